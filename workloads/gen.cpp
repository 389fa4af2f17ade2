// workloads/gen.cpp -- seeded synthetic INPUT generators (host side).
//
// This module holds none of the traced method's arithmetic (no interpolation,
// no integrator, no termination logic). It only produces the inputs that both
// the CPU oracle (oracle/) and the CUDA library (paper_2606_02627_b200/) are
// fed with: uniform random numbers, seed positions and sampled vector fields.
// Recipes: SURVEY.md 8(d) "Synthetic inputs"; restated in DESIGN.md section 4.
//
// Randomness: std::mt19937_64 raw 64-bit outputs only, u = (raw >> 11) * 2^-53
// (the engine is fixed by the C++ standard; std:: distributions are not
// portable and are not used). Field values are computed in fp64 and rounded
// once to fp32.
#include <cmath>
#include <cstdint>
#include <cstddef>
#include <random>
#include <vector>

extern "C" {

// n uniforms in [0,1) from engine seed `seed`, skipping the first `skip` draws.
void wl_uniform(uint64_t seed, uint64_t skip, uint64_t n, double* out) {
  std::mt19937_64 eng(seed);
  if (skip) eng.discard(skip);
  for (uint64_t i = 0; i < n; ++i) out[i] = double(eng() >> 11) * 0x1.0p-53;
}

// n seeds, three uniforms per seed in x,y,z order: p_a = u * ext_a (fp64),
// rounded to fp32, clamped to (float)ext_a. out is [n][3] fp32 (AoS).
void wl_seeds_uniform(uint64_t seed, uint64_t n, const double ext[3], float* out) {
  std::mt19937_64 eng(seed);
  for (uint64_t i = 0; i < n; ++i)
    for (int a = 0; a < 3; ++a) {
      double u = double(eng() >> 11) * 0x1.0p-53;
      float p = float(u * ext[a]);
      float top = float(ext[a]);
      out[3 * i + a] = p > top ? top : p;
    }
}

// ABC flow u = A sin z + C cos y, v = B sin x + A cos z, w = C sin y + B cos x
// at the N^3 vertices of [0,L]^3, vertex i at i * L/(N-1). out [N][N][N][3], x fastest.
void wl_abc_fill(int N, double L, double A, double B, double C, float* out) {
  const double d = L / double(N - 1);
#pragma omp parallel for schedule(static)
  for (int z = 0; z < N; ++z)
    for (int y = 0; y < N; ++y)
      for (int x = 0; x < N; ++x) {
        double X = x * d, Y = y * d, Z = z * d;
        size_t o = 3 * ((size_t(z) * N + y) * N + x);
        out[o + 0] = float(A * std::sin(Z) + C * std::cos(Y));
        out[o + 1] = float(B * std::sin(X) + A * std::cos(Z));
        out[o + 2] = float(C * std::sin(Y) + B * std::cos(X));
      }
}

// Turbulence mode table (SURVEY.md 8(d) "Turbulence generator"). For mode m draw
// five uniforms in this order: kmag, cos(theta), azimuth, polarisation, phase.
// Row m of `table` (8 doubles): kvec[3] = 2 pi kmag khat / N (radians per vertex),
// ampvec[3] = kmag^(-5/6) * e (e unit, e . khat = 0), phi, kmag.
void wl_turb_modes(uint64_t seed, int M, double kmin, double kmax, int N, double* table) {
  std::mt19937_64 eng(seed);
  auto U = [&]() { return double(eng() >> 11) * 0x1.0p-53; };
  const double PI = 3.14159265358979323846;
  for (int m = 0; m < M; ++m) {
    double u1 = U(), u2 = U(), u3 = U(), u4 = U(), u5 = U();
    double kmag = kmin + (kmax - kmin) * u1;
    double ct = 2.0 * u2 - 1.0, st = std::sqrt(std::fmax(0.0, 1.0 - ct * ct));
    double ph = 2.0 * PI * u3;
    double kh[3] = {st * std::cos(ph), st * std::sin(ph), ct};
    double ps = 2.0 * PI * u4, phi = 2.0 * PI * u5;
    // e1 = normalize(khat x z) (khat x x if |ct| > 0.999), e2 = khat x e1
    double ax[3] = {0, 0, 1};
    if (std::fabs(ct) > 0.999) { ax[0] = 1; ax[2] = 0; }
    double e1[3] = {kh[1] * ax[2] - kh[2] * ax[1], kh[2] * ax[0] - kh[0] * ax[2],
                    kh[0] * ax[1] - kh[1] * ax[0]};
    double n1 = std::sqrt(e1[0] * e1[0] + e1[1] * e1[1] + e1[2] * e1[2]);
    for (double& c : e1) c /= n1;
    double e2[3] = {kh[1] * e1[2] - kh[2] * e1[1], kh[2] * e1[0] - kh[0] * e1[2],
                    kh[0] * e1[1] - kh[1] * e1[0]};
    double amp = std::pow(kmag, -5.0 / 6.0);
    double* r = table + 8 * size_t(m);
    for (int a = 0; a < 3; ++a) {
      r[a] = 2.0 * PI * kmag * kh[a] / double(N);
      r[3 + a] = amp * (std::cos(ps) * e1[a] + std::sin(ps) * e2[a]);
    }
    r[6] = phi;
    r[7] = kmag;
  }
}

// Direct (one cos per vertex and mode) unnormalised fill in fp64:
// v(x) = sum_m ampvec_m cos(kvec_m . x + phi_m) at integer vertex coordinates of
// the box [lo, lo+dims). out64 is [dz][dy][dx][3] doubles. Returns sum |v|^2.
double wl_turb_fill_direct(const int dims[3], const int lo[3], int M, const double* table,
                           double* out64) {
  const int nx = dims[0], ny = dims[1], nz = dims[2];
  double total = 0.0;
#pragma omp parallel for schedule(static) reduction(+ : total)
  for (int z = 0; z < nz; ++z)
    for (int y = 0; y < ny; ++y)
      for (int x = 0; x < nx; ++x) {
        double X = x + lo[0], Y = y + lo[1], Z = z + lo[2];
        double v[3] = {0, 0, 0};
        for (int m = 0; m < M; ++m) {
          const double* r = table + 8 * size_t(m);
          double c = std::cos(r[0] * X + r[1] * Y + r[2] * Z + r[6]);
          v[0] += r[3] * c; v[1] += r[4] * c; v[2] += r[5] * c;
        }
        size_t o = 3 * ((size_t(z) * ny + y) * nx + x);
        out64[o] = v[0]; out64[o + 1] = v[1]; out64[o + 2] = v[2];
        total += v[0] * v[0] + v[1] * v[1] + v[2] * v[2];
      }
  return total;
}

// out32 = float(scale * in64), elementwise.
void wl_scale_round(size_t n, const double* in64, double scale, float* out32) {
#pragma omp parallel for schedule(static)
  for (size_t i = 0; i < n; ++i) out32[i] = float(scale * in64[i]);
}

// 3D-extended double gyre (BASELINE.json config 4): stream function
// psi = A sin(pi f) sin(pi y), f = a x^2 + b x, a = eps sin(omega t), b = 1 - 2 a:
// u = -pi A sin(pi f) cos(pi y), v = pi A cos(pi f) sin(pi y) (2 a x + b),
// w = wamp sin(pi z). Vertices over [0,2]x[0,1]x[0,1]; slice k at t = k*dt.
// out is [nslices][nz][ny][nx][3].
void wl_double_gyre_fill(const int dims[3], int nslices, double dt, double A, double eps,
                         double omega, double wamp, float* out) {
  const int nx = dims[0], ny = dims[1], nz = dims[2];
  const double PI = 3.14159265358979323846;
  const double dx = 2.0 / (nx - 1), dy = 1.0 / (ny - 1), dz = 1.0 / (nz - 1);
#pragma omp parallel for schedule(static) collapse(2)
  for (int s = 0; s < nslices; ++s)
    for (int z = 0; z < nz; ++z) {
      double t = s * dt;
      double a = eps * std::sin(omega * t), b = 1.0 - 2.0 * a;
      for (int y = 0; y < ny; ++y)
        for (int x = 0; x < nx; ++x) {
          double X = x * dx, Y = y * dy, Z = z * dz;
          double f = a * X * X + b * X;
          size_t o = 3 * (((size_t(s) * nz + z) * ny + y) * nx + x);
          // wall rows are set to exact zeros where the analytic value is zero
          double sy = (y == 0 || y == ny - 1) ? 0.0 : std::sin(PI * Y);
          double sz = (z == 0 || z == nz - 1) ? 0.0 : std::sin(PI * Z);
          out[o + 0] = float(-PI * A * std::sin(PI * f) * std::cos(PI * Y));
          out[o + 1] = float(PI * A * std::cos(PI * f) * sy * (2.0 * a * X + b));
          out[o + 2] = float(wamp * sz);
        }
    }
}

}  // extern "C"
