// oracle/streami_oracle.hpp
//
// TEST INFRASTRUCTURE ONLY.  Plain, slow, obviously-correct CPU implementation of the
// particle-update path of Streami (arxiv/paper_2606_02627): cell location + trilinear
// interpolation on a structured grid, linear interpolation in time, RK4 / Dormand-Prince
// 5(4) stepping, termination tests, vertex recording, streakline schedule and the
// brick (macrocell) hand-off rounds.  Only tests/, __graft_entry__.smoke() and bench.py's
// cpu_baseline / --impl reference legs may use it.  It shares no code with the CUDA
// library in paper_2606_02627_b200/ and neither includes the other.
//
// What it follows (file:line = /root/reference/PAPER.md; A1..A9 = the fp32 formula sheet of
// SURVEY.md 8(c), restated in DESIGN.md section 3):
//   * RK4 skeleton, "a failed sample ends the particle": Listing 1.
//   * trace loop / streakline schedule: Listing 2.
//   * sample() / destinationID() / macrocell + halo: PAPER.md:63-65; voxel array: PAPER.md:155.
//   * trilinear filter, time interpolation, |v| floor, DP5(4): the paper is silent,
//     BASELINE.json binds; readings Q1..Q21 of DESIGN.md.
//
// Every function is templated on the arithmetic type T (float = the parity reference for the
// GPU path, double = closed-form / convergence checks) and follows the sheet operation by
// operation: lerp(a,b,w) := fma(w, b-a, a); no blocking, fusion or reordering.  Compile with
// -ffp-contract=off so that only the fma's written here are fused.
//
// Pins (tests/test_oracle_pins.py): P1 constant field, P2 linear field, P3 8-term sum,
// P4 rigid rotation, P5 ABC(C=0) invariant, P6 v=a+bt, P7 double gyre, P8 DP5(4) tableau /
// polynomial / library cross-check / rp10, P9 bricks == monolithic, P10 invariants,
// P11 streakline == pathline.  Absolute trajectories in the turbulent fields and in chaotic
// ABC are "parity unpinned" by any closed form (pinned only by composition of the above).
#pragma once
#include <cmath>
#include <cstdint>
#include <cstring>
#include <vector>
#include <algorithm>

namespace oracle {

enum : uint32_t { ALIVE = 0, OUT_OF_DOMAIN = 1, MAX_STEPS = 2, STAGNANT = 3, HALO_MISS = 4 };
// internal return code of advance(): the particle left the brick's owned region (A9 rounds)
enum : uint32_t { HANDOFF = 100 };

template <class T> inline T lerp(T a, T b, T w) { return std::fma(w, b - a, a); }

// ---------------------------------------------------------------------------------------
// A1. Field and coordinates.  One stored array = the global grid (lo = 0, hi = N-1) or one
// brick's stored box [lo, hi] (A9).  `data` is the caller's packed fp32 AoS array with the
// dims of the STORED box, x fastest, slices outermost.
// ---------------------------------------------------------------------------------------
template <class T> struct GridField {
  int N[3];          // global vertex counts
  int lo[3], hi[3];  // stored box in global vertex indices (inclusive)
  T o[3], r[3], top[3];
  int nslices; T q, top_s; int time_mode;
  const float* data;

  void init(const int gdims[3], const int lo_[3], const int hi_[3], const float origin[3],
            const float spacing[3], int nslices_, float slice_dt, int time_mode_,
            const float* data_) {
    for (int a = 0; a < 3; ++a) {
      N[a] = gdims[a]; lo[a] = lo_[a]; hi[a] = hi_[a];
      o[a] = T(origin[a]);
      r[a] = T(1) / T(spacing[a]);   // A1: r_a = 1/d_a, computed once
      top[a] = T(N[a] - 1);
    }
    nslices = nslices_; q = T(1) / T(slice_dt); top_s = T(nslices - 1);
    time_mode = time_mode_; data = data_;
  }

  // A2 (+A9 brick form).  Returns 0 = ok, OUT_OF_DOMAIN or HALO_MISS.
  uint32_t sample_slice(int s, const T p[3], T v[3]) const {
    T g[3];
    for (int a = 0; a < 3; ++a) g[a] = (p[a] - o[a]) * r[a];               // A2.1
    bool ok = (g[0] >= T(0) && g[0] <= top[0]) && (g[1] >= T(0) && g[1] <= top[1]) &&
              (g[2] >= T(0) && g[2] <= top[2]);                            // A2.2 (NaN -> false)
    if (!ok) return OUT_OF_DOMAIN;
    int i[3]; T f[3];
    for (int a = 0; a < 3; ++a) {
      // A9: a brick serves lo <= g < hi, and g == hi only at the global top.
      bool in = g[a] >= T(lo[a]) && (g[a] < T(hi[a]) || (hi[a] == N[a] - 1 && g[a] <= T(hi[a])));
      if (!in) return HALO_MISS;
      i[a] = std::min(int(std::floor(g[a])), hi[a] - 1);                   // A2.3
      f[a] = g[a] - T(i[a]);
    }
    const size_t sx = size_t(hi[0] - lo[0] + 1), sy = size_t(hi[1] - lo[1] + 1),
                 sz = size_t(hi[2] - lo[2] + 1);
    const float* base = data + 3 * (size_t(s) * sz * sy * sx);
    T V[2][2][2][3];
    for (int dz = 0; dz < 2; ++dz)
      for (int dy = 0; dy < 2; ++dy)
        for (int dx = 0; dx < 2; ++dx) {                                   // A2.4
          size_t idx = (size_t(i[2] - lo[2] + dz) * sy + size_t(i[1] - lo[1] + dy)) * sx +
                       size_t(i[0] - lo[0] + dx);
          for (int c = 0; c < 3; ++c) V[dz][dy][dx][c] = T(base[3 * idx + c]);
        }
    for (int c = 0; c < 3; ++c) {                                          // A2.5: x, y, z
      T c00 = lerp(V[0][0][0][c], V[0][0][1][c], f[0]);
      T c01 = lerp(V[0][1][0][c], V[0][1][1][c], f[0]);
      T c10 = lerp(V[1][0][0][c], V[1][0][1][c], f[0]);
      T c11 = lerp(V[1][1][0][c], V[1][1][1][c], f[0]);
      T c0 = lerp(c00, c01, f[1]);
      T c1 = lerp(c10, c11, f[1]);
      v[c] = lerp(c0, c1, f[2]);
    }
    return 0;
  }

  // A3. Unsteady sample: space first, time last.
  uint32_t sample(const T p[3], T t, T v[3]) const {
    if (nslices == 1) return sample_slice(0, p, v);
    T s = t * q;
    s = std::min(std::max(s, T(0)), top_s);
    if (time_mode == 1) {                       // the paper's fields[(int)simTime]
      int j = std::min(int(std::floor(s)), nslices - 1);
      return sample_slice(j, p, v);
    }
    int j = std::min(int(std::floor(s)), nslices - 2);
    T a = s - T(j);
    T u0[3], u1[3];
    uint32_t rc = sample_slice(j, p, u0);
    if (rc) return rc;
    sample_slice(j + 1, p, u1);
    for (int c = 0; c < 3; ++c) v[c] = lerp(u0[c], u1[c], a);
    return 0;
  }

  // A2.2 alone: is p inside the global domain (used for p_new and for seeds).
  bool inside(const T p[3]) const {
    T g[3];
    for (int a = 0; a < 3; ++a) g[a] = (p[a] - o[a]) * r[a];
    return (g[0] >= T(0) && g[0] <= top[0]) && (g[1] >= T(0) && g[1] <= top[1]) &&
           (g[2] >= T(0) && g[2] <= top[2]);
  }
};

// A9. Owner of an in-domain position (destinationID, a "simple offset
// computation given the projected cell position and grid dimensions").
template <class T> struct BrickGrid {
  int N[3], nb[3], B[3];
  T o[3], r[3];
  int owner(const T p[3]) const {
    int b[3];
    for (int a = 0; a < 3; ++a) {
      T g = (p[a] - o[a]) * r[a];
      b[a] = std::min(int(std::floor(g)) / B[a], nb[a] - 1);
    }
    return (b[2] * nb[1] + b[1]) * nb[0] + b[0];
  }
};

// ---------------------------------------------------------------------------------------
// Analytic samplers (fp64/fp32 closed-form fields for the pins; never used for parity).
// kind: 0 constant c[0..2]; 1 linear v = A x + b (c[0..8] row-major A, c[9..11] b);
// 2 ABC (A,B,C = c[0..2]); 3 uniform-in-space polynomial in t: v_a = c[a] + c[3+a] t + c[6+a] t^4;
// 4 double gyre (A, eps, omega, wamp = c[0..3]).  Domain = world box [c_lo, c_hi].
// ---------------------------------------------------------------------------------------
template <class T> struct AnalyticField {
  int kind; double c[16]; double blo[3], bhi[3];
  bool inside(const T p[3]) const {
    for (int a = 0; a < 3; ++a)
      if (!(p[a] >= T(blo[a]) && p[a] <= T(bhi[a]))) return false;
    return true;
  }
  uint32_t sample(const T p[3], T t, T v[3]) const {
    if (!inside(p)) return OUT_OF_DOMAIN;
    const T PI = T(3.14159265358979323846);
    switch (kind) {
      case 0: for (int a = 0; a < 3; ++a) v[a] = T(c[a]); break;
      case 1: for (int a = 0; a < 3; ++a)
                v[a] = T(c[3 * a]) * p[0] + T(c[3 * a + 1]) * p[1] + T(c[3 * a + 2]) * p[2] + T(c[9 + a]);
              break;
      case 2: v[0] = T(c[0]) * std::sin(p[2]) + T(c[2]) * std::cos(p[1]);
              v[1] = T(c[1]) * std::sin(p[0]) + T(c[0]) * std::cos(p[2]);
              v[2] = T(c[2]) * std::sin(p[1]) + T(c[1]) * std::cos(p[0]);
              break;
      case 3: { T t2 = t * t, t4 = t2 * t2;
                for (int a = 0; a < 3; ++a) v[a] = T(c[a]) + T(c[3 + a]) * t + T(c[6 + a]) * t4; }
              break;
      case 4: { T A = T(c[0]), eps = T(c[1]), om = T(c[2]), wamp = T(c[3]);
                T a = eps * std::sin(om * t), b = T(1) - T(2) * a;
                T f = a * p[0] * p[0] + b * p[0];
                v[0] = -PI * A * std::sin(PI * f) * std::cos(PI * p[1]);
                v[1] = PI * A * std::cos(PI * f) * std::sin(PI * p[1]) * (T(2) * a * p[0] + b);
                v[2] = wamp * std::sin(PI * p[2]); }
              break;
      default: return OUT_OF_DOMAIN;
    }
    return 0;
  }
};

// ---------------------------------------------------------------------------------------
// Parameters, recording (A6) and per-run totals.
// ---------------------------------------------------------------------------------------
template <class T> struct Params {
  int integrator;      // 0 = RK4, 1 = DP5(4)
  T h, h_min, h_max, atol, rtol;
  uint32_t max_steps;
  T vmin, t0;
  uint32_t capacity, stride;
};

struct Totals { unsigned long long attempted = 0, accepted = 0, samples = 0, handoffs = 0; };

// A6: vertex k of particle `id` is stored iff k % stride == 0 and k/stride < capacity, at
// plane c element c*n*capacity + id*capacity + k/stride.
template <class T> struct Recorder {
  T* vertices; uint32_t* counts; size_t n; uint32_t capacity, stride;
  void record(size_t id, uint32_t k, const T p[3]) const {
    if (!vertices) return;
    if (k % stride != 0) return;
    uint32_t slot = k / stride;
    if (slot >= capacity) return;
    for (int c = 0; c < 3; ++c) vertices[(size_t(c) * n + id) * capacity + slot] = p[c];
    counts[id] = slot + 1;
  }
};

// Per-particle integrator state (what a hand-off record carries: position, id, step count;
// plus t, h for DP5(4)).
template <class T> struct State {
  T p[3]; uint32_t n; T t, h; T k1[3]; bool have_k1, rejected;
};

// ---------------------------------------------------------------------------------------
// A4 + A5 steps 2-6: fixed-step RK4 (Listing 1, with explicit h).
// step_base: the global step index of the particle's step 0 (streaklines: its birth step).
// Runs until the particle ends (returns its status) or `leaves(p)` says it left the brick
// (returns HANDOFF).  `cap` = number of steps after which status is MAX_STEPS.
// ---------------------------------------------------------------------------------------
template <class T, class F, class Leaves>
uint32_t advance_rk4(const F& fld, State<T>& st, const Params<T>& prm, uint32_t cap,
                     uint32_t step_base, size_t id, const Recorder<T>& rec, Totals& tot,
                     Leaves leaves) {
  const T h = prm.h, h2 = T(0.5) * h, h6 = h / T(6);       // A4: computed once
  const T vmin2 = prm.vmin * prm.vmin;
  T* p = st.p;
  for (;;) {
    if (st.n == cap) return MAX_STEPS;                                        // A5.2
    const T tn = prm.t0 + T(step_base + st.n) * h;                            // A4: not accumulated
    T k1[3], k2[3], k3[3], k4[3], q[3];
    uint32_t rc = fld.sample(p, tn, k1); tot.samples++;                       // A5.3
    if (rc) return rc;  // cannot happen for a p that passed the inside test (monolithic)
    T m = std::fma(k1[2], k1[2], std::fma(k1[1], k1[1], k1[0] * k1[0]));
    if (m < vmin2) return STAGNANT;
    tot.attempted++;
    for (int c = 0; c < 3; ++c) q[c] = std::fma(h2, k1[c], p[c]);             // A5.4
    rc = fld.sample(q, tn + h2, k2); tot.samples++; if (rc) return rc;
    for (int c = 0; c < 3; ++c) q[c] = std::fma(h2, k2[c], p[c]);
    rc = fld.sample(q, tn + h2, k3); tot.samples++; if (rc) return rc;
    for (int c = 0; c < 3; ++c) q[c] = std::fma(h, k3[c], p[c]);
    rc = fld.sample(q, tn + h, k4); tot.samples++; if (rc) return rc;
    T pn[3];
    for (int c = 0; c < 3; ++c) {
      T sum = (k1[c] + k4[c]) + T(2) * (k2[c] + k3[c]);
      pn[c] = std::fma(h6, sum, p[c]);
    }
    if (!fld.inside(pn)) return OUT_OF_DOMAIN;                                // A5.5: not recorded
    for (int c = 0; c < 3; ++c) p[c] = pn[c];                                 // A5.6
    st.n++; tot.accepted++;
    rec.record(id, st.n, p);
    if (leaves(p)) return HANDOFF;
  }
}

// ---------------------------------------------------------------------------------------
// A8: rp10(x) = x^(-1/10) without libm, identical op sequence on both sides.
// ---------------------------------------------------------------------------------------
inline float rp10(float x) {
  uint32_t bits; std::memcpy(&bits, &x, 4);
  int e = int((bits >> 23) & 0xffu) - 127;
  uint32_t mb = (bits & 0x007fffffu) | 0x3f800000u;
  float mnt; std::memcpy(&mnt, &mb, 4);
  int qd = (e >= 0) ? e / 10 : -((-e + 9) / 10);   // floor division
  int r = e - 10 * qd;
  static const float Tr[10] = {1.0f, 0.93303299f, 0.87055056f, 0.81225240f, 0.75785828f,
                               0.70710678f, 0.65975396f, 0.61557221f, 0.57434918f, 0.53588673f};
  float y = (0.02477176f * mnt + -0.14006647f) * mnt + 1.1145945f;
  y = y * Tr[r];
  y = std::ldexp(y, -qd);
  for (int it = 0; it < 2; ++it) {
    float y2 = y * y, y4 = y2 * y2, y8 = y4 * y4, y10 = y8 * y2;
    y = y * (1.1f - 0.1f * (x * y10));
  }
  return y;
}
inline double rp10(double x) {
  uint64_t bits; std::memcpy(&bits, &x, 8);
  int e = int((bits >> 52) & 0x7ffull) - 1023;
  uint64_t mb = (bits & 0x000fffffffffffffull) | 0x3ff0000000000000ull;
  double mnt; std::memcpy(&mnt, &mb, 8);
  int qd = (e >= 0) ? e / 10 : -((-e + 9) / 10);
  int r = e - 10 * qd;
  static const double Tr[10] = {1.0, 0.93303299, 0.87055056, 0.81225240, 0.75785828,
                                0.70710678, 0.65975396, 0.61557221, 0.57434918, 0.53588673};
  double y = (0.02477176 * mnt + -0.14006647) * mnt + 1.1145945;
  y = y * Tr[r];
  y = std::ldexp(y, -qd);
  for (int it = 0; it < 2; ++it) {
    double y2 = y * y, y4 = y2 * y2, y8 = y4 * y4, y10 = y8 * y2;
    y = y * (1.1 - 0.1 * (x * y10));
  }
  return y;
}

// Dormand-Prince 5(4) tableau as exact rationals rounded once to T (A8).
template <class T> struct DP {
  static constexpr T c2 = T(1.0 / 5.0), c3 = T(3.0 / 10.0), c4 = T(4.0 / 5.0), c5 = T(8.0 / 9.0);
  static constexpr T a21 = T(1.0 / 5.0);
  static constexpr T a31 = T(3.0 / 40.0), a32 = T(9.0 / 40.0);
  static constexpr T a41 = T(44.0 / 45.0), a42 = T(-56.0 / 15.0), a43 = T(32.0 / 9.0);
  static constexpr T a51 = T(19372.0 / 6561.0), a52 = T(-25360.0 / 2187.0),
                     a53 = T(64448.0 / 6561.0), a54 = T(-212.0 / 729.0);
  static constexpr T a61 = T(9017.0 / 3168.0), a62 = T(-355.0 / 33.0), a63 = T(46732.0 / 5247.0),
                     a64 = T(49.0 / 176.0), a65 = T(-5103.0 / 18656.0);
  static constexpr T b1 = T(35.0 / 384.0), b3 = T(500.0 / 1113.0), b4 = T(125.0 / 192.0),
                     b5 = T(-2187.0 / 6784.0), b6 = T(11.0 / 84.0);
  static constexpr T e1 = T(71.0 / 57600.0), e3 = T(-71.0 / 16695.0), e4 = T(71.0 / 1920.0),
                     e5 = T(-17253.0 / 339200.0), e6 = T(22.0 / 525.0), e7 = T(-1.0 / 40.0);
};

// ---------------------------------------------------------------------------------------
// A8: adaptive DP5(4) with the elementary controller.  Paper silent; BASELINE.json config 5.
// ---------------------------------------------------------------------------------------
template <class T, class F, class Leaves>
uint32_t advance_dp5(const F& fld, State<T>& st, const Params<T>& prm, uint32_t cap, size_t id,
                     const Recorder<T>& rec, Totals& tot, Leaves leaves) {
  typedef DP<T> D;
  const T vmin2 = prm.vmin * prm.vmin;
  const T LO = T(3.4867844e-11f), HI = T(3405062.9f), THIRD = T(1) / T(3);
  T* p = st.p;
  if (!st.have_k1) {
    uint32_t rc = fld.sample(p, st.t, st.k1); tot.samples++;
    if (rc) return rc;
    st.have_k1 = true;
  }
  for (;;) {
    if (st.n == cap) return MAX_STEPS;
    const T* k1 = st.k1;
    T m = std::fma(k1[2], k1[2], std::fma(k1[1], k1[1], k1[0] * k1[0]));
    if (m < vmin2) return STAGNANT;
    tot.attempted++;
    const T h = st.h, t = st.t;
    T k2[3], k3[3], k4[3], k5[3], k6[3], k7[3], P[3], pn[3], acc;
    uint32_t rc;
    for (int c = 0; c < 3; ++c) { acc = D::a21 * k1[c]; P[c] = std::fma(h, acc, p[c]); }
    rc = fld.sample(P, t + D::c2 * h, k2); tot.samples++; if (rc) return rc;
    for (int c = 0; c < 3; ++c) {
      acc = D::a31 * k1[c]; acc = std::fma(D::a32, k2[c], acc); P[c] = std::fma(h, acc, p[c]);
    }
    rc = fld.sample(P, t + D::c3 * h, k3); tot.samples++; if (rc) return rc;
    for (int c = 0; c < 3; ++c) {
      acc = D::a41 * k1[c]; acc = std::fma(D::a42, k2[c], acc); acc = std::fma(D::a43, k3[c], acc);
      P[c] = std::fma(h, acc, p[c]);
    }
    rc = fld.sample(P, t + D::c4 * h, k4); tot.samples++; if (rc) return rc;
    for (int c = 0; c < 3; ++c) {
      acc = D::a51 * k1[c]; acc = std::fma(D::a52, k2[c], acc); acc = std::fma(D::a53, k3[c], acc);
      acc = std::fma(D::a54, k4[c], acc); P[c] = std::fma(h, acc, p[c]);
    }
    rc = fld.sample(P, t + D::c5 * h, k5); tot.samples++; if (rc) return rc;
    for (int c = 0; c < 3; ++c) {
      acc = D::a61 * k1[c]; acc = std::fma(D::a62, k2[c], acc); acc = std::fma(D::a63, k3[c], acc);
      acc = std::fma(D::a64, k4[c], acc); acc = std::fma(D::a65, k5[c], acc);
      P[c] = std::fma(h, acc, p[c]);
    }
    rc = fld.sample(P, t + h, k6); tot.samples++; if (rc) return rc;
    for (int c = 0; c < 3; ++c) {
      acc = D::b1 * k1[c]; acc = std::fma(D::b3, k3[c], acc); acc = std::fma(D::b4, k4[c], acc);
      acc = std::fma(D::b5, k5[c], acc); acc = std::fma(D::b6, k6[c], acc);
      pn[c] = std::fma(h, acc, p[c]);
    }
    if (!fld.inside(pn)) return OUT_OF_DOMAIN;
    rc = fld.sample(pn, t + h, k7); tot.samples++; if (rc) return rc;
    T w[3];
    for (int c = 0; c < 3; ++c) {
      acc = D::e1 * k1[c]; acc = std::fma(D::e3, k3[c], acc); acc = std::fma(D::e4, k4[c], acc);
      acc = std::fma(D::e5, k5[c], acc); acc = std::fma(D::e6, k6[c], acc);
      acc = std::fma(D::e7, k7[c], acc);
      T E = h * acc;
      T sc = std::fma(prm.rtol, std::max(std::fabs(p[c]), std::fabs(pn[c])), prm.atol);
      w[c] = E / sc;
    }
    T err2 = std::fma(w[2], w[2], std::fma(w[1], w[1], w[0] * w[0])) * THIRD;
    bool accept = (err2 <= T(1)) || (h <= prm.h_min);
    T fac;
    if (err2 <= LO) fac = T(10);
    else if (err2 < HI) fac = T(0.9) * rp10(err2);
    else fac = T(0.2);
    if (accept) {
      for (int c = 0; c < 3; ++c) { p[c] = pn[c]; st.k1[c] = k7[c]; }
      st.t = t + h; st.n++; tot.accepted++;
      rec.record(id, st.n, p);
      if (st.rejected) fac = std::min(fac, T(1));
      st.h = std::min(std::max(h * fac, prm.h_min), prm.h_max);
      st.rejected = false;
      if (leaves(p)) return HANDOFF;
    } else {
      st.h = std::max(h * fac, prm.h_min);
      st.rejected = true;
    }
  }
}

struct NeverLeaves { template <class T> bool operator()(const T*) const { return false; } };

// ---------------------------------------------------------------------------------------
// A5: one streamline from seed to termination (monolithic field).
// ---------------------------------------------------------------------------------------
template <class T, class F>
void trace_one(const F& fld, const T seed[3], const Params<T>& prm, uint32_t cap,
               uint32_t step_base, size_t id, const Recorder<T>& rec, Totals& tot,
               uint32_t& steps, uint32_t& status, T fin[3]) {
  State<T> st;
  for (int c = 0; c < 3; ++c) st.p[c] = seed[c];
  st.n = 0; st.have_k1 = false; st.rejected = false;
  st.t = prm.t0; st.h = std::min(std::max(prm.h, prm.h_min), prm.h_max);
  if (!fld.inside(st.p)) {                                                    // A5.1
    steps = 0; status = OUT_OF_DOMAIN;
    for (int c = 0; c < 3; ++c) fin[c] = seed[c];
    return;
  }
  rec.record(id, 0, st.p);
  uint32_t rc = (prm.integrator == 0)
                    ? advance_rk4(fld, st, prm, cap, step_base, id, rec, tot, NeverLeaves())
                    : advance_dp5(fld, st, prm, cap, id, rec, tot, NeverLeaves());
  steps = st.n; status = rc;
  for (int c = 0; c < 3; ++c) fin[c] = st.p[c];
}

}  // namespace oracle
