// csrc/dp5.cuh -- adaptive Dormand-Prince 5(4) attempt (a5, config 5).  The paper has no
// adaptive integrator (Listing 1 is classical RK4); BASELINE.json config 5 asks for one and the
// formula sheet A8 fixes tableau, error norm, controller and the libm-free
// x^(-1/10).  Written from that sheet; -fmad=false, explicit __fmaf_rn only.
#pragma once
#include "trace.cuh"

namespace streami {

namespace dp {
constexpr float c2 = (float)(1.0 / 5.0), c3 = (float)(3.0 / 10.0), c4 = (float)(4.0 / 5.0),
                c5 = (float)(8.0 / 9.0);
constexpr float a21 = (float)(1.0 / 5.0);
constexpr float a31 = (float)(3.0 / 40.0), a32 = (float)(9.0 / 40.0);
constexpr float a41 = (float)(44.0 / 45.0), a42 = (float)(-56.0 / 15.0), a43 = (float)(32.0 / 9.0);
constexpr float a51 = (float)(19372.0 / 6561.0), a52 = (float)(-25360.0 / 2187.0),
                a53 = (float)(64448.0 / 6561.0), a54 = (float)(-212.0 / 729.0);
constexpr float a61 = (float)(9017.0 / 3168.0), a62 = (float)(-355.0 / 33.0),
                a63 = (float)(46732.0 / 5247.0), a64 = (float)(49.0 / 176.0),
                a65 = (float)(-5103.0 / 18656.0);
constexpr float b1 = (float)(35.0 / 384.0), b3 = (float)(500.0 / 1113.0), b4 = (float)(125.0 / 192.0),
                b5 = (float)(-2187.0 / 6784.0), b6 = (float)(11.0 / 84.0);
constexpr float e1 = (float)(71.0 / 57600.0), e3 = (float)(-71.0 / 16695.0),
                e4 = (float)(71.0 / 1920.0), e5 = (float)(-17253.0 / 339200.0),
                e6 = (float)(22.0 / 525.0), e7 = (float)(-1.0 / 40.0);
}  // namespace dp

// A8: x^(-1/10) from the bits of x: quadratic seed on the mantissa, a table for the exponent
// residue, two Newton rounds.  Only IEEE mul/add/sub, so it is reproducible anywhere.
__device__ __forceinline__ float rp10(float x) {
  unsigned bits = __float_as_uint(x);
  int e = (int)((bits >> 23) & 0xffu) - 127;
  float mnt = __uint_as_float((bits & 0x007fffffu) | 0x3f800000u);
  int qd = (e >= 0) ? e / 10 : -((-e + 9) / 10);
  int r = e - 10 * qd;
  float tr;
  switch (r) {
    case 0: tr = 1.0f; break;        case 1: tr = 0.93303299f; break;
    case 2: tr = 0.87055056f; break; case 3: tr = 0.81225240f; break;
    case 4: tr = 0.75785828f; break; case 5: tr = 0.70710678f; break;
    case 6: tr = 0.65975396f; break; case 7: tr = 0.61557221f; break;
    case 8: tr = 0.57434918f; break; default: tr = 0.53588673f; break;
  }
  float y = (0.02477176f * mnt + -0.14006647f) * mnt + 1.1145945f;
  y = y * tr;
  y = y * __uint_as_float((unsigned)(127 - qd) << 23);   // exact scaling by 2^-qd
#pragma unroll
  for (int it = 0; it < 2; ++it) {
    float y2 = y * y, y4 = y2 * y2, y8 = y4 * y4, y10 = y8 * y2;
    y = y * (1.1f - 0.1f * (x * y10));
  }
  return y;
}

#define STREAMI_S(PX, PY, PZ, T, KX, KY, KZ)                                                   \
  rc = sample<LAYOUT, UNSTEADY, BRICK, CACHE, UNIT>(a.g, s, cc, PX, PY, PZ, T, KX, KY, KZ);    \
  n_samples++;                                                                                 \
  if (rc) return rc;

// One DP5(4) attempt.  L.k1 holds k1 (FSAL).  Returns 0 to continue, else the final status.
template <int LAYOUT, bool UNSTEADY, bool BRICK, bool CACHE, bool UNIT, class CC = CellCache>
__device__ __forceinline__ unsigned dp5_attempt(const TraceArgs& a, const Store& s, CC& cc,
                                                Lane& L, unsigned& n_samples, unsigned& n_attempts) {
  if (L.n == a.max_steps) return ST_MAXSTEPS;
  const float k1x = L.k1x, k1y = L.k1y, k1z = L.k1z;
  float m = __fmaf_rn(k1z, k1z, __fmaf_rn(k1y, k1y, k1x * k1x));
  if (m < a.vmin2) return ST_STAGNANT;
  n_attempts++;
  const float h = L.h, t = L.t, px = L.px, py = L.py, pz = L.pz;
  unsigned rc;
  float k2x, k2y, k2z, k3x, k3y, k3z, k4x, k4y, k4z, k5x, k5y, k5z, k6x, k6y, k6z, k7x, k7y, k7z;
  float ax, ay, az;
  ax = dp::a21 * k1x; ay = dp::a21 * k1y; az = dp::a21 * k1z;
  STREAMI_S(__fmaf_rn(h, ax, px), __fmaf_rn(h, ay, py), __fmaf_rn(h, az, pz), t + dp::c2 * h, k2x, k2y, k2z)
  ax = __fmaf_rn(dp::a32, k2x, dp::a31 * k1x); ay = __fmaf_rn(dp::a32, k2y, dp::a31 * k1y);
  az = __fmaf_rn(dp::a32, k2z, dp::a31 * k1z);
  STREAMI_S(__fmaf_rn(h, ax, px), __fmaf_rn(h, ay, py), __fmaf_rn(h, az, pz), t + dp::c3 * h, k3x, k3y, k3z)
  ax = __fmaf_rn(dp::a43, k3x, __fmaf_rn(dp::a42, k2x, dp::a41 * k1x));
  ay = __fmaf_rn(dp::a43, k3y, __fmaf_rn(dp::a42, k2y, dp::a41 * k1y));
  az = __fmaf_rn(dp::a43, k3z, __fmaf_rn(dp::a42, k2z, dp::a41 * k1z));
  STREAMI_S(__fmaf_rn(h, ax, px), __fmaf_rn(h, ay, py), __fmaf_rn(h, az, pz), t + dp::c4 * h, k4x, k4y, k4z)
  ax = __fmaf_rn(dp::a54, k4x, __fmaf_rn(dp::a53, k3x, __fmaf_rn(dp::a52, k2x, dp::a51 * k1x)));
  ay = __fmaf_rn(dp::a54, k4y, __fmaf_rn(dp::a53, k3y, __fmaf_rn(dp::a52, k2y, dp::a51 * k1y)));
  az = __fmaf_rn(dp::a54, k4z, __fmaf_rn(dp::a53, k3z, __fmaf_rn(dp::a52, k2z, dp::a51 * k1z)));
  STREAMI_S(__fmaf_rn(h, ax, px), __fmaf_rn(h, ay, py), __fmaf_rn(h, az, pz), t + dp::c5 * h, k5x, k5y, k5z)
  ax = __fmaf_rn(dp::a65, k5x, __fmaf_rn(dp::a64, k4x, __fmaf_rn(dp::a63, k3x, __fmaf_rn(dp::a62, k2x, dp::a61 * k1x))));
  ay = __fmaf_rn(dp::a65, k5y, __fmaf_rn(dp::a64, k4y, __fmaf_rn(dp::a63, k3y, __fmaf_rn(dp::a62, k2y, dp::a61 * k1y))));
  az = __fmaf_rn(dp::a65, k5z, __fmaf_rn(dp::a64, k4z, __fmaf_rn(dp::a63, k3z, __fmaf_rn(dp::a62, k2z, dp::a61 * k1z))));
  STREAMI_S(__fmaf_rn(h, ax, px), __fmaf_rn(h, ay, py), __fmaf_rn(h, az, pz), t + h, k6x, k6y, k6z)
  ax = __fmaf_rn(dp::b6, k6x, __fmaf_rn(dp::b5, k5x, __fmaf_rn(dp::b4, k4x, __fmaf_rn(dp::b3, k3x, dp::b1 * k1x))));
  ay = __fmaf_rn(dp::b6, k6y, __fmaf_rn(dp::b5, k5y, __fmaf_rn(dp::b4, k4y, __fmaf_rn(dp::b3, k3y, dp::b1 * k1y))));
  az = __fmaf_rn(dp::b6, k6z, __fmaf_rn(dp::b5, k5z, __fmaf_rn(dp::b4, k4z, __fmaf_rn(dp::b3, k3z, dp::b1 * k1z))));
  const float nx = __fmaf_rn(h, ax, px), ny = __fmaf_rn(h, ay, py), nz = __fmaf_rn(h, az, pz);
  {
    float gx, gy, gz;
    if (!to_index<UNIT>(a.g, nx, ny, nz, gx, gy, gz)) return ST_OUT;
  }
  STREAMI_S(nx, ny, nz, t + h, k7x, k7y, k7z)
  // error vector, scale, RMS norm (squared)
  float Ex = h * __fmaf_rn(dp::e7, k7x, __fmaf_rn(dp::e6, k6x, __fmaf_rn(dp::e5, k5x, __fmaf_rn(dp::e4, k4x, __fmaf_rn(dp::e3, k3x, dp::e1 * k1x)))));
  float Ey = h * __fmaf_rn(dp::e7, k7y, __fmaf_rn(dp::e6, k6y, __fmaf_rn(dp::e5, k5y, __fmaf_rn(dp::e4, k4y, __fmaf_rn(dp::e3, k3y, dp::e1 * k1y)))));
  float Ez = h * __fmaf_rn(dp::e7, k7z, __fmaf_rn(dp::e6, k6z, __fmaf_rn(dp::e5, k5z, __fmaf_rn(dp::e4, k4z, __fmaf_rn(dp::e3, k3z, dp::e1 * k1z)))));
  float wx = __fdiv_rn(Ex, __fmaf_rn(a.rtol, fmaxf(fabsf(px), fabsf(nx)), a.atol));
  float wy = __fdiv_rn(Ey, __fmaf_rn(a.rtol, fmaxf(fabsf(py), fabsf(ny)), a.atol));
  float wz = __fdiv_rn(Ez, __fmaf_rn(a.rtol, fmaxf(fabsf(pz), fabsf(nz)), a.atol));
  const float THIRD = 1.0f / 3.0f;
  float err2 = __fmaf_rn(wz, wz, __fmaf_rn(wy, wy, wx * wx)) * THIRD;
  bool accept = (err2 <= 1.0f) || (h <= a.hmin);
  float fac;
  if (err2 <= 3.4867844e-11f) fac = 10.0f;
  else if (err2 < 3405062.9f) fac = 0.9f * rp10(err2);
  else fac = 0.2f;                                       // NaN lands here
  if (accept) {
    L.px = nx; L.py = ny; L.pz = nz; L.k1x = k7x; L.k1y = k7y; L.k1z = k7z;   // FSAL
    L.t = t + h; L.n++;
    record_vertex<true, DP5_THREADS>(a, L);
    if (L.rejected) fac = fminf(fac, 1.0f);
    L.h = fminf(fmaxf(h * fac, a.hmin), a.hmax);
    L.rejected = false;
  } else {
    L.h = fmaxf(h * fac, a.hmin);
    L.rejected = true;
  }
  return 0;
}
#undef STREAMI_S

}  // namespace streami
