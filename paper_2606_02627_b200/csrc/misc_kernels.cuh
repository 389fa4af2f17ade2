// csrc/misc_kernels.cuh -- layout repack, the stand-alone sampler entry and the streakline kernel.
#pragma once
#include "trace.cuh"

namespace streami {

// ---- field repack: caller's packed float3 -> library-owned layout (D6 of SURVEY.md) ---------
// One thread per vertex; reads are contiguous 12-byte triples, writes are 16/32-byte records.
static __global__ void repack_float4_kernel(const float* __restrict__ src, float4* __restrict__ dst,
                                     unsigned long long nvert) {
  unsigned long long v = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;
  const unsigned long long step = (unsigned long long)gridDim.x * blockDim.x;
  for (; v < nvert; v += step)
    dst[v] = make_float4(src[3 * v], src[3 * v + 1], src[3 * v + 2], 0.0f);
}

// SOA: three component planes of nvert floats each (nvert = all vertices of all slices).
static __global__ void repack_soa_kernel(const float* __restrict__ src, float* __restrict__ dst,
                                         unsigned long long nvert) {
  unsigned long long v = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;
  const unsigned long long step = (unsigned long long)gridDim.x * blockDim.x;
  for (; v < nvert; v += step) {
    dst[v] = src[3 * v]; dst[nvert + v] = src[3 * v + 1]; dst[2 * nvert + v] = src[3 * v + 2];
  }
}

// Tame scan: *flag |= 1 if any of the n floats is NaN, infinite or above 2^60 in magnitude.
static __global__ void tame_scan_kernel(const float* __restrict__ src, unsigned long long n, unsigned* flag) {
  unsigned long long i = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;
  const unsigned long long step = (unsigned long long)gridDim.x * blockDim.x;
  bool bad = false;
  for (; i < n; i += step) bad |= !(fabsf(src[i]) <= 1.152921504606846976e18f);
  if (__syncthreads_or(bad) && threadIdx.x == 0) atomicOr(flag, 1u);
}

// XPAIR record v = {Vx, Vy, Dx, Dy, Vz, Dz, 0, 0} with V = V[v], D = V[v+1] - V[v] (the difference is the x-lerp's own
// subtraction, done once here in fp32; see LayoutTraits in field.cuh); the last vertex of a row
// pairs with itself (its upper half is never used: i_x <= nx-2).
static __global__ void repack_xpair_kernel(const float* __restrict__ src, float4* __restrict__ dst,
                                    unsigned long long nvert, unsigned nx) {
  unsigned long long v = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;
  const unsigned long long step = (unsigned long long)gridDim.x * blockDim.x;
  for (; v < nvert; v += step) {
    unsigned long long w = ((v % nx) == nx - 1) ? v : v + 1;
    float a0 = src[3 * v], a1 = src[3 * v + 1], a2 = src[3 * v + 2];
    float b0 = src[3 * w], b1 = src[3 * w + 1], b2 = src[3 * w + 2];
    dst[2 * v] = make_float4(a0, a1, b0 - a0, b1 - a1);
    dst[2 * v + 1] = make_float4(a2, b2 - a2, 0.0f, 0.0f);
  }
}

// XYQUAD record v = {XPAIR row of vertex v, XPAIR row of the vertex one y-row up}: 64 bytes.  The
// last x of a row and the last y-row of a plane pair with themselves (never used: i <= N-2).
static __global__ void repack_xyquad_kernel(const float* __restrict__ src, float4* __restrict__ dst,
                                            unsigned long long nvert, unsigned nx, unsigned ny) {
  unsigned long long t = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;   // (vertex, half)
  const unsigned long long step = (unsigned long long)gridDim.x * blockDim.x;
  for (; t < 2ull * nvert; t += step) {
    unsigned long long v = t >> 1;
    const unsigned x = (unsigned)(v % nx), y = (unsigned)((v / nx) % ny);
    if ((t & 1ull) && y + 1 < ny) v += nx;
    const unsigned long long w = (x == nx - 1) ? v : v + 1;
    const float a0 = src[3 * v], a1 = src[3 * v + 1], a2 = src[3 * v + 2];
    const float b0 = src[3 * w], b1 = src[3 * w + 1], b2 = src[3 * w + 2];
    dst[2 * t] = make_float4(a0, a1, b0 - a0, b1 - a1);
    dst[2 * t + 1] = make_float4(a2, b2 - a2, 0.0f, 0.0f);
  }
}

// CELL record c = the four DIFF rows (dz*2+dy) of cell c as 24 consecutive floats {Vx, Vy, Dx, Dy, Vz, Dz} x 4,
// then 32 bytes of zero padding: 128 bytes, 8 corners, one L2 line (field.cuh).  One thread per (cell, row).
static __global__ void repack_cell_kernel(const float* __restrict__ src, float4* __restrict__ dst,
                                          unsigned nx, unsigned ny, unsigned nz, unsigned nslices) {
  const unsigned cx = nx - 1, cy = ny - 1, cz = nz - 1;
  const unsigned long long per_slice = (unsigned long long)cx * cy * cz;
  const unsigned long long total = 4ull * per_slice * nslices;
  unsigned long long t = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;
  const unsigned long long step = (unsigned long long)gridDim.x * blockDim.x;
  float2* out = reinterpret_cast<float2*>(dst);
  for (; t < total; t += step) {
    const unsigned r = (unsigned)(t & 3ull);
    unsigned long long c = t >> 2;
    const unsigned long long rec = c;
    const unsigned sl = (unsigned)(c / per_slice);
    c -= (unsigned long long)sl * per_slice;
    const unsigned ix = (unsigned)(c % cx), iy = (unsigned)((c / cx) % cy), iz = (unsigned)(c / ((unsigned long long)cx * cy));
    const unsigned long long v = (((unsigned long long)sl * nz + iz + (r >> 1)) * ny + iy + (r & 1u)) * nx + ix;
    const float* p = src + 3ull * v;
    float2* o = out + 16ull * rec + 3u * r;
    o[0] = make_float2(p[0], p[1]);
    o[1] = make_float2(p[3] - p[0], p[4] - p[1]);
    o[2] = make_float2(p[2], p[5] - p[2]);
    if (r == 3u) { dst[8ull * rec + 6] = make_float4(0.f, 0.f, 0.f, 0.f); dst[8ull * rec + 7] = make_float4(0.f, 0.f, 0.f, 0.f); }
  }
}

// ---- seed generation on a control shape (the paper's convenience kernels) ---
// Shape = o + u*eu + v*ev + w*ew, (u,v,w) in [0,1)^3, nu x nv x nw seeds, s = (k*nv + j)*nu + i.
// mode 0: lattice, u = ((float)i + 0.5f)/(float)nu (IEEE division).  mode 1: uniform random from a
// counter-based generator: U(s, a) = (float)(z >> 40) * 2^-24 with z the splitmix64 finaliser of
// rng_seed + (3 s + a + 1) * 0x9E3779B97F4A7C15.  p_c = fma(w, ew_c, fma(v, ev_c, fma(u, eu_c, o_c))).
struct SeedShape { float o[3], eu[3], ev[3], ew[3]; unsigned nu, nv, nw; int mode; unsigned long long rng_seed; };

__device__ __forceinline__ unsigned long long mix64(unsigned long long z) {
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
  return z ^ (z >> 31);
}

static __global__ void seed_shape_kernel(const SeedShape sh, float* __restrict__ out) {
  const unsigned long long total = (unsigned long long)sh.nu * sh.nv * sh.nw;
  unsigned long long s = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;
  const unsigned long long step = (unsigned long long)gridDim.x * blockDim.x;
  for (; s < total; s += step) {
    float u, v, w;
    if (sh.mode == 0) {
      const unsigned i = (unsigned)(s % sh.nu), j = (unsigned)((s / sh.nu) % sh.nv),
                     k = (unsigned)(s / ((unsigned long long)sh.nu * sh.nv));
      u = __fdiv_rn((float)i + 0.5f, (float)sh.nu); v = __fdiv_rn((float)j + 0.5f, (float)sh.nv);
      w = __fdiv_rn((float)k + 0.5f, (float)sh.nw);
    } else {
      const float S24 = 5.9604644775390625e-08f;   // 2^-24
      u = (float)(mix64(sh.rng_seed + (3ull * s + 1ull) * 0x9E3779B97F4A7C15ull) >> 40) * S24;
      v = (float)(mix64(sh.rng_seed + (3ull * s + 2ull) * 0x9E3779B97F4A7C15ull) >> 40) * S24;
      w = (float)(mix64(sh.rng_seed + (3ull * s + 3ull) * 0x9E3779B97F4A7C15ull) >> 40) * S24;
    }
#pragma unroll
    for (int c = 0; c < 3; ++c)
      out[3 * s + c] = __fmaf_rn(w, sh.ew[c], __fmaf_rn(v, sh.ev[c], __fmaf_rn(u, sh.eu[c], sh.o[c])));
  }
}

// ---- a2-a4 alone ----------------------------------------------------------------------------
template <int LAYOUT, bool UNSTEADY>
__global__ void sample_kernel(Geom g, Store s, const float* __restrict__ pts, unsigned long long n,
                              float t, float* __restrict__ out_v, unsigned* __restrict__ out_rc) {
  unsigned long long i = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  CellCache cc; cc.invalidate();
  float vx = 0.f, vy = 0.f, vz = 0.f;
  unsigned rc = sample<LAYOUT, UNSTEADY, false, false>(g, s, cc, pts[3 * i], pts[3 * i + 1],
                                                       pts[3 * i + 2], t, vx, vy, vz);
  if (rc) { vx = 0.f; vy = 0.f; vz = 0.f; }
  out_v[3 * i] = vx; out_v[3 * i + 1] = vy; out_v[3 * i + 2] = vz;
  out_rc[i] = rc;
}

// ---- a11 + a10 for streaklines (A7; Listing 2) -----------------------------
// One launch covers the global steps [s0, s1).  Particle id = j*m + i (release j, point i) is
// born at point i at global step j.  Its state between launches is its output slot (the last
// inside position is what the slot must hold anyway) plus one status byte.
template <bool T> struct StreakCache { typedef CellCache type; };
template <> struct StreakCache<true> { typedef CellCacheT type; };

struct StreakArgs {
  Geom g; Store s;
  const float* points; unsigned long long m; unsigned nsteps, s0, s1;
  float h, h2, h6, vmin2, t0;
  float* verts;                  // [3][nsteps][m]
  unsigned char* state;          // [nsteps*m] status, 0 = alive
  unsigned* steps;               // optional [nsteps*m]
  unsigned long long* totals;
};

// TCACHE (option "cell_cache"): the copy of the current cell (field.cuh; both slices of it for an
// unsteady field) stays in registers across the stages and steps of a window.
template <int LAYOUT, bool UNSTEADY, bool TCACHE>
__global__ void __launch_bounds__(256) streak_kernel(const StreakArgs a) {
  __shared__ unsigned long long s_tot[3];
  if (threadIdx.x < 3) s_tot[threadIdx.x] = 0ull;
  __syncthreads();
  const unsigned long long total = a.m * (unsigned long long)min(a.s1, a.nsteps);
  unsigned long long id = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (id < total) {
    const unsigned j = (unsigned)(id / a.m);
    const unsigned long long i = id - (unsigned long long)j * a.m;
    const unsigned long long plane = a.m * (unsigned long long)a.nsteps;
    float px, py, pz; unsigned st = ST_ALIVE; unsigned s = a.s0;
    bool run = true;
    if (j >= a.s0) {                                             // born in this window
      px = a.points[3 * i]; py = a.points[3 * i + 1]; pz = a.points[3 * i + 2];
      s = j;
      float gx, gy, gz;
      if (!to_index(a.g, px, py, pz, gx, gy, gz)) { st = ST_OUT; run = false; }
    } else {
      st = a.state[id];
      if (st != ST_ALIVE) run = false;
      else { px = a.verts[id]; py = a.verts[plane + id]; pz = a.verts[2 * plane + id]; }
    }
    if (run) {
      TraceArgs ta;                                              // only the fields rk4_step reads
      ta.g = a.g; ta.h = a.h; ta.h2 = a.h2; ta.h6 = a.h6; ta.vmin2 = a.vmin2;
      ta.max_steps = 0xffffffffu; ta.verts = nullptr; ta.cap = 0; ta.stride = 0xffffffffu; ta.prefetch = 0;
      Lane L; L.px = px; L.py = py; L.pz = pz; L.id = 0; L.slot = 0; L.rec_cd = 0xffffffffu;
      typename StreakCache<UNSTEADY && TCACHE>::type cc; cc.invalidate();
      unsigned n_samples = 0, n_attempts = 0;
      const unsigned s_first = s;
      for (; s < a.s1; ++s) {
        L.n = s;                                                 // t_s = t0 + (float)s*h, shared by all
        ta.t0 = a.t0;
        unsigned done;
        unsigned rc = rk4_step<LAYOUT, UNSTEADY, false, TCACHE, false, false>(ta, a.s, cc, L, done);
        if (rc) { st = rc; n_attempts = done >= 2u ? 1u : 0u; n_samples = min(done, 4u); break; }
      }
      n_attempts += s - s_first; n_samples += 4u * (s - s_first);
      if (st == ST_ALIVE && a.s1 >= a.nsteps) st = ST_MAXSTEPS;  // alive at the end
      px = L.px; py = L.py; pz = L.pz;
      atomicAdd(&s_tot[0], (unsigned long long)n_attempts);
      atomicAdd(&s_tot[1], (unsigned long long)(s - max(j, a.s0)));
      atomicAdd(&s_tot[2], (unsigned long long)n_samples);
    }
    if (run || j >= a.s0) {
      a.verts[id] = px; a.verts[plane + id] = py; a.verts[2 * plane + id] = pz;
      a.state[id] = (unsigned char)st;
      if (a.steps && st != ST_ALIVE) a.steps[id] = s - j;
    }
  }
  __syncthreads();
  if (a.totals && threadIdx.x < 3 && s_tot[threadIdx.x]) atomicAdd(a.totals + threadIdx.x, s_tot[threadIdx.x]);
}

// out_counts[i] = number of particles of point i alive at the end; copy status to u32.
// `released` = global steps executed (= nsteps for a complete run): later releases do not exist
// yet and report status 0; a particle still ALIVE in an unfinished run counts as alive.
static __global__ void streak_finalize_kernel(const unsigned char* __restrict__ state, unsigned long long m,
                                       unsigned nsteps, unsigned released, unsigned* __restrict__ counts,
                                       unsigned* __restrict__ status) {
  unsigned long long i = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= m) return;
  unsigned c = 0;
  for (unsigned j = 0; j < nsteps; ++j) {
    unsigned st = j < released ? state[(unsigned long long)j * m + i] : 0u;
    c += (j < released) && (st == ST_MAXSTEPS || st == ST_ALIVE);
    if (status) status[(unsigned long long)j * m + i] = st;
  }
  if (counts) counts[i] = c;
}

}  // namespace streami
