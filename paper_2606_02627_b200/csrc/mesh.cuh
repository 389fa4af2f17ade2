// csrc/mesh.cuh -- vector fields on hexahedral meshes: the paper's other field type
// ("unstructured meshes", cell location + interpolation).
// Written from the formula sheet U1-U4; shares nothing with oracle/.
// The translation unit is compiled with -fmad=false: every fused multiply-add is an explicit
// __fmaf_rn.  The paper locates cells with a BVH point query; a uniform bin grid gives the same
// located cell ("the first listed cell of the point's bin that contains it") with one table lookup.
//
// Layout: one 224-byte record per CELL -- the 8 corner positions [a][l] (24 floats), the 8 corner
// values [a][l] (24 floats), the cell's bounding box (6 floats), 2 pad -- so that testing and
// sampling a candidate cell is 7 contiguous sectors and no index indirection (the connectivity
// array H is consumed at create time).
#pragma once
#include <cuda_runtime.h>

#include "trace.cuh"

namespace streami {

constexpr int MESH_REC = 56;            // floats per cell record
constexpr int MESH_NEWTON = 6;          // U3: at most this many Newton steps
constexpr float MESH_TOL = 2e-5f;       // U3
// A list entry carries, next to the cell id, the cell's bounding box (grown by `margin` and a slack
// of MESH_BOX_SLACK bin widths, rounded outwards) in the coordinates of ITS bin, 1/256 bin width per
// unit, six int16: one 16-byte load per candidate decides whether the cell record is worth
// fetching.  The box only filters (any superset of the cells that can pass U3 gives the same
// located cell), so its own rounding does not matter as long as it errs outwards; the slack covers
// the fp32 rounding of the point's bin coordinate (<= 2 nb 2^-24 bin widths).
constexpr float MESH_BOX_SCALE = 256.0f;
#ifndef MESH_WALK
#define MESH_WALK 4                      // list entries fetched per round trip
#endif
constexpr double MESH_BOX_SLACK = 1.0 / 1024.0;

struct MeshDev {
  const float* cells;                   // [nc][MESH_REC]
  const unsigned* bin_start;            // [nbins + 1]
  const uint4* bin_items;               // {cell id, packed box}: see MESH_BOX_SCALE
  float lox, loy, loz, hix, hiy, hiz, sx, sy, sz;
  int nbx, nby, nbz;
  float margin;                         // what the packed boxes were grown by (build's choice, see hx_locate)
};

__device__ __forceinline__ void ldg256(const float* p, float* o) {   // p 32-byte aligned
  asm volatile("ld.global.nc.v8.f32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
               : "=f"(o[0]), "=f"(o[1]), "=f"(o[2]), "=f"(o[3]), "=f"(o[4]), "=f"(o[5]), "=f"(o[6]), "=f"(o[7])
               : "l"(p));
}

__device__ __forceinline__ float hx_tri(const float* Q, float x, float y, float z) {
  const float c00 = lerp(Q[0], Q[1], x), c01 = lerp(Q[2], Q[3], x);
  const float c10 = lerp(Q[4], Q[5], x), c11 = lerp(Q[6], Q[7], x);
  return lerp(lerp(c00, c01, y), lerp(c10, c11, y), z);
}
__device__ __forceinline__ float hx_cof(float u, float v, float w, float z) { return __fmaf_rn(u, v, -(w * z)); }

// U3: reference coordinates of p in the cell whose corner positions are P[a*8 + l].
__device__ __forceinline__ bool hx_invert(const float* __restrict__ P, float px, float py, float pz,
                                          float& x, float& y, float& z) {
  x = 0.5f; y = 0.5f; z = 0.5f;
  float dx = 0.0f, dy = 0.0f, dz = 0.0f;
  const float p[3] = {px, py, pz};
#pragma unroll 1
  for (int it = 0; it < MESH_NEWTON; ++it) {
    float G[3], Jx[3], Jy[3], Jz[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      const float* q = P + 8 * a;
      G[a] = hx_tri(q, x, y, z) - p[a];
      Jx[a] = lerp(lerp(q[1] - q[0], q[3] - q[2], y), lerp(q[5] - q[4], q[7] - q[6], y), z);
      Jy[a] = lerp(lerp(q[2] - q[0], q[3] - q[1], x), lerp(q[6] - q[4], q[7] - q[5], x), z);
      Jz[a] = lerp(lerp(q[4] - q[0], q[5] - q[1], x), lerp(q[6] - q[2], q[7] - q[3], x), y);
    }
    const float cxx = hx_cof(Jy[1], Jz[2], Jz[1], Jy[2]), cxy = hx_cof(Jz[0], Jy[2], Jy[0], Jz[2]),
                cxz = hx_cof(Jy[0], Jz[1], Jz[0], Jy[1]);
    const float cyx = hx_cof(Jz[1], Jx[2], Jx[1], Jz[2]), cyy = hx_cof(Jx[0], Jz[2], Jz[0], Jx[2]),
                cyz = hx_cof(Jz[0], Jx[1], Jx[0], Jz[1]);
    const float czx = hx_cof(Jx[1], Jy[2], Jy[1], Jx[2]), czy = hx_cof(Jy[0], Jx[2], Jx[0], Jy[2]),
                czz = hx_cof(Jx[0], Jy[1], Jy[0], Jx[1]);
    const float det = __fmaf_rn(Jx[2], cxz, __fmaf_rn(Jx[1], cxy, Jx[0] * cxx));
    const float r = __fdiv_rn(1.0f, det);
    dx = r * __fmaf_rn(G[2], cxz, __fmaf_rn(G[1], cxy, G[0] * cxx));
    dy = r * __fmaf_rn(G[2], cyz, __fmaf_rn(G[1], cyy, G[0] * cyx));
    dz = r * __fmaf_rn(G[2], czz, __fmaf_rn(G[1], czy, G[0] * czx));
    x = x - dx; y = y - dy; z = z - dz;
    if (fabsf(dx) <= MESH_TOL && fabsf(dy) <= MESH_TOL && fabsf(dz) <= MESH_TOL) break;   // U3: converged
  }
  const float t = MESH_TOL;
  const bool converged = fabsf(dx) <= t && fabsf(dy) <= t && fabsf(dz) <= t;
  return converged && (x >= -t && x <= 1.0f + t) && (y >= -t && y <= 1.0f + t) && (z >= -t && z <= 1.0f + t);
}

// U2 + U3.  Returns the located cell or -1; xi is valid when a cell is returned.
// The box pre-test only skips cells that cannot pass U3 (a converged xi inside the unit cube +- TOL
// maps into the bounding box +- TOL x its extent; the packed boxes are grown by `margin` = 50 times
// that, plus their own slack), so the located cell is the same with and without it.
template <bool VALUE>
__device__ __forceinline__ long long hx_locate_body(const MeshDev& m, float px, float py, float pz, float& x,
                                                    float& y, float& z, float* v) {
  if (!((px >= m.lox && px <= m.hix) && (py >= m.loy && py <= m.hiy) && (pz >= m.loz && pz <= m.hiz))) return -1;
  const int bx = min(__float2int_rd((px - m.lox) * m.sx), m.nbx - 1);
  const int by = min(__float2int_rd((py - m.loy) * m.sy), m.nby - 1);
  const int bz = min(__float2int_rd((pz - m.loz) * m.sz), m.nbz - 1);
  const unsigned id = ((unsigned)bz * m.nby + by) * m.nbx + bx;
  const unsigned k0 = m.bin_start[id], k1 = m.bin_start[id + 1];
  // the point in the coordinates of its bin, in box units (t - b is exact: both lie in [b, b+1])
  const float ux = ((px - m.lox) * m.sx - (float)bx) * MESH_BOX_SCALE;
  const float uy = ((py - m.loy) * m.sy - (float)by) * MESH_BOX_SCALE;
  const float uz = ((pz - m.loz) * m.sz - (float)bz) * MESH_BOX_SCALE;
  // The list is walked in order, MESH_WALK candidates at a time: the entries are fetched with independent
  // loads (the walk is a chain of dependent L2 reads and the kernel is bound by their latency), the
  // boxes are tested, and the survivors -- normally one -- go through U3 in list order.
  for (unsigned kb = k0; kb < k1; kb += (unsigned)MESH_WALK) {
    uint4 ent[MESH_WALK];
#pragma unroll
    for (int j = 0; j < MESH_WALK; ++j) ent[j] = kb + j < k1 ? __ldg(m.bin_items + kb + j) : make_uint4(0xffffffffu, 0u, 0u, 0u);
#pragma unroll
    for (int j = 0; j < MESH_WALK; ++j) {
      const unsigned cand = ent[j].x;
      if (cand == 0xffffffffu) continue;
      const float lx = (float)(short)(ent[j].y & 0xffffu), ly = (float)(short)(ent[j].y >> 16);
      const float lz = (float)(short)(ent[j].z & 0xffffu), hx = (float)(short)(ent[j].z >> 16);
      const float hy = (float)(short)(ent[j].w & 0xffffu), hz = (float)(short)(ent[j].w >> 16);
      if (ux < lx || ux > hx || uy < ly || uy > hy || uz < lz || uz > hz) continue;
      const float* rec = m.cells + (size_t)cand * MESH_REC;
      float P[24];             // records are 224 = 7 x 32 bytes: one 256-bit load per sector
#pragma unroll
      for (int i = 0; i < 24; i += 8) ldg256(rec + i, P + i);
      float Q[24];
      if (VALUE) {             // U4's operands, requested together with U3's (one round trip, not two)
#pragma unroll
        for (int i = 0; i < 24; i += 8) ldg256(rec + 24 + i, Q + i);
      }
      if (hx_invert(P, px, py, pz, x, y, z)) {
        if (VALUE) { v[0] = hx_tri(Q, x, y, z); v[1] = hx_tri(Q + 8, x, y, z); v[2] = hx_tri(Q + 16, x, y, z); }
        return (long long)cand;
      }
    }
  }
  return -1;
}

// S(p) on a mesh: located cell (or -1) and value.  One out-of-line copy serves the five call sites
// of the advection kernel (the inlined copies made it spill at 128 registers); the result comes back
// in registers.
struct HxSample { long long c; float vx, vy, vz; };
static __device__ __noinline__ HxSample hx_sample_call(const MeshDev& m, float px, float py, float pz) {
  HxSample r; float x, y, z, v[3] = {0.f, 0.f, 0.f};
  r.c = hx_locate_body<true>(m, px, py, pz, x, y, z, v);
  r.vx = v[0]; r.vy = v[1]; r.vz = v[2];
  return r;
}

// U4: value at reference coordinates xi of cell c.
__device__ __forceinline__ void hx_value(const MeshDev& m, long long c, float x, float y, float z, float& vx,
                                         float& vy, float& vz) {
  const float* rec = m.cells + (size_t)c * MESH_REC + 24;
  float Q[24];
#pragma unroll
  for (int i = 0; i < 24; i += 4) {
    const float4 q = __ldg(reinterpret_cast<const float4*>(rec + i));
    Q[i] = q.x; Q[i + 1] = q.y; Q[i + 2] = q.z; Q[i + 3] = q.w;
  }
  vx = hx_tri(Q, x, y, z); vy = hx_tri(Q + 8, x, y, z); vz = hx_tri(Q + 16, x, y, z);
}

// a2-a4 alone on a mesh
static __global__ void mesh_sample_kernel(const MeshDev m, const float* __restrict__ pts, unsigned long long n,
                                          float* __restrict__ out_v, long long* __restrict__ out_cell) {
  unsigned long long i = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  float x, y, z, vx = 0.f, vy = 0.f, vz = 0.f;
  const long long c = hx_locate_body<false>(m, pts[3 * i], pts[3 * i + 1], pts[3 * i + 2], x, y, z, nullptr);
  if (c >= 0) hx_value(m, c, x, y, z, vx, vy, vz);
  out_v[3 * i] = vx; out_v[3 * i + 1] = vy; out_v[3 * i + 2] = vz;
  if (out_cell) out_cell[i] = c;
}

struct MeshTraceArgs {
  MeshDev m;
  const float* seeds; unsigned long long n;
  const unsigned* perm;                 // optional processing order (Morton sort of the seeds' bins), or NULL
  unsigned long long* next;             // global work counter (zeroed by the host)
  float h, h2, h6, vmin2; unsigned max_steps;
  float* verts; unsigned cap, stride;
  unsigned* counts; unsigned* steps; unsigned* status; float* fin;
  unsigned long long* totals;
};

// RK4 streamlines on a mesh (A4-A6 with S := the mesh sample, "inside" := a cell is located).
// Persistent grid, one lane per particle; a lane whose particle has ended takes the next work item
// from a global counter, so that all lanes of a warp take one RK4 step per iteration.  The sample
// taken at p_new for the exit test (A5.5) is the next step's k1 (the same point: the same result).
static __global__ void __launch_bounds__(128) mesh_trace_kernel(const __grid_constant__ MeshTraceArgs a) {
  __shared__ unsigned long long s_tot[3];
  if (threadIdx.x < 3) s_tot[threadIdx.x] = 0ull;
  __syncthreads();
  const unsigned long long plane = a.n * a.cap;
  unsigned long long id = 0;
  float px = 0.f, py = 0.f, pz = 0.f, k1x = 0.f, k1y = 0.f, k1z = 0.f;
  unsigned n = 0, slot = 0, samples = 0, attempts = 0;
  bool active = false, exhausted = false;
  auto record = [&](unsigned k) {
    if (k % a.stride == 0u && k / a.stride < a.cap) {
      if (a.verts) { const unsigned long long o = id * a.cap + k / a.stride; a.verts[o] = px; a.verts[plane + o] = py; a.verts[2 * plane + o] = pz; }
      slot = k / a.stride + 1u;
    }
  };
  auto finish = [&](unsigned st) {
    if (a.counts) a.counts[id] = slot;
    if (a.steps) a.steps[id] = n;
    if (a.status) a.status[id] = st;
    if (a.fin) { a.fin[id] = px; a.fin[a.n + id] = py; a.fin[2 * a.n + id] = pz; }
    atomicAdd(&s_tot[0], (unsigned long long)attempts);
    atomicAdd(&s_tot[1], (unsigned long long)n);
    atomicAdd(&s_tot[2], (unsigned long long)samples);
    active = false;
  };
  for (;;) {
    if (!active && !exhausted) {                                                // a1: refill
      const unsigned long long w = atomicAdd(a.next, 1ull);
      if (w >= a.n) exhausted = true;
      else {
        id = a.perm ? a.perm[w] : w;
        px = a.seeds[3 * id]; py = a.seeds[3 * id + 1]; pz = a.seeds[3 * id + 2];
        n = 0; slot = 0; samples = 0; attempts = 0; active = true;
        const HxSample s0 = hx_sample_call(a.m, px, py, pz);
        k1x = s0.vx; k1y = s0.vy; k1z = s0.vz;
        if (s0.c < 0) finish(ST_OUT);                                           // A5.1
        else record(0u);
      }
    }
    if (__all_sync(0xffffffffu, !active)) {
      if (__all_sync(0xffffffffu, exhausted)) break;
      continue;
    }
    if (active) {
      unsigned st = ST_ALIVE;
      do {
        if (n == a.max_steps) { st = ST_MAXSTEPS; break; }                      // A5.2
        samples++;                                                              // k1 = S(p), carried
        const float mm = __fmaf_rn(k1z, k1z, __fmaf_rn(k1y, k1y, k1x * k1x));   // A5.3
        if (mm < a.vmin2) { st = ST_STAGNANT; break; }
        attempts++;
        float qx = __fmaf_rn(a.h2, k1x, px), qy = __fmaf_rn(a.h2, k1y, py), qz = __fmaf_rn(a.h2, k1z, pz);
        const HxSample s2 = hx_sample_call(a.m, qx, qy, qz); samples++;
        if (s2.c < 0) { st = ST_OUT; break; }
        qx = __fmaf_rn(a.h2, s2.vx, px); qy = __fmaf_rn(a.h2, s2.vy, py); qz = __fmaf_rn(a.h2, s2.vz, pz);
        const HxSample s3 = hx_sample_call(a.m, qx, qy, qz); samples++;
        if (s3.c < 0) { st = ST_OUT; break; }
        qx = __fmaf_rn(a.h, s3.vx, px); qy = __fmaf_rn(a.h, s3.vy, py); qz = __fmaf_rn(a.h, s3.vz, pz);
        const HxSample s4 = hx_sample_call(a.m, qx, qy, qz); samples++;
        if (s4.c < 0) { st = ST_OUT; break; }
        const float sx = (k1x + s4.vx) + 2.0f * (s2.vx + s3.vx);
        const float sy = (k1y + s4.vy) + 2.0f * (s2.vy + s3.vy);
        const float sz = (k1z + s4.vz) + 2.0f * (s2.vz + s3.vz);
        const float nx = __fmaf_rn(a.h6, sx, px), ny = __fmaf_rn(a.h6, sy, py), nz = __fmaf_rn(a.h6, sz, pz);
        const HxSample s5 = hx_sample_call(a.m, nx, ny, nz);                    // A5.5
        if (s5.c < 0) { st = ST_OUT; break; }
        px = nx; py = ny; pz = nz; k1x = s5.vx; k1y = s5.vy; k1z = s5.vz; n++;  // A5.6
        record(n);
      } while (false);
      if (st != ST_ALIVE) finish(st);
    }
  }
  __syncthreads();
  if (a.totals && threadIdx.x < 3 && s_tot[threadIdx.x]) atomicAdd(a.totals + threadIdx.x, s_tot[threadIdx.x]);
}

}  // namespace streami
