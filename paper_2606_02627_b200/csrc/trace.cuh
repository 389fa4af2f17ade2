// csrc/trace.cuh -- the advection kernel (a1, a5-a10 of SURVEY.md 8(a)).
//
// The paper's update() kernel (Listing 1) advances every particle by ONE RK4
// step per launch and hands all of them to an all-to-all after each step.
// This kernel is a B200 re-design of the same computation: a persistent grid sized to the
// machine, one lane per particle, the particle kept in registers from seed to termination, and
// a lane that loses its particle (terminated, or handed to another brick) immediately refills
// from a global work counter (warp ballot + one atomic per warp).  No compaction pass and no
// state round trip through memory is needed, and lanes stay busy although lifetimes differ by
// orders of magnitude.  Results follow the formula sheet A4-A9 operation by operation.
#pragma once
#include "field.cuh"

namespace streami {

// hand-off record: what a particle carries to another brick or into the next segment (position +
// unique id; plus its step count; DP5(4): t and h as bits in pad0/pad1).  32 bytes,
// read and written as two 16-byte accesses.
struct __align__(16) QRec {
  float px, py, pz; unsigned id;
  unsigned n; unsigned brick; unsigned pad0, pad1;
};

struct TraceArgs {
  Geom g;
  Store s;                         // monolithic store
  const Store* bricks; BrickMap bm; int nbricks;   // brick mode
  // work
  const float* seeds;              // [n][3]
  const float4* seeds4;            // optional: the seeds in processing order as {x, y, z, id}; perm is then unused
  const unsigned* perm;            // optional processing order of the work items (Morton sort), or NULL
  const QRec* qin;                 // work = queue records (brick rounds >= 1, segments >= 1), else seeds
  unsigned long long nwork;
  const unsigned* nwork_dev;       // if set, the work count is read from device memory instead
  unsigned seg_budget;             // step attempts per particle per launch, 0 = unlimited
  unsigned phase;                  // RK4: steps per phase of the advection loop (power of two dividing stride; trace_kernel.cuh)
  unsigned long long* next;        // global work counter
  int round;
  // integrator (host-computed fp32 constants, A4/A8)
  float h, h2, h6, hmin, hmax, atol, rtol, vmin2, t0;
  unsigned max_steps;
  // outputs (A6)
  float* verts; unsigned long long n; unsigned cap, stride;
  int vec_ok;                      // capacity % 8 == 0 and verts 32-byte aligned: full-sector vertex stores
  int prefetch;                    // 1 = one-step-ahead cell prefetch (field.cuh), 0 = off
  int staging;                     // 1 = stage vertices in shared memory (default), 0 = store each directly
  int brick_fast;                  // 0 = clear the bricks' integer-accept ranges (option "integer_accept" = 0)
  unsigned* counts; unsigned* steps; unsigned* status; float* fin;
  unsigned long long* totals;      // [4]
  // brick outputs
  QRec* qout; unsigned* qout_count;
  // in-kernel continuation queue (trace_kernel.cuh, INQ): qout, zero-initialised, is consumed by the same launch
  unsigned long long* cq_tail;     // next ring position to publish at (64-bit: positions never wrap)
  unsigned long long* cq_head;     // next ring position to claim
  unsigned* cq_done;               // particles terminated so far
  unsigned cq_total;               // the launch ends when cq_done reaches this (the particles it was given)
  unsigned* cq_error;              // set if a warp gave up waiting (never, unless a record was lost)
  unsigned cq_mask, cq_shift;      // ring of 2^cq_shift records
  unsigned* rc_this;               // round_counts row of this round (round 0 only), or NULL
  unsigned* rc_next;               // round_counts row of the next round, or NULL
  unsigned long long* log; unsigned long long log_cap; unsigned long long* log_count;
};

constexpr unsigned RC_HANDOFF = 100;

struct Lane {
  float px, py, pz;
  unsigned id, n;
  unsigned slot, rec_cd;           // next vertex slot, steps until the next recorded vertex
  unsigned pf;                     // cell most recently requested by the prefetcher
  unsigned stage0;                 // first slot held in the shared-memory staging group (<= slot)
  // DP5(4) only
  float t, h, k1x, k1y, k1z; bool rejected;
};

// a7, the output writer.  A vertex is 3 x 4 bytes into three planes; written one at a time each
// store dirties 4 bytes of a 32-byte sector that is evicted long before the particle's next vertex
// arrives (measured on C2: 6.6 GB of DRAM writes plus read-modify-write reads for 1.3 GB of
// vertices, 13-24 % of the kernel).  So vertices are staged per lane in shared memory, 8 slots per
// plane, and written as ONE full 32-byte sector per plane when the group of 8 is complete; a
// partial group (at termination, at a hand-off, or for a capacity that is not a multiple of 8)
// goes out with scalar stores.  Slots beyond the count stay untouched (A6).
constexpr int REC_GROUP = 8;
#ifndef STREAMI_RK4_BLOCK
#define STREAMI_RK4_BLOCK 256      // threads per block of the RK4 kernels (the staging arrays are sized by it)
#define STREAMI_RK4_MIN_BLOCKS 3  // resident blocks per SM the register allocation must allow
#endif
constexpr int REC_THREADS = STREAMI_RK4_BLOCK;
constexpr int DP5_THREADS = 128;   // threads per block of the DP5(4) kernels (trace_block in trace_kernel.cuh)
template <int BT>
__device__ __forceinline__ float* rec_stage() {
  // [thread][plane][slot & 7]: a lane's group is 96 contiguous bytes, read back as 6 LDS.128
  __shared__ __align__(16) float s_rec[3 * REC_GROUP * BT];
  return s_rec + 3 * REC_GROUP * threadIdx.x;
}

__device__ __forceinline__ float* rec_scratch() {              // never read: cp.async prefetch target
  __shared__ float s_scr[REC_THREADS];
  return s_scr + threadIdx.x;
}

template <int BT = REC_THREADS>
__device__ __forceinline__ void flush_vertices(const TraceArgs& a, Lane& L) {
  const unsigned cnt = L.slot - L.stage0;
  if (cnt != 0u && a.verts) {
    const float* s = rec_stage<BT>();
    const unsigned long long plane = a.n * a.cap;
    float* dst = a.verts + (unsigned long long)L.id * a.cap + L.stage0;
    if (cnt == (unsigned)REC_GROUP && a.vec_ok) {               // stage0 is then a multiple of 8
#pragma unroll
      for (int c = 0; c < 3; ++c) {
        const float4 lo = *reinterpret_cast<const float4*>(s + c * REC_GROUP);
        const float4 hi = *reinterpret_cast<const float4*>(s + c * REC_GROUP + 4);
        asm volatile("st.global.v8.f32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};" ::"l"(dst + c * plane),
                     "f"(lo.x), "f"(lo.y), "f"(lo.z), "f"(lo.w), "f"(hi.x), "f"(hi.y), "f"(hi.z), "f"(hi.w)
                     : "memory");
      }
    } else {
      const unsigned j0 = L.stage0 & (REC_GROUP - 1);
#pragma unroll 1
      for (unsigned j = 0; j < cnt; ++j) {
#pragma unroll
        for (int c = 0; c < 3; ++c) dst[c * plane + j] = s[c * REC_GROUP + j0 + j];
      }
    }
  }
  L.stage0 = L.slot;
}

// Called once per accepted step.  The staged path has no branch up to the flush: some lane of a warp
// records in almost every iteration (27 lanes, stride 8, phases apart), so a branch around the
// three shared-memory stores was taken -- and its whole body issued for 3 lanes -- nearly always.
// Without an output array the stores still go to the staging words, which are then never read.
template <bool REC = true, int BT = REC_THREADS>
__device__ __forceinline__ void record_vertex(const TraceArgs& a, Lane& L) {
  if (!REC) return;
  if (a.staging) {
    const bool due = --L.rec_cd == 0u;
    L.rec_cd = due ? a.stride : L.rec_cd;
    const bool rec = due && L.slot < a.cap;
    float* s = rec_stage<BT>() + (L.slot & (REC_GROUP - 1));
    if (rec) { s[0] = L.px; s[REC_GROUP] = L.py; s[2 * REC_GROUP] = L.pz; }
    L.slot += rec ? 1u : 0u;
    if (rec && (L.slot & (REC_GROUP - 1)) == 0u) flush_vertices<BT>(a, L);
  } else if (--L.rec_cd == 0) {                  // option "vertex_staging" = 0 (for A/B measurement)
    L.rec_cd = a.stride;
    if (L.slot < a.cap) {
      if (a.verts) {
        unsigned long long o = (unsigned long long)L.id * a.cap + L.slot;
        unsigned long long plane = a.n * a.cap;
        a.verts[o] = L.px; a.verts[plane + o] = L.py; a.verts[2 * plane + o] = L.pz;
      }
      L.slot++; L.stage0 = L.slot;
    }
  }
}

// The phased loop (trace_kernel.cuh) counts rec_cd down inside the step and records at the phase boundary.
template <int BT = REC_THREADS>
__device__ __forceinline__ void record_due(const TraceArgs& a, Lane& L) {
  if (L.rec_cd != 0u) return;
  L.rec_cd = a.stride;
  if (L.slot >= a.cap) return;
  if (a.staging) {
    float* s = rec_stage<BT>() + (L.slot & (REC_GROUP - 1));
    s[0] = L.px; s[REC_GROUP] = L.py; s[2 * REC_GROUP] = L.pz;
    L.slot++;
    if ((L.slot & (REC_GROUP - 1)) == 0u) flush_vertices<BT>(a, L);
  } else {
    if (a.verts) {
      unsigned long long o = (unsigned long long)L.id * a.cap + L.slot;
      unsigned long long plane = a.n * a.cap;
      a.verts[o] = L.px; a.verts[plane + o] = L.py; a.verts[2 * plane + o] = L.pz;
    }
    L.slot++; L.stage0 = L.slot;
  }
}

// ---- A4 + A5 steps 2-6: one RK4 step.  Returns 0 to continue, else the final status. -------
// `done` = field samples taken in this call (0..4); the caller derives its counters from it:
// a call that returns 0 took 4 samples and is one attempt; a call that ends the particle took
// `done` samples and is an attempt iff done >= 2 or the new position left the domain (A5.3
// comes before the attempt is counted).  The stage-1 sample does not repeat the domain test:
// p passed it at the end of the previous step (A5.5) or at the seed (A5.1).
// REC: record the new vertex here (record_vertex).  !REC && COUNT: only count rec_cd down; the caller records at
// its phase boundary (record_due).
template <int LAYOUT, bool UNSTEADY, bool BRICK, bool CACHE, bool UNIT, bool REC = true, class CC = CellCache, bool COUNT = false>
__device__ __forceinline__ unsigned rk4_step(const TraceArgs& a, const Store& s, CC& cc,
                                             Lane& L, unsigned& done) {
  done = 0;
  if (L.n == a.max_steps) return ST_MAXSTEPS;                                   // A5.2
  if constexpr (!UNSTEADY && !BRICK) {
    // Steady monolithic fields: all four stages run without a branch (sample_nb), one decision at
    // the end (C2 18.8 -> 18.6 ms; the brick kernel keeps the early returns: with the store
    // descriptor live it spills otherwise, C3 190 -> 201 ms).
    // Precedence as in A5: stagnation (after k1), then the first failing stage, then the exit test.
    float k1x, k1y, k1z, k2x, k2y, k2z, k3x, k3y, k3z, k4x, k4y, k4z;
    const unsigned r1 = sample_nb<LAYOUT, BRICK, CACHE, UNIT, true>(a.g, s, cc, L.px, L.py, L.pz, k1x, k1y, k1z);
    const float m = __fmaf_rn(k1z, k1z, __fmaf_rn(k1y, k1y, k1x * k1x));        // A5.3
    float qx = __fmaf_rn(a.h2, k1x, L.px), qy = __fmaf_rn(a.h2, k1y, L.py), qz = __fmaf_rn(a.h2, k1z, L.pz);
    const unsigned r2 = sample_nb<LAYOUT, BRICK, CACHE, UNIT, false>(a.g, s, cc, qx, qy, qz, k2x, k2y, k2z);
    if (CACHE && a.prefetch >= 3) {
      // Early form of the one-step-ahead prefetch: k2 is the midpoint slope, so p + 2 h k2 predicts the END of the NEXT
      // step to O(h^3) already now, three quarters of a step before this step's own end point is known.  The request
      // then has a whole step to arrive before the next step's stage 2 touches that cell (the end-of-step form leaves
      // it a quarter of a step, and the first use stalls: 23 % of all stall samples on C2).
      const float h2x = a.h + a.h;
      float ex, ey, ez;
      index_pos<UNIT>(a.g, __fmaf_rn(h2x, k2x, L.px), __fmaf_rn(h2x, k2y, L.py), __fmaf_rn(h2x, k2z, L.pz), ex, ey, ez);
      const unsigned ve = clamped_cell<BRICK>(s, ex, ey, ez);
      if (a.prefetch == 4) {                    // also the next step's mid point, p + 1.5 h k2 (steps that cross two faces)
        const float h15 = a.h + a.h2;
        float mx, my, mz;
        index_pos<UNIT>(a.g, __fmaf_rn(h15, k2x, L.px), __fmaf_rn(h15, k2y, L.py), __fmaf_rn(h15, k2z, L.pz), mx, my, mz);
        const unsigned vm = clamped_cell<BRICK>(s, mx, my, mz);
        if (vm != cc.key && vm != L.pf && vm != ve) prefetch_cell32<LAYOUT>(s, vm, (unsigned)__cvta_generic_to_shared(rec_scratch()));
      }
      if (ve != cc.key && ve != L.pf) prefetch_cell32<LAYOUT>(s, ve, (unsigned)__cvta_generic_to_shared(rec_scratch()));
      L.pf = ve;
    }
    qx = __fmaf_rn(a.h2, k2x, L.px); qy = __fmaf_rn(a.h2, k2y, L.py); qz = __fmaf_rn(a.h2, k2z, L.pz);
    const unsigned r3 = sample_nb<LAYOUT, BRICK, CACHE, UNIT, false>(a.g, s, cc, qx, qy, qz, k3x, k3y, k3z);
    qx = __fmaf_rn(a.h, k3x, L.px); qy = __fmaf_rn(a.h, k3y, L.py); qz = __fmaf_rn(a.h, k3z, L.pz);
    const unsigned r4 = sample_nb<LAYOUT, BRICK, CACHE, UNIT, false>(a.g, s, cc, qx, qy, qz, k4x, k4y, k4z);
    const float sx = (k1x + k4x) + 2.0f * (k2x + k3x);
    const float sy = (k1y + k4y) + 2.0f * (k2y + k3y);
    const float sz = (k1z + k4z) + 2.0f * (k2z + k3z);
    const float nx = __fmaf_rn(a.h6, sx, L.px), ny = __fmaf_rn(a.h6, sy, L.py), nz = __fmaf_rn(a.h6, sz, L.pz);
    float gx, gy, gz;
    index_pos<UNIT>(a.g, nx, ny, nz, gx, gy, gz);
    // A5.5 with the integer accept of sample_nb (fast = 0 unless the field is tame): floor(g) inside
    // the cell range decides; the faces g = N-1, the outside and +-inf take the float test.
    bool in5 = ((unsigned)__float2int_rd(gx) < s.fastx) & ((unsigned)__float2int_rd(gy) < s.fasty) &
               ((unsigned)__float2int_rd(gz) < s.fastz);
    if (__builtin_expect(!in5, 0)) in5 = in_domain(a.g, gx, gy, gz);
    const bool stag = m < a.vmin2;
    if ((r1 | r2 | r3 | r4) != 0u || stag || !in5) {                            // rare: the particle ends
      if (r1) { done = 1; return r1; }
      if (stag) { done = 1; return ST_STAGNANT; }
      if (r2) { done = 2; return r2; }
      if (r3) { done = 3; return r3; }
      if (r4) { done = 4; return r4; }
      done = 5; return ST_OUT;                                                  // A5.5: not recorded
    }
    done = 4;
    if (CACHE && a.prefetch && a.prefetch < 3) {
      float ox, oy, oz;
      index_pos<UNIT>(a.g, L.px, L.py, L.pz, ox, oy, oz);
      const float dx = gx - ox, dy = gy - oy, dz = gz - oz;
      const unsigned scratch = (unsigned)__cvta_generic_to_shared(rec_scratch());
      const unsigned vf = clamped_cell<BRICK>(s, gx + dx, gy + dy, gz + dz);
      if (a.prefetch == 2) {                    // also the half-step point (A/B: not worth its cost)
        const unsigned vh = clamped_cell<BRICK>(s, __fmaf_rn(0.5f, dx, gx), __fmaf_rn(0.5f, dy, gy), __fmaf_rn(0.5f, dz, gz));
        if (vh != cc.key && vh != L.pf && vh != vf) prefetch_cell32<LAYOUT>(s, vh, scratch);
      }
      if (vf != cc.key && vf != L.pf) prefetch_cell32<LAYOUT>(s, vf, scratch);
      L.pf = vf;
    }
    L.px = nx; L.py = ny; L.pz = nz; L.n++;                                     // A5.6
    record_vertex<REC>(a, L);
    if (!REC && COUNT) L.rec_cd--;
    return 0;
  }
  float tn = 0.0f;
  if (UNSTEADY) tn = a.t0 + (float)L.n * a.h;                                   // A4, not accumulated
  float k1x, k1y, k1z, k2x, k2y, k2z, k3x, k3y, k3z, k4x, k4y, k4z;
  unsigned rc = sample<LAYOUT, UNSTEADY, BRICK, CACHE, UNIT, true>(a.g, s, cc, L.px, L.py, L.pz, tn, k1x, k1y, k1z);
  done = 1;
  if (BRICK) { if (rc) return rc; }
  float m = __fmaf_rn(k1z, k1z, __fmaf_rn(k1y, k1y, k1x * k1x));                // A5.3
  if (m < a.vmin2) return ST_STAGNANT;
  float qx = __fmaf_rn(a.h2, k1x, L.px), qy = __fmaf_rn(a.h2, k1y, L.py), qz = __fmaf_rn(a.h2, k1z, L.pz);
  rc = sample<LAYOUT, UNSTEADY, BRICK, CACHE, UNIT>(a.g, s, cc, qx, qy, qz, tn + a.h2, k2x, k2y, k2z);
  done = 2;
  if (rc) return rc;
  qx = __fmaf_rn(a.h2, k2x, L.px); qy = __fmaf_rn(a.h2, k2y, L.py); qz = __fmaf_rn(a.h2, k2z, L.pz);
  rc = sample<LAYOUT, UNSTEADY, BRICK, CACHE, UNIT>(a.g, s, cc, qx, qy, qz, tn + a.h2, k3x, k3y, k3z);
  done = 3;
  if (rc) return rc;
  qx = __fmaf_rn(a.h, k3x, L.px); qy = __fmaf_rn(a.h, k3y, L.py); qz = __fmaf_rn(a.h, k3z, L.pz);
  rc = sample<LAYOUT, UNSTEADY, BRICK, CACHE, UNIT>(a.g, s, cc, qx, qy, qz, tn + a.h, k4x, k4y, k4z);
  done = 4;
  if (rc) return rc;
  float sx = (k1x + k4x) + 2.0f * (k2x + k3x);
  float sy = (k1y + k4y) + 2.0f * (k2y + k3y);
  float sz = (k1z + k4z) + 2.0f * (k2z + k3z);
  float nx = __fmaf_rn(a.h6, sx, L.px), ny = __fmaf_rn(a.h6, sy, L.py), nz = __fmaf_rn(a.h6, sz, L.pz);
  float gx, gy, gz;
  if (!to_index<UNIT>(a.g, nx, ny, nz, gx, gy, gz)) { done = 5; return ST_OUT; }  // A5.5: not recorded
  if (CACHE && !UNSTEADY && a.prefetch) {
    // predicted stage points of the NEXT step, in index space: g + 0.5 d and g + d
    float ox, oy, oz;
    index_pos<UNIT>(a.g, L.px, L.py, L.pz, ox, oy, oz);
    const float dx = gx - ox, dy = gy - oy, dz = gz - oz;
    const unsigned scratch = (unsigned)__cvta_generic_to_shared(rec_scratch());
    const unsigned vf = clamped_cell<BRICK>(s, gx + dx, gy + dy, gz + dz);
    if (a.prefetch == 2) {                      // also the half-step point (A/B: not worth its cost)
      const unsigned vh = clamped_cell<BRICK>(s, __fmaf_rn(0.5f, dx, gx), __fmaf_rn(0.5f, dy, gy), __fmaf_rn(0.5f, dz, gz));
      if (vh != cc.key && vh != L.pf && vh != vf) prefetch_cell32<LAYOUT>(s, vh, scratch);
    }
    if (vf != cc.key && vf != L.pf) prefetch_cell32<LAYOUT>(s, vf, scratch);
    L.pf = vf;
  }
  L.px = nx; L.py = ny; L.pz = nz; L.n++;                                       // A5.6
  record_vertex<REC>(a, L);
  if (!REC && COUNT) L.rec_cd--;
  return 0;
}

}  // namespace streami
