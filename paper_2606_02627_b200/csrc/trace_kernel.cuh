// csrc/trace_kernel.cuh -- the persistent advection kernel: refill, step, terminate / hand off.
//
// Segments (the build's choice, a12 of SURVEY.md 8(a); not in the paper).  A launch may give every
// particle a budget of `seg_budget` step attempts; a particle that is still alive when its budget
// is spent is appended to the out queue exactly like a brick leaver, the host re-sorts the queue
// by Morton cell block and launches the next segment.  The lanes that run at the same time then
// work in the same region of the field at ALL times of the trace, not only at the seeds: their
// gathers share TLB entries, DRAM pages and L2 lines.  It is a schedule only: a particle's
// arithmetic does not depend on where its trajectory is cut, and every output is indexed by id.
#pragma once
#include "dp5.cuh"

namespace streami {

// Threads per block: 256 for RK4; DP5(4) keeps six stage vectors, and blocks of 128 give the
// register allocator a finer occupancy grid (6 to 8 blocks = 24 to 32 warps, see trace_min_blocks).
__host__ __device__ constexpr int trace_block(int integ) { return integ == 1 ? DP5_THREADS : STREAMI_RK4_BLOCK; }

template <int BT>
__device__ __forceinline__ void finish_particle(const TraceArgs& a, Lane& L, unsigned st) {
  flush_vertices<BT>(a, L);
  if (a.counts) a.counts[L.id] = L.slot;
  if (a.steps) a.steps[L.id] = L.n;
  if (a.status) a.status[L.id] = st;
  if (a.fin) { a.fin[L.id] = L.px; a.fin[a.n + L.id] = L.py; a.fin[2 * a.n + L.id] = L.pz; }
}

// a9: append a particle to the next launch's queue: a brick leaver (the device-side stand-in for
// emitOutgoing + forward) or a particle whose segment budget is spent.
// One atomic per warp for the slot range.  `handoff` = it changes brick (counted and logged, A9).
template <int INTEG, bool INQ = false>
__device__ __forceinline__ void emit_outgoing(const TraceArgs& a, Lane& L, int dest, bool emit,
                                              bool handoff) {
  unsigned mask = __ballot_sync(__activemask(), emit);
  if (!emit) return;
  flush_vertices<trace_block(INTEG)>(a, L);
  int lane = threadIdx.x & 31;
  int leader = __ffs(mask) - 1;
  QRec r; r.px = L.px; r.py = L.py; r.pz = L.pz; r.id = L.id; r.n = L.n; r.brick = (unsigned)dest;
  r.pad0 = 0; r.pad1 = 0;
  if (INTEG == 1) { r.pad0 = __float_as_uint(L.t); r.pad1 = __float_as_uint(L.h); }
  else { r.pad0 = L.slot; r.pad1 = L.rec_cd; }     // RK4: the writer's position, so that the pick-up needs no division
  if (INQ) {
    // Ring slot pos & mask.  The payload {px, py, pz, id | n, brick} goes out with plain stores; the
    // record is PUBLISHED by a release store (gpu scope) of the tag word, (pos >> shift) + 1 = the pass
    // through the ring (the memory starts zeroed, tags start at 1).  The consumer reads the tag with an
    // acquire load before it touches the payload (PTX memory model: release / acquire pattern on one
    // word; nothing relies on the atomicity of a vector store).
    unsigned long long base = 0;
    if (lane == leader) base = atomicAdd(a.cq_tail, (unsigned long long)__popc(mask));
    base = __shfl_sync(mask, base, leader);
    const unsigned long long pos = base + __popc(mask & ((1u << lane) - 1u));
    unsigned* q = reinterpret_cast<unsigned*>(a.qout + (pos & (unsigned long long)a.cq_mask));
    const unsigned tag = (unsigned)(pos >> a.cq_shift) + 1u;
    *reinterpret_cast<uint4*>(q) = make_uint4(__float_as_uint(r.px), __float_as_uint(r.py), __float_as_uint(r.pz), r.id);
    *reinterpret_cast<uint2*>(q + 4) = make_uint2(r.n, r.brick);
    asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(q + 7), "r"(tag) : "memory");
  } else {
    unsigned base = 0;
    if (lane == leader) base = atomicAdd(a.qout_count, (unsigned)__popc(mask));
    base = __shfl_sync(mask, base, leader);
    a.qout[base + __popc(mask & ((1u << lane) - 1u))] = r;
  }
  // |Q_r+1[dest]| counts every queued particle; with a step budget per round (the paper's
  // one-step rounds) that includes particles that stay in their brick.  The log holds brick
  // changes only.
  if (a.rc_next && (handoff || a.seg_budget)) atomicAdd(a.rc_next + dest, 1u);
  if (handoff) {
    if (a.log_count) {
      unsigned long long k = atomicAdd(a.log_count, 1ull);
      if (a.log && k < a.log_cap)
        a.log[k] = ((unsigned long long)(a.round + 1) << 48) | ((unsigned long long)dest << 32) | L.id;
    }
  }
}

// Resident blocks per SM the compiler must allow for.  3 blocks of 256 (<= 80 registers): capping
// the steady RK4 kernel at 64 registers for a 4th block was measured on C2 and lost to its spills.
// Pathlines with the two-slice cell copy (48 more registers): 2 blocks of 256 (RK4), 3 of 128 (DP5(4)).
// Steady DP5(4) is latency-bound -- every stage of an attempt waits for the slowest lane's DRAM round
// trip -- and scales with resident warps as long as the memory system takes the requests: on
// LAYOUT_CELL (a cell = 3 loads from ONE line, ~1.4 L2 requests) C5 takes 933 / 774 / 746 / 741 ms
// at 5 / 6 / 7 / 8 blocks of 128 (64 registers, 64 bytes of stack at 8); on XYQUAD (4 requests per cell)
// 956 / 885 / 1194 / 1214 ms: past 6 blocks its requests saturate the L2 miss path.  The brick form
// (descriptor live, spills at 80 registers already) stays at 5.
constexpr int trace_min_blocks(int layout, int integ, bool unsteady, bool brick, bool cache) {
  return (unsteady && cache) ? (integ == 1 ? 3 : 2)
                             : (integ == 1 ? (brick ? 5 : (layout == LAYOUT_CELL ? 8 : 6)) : STREAMI_RK4_MIN_BLOCKS);
}
template <bool T> struct TraceCache { typedef CellCache type; };
template <> struct TraceCache<true> { typedef CellCacheT type; };

// INQ (build's choice; results unchanged): the continuation queue is consumed by the SAME launch.
// A particle that has spent its step budget is appended to the queue as above; a lane that finds
// the seed counter dry claims the next queue index and takes that record as soon as it is
// published.  Seeds first, continuations in the order they were queued: the trace runs breadth
// first, every particle gets its first K steps before any gets its second K, and when the queue
// runs dry nobody has more than K steps left.  Without it the launch ends with the lanes that
// happened to pick a long-lived particle late: a 2,000-step particle started when the counter runs
// dry keeps its SM waiting ~2,000 latency-bound steps (C2: 2.6 of 15.6 ms).  A claim never blocks:
// the lane keeps its index and looks again in the next iteration, so a warp whose other lanes hold
// particles (one of which may be the producer) keeps stepping.  The launch ends when every
// particle has terminated (`cq_done` == `cq_total`).
__device__ __forceinline__ unsigned ld_relaxed_u32(const unsigned* p) {      // strong (L2-coherent) load, no ordering
  unsigned v;
  asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ unsigned ld_acquire_u32(const unsigned* p) {      // orders every later access after it
  unsigned v;
  asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}

template <int LAYOUT, int INTEG, bool UNSTEADY, bool BRICK, bool CACHE, bool UNIT, bool INQ = false>
__global__ void __launch_bounds__(trace_block(INTEG), trace_min_blocks(LAYOUT, INTEG, UNSTEADY, BRICK, CACHE))
trace_kernel(const TraceArgs a) {
  __shared__ unsigned long long s_tot[4];
  if (threadIdx.x < 4) s_tot[threadIdx.x] = 0ull;
  __syncthreads();

  const int lane = threadIdx.x & 31;
  const unsigned FULL = 0xffffffffu;
  const unsigned long long nwork = a.nwork_dev ? (unsigned long long)*a.nwork_dev : a.nwork;
  Lane L; L.rejected = false; L.pf = 0xffffffffu;
  typename TraceCache<UNSTEADY && CACHE>::type cc; cc.invalidate();
  Store st = a.s;                 // brick mode: replaced per particle
  int my_brick = 0;
  bool active = false, exhausted = false;
  unsigned n_samples = 0, n_attempts = 0, n_start = 0, budget = 0;
  constexpr bool PH = INTEG == 0 && !INQ;   // phased loop (below)
  unsigned skip = 0;              // PH: steps of its first phase a continued particle sits out
  unsigned long long pend = ~0ull; // INQ: claimed ring position whose record is not published yet
  bool term = false;              // INQ: this lane's particle terminated since the last count
  unsigned spins = 0, seen_done = 0;   // INQ: polls of an idle warp since the launch last made progress

  for (;;) {
    if (INQ) {
      const unsigned tm = __ballot_sync(FULL, term);
      if (tm) { if (lane == 0) atomicAdd(a.cq_done, (unsigned)__popc(tm)); term = false; }
    }
    // ---- a1: refill idle lanes from the global work counter --------------------------------
    unsigned need = __ballot_sync(FULL, !active && !exhausted);
    if (need) {
      int leader = __ffs(need) - 1;
      unsigned long long base = 0;
      if (lane == leader) base = atomicAdd(a.next, (unsigned long long)__popc(need));
      base = __shfl_sync(FULL, base, leader);
      if (!active && !exhausted) {
        unsigned long long w = base + __popc(need & ((1u << lane) - 1u));
        if (w >= nwork) {
          exhausted = true;
        } else {
          n_samples = 0; n_attempts = 0;
          budget = a.seg_budget;
          const unsigned src = a.perm ? a.perm[w] : (unsigned)w;
          bool fresh = true;
          if (a.qin) {                                        // a continued or handed-over particle
            const QRec r = a.qin[src];
            L.px = r.px; L.py = r.py; L.pz = r.pz; L.id = r.id; L.n = r.n; my_brick = (int)r.brick;
            if (INTEG == 1) {
              L.t = __uint_as_float(r.pad0); L.h = __uint_as_float(r.pad1); L.rejected = false;
              L.slot = min(a.cap, L.n / a.stride + 1u);
              L.rec_cd = a.stride - L.n % a.stride;
            } else {                               // = min(cap, n / stride + 1) and stride - n % stride
              L.slot = r.pad0; L.rec_cd = r.pad1;
            }
            L.stage0 = L.slot;
            fresh = false;
          } else {
            if (a.seeds4) {
              const float4 s4 = __ldg(a.seeds4 + w);
              L.id = __float_as_uint(s4.w); L.px = s4.x; L.py = s4.y; L.pz = s4.z;
            } else {
              L.id = src;
              L.px = a.seeds[3ull * L.id]; L.py = a.seeds[3ull * L.id + 1]; L.pz = a.seeds[3ull * L.id + 2];
            }
            L.n = 0; L.slot = 0; L.rec_cd = 1; L.stage0 = 0;
            if (INTEG == 1) { L.t = a.t0; L.h = fminf(fmaxf(a.h, a.hmin), a.hmax); L.rejected = false; }
          }
          n_start = L.n;
          if (PH) skip = L.n & (a.phase - 1u);
          active = true;
          if (fresh) {
            float gx, gy, gz;
            if (!to_index<UNIT>(a.g, L.px, L.py, L.pz, gx, gy, gz)) {           // A5.1
              finish_particle<trace_block(INTEG)>(a, L, ST_OUT);
              active = false; term = true;
            } else {
              record_vertex<true, trace_block(INTEG)>(a, L);                    // vertex 0 = seed
              if (BRICK) {
                my_brick = owner_of<UNIT>(a.g, a.bm, L.px, L.py, L.pz);
                if (a.rc_this) atomicAdd(a.rc_this + my_brick, 1u);
              }
            }
          }
          if (active) {
            if (BRICK) {
              st = a.bricks[my_brick];
              if (!a.brick_fast) { st.fastx = 0u; st.fasty = 0u; st.fastz = 0u; }
            }
            cc.invalidate();
            if (INTEG == 1) {
              // k1 of the first attempt.  For a continued particle this recomputes the FSAL value
              // S(p, t) it carried (same operands, same operations), so it is not counted again.
              unsigned rc = sample<LAYOUT, UNSTEADY, BRICK, CACHE, UNIT, true>(a.g, st, cc, L.px, L.py, L.pz, L.t,
                                                                               L.k1x, L.k1y, L.k1z);
              if (fresh) n_samples++;
              if (rc) { finish_particle<trace_block(INTEG)>(a, L, rc); active = false; term = true; atomicAdd(&s_tot[2], 1ull); }
            }
          }
        }
      }
    }
    if (INQ) {
      // seeds are dry for this lane: claim a queue position (one atomic per warp), take the record once published
      const unsigned want = __ballot_sync(FULL, !active && exhausted && pend == ~0ull);
      if (want) {
        const int leader = __ffs(want) - 1;
        unsigned long long base = 0;
        if (lane == leader) base = atomicAdd(a.cq_head, (unsigned long long)__popc(want));
        base = __shfl_sync(FULL, base, leader);
        if (!active && exhausted && pend == ~0ull) pend = base + __popc(want & ((1u << lane) - 1u));
      }
      const bool look = !active && pend != ~0ull;
      const unsigned* q = reinterpret_cast<const unsigned*>(a.qout + (pend & (unsigned long long)a.cq_mask));
      const unsigned tag = (unsigned)(pend >> a.cq_shift) + 1u;
      // Poll with a relaxed load (an acquire load at gpu scope invalidates the SM's L1, and with it the
      // cells the prefetcher has brought in: not on every poll); once the tag of this pass is there, the
      // acquire load of the same word orders the payload reads behind the publisher's release store.
      const unsigned seen = look ? ld_relaxed_u32(q + 7) : 0u;
      // a tag of a LATER pass means the ring was lapped before this record was read (its size makes that impossible:
      // at most cq_total records are queued at any time and the ring holds twice that); never read on silently
      if (look && (int)(seen - tag) > 0) atomicExch(a.cq_error, 1u);
      if (look && seen == tag && ld_acquire_u32(q + 7) == tag) {
        uint4 r0; uint2 r1;            // after the acquire: plain (weak) loads are ordered behind it
        asm volatile("ld.global.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(r0.x), "=r"(r0.y), "=r"(r0.z), "=r"(r0.w) : "l"(q) : "memory");
        asm volatile("ld.global.v2.u32 {%0,%1}, [%2];" : "=r"(r1.x), "=r"(r1.y) : "l"(q + 4) : "memory");
        L.px = __uint_as_float(r0.x); L.py = __uint_as_float(r0.y); L.pz = __uint_as_float(r0.z);
        L.id = r0.w; L.n = r1.x; my_brick = (int)r1.y;
        if (BRICK) {
          st = a.bricks[my_brick];
          if (!a.brick_fast) { st.fastx = 0u; st.fasty = 0u; st.fastz = 0u; }
        }
        L.slot = min(a.cap, L.n / a.stride + 1u);
        L.rec_cd = a.stride - L.n % a.stride;
        L.stage0 = L.slot;
        n_samples = 0; n_attempts = 0; n_start = L.n; budget = a.seg_budget;
        cc.invalidate(); L.pf = 0xffffffffu;
        pend = ~0ull; active = true;
      }
    }
    if (__all_sync(FULL, !active)) {
      if (__all_sync(FULL, exhausted)) {
        if (!INQ) break;
        unsigned dn = 0;
        if (lane == 0) dn = ld_relaxed_u32(a.cq_done);
        dn = __shfl_sync(FULL, dn, 0);
        if (dn >= a.cq_total && !__any_sync(FULL, term)) break;
        // An idle warp polls ~5 times per microsecond.  2^26 polls (a quarter of a minute) during which NO particle
        // of the whole launch terminated means a record was lost (it cannot be, see the ring's size in the
        // host code): give up loudly instead of hanging the device.  Progress anywhere restarts the count, so a
        // long launch with a few stragglers is never cut short.
        if (dn != seen_done) { seen_done = dn; spins = 0; }
        if (++spins > (1u << 26)) { if (lane == 0) atomicExch(a.cq_error, 1u); break; }
        unsigned er = 0;
        if (lane == 0) er = ld_relaxed_u32(a.cq_error);
        if (__shfl_sync(FULL, er, 0)) break;                 // some warp has given up: end the launch, the host reports it
        __nanosleep(200);
      }
      continue;
    }
    // ---- a2-a8: one step (RK4) or one attempt (DP5(4)) --------------------------------------
    bool emit = false, handoff = false; int dest = my_brick;
    if constexpr (PH) {
      // Phased loop (RK4): a.phase = U steps between two passes through the warp-level code above and below (refill
      // ballots, vertex staging, emit), U a power of two that divides `stride`, so a vertex can only fall due on the
      // last step of a phase and is recorded at the boundary.  Lanes keep n = 0 (mod U) at boundaries: a fresh particle
      // starts there with n = 0, a continued one (n = r mod U) sits out the first r steps of its first phase.  A lane
      // that loses its particle inside a phase idles until the boundary (U/2 of ~800 steps on average).  Schedule only.
      const unsigned U = a.phase;
#pragma unroll 1
      for (unsigned u = 0; u < U; ++u) {
        if (active && u >= skip) {
          unsigned done = 0;
          unsigned rc = rk4_step<LAYOUT, UNSTEADY, BRICK, CACHE, UNIT, false, typename TraceCache<UNSTEADY && CACHE>::type, true>(a, st, cc, L, done);
          if (BRICK && rc == 0) {                                                 // a8: owner of p_new
            if (!still_owned<UNIT>(a.g, st, L.px, L.py, L.pz)) dest = owner_of<UNIT>(a.g, a.bm, L.px, L.py, L.pz);
            if (dest != my_brick) { rc = (L.n == a.max_steps) ? ST_MAXSTEPS : RC_HANDOFF; done = 0; handoff = rc == RC_HANDOFF; }
          }
          if (rc == 0 && --budget == 0u) { rc = RC_HANDOFF; done = 0; }           // segment budget spent
          if (rc) {
            active = false;
            // a vertex that fell due on this very step (n = 0 mod stride) is recorded before the particle goes
            record_due<trace_block(INTEG)>(a, L);
            if (rc == RC_HANDOFF) emit = true; else { finish_particle<trace_block(INTEG)>(a, L, rc); term = true; }
            n_attempts = (L.n - n_start) + (done >= 2u ? 1u : 0u);
            n_samples = 4u * (L.n - n_start) + min(done, 4u);
            atomicAdd(&s_tot[0], (unsigned long long)n_attempts);
            atomicAdd(&s_tot[1], (unsigned long long)(L.n - n_start));
            atomicAdd(&s_tot[2], (unsigned long long)n_samples);
            if (handoff) atomicAdd(&s_tot[3], 1ull);
          }
        }
      }
      skip = 0u;
      if (active) record_due<trace_block(INTEG)>(a, L);
    } else
    if (active) {
      unsigned rc, done = 0;
      if (INTEG == 0) rc = rk4_step<LAYOUT, UNSTEADY, BRICK, CACHE, UNIT>(a, st, cc, L, done);
      else            rc = dp5_attempt<LAYOUT, UNSTEADY, BRICK, CACHE, UNIT>(a, st, cc, L, n_samples, n_attempts);
      if (BRICK && rc == 0) {                                                   // a8: owner of p_new
        if (!still_owned<UNIT>(a.g, st, L.px, L.py, L.pz)) dest = owner_of<UNIT>(a.g, a.bm, L.px, L.py, L.pz);
        if (dest != my_brick) { rc = (L.n == a.max_steps) ? ST_MAXSTEPS : RC_HANDOFF; done = 0; handoff = rc == RC_HANDOFF; }
      }
      if (rc == 0 && --budget == 0u) {                                          // segment budget spent
        // (seg_budget == 0 wraps to 2^32-1: no segments.)  A rejected DP5(4) attempt must retry
        // with the flag it carries, so the cut waits for the next accepted step.
        if (INTEG == 1 && L.rejected) budget = 1u; else { rc = RC_HANDOFF; done = 0; }
      }
      if (rc) {
        active = false;
        if (rc == RC_HANDOFF) emit = true; else { finish_particle<trace_block(INTEG)>(a, L, rc); term = true; }
        if (INTEG == 0) {                       // RK4 counters are derived (see rk4_step)
          n_attempts = (L.n - n_start) + (done >= 2u ? 1u : 0u);
          n_samples = 4u * (L.n - n_start) + min(done, 4u);
        }
        atomicAdd(&s_tot[0], (unsigned long long)n_attempts);
        atomicAdd(&s_tot[1], (unsigned long long)(L.n - n_start));
        atomicAdd(&s_tot[2], (unsigned long long)n_samples);
        if (handoff) atomicAdd(&s_tot[3], 1ull);
      }
    }
    if (a.qout) {
      unsigned any = __ballot_sync(FULL, emit);
      if (any) emit_outgoing<INTEG, INQ>(a, L, dest, emit, handoff);
    }
  }
  asm volatile("cp.async.wait_all;" ::: "memory");   // prefetch copies still in flight target our shared memory
  __syncthreads();
  if (a.totals && threadIdx.x < 4 && s_tot[threadIdx.x]) atomicAdd(a.totals + threadIdx.x, s_tot[threadIdx.x]);
}

}  // namespace streami
