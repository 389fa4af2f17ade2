// csrc/api_rounds.cu -- the two round loops (a10): streaklines (Listing 2: a
// new batch of particles per advection step) and brick advection with hand-off (PAPER.md:96-101,
// 142-144: advance, emitOutgoing, forward, repeat while any particle is active anywhere).
#include <cmath>
#include <vector>

#include "internal.h"
#include "host_lines.cuh"
#include "lines.cuh"
#include "misc_kernels.cuh"
#include "sorter.cuh"
#include "trace_kernel.cuh"

namespace streami {
typedef void (*TraceKernel)(const TraceArgs);
TraceKernel pick_trace_kernel(int layout, int integ, bool unsteady, bool brick, bool cache, bool unit);
TraceKernel pick_trace_kernel_inq(int layout, bool unit, bool brick);
bool unit_geometry(const Geom& g);
int trace_grid(TraceKernel k, unsigned long long nwork, int block, int* grid);
int check_params(const streami_params* p, bool need_capacity);
void fill_integrator(TraceArgs& a, const streami_params* p);

typedef void (*StreakKernel)(const StreakArgs);
template <int LAYOUT>
static StreakKernel pick_streak_l(bool unsteady, bool tcache) {
  if (!unsteady) return tcache ? streak_kernel<LAYOUT, false, true> : streak_kernel<LAYOUT, false, false>;
  return tcache ? streak_kernel<LAYOUT, true, true> : streak_kernel<LAYOUT, true, false>;
}
static StreakKernel pick_streak(int layout, bool unsteady, bool tcache) {
  switch (layout) {
    case LAYOUT_PACKED3: return pick_streak_l<LAYOUT_PACKED3>(unsteady, tcache);
    case LAYOUT_FLOAT4: return pick_streak_l<LAYOUT_FLOAT4>(unsteady, tcache);
    case LAYOUT_CELL: return pick_streak_l<LAYOUT_CELL>(unsteady, tcache);
    case LAYOUT_XYQUAD: return pick_streak_l<LAYOUT_XYQUAD>(unsteady, tcache);
    case LAYOUT_SOA: return pick_streak_l<LAYOUT_SOA>(unsteady, tcache);
    case LAYOUT_TEX: return pick_streak_l<LAYOUT_TEX>(unsteady, tcache);
    default: return pick_streak_l<LAYOUT_XPAIR>(unsteady, tcache);
  }
}
}  // namespace streami

using namespace streami;

// Brick advection in ONE launch (trace_kernel.cuh, INQ): a particle that leaves its brick, or has
// spent its step budget, is appended to a device ring that the lanes of the same launch consume once
// the seeds are gone.  The hand-off itself is unchanged (32-byte record into the queue, one atomic
// per warp, picked up with the destination brick's descriptor); what goes away is
// the round structure: one sort, launch, count readback and tail per round (C3: 37 rounds).  Used
// only on request (option "brick_round_steps" = -2) and when the caller does not observe A9's rounds
// (no round table, no hand-off log).  The ring holds 2^shift >= 2n records: at most n are queued at any time (a
// particle is in at most one), and a slot is overwritten only after 2^shift later records.
static int brick_advect_inq(streami_field f, const float* seeds, size_t n, const streami_params* params,
                            float* out_vertices, unsigned* out_counts, unsigned* out_nrounds, cudaStream_t st) {
  TraceKernel k = pick_trace_kernel_inq(f->layout, unit_geometry(f->g), true);
  const int block = trace_block(0);
  unsigned shift = 10;
  while ((1ull << shift) < 2ull * n) ++shift;
  if (shift > 31) return STREAMI_E_INVALID;
  const size_t cap = (size_t)1 << shift;
  char* ctr = nullptr; QRec* cq = nullptr; unsigned* perm = nullptr; float4* seeds4 = nullptr;
  MortonSorter sorter{}; bool have_sorter = false;
  const bool sorting = options().presort && n >= 65536;
  auto cleanup = [&]() {
    if (ctr) cudaFreeAsync(ctr, st);
    if (seeds4) cudaFreeAsync(seeds4, st);
    if (cq) cudaFreeAsync(cq, st);
    if (perm) cudaFreeAsync(perm, st);
    if (have_sorter) sorter.release();
  };
  // scratch: [0] work counter u64, [8] ring tail u64, [16] ring head u64, [24] particles done u32, [28] error u32
  cudaError_t e = cudaMallocAsync((void**)&ctr, 32, st);
  if (e == cudaSuccess) e = cudaMemsetAsync(ctr, 0, 32, st);
  if (e == cudaSuccess) e = cudaMallocAsync((void**)&cq, sizeof(QRec) * cap, st);
  if (e == cudaSuccess) e = cudaMemsetAsync(cq, 0, sizeof(QRec) * cap, st);
  if (e == cudaSuccess && sorting) e = cudaMallocAsync((void**)&perm, sizeof(unsigned) * n, st);
  if (e != cudaSuccess) { cleanup(); return check(e); }
  int rc = STREAMI_OK;
  if (sorting) {
    rc = sorter.init(f, n, st, true);
    if (rc) { cleanup(); return rc; }
    have_sorter = true;
    rc = sorter.sort(f->g, seeds, 3, n, nullptr, perm);
    if (rc) { cleanup(); return rc; }
    e = cudaMallocAsync((void**)&seeds4, sizeof(float4) * n, st);
    if (e != cudaSuccess) { cleanup(); return check(e); }
    rc = sorter.gather_seeds(seeds, perm, n, seeds4);
    if (rc) { cleanup(); return rc; }
  }
  TraceArgs a{};
  a.g = f->g; a.g.time_mode = 0; a.s = f->bricks[0];
  a.bricks = f->d_bricks; a.bm = f->bm; a.nbricks = (int)f->bricks.size();
  a.brick_fast = options().integer_accept;
  a.seeds = seeds; a.seeds4 = seeds4; a.perm = seeds4 ? nullptr : perm; a.qin = nullptr; a.nwork = n; a.nwork_dev = nullptr;
  a.next = (unsigned long long*)ctr; a.round = 0;
  a.seg_budget = options().queue_steps > 0 ? (unsigned)options().queue_steps : 0u;   // 0 = until the particle leaves its brick
  fill_integrator(a, params);
  a.verts = out_vertices; a.n = n; a.counts = out_counts;
  a.vec_ok = out_vertices && (params->capacity % 8u) == 0u && ((unsigned long long)out_vertices % 32ull) == 0ull;
  a.qout = cq; a.qout_count = nullptr;
  a.cq_tail = (unsigned long long*)(ctr + 8); a.cq_head = (unsigned long long*)(ctr + 16);
  a.cq_done = (unsigned*)(ctr + 24); a.cq_total = (unsigned)n; a.cq_error = (unsigned*)(ctr + 28);
  a.cq_mask = (unsigned)(cap - 1); a.cq_shift = shift;
  int grid = 0;
  rc = trace_grid(k, n, block, &grid);
  if (rc) { cleanup(); return rc; }
  timing_begin(st);
  k<<<grid, block, 0, st>>>(a);
  timing_end(st);
  launch_counter()++;
  e = cudaGetLastError();
  unsigned err = 0;
  if (e == cudaSuccess) e = cudaMemcpyAsync(&err, ctr + 28, sizeof(unsigned), cudaMemcpyDeviceToHost, st);
  cleanup();
  if (e == cudaSuccess) e = cudaStreamSynchronize(st);     // streami_brick_advect synchronises its stream (streami.h)
  if (e != cudaSuccess) return check(e);
  if (err) return STREAMI_E_CUDA;
  if (out_nrounds) *out_nrounds = 1;
  return STREAMI_OK;
}

extern "C" {

// ---- step-synchronous streaklines (Tracer::step() of Listing 2) ---------------
struct streami_streak_s {
  streami::StreakArgs a;
  streami::StreakKernel k;
  unsigned done;          // global steps executed so far
  unsigned window;        // global steps per launch
  unsigned* out_status;   // optional [nsteps*m]
};

int streami_streak_begin(streami_field f, const float* points, size_t m, unsigned nsteps,
                         const streami_params* params, float* out_vertices, void* cuda_stream,
                         streami_streak* out) {
  OptionsScope options_scope;
  if (!out) return STREAMI_E_INVALID;
  *out = nullptr;
  if (!f || f->bricked || m == 0 || nsteps == 0 || !points || !out_vertices) return STREAMI_E_INVALID;
  int rc = check_params(params, false);
  if (rc) return rc;
  if (params->integrator != 0) return STREAMI_E_INVALID;      // shared stage times need a fixed step
  if ((unsigned long long)m * nsteps > 0xffffffffull) return STREAMI_E_INVALID;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  if (params->out_totals) STREAMI_TRY(cudaMemsetAsync(params->out_totals, 0, 4 * sizeof(unsigned long long), st));
  const bool unsteady = f->g.nslices > 1;
  // Window = global steps per launch.  A particle lives in registers inside a window (with the
  // two-slice copy of its cell) and goes through its output slot between windows, so long windows
  // win: C4 at 10 / 40 / 100 / 200 / 1000 steps per launch takes 155 / 99 / 88 / 86 / 86 ms.  The
  // earlier rule (two slice intervals per launch, to keep the slices of a launch L2-resident) cost
  // more in relaunches and cold caches than the residency bought.  256 bounds the state a caller
  // waits for between launches; steady fields take everything in one launch.
  unsigned K = (unsigned)options().streak_window;
  if (K == 0) K = unsteady ? std::min(nsteps, 256u) : nsteps;
  unsigned char* state = nullptr;
  STREAMI_TRY(cudaMallocAsync((void**)&state, (size_t)m * nsteps, st));
  streami_streak_s* h = new streami_streak_s();
  StreakArgs& a = h->a;
  a.g = f->g; a.g.time_mode = params->time_mode; a.s = launch_store(f);
  a.points = points; a.m = m; a.nsteps = nsteps;
  a.h = params->h; a.h2 = 0.5f * params->h; a.h6 = params->h / 6.0f;
  a.vmin2 = params->vmin * params->vmin; a.t0 = params->t0;
  a.verts = out_vertices; a.state = state; a.steps = params->out_steps; a.totals = params->out_totals;
  h->k = pick_streak(f->layout, unsteady, options().cell_cache != 0);
  h->done = 0; h->window = K; h->out_status = params->out_status;
  *out = h;
  return STREAMI_OK;
}

int streami_streak_step(streami_streak h, unsigned k, void* cuda_stream) {
  OptionsScope options_scope;
  if (!h) return STREAMI_E_INVALID;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  StreakArgs& a = h->a;
  const unsigned target = (unsigned)std::min<unsigned long long>((unsigned long long)h->done + k, a.nsteps);
  cudaError_t e = cudaSuccess;
  while (h->done < target && e == cudaSuccess) {
    a.s0 = h->done; a.s1 = std::min(target, h->done + h->window);
    unsigned long long threads = a.m * (unsigned long long)a.s1;
    timing_begin(st);
    h->k<<<(unsigned)((threads + 255) / 256), 256, 0, st>>>(a);
    timing_end(st);
    launch_counter()++;
    e = cudaGetLastError();
    h->done = a.s1;
  }
  return check(e);
}

int streami_streak_position(streami_streak h, unsigned* steps_done) {
  if (!h || !steps_done) return STREAMI_E_INVALID;
  *steps_done = h->done;
  return STREAMI_OK;
}

int streami_streak_lines(streami_streak h, unsigned long long* out_offsets, float* out_points,
                         unsigned long long* out_total, void* cuda_stream) {
  OptionsScope options_scope;
  if (!h || !out_offsets) return STREAMI_E_INVALID;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const StreakArgs& a = h->a;
  unsigned* counts = nullptr;
  STREAMI_TRY(cudaMallocAsync((void**)&counts, sizeof(unsigned) * a.m, st));
  const unsigned blocks = (unsigned)((a.m + 255) / 256);
  count_streak_kernel<<<blocks, 256, 0, st>>>(a.state, a.m, h->done, counts);
  launch_counter()++;
  int rc = check(cudaGetLastError());
  if (rc == STREAMI_OK) rc = scan_counts(counts, a.m, out_offsets, st);
  if (rc == STREAMI_OK && out_points) {
    gather_streak_kernel<<<blocks, 256, 0, st>>>(a.verts, a.state, a.m, a.nsteps, h->done, out_offsets, out_points);
    launch_counter()++;
    rc = check(cudaGetLastError());
  }
  cudaFreeAsync(counts, st);
  if (rc == STREAMI_OK && out_total) {
    cudaError_t e = cudaMemcpyAsync(out_total, out_offsets + a.m, sizeof(unsigned long long), cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    rc = check(e);
  }
  return rc;
}

int streami_streak_end(streami_streak h, unsigned* out_counts, void* cuda_stream) {
  OptionsScope options_scope;
  if (!h) return STREAMI_E_INVALID;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  cudaError_t e = cudaSuccess;
  if (out_counts || h->out_status) {       // out_counts may be NULL; params->out_status is written either way
    streak_finalize_kernel<<<(unsigned)((h->a.m + 255) / 256), 256, 0, st>>>(h->a.state, h->a.m, h->a.nsteps, h->done,
                                                                             out_counts, h->out_status);
    launch_counter()++;
    e = cudaGetLastError();
  }
  cudaFreeAsync(h->a.state, st);
  delete h;
  return check(e);
}

int streami_trace_streaklines(streami_field f, const float* points, size_t m, unsigned nsteps,
                              const streami_params* params, float* out_vertices,
                              unsigned* out_counts, void* cuda_stream) {
  OptionsScope options_scope;
  if (!f || f->bricked || (m > 0 && nsteps > 0 && (!points || !out_vertices || !out_counts))) return STREAMI_E_INVALID;
  int rc = check_params(params, false);
  if (rc) return rc;
  if (params->integrator != 0) return STREAMI_E_INVALID;
  if ((unsigned long long)m * nsteps > 0xffffffffull) return STREAMI_E_INVALID;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  if (m == 0 || nsteps == 0) {
    if (params->out_totals) STREAMI_TRY(cudaMemsetAsync(params->out_totals, 0, 4 * sizeof(unsigned long long), st));
    return STREAMI_OK;
  }
  streami_streak h = nullptr;
  rc = streami_streak_begin(f, points, m, nsteps, params, out_vertices, cuda_stream, &h);
  if (rc) return rc;
  rc = streami_streak_step(h, nsteps, cuda_stream);
  int rc2 = streami_streak_end(h, rc ? nullptr : out_counts, cuda_stream);
  return rc ? rc : rc2;
}

int streami_streamline_lines(const float* vertices, const unsigned* counts, size_t n, unsigned capacity,
                             unsigned long long* out_offsets, float* out_points,
                             unsigned long long* out_total, void* cuda_stream) {
  OptionsScope options_scope;
  if ((n > 0 && !counts) || !out_offsets || capacity == 0 || (n > 0 && out_points && !vertices)) return STREAMI_E_INVALID;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  int rc = scan_counts(counts, n, out_offsets, st);
  if (rc == STREAMI_OK && out_points && n) {
    gather_streamlines_kernel<<<148 * 8, 256, 0, st>>>(vertices, counts, n, capacity, out_offsets, out_points);
    launch_counter()++;
    rc = check(cudaGetLastError());
  }
  if (rc == STREAMI_OK && out_total) {
    cudaError_t e = cudaMemcpyAsync(out_total, out_offsets + n, sizeof(unsigned long long), cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    rc = check(e);
  }
  return rc;
}

int streami_partition_seeds(streami_field f, const float* seeds, size_t n, unsigned* out_perm,
                            unsigned long long* out_offsets, void* cuda_stream) {
  OptionsScope options_scope;
  if (!f || !f->bricked || !out_offsets || (n > 0 && (!seeds || !out_perm))) return STREAMI_E_INVALID;
  if (n > 0xffffffffull) return STREAMI_E_INVALID;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const unsigned nb = (unsigned)f->bricks.size();
  if (n == 0) return check(cudaMemsetAsync(out_offsets, 0, sizeof(unsigned long long) * (nb + 1), st));
  MortonSorter sorter{};
  int rc = sorter.init(f, n, st, true);
  if (rc) return rc;
  rc = sorter.sort(f->g, seeds, 3, n, nullptr, out_perm, out_offsets);
  sorter.release();
  return rc;
}

int streami_brick_advect(streami_field f, const float* seeds, size_t n,
                         const streami_params* params, float* out_vertices, unsigned* out_counts,
                         unsigned* out_round_counts, unsigned max_rounds,
                         unsigned long long* out_handoff_log, size_t log_capacity,
                         unsigned long long* out_log_count, unsigned* out_nrounds,
                         void* cuda_stream) {
  OptionsScope options_scope;
  if (!f || !f->bricked || (n > 0 && (!seeds || !out_counts))) return STREAMI_E_INVALID;
  int rc = check_params(params, true);
  if (rc) return rc;
  if (n > 0xffffffffull) return STREAMI_E_INVALID;
  if (out_round_counts && max_rounds == 0) return STREAMI_E_INVALID;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const int nb = (int)f->bricks.size();
  if (out_nrounds) *out_nrounds = 0;
  if (params->out_totals) STREAMI_TRY(cudaMemsetAsync(params->out_totals, 0, 4 * sizeof(unsigned long long), st));
  if (out_log_count) STREAMI_TRY(cudaMemsetAsync(out_log_count, 0, sizeof(unsigned long long), st));
  if (n == 0) return check(cudaStreamSynchronize(st));

  const bool cache = options().cell_cache != 0;
  // brick_round_steps = -2: one launch with the in-kernel ring instead of rounds (measured on C3: 158 ms
  // against 157 ms for sorted rounds -- the Morton sort of every round is worth what the rounds cost)
  const bool ring_ok = f->layout != LAYOUT_SOA && f->layout != LAYOUT_TEX;    // the comparison layouts have no ring kernels
  if (options().brick_round_steps == -2 && !out_round_counts && !out_handoff_log && params->integrator == 0 && cache && ring_ok)
    return brick_advect_inq(f, seeds, n, params, out_vertices, out_counts, out_nrounds, st);
  TraceKernel k = pick_trace_kernel(f->layout, params->integrator, false, true, cache, unit_geometry(f->g));
  const int block = trace_block(params->integrator);

  // scratch: [next u64][log count u64][qcount u32][pad u32][row0: nb x u32], two queues of n records
  const size_t ctr_bytes = 24 + sizeof(unsigned) * (size_t)nb;
  char* ctr = nullptr; QRec* q[2] = {nullptr, nullptr};
  STREAMI_TRY(cudaMallocAsync((void**)&ctr, ctr_bytes, st));
  cudaError_t e = cudaMallocAsync((void**)&q[0], sizeof(QRec) * n, st);
  if (e == cudaSuccess) e = cudaMallocAsync((void**)&q[1], sizeof(QRec) * n, st);
  unsigned* perm = nullptr; MortonSorter sorter{}; bool have_sorter = false;
  QRec* qs = nullptr;               // the round's work items in processing order (round 0: seeds as float4)
  const bool sorting = options().presort && n >= 65536;
  auto cleanup = [&]() {
    cudaFreeAsync(ctr, st); if (q[0]) cudaFreeAsync(q[0], st); if (q[1]) cudaFreeAsync(q[1], st);
    if (qs) cudaFreeAsync(qs, st);
    if (perm) cudaFreeAsync(perm, st);
    if (have_sorter) sorter.release();
  };
  if (e == cudaSuccess && sorting) e = cudaMallocAsync((void**)&perm, sizeof(unsigned) * n, st);
  if (e == cudaSuccess && sorting) e = cudaMallocAsync((void**)&qs, sizeof(QRec) * n, st);
  if (e != cudaSuccess) { if (e != cudaSuccess && !q[0]) q[0] = nullptr; cleanup(); return check(e); }
  unsigned long long* d_next = (unsigned long long*)ctr;
  unsigned long long* d_logc = out_log_count ? out_log_count : (unsigned long long*)(ctr + 8);
  unsigned* d_qcount = (unsigned*)(ctr + 16);
  unsigned* d_row0 = (unsigned*)(ctr + 24);
  e = cudaMemsetAsync(ctr, 0, ctr_bytes, st);
  if (e != cudaSuccess) { cleanup(); return check(e); }

  TraceArgs a{};
  a.g = f->g; a.g.time_mode = 0; a.s = f->bricks[0];
  a.bricks = f->d_bricks; a.bm = f->bm; a.nbricks = nb;
  a.brick_fast = options().integer_accept;
  a.seeds = seeds; a.perm = nullptr; a.next = d_next; a.nwork_dev = nullptr;
  // the paper re-queues EVERY particle after every RK step (Listing 1 ends in
  // emitOutgoing; one forward per step).  brick_round_steps = 1
  // reproduces that schedule; -1 advances until the particle leaves its brick (A9 / Q15, the round
  // structure the oracle reports); 0 = automatic: A9's rounds whenever the caller observes them
  // (round table or hand-off log requested), else a budget of 256 steps per round, which re-sorts
  // and re-balances the survivors (measured on C3: 241 -> 190 ms).  Per-particle results are the
  // same for every choice.
  {
    const int o = options().brick_round_steps;
    const bool observed = out_round_counts || out_handoff_log;
    a.seg_budget = o > 0 ? (unsigned)o : ((o == 0 && !observed) ? 256u : 0u);   // o < 0: A9's rounds
  }
  fill_integrator(a, params);
  a.verts = out_vertices; a.n = n; a.counts = out_counts;
  a.vec_ok = out_vertices && (params->capacity % 8u) == 0u && ((unsigned long long)out_vertices % 32ull) == 0ull;
  a.qout_count = d_qcount;
  a.log = out_handoff_log; a.log_cap = log_capacity; a.log_count = d_logc;

  if (sorting) {            // a12 + a9: each round's work is ONE contiguous segment per destination brick (Q_r[b] of A9:
                            // what a data-sharded run would send to rank b), in Morton order inside the segment
    rc = sorter.init(f, n, st, true);
    if (rc) { cleanup(); return rc; }
    have_sorter = true;
  }
  bool truncated = false;
  unsigned round = 0;
  unsigned long long nwork = n;
  std::vector<unsigned> h_buf(1 + nb);
  // Automatic rounds only (nobody observes A9's round structure): once a round has less than n/16 particles
  // left, the rest -- on C3 some twenty rounds of stragglers that changed brick often, each a launch that
  // waits for its slowest particle -- is finished by ONE launch that consumes its own hand-off ring
  // (trace_kernel.cuh, INQ).
  const bool ring_finish = options().brick_round_steps == 0 && !out_round_counts && !out_handoff_log &&
                           params->integrator == 0 && cache && ring_ok;
  for (;;) {
    a.round = (int)round; a.nwork = nwork;
    a.qin = round ? q[round & 1] : nullptr; a.qout = q[(round + 1) & 1];
    if (ring_finish && round > 0 && nwork * 16ull <= (unsigned long long)n) {
      unsigned shift = 10;
      while ((1ull << shift) < 2ull * nwork) ++shift;
      const size_t cap = (size_t)1 << shift;
      char* rctr = nullptr; QRec* ring = nullptr;       // [0] ring tail u64, [8] head u64, [16] done u32, [20] error u32
      e = cudaMallocAsync((void**)&rctr, 32, st);
      if (e == cudaSuccess) e = cudaMemsetAsync(rctr, 0, 32, st);
      if (e == cudaSuccess) e = cudaMallocAsync((void**)&ring, sizeof(QRec) * cap, st);
      if (e == cudaSuccess) e = cudaMemsetAsync(ring, 0, sizeof(QRec) * cap, st);
      if (e == cudaSuccess) e = cudaMemsetAsync(d_next, 0, sizeof(unsigned long long), st);
      unsigned err = 0;
      if (e == cudaSuccess) {
        TraceKernel kr = pick_trace_kernel_inq(f->layout, unit_geometry(f->g), true);
        a.perm = nullptr; a.seeds4 = nullptr; a.rc_this = nullptr; a.rc_next = nullptr;
        a.seg_budget = 0;                               // until the particle leaves its brick
        a.qout = ring; a.qout_count = nullptr; a.cq_tail = (unsigned long long*)rctr; a.cq_head = (unsigned long long*)(rctr + 8);
        a.cq_done = (unsigned*)(rctr + 16); a.cq_error = (unsigned*)(rctr + 20); a.cq_total = (unsigned)nwork;
        a.cq_mask = (unsigned)(cap - 1); a.cq_shift = shift;
        int grid = 0;
        rc = trace_grid(kr, nwork, block, &grid);
        if (rc == STREAMI_OK) {
          timing_begin(st);
          kr<<<grid, block, 0, st>>>(a);
          timing_end(st);
          launch_counter()++;
          e = cudaGetLastError();
          if (e == cudaSuccess) e = cudaMemcpyAsync(&err, rctr + 20, sizeof(unsigned), cudaMemcpyDeviceToHost, st);
          if (e == cudaSuccess) e = cudaStreamSynchronize(st);
        }
      }
      if (rctr) cudaFreeAsync(rctr, st);
      if (ring) cudaFreeAsync(ring, st);
      if (rc) { cleanup(); return rc; }
      if (e == cudaSuccess && err) { cleanup(); return STREAMI_E_CUDA; }
      round++;
      break;
    }
    a.perm = nullptr; a.seeds4 = nullptr;
    if (sorting && nwork >= 65536) {
      // the round's work in processing order: sort, then gather the items themselves (sorter.cuh)
      rc = round ? sorter.sort(f->g, (const float*)q[round & 1], 8, nwork, nullptr, perm)
                 : sorter.sort(f->g, seeds, 3, nwork, nullptr, perm);
      if (rc == STREAMI_OK)
        rc = round ? sorter.gather_rec32(q[round & 1], perm, nwork, qs) : sorter.gather_seeds(seeds, perm, nwork, (float4*)qs);
      if (rc) { cleanup(); return rc; }
      if (round) a.qin = qs; else a.seeds4 = (const float4*)qs;
    }
    a.rc_this = nullptr; a.rc_next = nullptr;
    if (round == 0) {
      a.rc_this = out_round_counts ? out_round_counts : d_row0;
      if (out_round_counts) e = cudaMemsetAsync(out_round_counts, 0, sizeof(unsigned) * nb, st);
    }
    if (out_round_counts && round + 1 < max_rounds) {
      a.rc_next = out_round_counts + (size_t)(round + 1) * nb;
      if (e == cudaSuccess) e = cudaMemsetAsync(a.rc_next, 0, sizeof(unsigned) * nb, st);
    }
    if (e == cudaSuccess) e = cudaMemsetAsync(d_next, 0, sizeof(unsigned long long), st);
    if (e == cudaSuccess) e = cudaMemsetAsync(d_qcount, 0, sizeof(unsigned), st);
    if (e != cudaSuccess) break;
    int grid = 0;
    rc = trace_grid(k, nwork, block, &grid);
    if (rc) { cleanup(); return rc; }
    timing_begin(st);
    k<<<grid, block, 0, st>>>(a);
    timing_end(st);
    launch_counter()++;
    e = cudaGetLastError();
    if (e != cudaSuccess) break;
    // the paper's fwdResult.numActiveAcrossAllRanks: read the live count
    e = cudaMemcpyAsync(h_buf.data(), d_qcount, sizeof(unsigned), cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess && round == 0)
      e = cudaMemcpyAsync(h_buf.data() + 1, a.rc_this, sizeof(unsigned) * nb, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) break;
    if (round == 0) {
      unsigned long long inside = 0;
      for (int b = 0; b < nb; ++b) inside += h_buf[1 + b];
      if (inside == 0) break;                                  // nothing was ever queued
    }
    round++;
    if (h_buf[0] == 0) break;
    if (out_round_counts && round >= max_rounds) truncated = true;
    nwork = h_buf[0];
  }
  if (e == cudaSuccess && out_handoff_log) {
    unsigned long long h_logc = 0;
    e = cudaMemcpyAsync(&h_logc, d_logc, sizeof(h_logc), cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (h_logc > log_capacity) truncated = true;
  }
  cleanup();
  if (e == cudaSuccess) e = cudaStreamSynchronize(st);
  if (e != cudaSuccess) return check(e);
  if (out_nrounds) *out_nrounds = round;
  return truncated ? STREAMI_E_TRUNCATED : STREAMI_OK;
}

}  // extern "C"

// ---- host-buffer variants (same calls, every buffer in host memory) -----------------------------

extern "C" {

int streami_trace_streaklines_host(streami_field f, const float* points, size_t m, unsigned nsteps,
                                   const streami_params* params, float* out_vertices,
                                   unsigned* out_counts, void* cuda_stream) {
  OptionsScope options_scope;
  if (!f || !params || (m > 0 && nsteps > 0 && (!points || !out_vertices || !out_counts))) return STREAMI_E_INVALID;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const size_t np = m * (size_t)nsteps;
  int rc;
  {
    Mirror mr(st);
    streami_params dp = *params;
    float* d_pts = (float*)mr.make(points, nullptr, 3 * m * sizeof(float));
    float* d_v = (float*)mr.make(nullptr, out_vertices, 3 * np * sizeof(float));
    unsigned* d_c = (unsigned*)mr.make(nullptr, out_counts, m * sizeof(unsigned));
    dp.out_steps = (unsigned*)mr.make(nullptr, params->out_steps, np * sizeof(unsigned));
    dp.out_status = (unsigned*)mr.make(nullptr, params->out_status, np * sizeof(unsigned));
    dp.out_final = nullptr;
    dp.out_totals = (unsigned long long*)mr.make(nullptr, params->out_totals, 4 * sizeof(unsigned long long));
    if (mr.err != cudaSuccess) return check(mr.err);
    rc = streami_trace_streaklines(f, d_pts, m, nsteps, &dp, d_v, d_c, cuda_stream);
    if (rc == STREAMI_OK && mr.download() != cudaSuccess) rc = check(mr.err);
  }
  if (rc == STREAMI_OK) rc = check(cudaStreamSynchronize(st));
  return rc;
}

int streami_brick_advect_host(streami_field f, const float* seeds, size_t n,
                              const streami_params* params, float* out_vertices, unsigned* out_counts,
                              unsigned* out_round_counts, unsigned max_rounds,
                              unsigned long long* out_handoff_log, size_t log_capacity,
                              unsigned long long* out_log_count, unsigned* out_nrounds,
                              void* cuda_stream) {
  OptionsScope options_scope;
  if (!f || !params || (n > 0 && (!seeds || !out_counts))) return STREAMI_E_INVALID;
  if (params->capacity == 0) return STREAMI_E_INVALID;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const int nb = f->bricked ? (int)f->bricks.size() : 0;
  int rc;
  {
    Mirror mr(st);
    streami_params dp = *params;
    float* d_seeds = (float*)mr.make(seeds, nullptr, 3 * n * sizeof(float));
    // slots beyond out_counts stay untouched (A6): the mirror starts as the caller's array
    float* d_v = (float*)mr.make(out_vertices, out_vertices, 3 * n * (size_t)params->capacity * sizeof(float));
    unsigned* d_c = (unsigned*)mr.make(nullptr, out_counts, n * sizeof(unsigned));
    // the round table is only partly written by the call: upload the caller's content first
    unsigned* d_rc = (unsigned*)mr.make(out_round_counts, out_round_counts, (size_t)max_rounds * nb * sizeof(unsigned));
    unsigned long long* d_log = (unsigned long long*)mr.make(nullptr, out_handoff_log, log_capacity * sizeof(unsigned long long));
    unsigned long long* d_lc = (unsigned long long*)mr.make(nullptr, out_log_count, sizeof(unsigned long long));
    dp.out_steps = (unsigned*)mr.make(nullptr, params->out_steps, n * sizeof(unsigned));
    dp.out_status = (unsigned*)mr.make(nullptr, params->out_status, n * sizeof(unsigned));
    dp.out_final = (float*)mr.make(nullptr, params->out_final, 3 * n * sizeof(float));
    dp.out_totals = (unsigned long long*)mr.make(nullptr, params->out_totals, 4 * sizeof(unsigned long long));
    if (mr.err != cudaSuccess) return check(mr.err);
    rc = streami_brick_advect(f, d_seeds, n, &dp, d_v, d_c, d_rc, max_rounds, d_log, log_capacity, d_lc,
                              out_nrounds, cuda_stream);
    if ((rc == STREAMI_OK || rc == STREAMI_E_TRUNCATED) && mr.download() != cudaSuccess) rc = check(mr.err);
  }
  if (rc == STREAMI_OK || rc == STREAMI_E_TRUNCATED) { int s = check(cudaStreamSynchronize(st)); if (s) rc = s; }
  return rc;
}

}  // extern "C"

extern "C" {

// Streamlines end to end for a host application: seeds in host memory in, assembled polylines
// (offsets + AoS points, the paper's getLines) in host memory out.  Only the stored vertices cross
// the bus, not the capacity-padded slot array.
int streami_trace_streamlines_lines_host(streami_field f, const float* seeds, size_t n,
                                         const streami_params* params, unsigned long long* out_offsets,
                                         float* out_points, unsigned long long max_points,
                                         unsigned long long* out_total, void* cuda_stream) {
  OptionsScope options_scope;
  if (!f) return STREAMI_E_INVALID;
  // Bricked fields run as one batch: every batch would pay all the rounds (C3 267 -> 293 ms in 4).
  auto trace = [&](const float* d_seeds, size_t nb, const streami_params* dp, float* d_v, unsigned* d_c) {
    return f->bricked ? streami_brick_advect(f, d_seeds, nb, dp, d_v, d_c, nullptr, 0, nullptr, 0, nullptr, nullptr, cuda_stream)
                      : streami_trace_streamlines(f, d_seeds, nb, dp, d_v, d_c, cuda_stream);
  };
  return lines_host(trace, f->bricked, seeds, n, params, out_offsets, out_points, max_points, out_total, cuda_stream);
}

}  // extern "C"
