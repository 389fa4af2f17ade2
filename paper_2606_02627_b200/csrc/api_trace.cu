// csrc/api_trace.cu -- streami_trace_streamlines (+ host-buffer variant): argument checks,
// scratch from the stream-ordered allocator, optional Morton presort, one persistent launch.
// This is Tracer::trace() in Streamlines mode without the per-step host loop.
#include <cmath>

#include "internal.h"
#include "sorter.cuh"
#include "trace_kernel.cuh"

namespace streami {

typedef void (*TraceKernel)(const TraceArgs);

template <int L, bool U>
static TraceKernel pick_lu(int integ, bool brick, bool cache) {      // steady
  if (brick && integ) return cache ? trace_kernel<L, 1, false, true, true, U> : trace_kernel<L, 1, false, true, false, U>;
  if (brick) return cache ? trace_kernel<L, 0, false, true, true, U> : trace_kernel<L, 0, false, true, false, U>;
  if (integ) return cache ? trace_kernel<L, 1, false, false, true, U> : trace_kernel<L, 1, false, false, false, U>;
  return cache ? trace_kernel<L, 0, false, false, true, U> : trace_kernel<L, 0, false, false, false, U>;
}

template <int L>
static TraceKernel pick_l(int integ, bool unsteady, bool brick, bool cache, bool unit) {
  if (unsteady && cache) return integ ? trace_kernel<L, 1, true, false, true, false> : trace_kernel<L, 0, true, false, true, false>;
  if (unsteady) return integ ? trace_kernel<L, 1, true, false, false, false> : trace_kernel<L, 0, true, false, false, false>;
  return unit ? pick_lu<L, true>(integ, brick, cache) : pick_lu<L, false>(integ, brick, cache);
}

// unit = the grid is its own index space (origin 0, spacing 1): see index_pos in field.cuh.
TraceKernel pick_trace_kernel(int layout, int integ, bool unsteady, bool brick, bool cache, bool unit) {
  switch (layout) {
    case LAYOUT_PACKED3: return pick_l<LAYOUT_PACKED3>(integ, unsteady, brick, cache, unit);
    case LAYOUT_FLOAT4: return pick_l<LAYOUT_FLOAT4>(integ, unsteady, brick, cache, unit);
    case LAYOUT_CELL: return pick_l<LAYOUT_CELL>(integ, unsteady, brick, cache, unit);
    case LAYOUT_XYQUAD: return pick_l<LAYOUT_XYQUAD>(integ, unsteady, brick, cache, unit);
    case LAYOUT_SOA: return pick_l<LAYOUT_SOA>(integ, unsteady, brick, cache, unit);
    case LAYOUT_TEX: return pick_l<LAYOUT_TEX>(integ, unsteady, brick, cache, unit);
    default: return pick_l<LAYOUT_XPAIR>(integ, unsteady, brick, cache, unit);
  }
}

// Steady monolithic RK4 with the cell cache and the in-kernel continuation queue (trace_kernel.cuh, INQ).
template <int L>
static TraceKernel pick_inq_l(bool unit, bool brick) {
  if (brick) return unit ? trace_kernel<L, 0, false, true, true, true, true> : trace_kernel<L, 0, false, true, true, false, true>;
  return unit ? trace_kernel<L, 0, false, false, true, true, true> : trace_kernel<L, 0, false, false, true, false, true>;
}
TraceKernel pick_trace_kernel_inq(int layout, bool unit, bool brick) {
  switch (layout) {
    case LAYOUT_PACKED3: return pick_inq_l<LAYOUT_PACKED3>(unit, brick);
    case LAYOUT_FLOAT4: return pick_inq_l<LAYOUT_FLOAT4>(unit, brick);
    case LAYOUT_CELL: return pick_inq_l<LAYOUT_CELL>(unit, brick);
    case LAYOUT_XYQUAD: return pick_inq_l<LAYOUT_XYQUAD>(unit, brick);
    default: return pick_inq_l<LAYOUT_XPAIR>(unit, brick);
  }
}

bool unit_geometry(const Geom& g) {
  return g.ox == 0.0f && g.oy == 0.0f && g.oz == 0.0f && g.rx == 1.0f && g.ry == 1.0f && g.rz == 1.0f;
}

// Persistent grid: as many blocks as are resident at once (a multiple of the SM count).
int trace_grid(TraceKernel k, unsigned long long nwork, int block, int* grid) {
  int per_sm = 0;
  STREAMI_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k, block, 0));
  int sms = num_sms();
  if (per_sm < 1 || sms < 1) return STREAMI_E_CUDA;
  if (options().max_blocks_per_sm > 0) per_sm = std::min(per_sm, options().max_blocks_per_sm);
  unsigned long long want = (nwork + block - 1) / block;
  unsigned long long full = (unsigned long long)per_sm * sms;
  *grid = (int)std::max(1ull, std::min(want, full));
  return STREAMI_OK;
}

int check_params(const streami_params* p, bool need_capacity) {
  if (!p) return STREAMI_E_INVALID;
  if (p->integrator != 0 && p->integrator != 1) return STREAMI_E_INVALID;
  if (!(std::isfinite(p->h) && p->h > 0.0f)) return STREAMI_E_INVALID;
  if (need_capacity && (p->capacity == 0 || p->stride == 0)) return STREAMI_E_INVALID;
  if (!(p->vmin >= 0.0f) || !std::isfinite(p->t0)) return STREAMI_E_INVALID;
  if (p->time_mode != 0 && p->time_mode != 1) return STREAMI_E_INVALID;
  if (p->integrator == 1) {
    if (!(p->h_min >= 0.0f) || !(p->h_max >= p->h_min) || !(p->atol >= 0.0f) || !(p->rtol >= 0.0f))
      return STREAMI_E_INVALID;
    if (!(p->atol > 0.0f || p->rtol > 0.0f)) return STREAMI_E_INVALID;
  }
  return STREAMI_OK;
}

void fill_integrator(TraceArgs& a, const streami_params* p) {
  a.h = p->h; a.h2 = 0.5f * p->h; a.h6 = p->h / 6.0f;        // A4: computed once, fp32
  a.hmin = p->h_min; a.hmax = p->h_max; a.atol = p->atol; a.rtol = p->rtol;
  a.vmin2 = p->vmin * p->vmin; a.t0 = p->t0; a.max_steps = p->max_steps;
  a.cap = p->capacity; a.stride = p->stride; a.vec_ok = 0; a.staging = options().vertex_staging;
  a.prefetch = options().prefetch;
  // RK4 phase length (trace_kernel.cuh): the largest power of two <= 8 that divides the recording stride (a vertex can
  // then only fall due on the last step of a phase) and the step budget of a segment / round, if there is one
  a.phase = 1u;
  while (a.phase < 8u && p->stride % (2u * a.phase) == 0u && (a.seg_budget == 0u || a.seg_budget % (2u * a.phase) == 0u)) a.phase *= 2u;
  a.steps = p->out_steps; a.status = p->out_status; a.fin = p->out_final; a.totals = p->out_totals;
}

}  // namespace streami

using namespace streami;

extern "C" {

int streami_trace_streamlines(streami_field f, const float* seeds, size_t n,
                              const streami_params* params, float* out_vertices,
                              unsigned* out_counts, void* cuda_stream) {
  OptionsScope options_scope;
  if (!f || f->bricked || (n > 0 && (!seeds || !out_counts))) return STREAMI_E_INVALID;
  int rc = check_params(params, true);
  if (rc) return rc;
  if (n > 0xffffffffull) return STREAMI_E_INVALID;           // particle ids are u32
  cudaStream_t st = (cudaStream_t)cuda_stream;
  if (params->out_totals) STREAMI_TRY(cudaMemsetAsync(params->out_totals, 0, 4 * sizeof(unsigned long long), st));
  if (n == 0) return STREAMI_OK;

  const bool unsteady = f->g.nslices > 1;
  const bool cache = options().cell_cache != 0;     // unsteady fields: the two-slice copy (CellCacheT)
  TraceKernel k = pick_trace_kernel(f->layout, params->integrator, unsteady, false, cache, unit_geometry(f->g));

  // Segments: K step attempts per particle per launch, Morton re-sort of the survivors between
  // launches (trace_kernel.cuh).  K = 0, or a trace too short or too small to need it: one launch.
  const bool sorting = options().presort && n >= 65536;
  unsigned K = (unsigned)options().segment_steps;
  if (!sorting || K >= params->max_steps) K = 0;
  const bool dp5 = params->integrator == 1;

  // In-kernel continuation queue (trace_kernel.cuh, INQ): steady RK4 with the cell cache, one launch.
  // Option "queue_steps" = Q > 0: steps per particle between two passes through the queue (0 = off, the
  // default: on C2 the shorter tail does not pay for the passes).  A particle
  // is queued at most floor(max_steps / Q) times, which sizes the queue; if that does not fit, the
  // launch runs without.
  unsigned Q = 0;
  if (!dp5 && !unsteady && cache && K == 0 && options().queue_steps > 0 && f->layout != LAYOUT_SOA && f->layout != LAYOUT_TEX) {
    Q = (unsigned)options().queue_steps;
    if (Q >= params->max_steps) Q = 0;
  }
  // ring of 2^shift records >= the passes of all particles: a slot is written once, its tag is always 1
  unsigned long long qcap = 0; unsigned qshift = 0;
  if (Q) {
    const unsigned long long need = (unsigned long long)n * (params->max_steps / Q);
    while ((1ull << qshift) < need) ++qshift;
    qcap = 1ull << qshift;
    if (qshift > 31) { Q = 0; qcap = 0; }
  }
  QRec* cq = nullptr;
  if (Q) {
    cudaError_t qe = cudaMallocAsync((void**)&cq, sizeof(QRec) * qcap, st);
    if (qe == cudaSuccess) qe = cudaMemsetAsync(cq, 0, sizeof(QRec) * qcap, st);   // all-zero = not written yet
    if (qe != cudaSuccess) {
      cudaGetLastError();
      if (cq) cudaFreeAsync(cq, st);
      cq = nullptr; Q = 0;
    } else {
      k = pick_trace_kernel_inq(f->layout, unit_geometry(f->g), false);
    }
  }
  int grid = 0;
  const int block = trace_block(params->integrator);
  rc = trace_grid(k, n, block, &grid);
  if (rc) { if (cq) cudaFreeAsync(cq, st); return rc; }

  // scratch: [0] work counter u64, [8] queue counts u32 x 2, INQ: [16] ring tail u64, [24] ring head u64,
  // [32] particles terminated u32, [36] error flag u32
  char* ctr = nullptr;
  {
    cudaError_t ce = cudaMallocAsync((void**)&ctr, 48, st);
    if (ce != cudaSuccess) { if (cq) cudaFreeAsync(cq, st); return check(ce); }
  }
  unsigned long long* next = (unsigned long long*)ctr;
  unsigned* qcount = (unsigned*)(ctr + 8);
  unsigned* perm = nullptr; QRec* q[2] = {nullptr, nullptr}; float4* seeds4 = nullptr;
  MortonSorter sorter{}; bool have_sorter = false;
  auto cleanup = [&]() {
    cudaFreeAsync(ctr, st);
    if (seeds4) cudaFreeAsync(seeds4, st);
    if (cq) cudaFreeAsync(cq, st);
    if (perm) cudaFreeAsync(perm, st);
    if (q[0]) cudaFreeAsync(q[0], st);
    if (q[1]) cudaFreeAsync(q[1], st);
    if (have_sorter) sorter.release();
  };
  cudaError_t e = cudaMemsetAsync(ctr, 0, 48, st);
  if (e == cudaSuccess && sorting) e = cudaMallocAsync((void**)&perm, sizeof(unsigned) * n, st);
  if (e == cudaSuccess && K) e = cudaMallocAsync((void**)&q[0], sizeof(QRec) * n, st);
  if (e == cudaSuccess && K) e = cudaMallocAsync((void**)&q[1], sizeof(QRec) * n, st);
  if (e != cudaSuccess) { cleanup(); return check(e); }
  if (sorting) {
    rc = sorter.init(f, n, st);
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
  a.g = f->g; a.g.time_mode = params->time_mode; a.s = launch_store(f);
  a.bricks = nullptr; a.nbricks = 0;
  a.seeds = seeds; a.seeds4 = seeds4; a.perm = seeds4 ? nullptr : perm; a.qin = nullptr; a.nwork = n; a.nwork_dev = nullptr; a.next = next; a.round = 0;
  a.seg_budget = K;
  fill_integrator(a, params);
  a.verts = out_vertices; a.n = n; a.counts = out_counts;
  a.vec_ok = out_vertices && (params->capacity % 8u) == 0u && ((unsigned long long)out_vertices % 32ull) == 0ull;
  a.qout = K ? q[0] : nullptr; a.qout_count = qcount;
  if (Q) {
    a.seg_budget = Q; a.qout = cq; a.qout_count = qcount;
    a.cq_tail = (unsigned long long*)(ctr + 16); a.cq_head = (unsigned long long*)(ctr + 24);
    a.cq_done = (unsigned*)(ctr + 32); a.cq_total = (unsigned)n; a.cq_error = (unsigned*)(ctr + 36);
    a.cq_mask = (unsigned)(qcap - 1ull); a.cq_shift = qshift;
  }
  timing_begin(st);
  k<<<grid, block, 0, st>>>(a);
  timing_end(st);
  launch_counter()++;
  e = cudaGetLastError();

  if (K && e == cudaSuccess) {
    // RK4: a particle takes exactly K steps per segment, so floor(max_steps / K) + 1 launches finish
    // everything (floor(max_steps / K) + 1 launches) and no count has to come back to the host (the call stays asynchronous; a launch
    // whose queue is empty exits at once).  DP5(4): rejected attempts spend budget too, so the live
    // count is read back every few segments (this synchronises the stream).
    const unsigned planned = params->max_steps / K + 1;   // the last one also turns n == max_steps into MAX_STEPS
    for (unsigned r = 1; e == cudaSuccess; ++r) {
      if (!dp5 && r >= planned) break;
      const unsigned in = (r - 1) & 1u, out = r & 1u;
      if (dp5 && (r % 4u) == 0u) {
        unsigned live = 0;
        e = cudaMemcpyAsync(&live, qcount + in, sizeof(unsigned), cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess) e = cudaStreamSynchronize(st);
        if (e != cudaSuccess || live == 0) break;
      }
      e = cudaMemsetAsync(qcount + out, 0, sizeof(unsigned), st);
      if (e == cudaSuccess) e = cudaMemsetAsync(next, 0, sizeof(unsigned long long), st);
      if (e != cudaSuccess) break;
      rc = sorter.sort(f->g, (const float*)q[in], 8, 0, qcount + in, perm);
      if (rc) { cleanup(); return rc; }
      a.seeds = nullptr; a.seeds4 = nullptr; a.perm = perm; a.qin = q[in]; a.nwork_dev = qcount + in; a.qout = q[out]; a.qout_count = qcount + out;
      a.round = (int)r;
      timing_begin(st);
      k<<<grid, block, 0, st>>>(a);
      timing_end(st);
      launch_counter()++;
      e = cudaGetLastError();
    }
  }
  unsigned cq_err = 0;
  if (Q && e == cudaSuccess) {
    // the in-kernel queue can give up (a lost record would otherwise hang the device): that must not pass for
    // success, so a call that used it reads the flag back and therefore synchronises its stream
    e = cudaMemcpyAsync(&cq_err, ctr + 36, sizeof(unsigned), cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
  }
  cleanup();
  if (e == cudaSuccess && cq_err) return STREAMI_E_CUDA;
  return check(e);
}

int streami_trace_streamlines_host(streami_field f, const float* seeds, size_t n,
                                   const streami_params* params, float* out_vertices,
                                   unsigned* out_counts, void* cuda_stream) {
  OptionsScope options_scope;
  if (!f || f->bricked || (n > 0 && (!seeds || !out_counts))) return STREAMI_E_INVALID;
  int rc = check_params(params, true);
  if (rc) return rc;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  if (n == 0) {
    if (params->out_totals) for (int i = 0; i < 4; ++i) params->out_totals[i] = 0;
    return STREAMI_OK;
  }
  const size_t nv = out_vertices ? 3 * n * (size_t)params->capacity : 0;
  float *d_seeds = nullptr, *d_verts = nullptr, *d_final = nullptr;
  unsigned *d_counts = nullptr, *d_steps = nullptr, *d_status = nullptr;
  unsigned long long* d_totals = nullptr;
  void* allocs[7] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};
  int na = 0;
  auto alloc = [&](void** p, size_t bytes) {
    cudaError_t e = cudaMallocAsync(p, bytes, st);
    if (e == cudaSuccess) allocs[na++] = *p;
    return e;
  };
  auto cleanup = [&]() { for (int i = 0; i < na; ++i) cudaFreeAsync(allocs[i], st); };
  cudaError_t e = alloc((void**)&d_seeds, 3 * n * sizeof(float));
  if (e == cudaSuccess) e = alloc((void**)&d_counts, n * sizeof(unsigned));
  if (e == cudaSuccess && nv) e = alloc((void**)&d_verts, nv * sizeof(float));
  if (e == cudaSuccess && params->out_steps) e = alloc((void**)&d_steps, n * sizeof(unsigned));
  if (e == cudaSuccess && params->out_status) e = alloc((void**)&d_status, n * sizeof(unsigned));
  if (e == cudaSuccess && params->out_final) e = alloc((void**)&d_final, 3 * n * sizeof(float));
  if (e == cudaSuccess && params->out_totals) e = alloc((void**)&d_totals, 4 * sizeof(unsigned long long));
  if (e == cudaSuccess) e = cudaMemcpyAsync(d_seeds, seeds, 3 * n * sizeof(float), cudaMemcpyHostToDevice, st);
  // Slots beyond out_counts are "left untouched" (A6): the device mirror starts as a copy of the caller's array, so
  // that the download below returns the caller's own values there, not whatever the allocator handed out.
  if (e == cudaSuccess && nv) e = cudaMemcpyAsync(d_verts, out_vertices, nv * sizeof(float), cudaMemcpyHostToDevice, st);
  if (e != cudaSuccess) { cleanup(); return check(e); }
  streami_params dp = *params;
  dp.out_steps = d_steps; dp.out_status = d_status; dp.out_final = d_final; dp.out_totals = d_totals;
  rc = streami_trace_streamlines(f, d_seeds, n, &dp, d_verts, d_counts, cuda_stream);
  if (rc) { cleanup(); return rc; }
  e = cudaMemcpyAsync(out_counts, d_counts, n * sizeof(unsigned), cudaMemcpyDeviceToHost, st);
  if (e == cudaSuccess && nv) e = cudaMemcpyAsync(out_vertices, d_verts, nv * sizeof(float), cudaMemcpyDeviceToHost, st);
  if (e == cudaSuccess && d_steps) e = cudaMemcpyAsync(params->out_steps, d_steps, n * sizeof(unsigned), cudaMemcpyDeviceToHost, st);
  if (e == cudaSuccess && d_status) e = cudaMemcpyAsync(params->out_status, d_status, n * sizeof(unsigned), cudaMemcpyDeviceToHost, st);
  if (e == cudaSuccess && d_final) e = cudaMemcpyAsync(params->out_final, d_final, 3 * n * sizeof(float), cudaMemcpyDeviceToHost, st);
  if (e == cudaSuccess && d_totals) e = cudaMemcpyAsync(params->out_totals, d_totals, 4 * sizeof(unsigned long long), cudaMemcpyDeviceToHost, st);
  cleanup();
  if (e == cudaSuccess) e = cudaStreamSynchronize(st);
  return check(e);
}

}  // extern "C"
