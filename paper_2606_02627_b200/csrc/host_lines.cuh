// csrc/host_lines.cuh -- host-buffer plumbing shared by the API translation units: device mirrors of
// host arrays, and the "seeds (host) in, assembled polylines (host) out" call for any tracer
// (structured fields, bricks, meshes).
#pragma once
#include <algorithm>
#include <vector>

#include "internal.h"
#include "lines.cuh"

namespace streami {

// Device mirrors of host buffers on one stream: allocate (+ upload), download, free.
struct Mirror {
  cudaStream_t st;
  std::vector<void*> dev;
  std::vector<std::pair<void*, std::pair<void*, size_t>>> back;   // device -> (host, bytes)
  cudaError_t err = cudaSuccess;
  explicit Mirror(cudaStream_t s) : st(s) {}
  void* make(const void* host_in, void* host_out, size_t bytes) {
    if (err != cudaSuccess || bytes == 0 || (!host_in && !host_out)) return nullptr;
    void* d = nullptr;
    err = cudaMallocAsync(&d, bytes, st);
    if (err != cudaSuccess) return nullptr;
    dev.push_back(d);
    if (host_in) err = cudaMemcpyAsync(d, host_in, bytes, cudaMemcpyHostToDevice, st);
    if (host_out) back.push_back({d, {host_out, bytes}});
    return d;
  }
  cudaError_t download() {
    for (auto& b : back)
      if (err == cudaSuccess) err = cudaMemcpyAsync(b.second.first, b.first, b.second.second, cudaMemcpyDeviceToHost, st);
    return err;
  }
  ~Mirror() { for (void* d : dev) cudaFreeAsync(d, st); }
};

// trace(d_seeds, n, params, d_vertices, d_counts) -> status runs one tracing call on cuda_stream.
template <class Trace>
int lines_host(Trace&& trace, bool one_batch, const float* seeds, size_t n, const streami_params* params,
               unsigned long long* out_offsets, float* out_points, unsigned long long max_points,
               unsigned long long* out_total, void* cuda_stream) {
  if (!params || !out_offsets || (n > 0 && !seeds) || (max_points > 0 && !out_points)) return STREAMI_E_INVALID;
  if (params->capacity == 0) return STREAMI_E_INVALID;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  if (out_total) *out_total = 0;
  if (n == 0) { out_offsets[0] = 0; return STREAMI_OK; }
  // Batches: the polylines of batch b cross the bus on a second stream while batch b+1 is traced
  // (on C2 the 1.33 GB of points take longer than the trace itself).  A batch must still hold a few
  // particles per resident lane, or the persistent kernel has nothing to balance: automatic = at
  // most 4 batches of at least 262,144 seeds.  Results do not depend on the split (ids are local to
  // a batch only inside the library).
  size_t per = (size_t)options().host_batch;
  // Points cost 12 B per `stride` steps on a ~50 GB/s bus against ~2e-11 s per RK4 step: only a dense
  // recording (C2, stride 8: the copy takes 1.5x the trace) has a copy worth hiding; with a sparse one
  // (C5, stride 128: 3 %) the extra kernel tails of the batches are all that is left (998 -> 1,077 ms).
  if (per == 0) per = (one_batch || params->stride > 32u) ? n : std::max<size_t>((n + 3) / 4, 262144);
  per = std::min(per, n);
  const size_t nbatch = (n + per - 1) / per;
  cudaStream_t cs = st;
  if (nbatch > 1) { cs = copy_stream(); if (!cs) return STREAMI_E_CUDA; }

  int rc = STREAMI_OK;
  unsigned long long total = 0;
  std::vector<cudaEvent_t> events;
  {
    Mirror mr(st);
    float* d_seeds = (float*)mr.make(seeds, nullptr, 3 * n * sizeof(float));
    unsigned* d_steps = (unsigned*)mr.make(nullptr, params->out_steps, n * sizeof(unsigned));
    unsigned* d_status = (unsigned*)mr.make(nullptr, params->out_status, n * sizeof(unsigned));
    unsigned long long* d_totals = (unsigned long long*)mr.make(nullptr, params->out_totals, 4 * sizeof(unsigned long long));
    unsigned long long* d_off = (unsigned long long*)mr.make(nullptr, out_offsets, (n + 1) * sizeof(unsigned long long));
    if (mr.err != cudaSuccess) return check(mr.err);
    if (d_totals) STREAMI_TRY(cudaMemsetAsync(d_totals, 0, 4 * sizeof(unsigned long long), st));
    for (size_t b = 0; b < nbatch && rc == STREAMI_OK; ++b) {
      const size_t s0 = b * per, nb = std::min(per, n - s0);
      float *d_v = nullptr, *d_pts = nullptr, *d_fin = nullptr; unsigned* d_c = nullptr;
      unsigned long long *d_loc = nullptr, *d_tot = nullptr;
      cudaError_t e = cudaMallocAsync((void**)&d_v, 3 * nb * (size_t)params->capacity * sizeof(float), st);
      if (e == cudaSuccess) e = cudaMallocAsync((void**)&d_c, nb * sizeof(unsigned), st);
      if (e == cudaSuccess) e = cudaMallocAsync((void**)&d_loc, (nb + 1) * sizeof(unsigned long long), st);
      if (e == cudaSuccess && params->out_final) e = cudaMallocAsync((void**)&d_fin, 3 * nb * sizeof(float), st);
      if (e == cudaSuccess && d_totals) e = cudaMallocAsync((void**)&d_tot, 4 * sizeof(unsigned long long), st);
      if (e != cudaSuccess) rc = check(e);
      unsigned long long tb = 0;
      if (rc == STREAMI_OK) {
        streami_params dp = *params;
        dp.out_steps = d_steps ? d_steps + s0 : nullptr; dp.out_status = d_status ? d_status + s0 : nullptr;
        dp.out_final = d_fin; dp.out_totals = d_tot;
        rc = trace(d_seeds + 3 * s0, nb, &dp, d_v, d_c);
      }
      if (rc == STREAMI_OK) rc = streami_streamline_lines(d_v, d_c, nb, params->capacity, d_loc, nullptr, &tb, cuda_stream);
      if (rc == STREAMI_OK && tb > 0) {
        e = cudaMallocAsync((void**)&d_pts, 3 * tb * sizeof(float), st);
        if (e != cudaSuccess) rc = check(e);
        else rc = streami_streamline_lines(d_v, d_c, nb, params->capacity, d_loc, d_pts, nullptr, cuda_stream);
      }
      if (rc == STREAMI_OK) {
        rebase_offsets_kernel<<<(unsigned)((nb + 1 + 255) / 256), 256, 0, st>>>(d_loc, total, d_off + s0, nb + 1);
        launch_counter()++;
        if (d_tot) { accumulate_totals_kernel<<<1, 32, 0, st>>>(d_totals, d_tot); launch_counter()++; }
        rc = check(cudaGetLastError());
      }
      if (d_v) cudaFreeAsync(d_v, st);
      if (d_c) cudaFreeAsync(d_c, st);
      if (d_loc) cudaFreeAsync(d_loc, st);
      if (d_tot) cudaFreeAsync(d_tot, st);
      // the batch's points (and final positions) go out on the copy stream
      if (rc == STREAMI_OK && cs != st) {
        cudaEvent_t ev = nullptr;
        e = cudaEventCreateWithFlags(&ev, cudaEventDisableTiming);
        if (e == cudaSuccess) { events.push_back(ev); e = cudaEventRecord(ev, st); }
        if (e == cudaSuccess) e = cudaStreamWaitEvent(cs, ev, 0);
        if (e != cudaSuccess) rc = check(e);
      }
      if (rc == STREAMI_OK) {
        const unsigned long long room = total < max_points ? max_points - total : 0ull;
        const unsigned long long copy = tb < room ? tb : room;
        e = cudaSuccess;
        if (copy) e = cudaMemcpyAsync(out_points + 3 * total, d_pts, 3 * copy * sizeof(float), cudaMemcpyDeviceToHost, cs);
        for (int c = 0; c < 3 && d_fin && e == cudaSuccess; ++c)
          e = cudaMemcpyAsync(params->out_final + c * n + s0, d_fin + c * nb, nb * sizeof(float), cudaMemcpyDeviceToHost, cs);
        if (e != cudaSuccess) rc = check(e);
      }
      // freed on the copy stream only if that stream was made to wait for the tracing stream above (rc == OK);
      // on an error path the tracing stream itself frees them, in order behind the kernels that write them
      if (d_pts) cudaFreeAsync(d_pts, rc == STREAMI_OK ? cs : st);
      if (d_fin) cudaFreeAsync(d_fin, rc == STREAMI_OK ? cs : st);
      total += tb;
    }
    if (cs != st) {                               // the caller's stream covers the copies as well
      cudaEvent_t ev = nullptr;
      cudaError_t e = cudaEventCreateWithFlags(&ev, cudaEventDisableTiming);
      if (e == cudaSuccess) { events.push_back(ev); e = cudaEventRecord(ev, cs); }
      if (e == cudaSuccess) e = cudaStreamWaitEvent(st, ev, 0);
      if (e != cudaSuccess && rc == STREAMI_OK) rc = check(e);
    }
    if (rc == STREAMI_OK && mr.download() != cudaSuccess) rc = check(mr.err);
  }
  {
    cudaError_t e = cudaStreamSynchronize(st);
    if (cs != st) { cudaError_t e2 = cudaStreamSynchronize(cs); if (e == cudaSuccess) e = e2; }
    if (rc == STREAMI_OK) rc = check(e);
  }
  for (cudaEvent_t ev : events) cudaEventDestroy(ev);
  if (out_total) *out_total = total;
  if (rc == STREAMI_OK && total > max_points) rc = STREAMI_E_TRUNCATED;
  return rc;
}


}  // namespace streami
