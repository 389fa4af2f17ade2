// csrc/lines.cuh -- polyline assembly (the paper's assembleOutput /
// getLines: "field lines are assembled ... streamlines in the order of the advection steps,
// streaklines from the youngest to the oldest particle").
//
// The tracing calls leave vertices in per-particle capacity slots (A6) or per-release slots (A7);
// these calls turn them into what a renderer or a file writer takes: one contiguous AoS point
// buffer plus a per-line offset table.  Pure data movement: an exclusive scan of the line lengths
// and a gather.
#pragma once
#include "internal.h"

namespace streami {

constexpr int SCAN_BLOCK = 256, SCAN_ITEMS = 4, SCAN_TILE = SCAN_BLOCK * SCAN_ITEMS;

// level 1: exclusive scan inside tiles of 1024 counts, tile totals out
static __global__ void __launch_bounds__(SCAN_BLOCK)
scan_tiles_kernel(const unsigned* __restrict__ counts, unsigned long long n,
                  unsigned long long* __restrict__ offsets, unsigned long long* __restrict__ tile_total) {
  __shared__ unsigned long long s_warp[SCAN_BLOCK / 32];
  const unsigned long long base = (unsigned long long)blockIdx.x * SCAN_TILE + threadIdx.x * SCAN_ITEMS;
  unsigned c[SCAN_ITEMS];
  unsigned long long mine = 0;
#pragma unroll
  for (int k = 0; k < SCAN_ITEMS; ++k) { c[k] = base + k < n ? counts[base + k] : 0u; mine += c[k]; }
  unsigned long long incl = mine;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    unsigned long long v = __shfl_up_sync(0xffffffffu, incl, d);
    if (lane >= d) incl += v;
  }
  if (lane == 31) s_warp[warp] = incl;
  __syncthreads();
  unsigned long long run = incl - mine;
  for (int w = 0; w < warp; ++w) run += s_warp[w];
#pragma unroll
  for (int k = 0; k < SCAN_ITEMS; ++k) { if (base + k < n) offsets[base + k] = run; run += c[k]; }
  if (threadIdx.x == SCAN_BLOCK - 1) tile_total[blockIdx.x] = run;
}

// level 2: one block turns the tile totals into tile bases and writes the grand total to offsets[n]
static __global__ void __launch_bounds__(1024)
scan_totals_kernel(unsigned long long* __restrict__ tile_total, unsigned ntiles,
                   unsigned long long* __restrict__ offsets, unsigned long long n) {
  __shared__ unsigned long long s_part[1024];
  const unsigned per = (ntiles + 1023u) / 1024u;
  const unsigned lo = threadIdx.x * per, hi = min(lo + per, ntiles);
  unsigned long long sum = 0;
  for (unsigned k = lo; k < hi; ++k) sum += tile_total[k];
  s_part[threadIdx.x] = sum;
  __syncthreads();
  for (unsigned d = 1; d < 1024; d <<= 1) {
    unsigned long long v = threadIdx.x >= d ? s_part[threadIdx.x - d] : 0ull;
    __syncthreads();
    s_part[threadIdx.x] += v;
    __syncthreads();
  }
  unsigned long long run = s_part[threadIdx.x] - sum;
  for (unsigned k = lo; k < hi; ++k) { unsigned long long c = tile_total[k]; tile_total[k] = run; run += c; }
  if (threadIdx.x == 1023) offsets[n] = s_part[1023];
}

static __global__ void add_bases_kernel(unsigned long long* __restrict__ offsets, unsigned long long n,
                                        const unsigned long long* __restrict__ tile_base) {
  unsigned long long i = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) offsets[i] += tile_base[i / SCAN_TILE];
}

// batches of the host polyline call: out[i] = local[i] + base (i < count), totals += part
static __global__ void rebase_offsets_kernel(const unsigned long long* __restrict__ local, unsigned long long base,
                                             unsigned long long* __restrict__ out, unsigned long long count) {
  unsigned long long i = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < count) out[i] = local[i] + base;
}
static __global__ void accumulate_totals_kernel(unsigned long long* __restrict__ dst, const unsigned long long* __restrict__ part) {
  if (threadIdx.x < 4) dst[threadIdx.x] += part[threadIdx.x];
}

// streamlines: point (line id, slot k) -> out_points[offsets[id] + k]; consecutive threads read
// consecutive slots of one particle (coalesced in each SoA plane).
static __global__ void gather_streamlines_kernel(const float* __restrict__ verts, const unsigned* __restrict__ counts,
                                                 unsigned long long n, unsigned cap,
                                                 const unsigned long long* __restrict__ offsets,
                                                 float* __restrict__ out_points) {
  const unsigned long long total = n * cap, plane = total;
  unsigned long long t = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;
  const unsigned long long step = (unsigned long long)gridDim.x * blockDim.x;
  for (; t < total; t += step) {
    const unsigned long long id = t / cap;
    const unsigned k = (unsigned)(t - id * cap);
    if (k < counts[id]) {
      float* o = out_points + 3ull * (offsets[id] + k);
      o[0] = verts[t]; o[1] = verts[plane + t]; o[2] = verts[2 * plane + t];
    }
  }
}

// streaklines: the line of rake point i = its particles that are alive (state ALIVE during a
// run, MAX_STEPS after the last step), youngest release first.
static __global__ void count_streak_kernel(const unsigned char* __restrict__ state, unsigned long long m,
                                           unsigned released, unsigned* __restrict__ counts) {
  unsigned long long i = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= m) return;
  unsigned c = 0;
  for (unsigned j = 0; j < released; ++j) { unsigned s = state[(unsigned long long)j * m + i]; c += (s == 0u || s == 2u); }
  counts[i] = c;
}
static __global__ void gather_streak_kernel(const float* __restrict__ verts, const unsigned char* __restrict__ state,
                                            unsigned long long m, unsigned nsteps, unsigned released,
                                            const unsigned long long* __restrict__ offsets,
                                            float* __restrict__ out_points) {
  unsigned long long i = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= m) return;
  const unsigned long long plane = m * (unsigned long long)nsteps;
  float* o = out_points + 3ull * offsets[i];
  for (unsigned j = released; j-- > 0;) {
    const unsigned long long id = (unsigned long long)j * m + i;
    const unsigned s = state[id];
    if (s == 0u || s == 2u) { o[0] = verts[id]; o[1] = verts[plane + id]; o[2] = verts[2 * plane + id]; o += 3; }
  }
}

// offsets[0..n] = exclusive scan of counts[0..n), offsets[n] = total.  Scratch from the stream pool.
static inline int scan_counts(const unsigned* counts, unsigned long long n, unsigned long long* offsets, cudaStream_t st) {
  if (n == 0) return check(cudaMemsetAsync(offsets, 0, sizeof(unsigned long long), st));
  const unsigned ntiles = (unsigned)((n + SCAN_TILE - 1) / SCAN_TILE);
  unsigned long long* tiles = nullptr;
  STREAMI_TRY(cudaMallocAsync((void**)&tiles, sizeof(unsigned long long) * ntiles, st));
  scan_tiles_kernel<<<ntiles, SCAN_BLOCK, 0, st>>>(counts, n, offsets, tiles);
  scan_totals_kernel<<<1, 1024, 0, st>>>(tiles, ntiles, offsets, n);
  add_bases_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(offsets, n, tiles);
  launch_counter() += 3;
  cudaError_t e = cudaGetLastError();
  cudaFreeAsync(tiles, st);
  return check(e);
}

}  // namespace streami
