// csrc/presort.cuh -- a12 of SURVEY.md 8(a): order the seeds by the Morton code of their coarse
// cell block before tracing (the build's choice; not in the paper).  It is a permutation only:
// every output is indexed by particle id, so results do not change.  Purpose: lanes that run at
// the same time work in the same region of the field, so the gathers of concurrently resident
// warps hit the same L2 lines / DRAM pages / TLB entries.  Counting sort: histogram over bins,
// exclusive scan, scatter.  Order inside a bin is unspecified.
#pragma once
#include "field.cuh"

namespace streami {

constexpr unsigned PRESORT_SEG = 1024;   // bins per scan segment (see the scan kernels below)

__device__ __forceinline__ unsigned spread3(unsigned x) {   // 10 bits -> every third bit
  x &= 0x3ffu;
  x = (x | (x << 16)) & 0x030000ffu;
  x = (x | (x << 8)) & 0x0300f00fu;
  x = (x | (x << 4)) & 0x030c30c3u;
  x = (x | (x << 2)) & 0x09249249u;
  return x;
}

// Positions are read with a stride in floats: 3 for the seed array, 8 for queue records.
__device__ __forceinline__ unsigned seed_bin(const Geom& g, int shift, const float* pos, unsigned stride,
                                             unsigned long long i) {
  float gx, gy, gz;
  const float* p = pos + (unsigned long long)stride * i;
  if (!to_index(g, p[0], p[1], p[2], gx, gy, gz)) return 0u;
  unsigned bx = (unsigned)__float2int_rz(gx) >> shift, by = (unsigned)__float2int_rz(gy) >> shift,
           bz = (unsigned)__float2int_rz(gz) >> shift;
  return spread3(bx) | (spread3(by) << 1) | (spread3(bz) << 2);
}

// Brick-major key (a9: per-destination segments): key = brick * 2^(3 lbits) + Morton code of the item's cell
// block RELATIVE to its brick's owned box, so that the sorted work of a round is one contiguous range per
// destination brick -- Q_r[b] of A9, the "send buffer" a data-sharded run would hand to rank b (PAPER.md:63-65,
// 101) -- and Morton-ordered inside it.  The brick of a queue record is its word 5 (written by emit_outgoing),
// the brick of a seed is its owner (A9).  Items outside the domain go to bin 0.
__device__ __forceinline__ unsigned brick_bin(const Geom& g, const BrickMap& m, int shift, int lbits, const float* pos,
                                              unsigned stride, unsigned long long i) {
  float gx, gy, gz;
  const float* p = pos + (unsigned long long)stride * i;
  if (!to_index(g, p[0], p[1], p[2], gx, gy, gz)) return 0u;
  const int ix = __float2int_rz(gx), iy = __float2int_rz(gy), iz = __float2int_rz(gz);
  int bx, by, bz;
  if (stride == 8u) {                        // queue record: destination brick as stored
    const unsigned b = __float_as_uint(p[5]);
    bx = (int)(b % (unsigned)m.nbx); by = (int)((b / (unsigned)m.nbx) % (unsigned)m.nby); bz = (int)(b / (unsigned)(m.nbx * m.nby));
  } else {
    bx = min(ix / m.Bx, m.nbx - 1); by = min(iy / m.By, m.nby - 1); bz = min(iz / m.Bz, m.nbz - 1);
  }
  const unsigned lim = (1u << lbits) - 1u;
  const unsigned lx = min((unsigned)max(ix - bx * m.Bx, 0) >> shift, lim), ly = min((unsigned)max(iy - by * m.By, 0) >> shift, lim),
                 lz = min((unsigned)max(iz - bz * m.Bz, 0) >> shift, lim);
  const unsigned b = (unsigned)((bz * m.nby + by) * m.nbx + bx);
  return (b << (3 * lbits)) | spread3(lx) | (spread3(ly) << 1) | (spread3(lz) << 2);
}

// The item count is `n`, or *n_dev when n_dev is set (a queue whose size only the device knows).
// lbits > 0: brick-major keys (brick_bin), else plain Morton keys of the global grid.
static __global__ void presort_hist_kernel(Geom g, BrickMap bm, int shift, int lbits, const float* __restrict__ pos, unsigned stride,
                                    unsigned long long n, const unsigned* __restrict__ n_dev,
                                    unsigned* __restrict__ hist, unsigned* __restrict__ keys) {
  if (n_dev) n = *n_dev;
  unsigned long long i = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;
  const unsigned long long step = (unsigned long long)gridDim.x * blockDim.x;
  for (; i < n; i += step) {
    unsigned k = lbits > 0 ? brick_bin(g, bm, shift, lbits, pos, stride, i) : seed_bin(g, shift, pos, stride, i);
    keys[i] = k;
    atomicAdd(hist + k, 1u);
  }
}

// Start of every brick's segment in the sorted order (brick-major keys): offsets[b] for b = 0..nb, read from the
// exclusive scan BEFORE the scatter advances it.
static __global__ void presort_segments_kernel(const unsigned* __restrict__ scanned, const unsigned* __restrict__ seg_base,
                                               unsigned bins_per_brick, unsigned nbricks, unsigned long long n,
                                               const unsigned* __restrict__ n_dev, unsigned long long* __restrict__ offsets) {
  if (n_dev) n = *n_dev;
  const unsigned b = blockIdx.x * blockDim.x + threadIdx.x;
  if (b < nbricks) {
    const unsigned k = b * bins_per_brick;
    offsets[b] = (unsigned long long)scanned[k] + seg_base[k / PRESORT_SEG];
  } else if (b == nbricks) {
    offsets[b] = n;
  }
}

// Exclusive scan of `hist` in two levels.  Level 1: each block scans one segment of 1024 bins in
// place (4 consecutive bins per thread, warp shuffles, one shared-memory hop) and writes the
// segment total.  Level 2: one block scans the <= 2048 segment totals.  The scatter adds both.

static __global__ void __launch_bounds__(256)
presort_scan_seg_kernel(unsigned* __restrict__ hist, unsigned nbins, unsigned* __restrict__ seg_total) {
  __shared__ unsigned s_warp[8];
  const unsigned base = blockIdx.x * PRESORT_SEG + threadIdx.x * 4u;
  unsigned c[4];
#pragma unroll
  for (int k = 0; k < 4; ++k) c[k] = (base + k < nbins) ? hist[base + k] : 0u;
  const unsigned mine = c[0] + c[1] + c[2] + c[3];
  unsigned incl = mine;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    unsigned v = __shfl_up_sync(0xffffffffu, incl, d);
    if (lane >= d) incl += v;
  }
  if (lane == 31) s_warp[warp] = incl;
  __syncthreads();
  unsigned woff = 0;
  for (int w = 0; w < warp; ++w) woff += s_warp[w];
  unsigned run = woff + incl - mine;
#pragma unroll
  for (int k = 0; k < 4; ++k) {
    if (base + k < nbins) hist[base + k] = run;
    run += c[k];
  }
  if (threadIdx.x == 255) seg_total[blockIdx.x] = run;
}

static __global__ void __launch_bounds__(1024)
presort_scan_top_kernel(unsigned* __restrict__ seg_total, unsigned nseg) {
  __shared__ unsigned s_part[1024];
  const unsigned per = (nseg + 1023u) / 1024u;
  const unsigned lo = threadIdx.x * per, hi = min(lo + per, nseg);
  unsigned sum = 0;
  for (unsigned k = lo; k < hi; ++k) sum += seg_total[k];
  s_part[threadIdx.x] = sum;
  __syncthreads();
  for (unsigned d = 1; d < 1024; d <<= 1) {                 // Hillis-Steele inclusive scan
    unsigned v = threadIdx.x >= d ? s_part[threadIdx.x - d] : 0u;
    __syncthreads();
    s_part[threadIdx.x] += v;
    __syncthreads();
  }
  unsigned run = s_part[threadIdx.x] - sum;
  for (unsigned k = lo; k < hi; ++k) { unsigned c = seg_total[k]; seg_total[k] = run; run += c; }
}

static __global__ void presort_scatter_kernel(const unsigned* __restrict__ keys, unsigned long long n,
                                       const unsigned* __restrict__ n_dev,
                                       unsigned* __restrict__ offsets,
                                       const unsigned* __restrict__ seg_base,
                                       unsigned* __restrict__ perm) {
  if (n_dev) n = *n_dev;
  unsigned long long i = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;
  const unsigned long long step = (unsigned long long)gridDim.x * blockDim.x;
  for (; i < n; i += step) {
    const unsigned k = keys[i];
    unsigned pos = atomicAdd(offsets + k, 1u) + seg_base[k / PRESORT_SEG];
    perm[pos] = (unsigned)i;
  }
}

// The work items in processing order, so that a refilling lane reads ONE record at its work index
// instead of perm[w] and then the item (one dependent L2 round trip less per refill, with the whole
// warp waiting).  Seeds become {x, y, z, id}; 32-byte queue records are copied as they are.
static __global__ void gather_seeds_kernel(const float* __restrict__ seeds, const unsigned* __restrict__ perm,
                                           unsigned long long n, float4* __restrict__ out) {
  unsigned long long i = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;
  const unsigned long long step = (unsigned long long)gridDim.x * blockDim.x;
  for (; i < n; i += step) {
    const unsigned id = perm[i];
    out[i] = make_float4(seeds[3ull * id], seeds[3ull * id + 1], seeds[3ull * id + 2], __uint_as_float(id));
  }
}

static __global__ void gather_rec32_kernel(const uint4* __restrict__ in, const unsigned* __restrict__ perm,
                                           unsigned long long n, uint4* __restrict__ out) {
  unsigned long long i = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;
  const unsigned long long step = (unsigned long long)gridDim.x * blockDim.x;
  for (; i < n; i += step) {
    const unsigned long long src = perm[i];
    out[2 * i] = in[2 * src]; out[2 * i + 1] = in[2 * src + 1];
  }
}

}  // namespace streami
