// csrc/sorter.cuh -- host driver of the Morton counting sort (a12), shared by the streamline and
// the brick round loops.
#pragma once
#include <algorithm>

#include "internal.h"
#include "presort.cuh"

namespace streami {

// Morton sort of work items (a12): a counting sort by the Morton code of the item's coarse cell
// block.  Scratch is allocated once per trace call and reused by every segment.
struct MortonSorter {
  int shift, lbits; unsigned nbins, nseg, nbricks;
  unsigned* hist; unsigned* keys; size_t cap;
  BrickMap bm;
  cudaStream_t st;

  // brick_major (bricked fields): keys are (destination brick, Morton code inside the brick), see presort.cuh
  int init(const streami_field_s* f, size_t n, cudaStream_t stream, bool brick_major = false) {
    st = stream; cap = n; hist = nullptr; keys = nullptr; lbits = 0; nbricks = 0; bm = BrickMap{1, 1, 1, 1, 1, 1};
    int maxdim = std::max(f->dims[0], std::max(f->dims[1], f->dims[2]));
    shift = 2;                                     // 4^3-cell blocks, at most 128 blocks per axis
    while (((maxdim - 1) >> shift) >= 128) shift++;
    unsigned bits = 0;
    while ((1u << bits) <= (unsigned)((maxdim - 1) >> shift)) bits++;
    nbins = 1u << (3 * bits);
    if (brick_major && f->bricked) {
      bm = f->bm; nbricks = (unsigned)f->bricks.size();
      int ext = 1;                                 // largest owned extent of a brick along any axis (the top brick takes the remainder)
      const int B[3] = {bm.Bx, bm.By, bm.Bz}, nb3[3] = {bm.nbx, bm.nby, bm.nbz};
      for (int a = 0; a < 3; ++a) ext = std::max(ext, f->dims[a] - B[a] * (nb3[a] - 1));
      lbits = 1;
      while ((1 << lbits) <= ((ext - 1) >> shift)) lbits++;
      // keep the table small: coarser blocks until nbricks * 8^lbits fits 2^24 bins
      while ((unsigned long long)nbricks << (3 * lbits) > (1ull << 24)) { shift++; lbits = 1; while ((1 << lbits) <= ((ext - 1) >> shift)) lbits++; }
      nbins = nbricks << (3 * lbits);
    }
    nseg = (nbins + PRESORT_SEG - 1) / PRESORT_SEG;
    STREAMI_TRY(cudaMallocAsync((void**)&hist, sizeof(unsigned) * ((size_t)nbins + nseg), st));   // counts + totals
    cudaError_t e = cudaMallocAsync((void**)&keys, sizeof(unsigned) * n, st);
    if (e != cudaSuccess) { cudaFreeAsync(hist, st); hist = nullptr; return check(e); }
    return STREAMI_OK;
  }
  void release() { if (hist) cudaFreeAsync(hist, st); if (keys) cudaFreeAsync(keys, st); hist = keys = nullptr; }

  // perm[0..count) = the items ordered by bin; count = n, or *n_dev (<= cap) when n_dev is set.
  // seg_offsets (brick-major only, may be NULL): [nbricks + 1] starts of the per-brick segments in perm
  int sort(const Geom& g, const float* pos, unsigned stride_floats, size_t n, const unsigned* n_dev,
           unsigned* perm, unsigned long long* seg_offsets = nullptr) {
    STREAMI_TRY(cudaMemsetAsync(hist, 0, sizeof(unsigned) * nbins, st));
    size_t items = n_dev ? cap : n;
    unsigned blocks = (unsigned)std::min<size_t>((items + 255) / 256, (size_t)num_sms() * 16);
    if (blocks == 0) blocks = 1;
    presort_hist_kernel<<<blocks, 256, 0, st>>>(g, bm, shift, lbits, pos, stride_floats, n, n_dev, hist, keys);
    presort_scan_seg_kernel<<<nseg, 256, 0, st>>>(hist, nbins, hist + nbins);
    presort_scan_top_kernel<<<1, 1024, 0, st>>>(hist + nbins, nseg);
    if (seg_offsets && lbits > 0) {
      presort_segments_kernel<<<(nbricks + 1 + 255) / 256, 256, 0, st>>>(hist, hist + nbins, 1u << (3 * lbits), nbricks, n, n_dev, seg_offsets);
      launch_counter()++;
    }
    presort_scatter_kernel<<<blocks, 256, 0, st>>>(keys, n, n_dev, hist, hist + nbins, perm);
    launch_counter() += 4;
    return check(cudaGetLastError());
  }

  // out[i] = {seed perm[i], perm[i]} / the 32-byte record perm[i]: the work items in processing order
  int gather_seeds(const float* seeds, const unsigned* perm, size_t n, float4* out) {
    unsigned blocks = (unsigned)std::min<size_t>((n + 255) / 256, (size_t)num_sms() * 16);
    gather_seeds_kernel<<<blocks ? blocks : 1, 256, 0, st>>>(seeds, perm, n, out);
    launch_counter()++;
    return check(cudaGetLastError());
  }
  int gather_rec32(const void* in, const unsigned* perm, size_t n, void* out) {
    unsigned blocks = (unsigned)std::min<size_t>((n + 255) / 256, (size_t)num_sms() * 16);
    gather_rec32_kernel<<<blocks ? blocks : 1, 256, 0, st>>>((const uint4*)in, perm, n, (uint4*)out);
    launch_counter()++;
    return check(cudaGetLastError());
  }
};

}  // namespace streami
