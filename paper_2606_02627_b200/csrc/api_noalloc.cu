// csrc/api_noalloc.cu -- streami_trace_streamlines_noalloc: the streamline trace for callers that cannot
// allocate (code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc).
//
// It is streami_trace_streamlines (api_trace.cu: Tracer::trace() in Streamlines mode) with
// every piece of scratch that call takes from the stream-ordered allocator -- the global work counter of the
// persistent kernel, and for n >= 65,536 seeds the Morton presort's histogram, keys, permutation and the seeds
// gathered into processing order (a12) -- placed in ONE file-scope device array of fixed size instead.  The same
// kernels run (trace_kernel via pick_trace_kernel, the presort kernels of presort.cuh), so every per-particle
// output is identical to the allocating call's.  No cudaMalloc / cudaMallocAsync / cudaFree / event creation and
// no allocating library routine is called.
//
// The array is shared by every call on a device and keeps the last call's contents: the counters and the
// histogram are cleared at the start of each call (on the caller's stream); calls that overlap on the GPU
// (different streams, or different host threads without ordering between their streams) RACE on it and must
// not be issued.  Every GPU that loads the library holds the array (NOALLOC_SCRATCH_BYTES, ~7.0 MiB) until exit.
#include <mutex>

#include "internal.h"
#include "presort.cuh"
#include "trace_kernel.cuh"

namespace streami {

typedef void (*TraceKernel)(const TraceArgs);
TraceKernel pick_trace_kernel(int layout, int integ, bool unsteady, bool brick, bool cache, bool unit);
bool unit_geometry(const Geom& g);
int trace_grid(TraceKernel k, unsigned long long nwork, int block, int* grid);
int check_params(const streami_params* p, bool need_capacity);
void fill_integrator(TraceArgs& a, const streami_params* p);

// ---- the static scratch: layout in bytes, every part 256-byte aligned --------------------------------------
constexpr size_t NOALLOC_MAX_SEEDS = STREAMI_NOALLOC_MAX_SEEDS;          // 262,144
constexpr unsigned NOALLOC_MAX_BITS = 6;                                 // Morton blocks: at most 64 per axis
constexpr unsigned NOALLOC_MAX_BINS = 1u << (3 * NOALLOC_MAX_BITS);      // 262,144 bins
constexpr unsigned NOALLOC_MAX_SEG = NOALLOC_MAX_BINS / PRESORT_SEG;     // 256 scan segments
constexpr size_t OFF_CTR = 0;                                            // work counter u64 (+ spare), 256 B
constexpr size_t OFF_HIST = 256;                                         // (bins + segments) x u32
constexpr size_t OFF_KEYS = OFF_HIST + sizeof(unsigned) * ((size_t)NOALLOC_MAX_BINS + NOALLOC_MAX_SEG);
constexpr size_t OFF_PERM = OFF_KEYS + sizeof(unsigned) * NOALLOC_MAX_SEEDS;
constexpr size_t OFF_SEEDS4 = OFF_PERM + sizeof(unsigned) * NOALLOC_MAX_SEEDS;
constexpr size_t NOALLOC_SCRATCH_BYTES = OFF_SEEDS4 + sizeof(float4) * NOALLOC_MAX_SEEDS;   // 7,341,312
static_assert(OFF_KEYS % 256 == 0 && OFF_PERM % 256 == 0 && OFF_SEEDS4 % 256 == 0, "scratch parts are 256-byte aligned");

// In HOST code this name is a host-side stand-in, not a device address: only cudaGetSymbolAddress (below) gives
// the pointer a kernel may be handed.
static __device__ __align__(256) unsigned char g_noalloc_scratch[NOALLOC_SCRATCH_BYTES];

// Device address of the array, resolved once per device with that device current.
static int noalloc_scratch(unsigned char** out) {
  constexpr int MAX_DEV = 64;
  static std::mutex mu;
  static unsigned char* ptr[MAX_DEV] = {};
  int dev = 0;
  STREAMI_TRY(cudaGetDevice(&dev));
  if (dev < 0 || dev >= MAX_DEV) return STREAMI_E_INVALID;
  std::lock_guard<std::mutex> lk(mu);
  if (!ptr[dev]) {
    void* p = nullptr;
    STREAMI_TRY(cudaGetSymbolAddress(&p, g_noalloc_scratch));     // `dev` is current: its copy of the array
    if (!p) return STREAMI_E_CUDA;
    ptr[dev] = (unsigned char*)p;
  }
  *out = ptr[dev];
  return STREAMI_OK;
}

}  // namespace streami

using namespace streami;

extern "C" {

int streami_trace_streamlines_noalloc(streami_field f, const float* seeds, size_t n,
                                      const streami_params* params, float* out_vertices,
                                      unsigned* out_counts, void* cuda_stream) {
  OptionsScope options_scope;
  if (!f || f->bricked || (n > 0 && (!seeds || !out_counts))) return STREAMI_E_INVALID;
  int rc = check_params(params, true);
  if (rc) return rc;
  if (n > NOALLOC_MAX_SEEDS) return STREAMI_E_TOO_LARGE;           // the static scratch holds no more
  cudaStream_t st = (cudaStream_t)cuda_stream;
  if (params->out_totals) STREAMI_TRY(cudaMemsetAsync(params->out_totals, 0, 4 * sizeof(unsigned long long), st));
  if (n == 0) return STREAMI_OK;

  unsigned char* scratch = nullptr;
  rc = noalloc_scratch(&scratch);
  if (rc) return rc;
  unsigned long long* next = (unsigned long long*)(scratch + OFF_CTR);
  unsigned* hist = (unsigned*)(scratch + OFF_HIST);
  unsigned* keys = (unsigned*)(scratch + OFF_KEYS);
  unsigned* perm = (unsigned*)(scratch + OFF_PERM);
  float4* seeds4 = (float4*)(scratch + OFF_SEEDS4);

  const bool unsteady = f->g.nslices > 1;
  const bool cache = options().cell_cache != 0;
  TraceKernel k = pick_trace_kernel(f->layout, params->integrator, unsteady, false, cache, unit_geometry(f->g));
  int grid = 0;
  const int block = trace_block(params->integrator);
  rc = trace_grid(k, n, block, &grid);                             // occupancy query only, nothing allocated
  if (rc) return rc;

  // what must start at zero: the work counter (the array keeps the last call's contents)
  STREAMI_TRY(cudaMemsetAsync(scratch + OFF_CTR, 0, 256, st));

  // a12: Morton presort, under the same rule as the allocating call (n >= 65,536).  Block size: 4^3 cells, coarser
  // until at most 64 blocks per axis remain (the allocating call allows 128: its histogram is allocated to fit).
  const bool sorting = options().presort && n >= 65536;
  if (sorting) {
    const int maxdim = std::max(f->dims[0], std::max(f->dims[1], f->dims[2]));
    int shift = 2;
    while (((maxdim - 1) >> shift) >= (1 << NOALLOC_MAX_BITS)) shift++;
    unsigned bits = 0;
    while ((1u << bits) <= (unsigned)((maxdim - 1) >> shift)) bits++;
    const unsigned nbins = 1u << (3 * bits);                       // <= NOALLOC_MAX_BINS
    const unsigned nseg = (nbins + PRESORT_SEG - 1) / PRESORT_SEG;
    STREAMI_TRY(cudaMemsetAsync(hist, 0, sizeof(unsigned) * nbins, st));
    const unsigned blocks = (unsigned)std::min<size_t>((n + 255) / 256, (size_t)num_sms() * 16);
    const BrickMap nobricks{1, 1, 1, 1, 1, 1};
    presort_hist_kernel<<<blocks, 256, 0, st>>>(f->g, nobricks, shift, 0, seeds, 3u, n, nullptr, hist, keys);
    presort_scan_seg_kernel<<<nseg, 256, 0, st>>>(hist, nbins, hist + nbins);
    presort_scan_top_kernel<<<1, 1024, 0, st>>>(hist + nbins, nseg);
    presort_scatter_kernel<<<blocks, 256, 0, st>>>(keys, n, nullptr, hist, hist + nbins, perm);
    gather_seeds_kernel<<<blocks, 256, 0, st>>>(seeds, perm, n, seeds4);
    launch_counter() += 5;
    STREAMI_TRY(cudaGetLastError());
  }

  TraceArgs a{};
  a.g = f->g; a.g.time_mode = params->time_mode; a.s = launch_store(f);
  a.bricks = nullptr; a.nbricks = 0;
  a.seeds = seeds; a.seeds4 = sorting ? seeds4 : nullptr; a.perm = nullptr; a.qin = nullptr;
  a.nwork = n; a.nwork_dev = nullptr; a.next = next; a.round = 0;
  a.seg_budget = 0;                                                // one launch: no segments, no in-kernel queue
  fill_integrator(a, params);
  a.verts = out_vertices; a.n = n; a.counts = out_counts;
  a.vec_ok = out_vertices && (params->capacity % 8u) == 0u && ((unsigned long long)out_vertices % 32ull) == 0ull;
  a.qout = nullptr; a.qout_count = nullptr;
  k<<<grid, block, 0, st>>>(a);
  launch_counter()++;
  return check(cudaGetLastError());
}

}  // extern "C"
