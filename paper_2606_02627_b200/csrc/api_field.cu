// csrc/api_field.cu -- field handles (D2/D3 of SURVEY.md: the host class that "is primarily
// responsible for data handling"), layout repack, options, streami_sample.
#include <cmath>
#include <cstring>
#include <limits>
#include <mutex>
#include <utility>
#include <vector>

#include "internal.h"
#include "misc_kernels.cuh"

namespace streami {

// process-wide option values, in the member order of Options (internal.h)
static std::atomic<int> g_options[N_OPTIONS] = {{1}, {1}, {0}, {0}, {0}, {1}, {3}, {0}, {0}, {1}, {0}, {0}};
static const char* const g_option_names[N_OPTIONS] = {"cell_cache", "presort", "streak_window", "kernel_timing", "segment_steps",
                                                      "vertex_staging", "prefetch", "max_blocks_per_sm", "brick_round_steps",
                                                      "integer_accept", "host_batch", "queue_steps"};
static_assert(sizeof(Options) == N_OPTIONS * sizeof(int), "Options is N_OPTIONS ints");
static thread_local Options tl_options;
static thread_local int tl_options_depth = 0;
static void options_snapshot(Options& o) {
  int* v = reinterpret_cast<int*>(&o);
  for (int i = 0; i < N_OPTIONS; ++i) v[i] = g_options[i].load(std::memory_order_relaxed);
}
const Options& options() {
  if (tl_options_depth == 0) options_snapshot(tl_options);
  return tl_options;
}
OptionsScope::OptionsScope() { if (tl_options_depth++ == 0) options_snapshot(tl_options); }
OptionsScope::~OptionsScope() { --tl_options_depth; }
int option_index(const char* name) {
  for (int i = 0; i < N_OPTIONS; ++i) if (!strcmp(name, g_option_names[i])) return i;
  return -1;
}
void option_store(int index, int value) { g_options[index].store(value, std::memory_order_relaxed); }
int option_load(int index) { return g_options[index].load(std::memory_order_relaxed); }
std::atomic<unsigned long long>& launch_counter() { static std::atomic<unsigned long long> c{0}; return c; }

static std::mutex g_err_mutex;
static std::string g_cuda_err = "CUDA error";
void set_cuda_error(cudaError_t e) {
  std::lock_guard<std::mutex> lk(g_err_mutex);
  g_cuda_err = std::string("CUDA error: ") + cudaGetErrorName(e) + ": " + cudaGetErrorString(e);
  cudaGetLastError();   // clear the sticky-less error state
}

int num_sms() {
  static int n = 0;
  if (n == 0) {
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return 0;
    if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) n = 0;
  }
  return n;
}

cudaStream_t copy_stream() {
  static cudaStream_t s = [] {
    cudaStream_t c = nullptr;
    if (cudaStreamCreateWithFlags(&c, cudaStreamNonBlocking) != cudaSuccess) { cudaGetLastError(); c = nullptr; }
    return c;
  }();
  return s;
}

static std::mutex g_time_mutex;
static std::vector<std::pair<cudaEvent_t, cudaEvent_t>> g_time_pairs;   // recorded, not yet read
static std::vector<cudaEvent_t> g_time_free;
static cudaEvent_t g_time_open = nullptr;

static cudaEvent_t take_event() {
  if (!g_time_free.empty()) { cudaEvent_t e = g_time_free.back(); g_time_free.pop_back(); return e; }
  cudaEvent_t e = nullptr;
  if (cudaEventCreate(&e) != cudaSuccess) return nullptr;
  return e;
}

void timing_begin(cudaStream_t st) {
  if (!options().kernel_timing) return;
  std::lock_guard<std::mutex> lk(g_time_mutex);
  g_time_open = take_event();
  if (g_time_open) cudaEventRecord(g_time_open, st);
}

void timing_end(cudaStream_t st) {
  if (!options().kernel_timing) return;
  std::lock_guard<std::mutex> lk(g_time_mutex);
  if (!g_time_open) return;
  cudaEvent_t e = take_event();
  if (e) { cudaEventRecord(e, st); g_time_pairs.emplace_back(g_time_open, e); }
  else g_time_free.push_back(g_time_open);
  g_time_open = nullptr;
}

static bool finite_pos(float x) { return std::isfinite(x) && x > 0.0f; }

// Scratch comes from the stream-ordered allocator.  Its default pool hands freed memory back to
// the driver at every synchronisation (release threshold 0), so a call that needs gigabytes of
// scratch (the host-buffer variants) would pay for fresh mappings each time; keep it cached.
static void keep_pool_cached() {
  static std::once_flag once;
  std::call_once(once, [] {
    int dev = 0; cudaMemPool_t pool = nullptr;
    if (cudaGetDevice(&dev) == cudaSuccess && cudaDeviceGetDefaultMemPool(&pool, dev) == cudaSuccess) {
      unsigned long long keep = ~0ull;
      cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &keep);
    }
    cudaGetLastError();
  });
}

// Records of the library-owned copy of a stored box of nx*ny*nz vertices x nslices.
static unsigned long long layout_records(int layout, unsigned nx, unsigned ny, unsigned nz, unsigned nslices) {
  if (layout == LAYOUT_CELL) return (unsigned long long)(nx - 1) * (ny - 1) * (nz - 1) * nslices;
  return (unsigned long long)nx * ny * nz * nslices;
}
static size_t layout_record_bytes(int layout) {
  return (layout == LAYOUT_FLOAT4 || layout == LAYOUT_TEX) ? 16 : (layout == LAYOUT_XPAIR ? 32 : (layout == LAYOUT_CELL ? 128 : (layout == LAYOUT_XYQUAD ? 64 : 12)));
}

// Build the library-owned copy of one packed float3 array (stored box nx*ny*nz, nslices slices).
static int repack(const float* src, unsigned nx, unsigned ny, unsigned nz, unsigned nslices, int layout,
                  void** out, size_t* bytes) {
  *out = nullptr; *bytes = 0;
  if (layout == LAYOUT_PACKED3) { *out = const_cast<float*>(src); return STREAMI_OK; }
  const unsigned long long nvert = (unsigned long long)nx * ny * nz * nslices;
  const unsigned long long nrec = layout_records(layout, nx, ny, nz, nslices);
  const size_t rec = layout_record_bytes(layout);
  void* dst = nullptr;
  STREAMI_TRY(cudaMalloc(&dst, rec * nrec + 32));   // +32: FLOAT4 reads p[1] of the last vertex
  int blocks = 148 * 8;
  if (layout == LAYOUT_FLOAT4 || layout == LAYOUT_TEX)
    repack_float4_kernel<<<blocks, 256>>>(src, (float4*)dst, nvert);
  else if (layout == LAYOUT_SOA)
    repack_soa_kernel<<<blocks, 256>>>(src, (float*)dst, nvert);
  else if (layout == LAYOUT_XPAIR)
    repack_xpair_kernel<<<blocks, 256>>>(src, (float4*)dst, nvert, nx);
  else if (layout == LAYOUT_XYQUAD)
    repack_xyquad_kernel<<<blocks, 256>>>(src, (float4*)dst, nvert, nx, ny);
  else
    repack_cell_kernel<<<blocks, 256>>>(src, (float4*)dst, nx, ny, nz, nslices);
  launch_counter()++;
  cudaError_t e = cudaGetLastError();
  if (e == cudaSuccess) e = cudaMemset((char*)dst + rec * nrec, 0, 32);
  if (e == cudaSuccess) e = cudaStreamSynchronize(0);
  if (e != cudaSuccess) { cudaFree(dst); return check(e); }
  *out = dst; *bytes = rec * nrec + 32;
  return STREAMI_OK;
}

// LAYOUT_TEX: a texture object in point mode over the float4 copy (tex1Dfetch).  A linear texture holds at most
// maxTexture1DLinear texels; larger stores are refused (INVALID).
static int make_texture(void* data, unsigned long long nvert, unsigned long long* tex) {
  int dev = 0, lim = 0;
  STREAMI_TRY(cudaGetDevice(&dev));
  STREAMI_TRY(cudaDeviceGetAttribute(&lim, cudaDevAttrMaxTexture1DLinearWidth, dev));
  if (nvert + 2 > (unsigned long long)lim) return STREAMI_E_INVALID;
  cudaResourceDesc rd; memset(&rd, 0, sizeof(rd));
  rd.resType = cudaResourceTypeLinear; rd.res.linear.devPtr = data;
  rd.res.linear.desc = cudaCreateChannelDesc<float4>(); rd.res.linear.sizeInBytes = 16ull * (nvert + 2);
  cudaTextureDesc td; memset(&td, 0, sizeof(td));
  td.filterMode = cudaFilterModePoint; td.readMode = cudaReadModeElementType; td.addressMode[0] = cudaAddressModeClamp;
  cudaTextureObject_t t = 0;
  STREAMI_TRY(cudaCreateTextureObject(&t, &rd, &td, nullptr));
  *tex = (unsigned long long)t;
  return STREAMI_OK;
}

// LAYOUT_CELL addresses cells, not vertices: the strides of the store become those of the cell grid.
static void cell_strides(Store& s, unsigned nx, unsigned ny, unsigned nz) {
  s.nx = nx - 1; s.nxy = (nx - 1) * (ny - 1);
  s.slice_stride = (unsigned long long)(nx - 1) * (ny - 1) * (nz - 1);
}

static int fill_geom(Geom& g, const int dims[3], const float origin[3], const float spacing[3],
                     int nslices, float slice_dt) {
  for (int a = 0; a < 3; ++a) {
    if (dims[a] < 2 || !finite_pos(spacing[a]) || !std::isfinite(origin[a])) return STREAMI_E_INVALID;
  }
  if (nslices < 1) return STREAMI_E_INVALID;
  if (nslices > 1 && !finite_pos(slice_dt)) return STREAMI_E_INVALID;
  if ((unsigned long long)dims[0] * dims[1] * dims[2] > 0xffffffffull) return STREAMI_E_INVALID;
  g.ox = origin[0]; g.oy = origin[1]; g.oz = origin[2];
  g.rx = 1.0f / spacing[0]; g.ry = 1.0f / spacing[1]; g.rz = 1.0f / spacing[2];   // A1, fp32 IEEE
  g.topx = (float)(dims[0] - 1); g.topy = (float)(dims[1] - 1); g.topz = (float)(dims[2] - 1);
  g.nslices = nslices;
  g.q = nslices > 1 ? 1.0f / slice_dt : 1.0f;
  g.top_s = (float)(nslices - 1);
  g.time_mode = 0;
  return STREAMI_OK;
}

// AUTO: the fastest layout whose library-owned copy fits HALF of the free device
// memory (the caller still has outputs to allocate).  Steady fields: CELL (128 B per cell, one L2 line
// per cell: C2 15.6 -> 15.2 ms, C3 149.6 -> 139.3 ms, C5 939 -> 741 ms against XYQUAD), else XYQUAD
// (64 B per vertex), else XPAIR (32 B per vertex).  Unsteady fields (two slices per sample: C4 249 vs
// 264 ms on XYQUAD): XPAIR.  A caller that cannot spare the memory passes PACKED3 (no copy) or FLOAT4.
static int auto_layout(unsigned long long nvert, unsigned long long ncell, int nslices) {
  if (nslices == 1) {
    size_t free_b = 0, total_b = 0;
    if (cudaMemGetInfo(&free_b, &total_b) == cudaSuccess) {
      if (128ull * ncell <= free_b / 2) return LAYOUT_CELL;
      if (64ull * nvert <= free_b / 2) return LAYOUT_XYQUAD;
    }
    cudaGetLastError();
  }
  return LAYOUT_XPAIR;
}

// Tame scan of n packed floats (sample_nb in field.cuh says what it licenses).
static int scan_tame(const float* dev_ptr, unsigned long long n, bool* tame) {
  unsigned* flag = nullptr; unsigned bad = 1u;
  cudaError_t e = cudaMalloc((void**)&flag, sizeof(unsigned));
  if (e == cudaSuccess) e = cudaMemset(flag, 0, sizeof(unsigned));
  if (e == cudaSuccess) {
    tame_scan_kernel<<<148 * 8, 256>>>(dev_ptr, n, flag);
    launch_counter()++;
    e = cudaMemcpy(&bad, flag, sizeof(unsigned), cudaMemcpyDeviceToHost);
  }
  cudaFree(flag);
  *tame = bad == 0u;
  return check(e);
}

static int pick_layout(int hint) {
  if (hint == STREAMI_LAYOUT_AUTO) return 0;              // decided per stored array (auto_layout)
  if (hint == STREAMI_LAYOUT_PACKED3 || hint == STREAMI_LAYOUT_FLOAT4 || hint == STREAMI_LAYOUT_XPAIR ||
      hint == STREAMI_LAYOUT_CELL || hint == STREAMI_LAYOUT_XYQUAD || hint == STREAMI_LAYOUT_SOA || hint == STREAMI_LAYOUT_TEX)
    return hint;
  return -1;
}

}  // namespace streami

using namespace streami;

extern "C" {

int streami_field_create(const int dims[3], const float origin[3], const float spacing[3],
                         int nslices, float slice_dt, const float* dev_ptr, int layout_hint,
                         streami_field* out) {
  OptionsScope options_scope;
  if (!dims || !origin || !spacing || !dev_ptr || !out) return STREAMI_E_INVALID;
  *out = nullptr;
  int layout = pick_layout(layout_hint);
  if (layout < 0) return STREAMI_E_INVALID;
  keep_pool_cached();
  streami_field_s* f = new streami_field_s();
  int rc = fill_geom(f->g, dims, origin, spacing, nslices, slice_dt);
  if (rc) { delete f; return rc; }
  for (int a = 0; a < 3; ++a) f->dims[a] = dims[a];
  f->layout = layout; f->bricked = false; f->d_bricks = nullptr; f->owned_bytes = 0;
  Store& s = f->store;
  s.lox = s.loy = s.loz = 0;
  s.hix = dims[0] - 1; s.hiy = dims[1] - 1; s.hiz = dims[2] - 1;
  s.topflagx = s.topflagy = s.topflagz = 1;
  s.cmx = s.hix - 1; s.cmy = s.hiy - 1; s.cmz = s.hiz - 1;
  s.fastx = s.fasty = s.fastz = 0u; s.self = nullptr;
  s.nx = (unsigned)dims[0]; s.nxy = (unsigned)dims[0] * (unsigned)dims[1];
  s.slice_stride = (unsigned long long)dims[0] * dims[1] * dims[2];
  void* data = nullptr; size_t bytes = 0;
  const bool automatic = layout == 0;
  if (automatic) layout = auto_layout(s.slice_stride, (unsigned long long)(dims[0] - 1) * (dims[1] - 1) * (dims[2] - 1), nslices);
  rc = repack(dev_ptr, (unsigned)dims[0], (unsigned)dims[1], (unsigned)dims[2], (unsigned)nslices, layout, &data, &bytes);
  if (rc == STREAMI_E_NOMEM && automatic && layout == LAYOUT_CELL) {      // AUTO never fails for its own ambition
    layout = LAYOUT_XYQUAD;
    rc = repack(dev_ptr, (unsigned)dims[0], (unsigned)dims[1], (unsigned)dims[2], (unsigned)nslices, layout, &data, &bytes);
  }
  if (rc == STREAMI_E_NOMEM && automatic && layout != LAYOUT_XPAIR) {
    layout = LAYOUT_XPAIR;
    rc = repack(dev_ptr, (unsigned)dims[0], (unsigned)dims[1], (unsigned)dims[2], (unsigned)nslices, layout, &data, &bytes);
  }
  if (rc == STREAMI_E_NOMEM && automatic) {                               // last resort: the caller's array in place
    layout = LAYOUT_PACKED3;
    rc = repack(dev_ptr, (unsigned)dims[0], (unsigned)dims[1], (unsigned)dims[2], (unsigned)nslices, layout, &data, &bytes);
  }
  f->layout = layout;
  if (rc) { delete f; return rc; }
  f->tame = false;
  // PACKED3 reads the caller's BORROWED array live (the in-situ use the paper targets): the
  // application may write NaN or Inf into it after this scan, so the integer accept is not licensed there.
  if (nslices == 1 && layout != LAYOUT_PACKED3) {                 // only the steady paths ask
    rc = scan_tame(dev_ptr, 3ull * s.slice_stride, &f->tame);
    if (rc) { if (bytes) cudaFree(data); delete f; return rc; }
  }
  if (layout == LAYOUT_CELL) cell_strides(s, (unsigned)dims[0], (unsigned)dims[1], (unsigned)dims[2]);
  s.data = data;
  s.plane = s.slice_stride * (unsigned long long)nslices; s.tex = 0ull;
  if (bytes) { f->owned.push_back(data); f->owned_bytes += bytes; }
  if (layout == LAYOUT_TEX) {
    rc = make_texture(data, s.slice_stride * (unsigned long long)nslices, &s.tex);
    if (rc) { cudaFree(data); delete f; return rc; }
    f->textures.push_back(s.tex);
  }
  *out = f;
  return STREAMI_OK;
}

int streami_field_create_bricked(const int global_dims[3], const float origin[3],
                                 const float spacing[3], const int brick_grid[3], int ghost_cells,
                                 const float* const* brick_dev_ptrs, int layout_hint,
                                 streami_field* out) {
  OptionsScope options_scope;
  if (!global_dims || !origin || !spacing || !brick_grid || !brick_dev_ptrs || !out)
    return STREAMI_E_INVALID;
  *out = nullptr;
  int layout = pick_layout(layout_hint);
  if (layout < 0 || ghost_cells < 1) return STREAMI_E_INVALID;
  if (layout == 0) {       // one layout for all bricks (one kernel serves them): decided on the whole grid
    const unsigned long long nv = (unsigned long long)global_dims[0] * global_dims[1] * global_dims[2];
    layout = auto_layout(nv, nv, 1);     // the bricks' cells (ghost layers included) are about as many as the vertices
  }
  for (int a = 0; a < 3; ++a)
    if (brick_grid[a] < 1 || brick_grid[a] > global_dims[a] - 1) return STREAMI_E_INVALID;
  const int nb = brick_grid[0] * brick_grid[1] * brick_grid[2];
  if (nb > 65535) return STREAMI_E_INVALID;   // the hand-off log packs dest into 16 bits
  keep_pool_cached();
  streami_field_s* f = new streami_field_s();
  int rc = fill_geom(f->g, global_dims, origin, spacing, 1, 1.0f);
  if (rc) { delete f; return rc; }
  for (int a = 0; a < 3; ++a) f->dims[a] = global_dims[a];
  f->layout = layout; f->bricked = true; f->d_bricks = nullptr; f->owned_bytes = 0; f->tame = true;
  BrickMap& m = f->bm;
  m.nbx = brick_grid[0]; m.nby = brick_grid[1]; m.nbz = brick_grid[2];
  m.Bx = global_dims[0] / m.nbx; m.By = global_dims[1] / m.nby; m.Bz = global_dims[2] / m.nbz;
  const int B[3] = {m.Bx, m.By, m.Bz};
  auto fail = [&](int code) {
    for (unsigned long long t : f->textures) cudaDestroyTextureObject((cudaTextureObject_t)t);
    for (void* p : f->owned) cudaFree(p);
    delete f;
    return code;
  };
  for (int bz = 0; bz < m.nbz; ++bz)
    for (int by = 0; by < m.nby; ++by)
      for (int bx = 0; bx < m.nbx; ++bx) {
        const int b[3] = {bx, by, bz};
        int lo[3], hi[3];
        for (int a = 0; a < 3; ++a) {
          lo[a] = std::max(B[a] * b[a] - ghost_cells, 0);
          hi[a] = std::min(B[a] * (b[a] + 1) + ghost_cells, global_dims[a] - 1);
          if (b[a] == brick_grid[a] - 1) hi[a] = global_dims[a] - 1;
          if (hi[a] - lo[a] < 1) return fail(STREAMI_E_INVALID);
        }
        const float* src = brick_dev_ptrs[(bz * m.nby + by) * m.nbx + bx];
        if (!src) return fail(STREAMI_E_INVALID);
        Store s;
        s.lox = lo[0]; s.loy = lo[1]; s.loz = lo[2];
        s.hix = hi[0]; s.hiy = hi[1]; s.hiz = hi[2];
        s.cmx = hi[0] - 1; s.cmy = hi[1] - 1; s.cmz = hi[2] - 1;
        s.topflagx = hi[0] == global_dims[0] - 1; s.topflagy = hi[1] == global_dims[1] - 1;
        s.topflagz = hi[2] == global_dims[2] - 1;
        {
          const float inf = std::numeric_limits<float>::infinity();
          s.flox = (float)lo[0]; s.floy = (float)lo[1]; s.floz = (float)lo[2];
          s.fhix = s.topflagx ? inf : (float)hi[0]; s.fhiy = s.topflagy ? inf : (float)hi[1];
          s.fhiz = s.topflagz ? inf : (float)hi[2];
          int ol[3], oh[3];
          for (int a = 0; a < 3; ++a) {
            ol[a] = B[a] * b[a];
            oh[a] = (b[a] == brick_grid[a] - 1) ? std::numeric_limits<int>::max() : B[a] * (b[a] + 1);
          }
          s.olox = ol[0]; s.oloy = ol[1]; s.oloz = ol[2]; s.ohix = oh[0]; s.ohiy = oh[1]; s.ohiz = oh[2];
        }
        s.fastx = s.fasty = s.fastz = 0u; s.self = nullptr;
        s.nx = (unsigned)(hi[0] - lo[0] + 1);
        s.nxy = s.nx * (unsigned)(hi[1] - lo[1] + 1);
        s.slice_stride = (unsigned long long)s.nxy * (unsigned)(hi[2] - lo[2] + 1);
        void* data = nullptr; size_t bytes = 0;
        const unsigned bnx = (unsigned)(hi[0] - lo[0] + 1), bny = (unsigned)(hi[1] - lo[1] + 1),
                       bnz = (unsigned)(hi[2] - lo[2] + 1);
        rc = repack(src, bnx, bny, bnz, 1u, layout, &data, &bytes);
        if (rc) return fail(rc);
        if (layout == LAYOUT_CELL) cell_strides(s, bnx, bny, bnz);
        s.data = data;
        s.plane = s.slice_stride; s.tex = 0ull;
        if (bytes) { f->owned.push_back(data); f->owned_bytes += bytes; }
        if (layout == LAYOUT_TEX) {
          rc = make_texture(data, s.slice_stride, &s.tex);
          if (rc) return fail(rc);
          f->textures.push_back(s.tex);
        }
        bool brick_tame = false;
        if (layout != LAYOUT_PACKED3) {      // a borrowed array can change after the scan (see streami_field_create)
          rc = scan_tame(src, 3ull * bnx * bny * bnz, &brick_tame);
          if (rc) return fail(rc);
        }
        f->tame = f->tame && brick_tame;
        f->bricks.push_back(s);
      }
  void* tbl = nullptr;
  if (check(cudaMalloc(&tbl, sizeof(Store) * nb)) != STREAMI_OK) return fail(STREAMI_E_NOMEM);
  f->owned.push_back(tbl);
  for (int i = 0; i < nb; ++i) {
    Store& s = f->bricks[i];
    s.self = (const Store*)tbl + i;
    if (f->tame) { s.fastx = (unsigned)(s.hix - s.lox); s.fasty = (unsigned)(s.hiy - s.loy); s.fastz = (unsigned)(s.hiz - s.loz); }
  }
  cudaError_t e = cudaMemcpy(tbl, f->bricks.data(), sizeof(Store) * nb, cudaMemcpyHostToDevice);
  if (e != cudaSuccess) return fail(check(e));
  f->d_bricks = (Store*)tbl;
  *out = f;
  return STREAMI_OK;
}

int streami_field_destroy(streami_field f) {
  if (!f) return STREAMI_E_INVALID;
  for (unsigned long long t : f->textures) cudaDestroyTextureObject((cudaTextureObject_t)t);
  for (void* p : f->owned) cudaFree(p);
  delete f;
  return STREAMI_OK;
}

int streami_field_info(streami_field f, int* layout, size_t* owned_bytes) {
  if (!f) return STREAMI_E_INVALID;
  if (layout) *layout = f->layout;
  if (owned_bytes) *owned_bytes = f->owned_bytes;
  return STREAMI_OK;
}

int streami_sample(streami_field f, const float* points, size_t n, float t, int time_mode,
                   float* out_v, unsigned* out_rc, void* cuda_stream) {
  OptionsScope options_scope;
  if (!f || f->bricked || !points || !out_v || !out_rc) return STREAMI_E_INVALID;
  if (time_mode != 0 && time_mode != 1) return STREAMI_E_INVALID;
  if (n == 0) return STREAMI_OK;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  Geom g = f->g; g.time_mode = time_mode;
  const bool unsteady = g.nslices > 1;
  unsigned blocks = (unsigned)((n + 255) / 256);
#define GO(L, U) sample_kernel<L, U><<<blocks, 256, 0, st>>>(g, f->store, points, n, t, out_v, out_rc)
  switch (f->layout * 2 + (unsteady ? 1 : 0)) {
    case LAYOUT_PACKED3 * 2: GO(LAYOUT_PACKED3, false); break;
    case LAYOUT_PACKED3 * 2 + 1: GO(LAYOUT_PACKED3, true); break;
    case LAYOUT_FLOAT4 * 2: GO(LAYOUT_FLOAT4, false); break;
    case LAYOUT_FLOAT4 * 2 + 1: GO(LAYOUT_FLOAT4, true); break;
    case LAYOUT_XPAIR * 2: GO(LAYOUT_XPAIR, false); break;
    case LAYOUT_XPAIR * 2 + 1: GO(LAYOUT_XPAIR, true); break;
    case LAYOUT_CELL * 2: GO(LAYOUT_CELL, false); break;
    case LAYOUT_CELL * 2 + 1: GO(LAYOUT_CELL, true); break;
    case LAYOUT_XYQUAD * 2: GO(LAYOUT_XYQUAD, false); break;
    case LAYOUT_XYQUAD * 2 + 1: GO(LAYOUT_XYQUAD, true); break;
    case LAYOUT_SOA * 2: GO(LAYOUT_SOA, false); break;
    case LAYOUT_SOA * 2 + 1: GO(LAYOUT_SOA, true); break;
    case LAYOUT_TEX * 2: GO(LAYOUT_TEX, false); break;
    default: GO(LAYOUT_TEX, true); break;
  }
#undef GO
  STREAMI_LAUNCHED();
  return STREAMI_OK;
}

int streami_seed_shape(const float origin[3], const float edge_u[3], const float edge_v[3],
                       const float edge_w[3], unsigned nu, unsigned nv, unsigned nw, int mode,
                       unsigned long long rng_seed, float* out_seeds, void* cuda_stream) {
  if (!origin || !edge_u || !edge_v || !edge_w || (mode != 0 && mode != 1)) return STREAMI_E_INVALID;
  const unsigned long long total = (unsigned long long)nu * nv * nw;
  if (total > 0xffffffffull) return STREAMI_E_INVALID;
  if (total == 0) return STREAMI_OK;
  if (!out_seeds) return STREAMI_E_INVALID;
  SeedShape sh;
  for (int c = 0; c < 3; ++c) { sh.o[c] = origin[c]; sh.eu[c] = edge_u[c]; sh.ev[c] = edge_v[c]; sh.ew[c] = edge_w[c]; }
  sh.nu = nu; sh.nv = nv; sh.nw = nw; sh.mode = mode; sh.rng_seed = rng_seed;
  const unsigned blocks = (unsigned)std::min<unsigned long long>((total + 255) / 256, 148ull * 16);
  seed_shape_kernel<<<blocks, 256, 0, (cudaStream_t)cuda_stream>>>(sh, out_seeds);
  STREAMI_LAUNCHED();
  return STREAMI_OK;
}

int streami_set_option(const char* name, int value) {
  if (!name) return STREAMI_E_INVALID;
  const int i = option_index(name);
  if (i < 0) return STREAMI_E_INVALID;
  Options lim{};    // member offsets only
  int* base = reinterpret_cast<int*>(&lim);
  int v = value;
  if (&base[i] == &lim.cell_cache || &base[i] == &lim.presort || &base[i] == &lim.kernel_timing ||
      &base[i] == &lim.vertex_staging || &base[i] == &lim.integer_accept) v = value != 0;
  else if (&base[i] == &lim.brick_round_steps) v = value < -2 ? -2 : value;
  else if (&base[i] == &lim.prefetch) v = value < 0 ? 0 : (value > 4 ? 4 : value);
  else v = value < 0 ? 0 : value;
  option_store(i, v);
  return STREAMI_OK;
}

int streami_get_option(const char* name, int* value) {
  if (!name || !value) return STREAMI_E_INVALID;
  const int i = option_index(name);
  if (i < 0) return STREAMI_E_INVALID;
  *value = option_load(i);
  return STREAMI_OK;
}

unsigned long long streami_launch_count(void) { return launch_counter().load(); }

int streami_kernel_time(float* total_ms, unsigned* launches) {
  if (!total_ms) return STREAMI_E_INVALID;
  std::lock_guard<std::mutex> lk(g_time_mutex);
  float sum = 0.0f; unsigned cnt = 0;
  cudaError_t err = cudaSuccess;
  for (auto& pr : g_time_pairs) {
    float ms = 0.0f;
    cudaError_t e = cudaEventSynchronize(pr.second);
    if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, pr.first, pr.second);
    if (e == cudaSuccess) { sum += ms; cnt++; } else err = e;
    g_time_free.push_back(pr.first); g_time_free.push_back(pr.second);
  }
  g_time_pairs.clear();
  *total_ms = sum;
  if (launches) *launches = cnt;
  return check(err);
}

const char* streami_error_string(int code) {
  switch (code) {
    case STREAMI_OK: return "ok";
    case STREAMI_E_INVALID: return "invalid argument";
    case STREAMI_E_NOMEM: return "out of device memory";
    case STREAMI_E_TRUNCATED: return "hand-off log or round table truncated (results valid)";
    case STREAMI_E_TOO_LARGE: return "too many seeds for the static scratch of streami_trace_streamlines_noalloc (max 262,144)";
    case STREAMI_E_CUDA: {
      static thread_local std::string copy;
      std::lock_guard<std::mutex> lk(g_err_mutex);
      copy = g_cuda_err;
      return copy.c_str();
    }
    default: return "unknown error code";
  }
}

}  // extern "C"
