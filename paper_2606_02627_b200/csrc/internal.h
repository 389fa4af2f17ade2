// csrc/internal.h -- host-side state shared by the API translation units.
#pragma once
#include <atomic>
#include <string>
#include <vector>

#include "../../include/streami.h"
#include "field.cuh"

struct streami_field_s {
  streami::Geom g;
  int dims[3];                       // global vertex counts
  int layout;
  bool bricked;
  bool tame;                         // every stored value finite and <= 2^60 (monolithic; see sample_nb)
  streami::Store store;              // monolithic
  std::vector<streami::Store> bricks;  // host copies
  streami::Store* d_bricks;          // device table
  streami::BrickMap bm;
  std::vector<void*> owned;          // device allocations owned by the handle
  std::vector<unsigned long long> textures;   // texture objects owned by the handle (LAYOUT_TEX)
  size_t owned_bytes;
};

namespace streami {

// Library options (streami_set_option).  The process-wide values are atomics; an API call works on ONE
// snapshot of them, taken when it is entered (OptionsScope), so that a setter running on another host
// thread can neither tear a value nor change the schedule of a call half way through.
struct Options { int cell_cache; int presort; int streak_window; int kernel_timing; int segment_steps; int vertex_staging; int prefetch; int max_blocks_per_sm; int brick_round_steps; int integer_accept; int host_batch; int queue_steps; };
constexpr int N_OPTIONS = 12;
const Options& options();            // the snapshot of the API call in progress on this thread, else a fresh one
int option_index(const char* name);  // -1 if unknown
void option_store(int index, int value);
int option_load(int index);
struct OptionsScope { OptionsScope(); ~OptionsScope(); };
std::atomic<unsigned long long>& launch_counter();
void set_cuda_error(cudaError_t e);

inline int check(cudaError_t e) {
  if (e == cudaSuccess) return STREAMI_OK;
  set_cuda_error(e);
  return e == cudaErrorMemoryAllocation ? STREAMI_E_NOMEM : STREAMI_E_CUDA;
}

#define STREAMI_TRY(expr)                         \
  do {                                            \
    int rc__ = streami::check(expr);              \
    if (rc__ != STREAMI_OK) return rc__;          \
  } while (0)

#define STREAMI_LAUNCHED()                        \
  do {                                            \
    streami::launch_counter()++;                  \
    STREAMI_TRY(cudaGetLastError());              \
  } while (0)

int num_sms();
cudaStream_t copy_stream();      // the library's own non-blocking stream for overlapped D2H copies (created once)

// The monolithic store as a launch sees it: with the integer-accept ranges of sample_nb (field.cuh)
// filled in when the field is tame and option "integer_accept" is on.
inline Store launch_store(const streami_field_s* f) {
  Store s = f->store;
  if (f->tame && options().integer_accept) {
    s.fastx = (unsigned)(s.cmx + 1); s.fasty = (unsigned)(s.cmy + 1); s.fastz = (unsigned)(s.cmz + 1);
  }
  return s;
}

// Optional device timing of the advection kernel alone (option "kernel_timing"): a pair of CUDA
// events recorded on the launching stream around each advection launch, summed by
// streami_kernel_time().  Off by default; bench.py's roofline leg turns it on.
void timing_begin(cudaStream_t st);
void timing_end(cudaStream_t st);

}  // namespace streami
