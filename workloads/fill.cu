// workloads/fill.cu -- CUDA INPUT generators for the large synthetic fields (C2, C3, C5).
//
// Input generation only: no interpolation, no integrator, no termination logic -- none of the
// traced method's arithmetic lives here.  The turbulence field of SURVEY.md 8(d) is
//   v(x) = s * sum_m ampvec_m cos(kvec_m . x + phi_m)   at integer vertex coordinates x,
// evaluated in fp64 and rounded once to fp32; 1024^3 vertices x 1,024 modes is ~1e12 cosines,
// which is why this runs on the GPU.  The mode table comes from workloads/gen.cpp
// (wl_turb_modes: 8 doubles per mode = kvec[3], ampvec[3], phi, kmag).  The result is checked
// against the direct CPU fill of gen.cpp on small grids (tests/test_gpu_workloads.py).
// The bytes produced here are the ones BOTH the oracle and the CUDA library are fed with.
#include <cuda_runtime.h>
#include <stddef.h>

namespace {

constexpr int FILL_BLOCK = 256;

// One thread per vertex of the box [lo, lo+dims).  out64[v*3 + c] = unnormalised component c.
// partial[block] = sum over the block's vertices of |v|^2 (fixed tree order -> deterministic).
__global__ void __launch_bounds__(FILL_BLOCK)
turb_fill_kernel(int nx, int ny, int nz, int lox, int loy, int loz, int M,
                 const double* __restrict__ table, double* __restrict__ out64,
                 double* __restrict__ partial) {
  extern __shared__ double s_tab[];            // [M][7]: kvec, ampvec, phi
  for (int i = threadIdx.x; i < M * 7; i += blockDim.x) {
    int m = i / 7, c = i - 7 * m;
    s_tab[i] = table[8 * (size_t)m + c];
  }
  __syncthreads();
  const size_t nvert = (size_t)nx * ny * nz;
  const size_t v = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  double sq = 0.0;
  if (v < nvert) {
    const int x = (int)(v % nx), y = (int)((v / nx) % ny), z = (int)(v / ((size_t)nx * ny));
    const double X = x + lox, Y = y + loy, Z = z + loz;
    double a0 = 0.0, a1 = 0.0, a2 = 0.0;
    for (int m = 0; m < M; ++m) {
      const double* r = s_tab + 7 * m;
      const double c = cos(r[0] * X + r[1] * Y + r[2] * Z + r[6]);
      a0 += r[3] * c; a1 += r[4] * c; a2 += r[5] * c;
    }
    out64[3 * v] = a0; out64[3 * v + 1] = a1; out64[3 * v + 2] = a2;
    sq = a0 * a0 + a1 * a1 + a2 * a2;
  }
  __shared__ double s_red[FILL_BLOCK];
  s_red[threadIdx.x] = sq;
  __syncthreads();
  for (int d = FILL_BLOCK / 2; d > 0; d >>= 1) {
    if (threadIdx.x < d) s_red[threadIdx.x] += s_red[threadIdx.x + d];
    __syncthreads();
  }
  if (threadIdx.x == 0) partial[blockIdx.x] = s_red[0];
}

__global__ void scale_round_kernel(size_t n, const double* __restrict__ in64, double scale,
                                   float* __restrict__ out32) {
  size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  const size_t step = (size_t)gridDim.x * blockDim.x;
  for (; i < n; i += step) out32[i] = (float)(scale * in64[i]);
}

// Copy the stored box [lo, hi] of a packed float3 volume into its own packed array (brick cut).
__global__ void cut_box_kernel(const float* __restrict__ vol, int Nx, int Ny, int lox, int loy,
                               int loz, int bx, int by, int bz, float* __restrict__ out) {
  const size_t n = (size_t)bx * by * bz;
  size_t v = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  const size_t step = (size_t)gridDim.x * blockDim.x;
  for (; v < n; v += step) {
    const int x = (int)(v % bx), y = (int)((v / bx) % by), z = (int)(v / ((size_t)bx * by));
    const size_t s = ((size_t)(z + loz) * Ny + (y + loy)) * Nx + (x + lox);
    out[3 * v] = vol[3 * s]; out[3 * v + 1] = vol[3 * s + 1]; out[3 * v + 2] = vol[3 * s + 2];
  }
}

}  // namespace

extern "C" {

// Number of per-block partial sums wl_cuda_turb_fill writes for a box of nvert vertices.
size_t wl_cuda_turb_partials(size_t nvert) { return (nvert + FILL_BLOCK - 1) / FILL_BLOCK; }

// All pointers are DEVICE pointers; table is [M][8] doubles.  Returns a cudaError_t as int.
int wl_cuda_turb_fill(const int dims[3], const int lo[3], int M, const double* d_table,
                      double* d_out64, double* d_partial, void* stream) {
  const size_t nvert = (size_t)dims[0] * dims[1] * dims[2];
  const size_t smem = sizeof(double) * 7 * (size_t)M;
  cudaError_t e = cudaFuncSetAttribute(turb_fill_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                       (int)smem);
  if (e != cudaSuccess) return (int)e;
  const unsigned blocks = (unsigned)((nvert + FILL_BLOCK - 1) / FILL_BLOCK);
  turb_fill_kernel<<<blocks, FILL_BLOCK, smem, (cudaStream_t)stream>>>(
      dims[0], dims[1], dims[2], lo[0], lo[1], lo[2], M, d_table, d_out64, d_partial);
  return (int)cudaGetLastError();
}

int wl_cuda_scale_round(size_t n, const double* d_in64, double scale, float* d_out32, void* stream) {
  scale_round_kernel<<<148 * 8, 256, 0, (cudaStream_t)stream>>>(n, d_in64, scale, d_out32);
  return (int)cudaGetLastError();
}

int wl_cuda_cut_box(const float* d_vol, const int N[3], const int lo[3], const int hi[3],
                    float* d_out, void* stream) {
  cut_box_kernel<<<148 * 8, 256, 0, (cudaStream_t)stream>>>(
      d_vol, N[0], N[1], lo[0], lo[1], lo[2], hi[0] - lo[0] + 1, hi[1] - lo[1] + 1,
      hi[2] - lo[2] + 1, d_out);
  return (int)cudaGetLastError();
}

}  // extern "C"
