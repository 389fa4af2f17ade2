// csrc/api_mesh.cu -- hexahedral-mesh fields: handle, bin grid (built on the host at create time),
// streami_mesh_sample, streami_mesh_trace_streamlines.  Formula sheet U1-U4, DESIGN.md section 13.
#include <algorithm>
#include <cmath>
#include <vector>

#include "host_lines.cuh"
#include "internal.h"
#include "mesh.cuh"
#include "sorter.cuh"

struct streami_mesh_s {
  streami::MeshDev d;
  size_t nc;
  void* dev_cells; void* dev_start; void* dev_items;
};

namespace streami {
int check_params(const streami_params* p, bool need_capacity);

// U2 bin index of a coordinate already known to be inside [lo, hi] (fp32, as on the device)
static int bin_index(float x, float lo, float s, int nb) { return std::min((int)std::floor((x - lo) * s), nb - 1); }
}  // namespace streami

using namespace streami;

extern "C" {

// Host-only helpers for applications that hold their hexahedra in another corner order or are not sure of their
// orientation (a cell with a non-positive Jacobian never converges in U3: its points would silently report
// OUT_OF_DOMAIN).  VTK_HEXAHEDRON order: nodes 0-3 = the bottom face counter-clockwise, 4-7 = the top face above them.
int streami_mesh_reorder_vtk_hex(size_t nc, const unsigned* H_vtk, unsigned* H_out) {
  if (!H_vtk || !H_out) return STREAMI_E_INVALID;
  static const int from_vtk[8] = {0, 1, 3, 2, 4, 5, 7, 6};        // lattice corner l = dx + 2 dy + 4 dz <- VTK node
  for (size_t c = 0; c < nc; ++c) {
    unsigned t[8];
    for (int l = 0; l < 8; ++l) t[l] = H_vtk[8 * c + from_vtk[l]];
    for (int l = 0; l < 8; ++l) H_out[8 * c + l] = t[l];          // in place is fine
  }
  return STREAMI_OK;
}

int streami_mesh_check_hex(size_t nv, size_t nc, const float* X, const unsigned* H, unsigned long long* out_bad,
                           long long* out_first_bad) {
  if (!X || !H || !out_bad || nv == 0) return STREAMI_E_INVALID;
  unsigned long long bad = 0; long long first = -1;
  for (size_t c = 0; c < nc; ++c) {
    bool ok = true;
    for (int l = 0; l < 8 && ok; ++l) ok = H[8 * c + l] < nv;
    // Jacobian determinant of the trilinear map at the centre and at the 8 corners (the usual validity test of a
    // hexahedron): dX_a/dxi_b = sum_l X_l[a] dN_l/dxi_b with N_l = prod_b (bit b of l ? xi_b : 1 - xi_b)
    for (int q = 0; q < 9 && ok; ++q) {
      const double xi[3] = {q == 8 ? 0.5 : (double)(q & 1), q == 8 ? 0.5 : (double)((q >> 1) & 1), q == 8 ? 0.5 : (double)((q >> 2) & 1)};
      double J[3][3] = {{0, 0, 0}, {0, 0, 0}, {0, 0, 0}};
      for (int l = 0; l < 8; ++l) {
        const float* x = X + 3 * (size_t)H[8 * c + l];
        for (int b = 0; b < 3; ++b) {
          double w = ((l >> b) & 1) ? 1.0 : -1.0;
          for (int o = 0; o < 3; ++o) if (o != b) w *= ((l >> o) & 1) ? xi[o] : 1.0 - xi[o];
          for (int a = 0; a < 3; ++a) J[a][b] += w * (double)x[a];
        }
      }
      const double det = J[0][0] * (J[1][1] * J[2][2] - J[1][2] * J[2][1]) - J[0][1] * (J[1][0] * J[2][2] - J[1][2] * J[2][0]) +
                         J[0][2] * (J[1][0] * J[2][1] - J[1][1] * J[2][0]);
      ok = det > 0.0;                                             // NaN -> bad
    }
    if (!ok) { if (first < 0) first = (long long)c; ++bad; }
  }
  *out_bad = bad;
  if (out_first_bad) *out_first_bad = first;
  return STREAMI_OK;
}

int streami_mesh_create_hex(size_t nv, size_t nc, const float* X, const float* V, const unsigned* H,
                            const float lo[3], const float hi[3], const int nb[3], streami_mesh* out) {
  OptionsScope options_scope;
  if (!out) return STREAMI_E_INVALID;
  *out = nullptr;
  if (!X || !V || !H || !lo || !hi || !nb || nv == 0 || nc == 0 || nc > 0xffffffffull) return STREAMI_E_INVALID;
  for (int a = 0; a < 3; ++a)
    if (nb[a] < 1 || !(hi[a] > lo[a]) || !std::isfinite(lo[a]) || !std::isfinite(hi[a])) return STREAMI_E_INVALID;
  const size_t nbins = (size_t)nb[0] * nb[1] * nb[2];
  if (nbins > 0x7fffffffull) return STREAMI_E_INVALID;
  for (size_t i = 0; i < 8 * nc; ++i) if (H[i] >= nv) return STREAMI_E_INVALID;

  float s[3];
  for (int a = 0; a < 3; ++a) s[a] = (float)nb[a] / (hi[a] - lo[a]);       // U2, fp32
  // cell records + bin ranges
  std::vector<float> cells(nc * (size_t)MESH_REC, 0.0f);
  std::vector<int> range(nc * 6);
  float extent = 0.0f;
  for (size_t c = 0; c < nc; ++c) {
    float* rec = cells.data() + c * MESH_REC;
    float mn[3], mx[3];
    for (int l = 0; l < 8; ++l) {
      const unsigned v = H[8 * c + l];
      for (int a = 0; a < 3; ++a) {
        const float x = X[3 * (size_t)v + a];
        rec[8 * a + l] = x; rec[24 + 8 * a + l] = V[3 * (size_t)v + a];
        mn[a] = l ? std::min(mn[a], x) : x; mx[a] = l ? std::max(mx[a], x) : x;
      }
    }
    for (int a = 0; a < 3; ++a) {
      rec[48 + a] = mn[a]; rec[51 + a] = mx[a];
      extent = std::max(extent, mx[a] - mn[a]);
      const float x0 = std::min(std::max(mn[a], lo[a]), hi[a]), x1 = std::min(std::max(mx[a], lo[a]), hi[a]);
      range[6 * c + a] = bin_index(x0, lo[a], s[a], nb[a]);
      range[6 * c + 3 + a] = bin_index(x1, lo[a], s[a], nb[a]);
    }
  }
  // CSR lists, cells in ascending order inside every bin (count, scan, fill)
  std::vector<unsigned> start(nbins + 1, 0u);
  auto for_bins = [&](size_t c, auto&& fn) {
    const int* r = range.data() + 6 * c;
    for (int z = r[2]; z <= r[5]; ++z)
      for (int y = r[1]; y <= r[4]; ++y)
        for (int x = r[0]; x <= r[3]; ++x) fn(((size_t)z * nb[1] + y) * nb[0] + x);
  };
  unsigned long long total = 0;
  for (size_t c = 0; c < nc; ++c) for_bins(c, [&](size_t b) { start[b + 1]++; total++; });
  if (total > 0xffffffffull) return STREAMI_E_INVALID;
  for (size_t b = 0; b < nbins; ++b) start[b + 1] += start[b];
  // list entries: cell id + the cell's box in the coordinates of the bin (MESH_BOX_SCALE in mesh.cuh)
  const float margin = 50.0f * MESH_TOL * extent;
  std::vector<uint4> items(std::max<size_t>(total, 1));
  std::vector<unsigned> fill(start.begin(), start.end() - 1);
  auto pack = [](double u_lo, double u_hi, unsigned& lo16, unsigned& hi16) {
    const double a = std::floor((u_lo - MESH_BOX_SLACK) * (double)MESH_BOX_SCALE);
    const double b = std::ceil((u_hi + MESH_BOX_SLACK) * (double)MESH_BOX_SCALE);
    lo16 = (unsigned)(unsigned short)(short)std::min(std::max(a, -32768.0), 32767.0);
    hi16 = (unsigned)(unsigned short)(short)std::min(std::max(b, -32768.0), 32767.0);
  };
  for (size_t c = 0; c < nc; ++c) {
    const float* rec = cells.data() + c * MESH_REC;
    for_bins(c, [&](size_t b) {
      const int bi[3] = {(int)(b % nb[0]), (int)((b / nb[0]) % nb[1]), (int)(b / ((size_t)nb[0] * nb[1]))};
      unsigned l16[3], h16[3];
      for (int a = 0; a < 3; ++a)
        pack(((double)rec[48 + a] - margin - lo[a]) * s[a] - bi[a], ((double)rec[51 + a] + margin - lo[a]) * s[a] - bi[a],
             l16[a], h16[a]);
      items[fill[b]++] = make_uint4((unsigned)c, l16[0] | (l16[1] << 16), l16[2] | (h16[0] << 16), h16[1] | (h16[2] << 16));
    });
  }

  streami_mesh_s* m = new streami_mesh_s();
  m->nc = nc; m->dev_cells = m->dev_start = m->dev_items = nullptr;
  cudaError_t e = cudaMalloc(&m->dev_cells, cells.size() * sizeof(float));
  if (e == cudaSuccess) e = cudaMalloc(&m->dev_start, start.size() * sizeof(unsigned));
  if (e == cudaSuccess) e = cudaMalloc(&m->dev_items, items.size() * sizeof(uint4));
  if (e == cudaSuccess) e = cudaMemcpy(m->dev_cells, cells.data(), cells.size() * sizeof(float), cudaMemcpyHostToDevice);
  if (e == cudaSuccess) e = cudaMemcpy(m->dev_start, start.data(), start.size() * sizeof(unsigned), cudaMemcpyHostToDevice);
  if (e == cudaSuccess) e = cudaMemcpy(m->dev_items, items.data(), items.size() * sizeof(uint4), cudaMemcpyHostToDevice);
  if (e != cudaSuccess) {
    cudaFree(m->dev_cells); cudaFree(m->dev_start); cudaFree(m->dev_items);
    delete m;
    return check(e);
  }
  MeshDev& d = m->d;
  d.cells = (const float*)m->dev_cells; d.bin_start = (const unsigned*)m->dev_start; d.bin_items = (const uint4*)m->dev_items;
  d.lox = lo[0]; d.loy = lo[1]; d.loz = lo[2]; d.hix = hi[0]; d.hiy = hi[1]; d.hiz = hi[2];
  d.sx = s[0]; d.sy = s[1]; d.sz = s[2]; d.nbx = nb[0]; d.nby = nb[1]; d.nbz = nb[2];
  d.margin = margin;
  *out = m;
  return STREAMI_OK;
}

int streami_mesh_destroy(streami_mesh m) {
  if (!m) return STREAMI_E_INVALID;
  cudaFree(m->dev_cells); cudaFree(m->dev_start); cudaFree(m->dev_items);
  delete m;
  return STREAMI_OK;
}

int streami_mesh_sample(streami_mesh m, const float* points, size_t n, float* out_v, long long* out_cell,
                        void* cuda_stream) {
  OptionsScope options_scope;
  if (!m || (n > 0 && (!points || !out_v))) return STREAMI_E_INVALID;
  if (n == 0) return STREAMI_OK;
  mesh_sample_kernel<<<(unsigned)((n + 127) / 128), 128, 0, (cudaStream_t)cuda_stream>>>(m->d, points, n, out_v, out_cell);
  STREAMI_LAUNCHED();
  return STREAMI_OK;
}

int streami_mesh_trace_streamlines(streami_mesh m, const float* seeds, size_t n, const streami_params* params,
                                   float* out_vertices, unsigned* out_counts, void* cuda_stream) {
  OptionsScope options_scope;
  if (!m || (n > 0 && (!seeds || !out_counts))) return STREAMI_E_INVALID;
  int rc = check_params(params, true);
  if (rc) return rc;
  if (params->integrator != 0 || n > 0xffffffffull) return STREAMI_E_INVALID;   // RK4 (Listing 1)
  cudaStream_t st = (cudaStream_t)cuda_stream;
  if (params->out_totals) STREAMI_TRY(cudaMemsetAsync(params->out_totals, 0, 4 * sizeof(unsigned long long), st));
  if (n == 0) return STREAMI_OK;
  MeshTraceArgs a{};
  a.m = m->d; a.seeds = seeds; a.n = n;
  a.h = params->h; a.h2 = 0.5f * params->h; a.h6 = params->h / 6.0f; a.vmin2 = params->vmin * params->vmin;
  a.max_steps = params->max_steps; a.verts = out_vertices; a.cap = params->capacity; a.stride = params->stride;
  a.counts = out_counts; a.steps = params->out_steps; a.status = params->out_status; a.fin = params->out_final;
  a.totals = params->out_totals;
  // a12: process the seeds in Morton order of their bins (order only; outputs are indexed by id)
  unsigned* perm = nullptr; MortonSorter sorter{}; bool have_sorter = false;
  if (options().presort && n >= 65536) {
    streami_field_s shape{};               // the bin grid as an index space for the sort keys
    shape.dims[0] = m->d.nbx + 1; shape.dims[1] = m->d.nby + 1; shape.dims[2] = m->d.nbz + 1;
    shape.g.ox = m->d.lox; shape.g.oy = m->d.loy; shape.g.oz = m->d.loz;
    shape.g.rx = m->d.sx; shape.g.ry = m->d.sy; shape.g.rz = m->d.sz;
    shape.g.topx = (float)m->d.nbx; shape.g.topy = (float)m->d.nby; shape.g.topz = (float)m->d.nbz;
    cudaError_t e0 = cudaMallocAsync((void**)&perm, sizeof(unsigned) * n, st);
    if (e0 != cudaSuccess) return check(e0);
    rc = sorter.init(&shape, n, st);
    if (rc == STREAMI_OK) { have_sorter = true; rc = sorter.sort(shape.g, seeds, 3, n, nullptr, perm); }
    if (rc) { cudaFreeAsync(perm, st); if (have_sorter) sorter.release(); return rc; }
    a.perm = perm;
  }
  unsigned long long* next = nullptr;
  cudaError_t e = cudaMallocAsync((void**)&next, sizeof(unsigned long long), st);
  if (e == cudaSuccess) e = cudaMemsetAsync(next, 0, sizeof(unsigned long long), st);
  int per_sm = 0;
  if (e == cudaSuccess) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, mesh_trace_kernel, 128, 0);
  if (e == cudaSuccess) {
    a.next = next;
    const unsigned long long want = (n + 127) / 128, full = (unsigned long long)std::max(per_sm, 1) * num_sms();
    timing_begin(st);
    mesh_trace_kernel<<<(unsigned)std::max(1ull, std::min(want, full)), 128, 0, st>>>(a);   // persistent grid
    timing_end(st);
    launch_counter()++;
    e = cudaGetLastError();
  }
  if (next) cudaFreeAsync(next, st);
  if (perm) cudaFreeAsync(perm, st);
  if (have_sorter) sorter.release();
  return check(e);
}

int streami_mesh_trace_streamlines_lines_host(streami_mesh m, const float* seeds, size_t n,
                                              const streami_params* params, unsigned long long* out_offsets,
                                              float* out_points, unsigned long long max_points,
                                              unsigned long long* out_total, void* cuda_stream) {
  OptionsScope options_scope;
  if (!m) return STREAMI_E_INVALID;
  auto trace = [&](const float* d_seeds, size_t nb, const streami_params* dp, float* d_v, unsigned* d_c) {
    return streami_mesh_trace_streamlines(m, d_seeds, nb, dp, d_v, d_c, cuda_stream);
  };
  return lines_host(trace, false, seeds, n, params, out_offsets, out_points, max_points, out_total, cuda_stream);
}

}  // extern "C"
