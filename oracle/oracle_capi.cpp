// oracle/oracle_capi.cpp -- C entry points of the CPU oracle, for ctypes (oracle/__init__.py).
//
// TEST INFRASTRUCTURE ONLY (see streami_oracle.hpp).  Drivers here add nothing to the
// arithmetic: they loop over particles (OpenMP, particles are independent), apply the
// streakline schedule of A7 (Listing 2) and the brick rounds of A9
// (PAPER.md:63-65, 96-101, 142-144), and copy results into the caller's arrays.
#include "streami_oracle.hpp"
#include <omp.h>

using namespace oracle;

extern "C" {

struct OGrid {
  int gdims[3]; int lo[3]; int hi[3];
  float origin[3]; float spacing[3];
  int nslices; float slice_dt; int time_mode;
  const float* data;
};

struct OParams {
  int integrator;
  double h, h_min, h_max, atol, rtol;
  uint32_t max_steps;
  double vmin, t0;
  uint32_t capacity, stride;
};

struct OAnalytic { int kind; double c[16]; double blo[3]; double bhi[3]; };

int oracle_num_threads() { return omp_get_max_threads(); }

}  // extern "C"

namespace {

template <class T> GridField<T> make_grid(const OGrid* g) {
  GridField<T> f;
  f.init(g->gdims, g->lo, g->hi, g->origin, g->spacing, g->nslices, g->slice_dt, g->time_mode,
         g->data);
  return f;
}
template <class T> AnalyticField<T> make_analytic(const OAnalytic* a) {
  AnalyticField<T> f;
  f.kind = a->kind;
  for (int i = 0; i < 16; ++i) f.c[i] = a->c[i];
  for (int i = 0; i < 3; ++i) { f.blo[i] = a->blo[i]; f.bhi[i] = a->bhi[i]; }
  return f;
}
template <class T> Params<T> make_params(const OParams* p) {
  Params<T> q;
  q.integrator = p->integrator;
  q.h = T(p->h); q.h_min = T(p->h_min); q.h_max = T(p->h_max);
  q.atol = T(p->atol); q.rtol = T(p->rtol);
  q.max_steps = p->max_steps; q.vmin = T(p->vmin); q.t0 = T(p->t0);
  q.capacity = p->capacity; q.stride = p->stride;
  return q;
}
inline void add(Totals& a, const Totals& b) {
  a.attempted += b.attempted; a.accepted += b.accepted; a.samples += b.samples;
  a.handoffs += b.handoffs;
}
inline void put(unsigned long long* out, const Totals& t) {
  if (!out) return;
  out[0] = t.attempted; out[1] = t.accepted; out[2] = t.samples; out[3] = t.handoffs;
}

// A5 over all seeds.
template <class T, class F>
void run_streamlines(const F& fld, const T* seeds, size_t n, const OParams* op, T* out_vertices,
                     uint32_t* out_counts, uint32_t* out_steps, uint32_t* out_status,
                     T* out_final, unsigned long long* totals) {
  Params<T> prm = make_params<T>(op);
  Recorder<T> rec{out_vertices, out_counts, n, prm.capacity, prm.stride};
  Totals tot;
#pragma omp parallel
  {
    Totals mine;
#pragma omp for schedule(dynamic, 256)
    for (long long i = 0; i < (long long)n; ++i) {
      if (out_counts) out_counts[i] = 0;
      uint32_t steps, status; T fin[3];
      trace_one(fld, seeds + 3 * i, prm, prm.max_steps, 0u, size_t(i), rec, mine, steps, status,
                fin);
      if (out_steps) out_steps[i] = steps;
      if (out_status) out_status[i] = status;
      if (out_final) for (int c = 0; c < 3; ++c) out_final[size_t(c) * n + i] = fin[c];
    }
#pragma omp critical
    add(tot, mine);
  }
  put(totals, tot);
}

// A7: particle (i, j) is born at point i at global step j and steps at global indices
// j .. nsteps-1; slot [c][j][i] = its final position; counts[i] = particles alive at the end.
template <class T, class F>
void run_streaklines(const F& fld, const T* points, size_t m, uint32_t nsteps, const OParams* op,
                     T* out_vertices, uint32_t* out_counts, uint32_t* out_steps,
                     uint32_t* out_status, unsigned long long* totals) {
  Params<T> prm = make_params<T>(op);
  prm.integrator = 0;
  Recorder<T> rec{nullptr, nullptr, 0, 1, 1};
  Totals tot;
  const size_t total = m * size_t(nsteps);
  std::vector<uint32_t> status_all(total);
#pragma omp parallel
  {
    Totals mine;
#pragma omp for schedule(dynamic, 256)
    for (long long id = 0; id < (long long)total; ++id) {
      size_t j = size_t(id) / m, i = size_t(id) % m;
      uint32_t steps, status; T fin[3];
      trace_one(fld, points + 3 * i, prm, nsteps - uint32_t(j), uint32_t(j), size_t(id), rec, mine,
                steps, status, fin);
      for (int c = 0; c < 3; ++c) out_vertices[(size_t(c) * nsteps + j) * m + i] = fin[c];
      status_all[id] = status;
      if (out_steps) out_steps[id] = steps;
      if (out_status) out_status[id] = status;
    }
#pragma omp critical
    add(tot, mine);
  }
  for (size_t i = 0; i < m; ++i) {
    uint32_t c = 0;
    for (size_t j = 0; j < nsteps; ++j) c += (status_all[j * m + i] == MAX_STEPS);
    out_counts[i] = c;
  }
  put(totals, tot);
}

}  // namespace

#define ORACLE_INSTANTIATE(T, SFX)                                                               \
  extern "C" void oracle_sample_##SFX(const OGrid* g, const T* pts, size_t n, T t, T* out_v,     \
                                      uint32_t* out_rc) {                                        \
    GridField<T> f = make_grid<T>(g);                                                            \
    for (size_t i = 0; i < n; ++i) {                                                             \
      T v[3] = {0, 0, 0};                                                                        \
      out_rc[i] = f.sample(pts + 3 * i, t, v);                                                   \
      for (int c = 0; c < 3; ++c) out_v[3 * i + c] = v[c];                                       \
    }                                                                                            \
  }                                                                                              \
  extern "C" void oracle_streamlines_##SFX(                                                      \
      const OGrid* g, const T* seeds, size_t n, const OParams* p, T* out_vertices,               \
      uint32_t* out_counts, uint32_t* out_steps, uint32_t* out_status, T* out_final,             \
      unsigned long long* totals) {                                                              \
    run_streamlines<T>(make_grid<T>(g), seeds, n, p, out_vertices, out_counts, out_steps,        \
                       out_status, out_final, totals);                                           \
  }                                                                                              \
  extern "C" void oracle_streamlines_analytic_##SFX(                                             \
      const OAnalytic* a, const T* seeds, size_t n, const OParams* p, T* out_vertices,           \
      uint32_t* out_counts, uint32_t* out_steps, uint32_t* out_status, T* out_final,             \
      unsigned long long* totals) {                                                              \
    run_streamlines<T>(make_analytic<T>(a), seeds, n, p, out_vertices, out_counts, out_steps,    \
                       out_status, out_final, totals);                                           \
  }                                                                                              \
  extern "C" void oracle_streaklines_##SFX(                                                      \
      const OGrid* g, const T* points, size_t m, uint32_t nsteps, const OParams* p,              \
      T* out_vertices, uint32_t* out_counts, uint32_t* out_steps, uint32_t* out_status,          \
      unsigned long long* totals) {                                                              \
    run_streaklines<T>(make_grid<T>(g), points, m, nsteps, p, out_vertices, out_counts,          \
                       out_steps, out_status, totals);                                           \
  }                                                                                              \
  extern "C" void oracle_streaklines_analytic_##SFX(                                             \
      const OAnalytic* a, const T* points, size_t m, uint32_t nsteps, const OParams* p,          \
      T* out_vertices, uint32_t* out_counts, uint32_t* out_steps, uint32_t* out_status,          \
      unsigned long long* totals) {                                                              \
    run_streaklines<T>(make_analytic<T>(a), points, m, nsteps, p, out_vertices, out_counts,      \
                       out_steps, out_status, totals);                                           \
  }                                                                                              \
  extern "C" void oracle_rp10_##SFX(const T* x, size_t n, T* out) {                              \
    for (size_t i = 0; i < n; ++i) out[i] = rp10(x[i]);                                          \
  }

ORACLE_INSTANTIATE(float, f32)
ORACLE_INSTANTIATE(double, f64)

// Tableau as the oracle holds it, for the identity pins P8(i).  out[0..6] = c, out[7..27] = a
// (rows 2..7, row s has s-1 entries), out[28..34] = b (5th order = row 7), out[35..41] = e.
template <class T> static void tableau(double* o) {
  typedef DP<T> D;
  const double v[42] = {
      0, D::c2, D::c3, D::c4, D::c5, 1, 1,
      D::a21,
      D::a31, D::a32,
      D::a41, D::a42, D::a43,
      D::a51, D::a52, D::a53, D::a54,
      D::a61, D::a62, D::a63, D::a64, D::a65,
      D::b1, 0, D::b3, D::b4, D::b5, D::b6,
      D::b1, 0, D::b3, D::b4, D::b5, D::b6, 0,
      D::e1, 0, D::e3, D::e4, D::e5, D::e6, D::e7};
  for (int i = 0; i < 42; ++i) o[i] = v[i];
}
extern "C" void oracle_dp5_tableau_f64(double* out) { tableau<double>(out); }
extern "C" void oracle_dp5_tableau_f32(double* out) { tableau<float>(out); }

// ---------------------------------------------------------------------------------------
// A9 rounds (fp32 and fp64).  bricks[b] describes brick b's stored box and array; all bricks
// share gdims/origin/spacing.  Queue order inside a round is unspecified by the sheet; here
// it is ascending particle id within each brick (deterministic).
// ---------------------------------------------------------------------------------------
namespace {
template <class T>
void run_bricks(const OGrid* bricks, const int nbg[3], const T* seeds, size_t n, const OParams* op,
                T* out_vertices, uint32_t* out_counts, uint32_t* out_steps, uint32_t* out_status,
                T* out_final, uint32_t* out_round_counts, uint32_t max_rounds,
                unsigned long long* out_log, size_t log_capacity, unsigned long long* out_nlog,
                uint32_t* out_nrounds, unsigned long long* totals) {
  const int nbricks = nbg[0] * nbg[1] * nbg[2];
  Params<T> prm = make_params<T>(op);
  std::vector<GridField<T>> F(nbricks);
  for (int b = 0; b < nbricks; ++b) F[b] = make_grid<T>(&bricks[b]);
  BrickGrid<T> bg;
  for (int a = 0; a < 3; ++a) {
    bg.N[a] = bricks[0].gdims[a]; bg.nb[a] = nbg[a]; bg.B[a] = bg.N[a] / bg.nb[a];
    bg.o[a] = F[0].o[a]; bg.r[a] = F[0].r[a];
  }
  Recorder<T> rec{out_vertices, out_counts, n, prm.capacity, prm.stride};
  std::vector<State<T>> st(n);
  std::vector<std::vector<uint32_t>> Q(nbricks), Qn(nbricks);
  Totals tot;
  for (size_t i = 0; i < n; ++i) {
    if (out_counts) out_counts[i] = 0;
    State<T>& s = st[i];
    for (int c = 0; c < 3; ++c) s.p[c] = seeds[3 * i + c];
    s.n = 0; s.have_k1 = false; s.rejected = false; s.t = prm.t0;
    s.h = std::min(std::max(prm.h, prm.h_min), prm.h_max);
    if (!F[0].inside(s.p)) {
      if (out_steps) out_steps[i] = 0;
      if (out_status) out_status[i] = OUT_OF_DOMAIN;
      if (out_final) for (int c = 0; c < 3; ++c) out_final[size_t(c) * n + i] = s.p[c];
      continue;
    }
    rec.record(i, 0, s.p);
    Q[bg.owner(s.p)].push_back(uint32_t(i));
  }
  uint32_t round = 0;
  unsigned long long nlog = 0;
  for (;;) {
    size_t live = 0;
    for (int b = 0; b < nbricks; ++b) {
      live += Q[b].size();
      if (out_round_counts && round < max_rounds)
        out_round_counts[size_t(round) * nbricks + b] = uint32_t(Q[b].size());
    }
    if (live == 0) break;
    for (int b = 0; b < nbricks; ++b) {
      const std::vector<uint32_t>& q = Q[b];
      std::vector<int> dest(q.size(), -1);
#pragma omp parallel
      {
        Totals mine;
#pragma omp for schedule(dynamic, 256)
        for (long long k = 0; k < (long long)q.size(); ++k) {
          const uint32_t id = q[k];
          State<T>& s = st[id];
          auto leaves = [&](const T* p) { return bg.owner(p) != b; };
          uint32_t rc = (prm.integrator == 0)
                            ? advance_rk4(F[b], s, prm, prm.max_steps, 0u, id, rec, mine, leaves)
                            : advance_dp5(F[b], s, prm, prm.max_steps, id, rec, mine, leaves);
          if (rc == HANDOFF) {
            if (s.n == prm.max_steps) rc = MAX_STEPS;
            else { dest[k] = bg.owner(s.p); mine.handoffs++; continue; }
          }
          if (out_steps) out_steps[id] = s.n;
          if (out_status) out_status[id] = rc;
          if (out_final) for (int c = 0; c < 3; ++c) out_final[size_t(c) * n + id] = s.p[c];
        }
#pragma omp critical
        add(tot, mine);
      }
      for (size_t k = 0; k < q.size(); ++k)
        if (dest[k] >= 0) {
          Qn[dest[k]].push_back(q[k]);
          if (out_log && nlog < log_capacity)
            out_log[nlog] = ((unsigned long long)(round + 1) << 48) |
                            ((unsigned long long)dest[k] << 32) | q[k];
          nlog++;
        }
    }
    for (int b = 0; b < nbricks; ++b) {
      std::sort(Qn[b].begin(), Qn[b].end());
      Q[b].swap(Qn[b]); Qn[b].clear();
    }
    round++;
  }
  if (out_nrounds) *out_nrounds = round;
  if (out_nlog) *out_nlog = nlog;
  put(totals, tot);
}
}  // namespace

extern "C" void oracle_brick_advect_f32(
    const OGrid* bricks, const int nbg[3], const float* seeds, size_t n, const OParams* p,
    float* out_vertices, uint32_t* out_counts, uint32_t* out_steps, uint32_t* out_status,
    float* out_final, uint32_t* out_round_counts, uint32_t max_rounds, unsigned long long* out_log,
    size_t log_capacity, unsigned long long* out_nlog, uint32_t* out_nrounds,
    unsigned long long* totals) {
  run_bricks<float>(bricks, nbg, seeds, n, p, out_vertices, out_counts, out_steps, out_status,
                    out_final, out_round_counts, max_rounds, out_log, log_capacity, out_nlog,
                    out_nrounds, totals);
}
extern "C" void oracle_brick_advect_f64(
    const OGrid* bricks, const int nbg[3], const double* seeds, size_t n, const OParams* p,
    double* out_vertices, uint32_t* out_counts, uint32_t* out_steps, uint32_t* out_status,
    double* out_final, uint32_t* out_round_counts, uint32_t max_rounds, unsigned long long* out_log,
    size_t log_capacity, unsigned long long* out_nlog, uint32_t* out_nrounds,
    unsigned long long* totals) {
  run_bricks<double>(bricks, nbg, seeds, n, p, out_vertices, out_counts, out_steps, out_status,
                     out_final, out_round_counts, max_rounds, out_log, log_capacity, out_nlog,
                     out_nrounds, totals);
}

// ---------------------------------------------------------------------------------------
// Seed generation on a control shape (the paper's convenience kernels: "uniformly distributed seed
// points given simple control shapes such as planes or lines").  The shape is
// the parallelepiped o + u*eu + v*ev + w*ew, (u,v,w) in [0,1)^3, sampled nu x nv x nw times
// (a line has nv = nw = 1, a plane nw = 1); seed index s = (k*nv + j)*nu + i.  fp32 formula:
//   mode 0 (lattice): u = ((float)i + 0.5f) / (float)nu, likewise v, w (IEEE division);
//   mode 1 (random):  u, v, w = U(s,0), U(s,1), U(s,2) with U(s,a) = (float)(z >> 40) * 2^-24,
//                     z = splitmix64 finaliser of rng_seed + (3 s + a + 1) * 0x9E3779B97F4A7C15;
//   p_c = fma(w, ew_c, fma(v, ev_c, fma(u, eu_c, o_c))).
// ---------------------------------------------------------------------------------------
static inline uint64_t oracle_mix64(uint64_t z) {
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
  return z ^ (z >> 31);
}
extern "C" void oracle_seed_shape_f32(const float o[3], const float eu[3], const float ev[3],
                                      const float ew[3], uint32_t nu, uint32_t nv, uint32_t nw,
                                      int mode, uint64_t rng_seed, float* out) {
  for (uint32_t k = 0; k < nw; ++k)
    for (uint32_t j = 0; j < nv; ++j)
      for (uint32_t i = 0; i < nu; ++i) {
        const uint64_t s = ((uint64_t)k * nv + j) * nu + i;
        float u, v, w;
        if (mode == 0) {
          u = ((float)i + 0.5f) / (float)nu; v = ((float)j + 0.5f) / (float)nv; w = ((float)k + 0.5f) / (float)nw;
        } else {
          float r[3];
          for (int a = 0; a < 3; ++a) {
            uint64_t z = oracle_mix64(rng_seed + (3ull * s + (uint64_t)a + 1ull) * 0x9E3779B97F4A7C15ull);
            r[a] = (float)(z >> 40) * 0x1.0p-24f;
          }
          u = r[0]; v = r[1]; w = r[2];
        }
        for (int c = 0; c < 3; ++c)
          out[3 * s + c] = std::fma(w, ew[c], std::fma(v, ev[c], std::fma(u, eu[c], o[c])));
      }
}

// ---------------------------------------------------------------------------------------
// Hexahedral meshes (oracle/hexmesh_oracle.hpp, formula sheet U1-U4).
// ---------------------------------------------------------------------------------------
#include "hexmesh_oracle.hpp"

#define HEXMESH_CAPI(T, SFX)                                                                         \
  extern "C" void oracle_hexmesh_sample_##SFX(size_t nv, size_t nc, const float* X, const float* V,  \
      const uint32_t* H, const float* lo, const float* hi, const int* nb, const T* pts, size_t n,    \
      int brute, T* out_v, long long* out_cell, T* out_xi) {                                         \
    oracle::HexMesh<T> m; m.init(nv, nc, X, V, H, lo, hi, nb);                                       \
    oracle::HexField<T> f{&m};                                                                       \
    for (size_t i = 0; i < n; ++i) {                                                                 \
      T xi[3] = {0, 0, 0}; long long c = -1;                                                         \
      if (brute) {  /* definition of point location: the lowest-numbered cell that contains p */     \
        int b[3];                                                                                    \
        if (m.bin_of(pts + 3 * i, b))                                                                \
          for (size_t k = 0; k < nc && c < 0; ++k) if (oracle::hx_invert(m, k, pts + 3 * i, xi)) c = (long long)k; \
      } else c = oracle::hx_locate(m, pts + 3 * i, xi);                                              \
      out_cell[i] = c;                                                                               \
      for (int a = 0; a < 3; ++a) { out_xi[3 * i + a] = xi[a]; out_v[3 * i + a] = 0; }                \
      if (c >= 0 && !brute) f.sample(pts + 3 * i, T(0), out_v + 3 * i);                              \
    }                                                                                                \
  }                                                                                                  \
  extern "C" void oracle_hexmesh_streamlines_##SFX(size_t nv, size_t nc, const float* X,             \
      const float* V, const uint32_t* H, const float* lo, const float* hi, const int* nb,            \
      const T* seeds, size_t n, const OParams* p, T* out_vertices, uint32_t* out_counts,             \
      uint32_t* out_steps, uint32_t* out_status, T* out_final, unsigned long long* totals) {         \
    oracle::HexMesh<T> m; m.init(nv, nc, X, V, H, lo, hi, nb);                                       \
    oracle::HexField<T> f{&m};                                                                       \
    run_streamlines<T>(f, seeds, n, p, out_vertices, out_counts, out_steps, out_status, out_final,   \
                       totals);                                                                      \
  }
HEXMESH_CAPI(float, f32)
HEXMESH_CAPI(double, f64)
