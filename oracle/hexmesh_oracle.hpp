// oracle/hexmesh_oracle.hpp
//
// TEST INFRASTRUCTURE ONLY.  Plain CPU implementation of the paper's OTHER field type: a vector
// field on an unstructured mesh ("unstructured meshes ... cell location ... interpolation",
// PAPER.md:155, 159), restricted to hexahedra -- the element type of the
// paper's own experiment, which re-expresses a structured grid as hexahedral cells.
// The paper locates cells with a BVH point query; any exact point location gives the same
// result, and a uniform bin grid is used here.  Shares no code with paper_2606_02627_b200/.
//
// Formula sheet U1-U4 (T = float is the parity reference, T = double for closed-form checks;
// lerp(a,b,w) := fma(w, b-a, a); nothing else is fused):
//  U1 mesh.  nv vertices X[v] (3 T), values V[v] (3 T), nc hexahedra H[c][8] (vertex ids); local
//     corner l = dx + 2 dy + 4 dz sits at reference coordinates (dx, dy, dz) in {0,1}^3.
//  U2 bins.  Box lo..hi (given), nb = (nbx,nby,nbz) bins, s_a = (T)nb_a / (hi_a - lo_a).  bin_a(x) =
//     min((int)floor((x - lo_a) * s_a), nb_a - 1); a point with x < lo_a or x > hi_a (or NaN) is
//     outside.  Hexahedron c is listed, in ascending c, in every bin between the bins of the
//     componentwise min and max of its 8 vertices (both clamped into the box).
//  U3 inverse map.  G(xi) = tri(X, xi) - p with tri = 3 nested lerps (x, then y, then z) per
//     component.  Start xi = (1/2,1/2,1/2); at most NEWTON = 6 times, stopping after the first
//     update with |d_a| <= TOL for all a (the usual Newton termination; the paper does not specify
//     the inverse map, it calls a library point query): J columns
//       J_x = lerp(lerp(X1-X0, X3-X2, xi_y), lerp(X5-X4, X7-X6, xi_y), xi_z),
//       J_y = lerp(lerp(X2-X0, X3-X1, xi_x), lerp(X6-X4, X7-X5, xi_x), xi_z),
//       J_z = lerp(lerp(X4-X0, X5-X1, xi_x), lerp(X6-X2, X7-X3, xi_x), xi_y);
//     cofactors c_ij with fma(a, b, -(c*d)); det = fma(J_x.z, c_xz, fma(J_x.y, c_xy, J_x.x * c_xx));
//     r = 1/det; d_a = r * fma(G.z, ., fma(G.y, ., G.x * .)) (adjugate row a); xi = xi - d.
//     p is in c iff the last update has |d_a| <= TOL (the iteration stopped by convergence: a far cell's iterate may
//     otherwise pass through the unit cube) and -TOL <= xi_a <= 1 + TOL for all a (TOL = 2e-5 in fp32,
//     1e-11 in fp64: it only has to
//     exceed the error of the inverse map so that no point falls between two cells; NaN -> no).
//     The located cell is the FIRST listed cell of p's bin that contains p.
//  U4 sample.  v = tri(V, xi) with the xi of U3 as it is (not clamped).
#pragma once
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <vector>

namespace oracle {

template <class T> struct HexMesh {
  size_t nv = 0, nc = 0;
  const float* X = nullptr;       // [nv][3]
  const float* V = nullptr;       // [nv][3]
  const uint32_t* H = nullptr;    // [nc][8]
  T lo[3], hi[3], s[3];
  int nb[3];
  std::vector<uint32_t> bin_start, bin_items;

  static constexpr int NEWTON = 6;
  static T tol() { return sizeof(T) == 4 ? T(2e-5) : T(1e-11); }

  bool bin_of(const T* p, int* b) const {
    for (int a = 0; a < 3; ++a) {
      if (!(p[a] >= lo[a] && p[a] <= hi[a])) return false;
      b[a] = std::min((int)std::floor((p[a] - lo[a]) * s[a]), nb[a] - 1);
    }
    return true;
  }
  size_t bin_id(const int* b) const { return ((size_t)b[2] * nb[1] + b[1]) * nb[0] + b[0]; }

  void init(size_t nv_, size_t nc_, const float* X_, const float* V_, const uint32_t* H_,
            const float* lo_, const float* hi_, const int* nb_) {
    nv = nv_; nc = nc_; X = X_; V = V_; H = H_;
    for (int a = 0; a < 3; ++a) {
      lo[a] = T(lo_[a]); hi[a] = T(hi_[a]); nb[a] = nb_[a];
      s[a] = T(nb[a]) / (hi[a] - lo[a]);
    }
    const size_t nbins = (size_t)nb[0] * nb[1] * nb[2];
    std::vector<std::vector<uint32_t>> lists(nbins);
    for (size_t c = 0; c < nc; ++c) {                       // ascending c: lists come out sorted
      T mn[3], mx[3];
      for (int a = 0; a < 3; ++a) { mn[a] = T(X[3 * H[8 * c] + a]); mx[a] = mn[a]; }
      for (int l = 1; l < 8; ++l)
        for (int a = 0; a < 3; ++a) {
          T x = T(X[3 * H[8 * c + l] + a]);
          mn[a] = std::min(mn[a], x); mx[a] = std::max(mx[a], x);
        }
      int b0[3], b1[3];
      for (int a = 0; a < 3; ++a) {                         // clamp into the box, then bin
        T x0 = std::min(std::max(mn[a], lo[a]), hi[a]), x1 = std::min(std::max(mx[a], lo[a]), hi[a]);
        b0[a] = std::min((int)std::floor((x0 - lo[a]) * s[a]), nb[a] - 1);
        b1[a] = std::min((int)std::floor((x1 - lo[a]) * s[a]), nb[a] - 1);
      }
      for (int z = b0[2]; z <= b1[2]; ++z)
        for (int y = b0[1]; y <= b1[1]; ++y)
          for (int x = b0[0]; x <= b1[0]; ++x) lists[((size_t)z * nb[1] + y) * nb[0] + x].push_back((uint32_t)c);
    }
    bin_start.assign(nbins + 1, 0);
    for (size_t b = 0; b < nbins; ++b) bin_start[b + 1] = bin_start[b] + (uint32_t)lists[b].size();
    bin_items.resize(bin_start[nbins]);
    for (size_t b = 0; b < nbins; ++b) std::copy(lists[b].begin(), lists[b].end(), bin_items.begin() + bin_start[b]);
  }
};

template <class T> inline T hx_lerp(T a, T b, T w) { return std::fma(w, b - a, a); }

// tri(Q, xi) for one component: Q[l], l = dx + 2 dy + 4 dz
template <class T> inline T hx_tri(const T* Q, const T* xi) {
  T c00 = hx_lerp(Q[0], Q[1], xi[0]), c01 = hx_lerp(Q[2], Q[3], xi[0]);
  T c10 = hx_lerp(Q[4], Q[5], xi[0]), c11 = hx_lerp(Q[6], Q[7], xi[0]);
  return hx_lerp(hx_lerp(c00, c01, xi[1]), hx_lerp(c10, c11, xi[1]), xi[2]);
}

// U3: reference coordinates of p in hexahedron c; returns "p is in c".
template <class T> bool hx_invert(const HexMesh<T>& m, size_t c, const T* p, T* xi) {
  T Q[3][8];
  for (int l = 0; l < 8; ++l)
    for (int a = 0; a < 3; ++a) Q[a][l] = T(m.X[3 * m.H[8 * c + l] + a]);
  xi[0] = xi[1] = xi[2] = T(0.5);
  T d[3] = {T(0), T(0), T(0)};
  for (int it = 0; it < HexMesh<T>::NEWTON; ++it) {
    T G[3], Jx[3], Jy[3], Jz[3];
    for (int a = 0; a < 3; ++a) {
      const T* q = Q[a];
      G[a] = hx_tri(q, xi) - p[a];
      Jx[a] = hx_lerp(hx_lerp(q[1] - q[0], q[3] - q[2], xi[1]), hx_lerp(q[5] - q[4], q[7] - q[6], xi[1]), xi[2]);
      Jy[a] = hx_lerp(hx_lerp(q[2] - q[0], q[3] - q[1], xi[0]), hx_lerp(q[6] - q[4], q[7] - q[5], xi[0]), xi[2]);
      Jz[a] = hx_lerp(hx_lerp(q[4] - q[0], q[5] - q[1], xi[0]), hx_lerp(q[6] - q[2], q[7] - q[3], xi[0]), xi[1]);
    }
    // J = [Jx Jy Jz] (columns); cofactor(a,b) = fma(u, v, -(w*z))
    auto cof = [](T u, T v, T w, T z) { return std::fma(u, v, -(w * z)); };
    const T cxx = cof(Jy[1], Jz[2], Jz[1], Jy[2]), cxy = cof(Jz[0], Jy[2], Jy[0], Jz[2]), cxz = cof(Jy[0], Jz[1], Jz[0], Jy[1]);
    const T cyx = cof(Jz[1], Jx[2], Jx[1], Jz[2]), cyy = cof(Jx[0], Jz[2], Jz[0], Jx[2]), cyz = cof(Jz[0], Jx[1], Jx[0], Jz[1]);
    const T czx = cof(Jx[1], Jy[2], Jy[1], Jx[2]), czy = cof(Jy[0], Jx[2], Jx[0], Jy[2]), czz = cof(Jx[0], Jy[1], Jy[0], Jx[1]);
    const T det = std::fma(Jx[2], cxz, std::fma(Jx[1], cxy, Jx[0] * cxx));
    const T r = T(1) / det;
    d[0] = r * std::fma(G[2], cxz, std::fma(G[1], cxy, G[0] * cxx));
    d[1] = r * std::fma(G[2], cyz, std::fma(G[1], cyy, G[0] * cyx));
    d[2] = r * std::fma(G[2], czz, std::fma(G[1], czy, G[0] * czx));
    xi[0] = xi[0] - d[0]; xi[1] = xi[1] - d[1]; xi[2] = xi[2] - d[2];
    const T tt = HexMesh<T>::tol();
    if (std::fabs(d[0]) <= tt && std::fabs(d[1]) <= tt && std::fabs(d[2]) <= tt) break;   // converged
  }
  const T t = HexMesh<T>::tol();
  const bool converged = std::fabs(d[0]) <= t && std::fabs(d[1]) <= t && std::fabs(d[2]) <= t;
  return converged && (xi[0] >= -t && xi[0] <= T(1) + t) && (xi[1] >= -t && xi[1] <= T(1) + t) &&
         (xi[2] >= -t && xi[2] <= T(1) + t);
}

// U2 + U3: the first listed cell of p's bin that contains p; -1 if none.
template <class T> long long hx_locate(const HexMesh<T>& m, const T* p, T* xi) {
  int b[3];
  if (!m.bin_of(p, b)) return -1;
  const size_t id = m.bin_id(b);
  for (uint32_t k = m.bin_start[id]; k < m.bin_start[id + 1]; ++k)
    if (hx_invert(m, m.bin_items[k], p, xi)) return (long long)m.bin_items[k];
  return -1;
}

// Field with the interface the integrators expect (sample, inside): steady, t ignored.
template <class T> struct HexField {
  const HexMesh<T>* m;
  bool inside(const T p[3]) const { T xi[3]; return hx_locate(*m, p, xi) >= 0; }
  uint32_t sample(const T p[3], T /*t*/, T v[3]) const {      // 0 ok, 1 OUT_OF_DOMAIN
    T xi[3];
    long long c = hx_locate(*m, p, xi);
    if (c < 0) return 1u;
    T Q[8];
    for (int a = 0; a < 3; ++a) {
      for (int l = 0; l < 8; ++l) Q[l] = T(m->V[3 * m->H[8 * c + l] + a]);
      v[a] = hx_tri(Q, xi);
    }
    return 0u;
  }
};

}  // namespace oracle
