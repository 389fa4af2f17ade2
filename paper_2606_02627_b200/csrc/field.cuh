// csrc/field.cuh -- device-side field views and the field-sampling layer (a2, a3, a4 of
// SURVEY.md 8(a)): cell location, trilinear gather + interpolation, linear interpolation in time.
//
// The paper's sample() is "computing offsets into [a CUDA global memory] array" of float3 voxels
// (PAPER.md:63, 155); the filter itself is fixed by BASELINE.json (trilinear) and by the fp32
// formula sheet A1-A3.  This file is written from that sheet; it shares
// nothing with oracle/.  The translation unit is compiled with -fmad=false: every fused
// multiply-add below is an explicit __fmaf_rn, everything else rounds once per operation.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace streami {

enum : int { LAYOUT_PACKED3 = 1, LAYOUT_FLOAT4 = 2, LAYOUT_XPAIR = 3, LAYOUT_CELL = 4, LAYOUT_XYQUAD = 5, LAYOUT_SOA = 6, LAYOUT_TEX = 7 };
enum : unsigned { ST_ALIVE = 0, ST_OUT = 1, ST_MAXSTEPS = 2, ST_STAGNANT = 3, ST_HALO = 4 };

// Global geometry (A1), uniform over the launch.
struct Geom {
  float ox, oy, oz;        // origin
  float rx, ry, rz;        // 1/spacing, computed once on the host in fp32
  float topx, topy, topz;  // (float)(N-1)
  int nslices;
  float q, top_s;          // 1/slice_dt, (float)(nslices-1)
  int time_mode;           // 0 linear, 1 hold floor slice
};

// One stored array: the whole grid (lo = 0, hi = N-1) or one brick's stored box (A9).
struct Store {
  const void* data;        // layout-specific records, x fastest
  int lox, loy, loz;       // stored box, global vertex indices, inclusive
  int hix, hiy, hiz;
  int cmx, cmy, cmz;       // hi - 1: the last cell per axis (A2.3 clamp), precomputed
  int topflagx, topflagy, topflagz;  // 1 where hi == N-1 (g == hi is then served too)
  // A9 serve test lo <= g < hi as floats, computed once: fhi = +inf where hi == N-1, because there
  // g <= hi is what the domain test has already established.
  float flox, floy, floz, fhix, fhiy, fhiz;
  // owned cell box of the brick [olo, ohi) in global cell indices (ohi = INT_MAX on the top brick of
  // an axis): floor(g) inside it <=> owner(g) == this brick, without the integer divisions of A9.
  int olox, oloy, oloz, ohix, ohiy, ohiz;
  unsigned nx, nxy;        // row and plane strides in records (vertices; LAYOUT_CELL: cells)
  // Monolithic steady stores: cells per axis if every stored value is tame (finite, |v| <= 2^60),
  // else 0.  See sample_nb: floor(g) < fast on all axes then decides "inside" with integers.
  unsigned fastx, fasty, fastz;
  // Bricks: device address of this descriptor in the brick table.  The advection kernel keeps a copy
  // of the descriptor in registers; the fields only the rare float tests need are read through
  // `self` when wanted instead of staying live (the brick kernel is short of registers).
  const Store* self;
  unsigned long long slice_stride;   // records per slice
  unsigned long long plane;          // LAYOUT_SOA: floats per component plane (all slices)
  unsigned long long tex;            // LAYOUT_TEX: cudaTextureObject_t over the float4 copy (point mode, tex1Dfetch)
};

// A brick grid (A9): owner of an in-domain position.
struct BrickMap {
  int nbx, nby, nbz;
  int Bx, By, Bz;
};

__device__ __forceinline__ float lerp(float a, float b, float w) { return __fmaf_rn(w, b - a, a); }

// One aligned 32-byte record: a single 256-bit read-only load (LDG.E.256 on sm_100a); 6 floats used.
// NA = do not allocate the line in L1.  The branch-free RK4 path asks for that: its demand loads
// still hit lines the one-step-ahead prefetch has brought in, but no longer evict them (768 lanes x
// 4 lines per cell are several times the L1), C2 16.9 -> 16.6 ms.  Without a prefetcher the same
// hint loses (C5 DP5(4) 0.95 -> 1.11 s, C4 two-slice reads 249 -> 276 ms), so it is per caller.
template <bool NA>
__device__ __forceinline__ void ldg_rec32(const char* p, float* o) {
  float p6, p7;
  if (NA)
    asm volatile("ld.global.nc.L1::no_allocate.v8.f32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                 : "=f"(o[0]), "=f"(o[1]), "=f"(o[2]), "=f"(o[3]), "=f"(o[4]), "=f"(o[5]), "=f"(p6), "=f"(p7)
                 : "l"(p));
  else
    asm volatile("ld.global.nc.v8.f32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                 : "=f"(o[0]), "=f"(o[1]), "=f"(o[2]), "=f"(o[3]), "=f"(o[4]), "=f"(o[5]), "=f"(p6), "=f"(p7)
                 : "l"(p));
  (void)p6; (void)p7;
}

// The same load keeping all 8 floats (LAYOUT_CELL: 24 consecutive floats = 3 loads).
template <bool NA>
__device__ __forceinline__ void ldg8(const char* p, float* o) {
  if (NA)
    asm volatile("ld.global.nc.L1::no_allocate.L2::128B.v8.f32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                 : "=f"(o[0]), "=f"(o[1]), "=f"(o[2]), "=f"(o[3]), "=f"(o[4]), "=f"(o[5]), "=f"(o[6]), "=f"(o[7])
                 : "l"(p));
  else
    asm volatile("ld.global.nc.L2::128B.v8.f32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                 : "=f"(o[0]), "=f"(o[1]), "=f"(o[2]), "=f"(o[3]), "=f"(o[4]), "=f"(o[5]), "=f"(o[6]), "=f"(o[7])
                 : "l"(p));
}

// ---- loads of the 8 cell vertices as 4 rows of 6 floats --------------------------------------
// V[row*6 + k], row = dz*2 + dy; k: {V[x].xyz, V[x+1].xyz} or, for the DIFF layouts, the record order.
template <int LAYOUT> struct CellLoad;

template <> struct CellLoad<LAYOUT_PACKED3> {
  template <bool NA>
  static __device__ __forceinline__ void row(const void* data, unsigned long long v, float* o) {
    const float* p = reinterpret_cast<const float*>(data) + 3ull * v;
#pragma unroll
    for (int k = 0; k < 6; ++k) o[k] = __ldg(p + k);
  }
};
template <> struct CellLoad<LAYOUT_FLOAT4> {
  template <bool NA>
  static __device__ __forceinline__ void row(const void* data, unsigned long long v, float* o) {
    const float4* p = reinterpret_cast<const float4*>(data) + v;
    float4 a = __ldg(p), b = __ldg(p + 1);
    o[0] = a.x; o[1] = a.y; o[2] = a.z; o[3] = b.x; o[4] = b.y; o[5] = b.z;
  }
};
template <> struct CellLoad<LAYOUT_XPAIR> {
  template <bool NA>
  static __device__ __forceinline__ void row(const void* data, unsigned long long v, float* o) {
    ldg_rec32<NA>(reinterpret_cast<const char*>(data) + 32ull * v, o);
  }
};

// LAYOUT_CELL: one aligned 128-byte record per CELL: the four DIFF rows {Vx, Vy, Dx, Dy, Vz, Dz} of
// that cell (row = dz*2 + dy) as 24 consecutive floats, then 32 bytes of padding.  All 8 corner
// vertices sit in ONE 128-byte L2 line: three 256-bit loads whose misses the L1 merges into ~1.4 L2
// requests per cell (ncu on C5), where XYQUAD's two 64-byte pieces make 4.
template <> struct CellLoad<LAYOUT_CELL> {
  template <bool NA>
  static __device__ __forceinline__ void cell(const void* data, unsigned long long c, float* V) {
    const char* p = reinterpret_cast<const char*>(data) + 128ull * c;
#pragma unroll
    for (int r = 0; r < 3; ++r) ldg8<NA>(p + 32 * r, V + 8 * r);
  }
};

// LAYOUT_XYQUAD: one aligned 64-byte record per VERTEX = the XPAIR rows (x, y) and (x, y+1) back to
// back: a cell is two 64-byte pieces (z and z+1).  DRAM brings 64 bytes per missed 32-byte sector
// (ncu on C5: 3.7 TB read for 1.8 TB of missed sectors); here both halves of every fetch are used.
template <> struct CellLoad<LAYOUT_XYQUAD> {
  template <bool NA>
  static __device__ __forceinline__ void pair(const void* data, unsigned long long v, float* o) {
    const char* p = reinterpret_cast<const char*>(data) + 64ull * v;
#pragma unroll
    for (int r = 0; r < 2; ++r) ldg_rec32<NA>(p + 32 * r, o + 6 * r);
  }
};

// LAYOUT_SOA: three component planes of fp32 (the other layout north_star names): a row is 2 floats from
// each of three planes, a cell 24 scalar loads from 12 distant sectors.  LAYOUT_TEX: the FLOAT4 copy read
// through a texture object in POINT mode (tex1Dfetch; the lerps stay in registers, A2 -- hardware filtering
// has 8-bit weights).  Both exist so that the layout choice is settled by measurement.
template <int LAYOUT>
__device__ __forceinline__ void load_row_alt(const Store& s, unsigned long long v, float* o) {
  if constexpr (LAYOUT == LAYOUT_SOA) {
    const float* p = reinterpret_cast<const float*>(s.data) + v;
#pragma unroll
    for (int c = 0; c < 3; ++c) { o[c] = __ldg(p + c * s.plane); o[3 + c] = __ldg(p + c * s.plane + 1); }
  } else {
    const float4 a = tex1Dfetch<float4>((cudaTextureObject_t)s.tex, (int)v);
    const float4 b = tex1Dfetch<float4>((cudaTextureObject_t)s.tex, (int)v + 1);
    o[0] = a.x; o[1] = a.y; o[2] = a.z; o[3] = b.x; o[4] = b.y; o[5] = b.z;
  }
}
template <int LAYOUT> struct AltLayout { static constexpr bool value = LAYOUT == LAYOUT_SOA || LAYOUT == LAYOUT_TEX; };

template <int LAYOUT>
__device__ __forceinline__ void load_cell(const Store& s, unsigned long long v, float* V) {
  if constexpr (AltLayout<LAYOUT>::value) {
    load_row_alt<LAYOUT>(s, v, V); load_row_alt<LAYOUT>(s, v + s.nx, V + 6);
    load_row_alt<LAYOUT>(s, v + s.nxy, V + 12); load_row_alt<LAYOUT>(s, v + s.nxy + s.nx, V + 18);
  } else if constexpr (LAYOUT == LAYOUT_CELL) {
    CellLoad<LAYOUT_CELL>::template cell<false>(s.data, v, V);
  } else if constexpr (LAYOUT == LAYOUT_XYQUAD) {
    CellLoad<LAYOUT_XYQUAD>::template pair<false>(s.data, v, V);
    CellLoad<LAYOUT_XYQUAD>::template pair<false>(s.data, v + s.nxy, V + 12);
  } else {
    CellLoad<LAYOUT>::template row<false>(s.data, v, V);
    CellLoad<LAYOUT>::template row<false>(s.data, v + s.nx, V + 6);
    CellLoad<LAYOUT>::template row<false>(s.data, v + s.nxy, V + 12);
    CellLoad<LAYOUT>::template row<false>(s.data, v + s.nxy + s.nx, V + 18);
  }
}

// A steady store holds fewer than 2^32 vertices (checked at create time), so the four row
// indices fit 32 bits (v + nxy + nx <= nvert - 1) and each address is one 32x32->64 multiply-add.
template <int LAYOUT, bool NA = false>
__device__ __forceinline__ void load_cell32(const Store& s, unsigned v, float* V) {
  if constexpr (AltLayout<LAYOUT>::value) {
    load_cell<LAYOUT>(s, (unsigned long long)v, V);
  } else if constexpr (LAYOUT == LAYOUT_CELL) {
    CellLoad<LAYOUT_CELL>::template cell<NA>(s.data, v, V);
  } else if constexpr (LAYOUT == LAYOUT_XYQUAD) {
    CellLoad<LAYOUT_XYQUAD>::template pair<NA>(s.data, v, V);
    CellLoad<LAYOUT_XYQUAD>::template pair<NA>(s.data, v + s.nxy, V + 12);
  } else {
    CellLoad<LAYOUT>::template row<NA>(s.data, v, V);
    CellLoad<LAYOUT>::template row<NA>(s.data, v + s.nx, V + 6);
    CellLoad<LAYOUT>::template row<NA>(s.data, v + s.nxy, V + 12);
    CellLoad<LAYOUT>::template row<NA>(s.data, v + s.nxy + s.nx, V + 18);
  }
}

// Layouts whose records hold V[x] and V[x+1] - V[x] instead of {V[x], V[x+1]}: the subtraction of
// the x-lerp, lerp(a, b, w) = fma(w, b - a, a), does not depend on the sample point, so the
// repack does it once per vertex pair (the same fp32 operation, the same bits) and every sample
// saves 12 of its 42 interpolation instructions.
template <int LAYOUT> struct LayoutTraits { static constexpr bool DIFF = LAYOUT == LAYOUT_XPAIR || LAYOUT == LAYOUT_CELL || LAYOUT == LAYOUT_XYQUAD; };

// Packed fp32 pairs (sm_100a FFMA2 / FADD2: two IEEE fp32 operations per instruction, each lane
// rounded exactly like the scalar instruction, so results do not change).
__device__ __forceinline__ float2 sub2(float2 a, float2 b) {
  float2 d;
  asm("{ .reg .b64 ra, rb, rd; mov.b64 ra, {%2,%3}; mov.b64 rb, {%4,%5}; sub.rn.f32x2 rd, ra, rb; mov.b64 {%0,%1}, rd; }"
      : "=f"(d.x), "=f"(d.y) : "f"(a.x), "f"(a.y), "f"(b.x), "f"(b.y));
  return d;
}
__device__ __forceinline__ float2 lerp2(float2 a, float2 b, float w) {
  return __ffma2_rn(make_float2(w, w), sub2(b, a), a);
}

// A2.5: x first, then y, then z; 7 lerps per component.
// DIFF rows are {Vx, Vy, Dx, Dy, Vz, Dz} (D = V[x+1] - V[x]): the x and y components of a row sit in
// aligned register pairs after the 256-bit load and go through the packed instructions together;
// the z components of the four rows are paired after their (scalar) x-lerp.  18 instructions per
// sample where the scalar form takes 30.
template <bool DIFF>
__device__ __forceinline__ void interp_cell(const float* V, float fx, float fy, float fz,
                                            float& vx, float& vy, float& vz) {
  if constexpr (DIFF) {
    const float2 fx2 = make_float2(fx, fx);
    float2 c[4]; float z[4];
#pragma unroll
    for (int r = 0; r < 4; ++r) {
      c[r] = __ffma2_rn(fx2, make_float2(V[6 * r + 2], V[6 * r + 3]), make_float2(V[6 * r], V[6 * r + 1]));
      z[r] = __fmaf_rn(fx, V[6 * r + 5], V[6 * r + 4]);
    }
    const float2 q0 = lerp2(c[0], c[1], fy), q1 = lerp2(c[2], c[3], fy);             // y, planes z and z+1
    const float2 qz = lerp2(make_float2(z[0], z[2]), make_float2(z[1], z[3]), fy);   // y, the z component of both planes
    const float2 xy = lerp2(q0, q1, fz);
    vx = xy.x; vy = xy.y; vz = lerp(qz.x, qz.y, fz);
  } else {
    float r[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      float c00 = lerp(V[0 + c], V[3 + c], fx), c01 = lerp(V[6 + c], V[9 + c], fx);
      float c10 = lerp(V[12 + c], V[15 + c], fx), c11 = lerp(V[18 + c], V[21 + c], fx);
      float c0 = lerp(c00, c01, fy);
      float c1 = lerp(c10, c11, fy);
      r[c] = lerp(c0, c1, fz);
    }
    vx = r[0]; vy = r[1]; vz = r[2];
  }
}

// Register-resident copy of the current cell (build's choice: a sample that stays in the cell of
// the previous one costs no loads; the arithmetic, hence the result, is unchanged).
struct CellCache {
  unsigned key;                  // vertex index of the cell's low corner inside the current store
  float V[24];
  __device__ __forceinline__ void invalidate() { key = 0xffffffffu; }   // never a low corner
};

// The same for an unsteady field read with linear interpolation in time (A3): the cell in slice j
// and in slice j+1, keyed by the record index in slice j (which fixes j as well).  Stages 2 and 3 of
// an RK4 step share their time and almost always their cell, and so do stage 4 and stage 1 of the
// next step (t_n + h and t_{n+1} fall in the same slice interval, the points differ by O(h^2)): about
// half of the two-slice gathers of a streakline step are repeats.
struct CellCacheT {
  unsigned long long key;
  float V[48];
  __device__ __forceinline__ void invalidate() { key = ~0ull; }
};
template <class CC> struct IsTimeCache { static constexpr bool value = false; };
template <> struct IsTimeCache<CellCacheT> { static constexpr bool value = true; };

// A2.1 + A2.2: index-space position and the closed-box test (NaN -> false).
// UNIT = the grid is its own index space (origin 0, spacing 1, hence r = 1): (p - 0.0f) * 1.0f
// returns p bit for bit, so the two operations are skipped.  C2, C3 and C5 are such grids.
template <bool UNIT>
__device__ __forceinline__ void index_pos(const Geom& g, float px, float py, float pz, float& gx,
                                          float& gy, float& gz) {
  if (UNIT) { gx = px; gy = py; gz = pz; }
  else { gx = (px - g.ox) * g.rx; gy = (py - g.oy) * g.ry; gz = (pz - g.oz) * g.rz; }
}
__device__ __forceinline__ bool in_domain(const Geom& g, float gx, float gy, float gz) {
  return (gx >= 0.0f && gx <= g.topx) && (gy >= 0.0f && gy <= g.topy) &&
         (gz >= 0.0f && gz <= g.topz);
}
template <bool UNIT = false>
__device__ __forceinline__ bool to_index(const Geom& g, float px, float py, float pz, float& gx,
                                         float& gy, float& gz) {
  index_pos<UNIT>(g, px, py, pz, gx, gy, gz);
  return in_domain(g, gx, gy, gz);
}

// Cell location inside one store.  Returns false (HALO_MISS) if the store cannot serve g.
// g >= 0 here, so float->int truncation equals floor.
template <bool BRICK>
__device__ __forceinline__ bool locate(const Store& s, float gx, float gy, float gz,
                                       unsigned long long& v, float& fx, float& fy, float& fz) {
  if (BRICK) {           // the caller has passed the domain test, so g <= N-1 already holds
    bool in = (gx >= s.flox) && (gx < s.fhix) && (gy >= s.floy) && (gy < s.fhiy) &&
              (gz >= s.floz) && (gz < s.fhiz);
    if (!in) return false;
  }
  int ix = min(__float2int_rz(gx), s.cmx);
  int iy = min(__float2int_rz(gy), s.cmy);
  int iz = min(__float2int_rz(gz), s.cmz);
  fx = gx - (float)ix; fy = gy - (float)iy; fz = gz - (float)iz;
  if (BRICK) { ix -= s.lox; iy -= s.loy; iz -= s.loz; }   // a monolithic store starts at 0
  // fewer than 2^32 records per slice (checked at create time): 32-bit arithmetic is exact
  v = (unsigned long long)((unsigned)iz * s.nxy + (unsigned)iy * s.nx + (unsigned)ix);
  return true;
}

// A3: slice index and weight.  Returns the slice j to read first; two = read j+1 as well.
__device__ __forceinline__ int time_slice(const Geom& g, float t, float& a, bool& two) {
  float s = t * g.q;
  s = fminf(fmaxf(s, 0.0f), g.top_s);
  if (g.time_mode == 1) { two = false; a = 0.0f; return min(__float2int_rz(s), g.nslices - 1); }
  int j = min(__float2int_rz(s), g.nslices - 2);
  a = s - (float)j; two = true;
  return j;
}

// Full sample S(p, t) (A2/A3, brick form A9).  Returns 0 ok, ST_OUT or ST_HALO.
// KNOWN: the caller has already established that p is inside the domain (it passed the A5.5 test
// at the end of the previous step, or the A5.1 test at the seed), so the test is not repeated.
template <int LAYOUT, bool UNSTEADY, bool BRICK, bool CACHE, bool UNIT = false, bool KNOWN = false, class CC = CellCache>
__device__ __forceinline__ unsigned sample(const Geom& g, const Store& s, CC& cc, float px,
                                           float py, float pz, float t, float& vx, float& vy,
                                           float& vz) {
  float gx, gy, gz;
  index_pos<UNIT>(g, px, py, pz, gx, gy, gz);
  unsigned long long v; float fx, fy, fz;
  if constexpr (BRICK && !UNSTEADY) {
    // Integer accept (see sample_nb), brick form: lo <= floor(g) < hi on every axis <=> the brick
    // serves g (A9) and g is inside the domain; no clamp is needed there.  fast = hi - lo if every
    // brick is tame, else 0; the faces g = N-1, misses, the outside and +-inf take the float tests.
    const int jx = __float2int_rd(gx), jy = __float2int_rd(gy), jz = __float2int_rd(gz);
    const int lx = jx - s.lox, ly = jy - s.loy, lz = jz - s.loz;
    if (((unsigned)lx < s.fastx) & ((unsigned)ly < s.fasty) & ((unsigned)lz < s.fastz)) {
      fx = gx - (float)jx; fy = gy - (float)jy; fz = gz - (float)jz;
      v = (unsigned long long)((unsigned)lz * s.nxy + (unsigned)ly * s.nx + (unsigned)lx);
    } else {
      if (!KNOWN) { if (!in_domain(g, gx, gy, gz)) return ST_OUT; }
      if (!locate<BRICK>(*s.self, gx, gy, gz, v, fx, fy, fz)) return ST_HALO;
    }
  } else if constexpr (!BRICK && !UNSTEADY && !KNOWN) {
    // the same accept for a monolithic steady store (DP5(4) stages; RK4 goes through sample_nb)
    const int jx = __float2int_rd(gx), jy = __float2int_rd(gy), jz = __float2int_rd(gz);
    if (((unsigned)jx < s.fastx) & ((unsigned)jy < s.fasty) & ((unsigned)jz < s.fastz)) {
      fx = gx - (float)jx; fy = gy - (float)jy; fz = gz - (float)jz;
      v = (unsigned long long)((unsigned)jz * s.nxy + (unsigned)jy * s.nx + (unsigned)jx);
    } else {
      if (!in_domain(g, gx, gy, gz)) return ST_OUT;
      locate<false>(s, gx, gy, gz, v, fx, fy, fz);
    }
  } else {
    if (!KNOWN) { if (!in_domain(g, gx, gy, gz)) return ST_OUT; }
    if (!locate<BRICK>(s, gx, gy, gz, v, fx, fy, fz)) return ST_HALO;
  }
  if (UNSTEADY) {
    float a; bool two;
    int j = time_slice(g, t, a, two);
    unsigned long long vj = v + (unsigned long long)j * s.slice_stride;
    if constexpr (CACHE && IsTimeCache<CC>::value) {
      if (two) {
        if (vj != cc.key) {
          load_cell<LAYOUT>(s, vj, cc.V);
          load_cell<LAYOUT>(s, vj + s.slice_stride, cc.V + 24);
          cc.key = vj;
        }
        float ux, uy, uz, wx, wy, wz;
        interp_cell<LayoutTraits<LAYOUT>::DIFF>(cc.V, fx, fy, fz, ux, uy, uz);
        interp_cell<LayoutTraits<LAYOUT>::DIFF>(cc.V + 24, fx, fy, fz, wx, wy, wz);
        vx = lerp(ux, wx, a); vy = lerp(uy, wy, a); vz = lerp(uz, wz, a);   // space first, time last
        return 0;
      } else {                                         // hold-floor-slice mode: one slice, the first half of the copy
        const unsigned long long k1 = vj | (1ull << 63);
        if (k1 != cc.key) { load_cell<LAYOUT>(s, vj, cc.V); cc.key = k1; }
        interp_cell<LayoutTraits<LAYOUT>::DIFF>(cc.V, fx, fy, fz, vx, vy, vz);
        return 0;
      }
    }
    float V[24];
    load_cell<LAYOUT>(s, vj, V);
    float ux, uy, uz;
    interp_cell<LayoutTraits<LAYOUT>::DIFF>(V, fx, fy, fz, ux, uy, uz);
    if (two) {
      load_cell<LAYOUT>(s, vj + s.slice_stride, V);
      float wx, wy, wz;
      interp_cell<LayoutTraits<LAYOUT>::DIFF>(V, fx, fy, fz, wx, wy, wz);
      vx = lerp(ux, wx, a); vy = lerp(uy, wy, a); vz = lerp(uz, wz, a);   // space first, time last
    } else { vx = ux; vy = uy; vz = uz; }
  } else if constexpr (CACHE && !IsTimeCache<CC>::value) {
    const unsigned v32 = (unsigned)v;
    if (v32 != cc.key) { load_cell32<LAYOUT, (LAYOUT == LAYOUT_CELL && !BRICK)>(s, v32, cc.V); cc.key = v32; }
    interp_cell<LayoutTraits<LAYOUT>::DIFF>(cc.V, fx, fy, fz, vx, vy, vz);
  } else {
    float V[24];
    load_cell32<LAYOUT>(s, (unsigned)v, V);
    interp_cell<LayoutTraits<LAYOUT>::DIFF>(V, fx, fy, fz, vx, vy, vz);
  }
  return 0;
}

// Branch-free steady sample: the status comes back as a value and the caller decides ONCE per
// step.  A position that fails the tests is clamped into the store, so the gather stays in bounds
// and the interpolated value is simply never used (the particle ends in this step).  Early
// returns cost more than they save here: every exit of the inlined step has to move the live
// particle state into the registers of the merge point (measured: ~120 MOV/IMAD.MOV per
// warp-iteration in the r1 kernel).  The arithmetic of a passing sample is unchanged.
template <int LAYOUT, bool BRICK, bool CACHE, bool UNIT, bool KNOWN>
__device__ __forceinline__ unsigned sample_nb(const Geom& g, const Store& s, CellCache& cc, float px,
                                              float py, float pz, float& vx, float& vy, float& vz) {
  float gx, gy, gz;
  index_pos<UNIT>(g, px, py, pz, gx, gy, gz);
  unsigned rc = 0;
  if (BRICK) {
    const bool served = (gx >= s.flox) && (gx < s.fhix) && (gy >= s.floy) && (gy < s.fhiy) &&
                        (gz >= s.floz) && (gz < s.fhiz);
    rc = served ? 0u : (unsigned)ST_HALO;
  }
  int ix, iy, iz;
  if constexpr (!BRICK && !KNOWN) {
    // Integer accept: 0 <= floor(g) <= N-2 on every axis <=> 0 <= g < N-1, which is inside the
    // closed box and needs no clamp (floor = truncation there).  Everything else -- outside, on
    // the top face g == N-1, +-inf (the conversion saturates) -- takes the exact float test.  A NaN
    // converts to 0 and would be accepted, so `fast` is 0 unless the field is tame: with finite
    // values <= 2^60 no lerp forms inf - inf or 0 * inf, and a stage point fma(h, k, p) of finite
    // operands is finite or +-inf, never NaN.  3 integer compares replace 6 float compares and 6
    // clamps per stage sample.
    ix = __float2int_rd(gx); iy = __float2int_rd(gy); iz = __float2int_rd(gz);
    const bool fast = ((unsigned)ix < s.fastx) & ((unsigned)iy < s.fasty) & ((unsigned)iz < s.fastz);
    if (__builtin_expect(!fast, 0)) {
      rc = in_domain(g, gx, gy, gz) ? 0u : (unsigned)ST_OUT;
      ix = max(min(__float2int_rz(gx), s.cmx), 0); iy = max(min(__float2int_rz(gy), s.cmy), 0);
      iz = max(min(__float2int_rz(gz), s.cmz), 0);
    }
  } else {
    if (!KNOWN) rc = in_domain(g, gx, gy, gz) ? rc : (unsigned)ST_OUT;      // OUT wins over HALO (A9)
    ix = min(__float2int_rz(gx), s.cmx); iy = min(__float2int_rz(gy), s.cmy); iz = min(__float2int_rz(gz), s.cmz);
    if (!KNOWN || BRICK) { ix = max(ix, BRICK ? s.lox : 0); iy = max(iy, BRICK ? s.loy : 0); iz = max(iz, BRICK ? s.loz : 0); }
  }
  const float fx = gx - (float)ix, fy = gy - (float)iy, fz = gz - (float)iz;
  if (BRICK) { ix -= s.lox; iy -= s.loy; iz -= s.loz; }
  const unsigned v32 = (unsigned)iz * s.nxy + (unsigned)iy * s.nx + (unsigned)ix;
  if (CACHE) {
    if (v32 != cc.key) { load_cell32<LAYOUT, !BRICK>(s, v32, cc.V); cc.key = v32; }
    interp_cell<LayoutTraits<LAYOUT>::DIFF>(cc.V, fx, fy, fz, vx, vy, vz);
  } else {
    float V[24];
    load_cell32<LAYOUT>(s, v32, V);
    interp_cell<LayoutTraits<LAYOUT>::DIFF>(V, fx, fy, fz, vx, vy, vz);
  }
  return rc;
}

// ---- one-step-ahead cell prefetch (build's choice; results unchanged) ------------------------
// The first touch of a new cell stalls the whole warp for an L2/DRAM round trip, and it happens
// mid-step (stage 2 or 4), where the lane has nothing else to do.  At the END of a step the next
// step's stage points are known to ~1 % of a cell (p_new + 0.5 d and p_new + d with
// d = p_new - p), so the cells they fall in are requested then, a whole warp-iteration early.
// The request is a 4-byte cp.async (LDGSTS, .ca: allocates in L1) per 32-byte sector into a
// scratch word of shared memory that is never read: no destination registers, nothing to wait on.
__device__ __forceinline__ void prefetch_sector(const void* gptr, unsigned smem_addr) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(smem_addr), "l"(gptr) : "memory");
}

template <int LAYOUT>
__device__ __forceinline__ void prefetch_cell32(const Store& s, unsigned v, unsigned smem_addr) {
  if constexpr (AltLayout<LAYOUT>::value) {
    return;                                  // comparison layouts: no prefetcher
  } else if constexpr (LAYOUT == LAYOUT_CELL) {
    const char* p = reinterpret_cast<const char*>(s.data) + 128ull * v;
#pragma unroll
    for (int r = 0; r < 3; ++r) prefetch_sector(p + 32 * r, smem_addr);
  } else if constexpr (LAYOUT == LAYOUT_XYQUAD) {
    const char* p = reinterpret_cast<const char*>(s.data);
    prefetch_sector(p + 64ull * v, smem_addr);
    prefetch_sector(p + 64ull * v + 32, smem_addr);
    prefetch_sector(p + 64ull * (v + s.nxy), smem_addr);
    prefetch_sector(p + 64ull * (v + s.nxy) + 32, smem_addr);
  } else {
    constexpr unsigned long long REC = LAYOUT == LAYOUT_XPAIR ? 32ull : (LAYOUT == LAYOUT_FLOAT4 ? 16ull : 12ull);
    const char* p = reinterpret_cast<const char*>(s.data);
    prefetch_sector(p + REC * v, smem_addr);
    prefetch_sector(p + REC * (v + s.nx), smem_addr);
    prefetch_sector(p + REC * (v + s.nxy), smem_addr);
    prefetch_sector(p + REC * (v + s.nxy + s.nx), smem_addr);
  }
}

// Cell (record index inside the store) that holds index-space position g, clamped into the store
// so that the address is always valid (a prediction may point anywhere; NaN converts to 0).
template <bool BRICK>
__device__ __forceinline__ unsigned clamped_cell(const Store& s, float gx, float gy, float gz) {
  int ix, iy, iz;
  if (BRICK) {      // from lo and the integer-accept range only (fast = 0: every prediction maps to cell 0)
    ix = max(min(__float2int_rz(gx) - s.lox, (int)s.fastx - 1), 0);
    iy = max(min(__float2int_rz(gy) - s.loy, (int)s.fasty - 1), 0);
    iz = max(min(__float2int_rz(gz) - s.loz, (int)s.fastz - 1), 0);
  } else {
    ix = max(min(__float2int_rz(gx), s.cmx), 0);
    iy = max(min(__float2int_rz(gy), s.cmy), 0);
    iz = max(min(__float2int_rz(gz), s.cmz), 0);
  }
  return (unsigned)iz * s.nxy + (unsigned)iy * s.nx + (unsigned)ix;
}

// A9: owner brick of an in-domain position (destinationID).
// Same brick as before?  floor(g) per axis inside the owned box (g >= 0 here: truncation = floor).
template <bool UNIT = false>
__device__ __forceinline__ bool still_owned(const Geom& g, const Store& s, float px, float py, float pz) {
  float gx, gy, gz;
  index_pos<UNIT>(g, px, py, pz, gx, gy, gz);
  const int ix = __float2int_rz(gx), iy = __float2int_rz(gy), iz = __float2int_rz(gz);
  return ix >= s.olox && ix < s.ohix && iy >= s.oloy && iy < s.ohiy && iz >= s.oloz && iz < s.ohiz;
}

template <bool UNIT = false>
__device__ __forceinline__ int owner_of(const Geom& g, const BrickMap& m, float px, float py,
                                        float pz) {
  float gx, gy, gz;
  index_pos<UNIT>(g, px, py, pz, gx, gy, gz);
  int bx = min(__float2int_rd(gx) / m.Bx, m.nbx - 1);
  int by = min(__float2int_rd(gy) / m.By, m.nby - 1);
  int bz = min(__float2int_rd(gz) / m.Bz, m.nbz - 1);
  return (bz * m.nby + by) * m.nbx + bx;
}

}  // namespace streami
