"""ctypes binding of the CPU oracle (oracle/streami_oracle.hpp, oracle/oracle_capi.cpp).

TEST INFRASTRUCTURE ONLY: importable from tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs, never from paper_2606_02627_b200/.  It does not import
the CUDA package or workloads/; it takes plain numpy arrays.

Build: g++ -O2 -ffp-contract=off -mfma -fopenmp (only the std::fma calls written in the
header are fused; see SURVEY.md 8(c) "Parity principle").
"""
import ctypes
import os
import subprocess

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = [os.path.join(HERE, "oracle_capi.cpp"), os.path.join(HERE, "streami_oracle.hpp"),
        os.path.join(HERE, "hexmesh_oracle.hpp")]
_SO = os.path.join(HERE, "liboracle.so")

OUT_OF_DOMAIN, MAX_STEPS, STAGNANT, HALO_MISS = 1, 2, 3, 4


def build(force=False):
    stale = force or not os.path.exists(_SO) or any(
        os.path.getmtime(s) > os.path.getmtime(_SO) for s in _SRC)
    if stale:
        cmd = ["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-mfma", "-fopenmp", "-fPIC",
               "-shared", _SRC[0], "-o", _SO + ".tmp"]
        subprocess.run(cmd, check=True)
        os.replace(_SO + ".tmp", _SO)
    return _SO


class OGrid(ctypes.Structure):
    _fields_ = [("gdims", ctypes.c_int * 3), ("lo", ctypes.c_int * 3), ("hi", ctypes.c_int * 3),
                ("origin", ctypes.c_float * 3), ("spacing", ctypes.c_float * 3),
                ("nslices", ctypes.c_int), ("slice_dt", ctypes.c_float),
                ("time_mode", ctypes.c_int), ("data", ctypes.c_void_p)]


class OParams(ctypes.Structure):
    _fields_ = [("integrator", ctypes.c_int), ("h", ctypes.c_double), ("h_min", ctypes.c_double),
                ("h_max", ctypes.c_double), ("atol", ctypes.c_double), ("rtol", ctypes.c_double),
                ("max_steps", ctypes.c_uint32), ("vmin", ctypes.c_double), ("t0", ctypes.c_double),
                ("capacity", ctypes.c_uint32), ("stride", ctypes.c_uint32)]


class OAnalytic(ctypes.Structure):
    _fields_ = [("kind", ctypes.c_int), ("c", ctypes.c_double * 16), ("blo", ctypes.c_double * 3),
                ("bhi", ctypes.c_double * 3)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
        _lib.oracle_num_threads.restype = ctypes.c_int
    return _lib


def num_threads():
    return lib().oracle_num_threads()


def _p(a):
    return None if a is None else a.ctypes.data_as(ctypes.c_void_p)


def _dt(precision):
    return (np.float32, "f32") if precision == "f32" else (np.float64, "f64")


def grid(data, dims, origin, spacing, nslices=1, slice_dt=1.0, time_mode=0, gdims=None, lo=None,
         hi=None):
    """Describe one stored array.  Monolithic: the global grid.  Brick: pass gdims/lo/hi."""
    data = np.ascontiguousarray(data, dtype=np.float32)
    g = OGrid()
    gd = tuple(dims) if gdims is None else tuple(gdims)
    lo = (0, 0, 0) if lo is None else tuple(lo)
    hi = tuple(d - 1 for d in gd) if hi is None else tuple(hi)
    stored = tuple(hi[a] - lo[a] + 1 for a in range(3))
    assert data.size == 3 * nslices * stored[0] * stored[1] * stored[2], "data size != stored box"
    g.gdims[:] = gd; g.lo[:] = lo; g.hi[:] = hi
    g.origin[:] = [float(x) for x in origin]; g.spacing[:] = [float(x) for x in spacing]
    g.nslices = nslices; g.slice_dt = float(slice_dt); g.time_mode = time_mode
    g.data = data.ctypes.data
    g._keep = data
    return g


def analytic(kind, coef, blo, bhi):
    a = OAnalytic()
    a.kind = kind
    c = list(coef) + [0.0] * (16 - len(coef))
    a.c[:] = c; a.blo[:] = list(blo); a.bhi[:] = list(bhi)
    return a


def params(integrator=0, h=0.01, h_min=0.0, h_max=1e30, atol=1e-5, rtol=1e-5, max_steps=1000,
           vmin=0.0, t0=0.0, capacity=1, stride=1):
    if integrator == 0:
        h_min, h_max = h, h
    return OParams(integrator, h, h_min, h_max, atol, rtol, max_steps, vmin, t0, capacity, stride)


def sample(g, pts, t=0.0, precision="f32"):
    T, sfx = _dt(precision)
    pts = np.ascontiguousarray(pts, dtype=T).reshape(-1, 3)
    n = pts.shape[0]
    v = np.zeros((n, 3), dtype=T); rc = np.zeros(n, dtype=np.uint32)
    fn = getattr(lib(), "oracle_sample_" + sfx)
    ct = ctypes.c_float if T is np.float32 else ctypes.c_double
    fn.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_size_t, ct, ctypes.c_void_p,
                   ctypes.c_void_p]
    fn(ctypes.byref(g), _p(pts), n, float(t), _p(v), _p(rc))
    return v, rc


class Result(dict):
    __getattr__ = dict.__getitem__


def streamlines(field, seeds, prm, precision="f32", record=True):
    """A5/A6/A8.  `field` is an OGrid or an OAnalytic."""
    T, sfx = _dt(precision)
    seeds = np.ascontiguousarray(seeds, dtype=T).reshape(-1, 3)
    n = seeds.shape[0]
    cap = prm.capacity
    verts = np.full((3, n, cap), np.nan, dtype=T) if record else None
    counts = np.zeros(n, dtype=np.uint32)
    steps = np.zeros(n, dtype=np.uint32); status = np.zeros(n, dtype=np.uint32)
    final = np.zeros((3, n), dtype=T); totals = np.zeros(4, dtype=np.uint64)
    name = "oracle_streamlines_analytic_" if isinstance(field, OAnalytic) else "oracle_streamlines_"
    fn = getattr(lib(), name + sfx)
    fn.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_size_t, ctypes.c_void_p] + \
        [ctypes.c_void_p] * 6
    fn(ctypes.byref(field), _p(seeds), n, ctypes.byref(prm), _p(verts), _p(counts), _p(steps),
       _p(status), _p(final), _p(totals))
    return Result(vertices=verts, counts=counts, steps=steps, status=status, final=final,
                  totals=totals)


def streaklines(field, points, nsteps, prm, precision="f32"):
    """A7.  Returns vertices [3][nsteps][m] (release-major), counts [m], steps/status [nsteps*m]."""
    T, sfx = _dt(precision)
    points = np.ascontiguousarray(points, dtype=T).reshape(-1, 3)
    m = points.shape[0]
    verts = np.zeros((3, nsteps, m), dtype=T)
    counts = np.zeros(m, dtype=np.uint32)
    steps = np.zeros(nsteps * m, dtype=np.uint32); status = np.zeros(nsteps * m, dtype=np.uint32)
    totals = np.zeros(4, dtype=np.uint64)
    name = "oracle_streaklines_analytic_" if isinstance(field, OAnalytic) else "oracle_streaklines_"
    fn = getattr(lib(), name + sfx)
    fn.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_size_t, ctypes.c_uint32,
                   ctypes.c_void_p] + [ctypes.c_void_p] * 5
    fn(ctypes.byref(field), _p(points), m, nsteps, ctypes.byref(prm), _p(verts), _p(counts),
       _p(steps), _p(status), _p(totals))
    return Result(vertices=verts, counts=counts, steps=steps, status=status, totals=totals)


def brick_advect(bricks, brick_grid, seeds, prm, precision="f32", max_rounds=256,
                 log_capacity=None, record=True):
    """A9.  `bricks` = list of OGrid (one per brick, flat id order)."""
    T, sfx = _dt(precision)
    seeds = np.ascontiguousarray(seeds, dtype=T).reshape(-1, 3)
    n = seeds.shape[0]
    nb = len(bricks)
    arr = (OGrid * nb)(*bricks)
    cap = prm.capacity
    verts = np.full((3, n, cap), np.nan, dtype=T) if record else None
    counts = np.zeros(n, dtype=np.uint32)
    steps = np.zeros(n, dtype=np.uint32); status = np.zeros(n, dtype=np.uint32)
    final = np.zeros((3, n), dtype=T); totals = np.zeros(4, dtype=np.uint64)
    round_counts = np.zeros((max_rounds, nb), dtype=np.uint32)
    if log_capacity is None:
        log_capacity = 64 * n + 16
    log = np.zeros(log_capacity, dtype=np.uint64)
    nlog = ctypes.c_ulonglong(0); nrounds = ctypes.c_uint32(0)
    nbg = (ctypes.c_int * 3)(*brick_grid)
    fn = getattr(lib(), "oracle_brick_advect_" + sfx)
    fn.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_size_t,
                   ctypes.c_void_p] + [ctypes.c_void_p] * 6 + [ctypes.c_uint32, ctypes.c_void_p,
                   ctypes.c_size_t, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p]
    fn(arr, nbg, _p(seeds), n, ctypes.byref(prm), _p(verts), _p(counts), _p(steps), _p(status),
       _p(final), _p(round_counts), max_rounds, _p(log), log_capacity, ctypes.byref(nlog),
       ctypes.byref(nrounds), _p(totals))
    return Result(vertices=verts, counts=counts, steps=steps, status=status, final=final,
                  totals=totals, round_counts=round_counts[:nrounds.value + 1],
                  nrounds=nrounds.value, log=np.sort(log[:min(nlog.value, log_capacity)]),
                  nlog=nlog.value)


def rp10(x, precision="f32"):
    T, sfx = _dt(precision)
    x = np.ascontiguousarray(x, dtype=T)
    out = np.empty_like(x)
    fn = getattr(lib(), "oracle_rp10_" + sfx)
    fn.argtypes = [ctypes.c_void_p, ctypes.c_size_t, ctypes.c_void_p]
    fn(_p(x), x.size, _p(out))
    return out


def dp5_tableau(precision="f64"):
    out = np.zeros(42, dtype=np.float64)
    fn = getattr(lib(), "oracle_dp5_tableau_" + precision)
    fn.argtypes = [ctypes.c_void_p]
    fn(_p(out))
    return dict(c=out[0:7], a=out[7:28], b=out[28:35], e=out[35:42])


def seed_shape(o, eu, ev, ew, nu, nv=1, nw=1, mode=0, rng_seed=0):
    """Seeds on a line / plane / box; see oracle_capi.cpp for the fp32 formula."""
    f3 = lambda v: (ctypes.c_float * 3)(*[float(x) for x in v])
    out = np.empty((nu * nv * nw, 3), dtype=np.float32)
    fn = lib().oracle_seed_shape_f32
    fn.argtypes = [ctypes.c_void_p] * 4 + [ctypes.c_uint32] * 3 + [ctypes.c_int, ctypes.c_uint64, ctypes.c_void_p]
    fn(f3(o), f3(eu), f3(ev), f3(ew), nu, nv, nw, mode, rng_seed, _p(out))
    return out


# ---- hexahedral meshes (oracle/hexmesh_oracle.hpp) --------------------------------------------
class HexMesh:
    """X [nv,3] f32 vertex positions, V [nv,3] f32 values, H [nc,8] u32 (corner l = dx+2dy+4dz),
    bin grid nb over the box lo..hi."""

    def __init__(self, X, V, H, lo, hi, nb):
        self.X = np.ascontiguousarray(X, dtype=np.float32)
        self.V = np.ascontiguousarray(V, dtype=np.float32)
        self.H = np.ascontiguousarray(H, dtype=np.uint32)
        self.lo = np.ascontiguousarray(lo, dtype=np.float32)
        self.hi = np.ascontiguousarray(hi, dtype=np.float32)
        self.nb = np.ascontiguousarray(nb, dtype=np.int32)

    def _args(self):
        return [ctypes.c_size_t(self.X.shape[0]), ctypes.c_size_t(self.H.shape[0]), _p(self.X), _p(self.V),
                _p(self.H), _p(self.lo), _p(self.hi), _p(self.nb)]


def hexmesh_sample(mesh, pts, precision="f32", brute=False):
    """(v [n,3], cell [n] (-1 = outside), xi [n,3]); brute = search all cells (the definition)."""
    T, sfx = _dt(precision)
    pts = np.ascontiguousarray(pts, dtype=T).reshape(-1, 3)
    n = pts.shape[0]
    v = np.zeros((n, 3), dtype=T); cell = np.zeros(n, dtype=np.int64); xi = np.zeros((n, 3), dtype=T)
    fn = getattr(lib(), "oracle_hexmesh_sample_" + sfx)
    fn.argtypes = None
    fn(*mesh._args(), _p(pts), ctypes.c_size_t(n), ctypes.c_int(1 if brute else 0), _p(v), _p(cell), _p(xi))
    return v, cell, xi


def hexmesh_streamlines(mesh, seeds, prm, precision="f32", record=True):
    T, sfx = _dt(precision)
    seeds = np.ascontiguousarray(seeds, dtype=T).reshape(-1, 3)
    n = seeds.shape[0]
    cap = prm.capacity
    verts = np.full((3, n, cap), np.nan, dtype=T) if record else None
    counts = np.zeros(n, dtype=np.uint32)
    steps = np.zeros(n, dtype=np.uint32); status = np.zeros(n, dtype=np.uint32)
    final = np.zeros((3, n), dtype=T); totals = np.zeros(4, dtype=np.uint64)
    fn = getattr(lib(), "oracle_hexmesh_streamlines_" + sfx)
    fn.argtypes = None
    fn(*mesh._args(), _p(seeds), ctypes.c_size_t(n), ctypes.byref(prm), _p(verts), _p(counts), _p(steps),
       _p(status), _p(final), _p(totals))
    return Result(vertices=verts, counts=counts, steps=steps, status=status, final=final, totals=totals)
