"""Seeded synthetic inputs for the five BASELINE.json configs (C1..C5).

This package serves BOTH the CPU oracle (oracle/) and the CUDA library
(paper_2606_02627_b200/) with the same bytes. It holds none of the traced method's
arithmetic: no interpolation, no Runge-Kutta, no termination logic -- only random
numbers, seed positions, analytic fields sampled at grid vertices (computed in fp64,
rounded once to fp32) and the brick cut of an array.  Recipes: SURVEY.md 8(d), restated
in DESIGN.md section 4.  The paper's own data sets (Fig. 1/3/5) are not
available; these synthetic fields stand in for them.

Neither `oracle` nor `paper_2606_02627_b200` imports this package; tests and bench.py do.
"""
import ctypes
import math
from dataclasses import dataclass, field as _dc_field

import numpy as np

from . import _build

_host = None


def _lib():
    global _host
    if _host is None:
        L = ctypes.CDLL(_build.build_host())
        u64, i32, f64 = ctypes.c_uint64, ctypes.c_int, ctypes.c_double
        P = ctypes.c_void_p
        L.wl_uniform.argtypes = [u64, u64, u64, P]
        L.wl_seeds_uniform.argtypes = [u64, u64, P, P]
        L.wl_abc_fill.argtypes = [i32, f64, f64, f64, f64, P]
        L.wl_turb_modes.argtypes = [u64, i32, f64, f64, i32, P]
        L.wl_turb_fill_direct.argtypes = [P, P, i32, P, P]
        L.wl_turb_fill_direct.restype = f64
        L.wl_scale_round.argtypes = [ctypes.c_size_t, P, f64, P]
        L.wl_double_gyre_fill.argtypes = [P, i32, f64, f64, f64, f64, f64, P]
        _host = L
    return _host


def _p(a):
    return a.ctypes.data_as(ctypes.c_void_p)


@dataclass
class Field:
    """A structured vector field as the application hands it over:
    packed fp32 3-vectors, x fastest, slices outermost."""
    dims: tuple            # (Nx, Ny, Nz) vertices
    origin: tuple          # fp32 world position of vertex (0,0,0)
    spacing: tuple         # fp32 spacing per axis
    data: np.ndarray       # [nslices, Nz, Ny, Nx, 3] float32
    nslices: int = 1
    slice_dt: float = 1.0


def uniform(seed, n, skip=0):
    out = np.empty(n, dtype=np.float64)
    _lib().wl_uniform(seed, skip, n, _p(out))
    return out


def seeds_uniform(seed, n, ext):
    """n seeds, p_a = u * ext_a (fp64), rounded to fp32, clamped to float(ext_a)."""
    ext = np.asarray(ext, dtype=np.float64)
    out = np.empty((n, 3), dtype=np.float32)
    _lib().wl_seeds_uniform(seed, n, _p(ext), _p(out))
    return out


def abc_field(N=32, A=math.sqrt(3.0), B=math.sqrt(2.0), C=1.0):
    """C1: ABC flow on N^3 vertices of [0, 2pi]^3, origin 0, spacing fp32(2pi/(N-1))."""
    L = 2.0 * math.pi
    data = np.empty((1, N, N, N, 3), dtype=np.float32)
    _lib().wl_abc_fill(N, L, A, B, C, _p(data))
    sp = float(np.float32(L / (N - 1)))
    return Field((N, N, N), (0.0, 0.0, 0.0), (sp, sp, sp), data)


def turb_modes(seed, M, kmin, kmax, N):
    table = np.empty((M, 8), dtype=np.float64)
    _lib().wl_turb_modes(seed, M, float(kmin), float(kmax), N, _p(table))
    return table


def turb_field_cpu(N, M, kmin, kmax, seed=2606):
    """Turbulence generator, direct CPU evaluation (small N only: cost N^3 * M cosines).
    Index-space coordinates: origin 0, spacing 1; unit RMS speed over all vertices."""
    table = turb_modes(seed, M, kmin, kmax, N)
    dims = np.array([N, N, N], dtype=np.int32)
    lo = np.zeros(3, dtype=np.int32)
    tmp = np.empty((N, N, N, 3), dtype=np.float64)
    sumsq = _lib().wl_turb_fill_direct(_p(dims), _p(lo), M, _p(table), _p(tmp))
    scale = 1.0 / math.sqrt(sumsq / float(N) ** 3)
    data = np.empty((1, N, N, N, 3), dtype=np.float32)
    _lib().wl_scale_round(tmp.size, _p(tmp), scale, _p(data))
    return Field((N, N, N), (0.0, 0.0, 0.0), (1.0, 1.0, 1.0), data)


def double_gyre_field(dims=(256, 128, 64), nslices=64, dt=0.25, A=0.1, eps=0.25,
                      omega=2.0 * math.pi / 10.0, wamp=0.05):
    """C4: 3D-extended double gyre over [0,2]x[0,1]x[0,1], nslices slices at k*dt."""
    nx, ny, nz = dims
    d = np.array(dims, dtype=np.int32)
    data = np.empty((nslices, nz, ny, nx, 3), dtype=np.float32)
    _lib().wl_double_gyre_fill(_p(d), nslices, dt, A, eps, omega, wamp, _p(data))
    sp = (float(np.float32(2.0 / (nx - 1))), float(np.float32(1.0 / (ny - 1))),
          float(np.float32(1.0 / (nz - 1))))
    return Field(tuple(dims), (0.0, 0.0, 0.0), sp, data, nslices, float(dt))


def rake_c4(na=64, nb=64, y=0.25):
    """C4 rake: x_a = 2(a+0.5)/na, z_b = (b+0.5)/nb, point i = b*na + a."""
    a = (np.arange(na, dtype=np.float64) + 0.5) * 2.0 / na
    b = (np.arange(nb, dtype=np.float64) + 0.5) / nb
    pts = np.empty((nb, na, 3), dtype=np.float32)
    pts[..., 0] = a[None, :]
    pts[..., 1] = y
    pts[..., 2] = b[:, None]
    return pts.reshape(-1, 3)


def brick_boxes(global_dims, brick_grid, ghost):
    """Stored vertex box [lo, hi] (inclusive, global vertex indices) of every brick, flat id
    (bz*nby + by)*nbx + bx.  PAPER.md:65: a macrocell stores its bounds plus a halo."""
    N, nb = global_dims, brick_grid
    B = [N[a] // nb[a] for a in range(3)]
    boxes = []
    for bz in range(nb[2]):
        for by in range(nb[1]):
            for bx in range(nb[0]):
                b = (bx, by, bz)
                lo = [max(B[a] * b[a] - ghost, 0) for a in range(3)]
                hi = [min(B[a] * (b[a] + 1) + ghost, N[a] - 1) for a in range(3)]
                if b[0] == nb[0] - 1: hi[0] = N[0] - 1
                if b[1] == nb[1] - 1: hi[1] = N[1] - 1
                if b[2] == nb[2] - 1: hi[2] = N[2] - 1
                boxes.append((tuple(lo), tuple(hi)))
    return boxes


def cut_bricks(fld, brick_grid, ghost=1):
    """Cut a steady field into independent brick arrays (each its own allocation), the way
    each MPI rank of the paper would hold its partition plus halo."""
    assert fld.nslices == 1
    vol = fld.data[0]
    out = []
    for lo, hi in brick_boxes(fld.dims, brick_grid, ghost):
        out.append(np.ascontiguousarray(
            vol[lo[2]:hi[2] + 1, lo[1]:hi[1] + 1, lo[0]:hi[0] + 1, :]))
    return out


# ---- CUDA generators for the large fields (input generation only; see workloads/fill.cu) ------
_cuda = None


def _cuda_lib():
    global _cuda
    if _cuda is None:
        L = ctypes.CDLL(_build.build_cuda())
        P, i32, f64, Z = ctypes.c_void_p, ctypes.c_int, ctypes.c_double, ctypes.c_size_t
        L.wl_cuda_turb_partials.argtypes = [Z]
        L.wl_cuda_turb_partials.restype = Z
        L.wl_cuda_turb_fill.argtypes = [P, P, i32, P, P, P, P]
        L.wl_cuda_scale_round.argtypes = [Z, P, f64, P, P]
        L.wl_cuda_cut_box.argtypes = [P, P, P, P, P, P]
        _cuda = L
    return _cuda


def turb_field_cuda(N, M, kmin, kmax, seed=2606, host=True, zchunk=64):
    """Turbulence generator on the GPU (C2/C3/C5 sizes), same recipe and mode table as
    turb_field_cpu: fp64 evaluation, one normalisation over the whole grid, one rounding to
    fp32.  Returns (Field or None, cuda tensor [1,N,N,N,3]); Field.data is the host copy of the
    SAME bytes (host=False skips it).  The fp64 intermediate is produced in z-chunks; per-block
    sums of squares are added on the host in block order, so the result is deterministic."""
    import torch
    L = _cuda_lib()
    table = turb_modes(seed, M, kmin, kmax, N)
    d_table = torch.from_numpy(table).cuda()
    st = ctypes.c_void_p(torch.cuda.current_stream().cuda_stream)
    out = torch.empty((1, N, N, N, 3), dtype=torch.float32, device="cuda")
    # pass 1: sum of squares (fp64 values kept per chunk only when everything fits one chunk)
    zchunk = min(zchunk, N)
    tmp = torch.empty((zchunk, N, N, 3), dtype=torch.float64, device="cuda")
    part = torch.empty(L.wl_cuda_turb_partials(zchunk * N * N), dtype=torch.float64, device="cuda")
    sumsq = 0.0

    def fill(z0, nz):
        dims = (ctypes.c_int * 3)(N, N, nz)
        lo = (ctypes.c_int * 3)(0, 0, z0)
        rc = L.wl_cuda_turb_fill(dims, lo, M, d_table.data_ptr(), tmp.data_ptr(), part.data_ptr(), st)
        if rc:
            raise RuntimeError("wl_cuda_turb_fill: cudaError %d" % rc)
        return L.wl_cuda_turb_partials(nz * N * N)

    for z0 in range(0, N, zchunk):
        nz = min(zchunk, N - z0)
        nb = fill(z0, nz)
        sumsq += float(np.sum(part[:nb].cpu().numpy(), dtype=np.float64))
    scale = 1.0 / math.sqrt(sumsq / float(N) ** 3)
    # pass 2: (re)compute each chunk, scale in fp64, round once to fp32
    for z0 in range(0, N, zchunk):
        nz = min(zchunk, N - z0)
        if N > zchunk:
            fill(z0, nz)
        dst = out[0, z0:z0 + nz]
        rc = L.wl_cuda_scale_round(nz * N * N * 3, tmp.data_ptr(), scale, dst.data_ptr(), st)
        if rc:
            raise RuntimeError("wl_cuda_scale_round: cudaError %d" % rc)
    torch.cuda.synchronize()
    del tmp, part
    fld = None
    if host:
        fld = Field((N, N, N), (0.0, 0.0, 0.0), (1.0, 1.0, 1.0), out.cpu().numpy())
    return fld, out


def cut_bricks_cuda(vol, global_dims, brick_grid, ghost=1):
    """Brick cut on the device: vol is a cuda tensor [1,Nz,Ny,Nx,3]; returns one cuda tensor per
    brick (each its own allocation), same boxes as cut_bricks."""
    import torch
    L = _cuda_lib()
    st = ctypes.c_void_p(torch.cuda.current_stream().cuda_stream)
    N = (ctypes.c_int * 3)(*global_dims)
    out = []
    for lo, hi in brick_boxes(global_dims, brick_grid, ghost):
        shp = (hi[2] - lo[2] + 1, hi[1] - lo[1] + 1, hi[0] - lo[0] + 1, 3)
        t = torch.empty(shp, dtype=torch.float32, device="cuda")
        rc = L.wl_cuda_cut_box(vol.data_ptr(), N, (ctypes.c_int * 3)(*lo), (ctypes.c_int * 3)(*hi),
                               t.data_ptr(), st)
        if rc:
            raise RuntimeError("wl_cuda_cut_box: cudaError %d" % rc)
        out.append(t)
    torch.cuda.synchronize()
    return out


# ---- hexahedral meshes (the paper's other field type; input generation only) -------------------
def hexmesh_from_grid(dims, origin, spacing, values=None, jitter=0.0, seed=1, value_fn=None):
    """Re-express a structured grid as hexahedral cells (what the paper's own experiment does with
    its structured data).  Vertices sit at the grid points; `jitter` > 0 displaces the
    interior vertices by up to +-jitter*spacing per axis (uniform, mt19937_64) to make the cells
    general hexahedra.  Values: `values` [Nz,Ny,Nx,3] taken as they are, or value_fn(X) evaluated
    at the (displaced) vertices in fp64 and rounded once.  Returns X [nv,3] f32, V [nv,3] f32,
    H [nc,8] u32 with corner l = dx + 2*dy + 4*dz, and the bounding box (lo, hi)."""
    nx, ny, nz = dims
    z, y, x = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    X = np.stack([origin[0] + x * float(spacing[0]), origin[1] + y * float(spacing[1]),
                  origin[2] + z * float(spacing[2])], axis=-1).astype(np.float64)
    if jitter > 0.0:
        u = uniform(seed, 3 * nx * ny * nz).reshape(nz, ny, nx, 3)
        d = (2.0 * u - 1.0) * jitter * np.asarray(spacing, dtype=np.float64)
        interior = np.zeros((nz, ny, nx, 1), dtype=bool)
        interior[1:-1, 1:-1, 1:-1] = True
        X = X + np.where(interior, d, 0.0)
    Xf = X.reshape(-1, 3).astype(np.float32)
    if value_fn is not None:
        V = np.asarray(value_fn(Xf.astype(np.float64)), dtype=np.float64).astype(np.float32)
    else:
        V = np.ascontiguousarray(values, dtype=np.float32).reshape(-1, 3)
    vid = (z * ny + y) * nx + x
    corners = [vid[dz:nz - 1 + dz, dy:ny - 1 + dy, dx:nx - 1 + dx] for dz in (0, 1) for dy in (0, 1) for dx in (0, 1)]
    H = np.stack(corners, axis=-1).reshape(-1, 8).astype(np.uint32)     # l = dx + 2 dy + 4 dz
    lo = Xf.min(axis=0); hi = Xf.max(axis=0)
    return Xf, V, H, lo, hi
