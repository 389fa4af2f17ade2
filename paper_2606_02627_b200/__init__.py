"""Thin Python binding of libstreami_b200.so (C ABI in include/streami.h).

Argument marshalling only: every step of the particle-update path runs in the CUDA kernels of
csrc/.  PyTorch is used for device memory (`torch.empty(..., device="cuda")`) and streams.
There is no CPU fallback: if the library cannot be built/loaded, importing the functions raises.
Function names and argument meaning follow include/streami.h one to one.
"""
import ctypes
import os

import torch

from . import build as _build

HERE = os.path.dirname(os.path.abspath(__file__))

OK, E_INVALID, E_NOMEM, E_CUDA, E_TRUNCATED, E_TOO_LARGE = 0, -1, -2, -3, -4, -5
NOALLOC_MAX_SEEDS = 262144
OUT_OF_DOMAIN, MAX_STEPS, STAGNANT, HALO_MISS = 1, 2, 3, 4
LAYOUT_AUTO, LAYOUT_PACKED3, LAYOUT_FLOAT4, LAYOUT_XPAIR, LAYOUT_CELL, LAYOUT_XYQUAD = 0, 1, 2, 3, 4, 5


class StreamiError(RuntimeError):
    def __init__(self, code, text):
        super().__init__("streami error %d: %s" % (code, text))
        self.code = code


class Params(ctypes.Structure):
    """Mirror of streami_params."""
    _fields_ = [("integrator", ctypes.c_int), ("h", ctypes.c_float), ("h_min", ctypes.c_float),
                ("h_max", ctypes.c_float), ("atol", ctypes.c_float), ("rtol", ctypes.c_float),
                ("max_steps", ctypes.c_uint), ("vmin", ctypes.c_float), ("t0", ctypes.c_float),
                ("time_mode", ctypes.c_int), ("capacity", ctypes.c_uint), ("stride", ctypes.c_uint),
                ("out_steps", ctypes.c_void_p), ("out_status", ctypes.c_void_p),
                ("out_final", ctypes.c_void_p), ("out_totals", ctypes.c_void_p)]


_lib = None


def lib():
    """Load (building in-tree if stale) the CUDA library.  Raises if that is impossible."""
    global _lib
    if _lib is None:
        so = _build.build()
        L = ctypes.CDLL(so)
        P, I, U, F, Z = ctypes.c_void_p, ctypes.c_int, ctypes.c_uint, ctypes.c_float, ctypes.c_size_t
        L.streami_field_create.argtypes = [P, P, P, I, F, P, I, P]
        L.streami_field_create_bricked.argtypes = [P, P, P, P, I, P, I, P]
        L.streami_field_destroy.argtypes = [P]
        L.streami_field_info.argtypes = [P, P, P]
        L.streami_sample.argtypes = [P, P, Z, F, I, P, P, P]
        L.streami_trace_streamlines.argtypes = [P, P, Z, P, P, P, P]
        L.streami_trace_streamlines_host.argtypes = [P, P, Z, P, P, P, P]
        L.streami_trace_streamlines_noalloc.argtypes = [P, P, Z, P, P, P, P]
        L.streami_trace_streaklines.argtypes = [P, P, Z, U, P, P, P, P]
        L.streami_brick_advect.argtypes = [P, P, Z, P, P, P, P, U, P, Z, P, P, P]
        L.streami_partition_seeds.argtypes = [P, P, Z, P, P, P]
        L.streami_trace_streaklines_host.argtypes = [P, P, Z, U, P, P, P, P]
        L.streami_streak_begin.argtypes = [P, P, Z, U, P, P, P, P]
        L.streami_seed_shape.argtypes = [P, P, P, P, U, U, U, I, ctypes.c_ulonglong, P, P]
        L.streami_mesh_create_hex.argtypes = [Z, Z, P, P, P, P, P, P, P]
        L.streami_mesh_destroy.argtypes = [P]
        L.streami_mesh_reorder_vtk_hex.argtypes = [Z, P, P]
        L.streami_mesh_check_hex.argtypes = [Z, Z, P, P, P, P]
        L.streami_mesh_sample.argtypes = [P, P, Z, P, P, P]
        L.streami_mesh_trace_streamlines.argtypes = [P, P, Z, P, P, P, P]
        L.streami_mesh_trace_streamlines_lines_host.argtypes = [P, P, Z, P, P, P, ctypes.c_ulonglong, P, P]
        L.streami_trace_streamlines_lines_host.argtypes = [P, P, Z, P, P, P, ctypes.c_ulonglong, P, P]
        L.streami_streak_step.argtypes = [P, U, P]
        L.streami_streak_position.argtypes = [P, P]
        L.streami_streak_end.argtypes = [P, P, P]
        L.streami_streak_lines.argtypes = [P, P, P, P, P]
        L.streami_streamline_lines.argtypes = [P, P, Z, U, P, P, P, P]
        L.streami_brick_advect_host.argtypes = [P, P, Z, P, P, P, P, U, P, Z, P, P, P]
        L.streami_set_option.argtypes = [ctypes.c_char_p, I]
        L.streami_get_option.argtypes = [ctypes.c_char_p, P]
        L.streami_launch_count.restype = ctypes.c_ulonglong
        L.streami_kernel_time.argtypes = [P, P]
        L.streami_error_string.restype = ctypes.c_char_p
        L.streami_error_string.argtypes = [I]
        _lib = L
    return _lib


def _check(rc, allow=()):
    if rc != OK and rc not in allow:
        raise StreamiError(rc, lib().streami_error_string(rc).decode())
    return rc


def _ptr(t):
    return None if t is None else ctypes.c_void_p(t.data_ptr())


def _stream(stream):
    if stream is None:
        stream = torch.cuda.current_stream()
    return ctypes.c_void_p(stream.cuda_stream)


def _req(t, dtype, name):
    if t is None:
        return
    if not (t.is_cuda and t.dtype == dtype and t.is_contiguous()):
        raise ValueError("%s must be a contiguous CUDA tensor of %s" % (name, dtype))


def params(integrator=0, h=0.01, h_min=0.0, h_max=0.0, atol=0.0, rtol=0.0, max_steps=1000,
           vmin=0.0, t0=0.0, time_mode=0, capacity=1, stride=1, out_steps=None, out_status=None,
           out_final=None, out_totals=None):
    _req(out_steps, torch.int32, "out_steps"); _req(out_status, torch.int32, "out_status")
    _req(out_final, torch.float32, "out_final"); _req(out_totals, torch.int64, "out_totals")
    p = Params(integrator, h, h_min, h_max, atol, rtol, max_steps, vmin, t0, time_mode, capacity,
               stride, None, None, None, None)
    p.out_steps = None if out_steps is None else out_steps.data_ptr()
    p.out_status = None if out_status is None else out_status.data_ptr()
    p.out_final = None if out_final is None else out_final.data_ptr()
    p.out_totals = None if out_totals is None else out_totals.data_ptr()
    p._keep = (out_steps, out_status, out_final, out_totals)
    return p


class Field:
    """Owner of a streami_field handle; keeps the caller's tensors alive (dev_ptr is borrowed)."""

    def __init__(self, handle, keep, bricked):
        self.handle, self._keep, self.bricked = handle, keep, bricked

    def info(self):
        lay, nbytes = ctypes.c_int(0), ctypes.c_size_t(0)
        _check(lib().streami_field_info(self.handle, ctypes.byref(lay), ctypes.byref(nbytes)))
        return lay.value, nbytes.value

    def destroy(self):
        if self.handle:
            lib().streami_field_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


def _i3(v):
    return (ctypes.c_int * 3)(*[int(x) for x in v])


def _f3(v):
    return (ctypes.c_float * 3)(*[float(x) for x in v])


def streami_field_create(dims, origin, spacing, nslices, slice_dt, data, layout_hint=LAYOUT_AUTO):
    """data: CUDA float32 tensor [nslices, Nz, Ny, Nx, 3] (packed, x fastest)."""
    _req(data, torch.float32, "data")
    h = ctypes.c_void_p(None)
    _check(lib().streami_field_create(_i3(dims), _f3(origin), _f3(spacing), int(nslices),
                                      float(slice_dt), _ptr(data), int(layout_hint), ctypes.byref(h)))
    return Field(h, data, False)


def streami_field_create_bricked(global_dims, origin, spacing, brick_grid, ghost_cells, brick_data,
                                 layout_hint=LAYOUT_AUTO):
    """brick_data: list of CUDA float32 tensors, one per brick (flat id order), each the brick's
    stored box [nz, ny, nx, 3]."""
    for t in brick_data:
        _req(t, torch.float32, "brick")
    ptrs = (ctypes.c_void_p * len(brick_data))(*[t.data_ptr() for t in brick_data])
    h = ctypes.c_void_p(None)
    _check(lib().streami_field_create_bricked(_i3(global_dims), _f3(origin), _f3(spacing),
                                              _i3(brick_grid), int(ghost_cells), ptrs,
                                              int(layout_hint), ctypes.byref(h)))
    return Field(h, list(brick_data), True)


def streami_sample(field, points, t=0.0, time_mode=0, stream=None):
    _req(points, torch.float32, "points")
    n = points.shape[0]
    v = torch.empty((n, 3), dtype=torch.float32, device=points.device)
    rc = torch.empty(n, dtype=torch.int32, device=points.device)
    _check(lib().streami_sample(field.handle, _ptr(points), n, float(t), int(time_mode), _ptr(v),
                                _ptr(rc), _stream(stream)))
    return v, rc


def streami_trace_streamlines(field, seeds, prm, out_vertices, out_counts, stream=None):
    _req(seeds, torch.float32, "seeds"); _req(out_vertices, torch.float32, "out_vertices")
    _req(out_counts, torch.int32, "out_counts")
    _check(lib().streami_trace_streamlines(field.handle, _ptr(seeds), seeds.shape[0],
                                           ctypes.byref(prm), _ptr(out_vertices), _ptr(out_counts),
                                           _stream(stream)))


def streami_trace_streamlines_noalloc(field, seeds, prm, out_vertices, out_counts, stream=None):
    """streami_trace_streamlines with all scratch in the library's static device array (no allocation);
    at most NOALLOC_MAX_SEEDS seeds, calls must not overlap on the GPU (include/streami.h)."""
    _req(seeds, torch.float32, "seeds"); _req(out_vertices, torch.float32, "out_vertices")
    _req(out_counts, torch.int32, "out_counts")
    _check(lib().streami_trace_streamlines_noalloc(field.handle, _ptr(seeds), seeds.shape[0],
                                                   ctypes.byref(prm), _ptr(out_vertices), _ptr(out_counts),
                                                   _stream(stream)))


def streami_trace_streamlines_host(field, seeds, prm_host, out_vertices, out_counts, stream=None):
    """Host-buffer variant: seeds/out_* are CPU tensors (pinned for speed); prm_host must carry
    host pointers (or None) in its optional outputs."""
    for t in (seeds, out_vertices, out_counts):
        if t is not None and (t.is_cuda or not t.is_contiguous()):
            raise ValueError("host variant takes contiguous CPU tensors")
    _check(lib().streami_trace_streamlines_host(field.handle, _ptr(seeds), seeds.shape[0],
                                                ctypes.byref(prm_host), _ptr(out_vertices),
                                                _ptr(out_counts), _stream(stream)))


def streami_trace_streaklines(field, points, nsteps, prm, out_vertices, out_counts, stream=None):
    _req(points, torch.float32, "points"); _req(out_vertices, torch.float32, "out_vertices")
    _req(out_counts, torch.int32, "out_counts")
    _check(lib().streami_trace_streaklines(field.handle, _ptr(points), points.shape[0], int(nsteps),
                                           ctypes.byref(prm), _ptr(out_vertices), _ptr(out_counts),
                                           _stream(stream)))


def streami_brick_advect(field, seeds, prm, out_vertices, out_counts, out_round_counts=None,
                         out_handoff_log=None, out_log_count=None, stream=None):
    """Returns (nrounds, truncated)."""
    _req(seeds, torch.float32, "seeds"); _req(out_vertices, torch.float32, "out_vertices")
    _req(out_counts, torch.int32, "out_counts"); _req(out_round_counts, torch.int32, "round_counts")
    _req(out_handoff_log, torch.int64, "handoff_log"); _req(out_log_count, torch.int64, "log_count")
    max_rounds = 0 if out_round_counts is None else out_round_counts.shape[0]
    log_cap = 0 if out_handoff_log is None else out_handoff_log.numel()
    nrounds = ctypes.c_uint(0)
    rc = _check(lib().streami_brick_advect(field.handle, _ptr(seeds), seeds.shape[0],
                                           ctypes.byref(prm), _ptr(out_vertices), _ptr(out_counts),
                                           _ptr(out_round_counts), max_rounds, _ptr(out_handoff_log),
                                           log_cap, _ptr(out_log_count), ctypes.byref(nrounds),
                                           _stream(stream)), allow=(E_TRUNCATED,))
    return nrounds.value, rc == E_TRUNCATED


def streami_partition_seeds(field, seeds, nbricks, stream=None):
    """(perm [n] int32 cuda, offsets [nbricks+1] int64 cuda): seeds ordered by (owner brick, Morton code)."""
    _req(seeds, torch.float32, "seeds")
    n = seeds.shape[0]
    perm = torch.empty(n, dtype=torch.int32, device="cuda")
    off = torch.empty(nbricks + 1, dtype=torch.int64, device="cuda")
    _check(lib().streami_partition_seeds(field.handle, _ptr(seeds), n, _ptr(perm), _ptr(off), _stream(stream)))
    return perm, off


class Streak:
    """Step-synchronous streaklines (streami_streak_begin/_step/_lines/_end)."""

    def __init__(self, field, points, nsteps, prm, out_vertices, stream=None):
        _req(points, torch.float32, "points"); _req(out_vertices, torch.float32, "out_vertices")
        self._keep = (field, points, prm, out_vertices)
        self.m, self.nsteps = points.shape[0], int(nsteps)
        self.handle = ctypes.c_void_p(None)
        _check(lib().streami_streak_begin(field.handle, _ptr(points), self.m, self.nsteps, ctypes.byref(prm),
                                          _ptr(out_vertices), _stream(stream), ctypes.byref(self.handle)))

    def step(self, k=1, stream=None):
        _check(lib().streami_streak_step(self.handle, int(k), _stream(stream)))

    def position(self):
        s = ctypes.c_uint(0)
        _check(lib().streami_streak_position(self.handle, ctypes.byref(s)))
        return s.value

    def lines(self, stream=None):
        """(offsets [m+1] int64 cuda, points [total, 3] float32 cuda) of the current snapshot."""
        off = torch.empty(self.m + 1, dtype=torch.int64, device="cuda")
        total = ctypes.c_ulonglong(0)
        _check(lib().streami_streak_lines(self.handle, _ptr(off), None, ctypes.byref(total), _stream(stream)))
        pts = torch.empty((total.value, 3), dtype=torch.float32, device="cuda")
        _check(lib().streami_streak_lines(self.handle, _ptr(off), _ptr(pts), None, _stream(stream)))
        return off, pts

    def end(self, out_counts=None, stream=None):
        _req(out_counts, torch.int32, "out_counts")
        if self.handle:
            _check(lib().streami_streak_end(self.handle, _ptr(out_counts), _stream(stream)))
            self.handle = None


def streami_streamline_lines(vertices, counts, stream=None):
    """Polylines of a streamline result: (offsets [n+1] int64 cuda, points [total, 3] float32 cuda)."""
    _req(vertices, torch.float32, "vertices"); _req(counts, torch.int32, "counts")
    n, cap = counts.shape[0], vertices.shape[2]
    off = torch.empty(n + 1, dtype=torch.int64, device="cuda")
    total = ctypes.c_ulonglong(0)
    _check(lib().streami_streamline_lines(_ptr(vertices), _ptr(counts), n, cap, _ptr(off), None,
                                          ctypes.byref(total), _stream(stream)))
    pts = torch.empty((total.value, 3), dtype=torch.float32, device="cuda")
    _check(lib().streami_streamline_lines(_ptr(vertices), _ptr(counts), n, cap, _ptr(off), _ptr(pts), None,
                                          _stream(stream)))
    return off, pts


def streami_seed_shape(origin, edge_u, edge_v=(0, 0, 0), edge_w=(0, 0, 0), nu=1, nv=1, nw=1, mode=0,
                       rng_seed=0, stream=None):
    """Seeds on a line / plane / box; returns a CUDA float32 tensor [nu*nv*nw, 3]."""
    out = torch.empty((nu * nv * nw, 3), dtype=torch.float32, device="cuda")
    _check(lib().streami_seed_shape(_f3(origin), _f3(edge_u), _f3(edge_v), _f3(edge_w), nu, nv, nw, int(mode),
                                    int(rng_seed), _ptr(out), _stream(stream)))
    return out


def _lines_host(fn, handle, seeds, prm_host, out_offsets, out_points, stream):
    for t, nm in ((seeds, "seeds"), (out_offsets, "out_offsets"), (out_points, "out_points")):
        if t is not None and (t.is_cuda or not t.is_contiguous()):
            raise ValueError("%s: contiguous CPU tensor expected" % nm)
    total = ctypes.c_ulonglong(0)
    rc = _check(fn(handle, _ptr(seeds), seeds.shape[0], ctypes.byref(prm_host), _ptr(out_offsets),
                   _ptr(out_points), out_points.shape[0], ctypes.byref(total), _stream(stream)),
                allow=(E_TRUNCATED,))
    return total.value, rc == E_TRUNCATED


def streami_trace_streamlines_lines_host(field, seeds, prm_host, out_offsets, out_points, stream=None):
    """Host seeds in, host polylines out (offsets int64 [n+1], points float32 [max_points, 3]).
    Returns (total_points, truncated)."""
    return _lines_host(lib().streami_trace_streamlines_lines_host, field.handle, seeds, prm_host, out_offsets,
                       out_points, stream)


def streami_mesh_trace_streamlines_lines_host(mesh, seeds, prm_host, out_offsets, out_points, stream=None):
    """The same on a hexahedral mesh."""
    return _lines_host(lib().streami_mesh_trace_streamlines_lines_host, mesh.handle, seeds, prm_host, out_offsets,
                       out_points, stream)


def streami_mesh_reorder_vtk_hex(H_vtk):
    """[nc][8] uint32 in VTK_HEXAHEDRON node order -> the library's corner order (numpy, host)."""
    import numpy as np
    H = np.ascontiguousarray(H_vtk, dtype=np.uint32)
    out = np.empty_like(H)
    _check(lib().streami_mesh_reorder_vtk_hex(H.shape[0], H.ctypes.data, out.ctypes.data))
    return out


def streami_mesh_check_hex(X, H):
    """(number of cells with a non-positive centre Jacobian or a bad vertex index, first such cell or -1)."""
    import numpy as np
    X = np.ascontiguousarray(X, dtype=np.float32); H = np.ascontiguousarray(H, dtype=np.uint32)
    bad = ctypes.c_ulonglong(0); first = ctypes.c_longlong(-1)
    _check(lib().streami_mesh_check_hex(X.shape[0], H.shape[0], X.ctypes.data, H.ctypes.data, ctypes.byref(bad), ctypes.byref(first)))
    return bad.value, first.value


class Mesh:
    """Owner of a streami_mesh handle (hexahedral mesh field)."""

    def __init__(self, X, V, H, lo, hi, nb):
        import numpy as np
        X = np.ascontiguousarray(X, dtype=np.float32); V = np.ascontiguousarray(V, dtype=np.float32)
        H = np.ascontiguousarray(H, dtype=np.uint32)
        self.handle = ctypes.c_void_p(None)
        _check(lib().streami_mesh_create_hex(X.shape[0], H.shape[0], X.ctypes.data, V.ctypes.data, H.ctypes.data,
                                             _f3(lo), _f3(hi), _i3(nb), ctypes.byref(self.handle)))

    def destroy(self):
        if self.handle:
            lib().streami_mesh_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


def streami_mesh_sample(mesh, points, stream=None):
    _req(points, torch.float32, "points")
    n = points.shape[0]
    v = torch.empty((n, 3), dtype=torch.float32, device="cuda")
    cell = torch.empty(n, dtype=torch.int64, device="cuda")
    _check(lib().streami_mesh_sample(mesh.handle, _ptr(points), n, _ptr(v), _ptr(cell), _stream(stream)))
    return v, cell


def streami_mesh_trace_streamlines(mesh, seeds, prm, out_vertices, out_counts, stream=None):
    _req(seeds, torch.float32, "seeds"); _req(out_vertices, torch.float32, "out_vertices")
    _req(out_counts, torch.int32, "out_counts")
    _check(lib().streami_mesh_trace_streamlines(mesh.handle, _ptr(seeds), seeds.shape[0], ctypes.byref(prm),
                                                _ptr(out_vertices), _ptr(out_counts), _stream(stream)))


def _host(t, name):
    if t is not None and (t.is_cuda or not t.is_contiguous()):
        raise ValueError("%s: the host variants take contiguous CPU tensors" % name)


def streami_trace_streaklines_host(field, points, nsteps, prm_host, out_vertices, out_counts, stream=None):
    """Host-buffer variant; prm_host carries host pointers (or None) in its optional outputs."""
    for t, nm in ((points, "points"), (out_vertices, "out_vertices"), (out_counts, "out_counts")):
        _host(t, nm)
    _check(lib().streami_trace_streaklines_host(field.handle, _ptr(points), points.shape[0], int(nsteps),
                                                ctypes.byref(prm_host), _ptr(out_vertices),
                                                _ptr(out_counts), _stream(stream)))


def streami_brick_advect_host(field, seeds, prm_host, out_vertices, out_counts, out_round_counts=None,
                              out_handoff_log=None, out_log_count=None, stream=None):
    """Host-buffer variant.  Returns (nrounds, truncated)."""
    for t, nm in ((seeds, "seeds"), (out_vertices, "out_vertices"), (out_counts, "out_counts"),
                  (out_round_counts, "round_counts"), (out_handoff_log, "log"), (out_log_count, "log_count")):
        _host(t, nm)
    max_rounds = 0 if out_round_counts is None else out_round_counts.shape[0]
    log_cap = 0 if out_handoff_log is None else out_handoff_log.numel()
    nrounds = ctypes.c_uint(0)
    rc = _check(lib().streami_brick_advect_host(field.handle, _ptr(seeds), seeds.shape[0],
                                                ctypes.byref(prm_host), _ptr(out_vertices),
                                                _ptr(out_counts), _ptr(out_round_counts), max_rounds,
                                                _ptr(out_handoff_log), log_cap, _ptr(out_log_count),
                                                ctypes.byref(nrounds), _stream(stream)),
                allow=(E_TRUNCATED,))
    return nrounds.value, rc == E_TRUNCATED


def streami_set_option(name, value):
    _check(lib().streami_set_option(name.encode(), int(value)))


def streami_get_option(name):
    v = ctypes.c_int(0)
    _check(lib().streami_get_option(name.encode(), ctypes.byref(v)))
    return v.value


def streami_launch_count():
    return lib().streami_launch_count()


def streami_kernel_time():
    """(total_ms, launches) of the advection-kernel launches since the last call (option
    "kernel_timing" must be 1)."""
    ms, cnt = ctypes.c_float(0.0), ctypes.c_uint(0)
    _check(lib().streami_kernel_time(ctypes.byref(ms), ctypes.byref(cnt)))
    return ms.value, cnt.value


def write_obj(path, offsets, points):
    """Write assembled polylines as a Wavefront OBJ file (the paper hands its lines to a renderer or
    an OBJ file): one `v x y z` per point, one `l i j k ...` per line with at least two
    points (1-based indices).  offsets/points as returned by the *_lines calls (any device)."""
    off = offsets.detach().cpu().tolist()
    pts = points.detach().cpu().tolist()
    with open(path, "w") as f:
        for x, y, z in pts:
            f.write("v %.9g %.9g %.9g\n" % (x, y, z))
        for a, b in zip(off[:-1], off[1:]):
            if b - a >= 2:
                f.write("l " + " ".join(str(k + 1) for k in range(a, b)) + "\n")
