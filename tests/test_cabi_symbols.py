"""CPU-only: the C-ABI library builds, loads and exports every function include/streami.h
declares; host-only entry points behave (no compute call is made without a GPU)."""
import ctypes
import os
import re

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_functions():
    src = open(os.path.join(ROOT, "include", "streami.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(streami_[a-z_]+)\s*\(", src)))


def test_header_declares_the_boundary():
    names = declared_functions()
    for must in ("streami_field_create", "streami_field_create_bricked", "streami_field_destroy",
                 "streami_trace_streamlines", "streami_trace_streaklines", "streami_brick_advect",
                 "streami_error_string"):
        assert must in names


def test_library_exports_every_declared_symbol():
    import paper_2606_02627_b200 as S
    L = S.lib()
    for name in declared_functions():
        assert hasattr(L, name), name


def test_host_only_entry_points():
    import paper_2606_02627_b200 as S
    L = S.lib()
    assert L.streami_error_string(0) == b"ok"
    assert b"invalid" in L.streami_error_string(-1)
    assert S.streami_get_option("cell_cache") in (0, 1)
    S.streami_set_option("streak_window", 5)
    assert S.streami_get_option("streak_window") == 5
    S.streami_set_option("streak_window", 0)
    assert L.streami_set_option(b"no_such_option", 1) == S.E_INVALID
    # argument validation happens before any CUDA call
    h = ctypes.c_void_p(None)
    assert L.streami_field_create(None, None, None, 1, 1.0, None, 0, ctypes.byref(h)) == S.E_INVALID
    assert L.streami_field_destroy(None) == S.E_INVALID
    assert isinstance(S.streami_launch_count(), int)


def test_product_does_not_import_the_oracle():
    """The product path must not route through oracle/ (or any CPU fallback)."""
    pkg = os.path.join(ROOT, "paper_2606_02627_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                text = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in text and "from oracle" not in text, f
                assert "streami_oracle" not in text and "liboracle" not in text, f


def test_obj_writer(tmp_path):
    """Host-side OBJ writer of assembled lines (no GPU involved)."""
    import torch
    import paper_2606_02627_b200 as S
    off = torch.tensor([0, 2, 2, 3, 6], dtype=torch.int64)
    pts = torch.arange(18, dtype=torch.float32).reshape(6, 3)
    p = tmp_path / "lines.obj"
    S.write_obj(str(p), off, pts)
    rows = p.read_text().splitlines()
    assert rows[0] == "v 0 1 2" and rows[5] == "v 15 16 17"
    assert rows[6:] == ["l 1 2", "l 4 5 6"]          # empty and single-point lines are skipped


def test_argument_validation_without_a_gpu():
    """Host logic of the boundary: every entry point rejects bad arguments with STREAMI_E_INVALID
    before it touches CUDA (so this runs on a CPU-only box), and the option table round-trips."""
    import ctypes
    import paper_2606_02627_b200 as S
    L = S.lib()
    NULL = None
    h = ctypes.c_void_p(None)
    i3 = (ctypes.c_int * 3)(4, 4, 4); f3 = (ctypes.c_float * 3)(0, 0, 0); s3 = (ctypes.c_float * 3)(1, 1, 1)
    bad_sp = (ctypes.c_float * 3)(1, -1, 1)
    dummy = ctypes.c_void_p(16)                                   # never dereferenced on these paths
    assert L.streami_field_create(NULL, f3, s3, 1, 1.0, dummy, 0, ctypes.byref(h)) == S.E_INVALID
    assert L.streami_field_create(i3, f3, bad_sp, 1, 1.0, dummy, 0, ctypes.byref(h)) == S.E_INVALID
    assert L.streami_field_create(i3, f3, s3, 0, 1.0, dummy, 0, ctypes.byref(h)) == S.E_INVALID
    assert L.streami_field_create(i3, f3, s3, 1, 1.0, dummy, 99, ctypes.byref(h)) == S.E_INVALID
    assert L.streami_field_create(i3, f3, s3, 1, 1.0, NULL, 0, ctypes.byref(h)) == S.E_INVALID
    assert L.streami_field_destroy(NULL) == S.E_INVALID
    prm = S.Params()
    assert L.streami_trace_streamlines(NULL, dummy, 8, ctypes.byref(prm), NULL, dummy, NULL) == S.E_INVALID
    assert L.streami_trace_streaklines(NULL, dummy, 8, 8, ctypes.byref(prm), dummy, dummy, NULL) == S.E_INVALID
    assert L.streami_brick_advect(NULL, dummy, 8, ctypes.byref(prm), NULL, dummy, NULL, 0, NULL, 0, NULL, NULL, NULL) == S.E_INVALID
    assert L.streami_streak_begin(NULL, dummy, 8, 8, ctypes.byref(prm), dummy, NULL, ctypes.byref(h)) == S.E_INVALID
    assert L.streami_streak_step(NULL, 1, NULL) == S.E_INVALID
    assert L.streami_streak_end(NULL, NULL, NULL) == S.E_INVALID
    assert L.streami_streamline_lines(dummy, dummy, 8, 0, dummy, NULL, NULL, NULL) == S.E_INVALID   # capacity 0
    assert L.streami_streamline_lines(dummy, dummy, 8, 4, NULL, NULL, NULL, NULL) == S.E_INVALID
    assert L.streami_seed_shape(NULL, f3, f3, f3, 2, 2, 2, 0, 0, dummy, NULL) == S.E_INVALID
    assert L.streami_seed_shape(f3, f3, f3, f3, 2, 2, 2, 7, 0, dummy, NULL) == S.E_INVALID          # unknown mode
    assert L.streami_seed_shape(f3, f3, f3, f3, 0, 2, 2, 0, 0, NULL, NULL) == S.OK                  # no seeds: nothing to do
    assert L.streami_set_option(b"no_such_option", 1) == S.E_INVALID
    for name, v in (("segment_steps", 17), ("prefetch", 2), ("vertex_staging", 0), ("max_blocks_per_sm", 2),
                    ("brick_round_steps", -2), ("presort", 0), ("cell_cache", 0), ("queue_steps", 96),
                    ("streak_window", 12)):
        old = S.streami_get_option(name)
        S.streami_set_option(name, v)
        assert S.streami_get_option(name) == v, name
        S.streami_set_option(name, old)
    assert L.streami_error_string(-4).startswith(b"hand-off log")


def test_mesh_host_helpers(wl=None):
    """streami_mesh_reorder_vtk_hex / streami_mesh_check_hex are host-only: VTK node order -> lattice corner order,
    and the orientation check flags inverted, degenerate and wrongly ordered cells."""
    import numpy as np
    import workloads
    import paper_2606_02627_b200 as S
    X, V, H, lo, hi = workloads.hexmesh_from_grid((5, 4, 3), (0.0, 0.0, 0.0), (1.0, 0.5, 2.0), None, jitter=0.2, seed=3,
                                                  value_fn=lambda P: P)
    assert S.streami_mesh_check_hex(X, H) == (0, -1)
    # the same cells in VTK order: the check sees the wrong order, the reorder restores the library's
    to_vtk = [0, 1, 3, 2, 4, 5, 7, 6]
    H_vtk = H[:, to_vtk]
    bad, first = S.streami_mesh_check_hex(X, H_vtk)
    assert bad == H.shape[0] and first == 0
    assert np.array_equal(S.streami_mesh_reorder_vtk_hex(H_vtk), H)
    # one mirrored cell (x corners swapped) and one degenerate cell
    H2 = H.copy(); H2[7] = H2[7][[1, 0, 3, 2, 5, 4, 7, 6]]; H2[11] = H2[11, 0]
    assert S.streami_mesh_check_hex(X, H2) == (2, 7)
    H3 = H.copy(); H3[2, 5] = X.shape[0] + 5                                # index out of range
    assert S.streami_mesh_check_hex(X, H3) == (1, 2)
