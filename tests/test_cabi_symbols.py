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
