"""streami_trace_streamlines_noalloc: the streamline trace with all scratch in the library's static device
array (no cudaMalloc: for callers under graph capture or in serving loops).  Collected last on purpose (the
suite runs with pytest -x).  The new entry point is compared with the existing, allocating path bit for bit
(the tolerance of every GPU test in this repository: both run the same kernels) on two calls in a row that
share the array: 100,000 RK4 seeds (the presort lives in the array), then 70,000 DP5(4) seeds."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def S():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("gpu tests need a CUDA device")
    import paper_2606_02627_b200 as S_
    S_.lib()
    return S_


def _trace(S, torch, call, field, d_seeds, kw):
    n, cap = d_seeds.shape[0], kw["capacity"]
    out = dict(verts=torch.full((3, n, cap), float("nan"), dtype=torch.float32, device="cuda"),
               counts=torch.full((n,), -1, dtype=torch.int32, device="cuda"),
               steps=torch.full((n,), -1, dtype=torch.int32, device="cuda"),
               status=torch.full((n,), -1, dtype=torch.int32, device="cuda"),
               final=torch.zeros((3, n), dtype=torch.float32, device="cuda"),
               totals=torch.zeros(4, dtype=torch.int64, device="cuda"))
    prm = S.params(out_steps=out["steps"], out_status=out["status"], out_final=out["final"], out_totals=out["totals"], **kw)
    call(field, d_seeds, prm, out["verts"], out["counts"])
    return out


def _same(torch, a, b, what):
    for k in ("counts", "steps", "status", "totals"):
        assert bool((a[k] == b[k]).all()), what + " " + k
    for k in ("final", "verts"):                            # bit patterns (NaN = untouched slot on both sides)
        assert bool((a[k].view(torch.int32) == b[k].view(torch.int32)).all()), what + " " + k


def test_noalloc_equals_allocating_path_two_calls_in_a_row(S, wl):
    import torch
    from helpers import gpu_field
    fld = wl.turb_field_cpu(48, 64, 1, 12)
    field = gpu_field(S, torch, fld, 0)
    rk4 = dict(integrator=0, h=0.25, max_steps=300, vmin=1e-6, capacity=40, stride=8)
    dp5 = dict(integrator=1, h=0.25, h_min=0.01, h_max=1.0, atol=1e-5, rtol=1e-5, max_steps=200, vmin=1e-6,
               capacity=16, stride=16)
    s1 = wl.seeds_uniform(5, 100000, [47.0] * 3); s1[::7, 0] += 60.0      # some seeds start outside the domain
    s2 = wl.seeds_uniform(6, 70000, [47.0] * 3)
    d1, d2 = torch.from_numpy(s1).cuda(), torch.from_numpy(s2).cuda()
    # the existing path
    ref1 = _trace(S, torch, S.streami_trace_streamlines, field, d1, rk4)
    ref2 = _trace(S, torch, S.streami_trace_streamlines, field, d2, dp5)
    # the first call on a device resolves the array's address (and loads its module): not part of the check below
    _trace(S, torch, S.streami_trace_streamlines_noalloc, field, d2[:64].contiguous(), rk4)
    torch.cuda.synchronize()
    # two calls in a row on one stream, sharing the array (the second finds the first one's contents in it)
    out1 = _trace(S, torch, S.streami_trace_streamlines_noalloc, field, d1, rk4)
    out2 = _trace(S, torch, S.streami_trace_streamlines_noalloc, field, d2, dp5)
    torch.cuda.synchronize()
    _same(torch, out1, ref1, "noalloc call 1 (RK4, presorted)")
    _same(torch, out2, ref2, "noalloc call 2 (DP5(4))")
    assert int(out1["totals"][0]) > 10 * 100000 and int((out1["status"] == 1).sum()) > 100000 // 7
    # and a third call, sizes swapped, still matches (stale presort data of call 1 in the array)
    out3 = _trace(S, torch, S.streami_trace_streamlines_noalloc, field, d2, rk4)
    ref3 = _trace(S, torch, S.streami_trace_streamlines, field, d2, rk4)
    torch.cuda.synchronize()
    _same(torch, out3, ref3, "noalloc call 3")


def test_noalloc_rejects_sizes_beyond_the_static_scratch(S, wl):
    import torch
    from helpers import gpu_field
    fld = wl.turb_field_cpu(16, 8, 1, 4)
    field = gpu_field(S, torch, fld, 0)
    n = S.NOALLOC_MAX_SEEDS + 1
    seeds = torch.zeros((n, 3), dtype=torch.float32, device="cuda")
    counts = torch.full((n,), -7, dtype=torch.int32, device="cuda")
    prm = S.params(integrator=0, h=0.25, max_steps=10, vmin=0.0, capacity=1, stride=1)
    with pytest.raises(S.StreamiError) as e:
        S.streami_trace_streamlines_noalloc(field, seeds, prm, None, counts)
    assert e.value.code == S.E_TOO_LARGE and "262,144" in str(e.value)
    torch.cuda.synchronize()
    assert bool((counts == -7).all())                       # nothing was enqueued
    # exactly the maximum is accepted
    ok = seeds[:S.NOALLOC_MAX_SEEDS].contiguous() + 3.0
    c2 = torch.full((S.NOALLOC_MAX_SEEDS,), -7, dtype=torch.int32, device="cuda")
    S.streami_trace_streamlines_noalloc(field, ok, prm, None, c2)
    torch.cuda.synchronize()
    assert bool((c2 >= 0).all())                            # every count was written


def test_noalloc_source_calls_no_allocator():
    """The entry point's translation unit names no allocating CUDA call outside comments."""
    import os
    import re
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    src = open(os.path.join(root, "paper_2606_02627_b200", "csrc", "api_noalloc.cu")).read()
    code = re.sub(r"//[^\n]*", "", src)
    for word in ("cudaMalloc", "cudaFree", "cudaEventCreate", "cudaStreamCreate", "cudaHostAlloc", "new ", "std::vector"):
        assert word not in code, word
    assert "cudaGetSymbolAddress" in code and "__device__ __align__(256)" in code
