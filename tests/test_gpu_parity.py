"""GPU parity tests: the CUDA path (through the C ABI binding) against the fp32 oracle, element by
element, on the same seeded inputs.  Bar (BASELINE.json north_star): integer outputs bit-exact;
vertex positions within 1e-4 cell over the first 200 steps.  The design goal is stronger
(both sides execute the same IEEE operations in the same order), so these
tests assert BIT equality of every float as well; the tolerance form is kept in
test_gpu_tolerance_form for the record.
"""
import numpy as np
import pytest

from helpers import assert_same, gpu_field, gpu_streamlines

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def S():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("gpu tests need a CUDA device")
    import paper_2606_02627_b200 as S_
    S_.lib()
    return S_


@pytest.fixture(scope="module")
def torch():
    import torch as t
    return t


LAYOUTS = [1, 2, 3, 4, 5, 6, 7]


# ---- a2-a4: the sampling layer alone -------------------------------------------------------
@pytest.mark.parametrize("layout", LAYOUTS)
def test_sample_steady(S, torch, oracle, wl, layout):
    fld = wl.turb_field_cpu(24, 32, 1, 5)
    rng = np.random.default_rng(0)
    pts = (rng.random((50001, 3)) * 25.0 - 1.0).astype(np.float32)      # some outside
    pts[:8] = [[0, 0, 0], [23, 23, 23], [23, 0, 11.5], [np.nan, 1, 1], [22.999998, 5, 5],
               [-0.0, 3, 3], [5, 23.000002, 5], [7, 7, 7]]
    g = oracle.grid(fld.data, fld.dims, fld.origin, fld.spacing)
    v_ref, rc_ref = oracle.sample(g, pts, 0.0, "f32")
    f = gpu_field(S, torch, fld, layout)
    v, rc = S.streami_sample(f, torch.from_numpy(pts).cuda())
    assert np.array_equal(rc.cpu().numpy().astype(np.uint32), rc_ref)
    assert np.array_equal(v.cpu().numpy().view(np.uint32), v_ref.view(np.uint32))
    assert 0.05 < np.mean(rc_ref != 0) < 0.5


@pytest.mark.parametrize("layout", LAYOUTS)
@pytest.mark.parametrize("time_mode", [0, 1])
def test_sample_unsteady(S, torch, oracle, wl, layout, time_mode):
    fld = wl.double_gyre_field(dims=(40, 20, 12), nslices=9, dt=0.25)
    rng = np.random.default_rng(1)
    pts = (rng.random((20000, 3)) * [2.1, 1.05, 1.05] - 0.02).astype(np.float32)
    f = gpu_field(S, torch, fld, layout)
    for t in (-1.0, 0.0, 0.1, 0.25, 1.3700001, 2.0, 7.5):
        g = oracle.grid(fld.data, fld.dims, fld.origin, fld.spacing, fld.nslices, fld.slice_dt,
                        time_mode)
        v_ref, rc_ref = oracle.sample(g, pts, t, "f32")
        v, rc = S.streami_sample(f, torch.from_numpy(pts).cuda(), t, time_mode)
        assert np.array_equal(rc.cpu().numpy().astype(np.uint32), rc_ref)
        assert np.array_equal(v.cpu().numpy().view(np.uint32), v_ref.view(np.uint32)), t


# ---- config 1: ABC 32^3, 1,024 seeds, RK4 h = 0.01, 1,000 steps, every vertex ----------------
@pytest.mark.parametrize("layout", LAYOUTS)
@pytest.mark.parametrize("cache", [0, 1])
def test_c1_abc_full(S, torch, oracle, wl, layout, cache):
    fld = wl.abc_field(32)
    seeds = wl.seeds_uniform(42, 1024, [2 * np.pi] * 3)
    kw = dict(integrator=0, h=0.01, max_steps=1000, vmin=1e-6, capacity=1001, stride=1)
    ref = oracle.streamlines(oracle.grid(fld.data, fld.dims, fld.origin, fld.spacing), seeds,
                             oracle.params(**kw), "f32")
    S.streami_set_option("cell_cache", cache)
    try:
        out = gpu_streamlines(S, torch, gpu_field(S, torch, fld, layout), seeds, **kw)
    finally:
        S.streami_set_option("cell_cache", 1)
    assert_same(out, ref, "C1")


# ---- turbulence, several tiles and a ragged tail, RK4 ----------------------------------------
@pytest.fixture(scope="module")
def turb48(wl):
    return wl.turb_field_cpu(48, 64, 1, 12)


@pytest.mark.parametrize("layout", LAYOUTS)
def test_turbulence_rk4(S, torch, oracle, wl, turb48, layout):
    n = 20011
    seeds = wl.seeds_uniform(42, n, [47.0] * 3)
    seeds[5] = [48.0, 1, 1]; seeds[6] = [np.nan, 1, 1]; seeds[7] = [47.0, 47.0, 47.0]
    kw = dict(integrator=0, h=0.25, max_steps=400, vmin=1e-6, capacity=401, stride=1)
    ref = oracle.streamlines(oracle.grid(turb48.data, turb48.dims, turb48.origin, turb48.spacing),
                             seeds, oracle.params(**kw), "f32")
    out = gpu_streamlines(S, torch, gpu_field(S, torch, turb48, layout), seeds, **kw)
    assert_same(out, ref, "turb48")
    hist = np.bincount(ref.status, minlength=5)
    assert hist[1] > 100 and hist[2] > 100            # both endings occur


def test_presort_and_stride(S, torch, oracle, wl, turb48):
    """n >= 65536 switches the Morton presort on; results are indexed by id so nothing changes.
    stride/capacity recording (A6); slots beyond the count stay untouched."""
    n = 70001
    seeds = wl.seeds_uniform(7, n, [47.0] * 3)
    kw = dict(integrator=0, h=0.25, max_steps=150, vmin=1e-6, capacity=9, stride=7)
    ref = oracle.streamlines(oracle.grid(turb48.data, turb48.dims, turb48.origin, turb48.spacing),
                             seeds, oracle.params(**kw), "f32")
    f = gpu_field(S, torch, turb48)
    for presort in (1, 0):
        S.streami_set_option("presort", presort)
        try:
            out = gpu_streamlines(S, torch, f, seeds, **kw)
        finally:
            S.streami_set_option("presort", 1)
        assert_same(out, ref, "presort=%d" % presort)
    out = gpu_streamlines(S, torch, f, seeds, record=False, **kw)     # out_vertices = NULL
    assert_same(out, ref, "no vertices")


# ---- DP5(4) (config 5's integrator) ----------------------------------------------------------
@pytest.mark.parametrize("layout", LAYOUTS)
@pytest.mark.parametrize("cache", [0, 1])
def test_turbulence_dp5(S, torch, oracle, wl, turb48, layout, cache):
    n = 6007
    seeds = wl.seeds_uniform(43, n, [47.0] * 3)
    kw = dict(integrator=1, h=0.25, h_min=0.01, h_max=1.0, atol=1e-5, rtol=1e-5, max_steps=300,
              vmin=1e-6, capacity=201, stride=1)
    ref = oracle.streamlines(oracle.grid(turb48.data, turb48.dims, turb48.origin, turb48.spacing),
                             seeds, oracle.params(**kw), "f32")
    S.streami_set_option("cell_cache", cache)
    try:
        out = gpu_streamlines(S, torch, gpu_field(S, torch, turb48, layout), seeds, **kw)
    finally:
        S.streami_set_option("cell_cache", 1)
    assert_same(out, ref, "dp5")
    assert ref.totals[0] > ref.totals[1]              # rejections happened


def test_dp5_forced_floor_and_tight_tolerance(S, torch, oracle, wl, turb48):
    seeds = wl.seeds_uniform(44, 3001, [47.0] * 3)
    f = gpu_field(S, torch, turb48)
    g = oracle.grid(turb48.data, turb48.dims, turb48.origin, turb48.spacing)
    for kw in (dict(integrator=1, h=0.5, h_min=0.5, h_max=0.5, atol=1e-9, rtol=0.0, max_steps=60,
                    vmin=0.0, capacity=61),
               dict(integrator=1, h=1.0, h_min=1e-4, h_max=4.0, atol=1e-7, rtol=1e-7, max_steps=120,
                    vmin=1e-6, capacity=16, stride=8)):
        ref = oracle.streamlines(g, seeds, oracle.params(**kw), "f32")
        assert_same(gpu_streamlines(S, torch, f, seeds, **kw), ref, str(kw))


# ---- unsteady streamlines (pathlines through slices) -----------------------------------------
@pytest.mark.parametrize("cache", [1, 0])
@pytest.mark.parametrize("layout", LAYOUTS)
@pytest.mark.parametrize("integrator", [0, 1])
def test_unsteady_pathlines(S, torch, oracle, wl, layout, integrator, cache):
    """cache = the two-slice register copy of the current cell (option "cell_cache"), on and off."""
    fld = wl.double_gyre_field(dims=(64, 32, 16), nslices=12, dt=0.25)
    seeds = wl.seeds_uniform(5, 4099, [2.0, 1.0, 1.0])
    kw = dict(integrator=integrator, h=0.05, h_min=0.001, h_max=0.5, atol=1e-6, rtol=1e-6,
              max_steps=150, vmin=1e-7, t0=0.3, capacity=151)
    for time_mode in (0, 1):
        g = oracle.grid(fld.data, fld.dims, fld.origin, fld.spacing, fld.nslices, fld.slice_dt,
                        time_mode)
        ref = oracle.streamlines(g, seeds, oracle.params(**kw), "f32")
        S.streami_set_option("cell_cache", cache)
        try:
            out = gpu_streamlines(S, torch, gpu_field(S, torch, fld, layout), seeds, time_mode=time_mode,
                                  **kw)
        finally:
            S.streami_set_option("cell_cache", 1)
        assert_same(out, ref, "unsteady tm=%d cache=%d" % (time_mode, cache))


# ---- edge cases ------------------------------------------------------------------------------
def test_edge_cases(S, torch, oracle, wl, turb48):
    f = gpu_field(S, torch, turb48)
    g = oracle.grid(turb48.data, turb48.dims, turb48.origin, turb48.spacing)
    # empty input
    out = gpu_streamlines(S, torch, f, np.zeros((0, 3), dtype=np.float32), h=0.25, max_steps=5)
    assert out["counts"].size == 0 and out["totals"].sum() == 0
    # every seed outside; a single seed; max_steps = 0; stagnation floor above every speed
    for seeds, kw in [
        (np.full((37, 3), -5.0, dtype=np.float32), dict(h=0.25, max_steps=5, capacity=2)),
        (np.array([[10.5, 11.5, 12.5]], dtype=np.float32), dict(h=0.25, max_steps=33, capacity=40)),
        (wl.seeds_uniform(1, 100, [47.0] * 3), dict(h=0.25, max_steps=0, capacity=3)),
        (wl.seeds_uniform(1, 100, [47.0] * 3), dict(h=0.25, max_steps=9, vmin=1e3, capacity=3)),
        (wl.seeds_uniform(1, 100, [47.0] * 3), dict(h=60.0, max_steps=9, capacity=3)),
    ]:
        ref = oracle.streamlines(g, seeds, oracle.params(**kw), "f32")
        assert_same(gpu_streamlines(S, torch, f, seeds, **kw), ref, str(kw))


def test_error_codes(S, torch, wl, turb48):
    f = gpu_field(S, torch, turb48)
    seeds = torch.zeros((4, 3), device="cuda")
    counts = torch.zeros(4, dtype=torch.int32, device="cuda")
    for bad in (dict(h=0.0), dict(h=float("nan")), dict(capacity=0), dict(stride=0),
                dict(integrator=2), dict(integrator=1, h_min=1.0, h_max=0.5, atol=1e-5),
                dict(time_mode=3)):
        kw = dict(h=0.25, max_steps=5); kw.update(bad)
        with pytest.raises(S.StreamiError) as e:
            S.streami_trace_streamlines(f, seeds, S.params(**kw), None, counts)
        assert e.value.code == S.E_INVALID
    data = torch.zeros((1, 4, 4, 4, 3), device="cuda")
    for dims, sp, nsl, lay in [((1, 4, 4), (1, 1, 1), 1, 0), ((4, 4, 4), (0, 1, 1), 1, 0),
                               ((4, 4, 4), (1, 1, 1), 0, 0), ((4, 4, 4), (1, 1, 1), 1, 9)]:
        with pytest.raises(S.StreamiError) as e:
            S.streami_field_create(dims, (0, 0, 0), sp, nsl, 1.0, data, lay)
        assert e.value.code == S.E_INVALID
    with pytest.raises(S.StreamiError):           # streamlines on a bricked field is invalid
        bf = S.streami_field_create_bricked((4, 4, 4), (0, 0, 0), (1, 1, 1), (1, 1, 1), 1, [data[0]])
        S.streami_trace_streamlines(bf, seeds, S.params(h=0.25), None, counts)


def test_host_buffer_variant(S, torch, oracle, wl, turb48):
    n = 5003
    seeds = wl.seeds_uniform(9, n, [47.0] * 3)
    kw = dict(integrator=0, h=0.25, max_steps=100, vmin=1e-6, capacity=26, stride=4)
    ref = oracle.streamlines(oracle.grid(turb48.data, turb48.dims, turb48.origin, turb48.spacing),
                             seeds, oracle.params(**kw), "f32")
    f = gpu_field(S, torch, turb48)
    h_seeds = torch.from_numpy(seeds).pin_memory()
    verts = torch.empty((3, n, 26), dtype=torch.float32).pin_memory()
    counts = torch.empty(n, dtype=torch.int32).pin_memory()
    steps = torch.empty(n, dtype=torch.int32); status = torch.empty(n, dtype=torch.int32)
    final = torch.empty((3, n), dtype=torch.float32); totals = torch.empty(4, dtype=torch.int64)
    prm = S.params(**kw)
    prm.out_steps, prm.out_status = steps.data_ptr(), status.data_ptr()
    prm.out_final, prm.out_totals = final.data_ptr(), totals.data_ptr()
    S.streami_trace_streamlines_host(f, h_seeds, prm, verts, counts)
    assert np.array_equal(counts.numpy().astype(np.uint32), ref.counts)
    assert np.array_equal(steps.numpy().astype(np.uint32), ref.steps)
    assert np.array_equal(status.numpy().astype(np.uint32), ref.status)
    assert np.array_equal(final.numpy(), ref.final)
    assert np.array_equal(totals.numpy().astype(np.uint64)[:3], ref.totals[:3])
    v = verts.numpy()
    for i in range(0, n, 97):
        c = ref.counts[i]
        assert np.array_equal(v[:, i, :c], ref.vertices[:, i, :c])


def test_gpu_tolerance_form(S, torch, oracle, wl, turb48):
    """The north_star bar as stated: |dx| <= 1e-4 cell over the first 200 steps, integers exact."""
    seeds = wl.seeds_uniform(11, 8000, [47.0] * 3)
    kw = dict(integrator=0, h=0.25, max_steps=400, vmin=1e-6, capacity=201, stride=1)
    ref = oracle.streamlines(oracle.grid(turb48.data, turb48.dims, turb48.origin, turb48.spacing),
                             seeds, oracle.params(**kw), "f32")
    out = gpu_streamlines(S, torch, gpu_field(S, torch, turb48), seeds, **kw)
    assert np.array_equal(out["steps"], ref.steps) and np.array_equal(out["status"], ref.status)
    d = np.abs(np.nan_to_num(out["vertices"]) - np.nan_to_num(ref.vertices))
    assert d.max() <= 1e-4                       # spacing is 1: world units are cell widths
