"""Schedule-only options must not change any result: segments with Morton re-sort of the survivors
(`segment_steps`), the one-step-ahead cell prefetch (`prefetch`), the staged vertex writer
(`vertex_staging`), the occupancy limit (`max_blocks_per_sm`), the integer domain test
(`integer_accept`), the continuation queue consumed by the same launch (`queue_steps`).  Each combination is compared bit for
bit with the oracle (RK4 and DP5(4), every layout family), with capacities that are and are not a
multiple of the 8-slot staging group, and with a stride that cuts groups at segment boundaries."""
import numpy as np
import pytest

from helpers import assert_same, gpu_field, gpu_streamlines

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def torch():
    import torch as t
    if not t.cuda.is_available():
        pytest.skip("no CUDA device")
    return t


@pytest.fixture(scope="module")
def S(torch):
    import paper_2606_02627_b200 as s
    s.lib()
    return s


@pytest.fixture(scope="module")
def turb48(wl):
    return wl.turb_field_cpu(48, 64, 1, 12)


DEFAULTS = dict(segment_steps=0, prefetch=3, vertex_staging=1, max_blocks_per_sm=0, presort=1, queue_steps=0)


def _with(S, opts, fn):
    try:
        for k, v in opts.items():
            S.streami_set_option(k, v)
        return fn()
    finally:
        for k, v in DEFAULTS.items():
            S.streami_set_option(k, v)


@pytest.mark.parametrize("layout", [1, 3, 4, 5])
@pytest.mark.parametrize("opts", [dict(segment_steps=16), dict(segment_steps=37, prefetch=0),
                                  dict(vertex_staging=0), dict(prefetch=2, max_blocks_per_sm=1), dict(prefetch=1), dict(prefetch=4),
                                  dict(segment_steps=5, vertex_staging=0, presort=1),
                                  dict(queue_steps=16), dict(queue_steps=7, vertex_staging=0),
                                  dict(queue_steps=50, prefetch=0, max_blocks_per_sm=1)])
def test_rk4_schedule_options(S, torch, oracle, wl, turb48, layout, opts):
    n = 70001                                      # >= 65536: sorting and segments are active
    seeds = wl.seeds_uniform(11, n, [47.0] * 3)
    g = oracle.grid(turb48.data, turb48.dims, turb48.origin, turb48.spacing)
    f = gpu_field(S, torch, turb48, layout)
    for kw in (dict(integrator=0, h=0.25, max_steps=150, vmin=1e-6, capacity=24, stride=3),
               dict(integrator=0, h=0.25, max_steps=120, vmin=1e-6, capacity=13, stride=1)):
        ref = oracle.streamlines(g, seeds, oracle.params(**kw), "f32")
        out = _with(S, opts, lambda: gpu_streamlines(S, torch, f, seeds, **kw))
        assert_same(out, ref, "rk4 %s %s" % (opts, kw))


@pytest.mark.parametrize("n", [1, 37, 5000])
@pytest.mark.parametrize("q", [1, 10, 64])
def test_continuation_queue_small_launches(S, torch, oracle, wl, turb48, n, q):
    """`queue_steps` with fewer particles than lanes (most warps only ever poll), seeds outside the
    domain (terminated before their first step) and particles that are queued at step max_steps."""
    seeds = wl.seeds_uniform(13, n, [47.0] * 3)
    seeds[::5, 0] += 60.0                           # every fifth seed starts outside
    g = oracle.grid(turb48.data, turb48.dims, turb48.origin, turb48.spacing)
    f = gpu_field(S, torch, turb48, 5)
    kw = dict(integrator=0, h=0.25, max_steps=128, vmin=1e-6, capacity=40, stride=4)
    ref = oracle.streamlines(g, seeds, oracle.params(**kw), "f32")
    out = _with(S, dict(queue_steps=q), lambda: gpu_streamlines(S, torch, f, seeds, **kw))
    assert_same(out, ref, "queue n=%d q=%d" % (n, q))


@pytest.mark.parametrize("layout", [3, 4])
@pytest.mark.parametrize("opts", [dict(segment_steps=8), dict(segment_steps=25, vertex_staging=0),
                                  dict(max_blocks_per_sm=2)])
def test_dp5_schedule_options(S, torch, oracle, wl, turb48, layout, opts):
    """DP5(4): a segment cut carries t and h and recomputes the FSAL k1; rejected attempts spend
    budget but a cut waits for the next accepted step."""
    n = 66000
    seeds = wl.seeds_uniform(12, n, [47.0] * 3)
    g = oracle.grid(turb48.data, turb48.dims, turb48.origin, turb48.spacing)
    f = gpu_field(S, torch, turb48, layout)
    kw = dict(integrator=1, h=0.25, h_min=0.01, h_max=1.0, atol=1e-5, rtol=1e-5, max_steps=90,
              vmin=1e-6, capacity=16, stride=2)
    ref = oracle.streamlines(g, seeds, oracle.params(**kw), "f32")
    out = _with(S, opts, lambda: gpu_streamlines(S, torch, f, seeds, **kw))
    assert_same(out, ref, "dp5 %s" % opts)
    assert int(ref.totals[0]) > int(ref.totals[1]), "the case must contain rejected attempts"


def test_unaligned_vertex_array_uses_scalar_stores(S, torch, oracle, wl, turb48):
    """The full-sector vertex stores need a 32-byte aligned out_vertices and capacity % 8 == 0; an
    array that starts 4 bytes off must take the scalar path and give the same vertices."""
    n, cap = 4099, 24
    seeds = wl.seeds_uniform(13, n, [47.0] * 3)
    kw = dict(integrator=0, h=0.25, max_steps=100, vmin=1e-6, capacity=cap, stride=2)
    ref = oracle.streamlines(oracle.grid(turb48.data, turb48.dims, turb48.origin, turb48.spacing),
                             seeds, oracle.params(**kw), "f32")
    f = gpu_field(S, torch, turb48)
    flat = torch.full((3 * n * cap + 8,), float("nan"), dtype=torch.float32, device="cuda")
    for shift in (0, 1):
        verts = flat[shift:shift + 3 * n * cap].view(3, n, cap)
        assert verts.data_ptr() % 32 == 4 * shift and verts.is_contiguous()
        counts = torch.zeros(n, dtype=torch.int32, device="cuda")
        flat.fill_(float("nan"))
        S.streami_trace_streamlines(f, torch.from_numpy(seeds).cuda(), S.params(**kw), verts, counts)
        torch.cuda.synchronize()
        assert np.array_equal(counts.cpu().numpy().astype(np.uint32), ref.counts)
        assert np.array_equal(verts.cpu().numpy().view(np.uint32), ref.vertices.view(np.uint32)), shift


@pytest.mark.parametrize("layout", [1, 3, 5])
@pytest.mark.parametrize("kind", ["tame", "nan", "inf", "huge", "big_tame"])
def test_integer_accept_keeps_the_domain_test_exact(S, torch, oracle, wl, turb48, layout, kind):
    """`integer_accept` decides "inside" from floor(g) when every field value is finite and <= 2^60;
    a field with NaN, infinite or larger values must take the float test (the library finds out at
    create time).  Seeds sit on the faces g = 0 and g = N-1 as well; a step of 1e30 sends stage
    points to +-inf.  All of it is compared bit for bit with the oracle, option on and off."""
    import dataclasses
    data = turb48.data.copy()
    rng = np.random.default_rng(5)
    idx = rng.integers(0, 48, size=(400, 3))
    if kind == "nan":
        data[0, idx[:, 2], idx[:, 1], idx[:, 0], idx[:, 0] % 3] = np.nan
    elif kind == "inf":
        data[0, idx[:, 2], idx[:, 1], idx[:, 0], idx[:, 0] % 3] = np.where(idx[:, 1] % 2, np.inf, -np.inf)
    elif kind == "huge":
        data[0, idx[:, 2], idx[:, 1], idx[:, 0], idx[:, 0] % 3] = np.where(idx[:, 1] % 2, 3e38, -3e38)
    elif kind == "big_tame":
        data[0, idx[:, 2], idx[:, 1], idx[:, 0], idx[:, 0] % 3] = np.where(idx[:, 1] % 2, 1e18, -1e18)
    fld = dataclasses.replace(turb48, data=data)
    n = 6000
    seeds = wl.seeds_uniform(21, n, [47.0] * 3)
    seeds[:600] = np.round(seeds[:600])                     # on vertices, many on the faces 0 and 47
    seeds[600:900, 0] = 47.0; seeds[900:1200, 1] = 0.0; seeds[1200:1500, 2] = 47.0
    seeds[1500:1700] = idx[:200] + 0.5                      # next to the planted values
    g = oracle.grid(fld.data, fld.dims, fld.origin, fld.spacing)
    f = gpu_field(S, torch, fld, layout)
    for kw in (dict(integrator=0, h=0.25, max_steps=80, vmin=1e-6, capacity=16, stride=5),
               dict(integrator=0, h=1e30, max_steps=3, vmin=0.0, capacity=4, stride=1),
               dict(integrator=1, h=0.25, h_min=0.01, h_max=1.0, atol=1e-4, rtol=1e-4, max_steps=60, vmin=1e-6,
                    capacity=16, stride=5)):
        ref = oracle.streamlines(g, seeds, oracle.params(**kw), "f32")
        assert kw["h"] > 1.0 or len(set(ref.status.tolist())) >= 2       # (RK4, RK4 with stage points at +-inf, DP5(4))
        for on in (1, 0):
            try:
                S.streami_set_option("integer_accept", on)
                out = gpu_streamlines(S, torch, f, seeds, **kw)
            finally:
                S.streami_set_option("integer_accept", 1)
            assert_same(out, ref, "%s integer_accept=%d %s" % (kind, on, kw))


def test_packed3_array_poisoned_after_create(S, torch, oracle, wl, turb48):
    """PACKED3 traces the caller's BORROWED array in place (the in-situ use).  If the application
    writes NaN / Inf into it AFTER streami_field_create, the create-time scan is stale: the integer accept
    must not be licensed for that layout, or a NaN position would be judged inside and run to MAX_STEPS
    (ADVICE r1).  The trace of the poisoned array must equal the oracle's on the same poisoned bytes."""
    data = turb48.data.copy()
    dev = torch.from_numpy(data).cuda()
    f = S.streami_field_create(turb48.dims, turb48.origin, turb48.spacing, 1, 1.0, dev, 1)
    rng = np.random.default_rng(9)
    idx = rng.integers(0, 48, size=(600, 3))
    data[0, idx[:, 2], idx[:, 1], idx[:, 0], idx[:, 0] % 3] = np.where(idx[:, 1] % 2, np.nan, np.inf)
    dev.copy_(torch.from_numpy(data))                              # the application overwrites its own array
    n = 6000
    seeds = wl.seeds_uniform(33, n, [47.0] * 3)
    seeds[:400] = idx[:400] + 0.5
    g = oracle.grid(data, turb48.dims, turb48.origin, turb48.spacing)
    for kw in (dict(integrator=0, h=0.25, max_steps=80, vmin=1e-6, capacity=16, stride=5),
               dict(integrator=1, h=0.25, h_min=0.01, h_max=1.0, atol=1e-4, rtol=1e-4, max_steps=60, vmin=1e-6,
                    capacity=16, stride=5)):
        ref = oracle.streamlines(g, seeds, oracle.params(**kw), "f32")
        assert np.count_nonzero(ref.status == oracle.OUT_OF_DOMAIN) > 400
        out = gpu_streamlines(S, torch, f, seeds, **kw)
        assert_same(out, ref, "poisoned packed3 %s" % kw)
