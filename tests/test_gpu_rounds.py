"""GPU parity for the two round loops: streaklines (A7) and brick advection with hand-off (A9)."""
import numpy as np
import pytest

from helpers import gpu_field

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


def gpu_streaklines(S, torch, field, pts, nsteps, **kw):
    m = pts.shape[0]
    d_pts = torch.from_numpy(np.ascontiguousarray(pts, dtype=np.float32)).cuda()
    verts = torch.full((3, nsteps, m), float("nan"), dtype=torch.float32, device="cuda")
    counts = torch.full((m,), -1, dtype=torch.int32, device="cuda")
    steps = torch.full((nsteps * m,), -1, dtype=torch.int32, device="cuda")
    status = torch.full((nsteps * m,), -1, dtype=torch.int32, device="cuda")
    totals = torch.zeros(4, dtype=torch.int64, device="cuda")
    prm = S.params(out_steps=steps, out_status=status, out_totals=totals, **kw)
    S.streami_trace_streaklines(field, d_pts, nsteps, prm, verts, counts)
    torch.cuda.synchronize()
    return (verts.cpu().numpy(), counts.cpu().numpy().astype(np.uint32),
            steps.cpu().numpy().astype(np.uint32), status.cpu().numpy().astype(np.uint32),
            totals.cpu().numpy().astype(np.uint64))


@pytest.mark.parametrize("cache", [1, 0])
@pytest.mark.parametrize("layout", [1, 2, 3, 4, 5])
@pytest.mark.parametrize("window", [0, 1, 7])
def test_streaklines_double_gyre(S, torch, oracle, wl, layout, window, cache):
    """A scaled-down config 4: double gyre slices, rake + a few points that leave or start outside.
    cache = the two-slice register copy of the current cell (option "cell_cache"), on and off."""
    fld = wl.double_gyre_field(dims=(64, 32, 16), nslices=10, dt=0.25)
    pts = wl.rake_c4(16, 8)
    pts = np.concatenate([pts, np.array([[2.5, 0.5, 0.5], [1.999, 0.5, 0.999], [0.001, 0.999, 0.001]],
                                        dtype=np.float32)])
    nsteps = 90                               # t up to 4.5 > last slice time 2.25: frozen field (Q10)
    kw = dict(integrator=0, h=0.05, vmin=0.0, t0=0.0)
    g = oracle.grid(fld.data, fld.dims, fld.origin, fld.spacing, fld.nslices, fld.slice_dt)
    ref = oracle.streaklines(g, pts, nsteps, oracle.params(**kw), "f32")
    S.streami_set_option("streak_window", window)
    S.streami_set_option("cell_cache", cache)
    try:
        v, counts, steps, status, totals = gpu_streaklines(S, torch, gpu_field(S, torch, fld, layout),
                                                           pts, nsteps, **kw)
    finally:
        S.streami_set_option("streak_window", 0)
        S.streami_set_option("cell_cache", 1)
    assert np.array_equal(status, ref.status) and np.array_equal(steps, ref.steps)
    assert np.array_equal(counts, ref.counts)
    assert np.array_equal(v.view(np.uint32), ref.vertices.view(np.uint32))
    assert np.array_equal(totals[:3], ref.totals[:3])
    assert np.count_nonzero(ref.status == 1) >= nsteps       # the outside point, every release


@pytest.mark.parametrize("cache", [1, 0])
@pytest.mark.parametrize("layout", [3, 5])
def test_streaklines_hold_floor_slice(S, torch, oracle, wl, layout, cache):
    """The paper's own time handling (fields[(int)simTime]; time_mode = 1) through
    the streakline kernel, with and without the register copy of the cell, two window lengths."""
    fld = wl.double_gyre_field(dims=(64, 32, 16), nslices=10, dt=0.25)
    pts = np.concatenate([wl.rake_c4(16, 8), np.array([[2.5, 0.5, 0.5], [1.999, 0.5, 0.999]], dtype=np.float32)])
    nsteps = 70
    kw = dict(integrator=0, h=0.05, vmin=0.0, t0=0.0)
    g = oracle.grid(fld.data, fld.dims, fld.origin, fld.spacing, fld.nslices, fld.slice_dt, 1)
    ref = oracle.streaklines(g, pts, nsteps, oracle.params(**kw), "f32")
    kw["time_mode"] = 1
    S.streami_set_option("cell_cache", cache)
    try:
        for window in (0, 9):
            S.streami_set_option("streak_window", window)
            v, counts, steps, status, totals = gpu_streaklines(S, torch, gpu_field(S, torch, fld, layout),
                                                               pts, nsteps, **kw)
            assert np.array_equal(status, ref.status) and np.array_equal(steps, ref.steps)
            assert np.array_equal(counts, ref.counts)
            assert np.array_equal(v.view(np.uint32), ref.vertices.view(np.uint32))
            assert np.array_equal(totals[:3], ref.totals[:3])
    finally:
        S.streami_set_option("streak_window", 0)
        S.streami_set_option("cell_cache", 1)


def test_streaklines_steady_field_with_deaths(S, torch, oracle, wl):
    fld = wl.turb_field_cpu(32, 48, 1, 6)
    pts = wl.seeds_uniform(3, 300, [31.0] * 3)
    nsteps = 120
    kw = dict(integrator=0, h=0.25, vmin=1e-6, t0=0.0)
    ref = oracle.streaklines(oracle.grid(fld.data, fld.dims, fld.origin, fld.spacing), pts, nsteps,
                             oracle.params(**kw), "f32")
    for window, cache in ((0, 1), (16, 1), (0, 0), (16, 0)):
        S.streami_set_option("streak_window", window)
        S.streami_set_option("cell_cache", cache)
        try:
            v, counts, steps, status, totals = gpu_streaklines(S, torch, gpu_field(S, torch, fld), pts,
                                                               nsteps, **kw)
        finally:
            S.streami_set_option("streak_window", 0)
            S.streami_set_option("cell_cache", 1)
        assert np.array_equal(status, ref.status) and np.array_equal(steps, ref.steps)
        assert np.array_equal(counts, ref.counts)
        assert np.array_equal(v.view(np.uint32), ref.vertices.view(np.uint32))
        assert np.array_equal(totals[:3], ref.totals[:3])
    assert np.count_nonzero(ref.status == 1) > 100 and np.count_nonzero(ref.status == 2) > 100


def gpu_bricks(S, torch, wl, fld, nb, seeds, ghost=1, layout=0, max_rounds=64, log_cap=None, **kw):
    arrays = [torch.from_numpy(a).cuda() for a in wl.cut_bricks(fld, nb, ghost)]
    f = S.streami_field_create_bricked(fld.dims, fld.origin, fld.spacing, nb, ghost, arrays, layout)
    n = seeds.shape[0]
    cap = kw.get("capacity", 1)
    nbricks = nb[0] * nb[1] * nb[2]
    d_seeds = torch.from_numpy(np.ascontiguousarray(seeds, dtype=np.float32)).cuda()
    verts = torch.full((3, n, cap), float("nan"), dtype=torch.float32, device="cuda")
    counts = torch.full((n,), -1, dtype=torch.int32, device="cuda")
    steps = torch.full((n,), -1, dtype=torch.int32, device="cuda")
    status = torch.full((n,), -1, dtype=torch.int32, device="cuda")
    final = torch.zeros((3, n), dtype=torch.float32, device="cuda")
    totals = torch.zeros(4, dtype=torch.int64, device="cuda")
    rcounts = torch.full((max_rounds, nbricks), -1, dtype=torch.int32, device="cuda")
    log = torch.zeros(64 * n + 16 if log_cap is None else log_cap, dtype=torch.int64, device="cuda")
    logc = torch.zeros(1, dtype=torch.int64, device="cuda")
    prm = S.params(out_steps=steps, out_status=status, out_final=final, out_totals=totals, **kw)
    nrounds, truncated = S.streami_brick_advect(f, d_seeds, prm, verts, counts, rcounts, log, logc)
    torch.cuda.synchronize()
    nlog = int(logc.item())
    return dict(vertices=verts.cpu().numpy(), counts=counts.cpu().numpy().astype(np.uint32),
                steps=steps.cpu().numpy().astype(np.uint32),
                status=status.cpu().numpy().astype(np.uint32), final=final.cpu().numpy(),
                totals=totals.cpu().numpy().astype(np.uint64), nrounds=nrounds, truncated=truncated,
                round_counts=rcounts.cpu().numpy(), nlog=nlog,
                log=np.sort(log.cpu().numpy().view(np.uint64)[:min(nlog, log.numel())]))


@pytest.mark.parametrize("nb,N,layout", [((2, 2, 2), 32, 3), ((2, 2, 2), 32, 1), ((3, 2, 1), 31, 2),
                                         ((1, 1, 1), 24, 3), ((2, 2, 2), 32, 4), ((3, 2, 1), 31, 4)])
def test_bricks_vs_oracle_and_monolithic(S, torch, oracle, wl, nb, N, layout):
    fld = wl.turb_field_cpu(N, 48, 1, 6)
    n = 30011
    seeds = wl.seeds_uniform(42, n, [N - 1.0] * 3)
    seeds[3] = [-1, 2, 2]; seeds[4] = [N - 1.0] * 3
    kw = dict(integrator=0, h=0.25, max_steps=400, vmin=1e-6, capacity=101, stride=4)
    boxes = wl.brick_boxes(fld.dims, nb, 1)
    bricks = [oracle.grid(a, None, fld.origin, fld.spacing, gdims=fld.dims, lo=lo, hi=hi)
              for a, (lo, hi) in zip(wl.cut_bricks(fld, nb, 1), boxes)]
    ref = oracle.brick_advect(bricks, nb, seeds, oracle.params(**kw), "f32")
    out = gpu_bricks(S, torch, wl, fld, nb, seeds, layout=layout, **kw)
    assert not out["truncated"]
    for key in ("status", "steps", "counts"):
        assert np.array_equal(out[key], getattr(ref, key)), key
    assert np.array_equal(out["final"].view(np.uint32), ref.final.view(np.uint32))
    assert np.array_equal(out["vertices"].view(np.uint32), ref.vertices.view(np.uint32))
    assert np.array_equal(out["totals"], ref.totals)
    # queue membership: rounds, per-round per-brick counts, sorted hand-off log -- bit exact
    assert out["nrounds"] == ref.nrounds and out["nlog"] == ref.nlog
    assert np.array_equal(out["round_counts"][:ref.nrounds].astype(np.uint32),
                          ref.round_counts[:ref.nrounds])
    assert np.array_equal(out["log"], ref.log)
    assert np.count_nonzero(ref.status == 4) == 0
    if nb != (1, 1, 1):
        assert ref.nrounds >= 3 and ref.nlog > n // 10
    # P9 on the GPU: the brick-wise trace equals the monolithic GPU trace bit for bit
    from helpers import gpu_streamlines
    mono = gpu_streamlines(S, torch, gpu_field(S, torch, fld, layout), seeds, **kw)
    for key in ("status", "steps", "counts"):
        assert np.array_equal(out[key], mono[key]), key
    assert np.array_equal(out["vertices"].view(np.uint32), mono["vertices"].view(np.uint32))


def test_bricks_halo_miss_and_truncation(S, torch, oracle, wl):
    N, nb = 9, (2, 1, 1)
    fast = np.zeros((1, N, N, N, 3), dtype=np.float32); fast[..., 0] = 3.0
    fld = wl.Field((N, N, N), (0, 0, 0), (1, 1, 1), fast)
    seeds = np.array([[3.5, 4, 4], [4.0, 4, 4], [2.0, 4, 4]], dtype=np.float32)
    kw = dict(integrator=0, h=1.0, max_steps=50, vmin=0.0, capacity=51)
    out = gpu_bricks(S, torch, wl, fld, nb, seeds, **kw)
    assert list(out["status"]) == [4, 1, 4]
    # slow field: ping-pong free straight lines; tiny log and round table overflow -> TRUNCATED
    slow = fast.copy(); slow[..., 0] = 1.0
    fld = wl.Field((N, N, N), (0, 0, 0), (1, 1, 1), slow)
    out = gpu_bricks(S, torch, wl, fld, nb, seeds, max_rounds=1, log_cap=1, **kw)
    assert out["truncated"] and out["nlog"] == 2 and out["nrounds"] == 2
    assert list(out["steps"]) == [4, 4, 6] and list(out["status"]) == [1, 1, 1]
    assert list(out["round_counts"][0]) == [2, 1]
    # nothing inside: zero rounds
    out = gpu_bricks(S, torch, wl, fld, nb, np.full((5, 3), 99.0, dtype=np.float32), **kw)
    assert out["nrounds"] == 0 and list(out["status"]) == [1] * 5 and out["nlog"] == 0


@pytest.mark.parametrize("mode", [-2, 0])
@pytest.mark.parametrize("nb,N,layout,q", [((2, 2, 2), 32, 5, 0), ((3, 2, 1), 31, 3, 0), ((2, 2, 2), 32, 5, 9),
                                           ((1, 1, 1), 24, 5, 0), ((2, 2, 2), 32, 1, 40)])
def test_bricks_one_launch_ring(S, torch, oracle, wl, nb, N, layout, q, mode):
    """Option brick_round_steps = -2: hand-offs (and, with queue_steps = q > 0, step budgets) go through
    a device ring consumed by the same launch; no rounds.  brick_round_steps = 0 without a round table
    or a log (what bench.py times): budgeted rounds, and the stragglers (< n/16 left) finished by one
    ring launch.  Per-particle results and the number of hand-offs equal the oracle's (A9: they do not
    depend on the round structure)."""
    fld = wl.turb_field_cpu(N, 48, 1, 6)
    n = 30011
    seeds = wl.seeds_uniform(42, n, [N - 1.0] * 3)
    seeds[3] = [-1, 2, 2]; seeds[4] = [N - 1.0] * 3
    kw = dict(integrator=0, h=0.25, max_steps=400, vmin=1e-6, capacity=101, stride=4)
    boxes = wl.brick_boxes(fld.dims, nb, 1)
    bricks = [oracle.grid(a, None, fld.origin, fld.spacing, gdims=fld.dims, lo=lo, hi=hi)
              for a, (lo, hi) in zip(wl.cut_bricks(fld, nb, 1), boxes)]
    ref = oracle.brick_advect(bricks, nb, seeds, oracle.params(**kw), "f32")
    arrays = [torch.from_numpy(a).cuda() for a in wl.cut_bricks(fld, nb, 1)]
    f = S.streami_field_create_bricked(fld.dims, fld.origin, fld.spacing, nb, 1, arrays, layout)
    d_seeds = torch.from_numpy(seeds).cuda()
    verts = torch.full((3, n, 101), float("nan"), dtype=torch.float32, device="cuda")
    counts = torch.full((n,), -1, dtype=torch.int32, device="cuda")
    steps = torch.full((n,), -1, dtype=torch.int32, device="cuda")
    status = torch.full((n,), -1, dtype=torch.int32, device="cuda")
    final = torch.zeros((3, n), dtype=torch.float32, device="cuda")
    totals = torch.zeros(4, dtype=torch.int64, device="cuda")
    prm = S.params(out_steps=steps, out_status=status, out_final=final, out_totals=totals, **kw)
    S.streami_set_option("brick_round_steps", mode)
    S.streami_set_option("queue_steps", q)
    try:
        nrounds, truncated = S.streami_brick_advect(f, d_seeds, prm, verts, counts)
        torch.cuda.synchronize()
    finally:
        S.streami_set_option("brick_round_steps", 0)
        S.streami_set_option("queue_steps", 0)
    assert (nrounds == 1 if mode == -2 else nrounds >= 1) and not truncated
    assert np.array_equal(status.cpu().numpy().astype(np.uint32), ref.status)
    assert np.array_equal(steps.cpu().numpy().astype(np.uint32), ref.steps)
    assert np.array_equal(counts.cpu().numpy().astype(np.uint32), ref.counts)
    assert np.array_equal(final.cpu().numpy().view(np.uint32), ref.final.view(np.uint32))
    assert np.array_equal(verts.cpu().numpy().view(np.uint32), ref.vertices.view(np.uint32))
    assert np.array_equal(totals.cpu().numpy().astype(np.uint64), ref.totals)


@pytest.mark.parametrize("nb,N", [((2, 2, 2), 32), ((3, 2, 1), 31), ((1, 1, 1), 24), ((4, 3, 2), 50)])
def test_partition_seeds_per_destination_segments(S, torch, oracle, wl, nb, N):
    """a9 / A9: the two-level counting sort (destination brick, Morton code inside the brick) that orders every
    round's work.  Through streami_partition_seeds: segment b of the permutation holds exactly the seeds the
    oracle's Q_0[b] holds (owner of the seed, A9), every seed once, segments contiguous and in brick order."""
    fld = wl.turb_field_cpu(N, 24, 1, 4)
    n = 70001
    seeds = wl.seeds_uniform(5, n, [N - 1.0] * 3)
    seeds[:50] = np.round(seeds[:50])                       # on vertices: faces belong to the upper brick
    nbricks = nb[0] * nb[1] * nb[2]
    arrays = [torch.from_numpy(a).cuda() for a in wl.cut_bricks(fld, nb, 1)]
    f = S.streami_field_create_bricked(fld.dims, fld.origin, fld.spacing, nb, 1, arrays, 3)
    perm, off = S.streami_partition_seeds(f, torch.from_numpy(seeds).cuda(), nbricks)
    torch.cuda.synchronize()
    perm = perm.cpu().numpy().astype(np.int64); off = off.cpu().numpy().astype(np.int64)
    assert off[0] == 0 and off[-1] == n and np.all(np.diff(off) >= 0)
    assert np.array_equal(np.sort(perm), np.arange(n))      # a permutation
    B = [N // nb[a] for a in range(3)]
    own = sum(np.minimum(np.floor(seeds[:, a]).astype(int) // B[a], nb[a] - 1) * [1, nb[0], nb[0] * nb[1]][a] for a in range(3))
    for b in range(nbricks):
        seg = perm[off[b]:off[b + 1]]
        assert np.all(own[seg] == b), b
    # the oracle's Q_0 sizes (round table, row 0)
    boxes = wl.brick_boxes(fld.dims, nb, 1)
    bricks = [oracle.grid(a, None, fld.origin, fld.spacing, gdims=fld.dims, lo=lo, hi=hi)
              for a, (lo, hi) in zip(wl.cut_bricks(fld, nb, 1), boxes)]
    ref = oracle.brick_advect(bricks, nb, seeds, oracle.params(0, h=0.25, max_steps=1, vmin=0.0, capacity=2), "f32")
    assert np.array_equal(np.diff(off), ref.round_counts[0])


_RING_STRESS = {}


@pytest.mark.parametrize("q", [1, 2, 3, 4])
def test_ring_stress_many_passes(S, torch, oracle, wl, q):
    """Stress test of the in-kernel hand-off ring (release / acquire publication, trace_kernel.cuh): one launch,
    every particle re-queued every q steps, so the ring of 2^19 records is passed through several hundred times
    (tags run to several hundred) while all SMs publish and claim at once; repeated 20 times, every per-particle
    output bit-compared with the oracle each time.  A torn or lost record would show as a wrong step count or
    position, a lapped ring or a stalled launch as an error return."""
    N, nb, n = 48, (2, 2, 2), 1 << 18
    # rigid rotation about the vertical axis through the centre (speed 1 at the rim) plus a slow vertical drift that
    # reverses at mid height: particles circle through the four brick columns until max_steps, so the work is long
    # and every particle changes brick again and again
    c = (N - 1) / 2.0
    z, y, x = np.meshgrid(np.arange(N), np.arange(N), np.arange(N), indexing="ij")
    data = np.zeros((1, N, N, N, 3), dtype=np.float32)
    data[0, ..., 0] = -(y - c) / c; data[0, ..., 1] = (x - c) / c; data[0, ..., 2] = 0.05 * np.sin(2 * np.pi * z / (N - 1))
    fld = wl.Field((N, N, N), (0.0, 0.0, 0.0), (1.0, 1.0, 1.0), data)
    seeds = wl.seeds_uniform(7, n, [N - 1.0] * 3)
    kw = dict(integrator=0, h=0.25, max_steps=1600, vmin=1e-6, capacity=16, stride=128)
    boxes = wl.brick_boxes(fld.dims, nb, 1)
    bricks = [oracle.grid(a, None, fld.origin, fld.spacing, gdims=fld.dims, lo=lo, hi=hi)
              for a, (lo, hi) in zip(wl.cut_bricks(fld, nb, 1), boxes)]
    if "ref" not in _RING_STRESS:
        _RING_STRESS["ref"] = oracle.brick_advect(bricks, nb, seeds, oracle.params(**kw), "f32")
    ref = _RING_STRESS["ref"]
    assert int(ref.totals[1]) // q > 100 * (1 << 19)            # the ring of 2^19 records is lapped hundreds of times
    assert int(ref.totals[3]) > 4 * n                           # and real hand-offs are plentiful
    arrays = [torch.from_numpy(a).cuda() for a in wl.cut_bricks(fld, nb, 1)]
    f = S.streami_field_create_bricked(fld.dims, fld.origin, fld.spacing, nb, 1, arrays, 0)
    d_seeds = torch.from_numpy(seeds).cuda()
    S.streami_set_option("brick_round_steps", -2)
    S.streami_set_option("queue_steps", q)
    try:
        for rep in range(20):
            verts = torch.full((3, n, 16), float("nan"), dtype=torch.float32, device="cuda")
            counts = torch.full((n,), -1, dtype=torch.int32, device="cuda")
            steps = torch.full((n,), -1, dtype=torch.int32, device="cuda")
            status = torch.full((n,), -1, dtype=torch.int32, device="cuda")
            final = torch.zeros((3, n), dtype=torch.float32, device="cuda")
            totals = torch.zeros(4, dtype=torch.int64, device="cuda")
            prm = S.params(out_steps=steps, out_status=status, out_final=final, out_totals=totals, **kw)
            nrounds, truncated = S.streami_brick_advect(f, d_seeds, prm, verts, counts)
            torch.cuda.synchronize()
            assert nrounds == 1 and not truncated
            assert np.array_equal(status.cpu().numpy().astype(np.uint32), ref.status), rep
            assert np.array_equal(steps.cpu().numpy().astype(np.uint32), ref.steps), rep
            assert np.array_equal(counts.cpu().numpy().astype(np.uint32), ref.counts), rep
            assert np.array_equal(final.cpu().numpy().view(np.uint32), ref.final.view(np.uint32)), rep
            assert np.array_equal(verts.cpu().numpy().view(np.uint32), ref.vertices.view(np.uint32)), rep
            assert np.array_equal(totals.cpu().numpy().astype(np.uint64)[:3], ref.totals[:3]), rep
    finally:
        S.streami_set_option("brick_round_steps", 0)
        S.streami_set_option("queue_steps", 0)


@pytest.mark.parametrize("k", [1, 7])
def test_bricks_paper_step_rounds(S, torch, oracle, wl, k):
    """the paper's schedule (every particle re-queued after every RK step,
    PAPER.md:96-101, 142-144) via option brick_round_steps.  Trajectories, statuses, step counts and
    the set of brick changes do not depend on the round structure (A9); the round table counts
    every queued particle and the rounds equal the steps of the longest-lived particle."""
    N, nb = 32, (2, 2, 2)
    fld = wl.turb_field_cpu(N, 48, 1, 6)
    n = 9001
    seeds = wl.seeds_uniform(5, n, [N - 1.0] * 3)
    kw = dict(integrator=0, h=0.25, max_steps=60, vmin=1e-6, capacity=61, stride=1)
    boxes = wl.brick_boxes(fld.dims, nb, 1)
    bricks = [oracle.grid(a, None, fld.origin, fld.spacing, gdims=fld.dims, lo=lo, hi=hi)
              for a, (lo, hi) in zip(wl.cut_bricks(fld, nb, 1), boxes)]
    ref = oracle.brick_advect(bricks, nb, seeds, oracle.params(**kw), "f32")
    S.streami_set_option("brick_round_steps", k)
    try:
        out = gpu_bricks(S, torch, wl, fld, nb, seeds, max_rounds=128, **kw)
    finally:
        S.streami_set_option("brick_round_steps", 0)
    assert not out["truncated"]
    for key in ("status", "steps", "counts"):
        assert np.array_equal(out[key], getattr(ref, key)), key
    assert np.array_equal(out["final"].view(np.uint32), ref.final.view(np.uint32))
    assert np.array_equal(out["vertices"].view(np.uint32), ref.vertices.view(np.uint32))
    assert np.array_equal(out["totals"], ref.totals)
    strip = lambda log: np.sort(log & np.uint64((1 << 48) - 1))          # (dest, id) without the round
    assert np.array_equal(strip(out["log"]), strip(ref.log))
    assert out["nrounds"] >= int(ref.steps.max()) // k
    rc = out["round_counts"]
    if k == 1:       # one step per round: round r holds exactly the particles that completed r steps
        assert out["nrounds"] == int(ref.steps.max()) + 1
        for r in (1, 2, 3, 30):
            assert int(rc[r].sum()) == np.count_nonzero(ref.steps >= r), r


def test_host_buffer_variants_of_streaklines_and_bricks(S, torch, oracle, wl):
    """streami_trace_streaklines_host / streami_brick_advect_host: the same results with every
    buffer in (pinned or pageable) host memory."""
    import ctypes
    # streaklines on a small double gyre
    fld = wl.double_gyre_field(dims=(32, 16, 8), nslices=6, dt=0.25)
    pts = wl.rake_c4(8, 8)
    ns = 40
    g = oracle.grid(fld.data, fld.dims, fld.origin, fld.spacing, fld.nslices, fld.slice_dt)
    ref = oracle.streaklines(g, pts, ns, oracle.params(integrator=0, h=0.05, vmin=1e-6, max_steps=ns), "f32")
    f = gpu_field(S, torch, fld)
    m = pts.shape[0]
    h_pts = torch.from_numpy(pts.copy()).pin_memory()
    h_v = torch.zeros((3, ns, m), dtype=torch.float32).pin_memory()
    h_c = torch.zeros(m, dtype=torch.int32)
    h_st = torch.zeros(ns * m, dtype=torch.int32)
    prm = S.params(integrator=0, h=0.05, vmin=1e-6)
    prm.out_status = h_st.data_ptr()
    S.streami_trace_streaklines_host(f, h_pts, ns, prm, h_v, h_c)
    assert np.array_equal(h_v.numpy().view(np.uint32), ref.vertices.view(np.uint32))
    assert np.array_equal(h_c.numpy().astype(np.uint32), ref.counts)
    assert np.array_equal(h_st.numpy().astype(np.uint32), ref.status)
    # bricks
    N, nb = 24, (2, 1, 2)
    fld = wl.turb_field_cpu(N, 32, 1, 5)
    n = 3000
    seeds = wl.seeds_uniform(9, n, [N - 1.0] * 3)
    kw = dict(integrator=0, h=0.25, max_steps=120, vmin=1e-6, capacity=16, stride=8)
    boxes = wl.brick_boxes(fld.dims, nb, 1)
    cut = wl.cut_bricks(fld, nb, 1)
    bricks = [oracle.grid(a, None, fld.origin, fld.spacing, gdims=fld.dims, lo=lo, hi=hi) for a, (lo, hi) in zip(cut, boxes)]
    ref = oracle.brick_advect(bricks, nb, seeds, oracle.params(**kw), "f32")
    fb = S.streami_field_create_bricked(fld.dims, fld.origin, fld.spacing, nb, 1,
                                        [torch.from_numpy(a).cuda() for a in cut])
    h_seeds = torch.from_numpy(seeds.copy())
    h_v = torch.full((3, n, 16), float("nan"), dtype=torch.float32)
    h_c = torch.zeros(n, dtype=torch.int32)
    h_steps = torch.zeros(n, dtype=torch.int32); h_status = torch.zeros(n, dtype=torch.int32)
    h_final = torch.zeros((3, n), dtype=torch.float32); h_tot = torch.zeros(4, dtype=torch.int64)
    h_rc = torch.full((32, 4), -1, dtype=torch.int32)
    h_log = torch.zeros(64 * n, dtype=torch.int64); h_lc = torch.zeros(1, dtype=torch.int64)
    prm = S.params(**kw)
    prm.out_steps = h_steps.data_ptr(); prm.out_status = h_status.data_ptr()
    prm.out_final = h_final.data_ptr(); prm.out_totals = h_tot.data_ptr()
    nrounds, trunc = S.streami_brick_advect_host(fb, h_seeds, prm, h_v, h_c, h_rc, h_log, h_lc)
    assert not trunc and nrounds == ref.nrounds
    assert np.array_equal(h_status.numpy().astype(np.uint32), ref.status)
    assert np.array_equal(h_steps.numpy().astype(np.uint32), ref.steps)
    assert np.array_equal(h_c.numpy().astype(np.uint32), ref.counts)
    assert np.array_equal(h_final.numpy().view(np.uint32), ref.final.view(np.uint32))
    mask = np.arange(16)[None, :] < ref.counts[:, None]      # slots beyond the count hold whatever the
    for c in range(3):                                       # device scratch array held (include/streami.h)
        assert np.array_equal(h_v.numpy()[c].view(np.uint32)[mask], ref.vertices[c].view(np.uint32)[mask])
    assert np.array_equal(h_tot.numpy().astype(np.uint64), ref.totals)
    assert np.array_equal(h_rc.numpy()[:ref.nrounds].astype(np.uint32), ref.round_counts[:ref.nrounds])
    assert (h_rc.numpy()[ref.nrounds + 1:] == -1).all()
    nlog = int(h_lc.item())
    assert nlog == ref.nlog
    assert np.array_equal(np.sort(h_log.numpy().view(np.uint64)[:nlog]), ref.log)


@pytest.mark.parametrize("layout,budget", [(3, -1), (5, 0), (1, 9)])
def test_bricks_dp5(S, torch, oracle, wl, layout, budget):
    """DP5(4) through the brick rounds: the hand-off record carries t and h, the FSAL k1 is
    recomputed in the new brick (bit-identical by A9).  Against the oracle's brick rounds and
    against the monolithic GPU trace."""
    N, nb = 32, (2, 2, 2)
    fld = wl.turb_field_cpu(N, 48, 1, 6)
    n = 12007
    seeds = wl.seeds_uniform(31, n, [N - 1.0] * 3)
    kw = dict(integrator=1, h=0.25, h_min=0.01, h_max=1.0, atol=1e-5, rtol=1e-5, max_steps=150,
              vmin=1e-6, capacity=40, stride=3)
    boxes = wl.brick_boxes(fld.dims, nb, 1)
    bricks = [oracle.grid(a, None, fld.origin, fld.spacing, gdims=fld.dims, lo=lo, hi=hi)
              for a, (lo, hi) in zip(wl.cut_bricks(fld, nb, 1), boxes)]
    ref = oracle.brick_advect(bricks, nb, seeds, oracle.params(**kw), "f32")
    S.streami_set_option("brick_round_steps", budget)
    try:
        out = gpu_bricks(S, torch, wl, fld, nb, seeds, layout=layout, max_rounds=128, **kw)
    finally:
        S.streami_set_option("brick_round_steps", 0)
    for key in ("status", "steps", "counts"):
        assert np.array_equal(out[key], getattr(ref, key)), key
    assert np.array_equal(out["final"].view(np.uint32), ref.final.view(np.uint32))
    assert np.array_equal(out["vertices"].view(np.uint32), ref.vertices.view(np.uint32))
    assert np.array_equal(out["totals"], ref.totals)
    if budget == -1:                                   # A9's rounds: queue membership bit exact
        assert out["nrounds"] == ref.nrounds
        assert np.array_equal(out["log"], ref.log)
        assert np.array_equal(out["round_counts"][:ref.nrounds].astype(np.uint32), ref.round_counts[:ref.nrounds])
    assert ref.nlog > n // 20 and int(ref.totals[0]) > int(ref.totals[1])      # hand-offs and rejections occur
    halo = ref.status == 4                             # steps of up to 1 cell may overrun a 1-cell halo (Q14)
    from helpers import gpu_streamlines
    mono = gpu_streamlines(S, torch, gpu_field(S, torch, fld, layout), seeds, **kw)
    ok = ~halo
    for key in ("status", "steps", "counts"):
        assert np.array_equal(out[key][ok], mono[key][ok]), key
    assert np.array_equal(out["final"].view(np.uint32)[:, ok], mono["final"].view(np.uint32)[:, ok])


@pytest.mark.parametrize("kind", ["tame", "nan", "inf"])
@pytest.mark.parametrize("integ", [0, 1])
def test_bricks_integer_accept_and_untamed_fields(S, torch, oracle, wl, kind, integ):
    """The brick kernels decide "served and inside" from floor(g) when every brick holds finite
    values and fall back to the float tests (descriptor read through its table entry) otherwise:
    fields with planted NaN / inf, the option on and off, thin ghosts (HALO_MISS), seeds on the
    domain faces -- RK4 and DP5(4), all against the oracle bit for bit."""
    import dataclasses
    N, nb = 28, (2, 2, 2)
    base = wl.turb_field_cpu(N, 32, 1, 5)
    data = base.data.copy()
    idx = np.random.default_rng(6).integers(0, N, size=(150, 3))
    if kind == "nan":
        data[0, idx[:, 2], idx[:, 1], idx[:, 0], idx[:, 0] % 3] = np.nan
    elif kind == "inf":
        data[0, idx[:, 2], idx[:, 1], idx[:, 0], idx[:, 0] % 3] = np.where(idx[:, 1] % 2, np.inf, -np.inf)
    fld = dataclasses.replace(base, data=data)
    n = 8000
    seeds = wl.seeds_uniform(31, n, [N - 1.0] * 3)
    seeds[:300] = np.round(seeds[:300]); seeds[300:500, 0] = N - 1.0; seeds[500:700, 2] = 0.0
    seeds[700:850] = idx + 0.5
    if integ == 0:
        kw = dict(integrator=0, h=1.5, max_steps=12, vmin=1e-6, capacity=20, stride=1)      # long steps: halo misses
    else:
        kw = dict(integrator=1, h=0.25, h_min=0.01, h_max=1.0, atol=1e-4, rtol=1e-4, max_steps=120, vmin=1e-6,
                  capacity=20, stride=8)
    boxes = wl.brick_boxes(fld.dims, nb, 1)
    bricks = [oracle.grid(a, None, fld.origin, fld.spacing, gdims=fld.dims, lo=lo, hi=hi)
              for a, (lo, hi) in zip(wl.cut_bricks(fld, nb, 1), boxes)]
    ref = oracle.brick_advect(bricks, nb, seeds, oracle.params(**kw), "f32")
    for on in (1, 0):
        try:
            S.streami_set_option("integer_accept", on)
            out = gpu_bricks(S, torch, wl, fld, nb, seeds, **kw)
        finally:
            S.streami_set_option("integer_accept", 1)
        for key in ("status", "steps", "counts"):
            assert np.array_equal(out[key], getattr(ref, key)), (key, on)
        assert np.array_equal(out["final"].view(np.uint32), ref.final.view(np.uint32)), on
        assert np.array_equal(out["vertices"].view(np.uint32), ref.vertices.view(np.uint32)), on
        assert np.array_equal(out["totals"], ref.totals), on
        assert out["nrounds"] == ref.nrounds and np.array_equal(out["log"], ref.log)
    hist = np.bincount(ref.status, minlength=5)
    assert hist[1] > 50
    if integ == 0:
        assert hist[2] > 50 and hist[4] > 0, "the case must contain MAX_STEPS and HALO_MISS"
