"""the step-synchronous streakline API (Tracer::step(), Listing 2) with
per-step snapshots, and polyline assembly (getLines).  After s global steps the slots equal what the
oracle's A7 returns for nsteps = s; the assembled lines equal oracle/lines.py."""
import numpy as np
import pytest

from helpers import gpu_field, gpu_streamlines

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


@pytest.mark.parametrize("window", [0, 3])
def test_streak_step_snapshots(S, torch, oracle, wl, window):
    from oracle import lines
    fld = wl.double_gyre_field(dims=(48, 24, 12), nslices=8, dt=0.25)
    pts = wl.rake_c4(12, 6)
    pts[5] = [2.5, 0.2, 0.2]                               # a rake point outside: its particles are born dead
    m, ns, h = pts.shape[0], 60, 0.05
    g = oracle.grid(fld.data, fld.dims, fld.origin, fld.spacing, fld.nslices, fld.slice_dt)
    f = gpu_field(S, torch, fld)
    d_pts = torch.from_numpy(pts).cuda()
    verts = torch.zeros((3, ns, m), dtype=torch.float32, device="cuda")
    status = torch.full((ns * m,), -1, dtype=torch.int32, device="cuda")
    prm = S.params(integrator=0, h=h, vmin=1e-6, out_status=status)
    S.streami_set_option("streak_window", window)
    try:
        tr = S.Streak(f, d_pts, ns, prm, verts)
        done = 0
        for k in (1, 9, 15, 35):                           # snapshots at s = 1, 10, 25, 60
            tr.step(k)
            done += k
            assert tr.position() == done
            ref = oracle.streaklines(g, pts, done, oracle.params(integrator=0, h=h, vmin=1e-6, max_steps=done), "f32")
            torch.cuda.synchronize()
            got = verts.cpu().numpy()[:, :done, :]
            assert np.array_equal(got.view(np.uint32), ref.vertices.view(np.uint32)), "slots after %d steps" % done
            off, lp = tr.lines()
            roff, rp = lines.streak_lines(ref.vertices, ref.status)
            assert np.array_equal(off.cpu().numpy().astype(np.uint64), roff)
            assert np.array_equal(lp.cpu().numpy().view(np.uint32), rp.view(np.uint32)), "lines after %d steps" % done
        tr.step(1000)                                      # clamped
        assert tr.position() == ns
        counts = torch.zeros(m, dtype=torch.int32, device="cuda")
        tr.end(counts)
        torch.cuda.synchronize()
        assert np.array_equal(counts.cpu().numpy().astype(np.uint32), ref.counts)
        assert np.array_equal(status.cpu().numpy().astype(np.uint32), ref.status)
    finally:
        S.streami_set_option("streak_window", 0)


def test_streamline_lines(S, torch, oracle, wl):
    from oracle import lines
    fld = wl.turb_field_cpu(32, 32, 1, 6)
    n = 5003                                               # several scan tiles and a ragged tail
    seeds = wl.seeds_uniform(3, n, [31.0] * 3)
    seeds[7] = [40.0, 1, 1]                                # an empty line
    kw = dict(integrator=0, h=0.25, max_steps=90, vmin=1e-6, capacity=19, stride=5)
    f = gpu_field(S, torch, fld)
    d_seeds = torch.from_numpy(seeds).cuda()
    verts = torch.full((3, n, 19), float("nan"), dtype=torch.float32, device="cuda")
    counts = torch.zeros(n, dtype=torch.int32, device="cuda")
    S.streami_trace_streamlines(f, d_seeds, S.params(**kw), verts, counts)
    off, pts = S.streami_streamline_lines(verts, counts)
    torch.cuda.synchronize()
    ref = oracle.streamlines(oracle.grid(fld.data, fld.dims, fld.origin, fld.spacing), seeds, oracle.params(**kw), "f32")
    roff, rp = lines.streamline_lines(ref.vertices, ref.counts)
    assert np.array_equal(off.cpu().numpy().astype(np.uint64), roff)
    assert np.array_equal(pts.cpu().numpy().view(np.uint32), rp.view(np.uint32))
    assert int(roff[8]) == int(roff[7])                    # the empty line
    # n = 0 and offsets-only
    e_off, e_pts = S.streami_streamline_lines(verts[:, :0, :].contiguous(), counts[:0].contiguous())
    assert e_off.cpu().tolist() == [0] and e_pts.shape[0] == 0


@pytest.mark.parametrize("mode", [0, 1])
def test_seed_shape(S, torch, oracle, mode):
    """Seed-generation kernel against the oracle, bit for bit: line, skewed
    plane, box; and the seeds feed a trace."""
    shapes = [((0.5, 1.0, 2.0), (3.0, 0.25, -1.0), (0, 0, 0), (0, 0, 0), 1000, 1, 1),
              ((1.0, 1.0, 1.0), (2.0, 2.0, 0.0), (0.0, 3.0, 5.0), (0, 0, 0), 37, 91, 1),
              ((0.0, 0.0, 0.0), (31.0, 0, 0), (0, 31.0, 0), (0, 0, 31.0), 33, 17, 29)]
    for o, eu, ev, ew, nu, nv, nw in shapes:
        got = S.streami_seed_shape(o, eu, ev, ew, nu, nv, nw, mode, rng_seed=12345).cpu().numpy()
        ref = oracle.seed_shape(o, eu, ev, ew, nu, nv, nw, mode, 12345)
        assert np.array_equal(got.view(np.uint32), ref.view(np.uint32)), (mode, nu, nv, nw)
    assert S.streami_seed_shape((0, 0, 0), (1, 0, 0), nu=0).shape[0] == 0


def test_streamlines_lines_host(S, torch, oracle, wl):
    """Host seeds in, host polylines out: equals the oracle's trace + the line definition; a point
    buffer that is too small reports TRUNCATED and still delivers the first points."""
    from oracle import lines
    fld = wl.turb_field_cpu(32, 32, 1, 6)
    n = 3001
    seeds = wl.seeds_uniform(21, n, [31.0] * 3)
    kw = dict(integrator=0, h=0.25, max_steps=80, vmin=1e-6, capacity=16, stride=4)
    ref = oracle.streamlines(oracle.grid(fld.data, fld.dims, fld.origin, fld.spacing), seeds, oracle.params(**kw), "f32")
    roff, rp = lines.streamline_lines(ref.vertices, ref.counts)
    f = gpu_field(S, torch, fld)
    h_seeds = torch.from_numpy(seeds.copy())
    off = torch.zeros(n + 1, dtype=torch.int64)
    pts = torch.full((n * 16, 3), float("nan"), dtype=torch.float32)
    h_status = torch.zeros(n, dtype=torch.int32)
    prm = S.params(**kw)
    prm.out_status = h_status.data_ptr()
    total, trunc = S.streami_trace_streamlines_lines_host(f, h_seeds, prm, off, pts)
    assert not trunc and total == int(roff[-1])
    assert np.array_equal(off.numpy().astype(np.uint64), roff)
    assert np.array_equal(pts.numpy()[:total].view(np.uint32), rp.view(np.uint32))
    assert np.isnan(pts.numpy()[total:]).all()
    assert np.array_equal(h_status.numpy().astype(np.uint32), ref.status)
    small = torch.zeros((100, 3), dtype=torch.float32)
    total2, trunc2 = S.streami_trace_streamlines_lines_host(f, h_seeds, S.params(**kw), off, small)
    assert trunc2 and total2 == total
    assert np.array_equal(small.numpy().view(np.uint32), rp[:100].view(np.uint32))


def test_streamlines_lines_host_on_bricks(S, torch, oracle, wl):
    """The same host call on a bricked field runs the brick rounds."""
    from oracle import lines
    N, nb = 24, (2, 2, 1)
    fld = wl.turb_field_cpu(N, 32, 1, 5)
    n = 2500
    seeds = wl.seeds_uniform(22, n, [N - 1.0] * 3)
    kw = dict(integrator=0, h=0.25, max_steps=100, vmin=1e-6, capacity=16, stride=8)
    ref = oracle.streamlines(oracle.grid(fld.data, fld.dims, fld.origin, fld.spacing), seeds, oracle.params(**kw), "f32")
    roff, rp = lines.streamline_lines(ref.vertices, ref.counts)
    fb = S.streami_field_create_bricked(fld.dims, fld.origin, fld.spacing, nb, 1,
                                        [torch.from_numpy(a).cuda() for a in wl.cut_bricks(fld, nb, 1)])
    off = torch.zeros(n + 1, dtype=torch.int64)
    pts = torch.zeros((n * 16, 3), dtype=torch.float32)
    total, trunc = S.streami_trace_streamlines_lines_host(fb, torch.from_numpy(seeds.copy()), S.params(**kw), off, pts)
    assert not trunc and total == int(roff[-1])
    assert np.array_equal(off.numpy().astype(np.uint64), roff)
    assert np.array_equal(pts.numpy()[:total].view(np.uint32), rp.view(np.uint32))      # P9: bricks == monolithic


@pytest.mark.parametrize("bricked", [False, True])
@pytest.mark.parametrize("batch", [700, 1000, 5000])
def test_streamlines_lines_host_in_batches(S, torch, oracle, wl, bricked, batch):
    """`host_batch` splits the seeds into batches whose polylines are copied out while the next batch
    is traced; offsets, points, every optional per-particle output, the totals and the truncation
    rule must not depend on the split (3001 seeds in batches of 700 / 1000 / one batch)."""
    from oracle import lines
    N = 24
    fld = wl.turb_field_cpu(N, 32, 1, 5)
    n = 3001
    seeds = wl.seeds_uniform(23, n, [N - 1.0] * 3)
    seeds[5] = [N + 2.0, 1, 1]                                           # an empty line
    kw = dict(integrator=0, h=0.25, max_steps=90, vmin=1e-6, capacity=16, stride=4)
    ref = oracle.streamlines(oracle.grid(fld.data, fld.dims, fld.origin, fld.spacing), seeds, oracle.params(**kw), "f32")
    roff, rp = lines.streamline_lines(ref.vertices, ref.counts)
    if bricked:
        nbk = (2, 1, 2)
        f = S.streami_field_create_bricked(fld.dims, fld.origin, fld.spacing, nbk, 1,
                                           [torch.from_numpy(a).cuda() for a in wl.cut_bricks(fld, nbk, 1)])
    else:
        f = gpu_field(S, torch, fld)
    h_seeds = torch.from_numpy(seeds.copy()).pin_memory()
    off = torch.zeros(n + 1, dtype=torch.int64).pin_memory()
    pts = torch.full((n * 16, 3), float("nan"), dtype=torch.float32).pin_memory()
    h_status = torch.zeros(n, dtype=torch.int32); h_steps = torch.zeros(n, dtype=torch.int32)
    h_final = torch.zeros((3, n), dtype=torch.float32); h_totals = torch.zeros(4, dtype=torch.int64)
    prm = S.params(**kw)
    prm.out_status = h_status.data_ptr(); prm.out_steps = h_steps.data_ptr()
    prm.out_final = h_final.data_ptr(); prm.out_totals = h_totals.data_ptr()
    try:
        S.streami_set_option("host_batch", batch)
        total, trunc = S.streami_trace_streamlines_lines_host(f, h_seeds, prm, off, pts)
        small = torch.zeros((1234, 3), dtype=torch.float32)
        total2, trunc2 = S.streami_trace_streamlines_lines_host(f, h_seeds, S.params(**kw), off.clone(), small)
    finally:
        S.streami_set_option("host_batch", 0)
    assert not trunc and total == int(roff[-1])
    assert np.array_equal(off.numpy().astype(np.uint64), roff)
    assert np.array_equal(pts.numpy()[:total].view(np.uint32), rp.view(np.uint32))
    assert np.isnan(pts.numpy()[total:]).all()
    assert np.array_equal(h_status.numpy().astype(np.uint32), ref.status)
    assert np.array_equal(h_steps.numpy().astype(np.uint32), ref.steps)
    assert np.array_equal(h_final.numpy().view(np.uint32), ref.final.view(np.uint32))
    assert np.array_equal(h_totals.numpy()[:3].astype(np.uint64), ref.totals[:3])
    assert trunc2 and total2 == total
    assert np.array_equal(small.numpy().view(np.uint32), rp[:1234].view(np.uint32))
