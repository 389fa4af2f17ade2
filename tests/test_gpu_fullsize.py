"""Parity at BASELINE.json's FULL sizes.

C2, C4, C5, P4 and `test_c3_full_size_bench_config` run exactly the call bench.py times
(`bench.Job.step_device`: same field generator, seeds, parameters, layout and options).
`test_c3_full_size_sampled` additionally asks for the round table and the hand-off log, which
switches streami_brick_advect to A9's observable rounds (no step budget, no ring finish): it checks
the queue outputs, not the timed configuration.  The oracle runs a strided sample of the particles one by one on
the SAME field bytes (copied from the device) and every per-particle output of those ids is
compared bit for bit.  Properties that hold at any size (P10 invariants) are checked on all ids.
Tolerance: the formula sheet makes both sides execute the same IEEE operations, so the bar here is
bit-exact (stricter than north_star's 99.9 % / 1e-4 cell, which tests/test_gpu_parity.py
::test_gpu_tolerance_form also evaluates).
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def torch():
    import torch as t
    if not t.cuda.is_available():
        pytest.skip("no CUDA device")
    return t


@pytest.fixture(scope="module")
def bench():
    import bench as b
    return b


def _gpu_outputs(job, torch, ids):
    job.step_device()
    torch.cuda.synchronize()
    idx = torch.from_numpy(ids.astype(np.int64)).cuda()
    out = dict(counts=job.counts[idx].cpu().numpy().astype(np.uint32),
               steps=job.steps_o[idx].cpu().numpy().astype(np.uint32),
               status=job.status_o[idx].cpu().numpy().astype(np.uint32),
               final=job.final_o[:, idx].cpu().numpy(),
               vertices=job.verts[:, idx, :].cpu().numpy())
    return out


def _invariants(job, torch, max_steps, cap, N):
    """P10 on ALL particles: status in 1..4, steps <= max_steps, counts <= capacity, final inside."""
    st = job.status_o
    assert int(st.min()) >= 1 and int(st.max()) <= 4
    assert int(job.steps_o.max()) <= max_steps
    assert int(job.counts.max()) <= cap and int(job.counts.min()) >= 0
    f = job.final_o
    assert bool(((f >= 0) & (f <= N - 1)).all())
    tot = job.totals_o.cpu().numpy()
    assert int(tot[1]) == int(job.steps_o.to(torch.int64).sum().item())      # accepted steps
    assert tot[0] >= tot[1]


def _compare(gpu, ref, what):
    k = gpu["counts"].shape[0]
    assert np.array_equal(gpu["status"], ref.status), what + " status"
    assert np.array_equal(gpu["steps"], ref.steps), what + " steps"
    assert np.array_equal(gpu["counts"], ref.counts), what + " counts"
    assert np.array_equal(gpu["final"].view(np.uint32), ref.final.view(np.uint32)), what + " final"
    cap = gpu["vertices"].shape[2]
    mask = np.arange(cap)[None, :] < ref.counts[:, None]                      # stored slots only
    for c in range(3):
        a = gpu["vertices"][c].view(np.uint32)[mask]
        b = ref.vertices[c].view(np.uint32)[mask]
        assert np.array_equal(a, b), what + " vertices plane %d" % c
    assert k == ref.status.shape[0]


def test_c2_full_size_sampled(torch, bench, oracle):
    """C2 (the bench default): 256^3 turbulence, 1,048,576 seeds, RK4 h = 0.25, max 2,000 steps,
    capacity 256 stride 8; oracle on every 64th seed (16,384 particles)."""
    job = bench.Job("c2", 0, 0)
    fld = job.host_field
    ids = np.arange(0, job.n, 64)
    gpu = _gpu_outputs(job, torch, ids)
    _invariants(job, torch, 2000, 256, 256)
    g = oracle.grid(fld.data, fld.dims, fld.origin, fld.spacing)
    ref = oracle.streamlines(g, job.seeds_h[ids], oracle.params(**job.w["prm"]), "f32")
    _compare(gpu, ref, "c2")
    # workload shape, recorded in DESIGN.md section 4
    st = job.steps_o.float()
    print("C2 steps/particle mean %.1f median %.1f at cap %.3f" %
          (st.mean().item(), st.median().item(), (job.steps_o == 2000).float().mean().item()))


def test_p4_pathlines_full_size_sampled(torch, bench, oracle):
    """P4 (bench.py --workload p4): 1,048,576 RK4 pathlines through C4's 64-slice double gyre with the
    two-slice register copy of the cell; oracle on every 128th seed."""
    job = bench.Job("p4", 0, 0)
    fld = job.host_field
    ids = np.arange(0, job.n, 128)
    gpu = _gpu_outputs(job, torch, ids)
    st = job.status_o
    assert int(st.min()) >= 1 and int(st.max()) <= 3 and int(job.steps_o.max()) <= 1000
    g = oracle.grid(fld.data, fld.dims, fld.origin, fld.spacing, fld.nslices, fld.slice_dt)
    ref = oracle.streamlines(g, job.seeds_h[ids], oracle.params(**job.w["prm"]), "f32")
    _compare(gpu, ref, "p4")


def test_c2_parity_recording_first_200_vertices(torch, bench, oracle, wl):
    """C2 with the parity-run recording (capacity 201, stride 1): every one of the first 200
    vertices of every 256th particle, bit for bit, plus north_star's tolerance form."""
    import paper_2606_02627_b200 as S
    job = bench.Job("c2", 0, 0)
    fld = job.host_field
    prm = dict(job.w["prm"]); prm.update(capacity=201, stride=1)
    n = job.n
    verts = torch.empty((3, n, 201), dtype=torch.float32, device="cuda")
    job.verts = verts
    job.prm = S.params(out_steps=job.steps_o, out_status=job.status_o, out_final=job.final_o,
                       out_totals=job.totals_o, **prm)
    ids = np.arange(0, n, 256)
    gpu = _gpu_outputs(job, torch, ids)
    g = oracle.grid(fld.data, fld.dims, fld.origin, fld.spacing)
    ref = oracle.streamlines(g, job.seeds_h[ids], oracle.params(**prm), "f32")
    _compare(gpu, ref, "c2 parity run")
    mask = np.arange(201)[None, :] < ref.counts[:, None]
    d = np.abs(gpu["vertices"].astype(np.float64) - ref.vertices.astype(np.float64))
    assert float(d[:, mask].max()) <= 1e-4            # cell widths (spacing 1), first 200 steps
    assert np.mean(gpu["status"] == ref.status) >= 0.999


def test_c3_full_size_sampled(torch, bench, oracle, wl):
    """C3: 512^3 turbulence in 2x2x2 bricks, 4,194,304 seeds, rounds until all terminate; oracle
    (brick rounds, A9) on every 256th seed.  Also: no HALO_MISS anywhere (Q14) and the hand-off
    log restricted to the sampled ids equals the oracle's."""
    job = bench.Job("c3", 0, 0)
    fld = job.host_field
    n = job.n
    log = torch.zeros(16 * n, dtype=torch.int64, device="cuda")
    logc = torch.zeros(1, dtype=torch.int64, device="cuda")
    rcounts = torch.zeros((256, 8), dtype=torch.int32, device="cuda")
    import paper_2606_02627_b200 as S
    nrounds, trunc = S.streami_brick_advect(job.field, job.seeds, job.prm, job.verts, job.counts,
                                            rcounts, log, logc)
    torch.cuda.synchronize()
    assert not trunc
    ids = np.arange(0, n, 256)
    idx = torch.from_numpy(ids.astype(np.int64)).cuda()
    gpu = dict(counts=job.counts[idx].cpu().numpy().astype(np.uint32),
               steps=job.steps_o[idx].cpu().numpy().astype(np.uint32),
               status=job.status_o[idx].cpu().numpy().astype(np.uint32),
               final=job.final_o[:, idx].cpu().numpy(), vertices=job.verts[:, idx, :].cpu().numpy())
    _invariants(job, torch, 4000, 256, 512)
    assert int((job.status_o == 4).sum().item()) == 0, "HALO_MISS must not occur in C3 (Q14)"
    boxes = wl.brick_boxes(fld.dims, (2, 2, 2), 1)
    cut = wl.cut_bricks(fld, (2, 2, 2), 1)
    bricks = [oracle.grid(c, None, fld.origin, fld.spacing, gdims=fld.dims, lo=lo, hi=hi)
              for c, (lo, hi) in zip(cut, boxes)]
    ref = oracle.brick_advect(bricks, (2, 2, 2), job.seeds_h[ids], oracle.params(**job.w["prm"]), "f32")
    _compare(gpu, ref, "c3")
    # hand-off log: entries (round+1)<<48 | dest<<32 | id; restrict to sampled ids, renumber, sort
    nlog = int(logc.item())
    assert nlog <= log.numel()
    L = log[:nlog].cpu().numpy().astype(np.uint64)
    lid = (L & np.uint64(0xffffffff)).astype(np.int64)
    sel = (lid % 256) == 0
    mine = np.sort((L[sel] & ~np.uint64(0xffffffff)) | (lid[sel] // 256).astype(np.uint64))
    assert np.array_equal(mine, ref.log), "hand-off log membership"
    # P10: round table sums
    rc = rcounts.cpu().numpy().astype(np.int64)
    assert rc[0].sum() == n, "Q_0 holds every (inside) seed once"
    assert rc[1:nrounds + 1].sum() == nlog, "total hand-offs = sum of later queue sizes"
    assert int(job.totals_o[3].item()) == nlog


def test_c3_full_size_bench_config(torch, bench, oracle, wl):
    """C3 exactly as bench.py times it: `Job.step_device`, i.e. no round table and
    no log, so the library runs its automatic schedule -- 256-step budget per round, Morton sort +
    gather of every round's work (n >= 65,536), and the stragglers finished through the in-kernel
    hand-off ring.  Every per-particle output of every 256th id is compared with the oracle's brick
    rounds (A9) bit for bit; totals[0:3] and the hand-off count are schedule-independent and are
    compared with `test_c3_full_size_sampled`'s observable-rounds run of the same seeds."""
    import paper_2606_02627_b200 as S
    job = bench.Job("c3", 0, 0)
    fld = job.host_field
    n = job.n
    ids = np.arange(0, n, 256)
    gpu = _gpu_outputs(job, torch, ids)                  # = job.step_device(): the timed call
    tot_auto = job.totals_o.cpu().numpy().copy()
    _invariants(job, torch, 4000, 256, 512)
    assert int((job.status_o == 4).sum().item()) == 0, "HALO_MISS must not occur in C3 (Q14)"
    boxes = wl.brick_boxes(fld.dims, (2, 2, 2), 1)
    cut = wl.cut_bricks(fld, (2, 2, 2), 1)
    bricks = [oracle.grid(c, None, fld.origin, fld.spacing, gdims=fld.dims, lo=lo, hi=hi)
              for c, (lo, hi) in zip(cut, boxes)]
    ref = oracle.brick_advect(bricks, (2, 2, 2), job.seeds_h[ids], oracle.params(**job.w["prm"]), "f32")
    _compare(gpu, ref, "c3 bench config")
    # all particles: the automatic schedule and A9's rounds give the same per-particle results and totals
    auto = dict(counts=job.counts.clone(), steps=job.steps_o.clone(), status=job.status_o.clone(),
                final=job.final_o.clone())
    logc = torch.zeros(1, dtype=torch.int64, device="cuda")
    rcounts = torch.zeros((256, 8), dtype=torch.int32, device="cuda")
    job.counts.zero_(); job.steps_o.zero_(); job.status_o.zero_(); job.final_o.zero_()
    S.streami_brick_advect(job.field, job.seeds, job.prm, job.verts, job.counts, rcounts, None, logc)
    torch.cuda.synchronize()
    for k, t in (("counts", job.counts), ("steps", job.steps_o), ("status", job.status_o)):
        assert bool((auto[k] == t).all()), "c3 automatic vs A9 rounds: " + k
    assert bool((auto["final"].view(torch.int32) == job.final_o.view(torch.int32)).all())
    tot_a9 = job.totals_o.cpu().numpy()
    assert np.array_equal(tot_auto[:3], tot_a9[:3]), "attempts / accepted / samples"
    assert int(tot_auto[3]) == int(tot_a9[3]) == int(logc.item()), "hand-off count"


def test_c4_full_size_sampled(torch, bench, oracle):
    """C4: double gyre 256x128x64 x 64 slices, 4,096-point rake, 1,000 global steps; oracle on
    every 64th rake point (64 points x 1,000 releases)."""
    job = bench.Job("c4", 0, 0)
    fld = job.host_field
    job.step_device()
    torch.cuda.synchronize()
    m, ns = job.n, job.nsteps
    pts = np.arange(0, m, 64)
    g = oracle.grid(fld.data, fld.dims, fld.origin, fld.spacing, fld.nslices, fld.slice_dt)
    prm = oracle.params(integrator=0, h=0.05, vmin=1e-6, max_steps=ns, capacity=1, stride=1)
    ref = oracle.streaklines(g, job.seeds_h[pts], ns, prm, "f32")
    v = job.verts.cpu().numpy()[:, :, pts]                                   # [3][ns][k]
    assert np.array_equal(v.view(np.uint32), ref.vertices.view(np.uint32)), "c4 slots"
    st = job.status_o.cpu().numpy().astype(np.uint32).reshape(ns, m)[:, pts].reshape(-1)
    sp = job.steps_o.cpu().numpy().astype(np.uint32).reshape(ns, m)[:, pts].reshape(-1)
    assert np.array_equal(st, ref.status), "c4 status"
    dead = ref.status != 2
    assert np.array_equal(sp[dead], ref.steps[dead]), "c4 steps of the dead"
    assert np.array_equal(job.counts.cpu().numpy().astype(np.uint32)[pts], ref.counts), "c4 counts"


def test_c5_full_size_sampled(torch, bench, oracle):
    """C5: 1024^3 turbulence (12.9 GB), 16,777,216 seeds, DP5(4) tol 1e-5, h in [0.01, 1], max
    8,000 accepted steps, capacity 64 stride 128; oracle on every 2048th seed (8,192 particles)
    on a host copy of the same field bytes."""
    job = bench.Job("c5", 0, 0)
    ids = np.arange(0, job.n, 2048)
    gpu = _gpu_outputs(job, torch, ids)
    _invariants(job, torch, 8000, 64, 1024)
    data = job.data.cpu().numpy()                                            # the same bytes
    g = oracle.grid(data, (1024, 1024, 1024), (0, 0, 0), (1, 1, 1))
    ref = oracle.streamlines(g, job.seeds_h[ids], oracle.params(**job.w["prm"]), "f32")
    _compare(gpu, ref, "c5")
    tot = job.totals_o.cpu().numpy()
    print("C5 attempts %d accepted %d samples %d" % (tot[0], tot[1], tot[2]))
