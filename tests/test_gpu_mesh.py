"""Hexahedral-mesh fields (the paper's other field type) against the oracle
(oracle/hexmesh_oracle.hpp, formula sheet U1-U4), bit for bit: located cell, reference
coordinates through the sampled value, RK4 streamlines.  Distorted cells, bins coarser and finer than
the cells, points and seeds outside the mesh."""
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
def S(torch):
    import paper_2606_02627_b200 as s
    s.lib()
    return s


def _mesh(wl, oracle, S, N=20, jitter=0.3, nb=(7, 9, 5)):
    fld = wl.turb_field_cpu(N, 24, 1, 4)
    X, V, H, lo, hi = wl.hexmesh_from_grid(fld.dims, fld.origin, fld.spacing, fld.data[0], jitter=jitter, seed=11)
    return fld, oracle.HexMesh(X, V, H, lo, hi, nb), S.Mesh(X, V, H, lo, hi, nb), lo, hi


@pytest.mark.parametrize("jitter,nb", [(0.0, (4, 4, 4)), (0.3, (7, 9, 5)), (0.35, (40, 33, 37))])
def test_mesh_sample(S, torch, oracle, wl, jitter, nb):
    fld, om, gm, lo, hi = _mesh(wl, oracle, S, jitter=jitter, nb=nb)
    rng = np.random.default_rng(3)
    pts = (lo - 0.3 + rng.uniform(0.0, 1.0, size=(20011, 3)) * (hi - lo + 0.6)).astype(np.float32)
    pts[:4] = [lo, hi, [np.nan, 1, 1], (lo + hi) / 2]
    rv, rcell, _ = oracle.hexmesh_sample(om, pts, "f32")
    v, cell = S.streami_mesh_sample(gm, torch.from_numpy(pts).cuda())
    assert np.array_equal(cell.cpu().numpy(), rcell)
    assert np.array_equal(v.cpu().numpy().view(np.uint32), rv.view(np.uint32))
    assert np.count_nonzero(rcell < 0) > 500 and np.count_nonzero(rcell >= 0) > 10000


@pytest.mark.parametrize("jitter", [0.0, 0.3])
def test_mesh_streamlines(S, torch, oracle, wl, jitter):
    fld, om, gm, lo, hi = _mesh(wl, oracle, S, jitter=jitter)
    n = 6007
    seeds = wl.seeds_uniform(8, n, [19.0] * 3)
    seeds[3] = [25.0, 1, 1]
    kw = dict(integrator=0, h=0.25, max_steps=120, vmin=1e-6, capacity=25, stride=5)
    ref = oracle.hexmesh_streamlines(om, seeds, oracle.params(**kw), "f32")
    verts = torch.full((3, n, 25), float("nan"), dtype=torch.float32, device="cuda")
    counts = torch.full((n,), -1, dtype=torch.int32, device="cuda")
    steps = torch.zeros(n, dtype=torch.int32, device="cuda"); status = torch.zeros(n, dtype=torch.int32, device="cuda")
    final = torch.zeros((3, n), dtype=torch.float32, device="cuda"); totals = torch.zeros(4, dtype=torch.int64, device="cuda")
    prm = S.params(out_steps=steps, out_status=status, out_final=final, out_totals=totals, **kw)
    S.streami_mesh_trace_streamlines(gm, torch.from_numpy(seeds).cuda(), prm, verts, counts)
    torch.cuda.synchronize()
    assert np.array_equal(status.cpu().numpy().astype(np.uint32), ref.status)
    assert np.array_equal(steps.cpu().numpy().astype(np.uint32), ref.steps)
    assert np.array_equal(counts.cpu().numpy().astype(np.uint32), ref.counts)
    assert np.array_equal(final.cpu().numpy().view(np.uint32), ref.final.view(np.uint32))
    assert np.array_equal(verts.cpu().numpy().view(np.uint32), ref.vertices.view(np.uint32))
    assert np.array_equal(totals.cpu().numpy().astype(np.uint64)[:3], ref.totals[:3])
    hist = np.bincount(ref.status, minlength=4)
    assert hist[1] > 50 and hist[2] > 50
    if jitter == 0.0:      # the hexahedral re-expression of a grid tracks the structured trace
        from helpers import gpu_field, gpu_streamlines
        g = gpu_streamlines(S, torch, gpu_field(S, torch, fld), seeds, **kw)
        same = (g["status"] == ref.status) & (g["steps"] == ref.steps)
        assert same.mean() > 0.995
        d = np.abs(g["final"] - ref.final)[:, same]
        assert np.median(d) < 1e-4


@pytest.mark.parametrize("nb", [(1, 1, 1), (300, 2, 170), (2, 512, 3)])
def test_mesh_sample_with_extreme_bins(S, torch, oracle, wl, nb):
    """The packed candidate boxes in the bin lists are in bin coordinates with 16 bits per bound: one
    bin for the whole mesh (every cell a candidate, boxes at 1/256 of the domain) and bins hundreds
    of times finer than a cell (bounds saturate) must locate the same cells as the oracle."""
    fld, om, gm, lo, hi = _mesh(wl, oracle, S, N=10, jitter=0.35, nb=nb)
    rng = np.random.default_rng(4)
    pts = (lo - 0.2 + rng.uniform(0.0, 1.0, size=(4001, 3)) * (hi - lo + 0.4)).astype(np.float32)
    pts[:3] = [lo, hi, (lo + hi) / 2]
    rv, rcell, _ = oracle.hexmesh_sample(om, pts, "f32")
    v, cell = S.streami_mesh_sample(gm, torch.from_numpy(pts).cuda())
    assert np.array_equal(cell.cpu().numpy(), rcell)
    assert np.array_equal(v.cpu().numpy().view(np.uint32), rv.view(np.uint32))
    assert np.count_nonzero(rcell >= 0) > 2000


@pytest.mark.parametrize("batch", [0, 900])
def test_mesh_streamlines_lines_host(S, torch, oracle, wl, batch):
    """Host seeds in, host polylines out on a mesh (one batch and several): equals the oracle's mesh
    trace + the line definition, with the optional per-particle outputs."""
    from oracle import lines
    fld, om, gm, lo, hi = _mesh(wl, oracle, S, jitter=0.3)
    n = 3001
    seeds = wl.seeds_uniform(9, n, [19.0] * 3)
    seeds[7] = [-3.0, 1, 1]
    kw = dict(integrator=0, h=0.25, max_steps=100, vmin=1e-6, capacity=16, stride=4)
    ref = oracle.hexmesh_streamlines(om, seeds, oracle.params(**kw), "f32")
    roff, rp = lines.streamline_lines(ref.vertices, ref.counts)
    off = torch.zeros(n + 1, dtype=torch.int64).pin_memory()
    pts = torch.full((n * 16, 3), float("nan"), dtype=torch.float32).pin_memory()
    h_status = torch.zeros(n, dtype=torch.int32); h_final = torch.zeros((3, n), dtype=torch.float32)
    h_totals = torch.zeros(4, dtype=torch.int64)
    prm = S.params(**kw)
    prm.out_status = h_status.data_ptr(); prm.out_final = h_final.data_ptr(); prm.out_totals = h_totals.data_ptr()
    try:
        S.streami_set_option("host_batch", batch)
        total, trunc = S.streami_mesh_trace_streamlines_lines_host(gm, torch.from_numpy(seeds.copy()), prm, off, pts)
    finally:
        S.streami_set_option("host_batch", 0)
    assert not trunc and total == int(roff[-1])
    assert np.array_equal(off.numpy().astype(np.uint64), roff)
    assert np.array_equal(pts.numpy()[:total].view(np.uint32), rp.view(np.uint32))
    assert np.array_equal(h_status.numpy().astype(np.uint32), ref.status)
    assert np.array_equal(h_final.numpy().view(np.uint32), ref.final.view(np.uint32))
    assert np.array_equal(h_totals.numpy()[:3].astype(np.uint64), ref.totals[:3])
