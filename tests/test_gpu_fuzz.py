"""Randomised parity sweep: seeded random grids (anisotropic dims, non-unit origin and spacing, steady or
time-sliced), every layout, both integrators, random recording strides / capacities / step sizes and seed counts on
both sides of the presort threshold, traced by the CUDA path and by the fp32 oracle and compared bit for bit.
The hand-picked cases of test_gpu_parity.py / test_gpu_schedule_options.py fix one knob at a time; this sweep
crosses them (e.g. the phase length of the RK4 loop is derived from the stride, the unit-geometry and
integer-accept specialisations from the geometry and the field values)."""
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


def _random_field(wl, rng, unsteady):
    """A smooth random field on a random grid: a few Fourier modes per component, fp64, rounded once."""
    dims = tuple(int(x) for x in rng.integers(2, 28, size=3))
    unit = rng.random() < 0.3
    origin = (0.0, 0.0, 0.0) if unit else tuple(float(np.float32(x)) for x in rng.uniform(-3, 3, size=3))
    spacing = (1.0, 1.0, 1.0) if unit else tuple(float(np.float32(x)) for x in rng.uniform(0.05, 2.0, size=3))
    ns = int(rng.integers(2, 5)) if unsteady else 1
    z, y, x = np.meshgrid(*(np.arange(d, dtype=np.float64) for d in dims[::-1]), indexing="ij")
    data = np.zeros((ns, dims[2], dims[1], dims[0], 3), dtype=np.float64)
    for s in range(ns):
        for c in range(3):
            for _ in range(3):
                k = rng.uniform(-0.9, 0.9, size=3); ph = rng.uniform(0, 2 * np.pi); a = rng.uniform(0.3, 1.0)
                data[s, ..., c] += a * np.cos(k[0] * x + k[1] * y + k[2] * z + ph + 0.7 * s)
    # speeds of the order of one cell per unit time in every direction
    data *= np.array(spacing, dtype=np.float64)
    return wl.Field(dims, origin, spacing, data.astype(np.float32), ns, 0.5)


@pytest.mark.parametrize("case", range(28))
def test_random_configuration(S, oracle, wl, case):
    import torch
    rng = np.random.default_rng(1000 + case)
    layout = [1, 2, 3, 4, 5, 6, 7][case % 7]
    unsteady = (case // 7) % 2 == 1
    fld = _random_field(wl, rng, unsteady)
    n = int(rng.choice([1, 37, 3000, 66000, 70001]))
    ext = np.array([(d - 1) * s for d, s in zip(fld.dims, fld.spacing)], dtype=np.float64)
    seeds = (np.array(fld.origin) + rng.random((n, 3)) * ext * 1.02 - 0.01 * ext).astype(np.float32)   # a few start outside
    integ = int(rng.integers(0, 2))
    stride = int(rng.choice([1, 2, 3, 4, 6, 8, 16, 24]))
    kw = dict(integrator=integ, h=float(np.float32(rng.uniform(0.05, 0.6))), max_steps=int(rng.integers(1, 160)),
              vmin=float(rng.choice([0.0, 1e-6, 0.2])), capacity=int(rng.integers(1, 30)), stride=stride,
              t0=float(np.float32(rng.uniform(-0.5, 1.0))) if unsteady else 0.0)
    if integ == 1:
        kw.update(h_min=float(np.float32(rng.uniform(0.005, 0.05))), h_max=float(np.float32(rng.uniform(0.6, 1.5))),
                  atol=float(rng.choice([1e-3, 1e-5])), rtol=float(rng.choice([1e-3, 1e-5])))
    tm = int(rng.integers(0, 2)) if unsteady else 0
    g = oracle.grid(fld.data, fld.dims, fld.origin, fld.spacing, fld.nslices, fld.slice_dt, tm)
    ref = oracle.streamlines(g, seeds, oracle.params(**kw), "f32")
    f = gpu_field(S, torch, fld, layout)
    out = gpu_streamlines(S, torch, f, seeds, time_mode=tm, **kw) if unsteady else gpu_streamlines(S, torch, f, seeds, **kw)
    assert_same(out, ref, "case %d layout %d %s n=%d dims=%s" % (case, layout, kw, n, fld.dims))


@pytest.mark.parametrize("case", range(14))
def test_random_brick_configuration(S, oracle, wl, case):
    """The same for brick-decomposed fields: random brick grids (dims not divisible by the grid, 1-3 bricks per axis),
    ghost width 1 or 2, both integrators, the three round schedules (A9's observable rounds, budgeted rounds + ring
    finish, one launch over the ring) and seed counts on both sides of the sort threshold.  Per-particle outputs,
    totals and (where observed) the round table are compared with the oracle's brick rounds."""
    import torch
    rng = np.random.default_rng(5000 + case)
    N = tuple(int(x) for x in rng.integers(12, 34, size=3))
    nb = tuple(int(x) for x in rng.integers(1, 4, size=3))
    ghost = int(rng.integers(1, 3))
    z, y, x = np.meshgrid(*(np.arange(d, dtype=np.float64) for d in N[::-1]), indexing="ij")
    data = np.zeros((1, N[2], N[1], N[0], 3), dtype=np.float64)
    for c in range(3):
        for _ in range(3):
            k = rng.uniform(-0.7, 0.7, size=3); ph = rng.uniform(0, 2 * np.pi)
            data[0, ..., c] += rng.uniform(0.3, 0.9) * np.cos(k[0] * x + k[1] * y + k[2] * z + ph)
    fld = wl.Field(N, (0.0, 0.0, 0.0), (1.0, 1.0, 1.0), data.astype(np.float32))
    n = int(rng.choice([500, 20000, 66000]))
    seeds = (rng.random((n, 3)) * (np.array(N) - 1.0)).astype(np.float32)
    integ = int(rng.integers(0, 2))
    kw = dict(integrator=integ, h=0.25, max_steps=int(rng.integers(20, 200)), vmin=1e-6, capacity=int(rng.integers(2, 20)),
              stride=int(rng.choice([1, 3, 4, 8])))
    if integ == 1:
        kw.update(h_min=0.01, h_max=float(rng.choice([0.5, 1.0])), atol=1e-4, rtol=1e-4)
    boxes = wl.brick_boxes(fld.dims, nb, ghost)
    cut = wl.cut_bricks(fld, nb, ghost)
    bricks = [oracle.grid(a, None, fld.origin, fld.spacing, gdims=fld.dims, lo=lo, hi=hi) for a, (lo, hi) in zip(cut, boxes)]
    ref = oracle.brick_advect(bricks, nb, seeds, oracle.params(**kw), "f32")
    arrays = [torch.from_numpy(a).cuda() for a in cut]
    layout = int(rng.choice([0, 3, 4, 5]))
    f = S.streami_field_create_bricked(fld.dims, fld.origin, fld.spacing, nb, ghost, arrays, layout)
    d_seeds = torch.from_numpy(seeds).cuda()
    nbricks = nb[0] * nb[1] * nb[2]
    for mode in ("observed", "auto", "ring"):
        if mode == "ring" and integ == 1:
            continue                                      # the one-launch ring is RK4 only
        verts = torch.full((3, n, kw["capacity"]), float("nan"), dtype=torch.float32, device="cuda")
        counts = torch.full((n,), -1, dtype=torch.int32, device="cuda")
        steps = torch.full((n,), -1, dtype=torch.int32, device="cuda")
        status = torch.full((n,), -1, dtype=torch.int32, device="cuda")
        final = torch.zeros((3, n), dtype=torch.float32, device="cuda")
        totals = torch.zeros(4, dtype=torch.int64, device="cuda")
        prm = S.params(out_steps=steps, out_status=status, out_final=final, out_totals=totals, **kw)
        rcounts = torch.zeros((512, nbricks), dtype=torch.int32, device="cuda") if mode == "observed" else None
        try:
            if mode == "ring":
                S.streami_set_option("brick_round_steps", -2)
            nrounds, trunc = S.streami_brick_advect(f, d_seeds, prm, verts, counts, rcounts)
            torch.cuda.synchronize()
        finally:
            S.streami_set_option("brick_round_steps", 0)
        what = "brick case %d %s N=%s nb=%s ghost=%d %s" % (case, mode, N, nb, ghost, kw)
        out = dict(vertices=verts.cpu().numpy(), counts=counts.cpu().numpy().astype(np.uint32),
                   steps=steps.cpu().numpy().astype(np.uint32), status=status.cpu().numpy().astype(np.uint32),
                   final=final.cpu().numpy(), totals=totals.cpu().numpy().astype(np.uint64))
        assert not trunc, what
        assert_same(out, ref, what)
        assert int(out["totals"][3]) == int(ref.totals[3]), what + " hand-offs"
        if mode == "observed":
            assert nrounds == ref.nrounds, what
            assert np.array_equal(rcounts.cpu().numpy()[:nrounds].astype(np.int64), ref.round_counts[:nrounds].astype(np.int64)), what
