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
