"""Shared helpers for the GPU parity tests: run the CUDA path through the Python binding of the
C ABI and return numpy arrays shaped like the oracle's results."""
import numpy as np


def gpu_field(S, torch, fld, layout=0):
    data = torch.from_numpy(np.ascontiguousarray(fld.data)).cuda()
    return S.streami_field_create(fld.dims, fld.origin, fld.spacing, fld.nslices, fld.slice_dt, data,
                                  layout)


def gpu_streamlines(S, torch, field, seeds, record=True, fill=float("nan"), **kw):
    n = seeds.shape[0]
    cap = kw.get("capacity", 1)
    d_seeds = torch.from_numpy(np.ascontiguousarray(seeds, dtype=np.float32)).cuda()
    verts = torch.full((3, n, cap), fill, dtype=torch.float32, device="cuda") if record else None
    counts = torch.full((n,), -1, dtype=torch.int32, device="cuda")
    steps = torch.full((n,), -1, dtype=torch.int32, device="cuda")
    status = torch.full((n,), -1, dtype=torch.int32, device="cuda")
    final = torch.zeros((3, n), dtype=torch.float32, device="cuda")
    totals = torch.zeros(4, dtype=torch.int64, device="cuda")
    prm = S.params(out_steps=steps, out_status=status, out_final=final, out_totals=totals, **kw)
    S.streami_trace_streamlines(field, d_seeds, prm, verts, counts)
    torch.cuda.synchronize()
    return dict(vertices=None if verts is None else verts.cpu().numpy(),
                counts=counts.cpu().numpy().astype(np.uint32),
                steps=steps.cpu().numpy().astype(np.uint32),
                status=status.cpu().numpy().astype(np.uint32), final=final.cpu().numpy(),
                totals=totals.cpu().numpy().astype(np.uint64))


def assert_same(gpu, ref, what="", vertices=True):
    """Bit-exact comparison of a GPU result dict with an oracle Result."""
    assert np.array_equal(gpu["status"], ref.status), what + " status"
    assert np.array_equal(gpu["steps"], ref.steps), what + " steps"
    assert np.array_equal(gpu["counts"], ref.counts), what + " counts"
    assert np.array_equal(gpu["final"].view(np.uint32), ref.final.view(np.uint32)), what + " final"
    if vertices and gpu["vertices"] is not None:
        assert np.array_equal(gpu["vertices"].view(np.uint32), ref.vertices.view(np.uint32)), \
            what + " vertices"
    assert np.array_equal(gpu["totals"][:3], ref.totals[:3]), what + " totals"
