"""Writes tests/golden/c1_oracle_f32.txt: a digest of the fp32 ORACLE's output on config 1
(ABC flow 32^3, 1,024 seeds, RK4 h = 0.01, 1,000 steps).  Calls only oracle/ and the input
generators in workloads/; never the CUDA path.  The digest is a regression guard for the
oracle (a later change to its arithmetic must be deliberate and name the passage that
justifies it in the commit message); it is not a pin -- the pins are closed forms, see
tests/test_oracle_pins.py.

Run from the repo root:  python tests/golden/make_golden.py
"""
import hashlib
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
import oracle          # noqa: E402
import workloads as wl  # noqa: E402


def digest():
    f = wl.abc_field(32)
    g = oracle.grid(f.data, f.dims, f.origin, f.spacing)
    seeds = wl.seeds_uniform(42, 1024, [2 * np.pi] * 3)
    prm = oracle.params(0, h=0.01, max_steps=1000, vmin=1e-6, capacity=1001, stride=1)
    r = oracle.streamlines(g, seeds, prm, "f32")
    v = np.nan_to_num(r.vertices, nan=0.0)
    lines = [
        "# digest of the fp32 oracle on BASELINE.json config 1; written by tests/golden/make_golden.py",
        "field_sha256 " + hashlib.sha256(f.data.tobytes()).hexdigest(),
        "seeds_sha256 " + hashlib.sha256(seeds.tobytes()).hexdigest(),
        "status_hist " + " ".join(str(x) for x in np.bincount(r.status, minlength=5)),
        "steps_sum %d" % int(r.steps.sum()),
        "totals " + " ".join(str(int(x)) for x in r.totals),
        "steps_sha256 " + hashlib.sha256(r.steps.tobytes()).hexdigest(),
        "vertices_sha256 " + hashlib.sha256(v.tobytes()).hexdigest(),
    ]
    for i in (0, 1, 511, 1023):
        k = int(r.counts[i]) - 1
        lines.append("particle %d last_vertex %d %s" % (
            i, k, " ".join(float(r.vertices[c, i, k]).hex() for c in range(3))))
    return "\n".join(lines) + "\n"


if __name__ == "__main__":
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "c1_oracle_f32.txt")
    open(out, "w").write(digest())
    print(open(out).read())
