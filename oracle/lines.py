"""TEST INFRASTRUCTURE ONLY -- plain definitions of the polyline assembly (the paper's getLines /
assembleOutput), written out in numpy loops.

streamline_lines: line id = the stored vertices 0..counts[id]-1 of particle id, in step order.
streak_lines:     line i = the particles of rake point i that are alive (status 0 during a run,
                  2 = alive at the end), from the youngest release to the oldest.
Both return (offsets [lines+1] uint64, points [total, 3]): offsets = exclusive prefix sum of the line
lengths.  Pinned in tests/test_oracle_pins.py by a hand-written example.
"""
import numpy as np


def streamline_lines(vertices, counts):
    """vertices [3][n][capacity], counts [n]."""
    n = counts.shape[0]
    offsets = np.zeros(n + 1, dtype=np.uint64)
    pts = []
    for i in range(n):
        c = int(counts[i])
        offsets[i + 1] = offsets[i] + np.uint64(c)
        for k in range(c):
            pts.append((vertices[0, i, k], vertices[1, i, k], vertices[2, i, k]))
    return offsets, np.array(pts, dtype=vertices.dtype).reshape(-1, 3)


def streak_lines(vertices, status, released=None):
    """vertices [3][nsteps][m], status [nsteps*m] (release-major); only releases j < released exist."""
    nsteps, m = vertices.shape[1], vertices.shape[2]
    released = nsteps if released is None else released
    st = np.asarray(status).reshape(nsteps, m)
    offsets = np.zeros(m + 1, dtype=np.uint64)
    pts = []
    for i in range(m):
        c = 0
        for j in range(released - 1, -1, -1):
            if st[j, i] in (0, 2):
                pts.append((vertices[0, j, i], vertices[1, j, i], vertices[2, j, i]))
                c += 1
        offsets[i + 1] = offsets[i] + np.uint64(c)
    return offsets, np.array(pts, dtype=vertices.dtype).reshape(-1, 3)
