"""Full-map fp64 reference for config C5 by the exact x-collapse.  Calls only `oracle/`.

C5 has R = I, so a cell's detector-plane coordinates are (Y, Z) = (y, z) and q_x = 0 (Eq. 41): the 256 cells of
one x-row share one phase for every detector point, and the sums of Eq. 42-47 (L353-L368) over the row collapse
exactly to ONE term carrying the row's summed weights.  The summed weights are formed in fp64 and handed to the
oracle as a float32 pair hi + lo at the same position (hi = fp32(w), lo = fp32(w - hi): the oracle only takes
float32 arrays; the residual is below 2^-48 |w|), so `oracle.amplitudes` is called unchanged on 2 x 65 536 cells
instead of 16 777 216: the full 512 x 512 map is 3.4e10 pair evaluations -- about a minute on 16 cores.

    python tests/c5_reference.py        # self-check on the reduced C5 (plain oracle loop vs collapse)
"""
from __future__ import annotations

import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def collapse_x(wl):
    """(pos, N, m) float32 arrays of the collapsed sample: for each distinct (y, z) of `wl` (an unrotated sample)
    two cells at (0, y, z) carrying the hi and lo float32 parts of the row's fp64 weight sums."""
    assert np.array_equal(np.asarray(wl.R, dtype=np.float64), np.eye(3)), "the x-collapse needs R = I (q_x = 0)"
    yz = np.ascontiguousarray(wl.pos[:, 1:3])
    key = yz.view([("y", np.float32), ("z", np.float32)]).ravel()
    uniq, inv = np.unique(key, return_inverse=True)
    n = uniq.shape[0]
    w = np.zeros((n, 4), dtype=np.float64)
    if wl.N is not None:
        w[:, 0] = np.bincount(inv, weights=wl.N.astype(np.float64), minlength=n)
    if wl.m is not None:
        for c in range(3):
            w[:, 1 + c] = np.bincount(inv, weights=wl.m[:, c].astype(np.float64), minlength=n)
    hi = w.astype(np.float32)
    lo = (w - hi.astype(np.float64)).astype(np.float32)
    pos = np.zeros((2 * n, 3), dtype=np.float32)
    pos[:n, 1], pos[:n, 2] = uniq["y"], uniq["z"]
    pos[n:] = pos[:n]
    wc = np.concatenate([hi, lo], axis=0)
    return pos, np.ascontiguousarray(wc[:, 0]), np.ascontiguousarray(wc[:, 1:4])


def full_reference(oracle, wl, idx=None):
    """Oracle amplitudes A [8, n] (fp64) of the unrotated workload `wl` at the detector points `idx` (all by default)
    through the collapsed sample, plus the tolerance denominators sum_j |w_cj| of the ORIGINAL cells."""
    qy, qz, th = oracle.grid_points(wl.grid)
    if idx is not None:
        qy, qz, th = qy[idx], qz[idx], th[idx]
    pos, N, m = collapse_x(wl)
    A = oracle.amplitudes(pos, N if wl.N is not None else None, m if wl.m is not None else None, None, qy, qz)
    wsum = np.zeros(4)
    if wl.N is not None:
        wsum[0] = np.abs(wl.N.astype(np.float64)).sum()
    if wl.m is not None:
        wsum[1:] = np.abs(wl.m.astype(np.float64)).sum(axis=0)
    return A, wsum, th


def self_check():
    """Collapse vs the plain loop of the oracle on the reduced C5 (32^3 block, full detector)."""
    import nms_inputs as ni
    import oracle
    wl = ni.make_config("C5", small=True)
    qy, qz, th = oracle.grid_points(wl.grid)
    A_plain, wsum_plain = oracle.amplitudes(wl.pos, wl.N, wl.m, wl.R, qy, qz, return_wsum=True)
    A_col, wsum, _ = full_reference(oracle, wl)
    err = np.abs(A_col - A_plain).max(axis=1) / np.repeat(wsum_plain, 2)
    assert np.allclose(wsum, wsum_plain, rtol=1e-12)
    return float(err.max())


if __name__ == "__main__":
    print("max |A_collapse - A_plain| / sum|w| on the reduced C5:", self_check())
