"""The identity behind the interpolating amplitude kernel (csrc/k_amp_interp.cu), checked with the fp64 oracle (no GPU).

On a detector line of equally spaced abscissae q_k = q_0 + k d at a fixed direction, the phasors of one cell obey
z_{k-1} + z_{k+1} = 2 cos(d p) z_k (p: the cell's projection on the direction), so the sums of Eq. 42-47 (L353-L368)
at an odd point are the sums at its two neighbours taken with the weights w / (2 cos(d p)):

    A_c(q_k) = B_c(q_{k-1}) + B_c(q_{k+1}),    B_c(q) = sum_j (h_j w_cj) exp(-i q p_j),  h_j = 1 / (2 cos(d p_j)).

The kernel generates only the even points and relies on exactly this; here both sides come from `oracle.amplitudes`
(the right-hand side with h-weighted weight arrays), for a polar direction and for a Cartesian row.
"""
import numpy as np
import pytest

import nms_inputs as ni


@pytest.mark.parametrize("line", ["polar", "cartesian"])
def test_odd_points_are_sums_of_h_weighted_neighbours(oracle_mod, line):
    rng = np.random.Generator(np.random.Philox(777))
    W = 600
    pos = rng.uniform(-20, 20, size=(W, 3)).astype(np.float32)
    N = rng.uniform(0.5, 1.5, size=W).astype(np.float32)
    m = rng.normal(size=(W, 3)).astype(np.float32)
    R = ni.rot_z(25.0) @ ni.rot_y(40.0)
    rp = pos.astype(np.float64) @ R.T                      # r' = R r (Eq. 38-40): detector plane (Y, Z) = (r'_y, r'_z)
    mr = (m.astype(np.float64) @ R.T)                      # m' = R m (reading 2), rotated here so that R = I below
    pos_r, m_r = rp.astype(np.float32), mr.astype(np.float32)
    rp = pos_r.astype(np.float64)                          # the oracle sees the rounded rotated positions
    d, n = 0.021, 9                                        # step phase <= 0.021 * 35 rad = 0.12 cycle
    k = np.arange(n)
    if line == "polar":
        th = 0.83                                          # theta from +z towards +y (reading 5)
        q = 0.4 + d * k
        qy, qz = q * np.sin(th), q * np.cos(th)
        p = np.sin(th) * rp[:, 1] + np.cos(th) * rp[:, 2]
    else:
        qy, qz = np.full(n, 0.37), -0.05 + d * k           # a row of a Cartesian detector: the line runs along q_z
        p = rp[:, 2]
    assert np.abs(d * p).max() < 0.2 * 2 * np.pi           # the kernel's admission rule
    h = 1.0 / (2.0 * np.cos(d * p))
    A, wsum = oracle_mod.amplitudes(pos_r, N, m_r, None, qy, qz, return_wsum=True)
    Nh = (N.astype(np.float64) * h).astype(np.float32)
    mh = (m_r.astype(np.float64) * h[:, None]).astype(np.float32)
    B = oracle_mod.amplitudes(pos_r, Nh, mh, None, qy, qz)
    odd = k[1:-1:2]
    for c in range(4):
        got = B[2 * c:2 * c + 2, odd - 1] + B[2 * c:2 * c + 2, odd + 1]
        # the fp32 rounding of the h-weighted weights is the only difference: <= 2^-24 per weight
        assert np.abs(got - A[2 * c:2 * c + 2, odd]).max() <= 2.0 ** -23 * wsum[c]
    # and it is an identity of the odd points only: the same sum at an even point's neighbours does not give that point
    # unless its spacing is the line's
    wrong = B[0:2, 0] + B[0:2, 3]
    assert np.abs(wrong - A[0:2, 1]).max() > 1e-3 * wsum[0] / np.sqrt(W)
