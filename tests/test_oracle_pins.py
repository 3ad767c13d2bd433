"""Pins of the fp64 oracle against what the paper and the mathematics fix (no GPU).

Each test names the PAPER.md passage it checks.  None of them re-types the
oracle's own formula: closed forms, invariants, an independent brute force in
Python complex arithmetic with a differently derived epilogue (Appendix-A
T-form), expanded forms Eq. 9/15/19-22/28, and values printed in Table II.
"""
import cmath
import math
import os

import numpy as np
import pytest

import nms_inputs as ni
from nms_inputs import KIND_INDEX as KI

GOLD = os.path.join(os.path.dirname(__file__), "golden")
B_H = 2.91e8          # A^-1 m^-1


def _polar(nq=24, nth=32, q0=0.01, q1=3.0):
    return ni.polar_grid(np.linspace(q0, q1, nq), nth)


# --------------------------------------------------------------------------- O1
def test_dimer_closed_form(oracle_mod):
    """Two unit cells at +-d/2: |N~|^2 = 2 + 2 cos(q.d) (north_star; Eq. 42)."""
    d = np.array([0.3, 1.7, -0.9])
    pos = np.stack([d / 2, -d / 2]).astype(np.float32)
    dd = (pos[0].astype(np.float64) - pos[1].astype(np.float64))
    g = _polar()
    qy, qz, th = oracle_mod.grid_points(g)
    A = oracle_mod.amplitudes(pos, np.ones(2, np.float32), None, None, qy, qz)
    f2 = A[0] ** 2 + A[1] ** 2
    np.testing.assert_allclose(f2, 2 + 2 * np.cos(qy * dd[1] + qz * dd[2]), rtol=0, atol=1e-12)
    assert np.all(A[2:] == 0.0)


# --------------------------------------------------------------------------- O2
def test_cartesian_and_list_grid_axis_convention(oracle_mod):
    """include/nms.h: a Cartesian grid has u0 = q_z [n0] (slow index) and u1 = q_y [n1] (fast index); a list grid
    u0 = q_y, u1 = q_z; theta = atan2(q_y, q_z) from +z towards +y (Eq. 6).  Pinned with distinguishable axes: a
    dimer along y only has |N~|^2 = 2 + 2 cos(q_y d), which must vary along u1 and not along u0."""
    d = 3.0
    pos = np.array([[0.0, -d / 2, 0.0], [0.0, d / 2, 0.0]], dtype=np.float32)
    N = np.ones(2, dtype=np.float32)
    qz = np.array([-0.7, 0.1, 0.4], dtype=np.float32)              # u0, n0 = 3
    qy = np.array([-0.9, -0.2, 0.3, 0.8, 1.1], dtype=np.float32)   # u1, n1 = 5
    grid = ni.cartesian_grid(qz, qy)
    gy, gz, th = oracle_mod.grid_points(grid)
    assert np.array_equal(gz.reshape(3, 5), np.repeat(qz.astype(np.float64)[:, None], 5, axis=1))
    assert np.array_equal(gy.reshape(3, 5), np.repeat(qy.astype(np.float64)[None, :], 3, axis=0))
    np.testing.assert_allclose(th, np.arctan2(gy, gz), rtol=0, atol=1e-15)
    A = oracle_mod.amplitudes(pos, N, None, None, gy, gz)
    F2 = (A[0] ** 2 + A[1] ** 2).reshape(3, 5)
    np.testing.assert_allclose(F2, np.repeat((2 + 2 * np.cos(qy.astype(np.float64) * d))[None, :], 3, axis=0), rtol=1e-13)
    assert np.ptp(F2, axis=0).max() < 1e-12 and np.ptp(F2, axis=1).min() > 0.1      # constant along u0, varying along u1
    lst = ni.list_grid(qy[:3], qz)                                  # list: u0 = q_y, u1 = q_z
    ly, lz, lth = oracle_mod.grid_points(lst)
    assert np.array_equal(ly, qy[:3].astype(np.float64)) and np.array_equal(lz, qz.astype(np.float64))
    np.testing.assert_allclose(lth, np.arctan2(ly, lz), rtol=0, atol=1e-15)


def test_forward_amplitude_is_weight_sum(oracle_mod):
    """F(0) = sum w (north_star): at q = 0, A = (sum N, R sum m) with zero imaginary parts."""
    rng = np.random.default_rng(1)
    pos = rng.normal(size=(50, 3)).astype(np.float32)
    N = rng.normal(size=50).astype(np.float32)
    m = rng.normal(size=(50, 3)).astype(np.float32)
    R = ni.rotation_alpha_beta(33.0, -71.0)
    A = oracle_mod.amplitudes(pos, N, m, R, np.zeros(1), np.zeros(1))
    ms = R @ m.astype(np.float64).sum(axis=0)
    np.testing.assert_allclose(A[:, 0], [N.astype(np.float64).sum(), 0, ms[0], 0, ms[1], 0, ms[2], 0], atol=1e-12)


# --------------------------------------------------------------------------- O3
@pytest.mark.parametrize("R", [np.eye(3), ni.rotation_alpha_beta(25.0, 40.0)])
def test_cuboid_lattice_dirichlet_product(oracle_mod, R):
    """Uniform centred cuboid lattice: N~ = prod_d sin(n_d k_d a/2)/sin(k_d a/2), k = R^T q (exact for the lattice)."""
    n, a = (5, 4, 7), 0.5
    pos = ni.cuboid_lattice(*n, a).astype(np.float32)     # multiples of 0.25: exact in fp32
    g = _polar(17, 24, 0.05, 2.5)
    qy, qz, _ = oracle_mod.grid_points(g)
    A = oracle_mod.amplitudes(pos, np.ones(len(pos), np.float32), None, R, qy, qz)
    kap = np.stack([np.zeros_like(qy), qy, qz], axis=1) @ R     # rows: R^T q
    want = np.ones_like(qy)
    for d in range(3):
        den = np.sin(kap[:, d] * a / 2)
        safe = np.where(np.abs(den) < 1e-300, 1.0, den)
        want *= np.where(np.abs(den) < 1e-300, float(n[d]), np.sin(n[d] * kap[:, d] * a / 2) / safe)   # limit n_d at k_d = 0
    np.testing.assert_allclose(A[0], want, atol=1e-10)
    np.testing.assert_allclose(A[1], 0.0, atol=1e-10)


# --------------------------------------------------------------------------- O4
def test_translation_multiplies_by_phase(oracle_mod):
    """Translate all cells by d: A -> e^{-i q.d} A; every |.|^2-type kind is unchanged (north_star)."""
    rng = np.random.default_rng(2)
    pos = (rng.integers(-40, 40, size=(60, 3)) * 0.25).astype(np.float32)
    d = np.array([1.5, -2.25, 0.75], dtype=np.float32)
    N = rng.normal(size=60).astype(np.float32)
    m = rng.normal(size=(60, 3)).astype(np.float32)
    g = _polar(9, 16)
    qy, qz, th = oracle_mod.grid_points(g)
    A0 = oracle_mod.amplitudes(pos, N, m, None, qy, qz)
    A1 = oracle_mod.amplitudes(pos + d, N, m, None, qy, qz)       # exact in fp32 (quarter-integers)
    ph = np.exp(-1j * (qy * float(d[1]) + qz * float(d[2])))
    for c in range(4):
        z0 = A0[2 * c] + 1j * A0[2 * c + 1]
        z1 = A1[2 * c] + 1j * A1[2 * c + 1]
        np.testing.assert_allclose(z1, z0 * ph, atol=1e-11)
    k = ni.ALL_KINDS
    np.testing.assert_allclose(oracle_mod.response(A1, th, k), oracle_mod.response(A0, th, k), atol=1e-9)


# --------------------------------------------------------------------------- O5
def test_rotating_sample_equals_rotating_q(oracle_mod):
    """A_R(q) = (1, R) . A_I(R^T q): rotating the sample by R == rotating q by R^T (north_star; Eq. 38-40)."""
    rng = np.random.default_rng(3)
    pos = rng.normal(scale=3, size=(40, 3)).astype(np.float32)
    N = rng.normal(size=40).astype(np.float32)
    m = rng.normal(size=(40, 3)).astype(np.float32)
    R = ni.rot_z(30.0) @ ni.rot_y(45.0)
    g = _polar(7, 12)
    qy, qz, _ = oracle_mod.grid_points(g)
    AR = oracle_mod.amplitudes(pos, N, m, R, qy, qz)
    k3 = np.stack([np.zeros_like(qy), qy, qz], axis=1) @ R       # R^T q as rows
    AI = oracle_mod.amplitudes(pos, N, m, None, k3[:, 1].copy(), k3[:, 2].copy(), qx=k3[:, 0].copy())
    np.testing.assert_allclose(AR[0:2], AI[0:2], atol=1e-11)
    MI = np.stack([AI[2] + 1j * AI[3], AI[4] + 1j * AI[5], AI[6] + 1j * AI[7]])
    MR = R @ MI
    for a in range(3):
        np.testing.assert_allclose(AR[2 + 2 * a] + 1j * AR[3 + 2 * a], MR[a], atol=1e-11)


def test_rotation_convention_alpha90_sends_z_to_x():
    """L279: alpha = 90 deg, beta = 0 switches to the parallel geometry, i.e. the sample z axis goes onto the beam axis x."""
    R = ni.rotation_alpha_beta(90.0, 0.0)
    np.testing.assert_allclose(R @ np.array([0, 0, 1.0]), [1, 0, 0], atol=1e-15)
    np.testing.assert_allclose(ni.rotation_alpha_beta(20, 50), ni.rot_z(50) @ ni.rot_y(20))


# --------------------------------------------------------------------------- O6
def _brute_force(pos, N, m, R, P, sN, sM, invV, pts):
    """Independent restatement in Python complex arithmetic; epilogue via T = s Mz - c My (Appendix-A form)."""
    out = []
    P = np.asarray(P, float) / np.linalg.norm(P)
    for (qy, qz, th) in pts:
        A = [0j, 0j, 0j, 0j]
        for j in range(len(pos)):
            r = [sum(R[a][b] * float(pos[j][b]) for b in range(3)) for a in range(3)]
            mm = [sum(R[a][b] * float(m[j][b]) for b in range(3)) for a in range(3)]
            e = cmath.exp(-1j * (qy * r[1] + qz * r[2]))
            A[0] += float(N[j]) * e
            for a in range(3):
                A[1 + a] += mm[a] * e
        n_, mx, my, mz = A[0] * sN, A[1] * sM, A[2] * sM, A[3] * sM
        s, c = math.sin(th), math.cos(th)
        T = s * mz - c * my
        Pi = -P[0] * mx + (P[1] * c - P[2] * s) * T
        nuc = abs(n_) ** 2
        mag = abs(mx) ** 2 + abs(T) ** 2
        proj = abs(Pi) ** 2
        nm = 2 * (n_ * Pi.conjugate()).real
        sf = mag - proj
        chi = 2 * (P[1] * s + P[2] * c) * (T * mx.conjugate()).imag
        vals = {"NUC": nuc, "MAG": mag, "UNPOL": nuc + mag, "PROJ": proj, "NM": nm, "SF": sf, "CHI": chi,
                "PM": sf + chi, "MP": sf - chi, "PP": nuc + nm + proj, "MM": nuc - nm + proj,
                "POL_PLUS": nuc + nm + proj + sf + chi, "POL_MINUS": nuc - nm + proj + sf - chi}
        out.append((A, [invV * vals[k] for k in ni.KINDS]))
    return out


@pytest.mark.parametrize("P", [(0, 0, 1), (1, 0, 0), (0.3, -0.5, 0.81)])
def test_brute_force_tiny(oracle_mod, P):
    """Brute force on 7 cells x 12 points with general P, R, N, m, scales (north_star 'brute force on tiny inputs')."""
    rng = np.random.default_rng(4)
    pos = rng.normal(scale=2, size=(7, 3)).astype(np.float32)
    N = rng.normal(size=7).astype(np.float32)
    m = rng.normal(size=(7, 3)).astype(np.float32)
    R = ni.rotation_alpha_beta(17.0, 123.0)
    qyf = rng.normal(size=12).astype(np.float32)
    qzf = rng.normal(size=12).astype(np.float32)
    g = ni.list_grid(qyf, qzf)
    qy, qz, th = oracle_mod.grid_points(g)
    np.testing.assert_array_equal(qy, qyf.astype(np.float64))
    A = oracle_mod.amplitudes(pos, N, m, R, qy, qz)
    sN, sM, invV = 0.7, 1.9, 0.013
    resp = oracle_mod.response(A, th, ni.ALL_KINDS, P=P, sN=sN, sM=sM, invV=invV)
    ref = _brute_force(pos, N, m, R, P, sN, sM, invV, [(qy[i], qz[i], math.atan2(qy[i], qz[i])) for i in range(12)])
    for i, (Ai, vals) in enumerate(ref):
        for c in range(4):
            assert abs(complex(A[2 * c, i], A[2 * c + 1, i]) - Ai[c]) < 1e-12
        np.testing.assert_allclose(resp[:, i], vals, rtol=1e-10, atol=1e-12)


# --------------------------------------------------------------------------- O8
def test_halpern_johnson_vector_is_transverse(oracle_mod):
    """Q . q^ = 0 (Eq. 5) and Q equals the component form of Eq. 7 (L62)."""
    rng = np.random.default_rng(5)
    nq = 64
    amp = rng.normal(size=(8, nq))
    th = rng.uniform(0, 2 * np.pi, nq)
    _, Q = oracle_mod.response(amp, th, [0], return_Q=True)
    Qc = [Q[0] + 1j * Q[1], Q[2] + 1j * Q[3], Q[4] + 1j * Q[5]]
    Mx, My, Mz = amp[2] + 1j * amp[3], amp[4] + 1j * amp[5], amp[6] + 1j * amp[7]
    s, c = np.sin(th), np.cos(th)
    np.testing.assert_allclose(s * Qc[1] + c * Qc[2], 0, atol=1e-13)
    np.testing.assert_allclose(Qc[0], -Mx, atol=1e-13)
    np.testing.assert_allclose(Qc[1], -My * c * c + Mz * s * c, atol=1e-13)
    np.testing.assert_allclose(Qc[2], My * s * c - Mz * s * s, atol=1e-13)


# --------------------------------------------------------------------------- O9
def test_channel_sum_rules(oracle_mod):
    """Eq. 11-13, 16-17, 23-24, 27 (L84-L165): relations between the 13 kinds, general P."""
    rng = np.random.default_rng(6)
    nq = 50
    amp = rng.normal(size=(8, nq))
    th = rng.uniform(0, 2 * np.pi, nq)
    r = oracle_mod.response(amp, th, ni.ALL_KINDS, P=(0.2, 0.6, -0.7), sN=1.3, sM=0.4, invV=2.0)
    k = {n: r[i] for n, i in KI.items()}
    np.testing.assert_allclose(k["SF"], k["MAG"] - k["PROJ"], atol=1e-12)
    np.testing.assert_allclose(k["PM"] - k["MP"], 2 * k["CHI"], atol=1e-12)
    np.testing.assert_allclose(k["PM"] + k["MP"], 2 * k["SF"], atol=1e-12)
    np.testing.assert_allclose(k["PP"] - k["MM"], 2 * k["NM"], atol=1e-12)
    np.testing.assert_allclose(k["POL_PLUS"], k["PP"] + k["PM"], atol=1e-12)
    np.testing.assert_allclose(k["POL_MINUS"], k["MM"] + k["MP"], atol=1e-12)
    np.testing.assert_allclose(0.5 * (k["PP"] + k["MM"] + k["PM"] + k["MP"]), k["UNPOL"], atol=1e-12)
    np.testing.assert_allclose(k["UNPOL"], k["NUC"] + k["MAG"], atol=1e-12)     # Eq. 28: N + M
    assert np.all(k["MAG"] >= -1e-12) and np.all(k["PROJ"] >= -1e-12) and np.all(k["SF"] >= -1e-9)


# --------------------------------------------------------------------------- O10
def test_expanded_forms_perpendicular_and_parallel(oracle_mod):
    """Expanded forms Eq. 9, 15, 19-20, 25, 28 (P = e_z) and Eq. 10, 21-22, 26 (P = e_x), with the
    parenthesis fixes of DESIGN.md reading 6 (b_H folded into the scales)."""
    rng = np.random.default_rng(7)
    nq = 40
    amp = rng.normal(size=(8, nq))
    th = rng.uniform(0, 2 * np.pi, nq)
    Nn = amp[0] + 1j * amp[1]
    Mx, My, Mz = amp[2] + 1j * amp[3], amp[4] + 1j * amp[5], amp[6] + 1j * amp[7]
    s, c = np.sin(th), np.cos(th)
    a2 = lambda z: (z * z.conjugate()).real
    cr = lambda u, v: (u * v.conjugate() + u.conjugate() * v).real
    # ---- P = e_z
    r = oracle_mod.response(amp, th, ni.ALL_KINDS, P=(0, 0, 1))
    k = {n: r[i] for n, i in KI.items()}
    eq9 = a2(My) * s * s * c * c + a2(Mz) * s ** 4 - cr(My, Mz) * s ** 3 * c
    np.testing.assert_allclose(k["PROJ"], eq9, atol=1e-11)
    chi15 = (Mx * My.conjugate() - Mx.conjugate() * My) * c * c - (Mx * Mz.conjugate() - Mx.conjugate() * Mz) * s * c
    np.testing.assert_allclose(k["CHI"], (-1j * chi15).real, atol=1e-11)
    np.testing.assert_allclose((-1j * chi15).imag, 0, atol=1e-11)
    sf20 = a2(Mx) + a2(My) * c ** 4 + a2(Mz) * s * s * c * c - cr(My, Mz) * s * c ** 3
    np.testing.assert_allclose(k["PM"], sf20 + (-1j * chi15).real, atol=1e-11)
    np.testing.assert_allclose(k["MP"], sf20 - (-1j * chi15).real, atol=1e-11)
    nsf19 = a2(Nn) + eq9
    inter = -cr(Nn, Mz) * s * s + cr(Nn, My) * s * c
    np.testing.assert_allclose(k["PP"], nsf19 + inter, atol=1e-11)
    np.testing.assert_allclose(k["MM"], nsf19 - inter, atol=1e-11)
    eq28 = a2(Nn) + a2(Mx) + a2(My) * c * c + a2(Mz) * s * s - cr(My, Mz) * s * c
    np.testing.assert_allclose(k["UNPOL"], eq28, atol=1e-11)
    np.testing.assert_allclose(k["POL_PLUS"], eq28 + inter + (-1j * chi15).real, atol=1e-11)      # Eq. 25
    np.testing.assert_allclose(k["POL_MINUS"], eq28 - inter - (-1j * chi15).real, atol=1e-11)
    # ---- P = e_x
    r = oracle_mod.response(amp, th, ni.ALL_KINDS, P=(1, 0, 0))
    k = {n: r[i] for n, i in KI.items()}
    np.testing.assert_allclose(k["PROJ"], a2(Mx), atol=1e-11)                                   # Eq. 10
    np.testing.assert_allclose(k["CHI"], 0, atol=1e-11)                                          # L100, L132
    np.testing.assert_allclose(k["PP"], a2(Nn) + a2(Mx) - cr(Nn, Mx), atol=1e-11)                # Eq. 21 upper sign
    np.testing.assert_allclose(k["MM"], a2(Nn) + a2(Mx) + cr(Nn, Mx), atol=1e-11)
    sf22 = a2(My) * c * c + a2(Mz) * s * s - cr(My, Mz) * s * c
    np.testing.assert_allclose(k["PM"], sf22, atol=1e-11)                                        # Eq. 22
    np.testing.assert_allclose(k["MP"], sf22, atol=1e-11)
    np.testing.assert_allclose(k["UNPOL"], eq28, atol=1e-11)                                     # Eq. 29 == Eq. 28


# --------------------------------------------------------------------------- O11
@pytest.mark.parametrize("n", [(0, 0, 1), (0.36, -0.48, 0.8)])
def test_uniform_magnetisation_angular_factors(oracle_mod, n):
    """Uniform m = n on any lattice: M~ = n F, hence Eq. 60-63 (L451-L457) angular factors exactly;
    for n = e_z the magnetic cross section is |F|^2 sin^2(theta) (north_star)."""
    pos = ni.sphere_node_centred(6.0, 1.0).astype(np.float32)
    W = len(pos)
    m = np.tile(np.asarray(n, np.float32), (W, 1))
    g = _polar(20, 36, 0.02, 2.0)
    qy, qz, th = oracle_mod.grid_points(g)
    A = oracle_mod.amplitudes(pos, np.ones(W, np.float32), m, None, qy, qz)
    r = oracle_mod.response(A, th, ni.ALL_KINDS)
    k = {nm: r[i] for nm, i in KI.items()}
    F2 = k["NUC"]
    nn = np.asarray(n, np.float32).astype(np.float64)
    s, c = np.sin(th), np.cos(th)
    np.testing.assert_allclose(k["MAG"], F2 * (nn[0] ** 2 + nn[1] ** 2 * c * c + nn[2] ** 2 * s * s - 2 * nn[1] * nn[2] * s * c), rtol=1e-9, atol=1e-7)
    np.testing.assert_allclose(k["NM"], 2 * F2 * (nn[1] * s * c - nn[2] * s * s), rtol=1e-9, atol=1e-7)
    np.testing.assert_allclose(k["PROJ"], F2 * (nn[1] * s * c - nn[2] * s * s) ** 2, rtol=1e-9, atol=1e-7)
    np.testing.assert_allclose(k["CHI"], 0, atol=1e-7)
    if n == (0, 0, 1):
        np.testing.assert_allclose(k["SF"], F2 * s * s * c * c, rtol=1e-9, atol=1e-7)          # L124: sin^2 cos^2 at saturation


# --------------------------------------------------------------------------- O12
def test_chiral_symmetries(oracle_mod):
    """L100: chi = 0 for M(r) = M(-r) and for M(r) = -M(-r); chi = 0 for P || e_x; chi(-q) = -chi(q), others even (L183)."""
    pos = ni.sphere_node_centred(4.0, 1.0)
    rng = np.random.default_rng(8)
    # pair every cell with its inversion image
    key = {tuple(p): i for i, p in enumerate(pos)}
    inv = np.array([key[tuple(-p)] for p in pos])
    base = rng.normal(size=(len(pos), 3))
    m_even = base + base[inv]
    m_odd = base - base[inv]
    g = _polar(10, 16, 0.1, 2.5)
    qy, qz, th = oracle_mod.grid_points(g)
    for mm in (m_even, m_odd):
        A = oracle_mod.amplitudes(pos.astype(np.float32), None, mm.astype(np.float32), None, qy, qz)
        chi = oracle_mod.response(A, th, [KI["CHI"]])
        mag = oracle_mod.response(A, th, [KI["MAG"]])
        assert np.max(np.abs(chi)) < 1e-9 * np.max(mag)
    A = oracle_mod.amplitudes(pos.astype(np.float32), None, base.astype(np.float32), None, qy, qz)
    r = oracle_mod.response(A, th, ni.ALL_KINDS)
    assert np.max(np.abs(r[KI["CHI"]])) > 1e-3 * np.max(r[KI["MAG"]])          # generic texture: chi != 0
    np.testing.assert_allclose(oracle_mod.response(A, th, [KI["CHI"]], P=(1, 0, 0)), 0, atol=1e-10)
    # Friedel partner: theta -> theta + pi is index shift by n_theta/2 on the polar grid
    r2 = r.reshape(len(ni.KINDS), g.n0, g.n1)
    sh = np.roll(r2, -g.n1 // 2, axis=2)
    for name, i in KI.items():
        if name == "CHI":
            np.testing.assert_allclose(sh[i], -r2[i], atol=1e-6 * np.max(np.abs(r2[i])))
        elif name in ("NUC", "MAG", "UNPOL", "PROJ", "SF"):
            np.testing.assert_allclose(sh[i], r2[i], atol=1e-6 * np.max(np.abs(r2[i])))
    I = oracle_mod.azimuthal_polar(r, g.n0, g.n1)
    assert np.max(np.abs(I[KI["CHI"]])) < 1e-6 * np.max(np.abs(r[KI["CHI"]]))        # L183: chi averages to zero


# --------------------------------------------------------------------------- O13
def _read_golden(name):
    out = {}
    for line in open(os.path.join(GOLD, name)):
        if line.startswith("#") or not line.strip():
            continue
        k, v = line.split()
        out[k] = float(v)
    return out


def _table2_setup(oracle_mod, q, nth):
    pos, N, m = ni.uniform_sphere_sample(20.0, 1.0, (0, 0, 1))
    W = len(pos)
    assert W == 33401
    V_cell = 1e-27                        # m^3 (a = 1 nm)
    N0, M0 = 8.0e14, 1.7e6                # m^-2, A/m (L524)
    sN, sM, invV = N0 * V_cell, B_H * M0 * V_cell, 1.0 / (W * V_cell)
    g = ni.polar_grid(q, nth)
    qy, qz, th = oracle_mod.grid_points(g)
    A = oracle_mod.amplitudes(pos, N, m, None, qy, qz)
    r = oracle_mod.response(A, th, ni.ALL_KINDS, sN=sN, sM=sM, invV=invV)      # m^-1
    return g, r * 1e-2, W                 # cm^-1


def test_table2_forward_intensities(oracle_mod):
    """Table II (L526-L541): azimuthally averaged I(q -> 0) in cm^-1 for the D = 40 nm sphere; exact for
    the lattice sphere once V_s is replaced by W V_cell (0.3 % apart), so compare value / (W V_cell) * V_s."""
    gold = _read_golden("table2_I0.txt")
    g, r, W = _table2_setup(oracle_mod, np.array([1e-6]), 64)
    I = oracle_mod.azimuthal_polar(r, 1, 64)[:, 0]
    V_s = 4.0 / 3.0 * np.pi * 20.0 ** 3
    for name, val in gold.items():
        got = I[KI[name]] * V_s / W
        assert abs(got - val) <= 0.0006e5, (name, got, val)      # ~half a unit of the last printed digit (x.xxx e5)


def test_sphere_form_factor_shape(oracle_mod):
    """Eq. 59 (L449): lattice sphere vs 9 N0^2 V_s g(qR)^2 in the continuum limit, few-% level at qR <~ 6 maxima."""
    q = np.linspace(0.01, 0.42, 30)
    g, r, W = _table2_setup(oracle_mod, q, 8)
    I = oracle_mod.azimuthal_polar(r, len(q), 8)[KI["NUC"]]
    v = q.astype(np.float32).astype(np.float64) * 20.0
    gg = (np.sin(v) - v * np.cos(v)) / v ** 3
    want = 9 * (8.0e14) ** 2 * (W * 1e-27) * gg ** 2 * 1e-2
    assert np.max(np.abs(I - want)) < 0.01 * want[0]


def test_table2_pmax(oracle_mod):
    """Table II p_max column: 2 pi^2 x (Eq. 34-35 taken literally) at r = xi_max R (reading 9).
    Approximate pin (lattice + q-range truncation at q_max = 3 nm^-1): 4 %."""
    gold = _read_golden("table2_pmax.txt")
    q = np.linspace(0.0, 3.0, 601)
    g, r, W = _table2_setup(oracle_mod, q, 16)
    I = oracle_mod.azimuthal_polar(r, len(q), 16) * 1e-7          # cm^-1 -> nm^-1
    xi = math.sqrt(105.0) / 5.0 - 1.0
    c, p = oracle_mod.correlation(I, q.astype(np.float32).astype(np.float64), np.array([xi * 20.0]))
    for name, val in gold.items():
        got = 2 * np.pi ** 2 * p[KI[name], 0]
        assert abs(got - val) < 0.04 * val, (name, got, val)
    # c(r) = 0 beyond the largest distance (L270), within truncation ripples
    c2, _ = oracle_mod.correlation(I, q.astype(np.float32).astype(np.float64), np.array([0.0, 45.0, 60.0]))
    assert np.all(np.abs(c2[KI["NUC"], 1:]) < 0.01 * c2[KI["NUC"], 0])


# --------------------------------------------------------------------------- O14 (vortex)
def test_linear_vortex_sphere_chiral_sign_and_shape(oracle_mod):
    """Sec. IV B (Eq. 90-96) with the factor-R fix of reading 6:
    chi-term = 18 V_s M0 M1 R g g' sin^2(th) cos(th), N~ real, M~_x,y imaginary; continuum limit, 5 % of max."""
    Rr = 20.0
    pos, N, m = ni.linear_vortex_sphere_sample(Rr, 1.0)
    W = len(pos)
    q = np.linspace(0.02, 0.4, 12)
    g = ni.polar_grid(q, 24)
    qy, qz, th = oracle_mod.grid_points(g)
    A = oracle_mod.amplitudes(pos, N, m, None, qy, qz)
    r = oracle_mod.response(A, th, ni.ALL_KINDS, invV=1.0 / W)
    qq = np.repeat(q.astype(np.float32).astype(np.float64), 24)
    v = qq * Rr
    gg = (np.sin(v) - v * np.cos(v)) / v ** 3
    gp = ((v * v - 3) * np.sin(v) + 3 * v * np.cos(v)) / v ** 4
    M1 = 5.0 / Rr
    s, c = np.sin(th), np.cos(th)
    chi = 18 * W * 1.0 * M1 * Rr * gg * gp * s * s * c
    mag = 9 * W * (gg ** 2 + M1 ** 2 * Rr ** 2 * gp ** 2) * s * s                    # Eq. 93 with M1^2 R^2
    nmx = -18 * W * gg ** 2 * s * s                                                  # Eq. 94
    assert np.max(np.abs(r[KI["CHI"]] - chi)) < 0.05 * np.max(np.abs(chi))
    assert np.max(np.abs(r[KI["MAG"]] - mag)) < 0.05 * np.max(np.abs(mag))
    assert np.max(np.abs(r[KI["NM"]] - nmx)) < 0.05 * np.max(np.abs(nmx))
    # symmetric lattice: N~ and M~_z real, M~_x purely imaginary, M~_y ~ q^_x = 0 on the detector (Eq. 91)
    assert np.max(np.abs(A[1])) < 1e-9 * np.max(np.abs(A[0]))
    assert np.max(np.abs(A[2])) < 1e-9 * np.max(np.abs(A[3]))
    assert max(np.max(np.abs(A[4])), np.max(np.abs(A[5]))) < 1e-9 * np.max(np.abs(A[3]))
    assert np.max(np.abs(A[7])) < 1e-9 * np.max(np.abs(A[6]))


# --------------------------------------------------------------------------- O15
def test_azimuthal_mean_of_trigonometric_maps(oracle_mod):
    """Eq. 30 (L181) by the periodic trapezoid is exact for trigonometric polynomials of degree < n_theta:
    angular factors of Eq. 60-62 average to (2nx^2+ny^2+nz^2)/2, (ny^2+3nz^2)/8, -nz (Eq. 65-67)."""
    n0, n1 = 9, 16
    th = 2 * np.pi * np.arange(n1) / n1
    u = np.linspace(1.0, 2.0, n0)
    nx, ny, nz = 0.36, -0.48, 0.8
    s, c = np.sin(th), np.cos(th)
    fM = nx ** 2 + ny ** 2 * c * c + nz ** 2 * s * s - 2 * ny * nz * s * c
    fP = ny ** 2 * s * s * c * c + nz ** 2 * s ** 4 - 2 * ny * nz * s ** 3 * c
    fNM = 2 * (ny * s * c - nz * s * s)
    maps = np.stack([np.outer(u, f).ravel() for f in (fM, fP, fNM)])
    I = oracle_mod.azimuthal_polar(maps, n0, n1)
    np.testing.assert_allclose(I[0], u * (2 * nx ** 2 + ny ** 2 + nz ** 2) / 2, atol=1e-13)
    np.testing.assert_allclose(I[1], u * (ny ** 2 + 3 * nz ** 2) / 8, atol=1e-13)
    np.testing.assert_allclose(I[2], u * (-nz), atol=1e-13)


def test_azimuthal_histogram_by_hand(oracle_mod):
    """Histogram average (reading 8): bin = floor((|q|-q_lo)/(q_hi-q_lo) n_bins); outside dropped; empty bins 0/count 0."""
    qy = np.array([0.0, 0.3, 0.0, 0.6, 1.2, 0.05, 2.0])
    qz = np.array([0.1, 0.4, 0.5, 0.8, 0.0, 0.0, 0.0])       # |q| = .1 .5 .5 1.0 1.2 .05 2.0
    f = np.array([[1.0, 2.0, 4.0, 8.0, 16.0, 32.0, 64.0]])
    I, cnt = oracle_mod.azimuthal_hist(f, qy, qz, 4, 0.0, 2.0)          # bins [0,.5) [.5,1) [1,1.5) [1.5,2)
    np.testing.assert_array_equal(cnt, [2, 2, 2, 0])
    np.testing.assert_allclose(I[0], [(1 + 32) / 2, (2 + 4) / 2, (8 + 16) / 2, 0.0])
    np.testing.assert_allclose(oracle_mod.hist_bin_centres(4, 0.0, 2.0), [0.25, 0.75, 1.25, 1.75])


def test_c2_detector_binning_counts(oracle_mod):
    """C2's 128 x 128 cartesian detector, 128 bins on [0, 1.5): corner pixels are dropped and a few
    innermost bins are empty (generator + binning property used by the correlation pass)."""
    w = ni.config_c2()
    qy, qz, _ = oracle_mod.grid_points(w.grid)
    _, cnt = oracle_mod.azimuthal_hist(np.zeros((1, w.grid.n_q)), qy, qz, 128, 0.0, 1.5)
    qa = np.hypot(qy, qz)
    assert cnt.sum() == np.count_nonzero(qa < 1.5)
    assert cnt[0] == 0 and np.count_nonzero(cnt == 0) >= 1 and cnt.sum() < w.grid.n_q


# --------------------------------------------------------------------------- O16
def test_correlation_three_point_trapezoid(oracle_mod):
    """Eq. 34-35 (L205-L207) by hand on three abscissae, one of them empty."""
    q = np.array([0.5, 1.0, 1.5, 2.5])
    I = np.array([[2.0, 99.0, 1.0, 0.5]])
    cnt = np.array([3, 0, 1, 2], dtype=np.int32)
    r = np.array([0.0, 2.0])
    c, p = oracle_mod.correlation(I, q, r, count=cnt)
    def f(i, rr):
        x = q[i] * rr
        j0 = 1.0 if x == 0 else math.sin(x) / x
        return I[0, i] * j0 * q[i] ** 2
    for k, rr in enumerate(r):
        want = (0.5 * (f(0, rr) + f(2, rr)) * 1.0 + 0.5 * (f(2, rr) + f(3, rr)) * 1.0) / (2 * math.pi ** 2)
        assert abs(c[0, k] - want) < 1e-14
        assert abs(p[0, k] - rr * rr * want) < 1e-14


def test_correlation_of_sphere_form_factor_is_gamma0(oracle_mod):
    """I(q) = V_s 9 g(qR)^2 -> c(r) = gamma_0(r/R) = 1 - 3 xi/4 + xi^3/16 and p = r^2 c = R^2 f(xi)/4
    (Eq. 74; Eq. 77 is 2 pi^2 times this, reading 9).  q_max R = 400; converges like 1/q_max."""
    Rr = 1.0
    q = np.linspace(1e-6, 400.0, 400001)
    v = q * Rr
    gg = (np.sin(v) - v * np.cos(v)) / v ** 3
    I = (4 * np.pi / 3 * Rr ** 3) * 9 * gg ** 2
    r = np.array([0.0, 0.3, 0.8, 1.0494, 1.5, 1.9, 2.0, 2.5])
    c, p = oracle_mod.correlation(I[None, :], q, r)
    xi = r / Rr
    gam = np.where(xi < 2, 1 - 0.75 * xi + xi ** 3 / 16, 0.0)
    # r > 0: the truncated tail oscillates and cancels (1e-5); r = 0: the missing Porod tail
    # int_{qmax}^inf (9 V_s / 2 q^2 R^4) dq / (2 pi^2) = 3 / (pi qmax R) is known in closed form
    np.testing.assert_allclose(c[0][1:], gam[1:], atol=1e-5)
    assert abs(c[0][0] - (1.0 - 3.0 / (np.pi * 400.0 * Rr))) < 1e-5
    fxi = 0.25 * xi ** 2 * (xi - 2) ** 2 * (xi + 4)
    np.testing.assert_allclose(p[0][xi <= 2], (Rr ** 2 * fxi / 4)[xi <= 2], atol=1e-5)


# --------------------------------------------------------------------------- O17
def test_form_factor_split_two_identical_particles(oracle_mod):
    """Eq. 49 (L378): K = 1 -> form == total; two identical particles at +-d/2 -> form = 2 B(A1,A1),
    total = (2 + 2 cos q.d) B(A1,A1) for every kind (all are sesquilinear in the amplitudes)."""
    rng = np.random.default_rng(9)
    local = (rng.integers(-8, 8, size=(30, 3)) * 0.25).astype(np.float32)
    N1 = rng.normal(size=30).astype(np.float32)
    m1 = rng.normal(size=(30, 3)).astype(np.float32)
    g = _polar(8, 12, 0.05, 2.0)
    qy, qz, th = oracle_mod.grid_points(g)
    kinds = ni.ALL_KINDS
    A1 = oracle_mod.amplitudes(local, N1, m1, None, qy, qz)
    B1 = oracle_mod.response(A1, th, kinds)
    tot, frm = oracle_mod.form_factor_split(local, N1, m1, [0, 30], kinds, qy, qz, th)
    np.testing.assert_allclose(tot, B1, atol=1e-10)
    np.testing.assert_allclose(frm, B1, atol=1e-10)
    d = np.array([4.0, -6.5, 9.25])
    cen = np.stack([d / 2, -d / 2]).astype(np.float32)
    pos2 = np.concatenate([local, local])
    N2 = np.concatenate([N1, N1])
    m2 = np.concatenate([m1, m1])
    tot, frm = oracle_mod.form_factor_split(pos2, N2, m2, [0, 30, 60], kinds, qy, qz, th, centres=cen)
    np.testing.assert_allclose(frm, 2 * B1, rtol=1e-10, atol=1e-9)
    np.testing.assert_allclose(tot, (2 + 2 * np.cos(qy * d[1] + qz * d[2])) * B1, rtol=1e-9, atol=1e-8)
    # centres folded into global positions must give the same answer
    posg = np.concatenate([local + cen[0], local + cen[1]])
    tot2, frm2 = oracle_mod.form_factor_split(posg, N2, m2, [0, 30, 60], kinds, qy, qz, th)
    np.testing.assert_allclose(tot2, tot, rtol=1e-9, atol=1e-8)
    np.testing.assert_allclose(frm2, frm, rtol=1e-9, atol=1e-8)
    # total of the split == ordinary path on the whole sample
    A = oracle_mod.amplitudes(posg, N2, m2, None, qy, qz)
    np.testing.assert_allclose(oracle_mod.response(A, th, kinds), tot, rtol=1e-9, atol=1e-8)


# --------------------------------------------------------------------------- O18
def test_generator_cell_counts_and_table1_rows():
    """Lattice conventions: 4169 node-centred cells at R/a = 10 (L699), 4224 cell-centred (L684),
    33401 at R/a = 20; Table I rows (L293-L304) reproduced in order by the node-centred generator."""
    assert len(ni.sphere_node_centred(10.0, 1.0)) == 4169
    assert len(ni.sphere_node_centred(20.0, 2.0)) == 4169
    assert len(ni.sphere_cell_centred(5.0, 0.5)) == 4224
    p = ni.sphere_node_centred(20.0, 1.0)
    assert len(p) == 33401
    want = [(0, -20, 0), (-6, -19, -1), (-6, -19, 0), (-6, -19, 1), (-5, -19, -3), (-5, -19, -2), (-5, -19, -1),
            (-5, -19, 0), (-5, -19, 1), (-5, -19, 2)]
    np.testing.assert_array_equal(p[:10], np.array(want, dtype=float))
    assert ni.config_c1().W == 4169 and ni.config_c2().W == 12640
    w3 = ni.make_config("C3", small=True)
    assert w3.W == 6 * 4224 and w3.offsets[-1] == w3.W
    m = w3.m.astype(np.float64)
    np.testing.assert_allclose(np.linalg.norm(m, axis=1), 1.0, atol=1e-6)
    w5 = ni.make_config("C5", small=True)
    assert 0.05 <= np.mean(w5.N == 0) < 0.06
    np.testing.assert_allclose(np.linalg.norm(w5.m.astype(np.float64), axis=1), 1.0, atol=1e-6)


# ----------------------------------------------------------------------------------------------------
# angular modal decomposition, Eq. 31-33 (L187-L199)
# ----------------------------------------------------------------------------------------------------
def _theta(n):
    return (2.0 * np.pi * np.arange(n) / n).astype(np.float32).astype(np.float64)


def test_modal_two_and_four_fold_anisotropy_ratios(oracle_mod):
    """L199: 'a two-fold sin^2 theta anisotropy yields A_0^c / A_2^c = -1, whereas for the case of a four-fold
    sin^2 theta cos^2 theta anisotropy A_0^c / A_4^c = -1' -- sin^2 = (1 - cos 2 theta)/2 and
    sin^2 cos^2 = (1 - cos 4 theta)/8, so I_0^c = u/2, I_2^c = -u/2 resp. I_0^c = u/8, I_4^c = -u/8."""
    n0, n1, kmax = 7, 48, 6
    th = _theta(n1)
    u = np.linspace(1.0, 3.0, n0)
    f2 = (u[:, None] * np.sin(th)[None, :] ** 2).reshape(1, -1)
    f4 = (u[:, None] * (np.sin(th) * np.cos(th))[None, :] ** 2).reshape(1, -1)
    Is, Ic, a_s, a_c, A_s, A_c = oracle_mod.modal(np.concatenate([f2, f4]), n0, n1, th, kmax)
    np.testing.assert_allclose(Ic[0, 0], u / 2, rtol=1e-6)
    np.testing.assert_allclose(Ic[0, 2], -u / 2, rtol=1e-6)
    np.testing.assert_allclose(Ic[1, 0], u / 8, rtol=1e-6)
    np.testing.assert_allclose(Ic[1, 4], -u / 8, rtol=1e-6)
    assert A_c[0, 0] / A_c[0, 2] == pytest.approx(-1.0, rel=1e-6)
    assert A_c[1, 0] / A_c[1, 4] == pytest.approx(-1.0, rel=1e-6)
    other2 = [k for k in range(kmax + 1) if k not in (0, 2)]
    assert np.abs(Ic[0][other2]).max() < 1e-6 and np.abs(Is[0]).max() < 1e-6
    # Eq. 32-33: a_k = sum_i I_k(q_i); A_k normalised by sum_j sqrt(a_j^s^2 + a_j^c^2)
    np.testing.assert_allclose(a_c[0, 0], u.sum() / 2, rtol=1e-6)
    np.testing.assert_allclose(np.sqrt(A_s ** 2 + A_c ** 2).sum(axis=1), 1.0, rtol=1e-12)


def test_modal_recovers_a_trigonometric_polynomial(oracle_mod):
    """f = c0 + sum_k (c_k cos k theta + s_k sin k theta), k <= 5 < n_theta / 2: Eq. 31 by the periodic trapezoid
    returns exactly I_0^c = c0, I_k^c = c_k, I_k^s = s_k (prefactor (2 - delta_k0) / 2 pi); the fp32 rounding of
    the grid's theta_j limits the agreement to ~k * 2^-24 * 2 pi."""
    rng = np.random.Generator(np.random.Philox(31))
    n0, n1, kmax = 3, 40, 5
    th = _theta(n1)
    c = rng.normal(size=(n0, kmax + 1))
    s = rng.normal(size=(n0, kmax + 1)); s[:, 0] = 0.0
    f = sum(c[:, k, None] * np.cos(k * th)[None, :] + s[:, k, None] * np.sin(k * th)[None, :] for k in range(kmax + 1))
    Is, Ic, a_s, a_c, A_s, A_c = oracle_mod.modal(f.reshape(1, -1), n0, n1, th, kmax)
    np.testing.assert_allclose(Ic[0].T, c, atol=2e-5)
    np.testing.assert_allclose(Is[0].T, s, atol=2e-5)
    np.testing.assert_allclose(a_c[0], c.sum(axis=0), atol=1e-4)
    np.testing.assert_allclose(a_s[0], s.sum(axis=0), atol=1e-4)


def test_modal_order_zero_is_the_azimuthal_average_and_brute_force(oracle_mod):
    """k = 0 of Eq. 31 is Eq. 30; every entry against a literal Python loop on a random map."""
    rng = np.random.Generator(np.random.Philox(32))
    n0, n1, kmax = 4, 17, 3
    th = _theta(n1)
    f = rng.normal(size=(2, n0 * n1))
    Is, Ic, a_s, a_c, A_s, A_c = oracle_mod.modal(f, n0, n1, th, kmax)
    np.testing.assert_allclose(Ic[:, 0], oracle_mod.azimuthal_polar(f, n0, n1), rtol=1e-13, atol=1e-15)
    for a in range(2):
        for k in range(kmax + 1):
            for i in range(n0):
                ss = sum(f[a, i * n1 + j] * math.sin(k * th[j]) for j in range(n1))
                cc = sum(f[a, i * n1 + j] * math.cos(k * th[j]) for j in range(n1))
                pref = (1.0 if k == 0 else 2.0) / n1
                assert Is[a, k, i] == pytest.approx(pref * ss, rel=1e-12, abs=1e-14)
                assert Ic[a, k, i] == pytest.approx(pref * cc, rel=1e-12, abs=1e-14)
        norm = sum(math.hypot(Is[a, k].sum(), Ic[a, k].sum()) for k in range(kmax + 1))
        np.testing.assert_allclose(A_c[a], Ic[a].sum(axis=1) / norm, rtol=1e-12)
        np.testing.assert_allclose(A_s[a], Is[a].sum(axis=1) / norm, rtol=1e-12, atol=1e-15)


def test_modal_uniform_sphere_magnetic_channel(oracle_mod):
    """C1-type sample (uniform m = e_z): MAG = |F|^2 sin^2 theta (Eq. 60) up to the lattice's own weak angular
    dependence, hence A_0^c / A_2^c = -1 to that level and all sine amplitudes vanish (mirror symmetry)."""
    wl = ni.make_config("C1")
    qy, qz, th = oracle_mod.grid_points(wl.grid)
    A = oracle_mod.amplitudes(wl.pos, wl.N, wl.m, wl.R, qy, qz)
    M = oracle_mod.response(A, th, [KI["MAG"]], P=wl.P)
    Is, Ic, a_s, a_c, A_s, A_c = oracle_mod.modal(M, wl.grid.n0, wl.grid.n1, wl.grid.u1, 4)
    assert A_c[0, 0] / A_c[0, 2] == pytest.approx(-1.0, abs=0.02)
    assert np.abs(A_s[0]).max() < 1e-6


# ----------------------------------------------------------------------------------------------------
# two-dimensional correlation function, Eq. 36 (L213)
# ----------------------------------------------------------------------------------------------------
def test_correlation_2d_of_a_ring_is_bessel(oracle_mod):
    """A single detector ring (n_q = 1, weight 1): the theta integral of exp(i x cos(theta - alpha)) is 2 pi J0(x) and
    that of cos(2 theta) exp(i x cos(theta - alpha)) is 2 pi i^2 J2(x) cos 2 alpha (Jacobi-Anger); the periodic
    trapezoid is exact to rounding for n_theta well above x.  scipy supplies J0, J2 (library routine, independent)."""
    from scipy.special import jv
    n1, q0 = 96, 0.8
    th = _theta(n1)
    rho = np.linspace(0.0, 20.0, 33).astype(np.float32).astype(np.float64)
    al = _theta(12)
    re, im = oracle_mod.correlation_2d(np.ones(n1), [q0], th, rho, al)
    want = 2 * np.pi * q0 * jv(0, q0 * rho)                           # f q wq dtheta sum = q0 * 2 pi J0
    np.testing.assert_allclose(re, np.repeat(want[:, None], 12, axis=1), atol=1e-6)
    assert np.abs(im).max() < 1e-6
    re2, im2 = oracle_mod.correlation_2d(np.cos(2 * th), [q0], th, rho, al)
    want2 = -2 * np.pi * q0 * jv(2, q0 * rho)[:, None] * np.cos(2 * al)[None, :]
    np.testing.assert_allclose(re2, want2, atol=2e-6)
    assert np.abs(im2).max() < 2e-6
    # an odd harmonic gives a purely imaginary C: int sin(theta) e^{i x cos(theta - alpha)} = 2 pi i J1(x) sin alpha
    re3, im3 = oracle_mod.correlation_2d(np.sin(th), [q0], th, rho, al)
    np.testing.assert_allclose(im3, 2 * np.pi * q0 * jv(1, q0 * rho)[:, None] * np.sin(al)[None, :], atol=2e-6)
    assert np.abs(re3).max() < 2e-6


def test_correlation_2d_of_a_gaussian(oracle_mod):
    """f = exp(-q^2 s^2 / 2): C(rho) = 2 pi int f J0(q rho) q dq = (2 pi / s^2) exp(-rho^2 / (2 s^2)) (Hankel pair);
    fine, long q grid (q_max s = 8); the trapezoid in q leaves the Euler-Maclaurin end term 2 pi h^2 / 12 (f q)'(0)
    = 1.3e-5 for h = 0.005, a constant offset, which bounds the agreement."""
    s_ = 2.0
    q = np.linspace(0.0, 4.0, 801)
    th = _theta(64)
    f = np.repeat(np.exp(-0.5 * (q * s_) ** 2)[:, None], 64, axis=1)
    rho = np.linspace(0.0, 6.0, 13)
    re, im = oracle_mod.correlation_2d(f, q, th, rho, [0.0, 1.0])
    want = 2 * np.pi / s_ ** 2 * np.exp(-0.5 * (rho / s_) ** 2)
    np.testing.assert_allclose(re[:, 0], want, rtol=0, atol=2e-5)
    np.testing.assert_allclose(re[:, 1], want, rtol=0, atol=2e-5)
    assert re[0, 0] - want[0] == pytest.approx(-2 * np.pi * 0.005 ** 2 / 12, rel=0.05)     # the end term itself, at rho = 0
    assert np.abs(im).max() < 1e-7          # theta_j are float32 values: the inversion symmetry holds to 2^-24


def test_correlation_2d_brute_force_and_trapezoid_weights(oracle_mod):
    """Literal Python loops with the non-uniform trapezoid weights written out by hand, on a random map."""
    rng = np.random.Generator(np.random.Philox(36))
    q = np.array([0.1, 0.25, 0.7, 1.0]); wq = np.array([0.075, 0.3, 0.375, 0.15])
    n1 = 7
    th = _theta(n1)
    f = rng.normal(size=(4, n1))
    rho, al = np.array([0.0, 1.5, 4.0]), np.array([0.3, 2.0])
    re, im = oracle_mod.correlation_2d(f, q, th, rho, al)
    for a in range(3):
        for b in range(2):
            z = 0j
            for i in range(4):
                for j in range(n1):
                    z += f[i, j] * q[i] * wq[i] * (2 * math.pi / n1) * cmath.exp(1j * q[i] * rho[a] * math.cos(th[j] - al[b]))
            assert re[a, b] == pytest.approx(z.real, rel=1e-12, abs=1e-14)
            assert im[a, b] == pytest.approx(z.imag, rel=1e-12, abs=1e-14)
    # C(0) is the plain integral of f q; C(rho, alpha + pi) = conj C(rho, alpha) for a real map
    assert re[0, 0] == pytest.approx(float(((f * (q * wq)[:, None]).sum()) * 2 * math.pi / n1), rel=1e-12)
    re2, im2 = oracle_mod.correlation_2d(f, q, th, rho, al + math.pi)
    np.testing.assert_allclose(re2, re, atol=1e-12)
    np.testing.assert_allclose(im2, -im, atol=1e-12)


# ----------------------------------------------------------------------------------------------------
# Fourier cross-correlation components G_ab = M~_a M~_b^*, Eq. 51-52 (L397-L402)
# ----------------------------------------------------------------------------------------------------
def test_cross_spectra_reproduce_the_cross_sections(oracle_mod):
    """The magnetic cross sections are contractions of G: with q^ = (0, s, c), |Q|^2 = |M~|^2 - |q^.M~|^2 gives
    MAG = sum_ab (delta_ab - q^_a q^_b) G^R_ab (Eq. 4-5), and Eq. 14 gives CHI = 2 (P_y s + P_z c)(s G^I_zx - c G^I_yx);
    both against the independently coded response routine, general P, scales and rotation; G is Hermitian."""
    rng = np.random.Generator(np.random.Philox(51))
    W = 40
    pos = rng.uniform(-8, 8, size=(W, 3)).astype(np.float32)
    N = rng.uniform(0.5, 1.5, size=W).astype(np.float32)
    m = rng.normal(size=(W, 3)).astype(np.float32)
    grid = ni.polar_grid(np.linspace(0.05, 2.0, 9), 16)
    qy, qz, th = oracle_mod.grid_points(grid)
    R = ni.rot_z(25.0) @ ni.rot_y(40.0)
    P = np.array([0.3, -0.5, 0.8]); P /= np.linalg.norm(P)
    sM, invV = 1.7, 0.01
    A = oracle_mod.amplitudes(pos, N, m, R, qy, qz)
    GR, GI = oracle_mod.cross_spectra(A, sM=sM, invV=invV)
    MAG, CHI = oracle_mod.response(A, th, [KI["MAG"], KI["CHI"]], P=P, sM=sM, invV=invV)
    qh = np.stack([np.zeros_like(th), np.sin(th), np.cos(th)])
    mag = sum(((a == b) - qh[a] * qh[b]) * GR[3 * a + b] for a in range(3) for b in range(3))
    np.testing.assert_allclose(mag, MAG, rtol=1e-11, atol=1e-12 * np.abs(MAG).max())
    s, c = np.sin(th), np.cos(th)
    chi = 2 * (P[1] * s + P[2] * c) * (s * GI[3 * 2 + 0] - c * GI[3 * 1 + 0])
    np.testing.assert_allclose(chi, CHI, rtol=1e-10, atol=1e-12 * np.abs(MAG).max())
    for a in range(3):
        assert np.all(np.abs(GI[3 * a + a]) <= 1e-15 * GR[3 * a + a]) and np.all(GR[3 * a + a] >= 0.0)
        for b in range(3):
            np.testing.assert_allclose(GR[3 * a + b], GR[3 * b + a], rtol=1e-14, atol=1e-15 * np.abs(GR).max())
            if a != b:
                np.testing.assert_allclose(GI[3 * a + b], -GI[3 * b + a], rtol=1e-14, atol=1e-15 * np.abs(GR).max())


def test_cross_spectra_uniform_magnetisation(oracle_mod):
    """Uniform m = n: M~ = n F, so G_ab = n_a n_b |F|^2 is real (Eq. 51-52 with Eq. 60's M~), |F|^2 = NUC for N = 1."""
    pos, N, m = ni.uniform_sphere_sample(radius=6.0, a=1.0, n=(0.6, 0.0, 0.8))
    grid = ni.polar_grid(np.linspace(0.05, 1.5, 6), 12)
    qy, qz, th = oracle_mod.grid_points(grid)
    A = oracle_mod.amplitudes(pos, N, m, None, qy, qz)
    GR, GI = oracle_mod.cross_spectra(A)
    F2 = oracle_mod.response(A, th, [KI["NUC"]])[0]
    n = np.array([0.6, 0.0, 0.8])
    for a in range(3):
        for b in range(3):
            np.testing.assert_allclose(GR[3 * a + b], n[a] * n[b] * F2, rtol=1e-6, atol=1e-9 * F2.max())
            assert np.abs(GI[3 * a + b]).max() <= 1e-9 * F2.max()


# --------------------------------------------------------------------------- f-3: batched magnetisation fields
def test_batched_fields_share_the_nuclear_amplitude_and_are_linear(oracle_mod):
    """Loop mode (L254, L323, L391): B magnetisation fields on one geometry.  Pins that do not re-call the routine on the
    same data: (i) the nuclear planes do not depend on the field and equal the run without moments; (ii) M~ is linear in
    m -- fields chosen with exactly representable sums, m_2 = m_0 + m_1 and m_3 = -2 m_0; (iii) a uniform field m_b = n_b
    on N = 1 has M~ = (R n_b) N~ (Eq. 43 with constant moment); (iv) B = 1 is the single call."""
    rng = np.random.Generator(np.random.Philox(33))
    W = 257
    pos = rng.uniform(-12, 12, size=(W, 3)).astype(np.float32)
    N = np.ones(W, dtype=np.float32)
    m0 = (rng.integers(-8, 9, size=(W, 3)) / 8.0).astype(np.float32)            # dyadic: sums are exact in fp32
    m1 = (rng.integers(-8, 9, size=(W, 3)) / 16.0).astype(np.float32)
    n4, n5 = np.array([0.25, -0.5, 1.0], dtype=np.float32), np.array([1.0, 0.0, 0.0], dtype=np.float32)
    mb = np.stack([m0, m1, m0 + m1, -2.0 * m0, np.tile(n4, (W, 1)), np.tile(n5, (W, 1))]).astype(np.float32)
    R = ni.rotation_alpha_beta(25.0, 40.0)
    g = _polar(7, 9)
    qy, qz, th = oracle_mod.grid_points(g)
    A = oracle_mod.amplitudes_batch(pos, N, mb, R, qy, qz)
    assert A.shape == (6, 8, g.n_q)
    A_nuc = oracle_mod.amplitudes(pos, N, None, R, qy, qz)
    scale = np.abs(A).max()
    for b in range(6):
        np.testing.assert_allclose(A[b, 0:2], A_nuc[0:2], rtol=0, atol=1e-13 * scale)                 # (i)
    np.testing.assert_allclose(A[2, 2:], A[0, 2:] + A[1, 2:], rtol=0, atol=1e-12 * scale)             # (ii)
    np.testing.assert_allclose(A[3, 2:], -2.0 * A[0, 2:], rtol=0, atol=1e-12 * scale)
    for b, n in ((4, n4), (5, n5)):                                                                   # (iii)
        Rn = R @ n.astype(np.float64)
        for c in range(3):
            np.testing.assert_allclose(A[b, 2 + 2 * c], Rn[c] * A_nuc[0], rtol=0, atol=1e-12 * scale)
            np.testing.assert_allclose(A[b, 3 + 2 * c], Rn[c] * A_nuc[1], rtol=0, atol=1e-12 * scale)
    A1 = oracle_mod.amplitudes_batch(pos, N, mb[1:2], R, qy, qz)                                      # (iv)
    assert np.array_equal(A1[0], oracle_mod.amplitudes(pos, N, mb[1], R, qy, qz))


# --------------------------------------------------------------------------- f-4: Friedel symmetry
def test_friedel_symmetry_of_real_weights(oracle_mod):
    """Eq. 42-43 (L353-L356) with real N_j, m_j: A(-q) = A(q)^*, exactly; on a ring, theta -> theta + pi is -q (L183).
    Consequences for the responses: the |.|^2-type kinds are even, the chiral one is odd (pinned in
    test_chiral_symmetries); here the amplitude identity itself, at exactly negated q."""
    rng = np.random.Generator(np.random.Philox(404))
    W = 300
    pos = rng.uniform(-20, 20, size=(W, 3)).astype(np.float32)
    N = rng.normal(size=W).astype(np.float32)
    m = rng.normal(size=(W, 3)).astype(np.float32)
    R = ni.rotation_alpha_beta(12.0, 77.0)
    qy, qz = rng.uniform(-2, 2, size=50), rng.uniform(-2, 2, size=50)
    A = oracle_mod.amplitudes(pos, N, m, R, qy, qz)
    B = oracle_mod.amplitudes(pos, N, m, R, -qy, -qz)
    np.testing.assert_allclose(B[0::2], A[0::2], rtol=0, atol=1e-12 * np.abs(A).max())
    np.testing.assert_allclose(B[1::2], -A[1::2], rtol=0, atol=1e-12 * np.abs(A).max())
