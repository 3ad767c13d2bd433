"""fp64 CPU oracle of the NuMagSANS direct-summation core -- TEST INFRASTRUCTURE ONLY.

Thin ctypes binding over `oracle/nmso.c` (plain C99 + OpenMP, libm sin/cos).
Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s cpu_baseline /
`--impl reference` leg may import this package.  It imports nothing from
`paper_2601_18444_b200/` and the product never imports it.

Array conventions mirror PAPER.md: amplitudes are [8][n_q] planes
(Re N, Im N, Re Mx, Im Mx, Re My, Im My, Re Mz, Im Mz) of the raw sums of
Eq. 42-47 (L353-L368); response maps are [n_kinds][n_q].
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from typing import Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "nmso.c")
_LIB = os.path.join(_HERE, "libnmso.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile oracle/nmso.c -> oracle/libnmso.so with gcc (-O2, no fast-math, OpenMP)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-fopenmp", "-shared", "-fPIC", "-std=c99", "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


def lib():
    global _lib
    if _lib is None:
        build()
        _lib = C.CDLL(_LIB)
        _lib.nmso_num_threads.restype = C.c_int
    return _lib


def num_threads() -> int:
    return int(lib().nmso_num_threads())


def _p(a, typ):
    return None if a is None else a.ctypes.data_as(C.POINTER(typ))


def _f32(a):
    return None if a is None else np.ascontiguousarray(a, dtype=np.float32)


def _f64(a):
    return None if a is None else np.ascontiguousarray(a, dtype=np.float64)


def _chk(rc, what):
    if rc != 0:
        raise RuntimeError(f"oracle {what} failed with code {rc}")


def grid_points(grid):
    """(q_y, q_z, theta) in fp64 for every flat detector index of an nms_inputs Grid."""
    n = grid.n0 * grid.n1
    qy, qz, th = (np.empty(n, dtype=np.float64) for _ in range(3))
    u0, u1 = _f32(grid.u0), _f32(grid.u1)
    _chk(lib().nmso_grid_points(C.c_int(grid.type), C.c_int(grid.n0), C.c_int(grid.n1), _p(u0, C.c_float), _p(u1, C.c_float),
                                _p(qy, C.c_double), _p(qz, C.c_double), _p(th, C.c_double)), "grid_points")
    return qy, qz, th


def amplitudes(pos, N, m, R=None, qy=None, qz=None, qx=None, offsets=None, centres=None, return_wsum=False):
    """Raw direct sums A[8, n_q] (fp64) at the given detector points (Eq. 42-47)."""
    pos, N, m = _f32(pos), _f32(N), _f32(m)
    W = pos.shape[0]
    qy, qz, qx = _f64(qy), _f64(qz), _f64(qx)
    nq = qy.shape[0]
    Rm = None if R is None else _f64(np.asarray(R).reshape(9))
    off = None if offsets is None else np.ascontiguousarray(offsets, dtype=np.int64)
    cen = _f32(centres)
    K = 0 if off is None else off.shape[0] - 1
    out = np.empty((8, nq), dtype=np.float64)
    wsum = np.zeros(4, dtype=np.float64)
    _chk(lib().nmso_amplitudes(_p(pos, C.c_float), _p(N, C.c_float), _p(m, C.c_float), C.c_int64(W),
                               _p(off, C.c_int64), C.c_int64(K), _p(cen, C.c_float), _p(Rm, C.c_double),
                               _p(qx, C.c_double), _p(qy, C.c_double), _p(qz, C.c_double), C.c_int64(nq),
                               _p(out, C.c_double), _p(wsum, C.c_double)), "amplitudes")
    return (out, wsum) if return_wsum else out


def amplitudes_batch(pos, N, m_batch, R=None, qy=None, qz=None, offsets=None, centres=None):
    """Batched magnetisation fields on a fixed geometry (the paper's loop mode: one m_i file per field / temperature /
    time step on the same NucData and StructData, L254, L323, L391): the plain loop of `amplitudes` over the B fields
    m_batch [B, W, 3].  Returns A [B, 8, n_q]; the nuclear planes A[b, 0:2] are the same for every field."""
    m_batch = np.ascontiguousarray(m_batch, dtype=np.float32)
    return np.stack([amplitudes(pos, N, m_batch[b], R, qy, qz, offsets=offsets, centres=centres) for b in range(m_batch.shape[0])])


def response(amp, theta, kinds: Sequence[int], P=None, sN=1.0, sM=1.0, invV=1.0, return_Q=False):
    """Response maps [n_kinds, n_q] from amplitudes via the Halpern-Johnson vector (Eq. 3-29)."""
    amp, theta = _f64(amp), _f64(theta)
    nq = theta.shape[0]
    kk = np.ascontiguousarray(kinds, dtype=np.int32)
    Pv = None if P is None else _f64(P)
    out = np.empty((len(kk), nq), dtype=np.float64)
    Q = np.empty((6, nq), dtype=np.float64) if return_Q else None
    _chk(lib().nmso_response(_p(amp, C.c_double), _p(theta, C.c_double), C.c_int64(nq), _p(Pv, C.c_double),
                             C.c_double(sN), C.c_double(sM), C.c_double(invV), _p(kk, C.c_int), C.c_int(len(kk)),
                             _p(out, C.c_double), _p(Q, C.c_double)), "response")
    return (out, Q) if return_Q else out


def cross_spectra(amp, sM=1.0, invV=1.0):
    """Fourier cross-correlation components of the magnetisation (Eq. 51-52), plain NumPy complex arithmetic:
    G_ab = invV sM^2 M~_a M~_b^*, a, b in (x, y, z); returns (G^R, G^I) [9, n_q] with row 3 a + b.
    amp [8, n_q] are the raw amplitude planes (Re N, Im N, Re Mx, Im Mx, ...); scales as in DESIGN.md reading 4."""
    amp = _f64(amp)
    M = [sM * (amp[2 + 2 * c] + 1j * amp[3 + 2 * c]) for c in range(3)]
    G = np.stack([invV * M[a] * np.conj(M[b]) for a in range(3) for b in range(3)])
    return np.ascontiguousarray(G.real), np.ascontiguousarray(G.imag)


def form_factor_split(pos, N, m, offsets, kinds, qy, qz, theta, R=None, centres=None, P=None, sN=1.0, sM=1.0, invV=1.0):
    """(total, form) maps [n_kinds, n_q] (Eq. 49-50): total = B(sum A_p), form = sum B(A_p)."""
    pos, N, m = _f32(pos), _f32(N), _f32(m)
    W = pos.shape[0]
    qy, qz, theta = _f64(qy), _f64(qz), _f64(theta)
    nq = qy.shape[0]
    Rm = None if R is None else _f64(np.asarray(R).reshape(9))
    off = np.ascontiguousarray(offsets, dtype=np.int64)
    cen = _f32(centres)
    kk = np.ascontiguousarray(kinds, dtype=np.int32)
    Pv = None if P is None else _f64(P)
    tot = np.empty((len(kk), nq), dtype=np.float64)
    frm = np.empty((len(kk), nq), dtype=np.float64)
    _chk(lib().nmso_form_factor_split(_p(pos, C.c_float), _p(N, C.c_float), _p(m, C.c_float), C.c_int64(W),
                                      _p(off, C.c_int64), C.c_int64(off.shape[0] - 1), _p(cen, C.c_float), _p(Rm, C.c_double),
                                      _p(qy, C.c_double), _p(qz, C.c_double), _p(theta, C.c_double), C.c_int64(nq),
                                      _p(Pv, C.c_double), C.c_double(sN), C.c_double(sM), C.c_double(invV),
                                      _p(kk, C.c_int), C.c_int(len(kk)), _p(tot, C.c_double), _p(frm, C.c_double)), "form_factor_split")
    return tot, frm


def azimuthal_polar(maps, n0: int, n1: int):
    """Ring means [n_maps, n0] of maps [n_maps, n0*n1] on a polar grid (Eq. 30, periodic trapezoid)."""
    maps = _f64(maps).reshape(-1, n0 * n1)
    out = np.empty((maps.shape[0], n0), dtype=np.float64)
    _chk(lib().nmso_azimuthal_polar(_p(maps, C.c_double), C.c_int(maps.shape[0]), C.c_int(n0), C.c_int(n1), _p(out, C.c_double)), "azimuthal_polar")
    return out


def modal(maps, n0: int, n1: int, theta, k_max: int):
    """Angular modal decomposition (Eq. 31-33) of maps [n_maps, n0*n1] on a polar grid with angles theta [n1]:
    returns (Is, Ic) [n_maps, k_max+1, n0], (a_s, a_c) and (A_s, A_c) [n_maps, k_max+1]."""
    maps = _f64(maps).reshape(-1, n0 * n1)
    theta = _f64(theta)
    nm, nk = maps.shape[0], k_max + 1
    Is, Ic = np.empty((nm, nk, n0)), np.empty((nm, nk, n0))
    a_s, a_c, A_s, A_c = (np.empty((nm, nk)) for _ in range(4))
    _chk(lib().nmso_modal(_p(maps, C.c_double), C.c_int(nm), C.c_int(n0), C.c_int(n1), _p(theta, C.c_double),
                          C.c_int(k_max), _p(Is, C.c_double), _p(Ic, C.c_double), _p(a_s, C.c_double),
                          _p(a_c, C.c_double), _p(A_s, C.c_double), _p(A_c, C.c_double)), "modal")
    return Is, Ic, a_s, a_c, A_s, A_c


def azimuthal_hist(maps, qy, qz, n_bins: int, q_lo: float, q_hi: float):
    """(I [n_maps, n_bins], count [n_bins]) histogram means by |q| (reading 8)."""
    qy, qz = _f64(qy), _f64(qz)
    maps = _f64(maps).reshape(-1, qy.shape[0])
    out = np.empty((maps.shape[0], n_bins), dtype=np.float64)
    cnt = np.empty(n_bins, dtype=np.int32)
    _chk(lib().nmso_azimuthal_hist(_p(maps, C.c_double), C.c_int(maps.shape[0]), _p(qy, C.c_double), _p(qz, C.c_double),
                                   C.c_int64(qy.shape[0]), C.c_int(n_bins), C.c_double(q_lo), C.c_double(q_hi),
                                   _p(out, C.c_double), _p(cnt, C.c_int32)), "azimuthal_hist")
    return out, cnt


def correlation_2d(fmap, q, theta, rho, alpha):
    """(Re C, Im C) [len(rho), len(alpha)] of Eq. 36 for one map [len(q) * len(theta)] on a polar grid."""
    q, theta, rho, alpha = _f64(q), _f64(theta), _f64(rho), _f64(alpha)
    fmap = _f64(fmap).reshape(q.shape[0] * theta.shape[0])
    re, im = np.empty((rho.shape[0], alpha.shape[0])), np.empty((rho.shape[0], alpha.shape[0]))
    _chk(lib().nmso_correlation_2d(_p(fmap, C.c_double), C.c_int(q.shape[0]), C.c_int(theta.shape[0]), _p(q, C.c_double),
                                   _p(theta, C.c_double), C.c_int(rho.shape[0]), C.c_int(alpha.shape[0]),
                                   _p(rho, C.c_double), _p(alpha, C.c_double), _p(re, C.c_double), _p(im, C.c_double)),
         "correlation_2d")
    return re, im


def correlation(Iq, q, r, count=None):
    """(c, p) [n_maps, n_r] by the literal Eq. 34-35 trapezoid over the non-empty bins."""
    q, r = _f64(q), _f64(r)
    Iq = _f64(Iq).reshape(-1, q.shape[0])
    cnt = None if count is None else np.ascontiguousarray(count, dtype=np.int32)
    c = np.empty((Iq.shape[0], r.shape[0]), dtype=np.float64)
    p = np.empty_like(c)
    _chk(lib().nmso_correlation(_p(Iq, C.c_double), _p(q, C.c_double), _p(cnt, C.c_int32), C.c_int(Iq.shape[0]), C.c_int(q.shape[0]),
                                _p(r, C.c_double), C.c_int(r.shape[0]), _p(c, C.c_double), _p(p, C.c_double)), "correlation")
    return c, p


def hist_bin_centres(n_bins: int, q_lo: float, q_hi: float):
    """Abscissa of a histogram bin = its centre (reading 8)."""
    return q_lo + (np.arange(n_bins, dtype=np.float64) + 0.5) * (q_hi - q_lo) / n_bins
