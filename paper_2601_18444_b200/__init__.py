"""paper_2601_18444_b200 -- Python binding of libnms.so, the B200-native direct-summation SANS core.

The binding only marshals arguments: every numerical step (rotate + pack, the direct Fourier sums of
PAPER.md Eq. 42-47, the Section-II response functions, azimuthal average, c(r)/p(r), form-factor
split) runs in the hand-written sm_100a kernels behind the C ABI of ``include/nms.h``.  PyTorch is used
for device memory and streams only.  There is no CPU fallback: if the shared library is missing and
cannot be built, importing this package raises; without a CUDA device ``nms_create`` raises.

Functions carry the names of the C entry points (``nms_create``, ``nms_set_sample``,
``nms_amplitudes``, ``nms_response``, ``nms_compute``, ``nms_azimuthal_average``, ``nms_correlation``,
``nms_form_factor_split``, ``nms_run_host``, ...); device arrays are ``torch`` CUDA tensors, host
arrays are NumPy arrays.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional, Sequence

import numpy as np

from . import build as _build

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libnms.so")

KINDS = ["NUC", "MAG", "UNPOL", "PROJ", "NM", "SF", "CHI", "PM", "MP", "PP", "MM", "POL_PLUS", "POL_MINUS"]
NMS_OK, NMS_E_ARG, NMS_E_STATE, NMS_E_CUDA, NMS_E_NOMEM, NMS_E_UNSUPPORTED = range(6)
NMS_T_PREP, NMS_T_AMPLITUDE, NMS_T_EPILOGUE, NMS_T_AZIMUTHAL, NMS_T_CORRELATION, NMS_T_MODAL, NMS_T_CORR2D, NMS_T_BATCH = range(8)
_STATUS = {0: "NMS_OK", 1: "NMS_E_ARG", 2: "NMS_E_STATE", 3: "NMS_E_CUDA", 4: "NMS_E_NOMEM", 5: "NMS_E_UNSUPPORTED"}

EXPORTS = [
    "nms_create", "nms_destroy", "nms_last_error", "nms_synchronize", "nms_set_sample", "nms_set_particles",
    "nms_set_rotation", "nms_set_polarization", "nms_set_scales", "nms_amplitudes", "nms_response", "nms_compute",
    "nms_azimuthal_average", "nms_correlation", "nms_form_factor_split", "nms_run_host", "nms_get_weight_sums",
    "nms_set_option", "nms_get_info", "nms_kernel_time_ms", "nms_kernel_time_total", "nms_modal_decomposition",
    "nms_correlation_2d", "nms_cross_spectra", "nms_run_host_split", "nms_run_host_scan", "nms_pipe_rates", "nms_phasor_selftest", "nms_compute_batch",
    "nms_azimuthal_average_noalloc",
]


class NmsError(RuntimeError):
    def __init__(self, status: int, message: str):
        super().__init__(f"{_STATUS.get(status, status)}: {message}")
        self.status = status


class _QGrid(C.Structure):
    _fields_ = [("type", C.c_int), ("n0", C.c_int), ("n1", C.c_int),
                ("u0", C.POINTER(C.c_float)), ("u1", C.POINTER(C.c_float))]


def _load():
    if _build.needs_build():
        _build.build()          # raises if nvcc or the sources are missing: no fallback
    lib = C.CDLL(LIB_PATH)
    for name in EXPORTS:
        getattr(lib, name)      # AttributeError if a declared entry point is not exported
    lib.nms_last_error.restype = C.c_char_p
    lib.nms_last_error.argtypes = [C.c_void_p]
    lib.nms_destroy.restype = None
    lib.nms_destroy.argtypes = [C.c_void_p]
    return lib


_lib = _load()


def _dev(t):
    """Device pointer of a contiguous CUDA tensor (or None)."""
    if t is None:
        return C.c_void_p(None)
    if not t.is_cuda or not t.is_contiguous():
        raise ValueError("expected a contiguous CUDA tensor")
    return C.c_void_p(t.data_ptr())


def _host(a, dtype):
    if a is None:
        return None, C.c_void_p(None)
    arr = np.ascontiguousarray(a, dtype=dtype)
    return arr, C.c_void_p(arr.ctypes.data)


def _grid_struct(grid):
    """grid: object with .type .n0 .n1 .u0 .u1 (host float32 arrays), e.g. nms_inputs.Grid."""
    u0 = np.ascontiguousarray(grid.u0, dtype=np.float32)
    u1 = np.ascontiguousarray(grid.u1, dtype=np.float32)
    g = _QGrid(int(grid.type), int(grid.n0), int(grid.n1), u0.ctypes.data_as(C.POINTER(C.c_float)),
               u1.ctypes.data_as(C.POINTER(C.c_float)))
    return g, (u0, u1)


def _kinds(kinds: Sequence[int]):
    arr = (C.c_int * len(kinds))(*[int(k) for k in kinds])
    return arr, len(kinds)


def _check(ctx, st):
    if st != NMS_OK:
        msg = _lib.nms_last_error(ctx).decode() if ctx else ""
        raise NmsError(st, msg)


# ---- same-name wrappers ------------------------------------------------------------------------
def nms_create(device: int = 0, stream: Optional[int] = None):
    """Create a context on CUDA device `device` enqueuing on `stream` (a cudaStream_t as int; None = torch's current stream)."""
    if stream is None:
        import torch
        if not torch.cuda.is_available():
            raise NmsError(NMS_E_CUDA, "no CUDA device (there is no CPU fallback)")
        stream = torch.cuda.current_stream(device).cuda_stream
    out = C.c_void_p(None)
    st = _lib.nms_create(C.byref(out), C.c_int(device), C.c_void_p(stream))
    if st != NMS_OK:
        raise NmsError(st, "nms_create failed (no usable sm_100 device?)")
    return out


def nms_destroy(ctx):
    _lib.nms_destroy(ctx)


def nms_last_error(ctx) -> str:
    return _lib.nms_last_error(ctx).decode()


def nms_synchronize(ctx):
    _check(ctx, _lib.nms_synchronize(ctx))


def nms_set_sample(ctx, pos, N, m, R=None):
    W = int(pos.shape[0])
    Rh, Rp = _host(None if R is None else np.asarray(R, dtype=np.float64).reshape(9), np.float64)
    _check(ctx, _lib.nms_set_sample(ctx, _dev(pos), _dev(N), _dev(m), C.c_int64(W), Rp))


def nms_set_particles(ctx, offsets, centres=None):
    if offsets is None:
        _check(ctx, _lib.nms_set_particles(ctx, C.c_void_p(None), C.c_int64(0), C.c_void_p(None)))
        return
    oh, op = _host(offsets, np.int64)
    _check(ctx, _lib.nms_set_particles(ctx, op, C.c_int64(len(oh) - 1), _dev(centres)))


def nms_set_rotation(ctx, R):
    Rh, Rp = _host(None if R is None else np.asarray(R, dtype=np.float64).reshape(9), np.float64)
    _check(ctx, _lib.nms_set_rotation(ctx, Rp))


def nms_set_polarization(ctx, P):
    Ph, Pp = _host(np.asarray(P, dtype=np.float64).reshape(3), np.float64)
    _check(ctx, _lib.nms_set_polarization(ctx, Pp))


def nms_set_scales(ctx, sN=1.0, sM=1.0, invV=1.0):
    _check(ctx, _lib.nms_set_scales(ctx, C.c_double(sN), C.c_double(sM), C.c_double(invV)))


def nms_amplitudes(ctx, grid, out_amp=None):
    g, keep = _grid_struct(grid)
    _check(ctx, _lib.nms_amplitudes(ctx, C.byref(g), _dev(out_amp)))


def nms_response(ctx, kinds, out):
    k, n = _kinds(kinds)
    _check(ctx, _lib.nms_response(ctx, k, C.c_int(n), _dev(out)))


def nms_cross_spectra(ctx, out_GR=None, out_GI=None):
    _check(ctx, _lib.nms_cross_spectra(ctx, _dev(out_GR), _dev(out_GI)))


def nms_compute(ctx, grid, kinds, out):
    g, keep = _grid_struct(grid)
    k, n = _kinds(kinds)
    _check(ctx, _lib.nms_compute(ctx, C.byref(g), k, C.c_int(n), _dev(out)))


def nms_compute_batch(ctx, grid, m_batch, kinds, out_maps=None, out_amp=None):
    """Batched magnetisation fields m_batch [B, W, 3] (CUDA tensor) on the current sample's geometry (f-3)."""
    g, keep = _grid_struct(grid)
    k, n = _kinds(kinds)
    _check(ctx, _lib.nms_compute_batch(ctx, C.byref(g), _dev(m_batch), C.c_int(int(m_batch.shape[0])), k, C.c_int(n),
                                       _dev(out_maps), _dev(out_amp)))


def nms_form_factor_split(ctx, grid, kinds, out_total, out_form):
    g, keep = _grid_struct(grid)
    k, n = _kinds(kinds)
    _check(ctx, _lib.nms_form_factor_split(ctx, C.byref(g), k, C.c_int(n), _dev(out_total), _dev(out_form)))


def nms_azimuthal_average(ctx, maps, n_maps, n_bins, q_lo, q_hi, out_I, out_q=None, out_count=None):
    _check(ctx, _lib.nms_azimuthal_average(ctx, _dev(maps), C.c_int(n_maps), C.c_int(n_bins), C.c_double(q_lo),
                                           C.c_double(q_hi), _dev(out_I), _dev(out_q), _dev(out_count)))


def nms_azimuthal_average_noalloc(ctx, maps, n_maps, n_bins, q_lo, q_hi, out_I, out_q=None, out_count=None):
    """|q|-histogram average that allocates nothing (static 576 KB scratch in libnms.so; n_bins <= 16384, n_maps * n_bins
    <= 65536; calls that overlap on the GPU race on the scratch)."""
    _check(ctx, _lib.nms_azimuthal_average_noalloc(ctx, _dev(maps), C.c_int(n_maps), C.c_int(n_bins), C.c_double(q_lo),
                                                   C.c_double(q_hi), _dev(out_I), _dev(out_q), _dev(out_count)))


def nms_modal_decomposition(ctx, maps, n_maps, k_max, out_Is=None, out_Ic=None, out_a=None, out_A=None):
    _check(ctx, _lib.nms_modal_decomposition(ctx, _dev(maps), C.c_int(n_maps), C.c_int(k_max), _dev(out_Is), _dev(out_Ic),
                                             _dev(out_a), _dev(out_A)))


def nms_correlation_2d(ctx, fmap, rgrid, out_re=None, out_im=None):
    g, keep = _grid_struct(rgrid)
    _check(ctx, _lib.nms_correlation_2d(ctx, _dev(fmap), C.byref(g), _dev(out_re), _dev(out_im)))


def nms_correlation(ctx, I, q_of_bin, count, n_maps, n_bins, r, out_c, out_p):
    _check(ctx, _lib.nms_correlation(ctx, _dev(I), _dev(q_of_bin), _dev(count), C.c_int(n_maps), C.c_int(n_bins),
                                     _dev(r), C.c_int(int(r.shape[0])), _dev(out_c), _dev(out_p)))


def _hostbuf(t):
    """Host pointer of a NumPy array or a (pinned) CPU torch tensor; None -> NULL."""
    if t is None:
        return C.c_void_p(None)
    if isinstance(t, np.ndarray):
        if not t.flags["C_CONTIGUOUS"]:
            raise ValueError("host arrays must be contiguous")
        return C.c_void_p(t.ctypes.data)
    if t.is_cuda or not t.is_contiguous():
        raise ValueError("expected a contiguous host tensor")
    return C.c_void_p(t.data_ptr())


def nms_run_host(ctx, pos, N, m, R, grid, kinds, out_maps, n_bins=0, q_lo=0.0, q_hi=0.0, out_I=None, r=None,
                 out_c=None, out_p=None):
    """One whole step from HOST buffers (NumPy float32 arrays or pinned CPU tensors); synchronises."""
    g, keep = _grid_struct(grid)
    k, n = _kinds(kinds)
    Rh, Rp = _host(None if R is None else np.asarray(R, dtype=np.float64).reshape(9), np.float64)
    n_r = 0 if r is None else int(r.shape[0])
    _check(ctx, _lib.nms_run_host(ctx, _hostbuf(pos), _hostbuf(N), _hostbuf(m), C.c_int64(int(pos.shape[0])), Rp,
                                  C.byref(g), k, C.c_int(n), _hostbuf(out_maps), C.c_int(n_bins), C.c_double(q_lo),
                                  C.c_double(q_hi), _hostbuf(out_I), _hostbuf(r), C.c_int(n_r), _hostbuf(out_c),
                                  _hostbuf(out_p)))


def nms_run_host_split(ctx, pos, N, m, offsets, centres, R, grid, kinds, out_total, out_form):
    """nms_set_sample + nms_set_particles + nms_form_factor_split from HOST buffers; synchronises."""
    g, keep = _grid_struct(grid)
    k, n = _kinds(kinds)
    Rh, Rp = _host(None if R is None else np.asarray(R, dtype=np.float64).reshape(9), np.float64)
    off, offp = _host(offsets, np.int64)
    _check(ctx, _lib.nms_run_host_split(ctx, _hostbuf(pos), _hostbuf(N), _hostbuf(m), C.c_int64(int(pos.shape[0])), offp,
                                        C.c_int64(int(off.shape[0]) - 1), _hostbuf(centres), Rp, C.byref(g), k, C.c_int(n),
                                        _hostbuf(out_total), _hostbuf(out_form)))


def nms_run_host_scan(ctx, pos, N, m, rotations, grid, kinds, out_maps):
    """Rocking scan from HOST buffers: rotations [n_rot][3][3]; out_maps [n_rot][n_kinds][n_q]; synchronises."""
    g, keep = _grid_struct(grid)
    k, n = _kinds(kinds)
    Rs = np.ascontiguousarray(np.asarray(rotations, dtype=np.float64).reshape(-1, 9))
    _check(ctx, _lib.nms_run_host_scan(ctx, _hostbuf(pos), _hostbuf(N), _hostbuf(m), C.c_int64(int(pos.shape[0])),
                                       C.c_void_p(Rs.ctypes.data), C.c_int(int(Rs.shape[0])), C.byref(g), k, C.c_int(n),
                                       _hostbuf(out_maps)))


def nms_get_weight_sums(ctx) -> np.ndarray:
    out = np.zeros(4, dtype=np.float64)
    _check(ctx, _lib.nms_get_weight_sums(ctx, C.c_void_p(out.ctypes.data)))
    return out


PIPES = ["FFMA", "FFMA2_REG", "FFMA2_BCAST", "FMUL", "MUFU_SIN", "MUFU_EX2", "DFMA", "I2FP", "IALU", "LOP3", "F2F",
         "PHASOR_MUFU", "PHASOR_POLY"]


def nms_pipe_rates(ctx) -> dict:
    """Measured operations per clock and SM of the instruction classes the amplitude kernels are made of."""
    out = np.zeros(len(PIPES), dtype=np.float64)
    _check(ctx, _lib.nms_pipe_rates(ctx, C.c_void_p(out.ctypes.data)))
    return {k: float(v) for k, v in zip(PIPES, out)}


def nms_phasor_selftest(ctx, polynomial: bool, log2_n: int = 24) -> dict:
    """Error statistics of the kernels' phasor routine against fp64 (see include/nms.h)."""
    out = np.zeros(23, dtype=np.float64)
    _check(ctx, _lib.nms_phasor_selftest(ctx, C.c_int(1 if polynomial else 0), C.c_int(log2_n), C.c_void_p(out.ctypes.data)))
    return {"max_cos": out[0], "max_sin": out[1], "rms_cos": out[2], "rms_sin": out[3],
            "harmonics": {n: float(out[4 + n + 8]) for n in range(-8, 9)}, "mean_cos": float(out[21]), "mean_minus_sin": float(out[22])}


def nms_set_option(ctx, key: str, value: int):
    _check(ctx, _lib.nms_set_option(ctx, C.c_char_p(key.encode()), C.c_int64(value)))


def nms_get_info(ctx, key: str) -> int:
    v = C.c_int64(0)
    _check(ctx, _lib.nms_get_info(ctx, C.c_char_p(key.encode()), C.byref(v)))
    return int(v.value)


def nms_kernel_time_ms(ctx, which: int) -> float:
    ms = C.c_float(0.0)
    _check(ctx, _lib.nms_kernel_time_ms(ctx, C.c_int(which), C.byref(ms)))
    return float(ms.value)


def nms_kernel_time_total(ctx, which: int):
    """(total_ms, launches) of a kernel class since "timing" was last set."""
    tot, cnt = C.c_double(0.0), C.c_int64(0)
    _check(ctx, _lib.nms_kernel_time_total(ctx, C.c_int(which), C.byref(tot), C.byref(cnt)))
    return float(tot.value), int(cnt.value)


class Context:
    """RAII convenience around the functions above (`with Context() as ctx: nms_compute(ctx.h, ...)`)."""

    def __init__(self, device: int = 0, stream: Optional[int] = None):
        self.h = nms_create(device, stream)

    def close(self):
        if self.h is not None:
            nms_destroy(self.h)
            self.h = None

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
