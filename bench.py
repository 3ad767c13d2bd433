#!/usr/bin/env python3
"""bench.py -- throughput of the direct-summation SANS hot path on B200 (contract: see DESIGN.md section 8).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload C5] [--impl reference]

One "step" is one pass of the whole hot path over one synthetic workload whose raw arrays are already
resident in HBM: a-1 prep (rotate + order + pack), a-2 amplitude sums, a-3 reduce + response epilogue,
and, where the config asks for them, a-4 azimuthal average, a-5 correlation function, a-6 form-factor
split.  The metric is BASELINE.json's: Gpair/s = W * n_q * n_rotations * n_gpus / t, pairs actually
evaluated (no symmetry or merging tricks).  Rank 0 prints ONE JSON line.

 * value        device-resident inputs, CUDA events on the launching stream, max over ranks
 * e2e          same step through the C ABI with HOST buffers (pinned), H2D and D2H copies inside the
                timed region
 * roofline     the amplitude kernel: 12 FP32 lane-instructions per pair over its
                CUDA-event time inside the timed region, against N_SM * 128 lanes * sm_max_mhz
 * cpu_baseline the fp64 oracle as it stands, timed on this box's host cores on a bounded sample
 * --impl reference   the oracle alone (this tier's reference arm), same metric and config

N > 1: one process per GPU (under torchrun; `python bench.py --gpus N` alone starts the N ranks itself).  The detector
lines of ONE workload are split over the ranks where the workload admits it (--shard auto / lines: cells replicated,
all-gather of I(q) only; scaling = strong); otherwise, or with --shard replicas, every rank runs an independent
replica (no data-path collective; value = total pairs of all ranks / max-over-ranks time; scaling = weak).
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import nms_inputs as ni  # noqa: E402  (seeded input generators only; no arithmetic of the method)

FP32_LANE_INSTR_PER_PAIR = 12      # 8 accumulate FFMA + 4 for the phasor
LANES_PER_SM = 128
PREP_BYTES_PER_CELL = 60.0         # a-1: 28 B in (pos, N, m as float) + 32 B out (Cell record)


def ncu_traffic(workload: str):
    """dram__bytes_read.sum + dram__bytes_write.sum of ONE launch of the workload's amplitude kernel, from the
    committed summary of the `ncu --set full` captures (profiles/r2_traffic.json: workload -> kernel, bytes, commit);
    None if the workload was not captured.  The kernel is ALU-bound: the figure documents that DRAM traffic is
    irrelevant to the bound."""
    path = os.path.join(ROOT, "profiles", "r2_traffic.json")
    if not os.path.exists(path):
        return None
    with open(path) as f:
        rec = json.load(f).get(workload)
    return None if rec is None else float(rec["dram_bytes_read"]) + float(rec["dram_bytes_write"])


def _env_int(name, default):
    try:
        return int(os.environ.get(name, default))
    except ValueError:
        return default


def _peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            return json.load(f), "MEASURED_PEAKS.json"
    # fallback of /opt/skills/guides/B200_PROFILING.md: nominal B200 numbers
    return {"hbm_gbs": 7700.0, "sm_max_mhz": 1965.0}, "B200_PROFILING.md fallback (nominal)"


# ---------------------------------------------------------------------------------------------------
# clocks: sample NVML during the timed region
# ---------------------------------------------------------------------------------------------------
class ClockSampler:
    REASONS = {0x1: "gpu_idle", 0x2: "applications_clocks_setting", 0x4: "sw_power_cap", 0x8: "hw_slowdown",
               0x10: "sync_boost", 0x20: "sw_thermal_slowdown", 0x40: "hw_thermal_slowdown",
               0x80: "hw_power_brake_slowdown", 0x100: "display_clock_setting"}

    def __init__(self, index: int, period: float = 0.05):
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._stop = threading.Event()
        self._thr = None
        self.period = period
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
        except Exception:
            self.nv = None

    def _run(self):
        while not self._stop.is_set():
            try:
                self.samples.append(float(self.nv.nvmlDeviceGetClockInfo(self.h, self.nv.NVML_CLOCK_SM)))
                bits = int(self.nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h))
                for b, name in self.REASONS.items():
                    if bits & b and name != "gpu_idle":
                        self.reasons.add(name)
            except Exception:
                pass
            self._stop.wait(self.period)

    def start(self):
        if self.nv is not None:
            self._stop.clear()
            self._thr = threading.Thread(target=self._run, daemon=True)
            self._thr.start()

    def stop(self):
        if self._thr is not None:
            self._stop.set()
            self._thr.join()
            self._thr = None

    def summary(self):
        med = float(np.median(self.samples)) if self.samples else None
        return {"sm_mhz": med, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons), "samples": len(self.samples)}


# ---------------------------------------------------------------------------------------------------
# the CUDA arm
# ---------------------------------------------------------------------------------------------------
class Runner:
    """Owns one context, the device-resident raw arrays of one workload and its output buffers."""

    def __init__(self, nms, wl, device: int, shard=None):
        import torch
        self.nms, self.wl, self.torch = nms, wl, torch
        self.shard = shard                       # None, or (full workload, world, rank, dist) under --shard lines
        self.dev = torch.device("cuda", device)
        self.ctx = nms.Context(device)
        self.h = self.ctx.h
        pin = lambda a: None if a is None else torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
        self.h_pos, self.h_N, self.h_m = pin(wl.pos), pin(wl.N), pin(wl.m)
        self.h_cen = pin(wl.centres)
        up = lambda t: None if t is None else t.to(self.dev, non_blocking=True)
        self.d_pos, self.d_N, self.d_m, self.d_cen = up(self.h_pos), up(self.h_N), up(self.h_m), up(self.h_cen)
        nk, nq = len(wl.kinds), wl.grid.n_q
        f32 = dict(dtype=torch.float32, device=self.dev)
        self.maps = torch.empty((nk, nq), **f32)
        self.form = torch.empty((nk, nq), **f32) if wl.split else None
        self.h_maps = torch.empty((nk, nq), dtype=torch.float32).pin_memory()
        self.h_form = torch.empty((nk, nq), dtype=torch.float32).pin_memory() if wl.split else None
        self.nb = wl.n_bins
        if self.nb:
            self.I = torch.empty((nk, self.nb), **f32)
            self.qb = torch.empty(self.nb, **f32)
            self.cnt = torch.empty(self.nb, dtype=torch.int32, device=self.dev)
            self.h_I = torch.empty((nk, self.nb), dtype=torch.float32).pin_memory()
        self.nr = 0 if wl.r is None else len(wl.r)
        if self.nr:
            self.h_r = pin(wl.r)
            self.d_r = up(self.h_r)
            self.c = torch.empty((nk, self.nr), **f32)
            self.p = torch.empty((nk, self.nr), **f32)
            self.h_c = torch.empty((nk, self.nr), dtype=torch.float32).pin_memory()
            self.h_p = torch.empty((nk, self.nr), dtype=torch.float32).pin_memory()
        self.rots = wl.rotations if wl.rotations is not None else [wl.R]
        self.h_scan = torch.empty((len(self.rots), nk, nq), dtype=torch.float32).pin_memory() if len(self.rots) > 1 else None
        torch.cuda.synchronize(self.dev)

    # -- one pass of the hot path, raw arrays resident in HBM -------------------------------------------
    def _post(self):
        nms, wl, h = self.nms, self.wl, self.h
        if self.nb:
            nms.nms_azimuthal_average(h, self.maps, len(wl.kinds), self.nb, wl.q_lo, wl.q_hi, self.I, self.qb, self.cnt)
            if self.nr and self.shard is None:
                nms.nms_correlation(h, self.I, self.qb, self.cnt, len(wl.kinds), self.nb, self.d_r, self.c, self.p)
            elif self.nr:
                full, world, rank, dist = self.shard                  # every ring is needed: all-gather I(q)
                nms.nms_synchronize(h)
                I_full = gather_lines(self.I, full.grid.n0, world, rank, dist)
                if not hasattr(self, "q_full"):
                    self.q_full = self.torch.as_tensor(full.grid.u0, device=self.dev)
                    self.cnt_full = self.torch.full((full.grid.n0,), full.grid.n1, dtype=self.torch.int32, device=self.dev)
                nms.nms_correlation(h, I_full, self.q_full, self.cnt_full, len(wl.kinds), full.grid.n0, self.d_r, self.c, self.p)

    def step_device(self, d2h: bool = False):
        nms, wl, h = self.nms, self.wl, self.h
        nms.nms_set_sample(h, self.d_pos, self.d_N, self.d_m, self.rots[0])          # a-1
        if wl.offsets is not None:
            nms.nms_set_particles(h, wl.offsets, self.d_cen)
        nms.nms_set_polarization(h, wl.P)
        for i, R in enumerate(self.rots):
            if i > 0:
                nms.nms_set_rotation(h, R)                                            # a-1 again (rocking scan)
            if wl.split:
                nms.nms_form_factor_split(h, wl.grid, wl.kinds, self.maps, self.form)  # a-6 (+ a-2, a-3)
            else:
                nms.nms_compute(h, wl.grid, wl.kinds, self.maps)                       # a-2 + a-3
            self._post()                                                              # a-4, a-5
            if d2h:
                self.h_maps.copy_(self.maps, non_blocking=True)
                if wl.split:
                    self.h_form.copy_(self.form, non_blocking=True)
                if self.nb:
                    self.h_I.copy_(self.I, non_blocking=True)
                if self.nr:
                    self.h_c.copy_(self.c, non_blocking=True)
                    self.h_p.copy_(self.p, non_blocking=True)

    # -- the same step from HOST buffers: ONE C-ABI call, H2D of the raw arrays and D2H of every result inside ---------
    def step_host(self):
        nms, wl, h, torch = self.nms, self.wl, self.h, self.torch
        if self.shard is not None:
            # line sharding under torchrun: the exchange step (all-gather of I(q)) sits between the passes, so the
            # binding-level calls are used with explicit pinned copies (nms_set_sample accepts host pointers as well)
            self.d_pos.copy_(self.h_pos, non_blocking=True)
            if self.d_N is not None:
                self.d_N.copy_(self.h_N, non_blocking=True)
            if self.d_m is not None:
                self.d_m.copy_(self.h_m, non_blocking=True)
            if self.d_cen is not None:
                self.d_cen.copy_(self.h_cen, non_blocking=True)
            self.step_device(d2h=True)
            torch.cuda.current_stream(self.dev).synchronize()
        elif wl.split:
            nms.nms_set_polarization(h, wl.P)
            nms.nms_run_host_split(h, self.h_pos, self.h_N, self.h_m, wl.offsets, self.h_cen, wl.R, wl.grid, wl.kinds,
                                   self.h_maps, self.h_form)
        elif len(self.rots) > 1:
            nms.nms_set_polarization(h, wl.P)
            nms.nms_run_host_scan(h, self.h_pos, self.h_N, self.h_m, self.rots, wl.grid, wl.kinds, self.h_scan)
        else:
            nms.nms_set_polarization(h, wl.P)
            nms.nms_run_host(h, self.h_pos, self.h_N, self.h_m, wl.R, wl.grid, wl.kinds, self.h_maps, self.nb, wl.q_lo,
                             wl.q_hi, self.h_I if self.nb else None, self.h_r if self.nr else None,
                             self.h_c if self.nr else None, self.h_p if self.nr else None)

    def bytes_per_step(self):
        wl = self.wl
        h2d = sum(t.numel() * t.element_size() for t in (self.h_pos, self.h_N, self.h_m, self.h_cen) if t is not None)
        per_rot = self.h_maps.numel() * 4 + (self.h_form.numel() * 4 if wl.split else 0)
        if self.nb:
            per_rot += self.h_I.numel() * 4
        if self.nr:
            h2d += self.h_r.numel() * 4
            per_rot += 2 * self.h_c.numel() * 4
        return int(h2d), int(per_rot * len(self.rots))

    def close(self):
        self.ctx.close()


def time_next_rows(nms, run, wl, torch, dev, reps=3, step_ms=None):
    """SURVEY 8(f) rows built so far, timed OUTSIDE the step on the step's last maps (polar detectors only):
    f-2 angular modal decomposition of all maps (k_max = 8) and f-1 two-dimensional correlation function of the
    first map on a (rho, alpha) grid of the detector's own size -- the amplitude kernel with pixels as cells."""
    h, nk, g = run.h, len(wl.kinds), wl.grid
    k_max = 8
    f32 = dict(dtype=torch.float32, device=dev)
    Is, Ic = torch.empty((nk, k_max + 1, g.n0), **f32), torch.empty((nk, k_max + 1, g.n0), **f32)
    a, A = torch.empty((nk, 2, k_max + 1), **f32), torch.empty((nk, 2, k_max + 1), **f32)
    r_max = float(np.pi / max(float(g.u0[1] - g.u0[0]), 1e-30)) if g.n0 > 1 else 1.0      # Nyquist range of the q grid
    rgrid = ni.polar_grid(np.linspace(0.0, r_max, g.n0), g.n1)
    re, im = torch.empty(rgrid.n_q, **f32), torch.empty(rgrid.n_q, **f32)
    out = {}
    for name, fn, units in (("modal_f2", lambda: nms.nms_modal_decomposition(h, run.maps, nk, k_max, Is, Ic, a, A),
                             nk * g.n_q * (k_max + 1)),
                            ("correlation_2d_f1", lambda: nms.nms_correlation_2d(h, run.maps[0], rgrid, re, im),
                             g.n_q * rgrid.n_q)):
        fn()
        ms = _timed(torch, dev, fn, reps) / reps
        out[name] = {"ms": ms, "units": units, "gunits_per_s": units / (ms * 1e-3) / 1e9}
    # f-3: B = 6 magnetisation fields (two passes of 3) on the workload's geometry; the fields are the sample's own
    # moments with permuted components and flipped signs (made on the device; the kernel cannot tell)
    if run.d_m is not None:
        B = 6
        mb = torch.stack([torch.roll(run.d_m, b % 3, dims=1) * (1.0 if b < 3 else -1.0) for b in range(B)]).contiguous()
        bmaps = torch.empty((B, nk, g.n_q), **f32)
        fn = lambda: nms.nms_compute_batch(h, wl.grid, mb, wl.kinds, bmaps, None)
        fn()
        ms = _timed(torch, dev, fn, 1)
        units = B * wl.W * g.n_q
        out["batched_fields_f3"] = {"ms": ms, "fields": B, "units": units, "gunits_per_s": units / (ms * 1e-3) / 1e9,
                                    "unit": "cell x q x field triples (shared phasor and nuclear sum; whole call incl. packing and responses)",
                                    "speedup_vs_single_field_step": (units / ms) / (wl.pairs / wl.n_rot / step_ms) if step_ms else None}
        del mb, bmaps
    # f-4: Friedel halving, an EFFECTIVE rate (half of the pairs are taken from A(-q) = A(q)^*); never the headline
    nms.nms_set_option(h, "friedel", 1)
    try:
        fn = lambda: nms.nms_compute(h, wl.grid, wl.kinds, run.maps)
        fn()
        ms = _timed(torch, dev, fn, 2) / 2
        out["friedel_f4"] = {"ms": ms, "effective_gpair_s": wl.W * g.n_q / (ms * 1e-3) / 1e9, "evaluated_gpair_s": 0.5 * wl.W * g.n_q / (ms * 1e-3) / 1e9,
                             "unit": "EFFECTIVE cell x q pairs per second of nms_compute with option friedel = 1 (half evaluated, half by conjugation)"}
    except nms.NmsError as e:
        out["friedel_f4"] = {"unavailable": str(e)}
    nms.nms_set_option(h, "friedel", 0)
    out["modal_f2"]["unit"] = "map values x harmonics"
    out["correlation_2d_f1"]["unit"] = "pixel x r-point pairs (one complex amplitude)"
    out["correlation_2d_f1"]["r_grid"] = f"polar {rgrid.n0}x{rgrid.n1}, rho <= {r_max:.1f}"
    return out


def _timed(torch, dev, fn, steps, dist=None):
    """Time exactly `steps` calls of fn between barrier + synchronize on both sides; ms, max over ranks."""
    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize(dev)
    beg, end = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    beg.record()
    for _ in range(steps):
        fn()
    end.record()
    torch.cuda.synchronize(dev)
    ms = beg.elapsed_time(end)
    if dist is not None:
        dist.barrier()
    return max_over_ranks(ms, dist, torch, dev)


def max_over_ranks(value: float, dist=None, torch=None, dev=None) -> float:
    """MAX-reduce a scalar over the process group (identity without one).  Works on gloo (CPU) and nccl."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(value)
    import torch as _t
    t = _t.tensor([float(value)], dtype=_t.float64, device=dev if dist.get_backend() == "nccl" else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def shard_lines(n0: int, world: int, rank: int):
    """Contiguous, balanced share [i0, i1) of the n0 detector lines (rings of a polar grid, rows of a Cartesian one)
    of rank `rank` (the detector points are independent units; the cells are replicated)."""
    base, extra = divmod(n0, world)
    i0 = rank * base + min(rank, extra)
    return i0, i0 + base + (1 if rank < extra else 0)


def can_shard_lines(wl, world: int) -> bool:
    """Line sharding covers polar and Cartesian detectors with at least one line per rank, except
    |q| histograms on Cartesian detectors (bins straddle ranks)."""
    g = wl.grid
    return g.type != 2 and not (g.type == 1 and wl.n_bins) and g.n0 >= world


def shard_workload(wl, world: int, rank: int):
    """This rank's part of a workload under line sharding: same sample, the detector lines [i0, i1)."""
    import copy
    g = wl.grid
    if g.type == 2:
        raise SystemExit("bench.py: --shard lines needs a polar or Cartesian detector")
    if g.type == 1 and wl.n_bins:
        raise SystemExit("bench.py: --shard lines does not cover |q| histograms on Cartesian detectors (bins straddle ranks)")
    i0, i1 = shard_lines(g.n0, world, rank)
    if i1 <= i0:
        raise SystemExit("bench.py: more ranks than detector lines")
    part = copy.copy(wl)
    part.grid = ni.polar_grid(g.u0[i0:i1], g.n1) if g.type == 0 else ni.cartesian_grid(g.u0[i0:i1], g.u1)
    if g.type == 0:
        part.grid.u1 = g.u1                     # the very same float32 angles
    part.n_bins = (i1 - i0) if wl.n_bins else 0
    return part, i0, i1


def gather_lines(local, n0: int, world: int, rank: int, dist):
    """All-gather per-line results local [n_rows, n_local] (ring averages I(q_i)) into [n_rows, n0] on every rank --
    the one exchange step of the sharded path (the Fourier-Bessel transform needs every ring).  Equal-sized padded
    buffers, so it runs on nccl and gloo alike."""
    import torch
    n_max = -(-n0 // world)
    pad = torch.zeros((local.shape[0], n_max), dtype=local.dtype, device=local.device)
    pad[:, :local.shape[1]] = local
    parts = [torch.empty_like(pad) for _ in range(world)]
    dist.all_gather(parts, pad)
    out = torch.empty((local.shape[0], n0), dtype=local.dtype, device=local.device)
    for r in range(world):
        i0, i1 = shard_lines(n0, world, r)
        out[:, i0:i1] = parts[r][:, :i1 - i0]
    return out


def aggregate_rate(pairs_per_rank: int, world: int, ms_max: float) -> float:
    """Whole-job Gpair/s: every rank evaluated pairs_per_rank pairs in (max over ranks) ms_max."""
    return pairs_per_rank * world / (ms_max * 1e-3) / 1e9


# ---------------------------------------------------------------------------------------------------
# the oracle arm (cpu_baseline leg and --impl reference): the only places bench.py executes oracle/
# ---------------------------------------------------------------------------------------------------
def oracle_step(oracle, wl, qy, qz, th, idx):
    """One bounded sample of the workload through the fp64 oracle as it stands: all cells x the detector
    points idx (first rotation only), responses, and the 1-D passes when the sample is the full detector."""
    full = len(idx) == wl.grid.n_q
    R = wl.rotations[0] if wl.rotations is not None else wl.R
    if wl.split:
        tot, form = oracle.form_factor_split(wl.pos, wl.N, wl.m, wl.offsets, wl.kinds, qy[idx], qz[idx], th[idx], R=R,
                                             centres=wl.centres, P=wl.P)
        return tot
    A = oracle.amplitudes(wl.pos, wl.N, wl.m, R, qy[idx], qz[idx], offsets=wl.offsets, centres=wl.centres)
    M = oracle.response(A, th[idx], wl.kinds, P=wl.P)
    if full and wl.n_bins:
        if wl.grid.type == 0 and not (wl.q_hi > wl.q_lo):
            I = oracle.azimuthal_polar(M, wl.grid.n0, wl.grid.n1)
            qb, cnt = wl.grid.u0.astype(np.float64), None
        else:
            I, cnt = oracle.azimuthal_hist(M, qy, qz, wl.n_bins, wl.q_lo, wl.q_hi)
            qb = oracle.hist_bin_centres(wl.n_bins, wl.q_lo, wl.q_hi)
        if wl.r is not None:
            oracle.correlation(I, qb, wl.r, count=cnt)
    return M


def oracle_sample(wl, n_sample):
    n = min(n_sample, wl.grid.n_q)
    if n == wl.grid.n_q:
        return np.arange(n, dtype=np.int64)
    return ni.q_subset(wl.grid.n_q, n, 9000 + (int(wl.name[1]) if wl.name[1].isdigit() else 0))


def parity_report(wl, maps_gpu, idx, M_ref):
    """The step's GPU maps against the oracle maps on the timed sample of detector points, by the north_star criterion
    taken literally: relative error wherever |oracle| > 1e-6 of the (GPU) map's own maximum, tolerance 1e-3, for every
    kind.  The positive kinds and the signed difference kinds NM / CHI are reported separately; `signed_literal` says
    how many of the tested points of the signed kinds miss the tolerance and by how much."""
    names = [ni.KINDS[k] for k in wl.kinds]
    fmax = np.abs(maps_gpu).max(axis=1)
    worst_pos, tested_pos, fail_pos = 0.0, 0, 0
    worst_sig, tested_sig, fail_sig = 0.0, 0, 0
    for i, name in enumerate(names):
        sel = np.abs(M_ref[i]) > 1e-6 * fmax[i]
        if not sel.any():
            continue
        rel = np.abs(maps_gpu[i][idx][sel] - M_ref[i][sel]) / np.abs(M_ref[i][sel])
        if name in ("NM", "CHI"):
            worst_sig, tested_sig, fail_sig = max(worst_sig, float(rel.max())), tested_sig + int(sel.sum()), fail_sig + int((rel > 1e-3).sum())
        else:
            worst_pos, tested_pos, fail_pos = max(worst_pos, float(rel.max())), tested_pos + int(sel.sum()), fail_pos + int((rel > 1e-3).sum())
    return {"detector_points": int(len(idx)), "tolerance": 1e-3, "floor": "1e-6 of the map's own maximum",
            "positive_kinds": {"points_tested": tested_pos, "points_failing": fail_pos, "worst_rel": worst_pos},
            "signed_literal": {"points_tested": tested_sig, "points_failing": fail_sig, "worst_rel": worst_sig}}


def time_oracle(wl, target_s=12.0, steps=1, warmup=0, keep=None):
    """Gpair/s of the oracle on a sample sized for about target_s seconds per step (probe first, then scale).
    keep: dict that receives the sample indices and the oracle maps of the last step (for the parity report)."""
    import oracle
    oracle.build()
    qy, qz, th = oracle.grid_points(wl.grid)
    n = 8
    while True:                                        # probe with growing samples until the timing is meaningful
        probe = oracle_sample(wl, n)
        t0 = time.perf_counter()
        oracle_step(oracle, wl, qy, qz, th, probe)
        el = time.perf_counter() - t0
        if el >= 0.5 or len(probe) == wl.grid.n_q:
            break
        n *= 8
    rate = wl.W * len(probe) / max(el, 1e-9)
    n = int(max(8, min(wl.grid.n_q, rate * target_s / wl.W)))
    idx = oracle_sample(wl, n)
    for _ in range(warmup):
        oracle_step(oracle, wl, qy, qz, th, idx)
    t0 = time.perf_counter()
    for _ in range(steps):
        M = oracle_step(oracle, wl, qy, qz, th, idx)
    dt = (time.perf_counter() - t0) / steps
    if keep is not None:
        keep["idx"], keep["M"] = idx, M
    pairs = wl.W * len(idx)
    return {"value": pairs / dt / 1e9, "unit": "Gpair/s", "cores": oracle.num_threads(), "kind": "oracle",
            "sample": f"all {wl.W} cells x {len(idx)} of {wl.grid.n_q} detector points (seeded subset, first rotation), "
                      f"fp64, {dt:.2f} s per step"}, dt * 1e3


def metric_name():
    with open(os.path.join(ROOT, "BASELINE.json")) as f:
        return json.load(f)["metric"]


def workload_config(wl, extra=None):
    g = wl.grid
    cfg = {"workload": f"{wl.name}: {WORKLOAD_TEXT[wl.name]}", "cells": wl.W,
           "detector": f"{['polar', 'cartesian', 'list'][g.type]} {g.n0}x{g.n1}", "n_q": g.n_q, "rotations": wl.n_rot,
           "pairs_per_step": wl.pairs, "kinds": [ni.KINDS[k] for k in wl.kinds],
           "cache": "inputs larger than L2" if wl.W * 28 > 126e6 else "inputs fit in L2; each step re-packs them"}
    if extra:
        cfg.update(extra)
    return cfg


WORKLOAD_TEXT = {
    "C1": "uniformly magnetized sphere, 1 nm cells, R = 10 nm",
    "C2": "vortex disc, 2 nm cells, rotated ZYZ (30,45,0) deg, all responses, I(q), c(r), p(r)",
    "C3": "ensemble of 1000 spheres (R = 5 nm, 0.5 nm cells), total and form-factor outputs",
    "C4": "skyrmion-lattice film 512x512x8, rocking scan of 36 rotations about z",
    "C5": "micromagnetic block 256^3 with 5 % pores, all responses, I(q), c(r), p(r)",
}


def run_reference(args, rank):
    if rank != 0:
        return
    if _env_int("WORLD_SIZE", 1) > 1:
        # torchrun pins OMP_NUM_THREADS=1 for its workers; rank 0 alone runs the oracle, so give it the box's cores back
        try:
            import ctypes
            ctypes.CDLL("libgomp.so.1").omp_set_num_threads(len(os.sched_getaffinity(0)))
        except Exception:
            pass
    wl = ni.make_config(args.workload)
    cb, ms = time_oracle(wl, target_s=args.oracle_seconds, steps=max(args.steps, 1), warmup=min(args.warmup, 1))
    line = {"impl": "reference", "metric": metric_name(), "value": cb["value"], "unit": "Gpair/s", "n_gpus": args.gpus,
            "steps": args.steps, "warmup": min(args.warmup, 1), "ms_per_step": ms, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": workload_config(wl), "cpu_baseline": cb,
            "e2e": {"value": cb["value"], "unit": "Gpair/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def run_sweep(args):
    """Context measurement, not the contract line: the paper's runtime experiment (Fig. 10) re-created
    synthetically -- step time against the number of cells for K = 10 ... 25 600 identical vortex spheres of 4169
    cells (ni.config_fig10), all 13 responses + ring average + c(r), p(r) on a 256 x 256 polar detector."""
    import torch
    import paper_2601_18444_b200 as nms
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(dev)
    points = []
    for K in (10, 40, 160, 640, 2560, 10240, 25600):
        wl = ni.config_fig10(K)
        run = Runner(nms, wl, 0)
        for _ in range(2):
            run.step_device()
        steps = 3 if K <= 2560 else 2
        ms = _timed(torch, dev, run.step_device, steps) / steps
        points.append({"particles": K, "cells": wl.W, "ms_per_step": ms, "gpair_s": wl.pairs / (ms * 1e-3) / 1e9,
                       "variant": nms.nms_get_info(run.h, "variant_used")})
        run.close()
        del run, wl
        torch.cuda.empty_cache()
    print(json.dumps({"sweep": "fig10", "detector": "polar 256x256, |q| 0.01-1.5 linear", "kinds": 13,
                      "note": "whole step per point: prep + amplitudes + responses + I(q) + c(r), p(r); inputs resident",
                      "points": points}), flush=True)


def measure(nms, torch, wl_full, args, steps, warmup, dist, rank, local_rank, world, sharded, headline, precision=0):
    """Time one workload: device-resident arm with the roofline of the amplitude kernel and, for the headline
    workload, the end-to-end arm, the next rows, the oracle (cpu_baseline) and the parity of this very run."""
    dev = torch.device("cuda", local_rank)
    if sharded:
        wl, line0, line1 = shard_workload(wl_full, world, rank)
        run = Runner(nms, wl, local_rank, shard=(wl_full, world, rank, dist))
    else:
        wl = wl_full
        run = Runner(nms, wl, local_rank)
    h = run.h
    nms.nms_set_option(h, "precision", precision)         # 0: the library's own choice; 1: fast variant forced
    sampler = ClockSampler(local_rank)

    # ---- device-resident arm -------------------------------------------------------------------------
    for _ in range(warmup):
        run.step_device()
    nms.nms_synchronize(h)
    launches0 = nms.nms_get_info(h, "launches")
    nms.nms_set_option(h, "timing", 1)                 # event pair around every kernel; resets the record
    sampler.start()
    ms_total = _timed(torch, dev, run.step_device, steps, dist)
    sampler.stop()
    launches = nms.nms_get_info(h, "launches") - launches0
    kt = {name: nms.nms_kernel_time_total(h, idx) for name, idx in
          (("prep", nms.NMS_T_PREP), ("amplitude", nms.NMS_T_AMPLITUDE), ("epilogue", nms.NMS_T_EPILOGUE),
           ("azimuthal", nms.NMS_T_AZIMUTHAL), ("correlation", nms.NMS_T_CORRELATION))}
    nms.nms_set_option(h, "timing", 0)
    ms_step = ms_total / steps
    # replicas: every rank evaluates the whole workload (weak); line sharding: the ranks share ONE workload (strong)
    value = aggregate_rate(wl_full.pairs, 1 if sharded else world, ms_step)

    # ---- roofline of the dominant kernel (amplitude sums) --------------------------------------------
    peaks, peak_src = _peaks()
    sm_count = nms.nms_get_info(h, "sm_count")
    amp_ms, amp_n = kt["amplitude"]
    amp_ms_per_launch = amp_ms / max(amp_n, 1)
    pairs_per_launch = wl.W * wl.grid.n_q
    achieved = pairs_per_launch * FP32_LANE_INSTR_PER_PAIR / (amp_ms_per_launch * 1e-3) / 1e12
    peak = sm_count * LANES_PER_SM * peaks["sm_max_mhz"] * 1e6 / 1e12
    clocks = sampler.summary()
    roofline = {"bound": "alu", "kernel": "k_amp (a-2 amplitude sums)", "achieved": achieved, "peak": peak,
                "unit": "T FP32 lane-instr/s (12 per pair)", "frac": achieved / peak,
                "traffic": ncu_traffic(wl.name),
                "peak_source": f"{sm_count} SMs x 128 FP32 lanes x sm_max_mhz {peaks['sm_max_mhz']:.0f} ({peak_src})",
                "gpair_s_kernel": pairs_per_launch / (amp_ms_per_launch * 1e-3) / 1e9,
                "ms_per_launch": amp_ms_per_launch, "launches_timed": amp_n,
                "share_of_step": amp_ms / ms_total,
                "frac_at_sampled_clock": (achieved / (sm_count * LANES_PER_SM * clocks["sm_mhz"] * 1e6 / 1e12))
                if clocks.get("sm_mhz") else None,
                "variant": nms.nms_get_info(h, "variant_used"), "qt": nms.nms_get_info(h, "qt"),
                "bases": nms.nms_get_info(h, "bases"), "three_term": nms.nms_get_info(h, "three_term"),
                "poly_phasors": nms.nms_get_info(h, "poly_phasors"), "interpolating": nms.nms_get_info(h, "interp"),
                "cell_chunks": nms.nms_get_info(h, "n_chunks"), "blocks_per_sm": nms.nms_get_info(h, "blocks_per_sm")}
    res = {"value": value, "ms_per_step": ms_step, "steps": steps, "warmup": warmup, "roofline": roofline,
           "clocks": clocks, "gpu_launches": launches, "pairs_per_step": wl_full.pairs}
    if headline:
        passes = {}
        hbm = peaks.get("hbm_gbs", 0.0)
        nk, nq = len(wl.kinds), wl.grid.n_q
        alg_bytes = {"prep": wl.W * PREP_BYTES_PER_CELL,                        # 28 B in, 32 B out per cell (a-1)
                     "azimuthal": nk * nq * 4.0 + nk * max(wl.n_bins, 1) * 4.0,  # maps in, I(q) out (a-4)
                     "correlation": nk * max(wl.n_bins, 1) * 4.0 + 2.0 * nk * max(run.nr, 1) * 4.0}   # a-5
        for name in ("prep", "epilogue", "azimuthal", "correlation"):
            t, n = kt[name]
            if n:
                passes[name] = {"ms_per_launch": t / n, "launches": n}
                if name in alg_bytes:
                    gbs = alg_bytes[name] / (t / n * 1e-3) / 1e9
                    passes[name].update({"achieved_gbs": gbs, "frac_of_hbm_peak": gbs / hbm if hbm else None})
        res["passes"] = passes
        # ---- end-to-end arm: host buffers, copies inside the timed region ----------------------------
        for _ in range(min(warmup, 3)):
            run.step_host()
        e2e_steps = max(1, min(steps, 10))
        ms_e2e = _timed(torch, dev, run.step_host, e2e_steps, dist) / e2e_steps
        h2d, d2h = run.bytes_per_step()
        res["e2e"] = {"value": aggregate_rate(wl_full.pairs, 1 if sharded else world, ms_e2e), "unit": "Gpair/s",
                      "ms_per_step": ms_e2e, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h, "steps": e2e_steps}
        res["next_rows"] = time_next_rows(nms, run, wl, torch, dev, step_ms=ms_step) if (wl.grid.type == 0 and not sharded) else None
    # the maps of the FIRST rotation of one more (untimed) pass, for the parity object
    maps_host = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        nms.nms_set_sample(h, run.d_pos, run.d_N, run.d_m, run.rots[0])
        if wl.offsets is not None:
            nms.nms_set_particles(h, wl.offsets, run.d_cen)
        nms.nms_set_polarization(h, wl.P)
        if wl.split:
            nms.nms_form_factor_split(h, wl.grid, wl.kinds, run.maps, run.form)
        else:
            nms.nms_compute(h, wl.grid, wl.kinds, run.maps)
        nms.nms_synchronize(h)
        maps_host = run.maps.cpu().numpy().astype(np.float64)
    run.close()
    res["cpu_baseline"], res["parity"] = None, None
    if maps_host is not None:
        keep = {}
        res["cpu_baseline"], _ = time_oracle(wl, target_s=args.oracle_seconds if headline else min(args.oracle_seconds, 3.0), keep=keep)
        res["parity"] = parity_report(wl, maps_host, keep["idx"], keep["M"])   # the oracle sample doubles as a parity check
    return res


def run_cuda(args, rank, local_rank, world):
    import torch
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product has no CPU fallback (use --impl reference for the oracle)")
    import paper_2601_18444_b200 as nms       # raises if libnms.so is missing and cannot be built
    dist = None
    if world > 1:
        import torch.distributed as dist
        torch.cuda.set_device(local_rank)
        dist.init_process_group(backend="nccl", device_id=torch.device("cuda", local_rank))
    torch.cuda.set_device(torch.device("cuda", local_rank))

    wl_full = ni.make_config(args.workload)
    sharded = world > 1 and (args.shard == "lines" or (args.shard == "auto" and can_shard_lines(wl_full, world)))
    res = measure(nms, torch, wl_full, args, args.steps, args.warmup, dist, rank, local_rank, world, sharded, True,
                  precision=args.precision)
    # the other two throughput configs of the north-star target (>= 60 % on C3-C5), timed OUTSIDE the headline region
    configs = None
    if world == 1 and not args.no_configs:
        configs = {}
        for name in ("C3", "C4", "C5"):
            if name == args.workload:
                continue
            r = measure(nms, torch, ni.make_config(name), args, 3, 3, None, rank, local_rank, 1, False, False)
            configs[name] = {"value": r["value"], "unit": "Gpair/s", "ms_per_step": r["ms_per_step"], "steps": r["steps"],
                             "warmup": r["warmup"], "roofline_frac": r["roofline"]["frac"],
                             "kernel_ms_per_launch": r["roofline"]["ms_per_launch"], "variant": r["roofline"]["variant"],
                             "cell_chunks": r["roofline"]["cell_chunks"], "clocks": r["clocks"], "parity": r["parity"],
                             "pairs_per_step": r["pairs_per_step"]}

        # The headline workload asks for the signed kinds NM / CHI, so the library runs the ACCURATE variant of its fp32
        # kernels (polynomial phasors, fp64 sub-accumulation of the nuclear channel: the variant that meets the north-star
        # criterion for them at every detector point).  Beside it: the same workload with the FAST
        # variant forced (option "precision" = 1: MUFU phasors, three-term recurrence), with its own parity object.
        if any(ni.KINDS[k] in ("NM", "CHI") for k in wl_full.kinds):
            r = measure(nms, torch, wl_full, args, 3, 3, None, rank, local_rank, 1, False, False, precision=1)
            configs[args.workload + "_precision1_fast"] = {
                "value": r["value"], "unit": "Gpair/s", "ms_per_step": r["ms_per_step"], "steps": r["steps"], "warmup": r["warmup"],
                "roofline_frac": r["roofline"]["frac"], "kernel_ms_per_launch": r["roofline"]["ms_per_launch"],
                "variant": r["roofline"]["variant"], "poly_phasors": r["roofline"]["poly_phasors"],
                "three_term": r["roofline"]["three_term"],
                "cell_chunks": r["roofline"]["cell_chunks"], "clocks": r["clocks"], "parity": r["parity"],
                "pairs_per_step": r["pairs_per_step"]}

    if rank == 0:
        line = {"metric": metric_name(), "value": res["value"], "unit": "Gpair/s", "n_gpus": world, "steps": args.steps,
                "warmup": args.warmup, "ms_per_step": res["ms_per_step"], "higher_is_better": True,
                "scaling": "strong" if sharded else "weak",
                "vs_baseline": None, "dtype": "f32", "data": "synthetic",
                "config": workload_config(wl_full, {"precision_option": args.precision, "parallelism": ("detector lines sharded over ranks, cells replicated, all-gather of I(q) only"
                                                                    if sharded else "replicas only") if world > 1 else "single GPU"}),
                "clocks": res["clocks"], "e2e": res["e2e"], "gpu_launches": res["gpu_launches"], "roofline": res["roofline"],
                "passes": res["passes"], "next_rows": res["next_rows"], "cpu_baseline": res["cpu_baseline"],
                "parity": res["parity"], "configs": configs}
        print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser(description=__doc__, formatter_class=argparse.RawDescriptionHelpFormatter)
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="C5", choices=["C1", "C2", "C3", "C4", "C5"])
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--oracle-seconds", type=float, default=12.0, help="CPU seconds per oracle step (bounded sample)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--sweep", action="store_true",
                    help="context only: step time against cell count for the paper's Fig. 10 workload (one JSON line)")
    ap.add_argument("--shard", default="auto", choices=["auto", "replicas", "lines"],
                    help="N > 1: the detector lines of ONE workload shared by the ranks (strong scaling; DESIGN.md "
                         "section 9) or independent replicas (weak scaling); auto = lines where the workload admits it")
    ap.add_argument("--pipes", action="store_true",
                    help="measured issue rates of the instruction classes of the amplitude kernels and error statistics "
                         "of the two phasor routines (one JSON line; the table behind DESIGN.md section 6)")
    ap.add_argument("--precision", type=int, default=0, choices=[0, 1, 2],
                    help="kernel variant of the timed workload: 0 the library's own choice (default), 1 fast, 2 accurate")
    ap.add_argument("--no-configs", action="store_true", help="skip the C3 / C4 side measurements of the default line")
    args = ap.parse_args()
    rank, local_rank, world = _env_int("RANK", 0), _env_int("LOCAL_RANK", 0), _env_int("WORLD_SIZE", 1)
    if world != args.gpus and world > 1:
        raise SystemExit(f"bench.py: --gpus {args.gpus} but WORLD_SIZE={world}")
    if args.gpus > 1 and world == 1:
        # not under torchrun: start the N ranks ourselves (one process per GPU) and become their launcher
        import socket
        with socket.socket() as sk:
            sk.bind(("127.0.0.1", 0))
            port = sk.getsockname()[1]
        os.execv(sys.executable, [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(args.gpus),
                                  "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:])
    if args.pipes:
        if rank == 0:
            import torch
            import paper_2601_18444_b200 as nms
            peaks, src = _peaks()
            with nms.Context(0) as ctx:
                rates = nms.nms_pipe_rates(ctx.h)
                st = {name: nms.nms_phasor_selftest(ctx.h, poly, 24) for name, poly in (("mufu", False), ("polynomial", True))}
            for v in st.values():
                v["harmonics"] = {str(k): x for k, x in v["harmonics"].items()}
            print(json.dumps({"pipes": "operations per clock and SM (16 warps/SM, 8 independent chains, clock64)", "rates": rates,
                              "phasor_error": st, "gpu": torch.cuda.get_device_name(0), "sm_max_mhz": peaks.get("sm_max_mhz")}), flush=True)
    elif args.sweep:
        if rank == 0:
            run_sweep(args)
    elif args.impl == "reference":
        run_reference(args, rank)
    else:
        run_cuda(args, rank, local_rank, world)


if __name__ == "__main__":
    main()
