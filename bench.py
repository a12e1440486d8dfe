#!/usr/bin/env python
"""bench.py -- the hot path of arXiv 2412.07631 (Eq. 2-3) on B200.

One "step" = one pass of the whole hot path over one batch of synthetic input:
    ct_qr_factor(A_aug)            a1-a4  (Householder QR of the Tikhonov-augmented CT matrix)
  + ct_qr_solve(handle, B, S) -> X a6-a7  (X = R^-1 (Q^T B) for the config's S noisy sinograms)
`value` is BASELINE.json's metric, "QR factor TFLOP/s" (flops = 2mn^2 - 2n^3/3), taken over the
factorisation part of the K timed steps (CUDA events inside the library, inputs resident in
HBM); the solve part of the same steps is reported as `solve.slices_per_s`; `ms_per_step` is
the whole step.  `e2e` is the same metric through the same C-ABI calls with HOST (pinned)
buffers, host<->device copies inside the timed region.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config c4] [--dtype f64|f32]
                    [--impl ours|reference] [--no-also] [--time-budget SECONDS]

The default workload is BASELINE.json configs[3] (m = 109096, n = 65536: 57 GB fp64 in core), the
largest config whose K + W steps fit the driver's window in both precisions; configs[4] (m = 245376,
n = 147456) is one factorisation of 110 s or more, so it is run once, in fp32, out of core from
pinned host memory with a capped device budget, as `extras.out_of_core`.  Every optional leg (second
precision, e2e, extras, CPU baseline) is sized against --time-budget (seconds of wall time for the
whole run, default 1500) and says in its block what it ran.

N > 1 (torchrun): the factorisation does not shard on one node without an exchange step
(DESIGN.md "Multi-GPU"): every rank factors its own replica of A and solves its own S/N share
of the slices; no data-path collective; value = N * flops / max-over-ranks time ("weak").
--impl reference: the CPU oracle (oracle/), as it stands, on the host cores, on a bounded sample.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2412_07631_b200 import workload as wl  # noqa: E402

METRIC = "qr_factor_tflops"
UNIT = "TFLOP/s"


# --------------------------------------------------------------------------------------------
# clocks sampled DURING the timed region (B200_PROFILING.md "clocks line")
# --------------------------------------------------------------------------------------------
class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int = 0):
        self.lines, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                 "-lms", "100"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thr = threading.Thread(target=self._pump, daemon=True)
            self.thr.start()
        except Exception:
            self.proc = None

    def _pump(self):
        for ln in self.proc.stdout:
            self.lines.append(ln.strip())

    def stop(self) -> dict:
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1])); pw.append(float(f[2]))
            except ValueError:
                continue
            for nm, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        return {"sm_mhz": statistics.median(sm), "sm_max_mhz": max(mx), "power_w_max": max(pw),
                "samples": len(sm), "reasons": sorted(reasons)}


class PcieSampler:
    """Host-link throughput from the device's own PCIe counters (NVML nvmlDeviceGetPcieThroughput, a 20 ms hardware
    window per call), sampled from a thread while a leg runs.  ncu's per-kernel pcie__* counters cannot see this traffic:
    the out-of-core copies are copy-engine operations between (under ncu: serialised) kernels, see profiles/r2_ooc.md."""

    def __init__(self, index: int = 0):
        self.index, self.rx, self.tx, self.run, self.thr = index, [], [], False, None

    def start(self):
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv, self.h = pynvml, pynvml.nvmlDeviceGetHandleByIndex(self.index)
            self.run = True
            self.thr = threading.Thread(target=self._loop, daemon=True)
            self.thr.start()
        except Exception:
            self.thr = None

    def _loop(self):
        while self.run:
            try:
                self.rx.append(self.nv.nvmlDeviceGetPcieThroughput(self.h, self.nv.NVML_PCIE_UTIL_RX_BYTES))   # KB/s
                self.tx.append(self.nv.nvmlDeviceGetPcieThroughput(self.h, self.nv.NVML_PCIE_UTIL_TX_BYTES))
            except Exception:
                break

    def stop(self) -> dict:
        if not self.thr:
            return {"unavailable": "pynvml"}
        self.run = False
        self.thr.join(timeout=2)
        if not self.rx:
            return {"unavailable": "no samples"}
        g = lambda v: [x * 1e3 / 1e9 for x in v]
        rx, tx = g(self.rx), g(self.tx)
        return {"source": "NVML PCIe counters, 20 ms windows", "samples": len(rx),
                "rx_gbs_mean": sum(rx) / len(rx), "rx_gbs_peak": max(rx),
                "tx_gbs_mean": sum(tx) / len(tx), "tx_gbs_peak": max(tx)}


def load_peaks() -> dict:
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            d = json.load(f)
        d["_source"] = "measured"
        return d
    return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0, "sm_max_mhz": 1965.0,
            "_source": "fallback"}


# Arithmetic peak of the path's own dtype: B200 has 148 SMs x 64 FP64
# FMA lanes (DFMA and DMMA.8x8x4 share that rate) and 148 x 128 FP32 FMA lanes; x 2 flop x the
# maximum SM clock.  MEASURED_PEAKS.json holds no fp64/fp32 figure, so the bench also runs the
# library's register-resident probe (ct_qr_peak_probe) and reports it beside the nominal one.
def nominal_peak_tflops(dtype: str, sm_max_mhz: float) -> float:
    lanes = 64 if dtype == "f64" else 128
    return 148 * lanes * 2 * sm_max_mhz * 1e6 / 1e12


# --------------------------------------------------------------------------------------------
# inputs (seeded, synthetic; recipe in DESIGN.md "Input recipe")
# --------------------------------------------------------------------------------------------
def build_inputs(cfg, dtype: str, S: int, s_lo: int = 0):
    """A_aug resident in HBM (column-major m x n), B (m x S) as numpy fp64, phantoms X0."""
    import torch
    tdt = torch.float64 if dtype == "f64" else torch.float32
    coo = wl.siddon_coo(cfg.N, cfg.n_ang, cfg.n_bins)
    At, lam = wl.dense_augmented_device(cfg, tdt, coo)
    X0, B = wl.make_slices(cfg, S=s_lo + S, coo=coo, lam=lam)
    return At, X0[:, s_lo:], B[:, s_lo:], coo, lam


def quality(cfg, X0: np.ndarray, X: np.ndarray) -> dict:
    """PAPER.md Eq. 4-7 (L136-154): mean SNR / PSNR / SSIM of the reconstructions against the
    generating phantoms (reported only)."""
    N = cfg.N
    ps, ss, sn = [], [], []
    for s in range(X.shape[1]):
        r, i = X0[:, s].reshape(N, N), X[:, s].astype(np.float64).reshape(N, N)
        ps.append(wl.psnr(r, i)); ss.append(wl.ssim(r, i)); sn.append(wl.snr(r, i))
    return {"psnr_db_mean": float(np.mean(ps)), "ssim_mean": float(np.mean(ss)), "snr_db_mean": float(np.mean(sn)),
            "psnr_db_min": float(np.min(ps)), "slices": int(X.shape[1])}


T_START = time.perf_counter()


class Budget:
    """Wall-time budget of the whole run: optional legs ask before they start."""
    def __init__(self, seconds: float):
        self.seconds = float(seconds)

    def left(self) -> float:
        return self.seconds - (time.perf_counter() - T_START)

    def allows(self, cost_s: float) -> bool:
        return self.left() >= cost_s


def log(msg: str) -> None:
    """Progress line on stderr (stdout carries only the one JSON line)."""
    print("[bench %7.1f s] %s" % (time.perf_counter() - T_START, msg), file=sys.stderr, flush=True)


class PinnedBuffer:
    """Page-locked host tensor that bypasses torch's caching host allocator (which rounds every request up to a
    power of two -- 145 GB would ask for 256 GB -- and never returns blocks to the OS): plain pageable storage
    registered with cudaHostRegister, unregistered and freed by release()."""
    def __init__(self, shape, dtype, zero: bool = False):
        import torch
        self.t = torch.zeros(shape, dtype=dtype) if zero else torch.empty(shape, dtype=dtype)
        self.nbytes = self.t.numel() * self.t.element_size()
        rc = torch.cuda.cudart().cudaHostRegister(self.t.data_ptr(), self.nbytes, 0)
        if int(rc) != 0:
            self.t = None
            raise RuntimeError(f"cudaHostRegister of {self.nbytes} bytes failed: {rc}")

    def release(self):
        import torch
        if self.t is not None:
            torch.cuda.synchronize()
            torch.cuda.cudart().cudaHostUnregister(self.t.data_ptr())
            self.t = None


def pinned_like(t) -> PinnedBuffer:
    """Pinned host copy of a device tensor."""
    import torch
    h = PinnedBuffer(t.shape, t.dtype)
    h.t.copy_(t)
    torch.cuda.synchronize()
    return h


def run_ours(cfg, dtype: str, steps: int, warmup: int, rank: int, world: int, budget: Budget, do_e2e: bool = True,
             structured: bool = False, do_sweep: bool = False, e2e_steps: int = 2) -> dict:
    import torch
    import paper_2412_07631_b200 as ctqr
    dist = torch.distributed if world > 1 else None
    npdt = np.float64 if dtype == "f64" else np.float32
    S_all = cfg.S
    # slices are sharded over ranks (independent right-hand sides, no collective)
    s_lo, S = wl.shard_slices(S_all, rank, world)
    At, X0, B, coo, lam = build_inputs(cfg, dtype, S, s_lo)
    m, n = cfg.m, cfg.n
    w = At.element_size()
    Bt = ctqr.colmajor_from_numpy(B.astype(npdt))
    Xt = torch.zeros((S, n), dtype=At.dtype, device="cuda")
    flops = cfg.factor_flops()
    kl = (m - n) if structured else 0     # --structured: promise the identity block

    Aw = torch.empty_like(At)             # working copy, factored in place: no cudaMalloc / cudaFree of the matrix inside a step

    def one_step(profile: bool, keep: bool = False):
        Aw.copy_(At)                      # (device-to-device, part of the step; ct_qr_factor orders itself after it)
        f = ctqr.ct_qr_factor(Aw, m, n, in_place=True, profile=profile, lower_bandwidth=kl)
        factor_launches = f.stats()["kernel_launches"]      # the solve call restarts the counter
        ctqr.ct_qr_solve(f, Bt, S, Xt)
        st = f.stats()
        st["launches_step"] = factor_launches + st["kernel_launches"]
        if keep:
            return st, f
        f.destroy()
        return st, None

    # the first warm-up step is wall-clocked: if W + K steps of this size cannot fit the share of the
    # time budget given to this precision, K is cut (never below 1) and the line says so
    t0 = time.perf_counter()
    if warmup > 0:
        one_step(False)
    torch.cuda.synchronize()
    t_step = time.perf_counter() - t0
    share = 0.55 * budget.seconds if do_sweep else 0.12 * budget.seconds
    steps_req = steps
    if warmup > 0 and (warmup + steps) * t_step > share:
        steps = int(max(1, min(steps, share / t_step - warmup)))
    for _ in range(max(warmup - 1, 0)):
        one_step(False)
    torch.cuda.synchronize()
    if dist:
        dist.barrier()
    sampler = ClockSampler(torch.cuda.current_device())
    if rank == 0:
        sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    e0.record()
    stats, f_last = [], None
    for i in range(steps):
        st, f_last = one_step(True, keep=(i == steps - 1))
        stats.append(st)
    e1.record()
    flops = stats[0]["factor_flops_performed"] if structured else flops   # TFLOP/s on flops actually performed
    torch.cuda.synchronize()
    if dist:
        dist.barrier()
    clocks = sampler.stop() if rank == 0 else None
    total_ms = e0.elapsed_time(e1)
    factor_ms = sum(s["factor_ms"] for s in stats)
    solve_ms = sum(s["solve_ms"] for s in stats)
    launches = sum(s["launches_step"] for s in stats)
    X = ctqr.numpy_from_colmajor(Xt)
    # the paper's regime (Tables 3, 7, 9: consistent systems, quality limited by the arithmetic only):
    # b_aug = A_aug x for a few phantoms, solved with the factor of the last timed step
    Sc = min(8, S)
    X0c, Bc = wl.make_slices(cfg, S=Sc, coo=coo, lam=lam, consistent=True)
    Bct = ctqr.colmajor_from_numpy(Bc.astype(npdt))
    Xct = torch.zeros((Sc, n), dtype=At.dtype, device="cuda")
    ctqr.ct_qr_solve(f_last, Bct, Sc, Xct)
    Xc = ctqr.numpy_from_colmajor(Xct)
    resid = float(np.linalg.norm(Xc.astype(np.float64) - X0c) / np.linalg.norm(X0c))
    t = torch.tensor([total_ms, factor_ms, solve_ms], dtype=torch.float64, device="cuda")
    if dist:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    total_ms, factor_ms, solve_ms = (float(x) for x in t.tolist())
    out = {
        "value": world * steps * flops / (factor_ms * 1e-3) / 1e12,
        "steps": steps, "steps_requested": steps_req,
        "ms_per_step": total_ms / steps,
        "factor_ms_per_step": factor_ms / steps,
        "solve": {"S": S_all, "ms_per_batch": solve_ms / steps, "slices_per_s": S_all * steps / (solve_ms * 1e-3),
                  "apply_qt_ms": stats[-1]["apply_qt_ms"], "trsm_ms": stats[-1]["trsm_ms"],
                  "tflops": cfg.solve_flops(S_all) * steps / (solve_ms * 1e-3) / 1e12},
        "gpu_launches": int(launches),
        "clocks": clocks,
        "quality_noisy": quality(cfg, X0, X),
        "quality_consistent": dict(quality(cfg, X0c, Xc), rel_error_vs_phantom=resid),
        "nb": stats[-1]["nb"], "ib": stats[-1]["ib"], "flops_per_factor": flops,
    }
    # roofline of the dominant kernel: the two contractions of the trailing update (a3)
    vt = {"ms": sum(s["vtc_ms"] for s in stats), "flops": sum(s["vtc_flops"] for s in stats),
          "launches": sum(s["vtc_launches"] for s in stats)}
    up = {"ms": sum(s["upd_ms"] for s in stats), "flops": sum(s["upd_flops"] for s in stats),
          "launches": sum(s["upd_launches"] for s in stats)}
    out["_spans"] = {"vtc": vt, "upd": up}
    out["_X"] = X
    if dtype == "f32" and rank == 0:
        # fp32 factor + fp64 iterative refinement (Tables 3, 7, 9): fp64-quality solutions
        # from the factor of the last timed step; operator = CSR of A_aug in fp64
        try:
            import scipy.sparse as sp
            rows_, cols_, vals_ = coo
            A0 = sp.coo_matrix((vals_, (rows_, cols_)), shape=(cfg.m0, n)).tocsr()
            Acsr = sp.vstack([A0, np.sqrt(lam) * sp.identity(n, format="csr")]).tocsr()
            Xr = np.zeros((n, Sc), order="F")
            info_c = ctqr.ct_qr_solve_refined(f_last, np.asfortranarray(Bc), Sc, Xr, A_csr=Acsr, max_iters=6, tol=1e-13)
            rr = float(np.linalg.norm(Xr - X0c) / np.linalg.norm(X0c))
            Sn = min(S, 64)
            Xn = np.zeros((n, Sn), order="F")
            info_n = ctqr.ct_qr_solve_refined(f_last, np.asfortranarray(B[:, :Sn]), Sn, Xn, A_csr=Acsr, max_iters=6, tol=1e-12)
            out["refined"] = {
                "consistent": dict(quality(cfg, X0c, Xr), rel_error_vs_phantom=rr, S=Sc, sweeps=info_c["iters_done"],
                                   correction_per_sweep=info_c["correction"], ms_total=info_c["ms_total"]),
                "noisy": {"S": Sn, "sweeps": info_n["iters_done"], "converged": info_n["converged"],
                          "correction_per_sweep": info_n["correction"], "ms_total": info_n["ms_total"],
                          "ms_initial_solve": info_n["ms_initial_solve"], "ms_residual": info_n["ms_residual"],
                          "ms_correction": info_n["ms_correction"], "slices_per_s": Sn / (info_n["ms_total"] * 1e-3)},
                "note": "ct_qr_solve_refined on the fp32 factor of the last timed step, fp64 CSR operator (host arrays staged per call)"}
            out["_Xref"] = Xn
        except Exception as e:
            out["refined"] = {"failed": repr(e)[:300]}
    del Bct, Xct
    if do_sweep and rank == 0 and world == 1:
        out["_extras"] = run_resident_extras(cfg, dtype, f_last, At, Aw, B, budget, factor_ms / steps, structured)
    f_last.destroy()
    if do_e2e and rank == 0:
        per = t_step * 1.15 + 2.0
        k = int(max(0, min(e2e_steps, (budget.left() - 0.35 * budget.seconds) / per - 1))) if do_sweep else \
            int(max(0, min(e2e_steps, (budget.left() - 0.30 * budget.seconds) / per - 1)))
        if k >= 1:
            Ah = pinned_like(At)
            del At, Aw
            torch.cuda.empty_cache()
            try:
                out["e2e"] = run_e2e(cfg, dtype, Ah.t, B.astype(npdt), S, k, flops, kl)
            finally:
                Ah.release()
        else:
            out["e2e"] = None
            out["e2e_skipped"] = "time budget"
    elif do_e2e:
        out["e2e"] = None
    At = Aw = Bt = Xt = None
    torch.cuda.empty_cache()
    return out


def run_e2e(cfg, dtype: str, Ah, B: np.ndarray, S: int, steps: int, flops: float, kl: int = 0) -> dict:
    """Same metric through ct_qr_factor / ct_qr_solve with HOST buffers: every step copies A and
    B host->device and X device->host inside the timed region (the library does the copies)."""
    import torch
    import paper_2412_07631_b200 as ctqr
    m, n = cfg.m, cfg.n
    Bh = torch.from_numpy(np.ascontiguousarray(B.T)).pin_memory()
    Xh = torch.zeros((S, n), dtype=Ah.dtype).pin_memory()
    w = Ah.element_size()

    def step():
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        f = ctqr.ct_qr_factor(Ah, m, n, lower_bandwidth=kl)
        t1 = time.perf_counter()
        ctqr.ct_qr_solve(f, Bh, S, Xh)
        torch.cuda.synchronize()
        t2 = time.perf_counter()
        f.destroy()
        return t1 - t0, t2 - t1

    step()
    ts = [step() for _ in range(max(1, steps))]
    tf = sum(a for a, _ in ts) / len(ts)
    tsol = sum(b for _, b in ts) / len(ts)
    return {"value": flops / tf / 1e12, "unit": UNIT, "h2d_bytes_per_step": int(m * n * w + m * S * w),
            "d2h_bytes_per_step": int(n * S * w), "factor_s": tf, "solve_s": tsol,
            "solve_slices_per_s": S / tsol, "steps": len(ts),
            "factor_s_steps": [round(a, 4) for a, _ in ts], "solve_s_steps": [round(b, 4) for _, b in ts],
            "note": "A, B, X in pinned host memory; wall clock around the synchronous C-ABI calls (one untimed "
                    "warm-up call first); mean over the steps"}


SWEEP_S = (1, 8, 16, 32, 64, 256, 512, 1024, 2048)       # PAPER.md:L89, Fig. 1 (L117-130): up to 2048 simultaneous slices


def run_solve_only(cfg, dtype: str) -> list:
    """One factorisation, then the batched solve at S = 8, 1, 64 on random right-hand sides (timing only).
    factor_read_gbs = the factor's m*n*w bytes / batch time: the algorithmic HBM traffic of the small-S solve."""
    import torch
    import paper_2412_07631_b200 as ctqr
    tdt = torch.float64 if dtype == "f64" else torch.float32
    w = 8 if dtype == "f64" else 4
    At, _ = wl.dense_augmented_device(cfg, tdt)
    f = ctqr.ct_qr_factor(At, cfg.m, cfg.n, in_place=True)
    g = torch.Generator(device="cuda"); g.manual_seed(7)
    out = []
    for S in (8, 1, 64):
        Bt = torch.randn((S, cfg.m), device="cuda", dtype=tdt, generator=g)
        Xt = torch.zeros((S, cfg.n), device="cuda", dtype=tdt)
        ctqr.ct_qr_solve(f, Bt, S, Xt)
        best = None
        for _ in range(3):
            ctqr.ct_qr_solve(f, Bt, S, Xt)
            st = f.stats()
            if best is None or st["solve_ms"] < best["solve_ms"]:
                best = st
        out.append({"S": S, "ms": best["solve_ms"], "apply_qt_ms": best["apply_qt_ms"], "trsm_ms": best["trsm_ms"],
                    "apply_qt_path": best["apply_qt_path"], "launches": best["kernel_launches"],
                    "factor_read_gbs": cfg.m * cfg.n * w / (best["solve_ms"] * 1e-3) / 1e9,
                    "slices_per_s": S / (best["solve_ms"] * 1e-3)})
    f.destroy()
    return out


def run_resident_extras(cfg, dtype: str, f, At, Aw, B: np.ndarray, budget: Budget, incore_ms: float, structured: bool) -> dict:
    """Legs that reuse the resident factor of the last timed step (rank 0, N = 1):
    solve S-sweep (Fig. 1: throughput rises with the number of slices solved at once;
    small S is bound by reading the factor from HBM, m*n*w bytes per batch), then -- after that factor is
    dropped -- the structure-aware factorisation of the same matrix."""
    import torch
    import paper_2412_07631_b200 as ctqr
    tdt = torch.float64 if dtype == "f64" else torch.float32
    npdt = np.float64 if dtype == "f64" else np.float32
    w = 8 if dtype == "f64" else 4
    m, n = cfg.m, cfg.n
    out = {}
    sweep = []
    Smax = max(SWEEP_S)
    reps = -(-Smax // B.shape[1])
    Bt_all = ctqr.colmajor_from_numpy(np.tile(B.astype(npdt), (1, reps))[:, :Smax])   # the batch repeated: timing only
    for S in SWEEP_S:
        Bt = Bt_all[:S]
        Xt = torch.zeros((S, n), dtype=tdt, device="cuda")
        ctqr.ct_qr_solve(f, Bt, S, Xt)
        ms = []
        for _ in range(3):
            ctqr.ct_qr_solve(f, Bt, S, Xt)
            ms.append(f.stats()["solve_ms"])
        t = min(ms)
        st = f.stats()
        sweep.append({"S": S, "ms": t, "slices_per_s": S / (t * 1e-3),
                      "apply_qt_ms": st["apply_qt_ms"], "trsm_ms": st["trsm_ms"],
                      "factor_read_gbs": m * n * w / (t * 1e-3) / 1e9,
                      "tflops": (4.0 * m * n - n * n) * S / (t * 1e-3) / 1e12,
                      "launches": st["kernel_launches"]})
        del Xt
    out["solve_sweep"] = sweep
    del Bt_all
    if structured or not budget.allows(0.45 * budget.seconds + 0.6 * incore_ms * 1e-3):
        return out
    # structure-aware factorisation: the identity block of [A0; sqrt(lambda) I] promised through
    # opt->lower_bandwidth = m0; same factor, fewer flops -- TFLOP/s quoted on the flops actually performed
    m0 = m - n
    Ss = min(cfg.S, 256)
    Bt = ctqr.colmajor_from_numpy(B[:, :Ss].astype(npdt))
    Xd = torch.zeros((Ss, n), dtype=tdt, device="cuda")
    ctqr.ct_qr_solve(f, Bt, Ss, Xd)
    f.destroy()
    ms = []
    fs = None
    for _ in range(3 if incore_ms < 2000 else 1):
        if fs is not None:
            fs.destroy()
        Aw.copy_(At)
        fs = ctqr.ct_qr_factor(Aw, m, n, in_place=True, lower_bandwidth=m0)
        ms.append(fs.stats()["factor_ms"])
    sst = fs.stats()
    Xs = torch.zeros((Ss, n), dtype=tdt, device="cuda")
    ctqr.ct_qr_solve(fs, Bt, Ss, Xs); ctqr.ct_qr_solve(fs, Bt, Ss, Xs)
    solve_ms = fs.stats()["solve_ms"]
    B8 = ctqr.colmajor_from_numpy(B[:, :8].astype(npdt))
    X8 = torch.zeros((8, n), dtype=tdt, device="cuda")
    s8 = []
    for _ in range(4):
        ctqr.ct_qr_solve(fs, B8, 8, X8)
        s8.append(fs.stats()["solve_ms"])
    t = min(ms)
    out["structured"] = {"lower_bandwidth": m0, "factor_ms": t, "vs_dense_time": t / incore_ms, "runs": len(ms),
                         "flops_performed": sst["factor_flops_performed"],
                         "flops_performed_over_dense": sst["factor_flops_performed"] / sst["factor_flops"],
                         "tflops_on_performed_flops": sst["factor_flops_performed"] / (t * 1e-3) / 1e12,
                         "equivalent_dense_tflops": sst["factor_flops"] / (t * 1e-3) / 1e12,
                         "solve": {"S": Ss, "ms": solve_ms, "slices_per_s": Ss / (solve_ms * 1e-3)},
                         "solve_S8": {"ms": min(s8[1:]), "slices_per_s": 8 / (min(s8[1:]) * 1e-3)},
                         "solution_rel_diff_vs_dense_path": float((Xs - Xd).norm() / Xd.norm())}
    fs.destroy()
    return out


def run_persistence() -> dict:
    """Factor persistence (factor once per geometry, reuse): save, reload, first solve.
    Always on BASELINE.json configs[2] in fp64 (a 4.3 GB factor file in the box's temp directory)."""
    import tempfile
    import torch
    import paper_2412_07631_b200 as ctqr
    cfg = wl.CONFIGS["c3"]
    m, n, S = cfg.m, cfg.n, 64
    coo = wl.siddon_coo(cfg.N, cfg.n_ang, cfg.n_bins)
    At, lam = wl.dense_augmented_device(cfg, torch.float64, coo)
    _, B = wl.make_slices(cfg, S=S, coo=coo, lam=lam)
    f = ctqr.ct_qr_factor(At, m, n, in_place=True)
    incore_ms = f.stats()["factor_ms"]
    Bt = ctqr.colmajor_from_numpy(B)
    Xt = torch.zeros((S, n), dtype=torch.float64, device="cuda")
    ctqr.ct_qr_solve(f, Bt, S, Xt)
    with tempfile.TemporaryDirectory() as td:
        path = os.path.join(td, "factor.ctqr")
        t0 = time.perf_counter(); ctqr.ct_qr_save(f, path); t_save = time.perf_counter() - t0
        nbytes = os.path.getsize(path)
        t0 = time.perf_counter(); g = ctqr.ct_qr_load(path); t_load = time.perf_counter() - t0
        X2 = torch.zeros_like(Xt)
        ctqr.ct_qr_solve(g, Bt, S, X2)
        out = {"workload": "configs[2] fp64", "file_bytes": nbytes, "save_s": t_save, "save_gbs": nbytes / t_save / 1e9,
               "load_s": t_load, "load_gbs": nbytes / t_load / 1e9,
               "reloaded_solve_ms": g.stats()["solve_ms"],
               "reloaded_solve_max_abs_diff": float((X2 - Xt).abs().max()),
               "vs_refactor_time": t_load / (incore_ms * 1e-3),
               "note": "file in the box's temp dir; wall clock around ct_qr_save / ct_qr_load"}
        g.destroy()
    f.destroy()
    return out


def run_file_tier(cfg, dtype: str, budget_bytes: int, S: int) -> dict:
    """The paper's storage tier (matrix on disk, host RAM as a block cache over it): the matrix is
    written to a file, its pages are dropped from the page cache (fsync + posix_fadvise DONTNEED), and ct_qr_factor
    runs on the file path with a capped device budget -- the first pass over every super-panel is a cold disk read;
    the factor is left in the file and the solve streams it from there."""
    import tempfile
    import torch
    import paper_2412_07631_b200 as ctqr
    tdt = torch.float64 if dtype == "f64" else torch.float32
    npdt = np.float64 if dtype == "f64" else np.float32
    w = 8 if dtype == "f64" else 4
    m, n = cfg.m, cfg.n
    coo = wl.siddon_coo(cfg.N, cfg.n_ang, cfg.n_bins)
    buf, lam = host_augmented_pinned(cfg, tdt, coo)
    _, B = wl.make_slices(cfg, S=S, coo=coo, lam=lam)
    out = {"workload": workload_name(cfg), "dtype": dtype, "matrix_bytes": m * n * w, "device_budget_bytes": budget_bytes}
    with tempfile.TemporaryDirectory() as td:
        path = os.path.join(td, "A.bin")
        t0 = time.perf_counter()
        with open(path, "wb") as fh:
            buf.t.numpy().tofile(fh)
            fh.flush(); os.fsync(fh.fileno())
        out["file_write_s"] = time.perf_counter() - t0
        out["file_write_gbs"] = m * n * w / out["file_write_s"] / 1e9
        buf.release()
        fd = os.open(path, os.O_RDONLY)
        os.posix_fadvise(fd, 0, 0, os.POSIX_FADV_DONTNEED)       # cold: nothing of the file stays in the page cache
        os.close(fd)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        f = ctqr.ct_qr_factor(None, m, n, dtype=npdt, file_path=path, device_budget_bytes=budget_bytes)
        torch.cuda.synchronize()
        wall = time.perf_counter() - t0
        st = f.stats()
        Bh = torch.from_numpy(np.ascontiguousarray(B.astype(npdt).T)).pin_memory()
        Xh = torch.zeros((S, n), dtype=tdt).pin_memory()
        ctqr.ct_qr_solve(f, Bh, S, Xh)
        st2 = f.stats()
        out.update({
            "n_superpanels": st["n_superpanels"], "factor_ms": st["factor_ms"], "wall_s": wall,
            "tflops": cfg.factor_flops() / (st["factor_ms"] * 1e-3) / 1e12,
            "cold_read_bytes": m * n * w, "h2d_bytes": st["h2d_bytes"], "d2h_bytes": st["d2h_bytes"],
            "file_traffic_gbs_avg": (st["h2d_bytes"] + st["d2h_bytes"]) / (st["factor_ms"] * 1e-3) / 1e9,
            "cold_read_gbs_lower_bound": m * n * w / wall / 1e9,
            "copy_exposed_ms": st.get("copy_exposed_ms"), "copy_busy_ms": st.get("copy_busy_ms"),
            "solve_streamed_from_file": {"S": S, "ms": st2["solve_ms"], "slices_per_s": S / (st2["solve_ms"] * 1e-3),
                                         "gbs": st2["h2d_bytes"] / (st2["solve_ms"] * 1e-3) / 1e9},
            "note": "matrix file in the box's temp directory, page cache dropped before the factorisation; every super-panel is "
                    "first read from disk; later reads of written-back reflector panels may hit the page cache"})
        f.destroy()
    return out


def host_augmented_pinned(cfg, torch_dtype, coo):
    """A_aug of `cfg` built straight in pinned host memory (the matrices of the out-of-core legs do not fit, or
    need not touch, the device): same entries as wl.dense_augmented_device (duplicates summed in fp64, one
    rounding).  Returns (PinnedBuffer whose tensor (n, m) is the column-major m x n matrix, lambda)."""
    import torch
    rows, cols, vals = coo
    lam = wl.tikhonov_lambda(vals, cfg.n)
    buf = PinnedBuffer((cfg.n, cfg.m), torch_dtype, zero=True)
    Ah = buf.t
    flat = Ah.view(-1).numpy()
    key = cols * np.int64(cfg.m) + rows
    uk, inv = np.unique(key, return_inverse=True)
    acc = np.zeros(uk.shape[0], dtype=np.float64)
    np.add.at(acc, inv, vals)
    flat[uk] = acc.astype(flat.dtype)
    d = np.arange(cfg.n, dtype=np.int64)
    flat[d * cfg.m + cfg.m0 + d] = np.asarray(np.sqrt(lam), dtype=np.float64).astype(flat.dtype)
    return buf, lam


def run_out_of_core(cfg, dtype: str, budget_bytes: int, S: int, structured: bool = False) -> dict:
    """a5 under real load: the matrix lives in pinned host memory, the device may use `budget_bytes` for
    matrix tiles, the factor is written back in place and the solve streams it (section 2.2)."""
    import torch
    import paper_2412_07631_b200 as ctqr
    tdt = torch.float64 if dtype == "f64" else torch.float32
    npdt = np.float64 if dtype == "f64" else np.float32
    w = 8 if dtype == "f64" else 4
    m, n = cfg.m, cfg.n
    t0 = time.perf_counter()
    coo = wl.siddon_coo(cfg.N, cfg.n_ang, cfg.n_bins)
    buf, lam = host_augmented_pinned(cfg, tdt, coo)
    Ah = buf.t
    t_build = time.perf_counter() - t0
    log("out-of-core leg: %s %s built in pinned host memory (%.1f GB) in %.1f s" % (cfg.name, dtype, m * n * w / 1e9, t_build))
    _, B = wl.make_slices(cfg, S=S, coo=coo, lam=lam)
    torch.cuda.synchronize()
    pc = PcieSampler(torch.cuda.current_device()); pc.start()
    t0 = time.perf_counter()
    f = ctqr.ct_qr_factor(Ah, m, n, device_budget_bytes=budget_bytes, lower_bandwidth=(m - n) if structured else 0)
    torch.cuda.synchronize()
    wall = time.perf_counter() - t0
    pcie_factor = pc.stop()
    st = f.stats()
    Bh = torch.from_numpy(np.ascontiguousarray(B.astype(npdt).T)).pin_memory()
    Xh = torch.zeros((S, n), dtype=tdt).pin_memory()
    pc = PcieSampler(torch.cuda.current_device()); pc.start()
    ctqr.ct_qr_solve(f, Bh, S, Xh)
    pcie_solve = pc.stop()
    st2 = f.stats()
    # optimality residual of the streamed solve, from the sparse rows in fp64 (no device arithmetic)
    import scipy.sparse as sp
    rows, cols, vals = coo
    A0 = sp.coo_matrix((vals.astype(npdt).astype(np.float64), (rows, cols)), shape=(cfg.m0, n)).tocsr()
    sl = float(np.asarray(np.sqrt(lam), dtype=npdt))
    X = Xh.numpy().T.astype(np.float64)
    Bd = B.astype(npdt).astype(np.float64)
    g = A0.T @ (Bd[:cfg.m0] - A0 @ X) + sl * (Bd[cfg.m0:] - sl * X)
    opt = float(np.linalg.norm(g) / (np.sqrt(np.sum(A0.data ** 2) + n * sl * sl) * np.linalg.norm(Bd)))
    fl = st["factor_flops_performed"] if structured else cfg.factor_flops()
    link = (st["h2d_bytes"] + st["d2h_bytes"]) / (st["factor_ms"] * 1e-3) / 1e9
    out = {
        "workload": workload_name(cfg), "dtype": dtype, "matrix_bytes": m * n * w, "host_build_s": t_build,
        "device_budget_bytes": budget_bytes, "n_superpanels": st["n_superpanels"], "factor_ms": st["factor_ms"],
        "wall_s": wall, "tflops": fl / (st["factor_ms"] * 1e-3) / 1e12, "lower_bandwidth": st["lower_bandwidth"],
        "h2d_bytes": st["h2d_bytes"], "d2h_bytes": st["d2h_bytes"],
        "host_link_gbs_avg": link, "pcie_counters_factor": pcie_factor, "pcie_counters_solve": pcie_solve,
        "algorithmic_link_bytes": m * n * w * (st["n_superpanels"] + 3) / 2.0,
        "copy_exposed_ms": st.get("copy_exposed_ms"), "copy_busy_ms": st.get("copy_busy_ms"),
        "solve_streamed": {"S": S, "ms": st2["solve_ms"], "slices_per_s": S / (st2["solve_ms"] * 1e-3),
                           "h2d_gbs": st2["h2d_bytes"] / (st2["solve_ms"] * 1e-3) / 1e9,
                           "optimality_residual": opt},
        "note": "matrix in pinned host memory, factor written back in place; the link is shared by H2D and D2H streams"}
    f.destroy()
    del Ah
    buf.release()
    return out


# --------------------------------------------------------------------------------------------
# CPU oracle arm (cpu_baseline leg and --impl reference)
# --------------------------------------------------------------------------------------------
def oracle_sample(cfg, dtype: str, k_cols: int, s_cols: int, reps: int = 1) -> dict:
    """Time the oracle, as it stands, on a bounded sample of the same workload: the leading
    k_cols columns of A_aug at full height m (an m x k Householder QR, 2mk^2 - 2k^3/3 flop) and
    its solve of s_cols slices.  Inputs are built on the host; no GPU involved."""
    import oracle
    npdt = np.float64 if dtype == "f64" else np.float32
    coo = wl.siddon_coo(cfg.N, cfg.n_ang, cfg.n_bins)
    rows, cols, vals = coo
    lam = wl.tikhonov_lambda(vals, cfg.n)
    k = min(k_cols, cfg.n)
    A = np.zeros((cfg.m, k), dtype=np.float64, order="F")
    sel = cols < k
    np.add.at(A, (rows[sel], cols[sel]), vals[sel])
    A[cfg.m0 + np.arange(k), np.arange(k)] = np.sqrt(lam)
    A = np.asfortranarray(A.astype(npdt))
    _, B = wl.make_slices(cfg, S=s_cols, coo=coo, lam=lam)
    B = np.asfortranarray(B.astype(npdt))
    fl = 2.0 * cfg.m * k * k - 2.0 * k ** 3 / 3.0
    tq, ts = [], []
    for _ in range(reps):
        t0 = time.perf_counter()
        VR, tau = oracle.qr(A)
        t1 = time.perf_counter()
        oracle.solve(VR, tau, B)
        t2 = time.perf_counter()
        tq.append(t1 - t0); ts.append(t2 - t1)
    tqm, tsm = sum(tq) / reps, sum(ts) / reps
    return {"value": fl / tqm / 1e12, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
            "sample": f"{cfg.name} {dtype}: oracle.qr on the leading {k} of {cfg.n} columns of A_aug at full m={cfg.m} "
                      f"({fl:.3g} flop, {tqm:.2f} s) + oracle.solve of {s_cols} slices on that factor ({tsm:.2f} s)",
            "factor_s": tqm, "solve_s": tsm, "solve_slices_per_s_on_sample": s_cols / tsm,
            "sample_flops": fl}


def sample_size(cfg) -> tuple[int, int]:
    """Leading-column count giving roughly 10-20 s of oracle work at this config's m."""
    target = 4e11                               # flop; the unblocked oracle runs at 15-35 GFLOP/s
    k = int(min(cfg.n, max(64, (target / (2.0 * cfg.m)) ** 0.5)))
    return (k // 64) * 64 if k >= 64 else k, min(cfg.S, 8)


def run_reference(cfg, dtype: str, steps: int, warmup: int) -> dict:
    k, s = sample_size(cfg)
    # K timed steps, each on the bounded sample: the sample shrinks (time ~ k^2) so that the whole run stays within
    # about four minutes of oracle work whatever K is
    if steps > 12:
        k = max(64, int(k * (12.0 / steps) ** 0.5) // 64 * 64)
    for _ in range(min(warmup, 1)):
        oracle_sample(cfg, dtype, max(64, k // 4), 1)
    r = oracle_sample(cfg, dtype, k, s, reps=max(1, steps))
    ms = (r["factor_s"] + r["solve_s"]) * 1e3
    return {"impl": "reference", "metric": METRIC, "value": r["value"], "unit": UNIT, "n_gpus": 0, "steps": steps,
            "warmup": warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": dtype, "data": "synthetic",
            "config": {"workload": workload_name(cfg), "sample": r["sample"]},
            "cpu_baseline": {k2: r[k2] for k2 in ("value", "unit", "cores", "kind", "sample")},
            "e2e": {"value": r["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}


def workload_name(cfg) -> str:
    idx = cfg.cfg_id - 1
    return (f"BASELINE.json configs[{idx}]: {cfg.N}x{cfg.N} image, parallel-beam Siddon, {cfg.n_ang} angles x "
            f"{cfg.n_bins} bins + sqrt(lambda) I rows -> m={cfg.m}, n={cfg.n}; {cfg.S} noisy ellipse-phantom slices, "
            f"I0={cfg.I0:g}")


# per-launch DRAM traffic (dram__bytes_read.sum + dram__bytes_write.sum) of the dominant kernel from the committed
# `ncu --set full` captures under profiles/: the LARGEST launch of that kernel in a factorisation of that config (the
# launches shrink with the trailing matrix); null when no capture of that config / kernel is committed.
#   (config, dtype, kernel) -> (bytes, algorithmic bytes of that launch, profile file)
NCU_TRAFFIC = {("c3", "f64", "upd"): (13.68e9, 8.29e9, "profiles/r1_pairs_c3.md"),
               ("c3", "f64", "vtc"): (3.95e9, None, "profiles/r1_pairs_c3.md"),
               ("c3", "f32", "upd"): (3.57e9, None, "profiles/r1_final_c3.md"),
               ("c3", "f32", "vtc"): (1.91e9, None, "profiles/r1_final_c3.md"),
               ("c4", "f64", "upd"): (124.1e9, 113.4e9, "profiles/r2_c4_f64.md"),
               ("c4", "f64", "vtc"): (90.1e9, 56.8e9, "profiles/r2_c4_f64.md"),
               ("c4", "f32", "upd"): (89.6e9, 56.2e9, "profiles/r2_c4_f32.md")}

KERNEL_NAMES = {("f64", "upd"): "gemm_mma_kernel<double,TA=false,128,64,32,32,3,2> (C <- C - V W, larfb; DMMA.8x8x4)",
                ("f64", "vtc"): "gemm_mma_kernel<double,TA=true,128,64,32,32,3,2> (W = V^T C, larfb; DMMA.8x8x4)",
                ("f32", "upd"): "umma::upd_tma_kernel (C <- C - V W, larfb; 3xTF32 on tcgen05.mma kind::tf32 / TMEM, operands pre-split, TMA-fed)",
                ("f32", "vtc"): "umma::vtc_tma_kernel (W = V^T C, larfb; 3xTF32 on tcgen05.mma kind::tf32 / TMEM, V pre-split and TMA-fed)"}


def roofline(spans: dict, dtype: str, peaks: dict, probe_tflops, cfg) -> dict:
    dom = max(("upd", "vtc"), key=lambda k: spans[k]["ms"])
    oth = "vtc" if dom == "upd" else "upd"
    s, o = spans[dom], spans[oth]
    ach = s["flops"] / (s["ms"] * 1e-3) / 1e12 if s["ms"] > 0 else 0.0
    peak = nominal_peak_tflops(dtype, float(peaks.get("sm_max_mhz", 1965.0)))
    tr = NCU_TRAFFIC.get((cfg.name, dtype, dom))
    # fp64 runs on the FP64 tensor pipe (DMMA), whose peak equals the DFMA peak.  fp32 runs as a 3xTF32
    # split on the tensor cores, but the work it replaces is fp32 FMA work and north_star asks for the
    # fraction of the FP32 peak, so the denominator stays the FFMA peak ("alu"): a fraction above 1
    # would mean the tensor-core path beats what FFMA could ever do.
    return {"bound": "tensor" if dtype == "f64" else "alu", "kernel": KERNEL_NAMES[(dtype, dom)],
            "achieved": ach, "peak": peak, "unit": UNIT, "frac": ach / peak,
            "traffic": tr[0] if tr else None,
            "traffic_note": ("ncu --set full, largest launch of this kernel in this config (%s); algorithmic bytes of that "
                             "launch %s; the launches of a factorisation shrink with the trailing matrix"
                             % (tr[2], "%.3g" % tr[1] if tr[1] else "n/a")) if tr else "no committed capture for this config",
            "peak_source": ("derived: 148 SMs x %d %s FMA lanes x 2 x %.0f MHz max SM clock (MEASURED_PEAKS.json "
                            "holds no %s figure; sm_max_mhz %s)" % (64 if dtype == "f64" else 128,
                                                                   "FP64" if dtype == "f64" else "FP32",
                                                                   float(peaks.get("sm_max_mhz", 1965.0)), dtype,
                                                                   peaks.get("_source"))),
            "peak_probe_tflops": probe_tflops,
            "launches": int(s["launches"]), "avg_launch_ms": s["ms"] / max(1, s["launches"]),
            "flops_per_launch_avg": s["flops"] / max(1, s["launches"]),
            "other_contraction": {"kernel": KERNEL_NAMES[(dtype, oth)],
                                  "achieved": o["flops"] / (o["ms"] * 1e-3) / 1e12 if o["ms"] > 0 else 0.0,
                                  "launches": int(o["launches"]), "ms_total": o["ms"]},
            "share_of_factor_time": None,
            # fp32 only: the same work against the tensor roofline of the 3xTF32 split it actually runs as
            # (measured bf16 peak x nominal tf32/bf16 ratio 1.1/2.25, three MMAs per product)
            "tensor_roofline_3xtf32": (None if dtype == "f64" else {
                "peak": float(peaks.get("bf16_tflops", 1590.0)) * (1.1 / 2.25) / 3.0, "unit": UNIT,
                "frac": ach / (float(peaks.get("bf16_tflops", 1590.0)) * (1.1 / 2.25) / 3.0),
                "peak_source": "MEASURED_PEAKS.json bf16_tflops (%s) x 1.1/2.25 / 3" % peaks.get("_source")})}


def cpu_baseline_block(cfg, dtype: str, budget: Budget) -> dict:
    """BASELINE.md "CPU-baseline plan": the oracle as it stands on the box's host cores.  The headline `value` is a
    bounded sample of the bench workload (leading columns at full height; the whole factorisation at that rate is an
    EXTRAPOLATION by flop count and is labelled so); configs[0] and configs[1] are run in full, configs[0] also on
    one thread."""
    import oracle
    k, s = sample_size(cfg)
    r = oracle_sample(cfg, dtype, k, s)
    out = {k2: v for k2, v in r.items() if k2 in ("value", "unit", "cores", "kind", "sample", "solve_slices_per_s_on_sample")}
    out["whole_factorisation_extrapolated_s"] = cfg.factor_flops() / (r["value"] * 1e12)
    out["extrapolated"] = ("value is measured on the sample; whole_factorisation_extrapolated_s = 2mn^2-2n^3/3 of the "
                           "full config / that rate (extrapolated by flop count, not run)")
    full = {}
    for name in ("c1", "c2"):
        c = wl.CONFIGS[name]
        if not budget.allows(40.0 if name == "c2" else 5.0):
            full[name] = "skipped: time budget"
            continue
        fr = oracle_sample(c, dtype, c.n, c.S)
        full[name] = {"m": c.m, "n": c.n, "S": c.S, "factor_s": fr["factor_s"], "tflops": fr["value"],
                      "solve_s": fr["solve_s"], "solve_slices_per_s": c.S / fr["solve_s"], "cores": fr["cores"]}
        if name == "c1":
            nt = oracle.num_threads()
            oracle.set_num_threads(1)
            f1 = oracle_sample(c, dtype, c.n, c.S)
            oracle.set_num_threads(nt)
            full[name]["one_thread"] = {"factor_s": f1["factor_s"], "tflops": f1["value"], "solve_s": f1["solve_s"]}
    out["full_runs"] = full
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="c4", choices=sorted(wl.CONFIGS))
    ap.add_argument("--dtype", default="f64", choices=["f64", "f32"])
    ap.add_argument("--no-also", action="store_true", help="skip the second precision")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--short-warmup", action="store_true", help="honour --warmup < 3 (profiling runs under ncu only; not a valid bench number)")
    ap.add_argument("--structured", action="store_true",
                    help="promise the identity block of [A0; sqrt(lambda) I] (lower_bandwidth = m0): same factor, "
                         "TFLOP/s on the flops actually performed; not the BASELINE.json headline")
    ap.add_argument("--no-extras", action="store_true", help="skip the solve S-sweep, the structured run, persistence and the out-of-core run")
    ap.add_argument("--time-budget", type=float, default=1500.0,
                    help="wall seconds for the whole run; optional legs are sized against it")
    ap.add_argument("--ooc-config", default="c5", choices=sorted(wl.CONFIGS),
                    help="config of the out-of-core leg (fp32 from pinned host memory, --ooc-budget-gb device bytes)")
    ap.add_argument("--ooc-budget-gb", type=float, default=48.0)
    ap.add_argument("--only-ooc", action="store_true",
                    help="run only the out-of-core leg (--ooc-config, --ooc-dtype, --ooc-budget-gb) and print its block: the "
                         "command the host-link ncu capture of profiles/r2_ooc.md profiles")
    ap.add_argument("--ooc-dtype", default="f32", choices=["f64", "f32"])
    ap.add_argument("--only-solve", action="store_true",
                    help="one factorisation of --config in --dtype, then the solve at S = 8, 1 and 64 (three timed batches each): the "
                         "command the solve captures of profiles/r2_solve.md profile")
    ap.add_argument("--file-tier-config", default="c3", choices=sorted(wl.CONFIGS),
                    help="config of the cold file-tier leg (matrix written to the temp directory, page cache dropped)")
    ap.add_argument("--file-tier-dtype", default="f64", choices=["f64", "f32"])
    ap.add_argument("--file-tier-budget-gb", type=float, default=1.2)
    args = ap.parse_args()
    cfg = wl.CONFIGS[args.config]
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))

    if args.impl == "reference":
        if rank == 0:
            print(json.dumps(run_reference(cfg, args.dtype, args.steps, args.warmup)), flush=True)
        return 0

    import torch
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        torch.distributed.init_process_group("nccl", device_id=torch.device("cuda", local))
    from paper_2412_07631_b200 import build as _build
    if rank == 0:
        _build.build()
    if world > 1:
        torch.distributed.barrier()
    import paper_2412_07631_b200 as ctqr

    if args.only_ooc:
        if rank == 0:
            print(json.dumps({"out_of_core": run_out_of_core(wl.CONFIGS[args.ooc_config], args.ooc_dtype,
                                                              int(args.ooc_budget_gb * 1e9), 8)}), flush=True)
        return 0
    if args.only_solve:
        if rank == 0:
            print(json.dumps({"solve_only": run_solve_only(cfg, args.dtype)}), flush=True)
        return 0
    budget = Budget(args.time_budget)
    warm = args.warmup if args.short_warmup else max(args.warmup, 3)
    extras_on = not args.no_extras and world == 1
    res = run_ours(cfg, args.dtype, args.steps, warm, rank, world, budget, do_e2e=not args.no_e2e,
                   structured=args.structured, do_sweep=True if extras_on else False)
    if rank == 0:
        log("%s %s: %.2f TFLOP/s over %d steps, step %.1f ms" % (cfg.name, args.dtype, res["value"], res["steps"], res["ms_per_step"]))
    if not extras_on:
        res.pop("_extras", None)
    other = "f32" if args.dtype == "f64" else "f64"
    res2 = None
    if not args.no_also:
        # second precision: same step, W >= 3 warm-up steps, K cut to its share of the time budget
        res2 = run_ours(cfg, other, min(args.steps, 5), 3 if not args.short_warmup else warm, rank, world, budget,
                        do_e2e=not args.no_e2e, structured=args.structured, do_sweep=False, e2e_steps=1)
        if rank == 0:
            log("%s %s: %.2f TFLOP/s over %d steps" % (cfg.name, other, res2["value"], res2["steps"]))
    if rank != 0:
        if world > 1:
            torch.distributed.destroy_process_group()
        return 0

    peaks = load_peaks()
    probe = {}
    for kind, name in ((0, "ffma_f32"), (1, "dfma_f64"), (2, "dmma_f64")):
        probe[name] = round(ctqr.ct_qr_peak_probe(kind, 8192)[0], 2)

    def finish(r, dtype):
        rf = roofline(r.pop("_spans"), dtype, peaks, probe["dmma_f64" if dtype == "f64" else "ffma_f32"], cfg)
        rf["share_of_factor_time"] = (rf["launches"] * rf["avg_launch_ms"]) / (r["factor_ms_per_step"] * r["steps"])
        r["roofline"] = rf
        r["frac_of_peak_whole_factor"] = r["value"] / (world * rf["peak"])
        return r

    extras = res.pop("_extras", None)
    res = finish(res, args.dtype)
    w = 8 if args.dtype == "f64" else 4
    line = {"metric": METRIC, "value": res["value"], "unit": UNIT, "n_gpus": world, "steps": res["steps"],
            "warmup": warm, "ms_per_step": res["ms_per_step"], "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": args.dtype, "data": "synthetic",
            "config": {"workload": workload_name(cfg), "m": cfg.m, "n": cfg.n, "S": cfg.S, "nb": res["nb"],
                       "ib": res["ib"], "flops_per_factor": res["flops_per_factor"],
                       "lower_bandwidth": (cfg.m - cfg.n) if args.structured else 0,
                       "l2": "inputs larger than L2 (A is %.2f GB; every step re-reads it from HBM)" % (cfg.m * cfg.n * w / 1e9),
                       "parallelism": "1 GPU" if world == 1 else f"{world} replicas, slices sharded",
                       "steps_requested": args.steps, "time_budget_s": args.time_budget,
                       "steps_note": ("as requested" if res["steps"] == args.steps else
                                      "cut to fit --time-budget (one step is %.1f s)" % (res["ms_per_step"] * 1e-3))},
            "value_definition": ("sum over timed steps of the banded flop count sum_j 4 r_j (n-j-1) actually performed"
                                 if args.structured else "sum over timed steps of 2mn^2-2n^3/3")
                                + " / device time of ct_qr_factor (A resident in HBM)",
            "factor_ms_per_step": res["factor_ms_per_step"], "frac_of_peak_whole_factor": res["frac_of_peak_whole_factor"],
            "solve": res["solve"], "quality_noisy": res["quality_noisy"], "quality_consistent": res["quality_consistent"], "clocks": res["clocks"],
            "e2e": res.get("e2e"), "gpu_launches": res["gpu_launches"], "roofline": res["roofline"],
            "peak_probe_tflops": probe}
    if res.get("e2e_skipped"):
        line["e2e_skipped"] = res["e2e_skipped"]
    if res.get("refined"):
        line["refined"] = res["refined"]
    Xp = res.pop("_X", None); res.pop("_Xref", None)
    if res2 is not None:
        X2 = res2.pop("_X", None); Xref = res2.pop("_Xref", None)
        if other == "f32" and Xref is not None and Xp is not None and "noisy" in res2.get("refined", {}):
            k = Xref.shape[1]
            d64 = Xp[:, :k].astype(np.float64)
            res2["refined"]["noisy"]["rel_diff_vs_fp64_path"] = float(np.linalg.norm(Xref - d64) / np.linalg.norm(d64))
            res2["refined"]["noisy"]["plain_fp32_rel_diff_vs_fp64_path"] = float(
                np.linalg.norm(X2[:, :k].astype(np.float64) - d64) / np.linalg.norm(d64))
        res2 = finish(res2, other)
        line["also"] = {other: {k: res2.get(k) for k in ("value", "steps", "ms_per_step", "factor_ms_per_step",
                                                     "frac_of_peak_whole_factor", "solve", "quality_noisy", "quality_consistent", "refined", "e2e",
                                                     "gpu_launches", "roofline", "clocks")}}
    if extras_on:
        extras = extras or {}
        # the out-of-core leg at configs[4] comes first: it is the one leg no smaller run can stand in for
        oc = wl.CONFIGS[args.ooc_config]
        need_s = 45.0 + oc.factor_flops() / 75e12 * 1.2          # host build + a factorisation at ~75 TFLOP/s fp32 + solve
        if budget.allows(need_s + 30.0):
            torch.cuda.empty_cache()
            try:
                extras["out_of_core"] = run_out_of_core(oc, args.ooc_dtype, int(args.ooc_budget_gb * 1e9), 64)
            except Exception as e:                                # e.g. the box cannot pin that much host memory
                extras["out_of_core"] = {"failed": repr(e)[:300]}
            log("out-of-core leg done")
        else:
            extras["out_of_core"] = {"skipped": "time budget (%.0f s left, %.0f s needed)" % (budget.left(), need_s)}
        if budget.allows(60.0):
            try:
                extras["persistence"] = run_persistence()
            except Exception as e:                                # e.g. no room in the temp directory
                extras["persistence"] = {"skipped": repr(e)[:200]}
        if budget.allows(80.0):
            try:
                extras["file_tier"] = run_file_tier(wl.CONFIGS[args.file_tier_config], args.file_tier_dtype,
                                                    int(args.file_tier_budget_gb * 1e9), 8)
            except Exception as e:
                extras["file_tier"] = {"failed": repr(e)[:300]}
            log("file-tier leg done")
        line["extras"] = extras
    if not args.no_cpu_baseline and world == 1:
        line["cpu_baseline"] = cpu_baseline_block(cfg, args.dtype, budget)
    line["wall_s_total"] = time.perf_counter() - T_START
    print(json.dumps(line), flush=True)
    if world > 1:
        torch.distributed.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
