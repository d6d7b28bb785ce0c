#!/usr/bin/env python
"""bench.py — throughput of the TTSH hot path in grid-point-steps/s (BASELINE.json:metric).

One bench "step" = one diagnostics interval of the paper-shaped workload: 100 applications of Algorithm 1
(rows a1-a6 of SURVEY.md §8a) followed by one ttsh_diagnostics call (row a7), on config C5 of BASELINE.json
(4096x4096, dx=0.5, dt=1e-2, fp64, disk R=900, seeded Gaussian 1e-2 start).  `value` counts Nx*Ny*100 grid-point-steps
per bench step, state resident in HBM.  `e2e` is the same job through the C ABI from HOST buffers: every bench
step copies the initial velocity (pinned host memory) to the device, calls ttsh_set_velocity, runs the 100 steps
and reads the diagnostics record back.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload C5|C5-f32|C3|C3-f32|...]

N > 1 (torchrun, one rank per GPU): independent replicas, no collective on the data path ("replicas only", DESIGN.md
§9); value = units all ranks processed / max-over-ranks time.
"""
from __future__ import annotations

import argparse
import json
import math
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

INNER = 100   # Euler steps per bench step (diagnostics cadence of BASELINE.json configs[1])
METRIC = "TTSH grid-point-steps/s"


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="C5")
    ap.add_argument("--inner", type=int, default=100, help="Euler steps per bench step (profiling runs use fewer)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-extra", action="store_true", help="skip the 1024^2 / fp32 side measurements")
    return ap.parse_args()


def workload(name):
    from paper_2304_03306_b200 import workloads
    dtype = "f32" if name.endswith("-f32") else "f64"
    cfg = workloads.CONFIGS[name.replace("-f32", "")]
    return cfg, dtype


PARAM_TEXT = {"baseline": "lambda0=3.5 alpha=-0.5 beta=0.5 Gamma0=-1 Gamma2=1 gamma_v=40 gamma_w=4",
              "paper": "the paper's parameters (PAPER.md:61): lambda0=9 alpha=0.5 beta=1.6 Gamma0=-2 Gamma2=1 gamma_v=40 gamma_w=4"}


def describe(cfg, dtype):
    geom = {"disk": f"disk R={cfg.R:g}", "dumbbell": f"dumbbell R={cfg.R:g} d={cfg.d:g}", "none": "unconfined"}[cfg.geometry]
    return (f"{cfg.name}: {cfg.Ny}x{cfg.Nx} grid, dx={cfg.dx}, dt={cfg.dt}, {dtype}, {geom}, {PARAM_TEXT[cfg.preset]}, "
            f"Gaussian 1e-2 start, seed {cfg.seed}")


def gpu_params(ttsh, cfg):
    return ttsh.paper_params() if cfg.preset == "paper" else ttsh.baseline_params()


def oracle_params(cfg):
    from oracle import BASELINE_PRESET, PAPER_PRESET
    return PAPER_PRESET if cfg.preset == "paper" else BASELINE_PRESET


# --------------------------------------------------------------------------------------------------
# clocks sampling during the timed region
# --------------------------------------------------------------------------------------------------
class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.rows, self.proc, self.thread, self.index = [], None, None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except Exception:
            self.proc = None
            return
        def pump():
            for line in self.proc.stdout:
                self.rows.append(line.strip())
        self.thread = threading.Thread(target=pump, daemon=True)
        self.thread.start()

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons, power = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            parts = [p.strip() for p in r.split(",")]
            if len(parts) < 7:
                continue
            try:
                sm.append(float(parts[0])); mx.append(float(parts[1])); power.append(float(parts[2]))
            except ValueError:
                continue
            for n, v in zip(names, parts[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(power) if power else None, "samples": len(sm), "reasons": sorted(reasons)}


# --------------------------------------------------------------------------------------------------
# the oracle on the host cores (cpu_baseline leg and --impl reference)
# --------------------------------------------------------------------------------------------------
def oracle_threads():
    try:
        from threadpoolctl import threadpool_info
        n = [p.get("num_threads", 1) for p in threadpool_info() if p.get("user_api") == "blas"]
        if n:
            return max(n)
    except Exception:
        pass
    return len(os.sched_getaffinity(0))


def oracle_c(cfg):
    """The oracle-fft restatement of the oracle in plain C (oracle/ttsh_oracle_c.c: full complex spectra, radix-2 FFT, OpenMP over
    lines) at the workload's REAL size, with its mask and start.  The honest CPU baseline: the counterpart of the CPU curve of
    Fig. 9."""
    from oracle.c_oracle import TTSHOracleC
    mask = cfg.mask()
    vx, vy = cfg.initial_velocity(mask)
    o = TTSHOracleC(cfg.Nx, cfg.Ny, cfg.dx, cfg.dt, oracle_params(cfg), mask=mask)
    o.set_velocity(vx, vy)
    return o


def time_oracle_c(cfg, n_steps, warmup=1):
    """(grid-point-steps/s, sample description, seconds per Euler step, threads) of the C oracle-fft on the full grid."""
    from oracle.c_oracle import threads
    o = oracle_c(cfg)
    if warmup:
        o.step(warmup)
    t0 = time.perf_counter()
    o.step(n_steps)
    t_step = (time.perf_counter() - t0) / n_steps
    o.close()
    sample = (f"{n_steps} Euler step(s) of oracle/ttsh_oracle_c.c (Algorithm 1 in plain C, full complex spectra, radix-2 FFT, fp64, "
              f"OpenMP) on the full {cfg.Ny}x{cfg.Nx} grid of the workload")
    return cfg.Nx * cfg.Ny / t_step, sample, t_step, threads()


def time_oracle(cfg, n_steps, budget_s, warmup=0):
    """Times the oracle AS IT STANDS (naive-DFT transforms = explicit DFT-matrix products) on a bounded sample of
    the workload: the same geometry family, parameters and start, on the largest grid <= the workload's whose
    predicted cost fits the budget.  Returns (grid-point-steps/s, sample description, seconds per step)."""
    from oracle import TTSHOracle
    from paper_2304_03306_b200 import workloads
    BASELINE_PRESET = oracle_params(cfg)

    def run(Nx, Ny, steps, wu):
        scale = Nx / cfg.Nx
        if cfg.geometry == "disk":
            mask = workloads.disk_mask(Nx, Ny, cfg.dx, cfg.R * scale)
        elif cfg.geometry == "dumbbell":
            mask = workloads.dumbbell_mask(Nx, Ny, cfg.dx, cfg.R * scale, cfg.d * scale)
        else:
            mask = None
        vx, vy = workloads.gaussian_velocity(Nx, Ny, cfg.seed, 1e-2, mask)
        o = TTSHOracle(Nx, Ny, cfg.dx, cfg.dt, BASELINE_PRESET, mask=mask)
        o.set_velocity(vx, vy)
        if wu:
            o.step(wu)
        t0 = time.perf_counter()
        o.step(steps)
        return (time.perf_counter() - t0) / steps

    # probe at 1/8 of the linear size (cost ~ N^3 per transform), then pick the sample grid
    div = 8 if min(cfg.Nx, cfg.Ny) >= 512 else 1
    t_probe = run(cfg.Nx // div, cfg.Ny // div, 1, 1)
    f = 1
    while f < div and t_probe * ((div // f) ** 3) * (n_steps + warmup + 1.5) > budget_s:
        f *= 2
    Nx, Ny = cfg.Nx // f, cfg.Ny // f
    t_step = t_probe if f == div else run(Nx, Ny, n_steps, warmup)
    sample = (f"{n_steps} Euler step(s) of oracle/ttsh_oracle.py (naive DFT-matrix transforms, fp64) on a {Ny}x{Nx} grid"
              + ("" if f == 1 else f" (the {cfg.Ny}x{cfg.Nx} workload scaled by 1/{f}: same geometry family, parameters, start)"))
    return Nx * Ny / t_step, sample, t_step


# --------------------------------------------------------------------------------------------------
# our arm
# --------------------------------------------------------------------------------------------------
# what ttsh_step launches per Euler step in the default (conservative) form, and the stage ids of ttsh_run_stage
STAGE_NAMES = ["k_inv_col", "k_row_step", "k_fwd_col", "k_spectral_p2"]
STAGE_IDS = [0, 9, 7, 8]


def stage_bytes(Nx, Ny, w, conservative=True):
    """Algorithmic HBM bytes per launch of each kernel of one step: every input read once, every
    output written once, pruned widths Wx = Nx/4+1, Hy = Ny/2+1.  Conservative advection form (the default):
    3 inverse transforms (w, v_x, v_y); literal form: 5 (w, d_x w, d_y w, v_x, v_y)."""
    Wx, Hy = Nx // 4 + 1, Ny // 2 + 1
    real, inter, spec = Nx * Ny * w, Ny * Wx * 2 * w, Hy * Wx * 2 * w
    ninv_col, ninv_row = (3, 3) if conservative else (4, 5)
    nreal_in = 4 if conservative else 6
    return {
        "k_inv_col": 2 * spec + ninv_col * inter,               # w^ and psi^ in
        "k_inv_row": ninv_col * inter + ninv_row * real,
        "k_realspace": nreal_in * real + 3 * real,
        "k_fwd_row": 3 * real + 3 * inter,
        "k_fwd_row_fused": 4 * real + 2 * inter,                 # v_x, v_y, w, K in; A~ = i kx Gy~ + S'~ and B~ = Gx~ out
        "k_row_step": 3 * inter + real + 2 * inter,              # w~, v_x~, psi~ and K in; A~, B~ out (w, v stay on the SM)
        "k_spectral_p2": 3 * spec + 2 * spec,                    # A^, B^, w^ in; w^, psi^ out
        "k_fwd_col": (2 * inter + 2 * spec) if conservative else (3 * inter + 3 * spec),
        "k_spectral": (3 if conservative else 4) * spec + 2 * spec,   # A^, B^ (or F^x, F^y, S^), w^ in; w^, psi^ out
        "k_col_step": 2 * inter + spec + 2 * spec + 3 * inter,   # A~, B~, w^ in; w^, psi^ and the three inverse intermediates out
    }


def row_step_flops(Nx, Ny):
    """Algorithmic flops of one k_row_step launch: per row pair 6 packed complex transforms of length Nx at the
    textbook 5 N log2 N, plus 18 flops per grid point for lines 1-2 of Algorithm 1 (both rows)."""
    import math
    return (Ny // 2) * (6 * 5 * Nx * math.log2(Nx) + 2 * Nx * 18)


def measure(torch, ttsh, cfg, dtype, K, W, device, want_roofline=True, want_e2e=True, sampler=None):
    import numpy as np
    mask = cfg.mask()
    vx0, vy0 = cfg.initial_velocity(mask)
    s = ttsh.Solver(cfg.Nx, cfg.Ny, cfg.dx, cfg.dt, gpu_params(ttsh, cfg), dtype, mask=mask, device=device)
    s.set_velocity(vx0, vy0)
    cx, cy = (cfg.Nx // 2) * cfg.dx, (cfg.Ny // 2) * cfg.dx
    stream = torch.cuda.current_stream(device)

    def bench_step():
        s.step(INNER)
        return s.diagnostics(cx, cy)

    for _ in range(W):
        bench_step()
    torch.cuda.synchronize(device)
    if sampler:
        sampler.start()
    l0 = s.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for _ in range(K):
        d = bench_step()
    e1.record(stream)
    torch.cuda.synchronize(device)
    ms = e0.elapsed_time(e1)
    launches = s.launch_count() - l0
    clocks = sampler.stop() if sampler else None
    out = {"ms_total": ms, "launches": launches, "clocks": clocks, "diag": d}

    if want_roofline:
        reps = 20
        names, ids = STAGE_NAMES, STAGE_IDS
        try:
            s.run_stage(9)
        except Exception:     # grid / dtype without the fused row-step kernel: ttsh_step launches the 5-kernel sequence
            names, ids = ["k_inv_col", "k_inv_row", "k_fwd_row_fused", "k_fwd_col", "k_spectral_p2"], [0, 1, 6, 7, 8]
        if 128 <= cfg.Ny <= 1024 and ids[1] == 9:
            try:                  # grids whose step is k_row_step + k_col_step (col_step.cuh): time those two
                s.run_stage(0); s.run_stage(9); s.run_stage(10)
                names, ids = ["k_row_step", "k_col_step"], [9, 10]
            except Exception:
                pass
        ns = len(ids)
        ev = [[torch.cuda.Event(enable_timing=True) for _ in range(ns + 1)] for _ in range(reps)]
        for r in range(reps):
            for i, st in enumerate(ids):
                ev[r][i].record(stream)
                s.run_stage(st)
            ev[r][ns].record(stream)
        torch.cuda.synchronize(device)
        per = [sum(ev[r][i].elapsed_time(ev[r][i + 1]) for r in range(reps)) / reps for i in range(ns)]
        out["stage_ms"] = dict(zip(names, per))

    if want_e2e:
        w = 8 if dtype == "f64" else 4
        npdt = np.float64 if dtype == "f64" else np.float32
        hvx = torch.from_numpy(vx0.astype(npdt)).pin_memory()
        hvy = torch.from_numpy(vy0.astype(npdt)).pin_memory()
        dvx = torch.empty_like(hvx, device=device)
        dvy = torch.empty_like(hvy, device=device)

        # A user streaming fresh inputs would double-buffer them: the host->device copy of step k+1 runs on a copy stream
        # while the Euler steps of step k run (every step's copy is inside the timed region; only the first cannot hide).
        dbuf = [(dvx, dvy), (torch.empty_like(dvx), torch.empty_like(dvy))]
        copy_stream = torch.cuda.Stream(device)
        ready = [torch.cuda.Event(), torch.cuda.Event()]       # copy into buffer set b has finished
        consumed = [torch.cuda.Event(), torch.cuda.Event()]    # ttsh_set_velocity has read buffer set b

        def enqueue_copy(b):
            copy_stream.wait_event(consumed[b])
            with torch.cuda.stream(copy_stream):
                dbuf[b][0].copy_(hvx, non_blocking=True)
                dbuf[b][1].copy_(hvy, non_blocking=True)
                ready[b].record(copy_stream)

        def e2e_step(k, last):
            b = k & 1
            stream.wait_event(ready[b])
            rc = ttsh.ttsh_set_velocity(s.h, dbuf[b][0].data_ptr(), dbuf[b][1].data_ptr())
            assert rc == 0
            consumed[b].record(stream)
            if not last:
                enqueue_copy(b ^ 1)          # next step's inputs travel while this step computes
            s.step(INNER)
            return s.diagnostics(cx, cy)     # D2H of the diagnostics record + stream sync

        for b in (0, 1):
            consumed[b].record(stream)
        enqueue_copy(0)
        e2e_step(0, True)
        torch.cuda.synchronize(device)
        ke = max(3, K)
        e0.record(stream)
        enqueue_copy(0)
        for k in range(ke):
            e2e_step(k, k == ke - 1)
        e1.record(stream)
        torch.cuda.synchronize(device)
        out["e2e_ms_per_step"] = e0.elapsed_time(e1) / ke
        out["h2d"] = 2 * cfg.Nx * cfg.Ny * w
        out["d2h"] = 8 * 8
    s.close()
    return out


def measure_ensemble(torch, ttsh, name, count, device, nsteps=200):
    """`count` members of one config's R sweep (radii spread over the config's sweep range, one seed each), advanced together."""
    cfg, dtype = workload(name)
    lo, hi = (min(cfg.sweep), max(cfg.sweep)) if cfg.sweep else (0.5 * cfg.R, cfg.R)
    radii = [lo + (hi - lo) * i / max(1, count - 1) for i in range(count)]
    masks = [cfg.mask(R=r) for r in radii]
    ens = ttsh.Ensemble(count, cfg.Nx, cfg.Ny, cfg.dx, cfg.dt, ttsh.baseline_params(), dtype, masks=masks, device=device)
    from paper_2304_03306_b200 import workloads
    for i, m in enumerate(ens.members):
        m.set_velocity(*workloads.gaussian_velocity(cfg.Nx, cfg.Ny, cfg.seed + 1000 * (i + 1), 1e-2, masks[i]))
    stream = torch.cuda.current_stream(device)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ens.step(20)
    torch.cuda.synchronize(device)
    e0.record(stream)
    ens.step(nsteps)
    e1.record(stream)
    torch.cuda.synchronize(device)
    ms = e0.elapsed_time(e1) / nsteps
    bad = sum(m.diagnostics()["nonfinite"] for m in (ens.members[0], ens.members[-1]))
    ens.close()
    return {"value": cfg.Nx * cfg.Ny * count / (ms * 1e-3), "unit": "grid-point-steps/s", "euler_step_ms": ms, "members": count,
            "nonfinite": bad, "workload": f"{count} members of the {name} sweep, disk R = {lo:g}..{hi:g}, {dtype}, one ttsh_ensemble_step"}


def measure_psd(torch, ttsh, name, nfreq, device, hbm_peak, reps=10):
    """One ttsh_psd_accumulate = inverse transform of w^ + the streaming update of nfreq complex accumulators per grid point
    (Eq. 5).  Algorithmic bytes of the update kernel: read w once, read + write nfreq accumulators."""
    cfg, dtype = workload(name)
    mask = cfg.mask()
    s = ttsh.Solver(cfg.Nx, cfg.Ny, cfg.dx, cfg.dt, ttsh.baseline_params(), dtype, mask=mask, device=device)
    s.set_velocity(*cfg.initial_velocity(mask))
    psd = ttsh.TemporalPSD(s, [0.01 * m for m in range(nfreq)])
    stream = torch.cuda.current_stream(device)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    for _ in range(3):
        psd.accumulate()
    torch.cuda.synchronize(device)
    e0.record(stream)
    for _ in range(reps):
        psd.accumulate()
    e1.record(stream)
    torch.cuda.synchronize(device)
    ms = e0.elapsed_time(e1) / reps
    w = 8 if dtype == "f64" else 4
    nbytes = cfg.Nx * cfg.Ny * (w + nfreq * 2 * 2 * w)
    S, n = psd.result()
    psd.close(); s.close()
    return {"ms_per_accumulate": ms, "algorithmic_bytes": nbytes, "GBps_incl_inverse_transform": nbytes / (ms * 1e-3) / 1e9,
            "frac_of_hbm_peak": nbytes / (ms * 1e-3) / 1e9 / hbm_peak, "samples": n, "finite": bool(all(math.isfinite(x) for x in S)),
            "workload": f"{name} {dtype}, {nfreq} frequencies: {nfreq * 2 * w * cfg.Nx * cfg.Ny / 2**20:.0f} MiB of accumulators (> L2)"}


def measure_tangent(torch, ttsh, name, nvec, device, nsteps=100, qr_every=10):
    """Lyapunov-exponent workload: nvec perturbations carried along the trajectory by ttsh_tangent_step,
    re-orthonormalised every qr_every steps.  Reports the cost per step next to the plain ttsh_step."""
    from paper_2304_03306_b200 import workloads
    cfg, dtype = workload(name)
    mask = cfg.mask()
    s = ttsh.Solver(cfg.Nx, cfg.Ny, cfg.dx, cfg.dt, ttsh.baseline_params(), dtype, mask=mask, device=device)
    s.set_velocity(*cfg.initial_velocity(mask))
    tg = ttsh.Tangent(s, nvec)
    for i in range(nvec):
        tg.set(i, *workloads.gaussian_velocity(cfg.Nx, cfg.Ny, cfg.seed + 500 + i, 1.0))
    tg.orthonormalize()
    stream = torch.cuda.current_stream(device)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    tg.step(qr_every); tg.orthonormalize()
    torch.cuda.synchronize(device)
    acc = [0.0] * nvec
    e0.record(stream)
    for _ in range(nsteps // qr_every):
        tg.step(qr_every)
        acc = [a + b for a, b in zip(acc, tg.orthonormalize())]
    e1.record(stream)
    torch.cuda.synchronize(device)
    ms = e0.elapsed_time(e1) / nsteps
    s.step(nsteps)                                   # untimed: the first call captures the plain step's CUDA graph
    torch.cuda.synchronize(device)
    e0.record(stream); s.step(nsteps); e1.record(stream)
    torch.cuda.synchronize(device)
    ms_base = e0.elapsed_time(e1) / nsteps
    rates = [a / (nsteps * cfg.dt) for a in acc]
    tg.close(); s.close()
    return {"ms_per_step_with_qr": ms, "ms_per_plain_step": ms_base, "vectors": nvec, "qr_every": qr_every,
            "growth_rates_over_window": [round(r, 6) for r in rates], "finite": bool(all(math.isfinite(r) for r in rates)),
            "workload": f"{name} {dtype}, {nvec} tangent vectors, QR every {qr_every} steps, {nsteps} steps from the 1e-2 start"}


def measure_fma_peak(torch, ttsh, dtype, device, reps=5):
    """The ALU roof, measured: ttsh_microbench_fma (a dense register-resident FMA loop, csrc/microbench.cu) timed with CUDA events;
    best of `reps` launches of about 10 ms each.  Returns TFLOP/s."""
    props = torch.cuda.get_device_properties(device)
    code = ttsh.TTSH_F64 if dtype == "f64" else ttsh.TTSH_F32
    blocks = props.multi_processor_count * 8                  # 8 CTAs x 256 threads = 64 warps per SM
    rounds = 2000 if dtype == "f64" else 4000
    sink = torch.empty(blocks * 256, dtype=torch.float64 if dtype == "f64" else torch.float32, device=device)
    stream = torch.cuda.current_stream(device)
    best = 0.0
    for i in range(reps + 1):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        rc, flops = ttsh.ttsh_microbench_fma(code, blocks, rounds, 0.999999, 1e-6, sink.data_ptr(), stream.cuda_stream)
        e1.record(stream)
        torch.cuda.synchronize(device)
        if rc != ttsh.TTSH_OK:
            raise RuntimeError("ttsh_microbench_fma failed")
        if i > 0:                                             # the first launch is warm-up
            best = max(best, flops / (e0.elapsed_time(e1) * 1e-3) / 1e12)
    return best


def measure_cufft_reference(torch, cfg, dtype, device, reps=10):
    """north_star: 'cuFFT serves only as a side-by-side reference'.  The transforms of ONE Euler step in the conservative form
    (3 inverse + 3 forward dense 2-D real transforms, the paper's own design) through torch.fft = cuFFT, without
    any of the element-wise work, next to our whole step."""
    tdt = torch.float64 if dtype == "f64" else torch.float32
    x = torch.randn(3, cfg.Ny, cfg.Nx, dtype=tdt, device=device)
    stream = torch.cuda.current_stream(device)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)

    def six():
        X = torch.fft.rfft2(x, norm="ortho")
        return torch.fft.irfft2(X, s=(cfg.Ny, cfg.Nx), norm="ortho")

    six(); six()
    torch.cuda.synchronize(device)
    e0.record(stream)
    for _ in range(reps):
        y = six()
    e1.record(stream)
    torch.cuda.synchronize(device)
    ms = e0.elapsed_time(e1) / reps
    del y
    return {"ms_for_3_rfft2_plus_3_irfft2": ms, "workload": f"dense {cfg.Nx}x{cfg.Ny} {dtype} transforms of one step via torch.fft (cuFFT)"}


def reduce_over_ranks(dist, maxima, sums, device="cpu"):
    """Replicas only: the job time is the MAX over ranks, counts are SUMMED.  No data-path collective."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return list(maxima), list(sums)
    import torch
    t = torch.tensor(list(maxima), device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    c = torch.tensor(list(sums), device=device, dtype=torch.int64)
    dist.all_reduce(c, op=dist.ReduceOp.SUM)
    return [float(x) for x in t], [int(x) for x in c]


def job_throughput(Nx, Ny, inner, steps, world, ms_max):
    """Whole-job grid-point-steps/s of `world` replicas that each ran `steps` bench steps in at most ms_max."""
    return Nx * Ny * inner * world * steps / (ms_max * 1e-3)


def main():
    a = parse()
    global INNER
    INNER = a.inner
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    cfg, dtype = workload(a.workload)
    config = {"workload": describe(cfg, dtype), "bench_step": f"{INNER} Euler steps (Algorithm 1) + 1 diagnostics call",
              "l2": "working set (9 fields, >1 GB at 4096^2 fp64) exceeds the 126 MB L2; no explicit flush",
              "parallelism": "single GPU" if world == 1 else f"{world} independent replicas (no collective)"}

    # ------------------------------------------------------------------ reference arm = the oracle on host cores
    if a.impl == "reference":
        if rank != 0:
            return
        # The oracle-fft (plain C) on the REAL grid of the workload.  One reference "step" is a bounded sample of our bench step:
        # REF_INNER Euler steps instead of 100 (+ the diagnostics call), so that --steps K --warmup W ends within minutes;
        # ms_per_step is the time actually measured per such step, value the grid-point-steps/s it achieved.
        from oracle.c_oracle import threads
        REF_INNER = 2
        o = oracle_c(cfg)
        cx, cy = (cfg.Nx // 2) * cfg.dx, (cfg.Ny // 2) * cfg.dx
        for _ in range(a.warmup):
            o.step(REF_INNER); o.diagnostics(cx, cy)
        t0 = time.perf_counter()
        for _ in range(a.steps):
            o.step(REF_INNER); o.diagnostics(cx, cy)
        t_step = (time.perf_counter() - t0) / max(1, a.steps)
        o.close()
        val = cfg.Nx * cfg.Ny * REF_INNER / t_step
        cores = threads()
        sample = (f"each step = {REF_INNER} Euler steps + 1 diagnostics call of oracle/ttsh_oracle_c.c (plain C oracle-fft, fp64, OpenMP) on the "
                  f"full {cfg.Ny}x{cfg.Nx} grid (our arm's step is 100 Euler steps + 1 diagnostics call on the same grid)")
        config["bench_step"] = f"{REF_INNER} Euler steps (Algorithm 1) + 1 diagnostics call (bounded sample of the 100-step bench step)"
        config["parallelism"] = f"{cores} host threads (OpenMP)"
        config.pop("l2", None)
        line = {"impl": "reference", "metric": METRIC, "value": val, "unit": "grid-point-steps/s", "n_gpus": a.gpus,
                "steps": a.steps, "warmup": a.warmup, "ms_per_step": 1e3 * t_step, "higher_is_better": True,
                "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic", "config": config,
                "cpu_baseline": {"value": val, "unit": "grid-point-steps/s", "cores": cores, "kind": "oracle-fft", "sample": sample},
                "e2e": {"value": val, "unit": "grid-point-steps/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
                "gpu_launches": 0}
        print(json.dumps(line))
        return

    # ------------------------------------------------------------------ our arm
    import torch
    from paper_2304_03306_b200 import ttsh      # raises if libttsh.so is missing: no fallback
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (no CPU fallback)")
    torch.cuda.set_device(local)
    device = torch.device("cuda", local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=device)
    # replicas: each rank runs its own seed
    if world > 1:
        from dataclasses import replace
        cfg = replace(cfg, index=cfg.index + 16 * rank)

    def barrier():
        if dist:
            dist.barrier()
        torch.cuda.synchronize(device)

    sampler = ClockSampler(local) if rank == 0 else None
    barrier()
    res = measure(torch, ttsh, cfg, dtype, a.steps, a.warmup, device, sampler=sampler)
    barrier()
    ms = res["ms_total"]
    e2e_ms = res["e2e_ms_per_step"]
    launches = res["launches"]
    (ms, e2e_ms), (launches,) = reduce_over_ranks(dist, [ms, e2e_ms], [launches], device)
    value = job_throughput(cfg.Nx, cfg.Ny, INNER, a.steps, world, ms)
    e2e_value = job_throughput(cfg.Nx, cfg.Ny, INNER, 1, world, e2e_ms)
    if rank != 0:
        if dist:
            dist.destroy_process_group()
        return

    w = 8 if dtype == "f64" else 4
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        pass
    peak = float(peaks.get("hbm_gbs", 6650.0))
    peak_src = "MEASURED_PEAKS.json hbm_gbs (of measured)" if "hbm_gbs" in peaks else "fallback 6650 GB/s (of fallback)"
    st = res["stage_ms"]
    sb = {k: v for k, v in stage_bytes(cfg.Nx, cfg.Ny, w).items() if k in st}
    dom = max(st, key=st.get)
    step_ms = sum(st.values())
    hbm = {k: {"ms": st[k], "GBps": sb[k] / (st[k] * 1e-3) / 1e9, "frac": sb[k] / (st[k] * 1e-3) / 1e9 / peak, "bytes": sb[k]} for k in st}
    roofline = {"bound": "hbm", "kernel": dom, "achieved": hbm[dom]["GBps"], "peak": peak, "unit": "GB/s", "frac": hbm[dom]["frac"],
                "traffic": None, "peak_source": peak_src, "algorithmic_bytes_per_launch": sb[dom]}
    if dom == "k_row_step":
        # The fused row kernel keeps w, v on the SM: 3.5 U of HBM traffic against 6 packed Nx-point transforms per row pair,
        # so its binding roofline is the plain fp64 / fp32 ALU pipe: peak = SMs x lanes x 2 (FMA) x max clock.
        props = torch.cuda.get_device_properties(device)
        sm_mhz = float(peaks.get("sm_max_mhz", 1965.0))
        lanes = 64 if dtype == "f64" else 128
        derived_peak = props.multi_processor_count * lanes * 2 * sm_mhz * 1e6 / 1e12
        alu_peak = measure_fma_peak(torch, ttsh, dtype, device)       # measured in this run; the derived figure is kept beside it
        flops = row_step_flops(cfg.Nx, cfg.Ny)
        ach = flops / (st[dom] * 1e-3) / 1e12
        roofline = {"bound": "alu", "kernel": dom, "achieved": ach, "peak": alu_peak, "unit": "TFLOP/s", "frac": ach / alu_peak,
                    "traffic": None,
                    "peak_source": f"measured in this run: ttsh_microbench_fma, a dense {dtype} FMA loop in registers on "
                                   f"{props.multi_processor_count} SMs x 64 warps (csrc/microbench.cu), best of 5 launches, CUDA events",
                    "peak_derived": derived_peak,
                    "peak_derived_source": f"{props.multi_processor_count} SMs x {lanes} {dtype} lanes x 2 flop x {sm_mhz:.0f} MHz (DESIGN.md §6)",
                    "flop_count": "textbook 5 N log2 N per complex transform of a packed row pair, unpruned (6 per pair) + 18 flop per "
                                  "point of lines 1-2; counting one radix-2 level less for the 1/2-rule zeros gives about 0.91 of it",
                    "algorithmic_flops_per_launch": flops, "algorithmic_bytes_per_launch": sb[dom],
                    "hbm_GBps": hbm[dom]["GBps"], "hbm_frac": hbm[dom]["frac"], "hbm_peak": peak, "hbm_peak_source": peak_src}
    roofline.update({"kernel_ms": st[dom], "kernel_share_of_step": st[dom] / step_ms, "all_kernels_hbm": hbm,
                     "step_algorithmic_bytes": sum(sb.values()), "step_GBps": sum(sb.values()) / (step_ms * 1e-3) / 1e9,
                     "step_frac_hbm": sum(sb.values()) / (step_ms * 1e-3) / 1e9 / peak})
    # traffic from the committed ncu --set full capture of that kernel, when present (profiles/ncu_traffic.csv)
    try:
        import csv
        with open(os.path.join(ROOT, "profiles", "ncu_traffic.csv")) as fh:
            for row in csv.DictReader(fh):
                if row["kernel"] == dom and row["workload"] == a.workload:
                    roofline["traffic"] = float(row["dram_bytes_per_launch"])     # latest row wins
                    roofline["traffic_source"] = row["source"]
    except Exception:
        pass

    line = {"metric": METRIC, "value": value, "unit": "grid-point-steps/s", "n_gpus": world, "steps": a.steps, "warmup": a.warmup,
            "ms_per_step": ms / a.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": dtype,
            "data": "synthetic", "config": config, "clocks": res["clocks"],
            "e2e": {"value": e2e_value, "unit": "grid-point-steps/s", "h2d_bytes_per_step": res["h2d"],
                    "d2h_bytes_per_step": res["d2h"], "ms_per_step": e2e_ms,
                    "pipeline": "double-buffered inputs: the pinned host->device copy of step k+1 overlaps the Euler steps of step k"},
            "gpu_launches": launches, "roofline": roofline, "euler_step_ms": ms / a.steps / INNER}

    if not a.no_extra and world == 1:
        extra = {}
        # all five BASELINE.json configs as single systems (C1, C2, C4 beside C3 and C5), then the paper's own grids C6, C7
        for name in ("C5-f32", "C1", "C2", "C3", "C3-f32", "C4", "C5p", "C6", "C6-f32", "C7", "C7-f32"):
            if name == a.workload:
                continue
            c2, d2 = workload(name)
            k2 = max(2, a.steps // 2) if c2.Nx * c2.Ny <= 4096 * 4096 else 1
            r2 = measure(torch, ttsh, c2, d2, k2, 3 if k2 > 1 else 1, device, want_roofline=False, want_e2e=False)
            extra[name] = {"value": c2.Nx * c2.Ny * INNER * k2 / (r2["ms_total"] * 1e-3), "unit": "grid-point-steps/s",
                           "euler_step_ms": r2["ms_total"] / k2 / INNER, "workload": describe(c2, d2)}
        # the paper's sweeps (R sweep of C1 / C2 / C3) as ensembles: ttsh_ensemble_step, one launch of each hot
        # kernel per Euler step for all members
        for name, count in (("C1", 256), ("C2", 64), ("C3", 16), ("C3-f32", 16)):
            extra[f"{name} x{count} ensemble"] = measure_ensemble(torch, ttsh, name, count, device)
        extra["C3 temporal PSD, 64 frequencies"] = measure_psd(torch, ttsh, "C3", 64, device, peak)
        extra["C2 Lyapunov, 8 vectors"] = measure_tangent(torch, ttsh, "C2", 8, device)
        extra["cuFFT side-by-side (reference only, never in the product path)"] = measure_cufft_reference(torch, cfg, dtype, device)
        line["other_workloads"] = extra

    if not a.no_cpu_baseline and world == 1:
        # the honest CPU baseline: the oracle-fft (plain C) on the real grid, about 10-20 s of CPU work
        val, sample, t_step, cores = time_oracle_c(cfg, 8, warmup=1)
        line["cpu_baseline"] = {"value": val, "unit": "grid-point-steps/s", "cores": cores, "kind": "oracle", "variant": "oracle-fft",
                                "sample": sample, "seconds_per_euler_step": t_step}
        # aside: the definition-oracle (explicit DFT-matrix products, O(N^3) per transform) on the largest scaled copy that fits 30 s
        val, sample, t_step = time_oracle(cfg, 1, budget_s=30.0)
        line["cpu_baseline_definition_oracle"] = {"value": val, "unit": "grid-point-steps/s", "cores": oracle_threads(), "kind": "oracle",
                                                  "variant": "definition (DFT-matrix products)", "sample": sample,
                                                  "seconds_per_euler_step": t_step}
    print(json.dumps(line))
    if dist:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
