#!/usr/bin/env python
"""bench.py -- the headline measurement of BASELINE.json on one B200 (or N replicas).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]

One STEP = one pass of the whole hot path over one batch of synthetic input: one Navier-Stokes
right-hand-side evaluation psfft_hd_rhs at 512^3 fp64 (spectral curl, 6 inverse + 3 forward 3D
transforms, u x w, 2/3-rule dealias, projection: rows a1-a11 of SURVEY.md §8(a)), input and output
resident in HBM.  `value` = evaluations per second (whole job, all ranks).  The other half of
BASELINE.json's metric -- 512^3 fp64 batch-3 r2c + c2r milliseconds and % of the HBM roofline
(configs[2]) -- is timed in the same run and reported under "fft3d".

Prints ONE JSON line (rank 0).  See DESIGN.md "Measurement" for every field.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "fp64 N^3 r2c+c2r 3D FFT ms & % HBM roofline; HD-RHS evals/sec at 512^3"
UNIT = "evals/s"
FALLBACK_HBM_GBS = 6650.0      # /opt/skills/guides/B200_PROFILING.md fallback when MEASURED_PEAKS.json is absent


# ---- distributed plumbing (nccl on GPUs; gloo in the CPU tests) ----------------------------------------

def dist_env():
    return int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))


def dist_init(backend: str):
    import torch.distributed as dist
    rank, _, world = dist_env()
    if world > 1 and not dist.is_initialized():
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29511")
        dist.init_process_group(backend=backend, rank=rank, world_size=world)
    return rank, world


def dist_barrier():
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized():
        dist.barrier()


def dist_max(x: float, device="cpu") -> float:
    """Max over ranks of a device-measured time (the slowest rank sets the job's time)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return float(x)
    t = torch.tensor([float(x)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate(ms_per_step_max: float, units_per_rank_per_step: float, world: int) -> float:
    """Whole-job throughput: units all ranks processed per second (replicas: weak scaling)."""
    return world * units_per_rank_per_step / (ms_per_step_max * 1e-3)


# ---- clocks ---------------------------------------------------------------------------------------------

class ClockSampler:
    """nvidia-smi sampling DURING the timed region (B200_PROFILING.md clocks line)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
         "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        try:
            self.p = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                       "-lms", "100", "-i", str(index)], stdout=self.f, stderr=subprocess.DEVNULL)
        except OSError:
            self.p = None

    def stop(self) -> dict:
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.p is None:
            return out
        time.sleep(0.15)
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.p.kill()
        self.f.flush()
        self.f.seek(0)
        sm, mx, power, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in self.f:
            t = [s.strip() for s in line.split(",")]
            if len(t) < 9:
                continue
            try:
                sm.append(float(t[1])); mx.append(float(t[2])); power.append(float(t[3]))
            except ValueError:
                continue
            for nm, v in zip(names, t[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        self.f.close()
        os.unlink(self.f.name)
        if sm:
            sm.sort()
            out.update(sm_mhz=sm[len(sm) // 2], sm_max_mhz=max(mx), power_w_max=max(power), samples=len(sm))
        out["reasons"] = sorted(reasons)
        return out


# ---- peaks ---------------------------------------------------------------------------------------------

def hbm_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md 6.65 TB/s)"


def ncu_traffic(kernel: str):
    """dram bytes (read + write) per launch of `kernel` from the committed ncu --set full capture
    (profiles/traffic.csv: kernel,dram_bytes_per_launch,source), or None."""
    p = os.path.join(ROOT, "profiles", "traffic.csv")
    if not os.path.exists(p):
        return None
    try:
        for line in open(p).read().splitlines()[1:]:
            cols = line.split(",")
            if cols and cols[0] == kernel:
                return float(cols[1])
    except Exception:
        return None
    return None


# ---- the oracle as CPU baseline (bench.py is one of the three places allowed to run oracle/) -------------

SAMPLE_N = 256


def work_ratio(N: int, n: int) -> float:
    """N^3 log2 N^3 / n^3 log2 n^3: transform work of the full workload per sample."""
    import math
    return (N ** 3 * 3 * math.log2(N)) / (n ** 3 * 3 * math.log2(n))


def oracle_sample(N: int, n: int, seed: int = 1234):
    """One oracle hd_rhs at n^3 on all host cores; returns (seconds, cores)."""
    import numpy as np
    import oracle
    from paper_1808_01309_b200 import synth
    cores = oracle.set_threads(os.cpu_count() or 1)
    uh = synth.solenoidal_spectrum(n, 4.0, 32, seed)
    t0 = time.perf_counter()
    out = oracle.hd_rhs(uh, 0.0)
    dt = time.perf_counter() - t0
    assert np.isfinite(out).all()
    return dt, cores


def cpu_baseline(N: int) -> dict:
    dt, cores = oracle_sample(N, SAMPLE_N)
    return {"value": 1.0 / (dt * work_ratio(N, SAMPLE_N)), "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": f"one oracle hd_rhs at {SAMPLE_N}^3 (same field recipe) in {dt:.2f} s on {cores} threads, scaled "
                      f"to {N}^3 by the N^3 log2 N^3 work ratio {work_ratio(N, SAMPLE_N):.2f}"}


def run_reference(args) -> int:
    """--impl reference: the oracle, as it stands, on the host cores; each step a bounded sample."""
    rank, _, world = dist_env()
    if rank != 0:
        return 0
    N = args.N
    n = SAMPLE_N
    t_first, cores = oracle_sample(N, n)
    if t_first * (args.steps + args.warmup) > 240.0:
        n = 128
    for _ in range(max(0, args.warmup - 1)):
        oracle_sample(N, n)
    times = [oracle_sample(N, n)[0] for _ in range(args.steps)]
    dt = sum(times) / len(times)
    value = 1.0 / (dt * work_ratio(N, n))
    sample = (f"each step = one oracle hd_rhs at {n}^3 on {cores} threads ({dt:.2f} s), scaled to {N}^3 by the "
              f"N^3 log2 N^3 work ratio {work_ratio(N, n):.2f}")
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt * work_ratio(N, n) * 1e3,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": workload_config(N, world),
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)
    return 0


def workload_config(N: int, world: int) -> dict:
    return {"workload": f"{N}^3 fp64 HD RHS (the metric's evals/s; field of BASELINE.json configs[1] at N={N}: random-phase "
                        f"solenoidal, E(k)~k^4 exp(-2(k/4)^2), unit energy, seed 1234+rank) + configs[2] {N}^3 fp64 batch-3 "
                        "r2c+c2r under 'fft3d'",
            "N": N, "fields": 3, "transforms_per_step": 9,
            "l2": "no flush needed: every pass streams > 1 GiB per field, far above the 126 MB L2",
            "parallelism": "1 GPU" if world == 1 else f"{world} independent replicas (north_star: no multi-GPU path; no collective)"}


# ---- our arm -------------------------------------------------------------------------------------------

def time_loop(fn, steps: int, stream) -> float:
    import torch
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for _ in range(steps):
        fn()
    e1.record(stream)
    e1.synchronize()
    return e0.elapsed_time(e1) / steps


def run_ours(args) -> int:
    import numpy as np
    import torch
    from paper_1808_01309_b200 import build as psbuild
    from paper_1808_01309_b200 import psfft, synth

    rank, local, world = dist_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; libpsfft has no CPU fallback (use --impl reference for the oracle)")
    torch.cuda.set_device(local)
    dist_init("nccl")
    psbuild.build_library()
    N, K, W = args.N, args.steps, max(3, args.warmup)
    dev = torch.device("cuda", local)
    stream = torch.cuda.current_stream()

    # synthetic input (host, pinned) -> device
    kcut = min(32, N // 2 - 1)
    uh_host = torch.from_numpy(synth.solenoidal_spectrum(N, 4.0, kcut, 1234 + rank)).pin_memory()
    rhs_host = torch.empty_like(uh_host).pin_memory()
    plan = psfft.Plan(N, torch.float64, 3, device=dev, work="hd")
    uh = uh_host.to(dev, non_blocking=True)
    rhs = torch.empty_like(uh)
    work = plan.ensure_work("hd")
    h = plan.handle

    def step():
        psfft.hd_rhs(h, uh, rhs, 0.0, work)

    for _ in range(W):
        step()
    torch.cuda.synchronize()
    launches_per_step = psfft.last_launch_count(h)

    # ---- timed region: K steps, device-resident input, per-launch events recorded live ----------------
    psfft.profile_reset(h)
    psfft.profile_enable(h, True)
    clocks = ClockSampler(local)
    dist_barrier()
    torch.cuda.synchronize()
    ms = time_loop(step, K, stream)
    torch.cuda.synchronize()
    dist_barrier()
    psfft.profile_enable(h, False)
    recs = psfft.profile_records(h)
    ms_max = dist_max(ms, dev)
    value = aggregate(ms_max, 1.0, world)

    # ---- roofline of the dominant kernel, from the events of the timed region -------------------------
    tot = {}
    for name, t, b in recs:
        a = tot.setdefault(name, [0.0, 0.0, 0])
        a[0] += t; a[1] += b; a[2] += 1
    dom = max(tot, key=lambda k: tot[k][0])
    peak, peak_src = hbm_peak()
    achieved = tot[dom][1] / (tot[dom][0] * 1e-3) / 1e9
    spec_bytes = plan.layout.spec_bytes
    step_bytes = 42.0 * spec_bytes
    roofline = {"bound": "hbm", "kernel": dom, "achieved": achieved, "peak": peak, "unit": "GB/s",
                "frac": achieved / peak, "traffic": ncu_traffic(dom), "peak_source": peak_src,
                "launches_timed": tot[dom][2], "avg_launch_ms": tot[dom][0] / tot[dom][2],
                "algorithmic_bytes_per_launch": tot[dom][1] / tot[dom][2],
                "kernel_share_of_step": tot[dom][0] / sum(v[0] for v in tot.values()),
                "per_kernel": {k: {"ms_per_step": v[0] / K, "GBps": v[1] / (v[0] * 1e-3) / 1e9, "launches_per_step": v[2] / K}
                               for k, v in tot.items()},
                "step_model": {"algorithmic_bytes": step_bytes, "model": "fused 3-pass HD RHS = 42 C (SURVEY.md §8(a))",
                               "GBps": step_bytes / (ms_max * 1e-3) / 1e9, "frac": step_bytes / (ms_max * 1e-3) / 1e9 / peak}}

    # ---- end to end through the C ABI with HOST buffers (H2D + kernels + D2H per step) ----------------
    d_in, d_out = torch.empty_like(uh), torch.empty_like(uh)

    def step_e2e():
        psfft.hd_rhs_host(h, uh_host, rhs_host, 0.0, d_in, d_out, work)

    step_e2e()
    dist_barrier()
    torch.cuda.synchronize()
    ke = min(K, 10)
    ms_e2e = dist_max(time_loop(step_e2e, ke, stream), dev)
    e2e = {"value": aggregate(ms_e2e, 1.0, world), "unit": UNIT, "h2d_bytes_per_step": 3 * spec_bytes,
           "d2h_bytes_per_step": 3 * spec_bytes, "ms_per_step": ms_e2e, "steps": ke}
    clk = clocks.stop()
    del d_in, d_out

    # ---- the other half of the metric: 512^3 fp64 batch-3 r2c + c2r (configs[2]) ----------------------
    fft3d = None
    if rank == 0 or world > 1:
        x = torch.from_numpy(synth.uniform_field(N, 3, 1234 + rank)).to(dev)
        X = torch.empty(plan.spec_shape(3), dtype=torch.complex128, device=dev)
        y = torch.empty_like(x)
        fwork = plan.ensure_work("fft")
        f_fwd = lambda: psfft.fft3d_r2c(h, x, X, fwork)
        f_bwd = lambda: psfft.fft3d_c2r(h, X, y, fwork)
        for _ in range(3):
            f_fwd(); f_bwd()
        torch.cuda.synchronize()
        t_f = dist_max(time_loop(f_fwd, K, stream), dev)
        t_b = dist_max(time_loop(f_bwd, K, stream), dev)
        rt_err = float((y - x).abs().max())
        # side reference only (north_star: cuFFT "may be timed only as a side reference"; never on the product path)
        cufft = None
        try:
            c_f = lambda: torch.fft.rfftn(x, dim=(1, 2, 3))
            c_b = lambda: torch.fft.irfftn(X, s=(N, N, N), dim=(1, 2, 3))
            for _ in range(2):
                c_f(); c_b()
            torch.cuda.synchronize()
            cufft = {"ms_r2c": time_loop(c_f, min(K, 10), stream), "ms_c2r": time_loop(c_b, min(K, 10), stream),
                     "what": "torch.fft.rfftn / irfftn (cuFFT) on the same tensors, allocation of the result included"}
        except Exception as exc:     # out of memory on a busy device: the side reference is optional
            cufft = {"unavailable": str(exc)[:80]}
        fbytes = 3.0 * (plan.layout.real_bytes + 5.0 * spec_bytes)
        fft3d = {"workload": f"{N}^3 fp64 batch 3, uniform [-1,1) seed 1234 (BASELINE.json configs[2])",
                 "ms_r2c": t_f, "ms_c2r": t_b, "ms_r2c_plus_c2r": t_f + t_b, "ms_per_transform_per_field": (t_f + t_b) / 6.0,
                 "algorithmic_bytes_per_direction": fbytes, "GBps_r2c": fbytes / (t_f * 1e-3) / 1e9,
                 "GBps_c2r": fbytes / (t_b * 1e-3) / 1e9, "hbm_frac": 2 * fbytes / ((t_f + t_b) * 1e-3) / 1e9 / peak,
                 "hbm_frac_of_nominal_8TBps": 2 * fbytes / ((t_f + t_b) * 1e-3) / 1e9 / 8000.0,
                 "roundtrip_max_abs_err": rt_err, "side_reference_cufft": cufft}
        del x, X, y

    # ---- the rows SURVEY.md §8(f) marks "next", same size, same protocol (device-resident) --------------
    next_rows = None
    if world == 1:
        th = torch.from_numpy(synth.scalar_spectrum(N, 4.0, kcut, 1234)).to(dev)
        rt = torch.empty_like(th)
        bwork = plan.ensure_work("rk_boussinesq")
        f_b = lambda: psfft.boussinesq_rhs(h, uh, th, rhs, rt, 1e-3, 1e-3, 1.0, bwork)
        f_rk = lambda: psfft.rk_step(h, psfft.SYS_HD, uh, rhs, 2, 1e-3, (1e-3, 0.0, 0.0), bwork)
        f_g = lambda: psfft.gpe_rhs(h, uh, rhs, 0.3, 1.0, bwork)     # the first two fields as (p^, q^)
        for f in (f_b, f_rk, f_g):
            for _ in range(3):
                f()
        torch.cuda.synchronize()
        t_b = time_loop(f_b, K, stream)
        t_rk = time_loop(f_rk, K, stream)
        t_g = time_loop(f_g, K, stream)
        next_rows = {"boussinesq_rhs": {"ms": t_b, "evals_per_s": 1e3 / t_b,
                                        "workload": f"{N}^3 fp64, u as above + random-phase theta, nu = kappa = 1e-3, N_bv = 1"},
                     "hd_rk2_step": {"ms": t_rk, "steps_per_s": 1e3 / t_rk,
                                     "workload": f"{N}^3 fp64, two fused RHS stages, nu = 1e-3, dt = 1e-3"},
                     "gpe_rhs": {"ms": t_g, "evals_per_s": 1e3 / t_g,
                                 "workload": f"{N}^3 fp64, psi = p + i q as two real fields, alpha = 0.3, beta = 1"}}
        del th, rt

    if rank != 0:
        return 0
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
            "ms_per_step": ms_max, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "config": workload_config(N, world), "clocks": clk, "e2e": e2e,
            "gpu_launches": launches_per_step * K, "launches_per_step": launches_per_step,
            "roofline": roofline, "fft3d": fft3d, "next_rows": next_rows}
    if world == 1 and not args.no_cpu_baseline:
        line["cpu_baseline"] = cpu_baseline(N)
    print(json.dumps(line), flush=True)
    return 0


def main() -> int:
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--N", type=int, default=512, help="grid size (the metric is quoted at 512)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
