#!/usr/bin/env python
"""bench.py — whole-step throughput of the B200 pseudo-spectral MHD step (BASELINE.json metric:
fp64 MHD timestep wall time and grid-point updates/s at 512^3; HBM GB/s vs peak).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--n 512]

One "step" = one AB2 time step = one pass of the whole hot path over the
config-4 state (512^3 decaying MHD turbulence, seeded synthetic).  Multi-GPU: the path does not
shard (every 3-D FFT couples the whole box) => "replicas only": N independent runs, no collective
on the data path; value = all ranks' grid-point updates / max-over-ranks device time.

`--impl reference` times the CPU oracle (oracle/, as it stands) on the host cores on a bounded
sample of the same workload; it is a deliberately slow checker, not a competitor.
Prints ONE JSON line on rank 0.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "grid_point_updates_per_s"
UNIT = "grid-point updates/s"
FALLBACK_HBM_GBS = 6650.0      # /opt/skills/guides/B200_PROFILING.md fallback
NOMINAL_HBM_GBS = 8000.0       # figure named by BASELINE.json's north_star


# ------------------------------------------------------------------------------------------------
# host-side helpers (unit-tested on CPU in tests/test_bench_host.py)
# ------------------------------------------------------------------------------------------------
def measured_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md 6.65 TB/s)"


def geometry(nx, ny, nz, dealias=True):
    """stored-mode counts of the 2/3-rule-pruned layout (mirrors csrc/mhd_api.cu make_geometry)."""
    if dealias:
        nkx, nky, nkz = (nx - 1) // 3 + 1, 2 * ((ny - 1) // 3) + 1, 2 * ((nz - 1) // 3) + 1
    else:
        nkx, nky, nkz = nx // 2 + 1, ny, nz
    return dict(nx=nx, ny=ny, nz=nz, nkx=nkx, nky=nky, nkz=nkz)


def algorithmic_bytes(g, hydro=False):
    """Compulsory HBM bytes per launch of each kernel class: unpadded input read once + output
    written once.  Complex = 16 B, real = 8 B."""
    nin, nout = (4, 9) if hydro else (7, 12)
    c = 16
    spec = g["nkz"] * g["nky"] * g["nkx"] * c            # compact spectral field
    w1 = g["nz"] * g["nky"] * g["nkx"] * c               # after z inverse / before z forward
    w2 = g["nz"] * g["ny"] * g["nkx"] * c                # after y inverse / before y forward
    real = g["nz"] * g["ny"] * g["nx"] * 8
    b = {}
    if g["nz"] > 1:
        b["fft_z_inv"] = nin * (spec + w1)
        b["fft_z_fwd"] = nout * (w1 + spec)
    b["fft_y_inv"] = nin * ((w1 if g["nz"] > 1 else spec) + w2)
    b["fft_y_fwd"] = nout * (w2 + (w1 if g["nz"] > 1 else spec))
    b["fft_x_c2r"] = nin * (w2 + real)
    b["fft_x_r2c"] = nout * (real + w2)
    b["products"] = (nin + nout) * real
    b["x_fused"] = (nin + nout) * w2                     # C2R-x + products + R2C-x in one kernel: rows in, rows out
    b["stage"] = (nout + 2 * nin + 2 * nin) * spec       # read flux + state + history, write state + history
    return b


def survey_reference_bytes(nx, ny, nz):
    """SURVEY.md §8(d) fixed numerator: 111 F with F = one full (unpruned) half-spectrum field."""
    return 111 * 16 * (nx // 2 + 1) * ny * nz


def parse_clock_samples(text):
    """nvidia-smi csv,noheader,nounits rows: index, sm, sm_max, power, active-reasons bitmask, hw_slowdown,
    hw_thermal, sw_thermal, sw_power_cap."""
    sm, smmax, reasons = [], [], set()
    for line in text.strip().splitlines():
        parts = [p.strip() for p in line.split(",")]
        if len(parts) < 9:
            continue
        try:
            sm.append(float(parts[1])); smmax.append(float(parts[2]))
        except ValueError:
            continue
        for name, val in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), parts[5:9]):
            if val.lower().startswith("active"):
                reasons.add(name)
    if not sm:
        return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
    top = max(sm)
    loaded = [s for s in sm if s >= 0.5 * top] or sm
    return {"sm_mhz": statistics.median(loaded), "sm_max_mhz": max(smmax), "reasons": sorted(reasons), "samples": len(sm)}


class ClockSampler:
    FIELDS = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index):
        self.p = None
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(gpu_index), f"--query-gpu={self.FIELDS}",
                                       "--format=csv,noheader,nounits", "-lms", "100"],
                                      stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except Exception:
            self.p = None

    def stop(self):
        if self.p is None:
            return parse_clock_samples("")
        self.p.terminate()
        try:
            out, _ = self.p.communicate(timeout=5)
        except Exception:
            self.p.kill()
            out = ""
        return parse_clock_samples(out or "")


def dist_setup(n_gpus, use_cuda):
    """one process per GPU under torchrun; returns (rank, world, local_rank, dist or None)."""
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world <= 1:
        return 0, 1, 0, None
    import torch.distributed as dist
    os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
    dist.init_process_group(backend="nccl" if use_cuda else "gloo", rank=rank, world_size=world)
    return rank, world, local, dist


def max_over_ranks(value, dist, device):
    if dist is None:
        return value
    import torch
    t = torch.tensor([value], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def time_oracle(n, steps, warmup, threads=None):
    """The CPU oracle, as it stands, on a config-4-recipe state of size n^3: seconds per step."""
    from oracle import mhd_ref
    from paper_2402_05478_b200 import inputs
    if threads:
        mhd_ref.set_threads(threads)
    cfg = inputs.config4(n, steps)
    s = mhd_ref.RefSolver(n, n, n, cfg.nu, cfg.eta, cfg.cs, cfg.dt)
    s.set_fields(*cfg.arrays())
    if warmup:
        s.step(warmup)
    t0 = time.perf_counter()
    s.step(steps)
    dt = time.perf_counter() - t0
    cores = mhd_ref.get_threads()
    s.close()
    return dt / steps, cores


# ------------------------------------------------------------------------------------------------
def run_reference(args):
    """--impl reference: the oracle on the host cores (rank 0 only; other ranks exit 0 without work)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return 0
    n = args.ref_n
    sec, cores = time_oracle(n, args.steps, args.warmup)
    value = n ** 3 / sec
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": sec * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"config4 recipe (decaying MHD turbulence, AB2, 2/3 dealiasing) on a bounded {n}^3 sample of the 512^3 box",
                   "grid": [n, n, n], "integrator": "AB2"},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle",
                         "sample": f"{args.steps} AB2 steps at {n}^3 after {args.warmup} warm-up steps"},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)
    return 0


def run_gpu(args):
    import numpy as np
    import torch
    from paper_2402_05478_b200 import inputs, mhd

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device and no CPU fallback (use --impl reference for the oracle)")
    rank, world, local, dist = dist_setup(args.gpus, True)
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    n, K, W = args.n, args.steps, max(args.warmup, 0)
    cfg = inputs.config4(n, K)
    npts = n ** 3
    geo = geometry(n, n, n)
    peak, peak_src = measured_peak()

    host = [torch.from_numpy(a).pin_memory() for a in cfg.arrays()]
    s = mhd.Solver(n, n, n, cfg.nu, cfg.eta, cfg.cs, cfg.dt, device=dev)
    s.set_fields_host(*host)
    s.step(W)                                       # warm-up (includes the Euler first step)
    s.synchronize()

    # ---- timed region: K steps, state resident in HBM (7 fields x 2.3 GB >> 126 MB L2) ----
    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize()
    sampler = ClockSampler(local) if rank == 0 else None
    l0 = mhd.launch_count()
    s.profile_begin()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(s.stream)
    s.step(K)
    e1.record(s.stream)
    torch.cuda.synchronize()
    if dist is not None:
        dist.barrier()
    prof = s.profile_end()
    launches = mhd.launch_count() - l0
    clocks = sampler.stop() if sampler else None
    ms_total = max_over_ranks(e0.elapsed_time(e1), dist, dev)
    ms_step = ms_total / K
    value = world * npts * K / (ms_total * 1e-3)

    # ---- end to end through the C ABI with HOST buffers: H2D of the 7 fields, K steps, diagnostics, D2H ----
    s2 = s
    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    s2.set_fields_host(*host)
    s2.step(K)
    d = s2.diagnostics(0)
    s2.get_fields_host(host)
    torch.cuda.synchronize()
    e2e_s = max_over_ranks(time.perf_counter() - t0, dist, dev)
    nfield_bytes = 7 * 8 * npts
    e2e = {"value": world * npts * K / e2e_s, "unit": UNIT, "h2d_bytes_per_step": nfield_bytes / K,
           "d2h_bytes_per_step": (nfield_bytes + 128) / K,
           "what": f"mhd_set_fields_host (7 pinned fields) + mhd_step({K}) + mhd_diagnostics + mhd_get_fields_host, wall clock"}

    if rank != 0:
        return 0

    # ---- roofline of the dominant kernel, timed live with CUDA events inside the timed region ----
    abytes = algorithmic_bytes(geo)
    traffic = load_traffic()
    kernels = []
    for name, (count, ms) in prof.items():
        if count == 0 or name not in abytes:
            continue
        per = ms / count
        kernels.append({"kernel": name, "launches_per_step": count / K, "ms_per_launch": per,
                        "algorithmic_gb": abytes[name] / 1e9, "gbs": abytes[name] / 1e9 / (per * 1e-3),
                        "frac": abytes[name] / 1e9 / (per * 1e-3) / peak, "share_of_step": ms / ms_total,
                        "traffic": traffic.get(name)})
    kernels.sort(key=lambda k: -k["share_of_step"])
    top = kernels[0]
    roofline = {"bound": "hbm", "kernel": top["kernel"], "achieved": top["gbs"], "peak": peak, "unit": "GB/s",
                "frac": top["frac"], "traffic": top["traffic"], "peak_source": peak_src,
                "algorithmic_bytes_per_launch": abytes[top["kernel"]]}
    if top["kernel"] == "x_fused":
        # the whole path is HBM-bound by design and is reported against the HBM roofline; this one kernel is not:
        roofline["note"] = ("x_fused keeps 7 fields x 8 points per thread in registers (12 warps/SM) and is limited by the FP64 pipe "
                            "(53 % active) and shared-memory wavefronts (66 %), not by HBM: profiles/r01b_summary.md")
    own_bytes = sum(k["algorithmic_gb"] * 1e9 * k["launches_per_step"] for k in kernels)   # only the kernel classes that ran
    step_roofline = {
        "design_bytes_per_step": own_bytes, "design_gbs": own_bytes / 1e9 / (ms_step * 1e-3),
        "design_frac_of_measured_peak": own_bytes / 1e9 / (ms_step * 1e-3) / peak,
        "survey_111F_bytes": survey_reference_bytes(n, n, n),
        "survey_111F_frac_of_measured_peak": survey_reference_bytes(n, n, n) / 1e9 / peak / (ms_step * 1e-3),
        "survey_111F_frac_of_8TBs": survey_reference_bytes(n, n, n) / 1e9 / NOMINAL_HBM_GBS / (ms_step * 1e-3),
    }

    # ---- the oracle timed beside it on this box's host cores (bounded sample) ----
    cpu = None
    if not args.no_cpu_baseline:
        sec, cores = time_oracle(args.cpu_n, args.cpu_steps, 1)
        cpu = {"value": args.cpu_n ** 3 / sec, "unit": UNIT, "cores": cores, "kind": "oracle",
               "sample": f"{args.cpu_steps} AB2 steps (after 1 Euler warm-up step) of the config-4 recipe at {args.cpu_n}^3, {sec:.2f} s per step"}

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W, "ms_per_step": ms_step,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"config4: 3D MHD decaying turbulence {n}^3, AB2, 2/3 dealiasing, nu=eta=1e-3, dt=2e-4, cs=1",
                   "grid": [n, n, n], "integrator": "AB2", "multi_gpu": "replicas only (no data-path collective)",
                   "l2": "inputs larger than L2 (spectral state 2.2 GB + 18 GB of transients per step vs 126 MB L2)",
                   "ekin_after_run": d["ekin"], "emag_after_run": d["emag"]},
        "clocks": clocks, "e2e": e2e, "gpu_launches": launches,
        "roofline": roofline, "step_roofline": step_roofline, "kernels": kernels, "cpu_baseline": cpu,
    }
    print(json.dumps(line), flush=True)
    return 0


def run_fft_sweep(args):
    """--workload fft: BASELINE config 5, batched 3-D R2C + C2R of 7 fields; effective GB/s = 2 F batch / t
    (input read once + output written once) against the measured copy peak, round-trip error, and cuFFT
    (torch.fft, never on the product path) as the one permitted reference line."""
    import torch
    from paper_2402_05478_b200 import mhd
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device")
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(dev)
    peak, peak_src = measured_peak()
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)       # > 126 MB L2
    sweep, l0 = [], mhd.launch_count()
    for n in [int(v) for v in args.fft_sizes.split(",")]:
        batch = 7
        gen = torch.Generator(device=dev); gen.manual_seed(1005)
        a = torch.rand((batch, n, n, n), dtype=torch.float64, device=dev, generator=gen) * 2.0 - 1.0
        plan = mhd.FftPlan(n, n, n, batch, stream=torch.cuda.current_stream(dev))
        spec = plan.r2c(a)
        back = plan.c2r(spec)
        err = float(torch.linalg.norm(back - a) / torch.linalg.norm(a))

        def timed(fn, reps=5):
            ts = []
            for it in range(3 + reps):
                flush.zero_()
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(); fn(); e1.record(); torch.cuda.synchronize()
                if it >= 3:
                    ts.append(e0.elapsed_time(e1))
            return statistics.median(ts)
        t_r2c = timed(lambda: plan.r2c(a, out=spec))
        t_c2r = timed(lambda: plan.c2r(spec, out=back))
        fr, fc = 8.0 * n ** 3 * batch, 16.0 * (n // 2 + 1) * n * n * batch
        row = {"n": n, "batch": batch, "r2c_ms": t_r2c, "c2r_ms": t_c2r, "roundtrip_rel_err": err,
               "r2c_eff_gbs": (fr + fc) / 1e9 / (t_r2c * 1e-3), "c2r_eff_gbs": (fr + fc) / 1e9 / (t_c2r * 1e-3)}
        row["r2c_frac"] = row["r2c_eff_gbs"] / peak
        row["c2r_frac"] = row["c2r_eff_gbs"] / peak
        del plan, back
        try:   # reference line only: cuFFT through torch.fft
            t_ref = timed(lambda: torch.fft.rfftn(a, dim=(1, 2, 3)), reps=3)
            row["cufft_r2c_ms"] = t_ref
        except Exception as ex:   # out of memory at the largest size is not an error of this library
            row["cufft_r2c_ms"] = None
            row["cufft_note"] = type(ex).__name__
        del a, spec
        torch.cuda.empty_cache()
        sweep.append(row)
    line = {"metric": "fft_effective_gbs", "unit": "GB/s", "n_gpus": 1, "higher_is_better": True, "dtype": "f64", "data": "synthetic",
            "config": {"workload": "config5: batched 3-D R2C + C2R, batch 7, uniform[-1,1) reals", "l2": "256 MB flush between iterations"},
            "peak": peak, "peak_source": peak_src, "sweep": sweep, "gpu_launches": mhd.launch_count() - l0,
            "value": max(r["r2c_eff_gbs"] for r in sweep)}
    print(json.dumps(line), flush=True)
    return 0


def load_traffic():
    """per-launch DRAM bytes (dram__bytes_read.sum + dram__bytes_write.sum) per kernel class from the committed
    ncu summary profiles/traffic.csv (kernel,bytes_per_launch); empty if absent."""
    out = {}
    p = os.path.join(ROOT, "profiles", "traffic.csv")
    if os.path.exists(p):
        for line in open(p):
            parts = line.strip().split(",")
            if len(parts) >= 2 and parts[0] != "kernel":
                try:
                    out[parts[0]] = float(parts[1])
                except ValueError:
                    pass
    return out


def main(argv=None):
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--n", type=int, default=512, help="grid size of the timed workload (config 4 is 512)")
    ap.add_argument("--ref-n", type=int, default=128, help="grid size of the bounded sample the reference arm times")
    ap.add_argument("--cpu-n", type=int, default=256, help="grid size of the bounded cpu_baseline sample")
    ap.add_argument("--cpu-steps", type=int, default=4, help="timed oracle steps of the cpu_baseline sample (about 10-20 s of CPU work)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--workload", default="step", choices=["step", "fft"], help="step: the 512^3 MHD step (default); fft: the config-5 FFT sweep")
    ap.add_argument("--fft-sizes", default="128,256,512,768")
    args = ap.parse_args(argv)
    if args.steps < 1:
        raise SystemExit("--steps must be >= 1")
    if args.impl == "reference":
        return run_reference(args)
    return run_fft_sweep(args) if args.workload == "fft" else run_gpu(args)


if __name__ == "__main__":
    sys.exit(main())
