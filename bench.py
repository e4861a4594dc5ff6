#!/usr/bin/env python
"""bench.py — whole-step throughput of the B200 pseudo-spectral MHD step (BASELINE.json metric:
fp64 MHD timestep wall time and grid-point updates/s at 512^3; HBM GB/s vs peak).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--n 512]
    python bench.py --config 1|2|3        # BASELINE configs 1-3 at full length (CUDA-graph replay), oracle timed beside
    python bench.py --workload fft        # BASELINE config 5 (FFT sweep) alone
    python bench.py --workload peaks      # measured FP64 / shared-memory ceilings alone

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


# radices of the fused x pass per length, in execution order: the Plan<N> table of csrc/fft_core.cuh (8 points per thread)
XFUSED_RADICES = {8: (8,), 16: (8, 2), 32: (8, 4), 64: (8, 8), 128: (8, 4, 4), 256: (8, 8, 4), 512: (8, 8, 8),
                  1024: (8, 8, 4, 4)}
BUTTERFLY_FP64 = {8: 56, 4: 16, 2: 4}        # FP64 instructions of one radix-r butterfly (fft_core.cuh bfly8 / bfly4 / bfly2)


def xfused_onchip_model(g, hydro=False):
    """On-chip work of one x_fused launch that no implementation of this design can avoid:
    per (z,y) row 4 inverse + 6 forward complex transforms of length nx (two real rows share one); every pass of radix r is
    nx/r butterflies (56 / 16 / 4 FP64 instructions for r = 8 / 4 / 2) and, on every pass but the first, r-1 twiddle
    multiplications of 4 instructions per butterfly; ~35 FP64 instructions per grid point for the products; between passes
    every complex (16 B) is written to and read from shared memory once.  The radices are the kernel's own plan table
    (XFUSED_RADICES), so 128 = 8*4*4 counts 3 passes and 1024 = 8*8*4*4 counts 4.
    Returns (FP64 instruction slots, shared-memory bytes) per launch; raises for a length the fused pass does not take."""
    nx = g["nx"]
    if nx not in XFUSED_RADICES:
        raise ValueError(f"the fused x pass has no plan for nx = {nx}")
    radices = XFUSED_RADICES[nx]
    rows = g["ny"] * g["nz"]
    nfft = (2 + 5) if hydro else (4 + 6)
    passes = len(radices)
    dp_fft = 0
    for s_, r in enumerate(radices):
        dp_fft += (nx // r) * (BUTTERFLY_FP64[r] + (4 * (r - 1) if s_ > 0 else 0))
    dp = rows * (nfft * dp_fft + 35 * nx)
    smem = rows * (nfft * (passes - 1) * 2 * 16 * nx          # exchanges: store + load of every complex
                   + (4 if hydro else 7) * 16 * g["nkx"]      # staged input rows read once
                   + (5 if hydro else 6) * 2 * 16 * g["nkx"])  # Hermitian split: Z[N-k] published and read
    return dp, smem


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


def host_ram_available_gb():
    try:
        for line in open("/proc/meminfo"):
            if line.startswith("MemAvailable:"):
                return int(line.split()[1]) / 2 ** 20
    except (OSError, ValueError):
        pass
    return 0.0


ORACLE_512_GB = 80.0     # the oracle's arrays at 512^3 (about 57 GB) + the input fields, with headroom


def oracle_sample_grid(requested, total_steps, budget_s=240.0):
    """Grid of the bounded oracle sample.  BASELINE.md §4 asks for the metric's own grid (512^3): taken when the host has the
    memory and `total_steps` oracle steps fit the time budget (about 17 s per step at 512^3 and 2.1 s at 256^3 on the
    16 host cores of a B200 box); otherwise 256^3, then 128^3.  Returns (n, reason)."""
    if requested:
        return int(requested), "grid requested on the command line"
    avail = host_ram_available_gb()
    if avail >= ORACLE_512_GB and total_steps * 17.0 <= budget_s:
        return 512, "the metric's own grid"
    why = (f"only {avail:.0f} GB of host memory available (512^3 needs about {ORACLE_512_GB:.0f})" if avail < ORACLE_512_GB
           else f"{total_steps} oracle steps at 512^3 would take about {total_steps * 17.0:.0f} s")
    if total_steps * 2.1 <= budget_s:
        return 256, why
    return 128, why


# ------------------------------------------------------------------------------------------------
def run_reference(args):
    """--impl reference: the oracle on the host cores (rank 0 only; other ranks exit 0 without work)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return 0
    n, why = oracle_sample_grid(args.ref_n, args.steps + args.warmup)
    sec, cores = time_oracle(n, args.steps, args.warmup)
    value = n ** 3 / sec
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": sec * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": (f"config4: 3D MHD decaying turbulence {n}^3, AB2, 2/3 dealiasing, nu=eta=1e-3, dt=2e-4, cs=1" if n == 512 else
                                f"config4 recipe (decaying MHD turbulence, AB2, 2/3 dealiasing) on a bounded {n}^3 sample of the 512^3 box"),
                   "grid": [n, n, n], "integrator": "AB2", "grid_choice": why},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle",
                         "sample": f"{args.steps} AB2 steps at {n}^3 after {args.warmup} warm-up steps ({why})"},
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
    s = mhd.Solver(n, n, n, cfg.nu, cfg.eta, cfg.cs, cfg.dt, flags=args.flags, device=dev)
    s.set_fields_host(*host)
    s.step(max(W, 4))                               # warm-up: Euler first step, one eager step, graph capture, first replay
    s.synchronize()

    # ---- timed region: K steps on the SHIPPED path (mhd_step = CUDA-graph replay), state resident in HBM ----
    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize()
    sampler = ClockSampler(local) if rank == 0 else None
    l0 = mhd.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(s.stream)
    s.step(K)
    e1.record(s.stream)
    torch.cuda.synchronize()
    if dist is not None:
        dist.barrier()
    launches = mhd.launch_count() - l0
    ms_total = max_over_ranks(e0.elapsed_time(e1), dist, dev)
    ms_step = ms_total / K
    value = world * npts * K / (ms_total * 1e-3)

    # ---- second pass, same K steps, eager with a CUDA-event pair around every launch: the per-kernel table ----
    s.profile_begin()
    p0, p1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    p0.record(s.stream)
    s.step(K)
    p1.record(s.stream)
    torch.cuda.synchronize()
    prof = s.profile_end()
    ms_prof_total = p0.elapsed_time(p1)

    # ---- end to end through the C ABI with HOST buffers: H2D of the 7 fields, K steps, diagnostics, D2H ----
    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    s.set_fields_host(*host)
    s.step(K)
    d = s.diagnostics(0)
    s.get_fields_host(host)
    torch.cuda.synchronize()
    e2e_s = max_over_ranks(time.perf_counter() - t0, dist, dev)
    clocks = sampler.stop() if sampler else None      # sampled from the start of the timed region to the end of the e2e pass
    nfield_bytes = 7 * 8 * npts
    e2e = {"value": world * npts * K / e2e_s, "unit": UNIT, "h2d_bytes_per_step": nfield_bytes / K,
           "d2h_bytes_per_step": (nfield_bytes + 128) / K,
           "what": f"mhd_set_fields_host (7 pinned fields) + mhd_step({K}) + mhd_diagnostics + mhd_get_fields_host, wall clock"}
    s.close()
    del s

    if rank != 0:
        return 0

    # ---- measured on-chip ceilings (FP64 FMA pipe, shared-memory data path) for the kernels that are not HBM-bound ----
    fp64_tflops, smem_gbs = mhd.measure_peaks(dev)
    exch_gbs = mhd.measure_exchange(192, dev)       # the fused pass's exchange pattern alone, with its FP64 work per exchange

    # ---- per-kernel rooflines, timed live with CUDA events ----
    abytes = algorithmic_bytes(geo)
    traffic = load_traffic()
    kernels = []
    for name, (count, ms) in prof.items():
        if count == 0 or name not in abytes:
            continue
        per = ms / count
        k = {"kernel": name, "launches_per_step": count / K, "ms_per_launch": per,
             "algorithmic_gb": abytes[name] / 1e9, "gbs": abytes[name] / 1e9 / (per * 1e-3),
             "hbm_frac": abytes[name] / 1e9 / (per * 1e-3) / peak, "share_of_step": ms / ms_prof_total,
             "traffic": traffic.get(name)}
        # ALGORITHMIC floors only: bytes the method must move, FP64 instructions the method must issue.
        floors = {"hbm": abytes[name] / (peak * 1e9) * 1e3}               # ms
        if name == "x_fused":
            dp, smem = xfused_onchip_model(geo)
            floors["alu"] = dp * 2.0 / (fp64_tflops * 1e12) * 1e3          # every FP64 instruction occupies one DFMA slot (2 flop)
            k["fp64_instr"] = dp
            # this implementation's own shared-memory traffic (two exchanges per transform through padded buffers): a property
            # of the design, not of the method -- a diagnostic, never the roofline
            smem_gbs_kernel = smem / 1e9 / (per * 1e-3)
            k["design_model"] = {"smem_bytes": smem, "smem_floor_ms": smem / (smem_gbs * 1e9) * 1e3,
                                 "frac_of_smem_peak": smem_gbs_kernel / smem_gbs if smem_gbs > 0 else None,
                                 "smem_exchange_ceiling_gbs": exch_gbs,
                                 "frac_of_exchange_ceiling": smem_gbs_kernel / exch_gbs if exch_gbs > 0 else None}
        k["floors_ms"] = floors
        k["bound"] = max(floors, key=floors.get)
        k["frac"] = floors[k["bound"]] / per
        kernels.append(k)
    kernels.sort(key=lambda k: -k["share_of_step"])
    top = kernels[0]
    unit = {"hbm": "GB/s", "alu": "TFLOP/s"}[top["bound"]]
    if top["bound"] == "hbm":
        achieved, pk, what = top["gbs"], peak, peak_src
    else:
        achieved, pk = top["fp64_instr"] * 2.0 / 1e12 / (top["ms_per_launch"] * 1e-3), fp64_tflops
        what = "measured in this run by mhd_measure_peaks (independent DFMA chains; a DFMA slot = 2 flop)"
    roofline = {"bound": top["bound"], "kernel": top["kernel"], "achieved": achieved, "peak": pk, "unit": unit,
                "frac": top["frac"], "traffic": top["traffic"], "peak_source": what,
                "hbm_frac": top["hbm_frac"], "hbm_peak": peak, "hbm_peak_source": peak_src,
                "algorithmic_bytes_per_launch": abytes[top["kernel"]], "floors_ms": top["floors_ms"],
                "share_of_step": top["share_of_step"], "design_model": top.get("design_model"),
                "note": "bound = the higher of the kernel's ALGORITHMIC floors (HBM bytes of the pruned transforms; FP64 instruction "
                        "slots of the butterflies and products, DESIGN.md §6); frac = that floor / measured time; hbm_frac is kept "
                        "beside it.  design_model = this implementation's own shared-memory traffic against the measured "
                        "shared-memory peak and against what its barrier-synchronised exchange pattern reaches alone "
                        "(mhd_measure_exchange): a diagnostic of the design, not a roofline"}
    own_bytes = sum(k["algorithmic_gb"] * 1e9 * k["launches_per_step"] for k in kernels)   # only the kernel classes that ran
    step_roofline = {
        "design_bytes_per_step": own_bytes, "design_gbs": own_bytes / 1e9 / (ms_step * 1e-3),
        "design_frac_of_measured_peak": own_bytes / 1e9 / (ms_step * 1e-3) / peak,
        "design_frac_of_8TBs": own_bytes / 1e9 / (ms_step * 1e-3) / NOMINAL_HBM_GBS,
        "survey_111F_bytes": survey_reference_bytes(n, n, n),
        "survey_111F_frac_of_8TBs": survey_reference_bytes(n, n, n) / 1e9 / NOMINAL_HBM_GBS / (ms_step * 1e-3),
        "profiled_pass_ms_per_step": ms_prof_total / K,
    }

    # ---- BASELINE metric, second half ("FFT HBM GB/s vs peak"): compact config-5 sweep in the same line ----
    fft = None
    if not args.no_fft:
        torch.cuda.empty_cache()
        fft = fft_sweep_rows([int(v) for v in args.fft_sizes.split(",")], dev, peak, reps=3, cufft=False)

    # ---- BASELINE configs 1-3 (launch-bound, L2-resident grids) at full length, AB2, in the same line ----
    small = None
    if not args.no_small:
        from paper_2402_05478_b200 import inputs as _inputs
        small = []
        for cid, make in ((1, _inputs.config1), (2, _inputs.config2), (3, _inputs.config3)):
            c = make()
            row = time_small_config(c, dev, 2, args.flags, (("AB2", mhd.AB2),))[0]
            row.update({"config": cid, "grid": [c.nx, c.ny, c.nz], "hydro": bool(c.hydro)})
            small.append(row)

    # ---- the oracle timed beside it on this box's host cores (bounded sample) ----
    cpu = None
    if not args.no_cpu_baseline:
        host = None                                  # the pinned input copies (7 fields) are no longer needed
        import gc
        gc.collect()
        cpu_n, why = oracle_sample_grid(args.cpu_n, args.cpu_steps + 1, budget_s=90.0)
        sec, cores = time_oracle(cpu_n, args.cpu_steps, 1)
        cpu = {"value": cpu_n ** 3 / sec, "unit": UNIT, "cores": cores, "kind": "oracle",
               "sample": f"{args.cpu_steps} AB2 steps (after 1 Euler warm-up step) of the config-4 recipe at {cpu_n}^3 ({why}), {sec:.2f} s per step"}

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W, "ms_per_step": ms_step,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"config4: 3D MHD decaying turbulence {n}^3, AB2, 2/3 dealiasing, nu=eta=1e-3, dt=2e-4, cs=1",
                   "grid": [n, n, n], "integrator": "AB2", "multi_gpu": "replicas only (no data-path collective)",
                   "timed_path": "mhd_step(K): CUDA-graph replay (the shipped path); the per-kernel table comes from a second, eager pass",
                   "l2": "inputs larger than L2 (spectral state 2.2 GB + 18 GB of transients per step vs 126 MB L2)",
                   "flags": args.flags, "ekin_after_run": d["ekin"], "emag_after_run": d["emag"]},
        "clocks": clocks, "e2e": e2e, "gpu_launches": launches,
        "roofline": roofline, "step_roofline": step_roofline, "kernels": kernels,
        "peaks": {"hbm_gbs": peak, "hbm_source": peak_src, "fp64_tflops": fp64_tflops, "smem_gbs": smem_gbs,
                  "smem_exchange_gbs": exch_gbs, "onchip_source": "mhd_measure_peaks / mhd_measure_exchange(192), this run"},
        "fft": fft, "small_configs": small, "cpu_baseline": cpu,
    }
    print(json.dumps(line), flush=True)
    return 0


def time_small_config(cfg, dev, reps, extra_flags, integrators):
    """One BASELINE small config at its full step count on the shipped path (CUDA-graph replay), per integrator: median of
    `reps` timed runs after one untimed run, CUDA events on the solver's stream."""
    import torch
    from paper_2402_05478_b200 import mhd
    flags = (mhd.FLAG_HYDRO if cfg.hydro else 0) | extra_flags
    rows = []
    for name, integ in integrators:
        s = mhd.Solver(cfg.nx, cfg.ny, cfg.nz, cfg.nu, cfg.eta, cfg.cs, cfg.dt, integrator=integ, flags=flags, device=dev)
        arrs = [torch.from_numpy(a).to(dev) for a in cfg.arrays()]
        ts = []
        l0 = mhd.launch_count()
        for rep in range(1 + reps):
            s.set_fields(*arrs)
            s.step(4)                                   # Euler start, eager step, capture, first replay: not timed
            s.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(s.stream); s.step(cfg.steps); e1.record(s.stream)
            torch.cuda.synchronize()
            if rep:
                ts.append(e0.elapsed_time(e1))
        ms = statistics.median(ts)
        d = s.diagnostics(0)
        rows.append({"integrator": name, "steps": cfg.steps, "ms_per_step": ms / cfg.steps,
                     "grid_point_updates_per_s": cfg.nx * cfg.ny * cfg.nz * cfg.steps / (ms * 1e-3),
                     "launches": (mhd.launch_count() - l0) // (1 + reps), "ekin": d["ekin"], "emag": d["emag"]})
        s.close()
    return rows


def run_small_config(args):
    """--config 1|2|3: BASELINE configs 1-3 at their full step count on the shipped path (CUDA-graph replay), AB2, with the
    oracle timed beside it at FULL length on the host cores.  These grids are L2-resident and launch-bound."""
    import torch
    from paper_2402_05478_b200 import inputs, mhd
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device")
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(dev)
    cfg = {1: inputs.config1, 2: inputs.config2, 3: inputs.config3}[args.config]()
    rows = time_small_config(cfg, dev, args.reps, args.flags, (("AB2", mhd.AB2), ("RK4", mhd.RK4)))
    cpu = None
    if not args.no_cpu_baseline:
        from oracle import mhd_ref
        o = mhd_ref.RefSolver(cfg.nx, cfg.ny, cfg.nz, cfg.nu, cfg.eta, cfg.cs, cfg.dt, flags=1 if cfg.hydro else 0)
        o.set_fields(*cfg.arrays())
        t0 = time.perf_counter(); o.step(cfg.steps); sec = time.perf_counter() - t0
        cpu = {"value": cfg.nx * cfg.ny * cfg.nz * cfg.steps / sec, "unit": UNIT, "cores": mhd_ref.get_threads(), "kind": "oracle",
               "sample": f"the full config: {cfg.steps} AB2 steps at {cfg.nx}x{cfg.ny}x{cfg.nz}, {sec:.2f} s"}
        o.close()
    line = {"metric": METRIC, "value": rows[0]["grid_point_updates_per_s"], "unit": UNIT, "n_gpus": 1, "steps": cfg.steps,
            "ms_per_step": rows[0]["ms_per_step"], "higher_is_better": True, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"{cfg.name}: {cfg.nx}x{cfg.ny}x{cfg.nz}, {cfg.steps} steps, CUDA-graph replay",
                       "l2": "L2-resident by construction (the config's whole working set is smaller than L2); launch-bound"},
            "runs": rows, "cpu_baseline": cpu}
    print(json.dumps(line), flush=True)
    return 0


def run_peaks(args):
    import torch
    from paper_2402_05478_b200 import mhd
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device")
    sampler = ClockSampler(0)
    vals = [mhd.measure_peaks("cuda:0") for _ in range(3)]
    exch = {str(d): max(mhd.measure_exchange(d, "cuda:0") for _ in range(2)) for d in (0, 64, 128, 192, 256)}
    exch_modes = {name: max(mhd.measure_exchange(192, "cuda:0", m) for _ in range(2))
                  for m, name in enumerate(("write_barrier_read_barrier", "barrier_write_barrier_read", "double_buffer_one_barrier",
                                             "warp_shuffle_octet_transpose_no_smem"))}
    clocks = sampler.stop()
    f, sm = max(v[0] for v in vals), max(v[1] for v in vals)
    sms = torch.cuda.get_device_properties(0).multi_processor_count
    mhz = clocks["sm_mhz"] or 0.0
    line = {"metric": "onchip_peaks", "fp64_tflops": f, "smem_gbs": sm, "clocks": clocks, "sms": sms,
            "dfma_per_clk_per_sm": (f * 1e12 / 2 / sms / (mhz * 1e6)) if mhz else None,
            "smem_bytes_per_clk_per_sm": (sm * 1e9 / sms / (mhz * 1e6)) if mhz else None,
            "smem_exchange_gbs_by_dfma_per_exchange": exch, "smem_exchange_gbs_by_barrier_placement_at_192": exch_modes,
            "hbm_gbs": measured_peak()[0]}
    print(json.dumps(line), flush=True)
    return 0


def fft_sweep_rows(sizes, dev, peak, reps=5, cufft=True):
    """BASELINE config 5: batched 3-D R2C + C2R of 7 fields; effective GB/s = (input + output bytes) / t (the 2F ideal)."""
    import torch
    from paper_2402_05478_b200 import mhd
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)       # > 126 MB L2
    sweep = []
    for n in sizes:
        batch = 7
        gen = torch.Generator(device=dev); gen.manual_seed(1005)
        a = torch.rand((batch, n, n, n), dtype=torch.float64, device=dev, generator=gen) * 2.0 - 1.0
        plan = mhd.FftPlan(n, n, n, batch, stream=torch.cuda.current_stream(dev), plane_workspace=n in (64, 128, 256, 512))
        spec = plan.r2c(a)
        back = plan.c2r(spec)
        err = float(torch.linalg.norm(back - a) / torch.linalg.norm(a))

        def timed(fn, reps=reps):
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
        if n in (64, 128, 256, 512):     # the 2-sweep plan mode (x and y passes through an L2-resident ring), measured beside the default
            plan.set_mode(mhd.FFT_PLANE_PIPELINE)
            row["plane_pipeline_r2c_ms"] = timed(lambda: plan.r2c(a, out=spec))
            row["plane_pipeline_c2r_ms"] = timed(lambda: plan.c2r(spec, out=back))
            plan.set_mode(mhd.FFT_THREE_SWEEP)
        plan.close()
        del plan, back
        if cufft:
            try:   # reference line only: cuFFT through torch.fft
                row["cufft_r2c_ms"] = timed(lambda: torch.fft.rfftn(a, dim=(1, 2, 3)), reps=3)
            except Exception as ex:   # out of memory at the largest size is not an error of this library
                row["cufft_r2c_ms"] = None
                row["cufft_note"] = type(ex).__name__
        del a, spec
        torch.cuda.empty_cache()
        sweep.append(row)
    return sweep


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
    l0 = mhd.launch_count()
    sweep = fft_sweep_rows([int(v) for v in args.fft_sizes.split(",")], dev, peak)
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
    ap.add_argument("--ref-n", type=int, default=0, help="grid size the reference arm times (0: 512 when memory and the step count allow, else 256 / 128)")
    ap.add_argument("--cpu-n", type=int, default=0, help="grid size of the cpu_baseline sample (0: 512, the metric's grid, when the host has the memory, else 256)")
    ap.add_argument("--cpu-steps", type=int, default=3, help="timed oracle steps of the cpu_baseline sample (BASELINE.md §4: 3 steps at 512^3, about 60 s)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--workload", default="step", choices=["step", "fft", "peaks"],
                    help="step: the 512^3 MHD step (default, carries the compact FFT sweep too); fft: the config-5 FFT sweep with the cuFFT line; "
                         "peaks: the measured FP64 / shared-memory ceilings")
    ap.add_argument("--fft-sizes", default="128,256,512,768")
    ap.add_argument("--no-small", action="store_true", help="skip the BASELINE config 1-3 rows (small_configs) in the default line")
    ap.add_argument("--no-fft", action="store_true", help="skip the compact config-5 sweep in the default line")
    ap.add_argument("--config", type=int, default=0, choices=[0, 1, 2, 3], help="time BASELINE config 1, 2 or 3 at full length instead")
    ap.add_argument("--reps", type=int, default=3, help="--config: timed repetitions (median)")
    ap.add_argument("--flags", type=int, default=0, help="extra mhd_create flags (execution-plan switches of include/mhd.h)")
    args = ap.parse_args(argv)
    if args.steps < 1:
        raise SystemExit("--steps must be >= 1")
    if args.impl == "reference":
        return run_reference(args)
    if args.config:
        return run_small_config(args)
    if args.workload == "peaks":
        return run_peaks(args)
    return run_fft_sweep(args) if args.workload == "fft" else run_gpu(args)


if __name__ == "__main__":
    sys.exit(main())
