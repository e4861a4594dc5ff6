"""Host-side logic of bench.py on CPU: byte models, clock parsing, and the N>1 rank plumbing
(replicas only: barrier + max-over-ranks, no data-path collective) over gloo with world size 2."""
import json
import os
import socket
import subprocess
import sys

import pytest

import bench

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_geometry_is_the_two_thirds_rule():
    g = bench.geometry(512, 512, 512)
    assert (g["nkx"], g["nky"], g["nkz"]) == (171, 341, 341)        # |k| <= 170: 3*170 < 512 <= 3*171
    g = bench.geometry(32, 32, 32)
    assert (g["nkx"], g["nky"], g["nkz"]) == (11, 21, 21)           # |k| <= 10
    g = bench.geometry(256, 256, 1)
    assert (g["nkx"], g["nky"], g["nkz"]) == (86, 171, 1)
    g = bench.geometry(16, 16, 16, dealias=False)
    assert (g["nkx"], g["nky"], g["nkz"]) == (9, 16, 16)


def test_algorithmic_bytes_512_match_design_table():
    b = bench.algorithmic_bytes(bench.geometry(512, 512, 512))
    spec, w1, w2 = 341 * 341 * 171 * 16, 512 * 341 * 171 * 16, 512 * 512 * 171 * 16
    assert b["fft_z_inv"] == 7 * (spec + w1) and b["fft_z_fwd"] == 12 * (w1 + spec)
    assert b["fft_y_inv"] == 7 * (w1 + w2) and b["fft_y_fwd"] == 12 * (w2 + w1)
    assert b["x_fused"] == 19 * w2
    assert b["stage"] == (12 + 28) * spec
    # every byte count is "read once + write once": the fused step moves less than the survey's 111 F model
    fused = sum(b[k] for k in ("fft_z_inv", "fft_y_inv", "x_fused", "fft_y_fwd", "fft_z_fwd", "stage"))
    assert fused < bench.survey_reference_bytes(512, 512, 512)
    assert bench.survey_reference_bytes(512, 512, 512) == 111 * 16 * 257 * 512 * 512


def test_algorithmic_bytes_2d_hydro_has_no_z_pass():
    b = bench.algorithmic_bytes(bench.geometry(256, 256, 1), hydro=True)
    assert "fft_z_inv" not in b and "fft_z_fwd" not in b
    assert b["x_fused"] == (4 + 9) * 256 * 86 * 16


def test_xfused_onchip_model_matches_the_design_derivation():
    """per row 10 transforms of 3 radix-8 passes of 64 butterflies (56 FP64 instructions + 28 twiddle
    instructions on passes 2 and 3) + 35 per grid point; two exchanges of 2 x 16 B per point, 7 staged rows, 6 split pairs."""
    g = bench.geometry(512, 512, 512)
    dp, smem = bench.xfused_onchip_model(g)
    rows = 512 * 512
    assert dp == rows * (10 * 64 * (56 * 3 + 28 * 2) + 35 * 512)
    assert smem == rows * (10 * 2 * 2 * 16 * 512 + 7 * 16 * 171 + 6 * 2 * 16 * 171)
    # the floors they imply at the ceilings measured on B200 (34.1 TFLOP/s, 36.5 TB/s) bracket the HBM floor from above
    alu_ms, smem_ms, hbm_ms = dp * 2 / 34.1e12 * 1e3, smem / 36.5e12 * 1e3, bench.algorithmic_bytes(g)["x_fused"] / 6542.1e9 * 1e3
    assert 2.3 < alu_ms < 2.6 and 2.6 < smem_ms < 2.9 and 2.0 < hbm_ms < 2.2
    dph, _ = bench.xfused_onchip_model(bench.geometry(256, 256, 1), hydro=True)
    # 256 = 8*8*4 (the kernel's plan): two radix-8 passes of 32 butterflies, one radix-4 pass of 64; 2 inverse + 5 forward transforms
    assert dph == 256 * (7 * (32 * 56 + 32 * (56 + 28) + 64 * (16 + 12)) + 35 * 256)
    # lengths that are not powers of 8 take their pass count from the plan table, not from log8: 128 = 8*4*4, 1024 = 8*8*4*4
    dp128, sm128 = bench.xfused_onchip_model(bench.geometry(128, 128, 128))
    assert dp128 == 128 * 128 * (10 * (16 * 56 + 32 * (16 + 12) * 2) + 35 * 128)
    assert sm128 == 128 * 128 * (10 * 2 * 2 * 16 * 128 + 7 * 16 * 43 + 6 * 2 * 16 * 43)
    dp1024, sm1024 = bench.xfused_onchip_model(bench.geometry(1024, 8, 8))
    assert dp1024 == 64 * (10 * (128 * 56 + 128 * (56 + 28) + 256 * (16 + 12) * 2) + 35 * 1024)
    assert sm1024 == 64 * (10 * 3 * 2 * 16 * 1024 + 7 * 16 * 342 + 6 * 2 * 16 * 342)
    with pytest.raises(ValueError):
        bench.xfused_onchip_model(bench.geometry(384, 8, 8))         # 3*2^a lengths run the unfused plan


def test_parse_clock_samples():
    text = "\n".join([
        "0, 345, 1965, 180.1, 0x0000000000000000, Not Active, Not Active, Not Active, Not Active",
        "0, 1965, 1965, 720.5, 0x0000000000000004, Not Active, Not Active, Not Active, Active",
        "0, 1950, 1965, 910.0, 0x0000000000000004, Not Active, Not Active, Not Active, Active",
        "garbage line",
    ])
    c = bench.parse_clock_samples(text)
    assert c["sm_max_mhz"] == 1965.0 and c["samples"] == 3
    assert c["sm_mhz"] == pytest.approx(1957.5)          # median of the samples under load (>= half the top clock)
    assert c["reasons"] == ["sw_power_cap"]
    assert bench.parse_clock_samples("")["sm_mhz"] is None


def test_measured_peak_reads_the_driver_file_or_falls_back():
    peak, src = bench.measured_peak()
    assert peak > 1000.0 and ("measured" in src or "fallback" in src)


def test_load_traffic_reads_profiles_csv():
    t = bench.load_traffic()
    for v in t.values():
        assert v > 0


_WORKER = r"""
import os, sys, json
sys.path.insert(0, {root!r})
import bench, torch
rank, world, local, dist = bench.dist_setup(2, use_cuda=False)
assert world == 2 and dist is not None
dist.barrier()
ms = bench.max_over_ranks(10.0 + 5.0 * rank, dist, torch.device("cpu"))   # rank 1 is the slow replica
dist.barrier()
if rank == 0:
    print(json.dumps({{"ms": ms, "world": world}}))
dist.destroy_process_group()
"""


def test_replicas_only_rank_plumbing_gloo_world_size_2(tmp_path):
    """bench.py's N>1 path: one process per replica, barrier, MAX over ranks, rank 0 prints."""
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    script = tmp_path / "worker.py"
    script.write_text(_WORKER.format(root=ROOT))
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE="2",
                   MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True))
    outs = [p.communicate(timeout=180) for p in procs]
    for p, (o, e) in zip(procs, outs):
        assert p.returncode == 0, e[-2000:]
    line = json.loads(outs[0][0].strip().splitlines()[-1])
    assert line == {"ms": 15.0, "world": 2}          # the slower replica sets the time
    assert outs[1][0].strip() == ""                  # only rank 0 prints


def test_reference_arm_runs_on_rank0_only_and_prints_the_contract_line():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "1",
                        "--warmup", "0", "--ref-n", "16"], env=env, capture_output=True, text=True, timeout=300)
    assert r.returncode == 0 and r.stdout.strip() == ""
    env = dict(os.environ, RANK="0", WORLD_SIZE="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "1",
                        "--warmup", "1", "--ref-n", "16"], env=env, capture_output=True, text=True, timeout=300)
    assert r.returncode == 0, r.stderr[-2000:]
    line = json.loads(r.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["unit"] == bench.UNIT and line["value"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["e2e"]["h2d_bytes_per_step"] == 0
