"""GPU parity for SURVEY.md §8(f) rows #2 and #3: box lengths, the steady body force of eq. (2), and the paper's
diagnostics (Omega(t) PAPER.md:201, Rayleigh quotient eq. (14)), CUDA library vs CPU oracle."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

from paper_2402_05478_b200 import inputs

TWO_PI = 2 * np.pi
PER_STEP, ENERGY = 1e-11, 1e-10


@pytest.fixture(scope="module")
def gpu():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2402_05478_b200 import mhd
    mhd.lib()
    return mhd


def rel(got, want):
    g = np.concatenate([np.asarray(a).ravel() for a in got])
    w = np.concatenate([np.asarray(a).ravel() for a in want])
    return float(np.linalg.norm(g - w) / np.linalg.norm(w))


def both(gpu, ref, shape, f, nu, eta, cs, dt, integrator=0, flags=0, box=None, force=None):
    import torch
    nz, ny, nx = shape
    o = ref.RefSolver(nx, ny, nz, nu, eta, cs, dt, integrator=integrator, flags=flags & 3)
    g = gpu.Solver(nx, ny, nz, nu, eta, cs, dt, integrator=integrator, flags=flags)
    if box is not None:
        o.set_box(*box)
        g.set_box(*box)
    if force is not None:
        o.set_forcing(*force)
        g.set_forcing(*[torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in force])
    o.set_fields(*f)
    g.set_fields(*[torch.from_numpy(a).cuda() for a in f])
    return o, g


def fields_err(g, o):
    got = [t.cpu().numpy() for t in g.get_fields()]
    want = o.get_fields()
    return max(rel(got[0:1], want[0:1]), rel(got[1:4], want[1:4]), rel(got[4:7], want[4:7]))


def diag_close(dg, do):
    for k in ("ekin", "emag", "eiso", "mass", "enstrophy", "current2", "u2", "rayleigh_q"):
        assert abs(dg[k] - do[k]) <= ENERGY * max(abs(do[k]), 1e-300) + (1e-15 if k == "eiso" else 0.0), (k, dg[k], do[k])
    assert abs(dg["max_divb"] - do["max_divb"]) <= 1e-11


@pytest.mark.parametrize("integrator", [0, 1])
def test_stretched_box_matches_oracle(gpu, ref, integrator):
    shape = (16, 24, 32)
    f = inputs.smooth_random_state(32, 24, 16, seed=31)
    o, g = both(gpu, ref, shape, f, 2e-3, 3e-3, 1.2, 5e-4, integrator=integrator, box=(1.0, 2.0, 3.0))
    o.step(1); g.step(1)
    assert fields_err(g, o) <= PER_STEP
    o.step(9); g.step(9)                      # AB2: steps 4.. replay the captured graph with the box baked in
    assert fields_err(g, o) <= 1e-12
    diag_close(g.diagnostics(), o.diagnostics())


def test_set_box_after_graph_capture_takes_effect(gpu, ref):
    shape = (16, 16, 16)
    f = inputs.smooth_random_state(16, 16, 16, seed=32)
    o, g = both(gpu, ref, shape, f, 1e-2, 1e-2, 1.0, 1e-3)
    o.step(6); g.step(6)
    o.set_box(TWO_PI, 3.0, TWO_PI); g.set_box(TWO_PI, 3.0, TWO_PI)
    o.step(6); g.step(6)
    assert fields_err(g, o) <= 1e-12


@pytest.mark.parametrize("integrator", [0, 1])
def test_forced_run_matches_oracle(gpu, ref, integrator):
    """forced ABC flow of App. B eq. (B3) (alpha = 0.1) on a smooth random MHD state."""
    n = 32
    shape = (n, n, n)
    f = inputs.smooth_random_state(n, n, n, seed=33)
    force = [0.1 * c for c in inputs.abc_flow(n, n, n)]
    o, g = both(gpu, ref, shape, f, 1e-2, 1e-2, 1.0, 1e-3, integrator=integrator, flags=gpu.FLAG_FORCING, force=force)
    o.step(1); g.step(1)
    assert fields_err(g, o) <= PER_STEP
    o.step(11); g.step(11)
    assert fields_err(g, o) <= 1e-12
    diag_close(g.diagnostics(16), o.diagnostics(16))
    # switching the force off (after graph capture) is honoured too
    o.set_forcing(None, None, None); g.set_forcing(None, None, None)
    o.step(5); g.step(5)
    assert fields_err(g, o) <= 1e-12


def test_forced_2d_hydro_orszag_tang_b2(gpu, ref):
    """App. B eq. (B2): 2-D flow forced with its own shape, hydro flag, host-buffer forcing call."""
    n = 64
    x = TWO_PI * np.arange(n) / n
    Y, X = np.meshgrid(x, x, indexing="ij")
    ux = (-np.sin(Y))[None].copy(); uy = np.sin(X)[None].copy()
    one = np.ones((1, n, n)); zero = np.zeros((1, n, n))
    import torch
    fl = gpu.FLAG_FORCING | gpu.FLAG_HYDRO
    o = ref.RefSolver(n, n, 1, 5e-3, 0.0, 2.0, 1e-3, flags=1)
    g = gpu.Solver(n, n, 1, 5e-3, 0.0, 2.0, 1e-3, flags=fl)
    o.set_forcing(0.1 * ux, 0.1 * uy, zero)
    g.set_forcing_host(np.ascontiguousarray(0.1 * ux), np.ascontiguousarray(0.1 * uy), zero)
    o.set_fields(one, ux, uy, zero)
    g.set_fields(*[torch.from_numpy(a).cuda() for a in (one, ux, uy, zero)])
    o.step(40); g.step(40)
    got = [t.cpu().numpy() for t in g.get_fields()]
    want = o.get_fields()
    assert rel(got[0:4], want[0:4]) <= 1e-12
    diag_close(g.diagnostics(), o.diagnostics())


def test_forcing_needs_the_flag_and_spectra_need_the_2pi_box(gpu):
    import torch
    s = gpu.Solver(16, 16, 16, 0.01, 0.01, 1.0, 1e-3)
    z = torch.zeros((16, 16, 16), dtype=torch.float64, device="cuda")
    with pytest.raises(gpu.MhdError) as e:
        s.set_forcing(z, z, z)
    assert e.value.code == gpu.ESTATE
    with pytest.raises(gpu.MhdError):
        s.set_box(-1.0, 1.0, 1.0)
    s.set_box(1.0, TWO_PI, TWO_PI)
    s.set_fields(z + 1.0, z, z, z, z, z, z)
    with pytest.raises(gpu.MhdError) as e:
        s.diagnostics(8)
    assert e.value.code == gpu.EINVAL
    assert s.diagnostics(0)["rc"] == 0


def test_paper_diagnostics_on_config1_and_closed_forms(gpu, ref):
    import torch
    cfg = inputs.config1()
    o = ref.RefSolver(cfg.nx, cfg.ny, cfg.nz, cfg.nu, cfg.eta, cfg.cs, cfg.dt)
    g = gpu.Solver(cfg.nx, cfg.ny, cfg.nz, cfg.nu, cfg.eta, cfg.cs, cfg.dt)
    o.set_fields(*cfg.arrays()); g.set_fields(*[torch.from_numpy(a).cuda() for a in cfg.arrays()])
    o.step(5); g.step(5)
    diag_close(g.diagnostics(), o.diagnostics())
    # Beltrami closed form on the GPU alone: ABC flow and field, Q = k0^2 (eq. 14 with curl u = k0 u)
    n = 32
    u = inputs.abc_flow(n, n, n, k0=2.0, u0=0.7)
    b = inputs.abc_flow(n, n, n, k0=2.0, u0=0.2)
    s = gpu.Solver(n, n, n, 0.01, 0.01, 1.0, 1e-3)
    s.set_fields(*[torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in [np.ones((n, n, n))] + u + b])
    d = s.diagnostics()
    assert abs(d["enstrophy"] - 4 * 3 * 0.49) <= 1e-12 and abs(d["rayleigh_q"] - 4.0) <= 1e-12


def test_execution_plan_flags_do_not_change_the_result(gpu, ref):
    """MHD_FLAG_NO_GRAPH is bit-identical to the default plan (same kernels, launched one by one); MHD_FLAG_UNFUSED_X (x C2R,
    products kernel, x R2C through real arrays) agrees with it to roundoff and with the oracle at the per-step bar.
    Nothing is selected through the environment."""
    import torch
    cfg = inputs.config1()
    dev = [torch.from_numpy(a).cuda() for a in cfg.arrays()]
    res = {}
    for name, fl in (("default", 0), ("nograph", gpu.FLAG_NO_GRAPH), ("unfused", gpu.FLAG_UNFUSED_X),
                     ("all", gpu.FLAG_NO_GRAPH | gpu.FLAG_UNFUSED_X)):
        s = gpu.Solver(cfg.nx, cfg.ny, cfg.nz, cfg.nu, cfg.eta, cfg.cs, cfg.dt, flags=fl)
        s.set_fields(*dev); s.step(9)
        res[name] = [t.cpu().numpy() for t in s.get_fields()]
    for a, b in zip(res["default"], res["nograph"]):
        assert np.array_equal(a, b)
    o = ref.RefSolver(cfg.nx, cfg.ny, cfg.nz, cfg.nu, cfg.eta, cfg.cs, cfg.dt)
    o.set_fields(*cfg.arrays()); o.step(9)
    want = o.get_fields()
    for name in ("unfused", "all"):
        assert rel(res[name], res["default"]) <= 1e-13, name
        assert rel(res[name], want) <= 1e-12, name
    with pytest.raises(gpu.MhdError):
        gpu.Solver(cfg.nx, cfg.ny, cfg.nz, cfg.nu, cfg.eta, cfg.cs, cfg.dt, flags=1 << 20)      # unknown flag bits are refused


def test_solver_runs_while_the_current_stream_and_device_context_differ(gpu):
    """every ABI call makes the workspace's device current for its own duration (DeviceGuard) and enqueues on the context's
    stream only: driving a solver from inside another stream context, and closing it right after an asynchronous step,
    must neither fail nor corrupt a tensor allocated immediately afterwards (close() synchronises the private stream)."""
    import torch
    cfg = inputs.config1()
    dev = [torch.from_numpy(a).cuda() for a in cfg.arrays()]
    a = gpu.Solver(cfg.nx, cfg.ny, cfg.nz, cfg.nu, cfg.eta, cfg.cs, cfg.dt)
    a.set_fields(*dev); a.step(40)
    want = [t.clone() for t in a.get_fields()]
    side = torch.cuda.Stream()
    with torch.cuda.stream(side):
        b = gpu.Solver(cfg.nx, cfg.ny, cfg.nz, cfg.nu, cfg.eta, cfg.cs, cfg.dt)
        b.set_fields(*dev); b.step(40)
        got = b.get_fields()
        b.step(200)                   # asynchronous work still in flight ...
        b.close()                     # ... when the context and its workspace are released
        junk = torch.full((b.workspace_bytes // 8,), 7.0, dtype=torch.float64, device="cuda")   # likely reuses the block
    torch.cuda.synchronize()
    for x, y in zip(want, got):
        assert torch.equal(x, y)
    assert bool((junk == 7.0).all())


def test_solver_on_a_second_gpu_while_the_first_is_current(gpu):
    """include/mhd.h: contexts on different devices of one process are independent, and every call makes the device that
    owns the workspace current for its own duration.  A solver created on cuda:1 and driven while cuda:0 is current must
    equal a cuda:0 run bit for bit and leave cuda:0 current; a stream that lives on the other GPU is refused at create.
    Needs two GPUs (the round's boxes have one: skipped there, with the reason)."""
    import torch
    if torch.cuda.device_count() < 2:
        pytest.skip(f"needs 2 GPUs, this box has {torch.cuda.device_count()}")
    cfg = inputs.config1()
    torch.cuda.set_device(0)
    a = gpu.Solver(cfg.nx, cfg.ny, cfg.nz, cfg.nu, cfg.eta, cfg.cs, cfg.dt, device="cuda:0")
    a.set_fields(*[torch.from_numpy(x).to("cuda:0") for x in cfg.arrays()]); a.step(12)
    b = gpu.Solver(cfg.nx, cfg.ny, cfg.nz, cfg.nu, cfg.eta, cfg.cs, cfg.dt, device="cuda:1")
    assert torch.cuda.current_device() == 0
    b.set_fields(*[torch.from_numpy(x).to("cuda:1") for x in cfg.arrays()]); b.step(12)
    assert torch.cuda.current_device() == 0
    for x, y in zip(a.get_fields(), b.get_fields()):
        assert y.device.index == 1 and torch.equal(x.cpu(), y.cpu())
    da, db = a.diagnostics(8), b.diagnostics(8)
    assert da["ekin"] == db["ekin"] and np.array_equal(da["ekin_spec"], db["ekin_spec"])
    with pytest.raises(gpu.MhdError) as e:
        gpu.Solver(cfg.nx, cfg.ny, cfg.nz, cfg.nu, cfg.eta, cfg.cs, cfg.dt, device="cuda:1", stream=torch.cuda.Stream(device="cuda:0"))
    assert e.value.code == gpu.EINVAL


@pytest.mark.parametrize("integrator", [0, 1])
def test_exact_resume_is_bit_identical(gpu, integrator):
    """mhd_get_state / mhd_set_state: a run interrupted after 5 steps and continued in a fresh
    context equals the uninterrupted run bit for bit (the AB2 history travels with the state; a restart from grid
    fields would re-bootstrap with an Euler step and differ)."""
    import torch
    cfg = inputs.config1()
    dev = [torch.from_numpy(a).cuda() for a in cfg.arrays()]
    a = gpu.Solver(cfg.nx, cfg.ny, cfg.nz, cfg.nu, cfg.eta, cfg.cs, cfg.dt, integrator=integrator)
    a.set_fields(*dev); a.step(12)
    b = gpu.Solver(cfg.nx, cfg.ny, cfg.nz, cfg.nu, cfg.eta, cfg.cs, cfg.dt, integrator=integrator)
    b.set_fields(*dev); b.step(5)
    blob = b.get_state().clone()
    c = gpu.Solver(cfg.nx, cfg.ny, cfg.nz, cfg.nu, cfg.eta, cfg.cs, cfg.dt, integrator=integrator)
    c.set_state(blob); c.step(7)
    for x, y in zip(a.get_fields(), c.get_fields()):
        assert torch.equal(x, y)
    assert c.diagnostics()["step"] == 12
    if integrator == 0:          # the naive restart really is different (so the test above is not vacuous)
        d = gpu.Solver(cfg.nx, cfg.ny, cfg.nz, cfg.nu, cfg.eta, cfg.cs, cfg.dt)
        d.set_fields(*b.get_fields()); d.step(7)
        assert not torch.equal(a.get_fields()[1], d.get_fields()[1])
    # a blob from another configuration is refused
    other = gpu.Solver(16, 16, 16, cfg.nu, cfg.eta, cfg.cs, cfg.dt, integrator=integrator)
    with pytest.raises(gpu.MhdError) as e:
        other.set_state(blob)
    assert e.value.code == gpu.EINVAL
    with pytest.raises(gpu.MhdError) as e:
        other.get_state()
    assert e.value.code == gpu.ESTATE


def test_onchip_probes_are_consistent(gpu):
    """Instrumentation (bench.py's on-chip ceilings): the FP64 and shared-memory probes land near the hardware's nominal rates,
    and the fused pass's exchange pattern can never beat the free-running shared-memory probe."""
    import torch
    sms = torch.cuda.get_device_properties(0).multi_processor_count
    fp64, smem = gpu.measure_peaks("cuda:0")
    assert 10.0 < fp64 < 2.0 * 64 * sms * 2.2e9 / 1e12              # TFLOP/s: positive, below 64 DFMA/clk/SM at 2.2 GHz
    assert 5e3 < smem < 128.0 * sms * 2.2                            # GB/s: below 128 B/clk/SM at 2.2 GHz
    for mode in (0, 1, 2):
        ex = gpu.measure_exchange(192, "cuda:0", mode)
        assert 0.5 * smem < ex < 1.02 * smem, (mode, ex, smem)
    assert gpu.measure_exchange(0, "cuda:0") >= 0.95 * gpu.measure_exchange(256, "cuda:0")     # FP64 work never speeds the exchange up
    shuffle = gpu.measure_exchange(192, "cuda:0", 3)                 # mode 3: warp-shuffle octet transpose, no shared memory
    print(f"exchange probe at 192 DFMA: shared memory {ex:.0f} GB/s-equivalent, warp shuffle {shuffle:.0f}")
    assert 1e3 < shuffle < 4.0 * smem
    with pytest.raises(gpu.MhdError):
        gpu.measure_exchange(100, "cuda:0")
    with pytest.raises(gpu.MhdError):
        gpu.measure_exchange(192, "cuda:0", 4)
