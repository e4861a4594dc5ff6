"""Long-run physics validation on the GPU: the coherent kinetic <-> magnetic energy exchange of
the paper's Test 5 (3-D ABC flow, printed period T = 30.171) and Test 3 (2-D Orszag-Tang flow,
PAPER.md:219-226, T = 2.971).  These are WEAK pins: the paper does not state the direction of
the ambient field, nor Re/Rm and u0 of exactly these runs, so the runs below use the readings written in each test and
the bars are percent-level, not roundoff-level.  They validate physics (and exercise O(1e4-1e5)-step runs, RK4 at
Ms = 0.01, the 2-D path), not parity.  The printed periods come from tests/golden/paper_values.json."""
import json
import os

import numpy as np
import pytest

pytestmark = [pytest.mark.gpu, pytest.mark.slow]

from paper_2402_05478_b200 import inputs

TWO_PI = 2 * np.pi
GOLD = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "paper_values.json")))


@pytest.fixture(scope="module")
def gpu():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2402_05478_b200 import mhd
    mhd.lib()
    return mhd


def maxima(t, y):
    """times of the interior local maxima of a sampled series, refined with a parabola"""
    out = []
    for i in range(1, len(y) - 1):
        if y[i] > y[i - 1] and y[i] >= y[i + 1]:
            d = (y[i - 1] - y[i + 1]) / (2 * (y[i - 1] - 2 * y[i] + y[i + 1]))
            out.append(t[i] + d * (t[1] - t[0]))
    return out


def energy_series(gpu, shape, fields, nu, eta, cs, dt, tend, every, integrator):
    import torch
    nz, ny, nx = shape
    s = gpu.Solver(nx, ny, nz, nu, eta, cs, dt, integrator=integrator)
    s.set_fields(*[torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in fields])
    t, ek, em = [0.0], [], []
    d = s.diagnostics(); ek.append(d["ekin"]); em.append(d["emag"])
    for _ in range(int(round(tend / dt)) // every):
        s.step(every)
        d = s.diagnostics()
        assert d["rc"] == 0
        t.append(d["time"]); ek.append(d["ekin"]); em.append(d["emag"])
    return np.array(t), np.array(ek), np.array(em), d


def test_abc_flow_energy_exchange_period(gpu):
    """Reading: u0 = 0.1, Ms = 0.1 (Cs = 1), M_A = 1 (V_A = B0 = 0.1) as in App. A's text, uniform B0
    along x, Re = Rm = 1000, 64^3 (PAPER.md:352 finds 64^3 sufficient), dt = 1e-3.  Linear theory gives pi/(k0 V_A) =
    31.42 for the exchange period; the paper prints 30.171; this code gives 29.67 at 64^3 and 128^3, AB2 and RK4."""
    n = 64
    one = np.ones((n, n, n))
    u = inputs.abc_flow(n, n, n, u0=0.1)
    t, ek, em, d = energy_series(gpu, (n, n, n), [one] + u + [0.1 * one, 0 * one, 0 * one], 1e-3, 1e-3, 1.0, 1e-3, 55.0, 100, 0)
    pk = maxima(t, em)
    assert len(pk) >= 2
    T = pk[1] - pk[0]
    assert abs(T - GOLD["period_3d_abc"]["value"]) <= 0.03 * GOLD["period_3d_abc"]["value"], T
    assert abs(T - np.pi / 0.1) <= 0.07 * np.pi / 0.1
    assert em.max() > 2.0 * em[0] and ek.min() < 0.5 * ek[0]         # a real exchange, not a ripple
    assert d["max_divb"] <= 1e-12 and abs(d["mass"] - 1.0) <= 1e-12   # invariants after 55 000 steps


def test_orszag_tang_2d_energy_exchange_period(gpu):
    """Reading: A = 1, k0 = 1, u0 = 1, M_A = 1 (uniform B0 = 1 along x), Ms = 0.01 (Cs = 100), Re = Rm = 1000, 128^2,
    dt = 1e-4 (the paper's).  AB2 is unstable for sound waves at Cs kmax dt = 0.42 with no damping there, so RK4 is used.
    The paper prints T = 2.971; pi/(k0 V_A) = 3.14; this code gives 3.14-3.18."""
    n = 128
    x = TWO_PI * np.arange(n) / n
    Y, X = np.meshgrid(x, x, indexing="ij")
    one = np.ones((1, n, n))
    f = [one, (-np.sin(Y))[None], np.sin(X)[None], 0 * one, one.copy(), 0 * one, 0 * one]
    t, ek, em, d = energy_series(gpu, (1, n, n), f, 1e-3, 1e-3, 100.0, 1e-4, 7.0, 200, 1)
    pk = maxima(t, em)
    assert len(pk) >= 2
    T = pk[1] - pk[0]
    assert abs(T - GOLD["period_2d_orszag_tang"]["value"]) <= 0.08 * GOLD["period_2d_orszag_tang"]["value"], T
    assert abs(T - np.pi) <= 0.03 * np.pi
    assert d["max_divb"] <= 1e-10


def test_config2_kelvin_helmholtz_growth_rate_on_the_gpu(gpu):
    """BASELINE config 2 asks for the linear growth rate: 256^2 hydro KH (profile family of PAPER.md:163-172, eqs 6-7),
    snapshots every 50 steps; in the linear window t in [0.8, 1.4] the most unstable seeded mode kx = 4
    (kx a = 0.2, on the rising side of the paper's inverted parabola with its maximum at kx a = 0.4)
    must grow at the rate of the linear eigen-solve written in tests/test_oracle_kh.py (5 %)."""
    import torch
    from test_oracle_kh import amplitude, kh_eig
    c = inputs.config2(256, 2000)
    s = gpu.Solver(c.nx, c.ny, c.nz, c.nu, c.eta, c.cs, c.dt, flags=gpu.FLAG_HYDRO)
    s.set_fields(*[torch.from_numpy(a).cuda() for a in c.arrays()[:4]])
    s.step(800)
    ts, amps = [], {k: [] for k in (1, 2, 3, 4)}
    for i in range(13):
        uy = s.get_fields()[2][0].cpu().numpy()
        ts.append((800 + 50 * i) * c.dt)
        for k in amps:
            amps[k].append(np.log(amplitude(uy, k)))
        if i < 12:
            s.step(50)
    gam = {k: float(np.polyfit(ts, v, 1)[0]) for k, v in amps.items()}
    want = kh_eig(256, 0.05, 4, c.nu, c.cs)[0].real
    assert abs(gam[4] - want) <= 0.05 * want, (gam, want)
    assert gam[4] > gam[2] > 0.0          # growth increases with kx below the maximum at kx a = 0.4
