"""Pins 8-13 of SURVEY.md §8(c.4): exact invariants, div B, ideal-limit energy conservation to the
integrator's order, dissipative energy balance, cyclic axis permutation, temporal order, plus
diagnostics identities (Parseval for the spectra).  Expected values come from identities of
eqs (1)-(4), not from oracle code."""
import numpy as np
import pytest

from paper_2402_05478_b200 import inputs

TWO_PI = 2 * np.pi


def make(ref, n, nu, eta, cs, dt, integrator=0, seed=7, kmax=2.0, flags=0, shape=None):
    nz, ny, nx = shape if shape else (n, n, n)
    fields = inputs.smooth_random_state(nx, ny, nz, seed=seed, kmax=kmax, hydro=bool(flags & 1))
    s = ref.RefSolver(nx, ny, nz, nu, eta, cs, dt, integrator=integrator, flags=flags)
    s.set_fields(*fields)
    return s, fields


# ---------------------------------------------------------------- pin 8: exact invariants
@pytest.mark.parametrize("integrator", [0, 1])
def test_mass_momentum_meanB_are_conserved(ref, integrator):
    s, _ = make(ref, 16, 0.02, 0.03, 1.0, 2e-3, integrator)
    d0 = s.diagnostics()
    s.step(10)
    d1 = s.diagnostics()
    assert abs(d1["mass"] - d0["mass"]) <= 1e-14
    assert np.max(np.abs(d1["mom"] - d0["mom"])) <= 1e-14
    assert np.max(np.abs(d1["bmean"] - d0["bmean"])) <= 1e-14
    assert d1["step"] == 10 and abs(d1["time"] - 10 * 2e-3) <= 1e-15


# ---------------------------------------------------------------- pin 9: div B at roundoff
def test_divB_stays_at_roundoff(ref):
    s, _ = make(ref, 24, 0.01, 0.01, 1.0, 2e-3, kmax=3.0)
    assert s.diagnostics()["max_divb"] <= 1e-13
    s.step(25)
    assert s.diagnostics()["max_divb"] <= 1e-13


def test_divB_diagnostic_sees_a_monopole(ref):
    """max_divb is max_x |div B| -- checked on B = (sin x, 0, 0) whose divergence is cos x (max 1)."""
    n = 16
    x = TWO_PI * np.arange(n) / n
    X = np.broadcast_to(x, (n, n, n))
    one, zero = np.ones((n, n, n)), np.zeros((n, n, n))
    s = ref.RefSolver(n, n, n, 0.0, 0.0, 1.0, 1e-3)
    s.set_fields(one, zero, zero, zero, np.sin(2 * X), zero, zero)
    assert abs(s.diagnostics()["max_divb"] - 2.0) <= 1e-13


# ---------------------------------------------------------------- diagnostics identities
def test_energies_match_their_definitions(ref):
    s, f = make(ref, 16, 0.0, 0.0, 1.3, 1e-3)
    rho, ux, uy, uz, bx, by, bz = f
    d = s.diagnostics(nshell=16)
    assert abs(d["ekin"] - np.mean(0.5 * rho * (ux ** 2 + uy ** 2 + uz ** 2))) <= 1e-14
    assert abs(d["emag"] - np.mean(0.5 * (bx ** 2 + by ** 2 + bz ** 2))) <= 1e-15
    assert abs(d["eiso"] - 1.3 ** 2 * np.mean(rho * np.log(rho))) <= 1e-15
    assert abs(d["mass"] - np.mean(rho)) <= 1e-15
    assert abs(d["mom"][1] - np.mean(rho * uy)) <= 1e-15
    # Parseval: the shells partition the modes, so the spectra sum to the mean-square fields
    assert abs(d["emag_spec"].sum() - d["emag"]) <= 1e-14
    assert abs(d["ekin_spec"].sum() - np.mean(0.5 * (ux ** 2 + uy ** 2 + uz ** 2))) <= 1e-13


def test_spectrum_puts_a_single_mode_in_its_shell(ref):
    n = 16
    x = TWO_PI * np.arange(n) / n
    Z, Y, X = np.meshgrid(x, x, x, indexing="ij")
    one, zero = np.ones((n, n, n)), np.zeros((n, n, n))
    s = ref.RefSolver(n, n, n, 0.0, 0.0, 1.0, 1e-3)
    # |k| = sqrt(1+4+4) = 3 -> shell 3 ; |k| = sqrt(2) -> shell 1
    s.set_fields(one, 0.6 * np.cos(X + 2 * Y - 2 * Z), zero, zero, zero, 0.8 * np.sin(X + Z), zero)
    d = s.diagnostics(nshell=8)
    want_k = np.zeros(8); want_k[3] = 0.5 * 0.36 / 2
    want_m = np.zeros(8); want_m[1] = 0.5 * 0.64 / 2
    assert np.max(np.abs(d["ekin_spec"] - want_k)) <= 1e-15
    assert np.max(np.abs(d["emag_spec"] - want_m)) <= 1e-15


def test_diagnostics_flags_nonpositive_density(ref):
    n = 8
    one, zero = np.ones((n, n, n)), np.zeros((n, n, n))
    rho = one.copy(); rho[0, 0, 0] = -1.0
    s = ref.RefSolver(n, n, n, 0.0, 0.0, 1.0, 1e-3, flags=ref.FLAG_NO_DEALIAS)
    s.set_fields(rho, zero, zero, zero, zero, zero, zero)
    assert s.diagnostics()["rc"] == ref.ENONFINITE


# ---------------------------------------------------------------- pins 10 + 13: order in time
def _total_energy_after(ref, integrator, dt, T, nu=0.0, eta=0.0, n=16):
    s, _ = make(ref, n, nu, eta, 1.0, dt, integrator, seed=11)
    s.step(int(round(T / dt)))
    d = s.diagnostics()
    return d["ekin"] + d["emag"] + d["eiso"], s.get_fields()


@pytest.mark.parametrize("integrator,order", [(0, 2), (1, 4)])
def test_ideal_limit_energy_drift_has_integrator_order(ref, integrator, order):
    """nu = eta = 0: ekin + emag + eiso (eiso = cs^2 <rho ln rho>) is the invariant of the isothermal
    system; the time-integration part of its drift falls by 2^order per halving of dt (Richardson
    differences cancel the dt-independent spatial truncation error of the 16^3 grid)."""
    T = 0.4
    dts = [T / 16, T / 32, T / 64] if integrator == 1 else [T / 40, T / 80, T / 160]
    E = [_total_energy_after(ref, integrator, dt, T)[0] for dt in dts]
    rate = np.log2(abs(E[0] - E[1]) / abs(E[1] - E[2]))
    assert abs(rate - order) <= 0.3, (rate, E)


def test_ideal_limit_conserves_total_energy_up_to_spectrally_small_truncation(ref):
    """What is left as dt -> 0 is the spatial truncation error, which falls spectrally with n
    (measured 8e-5, 9e-6, 3e-7 relative at 16^3, 24^3, 32^3); kinetic + magnetic energy alone is not
    conserved: the compression work goes through eiso."""
    T, drift = 0.4, []
    for n in (16, 32):
        s, _ = make(ref, n, 0.0, 0.0, 1.0, T / 32, 1, seed=11)
        d0 = s.diagnostics()
        s.step(32)
        d1 = s.diagnostics()
        tot = lambda d: d["ekin"] + d["emag"] + d["eiso"]
        drift.append(abs(tot(d1) - tot(d0)) / tot(d0))
    assert drift[1] <= 1e-6 and drift[1] <= drift[0] / 50
    assert abs((d1["ekin"] + d1["emag"]) - (d0["ekin"] + d0["emag"])) > 1e-3 * tot(d0)


@pytest.mark.parametrize("integrator,order", [(0, 2), (1, 4)])
def test_temporal_self_convergence(ref, integrator, order):
    T = 0.2
    dts = [T / 10, T / 20, T / 40] if integrator == 1 else [T / 20, T / 40, T / 80]
    sol = [np.array(_total_energy_after(ref, integrator, dt, T, nu=0.01, eta=0.01)[1]) for dt in dts]
    e1 = np.linalg.norm(sol[0] - sol[1])
    e2 = np.linalg.norm(sol[1] - sol[2])
    assert abs(np.log2(e1 / e2) - order) <= 0.25, np.log2(e1 / e2)


def test_ab2_and_rk4_converge_to_the_same_solution(ref):
    T = 0.1
    a = np.array(_total_energy_after(ref, 0, T / 400, T, nu=0.01, eta=0.01)[1])
    b = np.array(_total_energy_after(ref, 1, T / 20, T, nu=0.01, eta=0.01)[1])
    assert np.linalg.norm(a - b) <= 2e-6 * np.linalg.norm(b)


# ---------------------------------------------------------------- pin 11: dissipative energy balance
def test_energy_balance_with_viscosity_and_resistivity(ref):
    """d/dt (ekin+emag+eiso) = -nu <|grad u|^2> - eta <|curl B|^2>, both evaluated here with numpy.fft."""
    n, nu, eta, dt = 16, 0.05, 0.08, 5e-4
    s, _ = make(ref, n, nu, eta, 1.0, dt, integrator=1, seed=5)
    s.step(20)
    tot = lambda d: d["ekin"] + d["emag"] + d["eiso"]
    Em = tot(s.diagnostics())
    s.step(1)
    f = s.get_fields()
    s.step(1)
    Ep = tot(s.diagnostics())
    k = np.fft.fftfreq(n, 1.0 / n)
    K = [np.arange(n // 2 + 1).reshape(1, 1, -1), k.reshape(1, -1, 1), k.reshape(-1, 1, 1)]   # x, y, z
    ddx = lambda a, ax: np.fft.irfftn(1j * K[ax] * np.fft.rfftn(a), s=(n, n, n), axes=(0, 1, 2))
    grad_u2 = sum(np.mean(ddx(f[1 + i], j) ** 2) for i in range(3) for j in range(3))
    bx, by, bz = f[4], f[5], f[6]
    J = [ddx(bz, 1) - ddx(by, 2), ddx(bx, 2) - ddx(bz, 0), ddx(by, 0) - ddx(bx, 1)]
    j2 = sum(np.mean(c ** 2) for c in J)
    want = -nu * grad_u2 - eta * j2
    got = (Ep - Em) / (2 * dt)
    assert abs(got - want) <= 1e-5 * abs(want), (got, want)


# ---------------------------------------------------------------- pin 12: cyclic permutation of the axes
@pytest.mark.parametrize("integrator", [0, 1])
def test_cyclic_axis_permutation(ref, integrator):
    """Rotating the initial condition x->y->z->x must rotate the result: pins axis handling in the
    3-D transforms and the index pattern of k x E^ and k_j T^_ij."""
    shape = (8, 12, 16)                              # (nz, ny, nx), all different on purpose
    nz, ny, nx = shape
    f = inputs.smooth_random_state(nx, ny, nz, seed=3, kmax=2.0)
    s = ref.RefSolver(nx, ny, nz, 0.02, 0.03, 1.1, 2e-3, integrator=integrator)
    s.set_fields(*f)
    s.step(5)
    out = s.get_fields()
    # primed frame: x' = z, y' = x, z' = y.  a'[z',y',x'] = a[x',z',y'] = a.transpose(1,2,0); v'_x = v_z, v'_y = v_x, v'_z = v_y
    P = lambda a: np.ascontiguousarray(a.transpose(1, 2, 0))
    rot = lambda g: [P(g[0]), P(g[3]), P(g[1]), P(g[2]), P(g[6]), P(g[4]), P(g[5])]
    fp = rot(f)
    nzp, nyp, nxp = fp[0].shape
    sp = ref.RefSolver(nxp, nyp, nzp, 0.02, 0.03, 1.1, 2e-3, integrator=integrator)
    sp.set_fields(*fp)
    sp.step(5)
    outp = sp.get_fields()
    want = rot(out)
    for a, b in zip(outp, want):
        assert np.max(np.abs(a - b)) <= 1e-13


# ---------------------------------------------------------------- 2-D and hydro are the same algorithm
def test_hydro_flag_equals_zero_field_run_and_keeps_B_zero(ref):
    n = 16
    f = inputs.smooth_random_state(n, n, n, seed=9, hydro=True)
    a = ref.RefSolver(n, n, n, 0.02, 0.0, 1.0, 2e-3, flags=ref.FLAG_HYDRO)
    b = ref.RefSolver(n, n, n, 0.02, 0.0, 1.0, 2e-3)
    a.set_fields(*f[:4])
    b.set_fields(*f)
    a.step(5); b.step(5)
    fa, fb = a.get_fields(), b.get_fields()
    for i in range(4):
        assert np.array_equal(fa[i], fb[i])
    for i in range(4, 7):
        assert not np.any(fa[i]) and not np.any(fb[i])


def test_2d_run_equals_3d_run_of_z_independent_state(ref):
    n = 16
    f2 = inputs.smooth_random_state(n, n, 1, seed=21)
    f3 = [np.ascontiguousarray(np.broadcast_to(a, (4, n, n))) for a in f2]
    a = ref.RefSolver(n, n, 1, 0.02, 0.03, 1.0, 2e-3)
    b = ref.RefSolver(n, n, 4, 0.02, 0.03, 1.0, 2e-3)
    a.set_fields(*f2); b.set_fields(*f3)
    a.step(5); b.step(5)
    for x, y in zip(a.get_fields(), b.get_fields()):
        assert np.max(np.abs(y - x)) <= 1e-13


def test_step_before_set_fields_is_a_state_error(ref):
    s = ref.RefSolver(8, 8, 8, 0.0, 0.0, 1.0, 1e-3)
    with pytest.raises(RuntimeError):
        s.step(1)
    with pytest.raises(ValueError):
        ref.RefSolver(8, 8, 8, 0.0, 0.0, 1.0, -1.0)
