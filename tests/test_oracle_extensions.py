"""Pins for the oracle's SURVEY.md §8(f) rows #2 and #3: general box lengths, the steady
body force f of eq. (2) (App. B eqs B2-B3), and the paper's diagnostics
Omega(t) = <|curl u|^2> and the Rayleigh quotient Q(t) of eq. (14).
Every expected value comes from mathematics written here (closed forms, recurrences, the exact rescaling
symmetry of the equations, a numpy.fft restatement), never from oracle code."""
import numpy as np
import pytest

from paper_2402_05478_b200 import inputs

TWO_PI = 2 * np.pi


def coords(nx, ny, nz, lx=TWO_PI, ly=TWO_PI, lz=TWO_PI):
    x = lx * np.arange(nx) / nx
    y = ly * np.arange(ny) / ny
    z = lz * np.arange(nz) / nz
    Z, Y, X = np.meshgrid(z, y, x, indexing="ij")
    return X, Y, Z


def ab2_forced_scalar(z, c, nsteps, y0=0.0):
    """y' = lambda*y + s with z = lambda*dt, c = s*dt, under Euler-started AB2."""
    r_prev = z * y0 + c
    y = y0 + r_prev
    for _ in range(nsteps - 1):
        r = z * y + c
        y = y + 1.5 * r - 0.5 * r_prev
        r_prev = r
    return y if nsteps >= 1 else y0


# ------------------------------------------------------------------ box lengths
def test_box_rescaling_symmetry(ref):
    """x' = kappa*x, t' = kappa*t maps a box of length L = 2*pi/kappa onto the 2*pi box with
    (nu, eta, dt, f) -> (kappa*nu, kappa*eta, kappa*dt, f/kappa) and cs unchanged: the two oracle runs
    must agree to roundoff.  Uses different kappa per axis in its anisotropic variant below."""
    n, kappa = 16, 2.5
    L = TWO_PI / kappa
    f = inputs.smooth_random_state(n, n, n, seed=3, kmax=2.0)
    nu, eta, cs, dt, nsteps = 0.03, 0.02, 1.3, 2e-3, 8
    a = ref.RefSolver(n, n, n, nu, eta, cs, dt)
    a.set_box(L, L, L)
    a.set_fields(*f)
    a.step(nsteps)
    b = ref.RefSolver(n, n, n, kappa * nu, kappa * eta, cs, kappa * dt)
    b.set_fields(*f)
    b.step(nsteps)
    for x, y in zip(a.get_fields(), b.get_fields()):
        assert np.max(np.abs(x - y)) <= 1e-13
    da, db = a.diagnostics(), b.diagnostics()
    assert abs(da["ekin"] - db["ekin"]) <= 1e-14 and abs(da["emag"] - db["emag"]) <= 1e-14
    assert abs(da["max_divb"] - kappa * db["max_divb"]) <= 1e-12          # a derivative: scales with kappa
    assert abs(da["enstrophy"] - kappa ** 2 * db["enstrophy"]) <= 1e-11 * db["enstrophy"] * kappa ** 2
    assert abs(da["rayleigh_q"] - kappa ** 2 * db["rayleigh_q"]) <= 1e-11 * db["rayleigh_q"] * kappa ** 2


def test_default_box_is_two_pi_exactly(ref):
    n = 12
    f = inputs.smooth_random_state(n, n, n, seed=5)
    a = ref.RefSolver(n, n, n, 0.01, 0.01, 1.0, 1e-3)
    b = ref.RefSolver(n, n, n, 0.01, 0.01, 1.0, 1e-3)
    b.set_box(TWO_PI, TWO_PI, TWO_PI)
    for s in (a, b):
        s.set_fields(*f)
        s.step(3)
    for x, y in zip(a.get_fields(), b.get_fields()):
        assert np.array_equal(x, y)
    with pytest.raises(ValueError):
        a.set_box(0.0, 1.0, 1.0)


@pytest.mark.parametrize("axis_x,length,k_int", [(0, 1.0, 2), (1, 2.0, 3), (2, 0.5, 1)])
def test_shear_wave_on_a_stretched_box_decays_with_physical_wavenumber(ref, axis_x, length, k_int):
    """rho = 1, u = a sin(k x_j) e_i on a box with L_j = length: k = 2*pi*k_int/L_j, amplitude obeys the
    AB2 recurrence with z = -nu k^2 dt (KH test box Lx = 1, Ly = 2: PAPER.md:161)."""
    n, nu, dt, a, nsteps = 16, 1e-3, 1e-3, 0.3, 20
    ls = [TWO_PI, TWO_PI, TWO_PI]
    ls[axis_x] = length
    Xs = coords(n, n, n, *ls)
    k = TWO_PI * k_int / length
    axis_u = (axis_x + 1) % 3
    u = [np.zeros((n, n, n)) for _ in range(3)]
    u[axis_u] = a * np.sin(k * Xs[axis_x])
    zero = np.zeros((n, n, n))
    s = ref.RefSolver(n, n, n, nu, 0.0, 1.0, dt)
    s.set_box(*ls)
    s.set_fields(np.ones((n, n, n)), u[0], u[1], u[2], zero, zero, zero)
    s.step(nsteps)
    out = s.get_fields()
    y_prev, y, z = 1.0, 1.0 - nu * k * k * dt, -nu * k * k * dt
    for _ in range(nsteps - 1):
        y_prev, y = y, y + z * (1.5 * y - 0.5 * y_prev)
    assert np.max(np.abs(out[1 + axis_u] - y * u[axis_u])) <= 1e-13
    d = s.diagnostics()
    assert abs(d["enstrophy"] - k * k * 0.5 * (a * y) ** 2) <= 1e-13 * k * k    # <|curl u|^2> = k^2 <u^2>
    assert abs(d["rayleigh_q"] - k * k) <= 1e-10 * k * k


def test_sound_speed_on_a_short_box(ref):
    """small plane sound wave on Lx = 1: omega = cs * 2*pi/Lx (eqs 1-3)."""
    n, cs, amp, dt = 32, 1.5, 1e-6, 1e-4
    L = 1.0
    X, Y, Z = coords(n, 4, 4, L, TWO_PI, TWO_PI)
    k = TWO_PI / L
    rho = 1.0 + amp * np.cos(k * X)
    ux = cs * amp * np.cos(k * X)                        # right-going wave
    zero = np.zeros_like(X)
    s = ref.RefSolver(n, 4, 4, 0.0, 0.0, cs, dt)
    s.set_box(L, TWO_PI, TWO_PI)
    s.set_fields(rho, ux, zero, zero, zero, zero, zero)
    nsteps = 400
    s.step(nsteps)
    out = s.get_fields()
    t = nsteps * dt
    want = 1.0 + amp * np.cos(k * X - cs * k * t)
    assert np.max(np.abs(out[0] - want)) <= 2e-3 * amp      # O(dt^2) + O(amp) corrections


# ------------------------------------------------------------------ forcing
def test_forced_shear_flow_follows_the_forced_ab2_recurrence(ref):
    """rho = 1, u = 0, B = 0, f = alpha sin(k y) x^: an exact solution of the discrete system with
    m_x = Y(t) sin(k y), Y' = -nu k^2 Y + alpha (eq. 2 with f)."""
    n, nu, dt, alpha, k, nsteps = 16, 0.05, 1e-2, 0.1, 2, 30
    X, Y, Z = coords(n, n, n)
    zero = np.zeros((n, n, n))
    fx = alpha * np.sin(k * Y)
    s = ref.RefSolver(n, n, n, nu, 0.0, 1.0, dt)
    s.set_forcing(fx, zero, zero)
    s.set_fields(np.ones((n, n, n)), zero, zero, zero, zero, zero, zero)
    s.step(nsteps)
    out = s.get_fields()
    amp = ab2_forced_scalar(-nu * k * k * dt, alpha * dt, nsteps)
    assert np.max(np.abs(out[1] - amp * np.sin(k * Y))) <= 1e-13
    assert np.max(np.abs(out[0] - 1.0)) <= 1e-13 and np.max(np.abs(out[2])) <= 1e-13
    # steady state of the continuous problem: Y = alpha / (nu k^2)
    assert abs(ab2_forced_scalar(-nu * k * k * dt, alpha * dt, 40000) - alpha / (nu * k * k)) <= 1e-9
    # switching the force off again gives free decay
    s.set_forcing(None, None, None)
    s.set_fields(np.ones((n, n, n)), out[1], zero, zero, zero, zero, zero)
    s.step(1)
    assert np.max(np.abs(s.get_fields()[1] - (1 - nu * k * k * dt) * out[1])) <= 1e-13


@pytest.mark.parametrize("integrator", [0, 1])
def test_momentum_budget_with_a_mean_force(ref, integrator):
    """d<m>/dt = <f> exactly (the k = 0 mode of every divergence is 0): <m>(t) = <m>(0) + t <f> for Euler, AB2 and RK4."""
    n, dt, nsteps = 12, 2e-3, 7
    f = inputs.smooth_random_state(n, n, n, seed=11)
    rng = np.random.default_rng(2)
    X, Y, Z = coords(n, n, n)
    force = [0.3 + 0.1 * np.sin(X + Y), -0.2 + 0.05 * np.cos(2 * Z), 0.1 * np.sin(Y)]
    s = ref.RefSolver(n, n, n, 0.02, 0.02, 1.0, dt, integrator=integrator)
    s.set_forcing(*force)
    s.set_fields(*f)
    m0 = s.diagnostics()["mom"]
    s.step(nsteps)
    m1 = s.diagnostics()["mom"]
    want = m0 + nsteps * dt * np.array([0.3, -0.2, 0.0])
    assert np.max(np.abs(m1 - want)) <= 1e-14


def test_forcing_is_dealiased_like_every_rhs_term(ref):
    """a force on a mode outside the 2/3 mask does nothing."""
    n = 12                                             # kmax = 3
    X, Y, Z = coords(n, n, n)
    zero = np.zeros((n, n, n))
    s = ref.RefSolver(n, n, n, 0.0, 0.0, 1.0, 1e-2)
    s.set_forcing(np.sin(5 * Y), zero, zero)
    s.set_fields(np.ones((n, n, n)), zero, zero, zero, zero, zero, zero)
    s.step(3)
    assert np.max(np.abs(s.get_fields()[1])) <= 1e-15          # only the roundoff of the sampled mean survives


def test_paper_forcing_profiles_b2_b3_are_beltrami_balanced(ref):
    """App. B: the flow is forced 'with itself', f = alpha * (flow shape).  For the ABC shape
    (eq. B3) with rho = 1 and u = u0 * ABC the advection term is a pure gradient (curl u = k0 u), so in the
    low-Mach limit the forced flow u0 = alpha / (nu k0^2) is steady up to O(Ms^2)."""
    n, nu, alpha, k0 = 16, 0.5, 0.1, 1.0
    shape = inputs.abc_flow(n, n, n)
    u0 = alpha / (nu * k0 * k0)
    zero = np.zeros((n, n, n))
    cs = 20.0                                          # Ms = u0*sqrt(3)/cs ~ 0.017
    s = ref.RefSolver(n, n, n, nu, 0.0, cs, 2e-4)
    s.set_forcing(*[alpha * c for c in shape])
    s.set_fields(np.ones((n, n, n)), *[u0 * c for c in shape], zero, zero, zero)
    s.step(500)
    out = s.get_fields()
    for i in range(3):
        assert np.max(np.abs(out[1 + i] - u0 * shape[i])) <= 5e-3 * u0      # acoustic adjustment O(Ms) only; no decay
    # without the force the same flow decays: after t the amplitude is exp(-nu k0^2 t)
    s2 = ref.RefSolver(n, n, n, nu, 0.0, cs, 2e-4)
    s2.set_fields(np.ones((n, n, n)), *[u0 * c for c in shape], zero, zero, zero)
    s2.step(500)
    assert abs(np.max(np.abs(s2.get_fields()[1])) / np.max(np.abs(u0 * shape[0])) - np.exp(-nu * 500 * 2e-4)) <= 5e-3   # 4.9 % decay


# ------------------------------------------------------------------ paper diagnostics
def test_beltrami_fields_have_q_equal_k0_squared(ref):
    """ABC flow and field (eq. 11): curl u = k0 u, so Omega = k0^2 <|u|^2> = 3 k0^2 u0^2 and Q = k0^2."""
    n = 16
    for k0 in (1.0, 2.0):
        u = inputs.abc_flow(n, n, n, k0=k0, u0=0.7)
        b = inputs.abc_flow(n, n, n, k0=k0, u0=0.2)
        s = ref.RefSolver(n, n, n, 0.01, 0.01, 1.0, 1e-3)
        s.set_fields(np.ones((n, n, n)), *u, *b)
        d = s.diagnostics()
        assert abs(d["u2"] - 3 * 0.49) <= 1e-13
        assert abs(d["enstrophy"] - k0 ** 2 * 3 * 0.49) <= 1e-12
        assert abs(d["current2"] - k0 ** 2 * 3 * 0.04) <= 1e-12
        assert abs(d["rayleigh_q"] - k0 ** 2) <= 1e-12


def test_taylor_green_initial_enstrophy(ref):
    """TG vortex (eq. 8): u = (sin x cos y cos z, -cos x sin y cos z, 0) is solenoidal with
    every mode on |k|^2 = 3: <|u|^2> = 1/4 and Omega(0) = 3/4."""
    n = 16
    X, Y, Z = coords(n, n, n)
    ux = np.sin(X) * np.cos(Y) * np.cos(Z)
    uy = -np.cos(X) * np.sin(Y) * np.cos(Z)
    zero = np.zeros((n, n, n))
    s = ref.RefSolver(n, n, n, 0.01, 0.0, 1.0, 1e-3, flags=1)
    s.set_fields(np.ones((n, n, n)), ux, uy, zero)
    d = s.diagnostics()
    assert abs(d["u2"] - 0.25) <= 1e-14 and abs(d["enstrophy"] - 0.75) <= 1e-13
    assert d["current2"] == 0.0 and abs(d["rayleigh_q"] - 3.0) <= 1e-12


def test_enstrophy_and_q_match_a_numpy_restatement(ref):
    """variable density, compressive u: Omega from numpy.fft of u = m/rho, mode by mode."""
    nz, ny, nx = 8, 12, 16
    f = inputs.smooth_random_state(nx, ny, nz, seed=21)
    s = ref.RefSolver(nx, ny, nz, 0.01, 0.01, 1.0, 1e-3, flags=2)      # no mask: the state is the input itself
    s.set_fields(*f)
    d = s.diagnostics()
    kx = np.fft.fftfreq(nx, 1.0 / nx)[None, None, :]
    ky = np.fft.fftfreq(ny, 1.0 / ny)[None, :, None]
    kz = np.fft.fftfreq(nz, 1.0 / nz)[:, None, None]
    N = nx * ny * nz

    def curl2(v):
        vh = [np.fft.fftn(c) for c in v]
        w = [ky * vh[2] - kz * vh[1], kz * vh[0] - kx * vh[2], kx * vh[1] - ky * vh[0]]
        return sum(np.sum(np.abs(c) ** 2) for c in w) / N ** 2

    u2 = sum(np.mean(c ** 2) for c in f[1:4])
    b2 = sum(np.mean(c ** 2) for c in f[4:7])
    en, cu = curl2(f[1:4]), curl2(f[4:7])
    assert abs(d["u2"] - u2) <= 1e-13 * u2
    assert abs(d["enstrophy"] - en) <= 1e-12 * en and abs(d["current2"] - cu) <= 1e-12 * cu
    assert abs(d["rayleigh_q"] - (en + 0.5 * cu) / (u2 + 0.5 * b2)) <= 1e-12


def test_spectra_are_refused_off_the_two_pi_box(ref):
    s = ref.RefSolver(8, 8, 8, 0.0, 0.0, 1.0, 1e-3)
    s.set_box(1.0, TWO_PI, TWO_PI)
    one = np.ones((8, 8, 8))
    s.set_fields(one, 0 * one, 0 * one, 0 * one, 0 * one, 0 * one, 0 * one)
    with pytest.raises(RuntimeError):
        s.diagnostics(4)
    assert s.diagnostics(0)["rc"] == 0
