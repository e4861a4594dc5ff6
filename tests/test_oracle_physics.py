"""Pins for the oracle's step (SURVEY.md §8(c.4) pins 2-13).  Every expected value here comes from
mathematics written in this file (closed forms, small recurrences, a numpy.fft restatement), never
from oracle code.  Citations: eqs (1)-(4) PAPER.md:39-47; 2/3 rule and Adams-Bashforth PAPER.md:78."""
import numpy as np
import pytest

from paper_2402_05478_b200 import inputs

TWO_PI = 2 * np.pi


def coords(n):
    x = TWO_PI * np.arange(n) / n
    Z, Y, X = np.meshgrid(x, x, x, indexing="ij")
    return X, Y, Z


def ab2_scalar(z, nsteps):
    """y' = lambda*y with z = lambda*dt under Euler-started AB2; returns y_n / y_0."""
    y_prev, y = 1.0, 1.0 + z
    for _ in range(nsteps - 1):
        y_prev, y = y, y + z * (1.5 * y - 0.5 * y_prev)
    return y if nsteps >= 1 else 1.0


# ---------------------------------------------------------------- pin 2: mask and derivative
@pytest.mark.parametrize("n,kmax", [(32, 10), (48, 15), (16, 5), (24, 7)])
def test_mask_is_two_thirds_rule_per_axis(ref, n, kmax):
    s = ref.RefSolver(n, n, n, 0.0, 0.0, 1.0, 1e-3)
    m = s.mask()
    k = np.fft.fftfreq(n, 1.0 / n)
    want = (np.abs(k)[:, None, None] <= kmax) & (np.abs(k)[None, :, None] <= kmax) & (np.arange(n // 2 + 1)[None, None, :] <= kmax)
    assert np.array_equal(m, want)
    w = np.full(n // 2 + 1, 2)
    w[0] = 1
    w[-1] = 1
    assert int(np.sum(m * w)) == (2 * kmax + 1) ** 3      # 9261 at 32^3 (SURVEY.md §8(c.4) pin 2)
    assert 3 * kmax < n <= 3 * (kmax + 1)


def test_mask_2d_and_no_dealias(ref):
    s = ref.RefSolver(32, 32, 1, 0.0, 0.0, 1.0, 1e-3)
    assert s.mask().sum() == 11 * 21                     # kz = 0 always passes
    s = ref.RefSolver(16, 16, 16, 0.0, 0.0, 1.0, 1e-3, flags=ref.FLAG_NO_DEALIAS)
    assert s.mask().all()


@pytest.mark.parametrize("axis", [0, 1, 2])
def test_spectral_derivative_of_every_retained_mode(ref, axis):
    """continuity: R_rho = -div m.  m = sin(k x_axis) e_axis  =>  R_rho = -k cos(k x_axis) if |k|<=kmax else 0."""
    n, kmax = 24, 7
    X = coords(n)[axis]
    for k in range(1, n // 2):
        s = ref.RefSolver(n, n, n, 0.0, 0.0, 1.0, 1e-3)
        u = [np.zeros((n, n, n)) for _ in range(3)]
        u[axis] = np.sin(k * X)
        zero = np.zeros((n, n, n))
        s.set_fields(np.ones((n, n, n)), u[0], u[1], u[2], zero, zero, zero)
        R = s.rhs()
        got = np.fft.irfftn(R[0], s=(n, n, n), axes=(0, 1, 2))
        want = -k * np.cos(k * X) if k <= kmax else np.zeros_like(X)
        assert np.max(np.abs(got - want)) <= 1e-12 * k


# ---------------------------------------------------------------- pin 3: one RHS vs numpy.fft restatement
def numpy_rhs(fields, nu, eta, cs, hydro=False):
    """Independent restatement of eqs (1)-(4) with numpy.fft (shares nothing with oracle or product)."""
    rho, ux, uy, uz, bx, by, bz = fields
    nz, ny, nx = rho.shape
    kx = np.arange(nx // 2 + 1).reshape(1, 1, -1).astype(float)
    ky = np.fft.fftfreq(ny, 1.0 / ny).reshape(1, -1, 1)
    kz = np.fft.fftfreq(nz, 1.0 / nz).reshape(-1, 1, 1)
    M = (3 * np.abs(kx) < nx) & (3 * np.abs(ky) < ny) & (3 * np.abs(kz) < nz)
    F = lambda a: np.fft.rfftn(a, axes=(0, 1, 2))
    Fi = lambda a: np.fft.irfftn(a, s=(nz, ny, nx), axes=(0, 1, 2))
    S = [M * F(a) for a in (rho, rho * ux, rho * uy, rho * uz, bx, by, bz)]
    r, mx, my, mz, Bx, By, Bz = [Fi(a) for a in S]
    u = [mx / r, my / r, mz / r]
    m = [mx, my, mz]
    B = [Bx, By, Bz]
    K = [kx, ky, kz]
    k2 = kx ** 2 + ky ** 2 + kz ** 2
    b2 = Bx ** 2 + By ** 2 + Bz ** 2
    R = [-1j * (kx * S[1] + ky * S[2] + kz * S[3])]
    for i in range(3):
        acc = 0
        for j in range(3):
            T = m[i] * u[j] - B[i] * B[j] + (0.5 * b2 if i == j else 0.0)
            acc = acc - 1j * K[j] * F(T)
        R.append(M * (acc - 1j * K[i] * cs ** 2 * S[0] - nu * k2 * F(u[i])))
    E = [u[1] * B[2] - u[2] * B[1], u[2] * B[0] - u[0] * B[2], u[0] * B[1] - u[1] * B[0]]
    Eh = [F(e) for e in E]
    curl = [1j * (ky * Eh[2] - kz * Eh[1]), 1j * (kz * Eh[0] - kx * Eh[2]), 1j * (kx * Eh[1] - ky * Eh[0])]
    for i in range(3):
        R.append(np.zeros_like(S[0]) if hydro else M * curl[i] - eta * k2 * S[4 + i])
    return np.array(S), np.array(R)


@pytest.mark.parametrize("shape,hydro", [((16, 16, 16), False), ((8, 12, 24), False), ((1, 16, 16), False), ((16, 16, 16), True)])
def test_rhs_matches_numpy_restatement(ref, shape, hydro):
    nz, ny, nx = shape
    fields = inputs.smooth_random_state(nx, ny, nz, seed=42, kmax=3.0, hydro=hydro)
    nu, eta, cs = 0.03, 0.02, 1.3
    s = ref.RefSolver(nx, ny, nz, nu, eta, cs, 1e-3, flags=ref.FLAG_HYDRO if hydro else 0)
    s.set_fields(*fields)
    S_want, R_want = numpy_rhs(fields, nu, eta, cs, hydro)
    S_got = np.array([s.get_spectral(i) for i in range(7)])
    R_got = s.rhs()
    assert np.linalg.norm(S_got - S_want) <= 1e-13 * np.linalg.norm(S_want)
    for i in range(7):
        scale = max(np.linalg.norm(R_want[i]), 1e-30)
        assert np.linalg.norm(R_got[i] - R_want[i]) <= 1e-12 * scale + 1e-9 * (scale < 1e-20), i


# ---------------------------------------------------------------- pin 4: viscous shear wave, exact
@pytest.mark.parametrize("k,axis_u,axis_x", [(3, 1, 0), (2, 2, 1), (4, 0, 2)])
def test_shear_wave_decays_by_ab2_recurrence(ref, k, axis_u, axis_x):
    """rho=1, u = a sin(k x_j) e_i (i != j), B=0 is an exact solution: amplitude obeys y' = -nu k^2 y."""
    n, nu, dt, a, nsteps = 16, 0.05, 1e-2, 0.7, 25
    Xs = coords(n)
    u = [np.zeros((n, n, n)) for _ in range(3)]
    u[axis_u] = a * np.sin(k * Xs[axis_x])
    zero = np.zeros((n, n, n))
    s = ref.RefSolver(n, n, n, nu, 0.0, 1.0, dt)
    s.set_fields(np.ones((n, n, n)), u[0], u[1], u[2], zero, zero, zero)
    s.step(nsteps)
    out = s.get_fields()
    amp = ab2_scalar(-nu * k * k * dt, nsteps)
    assert np.max(np.abs(out[1 + axis_u] - amp * u[axis_u])) <= 1e-13
    assert np.max(np.abs(out[0] - 1.0)) <= 1e-13
    for i in range(3):
        if i != axis_u:
            assert np.max(np.abs(out[1 + i])) <= 1e-13
    # and the recurrence itself approximates exp(-nu k^2 t) to O(dt^2)
    assert abs(amp - np.exp(-nu * k * k * dt * nsteps)) <= 2.0 * (nu * k * k * dt) ** 2 * nsteps


# ---------------------------------------------------------------- pin 5: resistive decay of a force-free field
def test_force_free_field_decays_resistively(ref):
    """B = ABC field (curl B = k0 B, so J x B = 0), u = 0, rho = 1: B^ decays with z = -eta k0^2 dt; u stays 0."""
    n, eta, dt, nsteps = 16, 0.08, 1e-2, 20
    B0 = inputs.abc_flow(n, n, n, u0=0.4)
    zero = np.zeros((n, n, n))
    s = ref.RefSolver(n, n, n, 0.01, eta, 1.0, dt)
    s.set_fields(np.ones((n, n, n)), zero, zero, zero, *B0)
    s.step(nsteps)
    out = s.get_fields()
    amp = ab2_scalar(-eta * dt, nsteps)
    for i in range(3):
        assert np.max(np.abs(out[4 + i] - amp * B0[i])) <= 1e-13
        assert np.max(np.abs(out[1 + i])) <= 1e-14
    assert np.max(np.abs(out[0] - 1.0)) <= 1e-14


# ---------------------------------------------------------------- pin 6: sound wave and fast magnetosonic wave
def _phase_speed(ref, B0y, cs, k, n=32, eps=1e-6, dt=1e-3, nsteps=200):
    X, Y, Z = coords(n)
    vf = np.sqrt(cs ** 2 + B0y ** 2)
    rho = 1.0 + eps * np.cos(k * X)
    ux = eps * vf * np.cos(k * X)
    zero = np.zeros((n, n, n))
    by = B0y * (1.0 + eps * np.cos(k * X))
    s = ref.RefSolver(n, n, n, 0.0, 0.0, cs, dt)
    s.set_fields(rho, ux, zero, zero, zero, by, zero)
    s.step(nsteps)
    rho_hat = np.fft.rfftn(s.get_fields()[0])[0, 0, k]
    return -np.angle(rho_hat) / (k * dt * nsteps), vf


def test_sound_wave_speed(ref):
    got, want = _phase_speed(ref, 0.0, 1.5, 2)
    assert abs(got - want) <= 2e-5 * want


def test_fast_magnetosonic_wave_speed(ref):
    """pins the +B^2/2 magnetic-pressure term of eq. (2) and the compressive part of eq. (4)."""
    got, want = _phase_speed(ref, 0.8, 1.2, 3)
    assert abs(got - want) <= 2e-5 * want


# ---------------------------------------------------------------- pin 7: circularly polarised Alfven wave
@pytest.mark.parametrize("nu,eta", [(0.0, 0.0), (0.02, 0.05)])
def test_circularly_polarised_alfven_wave(ref, nu, eta):
    """Exact at any amplitude: per mode d/dt (v, b) = [[-nu k^2, i k B0], [i k B0, -eta k^2]] (v, b).
    A wrong sign in eq. (4) or in the -B_i B_j tension turns the rotation into exponential growth."""
    n, k, B0, b, dt, nsteps = 16, 2, 1.0, 0.5, 2e-3, 100
    X, Y, Z = coords(n)
    one, zero = np.ones((n, n, n)), np.zeros((n, n, n))
    s = ref.RefSolver(n, n, n, nu, eta, 1.0, dt)
    s.set_fields(one, zero, -b * np.cos(k * X), -b * np.sin(k * X), B0 * one, b * np.cos(k * X), b * np.sin(k * X))
    s.step(nsteps)
    out = s.get_fields()
    A = np.array([[-nu * k * k, 1j * k * B0], [1j * k * B0, -eta * k * k]])
    v_prev = np.array([-b, b], dtype=complex)
    v = v_prev + dt * (A @ v_prev)
    for _ in range(nsteps - 1):
        v_prev, v = v, v + dt * (1.5 * (A @ v) - 0.5 * (A @ v_prev))
    e = np.exp(1j * k * X)
    want = {2: (v[0] * e).real, 3: (v[0] * e).imag, 5: (v[1] * e).real, 6: (v[1] * e).imag}
    for idx, w in want.items():
        assert np.max(np.abs(out[idx] - w)) <= 1e-12, idx
    assert np.max(np.abs(out[0] - 1.0)) <= 1e-13 and np.max(np.abs(out[1])) <= 1e-13
    assert np.max(np.abs(out[4] - B0)) <= 1e-13
    if nu == 0.0 and eta == 0.0:   # (-b, b) is the eigenvector of eigenvalue -i k B0: pure rotation, to O(dt^2)
        assert abs(abs(v[1]) - b) <= 1e-5 and abs(np.angle(v[1] / b) + k * B0 * dt * nsteps) <= 1e-5
