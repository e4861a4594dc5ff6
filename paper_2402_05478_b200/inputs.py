"""Seeded synthetic inputs for the BASELINE.json configs (SURVEY.md §8(d) recipes).

This module is the ONLY code shared by the CUDA path and the CPU checker (oracle).  It holds
none of the method's arithmetic: it only writes down initial conditions (closed
forms from PAPER.md and seeded random-phase Fourier sums) as plain numpy arrays
that are then handed, identically, to both sides.  numpy's FFT is used here for
input synthesis only (config 4); it never appears on the product path.

Array convention everywhere: shape (nz, ny, nx), C order, x fastest, float64,
grid x_j = 2*pi*j/n on the box [0, 2*pi)^3.

Citations: ABC flow PAPER.md:277-281 (eq. 11); Orszag-Tang flow PAPER.md:223
(eq. 9); KH shear profile and perturbation PAPER.md:163-170 (eqs 6-7); Table I
workload shape (512^3, 100 iterations) PAPER.md:61-68.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

TWO_PI = 2.0 * np.pi


@dataclass
class Config:
    """One BASELINE.json config: grid, parameters, and the seeded fields."""

    name: str
    nx: int
    ny: int
    nz: int
    nu: float
    eta: float
    cs: float
    dt: float
    steps: int
    hydro: bool = False
    seed: int = 0
    fields: dict = field(default_factory=dict)  # rho, ux, uy, uz, bx, by, bz

    @property
    def shape(self):
        return (self.nz, self.ny, self.nx)

    def arrays(self):
        """The seven arrays in ABI order (rho, ux, uy, uz, bx, by, bz)."""
        return [self.fields[k] for k in ("rho", "ux", "uy", "uz", "bx", "by", "bz")]


def grid(nx: int, ny: int, nz: int):
    """Broadcastable coordinate arrays X, Y, Z of shapes (1,1,nx), (1,ny,1), (nz,1,1)."""
    x = (TWO_PI * np.arange(nx) / nx).reshape(1, 1, nx)
    y = (TWO_PI * np.arange(ny) / ny).reshape(1, ny, 1)
    z = (TWO_PI * np.arange(nz) / nz).reshape(nz, 1, 1)
    return x, y, z


def half_space_modes(kmax: float):
    """Independent integer wavevectors with 0 < |k| <= kmax, one per +-k pair.

    Enumerated over {kx>0} U {kx=0, ky>0} U {kx=ky=0, kz>0} in lexicographic
    (kz, ky, kx) order.  Returns a list of (kx, ky, kz).
    """
    m = int(np.floor(kmax))
    out = []
    for kz in range(-m, m + 1):
        for ky in range(-m, m + 1):
            for kx in range(-m, m + 1):
                k2 = kx * kx + ky * ky + kz * kz
                if k2 == 0 or k2 > kmax * kmax:
                    continue
                if kx > 0 or (kx == 0 and ky > 0) or (kx == 0 and ky == 0 and kz > 0):
                    out.append((kx, ky, kz))
    return out


def _phase(kvec, x, y, z):
    kx, ky, kz = kvec
    return kx * x + ky * y + kz * z


def random_phase_scalar(nx, ny, nz, kmax, amp, rng):
    """sum_k amp*cos(k.x + phi_k) over half_space_modes(kmax); one uniform phase per mode."""
    x, y, z = grid(nx, ny, nz)
    f = np.zeros((nz, ny, nx))
    for kvec in half_space_modes(kmax):
        phi = rng.uniform(0.0, TWO_PI)
        f = f + amp * np.cos(_phase(kvec, x, y, z) + phi)
    return f


def random_phase_solenoidal(nx, ny, nz, kmax, rms, rng):
    """Solenoidal random-phase vector field on modes 0<|k|<=kmax, rescaled to sqrt(<|v|^2>) = rms.

    v = sum_k Re[(I - kk/k^2) c_k exp(i k.x)], c_k = (e^{i phi_1}, e^{i phi_2}, e^{i phi_3}).
    The projection makes k.v_k = 0 mode by mode, so div v = 0 analytically.
    """
    x, y, z = grid(nx, ny, nz)
    v = [np.zeros((nz, ny, nx)) for _ in range(3)]
    for kvec in half_space_modes(kmax):
        k = np.array(kvec, dtype=float)
        c = np.exp(1j * rng.uniform(0.0, TWO_PI, size=3))
        c = c - k * (k @ c) / (k @ k)
        e = np.exp(1j * _phase(kvec, x, y, z))
        for i in range(3):
            v[i] = v[i] + (c[i] * e).real
    cur = np.sqrt(np.mean(v[0] ** 2 + v[1] ** 2 + v[2] ** 2))
    return [vi * (rms / cur) for vi in v]


def abc_flow(nx, ny, nz, A=1.0, B=1.0, C=1.0, k0=1.0, u0=1.0):
    """Arnold-Beltrami-Childress flow, PAPER.md:277-281 (eq. 11)."""
    x, y, z = grid(nx, ny, nz)
    one = np.ones((nz, ny, nx))
    ux = u0 * (A * np.sin(k0 * z) + C * np.cos(k0 * y)) * one
    uy = u0 * (B * np.sin(k0 * x) + A * np.cos(k0 * z)) * one
    uz = u0 * (C * np.sin(k0 * y) + B * np.cos(k0 * x)) * one
    return [ux, uy, uz]


def spectrum_solenoidal(nx, ny, nz, kcut, k_peak, rms, rng):
    """Random-phase solenoidal field with E(k) ~ k^4 exp(-2 (k/k_peak)^2) on 0<|k|<=kcut.

    Per-mode amplitude^2 ~ E(|k|)/(4 pi |k|^2); complex random-phase vector projected with
    (I - kk/k^2); synthesised with numpy's inverse real FFT (input generation only);
    rescaled to sqrt(<|v|^2>) = rms.  (SURVEY.md §8(d) config 4.)
    """
    nxh = nx // 2 + 1
    kx = np.arange(nxh, dtype=float).reshape(1, 1, nxh)
    ky = np.fft.fftfreq(ny, 1.0 / ny).reshape(1, ny, 1)
    kz = np.fft.fftfreq(nz, 1.0 / nz).reshape(nz, 1, 1)
    k2 = kx * kx + ky * ky + kz * kz
    kk = np.sqrt(k2)
    sel = (k2 > 0) & (kk <= kcut)
    safe = np.where(k2 > 0, k2, 1.0)
    amp = np.where(sel, np.sqrt(kk ** 4 * np.exp(-2.0 * (kk / k_peak) ** 2) / (4.0 * np.pi * safe)), 0.0)
    c = [amp * np.exp(1j * rng.uniform(0.0, TWO_PI, size=(nz, ny, nxh))) for _ in range(3)]
    kdotc = (kx * c[0] + ky * c[1] + kz * c[2]) / safe
    kvec = (kx, ky, kz)
    v = []
    for i in range(3):
        ci = c[i] - kvec[i] * kdotc
        v.append(np.fft.irfftn(ci, s=(nz, ny, nx), axes=(0, 1, 2)))
    cur = np.sqrt(np.mean(v[0] ** 2 + v[1] ** 2 + v[2] ** 2))
    return [np.ascontiguousarray(vi * (rms / cur)) for vi in v]


# --------------------------------------------------------------------------------------
# The five BASELINE.json configs
# --------------------------------------------------------------------------------------

def config1(n: int = 32) -> Config:
    """3D compressible MHD, 32^3: rho = 1 + 0.01-amplitude modes |k|<=2, ABC velocity, B solenoidal rms 0.1."""
    rng = np.random.default_rng(1001)
    rho = 1.0 + random_phase_scalar(n, n, n, 2.0, 0.01, rng)
    u = abc_flow(n, n, n)
    b = random_phase_solenoidal(n, n, n, 2.0, 0.1, rng)
    c = Config("config1_mhd32", n, n, n, nu=1e-2, eta=1e-2, cs=1.0, dt=1e-3, steps=20, seed=1001)
    c.fields = dict(rho=rho, ux=u[0], uy=u[1], uz=u[2], bx=b[0], by=b[1], bz=b[2])
    return c


def config2(n: int = 256, steps: int = 2000) -> Config:
    """2D hydrodynamic Kelvin-Helmholtz, n^2 x 1 (eqs 6-7 profile family on the 2*pi box)."""
    rng = np.random.default_rng(1002)
    a = 0.05
    sigma = 4.0 * a
    x, y, z = grid(n, n, 1)
    one = np.ones((1, n, n))
    ux = (np.tanh((y - np.pi / 2) / a) - np.tanh((y - 3 * np.pi / 2) / a) - 1.0) * one
    env = np.exp(-((y - np.pi / 2) ** 2) / sigma ** 2) + np.exp(-((y - 3 * np.pi / 2) ** 2) / sigma ** 2)
    uy = np.zeros((1, n, n))
    for kx in range(1, 5):
        phi = rng.uniform(0.0, TWO_PI)
        uy = uy + 1e-3 * np.sin(kx * x + phi) * env
    zero = np.zeros((1, n, n))
    c = Config("config2_kh256", n, n, 1, nu=1e-4, eta=0.0, cs=2.0, dt=1e-3, steps=steps, hydro=True, seed=1002)
    c.fields = dict(rho=one.copy(), ux=ux, uy=uy, uz=zero.copy(), bx=zero.copy(), by=zero.copy(), bz=zero.copy())
    return c


def config3(n: int = 128, steps: int = 500) -> Config:
    """3D MHD Orszag-Tang-type vortex with a seeded z-modulation (eq. 9 family)."""
    rng = np.random.default_rng(1003)
    phi = rng.uniform(0.0, TWO_PI)
    x, y, z = grid(n, n, n)
    one = np.ones((n, n, n))
    mod = 1.0 + 0.01 * np.cos(z + phi)
    ux = -np.sin(y) * mod * one
    uy = np.sin(x) * mod * one
    bx = -np.sin(y) * one
    by = np.sin(2 * x) * one
    zero = np.zeros((n, n, n))
    c = Config("config3_ot128", n, n, n, nu=5e-3, eta=5e-3, cs=1.0, dt=5e-4, steps=steps, seed=1003)
    c.fields = dict(rho=one.copy(), ux=ux, uy=uy, uz=zero.copy(), bx=bx, by=by, bz=zero.copy())
    return c


def config4(n: int = 512, steps: int = 100) -> Config:
    """3D MHD decaying turbulence: E(k) ~ k^4 exp(-2 (k/4)^2), u_rms = 1, B_rms = 0.5, rho = 1."""
    rng = np.random.default_rng(1004)
    kcut = min(32.0, (n - 1) // 3)  # stay inside the 2/3 mask on small test grids
    u = spectrum_solenoidal(n, n, n, kcut, 4.0, 1.0, rng)
    b = spectrum_solenoidal(n, n, n, kcut, 4.0, 0.5, rng)
    c = Config(f"config4_turb{n}", n, n, n, nu=1e-3, eta=1e-3, cs=1.0, dt=2e-4, steps=steps, seed=1004)
    c.fields = dict(rho=np.ones((n, n, n)), ux=u[0], uy=u[1], uz=u[2], bx=b[0], by=b[1], bz=b[2])
    return c


def config5_batch(n: int, batch: int = 7, nz: int | None = None) -> np.ndarray:
    """Batched FFT sweep input: uniform[-1,1) reals, shape (batch, nz, n, n)."""
    rng = np.random.default_rng(1005)
    nz = n if nz is None else nz
    return rng.uniform(-1.0, 1.0, size=(batch, nz, n, n))


def smooth_random_state(nx, ny, nz, seed, kmax=2.0, hydro=False):
    """A small smooth MHD state for unit tests (config-1 recipe on any grid, any seed)."""
    rng = np.random.default_rng(seed)
    rho = 1.0 + random_phase_scalar(nx, ny, nz, kmax, 0.05, rng)
    u = random_phase_solenoidal(nx, ny, nz, kmax, 0.5, rng)
    u[0] = u[0] + 0.1 * random_phase_scalar(nx, ny, nz, kmax, 1.0, rng)  # make u compressive too
    if hydro:
        b = [np.zeros((nz, ny, nx)) for _ in range(3)]
    else:
        b = random_phase_solenoidal(nx, ny, nz, kmax, 0.3, rng)
    return [rho, u[0], u[1], u[2], b[0], b[1], b[2]]


def full_band_state(nx, ny, nz, seed, hydro=False):
    """White noise under a smooth envelope: O(1) content in EVERY Fourier mode up to the Nyquist index, so that the
    modes next to the 2/3-rule cut (index 170/171 on a 512 axis) and every pruned-index path carry full-size data.
    rho = 1 + 0.3 e(x) w(x) stays in [0.7, 1.3] on the grid (w uniform in [-1,1), e in [0.25, 1] a k = 1 cosine product);
    u and B are e(x) times independent uniform noise of amplitude 1 and 0.5.  Test input only (not a paper workload)."""
    rng = np.random.default_rng(seed)
    x, y, z = grid(nx, ny, nz)
    env = 0.25 + 0.75 * (0.5 + 0.5 * np.cos(x + 0.3)) * (0.5 + 0.5 * np.cos(y - 1.1)) * (0.5 + 0.5 * np.cos(z + 2.0))
    shape = (nz, ny, nx)
    rho = 1.0 + 0.3 * env * rng.uniform(-1.0, 1.0, size=shape)
    u = [env * rng.uniform(-1.0, 1.0, size=shape) for _ in range(3)]
    if hydro:
        b = [np.zeros(shape) for _ in range(3)]
    else:
        b = [0.5 * env * rng.uniform(-1.0, 1.0, size=shape) for _ in range(3)]
    return [np.ascontiguousarray(a) for a in [rho] + u + b]
