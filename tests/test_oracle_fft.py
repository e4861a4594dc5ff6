"""Pins for the oracle's FFT (SURVEY.md §8(c.4) pin 1): the DFT definition written out as a dense
matrix product (brute force), numpy.fft as an independent library routine, Parseval, round trip and
the closed-form transform of a single cosine.  None of these calls oracle code to make the
expected value."""
import numpy as np
import pytest

TWO_PI = 2 * np.pi


def dft_matrix(n, sign=-1):
    j = np.arange(n)
    return np.exp(sign * 1j * TWO_PI * np.outer(j, j) / n)


@pytest.mark.parametrize("n", [1, 2, 3, 4, 5, 6, 7, 8, 9, 12, 16, 24, 27, 32, 48, 64, 96, 128, 384])
@pytest.mark.parametrize("sign", [-1, 1])
def test_fft1d_matches_definition(ref, n, sign):
    rng = np.random.default_rng(n * 7 + sign)
    x = rng.standard_normal(n) + 1j * rng.standard_normal(n)
    want = dft_matrix(n, sign) @ x
    got = ref.fft1d(x, sign)
    assert np.linalg.norm(got - want) <= 1e-13 * max(1.0, np.linalg.norm(want))


def brute_r2c(a):
    """O(N^6)-equivalent definition: f^(kz,ky,kx) = sum_xyz f exp(-i k.x), kept for kx <= nx/2."""
    nz, ny, nx = a.shape
    Fz, Fy, Fx = dft_matrix(nz), dft_matrix(ny), dft_matrix(nx)[: nx // 2 + 1]
    return np.einsum("az,by,cx,zyx->abc", Fz, Fy, Fx, a, optimize=False if a.size <= 512 else True)


@pytest.mark.parametrize("shape", [(8, 8, 8), (6, 6, 6), (12, 6, 4), (1, 8, 8), (4, 12, 24)])
def test_r2c_matches_brute_force_dft(ref, shape):
    rng = np.random.default_rng(sum(shape))
    a = rng.uniform(-1, 1, size=shape)
    want = brute_r2c(a)
    got = ref.fft_r2c(a)
    assert got.shape == want.shape
    assert np.linalg.norm(got - want) <= 1e-13 * np.linalg.norm(want)


@pytest.mark.parametrize("shape", [(16, 16, 16), (8, 16, 32), (24, 24, 24), (1, 64, 64), (32, 32, 32), (12, 48, 96)])
def test_r2c_c2r_match_numpy(ref, shape):
    rng = np.random.default_rng(11 + sum(shape))
    a = rng.uniform(-1, 1, size=(2,) + shape)
    want = np.fft.rfftn(a, axes=(1, 2, 3))
    got = ref.fft_r2c(a)
    assert np.linalg.norm(got - want) <= 1e-13 * np.linalg.norm(want)
    back = ref.fft_c2r(got, shape[2])
    assert np.linalg.norm(back - a) <= 1e-13 * np.linalg.norm(a)
    # c2r of an independent spectrum (numpy's) equals numpy's inverse
    spec = np.fft.rfftn(rng.uniform(-1, 1, size=shape))
    assert np.allclose(ref.fft_c2r(spec, shape[2]), np.fft.irfftn(spec, s=shape, axes=(0, 1, 2)), rtol=0, atol=1e-13)


def test_parseval(ref):
    rng = np.random.default_rng(5)
    nz, ny, nx = 12, 16, 24
    a = rng.standard_normal((nz, ny, nx))
    A = ref.fft_r2c(a)
    w = np.full(nx // 2 + 1, 2.0)
    w[0] = 1.0
    w[-1] = 1.0
    lhs = np.sum(a * a)
    rhs = np.sum(w * np.abs(A) ** 2) / a.size
    assert abs(lhs - rhs) <= 1e-13 * lhs


@pytest.mark.parametrize("k,phi", [((1, 0, 0), 0.3), ((0, 2, 0), 1.1), ((0, 0, 3), 2.0), ((2, -1, 3), 0.7), ((1, 3, -2), 4.0)])
def test_single_cosine_closed_form(ref, k, phi):
    """FFT of cos(k.x + phi) is (N/2) e^{+i phi} at +k and (N/2) e^{-i phi} at -k, zero elsewhere."""
    n = 16
    x = TWO_PI * np.arange(n) / n
    Z, Y, X = np.meshgrid(x, x, x, indexing="ij")
    kx, ky, kz = k
    a = np.cos(kx * X + ky * Y + kz * Z + phi)
    A = ref.fft_r2c(a)
    want = np.zeros_like(A)
    N = n ** 3
    # half-spectrum holds kx >= 0 only
    if kx > 0:
        want[kz % n, ky % n, kx] = 0.5 * N * np.exp(1j * phi)
    elif kx == 0:
        want[kz % n, ky % n, 0] += 0.5 * N * np.exp(1j * phi)
        want[-kz % n, -ky % n, 0] += 0.5 * N * np.exp(-1j * phi)
    assert np.max(np.abs(A - want)) <= 1e-12 * N


def test_c2r_ignores_imaginary_part_of_self_conjugate_x_modes(ref):
    """Documented convention: the x inverse takes the real part of the Hermitian-extended
    row, so Im of the kx = 0 and kx = nx/2 entries of a 1-D row does not reach the output."""
    n = 8
    rng = np.random.default_rng(3)
    spec = np.fft.rfftn(rng.standard_normal((1, 1, n)))
    base = ref.fft_c2r(spec, n)
    spec2 = spec.copy()
    spec2[0, 0, 0] += 0.5j
    spec2[0, 0, n // 2] -= 0.25j
    assert np.array_equal(ref.fft_c2r(spec2, n), base)
