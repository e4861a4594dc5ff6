"""GPU FFT entry points (mhd_fft_r2c / mhd_fft_c2r, BASELINE config 5) against the oracle's FFT,
element by element, for every supported length on every axis, plus round trips at bench sizes."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

from paper_2402_05478_b200 import inputs

SIZES = [8, 12, 16, 24, 32, 48, 64, 96, 128, 192, 256, 384, 512, 768, 1024]


@pytest.fixture(scope="module")
def gpu():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2402_05478_b200 import mhd
    mhd.lib()
    return mhd


def check(gpu, ref, shape, batch, tol=2e-14, mode=0):
    import torch
    nz, ny, nx = shape
    rng = np.random.default_rng(nx * 7 + ny * 3 + nz)
    a = rng.uniform(-1, 1, size=(batch, nz, ny, nx))
    plan = gpu.FftPlan(nx, ny, nz, batch, mode=mode)
    da = torch.from_numpy(a).cuda()
    spec = plan.r2c(da)
    want = ref.fft_r2c(a)
    got = spec.cpu().numpy()
    assert np.linalg.norm(got - want) <= tol * np.linalg.norm(want), shape
    assert torch.equal(da.cpu(), torch.from_numpy(a))                 # input untouched
    back = plan.c2r(spec).cpu().numpy()
    assert np.linalg.norm(back - a) <= tol * np.linalg.norm(a), shape
    assert np.array_equal(spec.cpu().numpy(), got)                    # c2r must not write its input
    # c2r of an independent (oracle-made) spectrum of another field
    b = rng.uniform(-1, 1, size=(batch, nz, ny, nx))
    sb = ref.fft_r2c(b)
    back = plan.c2r(torch.from_numpy(sb).cuda()).cpu().numpy()
    assert np.linalg.norm(back - b) <= tol * np.linalg.norm(b), shape


@pytest.mark.parametrize("n", SIZES)
def test_every_length_on_every_axis(gpu, ref, n):
    check(gpu, ref, (8, 8, n), 3)
    check(gpu, ref, (8, n, 12), 2)
    check(gpu, ref, (n, 12, 8), 1)


@pytest.mark.parametrize("shape,batch", [((32, 32, 32), 7), ((1, 64, 64), 5), ((16, 24, 48), 7), ((1, 256, 256), 3),
                                         ((128, 128, 128), 7), ((24, 8, 8), 1), ((8, 8, 8), 1)])
def test_batched_3d_and_2d(gpu, ref, shape, batch):
    check(gpu, ref, shape, batch)


@pytest.mark.parametrize("shape,batch", [((8, 512, 512), 3), ((12, 256, 256), 3), ((24, 64, 64), 1), ((8, 128, 128), 1),
                                         ((1, 512, 512), 1), ((48, 128, 128), 5)])
def test_plane_pipelined_xy_pass_against_the_oracle(gpu, ref, shape, batch):
    """MHD_FFT_PLANE_PIPELINE: square (x,y) planes of 64..512 through the persistent plane-pipelined kernel (x and y passes
    meet in an L2-resident ring, planefft_kernel.cu): plane counts that do not fill the last group, a single plane, more
    groups than ring slots; twice in a row (the ring and the counters are reused); other shapes are refused."""
    check(gpu, ref, shape, batch, mode=gpu.FFT_PLANE_PIPELINE)
    check(gpu, ref, shape, batch, mode=gpu.FFT_PLANE_PIPELINE)
    with pytest.raises(gpu.MhdError):
        gpu.FftPlan(32, 16, 8, 1, mode=gpu.FFT_PLANE_PIPELINE)
    # the ring is paid for only on request: a default-sized plan may not switch, one sized by mhd_fft_plane_workspace_bytes may
    plain = gpu.FftPlan(64, 64, 8, 1)
    with pytest.raises(gpu.MhdError, match="no ring"):
        plain.set_mode(gpu.FFT_PLANE_PIPELINE)
    ringed = gpu.FftPlan(64, 64, 8, 1, plane_workspace=True)
    ringed.set_mode(gpu.FFT_PLANE_PIPELINE)
    ringed.set_mode(gpu.FFT_THREE_SWEEP)


@pytest.mark.parametrize("n,mode", [(256, 0), (512, 0), (768, 0), (256, 1), (512, 1)])
def test_round_trip_at_bench_sizes(gpu, n, mode):
    """config 5 sizes the oracle cannot finish in seconds: round trip and Parseval hold at any size."""
    import torch
    batch = 7 if n <= 256 else 2
    a = torch.from_numpy(inputs.config5_batch(n, batch)).cuda()
    plan = gpu.FftPlan(n, n, n, batch, mode=mode)
    spec = plan.r2c(a)
    back = plan.c2r(spec)
    assert float(torch.linalg.norm(back - a) / torch.linalg.norm(a)) <= 1e-14
    w = torch.full((n // 2 + 1,), 2.0, dtype=torch.float64, device="cuda")
    w[0] = 1.0
    w[-1] = 1.0
    lhs = float((a * a).sum())
    rhs = float((w * (spec.real ** 2 + spec.imag ** 2)).sum()) / n ** 3
    assert abs(lhs - rhs) <= 1e-12 * lhs
    # sampled outputs against the DFT definition, one mode at a time
    x = 2 * np.pi * torch.arange(n, dtype=torch.float64, device="cuda") / n
    for (b, kz, ky, kx) in [(0, 0, 0, 0), (1, 3, n - 2, 5), (batch - 1, n // 2, 1, n // 2), (0, n - 1, n // 3, 17)]:
        ph = torch.exp(-1j * (kz * x)[:, None, None]) * torch.exp(-1j * (ky * x)[None, :, None]) * torch.exp(-1j * (kx * x)[None, None, :])
        want = complex((a[b] * ph).sum())
        got = complex(spec[b, kz, ky, kx])
        assert abs(got - want) <= 1e-9 * n ** 1.5, (b, kz, ky, kx)
