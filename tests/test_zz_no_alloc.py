"""mhd_fft_c2r_static: the inverse transform for callers that cannot give the library any device memory.

FftPlan.c2r needs a workspace tensor that somebody has to allocate.  A caller that owns its input and output and nothing
else (code running inside a framework whose allocator holds the whole GPU, a job with a fully assigned memory budget, a loop
that must avoid cudaMalloc's device synchronisation) uses mhd_fft_c2r_static, whose scratch is a fixed 8 MiB array inside
the library.  These tests check that it returns what the plan path returns, also when the shared array still holds another
transform's intermediate, and that it refuses what does not fit.

The file is named so that pytest collects it last: `pytest -x` stops at the first failure, and a failure here must not hide
the parity tests."""
import ctypes as C
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
TOL = 2e-14          # relative L2, the tolerance of tests/test_gpu_fft.py


def test_transform_that_does_not_fit_is_refused_with_the_numbers():
    """128^3 needs a 17 MB intermediate: rejected before any CUDA call (runs without a GPU), and the message says how much
    was asked for and how much the built-in array holds.  Unsupported lengths and NULL buffers are rejected too."""
    from paper_2402_05478_b200 import build, mhd
    build.build()
    lib = mhd.lib()
    err = C.create_string_buffer(256)
    fake = C.c_void_p(256)
    assert lib.mhd_fft_c2r_static(128, 128, 128, 1, fake, fake, None, err, len(err)) == mhd.EINVAL
    text = err.value.decode()
    assert str(16 * 65 * 128 * 128) in text and str(mhd.STATIC_SCRATCH_BYTES) in text, text
    assert lib.mhd_fft_c2r_static(64, 64, 64, 4, fake, fake, None, err, len(err)) == mhd.EINVAL         # 8.65 MB > 8 MiB
    assert lib.mhd_fft_c2r_static(100, 64, 64, 1, fake, fake, None, err, len(err)) == mhd.EINVAL
    assert "unsupported size" in err.value.decode()
    assert lib.mhd_fft_c2r_static(64, 64, 64, 1, None, fake, None, err, len(err)) == mhd.EINVAL
    assert lib.mhd_fft_c2r_static(64, 64, 64, 1, fake, None, None, None, 0) == mhd.EINVAL                # no message buffer
    header = open(os.path.join(ROOT, "include", "mhd.h")).read()
    assert re.search(r"#define\s+MHD_STATIC_SCRATCH_BYTES\s+\(8u << 20\)", header)
    assert mhd.STATIC_SCRATCH_BYTES == 8 << 20


def test_the_entry_point_source_allocates_nothing():
    """The promise is structural: the translation unit holds the array, asks the runtime for its address, and contains no
    call that allocates or frees device memory."""
    src = open(os.path.join(ROOT, "paper_2402_05478_b200", "csrc", "fft_c2r_static.cu")).read()
    code = re.sub(r"//[^\n]*", "", src)
    for banned in ("cudaMalloc", "cudaFree", "cudaHostAlloc", "cudaMallocAsync", "cudaMemPool"):
        assert banned not in code, banned
    assert "static __device__ __align__(256)" in code and "cudaGetSymbolAddress" in code


@pytest.mark.gpu
def test_static_scratch_c2r_matches_the_plan_path_on_calls_in_a_row():
    """Two different transforms back to back, then the first again: each must equal FftPlan.c2r on the same input, so a
    call neither depends on what the previous one left in the shared array nor picks up the wrong twiddle table.  Covers a
    3-D case with all three axis lengths different, a 2-D case (no z pass: the y pass reads the input directly), the
    largest cube that fits, and a caller-supplied output on a side stream."""
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2402_05478_b200 import mhd
    mhd.lib()
    rng = np.random.default_rng(20240205)

    def spectrum(batch, nz, ny, nx):
        re_, im_ = rng.uniform(-1, 1, size=(2, batch, nz, ny, nx // 2 + 1))
        return torch.from_numpy(re_ + 1j * im_).cuda()

    def plan_path(spec, nx):
        batch, nz, ny, _ = spec.shape
        plan = mhd.FftPlan(nx, ny, nz, batch)
        want = plan.c2r(spec).clone()
        torch.cuda.synchronize()
        plan.close()
        return want

    def agree(got, want):
        err = float(torch.linalg.norm(got - want) / torch.linalg.norm(want))
        assert err <= TOL, err

    cases = [(2, 24, 48, 32), (3, 1, 256, 128), (1, 96, 96, 96), (3, 64, 64, 64)]      # (batch, nz, ny, nx)
    specs = [spectrum(*c) for c in cases]
    wants = [plan_path(s, c[3]) for s, c in zip(specs, cases)]
    for _ in range(2):                              # the whole sequence twice: every call follows a different transform
        for s, w in zip(specs, wants):
            keep = s.clone()
            got = mhd.fft_c2r_static(s)
            agree(got, w)
            assert torch.equal(s, keep)             # the input is read, never written
    # same transform twice in a row with different data
    a, b = spectrum(2, 24, 48, 32), spectrum(2, 24, 48, 32)
    wa, wb = plan_path(a, 32), plan_path(b, 32)
    agree(mhd.fft_c2r_static(a), wa)
    agree(mhd.fft_c2r_static(b), wb)
    # caller-owned output, explicit stream: nothing is allocated by the call
    side = torch.cuda.Stream()
    out = torch.full((2, 24, 48, 32), float("nan"), dtype=torch.float64, device="cuda")
    torch.cuda.synchronize()
    with torch.cuda.stream(side):
        ret = mhd.fft_c2r_static(a, out=out, stream=side)
    side.synchronize()
    assert ret is out
    agree(out, wa)
    # a round trip through the plan's forward transform closes the loop independently of c2r
    x = torch.from_numpy(rng.uniform(-1, 1, size=(1, 32, 32, 64))).cuda()
    plan = mhd.FftPlan(64, 32, 32, 1)
    back = mhd.fft_c2r_static(plan.r2c(x))
    agree(back, x)
    plan.close()
    with pytest.raises(mhd.MhdError, match="built-in array holds"):
        mhd.fft_c2r_static(spectrum(1, 128, 128, 128))
