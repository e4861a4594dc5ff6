"""CPU-side checks of the C-ABI boundary: the CUDA library builds for sm_100a, loads without a GPU,
exports every function include/mhd.h declares, and rejects bad arguments before touching CUDA."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2402_05478_b200 import build, mhd
    build.build()
    return mhd.lib()


def declared_functions():
    src = open(os.path.join(ROOT, "include", "mhd.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(mhd_[a-z0-9_]+)\s*\(", src)))


def test_header_declares_the_north_star_calls():
    names = declared_functions()
    for need in ("mhd_create", "mhd_set_fields", "mhd_step", "mhd_get_fields", "mhd_diagnostics", "mhd_destroy",
                 "mhd_fft_r2c", "mhd_fft_c2r"):
        assert need in names


def test_library_exports_every_declared_symbol(lib):
    from paper_2402_05478_b200 import mhd
    names = declared_functions()
    assert len(names) >= 17
    for n in names:
        assert hasattr(lib, n), n
    assert sorted(mhd.EXPORTS) == names


def test_library_is_sm100a_only():
    import subprocess
    from paper_2402_05478_b200 import mhd
    out = subprocess.run(["cuobjdump", "-lelf", mhd.LIB_PATH], capture_output=True, text=True).stdout
    archs = set(re.findall(r"sm_(\d+a?)", out))
    assert archs == {"100a"}, out


def test_workspace_bytes_and_size_validation(lib):
    w = lib.mhd_workspace_bytes(32, 32, 32, 0, 0)
    assert 1_000_000 < w < 64_000_000
    assert lib.mhd_workspace_bytes(32, 32, 32, 1, 0) > w                 # RK4 keeps one more state copy
    assert lib.mhd_workspace_bytes(256, 256, 1, 0, 1) > 0                # 2-D
    assert lib.mhd_workspace_bytes(30, 32, 32, 0, 0) == 0                # unsupported length
    assert lib.mhd_workspace_bytes(32, 32, 32, 7, 0) == 0                # unknown integrator
    w512 = lib.mhd_workspace_bytes(512, 512, 512, 0, 0)
    assert 20e9 < w512 < 60e9                                            # fits one B200 (180 GB) many times over
    assert lib.mhd_fft_workspace_bytes(768, 768, 768, 7) < 30e9
    assert lib.mhd_fft_workspace_bytes(100, 64, 64, 7) == 0


def test_bad_arguments_are_rejected_before_any_cuda_call(lib):
    from paper_2402_05478_b200 import mhd
    h = C.c_void_p()
    assert lib.mhd_create(C.byref(h), 32, 32, 32, 0.01, 0.01, 1.0, 1e-3, 0, 0, None, 0, None) == mhd.EINVAL
    assert lib.mhd_create(C.byref(h), 32, 32, 32, 0.01, 0.01, 1.0, -1.0, 0, 0, C.c_void_p(256), 1 << 40, None) == mhd.EINVAL
    assert lib.mhd_create(C.byref(h), 33, 32, 32, 0.01, 0.01, 1.0, 1e-3, 0, 0, C.c_void_p(256), 1 << 40, None) == mhd.EINVAL
    assert lib.mhd_create(C.byref(h), 32, 32, 32, 0.01, 0.01, 1.0, 1e-3, 0, 0, C.c_void_p(260), 1 << 40, None) == mhd.EINVAL  # misaligned
    assert lib.mhd_create(None, 32, 32, 32, 0.01, 0.01, 1.0, 1e-3, 0, 0, None, 0, None) == mhd.EINVAL
    assert not h.value
    assert lib.mhd_step(None, 1) == mhd.EINVAL
    assert lib.mhd_fft_r2c(None, None, None) == mhd.EINVAL
    assert lib.mhd_strerror(mhd.ESTATE).decode().startswith("call out of order")
    assert lib.mhd_last_error(None) == b""
    lib.mhd_destroy(None)
    lib.mhd_fft_plan_destroy(None)


def test_binding_fails_loudly_without_a_gpu():
    import torch
    from paper_2402_05478_b200 import mhd
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        mhd.Solver(32, 32, 32, 0.01, 0.01, 1.0, 1e-3)


def test_product_package_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_2402_05478_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle", text, flags=re.M), f
                assert "mhd_ref" not in text and "oracle/" not in text and "oracle." not in text, f


def test_library_has_no_hidden_dispatch_and_no_per_process_device_state():
    """The ABI is the only way to choose an execution plan (mhd_create flags): no translation unit reads the environment,
    and kernel attributes / SM counts are cached per DEVICE (DeviceOnce keyed by cudaGetDevice), never in a per-process
    static, so two contexts on two GPUs of one process cannot share a launch configuration by accident."""
    csrc = os.path.join(ROOT, "paper_2402_05478_b200", "csrc")
    for f in os.listdir(csrc):
        text = open(os.path.join(csrc, f)).read()
        assert "getenv" not in text, f
        assert not re.search(r"static\s+(int\s+sms|bool\s+attr_done)", text), f
    internal = open(os.path.join(csrc, "mhd_internal.h")).read()
    assert "struct DeviceOnce" in internal and "kMaxDevices" in internal
    for f in ("fft_kernels.cu", "xfused_kernel.cu", "planefft_kernel.cu"):
        text = open(os.path.join(csrc, f)).read()
        assert text.count("cudaFuncSetAttribute") > 0 and "once.done[dev]" in text, f


def test_peaks_probe_rejects_bad_arguments(lib):
    from paper_2402_05478_b200 import mhd
    f, s = C.c_double(), C.c_double()
    assert lib.mhd_measure_peaks(None, 1 << 23, None, C.byref(f), C.byref(s)) == mhd.EINVAL
    assert lib.mhd_measure_peaks(C.c_void_p(256), 16, None, C.byref(f), C.byref(s)) == mhd.EINVAL
    assert lib.mhd_measure_exchange(None, 1 << 23, None, 192, 1, C.byref(s)) == mhd.EINVAL
    assert lib.mhd_measure_exchange(C.c_void_p(256), 1 << 23, None, 100, 1, C.byref(s)) == mhd.EINVAL     # not a multiple of 64
    assert lib.mhd_measure_exchange(C.c_void_p(256), 1 << 23, None, 320, 1, C.byref(s)) == mhd.EINVAL
    assert lib.mhd_measure_exchange(C.c_void_p(256), 1 << 23, None, 192, 4, C.byref(s)) == mhd.EINVAL     # no such exchange mode
    assert lib.mhd_fft_last_error(None) == b""
    assert lib.mhd_fft_plan_set_mode(None, 0) == mhd.EINVAL
    # the plane pipeline's ring + counters are paid for only by a plan that asks for them, and only exist for square planes of 64..512
    plain = lib.mhd_fft_workspace_bytes(256, 256, 8, 1)
    assert 16 * 129 * 256 * 8 <= plain < 16 * 129 * 256 * 8 + 16 * 256 * 3 + 4096
    ring = lib.mhd_fft_plane_workspace_bytes(256, 256, 8, 1) - plain
    assert 15e6 < ring < 30e6                        # 5 slots of about 4 MB
    assert lib.mhd_fft_plane_workspace_bytes(512, 256, 8, 1) == 0 and lib.mhd_fft_plane_workspace_bytes(32, 32, 8, 1) == 0
    assert lib.mhd_fft_plane_workspace_bytes(100, 100, 8, 1) == 0
