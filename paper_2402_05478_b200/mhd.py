"""Thin ctypes binding of libmhd_b200.so (include/mhd.h).  Argument marshalling only: every step of
the path runs in the library's CUDA kernels.  PyTorch supplies device memory and the stream.

There is NO CPU fallback: importing is cheap, but any call raises if the CUDA library is missing.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libmhd_b200.so")

OK, EINVAL, ENOMEM, ECUDA, ESTATE, ENONFINITE = 0, -1, -2, -3, -4, -5
AB2, RK4 = 0, 1
FLAG_HYDRO, FLAG_NO_DEALIAS, FLAG_FORCING = 1, 2, 4
FLAG_UNFUSED_X, FLAG_NO_GRAPH = 8, 16
FFT_THREE_SWEEP, FFT_PLANE_PIPELINE = 0, 1
STATIC_SCRATCH_BYTES = 8 << 20          # MHD_STATIC_SCRATCH_BYTES: largest intermediate fft_c2r_static accepts

EXPORTS = [
    "mhd_workspace_bytes", "mhd_create", "mhd_destroy", "mhd_set_fields", "mhd_set_fields_host", "mhd_set_box",
    "mhd_set_forcing", "mhd_set_forcing_host", "mhd_step",
    "mhd_state_bytes", "mhd_get_state", "mhd_set_state",
    "mhd_get_fields", "mhd_get_fields_host", "mhd_diagnostics", "mhd_strerror", "mhd_last_error",
    "mhd_fft_workspace_bytes", "mhd_fft_plan_create", "mhd_fft_r2c", "mhd_fft_c2r", "mhd_fft_plan_destroy", "mhd_fft_last_error", "mhd_fft_plan_set_mode",
    "mhd_fft_plane_workspace_bytes",
    "mhd_fft_c2r_static",
    "mhd_launch_count", "mhd_profile_kernel_count", "mhd_profile_kernel_name", "mhd_profile_begin", "mhd_profile_end",
    "mhd_measure_peaks", "mhd_measure_exchange",
]


class Diag(C.Structure):
    _fields_ = [("step", C.c_longlong), ("time", C.c_double), ("ekin", C.c_double), ("emag", C.c_double),
                ("eiso", C.c_double), ("mass", C.c_double), ("mom", C.c_double * 3),
                ("bmean", C.c_double * 3), ("max_divb", C.c_double),
                ("enstrophy", C.c_double), ("current2", C.c_double), ("u2", C.c_double), ("rayleigh_q", C.c_double)]


class MhdError(RuntimeError):
    def __init__(self, code, where, detail=""):
        self.code = code
        msg = lib().mhd_strerror(code).decode() if _lib is not None else str(code)
        super().__init__(f"{where}: {msg} ({code})" + (f": {detail}" if detail else ""))


_lib = None
_vp = C.c_void_p


def lib():
    """Load the CUDA library; fail loudly if it has not been built (no fallback of any kind)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} is missing: run `python -m paper_2402_05478_b200.build` "
                              "(or __graft_entry__.build()); there is no CPU fallback")
        L = C.CDLL(LIB_PATH)
        L.mhd_workspace_bytes.restype = C.c_size_t
        L.mhd_workspace_bytes.argtypes = [C.c_int, C.c_int, C.c_int, C.c_int, C.c_uint]
        L.mhd_create.argtypes = [C.POINTER(_vp), C.c_int, C.c_int, C.c_int, C.c_double, C.c_double, C.c_double,
                                 C.c_double, C.c_int, C.c_uint, _vp, C.c_size_t, _vp]
        L.mhd_destroy.argtypes = [_vp]
        L.mhd_destroy.restype = None
        for name in ("mhd_set_fields", "mhd_set_fields_host", "mhd_get_fields", "mhd_get_fields_host"):
            getattr(L, name).argtypes = [_vp] * 8
        L.mhd_set_box.argtypes = [_vp, C.c_double, C.c_double, C.c_double]
        L.mhd_set_forcing.argtypes = [_vp] * 4
        L.mhd_set_forcing_host.argtypes = [_vp] * 4
        L.mhd_step.argtypes = [_vp, C.c_int]
        L.mhd_state_bytes.restype = C.c_size_t
        L.mhd_state_bytes.argtypes = [_vp]
        L.mhd_get_state.argtypes = [_vp, _vp, C.c_size_t]
        L.mhd_set_state.argtypes = [_vp, _vp, C.c_size_t]
        L.mhd_diagnostics.argtypes = [_vp, C.POINTER(Diag), _vp, _vp, C.c_int]
        L.mhd_strerror.restype = C.c_char_p
        L.mhd_strerror.argtypes = [C.c_int]
        L.mhd_last_error.restype = C.c_char_p
        L.mhd_last_error.argtypes = [_vp]
        L.mhd_fft_workspace_bytes.restype = C.c_size_t
        L.mhd_fft_workspace_bytes.argtypes = [C.c_int] * 4
        L.mhd_fft_plane_workspace_bytes.restype = C.c_size_t
        L.mhd_fft_plane_workspace_bytes.argtypes = [C.c_int] * 4
        L.mhd_fft_plan_create.argtypes = [C.POINTER(_vp), C.c_int, C.c_int, C.c_int, C.c_int, _vp, C.c_size_t, _vp]
        L.mhd_fft_r2c.argtypes = [_vp, _vp, _vp]
        L.mhd_fft_c2r.argtypes = [_vp, _vp, _vp]
        L.mhd_fft_plan_destroy.argtypes = [_vp]
        L.mhd_fft_plan_destroy.restype = None
        L.mhd_fft_plan_set_mode.argtypes = [_vp, C.c_int]
        L.mhd_fft_last_error.restype = C.c_char_p
        L.mhd_fft_last_error.argtypes = [_vp]
        L.mhd_fft_c2r_static.argtypes = [C.c_int, C.c_int, C.c_int, C.c_int, _vp, _vp, _vp, C.c_char_p, C.c_size_t]
        L.mhd_launch_count.restype = C.c_longlong
        L.mhd_profile_kernel_count.restype = C.c_int
        L.mhd_profile_kernel_name.restype = C.c_char_p
        L.mhd_profile_kernel_name.argtypes = [C.c_int]
        L.mhd_profile_begin.argtypes = [_vp]
        L.mhd_profile_end.argtypes = [_vp, C.POINTER(C.c_int), C.POINTER(C.c_double)]
        L.mhd_measure_peaks.argtypes = [_vp, C.c_size_t, _vp, C.POINTER(C.c_double), C.POINTER(C.c_double)]
        L.mhd_measure_exchange.argtypes = [_vp, C.c_size_t, _vp, C.c_int, C.c_int, C.POINTER(C.c_double)]
        _lib = L
    return _lib


def launch_count() -> int:
    return int(lib().mhd_launch_count())


def measure_peaks(device="cuda:0"):
    """(FP64 TFLOP/s, shared-memory GB/s) measured on `device` by the library's own probe kernels (mhd_measure_peaks)."""
    torch = _torch()
    dev = torch.device(device)
    with torch.cuda.device(dev):
        scratch = torch.empty(8 << 20, dtype=torch.uint8, device=dev)
        f, s = C.c_double(), C.c_double()
        torch.cuda.synchronize(dev)
        rc = lib().mhd_measure_peaks(_vp(scratch.data_ptr()), scratch.numel(), _vp(torch.cuda.current_stream(dev).cuda_stream),
                                     C.byref(f), C.byref(s))
    if rc != OK:
        raise MhdError(rc, "mhd_measure_peaks")
    return float(f.value), float(s.value)


def measure_exchange(dfma_per_exchange=192, device="cuda:0", barrier_mode=1):
    """shared-memory GB/s reached by the fused x pass's exchange pattern alone (mhd_measure_exchange)."""
    torch = _torch()
    dev = torch.device(device)
    with torch.cuda.device(dev):
        scratch = torch.empty(8 << 20, dtype=torch.uint8, device=dev)
        g = C.c_double()
        torch.cuda.synchronize(dev)
        rc = lib().mhd_measure_exchange(_vp(scratch.data_ptr()), scratch.numel(), _vp(torch.cuda.current_stream(dev).cuda_stream),
                                        int(dfma_per_exchange), int(barrier_mode), C.byref(g))
    if rc != OK:
        raise MhdError(rc, "mhd_measure_exchange")
    return float(g.value)


def _torch():
    import torch
    if not torch.cuda.is_available():
        raise RuntimeError("paper_2402_05478_b200 needs a CUDA device; there is no CPU fallback")
    return torch


def _stream_ptr(torch, stream, device):
    """The library enqueues on ONE stream.  By default the binding gives each object its own torch stream
    (CUDA graphs cannot be captured on the legacy default stream) and orders it against the caller's
    current stream around every call that consumes or produces caller tensors."""
    s = torch.cuda.Stream(device=device) if stream is None else stream
    return s, _vp(s.cuda_stream)


def _dev_ptr(t, n, name):
    import torch
    if t is None:
        return None
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float64 and t.is_contiguous() and t.numel() == n):
        raise ValueError(f"{name}: expected a contiguous CUDA float64 tensor with {n} elements")
    return _vp(t.data_ptr())


def _host_ptr(a, n, name, writable=False):
    """numpy array or CPU torch tensor (pinned or not) -> pointer; no copies are made."""
    if a is None:
        return None
    try:
        import torch
        if isinstance(a, torch.Tensor):
            if a.is_cuda or a.dtype != torch.float64 or not a.is_contiguous() or a.numel() != n:
                raise ValueError(f"{name}: expected a contiguous CPU float64 tensor with {n} elements")
            return _vp(a.data_ptr())
    except ImportError:
        pass
    if not (isinstance(a, np.ndarray) and a.dtype == np.float64 and a.flags.c_contiguous and a.size == n):
        raise ValueError(f"{name}: expected a C-contiguous float64 array with {n} elements")
    if writable and not a.flags.writeable:
        raise ValueError(f"{name}: array is read-only")
    return _vp(a.ctypes.data)


class Solver:
    """mhd_create / mhd_set_fields / mhd_step / mhd_get_fields / mhd_diagnostics on one GPU."""

    def __init__(self, nx, ny, nz, nu, eta, cs, dt, integrator=AB2, flags=0, stream=None, device="cuda:0"):
        torch = _torch()
        L = lib()
        self.nx, self.ny, self.nz = int(nx), int(ny), int(nz)
        self.shape = (self.nz, self.ny, self.nx)
        self.npts = self.nx * self.ny * self.nz
        self.flags = int(flags)
        self.hydro = bool(flags & FLAG_HYDRO)
        self.device = torch.device(device)
        nbytes = L.mhd_workspace_bytes(self.nx, self.ny, self.nz, int(integrator), self.flags)
        if nbytes == 0:
            raise MhdError(EINVAL, "mhd_workspace_bytes", f"unsupported size {nx}x{ny}x{nz}")
        self.workspace_bytes = int(nbytes)
        with torch.cuda.device(self.device):
            self._ws = torch.empty(self.workspace_bytes + 256, dtype=torch.uint8, device=self.device)
            off = (-self._ws.data_ptr()) % 256
            self._stream, sp = _stream_ptr(torch, stream, self.device)
            self._stream.wait_stream(torch.cuda.current_stream(self.device))   # workspace allocation
            self._h = _vp()
            rc = L.mhd_create(C.byref(self._h), self.nx, self.ny, self.nz, float(nu), float(eta), float(cs), float(dt),
                              int(integrator), self.flags, _vp(self._ws.data_ptr() + off), self.workspace_bytes, sp)
        if rc != OK:
            self._h = _vp()
            raise MhdError(rc, "mhd_create")

    @property
    def stream(self):
        return self._stream

    def _before(self):
        import torch
        self._stream.wait_stream(torch.cuda.current_stream(self.device))

    def _after(self):
        import torch
        torch.cuda.current_stream(self.device).wait_stream(self._stream)

    def profile_begin(self):
        self._check(lib().mhd_profile_begin(self._h), "mhd_profile_begin")

    def profile_end(self):
        """{kernel class: (launches, summed ms)} since profile_begin; synchronises."""
        L = lib()
        n = L.mhd_profile_kernel_count()
        counts = (C.c_int * n)()
        ms = (C.c_double * n)()
        self._check(L.mhd_profile_end(self._h, counts, ms), "mhd_profile_end")
        return {L.mhd_profile_kernel_name(i).decode(): (int(counts[i]), float(ms[i])) for i in range(n)}

    def _check(self, rc, where, allow=()):
        if rc != OK and rc not in allow:
            raise MhdError(rc, where, lib().mhd_last_error(self._h).decode())
        return rc

    def close(self):
        """mhd_step is asynchronous on the solver's own stream: wait for it before the context is destroyed and the
        workspace goes back to torch's caching allocator (which could hand it to another stream at once)."""
        if getattr(self, "_h", None):
            try:
                self._stream.synchronize()
            finally:
                lib().mhd_destroy(self._h)
                self._h = _vp()
        self._ws = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- device-resident fields (torch CUDA tensors) ----
    def set_fields(self, rho, ux, uy, uz, bx=None, by=None, bz=None):
        names = ("rho", "ux", "uy", "uz", "bx", "by", "bz")
        ptrs = [_dev_ptr(t, self.npts, n) for t, n in zip((rho, ux, uy, uz, bx, by, bz), names)]
        self._before()
        self._check(lib().mhd_set_fields(self._h, *ptrs), "mhd_set_fields")
        self._after()        # the caller may free or overwrite its tensors once its stream has passed this point

    def get_fields(self):
        torch = _torch()
        out = [torch.empty(self.shape, dtype=torch.float64, device=self.device) for _ in range(7)]
        ptrs = [_vp(t.data_ptr()) for t in out]
        self._before()
        self._check(lib().mhd_get_fields(self._h, *ptrs), "mhd_get_fields")
        self._after()
        return out

    # ---- host-resident fields (numpy arrays or pinned CPU tensors) ----
    def set_fields_host(self, rho, ux, uy, uz, bx=None, by=None, bz=None):
        names = ("rho", "ux", "uy", "uz", "bx", "by", "bz")
        ptrs = [_host_ptr(a, self.npts, n) for a, n in zip((rho, ux, uy, uz, bx, by, bz), names)]
        self._check(lib().mhd_set_fields_host(self._h, *ptrs), "mhd_set_fields_host")

    def get_fields_host(self, out=None):
        if out is None:
            out = [np.empty(self.shape) for _ in range(7)]
        ptrs = [_host_ptr(a, self.npts, f"out[{i}]", writable=True) for i, a in enumerate(out)]
        self._check(lib().mhd_get_fields_host(self._h, *ptrs), "mhd_get_fields_host")
        return out

    def set_box(self, lx, ly, lz):
        self._check(lib().mhd_set_box(self._h, float(lx), float(ly), float(lz)), "mhd_set_box")

    def set_forcing(self, fx=None, fy=None, fz=None):
        """steady body force f of eq. (2): CUDA tensors, or None x 3 to switch it off (needs FLAG_FORCING)."""
        ptrs = [_dev_ptr(t, self.npts, n) for t, n in zip((fx, fy, fz), ("fx", "fy", "fz"))]
        self._before()
        self._check(lib().mhd_set_forcing(self._h, *ptrs), "mhd_set_forcing")
        self._after()

    def set_forcing_host(self, fx=None, fy=None, fz=None):
        ptrs = [_host_ptr(a, self.npts, n) for a, n in zip((fx, fy, fz), ("fx", "fy", "fz"))]
        self._check(lib().mhd_set_forcing_host(self._h, *ptrs), "mhd_set_forcing_host")

    def get_state(self):
        """exact-resume blob (spectral state + integrator history + header) as a CUDA uint8 tensor"""
        torch = _torch()
        n = int(lib().mhd_state_bytes(self._h))
        blob = torch.empty(n, dtype=torch.uint8, device=self.device)
        self._before()
        self._check(lib().mhd_get_state(self._h, _vp(blob.data_ptr()), n), "mhd_get_state")
        self._after()
        return blob

    def set_state(self, blob):
        torch = _torch()
        if not (isinstance(blob, torch.Tensor) and blob.is_cuda and blob.dtype == torch.uint8 and blob.is_contiguous()):
            raise ValueError("blob: expected a contiguous CUDA uint8 tensor from get_state()")
        self._before()
        self._check(lib().mhd_set_state(self._h, _vp(blob.data_ptr()), int(blob.numel())), "mhd_set_state")
        self._after()

    def step(self, n=1):
        self._check(lib().mhd_step(self._h, int(n)), "mhd_step")

    def diagnostics(self, nshell=0):
        d = Diag()
        ek = np.zeros(max(int(nshell), 1))
        em = np.zeros(max(int(nshell), 1))
        rc = self._check(lib().mhd_diagnostics(self._h, C.byref(d), _vp(ek.ctypes.data), _vp(em.ctypes.data), int(nshell)),
                         "mhd_diagnostics", allow=(ENONFINITE,))
        out = dict(step=d.step, time=d.time, ekin=d.ekin, emag=d.emag, eiso=d.eiso, mass=d.mass,
                   mom=np.array(d.mom[:]), bmean=np.array(d.bmean[:]), max_divb=d.max_divb, rc=rc,
                   enstrophy=d.enstrophy, current2=d.current2, u2=d.u2, rayleigh_q=d.rayleigh_q)
        if nshell > 0:
            out["ekin_spec"] = ek[:nshell].copy()
            out["emag_spec"] = em[:nshell].copy()
        return out

    def synchronize(self):
        self._stream.synchronize()


class FftPlan:
    """mhd_fft_plan_create / mhd_fft_r2c / mhd_fft_c2r: batched 3-D real FFT, unpadded cuFFT-style layout."""

    @property
    def stream(self):
        return self._stream

    def __init__(self, nx, ny, nz, batch, stream=None, device="cuda:0", mode=FFT_THREE_SWEEP, plane_workspace=False):
        """plane_workspace (implied by mode=FFT_PLANE_PIPELINE): size the workspace for the plane pipeline's ring too
        (mhd_fft_plane_workspace_bytes), so that set_mode(FFT_PLANE_PIPELINE) is allowed later; the default plan does not pay."""
        torch = _torch()
        L = lib()
        self.nx, self.ny, self.nz, self.batch = int(nx), int(ny), int(nz), int(batch)
        self.device = torch.device(device)
        want_ring = bool(plane_workspace) or mode == FFT_PLANE_PIPELINE
        sizer = L.mhd_fft_plane_workspace_bytes if want_ring else L.mhd_fft_workspace_bytes
        nbytes = sizer(self.nx, self.ny, self.nz, self.batch)
        if nbytes == 0:
            raise MhdError(EINVAL, sizer.__name__, f"unsupported size {nx}x{ny}x{nz} batch {batch}")
        with torch.cuda.device(self.device):
            self._ws = torch.empty(int(nbytes) + 256, dtype=torch.uint8, device=self.device)
            off = (-self._ws.data_ptr()) % 256
            self._stream, sp = _stream_ptr(torch, stream, self.device)
            self._stream.wait_stream(torch.cuda.current_stream(self.device))
            self._h = _vp()
            rc = L.mhd_fft_plan_create(C.byref(self._h), self.nx, self.ny, self.nz, self.batch,
                                       _vp(self._ws.data_ptr() + off), int(nbytes), sp)
        if rc != OK:
            self._h = _vp()
            raise MhdError(rc, "mhd_fft_plan_create")
        self.real_shape = (self.batch, self.nz, self.ny, self.nx)
        self.spec_shape = (self.batch, self.nz, self.ny, self.nx // 2 + 1)
        if mode != FFT_THREE_SWEEP:
            self.set_mode(mode)

    def set_mode(self, mode):
        """FFT_THREE_SWEEP (default) or FFT_PLANE_PIPELINE (x and y passes through an L2-resident ring; square planes 64..512)"""
        rc = lib().mhd_fft_plan_set_mode(self._h, int(mode))
        if rc != OK:
            raise MhdError(rc, "mhd_fft_plan_set_mode", lib().mhd_fft_last_error(self._h).decode())

    def r2c(self, real, out=None):
        torch = _torch()
        n = int(np.prod(self.real_shape))
        if out is None:
            out = torch.empty(self.spec_shape, dtype=torch.complex128, device=self.device)
        self._stream.wait_stream(torch.cuda.current_stream(self.device))
        rc = lib().mhd_fft_r2c(self._h, _dev_ptr(real, n, "real"), _vp(out.data_ptr()))
        torch.cuda.current_stream(self.device).wait_stream(self._stream)
        if rc != OK:
            raise MhdError(rc, "mhd_fft_r2c", lib().mhd_fft_last_error(self._h).decode())
        return out

    def c2r(self, spec, out=None):
        torch = _torch()
        if not (spec.is_cuda and spec.dtype == torch.complex128 and spec.is_contiguous() and tuple(spec.shape) == self.spec_shape):
            raise ValueError("spec: expected a contiguous CUDA complex128 tensor of shape %r" % (self.spec_shape,))
        if out is None:
            out = torch.empty(self.real_shape, dtype=torch.float64, device=self.device)
        self._stream.wait_stream(torch.cuda.current_stream(self.device))
        rc = lib().mhd_fft_c2r(self._h, _vp(spec.data_ptr()), _vp(out.data_ptr()))
        torch.cuda.current_stream(self.device).wait_stream(self._stream)
        if rc != OK:
            raise MhdError(rc, "mhd_fft_c2r", lib().mhd_fft_last_error(self._h).decode())
        return out

    def close(self):
        if getattr(self, "_h", None):
            try:
                self._stream.synchronize()      # transforms may still be running on the plan's stream
            finally:
                lib().mhd_fft_plan_destroy(self._h)
                self._h = _vp()
        self._ws = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def fft_c2r_static(spec, out=None, stream=None):
    """mhd_fft_c2r_static: the inverse transform of FftPlan.c2r for code that cannot give the library a workspace.

    FftPlan allocates a workspace tensor; this call allocates nothing on the GPU once `out` is given.  It is meant for
    callers that own their input and output and no other device memory (a hook inside a framework whose allocator holds the
    whole GPU, a job with a fully assigned memory budget, a loop that must not hit cudaMalloc's device synchronisation).
    The scratch is a fixed array inside the library: the transform's intermediate, 16 bytes per element of `spec`, may not
    exceed STATIC_SCRATCH_BYTES (8 MiB), else MhdError says how much was asked for.

    spec: contiguous CUDA complex128 tensor [batch][nz][ny][nx/2+1] (nx is taken as 2*(last dim - 1)); out: contiguous CUDA
    float64 tensor [batch][nz][ny][nx] on the same GPU (created with torch.empty when None -- pass it if you cannot
    allocate).  Enqueued on `stream` (default: the current torch stream of spec's device).  The first call on a GPU also
    sets the scratch up and synchronises the stream: make it before any stream capture.  All calls on one GPU share the
    scratch, so calls on different streams must not overlap."""
    torch = _torch()
    if not (isinstance(spec, torch.Tensor) and spec.is_cuda and spec.dtype == torch.complex128 and spec.is_contiguous() and spec.dim() == 4):
        raise ValueError("spec: expected a contiguous CUDA complex128 tensor [batch][nz][ny][nx/2+1]")
    batch, nz, ny, nxh = (int(v) for v in spec.shape)
    nx = 2 * (nxh - 1)
    if out is None:
        out = torch.empty((batch, nz, ny, nx), dtype=torch.float64, device=spec.device)
    if out.device != spec.device:
        raise ValueError("out: must live on the same GPU as spec")
    optr = _dev_ptr(out, batch * nz * ny * nx, "out")
    s = torch.cuda.current_stream(spec.device) if stream is None else stream
    err = C.create_string_buffer(256)
    rc = lib().mhd_fft_c2r_static(nx, ny, nz, batch, _vp(spec.data_ptr()), optr, _vp(s.cuda_stream), err, len(err))
    if rc != OK:
        raise MhdError(rc, "mhd_fft_c2r_static", err.value.decode())
    return out
