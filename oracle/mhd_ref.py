"""ctypes binding of the CPU ORACLE (oracle/mhd_ref.c).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this module.  It shares no code with the CUDA path (paper_2402_05478_b200/).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "mhd_ref.c")
_HDR = os.path.join(_HERE, "mhd_ref.h")
_LIB = os.path.join(_HERE, "libmhd_ref.so")

OK, EINVAL, ENOMEM, ESTATE, ENONFINITE = 0, -1, -2, -4, -5
AB2, RK4 = 0, 1
FLAG_HYDRO, FLAG_NO_DEALIAS = 1, 2
FIELD_NAMES = ("rho", "mx", "my", "mz", "bx", "by", "bz")


_SAN_LIB = os.path.join(_HERE, "libmhd_ref_san.so")


def sanitize() -> bool:
    """MHD_REF_SANITIZE=1: the oracle built with AddressSanitizer + UndefinedBehaviourSanitizer.  The process
    must then be started with libasan preloaded, e.g.
        MHD_REF_SANITIZE=1 LD_PRELOAD=$(gcc -print-file-name=libasan.so) ASAN_OPTIONS=detect_leaks=0 \
            python -m pytest tests -m "not gpu" -q
    (the interpreter itself is not instrumented, so leak detection is switched off).  Test infrastructure only."""
    return os.environ.get("MHD_REF_SANITIZE", "") not in ("", "0")


def build(force: bool = False) -> str:
    """Compile oracle/mhd_ref.c into oracle/libmhd_ref.so with gcc (building the checker is not using it)."""
    lib_path = _SAN_LIB if sanitize() else _LIB
    stale = (not os.path.exists(lib_path)) or any(
        os.path.getmtime(p) > os.path.getmtime(lib_path) for p in (_SRC, _HDR))
    if force or stale:
        opt = ["-O1", "-g", "-fno-omit-frame-pointer", "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined"] \
            if sanitize() else ["-O2"]
        cmd = ["gcc"] + opt + ["-std=c99", "-fPIC", "-shared", "-fopenmp", "-fcx-limited-range",
                               "-Wall", "-Wextra", "-o", lib_path, _SRC, "-lm"]
        subprocess.run(cmd, check=True, cwd=_HERE)
    return lib_path


class Diag(C.Structure):
    _fields_ = [("step", C.c_longlong), ("time", C.c_double), ("ekin", C.c_double), ("emag", C.c_double),
                ("eiso", C.c_double), ("mass", C.c_double), ("mom", C.c_double * 3),
                ("bmean", C.c_double * 3), ("max_divb", C.c_double),
                ("enstrophy", C.c_double), ("current2", C.c_double), ("u2", C.c_double), ("rayleigh_q", C.c_double)]


_lib = None
_dp = C.POINTER(C.c_double)


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        L.mhd_ref_set_threads.argtypes = [C.c_int]
        L.mhd_ref_get_threads.restype = C.c_int
        L.mhd_ref_fft1d.argtypes = [C.c_int, C.c_int, _dp, _dp]
        L.mhd_ref_fft_r2c.argtypes = [C.c_int] * 4 + [_dp, _dp]
        L.mhd_ref_fft_c2r.argtypes = [C.c_int] * 4 + [_dp, _dp]
        L.mhd_ref_create.argtypes = [C.POINTER(C.c_void_p), C.c_int, C.c_int, C.c_int, C.c_double, C.c_double,
                                     C.c_double, C.c_double, C.c_int, C.c_uint]
        L.mhd_ref_destroy.argtypes = [C.c_void_p]
        L.mhd_ref_destroy.restype = None
        L.mhd_ref_set_fields.argtypes = [C.c_void_p] + [_dp] * 7
        L.mhd_ref_set_box.argtypes = [C.c_void_p, C.c_double, C.c_double, C.c_double]
        L.mhd_ref_set_forcing.argtypes = [C.c_void_p] + [_dp] * 3
        L.mhd_ref_get_fields.argtypes = [C.c_void_p] + [_dp] * 7
        L.mhd_ref_step.argtypes = [C.c_void_p, C.c_int]
        L.mhd_ref_diagnostics.argtypes = [C.c_void_p, C.POINTER(Diag), _dp, _dp, C.c_int]
        L.mhd_ref_get_spectral.argtypes = [C.c_void_p, C.c_int, _dp]
        L.mhd_ref_set_spectral.argtypes = [C.c_void_p, C.c_int, _dp]
        L.mhd_ref_rhs.argtypes = [C.c_void_p, _dp]
        L.mhd_ref_mask.argtypes = [C.c_void_p, C.POINTER(C.c_ubyte)]
        _lib = L
    return _lib


def _p(a):
    return None if a is None else a.ctypes.data_as(_dp)


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def set_threads(n: int) -> None:
    lib().mhd_ref_set_threads(int(n))


def get_threads() -> int:
    return int(lib().mhd_ref_get_threads())


def fft1d(x, sign=-1):
    x = np.ascontiguousarray(x, dtype=np.complex128)
    out = np.empty_like(x)
    rc = lib().mhd_ref_fft1d(x.size, sign, x.view(np.float64).ctypes.data_as(_dp),
                             out.view(np.float64).ctypes.data_as(_dp))
    assert rc == OK, rc
    return out


def fft_r2c(a):
    """a: (batch, nz, ny, nx) or (nz, ny, nx) real -> complex half-spectrum (..., nz, ny, nx/2+1), unnormalised."""
    a = _f64(a)
    squeeze = a.ndim == 3
    if squeeze:
        a = a[None]
    b, nz, ny, nx = a.shape
    out = np.empty((b, nz, ny, nx // 2 + 1), dtype=np.complex128)
    rc = lib().mhd_ref_fft_r2c(nx, ny, nz, b, _p(a), out.view(np.float64).ctypes.data_as(_dp))
    assert rc == OK, rc
    return out[0] if squeeze else out


def fft_c2r(a, nx):
    """inverse of fft_r2c (includes 1/(nx ny nz))."""
    a = np.ascontiguousarray(a, dtype=np.complex128)
    squeeze = a.ndim == 3
    if squeeze:
        a = a[None]
    b, nz, ny, nxh = a.shape
    assert nxh == nx // 2 + 1
    out = np.empty((b, nz, ny, nx), dtype=np.float64)
    rc = lib().mhd_ref_fft_c2r(nx, ny, nz, b, a.view(np.float64).ctypes.data_as(_dp), _p(out))
    assert rc == OK, rc
    return out[0] if squeeze else out


class RefSolver:
    """The oracle's mhd_ref_* calls on numpy arrays of shape (nz, ny, nx)."""

    def __init__(self, nx, ny, nz, nu, eta, cs, dt, integrator=AB2, flags=0):
        self.nx, self.ny, self.nz = nx, ny, nz
        self.shape = (nz, ny, nx)
        self.cshape = (nz, ny, nx // 2 + 1)
        self.flags = flags
        self._h = C.c_void_p()
        rc = lib().mhd_ref_create(C.byref(self._h), nx, ny, nz, nu, eta, cs, dt, integrator, flags)
        if rc != OK:
            raise ValueError(f"mhd_ref_create failed: {rc}")

    def close(self):
        if self._h:
            lib().mhd_ref_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_fields(self, rho, ux, uy, uz, bx=None, by=None, bz=None):
        arrs = [None if a is None else _f64(a) for a in (rho, ux, uy, uz, bx, by, bz)]
        for a in arrs:
            assert a is None or a.shape == self.shape, (a.shape, self.shape)
        rc = lib().mhd_ref_set_fields(self._h, *[_p(a) for a in arrs])
        if rc != OK:
            raise RuntimeError(f"mhd_ref_set_fields: {rc}")

    def set_box(self, lx, ly, lz):
        rc = lib().mhd_ref_set_box(self._h, float(lx), float(ly), float(lz))
        if rc != OK:
            raise ValueError(f"mhd_ref_set_box: {rc}")

    def set_forcing(self, fx=None, fy=None, fz=None):
        arrs = [None if a is None else _f64(a) for a in (fx, fy, fz)]
        for a in arrs:
            assert a is None or a.shape == self.shape
        rc = lib().mhd_ref_set_forcing(self._h, *[_p(a) for a in arrs])
        if rc != OK:
            raise ValueError(f"mhd_ref_set_forcing: {rc}")

    def step(self, n=1):
        rc = lib().mhd_ref_step(self._h, int(n))
        if rc != OK:
            raise RuntimeError(f"mhd_ref_step: {rc}")

    def get_fields(self):
        out = [np.empty(self.shape) for _ in range(7)]
        rc = lib().mhd_ref_get_fields(self._h, *[_p(a) for a in out])
        if rc != OK:
            raise RuntimeError(f"mhd_ref_get_fields: {rc}")
        return out

    def diagnostics(self, nshell=0):
        d = Diag()
        ek = np.zeros(max(nshell, 1))
        em = np.zeros(max(nshell, 1))
        rc = lib().mhd_ref_diagnostics(self._h, C.byref(d), _p(ek), _p(em), int(nshell))
        if rc not in (OK, ENONFINITE):
            raise RuntimeError(f"mhd_ref_diagnostics: {rc}")
        out = dict(step=d.step, time=d.time, ekin=d.ekin, emag=d.emag, eiso=d.eiso, mass=d.mass,
                   mom=np.array(d.mom[:]), bmean=np.array(d.bmean[:]), max_divb=d.max_divb, rc=rc,
                   enstrophy=d.enstrophy, current2=d.current2, u2=d.u2, rayleigh_q=d.rayleigh_q)
        if nshell > 0:
            out["ekin_spec"] = ek[:nshell].copy()
            out["emag_spec"] = em[:nshell].copy()
        return out

    def get_spectral(self, field):
        out = np.empty(self.cshape, dtype=np.complex128)
        rc = lib().mhd_ref_get_spectral(self._h, int(field), out.view(np.float64).ctypes.data_as(_dp))
        assert rc == OK, rc
        return out

    def set_spectral(self, field, a):
        a = np.ascontiguousarray(a, dtype=np.complex128)
        assert a.shape == self.cshape
        rc = lib().mhd_ref_set_spectral(self._h, int(field), a.view(np.float64).ctypes.data_as(_dp))
        assert rc == OK, rc

    def rhs(self):
        out = np.empty((7,) + self.cshape, dtype=np.complex128)
        rc = lib().mhd_ref_rhs(self._h, out.view(np.float64).ctypes.data_as(_dp))
        if rc != OK:
            raise RuntimeError(f"mhd_ref_rhs: {rc}")
        return out

    def mask(self):
        out = np.empty(self.cshape, dtype=np.uint8)
        rc = lib().mhd_ref_mask(self._h, out.ctypes.data_as(C.POINTER(C.c_ubyte)))
        assert rc == OK, rc
        return out.astype(bool)
