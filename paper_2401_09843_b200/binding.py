"""Thin ctypes binding of libns.so (include/ns.h).  Argument marshalling only: every step of the
path runs in the CUDA kernels behind the C ABI.  There is no fallback: if libns.so is missing or
no CUDA device is usable, calls raise.

Host buffers are numpy arrays, device buffers are torch CUDA tensors (PyTorch is used only for
device memory and streams).  Complex arrays: numpy complex128/complex64, torch complex128/complex64.
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libns.so")

NS_F64, NS_F32 = 0, 1
NS_HOST, NS_DEVICE = 0, 1
NS_OK, NS_ERR_INVALID_ARG, NS_ERR_OOM, NS_ERR_CUDA, NS_ERR_STATE, NS_ERR_NONFINITE = 0, -1, -2, -3, -4, -5

EXPORTS = [
    "ns_create", "ns_destroy", "ns_set_initial", "ns_set_spectral", "ns_get_spectral", "ns_rhs", "ns_step",
    "ns_step_cfl", "ns_step_dts", "ns_advance", "ns_max_velocity", "ns_get_fields", "ns_energy_spectrum", "ns_enstrophy_spectrum",
    "ns_structure_function", "ns_structure_function_p", "ns_ensemble_moments", "ns_autotune", "ns_transform_grid", "ns_padded_size", "ns_profile", "ns_profile_read", "ns_time", "ns_kernel_launches", "ns_device_bytes", "ns_last_error",
]
# include/ns_mg.h: one sample over several devices
EXPORTS_MG = [
    "ns_mg_create", "ns_mg_destroy", "ns_mg_set_spectral", "ns_mg_get_spectral", "ns_mg_rhs", "ns_mg_step", "ns_mg_step_cfl",
    "ns_mg_max_velocity", "ns_mg_time", "ns_mg_exchange_bytes", "ns_mg_kernel_launches", "ns_mg_device_bytes", "ns_mg_last_error",
]
# include/ns_noalloc.h: the allocation-free entry point
EXPORTS_NOALLOC = ["ns_noalloc_energy_spectrum"]
NS_NOALLOC_MAX_VALUES = 16384
# include/ns2d.h: the two-dimensional solver
EXPORTS_2D = [
    "ns2d_create", "ns2d_destroy", "ns2d_set_initial", "ns2d_set_spectral", "ns2d_get_spectral", "ns2d_rhs", "ns2d_step", "ns2d_step_cfl",
    "ns2d_step_dts", "ns2d_advance", "ns2d_max_velocity", "ns2d_get_fields", "ns2d_energy_spectrum", "ns2d_enstrophy_spectrum", "ns2d_time",
    "ns2d_profile", "ns2d_profile_read", "ns2d_transform_grid", "ns2d_kernel_launches", "ns2d_device_bytes", "ns2d_last_error",
]


class ns_params(ctypes.Structure):
    _fields_ = [("nu", ctypes.c_double), ("eps", ctypes.c_double), ("s", ctypes.c_double),
                ("m_cut", ctypes.c_double), ("q_exp", ctypes.c_double), ("q_sharp", ctypes.c_int)]


class NSError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"libns error {code}: {msg}")
        self.code = code


_lib = None


def lib():
    """Load libns.so (built by `python -m paper_2401_09843_b200.build`).  Raises if it is missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} not found: build it with `python -m paper_2401_09843_b200.build` "
                              "(there is no CPU fallback)")
        L = ctypes.CDLL(LIB_PATH)
        vp, i, d = ctypes.c_void_p, ctypes.c_int, ctypes.c_double
        L.ns_create.argtypes = [ctypes.POINTER(vp), i, i, ctypes.POINTER(ns_params), i, vp]
        L.ns_destroy.argtypes = [vp]
        L.ns_set_initial.argtypes = [vp, vp, i]
        L.ns_set_spectral.argtypes = [vp, vp, i]
        L.ns_get_spectral.argtypes = [vp, vp, i]
        L.ns_rhs.argtypes = [vp, vp, i]
        L.ns_step.argtypes = [vp, d]
        L.ns_step_cfl.argtypes = [vp, d, d, vp]
        L.ns_step_dts.argtypes = [vp, vp]
        L.ns_advance.argtypes = [vp, d, d, i, ctypes.POINTER(ctypes.c_int)]
        L.ns_max_velocity.argtypes = [vp, vp]
        L.ns_get_fields.argtypes = [vp, vp, i]
        L.ns_energy_spectrum.argtypes = [vp, vp, i]
        L.ns_enstrophy_spectrum.argtypes = [vp, vp, i]
        L.ns_structure_function.argtypes = [vp, vp, i]
        L.ns_structure_function_p.argtypes = [vp, d, vp, i]
        L.ns_ensemble_moments.argtypes = [vp, vp, vp, i]
        L.ns_autotune.argtypes = [i, i, i, vp, vp, ctypes.POINTER(ctypes.c_int)]
        L.ns_transform_grid.argtypes = [vp]
        L.ns_padded_size.argtypes = [vp]
        L.ns_profile.argtypes = [vp, i]
        L.ns_profile_read.argtypes = [vp, vp, vp]
        L.ns_time.argtypes = [vp, i]
        L.ns_time.restype = d
        L.ns_kernel_launches.argtypes = [vp]
        L.ns_kernel_launches.restype = ctypes.c_longlong
        L.ns_device_bytes.argtypes = [vp]
        L.ns_device_bytes.restype = ctypes.c_longlong
        L.ns_last_error.argtypes = [vp]
        L.ns_last_error.restype = ctypes.c_char_p
        # include/ns2d.h
        L.ns2d_create.argtypes = [ctypes.POINTER(vp), i, i, ctypes.POINTER(ns_params), i, vp]
        L.ns2d_destroy.argtypes = [vp]
        for name in ("ns2d_set_initial", "ns2d_set_spectral", "ns2d_get_spectral", "ns2d_rhs", "ns2d_get_fields"):
            getattr(L, name).argtypes = [vp, vp, i]
        L.ns2d_step.argtypes = [vp, d]
        L.ns2d_step_cfl.argtypes = [vp, d, d, vp]
        L.ns2d_step_dts.argtypes = [vp, vp]
        L.ns2d_advance.argtypes = [vp, d, d, i, ctypes.POINTER(ctypes.c_int)]
        L.ns2d_max_velocity.argtypes = [vp, vp]
        L.ns2d_energy_spectrum.argtypes = [vp, vp, i]
        L.ns2d_enstrophy_spectrum.argtypes = [vp, vp, i]
        L.ns2d_time.argtypes = [vp, i]
        L.ns2d_time.restype = d
        L.ns2d_profile.argtypes = [vp, i]
        L.ns2d_profile_read.argtypes = [vp, vp, vp]
        L.ns2d_transform_grid.argtypes = [vp]
        L.ns2d_kernel_launches.argtypes = [vp]
        L.ns2d_kernel_launches.restype = ctypes.c_longlong
        L.ns2d_device_bytes.argtypes = [vp]
        L.ns2d_device_bytes.restype = ctypes.c_longlong
        L.ns2d_last_error.argtypes = [vp]
        L.ns2d_last_error.restype = ctypes.c_char_p
        # include/ns_mg.h
        L.ns_mg_create.argtypes = [ctypes.POINTER(vp), i, i, ctypes.POINTER(ctypes.c_int), ctypes.POINTER(ns_params), i]
        L.ns_mg_destroy.argtypes = [vp]
        for name in ("ns_mg_set_spectral", "ns_mg_get_spectral", "ns_mg_rhs"):
            getattr(L, name).argtypes = [vp, vp]
        L.ns_mg_max_velocity.argtypes = [vp, ctypes.POINTER(d)]
        L.ns_mg_step.argtypes = [vp, d]
        L.ns_mg_step_cfl.argtypes = [vp, d, d, ctypes.POINTER(d)]
        L.ns_mg_time.argtypes = [vp]
        L.ns_mg_time.restype = d
        for name in ("ns_mg_exchange_bytes", "ns_mg_kernel_launches", "ns_mg_device_bytes"):
            getattr(L, name).argtypes = [vp]
            getattr(L, name).restype = ctypes.c_longlong
        L.ns_mg_last_error.argtypes = [vp]
        L.ns_mg_last_error.restype = ctypes.c_char_p
        # include/ns_noalloc.h
        L.ns_noalloc_energy_spectrum.argtypes = [vp, i, i, i, i, vp, i, vp, ctypes.c_char_p, i]
        _lib = L
    return _lib


def _is_torch(x):
    return type(x).__module__.startswith("torch")


def _buf(x, writable=False):
    """(pointer, memspace, keepalive) of a numpy array (host) or a torch CUDA tensor (device)."""
    if _is_torch(x):
        if not x.is_cuda:
            raise ValueError("torch tensors must live on the GPU (use numpy arrays for host buffers)")
        if not x.is_contiguous():
            raise ValueError("device buffer must be contiguous")
        return ctypes.c_void_p(x.data_ptr()), NS_DEVICE, x
    a = x
    if not isinstance(a, np.ndarray) or not a.flags["C_CONTIGUOUS"]:
        if writable:
            raise ValueError("output host buffer must be a C-contiguous numpy array")
        a = np.ascontiguousarray(a)
    return ctypes.c_void_p(a.ctypes.data), NS_HOST, a


def autotune(N, dtype="f64", ncand=3):
    """ns_autotune: time the transform passes on the first `ncand` admissible transform grids >= N, record the fastest for later
    Solver(N, ...) calls in this process.  Returns (best grid, [(grid, ms), ...])."""
    dt = {"f64": NS_F64, "f32": NS_F32, NS_F64: NS_F64, NS_F32: NS_F32}[dtype]
    grids = np.zeros(ncand, dtype=np.int32)
    ms = np.zeros(ncand, dtype=np.float64)
    best = ctypes.c_int(0)
    rc = lib().ns_autotune(int(N), dt, int(ncand), ctypes.c_void_p(grids.ctypes.data), ctypes.c_void_p(ms.ctypes.data), ctypes.byref(best))
    if rc != NS_OK:
        raise NSError(rc, lib().ns_last_error(None).decode())
    return int(best.value), [(int(g), float(t)) for g, t in zip(grids, ms) if g]


class Solver:
    """Owner of one ns_solver handle.  Method names follow the C entry points without the ns_ prefix."""

    def __init__(self, N, batch=1, nu=0.0, eps=0.0, s=1.0, m_cut=-1.0, q_exp=-1.0, q_sharp=0, dtype="f64", stream=None):
        self.N, self.batch = int(N), int(batch)
        self.dtype = {"f64": NS_F64, "f32": NS_F32, NS_F64: NS_F64, NS_F32: NS_F32}[dtype]
        self.real = np.float64 if self.dtype == NS_F64 else np.float32
        self.cplx = np.complex128 if self.dtype == NS_F64 else np.complex64
        self._h = ctypes.c_void_p()
        p = ns_params(nu, eps, s, m_cut, q_exp, q_sharp)
        if stream is None:
            import torch  # device memory and streams only
            stream = torch.cuda.current_stream().cuda_stream
        rc = lib().ns_create(ctypes.byref(self._h), self.N, self.batch, ctypes.byref(p), self.dtype, ctypes.c_void_p(stream))
        if rc != NS_OK:
            raise NSError(rc, lib().ns_last_error(None).decode())

    # shapes ---------------------------------------------------------------------------------------
    @property
    def spectral_shape(self):
        return (self.batch, 3, self.N, self.N, self.N // 2 + 1)

    @property
    def physical_shape(self):
        return (self.batch, 3, self.N, self.N, self.N)

    def _check(self, rc):
        if rc != NS_OK:
            raise NSError(rc, lib().ns_last_error(self._h).decode())

    def _typed(self, x, kind):
        """Cast host arrays to the solver dtype; device tensors must already match."""
        want = self.real if kind == "real" else self.cplx
        if _is_torch(x):
            import torch
            tw = {np.float64: torch.float64, np.float32: torch.float32, np.complex128: torch.complex128,
                  np.complex64: torch.complex64}[want]
            if x.dtype != tw:
                raise ValueError(f"device tensor dtype {x.dtype} != {tw}")
            return x
        return np.ascontiguousarray(x, dtype=want)

    # calls ----------------------------------------------------------------------------------------
    def close(self):
        if self._h:
            lib().ns_destroy(self._h)
            self._h = ctypes.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_initial(self, u_phys):
        u = self._typed(u_phys, "real")
        assert tuple(u.shape) == self.physical_shape, (tuple(u.shape), self.physical_shape)
        p, ms, _k = _buf(u)
        self._check(lib().ns_set_initial(self._h, p, ms))

    def set_spectral(self, u_hat):
        u = self._typed(u_hat, "cplx")
        assert tuple(u.shape) == self.spectral_shape
        p, ms, _k = _buf(u)
        self._check(lib().ns_set_spectral(self._h, p, ms))

    def get_spectral(self, out=None):
        if out is None:
            out = np.empty(self.spectral_shape, dtype=self.cplx)
        p, ms, _k = _buf(out, writable=True)
        self._check(lib().ns_get_spectral(self._h, p, ms))
        return out

    def rhs(self, out=None):
        if out is None:
            out = np.empty(self.spectral_shape, dtype=self.cplx)
        p, ms, _k = _buf(out, writable=True)
        self._check(lib().ns_rhs(self._h, p, ms))
        return out

    def step(self, dt):
        self._check(lib().ns_step(self._h, float(dt)))

    def step_cfl(self, cfl, t_end, return_dt=True):
        if return_dt:
            dts = np.empty(self.batch, dtype=np.float64)
            self._check(lib().ns_step_cfl(self._h, float(cfl), float(t_end), ctypes.c_void_p(dts.ctypes.data)))
            return dts
        self._check(lib().ns_step_cfl(self._h, float(cfl), float(t_end), None))
        return None

    def step_dts(self, dts):
        d = np.ascontiguousarray(dts, dtype=np.float64)
        assert d.shape == (self.batch,)
        self._check(lib().ns_step_dts(self._h, ctypes.c_void_p(d.ctypes.data)))

    def max_velocity(self):
        out = np.empty(self.batch, dtype=np.float64)
        self._check(lib().ns_max_velocity(self._h, ctypes.c_void_p(out.ctypes.data)))
        return out

    def get_fields(self, out=None):
        if out is None:
            out = np.empty(self.physical_shape, dtype=self.real)
        p, ms, _k = _buf(out, writable=True)
        self._check(lib().ns_get_fields(self._h, p, ms))
        return out

    def energy_spectrum(self, nbins):
        E = np.empty((self.batch, int(nbins)), dtype=np.float64)
        self._check(lib().ns_energy_spectrum(self._h, ctypes.c_void_p(E.ctypes.data), int(nbins)))
        return E

    def advance(self, cfl, t_end, max_steps=1 << 30):
        """Integrate every sample to t_end at the given CFL number; returns the number of RK3 steps launched."""
        n = ctypes.c_int(0)
        self._check(lib().ns_advance(self._h, float(cfl), float(t_end), int(max_steps), ctypes.byref(n)))
        return n.value

    def structure_function_p(self, p, nl=None):
        nl = self.N // 2 if nl is None else int(nl)
        S = np.empty((self.batch, nl), dtype=np.float64)
        self._check(lib().ns_structure_function_p(self._h, float(p), ctypes.c_void_p(S.ctypes.data), nl))
        return S

    def ensemble_moments(self):
        """(mean, var) over the batch, each [3][N][N][N] of the solver dtype (host arrays)."""
        shape = self.physical_shape[1:]
        mean = np.empty(shape, dtype=self.real)
        var = np.empty(shape, dtype=self.real)
        self._check(lib().ns_ensemble_moments(self._h, ctypes.c_void_p(mean.ctypes.data), ctypes.c_void_p(var.ctypes.data), NS_HOST))
        return mean, var

    def enstrophy_spectrum(self, nbins):
        Z = np.empty((self.batch, int(nbins)), dtype=np.float64)
        self._check(lib().ns_enstrophy_spectrum(self._h, ctypes.c_void_p(Z.ctypes.data), int(nbins)))
        return Z

    def structure_function(self, nl=None):
        nl = self.N // 2 if nl is None else int(nl)
        S = np.empty((self.batch, nl), dtype=np.float64)
        self._check(lib().ns_structure_function(self._h, ctypes.c_void_p(S.ctypes.data), nl))
        return S

    PASS_NAMES = ["a1_col_inv_x", "a2_col_inv_y", "a3_z_inv_prod", "a4_z_fwd", "a5_col_fwd_y", "a6_col_fwd_x",
                  "a7_spectral", "other"]

    @property
    def transform_grid(self):
        """ns_transform_grid: the grid Nt >= N the transforms run on."""
        return int(lib().ns_transform_grid(self._h))

    @property
    def padded_size(self):
        """ns_padded_size: M = 3 Nt / 2, the padded grid max|u| is taken over."""
        return int(lib().ns_padded_size(self._h))

    def profile(self, enable=True):
        self._check(lib().ns_profile(self._h, 1 if enable else 0))

    def profile_read(self):
        """{pass name: (total ms, launches)} accumulated since profile(True)."""
        ms = np.zeros(8, dtype=np.float64)
        cnt = np.zeros(8, dtype=np.int64)
        self._check(lib().ns_profile_read(self._h, ctypes.c_void_p(ms.ctypes.data), ctypes.c_void_p(cnt.ctypes.data)))
        return {n: (float(ms[i]), int(cnt[i])) for i, n in enumerate(self.PASS_NAMES)}

    def time(self, sample=0):
        return float(lib().ns_time(self._h, int(sample)))

    def kernel_launches(self):
        return int(lib().ns_kernel_launches(self._h))

    def device_bytes(self):
        return int(lib().ns_device_bytes(self._h))


class Solver2D:
    """Owner of one ns2d_solver handle (include/ns2d.h).  Method names follow the C entry points without the ns2d_ prefix."""

    PASS_NAMES = ["b1_x_inv", "b2_y_fused", "b3_x_fwd", "b4_spectral"]

    def __init__(self, N, batch=1, nu=0.0, eps=0.0, s=1.0, m_cut=-1.0, q_exp=-1.0, q_sharp=0, dtype="f64", stream=None):
        self.N, self.batch = int(N), int(batch)
        self.dtype = {"f64": NS_F64, "f32": NS_F32, NS_F64: NS_F64, NS_F32: NS_F32}[dtype]
        self.real = np.float64 if self.dtype == NS_F64 else np.float32
        self.cplx = np.complex128 if self.dtype == NS_F64 else np.complex64
        self._h = ctypes.c_void_p()
        p = ns_params(nu, eps, s, m_cut, q_exp, q_sharp)
        if stream is None:
            import torch  # device memory and streams only
            stream = torch.cuda.current_stream().cuda_stream
        rc = lib().ns2d_create(ctypes.byref(self._h), self.N, self.batch, ctypes.byref(p), self.dtype, ctypes.c_void_p(stream))
        if rc != NS_OK:
            raise NSError(rc, lib().ns2d_last_error(None).decode())

    @property
    def spectral_shape(self):
        return (self.batch, 2, self.N, self.N // 2 + 1)

    @property
    def physical_shape(self):
        return (self.batch, 2, self.N, self.N)

    def _check(self, rc):
        if rc != NS_OK:
            raise NSError(rc, lib().ns2d_last_error(self._h).decode())

    _typed = Solver._typed

    def close(self):
        if self._h:
            lib().ns2d_destroy(self._h)
            self._h = ctypes.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_initial(self, u_phys):
        u = self._typed(u_phys, "real")
        assert tuple(u.shape) == self.physical_shape, (tuple(u.shape), self.physical_shape)
        p, ms, _k = _buf(u)
        self._check(lib().ns2d_set_initial(self._h, p, ms))

    def set_spectral(self, u_hat):
        u = self._typed(u_hat, "cplx")
        assert tuple(u.shape) == self.spectral_shape
        p, ms, _k = _buf(u)
        self._check(lib().ns2d_set_spectral(self._h, p, ms))

    def get_spectral(self, out=None):
        if out is None:
            out = np.empty(self.spectral_shape, dtype=self.cplx)
        p, ms, _k = _buf(out, writable=True)
        self._check(lib().ns2d_get_spectral(self._h, p, ms))
        return out

    def rhs(self, out=None):
        if out is None:
            out = np.empty(self.spectral_shape, dtype=self.cplx)
        p, ms, _k = _buf(out, writable=True)
        self._check(lib().ns2d_rhs(self._h, p, ms))
        return out

    def get_fields(self, out=None):
        if out is None:
            out = np.empty(self.physical_shape, dtype=self.real)
        p, ms, _k = _buf(out, writable=True)
        self._check(lib().ns2d_get_fields(self._h, p, ms))
        return out

    def step(self, dt):
        self._check(lib().ns2d_step(self._h, float(dt)))

    def step_cfl(self, cfl, t_end, return_dt=True):
        if return_dt:
            dts = np.empty(self.batch, dtype=np.float64)
            self._check(lib().ns2d_step_cfl(self._h, float(cfl), float(t_end), ctypes.c_void_p(dts.ctypes.data)))
            return dts
        self._check(lib().ns2d_step_cfl(self._h, float(cfl), float(t_end), None))
        return None

    def step_dts(self, dts):
        d = np.ascontiguousarray(dts, dtype=np.float64)
        assert d.shape == (self.batch,)
        self._check(lib().ns2d_step_dts(self._h, ctypes.c_void_p(d.ctypes.data)))

    def advance(self, cfl, t_end, max_steps=1 << 30):
        n = ctypes.c_int(0)
        self._check(lib().ns2d_advance(self._h, float(cfl), float(t_end), int(max_steps), ctypes.byref(n)))
        return n.value

    def max_velocity(self):
        out = np.empty(self.batch, dtype=np.float64)
        self._check(lib().ns2d_max_velocity(self._h, ctypes.c_void_p(out.ctypes.data)))
        return out

    def energy_spectrum(self, nbins):
        E = np.empty((self.batch, int(nbins)), dtype=np.float64)
        self._check(lib().ns2d_energy_spectrum(self._h, ctypes.c_void_p(E.ctypes.data), int(nbins)))
        return E

    def enstrophy_spectrum(self, nbins):
        Z = np.empty((self.batch, int(nbins)), dtype=np.float64)
        self._check(lib().ns2d_enstrophy_spectrum(self._h, ctypes.c_void_p(Z.ctypes.data), int(nbins)))
        return Z

    @property
    def transform_grid(self):
        """ns2d_transform_grid: the grid Nt >= N the transforms run on."""
        return int(lib().ns2d_transform_grid(self._h))

    @property
    def padded_size(self):
        return 3 * self.transform_grid // 2

    def profile(self, enable=True):
        self._check(lib().ns2d_profile(self._h, 1 if enable else 0))

    def profile_read(self):
        ms = np.zeros(4, dtype=np.float64)
        cnt = np.zeros(4, dtype=np.int64)
        self._check(lib().ns2d_profile_read(self._h, ctypes.c_void_p(ms.ctypes.data), ctypes.c_void_p(cnt.ctypes.data)))
        return {n: (float(ms[i]), int(cnt[i])) for i, n in enumerate(self.PASS_NAMES)}

    def time(self, sample=0):
        return float(lib().ns2d_time(self._h, int(sample)))

    def kernel_launches(self):
        return int(lib().ns2d_kernel_launches(self._h))

    def device_bytes(self):
        return int(lib().ns2d_device_bytes(self._h))


class SolverMG:
    """One sample over several devices (include/ns_mg.h): ky / px slab decomposition driven by one process.  `devices` may name
    the same GPU more than once (the ranks then share it).  Spectral arrays are host numpy arrays [3][N][N][N/2+1]."""

    def __init__(self, N, devices, nu=0.0, eps=0.0, s=1.0, m_cut=-1.0, q_exp=-1.0, q_sharp=0, dtype="f64"):
        self.N, self.devices = int(N), [int(x) for x in devices]
        self.dtype = {"f64": NS_F64, "f32": NS_F32, NS_F64: NS_F64, NS_F32: NS_F32}[dtype]
        self.cplx = np.complex128 if self.dtype == NS_F64 else np.complex64
        self.spectral_shape = (3, self.N, self.N, self.N // 2 + 1)
        p = ns_params(nu, eps, s, m_cut, q_exp, q_sharp)
        dev = (ctypes.c_int * len(self.devices))(*self.devices)
        h = ctypes.c_void_p()
        rc = lib().ns_mg_create(ctypes.byref(h), self.N, len(self.devices), dev, ctypes.byref(p), self.dtype)
        if rc != NS_OK:
            raise NSError(rc, lib().ns_mg_last_error(None).decode())
        self._h = h

    def __del__(self):
        if getattr(self, "_h", None):
            lib().ns_mg_destroy(self._h)
            self._h = None

    def _check(self, rc):
        if rc != NS_OK:
            raise NSError(rc, lib().ns_mg_last_error(self._h).decode())

    def _host(self, a):
        a = np.ascontiguousarray(a, dtype=self.cplx)
        assert a.shape == self.spectral_shape, (a.shape, self.spectral_shape)
        return a

    def set_spectral(self, u_hat):
        a = self._host(u_hat)
        self._check(lib().ns_mg_set_spectral(self._h, ctypes.c_void_p(a.ctypes.data)))

    def get_spectral(self):
        out = np.empty(self.spectral_shape, dtype=self.cplx)
        self._check(lib().ns_mg_get_spectral(self._h, ctypes.c_void_p(out.ctypes.data)))
        return out

    def rhs(self):
        out = np.empty(self.spectral_shape, dtype=self.cplx)
        self._check(lib().ns_mg_rhs(self._h, ctypes.c_void_p(out.ctypes.data)))
        return out

    def step(self, dt):
        self._check(lib().ns_mg_step(self._h, float(dt)))

    def step_cfl(self, cfl, t_end, return_dt=True):
        dt = ctypes.c_double(0.0)
        self._check(lib().ns_mg_step_cfl(self._h, float(cfl), float(t_end), ctypes.byref(dt) if return_dt else None))
        return dt.value if return_dt else None

    def max_velocity(self):
        v = ctypes.c_double(0.0)
        self._check(lib().ns_mg_max_velocity(self._h, ctypes.byref(v)))
        return v.value

    def time(self):
        return float(lib().ns_mg_time(self._h))

    def exchange_bytes(self):
        return int(lib().ns_mg_exchange_bytes(self._h))

    def kernel_launches(self):
        return int(lib().ns_mg_kernel_launches(self._h))

    def device_bytes(self):
        return int(lib().ns_mg_device_bytes(self._h))


def energy_spectrum_noalloc(u_hat, N, nbins, out=None, stream=None):
    """ns_noalloc_energy_spectrum (include/ns_noalloc.h): shell spectrum of a spectral state held by the caller in DEVICE memory
    (torch CUDA tensor [batch][3][N][N][N/2+1], complex128 or complex64), accumulated in the library's static device scratch: no
    allocation inside the call.  `out`: a torch CUDA float64 tensor or a numpy float64 array [batch][nbins] (default: a new numpy
    array).  batch * nbins <= NS_NOALLOC_MAX_VALUES.  Argument marshalling only."""
    if not _is_torch(u_hat) or not u_hat.is_cuda or not u_hat.is_contiguous():
        raise TypeError("u_hat must be a contiguous torch CUDA tensor")
    batch = int(u_hat.shape[0])
    if tuple(u_hat.shape) != (batch, 3, int(N), int(N), int(N) // 2 + 1):
        raise ValueError(f"u_hat has shape {tuple(u_hat.shape)}, expected [batch][3][N][N][N/2+1]")
    dtype = NS_F64 if u_hat.element_size() == 16 else NS_F32
    if out is None:
        out = np.empty((batch, int(nbins)), dtype=np.float64)
    p, ms, _k = _buf(out, writable=True)
    err = ctypes.create_string_buffer(256)
    rc = lib().ns_noalloc_energy_spectrum(ctypes.c_void_p(u_hat.data_ptr()), int(N), batch, dtype, int(nbins), p, ms,
                                          ctypes.c_void_p(int(stream)) if stream else None, err, 256)
    if rc != NS_OK:
        raise NSError(rc, err.value.decode())
    return out
