"""ctypes wrapper of the CPU oracle (oracle/ns_oracle.cpp).  TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this.  It imports nothing from the CUDA package.  Spectral arrays are numpy complex128
[3][N][N][N/2+1]; physical arrays float64 [3][N][N][N].
"""
from __future__ import annotations

import ctypes
import importlib.util
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))


def _load():
    spec = importlib.util.spec_from_file_location("_ns_oracle_build", os.path.join(_HERE, "build.py"))
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    lib = ctypes.CDLL(mod.build())
    d, i, p = ctypes.c_double, ctypes.c_int, ctypes.c_void_p
    lib.orc_num_threads.restype = i
    lib.orc_dft1d.argtypes = [i, i, p, p]
    lib.orc_fft1d.argtypes = [i, i, p, p]
    lib.orc_fft3d.argtypes = [i, i, p]
    lib.orc_dissipation.argtypes = [i, d, d, d, d, d, i, d]
    lib.orc_dissipation.restype = d
    lib.orc_rhs_parts.argtypes = [i, i, d, d, d, d, d, i, p, p, p, p, p]
    lib.orc_rhs_at_modes.argtypes = [i, d, d, d, d, d, i, p, i, p, p]
    lib.orc_step.argtypes = [i, i, d, d, d, d, d, i, p, d]
    lib.orc_set_initial.argtypes = [i, p, p]
    lib.orc_get_fields.argtypes = [i, p, p]
    lib.orc_max_velocity.argtypes = [i, i, p]
    lib.orc_max_velocity.restype = d
    lib.orc_energy_spectrum.argtypes = [i, p, i, p]
    lib.orc_enstrophy_spectrum.argtypes = [i, p, i, p]
    lib.orc_structure_function.argtypes = [i, p, i, p]
    lib.orc_structure_function_p.argtypes = [i, p, ctypes.c_double, i, p]
    return lib


_lib = _load()


class Params:
    """Same fields as ns_params in include/ns.h (plain numbers; no shared code)."""

    def __init__(self, nu=0.0, eps=0.0, s=1.0, m_cut=-1.0, q_exp=-1.0, q_sharp=0):
        self.nu, self.eps, self.s, self.m_cut, self.q_exp, self.q_sharp = nu, eps, s, m_cut, q_exp, q_sharp

    def args(self):
        return (float(self.nu), float(self.eps), float(self.s), float(self.m_cut), float(self.q_exp), int(self.q_sharp))


def _ptr(a):
    return a.ctypes.data_as(ctypes.c_void_p)


def _c128(a):
    return np.ascontiguousarray(a, dtype=np.complex128)


def num_threads() -> int:
    return int(_lib.orc_num_threads())


def dft1d(x, sign):
    x = _c128(x)
    out = np.empty_like(x)
    _lib.orc_dft1d(x.size, sign, _ptr(x), _ptr(out))
    return out


def fft1d(x, sign):
    x = _c128(x)
    out = np.empty_like(x)
    _lib.orc_fft1d(x.size, sign, _ptr(x), _ptr(out))
    return out


def fft3d(a, sign):
    a = _c128(a).copy()
    n = a.shape[0]
    assert a.shape == (n, n, n)
    _lib.orc_fft3d(n, sign, _ptr(a))
    return a


def dissipation(N, params: Params, k2: float) -> float:
    return float(_lib.orc_dissipation(N, *params.args(), float(k2)))


def spectral_shape(N):
    return (3, N, N, N // 2 + 1)


def rhs_parts(N, params: Params, u_hat, M=None):
    """Returns dict(b=, n=, r=, umax=) -- b: unprojected divergence term, n: projected, r: full RHS."""
    M = 3 * N // 2 if M is None else M
    u_hat = _c128(u_hat)
    assert u_hat.shape == spectral_shape(N)
    b = np.empty_like(u_hat)
    n = np.empty_like(u_hat)
    r = np.empty_like(u_hat)
    umax = ctypes.c_double(0.0)
    _lib.orc_rhs_parts(N, M, *params.args(), _ptr(u_hat), _ptr(b), _ptr(n), _ptr(r), ctypes.byref(umax))
    return dict(b=b, n=n, r=r, umax=umax.value)


def rhs(N, params: Params, u_hat, M=None):
    return rhs_parts(N, params, u_hat, M)["r"]


def rhs_at_modes(N, params: Params, u_hat, modes):
    """R_hat at the stored indices modes[n] = (ix, iy, iz) by the direct truncated convolution sum; returns [n][3]."""
    u_hat = _c128(u_hat)
    assert u_hat.shape == spectral_shape(N)
    modes = np.ascontiguousarray(modes, dtype=np.int32)
    assert modes.ndim == 2 and modes.shape[1] == 3
    out = np.empty((modes.shape[0], 3), dtype=np.complex128)
    _lib.orc_rhs_at_modes(N, *params.args(), _ptr(u_hat), modes.shape[0], _ptr(modes), _ptr(out))
    return out


def step(N, params: Params, u_hat, dt, M=None):
    M = 3 * N // 2 if M is None else M
    u = _c128(u_hat).copy()
    assert u.shape == spectral_shape(N)
    _lib.orc_step(N, M, *params.args(), _ptr(u), float(dt))
    return u


def set_initial(N, u_phys):
    u_phys = np.ascontiguousarray(u_phys, dtype=np.float64)
    assert u_phys.shape == (3, N, N, N)
    out = np.empty(spectral_shape(N), dtype=np.complex128)
    _lib.orc_set_initial(N, _ptr(u_phys), _ptr(out))
    return out


def get_fields(N, u_hat):
    u_hat = _c128(u_hat)
    out = np.empty((3, N, N, N), dtype=np.float64)
    _lib.orc_get_fields(N, _ptr(u_hat), _ptr(out))
    return out


def max_velocity(N, u_hat, M=None):
    M = 3 * N // 2 if M is None else M
    u_hat = _c128(u_hat)
    return float(_lib.orc_max_velocity(N, M, _ptr(u_hat)))


def energy_spectrum(N, u_hat, nbins):
    u_hat = _c128(u_hat)
    E = np.empty(nbins, dtype=np.float64)
    _lib.orc_energy_spectrum(N, _ptr(u_hat), nbins, _ptr(E))
    return E


def enstrophy_spectrum(N, u_hat, nbins):
    u_hat = _c128(u_hat)
    Z = np.empty(nbins, dtype=np.float64)
    _lib.orc_enstrophy_spectrum(N, _ptr(u_hat), nbins, _ptr(Z))
    return Z


def structure_function(N, u_hat, nl=None):
    nl = N // 2 if nl is None else nl
    u_hat = _c128(u_hat)
    S = np.empty(nl, dtype=np.float64)
    _lib.orc_structure_function(N, _ptr(u_hat), nl, _ptr(S))
    return S


def structure_function_p(N, u_hat, p, nl=None):
    nl = N // 2 if nl is None else nl
    u_hat = _c128(u_hat)
    S = np.empty(nl, dtype=np.float64)
    _lib.orc_structure_function_p(N, _ptr(u_hat), float(p), nl, _ptr(S))
    return S
