"""ctypes wrapper of the TWO-DIMENSIONAL CPU oracle (oracle/ns2d_oracle.cpp).  TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's oracle legs may import this.  Spectral arrays are numpy complex128
[2][N][N/2+1] (index [comp][ikx][iky], iky >= 0 fastest); physical arrays float64 [2][N][N].
"""
from __future__ import annotations

import ctypes

import numpy as np

from . import ns_oracle as _o3

Params = _o3.Params
_lib = _o3._lib
d, i, p = ctypes.c_double, ctypes.c_int, ctypes.c_void_p
_lib.orc2_fft2d.argtypes = [i, i, p]
_lib.orc2_rhs_parts.argtypes = [i, i, d, d, d, d, d, i, p, p, p, p, p]
_lib.orc2_step.argtypes = [i, i, d, d, d, d, d, i, p, d]
_lib.orc2_set_initial.argtypes = [i, p, p]
_lib.orc2_get_fields.argtypes = [i, p, p]
_lib.orc2_max_velocity.argtypes = [i, i, p]
_lib.orc2_max_velocity.restype = d
_lib.orc2_spectrum.argtypes = [i, p, i, i, p]


def _ptr(a):
    return a.ctypes.data_as(ctypes.c_void_p)


def _c128(a):
    return np.ascontiguousarray(a, dtype=np.complex128)


def spectral_shape(N):
    return (2, N, N // 2 + 1)


def fft2d(a, sign):
    a = _c128(a).copy()
    n = a.shape[0]
    assert a.shape == (n, n)
    _lib.orc2_fft2d(n, sign, _ptr(a))
    return a


def rhs_parts(N, params: Params, u_hat, M=None):
    M = 3 * N // 2 if M is None else M
    u_hat = _c128(u_hat)
    assert u_hat.shape == spectral_shape(N)
    b, n, r = np.empty_like(u_hat), np.empty_like(u_hat), np.empty_like(u_hat)
    umax = ctypes.c_double(0.0)
    _lib.orc2_rhs_parts(N, M, *params.args(), _ptr(u_hat), _ptr(b), _ptr(n), _ptr(r), ctypes.byref(umax))
    return dict(b=b, n=n, r=r, umax=umax.value)


def rhs(N, params: Params, u_hat, M=None):
    return rhs_parts(N, params, u_hat, M)["r"]


def step(N, params: Params, u_hat, dt, M=None):
    M = 3 * N // 2 if M is None else M
    u = _c128(u_hat).copy()
    assert u.shape == spectral_shape(N)
    _lib.orc2_step(N, M, *params.args(), _ptr(u), float(dt))
    return u


def set_initial(N, u_phys):
    u_phys = np.ascontiguousarray(u_phys, dtype=np.float64)
    assert u_phys.shape == (2, N, N)
    out = np.empty(spectral_shape(N), dtype=np.complex128)
    _lib.orc2_set_initial(N, _ptr(u_phys), _ptr(out))
    return out


def get_fields(N, u_hat):
    u_hat = _c128(u_hat)
    out = np.empty((2, N, N), dtype=np.float64)
    _lib.orc2_get_fields(N, _ptr(u_hat), _ptr(out))
    return out


def max_velocity(N, u_hat, M=None):
    M = 3 * N // 2 if M is None else M
    return float(_lib.orc2_max_velocity(N, M, _ptr(_c128(u_hat))))


def energy_spectrum(N, u_hat, nbins):
    E = np.empty(nbins, dtype=np.float64)
    _lib.orc2_spectrum(N, _ptr(_c128(u_hat)), nbins, 0, _ptr(E))
    return E


def enstrophy_spectrum(N, u_hat, nbins):
    Z = np.empty(nbins, dtype=np.float64)
    _lib.orc2_spectrum(N, _ptr(_c128(u_hat)), nbins, 1, _ptr(Z))
    return Z
