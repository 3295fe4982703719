"""ctypes wrapper around oracle/vog_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this module.  It holds no arithmetic of its own: every number comes
from the C functions in vog_oracle.c (double precision, no FFT in any advection), each
of which cites the passage of the paper it restates.  Arrays are numpy float64,
row-major [Nv][Nx] (f[j, i] = value at (x_i, v_j)).
"""
import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "vog_oracle.c")
_LIB = os.path.join(_HERE, "libvog_oracle.so")

LAGRANGE = 0
BSPLINE = 1
SPLIT_XVX = 0
SPLIT_VXV = 1


class Feq(ctypes.Structure):
    """f_eq(v) = sum_g amp_g exp(-c_g (v - mu_g)^2); n = 0 means full-f."""
    _fields_ = [("n", ctypes.c_int), ("amp", ctypes.c_double * 4),
                ("mu", ctypes.c_double * 4), ("c", ctypes.c_double * 4)]

    @staticmethod
    def make(gaussians):
        q = Feq()
        q.n = len(gaussians)
        for g, (amp, mu, c) in enumerate(gaussians):
            q.amp[g], q.mu[g], q.c[g] = amp, mu, c
        return q


def build(force=False):
    """Compile the oracle with gcc (-O2 -fopenmp).  Building the checker is not using it."""
    if (not force and os.path.exists(_LIB)
            and os.path.getmtime(_LIB) >= os.path.getmtime(_SRC)):
        return _LIB
    subprocess.check_call(["gcc", "-O2", "-fopenmp", "-shared", "-fPIC", "-o", _LIB, _SRC, "-lm"])
    return _LIB


_lib = None
_dp = ctypes.POINTER(ctypes.c_double)


def lib():
    global _lib
    if _lib is None:
        build()
        L = ctypes.CDLL(_LIB)
        L.oracle_num_threads.restype = ctypes.c_int
        L.oracle_bspline.restype = ctypes.c_double
        L.oracle_bspline.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_double]
        L.oracle_electric_energy.restype = ctypes.c_double
        L.oracle_electric_energy.argtypes = [ctypes.c_int, _dp, ctypes.c_double]
        L.oracle_feq.restype = ctypes.c_double
        L.oracle_feq.argtypes = [ctypes.POINTER(Feq), ctypes.c_double]
        _lib = L
    return _lib


def _p(a):
    return a.ctypes.data_as(_dp)


def _c(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def num_threads():
    return int(lib().oracle_num_threads())


def split_shift(beta):
    b = ctypes.c_long()
    bs = ctypes.c_double()
    lib().oracle_split_shift(ctypes.c_double(beta), ctypes.byref(b), ctypes.byref(bs))
    return int(b.value), float(bs.value)


def lagrange_weights(d, bstar):
    w = np.zeros(2 * d + 2)
    lib().oracle_lagrange_weights(ctypes.c_int(d), ctypes.c_double(bstar), _p(w))
    return w


def bspline(i, k, x):
    return float(lib().oracle_bspline(i, k, x))


def lagrange_first_row(N, d, beta):
    a = np.zeros(N)
    lib().oracle_lagrange_first_row(ctypes.c_int(N), ctypes.c_int(d), ctypes.c_double(beta), _p(a))
    return a


def circulant(a):
    a = _c(a)
    N = a.size
    A = np.zeros((N, N))
    lib().oracle_circulant(ctypes.c_int(N), _p(a), _p(A))
    return A


def spline_first_rows(N, k, beta):
    cc = np.zeros(N)
    mm = np.zeros(N)
    lib().oracle_spline_first_rows(ctypes.c_int(N), ctypes.c_int(k), ctypes.c_double(beta), _p(cc), _p(mm))
    return cc, mm


def spline_dense_matrix(N, k, beta):
    A = np.zeros((N, N))
    rc = lib().oracle_spline_dense_matrix(ctypes.c_int(N), ctypes.c_int(k), ctypes.c_double(beta), _p(A))
    if rc:
        raise ArithmeticError("singular collocation matrix")
    return A


def advect_line(u, beta, kind, order):
    u = _c(u)
    out = np.zeros_like(u)
    rc = lib().oracle_advect_line(ctypes.c_int(u.size), _p(u), ctypes.c_long(1), ctypes.c_double(beta),
                                  ctypes.c_int(kind), ctypes.c_int(order), _p(out), ctypes.c_long(1))
    if rc:
        raise ValueError("bad kind/order")
    return out


def shift_x(f, beta, kind, order):
    f = _c(f)
    beta = _c(beta)
    Nv, Nx = f.shape
    assert beta.size == Nv
    out = np.empty_like(f)
    rc = lib().oracle_shift_x(ctypes.c_int(Nx), ctypes.c_int(Nv), _p(f), _p(beta),
                              ctypes.c_int(kind), ctypes.c_int(order), _p(out))
    if rc:
        raise ValueError("bad kind/order")
    return out


def shift_v(f, beta, kind, order):
    f = _c(f)
    beta = _c(beta)
    Nv, Nx = f.shape
    assert beta.size == Nx
    out = np.empty_like(f)
    rc = lib().oracle_shift_v(ctypes.c_int(Nx), ctypes.c_int(Nv), _p(f), _p(beta),
                              ctypes.c_int(kind), ctypes.c_int(order), _p(out))
    if rc:
        raise ValueError("bad kind/order")
    return out


def advect_x(f, L, vmin, vmax, dt, kind, order):
    f = _c(f)
    Nv, Nx = f.shape
    out = np.empty_like(f)
    rc = lib().oracle_advect_x(ctypes.c_int(Nx), ctypes.c_int(Nv), _p(f), ctypes.c_double(L),
                               ctypes.c_double(vmin), ctypes.c_double(vmax), ctypes.c_double(dt),
                               ctypes.c_int(kind), ctypes.c_int(order), _p(out))
    if rc:
        raise ValueError("bad kind/order")
    return out


def advect_v(f, E, vmin, vmax, dt, kind, order, feq=None):
    f = _c(f)
    E = _c(E)
    Nv, Nx = f.shape
    assert E.size == Nx
    out = np.empty_like(f)
    q = feq if feq is not None else Feq.make([])
    rc = lib().oracle_advect_v(ctypes.c_int(Nx), ctypes.c_int(Nv), _p(f), _p(E), ctypes.c_double(vmin),
                               ctypes.c_double(vmax), ctypes.c_double(dt), ctypes.c_int(kind),
                               ctypes.c_int(order), ctypes.byref(q), _p(out))
    if rc:
        raise ValueError("bad kind/order")
    return out


def feq_eval(feq, v):
    return float(lib().oracle_feq(ctypes.byref(feq), ctypes.c_double(v)))


def density(f, vmin, vmax):
    f = _c(f)
    Nv, Nx = f.shape
    rho = np.zeros(Nx)
    lib().oracle_density(ctypes.c_int(Nx), ctypes.c_int(Nv), _p(f), ctypes.c_double(vmin),
                         ctypes.c_double(vmax), _p(rho))
    return rho


def poisson(rho, L):
    rho = _c(rho)
    E = np.zeros_like(rho)
    lib().oracle_poisson(ctypes.c_int(rho.size), _p(rho), ctypes.c_double(L), _p(E))
    return E


def field(f, L, vmin, vmax):
    f = _c(f)
    Nv, Nx = f.shape
    E = np.zeros(Nx)
    lib().oracle_field(ctypes.c_int(Nx), ctypes.c_int(Nv), _p(f), ctypes.c_double(L),
                       ctypes.c_double(vmin), ctypes.c_double(vmax), _p(E))
    return E


def field_trapezoid(rho, L, zero_mean=True, background=0.0):
    """trapezoidal rule for E from rho, with (default) or without the zero-mean modifications."""
    rho = _c(rho)
    E = np.zeros_like(rho)
    lib().oracle_field_trapezoid(ctypes.c_int(rho.size), _p(rho), ctypes.c_double(L), ctypes.c_int(1 if zero_mean else 0),
                                 ctypes.c_double(background), _p(E))
    return E


def rho_modes(rho):
    """(rho^_0, |rho^_1|) of P:245, 261."""
    rho = _c(rho)
    out = np.zeros(2)
    lib().oracle_rho_modes(ctypes.c_int(rho.size), _p(rho), _p(out))
    return float(out[0]), float(out[1])


def kinetic_energy(f, L, vmin, vmax):
    f = _c(f)
    Nv, Nx = f.shape
    lib().oracle_kinetic_energy.restype = ctypes.c_double
    return float(lib().oracle_kinetic_energy(ctypes.c_int(Nx), ctypes.c_int(Nv), _p(f), ctypes.c_double(L),
                                             ctypes.c_double(vmin), ctypes.c_double(vmax)))


def electric_energy(E, L):
    E = _c(E)
    return float(lib().oracle_electric_energy(ctypes.c_int(E.size), _p(E), ctypes.c_double(L)))


def step(f, L, vmin, vmax, dt, kind, order, feq=None, split=SPLIT_XVX, E_ext=None, E_in=None):
    """One Strang step.  Returns (f_new, E_self_consistent_used)."""
    f = _c(f).copy()
    Nv, Nx = f.shape
    q = feq if feq is not None else Feq.make([])
    E_out = np.zeros(Nx)
    work = np.empty_like(f)
    ext = _c(E_ext) if E_ext is not None else None
    ein = _c(E_in) if E_in is not None else None
    if split == SPLIT_VXV and ein is None:
        ein = field(f, L, vmin, vmax)
    rc = lib().oracle_step(ctypes.c_int(Nx), ctypes.c_int(Nv), _p(f), ctypes.c_double(L),
                           ctypes.c_double(vmin), ctypes.c_double(vmax), ctypes.c_double(dt),
                           ctypes.c_int(kind), ctypes.c_int(order), ctypes.byref(q), ctypes.c_int(split),
                           _p(ext) if ext is not None else None,
                           _p(ein) if ein is not None else None, _p(E_out), _p(work))
    if rc:
        raise ValueError("bad kind/order")
    return f, E_out
