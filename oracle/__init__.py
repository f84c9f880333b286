"""ctypes binding of the CPU ORACLE (oracle/phx_oracle.cpp).

TEST INFRASTRUCTURE, NOT PRODUCT.  Only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference leg may import this package.  It does not import the CUDA
package and the CUDA package does not import it.  All state is numpy float64 / complex128.
"""
import ctypes as C
import os

import numpy as np

from . import build as _build

NCOEF = 18
COEF_NAMES = ("cx", "cy", "ih", "g", "gx", "gr", "Rr", "hgc", "gamr", "bxx", "byy", "bxy", "dt", "dt6", "dt3",
              "sig2", "doff", "omega")


class Params(C.Structure):
    """Mirror of orc_params (Eqs. (1), (16), (17), (22) of the paper)."""
    _fields_ = [(k, C.c_double) for k in ("hbar", "m", "g", "g_x", "g_r", "R", "gamma_c", "gamma_r", "beta", "dt",
                                          "noise_scale", "density_offset", "omega")]


class _Problem(C.Structure):
    _fields_ = [("nx", C.c_int32), ("ny", C.c_int32), ("batch", C.c_int32), ("spinor", C.c_int32),
                ("reservoir", C.c_int32), ("noise", C.c_int32), ("bc_x", C.c_int32), ("bc_y", C.c_int32),
                ("seed", C.c_uint32), ("coef", C.c_double * NCOEF), ("V", C.c_void_p), ("P", C.c_void_p),
                ("E", C.c_void_p), ("first_realisation", C.c_uint32)]


_lib = None


_omp = False


def select_build(openmp: bool):
    """openmp=True: use liboracle_omp.so (the same source with its OpenMP pragmas honoured) -- bench.py's all-cores
    cpu_baseline leg only; the parity oracle is the single-threaded build (the default)."""
    global _lib, _omp
    if bool(openmp) != _omp:
        _lib, _omp = None, bool(openmp)


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build.build_omp() if _omp else _build.build())
        _lib.orc_step_rk4.restype = C.c_int32
        _lib.orc_step_rk4.argtypes = [C.c_void_p] * 5 + [C.c_uint64, C.c_int64]
        _lib.orc_derivative.restype = None
        _lib.orc_derivative.argtypes = [C.c_void_p, C.c_double] + [C.c_void_p] * 8
        _lib.orc_derive_coeffs.restype = None
        _lib.orc_derive_coeffs.argtypes = [C.c_void_p, C.c_double, C.c_double, C.c_int32, C.c_void_p]
        _lib.orc_noise_u32.restype = None
        _lib.orc_noise_u32.argtypes = [C.c_int32, C.c_int32, C.c_int32, C.c_uint32, C.c_uint64, C.c_void_p]
        _lib.orc_normal_pair.restype = None
        _lib.orc_normal_pair.argtypes = [C.c_uint32, C.c_uint32, C.c_void_p, C.c_void_p]
        _lib.orc_philox4x32_10.restype = None
        _lib.orc_philox4x32_10.argtypes = [C.c_void_p] * 3
        _lib.orc_ensemble_mean_density.restype = None
        _lib.orc_ensemble_mean_density.argtypes = [C.c_int32] * 3 + [C.c_void_p] * 2
        _lib.orc_dp54_tableau.restype = None
        _lib.orc_dp54_tableau.argtypes = [C.c_int32] + [C.c_void_p] * 4
        _lib.orc_step_dp54.restype = C.c_int32
        _lib.orc_step_dp54.argtypes = [C.c_void_p] * 7 + [C.c_int32] + [C.c_void_p] * 4 + [C.c_int64, C.c_void_p]
    return _lib


def _ptr(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def make_params(**kw) -> Params:
    d = dict(hbar=1.0, m=0.5, g=0.0, g_x=0.0, g_r=0.0, R=0.0, gamma_c=0.0, gamma_r=0.0, beta=0.0, dt=0.0,
             noise_scale=1.0, density_offset=0.0, omega=0.0)
    for k in kw:
        if k not in d:
            raise KeyError(k)
    d.update(kw)
    return Params(**d)


def derive_coeffs(params: Params, dx: float, dy: float, prec32: bool) -> np.ndarray:
    out = np.zeros(NCOEF, dtype=np.float64)
    lib().orc_derive_coeffs(C.byref(params), dx, dy, int(bool(prec32)), _ptr(out))
    return out


class Adaptive(C.Structure):
    """Mirror of orc_adaptive (reading Q20)."""
    _fields_ = [("atol", C.c_double), ("rtol", C.c_double), ("h_init", C.c_double), ("h_min", C.c_double),
                ("h_max", C.c_double), ("t_end", C.c_double), ("max_attempts", C.c_int64)]


class AdaptiveState(C.Structure):
    _fields_ = [("t", C.c_double), ("h_next", C.c_double), ("n_accept", C.c_int64), ("n_reject", C.c_int64)]


def dp54_tableau(prec32=False):
    """(c[7], a[7][7], b[7], e[7]) of the Dormand-Prince 5(4) pair as the oracle uses them."""
    c, a, b, e = np.zeros(7), np.zeros((7, 7)), np.zeros(7), np.zeros(7)
    lib().orc_dp54_tableau(int(bool(prec32)), _ptr(c), _ptr(a), _ptr(b), _ptr(e))
    return c, a, b, e


class Oracle:
    """One oracle problem: grid, model switches, canonical coefficients, static fields, state.

    model: "scalar" | "reservoir" | "spinor" | "spinor_reservoir".
    prec32=True rounds the derived coefficients once to float (the arithmetic stays double).
    """

    def __init__(self, nx, ny, dx, dy, params, model="scalar", batch=1, prec32=False, noise=False, seed=0,
                 bc=(0, 0), V=None, P=None, E=None, coef=None, first_realisation=0):
        self.nx, self.ny, self.batch = int(nx), int(ny), int(batch)
        self.model = model
        self.spinor = model in ("spinor", "spinor_reservoir")
        self.reservoir = model in ("reservoir", "spinor_reservoir")
        if model not in ("scalar", "reservoir", "spinor", "spinor_reservoir"):
            raise ValueError(model)
        self.coef = derive_coeffs(params, dx, dy, prec32) if coef is None else np.asarray(coef, np.float64).copy()
        self.V = None if V is None else np.ascontiguousarray(V, dtype=np.float64).reshape(ny, nx)
        self.P = None if P is None else np.ascontiguousarray(P, dtype=np.float64).reshape(ny, nx)
        self.E = None if E is None else np.ascontiguousarray(E, dtype=np.complex128).reshape(ny, nx)
        self.pb = _Problem(self.nx, self.ny, self.batch, int(self.spinor), int(self.reservoir), int(bool(noise)),
                           int(bc[0]), int(bc[1]), int(seed), (C.c_double * NCOEF)(*self.coef), _ptr(self.V),
                           _ptr(self.P), _ptr(self.E), int(first_realisation))
        shape = (self.batch, self.ny, self.nx)
        self.psi_p = np.zeros(shape, np.complex128)
        self.psi_m = np.zeros(shape, np.complex128) if self.spinor else None
        self.n_p = np.zeros(shape, np.float64) if self.reservoir else None
        self.n_m = np.zeros(shape, np.float64) if (self.reservoir and self.spinor) else None
        self.step = 0
        self.prec32 = bool(prec32)
        self.ad = AdaptiveState(0.0, 0.0, 0, 0)          # adaptive integrator: time, next step size, counters

    def step_dp54(self, t_end, atol, rtol, h_init, h_min=1e-12, h_max=1e30, max_attempts=1 << 40, log_cap=1 << 16):
        """Adaptive Dormand-Prince 5(4) from self.ad.t to t_end; returns the attempt log (accept, q, h, err)."""
        ctl = Adaptive(atol, rtol, h_init, h_min, h_max, t_end, max_attempts)
        acc, q = np.zeros(log_cap, np.int32), np.zeros(log_cap, np.int32)
        h, err = np.zeros(log_cap), np.zeros(log_cap)
        n = C.c_int64(0)
        rc = lib().orc_step_dp54(C.byref(self.pb), _ptr(self.psi_p), _ptr(self.psi_m), _ptr(self.n_p), _ptr(self.n_m),
                                 C.byref(ctl), C.byref(self.ad), int(self.prec32), _ptr(acc), _ptr(q), _ptr(h), _ptr(err),
                                 log_cap, C.byref(n))
        if rc != 0:
            raise RuntimeError(f"orc_step_dp54: status {rc}")
        k = min(n.value, log_cap)
        return {"accept": acc[:k], "q": q[:k], "h": h[:k], "err": err[:k], "attempts": n.value}

    def set_field(self, name, arr):
        dst = getattr(self, name)
        if dst is None:
            raise ValueError(f"field {name} not present in model {self.model}")
        dst[...] = np.asarray(arr).reshape(dst.shape)

    def step_rk4(self, n_steps=1):
        rc = lib().orc_step_rk4(C.byref(self.pb), _ptr(self.psi_p), _ptr(self.psi_m), _ptr(self.n_p),
                                _ptr(self.n_m), self.step, int(n_steps))
        if rc != 0:
            raise RuntimeError("orc_step_rk4: bad arguments")
        self.step += int(n_steps)

    def derivative(self, t=0.0, r=0):
        """K (and Kn) of batch element r at time t; returns dict of arrays [ny][nx]."""
        out = {}
        Kp = np.zeros((self.ny, self.nx), np.complex128)
        Km = np.zeros_like(Kp) if self.spinor else None
        Knp = np.zeros((self.ny, self.nx), np.float64) if self.reservoir else None
        Knm = np.zeros_like(Knp) if (self.reservoir and self.spinor) else None
        sel = lambda a: None if a is None else np.ascontiguousarray(a[r])
        a, b, c, d = sel(self.psi_p), sel(self.psi_m), sel(self.n_p), sel(self.n_m)
        lib().orc_derivative(C.byref(self.pb), float(t), _ptr(a), _ptr(b), _ptr(c), _ptr(d), _ptr(Kp), _ptr(Km),
                             _ptr(Knp), _ptr(Knm))
        out.update(K_p=Kp, K_m=Km, Kn_p=Knp, Kn_m=Knm)
        return out

    def ensemble_mean_density(self, name="psi_p"):
        out = np.zeros((self.ny, self.nx), np.float64)
        psi = np.ascontiguousarray(getattr(self, name))
        lib().orc_ensemble_mean_density(self.nx, self.ny, self.batch, _ptr(psi), _ptr(out))
        return out


def philox4x32_10(ctr, key):
    c = np.asarray(ctr, dtype=np.uint32).copy()
    k = np.asarray(key, dtype=np.uint32).copy()
    out = np.zeros(4, dtype=np.uint32)
    lib().orc_philox4x32_10(_ptr(c), _ptr(k), _ptr(out))
    return out


def noise_u32(nx, ny, batch, seed, step):
    out = np.zeros((batch, ny, nx, 4), dtype=np.uint32)
    lib().orc_noise_u32(nx, ny, batch, int(seed), int(step), _ptr(out))
    return out


def normal_pair(w0, w1):
    a, b = C.c_double(), C.c_double()
    lib().orc_normal_pair(int(w0), int(w1), C.byref(a), C.byref(b))
    return a.value, b.value
