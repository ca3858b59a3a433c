"""ctypes wrapper of the CPU oracle (oracle/mg_oracle.cpp).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this.  It imports nothing from the CUDA package.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "mg_oracle.cpp")
_LIB = os.path.join(_HERE, "libmg_oracle.so")
_LIB_OMP = os.path.join(_HERE, "libmg_oracle_omp.so")
_lib = None
_lib_omp = None


def build(force: bool = False) -> str:
    """g++ -O2 -ffp-contract=off (no FMA contraction, no fast-math): plain fp64."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["g++", "-O2", "-ffp-contract=off", "-std=c++17", "-shared", "-fPIC",
                               "-o", _LIB, _SRC])
    return _LIB


def build_omp(force: bool = False) -> str:
    """The same source with -fopenmp: grid loops on all host cores (bench.py's `cpu_baseline_allcores`, a timing line only)."""
    if force or not os.path.exists(_LIB_OMP) or os.path.getmtime(_LIB_OMP) < os.path.getmtime(_SRC):
        subprocess.check_call(["g++", "-O2", "-ffp-contract=off", "-fopenmp", "-std=c++17", "-shared", "-fPIC", "-o", _LIB_OMP, _SRC])
    return _LIB_OMP


def _p(a, ct):
    return None if a is None else a.ctypes.data_as(C.POINTER(ct))


def _declare(_lib):
    _lib.orc_create.restype = C.c_void_p
    _lib.orc_create.argtypes = [C.c_int64, C.c_void_p, C.c_void_p, C.c_void_p, C.c_double,
                                C.c_int, C.c_int, C.c_int, C.c_int, C.c_int]
    _lib.orc_last_error.restype = C.c_char_p
    _lib.orc_level_n.restype = C.c_int64
    _lib.orc_level_h.restype = C.c_double
    for name in ("orc_destroy", "orc_num_levels", "orc_level_n", "orc_level_h", "orc_user_perm",
                 "orc_level_arrays", "orc_transfer_tables", "orc_update", "orc_update3", "orc_level_xi", "orc_level_coeffs",
                 "orc_apply", "orc_smooth", "orc_smooth_group", "orc_restrict", "orc_prolong_correct",
                 "orc_restrict_coeff", "orc_coarse_solve", "orc_cycle", "orc_solve_ex", "orc_solve_bicgstab"):
        getattr(_lib, name).argtypes = None
    return _lib


def lib():
    global _lib
    if _lib is None:
        _lib = _declare(C.CDLL(build()))
    return _lib


def use_openmp(on: bool = True):
    """Route the wrapper to the -fopenmp build (bench.py timing line) or back to the single-threaded oracle."""
    global _lib, _lib_omp
    if on:
        if _lib_omp is None:
            _lib_omp = _declare(C.CDLL(build_omp()))
        _lib = _lib_omp
    else:
        _lib = None


def _d(a):
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a


class Oracle:
    """create / update / solve plus single-step entry points for the pins."""

    def __init__(self, i, j, kind, h, levels=0, nu_pre=2, nu_post=2, m=30, max_iters=200, gamma=1):
        L = lib()
        i = np.ascontiguousarray(i, dtype=np.int32)
        j = np.ascontiguousarray(j, dtype=np.int32)
        kind = np.ascontiguousarray(kind, dtype=np.uint8)
        self.n = int(i.shape[0])
        self._h = L.orc_create(C.c_int64(self.n), i.ctypes.data, j.ctypes.data, kind.ctypes.data,
                               C.c_double(h), int(levels), int(nu_pre), int(nu_post), int(m), int(max_iters))
        if not self._h:
            raise ValueError("oracle: " + L.orc_last_error().decode())
        self._h = C.c_void_p(self._h)
        L.orc_set_gamma(self._h, int(gamma))
        self.levels = L.orc_num_levels(self._h)
        self.m = m
        perm = np.empty(self.n, dtype=np.int64)
        L.orc_user_perm(self._h, C.c_void_p(perm.ctypes.data))
        self.user2canon = perm

    def set_bc_transfer(self, mode):
        """Reading G9 experiment: 1 = transfers renormalised next to Neumann guards inside the cycle, 0 = rules T2 / T3."""
        lib().orc_set_bc_transfer(self._h, int(mode))

    def __del__(self):
        try:
            if getattr(self, "_h", None):
                lib().orc_destroy(self._h)
                self._h = None
        except Exception:
            pass

    # ---- inspection
    def level_n(self, s):
        return int(lib().orc_level_n(self._h, int(s)))

    def level_h(self, s):
        return float(lib().orc_level_h(self._h, int(s)))

    def level_arrays(self, s):
        n = self.level_n(s)
        out = dict(I=np.empty(n, np.int32), J=np.empty(n, np.int32), kind=np.empty(n, np.uint8),
                   colour=np.empty(n, np.uint8), nbr=np.empty((n, 4), np.int32),
                   ns_idx=np.empty((n, 4), np.int32), ns_w=np.empty((n, 4), np.float64),
                   ns_wself=np.empty(n, np.float64), ns_delta=np.empty(n, np.float64),
                   ns_tn=np.empty((n, 2), np.int8), ns_fallback=np.empty(n, np.uint8))
        lib().orc_level_arrays(self._h, int(s), *[C.c_void_p(out[k].ctypes.data) for k in
                               ("I", "J", "kind", "colour", "nbr", "ns_idx", "ns_w", "ns_wself",
                                "ns_delta", "ns_tn", "ns_fallback")])
        return out

    def transfer_tables(self, s):
        nf, nc = self.level_n(s), self.level_n(s + 1)
        out = dict(fine9=np.empty((nc, 9), np.int32), parent=np.empty((nf, 4), np.int32),
                   parent_w=np.empty((nf, 4), np.float64), ptype=np.empty(nf, np.uint8))
        lib().orc_transfer_tables(self._h, int(s), *[C.c_void_p(out[k].ctypes.data) for k in
                                  ("fine9", "parent", "parent_w", "ptype")])
        return out

    def level_coeffs(self, s):
        n = self.level_n(s)
        lam, c = np.empty(n), np.empty(n)
        lib().orc_level_coeffs(self._h, int(s), C.c_void_p(lam.ctypes.data), C.c_void_p(c.ctypes.data))
        return lam, c

    # ---- update / single steps (canonical level order)
    def update(self, lam, c):
        lam, c = _d(lam), _d(c)
        assert lam.shape[0] == self.n and c.shape[0] == self.n
        rc = lib().orc_update(self._h, C.c_void_p(lam.ctypes.data), C.c_void_p(c.ctypes.data))
        if rc != 0:
            raise ValueError("oracle update: " + lib().orc_last_error().decode())

    def update3(self, lam, xi, c):
        """Three-field form lambda*phi - xi*div(c grad phi) = rho (Eq. 3, Eq. 10)."""
        lam, xi, c = _d(lam), _d(xi), _d(c)
        assert lam.shape[0] == self.n and c.shape[0] == self.n and xi.shape[0] == self.n
        rc = lib().orc_update3(self._h, C.c_void_p(lam.ctypes.data), C.c_void_p(xi.ctypes.data), C.c_void_p(c.ctypes.data))
        if rc != 0:
            raise ValueError("oracle update: " + lib().orc_last_error().decode())

    def level_xi(self, s):
        xi = np.empty(self.level_n(s))
        lib().orc_level_xi(self._h, int(s), C.c_void_p(xi.ctypes.data))
        return xi

    def apply(self, s, x):
        x = _d(x); y = np.empty_like(x)
        assert x.shape[0] == self.level_n(s)
        lib().orc_apply(self._h, int(s), C.c_void_p(x.ctypes.data), C.c_void_p(y.ctypes.data))
        return y

    def smooth(self, s, x, b, sweeps=1):
        x = _d(x).copy(); b = _d(b)
        lib().orc_smooth(self._h, int(s), C.c_void_p(x.ctypes.data), C.c_void_p(b.ctypes.data), int(sweeps))
        return x

    def smooth_group(self, s, x, b, group):
        x = _d(x).copy(); b = _d(b)
        lib().orc_smooth_group(self._h, int(s), C.c_void_p(x.ctypes.data), C.c_void_p(b.ctypes.data), int(group))
        return x

    def restrict(self, s, d):
        d = _d(d); out = np.empty(self.level_n(s + 1))
        assert d.shape[0] == self.level_n(s)
        lib().orc_restrict(self._h, int(s), C.c_void_p(d.ctypes.data), C.c_void_p(out.ctypes.data))
        return out

    def prolong_correct(self, s, ec, x):
        ec = _d(ec); x = _d(x).copy()
        assert ec.shape[0] == self.level_n(s + 1) and x.shape[0] == self.level_n(s)
        lib().orc_prolong_correct(self._h, int(s), C.c_void_p(ec.ctypes.data), C.c_void_p(x.ctypes.data))
        return x

    def restrict_coeff(self, s, v):
        v = _d(v); out = np.empty(self.level_n(s + 1))
        lib().orc_restrict_coeff(self._h, int(s), C.c_void_p(v.ctypes.data), C.c_void_p(out.ctypes.data))
        return out

    def coarse_solve(self, b):
        b = _d(b); x = np.empty_like(b)
        lib().orc_coarse_solve(self._h, C.c_void_p(b.ctypes.data), C.c_void_p(x.ctypes.data))
        return x

    def cycle(self, s, x, b):
        x = _d(x).copy(); b = _d(b)
        lib().orc_cycle(self._h, int(s), C.c_void_p(x.ctypes.data), C.c_void_p(b.ctypes.data))
        return x

    # ---- solve (user order)
    def solve(self, f, x0, rtol, precond=0, debug=False):
        f, x0 = _d(f), _d(x0)
        x = np.empty(self.n)
        iters, relres = C.c_int(0), C.c_double(0.0)
        hist = np.zeros(4096)
        V = Z = H = None
        ncols = C.c_int(0)
        if debug:
            V = np.zeros((self.m + 1, self.n)); Z = np.zeros((self.m, self.n)); H = np.zeros((self.m + 1, self.m))
        vp = lambda a: C.c_void_p(a.ctypes.data) if a is not None else None
        st = lib().orc_solve_ex(self._h, vp(f), vp(x0), vp(x), C.c_double(rtol), int(precond),
                                C.byref(iters), C.byref(relres), vp(hist), vp(V), vp(Z), vp(H), C.byref(ncols))
        if st < 0:
            raise RuntimeError("oracle solve: " + lib().orc_last_error().decode())
        res = dict(x=x, iters=iters.value, relres=relres.value, status=st, hist=hist[:iters.value].copy())
        if debug:
            k = ncols.value
            res.update(V=V[:k + 1], Z=Z[:k], H=H[:k + 1, :k], ncols=k)
        return res

    def solve_bicgstab(self, f, x0, rtol, precond=0):
        """BiCGStab with the V-cycle as right preconditioner; iters counts preconditioner applications."""
        f, x0 = _d(f), _d(x0)
        x = np.empty(self.n)
        iters, relres = C.c_int(0), C.c_double(0.0)
        hist = np.zeros(8192)
        vp = lambda a: C.c_void_p(a.ctypes.data)
        st = lib().orc_solve_bicgstab(self._h, vp(f), vp(x0), vp(x), C.c_double(rtol), int(precond), C.byref(iters), C.byref(relres), vp(hist))
        if st < 0:
            raise RuntimeError("oracle bicgstab: " + lib().orc_last_error().decode())
        return dict(x=x, iters=iters.value, relres=relres.value, status=st, hist=hist[:iters.value].copy())
