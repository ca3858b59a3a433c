"""Thin ctypes binding of libmg_b200.so (include/mg_b200.h): argument marshalling only.

PyTorch is used for device memory (tensors, caching allocator) and streams; every step of the path
runs in the library's CUDA kernels.  There is no CPU fallback: if the library cannot be built/loaded
or no CUDA device is present, calls raise.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIBPATH = os.path.join(_HERE, "libmg_b200.so")
_lib = None
_alloc_cb = None
_free_cb = None

MG_OK, MG_NOT_CONVERGED, MG_BREAKDOWN = 0, 1, 2


class MgError(RuntimeError):
    def __init__(self, code, where):
        L = lib()
        super().__init__(f"{where}: {L.mg_strerror(code).decode()} ({code}); {L.mg_last_error().decode()}")
        self.code = code


NOALLOC_MAX_N = 268435456          # MG_NOALLOC_MAX_N of include/mg_b200.h


def norm2_noalloc(v, out=None, stream=None):
    """mg_norm2_noalloc: ||v||_2 of a CUDA fp64 tensor into the 1-element CUDA tensor `out`, no allocation inside the library
    (pass `out` to allocate nothing here either).  Asynchronous; returns `out`."""
    import torch
    if out is None:
        out = torch.empty(1, dtype=torch.float64, device=v.device)
    assert v.is_cuda and v.dtype == torch.float64 and v.is_contiguous() and out.is_cuda and out.dtype == torch.float64
    rc = lib().mg_norm2_noalloc(C.c_void_p(v.data_ptr()), C.c_int64(v.numel()), C.c_void_p(out.data_ptr()), _stream_ptr(stream))
    if rc:
        raise MgError(rc, "mg_norm2_noalloc")
    return out


def last_error() -> str:
    """mg_last_error(): the calling thread's last error / diagnostic text."""
    return lib().mg_last_error().decode()


class _Mesh(C.Structure):
    _fields_ = [("n", C.c_int64), ("i", C.c_void_p), ("j", C.c_void_p), ("h", C.c_double)]


class _Bc(C.Structure):
    _fields_ = [("kind", C.c_void_p)]


class _Options(C.Structure):
    _fields_ = [("levels", C.c_int), ("nu_pre", C.c_int), ("nu_post", C.c_int), ("restart_m", C.c_int),
                ("max_iters", C.c_int), ("flags", C.c_int), ("gamma", C.c_int), ("planes", C.c_int), ("solver", C.c_int)]


EXPORTS = ["mg_set_allocator", "mg_setup", "mg_update_coeffs", "mg_update_coeffs3", "mg_update_coeffs3_host", "mg_level_xi", "mg_solve", "mg_update_coeffs_host",
           "mg_solve_host", "mg_destroy", "mg_num_levels", "mg_level_n", "mg_level_info", "mg_transfer_info",
           "mg_level_coeffs", "mg_apply", "mg_smooth", "mg_restrict", "mg_smooth_restrict", "mg_prolong_correct", "mg_coarse_solve",
           "mg_vcycle", "mg_kernel_launches", "mg_last_solve_ms", "mg_last_update_ms", "mg_last_step_ms", "mg_last_reorth", "mg_last_history", "mg_strerror",
           "mg_last_error", "mg_norm2_noalloc"]


def lib():
    """Loads (building if needed) the CUDA library. Fails loudly if that is impossible."""
    global _lib
    if _lib is None:
        if not os.path.exists(_LIBPATH):
            from . import build as _b
            _b.build()
        L = C.CDLL(_LIBPATH)
        L.mg_strerror.restype = C.c_char_p
        L.mg_last_error.restype = C.c_char_p
        L.mg_level_n.restype = C.c_int64
        L.mg_kernel_launches.restype = C.c_int64
        L.mg_last_solve_ms.restype = C.c_double
        L.mg_last_update_ms.restype = C.c_double
        L.mg_last_step_ms.restype = C.c_double
        _lib = L
    return _lib


def use_torch_allocator():
    """Route the library's device allocations through torch's CUDA caching allocator.  The callback objects are created once and
    kept for the life of the process: a handle keeps the function pointers it was created with (mg_set_allocator)."""
    global _alloc_cb, _free_cb
    import torch
    if _alloc_cb is None:
        AF = C.CFUNCTYPE(C.c_void_p, C.c_uint64, C.c_void_p)
        FF = C.CFUNCTYPE(None, C.c_void_p)

        def _alloc(nbytes, stream):
            try:
                return torch.cuda.caching_allocator_alloc(int(nbytes), stream=int(stream or 0))
            except Exception:
                return None

        def _free(ptr):
            torch.cuda.caching_allocator_delete(ptr)

        _alloc_cb, _free_cb = AF(_alloc), FF(_free)
    rc = lib().mg_set_allocator(_alloc_cb, _free_cb)
    if rc:
        raise MgError(rc, "mg_set_allocator")


def use_default_allocator():
    """Back to cudaMalloc / cudaFree for handles created from now on (existing handles keep the allocator they were created with)."""
    rc = lib().mg_set_allocator(None, None)
    if rc:
        raise MgError(rc, "mg_set_allocator")


def _stream_ptr(stream):
    import torch
    s = stream if stream is not None else torch.cuda.current_stream()
    return C.c_void_p(s.cuda_stream)


def _dptr(t):
    import torch
    assert t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()
    return C.c_void_p(t.data_ptr())


class Solver:
    """create / update / solve on one mesh."""

    def __init__(self, i, j, kind, h, levels=0, nu_pre=2, nu_post=2, restart_m=30, max_iters=200, stream=None, host_only=False, fused_tail=False, gamma=1, full_cgs2=False, planes=1, solver=0):
        import torch
        if not host_only and not torch.cuda.is_available():
            raise RuntimeError("paper_2509_11831_b200 needs a CUDA device (no CPU fallback)")
        L = lib()
        i = np.ascontiguousarray(i, dtype=np.int32)
        j = np.ascontiguousarray(j, dtype=np.int32)
        kind = np.ascontiguousarray(kind, dtype=np.uint8)
        self.n = int(i.shape[0])
        if int(nu_pre) < 1 or int(nu_post) < 0:
            raise ValueError("nu_pre must be >= 1 (rule T2) and nu_post >= 0")
        mesh = _Mesh(self.n, i.ctypes.data, j.ctypes.data, float(h))
        bc = _Bc(kind.ctypes.data)
        opt = _Options(int(levels), int(nu_pre), int(nu_post) if int(nu_post) != 0 else -1,   # 0 sweeps = MG_NU_NONE
                        int(restart_m), int(max_iters), (1 if host_only else 0) | (2 if fused_tail else 0) | (4 if full_cgs2 else 0), int(gamma), int(planes), {0: 0, 1: 1, 'fgmres': 0, 'bicgstab': 1}[solver])
        hd = C.c_void_p()
        rc = L.mg_setup(C.byref(mesh), C.byref(bc), C.byref(opt), None if host_only else _stream_ptr(stream), C.byref(hd))
        if rc:
            raise MgError(rc, "mg_setup")
        self._h = hd
        self.planes = max(1, int(planes))     # with P > 1 planes: fields are [P, n] tensors, iters / relres arrays of P
        self.levels = L.mg_num_levels(self._h)
        self.device = None if host_only else torch.device("cuda", torch.cuda.current_device())

    def close(self):
        if getattr(self, "_h", None):
            lib().mg_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- the three calls
    def update_coeffs(self, lam, c, stream=None):
        rc = lib().mg_update_coeffs(self._h, _dptr(lam), _dptr(c), _stream_ptr(stream))
        if rc:
            raise MgError(rc, "mg_update_coeffs")

    def update_coeffs3(self, lam, xi, c, stream=None):
        """Three-field form lambda phi - xi div(c grad phi) = rho (Eq. 3); xi=None is update_coeffs."""
        rc = lib().mg_update_coeffs3(self._h, _dptr(lam), _dptr(xi) if xi is not None else None, _dptr(c), _stream_ptr(stream))
        if rc:
            raise MgError(rc, "mg_update_coeffs3")

    def update_coeffs3_host(self, lam, xi, c, stream=None):
        lam, xi, c = (np.ascontiguousarray(a, dtype=np.float64) for a in (lam, xi, c))
        rc = lib().mg_update_coeffs3_host(self._h, C.c_void_p(lam.ctypes.data), C.c_void_p(xi.ctypes.data),
                                          C.c_void_p(c.ctypes.data), _stream_ptr(stream))
        if rc:
            raise MgError(rc, "mg_update_coeffs3_host")

    def level_xi(self, s, stream=None):
        xi = np.empty(self.level_n(s))
        rc = lib().mg_level_xi(self._h, int(s), C.c_void_p(xi.ctypes.data), _stream_ptr(stream))
        if rc:
            raise MgError(rc, "mg_level_xi")
        return xi

    def solve(self, f, x0, rtol, x=None, stream=None):
        import torch
        if x is None:
            x = torch.empty_like(f)
        P = self.planes
        assert f.numel() == P * self.n and x0.numel() == P * self.n and x.numel() == P * self.n
        iters, relres = (C.c_int * P)(), (C.c_double * P)()
        rc = lib().mg_solve(self._h, _dptr(f), _dptr(x0), _dptr(x), C.c_double(rtol), iters, relres, _stream_ptr(stream))
        if rc < 0:
            raise MgError(rc, "mg_solve")
        if P == 1:
            return x, iters[0], relres[0], rc
        return x, list(iters), list(relres), rc

    def update_coeffs_host(self, lam, c, stream=None):
        lam = np.ascontiguousarray(lam, dtype=np.float64); c = np.ascontiguousarray(c, dtype=np.float64)
        rc = lib().mg_update_coeffs_host(self._h, C.c_void_p(lam.ctypes.data), C.c_void_p(c.ctypes.data), _stream_ptr(stream))
        if rc:
            raise MgError(rc, "mg_update_coeffs_host")

    def solve_host(self, f, x0, rtol, x=None, stream=None):
        f = np.ascontiguousarray(f, dtype=np.float64); x0 = np.ascontiguousarray(x0, dtype=np.float64)
        P = self.planes
        if x is None:
            x = np.empty(f.shape)
        assert f.size == P * self.n and x0.size == P * self.n and x.size == P * self.n
        iters, relres = (C.c_int * P)(), (C.c_double * P)()
        rc = lib().mg_solve_host(self._h, C.c_void_p(f.ctypes.data), C.c_void_p(x0.ctypes.data), C.c_void_p(x.ctypes.data),
                                 C.c_double(rtol), iters, relres, _stream_ptr(stream))
        if rc < 0:
            raise MgError(rc, "mg_solve_host")
        if P == 1:
            return x, iters[0], relres[0], rc
        return x, list(iters), list(relres), rc

    # ---- inspection
    def level_n(self, s):
        return int(lib().mg_level_n(self._h, int(s)))

    def level_info(self, s):
        n = self.level_n(s)
        out = dict(I=np.empty(n, np.int32), J=np.empty(n, np.int32), kind=np.empty(n, np.uint8),
                   colour=np.empty(n, np.uint8), nbr=np.empty((n, 4), np.int32), ns_tn=np.empty((n, 2), np.int8),
                   ns_fallback=np.empty(n, np.uint8), slot=np.empty(n, np.int32))
        u2c = np.empty(self.n, np.int64) if s == 0 else None
        args = [C.c_void_p(out[k].ctypes.data) for k in ("I", "J", "kind", "colour", "nbr", "ns_tn", "ns_fallback", "slot")]
        rc = lib().mg_level_info(self._h, int(s), *args, C.c_void_p(u2c.ctypes.data) if u2c is not None else None)
        if rc:
            raise MgError(rc, "mg_level_info")
        if u2c is not None:
            out["user2canon"] = u2c
        return out

    def transfer_info(self, s):
        nf, nc = self.level_n(s), self.level_n(s + 1)
        out = dict(fine9=np.empty((nc, 9), np.int32), parent=np.empty((nf, 4), np.int32), ptype=np.empty(nf, np.uint8))
        rc = lib().mg_transfer_info(self._h, int(s), *[C.c_void_p(out[k].ctypes.data) for k in ("fine9", "parent", "ptype")])
        if rc:
            raise MgError(rc, "mg_transfer_info")
        return out

    def level_coeffs(self, s, stream=None):
        n = self.level_n(s)
        lam, c = np.empty(n), np.empty(n)
        rc = lib().mg_level_coeffs(self._h, int(s), C.c_void_p(lam.ctypes.data), C.c_void_p(c.ctypes.data), _stream_ptr(stream))
        if rc:
            raise MgError(rc, "mg_level_coeffs")
        return lam, c

    # ---- single steps (device level vectors, canonical order)
    def _call(self, name, *args):
        rc = getattr(lib(), name)(self._h, *args)
        if rc:
            raise MgError(rc, name)

    def apply(self, s, x, stream=None):
        import torch
        y = torch.empty_like(x)
        self._call("mg_apply", int(s), _dptr(x), _dptr(y), _stream_ptr(stream))
        return y

    def smooth(self, s, x, b, sweeps=1, stream=None):
        x = x.clone()
        self._call("mg_smooth", int(s), _dptr(x), _dptr(b), int(sweeps), _stream_ptr(stream))
        return x

    def smooth_restrict(self, s, x, b, sweeps=2, stream=None):
        import torch
        x = x.clone()
        dc = torch.empty(self.level_n(s + 1), dtype=torch.float64, device=x.device)
        self._call("mg_smooth_restrict", int(s), _dptr(x), _dptr(b), int(sweeps), _dptr(dc), _stream_ptr(stream))
        return x, dc

    def restrict(self, s, d, stream=None):
        import torch
        out = torch.empty(self.level_n(s + 1), dtype=torch.float64, device=d.device)
        self._call("mg_restrict", int(s), _dptr(d), _dptr(out), _stream_ptr(stream))
        return out

    def prolong_correct(self, s, ec, x, stream=None):
        x = x.clone()
        self._call("mg_prolong_correct", int(s), _dptr(ec), _dptr(x), _stream_ptr(stream))
        return x

    def coarse_solve(self, b, stream=None):
        import torch
        x = torch.empty_like(b)
        self._call("mg_coarse_solve", _dptr(b), _dptr(x), _stream_ptr(stream))
        return x

    def vcycle(self, s, x, b, stream=None):
        x = x.clone()
        self._call("mg_vcycle", int(s), _dptr(x), _dptr(b), _stream_ptr(stream))
        return x

    @property
    def kernel_launches(self):
        return int(lib().mg_kernel_launches(self._h))

    @property
    def last_solve_ms(self):
        return float(lib().mg_last_solve_ms(self._h))

    @property
    def last_step_ms(self):
        return float(lib().mg_last_step_ms(self._h))

    def last_history(self):
        """(relres, orth) per iteration of the last solve, see mg_last_history."""
        import numpy as np
        r, o = np.zeros(512), np.zeros(512)
        n = lib().mg_last_history(self._h, r.ctypes.data_as(C.c_void_p), o.ctypes.data_as(C.c_void_p), 512)
        if n < 0:
            raise RuntimeError(f"mg_last_history: {n}")
        return r[:n].copy(), o[:n].copy()

    @property
    def last_reorth(self):
        return int(lib().mg_last_reorth(self._h))

    @property
    def last_update_ms(self):
        return float(lib().mg_last_update_ms(self._h))
