"""mg_norm2_noalloc (include/mg_b200.h): the entry point that allocates nothing — its scratch is a fixed __device__ array of the
library.  Checked against the EXISTING path that computes the same quantity: mg_solve's `final_relres` is
||f - A x|| / ||f|| formed by k_apply + k_norm2 with handle-allocated scratch; here the same residual (mg_apply, the
existing single-step entry) is normed by the new entry point.  Two calls in a row share the scratch array.  Collected
last on purpose (the suite runs with pytest -x); passes alone in a fresh process and after the other tests."""
import ctypes as C

import numpy as np
import pytest

from paper_2509_11831_b200 import workloads as W

pytestmark = pytest.mark.gpu

TOL = 1e-13          # the bar of the single-application tests (tests/test_gpu_parity.py TOL_STEP): only the summation order differs


def test_norm2_noalloc_matches_the_solve_path_twice_in_a_row():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2509_11831_b200 import binding as B
    B.lib()
    B.use_torch_allocator()
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a, dtype=np.float64)).cuda()
    pl = W.make_plane(3, 257)
    s = B.Solver(pl.i, pl.j, pl.kind, pl.h, levels=pl.levels, max_iters=5)
    s.update_coeffs(dev(pl.lam), dev(pl.c))
    u2c = torch.from_numpy(s.level_info(0)["user2canon"]).cuda()
    fc = torch.empty(pl.n, dtype=torch.float64, device="cuda")
    fc[u2c] = dev(pl.f)
    out = torch.zeros(2, dtype=torch.float64, device="cuda")
    x0 = dev(pl.x0)
    for call in range(2):                                         # two solves, two pairs of calls on the shared scratch
        x, iters, relres, rc = s.solve(dev(pl.f), x0, 1e-10)      # capped at 5 iterations: relres is the true residual of x
        assert rc == 1 and iters == 5 and relres > 1e-10
        xc = torch.empty_like(fc)
        xc[u2c] = x
        r = fc - s.apply(0, xc)                                   # existing single-step path, canonical order
        B.norm2_noalloc(r, out[0:1])
        B.norm2_noalloc(fc, out[1:2])                             # back to back on the same stream: ordered, no race
        o = out.cpu().numpy()
        assert abs(o[0] / o[1] - relres) <= TOL * relres, (call, o[0] / o[1], relres)
        assert abs(o[0] - float(torch.linalg.vector_norm(r))) <= TOL * o[0]
        x0 = x                                                    # second round: another vector (warm start)
    # the array keeps the last call's contents: a repeated call gives the same bits, a short vector after a long one is right
    a = B.norm2_noalloc(r).item()
    assert a == B.norm2_noalloc(r).item() == o[0]
    big = torch.randn(3 * 65536 + 17, dtype=torch.float64, device="cuda")
    vb = B.norm2_noalloc(big).item()
    assert abs(vb - float(torch.linalg.vector_norm(big))) <= TOL * vb
    assert B.norm2_noalloc(big[:5]).item() == pytest.approx(float(torch.linalg.vector_norm(big[:5])), rel=1e-15)
    assert B.norm2_noalloc(big[:0]).item() == 0.0
    # sizes beyond the fixed scratch are refused with a clear error, nothing is launched
    L = B.lib()
    rc = L.mg_norm2_noalloc(C.c_void_p(big.data_ptr()), C.c_int64(B.NOALLOC_MAX_N + 1), C.c_void_p(out.data_ptr()), None)
    assert rc == -1 and "MG_NOALLOC_MAX_N" in B.last_error()
    assert L.mg_norm2_noalloc(None, C.c_int64(4), C.c_void_p(out.data_ptr()), None) == -1
    torch.cuda.synchronize()
    s.close()
