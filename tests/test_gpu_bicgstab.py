"""BiCGStab as alternative outer solver (mg_options.solver = 1) against the oracle's
orc_solve_bicgstab: same preconditioner, same recurrence, same stop rules.  The solution bar is the solve bar (1e-8 relative
L2, true residual < rtol).  Iteration counts: BiCGStab's residual is not monotone and every scalar is a ratio of inner
products whose summation order differs between the two sides, so a threshold can be crossed one step (two applications)
apart: |iters - oracle| <= 2."""
import numpy as np
import pytest

from paper_2509_11831_b200 import workloads as W
from tests import helpers as H
from tests.test_gpu_parity import TOL_SOLVE, dev, gpu, host, rel  # noqa: F401  (gpu is a fixture)

pytestmark = pytest.mark.gpu

CASES = {
    "cfg1": lambda: W.make_plane(1),
    "cfg2_257": lambda: W.make_plane(2, 257),
    "cfg3_257": lambda: W.make_plane(3, 257),
    "cfg3_1025": lambda: W.make_plane(3),
    "blob_193": lambda: H.random_blob_plane(104, 193),
}


@pytest.mark.parametrize("case", list(CASES))
def test_bicgstab_parity(gpu, oracle_mod, case):
    pl = CASES[case]()
    o = oracle_mod.Oracle(pl.i, pl.j, pl.kind, pl.h, levels=pl.levels)
    o.update(pl.lam, pl.c)
    ro = o.solve_bicgstab(pl.f, pl.x0, 1e-10)
    s = gpu.Solver(pl.i, pl.j, pl.kind, pl.h, levels=pl.levels, solver="bicgstab")
    s.update_coeffs(dev(pl.lam), dev(pl.c))
    x, iters, relres, rc = s.solve(dev(pl.f), dev(pl.x0), 1e-10)
    print(f"{case}: applications gpu/oracle = {iters}/{ro['iters']}, rel.err {rel(host(x), ro['x']):.2e}, relres {relres:.2e}")
    assert rc == 0 and ro["status"] == 0 and abs(iters - ro["iters"]) <= 2
    assert rel(host(x), ro["x"]) <= TOL_SOLVE and relres < 1e-10
    r, _ = s.last_history()
    assert len(r) == iters and r[-1] < 1e-10
    k = min(len(r), len(ro["hist"])) // 2                         # the same recurrence: the residual histories coincide at first; later the
    assert np.allclose(r[:k], ro["hist"][:k], rtol=1e-3)          # rounding of the inner products is amplified (BiCGStab is not backward stable)
    # the fGMRES solution of the same system
    g = gpu.Solver(pl.i, pl.j, pl.kind, pl.h, levels=pl.levels)
    g.update_coeffs(dev(pl.lam), dev(pl.c))
    xg, itg, _, _ = g.solve(dev(pl.f), dev(pl.x0), 1e-10)
    assert rel(host(x), host(xg)) <= TOL_SOLVE
    g.close(); s.close()


def test_bicgstab_edge_cases_and_planes(gpu, oracle_mod):
    pl1 = H.small_annulus(17, 1)                    # one level: the cycle is the direct solve -> converged at the first half step
    s = gpu.Solver(pl1.i, pl1.j, pl1.kind, pl1.h, levels=1, solver=1)
    s.update_coeffs(dev(pl1.lam), dev(pl1.c))
    x, iters, relres, rc = s.solve(dev(pl1.f), dev(pl1.x0), 1e-10)
    o1 = oracle_mod.Oracle(pl1.i, pl1.j, pl1.kind, pl1.h, levels=1)
    o1.update(pl1.lam, pl1.c)
    assert rc == 0 and iters == 1 and rel(host(x), o1.solve_bicgstab(pl1.f, pl1.x0, 1e-10)["x"]) <= TOL_SOLVE
    x, iters, relres, rc = s.solve(dev(np.zeros(pl1.n)), dev(np.ones(pl1.n)), 1e-10)
    assert rc == 0 and iters == 0 and not host(x).any()
    s.close()
    # iteration cap (odd: the step ends at its half) and planes: batched == separate handles bit for bit
    P = 3
    pls = [W.make_plane(2, 129, seed=W.SEEDS[2] + 31 * p) for p in range(P)]
    p0 = pls[0]
    st = lambda k: np.stack([getattr(q, k) for q in pls])
    o = oracle_mod.Oracle(p0.i, p0.j, p0.kind, p0.h, levels=p0.levels, max_iters=7)
    o.update(pls[0].lam, pls[0].c)
    rcap = o.solve_bicgstab(pls[0].f, pls[0].x0, 1e-10)
    sc = gpu.Solver(p0.i, p0.j, p0.kind, p0.h, levels=p0.levels, solver=1, max_iters=7)
    sc.update_coeffs(dev(pls[0].lam), dev(pls[0].c))
    x, iters, relres, rc = sc.solve(dev(pls[0].f), dev(pls[0].x0), 1e-10)
    assert rc == 1 and iters == 7 == rcap["iters"] and rel(host(x), rcap["x"]) <= 1e-6
    sc.close()
    seq = []
    for q in pls:
        s1 = gpu.Solver(p0.i, p0.j, p0.kind, p0.h, levels=p0.levels, solver=1)
        s1.update_coeffs(dev(q.lam), dev(q.c))
        seq.append(s1.solve(dev(q.f), dev(q.x0), 1e-10))
        seq[-1] = (host(seq[-1][0]),) + seq[-1][1:]
        s1.close()
    sb = gpu.Solver(p0.i, p0.j, p0.kind, p0.h, levels=p0.levels, solver=1, planes=P)
    sb.update_coeffs(dev(st("lam")), dev(st("c")))
    xb, its, rrs, rc = sb.solve(dev(st("f")), dev(st("x0")), 1e-10)
    assert rc == 0
    for p in range(P):
        assert its[p] == seq[p][1] and rrs[p] == seq[p][2] and np.array_equal(host(xb)[p], seq[p][0])
    sb.close()
