"""Pins of the oracle's BiCGStab (orc_solve_bicgstab; PAPER.md:342 names BiCGStab as the alternative outer solver).  None of
them retypes the recurrence: the solution is checked against dense direct solves, against the fGMRES oracle, and through
properties that fix the algorithm — finite termination in exact arithmetic, one application with an exact
preconditioner, homogeneity, the recurrence residual agreeing with the recomputed one, restart behaviour."""
import numpy as np
import pytest

from paper_2509_11831_b200 import workloads as W
from tests import helpers as H


def _dense(o, lv=0):
    n = o.level_n(lv)
    return np.column_stack([o.apply(lv, e) for e in np.eye(n)])


@pytest.mark.parametrize("geom", ["square", "annulus", "dshape"])
def test_bicgstab_matches_dense_direct_solve(oracle_mod, geom):
    pl = {"square": lambda: H.square_plane(17, 2), "annulus": lambda: H.small_annulus(33, 2), "dshape": lambda: H.small_dshape(33, 2)}[geom]()
    o = H.make_oracle(oracle_mod, pl)
    f = np.random.default_rng(5).standard_normal(pl.n)
    r = o.solve_bicgstab(f, np.zeros(pl.n), 1e-11)
    xd = np.linalg.solve(_dense(o), H.canon(o, f))
    assert r["status"] == 0 and r["relres"] < 1e-11
    assert np.linalg.norm(H.canon(o, r["x"]) - xd) <= 1e-9 * np.linalg.norm(xd)
    # the reported residual is the true one
    true = np.linalg.norm(H.canon(o, f) - _dense(o) @ H.canon(o, r["x"])) / np.linalg.norm(f)
    assert r["relres"] == pytest.approx(true, rel=1e-2, abs=2e-14)


def test_bicgstab_special_cases(oracle_mod):
    pl = H.small_annulus(17, 1)
    o = H.make_oracle(oracle_mod, pl, m=60)
    # exact preconditioner: v = A A^-1 r = r, alpha = 1, s = 0 -> converged at the first half step, one application
    r = o.solve_bicgstab(pl.f, pl.x0, 1e-10, precond=2)
    assert r["iters"] == 1 and r["status"] == 0
    # one-level hierarchy: the cycle is the direct solve -> the same
    assert o.solve_bicgstab(pl.f, pl.x0, 1e-10)["iters"] == 1
    # zero right-hand side -> x = 0 without iterating (K1); converged initial guess -> returned untouched
    r0 = o.solve_bicgstab(np.zeros(pl.n), np.ones(pl.n), 1e-10)
    assert r0["iters"] == 0 and not r0["x"].any()
    xs = o.solve_bicgstab(pl.f, pl.x0, 1e-13)["x"]
    r1 = o.solve_bicgstab(pl.f, xs, 1e-10)
    assert r1["iters"] == 0 and np.array_equal(r1["x"], xs)
    # identity preconditioner on a small symmetric positive definite system: BiCGStab terminates within n steps
    # (2 n applications) in exact arithmetic; in fp64 it reaches 1e-10 well before
    pl2 = H.square_plane(7, 1)
    o2 = H.make_oracle(oracle_mod, pl2, max_iters=4 * pl2.n)
    f = np.random.default_rng(0).standard_normal(pl2.n)
    r2 = o2.solve_bicgstab(f, np.zeros(pl2.n), 1e-10, precond=1)
    assert r2["status"] == 0 and r2["iters"] <= 2 * pl2.n
    xd = np.linalg.solve(_dense(o2), H.canon(o2, f))
    assert np.linalg.norm(H.canon(o2, r2["x"]) - xd) <= 1e-8 * np.linalg.norm(xd)


def test_bicgstab_invariants_and_agreement_with_fgmres(oracle_mod):
    pl = W.make_plane(3, 129)
    o = H.make_oracle(oracle_mod, pl)
    g = o.solve(pl.f, pl.x0, 1e-10)
    b = o.solve_bicgstab(pl.f, pl.x0, 1e-10)
    assert b["status"] == 0 and b["relres"] < 1e-10
    assert np.linalg.norm(b["x"] - g["x"]) <= 1e-8 * np.linalg.norm(g["x"])
    # both are optimal-ish Krylov methods on the same preconditioned operator: comparable work (P:342 proposes the swap)
    assert 0.5 * g["iters"] <= b["iters"] <= 2.5 * g["iters"]
    # the recurrence residual at exit is the true residual to rounding (no drift), and the history ends below rtol
    assert b["hist"][-1] < 1e-10 and b["hist"][-1] == pytest.approx(b["relres"], rel=5e-2)
    # homogeneity: (A, 3 f) -> 3 x with the same number of applications (all scalars are ratios of inner products)
    b3 = o.solve_bicgstab(3.0 * pl.f, pl.x0, 1e-10)
    assert b3["iters"] == b["iters"] and np.linalg.norm(b3["x"] - 3.0 * b["x"]) <= 1e-12 * np.linalg.norm(b3["x"])
    # ordering independence
    q = W.make_plane(3, 129, order="shuffle")
    oq = H.make_oracle(oracle_mod, q)
    bq = oq.solve_bicgstab(q.f, q.x0, 1e-10)
    assert bq["iters"] == b["iters"] and np.array_equal(H.canon(oq, bq["x"]), H.canon(o, b["x"]))
    # iteration cap: stops at max_iters applications with status 1, the iterate is the one of the uncapped run's history
    oc = H.make_oracle(oracle_mod, pl, max_iters=7)
    bc = oc.solve_bicgstab(pl.f, pl.x0, 1e-10)
    assert bc["status"] == 1 and bc["iters"] == 7 and bc["relres"] == pytest.approx(b["hist"][6], rel=1e-6)
