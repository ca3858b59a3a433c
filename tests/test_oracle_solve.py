"""Pins P3, P4, P8, P9 for the oracle's coarse solve, V-cycle and fGMRES."""
import numpy as np
import pytest

from paper_2509_11831_b200 import workloads as W
from tests import helpers as H


def _dense(o, s=0):
    n = o.level_n(s)
    return np.column_stack([o.apply(s, e) for e in np.eye(n)])


def _square_mms(n):
    """config 1 at lattice n: discrete closed-form solution of the 5-point scheme."""
    pl = W.make_plane(1, n)
    h = pl.h
    amp = (1 + 2 * np.pi ** 2) / (1 + (8 / h ** 2) * np.sin(np.pi * h / 2) ** 2)
    u_cont = np.sin(np.pi * pl.x) * np.sin(np.pi * pl.y)
    u_cont[pl.kind != 0] = 0.0
    return pl, amp * u_cont, u_cont


def test_P3_discrete_closed_form_and_order(oracle_mod):
    """f = (1+2pi^2) sin sin, lambda=c=1, zero Dirichlet: the discrete solution is the continuous one
    times (1+2pi^2)/(1+(8/h^2) sin^2(pi h/2)) (sin sin is an eigenvector, P1).  Error vs continuous
    must fall by 4 per halving over 3 refinements (north_star: O(h^2))."""
    errs = []
    for n in (33, 65, 129, 257):
        pl, u_h, u_c = _square_mms(n)
        o = H.make_oracle(oracle_mod, pl)
        r = o.solve(pl.f, pl.x0, 1e-10)
        assert r["status"] == 0
        assert np.linalg.norm(r["x"] - u_h) <= 1e-9 * np.linalg.norm(u_h)
        errs.append(np.linalg.norm(r["x"] - u_c) / np.linalg.norm(u_c))
    for k in range(3):
        assert errs[k] / errs[k + 1] == pytest.approx(4.0, abs=0.05)


@pytest.mark.parametrize("geom", ["square", "annulus", "annulus_dirichlet", "dshape"])
def test_P4_dense_direct_solve(oracle_mod, geom):
    """fGMRES+MG solution == numpy dense solve of the assembled operator (lattices <= 33^2)."""
    pl = {"square": lambda: H.square_plane(17, 2, lam=0.3, c=2.0),
          "annulus": lambda: H.small_annulus(33, 2),
          "annulus_dirichlet": lambda: H.small_annulus(33, 3, neumann_inner=False),
          "dshape": lambda: H.small_dshape(33, 2)}[geom]()
    rng = np.random.default_rng(11)
    f = rng.standard_normal(pl.n)
    x0 = rng.standard_normal(pl.n)
    o = H.make_oracle(oracle_mod, pl)
    r = o.solve(f, x0, 1e-12)
    assert r["status"] == 0
    A = _dense(o)
    xd = np.linalg.solve(A, H.canon(o, f))
    assert np.linalg.norm(H.canon(o, r["x"]) - xd) <= 1e-9 * np.linalg.norm(xd)
    # reported residual is the true one (Eq. 23)
    true = np.linalg.norm(H.canon(o, f) - A @ H.canon(o, r["x"])) / np.linalg.norm(f)
    assert r["relres"] == pytest.approx(true, rel=1e-6, abs=2e-13)
    assert true < 1e-12


def test_coarse_solve_is_dense_solve(oracle_mod):
    pl = H.small_dshape(65, 3)
    o = H.make_oracle(oracle_mod, pl)
    s = o.levels - 1
    A = _dense(o, s)
    b = np.random.default_rng(2).standard_normal(o.level_n(s))
    assert np.linalg.norm(o.coarse_solve(b) - np.linalg.solve(A, b)) <= 1e-12 * np.linalg.norm(b) * np.linalg.cond(A)
    assert np.linalg.norm(A @ o.coarse_solve(b) - b) <= 1e-12 * np.linalg.norm(b)
    # a one-level "cycle" is the direct solve
    o1 = H.make_oracle(oracle_mod, H.small_dshape(17, 1))
    b1 = np.random.default_rng(3).standard_normal(o1.level_n(0))
    x1 = o1.cycle(0, np.zeros_like(b1), b1)
    assert np.linalg.norm(_dense(o1) @ x1 - b1) <= 1e-12 * np.linalg.norm(b1)


def test_two_grid_cycle_matches_matrix_formula(oracle_mod):
    """mg_cycle with 2 levels equals S^nu2 (I - P A_c^-1 R A) S^nu1 built from dense
    matrices of the single steps (each pinned separately) - pins the order and signs of the cycle."""
    pl = H.small_annulus(33, 2)
    o = H.make_oracle(oracle_mod, pl, nu_pre=1, nu_post=2)
    nf, nc = o.level_n(0), o.level_n(1)
    rng = np.random.default_rng(4)
    x0, b = rng.standard_normal(nf), rng.standard_normal(nf)
    x = o.smooth(0, x0, b, 1)
    d = o.apply(0, x) - b
    dc = o.restrict(0, d)
    ec = np.linalg.solve(_dense(o, 1), dc)
    x = o.prolong_correct(0, ec, x)
    x = o.smooth(0, x, b, 2)
    got = o.cycle(0, x0, b)
    assert np.linalg.norm(got - x) <= 1e-12 * np.linalg.norm(x)


def _vcycle_factor(o, n, cycles=15, seed=0):
    x = np.random.default_rng(seed).standard_normal(n)
    b = np.zeros(n)
    rs = []
    for _ in range(cycles + 1):
        rs.append(np.linalg.norm(o.apply(0, x)))
        x = o.cycle(0, x, b)
    rs = np.array(rs)
    return (rs[15] / rs[5]) ** (1.0 / 10.0)


def test_P8_convergence_factor_square(oracle_mod):
    """Poisson-like problem on the square: V(2,2) RB-GS + FW + bilinear converges with an h-independent
    factor well below 0.2 (textbook multigrid behaviour, P:143 / [13]) for 2..max levels."""
    fac = {}
    for n in (33, 65, 129, 257):
        pl = W.make_plane(1, n)
        o = H.make_oracle(oracle_mod, pl)
        fac[n] = _vcycle_factor(o, pl.n)
        assert fac[n] < 0.2
    v = np.array(list(fac.values()))
    assert v.max() / v.min() < 1.2 + 0.2
    pl = W.make_plane(1, 65)
    for L in (2, 3):
        assert _vcycle_factor(H.make_oracle(oracle_mod, pl, levels=L), pl.n) < 0.2


def test_P8_convergence_bounded_curved(oracle_mod):
    """Curved, re-fitted boundaries: the stationary V-cycle stays a contraction with a factor
    that does not grow under refinement on the annulus; as a preconditioner the iteration count stays
    in a narrow band (P:286 reports 11-17 for its own annulus at 1e-8 with V(5,5))."""
    its, facs = [], []
    for n in (65, 129, 257):
        pl = W.make_plane(2, n)
        o = H.make_oracle(oracle_mod, pl)
        facs.append(_vcycle_factor(o, pl.n))
        its.append(o.solve(pl.f, pl.x0, 1e-10)["iters"])
    assert max(facs) < 0.6
    assert facs[2] < facs[0] * 1.25
    assert max(its) <= 25 and its[2] - its[0] <= 6


def test_P9_krylov_invariants(oracle_mod):
    pl = H.small_dshape(65, 3)
    o = H.make_oracle(oracle_mod, pl, nu_pre=1, nu_post=1)
    A = _dense(o)
    r = o.solve(pl.f, pl.x0, 1e-10, debug=True)
    V, Z, Hh, k = r["V"], r["Z"], r["H"], r["ncols"]
    assert k >= 5 and r["status"] == 0
    Vk = V[:k]                                                     # v_{k+1} is not formed on exit
    # modified Gram-Schmidt applied TWICE (rule K2, reading G22): the basis is orthonormal to working precision in
    # every column, also near convergence where a single pass loses orthogonality like eps*cond/residual
    G = np.abs(Vk @ Vk.T - np.eye(k))
    assert G.max() <= 1e-13
    # Arnoldi relation A Z_k = V_{k+1} H_k (flexible GMRES, Saad [29]) on the first k-1 columns
    lhs = A @ Z[:k - 1].T
    rhs = V[:k].T @ Hh[:k, :k - 1]
    assert np.abs(lhs - rhs).max() <= 1e-12 * np.abs(A).max()
    # recurrence residual equals the recomputed one at every step; history is non-increasing
    b = H.canon(o, pl.f)
    bn = np.linalg.norm(b)
    hist = r["hist"]
    assert (np.diff(hist) <= 1e-15).all()
    beta = np.linalg.norm(b)                                       # x0 = 0
    for j in range(1, k + 1):
        Hj = Hh[:j + 1, :j]
        e1 = np.zeros(j + 1); e1[0] = beta
        y, res, *_ = np.linalg.lstsq(Hj, e1, rcond=None)
        xj = Z[:j].T @ y
        true = np.linalg.norm(b - A @ xj) / bn
        assert hist[j - 1] == pytest.approx(true, rel=(1e-8 if j <= 5 else (1e-4 if true > 1e-6 else 5e-2)), abs=1e-14)


def test_P9_preconditioner_special_cases(oracle_mod):
    pl = H.small_annulus(17, 1)
    o = H.make_oracle(oracle_mod, pl, m=60)
    # exact preconditioner -> one iteration
    r = o.solve(pl.f, pl.x0, 1e-10, precond=2)
    assert r["iters"] == 1 and r["status"] == 0
    # one-level hierarchy: the "cycle" is the direct solve -> one iteration
    assert o.solve(pl.f, pl.x0, 1e-10)["iters"] == 1
    # identity preconditioner: plain GMRES terminates within n steps (n <= m)
    pl2 = H.square_plane(7, 1)
    o2 = H.make_oracle(oracle_mod, pl2, m=60)
    f = np.random.default_rng(0).standard_normal(pl2.n)
    r = o2.solve(f, np.zeros(pl2.n), 1e-10, precond=1)
    assert r["status"] == 0 and r["iters"] <= pl2.n
    xd = np.linalg.solve(_dense(o2), H.canon(o2, f))
    assert np.linalg.norm(H.canon(o2, r["x"]) - xd) <= 1e-8 * np.linalg.norm(xd)


def test_solve_edge_cases(oracle_mod):
    pl = H.small_annulus(33, 2)
    o = H.make_oracle(oracle_mod, pl)
    r = o.solve(np.zeros(pl.n), np.ones(pl.n), 1e-10)               # K1: b = 0 -> x = 0, 0 iterations
    assert r["iters"] == 0 and not r["x"].any()
    xs = o.solve(pl.f, pl.x0, 1e-12)["x"]
    r = o.solve(pl.f, xs, 1e-10)                                    # already converged initial guess
    assert r["iters"] == 0 and np.array_equal(r["x"], xs)
    o3 = H.make_oracle(oracle_mod, pl, m=3, max_iters=200)          # restarts (K5)
    r3 = o3.solve(pl.f, pl.x0, 1e-10)
    assert r3["status"] == 0 and r3["iters"] > 3
    assert np.linalg.norm(r3["x"] - xs) <= 1e-8 * np.linalg.norm(xs)
    o4 = H.make_oracle(oracle_mod, pl, m=30, max_iters=2)           # iteration cap
    r4 = o4.solve(pl.f, pl.x0, 1e-10)
    assert r4["status"] == 1 and r4["iters"] == 2
    with pytest.raises(ValueError):
        o.update(pl.lam, -pl.c)                                     # c > 0 required


def test_w_cycle_gamma2(oracle_mod):
    """Cycle index gamma of PAPER.md:187-189, 197 (gamma = 2: W-cycle).  With two levels a W-cycle equals a V-cycle (the second
    exact coarse solve changes nothing).  With three levels the level-1 sub-cycle of a W-cycle is again a V-cycle, so the
    W-cycle can be composed from the oracle's single steps with gamma = 1: pre-smoothing, defect, restriction, TWO
    carried-over level-1 cycles, prolongation + correction, post-smoothing.  And it must contract at least as fast."""
    pl = H.small_annulus(65, 3)
    rng = np.random.default_rng(3)
    ov = H.make_oracle(oracle_mod, pl, levels=3)
    ow = H.make_oracle(oracle_mod, pl, levels=3, gamma=2)
    n = ov.level_n(0)
    x, b = rng.standard_normal(n), rng.standard_normal(n)
    xs = ov.smooth(0, x, b, 2)
    dc = ov.restrict(0, ov.apply(0, xs) - b)
    e = ov.cycle(1, np.zeros(ov.level_n(1)), dc)
    e = ov.cycle(1, e, dc)
    ref = ov.smooth(0, ov.prolong_correct(0, e, xs), b, 2)
    got = ow.cycle(0, x, b)
    assert np.linalg.norm(got - ref) <= 1e-13 * np.linalg.norm(ref)
    o2v, o2w = H.make_oracle(oracle_mod, pl, levels=2), H.make_oracle(oracle_mod, pl, levels=2, gamma=2)
    assert np.linalg.norm(o2w.cycle(0, x, b) - o2v.cycle(0, x, b)) <= 1e-12 * np.linalg.norm(x)
    # contraction of the error of A x = 0
    zero = np.zeros(n)
    ev, ew = x.copy(), x.copy()
    for _ in range(6):
        ev, ew = ov.cycle(0, ev, zero), ow.cycle(0, ew, zero)
    assert np.linalg.norm(ew) <= 1.05 * np.linalg.norm(ev)
    rv, rw = ov.solve(pl.f, pl.x0, 1e-10), ow.solve(pl.f, pl.x0, 1e-10)
    assert rw["status"] == 0 and rw["iters"] <= rv["iters"]


def test_f_cycle(oracle_mod):
    """F-cycle (via its ref. [33]): the next coarser level is visited by an F-cycle, then by a V-cycle.
    With two levels it equals the V-cycle, with three levels the W-cycle (below the top level both pay two visits to the
    exact coarsest solve).  With four levels the level-1 sub-cycles are a W-cycle (three levels: F = W) followed by a
    V-cycle, so the F-cycle can be composed from the separately pinned V- and W-cycle oracles.  Its contraction lies
    between theirs."""
    pl = H.small_annulus(129, 4)
    rng = np.random.default_rng(4)
    ov, ow, of = (H.make_oracle(oracle_mod, pl, levels=4, gamma=g) for g in (1, 2, 3))
    n = ov.level_n(0)
    x, b = rng.standard_normal(n), rng.standard_normal(n)
    xs = ov.smooth(0, x, b, 2)
    dc = ov.restrict(0, ov.apply(0, xs) - b)
    e = ow.cycle(1, np.zeros(ov.level_n(1)), dc)          # F-cycle on levels 1-3 = W-cycle
    e = ov.cycle(1, e, dc)                                # then a V-cycle, e carried over
    ref = ov.smooth(0, ov.prolong_correct(0, e, xs), b, 2)
    got = of.cycle(0, x, b)
    assert np.linalg.norm(got - ref) <= 1e-12 * np.linalg.norm(ref)
    assert np.linalg.norm(got - ov.cycle(0, x, b)) > 1e-6 * np.linalg.norm(ref)      # and it is not the V-cycle
    assert np.linalg.norm(got - ow.cycle(0, x, b)) > 1e-9 * np.linalg.norm(ref)      # nor the W-cycle
    for lv, other in ((2, 1), (3, 2)):
        pls = H.small_annulus(65, lv)
        oa, ob = H.make_oracle(oracle_mod, pls, levels=lv, gamma=3), H.make_oracle(oracle_mod, pls, levels=lv, gamma=other)
        xx, bb = rng.standard_normal(oa.level_n(0)), rng.standard_normal(oa.level_n(0))
        assert np.linalg.norm(oa.cycle(0, xx, bb) - ob.cycle(0, xx, bb)) <= 1e-12 * np.linalg.norm(xx)
    zero = np.zeros(n)
    ev, ew, ef = x.copy(), x.copy(), x.copy()
    for _ in range(6):
        ev, ew, ef = ov.cycle(0, ev, zero), ow.cycle(0, ew, zero), of.cycle(0, ef, zero)
    assert np.linalg.norm(ew) <= 1.05 * np.linalg.norm(ef) <= 1.05 * 1.05 * np.linalg.norm(ev)
    rf = of.solve(pl.f, pl.x0, 1e-10)
    assert rf["status"] == 0 and rf["iters"] <= ov.solve(pl.f, pl.x0, 1e-10)["iters"]


def test_G9_boundary_aware_transfer_experiment(oracle_mod):
    """Reading G9 ("stencil points may be missing"): the oracle's optional transfers that renormalise the weights next
    to NEUMANN guards.  Pins of the option itself: it changes nothing where no Neumann guard exists (all-Dirichlet mesh:
    identical cycle, bit for bit), the solution of a solve does not depend on it, and on the annulus with a Neumann inner
    circle it lowers the stationary V-cycle factor.  The numbers behind DESIGN.md G9 (why the CUDA path keeps T2 / T3)."""
    pl = H.small_annulus(65, 3, neumann_inner=False)
    o = H.make_oracle(oracle_mod, pl)
    rng = np.random.default_rng(3)
    x, b = rng.standard_normal(pl.n), rng.standard_normal(pl.n)
    c0 = o.cycle(0, x, b)
    o.set_bc_transfer(1)
    assert np.array_equal(o.cycle(0, x, b), c0)
    pl = W.make_plane(2, 129)
    res = {}
    for mode in (0, 1):
        o = H.make_oracle(oracle_mod, pl)
        o.set_bc_transfer(mode)
        r = o.solve(pl.f, pl.x0, 1e-10)
        res[mode] = (_vcycle_factor(o, pl.n), r["iters"], r["x"])
    assert res[1][0] < res[0][0] - 0.03 and res[1][1] <= res[0][1]
    assert np.linalg.norm(res[1][2] - res[0][2]) <= 1e-8 * np.linalg.norm(res[0][2])
