"""Pins P12 for the oracle's three-field form lambda*phi - xi*div(c grad phi) = rho (Eq. 3,
PAPER.md:82 Eq. 10: the bracket of row (i,j) carries xi_{i,j}/2).  Checked against closed forms, the
absorption property the paper states, a dense direct solve and a manufactured solution;
never against the oracle's own formulae."""
import numpy as np
import pytest

from paper_2509_11831_b200 import workloads as W
from tests import helpers as H


def _dense(o, s=0):
    n = o.level_n(s)
    return np.column_stack([o.apply(s, e) for e in np.eye(n)])


def _xi_field(pl, seed=2):
    rng = np.random.default_rng(seed)
    return np.exp(0.6 * rng.standard_normal(pl.n))


def test_P12_eigenpairs_constant_xi(oracle_mod):
    """Square, c = 1, constant lambda and xi, zero guards: sin sin is an eigenvector with eigenvalue
    lam + xi (4/h^2)(sin^2(k pi h/2) + sin^2(l pi h/2)): xi scales the difference part and not lambda."""
    n, lam0, xi0 = 33, 0.7, 2.5
    pl = H.square_plane(n, 1, lam=lam0, c=1.0)
    o = oracle_mod.Oracle(pl.i, pl.j, pl.kind, pl.h, levels=1)
    o.update3(pl.lam, np.full(pl.n, xi0), pl.c)
    a = o.level_arrays(0)
    h = pl.h
    inner = a["kind"] == 0
    for k, l in [(1, 1), (2, 5), (n - 2, 3)]:
        v = np.sin(k * np.pi * a["I"] * h) * np.sin(l * np.pi * a["J"] * h)
        v[~inner] = 0.0
        ev = lam0 + xi0 * (4.0 / h ** 2) * (np.sin(k * np.pi * h / 2) ** 2 + np.sin(l * np.pi * h / 2) ** 2)
        Av = o.apply(0, v)
        assert np.abs(Av[inner] - ev * v[inner]).max() <= 1e-12 * ev
        assert np.array_equal(Av[~inner], v[~inner])


@pytest.mark.parametrize("geom", ["annulus", "dshape"])
def test_P12_row_scaling_structure(oracle_mod, geom):
    """Eq. 10: A3 = Lambda + diag(xi) (A2 - Lambda) on inner rows, with the xi of the ROW's point (so A3 is not
    symmetric for variable xi); Dirichlet and Neumann rows (Eq. 11, 16) do not see xi.  Every level."""
    pl = H.small_annulus(33, 3) if geom == "annulus" else H.small_dshape(33, 3)
    xi = _xi_field(pl)
    o2 = H.make_oracle(oracle_mod, pl)
    o3 = oracle_mod.Oracle(pl.i, pl.j, pl.kind, pl.h, levels=pl.levels)
    o3.update3(pl.lam, xi, pl.c)
    for s in range(o3.levels):
        A2, A3 = _dense(o2, s), _dense(o3, s)
        lam_s, c_s = o3.level_coeffs(s)
        assert np.array_equal(lam_s, o2.level_coeffs(s)[0]) and np.array_equal(c_s, o2.level_coeffs(s)[1])
        xi_s = o3.level_xi(s)
        inner = o3.level_arrays(s)["kind"] == 0
        L = np.diag(lam_s)
        expect = L + xi_s[:, None] * (A2 - L)
        scale = np.abs(A3).max()
        assert np.abs(A3[inner] - expect[inner]).max() <= 1e-14 * scale
        assert np.array_equal(A3[~inner], A2[~inner])
        if s == 0:
            assert np.array_equal(xi_s, H.canon(o3, xi))
            assert np.abs(A3 - A3.T).max() > 1e-3 * scale       # row scaling, not a symmetric scaling


def test_P12_xi_is_grid_transferred_like_lambda(oracle_mod):
    """P:153 / P:207: lambda, xi and c are all transferred to the coarser levels by the same rule (T4)."""
    pl = H.small_dshape(65, 4)
    xi = _xi_field(pl)
    o = oracle_mod.Oracle(pl.i, pl.j, pl.kind, pl.h, levels=pl.levels)
    o.update3(xi, xi, pl.c)                                      # lambda := xi, so both must stay equal on all levels
    for s in range(o.levels):
        assert np.array_equal(o.level_xi(s), o.level_coeffs(s)[0])
        assert xi.min() - 1e-15 <= o.level_xi(s).min() and o.level_xi(s).max() <= xi.max() + 1e-15
    o.update3(pl.lam, np.full(pl.n, 3.25), pl.c)
    for s in range(o.levels):
        assert np.abs(o.level_xi(s) - 3.25).max() <= 1e-14


@pytest.mark.parametrize("geom", ["annulus", "dshape"])
def test_P12_absorption_and_dense_solve(oracle_mod, geom):
    """xi "can be absorbed into lambda and rho".  The multi-level three-field solve must equal the dense
    direct solve of the TWO-field operator with lambda/xi and rho/xi on the inner rows (guard rows unchanged)."""
    pl = H.small_annulus(33, 3) if geom == "annulus" else H.small_dshape(33, 3)
    xi = _xi_field(pl, seed=9)
    rng = np.random.default_rng(4)
    f, x0 = rng.standard_normal(pl.n), rng.standard_normal(pl.n)
    o3 = oracle_mod.Oracle(pl.i, pl.j, pl.kind, pl.h, levels=pl.levels)
    o3.update3(pl.lam, xi, pl.c)
    r = o3.solve(f, x0, 1e-12)
    assert r["status"] == 0
    o2 = oracle_mod.Oracle(pl.i, pl.j, pl.kind, pl.h, levels=1)
    o2.update(pl.lam / xi, pl.c)
    inner = pl.kind == 0
    f2 = np.where(inner, f / xi, f)
    xd = np.linalg.solve(_dense(o2), H.canon(o2, f2))
    assert np.linalg.norm(H.canon(o3, r["x"]) - xd) <= 1e-9 * np.linalg.norm(xd)
    # and the reported residual is the three-field one (Eq. 23); looser rtol keeps it above the rounding floor
    r = o3.solve(f, x0, 1e-8)
    A3 = _dense(o3)
    true = np.linalg.norm(H.canon(o3, f) - A3 @ H.canon(o3, r["x"])) / np.linalg.norm(f)
    assert r["relres"] == pytest.approx(true, rel=1e-3) and true < 1e-8


def test_P12_manufactured_solution_order(oracle_mod):
    """u = sin(pi x) sin(pi y), lambda = c = 1, xi = 1 + x + y/2 on the unit square:
    rho = (1 + 2 pi^2 xi) u.  Error vs the continuous solution falls by 4 per halving (O(h^2))."""
    errs, its = [], []
    for n in (33, 65, 129):
        pl = W.make_plane(1, n)
        xi = 1.0 + pl.x + 0.5 * pl.y
        u = np.sin(np.pi * pl.x) * np.sin(np.pi * pl.y)
        u[pl.kind != 0] = 0.0
        f = np.where(pl.kind == 0, (1.0 + 2.0 * np.pi ** 2 * xi) * u, 0.0)
        o = oracle_mod.Oracle(pl.i, pl.j, pl.kind, pl.h, levels=pl.levels)
        o.update3(pl.lam, xi, pl.c)
        r = o.solve(f, np.zeros(pl.n), 1e-11)
        assert r["status"] == 0
        errs.append(np.linalg.norm(r["x"] - u) / np.linalg.norm(u))
        its.append(r["iters"])
    assert errs[0] / errs[1] == pytest.approx(4.0, abs=0.1) and errs[1] / errs[2] == pytest.approx(4.0, abs=0.1)
    assert max(its) <= min(its) + 2                              # h-independent iteration count


def test_P12_smoother_solves_its_rows(oracle_mod):
    """Gauss-Seidel with xi: after the loop over a group the residual of the three-field rows of that group is zero."""
    pl = H.small_dshape(65, 2)
    o = oracle_mod.Oracle(pl.i, pl.j, pl.kind, pl.h, levels=pl.levels)
    o.update3(pl.lam, _xi_field(pl), pl.c)
    rng = np.random.default_rng(1)
    for s in range(o.levels):
        a = o.level_arrays(s)
        x, b = rng.standard_normal(o.level_n(s)), rng.standard_normal(o.level_n(s))
        for g in (0, 1, 2):
            x = o.smooth_group(s, x, b, g)
            rows = a["colour"] == g
            r = b - o.apply(s, x)
            assert np.abs(r[rows]).max() <= 1e-13 * (np.abs(b).max() + np.abs(o.apply(s, np.abs(x))).max())


def test_P12_unit_xi_is_the_two_field_form_bit_for_bit(oracle_mod):
    pl = H.small_annulus(65, 3)
    o2 = H.make_oracle(oracle_mod, pl)
    o3 = oracle_mod.Oracle(pl.i, pl.j, pl.kind, pl.h, levels=pl.levels)
    o3.update3(pl.lam, np.ones(pl.n), pl.c)
    r2, r3 = o2.solve(pl.f, pl.x0, 1e-10), o3.solve(pl.f, pl.x0, 1e-10)
    assert r2["iters"] == r3["iters"] and np.array_equal(r2["x"], r3["x"])
    with pytest.raises(ValueError):
        o3.update3(pl.lam, np.zeros(pl.n), pl.c)
