"""Pins P1, P2, P5, P6, P7 for the oracle's operator, transfers and smoother.
Everything is checked against closed forms / invariants, never against the oracle's own formulae."""
import numpy as np
import pytest

from tests import helpers as H


def test_P1_eigenpairs_closed_form(oracle_mod):
    """5-point Laplacian on the square, c=1, lambda=const, zero guards: sin(k pi x) sin(l pi y) is an
    eigenvector with eigenvalue lam + (4/h^2)(sin^2(k pi h/2) + sin^2(l pi h/2))  (textbook).
    Pins Eq. 10 with the 1/h^2 of reading G1, and the neighbour maps."""
    n = 33
    lam0 = 0.7
    pl = H.square_plane(n, 1, lam=lam0, c=1.0)
    o = H.make_oracle(oracle_mod, pl)
    a = o.level_arrays(0)
    h = pl.h
    x, y = a["I"] * h, a["J"] * h
    inner = a["kind"] == 0
    for k, l in [(1, 1), (2, 5), (7, 3), (n - 2, n - 2), (n - 2, 1), (13, 29)]:
        v = np.sin(k * np.pi * x) * np.sin(l * np.pi * y)
        v[~inner] = 0.0
        ev = lam0 + (4.0 / h ** 2) * (np.sin(k * np.pi * h / 2) ** 2 + np.sin(l * np.pi * h / 2) ** 2)
        Av = o.apply(0, v)
        assert np.abs(Av[inner] - ev * v[inner]).max() <= 1e-12 * ev
        assert np.array_equal(Av[~inner], v[~inner])            # Dirichlet rows: Eq. 11


@pytest.mark.parametrize("geom", ["annulus", "dshape"])
def test_P2_constants_and_linear_functions(oracle_mod, geom):
    pl = H.small_annulus(65, 3) if geom == "annulus" else H.small_dshape(129, 4)
    o = oracle_mod.Oracle(pl.i, pl.j, pl.kind, pl.h, levels=pl.levels)
    rng = np.random.default_rng(3)
    lam = rng.uniform(0.1, 2.0, pl.n)
    o.update(lam, np.full(pl.n, 1.7))                             # constant c on the finest level
    for s in range(o.levels):
        a = o.level_arrays(s)
        lam_s, c_s = o.level_coeffs(s)
        assert np.abs(c_s - 1.7).max() < 1e-14                    # T4 of a constant is that constant (P6)
        h = o.level_h(s)
        inner, dirich, neum = a["kind"] == 0, a["kind"] == 1, a["kind"] == 2
        one = np.ones(o.level_n(s))
        A1 = o.apply(s, one)
        scale = 4 * 1.7 / h ** 2
        assert np.abs(A1[inner] - lam_s[inner]).max() <= 1e-13 * scale      # stencil sums to lambda
        assert np.array_equal(A1[dirich], one[dirich])
        assert np.abs(A1[neum]).max() <= 1e-13 / h                          # Neumann rows annihilate constants
        al, be = 0.3, -1.1
        u = al * a["I"] * h + be * a["J"] * h
        Au = o.apply(s, u)
        assert np.abs(Au[inner] - lam_s[inner] * u[inner]).max() <= 1e-11 * scale
        # Neumann rows on linear functions: (alpha nR + beta nZ)/|n| exactly (bilinear phi^N), Eq. 16
        reg = neum & (a["ns_fallback"] == 0)
        tn = a["ns_tn"][reg].astype(float) / 2
        expect = (al * tn[:, 0] + be * tn[:, 1]) / np.sqrt((tn ** 2).sum(axis=1))
        assert np.abs(Au[reg] - expect).max() <= 1e-11
        assert reg.sum() > 0 or neum.sum() == 0


def test_P2_row_structure(oracle_mod):
    """5 nnz per inner row, <=3 in the paper's printed boundary cases, diag>0, offdiag<=0."""
    pl = H.small_dshape(33, 1)
    o = H.make_oracle(oracle_mod, pl)
    a = o.level_arrays(0)
    n = pl.n
    A = np.column_stack([o.apply(0, e) for e in np.eye(n)])
    inner = a["kind"] == 0
    nnz = (A != 0).sum(axis=1)
    assert (nnz[inner] == 5).all()
    assert (np.diag(A)[inner] > 0).all()
    off = A - np.diag(np.diag(A))
    assert (off[inner] <= 0).all()
    guards = np.nonzero(~inner)[0]
    for l in guards:
        if a["kind"][l] == 1:
            assert nnz[l] == 1 and A[l, l] == 1.0
        elif not a["ns_fallback"][l] and (np.abs(a["ns_tn"][l]) % 2).sum() <= 1:
            assert nnz[l] <= 3
        else:
            assert nnz[l] <= 5
        cols = np.nonzero(A[l])[0]
        assert all(c == l or a["kind"][c] == 0 for c in cols)


def test_P5_symmetric_positive_definite(oracle_mod):
    """All-Dirichlet: eliminating the guard rows leaves a symmetric positive definite inner block
    (Eq. 4).  A wrong face average (e.g. c_l only) breaks the symmetry."""
    pl = H.small_annulus(33, 1, neumann_inner=False)
    o = H.make_oracle(oracle_mod, pl)
    a = o.level_arrays(0)
    A = np.column_stack([o.apply(0, e) for e in np.eye(pl.n)])
    inner = a["kind"] == 0
    Aii = A[np.ix_(inner, inner)]
    assert np.abs(Aii - Aii.T).max() <= 1e-14 * np.abs(Aii).max()
    np.linalg.cholesky(Aii)
    # with Neumann rows: strictly diagonally dominant M-matrix after eliminating guards (lambda > 0)
    pl = H.small_annulus(33, 1, neumann_inner=True)
    o = H.make_oracle(oracle_mod, pl)
    a = o.level_arrays(0)
    A = np.column_stack([o.apply(0, e) for e in np.eye(pl.n)])
    inner = a["kind"] == 0
    Agg = A[np.ix_(~inner, ~inner)]
    red = A[np.ix_(inner, inner)] - A[np.ix_(inner, ~inner)] @ np.linalg.solve(Agg, A[np.ix_(~inner, inner)])
    d = np.diag(red)
    off = red - np.diag(d)
    assert (off <= 1e-9 * d.max()).all()
    assert (d > np.abs(off).sum(axis=1)).all()


def test_P6_transfer_identities(oracle_mod):
    n = 33
    pl = H.square_plane(n, 2)
    o = H.make_oracle(oracle_mod, pl)
    nf, nc = o.level_n(0), o.level_n(1)
    fa, ca = o.level_arrays(0), o.level_arrays(1)
    # P as a matrix: x - prolong_correct(e_c, x) with x = 0  ->  -(-P e_c)
    P = np.column_stack([-o.prolong_correct(0, e, np.zeros(nf)) for e in np.eye(nc)])
    R = np.column_stack([o.restrict(0, e) for e in np.eye(nf)])
    fin, cin = fa["kind"] == 0, ca["kind"] == 0
    # away from guards R = 1/4 P^T entrywise (full weighting is the scaled adjoint of bilinear)
    deep_c = cin & (ca["I"] > 1) & (ca["I"] < (n - 1) // 2 - 1) & (ca["J"] > 1) & (ca["J"] < (n - 1) // 2 - 1)
    assert np.abs(R[np.ix_(deep_c, fin)] - 0.25 * P[np.ix_(fin, deep_c)].T).max() <= 1e-16
    # bilinear P is exact on linear functions at fine inner points whose parents are all inner
    u_c = 0.4 * ca["I"] * 2 - 0.9 * ca["J"] * 2 + 0.2
    u_f = 0.4 * fa["I"] - 0.9 * fa["J"] + 0.2
    Pu = P @ u_c
    deep_f = fin & (fa["I"] > 2) & (fa["I"] < n - 3) & (fa["J"] > 2) & (fa["J"] < n - 3)
    assert np.abs(Pu[deep_f] - u_f[deep_f]).max() <= 1e-13
    # zero Dirichlet data: guards of the correction are zero (set_bnds_hom)
    assert np.array_equal(Pu[~fin], np.zeros((~fin).sum()))
    # R of a constant is the constant away from guards; coarse guard rows are 0
    Rc = R @ np.ones(nf)
    assert np.abs(Rc[deep_c] - 1.0).max() <= 1e-15
    assert np.array_equal(Rc[~cin], np.zeros((~cin).sum()))
    # weights: a unit impulse at a coincident fine point restricts to 4/16 there, 2/16 edge, 1/16 corner
    q = int(np.nonzero(deep_c)[0][5])
    Ic, Jc = int(ca["I"][q]), int(ca["J"][q])
    fidx = {(int(i), int(j)): k for k, (i, j) in enumerate(zip(fa["I"], fa["J"]))}
    for (dx, dy), w in {(0, 0): 0.25, (1, 0): 0.125, (0, -1): 0.125, (1, 1): 0.0625, (-1, 1): 0.0625}.items():
        assert R[q, fidx[(2 * Ic + dx, 2 * Jc + dy)]] == w


def test_P6_coefficient_restriction_bounds(oracle_mod):
    pl = H.small_dshape(65, 3)
    o = H.make_oracle(oracle_mod, pl)
    for s in range(o.levels - 1):
        lam_f, c_f = o.level_coeffs(s)
        lam_c, c_c = o.level_coeffs(s + 1)
        t = o.transfer_tables(s)
        for q in range(o.level_n(s + 1)):
            idx = t["fine9"][q][t["fine9"][q] >= 0]
            assert len(idx) >= 1
            assert c_f[idx].min() * (1 - 1e-15) <= c_c[q] <= c_f[idx].max() * (1 + 1e-15)
            assert lam_f[idx].min() * (1 - 1e-15) <= lam_c[q] <= lam_f[idx].max() * (1 + 1e-15)
        assert (c_c > 0).all()
    # exact value on one interior coarse point: full weighting 1/16 [1 2 1; 2 4 2; 1 2 1]
    t = o.transfer_tables(0)
    full = np.nonzero((t["fine9"] >= 0).all(axis=1))[0][3]
    lam_f, c_f = o.level_coeffs(0)
    w = np.array([1, 2, 1, 2, 4, 2, 1, 2, 1]) / 16.0
    assert o.level_coeffs(1)[1][full] == pytest.approx((w * c_f[t["fine9"][full]]).sum(), rel=1e-15)


@pytest.mark.parametrize("geom", ["annulus", "dshape"])
def test_P7_smoother_group_residuals(oracle_mod, geom):
    """After the loop over a group, the residual on that group's rows is zero (Gauss-Seidel);
    the other groups' values are untouched."""
    pl = H.small_annulus(65, 2) if geom == "annulus" else H.small_dshape(65, 2)
    o = H.make_oracle(oracle_mod, pl)
    rng = np.random.default_rng(1)
    for s in range(o.levels):
        a = o.level_arrays(s)
        n = o.level_n(s)
        x = rng.standard_normal(n)
        b = rng.standard_normal(n)
        for g in (0, 1, 2):
            xn = o.smooth_group(s, x, b, g)
            rows = a["colour"] == g
            assert np.array_equal(xn[~rows], x[~rows])
            r = b - o.apply(s, xn)
            rowscale = np.abs(b).max() + np.abs(o.apply(s, np.abs(xn))).max()
            assert np.abs(r[rows]).max() <= 1e-13 * rowscale
            x = xn
        # one sweep == the three groups in order red, black, boundary
        x0 = rng.standard_normal(n)
        y = x0
        for g in (0, 1, 2):
            y = o.smooth_group(s, y, b, g)
        assert np.array_equal(o.smooth(s, x0, b, 1), y)


def test_P7_ordering_independence(oracle_mod):
    """the algorithms do not depend on the mesh ordering."""
    a = H.small_dshape(65, 3, order="rowmajor")
    b = H.small_dshape(65, 3, order="shuffle")
    oa, ob = H.make_oracle(oracle_mod, a), H.make_oracle(oracle_mod, b)
    ra, rb = oa.solve(a.f, a.x0, 1e-10), ob.solve(b.f, b.x0, 1e-10)
    assert ra["iters"] == rb["iters"]
    assert np.array_equal(H.canon(oa, ra["x"]), H.canon(ob, rb["x"]))


def _geoms():
    return [H.small_annulus(65, 3), H.small_dshape(129, 4), H.random_blob_plane(3), H.random_blob_plane(4)]


def test_P6_set_bnds_hom_and_prolongation_brute_force(oracle_mod):
    """Rule T3 on ragged meshes with Neumann guards, every level.  The correction e = P e_c must (i) equal the
    bilinear interpolation of P:153 / Fig. 3 on fine inner points, parents absent from the coarse mesh counting 0
    (written here from the weights 1 / (1/2, 1/2) / (1/4 x 4) with a dict on (I, J)); (ii) vanish on Dirichlet guards
    (homogeneous Eq. 11); (iii) satisfy the HOMOGENEOUS Neumann row on Neumann guards: (A e)_l = 0
    (Eq. 16, with Gamma = 0; set_bnds_hom) — fallback guards included.  Dropping the 1/(1 - w_self)
    of half-integer normals, or leaving Neumann guards at 0, fails (iii)."""
    rng = np.random.default_rng(11)
    n_neu = n_fb = n_half = 0
    for pl in _geoms():
        o = H.make_oracle(oracle_mod, pl)
        for s in range(o.levels - 1):
            fa, ca = o.level_arrays(s), o.level_arrays(s + 1)
            nf, nc = o.level_n(s), o.level_n(s + 1)
            ec = rng.standard_normal(nc)
            e = -o.prolong_correct(s, ec, np.zeros(nf))
            cmap = {(int(i), int(j)): k for k, (i, j) in enumerate(zip(ca["I"], ca["J"]))}
            val = lambda ci, cj: ec[cmap[(ci, cj)]] if (ci, cj) in cmap else 0.0
            exp = np.zeros(nf)
            for l in np.nonzero(fa["kind"] == 0)[0]:
                I, J = int(fa["I"][l]), int(fa["J"][l])
                Il, Jl = I // 2, J // 2                             # Python floor division: lower coarse index
                if I % 2 == 0 and J % 2 == 0:
                    exp[l] = val(Il, Jl)
                elif J % 2 == 0:
                    exp[l] = 0.5 * val(Il, Jl) + 0.5 * val(Il + 1, Jl)
                elif I % 2 == 0:
                    exp[l] = 0.5 * val(Il, Jl) + 0.5 * val(Il, Jl + 1)
                else:
                    exp[l] = 0.25 * (val(Il, Jl) + val(Il + 1, Jl) + val(Il, Jl + 1) + val(Il + 1, Jl + 1))
            inner, dirich, neum = fa["kind"] == 0, fa["kind"] == 1, fa["kind"] == 2
            assert np.abs(e[inner] - exp[inner]).max() <= 1e-15 * np.abs(ec).max()
            assert np.array_equal(e[dirich], np.zeros(dirich.sum()))
            Ae = o.apply(s, e)
            h = o.level_h(s)
            assert np.abs(Ae[neum]).max(initial=0.0) <= 4e-16 * np.abs(ec).max() / h
            if neum.any():                                       # the guards really carry the interpolated values
                assert np.abs(e[neum]).max() > 0.0
            n_neu += int(neum.sum())
            n_fb += int((neum & (fa["ns_fallback"] == 1)).sum())
            n_half += int((neum & (fa["ns_fallback"] == 0) & ((np.abs(fa["ns_tn"]) % 2).sum(axis=1) > 0)).sum())
    assert n_neu > 500 and n_fb > 0 and n_half > 50              # every branch of set_bnds_hom was exercised


def test_P6_restriction_brute_force_ragged(oracle_mod):
    """Rule T2 next to ragged boundaries, every level: d_c(I, J) = 1/16 [1 2 1; 2 4 2; 1 2 1] over the fine INNER
    points (2I+dx, 2J+dy) present (fine guards and absent points contribute 0) on coarse inner rows; coarse
    guard rows are 0.  Written here with dicts on (I, J), independent of the oracle's fine9 tables."""
    rng = np.random.default_rng(12)
    near = 0
    for pl in _geoms():
        o = H.make_oracle(oracle_mod, pl)
        for s in range(o.levels - 1):
            fa, ca = o.level_arrays(s), o.level_arrays(s + 1)
            d = rng.standard_normal(o.level_n(s))
            got = o.restrict(s, d)
            fmap = {(int(i), int(j)): k for k, (i, j) in enumerate(zip(fa["I"], fa["J"]))}
            exp = np.zeros(o.level_n(s + 1))
            for q in np.nonzero(ca["kind"] == 0)[0]:
                I, J = int(ca["I"][q]), int(ca["J"][q])
                acc = 0.0
                for dy in (-1, 0, 1):
                    for dx in (-1, 0, 1):
                        l = fmap.get((2 * I + dx, 2 * J + dy), -1)
                        if l >= 0 and fa["kind"][l] == 0:
                            acc += (2 - abs(dx)) * (2 - abs(dy)) / 16.0 * d[l]
                        else:
                            near += 1
                exp[q] = acc
            assert np.abs(got - exp).max() <= 2e-16 * 4
            assert np.array_equal(got[ca["kind"] != 0], np.zeros((ca["kind"] != 0).sum()))
    assert near > 1000                                             # stencils with missing / guard fine points were hit
