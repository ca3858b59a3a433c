"""Shared test helpers: small geometries and an independent brute-force mesh checker (pure Python
dicts; shares nothing with oracle/ or the CUDA package)."""
import numpy as np

from paper_2509_11831_b200 import workloads as W
from tests import cases as TC


def make_oracle(om, pl, **kw):
    kw.setdefault("levels", pl.levels)
    o = om.Oracle(pl.i, pl.j, pl.kind, pl.h, **kw)
    o.update(pl.lam, pl.c)
    return o


def canon(o, v_user):
    """user-order vector -> canonical level-0 order"""
    out = np.empty_like(v_user)
    out[o.user2canon] = v_user
    return out


def square_plane(n, levels, lam=1.0, c=1.0):
    inner = W.square_mask(n)
    h = 1.0 / (n - 1)
    neu = np.zeros((n, n), bool)
    return TC.mask_plane(inner, neu, h, lam_f=np.full((n, n), lam), c_f=np.full((n, n), c), levels=levels)


def small_annulus(n=33, levels=2, seed=5, neumann_inner=True, i0=0, j0=0, order="rowmajor"):
    h = 2.0 / (n - 1)
    x = -1 + np.arange(n) * h
    X, Y = np.meshgrid(x, x, indexing="xy")
    inner, r = W.annulus_mask(X, Y, 0.35, 1.0)
    rng = np.random.default_rng(seed)
    neu = (r <= 0.35) & neumann_inner
    lam = 0.5 + rng.uniform(0, 1, (n, n))
    c = np.exp(0.5 * rng.standard_normal((n, n)))
    f = rng.standard_normal((n, n))
    return TC.mask_plane(inner, neu, h, lam, c, f, levels=levels, i0=i0, j0=j0, order=order, seed=seed)


def small_dshape(n=33, levels=2, seed=7, order="rowmajor"):
    h = 2.0 / (n - 1)
    x = -1 + np.arange(n) * h
    X, Y = np.meshgrid(x, x, indexing="xy")
    inner, psi, closed = W.dshape_mask(X, Y)
    rng = np.random.default_rng(seed)
    neu = psi <= W._D["pin"]
    lam = 0.01 + rng.uniform(0, 1, (n, n))
    c = np.exp(rng.standard_normal((n, n)) + np.log(10.0) * closed)
    f = rng.standard_normal((n, n))
    return TC.mask_plane(inner, neu, h, lam, c, f, levels=levels, order=order, seed=seed)


def random_blob_plane(seed, n=97):
    """Ragged random domain: thresholded smooth noise with holes, islands and thin necks; random Dirichlet / Neumann
    guards; random coefficients and right-hand side; odd negative lattice origin; auto level count.  Stresses the
    coarse levels (inner sets that split, degenerate normals, guards that coincide with no fine point)."""
    rng = np.random.default_rng(seed)
    h = 2.0 / (n - 1)
    g = W.gaussian_field(rng, n, 0.12 + 0.1 * rng.uniform(), h)
    inner = g > rng.uniform(-0.4, 0.3)
    inner[:2, :] = inner[-2:, :] = False
    inner[:, :2] = inner[:, -2:] = False
    neu = W.gaussian_field(rng, n, 0.3, h) > 0
    lam = 0.2 + rng.uniform(0, 1, (n, n))
    c = np.exp(0.7 * W.gaussian_field(rng, n, 0.1, h))
    f = rng.standard_normal((n, n))
    return TC.mask_plane(inner, neu, h, lam, c, f, levels=0, i0=-41 - seed, j0=-13 + 2 * seed, seed=seed,
                        order="shuffle" if seed % 2 else "rowmajor")


def brute_hierarchy(i, j, kind, levels):
    """Re-derive every level (rules M1-M6) with dicts keyed on (I,J).
    Returns a list of dicts: pts (sorted by (J,I)), kind, colour, nbr."""
    cur = {(int(a), int(b)): int(k) for a, b, k in zip(i, j, kind)}
    out = []
    D4 = [(-1, 0), (1, 0), (0, -1), (0, 1)]
    for s in range(levels):
        pts = sorted(cur.keys(), key=lambda p: (p[1], p[0]))
        idx = {p: k for k, p in enumerate(pts)}
        kd = np.array([cur[p] for p in pts], np.uint8)
        col = np.array([2 if cur[p] != 0 else ((p[0] + p[1]) % 2) for p in pts], np.uint8)
        nbr = np.array([[idx.get((p[0] + d[0], p[1] + d[1]), -1) for d in D4] for p in pts], np.int32)
        out.append(dict(pts=pts, kind=kd, colour=col, nbr=nbr, map=cur))
        if s == levels - 1:
            break
        inner_c = {(p[0] // 2, p[1] // 2) for p, k in cur.items() if k == 0 and p[0] % 2 == 0 and p[1] % 2 == 0}
        nxt = {p: 0 for p in inner_c}
        for q in inner_c:
            for d in D4:
                g = (q[0] + d[0], q[1] + d[1])
                if g in inner_c or g in nxt:
                    continue
                any_dir = False
                for e in D4:
                    qq = (g[0] + e[0], g[1] + e[1])
                    if qq not in inner_c:
                        continue
                    m = (g[0] + qq[0], g[1] + qq[1])
                    if cur.get(m, -1) == 0:
                        cand = cur[(2 * g[0], 2 * g[1])]
                    else:
                        cand = cur[m]
                    assert cand in (1, 2)
                    any_dir |= cand == 1
                nxt[g] = 1 if any_dir else 2
        cur = nxt
    return out
