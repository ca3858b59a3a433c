"""Pins P11 (hierarchy) and the structural part of P2 for the oracle's host-side mesh construction.
Checked against: counts that follow from PAPER.md:78's definitions (tests/golden), an independent
dict-based brute-force re-derivation (tests/helpers.py), the paper's printed Neumann stencils
(Eq. 14/15, tests/golden/neumann_stencils.txt) and invariants stated at PAPER.md:123, 131, 163."""
import os

import numpy as np
import pytest

from paper_2509_11831_b200 import workloads as W
from tests import helpers as H

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _read_counts():
    rows = []
    for line in open(os.path.join(GOLD, "config1_level_counts.txt")):
        if line.strip() and not line.startswith("#"):
            rows.append(tuple(int(t) for t in line.split()))
    return rows


def _read_stencils():
    tab = {}
    for line in open(os.path.join(GOLD, "neumann_stencils.txt")):
        if not line.strip() or line.startswith("#"):
            continue
        a, b, c = line.split("|")
        tn = tuple(int(t) for t in a.split())
        t = b.split()
        nodes = sorted((int(t[k]), int(t[k + 1]), float(t[k + 2])) for k in range(0, len(t), 3))
        tab[tn] = (nodes, int(c))
    return tab


def test_config1_counts(oracle_mod):
    pl = W.make_plane(1)
    o = oracle_mod.Oracle(pl.i, pl.j, pl.kind, pl.h, levels=4)
    assert o.levels == 4
    for s, n, nin in _read_counts():
        a = o.level_arrays(s)
        assert o.level_n(s) == n
        assert int((a["kind"] == 0).sum()) == nin
        assert o.level_h(s) == pytest.approx(pl.h * 2 ** s, rel=0, abs=0)


def test_annulus_inner_count_bruteforce():
    pl = W.make_plane(2, 129)
    n, h = 129, 2.0 / 128
    cnt = 0
    for j in range(n):
        for i in range(n):
            r2 = (-1 + i * h) ** 2 + (-1 + j * h) ** 2
            cnt += (0.09 < r2 < 1.0) and 0 < i < n - 1 and 0 < j < n - 1
    assert abs(pl.n_inner - cnt) <= 4          # sqrt rounding on the circle itself


@pytest.mark.parametrize("geom", ["square", "annulus", "annulus_neg", "dshape", "dshape_shuffled"])
def test_hierarchy_vs_bruteforce(oracle_mod, geom):
    if geom == "square":
        pl = H.square_plane(33, 4)
    elif geom == "annulus":
        pl = H.small_annulus(65, 4)
    elif geom == "annulus_neg":
        pl = H.small_annulus(65, 4, i0=-37, j0=-22)       # negative and odd lattice origin (rule M1)
    elif geom == "dshape":
        pl = H.small_dshape(129, 5)
    else:
        pl = H.small_dshape(65, 4, order="shuffle")
    o = oracle_mod.Oracle(pl.i, pl.j, pl.kind, pl.h, levels=pl.levels)
    ref = H.brute_hierarchy(pl.i, pl.j, pl.kind, o.levels)
    for s in range(o.levels):
        a, r = o.level_arrays(s), ref[s]
        assert o.level_n(s) == len(r["pts"])
        assert np.array_equal(a["I"], np.array([p[0] for p in r["pts"]], np.int32))
        assert np.array_equal(a["J"], np.array([p[1] for p in r["pts"]], np.int32))
        assert np.array_equal(a["kind"], r["kind"])
        assert np.array_equal(a["colour"], r["colour"])
        assert np.array_equal(a["nbr"], r["nbr"])
        # invariants: inner points have 4 neighbours; guards have an inner 4-neighbour (M2)
        inner = a["kind"] == 0
        assert (a["nbr"][inner] >= 0).all()
        nb_inner = np.where(a["nbr"] >= 0, inner[np.maximum(a["nbr"], 0)], False)
        assert nb_inner[~inner].any(axis=1).all()
        # red-black independence: no inner neighbour of an inner point has its colour
        for d in range(4):
            q = a["nbr"][inner, d]
            same = (a["colour"][q] == a["colour"][inner]) & (a["kind"][q] == 0)
            assert not same.any()
        # E(W(l)) = l
        w = a["nbr"][:, 0]
        ok = w >= 0
        assert np.array_equal(a["nbr"][w[ok], 1], np.nonzero(ok)[0].astype(np.int32))
    # Inner_{s+1} subset of Inner_s at doubled indices
    for s in range(o.levels - 1):
        fa, ca = o.level_arrays(s), o.level_arrays(s + 1)
        fine_inner = {(int(i), int(j)) for i, j, k in zip(fa["I"], fa["J"], fa["kind"]) if k == 0}
        for i, j, k in zip(ca["I"], ca["J"], ca["kind"]):
            if k == 0:
                assert (2 * int(i), 2 * int(j)) in fine_inner


@pytest.mark.parametrize("geom", ["annulus", "dshape"])
def test_neumann_stencils(oracle_mod, geom):
    tab = _read_stencils()
    pl = H.small_annulus(129, 5) if geom == "annulus" else H.small_dshape(257, 6)
    o = oracle_mod.Oracle(pl.i, pl.j, pl.kind, pl.h, levels=pl.levels)
    seen = set()
    for s in range(o.levels):
        a = o.level_arrays(s)
        h = o.level_h(s)
        mp = {(int(i), int(j)): int(k) for i, j, k in zip(a["I"], a["J"], a["kind"])}
        psi2 = lambda p: {0: 2, 1: 1, 2: 1}.get(mp.get(p, -1), 0)          # Eq. 12 doubled
        for l in np.nonzero(a["kind"] == 2)[0]:
            I, J = int(a["I"][l]), int(a["J"][l])
            tn = (psi2((I + 1, J)) - psi2((I - 1, J)), psi2((I, J + 1)) - psi2((I, J - 1)))   # Eq. 13
            assert tuple(int(t) for t in a["ns_tn"][l]) == tn
            nodes = sorted((int(a["I"][q]) - I, int(a["J"][q]) - J, float(w))
                           for q, w in zip(a["ns_idx"][l], a["ns_w"][l]) if q >= 0)
            # a boundary row depends on inner points only
            assert all(a["kind"][q] == 0 for q in a["ns_idx"][l] if q >= 0)
            assert len(nodes) >= 1
            wsum = sum(w for _, _, w in nodes) + a["ns_wself"][l]
            assert wsum == pytest.approx(1.0, abs=1e-15)
            if a["ns_fallback"][l]:
                assert a["ns_delta"][l] == h and a["ns_wself"][l] == 0.0
                assert all(abs(dx) + abs(dy) == 1 for dx, dy, _ in nodes)
                continue
            assert a["ns_delta"][l] == pytest.approx(h * np.sqrt(tn[0] ** 2 + tn[1] ** 2) / 2, rel=1e-15)
            if tn in tab:
                exp_nodes, n2 = tab[tn]
                assert nodes == exp_nodes and a["ns_wself"][l] == 0.0
                assert tn[0] ** 2 + tn[1] ** 2 == n2
                seen.add(tn)
            assert len(nodes) + (a["ns_wself"][l] > 0) <= 4
    assert len(seen) >= 6          # the printed cases do occur in these geometries


def test_transfer_tables(oracle_mod):
    pl = H.small_annulus(65, 3, i0=-11, j0=5)
    o = oracle_mod.Oracle(pl.i, pl.j, pl.kind, pl.h, levels=3)
    for s in range(o.levels - 1):
        fa, ca, t = o.level_arrays(s), o.level_arrays(s + 1), o.transfer_tables(s)
        fmap = {(int(i), int(j)): k for k, (i, j) in enumerate(zip(fa["I"], fa["J"]))}
        cmap = {(int(i), int(j)): k for k, (i, j) in enumerate(zip(ca["I"], ca["J"]))}
        for q in range(o.level_n(s + 1)):
            exp = [fmap.get((2 * int(ca["I"][q]) + dx, 2 * int(ca["J"][q]) + dy), -1)
                   for dy in (-1, 0, 1) for dx in (-1, 0, 1)]
            assert list(t["fine9"][q]) == exp
        for l in range(o.level_n(s)):
            I, J = int(fa["I"][l]), int(fa["J"][l])
            cands = [((I + a) // 2, (J + b) // 2) for b in ((0,) if J % 2 == 0 else (-1, 1))
                     for a in ((0,) if I % 2 == 0 else (-1, 1))]
            exp = sorted(cmap.get(p, -1) for p in cands)
            got = sorted(int(v) for v, w in zip(t["parent"][l], t["parent_w"][l]) if w > 0)
            assert got == exp
            assert t["parent_w"][l].sum() == 1.0
            assert t["ptype"][l] == (I % 2) + 2 * (J % 2)


def test_invalid_meshes(oracle_mod):
    pl = H.square_plane(9, 1)
    with pytest.raises(ValueError):                      # duplicate point
        oracle_mod.Oracle(np.append(pl.i, pl.i[0]), np.append(pl.j, pl.j[0]), np.append(pl.kind, pl.kind[0]), pl.h)
    keep = np.ones(pl.n, bool)
    keep[np.nonzero(pl.kind != 0)[0][0]] = False         # drop a guard: an inner point lacks a neighbour
    with pytest.raises(ValueError):
        oracle_mod.Oracle(pl.i[keep], pl.j[keep], pl.kind[keep], pl.h)
    with pytest.raises(ValueError):                      # stray guard with no inner neighbour
        oracle_mod.Oracle(np.append(pl.i, 40), np.append(pl.j, 40), np.append(pl.kind, 1).astype(np.uint8), pl.h)


def test_auto_levels(oracle_mod):
    pl = W.make_plane(1)
    o = oracle_mod.Oracle(pl.i, pl.j, pl.kind, pl.h, levels=0)
    assert o.levels == 4                                  # 65 -> 33 -> 17 -> 9 (rule M8)
    o = oracle_mod.Oracle(pl.i, pl.j, pl.kind, pl.h, levels=12)
    assert o.levels == 6                                  # 3x3 lattice keeps one inner point; next is empty
