"""CPU tests of the product's host side (-m "not gpu"): the C-ABI library loads and exports every
symbol include/mg_b200.h declares, and its host setup (level point lists, guard classification,
colours, neighbour maps, Neumann stencil codes, transfer tables) is BIT-EXACT against the oracle
(north_star: "mesh/level index construction bit-exact").  No compute call is made."""
import os
import re

import numpy as np
import pytest

from paper_2509_11831_b200 import binding as B
from paper_2509_11831_b200 import workloads as W
from tests import helpers as H

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_exports_every_declared_symbol():
    hdr = open(os.path.join(ROOT, "include", "mg_b200.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(mg_[a-z_0-9]+)\s*\(", hdr)) - {"mg_alloc_fn", "mg_free_fn"}
    assert declared == set(B.EXPORTS)
    L = B.lib()
    for name in declared:
        assert hasattr(L, name), name


def test_error_codes_without_device():
    L = B.lib()
    assert L.mg_strerror(0) == b"ok"
    pl = H.square_plane(9, 1)
    s = B.Solver(pl.i, pl.j, pl.kind, pl.h, levels=1, host_only=True)
    assert s.levels == 1 and s.level_n(0) == pl.n
    import ctypes as C
    # compute calls on a host-only handle fail loudly (no CPU fallback)
    assert L.mg_update_coeffs(s._h, C.c_void_p(8), C.c_void_p(8), None) == -5
    assert L.mg_apply(s._h, 0, C.c_void_p(8), C.c_void_p(8), None) == -5
    # ... including the solve and the host-buffer entry points (MG_ECUDA, not an allocation failure)
    buf = np.zeros(pl.n)
    p = C.c_void_p(buf.ctypes.data)
    assert L.mg_solve(s._h, p, p, p, C.c_double(1e-10), None, None, None) == -5
    assert L.mg_solve_host(s._h, p, p, p, C.c_double(1e-10), None, None, None) == -5
    assert L.mg_update_coeffs_host(s._h, p, p, None) == -5
    assert L.mg_update_coeffs3_host(s._h, p, p, p, None) == -5
    # diagnostics before the first solve; option range (gamma 0..3, flag bits 0..2)
    assert s.last_reorth == -1 and len(s.last_history()[0]) == 0
    assert L.mg_last_history(None, None, None, 4) == -1 and L.mg_last_reorth(None) == -1
    for g in (0, 1, 2, 3):
        B.Solver(pl.i, pl.j, pl.kind, pl.h, levels=1, host_only=True, gamma=g, full_cgs2=True).close()
    with pytest.raises(B.MgError):
        B.Solver(pl.i, pl.j, pl.kind, pl.h, levels=1, host_only=True, gamma=4)
    with pytest.raises(B.MgError):
        B.Solver(pl.i, pl.j, pl.kind, -1.0, host_only=True)
    with pytest.raises(B.MgError):
        B.Solver(np.append(pl.i, pl.i[0]), np.append(pl.j, pl.j[0]), np.append(pl.kind, pl.kind[0]), pl.h, host_only=True)
    keep = np.ones(pl.n, bool)
    keep[np.nonzero(pl.kind != 0)[0][0]] = False
    with pytest.raises(B.MgError):
        B.Solver(pl.i[keep], pl.j[keep], pl.kind[keep], pl.h, host_only=True)


CASES = {
    "square65": lambda: W.make_plane(1),
    "annulus129_shuffled": lambda: W.make_plane(2, 129, order="shuffle"),
    "annulus65_negative_origin": lambda: H.small_annulus(65, 4, i0=-37, j0=-22),
    "dshape257": lambda: W.make_plane(3, 257),
    "dshape129_auto": lambda: W.make_plane(3, 129, levels=0),
}


for _k in range(8):
    CASES[f"random_blob_{_k}"] = (lambda k: (lambda: H.random_blob_plane(100 + k)))(_k)


@pytest.mark.parametrize("case", list(CASES))
def test_hierarchy_bit_exact_vs_oracle(oracle_mod, case):
    pl = CASES[case]()
    o = oracle_mod.Oracle(pl.i, pl.j, pl.kind, pl.h, levels=pl.levels)
    s = B.Solver(pl.i, pl.j, pl.kind, pl.h, levels=pl.levels, host_only=True)
    assert s.levels == o.levels
    for lv in range(o.levels):
        a, g = o.level_arrays(lv), s.level_info(lv)
        assert s.level_n(lv) == o.level_n(lv)
        for k in ("I", "J", "kind", "colour", "nbr", "ns_fallback"):
            assert np.array_equal(a[k], g[k]), (lv, k)
        neu = a["kind"] == 2
        assert np.array_equal(a["ns_tn"][neu], g["ns_tn"][neu])
        assert len(np.unique(g["slot"])) == len(g["slot"])
    assert np.array_equal(o.user2canon, s.level_info(0)["user2canon"])
    for lv in range(o.levels - 1):
        a, g = o.transfer_tables(lv), s.transfer_info(lv)
        assert np.array_equal(a["fine9"], g["fine9"])
        assert np.array_equal(a["ptype"], g["ptype"])
        # the oracle lists parents with their weights; the library lists them in the same order, -1 padded
        exp = np.where(a["parent_w"] > 0, a["parent"], -1)
        assert np.array_equal(exp, g["parent"])
    s.close()


@pytest.mark.parametrize("order", [1, 2])
def test_tile_order_is_a_layout_choice_only(order):
    """MG_B200_TILE_ORDER (Morton / parent-grouped tile ids; the ordering study of profiles/r02_layout.md) changes where a tile
    lives in memory, nothing else: every canonical index array stays bit-exact against the oracle and the slot map stays a
    permutation.  The variable is read once per process, hence the subprocess."""
    import subprocess
    import sys
    code = (
        "import numpy as np\n"
        "from oracle import oracle as om\n"
        "from paper_2509_11831_b200 import binding as B, workloads as W\n"
        "from tests import helpers as H\n"
        "for pl in (W.make_plane(3, 257), H.random_blob_plane(103), H.small_annulus(65, 4, i0=-37, j0=-22)):\n"
        "    o = om.Oracle(pl.i, pl.j, pl.kind, pl.h, levels=pl.levels)\n"
        "    s = B.Solver(pl.i, pl.j, pl.kind, pl.h, levels=pl.levels, host_only=True)\n"
        "    assert s.levels == o.levels\n"
        "    slots = []\n"
        "    for lv in range(o.levels):\n"
        "        a, g = o.level_arrays(lv), s.level_info(lv)\n"
        "        for k in ('I', 'J', 'kind', 'colour', 'nbr', 'ns_fallback'):\n"
        "            assert np.array_equal(a[k], g[k]), (lv, k)\n"
        "        assert len(np.unique(g['slot'])) == len(g['slot'])\n"
        "        slots.append(g['slot'])\n"
        "    assert np.array_equal(o.user2canon, s.level_info(0)['user2canon'])\n"
        "    for lv in range(o.levels - 1):\n"
        "        a, g = o.transfer_tables(lv), s.transfer_info(lv)\n"
        "        assert np.array_equal(a['fine9'], g['fine9']) and np.array_equal(a['ptype'], g['ptype'])\n"
        "print('ok', sum(int(x.sum()) for x in slots))\n")
    outs = {}
    for o in (0, order):
        env = dict(os.environ, MG_B200_TILE_ORDER=str(o))
        r = subprocess.run([sys.executable, "-c", code], env=env, cwd=ROOT, capture_output=True, text=True, timeout=600)
        assert r.returncode == 0 and r.stdout.startswith("ok"), r.stderr[-2000:]
        outs[o] = r.stdout
    assert outs[0] != outs[order]          # the slots really moved (last mesh has several tiles on level 0)
