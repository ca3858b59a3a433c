"""The measurement switches that select another kernel variant or another memory order (environment variables read once per
process, hence subprocesses) must not change results: MG_B200_NO_STRIPS (shared-memory tile code instead of the register-tiled
smoother) gives the SAME BITS everywhere — both evaluate rows through row_d1 / neumann_point in the same order — and the tile orders
of the layout study (MG_B200_TILE_ORDER, profiles/r02_layout.md) give the same bits in every grid operation (a tile's arithmetic
does not depend on where the tile lives) and the same solve up to the summation order of the Krylov inner products, which run
over memory order; each variant also meets the oracle bar."""
import os
import subprocess
import sys

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

CODE = r"""
import sys, numpy as np, torch
from oracle import oracle as om
from paper_2509_11831_b200 import binding as B
from tests import helpers as H
out = sys.argv[1]
B.lib(); B.use_torch_allocator()
dev = lambda a: torch.from_numpy(np.ascontiguousarray(a, dtype=np.float64)).cuda()
pl = H.random_blob_plane(302, 769)
s = B.Solver(pl.i, pl.j, pl.kind, pl.h, levels=pl.levels)
s.update_coeffs(dev(pl.lam), dev(pl.c))
rng = np.random.default_rng(5)
n0 = s.level_n(0)
x, b = rng.standard_normal(n0), rng.standard_normal(n0)
xs, dc = s.smooth_restrict(0, dev(x), dev(b), 2)
vc = s.vcycle(0, dev(x), dev(b))
sol, iters, relres, rc = s.solve(dev(pl.f), dev(pl.x0), 1e-10)
o = om.Oracle(pl.i, pl.j, pl.kind, pl.h, levels=pl.levels)
o.update(pl.lam, pl.c)
ro = o.solve(pl.f, pl.x0, 1e-10)
err = np.linalg.norm(sol.cpu().numpy() - ro["x"]) / np.linalg.norm(ro["x"])
assert rc == 0 and abs(iters - ro["iters"]) <= 1 and err <= 1e-8, (rc, iters, ro["iters"], err)
np.savez(out, xs=xs.cpu().numpy(), dc=dc.cpu().numpy(), vc=vc.cpu().numpy(), sol=sol.cpu().numpy(), iters=iters, relres=relres)
print("ok", iters, err)
"""


def _run(tmp_path, name, **env):
    out = str(tmp_path / (name + ".npz"))
    e = dict(os.environ, **env)
    for k in ("MG_B200_NO_STRIPS", "MG_B200_TILE_ORDER", "MG_B200_FORCE_BLOCK"):
        if k not in env:
            e.pop(k, None)
    r = subprocess.run([sys.executable, "-c", CODE, out], env=e, cwd=ROOT, capture_output=True, text=True, timeout=900)
    assert r.returncode == 0 and r.stdout.strip().startswith("ok"), r.stderr[-3000:]
    return np.load(out)


def test_kernel_variants_and_tile_orders_give_the_same_bits(tmp_path):
    base = _run(tmp_path, "default")
    for name, env in (("no_strips", {"MG_B200_NO_STRIPS": "1"}), ("morton", {"MG_B200_TILE_ORDER": "1"}),
                      ("parent_grouped", {"MG_B200_TILE_ORDER": "2"})):
        v = _run(tmp_path, name, **env)
        for k in ("xs", "dc", "vc"):
            assert np.array_equal(base[k], v[k]), (name, k, float(np.abs(base[k] - v[k]).max()))
        assert int(base["iters"]) == int(v["iters"]), name
        if name == "no_strips":
            assert np.array_equal(base["sol"], v["sol"]) and float(base["relres"]) == float(v["relres"])
        else:
            assert np.linalg.norm(base["sol"] - v["sol"]) <= 1e-12 * np.linalg.norm(base["sol"])
