"""Planes batched inside the kernels (one elliptic solve per poloidal
plane, all planes on the same mesh).  A handle with P planes keeps the mesh tables once, every vector P times, and
launches every kernel once for all planes (gridDim.y = P) with one fGMRES state per plane.  The bar: batched == P
separate handles BIT FOR BIT (x, iteration counts, residuals), and each plane matches the oracle."""
import numpy as np
import pytest

from paper_2509_11831_b200 import workloads as W
from tests import helpers as H
from tests.test_gpu_parity import TOL_SOLVE, dev, gpu, host, rel  # noqa: F401  (gpu is a fixture)

pytestmark = pytest.mark.gpu


def _planes(cfg, lattice, P):
    pls = [W.make_plane(cfg, lattice, seed=W.SEEDS[cfg] + 31 * p) for p in range(P)]
    for pl in pls[1:]:
        assert np.array_equal(pl.i, pls[0].i) and np.array_equal(pl.kind, pls[0].kind)
    return pls


def _stack(pls, name):
    return np.stack([getattr(pl, name) for pl in pls])


@pytest.mark.parametrize("cfg,lattice,P,kw", [(2, 257, 5, {}), (3, 257, 3, dict(nu_pre=3, nu_post=1, restart_m=8)),
                                              (3, 1025, 2, {}), (2, 129, 16, dict(gamma=2)), (3, 257, 3, dict(restart_m=40))])
def test_batched_planes_equal_separate_handles(gpu, oracle_mod, cfg, lattice, P, kw):
    import torch
    pls = _planes(cfg, lattice, P)
    p0 = pls[0]
    lam, c, f, x0 = (_stack(pls, k) for k in ("lam", "c", "f", "x0"))
    if P >= 3:
        f[1] = 0.0                                   # K1: zero right-hand side on one plane -> x = 0, 0 iterations
        x0[1] = 1.0
    okw = dict(levels=p0.levels, nu_pre=kw.get("nu_pre", 2), nu_post=kw.get("nu_post", 2), m=kw.get("restart_m", 30), gamma=kw.get("gamma", 1))
    ref = []
    for p in range(P):                               # oracle per plane
        o = oracle_mod.Oracle(p0.i, p0.j, p0.kind, p0.h, **okw)
        o.update(lam[p], c[p])
        ref.append(o.solve(f[p], x0[p], 1e-10))
    if P >= 3:
        x0[2] = ref[2]["x"]                          # one plane starts from its solution: converged before the first cycle
        ref[2] = dict(x=ref[2]["x"], iters=0, status=0)
    seq = []
    for p in range(P):                               # P separate single-plane handles
        s = gpu.Solver(p0.i, p0.j, p0.kind, p0.h, levels=p0.levels, **kw)
        s.update_coeffs(dev(lam[p]), dev(c[p]))
        x, it, rr, rc = s.solve(dev(f[p]), dev(x0[p]), 1e-10)
        seq.append((host(x), it, rr, rc))
        s.close()
    sb = gpu.Solver(p0.i, p0.j, p0.kind, p0.h, levels=p0.levels, planes=P, **kw)
    for rep in range(2):                             # twice: the state of every plane is re-initialised per solve
        sb.update_coeffs(dev(lam), dev(c))
        xb, its, rrs, rc = sb.solve(dev(f), dev(x0), 1e-10)
        xb = host(xb)
        assert rc == 0 and xb.shape == (P, p0.n)
        for p in range(P):
            assert its[p] == seq[p][1] and rrs[p] == seq[p][2], (p, its, [q[1] for q in seq])
            assert np.array_equal(xb[p], seq[p][0]), p
            assert abs(its[p] - ref[p]["iters"]) <= 1 and rel(xb[p], ref[p]["x"]) <= TOL_SOLVE
    assert len(set(its)) > 1                         # the planes really stop at different iterations
    # host-buffer entry points carry all planes too
    sb.update_coeffs_host(lam, c)
    xh, its2, rrs2, rc2 = sb.solve_host(f, x0, 1e-10)
    assert rc2 == 0 and list(its2) == list(its) and np.array_equal(xh, xb)
    torch.cuda.synchronize()
    sb.close()


def test_batched_planes_per_plane_status(gpu):
    """One plane cannot reach rtol within max_iters, the others can: the call returns the worst status, every plane
    reports its own count, and the converged planes are unaffected (bit for bit) by the one that keeps iterating."""
    P = 3
    pls = _planes(2, 129, P)
    p0 = pls[0]
    lam, c, f, x0 = (_stack(pls, k) for k in ("lam", "c", "f", "x0"))
    f[1] *= 1e-6                                    # scaling f does not change the iteration count ...
    s = gpu.Solver(p0.i, p0.j, p0.kind, p0.h, levels=p0.levels, planes=P, max_iters=200)
    s.update_coeffs(dev(lam), dev(c))
    x_ok, its_ok, _, rc = s.solve(dev(f), dev(x0), 1e-10)
    assert rc == 0
    s.close()
    cap = min(its_ok) - 2                           # ... so cap below what every plane needs except none: all capped
    s = gpu.Solver(p0.i, p0.j, p0.kind, p0.h, levels=p0.levels, planes=P, max_iters=cap)
    s.update_coeffs(dev(lam), dev(c))
    x, its, rrs, rc = s.solve(dev(f), dev(x0), 1e-10)
    assert rc == 1 and list(its) == [cap] * P and all(r >= 1e-10 for r in rrs)
    s.close()
    # a mixed outcome: plane 0 starts from the converged solution (0 iterations), plane 1, 2 are capped
    x0m = x0.copy(); x0m[0] = host(x_ok)[0]
    s = gpu.Solver(p0.i, p0.j, p0.kind, p0.h, levels=p0.levels, planes=P, max_iters=cap)
    s.update_coeffs(dev(lam), dev(c))
    x, its, rrs, rc = s.solve(dev(f), dev(x0m), 1e-10)
    assert rc == 1 and its[0] == 0 and its[1] == cap and its[2] == cap and rrs[0] < 1e-10
    assert np.array_equal(host(x)[0], host(x_ok)[0])
    assert "plane" in gpu.last_error()
    s.close()


def test_batched_planes_three_field_form(gpu, oracle_mod):
    """The three-field form (Eq. 3) with planes: every plane has its own xi; batched == separate handles bit for bit on a
    mesh large enough for the register-tiled kernels (their multi-plane, xi-carrying instantiation), and each plane matches the oracle."""
    P = 2
    pls = _planes(3, 1025, P)
    p0 = pls[0]
    lam, c, f, x0 = (_stack(pls, k) for k in ("lam", "c", "f", "x0"))
    xi = np.stack([W.xi_field(pl, seed=40 + p) for p, pl in enumerate(pls)])
    seq = []
    for p in range(P):
        s = gpu.Solver(p0.i, p0.j, p0.kind, p0.h, levels=p0.levels)
        s.update_coeffs3(dev(lam[p]), dev(xi[p]), dev(c[p]))
        x, it, rr, rc = s.solve(dev(f[p]), dev(x0[p]), 1e-10)
        seq.append((host(x), it, rr, rc))
        s.close()
    sb = gpu.Solver(p0.i, p0.j, p0.kind, p0.h, levels=p0.levels, planes=P)
    sb.update_coeffs3(dev(lam), dev(xi), dev(c))
    xb, its, rrs, rc = sb.solve(dev(f), dev(x0), 1e-10)
    assert rc == 0
    for p in range(P):
        assert its[p] == seq[p][1] and rrs[p] == seq[p][2] and np.array_equal(host(xb)[p], seq[p][0])
    o = oracle_mod.Oracle(p0.i, p0.j, p0.kind, p0.h, levels=p0.levels)
    o.update3(lam[1], xi[1], c[1])
    ro = o.solve(f[1], x0[1], 1e-10)
    assert abs(its[1] - ro["iters"]) <= 1 and rel(host(xb)[1], ro["x"]) <= TOL_SOLVE
    sb.close()


@pytest.mark.parametrize("seed", list(range(230, 238)))
def test_random_mesh_options_planes_and_solvers(gpu, oracle_mod, seed):
    """Seeded sweep: ragged random domain x V(nu1,nu2) x V/W/F cycle x restart length x outer solver (fGMRES / BiCGStab) x 2-4 planes
    with per-plane coefficients and right-hand sides.  Batched == separate handles bit for bit; every plane against the oracle
    (fGMRES: iterations +-1; BiCGStab: applications +-2, see tests/test_gpu_bicgstab.py)."""
    rng = np.random.default_rng(seed)
    n = int(rng.choice([97, 129, 193, 257]))
    nu1, nu2 = max(1, int(rng.integers(0, 4))), int(rng.integers(0, 4))
    gamma, m = int(rng.choice([1, 1, 2, 3])), int(rng.choice([5, 12, 30]))
    solver, P = int(rng.integers(0, 2)), int(rng.integers(2, 5))
    pl = H.random_blob_plane(seed, n)
    lam = np.stack([pl.lam * (1.0 + 0.3 * rng.uniform(-1, 1, pl.n)) for _ in range(P)])
    c = np.stack([pl.c * np.exp(0.3 * rng.standard_normal(pl.n)) for _ in range(P)])
    f = np.stack([pl.f if p == 0 else rng.standard_normal(pl.n) for p in range(P)])
    x0 = np.zeros((P, pl.n))
    kw = dict(levels=pl.levels, nu_pre=nu1, nu_post=nu2, restart_m=m, gamma=gamma, max_iters=150, solver=solver)
    seq = []
    for p in range(P):
        s = gpu.Solver(pl.i, pl.j, pl.kind, pl.h, **kw)
        s.update_coeffs(dev(lam[p]), dev(c[p]))
        x, it, rr, rc = s.solve(dev(f[p]), dev(x0[p]), 1e-10)
        seq.append((host(x), it, rr, rc))
        s.close()
    sb = gpu.Solver(pl.i, pl.j, pl.kind, pl.h, planes=P, **kw)
    sb.update_coeffs(dev(lam), dev(c))
    xb, its, rrs, rcb = sb.solve(dev(f), dev(x0), 1e-10)
    sb.close()
    assert rcb == max(q[3] for q in seq)
    for p in range(P):
        assert its[p] == seq[p][1] and rrs[p] == seq[p][2] and np.array_equal(host(xb)[p], seq[p][0]), (p, its, [q[1] for q in seq])
    o = oracle_mod.Oracle(pl.i, pl.j, pl.kind, pl.h, levels=pl.levels, nu_pre=nu1, nu_post=nu2, m=m, gamma=gamma, max_iters=150)
    for p in (0, P - 1):
        o.update(lam[p], c[p])
        ro = o.solve_bicgstab(f[p], x0[p], 1e-10) if solver else o.solve(f[p], x0[p], 1e-10)
        if ro["status"] == 0 and seq[p][3] == 0:
            assert abs(its[p] - ro["iters"]) <= (2 if solver else 1) and rel(host(xb)[p], ro["x"]) <= TOL_SOLVE, (p, its[p], ro["iters"])
        else:
            assert ro["status"] == seq[p][3] or solver == 1, (ro["status"], seq[p][3])
