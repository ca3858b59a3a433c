"""GPU parity at BASELINE.json's FULL sizes (-m gpu), in the configuration bench.py times: the oracle's complete solve of
configs 3, 4 and 5 (first three time steps) beside the CUDA path's — iteration counts equal +-1, solutions within 1e-8
relative L2, per-level coefficients within 1e-13 (north_star) — plus the coarsest-level direct solve at the sizes where
the cooperative multi-CTA inverse runs, and the error paths that need a device."""
import numpy as np
import pytest

from paper_2509_11831_b200 import workloads as W
from tests import cases as TC
from tests import helpers as H
from tests.test_gpu_parity import TOL_SOLVE, TOL_STEP, dev, gpu, host, rel  # noqa: F401  (gpu is a fixture)

pytestmark = pytest.mark.gpu


def _coeff_parity(o, s):
    for lv in range(o.levels):
        lo, co = o.level_coeffs(lv)
        lg, cg = s.level_coeffs(lv)
        assert rel(lg, lo) <= TOL_STEP and rel(cg, co) <= TOL_STEP


def test_full_size_config3(gpu, oracle_mod):
    """BASELINE.json configs[2]: 1025^2 D-shape, 10^3 coefficient contrast with a jump, 8 levels."""
    pl = W.make_plane(3)
    assert pl.lattice == 1025 and pl.levels == 8
    o = oracle_mod.Oracle(pl.i, pl.j, pl.kind, pl.h, levels=pl.levels)
    o.update(pl.lam, pl.c)
    ro = o.solve(pl.f, pl.x0, 1e-10)
    s = gpu.Solver(pl.i, pl.j, pl.kind, pl.h, levels=pl.levels)
    s.update_coeffs(dev(pl.lam), dev(pl.c))
    _coeff_parity(o, s)
    x, iters, relres, rc = s.solve(dev(pl.f), dev(pl.x0), 1e-10)
    print(f"config 3 full size: n={pl.n} iters gpu/oracle={iters}/{ro['iters']} rel.err={rel(host(x), ro['x']):.2e}")
    assert rc == 0 and ro["status"] == 0 and abs(iters - ro["iters"]) <= 1
    assert rel(host(x), ro["x"]) <= TOL_SOLVE and relres < 1e-10
    s.close()


def test_full_size_config5_first_steps(gpu, oracle_mod):
    """BASELINE.json configs[4] at 2049^2 (2.8 M points, 9 levels): the first 3 of the 64 time steps, coefficients and
    right-hand side regenerated every step, each solve warm-started from the previous solution of its own side."""
    pl = W.make_plane(5)
    assert pl.lattice == 2049 and pl.levels == 9
    o = oracle_mod.Oracle(pl.i, pl.j, pl.kind, pl.h, levels=pl.levels)
    s = gpu.Solver(pl.i, pl.j, pl.kind, pl.h, levels=pl.levels)
    xo, xg, cur = pl.x0.copy(), dev(pl.x0), pl
    for k in range(3):
        o.update(cur.lam, cur.c)
        ro = o.solve(cur.f, xo, 1e-10)
        s.update_coeffs(dev(cur.lam), dev(cur.c))
        _coeff_parity(o, s)
        _, iters, relres, rc = s.solve(dev(cur.f), xg, 1e-10, x=xg)
        print(f"config 5 step {k}: iters gpu/oracle={iters}/{ro['iters']} rel.err={rel(host(xg), ro['x']):.2e}")
        assert rc == 0 and ro["status"] == 0 and abs(iters - ro["iters"]) <= 1
        assert rel(host(xg), ro["x"]) <= TOL_SOLVE and relres < 1e-10
        xo = ro["x"]
        cur = W.next_step(cur, k)
    s.close()


def test_full_size_config4_solve_vs_oracle(gpu, oracle_mod):
    """BASELINE.json configs[3] (4097^2, 11.3 M points, 10 levels), the bench workload: the oracle's complete
    fGMRES(30) + V(2,2) solve (about a minute and 6 GB of host memory) against the CUDA path's."""
    pl = W.make_plane(4)
    o = oracle_mod.Oracle(pl.i, pl.j, pl.kind, pl.h, levels=pl.levels)
    o.update(pl.lam, pl.c)
    ro = o.solve(pl.f, pl.x0, 1e-10)
    s = gpu.Solver(pl.i, pl.j, pl.kind, pl.h, levels=pl.levels)
    s.update_coeffs(dev(pl.lam), dev(pl.c))
    _coeff_parity(o, s)
    x, iters, relres, rc = s.solve(dev(pl.f), dev(pl.x0), 1e-10)
    print(f"config 4 full size: n={pl.n} iters gpu/oracle={iters}/{ro['iters']} rel.err={rel(host(x), ro['x']):.2e} "
          f"relres gpu/oracle={relres:.3e}/{ro['relres']:.3e}")
    assert rc == 0 and ro["status"] == 0 and abs(iters - ro["iters"]) <= 1
    assert rel(host(x), ro["x"]) <= TOL_SOLVE and relres < 1e-10
    s.close()


@pytest.mark.parametrize("lattice,n_expect", [(97, 468), (145, 1020)])
def test_coarse_solve_cooperative_inverse(gpu, oracle_mod, lattice, n_expect):
    """Rule C at the coarsest-level sizes the paper keeps (~400 points) and near the library's limit of
    1024: [A | I] no longer fits one CTA's shared memory, so the cooperative column-slab Gauss-Jordan runs.  Both sides
    are backward-stable direct solves of the same dense system: forward error <= O(cond(A) eps) (DESIGN.md tolerances);
    cond is computed here from the oracle's rows."""
    pl = H.small_annulus(lattice, 3)
    o = H.make_oracle(oracle_mod, pl)
    n = o.level_n(2)
    assert n == n_expect
    A = np.column_stack([o.apply(2, e) for e in np.eye(n)])
    cond = np.linalg.cond(A)
    s = gpu.Solver(pl.i, pl.j, pl.kind, pl.h, levels=3)
    s.update_coeffs(dev(pl.lam), dev(pl.c))
    rng = np.random.default_rng(40)
    for _ in range(3):
        b = rng.standard_normal(n)
        xg = host(s.coarse_solve(dev(b)))
        err_o, err_d = rel(xg, o.coarse_solve(b)), rel(xg, np.linalg.solve(A, b))
        print(f"coarse n={n} cond={cond:.3g} rel.err vs oracle={err_o:.2e} vs numpy={err_d:.2e}")
        assert err_o <= 20 * cond * np.finfo(float).eps and err_d <= 20 * cond * np.finfo(float).eps
    # and the cycle / solve built on it
    x, b = rng.standard_normal(o.level_n(0)), rng.standard_normal(o.level_n(0))
    assert rel(host(s.vcycle(0, dev(x), dev(b))), o.cycle(0, x, b)) <= 1e-12
    ro = o.solve(pl.f, pl.x0, 1e-10)
    xs, iters, relres, rc = s.solve(dev(pl.f), dev(pl.x0), 1e-10)
    assert rc == 0 and abs(iters - ro["iters"]) <= 1 and rel(host(xs), ro["x"]) <= TOL_SOLVE
    s.close()


@pytest.mark.parametrize("levels", [1, 2])
def test_singular_coarsest_operator_is_reported(gpu, oracle_mod, levels):
    """The oracle refuses a singular coarsest operator at update (-2).  The CUDA update is asynchronous: the zero pivot is
    flagged on the device and the next call that uses the operators returns MG_ECOEFF.  Exactly singular case: one
    coarsest inner point with Dirichlet guards and lambda = -(a_W + a_E + a_S + a_N), so a_ll = 0 and the point's
    column is zero (lambda < 0 is admissible as such, Eq. 21); all values are powers of two, so the
    restricted coefficients (rule T4) and a_ll are exact on both sides."""
    n = 3 if levels == 1 else 5
    h = 1.0 if levels == 1 else 0.5                      # coarsest spacing 1: kappa = 1/2, a_X = kappa (1 + 1) = 1
    pl = TC.mask_plane(W.square_mask(n), np.zeros((n, n), bool), h, lam_f=np.full((n, n), -4.0), c_f=np.ones((n, n)), levels=levels)
    o = oracle_mod.Oracle(pl.i, pl.j, pl.kind, pl.h, levels=levels)
    with pytest.raises(ValueError, match="singular"):
        o.update(pl.lam, pl.c)
    s = gpu.Solver(pl.i, pl.j, pl.kind, pl.h, levels=levels)
    s.update_coeffs(dev(pl.lam), dev(pl.c))
    f = np.ones(pl.n)
    with pytest.raises(gpu.MgError) as e:
        s.solve(dev(f), dev(np.zeros(pl.n)), 1e-10)
    assert e.value.code == -3 and "singular" in str(e.value)
    with pytest.raises(gpu.MgError) as e:               # single-step entry points consult the same flag
        s.coarse_solve(dev(np.ones(s.level_n(levels - 1))))
    assert e.value.code == -3
    lam_ok = np.full(pl.n, 1.0)                           # a valid update clears it
    s.update_coeffs(dev(lam_ok), dev(pl.c))
    o.update(lam_ok, pl.c)
    x, iters, relres, rc = s.solve(dev(f), dev(np.zeros(pl.n)), 1e-10)
    assert rc == 0 and rel(host(x), o.solve(f, np.zeros(pl.n), 1e-10)["x"]) <= TOL_SOLVE
    s.close()


def test_inadmissible_coefficients_block_single_steps(gpu):
    """mg_apply / mg_smooth / mg_vcycle after an update with c <= 0 return MG_ECOEFF like mg_solve."""
    pl = H.small_annulus(33, 2)
    s = gpu.Solver(pl.i, pl.j, pl.kind, pl.h, levels=2)
    c = pl.c.copy(); c[5] = -1.0
    s.update_coeffs(dev(pl.lam), dev(c))
    x = dev(np.ones(s.level_n(0)))
    for call in (lambda: s.apply(0, x), lambda: s.smooth(0, x, x, 1), lambda: s.vcycle(0, x, x)):
        with pytest.raises(gpu.MgError) as e:
            call()
        assert e.value.code == -3
    with pytest.raises(gpu.MgError) as e:
        s.solve(dev(pl.f), dev(pl.x0), 1e-10)
    assert e.value.code == -3 and s.last_solve_ms < 0     # no stale timing after the early return
    s.update_coeffs(dev(pl.lam), dev(pl.c))
    s.apply(0, x)
    s.close()


def test_not_converged_says_why(gpu):
    """rtol below the fp64 floor of the true residual: the recurrence residual passes it, the recomputed one cannot; the
    call returns MG_NOT_CONVERGED (the method has no stagnation exit) and mg_last_error says so."""
    pl = W.make_plane(3, 257)
    s = gpu.Solver(pl.i, pl.j, pl.kind, pl.h, levels=pl.levels, max_iters=60)
    s.update_coeffs(dev(pl.lam), dev(pl.c))
    x, iters, relres, rc = s.solve(dev(pl.f), dev(pl.x0), 1e-18)
    assert rc == 1 and iters == 60 and relres < 1e-11
    assert "attainable" in gpu.last_error()
    s.close()


@pytest.mark.parametrize("seed,lattice", [(301, 1025), (302, 769), (303, 1281)])
def test_register_tiled_smoother_on_ragged_large_meshes(gpu, oracle_mod, seed, lattice):
    """Levels of more than one tile per SM run the register-tiled smoother kernels (k_gs_strip): interior tiles and,
    with guard lists, masks and the boundary phase, general tiles.  Ragged random domains with holes, islands, mixed
    Dirichlet / Neumann guards, half-integer normals and fallback stencils at a size where level 0 (and 1) take that
    path: every fused variant against the oracle — plain sweeps, sweeps + restricted defect, correction + sweeps inside
    the cycle, and correction + sweeps + w = A x inside the solve."""
    pl = H.random_blob_plane(seed, lattice)
    o = oracle_mod.Oracle(pl.i, pl.j, pl.kind, pl.h, levels=pl.levels)
    o.update(pl.lam, pl.c)
    s = gpu.Solver(pl.i, pl.j, pl.kind, pl.h, levels=pl.levels)
    s.update_coeffs(dev(pl.lam), dev(pl.c))
    assert s.levels == o.levels
    rng = np.random.default_rng(seed)
    for lv in (0, 1):
        n = o.level_n(lv)
        x, b = rng.standard_normal(n), rng.standard_normal(n)
        for sweeps in (2, 3, 4):
            assert rel(host(s.smooth(lv, dev(x), dev(b), sweeps)), o.smooth(lv, x, b, sweeps)) <= TOL_STEP
        xo = o.smooth(lv, x, b, 2)
        do = o.restrict(lv, o.apply(lv, xo) - b)
        xg, dg = s.smooth_restrict(lv, dev(x), dev(b), 2)
        scale = np.linalg.norm(o.restrict(lv, np.abs(o.apply(lv, xo)) + np.abs(b)))
        assert rel(host(xg), xo) <= TOL_STEP and np.linalg.norm(host(dg) - do) <= TOL_STEP * max(scale, np.linalg.norm(do))
        assert rel(host(s.vcycle(lv, dev(x), dev(b))), o.cycle(lv, x, b)) <= 1e-12
    ro = o.solve(pl.f, pl.x0, 1e-10)
    xs, iters, relres, rc = s.solve(dev(pl.f), dev(pl.x0), 1e-10)
    print(f"blob {seed} {lattice}: n={pl.n} levels={o.levels} iters gpu/oracle={iters}/{ro['iters']} rel.err={rel(host(xs), ro['x']):.2e}")
    assert rc == ro["status"] == 0 and abs(iters - ro["iters"]) <= 1 and rel(host(xs), ro["x"]) <= TOL_SOLVE
    s.close()
    # odd sweep counts: the single-sweep forms of the same kernels (sweep + restricted defect, correction + sweep, correction + sweep +
    # apply) — V(3,1): pre-smoothing 2 + 1, post-smoothing 1
    o31 = oracle_mod.Oracle(pl.i, pl.j, pl.kind, pl.h, levels=pl.levels, nu_pre=3, nu_post=1)
    o31.update(pl.lam, pl.c)
    s31 = gpu.Solver(pl.i, pl.j, pl.kind, pl.h, levels=pl.levels, nu_pre=3, nu_post=1)
    s31.update_coeffs(dev(pl.lam), dev(pl.c))
    for lv in (0, 1):
        n = o31.level_n(lv)
        x, b = rng.standard_normal(n), rng.standard_normal(n)
        xo = o31.smooth(lv, x, b, 1)
        do = o31.restrict(lv, o31.apply(lv, xo) - b)
        xg, dg = s31.smooth_restrict(lv, dev(x), dev(b), 1)
        scale = np.linalg.norm(o31.restrict(lv, np.abs(o31.apply(lv, xo)) + np.abs(b)))
        assert rel(host(xg), xo) <= TOL_STEP and np.linalg.norm(host(dg) - do) <= TOL_STEP * max(scale, np.linalg.norm(do))
        assert rel(host(s31.vcycle(lv, dev(x), dev(b))), o31.cycle(lv, x, b)) <= 1e-12
    r31 = o31.solve(pl.f, pl.x0, 1e-10)
    x31, it31, _, rc31 = s31.solve(dev(pl.f), dev(pl.x0), 1e-10)
    assert rc31 == r31["status"] == 0 and abs(it31 - r31["iters"]) <= 1 and rel(host(x31), r31["x"]) <= TOL_SOLVE
    s31.close()


def test_allocator_is_captured_per_handle(gpu, oracle_mod):
    """a handle allocates and frees with the allocator pair that was installed when it was created, whatever
    mg_set_allocator is called with in between — also for its late allocations (host-buffer staging, the xi arrays of the first
    three-field update)."""
    import torch
    pl = H.small_annulus(65, 3)
    o = H.make_oracle(oracle_mod, pl)
    ro = o.solve(pl.f, pl.x0, 1e-10)
    gpu.use_torch_allocator()
    a = gpu.Solver(pl.i, pl.j, pl.kind, pl.h, levels=3)               # torch's caching allocator
    gpu.use_default_allocator()
    b = gpu.Solver(pl.i, pl.j, pl.kind, pl.h, levels=3)               # cudaMalloc
    gpu.use_torch_allocator()
    for s in (a, b):
        s.update_coeffs_host(pl.lam, pl.c)                            # late allocation: staging buffers
        x, iters, relres, rc = s.solve_host(pl.f, pl.x0, 1e-10)
        assert rc == 0 and abs(iters - ro["iters"]) <= 1 and rel(x, ro["x"]) <= TOL_SOLVE
        s.update_coeffs3(dev(pl.lam), dev(np.ones(pl.n)), dev(pl.c))  # late allocation: xi on every level
        x3, it3, _, rc3 = s.solve(dev(pl.f), dev(pl.x0), 1e-10)
        assert rc3 == 0 and rel(host(x3), ro["x"]) <= TOL_SOLVE
    gpu.use_default_allocator()
    a.close()                                                         # frees torch-cached pointers through torch although cudaFree is installed now
    gpu.use_torch_allocator()
    b.close()                                                         # and the other way round
    torch.cuda.synchronize()
    assert torch.zeros(4, device="cuda").sum().item() == 0.0          # the context is healthy
