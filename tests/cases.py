"""Test-only inputs (not part of the product package): planes from arbitrary masks and the paper's own
verification case.  `neumann_offsets` reads the discrete normal off the mesh classification a solver
reports (reading D3 of DESIGN.md), so it lives here with the tests, not in the shared input generator."""
import numpy as np

from paper_2509_11831_b200.workloads import KIND_DIRICHLET, KIND_INNER, KIND_NEUMANN, Plane, _collect, guards_of


def mask_plane(inner: np.ndarray, neumann: np.ndarray, h: float, lam_f=None, c_f=None, f_f=None,
               levels: int = 2, i0: int = 0, j0: int = 0, order="rowmajor", seed=0) -> Plane:
    """Test helper: a plane from an arbitrary bool inner mask [j, i] (lattice origin offset i0, j0)."""
    n_j, n_i = inner.shape
    assert n_j == n_i, "square lattice arrays only"
    n = n_j
    X, Y = np.meshgrid(np.arange(n) * h + i0 * h, np.arange(n) * h + j0 * h, indexing="xy")
    one = np.ones((n, n))
    pl = _collect(0, n, h, X, Y, inner, neumann, one if lam_f is None else lam_f,
                  one if c_f is None else c_f, np.zeros((n, n)) if f_f is None else f_f,
                  levels, order, seed, {})
    pl.i = (pl.i + i0).astype(np.int32)
    pl.j = (pl.j + j0).astype(np.int32)
    return pl


# --------------------------------------------------------------------------- the paper's own verification case
def make_paper_annulus(h: float, levels: int, neumann_inner: bool = False, R0: float = 1.0, absorb_xi: bool = True) -> Plane:
    """PAPER.md:233-252 (Eq. 19-22): circular flux surfaces, domain 0.2 < r < 0.4 with
    r = sqrt((R-R0)^2 + Z^2)/R0, coefficients Eq. 21, manufactured solution Eq. 22.  The three-field
    form lambda*phi - xi*div(c grad phi) = rho (Eq. 6) is handed over with xi absorbed (PAPER.md:47:
    "it can be absorbed as well into lambda and rho"): lam = lambda/xi, f = rho/xi; with `absorb_xi=False` the three
    fields are handed over as printed (lam = lambda, f = rho on inner rows, xi of Eq. 21 in meta["xi"]).  rho is derived
    symbolically from Eq. 6.  R0 is not printed; R0 = 1 reproduces the paper's point counts to within the
    guard layer (G10, G12).  Guard values: phi_MMS on Dirichlet guards; for Neumann guards
    (inner circle, if `neumann_inner`) f is left 0 and `meta` carries grad phi_MMS at every point so that
    the caller can form Gamma along the DISCRETE normal the mesh rules define (`neumann_gamma`)."""
    import sympy as sp
    Rs, Zs = sp.symbols("R Z", real=True)
    xs = Rs - R0
    r = sp.sqrt(xs ** 2 + Zs ** 2) / R0
    th = sp.atan2(Zs, xs)
    rhat = (r - sp.Rational(1, 5)) / (sp.Rational(2, 5) - sp.Rational(1, 5))
    lam_s = r * sp.sin(th)
    xi_s = Rs * sp.sqrt(r) * (2 + sp.cos(th))
    c_s = (sp.Rational(11, 10) + sp.cos(sp.pi / 2 * rhat) * sp.cos(3 * th)) / Rs
    phi_s = sp.Rational(13, 10) + sp.cos(sp.Rational(3, 2) * sp.pi * rhat) * sp.sin(4 * th)
    rho_s = lam_s * phi_s - xi_s * (sp.diff(c_s * sp.diff(phi_s, Rs), Rs) + sp.diff(c_s * sp.diff(phi_s, Zs), Zs))
    fn = {k: sp.lambdify((Rs, Zs), e, "numpy") for k, e in
          dict(lam=lam_s, xi=xi_s, c=c_s, phi=phi_s, rho=rho_s, pR=sp.diff(phi_s, Rs), pZ=sp.diff(phi_s, Zs)).items()}
    L = int(np.ceil(0.4 * R0 / h)) + 3
    idx = np.arange(-L, L + 1)
    n = idx.shape[0]
    X, Zc = np.meshgrid(idx * h, idx * h, indexing="xy")       # arrays indexed [j, i]; x = R - R0
    rr = np.sqrt(X * X + Zc * Zc) / R0
    inner = (rr > 0.2) & (rr < 0.4)
    guard = guards_of(inner)
    jj, ii = np.nonzero(inner | guard)
    Rp, Zp = R0 + X[jj, ii], Zc[jj, ii]
    is_inner = inner[jj, ii]
    neu = (~is_inner) & (rr[jj, ii] <= 0.2) & neumann_inner
    kind = np.where(is_inner, KIND_INNER, np.where(neu, KIND_NEUMANN, KIND_DIRICHLET)).astype(np.uint8)
    xi = fn["xi"](Rp, Zp)
    phi = fn["phi"](Rp, Zp)
    div = xi if absorb_xi else 1.0
    f = np.where(is_inner, fn["rho"](Rp, Zp) / div, np.where(neu, 0.0, phi))
    meta = {"phi": phi, "phi_R": fn["pR"](Rp, Zp), "phi_Z": fn["pZ"](Rp, Zp), "xi": np.ascontiguousarray(xi)}
    return Plane(cfg=0, lattice=n, h=h, i=(ii - L).astype(np.int32), j=(jj - L).astype(np.int32), kind=kind,
                 lam=np.ascontiguousarray(fn["lam"](Rp, Zp) / div), c=np.ascontiguousarray(fn["c"](Rp, Zp)),
                 f=np.ascontiguousarray(f), x0=np.zeros(jj.shape[0]), levels=levels, x=Rp, y=Zp, meta=meta)


def neumann_gamma(plane: Plane, offset_R: np.ndarray, offset_Z: np.ndarray) -> np.ndarray:
    """Right-hand side with the Neumann rows filled for the manufactured solution: Gamma_l = (o_l . grad phi)(x_l),
    o_l = n/|n| for a guard with discrete normal n (Eq. 13-16: upstream value at distance h|n| along n), or the mean
    offset of the inner 4-neighbours in units of h for the degenerate fallback (distance h).  The offsets come from
    the mesh classification of the side under test; this function holds no discretisation arithmetic."""
    f = plane.f.copy()
    m = plane.kind == KIND_NEUMANN
    g = offset_R * plane.meta["phi_R"] + offset_Z * plane.meta["phi_Z"]
    f[m] = g[m]
    return f


def neumann_offsets(kind, ns_tn, ns_fallback, nbr):
    """Per point of a level (canonical order), the offset in units of h from a Neumann guard to the place where the
    discretisation evaluates the upstream value, read off the mesh classification a solver (oracle or library)
    reports: n/|n| with n = ns_tn / 2 the discrete normal (Eq. 13), or, for guards flagged `ns_fallback`, the mean
    offset of their inner 4-neighbours (`nbr`: W, E, S, N indices, -1 absent).  Zero elsewhere."""
    n = kind.shape[0]
    oR, oZ = np.zeros(n), np.zeros(n)
    tn = ns_tn.astype(float) / 2.0
    nrm = np.hypot(tn[:, 0], tn[:, 1])
    reg = (kind == KIND_NEUMANN) & (ns_fallback == 0)
    oR[reg], oZ[reg] = tn[reg, 0] / nrm[reg], tn[reg, 1] / nrm[reg]
    D = [(-1, 0), (1, 0), (0, -1), (0, 1)]
    for l in np.nonzero((kind == KIND_NEUMANN) & (ns_fallback == 1))[0]:
        nb = [d for d, q in zip(D, nbr[l]) if q >= 0 and kind[q] == KIND_INNER]
        oR[l], oZ[l] = np.mean([d[0] for d in nb]), np.mean([d[1] for d in nb])
    return oR, oZ
