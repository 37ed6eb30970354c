"""Pins of the CPU oracle (oracle/snk_oracle.cpp) against things the paper and the mathematics fix.

None of these re-type the oracle's own formulae: Boys is checked against mpmath's incomplete gamma,
A against closed forms / brute-force 3-D quadrature / the Poisson equation, collocation against
closed-form overlaps, K against the analytic exchange matrix from closed-form (ss|ss) ERIs.
PAPER.md = /root/reference/PAPER.md (arXiv 2303.14280).  No value printed by the paper exists
for F_m, A or K, so there are no paper-number fixtures.
"""
import math

import mpmath as mp
import numpy as np
import pytest
from scipy.special import erf

from paper_2303_14280_b200 import inputs


def _boys_ref(m, x):
    """Eq. 22 in closed form: F_m(x) = gamma(m+1/2, x) / (2 x^(m+1/2))."""
    mp.mp.dps = 40
    if x == 0:
        return mp.mpf(1) / (2 * m + 1)
    x = mp.mpf(x)
    return mp.gammainc(m + mp.mpf(1) / 2, 0, x) / (2 * x ** (m + mp.mpf(1) / 2))


def test_boys_vs_mpmath(oracle_mod):
    xs = [0.0, 1e-12, 1e-8, 1e-4, 1e-2, 0.1, 0.37, 1.0, 2.5, 5.0, 9.99, 17.3, 25.0, 30.0, 34.0, 34.999, 35.0,
          35.001, 36.0, 40.0, 55.5, 100.0, 333.3, 1e3]
    worst = 0.0
    for x in xs:
        for mmax in (0, 3, 6):
            F = oracle_mod.boys(mmax, x)
            for m in range(mmax + 1):
                ref = float(_boys_ref(m, x))
                worst = max(worst, abs(F[m] / ref - 1.0))
    assert worst <= 4e-15, worst


def test_boys_special_cases(oracle_mod):
    # F_m(0) = 1/(2m+1);  F_0 = sqrt(pi/x)/2 erf(sqrt x);  large-x asymptote (2m-1)!!/2^(m+1) sqrt(pi/x^(2m+1))
    F = oracle_mod.boys(6, 0.0)
    assert np.allclose(F, [1.0 / (2 * m + 1) for m in range(7)], rtol=1e-15)
    for x in (0.3, 4.0, 20.0, 60.0):
        assert abs(oracle_mod.boys(0, x)[0] / (0.5 * math.sqrt(math.pi / x) * erf(math.sqrt(x))) - 1) < 4e-15
    x = 200.0
    F = oracle_mod.boys(4, x)
    df = 1.0
    for m in range(5):
        asym = df / 2 ** (m + 1) * math.sqrt(math.pi / x ** (2 * m + 1))
        assert abs(F[m] / asym - 1) < 1e-14
        df *= (2 * m + 1)
    # downward-recursion identity  (2m+1) F_m = 2x F_{m+1} + e^{-x}
    for x in (0.7, 12.0, 33.0, 48.0):
        F = oracle_mod.boys(6, x)
        for m in range(6):
            assert abs((2 * m + 1) * F[m] - (2 * x * F[m + 1] + math.exp(-x))) <= 4e-15 * (2 * m + 1) * F[m]


def _basis(atoms, shells):
    """shells: list of (atom, l, exps, coefs) -> inputs.Basis with the coefficients used verbatim."""
    return inputs.Basis(
        atom_xyz=np.array(atoms, dtype=np.float64),
        shell_atom=np.array([s[0] for s in shells], dtype=np.int32),
        shell_l=np.array([s[1] for s in shells], dtype=np.int32),
        shell_nprim=np.array([len(s[2]) for s in shells], dtype=np.int32),
        prim_exp=np.concatenate([np.asarray(s[2], dtype=np.float64) for s in shells]),
        prim_coef=np.concatenate([np.asarray(s[3], dtype=np.float64) for s in shells]))


def test_A_s_type_closed_form(oracle_mod):
    """Eq. 37 for two s primitives: c_a c_b (2 pi/p) exp(-mu |AB|^2) F_0(p |P - r_g|^2), F_0 via erf."""
    A, B = [0.1, -0.2, 0.3], [1.0, 0.7, -0.4]
    za, zb, ca, cb = 0.9, 2.3, 0.7, 1.3
    o = oracle_mod.Oracle(_basis([A, B], [(0, 0, [za], [ca]), (1, 0, [zb], [cb])]))
    rng = np.random.default_rng(1)
    pts = rng.uniform(-3, 3, (50, 3))
    got = o.A_pair(0, 1, pts)[:, 0, 0]
    p = za + zb
    Pc = (za * np.array(A) + zb * np.array(B)) / p
    x = p * ((pts - Pc) ** 2).sum(1)
    ref = ca * cb * 2 * math.pi / p * math.exp(-za * zb / p * ((np.array(A) - np.array(B)) ** 2).sum()) \
        * 0.5 * np.sqrt(math.pi / x) * erf(np.sqrt(x))
    assert np.max(np.abs(got / ref - 1)) < 1e-14


def _phi_direct(center, comp, exps, coefs, r):
    d = r - np.asarray(center)
    r2 = (d ** 2).sum(-1)
    rad = sum(c * np.exp(-e * r2) for e, c in zip(exps, coefs))
    return d[..., 0] ** comp[0] * d[..., 1] ** comp[1] * d[..., 2] ** comp[2] * rad


def _quad_A(sa, sb, atoms, rg, nr=140, nth=40, nph=80):
    """Brute-force Eq. 37 in spherical coordinates about r_g: the r^2 Jacobian cancels 1/r."""
    xr, wr = np.polynomial.legendre.leggauss(nr)
    rmax = 14.0
    r = 0.5 * rmax * (xr + 1)
    wr = 0.5 * rmax * wr
    ct, wt = np.polynomial.legendre.leggauss(nth)
    st = np.sqrt(1 - ct ** 2)
    ph = np.arange(nph) * 2 * math.pi / nph
    u = np.stack([st[:, None] * np.cos(ph)[None], st[:, None] * np.sin(ph)[None], np.broadcast_to(ct[:, None], (nth, nph))], -1)
    wang = np.broadcast_to(wt[:, None] * 2 * math.pi / nph, (nth, nph))
    pts = rg + r[:, None, None, None] * u[None]
    wgt = (wr * r)[:, None, None] * wang[None]          # r^2 dr dOmega / r
    ca, cb = inputs.cart_components(sa[1]), inputs.cart_components(sb[1])
    out = np.zeros((len(ca), len(cb)))
    for i, a in enumerate(ca):
        fa = _phi_direct(atoms[sa[0]], a, sa[2], sa[3], pts)
        for k, b in enumerate(cb):
            out[i, k] = (wgt * fa * _phi_direct(atoms[sb[0]], b, sb[2], sb[3], pts)).sum()
    return out


@pytest.mark.parametrize("la,lb", [(0, 0), (1, 0), (1, 1), (2, 1), (2, 2), (3, 1), (3, 3)])
def test_A_vs_bruteforce_quadrature(oracle_mod, la, lb):
    atoms = [[0.0, 0.1, -0.2], [0.8, -0.5, 0.6]]
    sa = (0, la, [1.1, 0.6], [0.8, 0.5])
    sb = (1, lb, [0.9], [1.2])
    o = oracle_mod.Oracle(_basis(atoms, [sa, sb]))
    for rg in ([0.3, 0.4, 0.1], [2.0, -1.0, 0.5]):
        got = o.A_pair(0, 1, np.array([rg]))[0]
        ref = _quad_A(sa, sb, atoms, np.array(rg))
        assert np.max(np.abs(got - ref)) < 2e-9 * max(1.0, np.abs(ref).max()), (la, lb, rg, np.abs(got - ref).max())
        # symmetry A_ab = A_ba^T
        assert np.max(np.abs(o.A_pair(1, 0, np.array([rg]))[0].T - got)) < 1e-14 * max(1.0, np.abs(got).max())


def test_A_far_field_and_poisson(oracle_mod):
    """(iii) A_ab(r_g) |r_g - P| -> S_ab for s-s;  (iv) laplacian_{r_g} A_ab = -4 pi phi_a phi_b ties A to collocation."""
    atoms = [[0.0, 0.0, 0.0], [0.9, 0.3, -0.2]]
    shells = [(0, 0, [1.3], [0.9]), (1, 0, [0.7], [1.1]), (0, 2, [0.8, 0.5], [0.6, 0.4]), (1, 1, [1.0], [0.7])]
    o = oracle_mod.Oracle(_basis(atoms, shells))
    za, zb = 1.3, 0.7
    p = za + zb
    AB2 = sum((a - b) ** 2 for a, b in zip(*atoms))
    S = 0.9 * 1.1 * (math.pi / p) ** 1.5 * math.exp(-za * zb / p * AB2)
    Pc = (za * np.array(atoms[0]) + zb * np.array(atoms[1])) / p
    rg = Pc + np.array([300.0, 0, 0])
    assert abs(o.A_pair(0, 1, rg[None])[0, 0, 0] * 300.0 / S - 1) < 1e-4       # monopole, O(1/R^2) corrections
    # Poisson, 4th-order central differences
    h = 2e-2
    r0 = np.array([0.4, 0.2, -0.3])
    Phi = o.collocation(r0[None])[0]
    off = [0, 1, 2, 8, 11]
    for (a, b) in [(0, 1), (2, 3), (2, 2), (3, 1)]:
        lap = 0.0
        A0 = o.A_pair(a, b, r0[None])[0]
        for q in range(3):
            e = np.zeros(3); e[q] = h
            pts = np.array([r0 - 2 * e, r0 - e, r0 + e, r0 + 2 * e])
            Aq = o.A_pair(a, b, pts)
            lap = lap + (-Aq[0] + 16 * Aq[1] - 30 * A0 + 16 * Aq[2] - Aq[3]) / (12 * h * h)
        la, lb = shells[a][1], shells[b][1]
        fa = Phi[off[a]:off[a] + inputs.ncart(la)]
        fb = Phi[off[b]:off[b] + inputs.ncart(lb)]
        ref = -4 * math.pi * np.outer(fa, fb)
        assert np.max(np.abs(lap - ref)) < 5e-6 * max(1.0, np.abs(ref).max()), (a, b, np.abs(lap - ref).max())


def test_A_derivative_relation(oracle_mod):
    """(v) d/dA_x (s_a s_b | r_g) = 2 zeta_a (p_x,a s_b | r_g): links l and l+1 on the same centre."""
    za, zb = 0.8, 1.4
    B = [0.5, -0.3, 0.2]
    rg = np.array([[0.7, 0.9, -0.4]])
    h = 1e-4
    vals = []
    for dx in (-2 * h, -h, h, 2 * h):
        o = oracle_mod.Oracle(_basis([[dx, 0, 0], B], [(0, 0, [za], [1.0]), (1, 0, [zb], [1.0])]))
        vals.append(o.A_pair(0, 1, rg)[0, 0, 0])
    deriv = (vals[0] - 8 * vals[1] + 8 * vals[2] - vals[3]) / (12 * h)
    o = oracle_mod.Oracle(_basis([[0, 0, 0], B], [(0, 1, [za], [1.0]), (1, 0, [zb], [1.0])]))
    px = o.A_pair(0, 1, rg)[0, 0, 0]
    assert abs(deriv - 2 * za * px) < 1e-9


def _overlap_ss(za, A, zb, B):
    p = za + zb
    return (math.pi / p) ** 1.5 * math.exp(-za * zb / p * ((np.asarray(A) - np.asarray(B)) ** 2).sum())


def test_collocation_overlap_and_normalisation(oracle_mod):
    """sum_g w_g Phi[g,mu] Phi[g,nu] -> S_mu,nu as the grid is refined; normalised (l,0,0) diag -> 1 (R5)."""
    w = inputs.make_workload(1, grid=(50, 20, 40))
    o = oracle_mod.Oracle(w.basis)
    Phi = o.collocation(w.points)
    S = (Phi * w.weights[:, None]).T @ Phi
    b = w.basis
    # diagonal: s functions and the (l,0,0)-type p components are unit-normalised by the harness
    assert np.max(np.abs(np.diag(S) - 1.0)) < 2e-6
    # off-diagonal s-s closed form between shells 0 (O, contracted s) and 5 (H, contracted s)
    po = b.prim_offset
    ref = 0.0
    for k in range(po[0], po[1]):
        for l in range(po[5], po[6]):
            ref += b.prim_coef[k] * b.prim_coef[l] * _overlap_ss(b.prim_exp[k], b.atom_xyz[0], b.prim_exp[l], b.atom_xyz[1])
    fo = b.shell_offset
    assert abs(S[fo[0], fo[5]] - ref) < 2e-6
    coarse = inputs.make_workload(1, grid=(20, 8, 16))
    Phic = o.collocation(coarse.points)
    Sc = (Phic * coarse.weights[:, None]).T @ Phic
    assert np.max(np.abs(np.diag(S) - 1.0)) < np.max(np.abs(np.diag(Sc) - 1.0))


def _eri_ssss_K(atoms, exps, cent, P):
    """Exact K_mu,nu = sum_{lam,kap} (mu lam | nu kap) P_lam,kap (Eq. 3) for unit-coefficient
    s primitives, (ab|cd) = 2 pi^(5/2)/(pq sqrt(p+q)) K_ab K_cd F_0(rho |P-Q|^2) (Eq. 21 with m = 0)."""
    n = len(exps)
    R = np.array([atoms[c] for c in cent])
    z = np.array(exps)
    p = z[:, None] + z[None, :]
    Kab = np.exp(-z[:, None] * z[None, :] / p * ((R[:, None] - R[None]) ** 2).sum(-1))
    Pc = (z[:, None, None] * R[:, None] + z[None, :, None] * R[None]) / p[..., None]
    K = np.zeros((n, n))
    for m in range(n):
        for nu in range(n):
            # (m lam | nu kap) for all lam, kap
            pp = p[m][:, None]; qq = p[nu][None, :]
            rho = pp * qq / (pp + qq)
            d2 = ((Pc[m][:, None] - Pc[nu][None, :]) ** 2).sum(-1)
            x = rho * d2
            F0 = np.where(x < 1e-14, 1.0 - x / 3.0, 0.5 * np.sqrt(math.pi / np.maximum(x, 1e-300)) * erf(np.sqrt(x)))
            eri = 2 * math.pi ** 2.5 / (pp * qq * np.sqrt(pp + qq)) * Kab[m][:, None] * Kab[nu][None, :] * F0
            K[m, nu] = (eri * P).sum()
    return K


def test_snK_converges_to_analytic_exchange(oracle_mod):
    """Fourth north_star check: all-s water-shaped system, error falls monotonically with grid level,
    K~ asymmetry tracks it (third check), K symmetric exactly after Eq. 40."""
    atoms_ang = np.array([[0.0, 0.0, 0.0], [0.757, 0.587, 0.0], [-0.757, 0.587, 0.0]])
    atoms = atoms_ang * inputs.BOHR_PER_ANGSTROM
    exps = [5.0, 1.2, 0.35, 1.5, 0.4, 1.5, 0.4]
    cent = [0, 0, 0, 1, 1, 2, 2]
    coef = [(2 * e / math.pi) ** 0.75 for e in exps]
    basis = _basis(atoms, [(c, 0, [e], [k]) for c, e, k in zip(cent, exps, coef)])
    rng = np.random.default_rng(7)
    Cm = rng.standard_normal((7, 3)) * 0.5
    P = Cm @ Cm.T
    Kex = _eri_ssss_K(atoms, exps, cent, P * np.outer(coef, coef)) * np.outer(coef, coef)
    o = oracle_mod.Oracle(basis)
    errs, asym = [], []
    for g in [(20, 8, 16), (40, 14, 28), (60, 20, 40)]:
        pts, w = inputs.becke_grid(atoms, *g)
        o.set_grid(pts, w, eps=0.0)
        K = o.build_K(P)
        assert np.array_equal(K, K.T)
        errs.append(np.abs(K - Kex).max())
        sel = np.arange(7, dtype=np.int32)
        Kt = o.build_K(P, sel_shells=sel)       # unsymmetrised K~
        asym.append(np.abs(Kt - Kt.T).max())
        assert np.abs(0.5 * (Kt + Kt.T) - K).max() < 1e-13
    assert errs[0] > errs[1] > errs[2], errs
    assert errs[0] < 1e-3 and errs[1] < 1e-5 and errs[2] < 1e-7, errs
    assert asym[0] > asym[1] > asym[2], asym


def test_K_linearity_translation_permutation(oracle_mod):
    w = inputs.make_workload(1, grid=(12, 6, 12))
    o = oracle_mod.Oracle(w.basis)
    o.set_grid(w.points, w.weights, eps=0.0, batch_max=300)
    rng = np.random.default_rng(3)
    n = w.basis.nbf
    P1 = w.P
    C2 = rng.standard_normal((n, 2)); P2 = C2 @ C2.T
    K1, K2 = o.build_K(P1), o.build_K(P2)
    K12 = o.build_K(0.7 * P1 - 1.9 * P2)
    scale = np.abs(K12).max()
    assert np.abs(K12 - (0.7 * K1 - 1.9 * K2)).max() < 1e-13 * scale
    # permutation of grid points (eps = 0)
    perm = rng.permutation(w.points.shape[0])
    o.set_grid(w.points[perm], w.weights[perm], eps=0.0, batch_max=300)
    assert np.abs(o.build_K(P1) - K1).max() < 1e-12 * np.abs(K1).max()
    # rigid translation of atoms + grid
    t = np.array([0.31, -1.7, 2.2])
    b2 = inputs.Basis(w.basis.atom_xyz + t, w.basis.shell_atom, w.basis.shell_l, w.basis.shell_nprim, w.basis.prim_exp, w.basis.prim_coef)
    o2 = oracle_mod.Oracle(b2)
    o2.set_grid(w.points + t, w.weights, eps=0.0, batch_max=300)
    assert np.abs(o2.build_K(P1) - K1).max() < 1e-11 * np.abs(K1).max()


def test_K_dense_numpy_definition(oracle_mod):
    """The batched/packed oracle K equals the unbatched dense definition (Eqs. 35, 38-40) assembled in numpy
    from the oracle's own A blocks and collocation: pins the batching / packing / two-direction bookkeeping."""
    w = inputs.make_workload(1, grid=(8, 4, 8))
    o = oracle_mod.Oracle(w.basis)
    o.set_grid(w.points, w.weights, eps=0.0, batch_max=64)
    K = o.build_K(w.P)
    n, ns = w.basis.nbf, w.basis.nshells
    fo = w.basis.shell_offset
    Phi = o.collocation(w.points)
    A = np.zeros((w.points.shape[0], n, n))
    for a in range(ns):
        for b in range(ns):
            A[:, fo[a]:fo[a + 1], fo[b]:fo[b + 1]] = o.A_pair(a, b, w.points)
    F = Phi @ w.P.T
    G = w.weights[:, None] * np.einsum("gnl,gl->gn", A, F)
    Kt = Phi.T @ G
    Kd = 0.5 * (Kt + Kt.T)
    assert np.abs(K - Kd).max() < 1e-12 * np.abs(Kd).max()


def test_batching_determinism_and_root_cell_subsets(oracle_mod):
    """R13: same batches from shuffled input; a subset made of whole root cells reproduces its batches."""
    w = inputs.make_workload(2, grid=(10, 6, 12), lattice=1)
    o = oracle_mod.Oracle(w.basis)
    o.set_grid(w.points, w.weights, eps=0.0, batch_max=200, batch_cell=4.0)
    off, perm, bbox = o.batches()
    assert off[-1] == w.points.shape[0] and len(set(perm.tolist())) == len(perm)
    assert np.all(np.diff(off) <= 200) and np.all(np.diff(off) > 0)
    sets = [frozenset(perm[off[j]:off[j + 1]].tolist()) for j in range(len(off) - 1)]
    for j in range(len(off) - 1):     # input order kept inside a batch
        assert np.all(np.diff(perm[off[j]:off[j + 1]]) > 0)
    rng = np.random.default_rng(0)
    sh = rng.permutation(w.points.shape[0])
    o.set_grid(w.points[sh], w.weights[sh], eps=0.0, batch_max=200, batch_cell=4.0)
    off2, perm2, _ = o.batches()
    sets2 = [frozenset(sh[perm2[off2[j]:off2[j + 1]]].tolist()) for j in range(len(off2) - 1)]
    assert sets == sets2                                   # same batches, same order
    # whole-root-cell subset
    cell = np.floor(w.points / 4.0).astype(np.int64)
    keys = [tuple(c) for c in cell]
    chosen = set(sorted(set(keys))[::3])
    mask = np.array([k in chosen for k in keys])
    idx = np.nonzero(mask)[0]
    o.set_grid(w.points[idx], w.weights[idx], eps=0.0, batch_max=200, batch_cell=4.0)
    off3, perm3, _ = o.batches()
    sets3 = [frozenset(idx[perm3[off3[j]:off3[j + 1]]].tolist()) for j in range(len(off3) - 1)]
    expect = [s for s in sets if next(iter(s)) in set(idx.tolist())]
    assert sets3 == expect


def test_screening_bounds_and_error(oracle_mod):
    """R10/R11 are true bounds; ||K_eps - K_0||_max <= c * eps (Eqs. 41-47 only delete small terms)."""
    w = inputs.make_workload(2, grid=(8, 6, 10), lattice=1)
    b = w.basis
    o = oracle_mod.Oracle(b)
    rng = np.random.default_rng(5)
    # R11: Atilde_ab >= |A| at random points
    pts = rng.uniform(-4, 8, (40, 3))
    for a in range(b.nshells):
        for bb in range(a, b.nshells):
            assert np.abs(o.A_pair(a, bb, pts)).max() <= o.A_bound(a, bb) * (1 + 1e-12)
    # R10: |phi| < eps outside rcut
    eps = 1e-8
    fo = b.shell_offset
    for a in range(b.nshells):
        rc = o.rcut(a, eps)
        assert rc == 0.25 * round(rc / 0.25)
        u = rng.standard_normal((30, 3)); u /= np.linalg.norm(u, axis=1)[:, None]
        p = b.atom_xyz[b.shell_atom[a]] + u * rc * rng.uniform(1.0, 1.5, (30, 1))
        assert np.abs(o.collocation(p)[:, fo[a]:fo[a + 1]]).max() < eps
    o.set_grid(w.points, w.weights, eps=0.0, batch_max=256)
    K0 = o.build_K(w.P)
    n0 = o.stats()["n_pairpoints"]
    for eps in (1e-6, 1e-9):
        o.set_grid(w.points, w.weights, eps=eps, batch_max=256)
        Ke = o.build_K(w.P)
        assert o.stats()["n_pairpoints"] <= n0
        assert np.abs(Ke - K0).max() <= 300 * eps, (eps, np.abs(Ke - K0).max())
    # a large threshold really deletes work
    o.set_grid(w.points, w.weights, eps=1e-3, batch_max=256)
    o.build_K(w.P)
    assert o.stats()["n_pairpoints"] < n0
