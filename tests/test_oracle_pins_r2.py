"""More pins of the CPU oracle: the screening quantities R10 / R11 recomputed from their definitions with mpmath
(neither side's C++), and the oracle's column-subset path.

SURVEY.md section 8(c): R10 = envelope r^l sum_k |c_k| exp(-z_k r^2), r_cut = SMALLEST value of the ladder 0.25 n bohr
(n >= 1) with r >= sqrt(l / (2 z_min)) and envelope < eps;  R11 = A~_ab = sum_kl c'_k c'_l (2 pi / p') exp(-(z'_k z'_l / p') |AB|^2),
s shells (c', z') = (|c|, z), l > 0 shells z' = z / 2, c' = |c| (l / (e z))^(l/2).  PAPER.md:245 (cut-off sphere), 269 (bound).
"""
import numpy as np
import mpmath as mp
import pytest

from paper_2303_14280_b200 import inputs


def _shell(b, a):
    po = b.prim_offset
    return (int(b.shell_l[a]), [float(x) for x in b.prim_exp[po[a]:po[a + 1]]], [float(x) for x in b.prim_coef[po[a]:po[a + 1]]],
            np.asarray(b.atom_xyz[b.shell_atom[a]], dtype=float))


def _envelope(l, exps, coefs, r):
    r = mp.mpf(r)
    return r ** l * mp.fsum(abs(mp.mpf(c)) * mp.e ** (-mp.mpf(z) * r * r) for z, c in zip(exps, coefs))


def _rcut_from_definition(l, exps, coefs, eps):
    rmin = mp.sqrt(mp.mpf(l) / (2 * min(exps)))
    n = 1
    while True:
        r = mp.mpf(n) / 4
        if r >= rmin and _envelope(l, exps, coefs, r) < eps:
            return n
        n += 1


@pytest.mark.parametrize("cfg,lattice", [(2, 1), (5, None)])
def test_rcut_is_the_smallest_ladder_value(oracle_mod, cfg, lattice):
    """R10: orc_rcut is ON the ladder, satisfies both conditions, and the ladder value below it violates one."""
    mp.mp.dps = 40
    kw = dict(grid=(6, 4, 6))
    if lattice:
        kw["lattice"] = lattice
    else:
        kw["natoms"] = 2
    w = inputs.make_workload(cfg, **kw)
    b = w.basis
    o = oracle_mod.Oracle(b)
    seen = set()
    for a in range(b.nshells):
        l, ex, co, _ = _shell(b, a)
        key = (l, tuple(ex), tuple(co))
        if key in seen:
            continue
        seen.add(key)
        for eps in (1e-6, 1e-10, 1e-12):
            n = _rcut_from_definition(l, ex, co, eps)
            # the decision must not sit within rounding of eps, else libm vs mpmath could legitimately differ
            e_at, e_below = _envelope(l, ex, co, mp.mpf(n) / 4), _envelope(l, ex, co, mp.mpf(n - 1) / 4)
            assert abs(e_at / eps - 1) > 1e-9 and abs(e_below / eps - 1) > 1e-9
            assert o.rcut(a, eps) == 0.25 * n, (a, l, eps, o.rcut(a, eps), 0.25 * n)
    assert np.isinf(o.rcut(0, 0.0))


def _sgauss(l, z, c):
    z, c = mp.mpf(z), abs(mp.mpf(c))
    if l == 0:
        return c, z
    return c * (mp.mpf(l) / (mp.e * z)) ** (mp.mpf(l) / 2), z / 2


def test_A_bound_from_definition_and_tightness(oracle_mod):
    """R11 from its formula (mpmath, 40 digits) for every shell pair of a small s..f basis; and the bound is attained
    (not merely an upper bound) by an s-s pair of single positive primitives at the product centre, where F_0(0) = 1."""
    mp.mp.dps = 40
    w = inputs.make_workload(5, grid=(6, 4, 6), natoms=3)
    b = w.basis
    o = oracle_mod.Oracle(b)
    for a in range(b.nshells):
        la, ea, ca, A = _shell(b, a)
        for bb in range(b.nshells):
            lb, eb, cb, B = _shell(b, bb)
            AB2 = mp.fsum((mp.mpf(x) - mp.mpf(y)) ** 2 for x, y in zip(A, B))
            ref = mp.mpf(0)
            for z1, c1 in zip(ea, ca):
                for z2, c2 in zip(eb, cb):
                    k1, q1 = _sgauss(la, z1, c1)
                    k2, q2 = _sgauss(lb, z2, c2)
                    p = q1 + q2
                    ref += k1 * k2 * (2 * mp.pi / p) * mp.e ** (-(q1 * q2 / p) * AB2)
            got = o.A_bound(a, bb)
            # exp(-x) carries the rounding of its argument: relative accuracy u * x, x = -ln(term) up to several hundred here
            assert abs(got - float(ref)) <= (1e-13 + 1e-15 * abs(float(mp.log(ref)))) * float(ref), (a, bb, got, float(ref))
            assert abs(got - o.A_bound(bb, a)) <= 4e-16 * got      # same terms, other summation order
    # tightness
    atoms = np.array([[0.0, 0.0, 0.0], [0.9, -0.4, 0.7]])
    za, zb, ka, kb = 1.3, 0.45, 0.8, 1.1
    basis = inputs.Basis(atom_xyz=atoms, shell_atom=np.array([0, 1], dtype=np.int32), shell_l=np.array([0, 0], dtype=np.int32),
                         shell_nprim=np.array([1, 1], dtype=np.int32), prim_exp=np.array([za, zb]), prim_coef=np.array([ka, kb]))
    o2 = oracle_mod.Oracle(basis)
    P = (za * atoms[0] + zb * atoms[1]) / (za + zb)
    val = o2.A_pair(0, 1, P[None, :])[0, 0, 0]
    assert abs(val - o2.A_bound(0, 1)) <= 1e-14 * val
    # and it is a strict over-estimate anywhere else
    assert o2.A_pair(0, 1, (P + 0.3)[None, :])[0, 0, 0] < o2.A_bound(0, 1)


def test_column_subset_path(oracle_mod):
    """orc_build_K(sel_shells = S), S a STRICT subset: the columns of the unsymmetrised K~ that belong to S equal those
    of the all-shell K~, every other column is exactly zero, and the symmetrised K is recovered from the all-shell K~."""
    w = inputs.make_workload(2, grid=(8, 6, 10), lattice=1)
    b = w.basis
    o = oracle_mod.Oracle(b)
    o.set_grid(w.points, w.weights, eps=w.eps, batch_max=256)
    K = o.build_K(w.P)
    Kt_all = o.build_K(w.P, sel_shells=np.arange(b.nshells, dtype=np.int32))
    assert np.abs(0.5 * (Kt_all + Kt_all.T) - K).max() <= 1e-13 * max(1.0, np.abs(K).max())
    fo = b.shell_offset
    S = np.array([1, 4, b.nshells - 1], dtype=np.int32)
    Kt_S = o.build_K(w.P, sel_shells=S)
    cols = np.zeros(b.nbf, dtype=bool)
    for s in S:
        cols[fo[s]:fo[s + 1]] = True
    assert np.array_equal(Kt_S[:, ~cols], np.zeros_like(Kt_S[:, ~cols]))
    assert np.abs(Kt_S[:, cols] - Kt_all[:, cols]).max() <= 1e-13 * max(1.0, np.abs(Kt_all).max())
    assert np.abs(Kt_S[:, cols]).max() > 0
