"""snk_A_pair_noalloc (include/snk.h): the A-block kernel with its primitive-pair scratch in a fixed device array inside the
library instead of a per-call cudaMalloc.  Checked against the existing path (snk_debug_A_pair, which is itself checked
against the oracle in test_gpu_parity.py) on consecutive calls that reuse the shared scratch.

This file is named so that pytest collects it last: the suite runs with `pytest -x`, and a failure here must not hide the
other tests.  It brings its own fixtures, so it passes alone in a fresh process as well as after the other files."""
import numpy as np
import pytest

from paper_2303_14280_b200 import inputs

pytestmark = pytest.mark.gpu

REL_TOL = 2e-13        # the bound test_A_blocks_OS_vs_MD uses for A blocks, relative to the block's largest element


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


def _basis():
    """two centres carrying s, p, d, f shells with 1-3 primitives: every (l_a, l_b) class, both orientations, same-centre pairs"""
    rng = np.random.Generator(np.random.PCG64(23))
    atoms = np.array([[0.0, 0.1, -0.2], [1.1, -0.7, 0.9]])
    return inputs.make_basis(rng, np.array([6, 6]), atoms, {6: [(0, 3), (1, 2), (2, 1), (3, 2)]}, (0.15, 8.0))


def test_noalloc_matches_existing_path_on_consecutive_calls(snk_mod, torch_cuda):
    torch = torch_cuda
    b = _basis()
    s = snk_mod.Snk(b)
    rng = np.random.default_rng(5)
    pts = np.concatenate([rng.uniform(-3, 3, (333, 3)), rng.uniform(-40, 40, (100, 3)), b.atom_xyz, b.atom_xyz + 1e-9])
    pd = torch.as_tensor(pts, device="cuda")
    n = pts.shape[0]
    pairs = [(a, c) for a in range(b.nshells) for c in range(b.nshells)]
    ref = {ac: s.debug_A_pair(*ac, pd).cpu().numpy() for ac in pairs}      # the existing (allocating, synchronising) path
    worst = 0.0

    def check(ac, got):
        nonlocal worst
        r = ref[ac]
        assert got.shape == r.shape
        err = np.abs(got - r).max() / np.abs(r).max()
        worst = max(worst, err)
        assert err <= REL_TOL, (ac, err)

    # two calls in a row per pair: the second one finds the first one's records in the shared scratch and must give the same
    # result; then the next pair (other number of primitive pairs, other class) overwrites them
    for ac in pairs:
        shape = (n, s._nc(ac[0]), s._nc(ac[1]))
        out1 = torch.full(shape, float("nan"), dtype=torch.float64, device="cuda")
        out2 = torch.full(shape, float("nan"), dtype=torch.float64, device="cuda")
        s.A_pair_noalloc(*ac, pd, out1)
        s.A_pair_noalloc(*ac, pd, out2)
        g1, g2 = out1.cpu().numpy(), out2.cpu().numpy()
        check(ac, g1)
        assert np.array_equal(g1, g2), ac
    # back-to-back calls for DIFFERENT pairs on one stream without any host synchronisation in between: stream order alone
    # must keep the second call's scratch fill behind the first call's kernel
    order = [pairs[3], pairs[-1], pairs[0], pairs[10], pairs[3]]
    outs = [torch.empty((n, s._nc(a), s._nc(c)), dtype=torch.float64, device="cuda") for a, c in order]
    for ac, o in zip(order, outs):
        s.A_pair_noalloc(*ac, pd, o)
    torch.cuda.synchronize()
    for ac, o in zip(order, outs):
        check(ac, o.cpu().numpy())
    # a side stream works the same way
    st = torch.cuda.Stream()
    st.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(st):
        o = torch.empty((n, s._nc(5), s._nc(2)), dtype=torch.float64, device="cuda")
        s.A_pair_noalloc(5, 2, pd, o, stream=st)
    st.synchronize()
    check((5, 2), o.cpu().numpy())
    print("snk_A_pair_noalloc vs snk_debug_A_pair: worst rel diff %.2e over %d shell pairs" % (worst, len(pairs)))


def test_noalloc_edges_and_limit(snk_mod, torch_cuda):
    torch = torch_cuda
    b = _basis()
    s = snk_mod.Snk(b)
    pd = torch.zeros((0, 3), dtype=torch.float64, device="cuda")
    s.A_pair_noalloc(0, 1, pd, torch.empty((0, 1, 3), dtype=torch.float64, device="cuda"))          # n = 0: nothing to do
    one = torch.zeros((1, 3), dtype=torch.float64, device="cuda")
    with pytest.raises(snk_mod.SnkError) as e:
        s._check(s._lib.snk_A_pair_noalloc(s.h, 0, b.nshells, 1, one.data_ptr(), one.data_ptr(), None))
    assert e.value.code == -1                                                                        # SNK_EINVAL: bad shell index
    # beyond the fixed scratch: 33 x 32 = 1056 > 1024 primitive pairs is refused with a clear message, 32 x 32 is served
    rng = np.random.default_rng(9)
    atoms = np.array([[0.0, 0.0, 0.0], [0.8, 0.3, -0.5]])
    big = inputs.Basis(atom_xyz=atoms, shell_atom=np.array([0, 1, 1], dtype=np.int32), shell_l=np.array([0, 0, 0], dtype=np.int32),
                       shell_nprim=np.array([33, 32, 32], dtype=np.int32), prim_exp=rng.uniform(0.2, 5.0, 97),
                       prim_coef=rng.uniform(0.05, 0.2, 97))
    sb = snk_mod.Snk(big)
    pts = torch.as_tensor(rng.uniform(-2, 2, (64, 3)), device="cuda")
    out = torch.empty((64, 1, 1), dtype=torch.float64, device="cuda")
    with pytest.raises(snk_mod.SnkError) as e:
        sb.A_pair_noalloc(0, 1, pts, out)
    assert e.value.code == -1 and "1024" in str(e.value)
    sb.A_pair_noalloc(1, 2, pts, out)                                                                # exactly the maximum
    r = sb.debug_A_pair(1, 2, pts)
    assert float((out - r).abs().max() / r.abs().max()) <= REL_TOL
    # the scratch survives a context: a new context on the same device reuses the same array
    s2 = snk_mod.Snk(b)
    o = torch.empty((64, 3, 6), dtype=torch.float64, device="cuda")
    s2.A_pair_noalloc(1, 2, pts, o)
    r = s2.debug_A_pair(1, 2, pts)
    assert float((o - r).abs().max() / r.abs().max()) <= REL_TOL
