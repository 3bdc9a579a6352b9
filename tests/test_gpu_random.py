"""-m gpu: randomised sizes and inputs for the two build kernels whose scans are single-pass look-backs (the one-sweep radix
pass and the one-pass octree level): many small and mid-size cases with ragged tails, heavy duplicates, skewed digits and
odd bucket sizes, each bit-exact against the oracle (stable sort with index tie-break, C2; canonical octree, C3).  A
look-back that reads a stale or half-published status word shows up as a wrong permutation or a wrong child index."""
import numpy as np
import pytest

import oracle

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B(cuda_device):
    from paper_2606_17145_b200 import binding
    return binding


def _keys(rng, n, kind):
    if kind == 0:                                   # all bits random
        return rng.integers(0, 1 << 63, size=n, dtype=np.uint64)
    if kind == 1:                                   # few distinct keys: long runs of duplicates
        return rng.choice(rng.integers(0, 1 << 63, size=max(1, n // 50 + 1), dtype=np.uint64), size=n)
    if kind == 2:                                   # skewed: most keys share their high digits
        return (rng.integers(0, 1 << 20, size=n, dtype=np.uint64) | (np.uint64(0x1234567) << np.uint64(36)))
    return np.sort(rng.integers(0, 1 << 63, size=n, dtype=np.uint64))[::-1].copy()      # descending


def test_one_sweep_sort_random_cases(B):
    import torch
    rng = np.random.default_rng(2026)
    sizes = [1, 2, 31, 32, 33, 2047, 2048, 2049, 4097, 65536 + 7] + [int(x) for x in rng.integers(1, 300000, size=30)]
    for t, n in enumerate(sizes):
        k = _keys(rng, n, t % 4)
        v = np.arange(n, dtype=np.uint32)
        b, e = (0, 64) if t % 3 == 0 else (int(rng.integers(0, 30)), int(rng.integers(31, 65)))
        ks, vs = B.og_radix_sort_pairs(torch.from_numpy(k.view(np.int64)).cuda(), torch.from_numpy(v.view(np.int32)).cuda(), b, e)
        mask = np.uint64(((1 << (e - b)) - 1) << b) if e - b < 64 else np.uint64(0xFFFFFFFFFFFFFFFF)
        order = np.argsort(k & mask, kind="stable")
        assert np.array_equal(vs.cpu().numpy().view(np.uint32), order.astype(np.uint32)), (n, t, b, e)
        assert np.array_equal(ks.cpu().numpy().view(np.uint64), k[order]), (n, t, b, e)


def test_octree_random_cases(B):
    import torch
    from paper_2606_17145_b200 import workloads as W
    rng = np.random.default_rng(77)
    for t in range(24):
        n = int(rng.integers(1, 60000))
        L = float(rng.choice([1.0, 7.5, 100.0]))
        kind = t % 3
        if kind == 0:
            x = rng.random((n, 3)) * L
        elif kind == 1:                             # tight clumps: deep single-child chains, big leaves at level 21
            c = rng.random((max(1, n // 500), 3)) * L
            x = c[rng.integers(0, c.shape[0], size=n)] + rng.standard_normal((n, 3)) * 1e-6 * L
        else:                                       # a sheet: many empty octants
            x = rng.random((n, 3)) * L
            x[:, 2] = 0.3 * L + rng.random(n) * 1e-3 * L
        pos = np.mod(x, L).astype(np.float32)
        pos[pos >= L] = 0.0
        mass = (rng.random(n) + 0.5).astype(np.float32)
        eps = np.full(n, 1e-3 * L, np.float32)
        leaf_max = int(rng.choice([1, 2, 8, 13, 32]))
        r_s = 0.01 * L
        prm = B.make_params(r_s, leaf_max=leaf_max)
        tree = B.og_tree_build(torch.from_numpy(pos).cuda(), torch.from_numpy(mass).cuda(), torch.from_numpy(eps).cuda(), L, prm)
        assert B.og_tree_status(tree) == B.OG_OK, (t, B.og_last_error())
        ot = oracle.build_tree(pos, mass, eps, oracle.make_params(L, r_s, leaf_max=leaf_max))
        assert B.og_tree_stats(tree)["n_nodes"] == ot.n_nodes, (t, n, leaf_max)
        for f, ref in ((B.OG_F_PERM, ot.perm), (B.OG_F_NODE_FIRST, ot.first), (B.OG_F_NODE_COUNT, ot.count),
                       (B.OG_F_NODE_FIRST_CHILD, ot.first_child)):
            assert np.array_equal(B.og_tree_get(tree, f).cpu().numpy().view(np.uint32), ref), (t, n, leaf_max, f)
        assert np.array_equal(B.og_tree_get(tree, B.OG_F_NODE_LEVEL).cpu().numpy(), ot.level)
        assert np.array_equal(B.og_tree_get(tree, B.OG_F_NODE_NCHILD).cpu().numpy(), ot.n_child)
        com = B.og_tree_get(tree, B.OG_F_NODE_COM).cpu().numpy()
        assert np.array_equal(com[:, 3].view(np.uint32), ot.M.view(np.uint32)) and np.array_equal(com[:, :3].view(np.uint32), ot.s.view(np.uint32))
        lo = B.og_tree_get(tree, B.OG_F_NODE_LO).cpu().numpy()
        assert np.array_equal(lo[:, :3].view(np.uint32), ot.lo.view(np.uint32)) and np.array_equal(lo[:, 3].view(np.uint32), ot.hmax.view(np.uint32))
        B.og_tree_free(tree)
