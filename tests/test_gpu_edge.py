"""-m gpu: edge and degenerate cases of the path through the C ABI, each against the oracle
(or its closed form): tiny and ragged sizes, coincident particles, deep single-child chains and the
node-capacity latch, groups that straddle the periodic wall (per-lane nearest-image path), targets with
a_old = 0, arbitrary / duplicated / empty / invalid active lists, caller-supplied workspace, the
HOST-buffer entry point, position validation."""
import numpy as np
import pytest

import oracle
from paper_2606_17145_b200 import workloads as W
from gpu_common import check_acc, rel_err_scalar

pytestmark = pytest.mark.gpu

L, RS = 1.0, 1.25 / 64
EPS = 0.02 / 32


@pytest.fixture(scope="module")
def B(cuda_device):
    from paper_2606_17145_b200 import binding
    return binding


def _wl(pos, mass=None, eps=None, L=L, r_s=RS, alpha=0.005):
    pos = np.ascontiguousarray(pos, np.float32)
    n = pos.shape[0]
    mass = np.full(n, 1.0 / max(n, 1), np.float32) if mass is None else np.asarray(mass, np.float32)
    eps = np.full(n, EPS, np.float32) if eps is None else np.asarray(eps, np.float32)
    return W.Workload("edge", pos, mass, eps, L, r_s, alpha=alpha)


def _both(B, w, active=None, a_old=None, leaf_max=8, flags=0, max_nodes=0):
    """GPU and oracle results for the same inputs -> (acc_gpu, pot_gpu, acc_orc, pot_orc)."""
    import torch
    prm = B.make_params(w.r_s, G=w.G, rcut_over_rs=w.rcut_over_rs, alpha=w.alpha, theta=w.theta, leaf_max=leaf_max,
                        max_nodes=max_nodes, flags=B.OG_PERIODIC | flags)
    pos, mass, eps = (torch.from_numpy(x).cuda() for x in (w.pos, w.mass, w.eps))
    tree = B.og_tree_build(pos, mass, eps, w.L, prm)
    act = None if active is None else torch.from_numpy(np.asarray(active, np.uint32).view(np.int32)).cuda()
    ao = None if a_old is None else torch.from_numpy(np.asarray(a_old, np.float32)).cuda()
    a, p = B.og_shortrange_accel(tree, act, ao)
    assert B.og_tree_status(tree) == B.OG_OK, B.og_last_error()
    oprm = oracle.make_params(w.L, w.r_s, G=w.G, rcut_over_rs=w.rcut_over_rs, alpha=w.alpha, theta=w.theta,
                              leaf_max=leaf_max)
    ot = oracle.build_tree(w.pos, w.mass, w.eps, oprm)
    assert B.og_tree_stats(tree)["n_nodes"] == ot.n_nodes
    ao_, po_, _ = oracle.walk(ot, None if active is None else np.asarray(active, np.uint32),
                              None if a_old is None else np.asarray(a_old, np.float32), want_counters=False)
    B.og_tree_free(tree)
    return a.cpu().numpy(), p.cpu().numpy(), ao_, po_


def test_single_particle(B):
    a, p, ao, po = _both(B, _wl([[0.3, 0.4, 0.5]]))
    assert np.all(a == 0) and np.all(p == 0) and np.all(ao == 0)


def test_two_coincident_particles(B):
    """C5: distinct coincident particles: force 0, potential -(14/5) G m / h."""
    w = _wl([[0.5, 0.5, 0.5], [0.5, 0.5, 0.5]])
    a, p, ao, po = _both(B, w)
    h = np.float32(2.8) * np.float32(EPS)
    assert np.all(a == 0) and np.all(ao == 0)
    assert np.allclose(p, -2.8 * 0.5 / h, rtol=1e-6) and np.allclose(po, -2.8 * 0.5 / float(h), rtol=1e-6)


@pytest.mark.parametrize("n", [2, 9, 31, 32, 33, 65, 1000])
def test_ragged_sizes(B, n):
    rng = np.random.default_rng(n)
    c = rng.random(3) * 0.8 + 0.1
    pos = np.mod(c + 0.02 * rng.standard_normal((n, 3)), 1.0)
    a, p, ao, po = _both(B, _wl(pos))
    check_acc(a, ao, what=f"n={n}")
    ep = rel_err_scalar(p, po)
    assert ep.size == 0 or ep.max() <= 1e-4


def test_group_straddles_periodic_wall(B):
    """A tight cluster cut by the faces x = 0 / L in all three axes: Morton-consecutive targets sit on both
    sides of the wall, so sources cannot be pre-shifted for the whole group (per-lane nearest-image path)."""
    rng = np.random.default_rng(5)
    pos = np.mod(0.015 * rng.standard_normal((4000, 3)), 1.0)
    w = _wl(pos)
    a1, p1, ao1, po1 = _both(B, w)
    check_acc(a1, ao1, what="wall geometric")
    a_old = np.linalg.norm(ao1, axis=1).astype(np.float32)
    a2, p2, ao2, po2 = _both(B, w, a_old=a_old)
    check_acc(a2, ao2, what="wall relative")
    ep = rel_err_scalar(p2, po2)
    assert np.percentile(ep, 99) <= 1e-4 and ep.max() <= 1e-2


def test_deep_chain_and_node_overflow_latch(B):
    """Near-coincident particles create single-child chains down to level 21 (R6); a too small node
    capacity latches OG_ERR_NODE_OVERFLOW instead of writing out of bounds."""
    import torch
    rng = np.random.default_rng(11)
    base = np.array([0.123456, 0.654321, 0.333333])
    pos = np.concatenate([base + 3e-7 * rng.random((64, 3)), rng.random((200, 3))])
    w = _wl(pos)
    a, p, ao, po = _both(B, w, leaf_max=1, max_nodes=4096)
    check_acc(a, ao, what="deep chain")
    prm = B.make_params(w.r_s, leaf_max=1, max_nodes=64)
    t = B.og_tree_build(*(torch.from_numpy(x).cuda() for x in (w.pos, w.mass, w.eps)), w.L, prm)
    assert B.og_tree_status(t) == B.OG_ERR_NODE_OVERFLOW
    assert "status" in B.og_last_error()
    B.og_tree_free(t)


def test_a_old_zero_opens_everything(B):
    """A = 0 => G M l^2 > 0 always opens (R14): those targets get the direct sum within r_cut."""
    w = W.make("uniform32", small=True)
    a_old = np.zeros(w.n, np.float32)
    a_old[::2] = 1.0
    a, p, ao, po = _both(B, w, a_old=a_old)
    check_acc(a, ao, what="a_old mixed zero")
    ad, _ = oracle.direct(w.pos, w.mass, w.eps, oracle.make_params(w.L, w.r_s))
    check_acc(a[1::2], ad[1::2], p99=2e-5, mx=1e-3, what="a_old=0 vs direct")


def test_active_lists(B):
    """Arbitrary order, duplicates, a single target, and the empty list."""
    import torch
    w = W.make("nfw256", small=True)
    rng = np.random.default_rng(3)
    act = rng.permutation(w.n)[:777].astype(np.uint32)
    act[10] = act[500]                      # duplicate
    a, p, ao, po = _both(B, w, active=act)
    check_acc(a, ao, what="active subset")
    assert np.array_equal(a[10], a[500])
    a1, p1, ao1, po1 = _both(B, w, active=act[:1])
    check_acc(a1, ao1, what="one target")
    prm = B.make_params(w.r_s)
    t = B.og_tree_build(*(torch.from_numpy(x).cuda() for x in (w.pos, w.mass, w.eps)), w.L, prm)
    empty = torch.empty(0, dtype=torch.int32, device="cuda")
    out = torch.empty((0, 3), dtype=torch.float32, device="cuda")
    B.og_shortrange_accel(t, empty, None, acc_out=out, want_pot=False)
    assert B.og_tree_status(t) == B.OG_OK
    bad = torch.tensor([0, w.n + 5], dtype=torch.int32, device="cuda")     # out of range -> latched
    B.og_shortrange_accel(t, bad, None)
    assert B.og_tree_status(t) == B.OG_ERR_INVALID_ARG
    B.og_tree_free(t)


def test_workspace_validate_and_host_entry(B):
    import torch
    w = W.make("lattice128", small=True)
    prm = B.make_params(w.r_s, alpha=w.alpha, flags=B.OG_PERIODIC | B.OG_VALIDATE_POS)
    pos, mass, eps = (torch.from_numpy(x).cuda() for x in (w.pos, w.mass, w.eps))
    ws = torch.empty(B.og_tree_workspace_bytes(w.n, prm) + 256, dtype=torch.uint8, device="cuda")
    off = (-ws.data_ptr()) % 256
    t = B.og_tree_build(pos, mass, eps, w.L, prm, workspace=ws[off:])
    a_ws, p_ws = B.og_shortrange_accel(t, None, None)
    assert B.og_tree_status(t) == B.OG_OK
    t2 = B.og_tree_build(pos, mass, eps, w.L, prm)
    a_pool, p_pool = B.og_shortrange_accel(t2, None, None)
    assert torch.equal(a_ws, a_pool) and torch.equal(p_ws, p_pool)
    with pytest.raises(B.OgError):
        B.og_tree_build(pos, mass, eps, w.L, prm, workspace=ws[off:off + 4096])
    # HOST-buffer entry point = the two device calls
    a_h, p_h = B.og_shortrange_accel_host(torch.from_numpy(w.pos), torch.from_numpy(w.mass), torch.from_numpy(w.eps),
                                          w.L, prm)
    assert torch.equal(a_h, a_pool.cpu()) and torch.equal(p_h, p_pool.cpu())
    # pot_out = NULL gives the same accelerations
    a_np, none = B.og_shortrange_accel(t2, None, None, want_pot=False)
    assert none is None and torch.equal(a_np, a_pool)
    B.og_tree_free(t)
    B.og_tree_free(t2)
    # position outside [0, box) is latched when OG_VALIDATE_POS is set
    badpos = pos.clone()
    badpos[7, 1] = w.L
    t3 = B.og_tree_build(badpos, mass, eps, w.L, prm)
    assert B.og_tree_status(t3) == B.OG_ERR_BAD_POSITION
    B.og_tree_free(t3)


@pytest.mark.parametrize("G,rcut_over_rs,theta,alpha", [(2.5, 4.5, 0.5, 0.005), (1.0, 4.0, 0.7, 0.02), (0.3, 5.0, 0.3, 0.001)])
def test_parameter_plumbing(B, G, rcut_over_rs, theta, alpha):
    """G, rcut_over_rs (up to the polynomial's limit 5), theta and alpha other than the configs' values."""
    w0 = W.make("nfw256", small=True)
    w = W.Workload("params", w0.pos, w0.mass, w0.eps, w0.L, w0.r_s, alpha=alpha, theta=theta,
                   rcut_over_rs=rcut_over_rs, G=G)
    a1, p1, ao1, po1 = _both(B, w)
    check_acc(a1, ao1, what="params geometric")
    a_old = np.linalg.norm(ao1, axis=1).astype(np.float32)
    a2, p2, ao2, po2 = _both(B, w, a_old=a_old)
    check_acc(a2, ao2, what="params relative")
    ep = rel_err_scalar(p2, po2)
    assert np.percentile(ep, 99) <= 1e-4 and ep.max() <= 1e-2


def test_rcut_over_rs_above_polynomial_range_is_rejected(B):
    import torch
    w = W.make("uniform32", small=True)
    prm = B.make_params(w.r_s, rcut_over_rs=5.5)
    with pytest.raises(B.OgError):
        B.og_tree_build(*(torch.from_numpy(x).cuda() for x in (w.pos, w.mass, w.eps)), w.L, prm)
    assert "rcut_over_rs" in B.og_last_error()


def test_mixed_softening_species(B):
    """Two species with very different softening (h of the heavy one comparable to r_cut), all active and a
    sparse subset: spline branches, R16 guard with mixed h_max, both walk instantiations."""
    rng = np.random.default_rng(21)
    n_hi, n_lo = 30000, 6000
    pos = np.concatenate([np.mod(0.5 + 0.05 * rng.standard_normal((n_hi, 3)), 1.0), rng.random((n_lo, 3))])
    mass = np.concatenate([np.full(n_hi, 1.0), np.full(n_lo, 8.0)]) / (n_hi + 8.0 * n_lo)
    eps = np.concatenate([np.full(n_hi, 0.001), np.full(n_lo, 0.012)])
    w = _wl(pos, mass, eps)                      # r_cut = 0.0879, h_lo = 0.0336
    a1, p1, ao1, po1 = _both(B, w)
    check_acc(a1, ao1, what="species geometric")
    a_old = np.linalg.norm(ao1, axis=1).astype(np.float32)
    a2, p2, ao2, po2 = _both(B, w, a_old=a_old)
    check_acc(a2, ao2, what="species relative")
    act = np.sort(rng.choice(n_hi, 1500, replace=False)).astype(np.uint32)     # < n / 16: 8 targets per warp
    a3, p3, ao3, po3 = _both(B, w, active=act, a_old=a_old[act])
    check_acc(a3, ao3, what="species sparse")
    ep = rel_err_scalar(p3, po3)
    assert np.percentile(ep, 99) <= 1e-4 and ep.max() <= 1e-2


# ---- traversal stack: spill / reload path and the capacity latch (og_params.walk_stack_entries / walk_spill_entries) ----
def _spill_case(B, stack_entries, spill_entries):
    import torch
    w = W.make("nfw256", small=True)
    prm = B.make_params(w.r_s, G=w.G, rcut_over_rs=w.rcut_over_rs, alpha=w.alpha, theta=w.theta, leaf_max=1,
                        max_nodes=3 * w.n, flags=B.OG_PERIODIC | B.OG_COUNT, walk_stack_entries=stack_entries,
                        walk_spill_entries=spill_entries)
    pos, mass, eps = (torch.from_numpy(x).cuda() for x in (w.pos, w.mass, w.eps))
    tree = B.og_tree_build(pos, mass, eps, w.L, prm)
    a, p = B.og_shortrange_accel(tree, None, None)
    st = B.og_tree_stats(tree)
    status = B.og_tree_status(tree)
    B.og_tree_free(tree)
    return w, a.cpu().numpy(), p.cpu().numpy(), st, status


def test_stack_spill_and_reload_keep_parity(B):
    """A 64-entry shared-memory stack on a leaf_max = 1 tree forces the warps to move ranges to their global slabs
    and back (stack_spills > 0); the walk still equals the oracle's, and visits exactly the same nodes as the run
    with the default stack (equal counters)."""
    w, a, p, st, status = _spill_case(B, 64, 0)
    assert status == B.OG_OK, B.og_last_error()
    assert st["stack_spills"] > 0, st
    w2, a2, p2, st2, status2 = _spill_case(B, 0, 0)
    assert status2 == B.OG_OK and st2["stack_spills"] == 0
    for k in ("V_full", "V_cull", "A_in", "P_in", "P_soft", "P_out"):
        assert st[k] == st2[k], (k, st[k], st2[k])
    ot = oracle.build_tree(w.pos, w.mass, w.eps, oracle.make_params(w.L, w.r_s, G=w.G, alpha=w.alpha, theta=w.theta,
                                                                     leaf_max=1))
    ao, po, _ = oracle.walk(ot, None, None, want_counters=False)
    check_acc(a, ao, what="spilled stack")
    ep = rel_err_scalar(p, po)
    assert np.percentile(ep, 99) <= 1e-4 and ep.max() <= 1e-2


def test_stack_overflow_is_latched(B):
    """A slab too small for the first spill (16 < 64 / 2 ranges): OG_ERR_STACK_OVERFLOW is latched, nothing faults."""
    _, a, p, st, status = _spill_case(B, 64, 16)
    assert status == B.OG_ERR_STACK_OVERFLOW
    assert np.all(np.isfinite(a))


def test_bad_stack_knobs_are_rejected(B):
    import torch
    w = W.make("uniform32", small=True)
    pos, mass, eps = (torch.from_numpy(x).cuda() for x in (w.pos, w.mass, w.eps))
    for bad in (32, 65, 512):
        with pytest.raises(B.OgError):
            B.og_tree_build(pos, mass, eps, w.L, B.make_params(w.r_s, walk_stack_entries=bad))


# ---- streams (og.h "Streams and a tree") ---------------------------------------------------------------
def test_walks_on_other_streams_are_ordered_after_build_and_each_other(B):
    """Build on one stream, walk at once on two others without any host synchronisation in between: the library
    orders the walks after the build and after each other (they share the tree's scratch state), so the results
    are bit-identical to the single-stream run."""
    import torch
    w = W.make("nfw256", small=True)
    pos, mass, eps = (torch.from_numpy(x).cuda() for x in (w.pos, w.mass, w.eps))
    prm = B.make_params(w.r_s, G=w.G, alpha=w.alpha, theta=w.theta)
    tree = B.og_tree_build(pos, mass, eps, w.L, prm)
    a_ref, p_ref = B.og_shortrange_accel(tree, None, None)
    a_old = torch.linalg.vector_norm(a_ref, dim=1).contiguous()
    a_ref2, p_ref2 = B.og_shortrange_accel(tree, None, a_old)
    torch.cuda.synchronize()
    B.og_tree_free(tree)
    s0, s1, s2 = torch.cuda.Stream(), torch.cuda.Stream(), torch.cuda.Stream()
    for rep in range(3):
        torch.cuda.synchronize()
        tree = B.og_tree_build(pos, mass, eps, w.L, prm, stream=s0)
        a1, p1 = B.og_shortrange_accel(tree, None, None, stream=s1)
        a2, p2 = B.og_shortrange_accel(tree, None, a_old, stream=s2)
        B.og_tree_free(tree, stream=s0)          # ordered after the last walk by the library
        torch.cuda.synchronize()
        assert torch.equal(a1, a_ref) and torch.equal(p1, p_ref)
        assert torch.equal(a2, a_ref2) and torch.equal(p2, p_ref2)
    B.og_trim()


# ---- sub-lists, device-side grouping decision, per-target work figure -------------------------------------
def test_sublist_of_whole_warps_returns_the_same_bits_and_cost_field(B):
    """og.h: a call on a sub-list that covers whole warps (multiples of 32 consecutive targets) of the sorted active
    order returns the same bits as the full call -- also when the sub-list is a small part of the box (the grouping is
    decided from the density of the list in ITS Morton range, not from n_active / n).  With OG_COUNT the tree also
    records the interactions evaluated per target (OG_F_WALK_COST), whose sum is A_in + P_in + P_out."""
    import torch
    w = W.make("nfw256", small=True)
    pos, mass, eps = (torch.from_numpy(x).cuda() for x in (w.pos, w.mass, w.eps))
    prm = B.make_params(w.r_s, G=w.G, alpha=w.alpha, theta=w.theta, flags=B.OG_PERIODIC | B.OG_COUNT)
    tree = B.og_tree_build(pos, mass, eps, w.L, prm)
    a_full, p_full = B.og_shortrange_accel(tree, None, None)
    st = B.og_tree_stats(tree)
    cost = B.og_tree_get(tree, B.OG_F_WALK_COST).cpu().numpy().view(np.uint32)
    assert int(cost.astype(np.int64).sum()) == st["A_in"] + st["P_in"] + st["P_out"]
    assert cost.min() > 0
    perm = B.og_tree_get(tree, B.OG_F_PERM).cpu().numpy().view(np.uint32)
    n = w.n
    for lo, hi in ((0, 32 * 5), (32 * 100, 32 * 163), (n - (n % 32) - 64, n)):      # the last one includes the ragged tail
        sub = perm[lo:hi].copy()
        rng = np.random.default_rng(lo)
        rng.shuffle(sub)                                                        # any order: the library sorts by slot
        act = torch.from_numpy(sub.view(np.int32)).cuda()
        a_sub, p_sub = B.og_shortrange_accel(tree, act, None)
        idx = torch.from_numpy(sub.astype(np.int64)).cuda()
        assert torch.equal(a_sub, a_full[idx]) and torch.equal(p_sub, p_full[idx]), (lo, hi)
        c2 = B.og_tree_get(tree, B.OG_F_WALK_COST).cpu().numpy().view(np.uint32)[: hi - lo]
        assert np.array_equal(c2, cost[sub])
    assert B.og_tree_status(tree) == B.OG_OK
    B.og_tree_free(tree)
    # a tree built without OG_COUNT has no such field
    tree = B.og_tree_build(pos, mass, eps, w.L, B.make_params(w.r_s))
    with pytest.raises(B.OgError):
        B.og_tree_get(tree, B.OG_F_WALK_COST)
    B.og_tree_free(tree)


def test_sparse_full_list_and_its_sub_ranges_agree_under_the_same_grouping(B):
    """og.h (og_shortrange_accel): the bits of a whole-warp sub-list equal the full call's PROVIDED both use the same
    grouping.  A list of two dense clumps at the two ends of the Morton curve counts as sparse (8 targets per warp),
    each clump alone as dense (32 per warp): the automatic choice differs, og_stats.walk_targets_per_warp says so, and
    OG_WALK_G8 / OG_WALK_G32 on the sub-list's tree restore the full call's bits."""
    import torch
    w = W.make("nfw256", small=True)
    pos, mass, eps = (torch.from_numpy(x).cuda() for x in (w.pos, w.mass, w.eps))

    def build(extra=0):
        return B.og_tree_build(pos, mass, eps, w.L, B.make_params(w.r_s, G=w.G, alpha=w.alpha, theta=w.theta,
                                                                  flags=B.OG_PERIODIC | extra))
    tree = build()
    assert B.og_tree_stats(tree)["walk_targets_per_warp"] == 0            # no walk yet
    a_id, p_id = B.og_shortrange_accel(tree, None, None)                  # identity list: 32 per warp
    assert B.og_tree_stats(tree)["walk_targets_per_warp"] == 32
    perm = B.og_tree_get(tree, B.OG_F_PERM).cpu().numpy().view(np.uint32)
    n, m = w.n, 32 * 20
    clump_a, clump_b = perm[:m].copy(), perm[n - m:].copy()               # sorted slots [0, m) and [n - m, n)
    full = np.concatenate([clump_b, clump_a])                             # any order: the library sorts by slot
    np.random.default_rng(5).shuffle(full)
    assert full.size * 16 < n                                             # the rule of og.h: sparse
    dev = lambda x: torch.from_numpy(np.ascontiguousarray(x).view(np.int32)).cuda()
    a_full, p_full = B.og_shortrange_accel(tree, dev(full), None)
    assert B.og_tree_stats(tree)["walk_targets_per_warp"] == 8
    res = {int(i): (a_full[k].clone(), float(p_full[k])) for k, i in enumerate(full)}

    def same_bits(a, p, idx, ref_a=None):
        for k, i in enumerate(idx):
            ra, rp = res[int(i)]
            if not (torch.equal(a[k], ra) and float(p[k]) == rp):
                return False
        return True

    # automatic choice on a clump alone: dense -- a different grouping than the full call's (bits are then not promised)
    B.og_shortrange_accel(tree, dev(clump_a), None)
    assert B.og_tree_stats(tree)["walk_targets_per_warp"] == 32
    B.og_tree_free(tree)
    # the full call's grouping fixed by the flag: the clumps and 32-aligned pieces of the sorted order return its bits
    t8 = build(B.OG_WALK_G8)
    for sub in (clump_a, clump_b, perm[32 * 3:32 * 9].copy(), np.concatenate([perm[32 * 17:m], perm[n - m:n - m + 64]])):
        a_s, p_s = B.og_shortrange_accel(t8, dev(sub), None)
        assert B.og_tree_stats(t8)["walk_targets_per_warp"] == 8
        assert same_bits(a_s, p_s, sub), "sub-list under OG_WALK_G8 differs from the sparse full call"
    B.og_tree_free(t8)
    # and the other way round: the sparse list forced to 32 per warp returns the identity call's bits
    t32 = build(B.OG_WALK_G32)
    a_f, p_f = B.og_shortrange_accel(t32, dev(full), None)
    assert B.og_tree_stats(t32)["walk_targets_per_warp"] == 32
    idx = torch.from_numpy(full.astype(np.int64)).cuda()
    assert torch.equal(a_f, a_id[idx]) and torch.equal(p_f, p_id[idx])
    assert B.og_tree_status(t32) == B.OG_OK
    B.og_tree_free(t32)
    with pytest.raises(B.OgError):
        build(B.OG_WALK_G8 | B.OG_WALK_G32)
