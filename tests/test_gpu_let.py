"""-m gpu: row f4 on the device against oracle/let.py and oracle.walk_ext on the same seeded inputs.
 * og_shortrange_accel_ext (walk for targets that are not particles of the tree) vs oracle.walk_ext: the walk's gates
   (p99 <= 1e-4, max <= 1e-2 relative acceleration error; same for the potential);
 * og_domain_cell_hist / og_domain_owner: bit-exact; og_let_export_list: the oracle's set, plus at most targets within
   the kernel's conservative 1e-5 band of r_cut; og_let_accumulate: exact;
 * the whole pipeline (paper_2606_17145_b200/let.py with LocalExchange: R domains one after the other on one GPU, no rank
   waits on another) vs oracle.let.let_walk: the same gates, owners and export counts equal."""
import numpy as np
import pytest

import oracle
from oracle import let as olet
from paper_2606_17145_b200 import workloads as W
from gpu_common import check_acc, gpu_params, oracle_params, rel_err_scalar, to_dev

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B(cuda_device):
    from paper_2606_17145_b200 import binding
    return binding


@pytest.mark.parametrize("name", ["nfw256", "zoom", "uniform32"])
def test_external_targets_walk_matches_oracle(B, name):
    import torch
    w = W.make(name, small=True)
    rng = np.random.default_rng(17)
    n_t = 5000 + 13                                          # ragged
    # half of the external targets sit on top of the particle distribution (displaced particles), half anywhere
    k = rng.choice(w.n, n_t // 2, replace=False)
    near = np.mod(w.pos[k].astype(np.float64) + rng.standard_normal((n_t // 2, 3)) * 0.3 * w.r_s, w.L)
    tpos = np.vstack([near, rng.random((n_t - n_t // 2, 3)) * w.L]).astype(np.float32)
    tpos[tpos >= w.L] = 0.0
    teps = rng.choice(np.unique(w.eps), n_t).astype(np.float32)
    pos, mass, eps = to_dev(w)
    tree = B.og_tree_build(pos, mass, eps, w.L, gpu_params(w))
    ot = oracle.build_tree(w.pos, w.mass, w.eps, oracle_params(w))
    th = oracle.particle_h(teps)
    tp_d, te_d = torch.from_numpy(tpos).cuda(), torch.from_numpy(teps).cuda()
    # geometric pass, then relative pass with the oracle's |a| as a_old (R23)
    a_g, p_g = B.og_shortrange_accel_ext(tree, tp_d, te_d, None)
    ao_g, po_g, _ = oracle.walk_ext(ot, tpos, th, None)
    check_acc(a_g.cpu().numpy(), ao_g, what=f"{name} ext geometric")
    a_old = np.linalg.norm(ao_g, axis=1).astype(np.float32)
    a_r, p_r = B.og_shortrange_accel_ext(tree, tp_d, te_d, torch.from_numpy(a_old).cuda())
    ao_r, po_r, _ = oracle.walk_ext(ot, tpos, th, a_old)
    q99, mx = check_acc(a_r.cpu().numpy(), ao_r, what=f"{name} ext relative")
    ep = rel_err_scalar(p_r.cpu().numpy(), po_r)
    assert np.percentile(ep, 99) <= 1e-4 and ep.max() <= 1e-2
    # a target far from everything gets exactly zero; results come back in the caller's order
    zero = np.linalg.norm(ao_r, axis=1) == 0
    assert np.all(a_r.cpu().numpy()[zero] == 0)
    assert B.og_tree_status(tree) == B.OG_OK, B.og_last_error()
    print(f"{name}: ext walk p99 {q99:.2e} max {mx:.2e}; {int(zero.sum())} targets out of reach")
    B.og_tree_free(tree)


def test_domain_kernels_bit_exact(B):
    import torch
    from paper_2606_17145_b200 import let
    w = W.make("nfw256", small=True)
    pos = torch.from_numpy(w.pos).cuda()
    keys = oracle.keys(w.pos, w.L)
    hist = B.og_domain_cell_hist(pos, w.L).cpu().numpy()
    assert np.array_equal(hist, np.bincount((keys >> np.uint64(48)).astype(np.int64), minlength=1 << 15))
    for R in (1, 2, 3, 7, 8):
        own_o, S_o = olet.owners(keys, R)
        S = let.splitters(hist, R)
        assert np.array_equal(S, S_o)
        own = B.og_domain_owner(pos, w.L, torch.from_numpy(S.astype(np.int32)).cuda()).cpu().numpy()
        assert np.array_equal(own, own_o)
    # export list against the oracle's rule
    ot = oracle.build_tree(w.pos[own_o == 2], w.mass[own_o == 2], w.eps[own_o == 2], oracle_params(w))
    lo, hi = olet.top_boxes(ot)
    r_cut = 4.5 * w.r_s
    t = np.flatnonzero(own_o != 2)
    ref = olet.within_reach(w.pos[t], lo, hi, r_cut, w.L)
    boxes = torch.from_numpy(np.hstack([lo, hi]).astype(np.float32)).cuda()
    lst = B.og_let_export_list(torch.from_numpy(w.pos[t]).cuda(), boxes, r_cut, w.L).cpu().numpy()
    assert np.all(np.diff(lst) > 0)
    got = np.zeros(len(t), bool)
    got[lst] = True
    assert not np.any(ref & ~got)                                            # nothing the oracle exports is missing
    extra = np.flatnonzero(got & ~ref)
    assert np.all(olet.within_reach(w.pos[t][extra], lo, hi, r_cut * (1 + 3e-5) + 1e-6 * w.L, w.L))
    assert 0 < ref.sum() < len(t)
    # empty inputs
    assert B.og_let_export_list(torch.empty((0, 3), device="cuda"), boxes, r_cut, w.L).numel() == 0
    # accumulate
    acc = torch.zeros((10, 3), device="cuda"); pot = torch.ones(10, device="cuda")
    idx = torch.tensor([7, 2, 9], dtype=torch.int32, device="cuda")
    B.og_let_accumulate(acc, pot, idx, torch.arange(9, dtype=torch.float32, device="cuda").view(3, 3).contiguous(),
                        torch.tensor([1.0, 2.0, 3.0], device="cuda"))
    assert acc[7].tolist() == [0, 1, 2] and acc[2].tolist() == [3, 4, 5] and acc[9].tolist() == [6, 7, 8]
    assert pot.tolist() == [1, 1, 3, 1, 1, 1, 1, 2, 1, 4]


@pytest.mark.parametrize("name,R", [("nfw256", 3), ("nfw256", 8), ("zoom", 4), ("lattice128", 2)])
def test_let_pipeline_matches_oracle(B, name, R):
    import torch
    from paper_2606_17145_b200 import let
    w = W.make(name, small=True)
    prm_o = oracle_params(w)
    act = np.arange(w.n, dtype=np.uint32) if w.active_idx is None else w.active_idx
    # a_old (R23): |a| of the oracle's geometric LET pass, per target
    a_g, _, _ = olet.let_walk(w.pos, w.mass, w.eps, prm_o, R, active_idx=act, a_old=None)
    a_old = np.linalg.norm(a_g, axis=1).astype(np.float32)
    a_ref, p_ref, oinfo = olet.let_walk(w.pos, w.mass, w.eps, prm_o, R, active_idx=act, a_old=a_old)
    # device: everything starts on "rank" r = gid mod R, is decomposed, walked, exchanged, summed
    ex = let.LocalExchange(R)
    active_mask = np.zeros(w.n, bool); active_mask[act] = True
    aold_pp = np.zeros(w.n, np.float32); aold_pp[act] = a_old
    parts = {}
    for r in range(R):
        sel = np.arange(r, w.n, R)
        parts[r] = let.Domain(*(torch.from_numpy(x[sel]).cuda() for x in (w.pos, w.mass, w.eps)),
                              torch.from_numpy(sel.astype(np.int64)).cuda(), torch.from_numpy(active_mask[sel]).cuda(),
                              torch.from_numpy(aold_pp[sel]).cuda())
    doms, S = let.decompose(B, parts, ex, w.L)
    assert np.array_equal(S, oinfo["splitters"])
    for r in range(R):
        assert np.array_equal(doms[r].gid.cpu().numpy(), np.flatnonzero(oinfo["owner"] == r))
    res, info = let.let_forces(B, doms, ex, w.L, gpu_params(w))
    acc = np.zeros((w.n, 3)); pot = np.zeros(w.n)
    for r in range(R):
        g = doms[r].gid[doms[r].active.long()].cpu().numpy()
        acc[g] = res[r][0].cpu().numpy(); pot[g] = res[r][1].cpu().numpy()
    q99, mx = check_acc(acc[act], a_ref, what=f"{name} LET R={R}")
    ep = rel_err_scalar(pot[act], p_ref)
    assert np.percentile(ep, 99) <= 1e-4 and ep.max() <= 1e-2
    n_exp = sum(info["n_exported"].values())
    assert oinfo["n_exported"].sum() <= n_exp <= oinfo["n_exported"].sum() * 1.001 + 2     # (the kernel's 1e-5 band)
    print(f"{name} R={R}: LET acc p99 {q99:.2e} max {mx:.2e}; pot p99 {np.percentile(ep, 99):.2e}; exported {n_exp} "
          f"target copies for {len(act)} targets")


def test_let_empty_domains_active_subset_geometric_on_device(B):
    """As tests/test_let_dist.py::test_empty_domains_..., through the kernels: 7 domains over three occupied cells."""
    import torch
    from paper_2606_17145_b200 import let
    rng = np.random.default_rng(12)
    L = 10.0
    centres = np.array([[1.1, 1.1, 1.1], [1.3, 1.1, 1.1], [7.7, 3.3, 9.1]])
    pos = np.vstack([c + rng.random((40, 3)) * 0.05 for c in centres]).astype(np.float32)
    n = pos.shape[0]
    mass = (rng.random(n) + 0.5).astype(np.float32)
    eps = np.full(n, 1e-3, np.float32)
    prm_o = oracle.make_params(L, 0.2, alpha=0.005, theta=0.5, leaf_max=4)
    prm = B.make_params(0.2, alpha=0.005, theta=0.5, leaf_max=4)
    R = 7
    act = np.sort(rng.choice(n, 50, replace=False)).astype(np.uint32)
    mask = np.zeros(n, bool); mask[act] = True
    ex = let.LocalExchange(R)
    parts = {}
    for r in range(R):
        sel = np.arange(r, n, R)
        parts[r] = let.Domain(*(torch.from_numpy(x[sel]).cuda() for x in (pos, mass, eps)),
                              torch.from_numpy(sel.astype(np.int64)).cuda(), torch.from_numpy(mask[sel]).cuda(), None)
    doms, S = let.decompose(B, parts, ex, L)
    assert [int(doms[r].pos.shape[0]) for r in range(R)].count(0) >= 3
    res, info = let.let_forces(B, doms, ex, L, prm, geometric=True)
    a_ref, p_ref, oinfo = olet.let_walk(pos, mass, eps, prm_o, R, active_idx=act, a_old=None)
    assert np.array_equal(S, oinfo["splitters"])
    got = np.zeros((n, 3)); gp = np.zeros(n)
    for r in range(R):
        g = doms[r].gid[doms[r].active.long()].cpu().numpy()
        got[g] = res[r][0].cpu().numpy(); gp[g] = res[r][1].cpu().numpy()
    check_acc(got[act], a_ref, what="LET with empty domains")
    ep = rel_err_scalar(gp[act], p_ref)
    assert np.percentile(ep, 99) <= 1e-4 and ep.max() <= 1e-2


def test_external_targets_on_top_of_tree_particles_and_across_the_wall(B):
    """External targets that coincide with particles of the tree (r = 0 pairs: force 0, potential -(14/5) G m / h, C5;
    nothing is excluded) and targets within r_cut of the periodic wall."""
    import torch
    w = W.make("uniform32", small=True)
    rng = np.random.default_rng(3)
    k = rng.choice(w.n, 300, replace=False)
    wall = rng.random((300, 3)).astype(np.float32) * w.L
    wall[:, 0] = (rng.random(300) * 0.5 * w.r_s).astype(np.float32)             # hugging x = 0
    wall[150:, 1] = np.float32(w.L) - (rng.random(150) * 0.5 * w.r_s).astype(np.float32)
    wall[wall >= w.L] = 0.0
    tpos = np.vstack([w.pos[k], wall]).astype(np.float32)
    teps = np.full(600, float(w.eps[0]), np.float32)
    pos, mass, eps = to_dev(w)
    tree = B.og_tree_build(pos, mass, eps, w.L, gpu_params(w))
    ot = oracle.build_tree(w.pos, w.mass, w.eps, oracle_params(w))
    th = oracle.particle_h(teps)
    ao_g, _, _ = oracle.walk_ext(ot, tpos, th, None)
    a_old = np.linalg.norm(ao_g, axis=1).astype(np.float32)
    ao, po, _ = oracle.walk_ext(ot, tpos, th, a_old)
    a, p = B.og_shortrange_accel_ext(tree, torch.from_numpy(tpos).cuda(), torch.from_numpy(teps).cuda(),
                                     torch.from_numpy(a_old).cuda())
    check_acc(a.cpu().numpy(), ao, what="ext coincident / wall")
    ep = rel_err_scalar(p.cpu().numpy(), po)
    assert np.percentile(ep, 99) <= 1e-4 and ep.max() <= 1e-2
    # the coincident pair really is in the sum: the potential of such a target is lower than without its twin
    d, pd = oracle.direct_ext(np.delete(w.pos, k[:1], 0), np.delete(w.mass, k[:1]), np.delete(w.eps, k[:1]), oracle_params(w),
                              tpos[:1], teps[:1])
    assert po[0] < pd[0]
    assert B.og_tree_status(tree) == B.OG_OK
    B.og_tree_free(tree)
    # a counting tree (OG_COUNT) and MORE external targets than the tree has particles: same numbers, nothing overrun
    small = W.Workload("few", w.pos[:200].copy(), w.mass[:200].copy(), w.eps[:200].copy(), w.L, w.r_s)
    tc = B.og_tree_build(*(torch.from_numpy(x).cuda() for x in (small.pos, small.mass, small.eps)), small.L,
                         gpu_params(small, flags=B.OG_COUNT))
    guard = torch.full((4096,), 7.0, device="cuda")                              # allocated right after the tree
    a2, p2 = B.og_shortrange_accel_ext(tc, torch.from_numpy(tpos).cuda(), torch.from_numpy(teps).cuda(), None)
    oc = oracle.build_tree(small.pos, small.mass, small.eps, oracle_params(small))
    ao2, po2, _ = oracle.walk_ext(oc, tpos, th, None)
    nz = np.linalg.norm(ao2, axis=1) > 0
    check_acc(a2.cpu().numpy()[nz], ao2[nz], what="ext on a counting tree")
    assert B.og_tree_status(tc) == B.OG_OK and float(guard.min()) == 7.0
    B.og_tree_free(tc)


def test_external_targets_grouping_follows_their_density_against_the_tree(B):
    """og.h (og_shortrange_accel_ext): external targets are walked 8 per warp when they are fewer than 1 / 16 of the
    tree's particles in the key range they span, else 32 per warp; OG_WALK_G32 / OG_WALK_G8 fix it and
    og_stats.walk_targets_per_warp reports it.  Either grouping meets the oracle within the walk's gates."""
    import torch
    w = W.make("nfw256", small=True)
    rng = np.random.default_rng(23)
    pos, mass, eps = to_dev(w)
    ot = oracle.build_tree(w.pos, w.mass, w.eps, oracle_params(w))
    few = (rng.random((300, 3)) * w.L).astype(np.float32)                    # 300 x 16 << n: sparse
    many = np.mod(w.pos[rng.choice(w.n, 20000, replace=False)].astype(np.float64) + 0.01, w.L).astype(np.float32)   # dense
    many[many >= w.L] = 0.0
    for tpos, expect in ((few, 8), (many, 32)):
        teps = np.full(tpos.shape[0], float(w.eps[0]), np.float32)
        ao, po, _ = oracle.walk_ext(ot, tpos, oracle.particle_h(teps), None)
        tp_d, te_d = torch.from_numpy(tpos).cuda(), torch.from_numpy(teps).cuda()
        for flags, tpw in ((0, expect), (B.OG_WALK_G32, 32), (B.OG_WALK_G8, 8)):
            tree = B.og_tree_build(pos, mass, eps, w.L, gpu_params(w, flags=flags))
            a, p = B.og_shortrange_accel_ext(tree, tp_d, te_d, None)
            assert B.og_tree_stats(tree)["walk_targets_per_warp"] == tpw, (tpos.shape[0], flags)
            check_acc(a.cpu().numpy(), ao, what=f"ext {tpos.shape[0]} targets, {tpw} per warp")
            assert B.og_tree_status(tree) == B.OG_OK, B.og_last_error()
            B.og_tree_free(tree)
