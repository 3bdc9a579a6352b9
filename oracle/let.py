"""oracle.let -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Plain NumPy restatement of row f4: the short-range force when the particles are
split over R domains, each with its own tree ("the tree walk is executed for particles that reside on
the same MPI rank ('primary') ... particles that require tree nodes of other MPI ranks are exported ... ('secondary')",
:80 export buffers).  The paper prints no rule; readings R49..R53 of DESIGN.md Sec. 13 (Gadget-2's domain
decomposition, Springel 2005):

  R49  domains are contiguous ranges of the Morton order (space-filling-curve segments): with B = 15 key bits (the
       level-5 cells) domain d owns the cells [S_d, S_{d+1}), S_d = the first cell at which the cumulative particle
       count reaches ceil(d N / R)  (S_0 = 0, S_R = 2^15); whole cells only, so the rule is pure integer work.
  R50  every domain builds the canonical tree of its OWN particles in the full box (C1..C4 unchanged).
  R51  the force on a target is the sum over domains of the walk (C6) of that domain's tree with the target's own
       (x, h, a_old): its home domain's walk excludes the target itself by slot (primary), the other domains' walks
       treat it as an external point (secondary, oracle.walk_ext).  Summed in the order home, then domains ascending.
  R52  a target is exported to domain q only if it lies within r_cut of the bounding box of one of q's "top cells"
       (the nodes of q's tree at level 2 when r_cut <= 0.05 L, else at level 1, or shallower leaves; nearest periodic
       image, box-to-point distance).  A domain farther than that contributes exactly nothing, so the filter is exact:
       the nodes at the chosen level and below are culled (R17); a node ABOVE that level which is not opened has the
       target outside its 0.6 l guard box (R15), i.e. at least 0.1 l away from its cell and hence from its centre of
       mass -- the root (l = L) is therefore always opened, and a level-1 node (l = L / 2) that is accepted lies
       >= 0.05 L >= r_cut away and adds nothing (R21: nothing beyond r_cut).  With r_cut > 0.05 L that last step fails
       (an accepted level-1 node can be within r_cut although none of its level-2 children's boxes is), hence level 1.
  R53  a_old of a target is one number (R23) used in every domain's walk.

Only tests/ may import this module; it calls oracle/ only.
"""
from __future__ import annotations

import numpy as np

import oracle

KEY_SHIFT = 48          # 63-bit keys: the top 15 bits are the level-5 cell
N_CELLS = 1 << 15


def splitters(cell_hist: np.ndarray, R: int) -> np.ndarray:
    """R49: S[0..R] from the global histogram of particles per level-5 cell."""
    cum = np.cumsum(cell_hist.astype(np.int64))
    N = int(cum[-1])
    S = np.zeros(R + 1, np.int64)
    S[R] = N_CELLS
    for d in range(1, R):
        want = -(-d * N // R)                         # ceil(d N / R)
        # the first cell c with (particles in cells < c) >= want
        before = np.concatenate([[0], cum[:-1]])
        S[d] = int(np.argmax(before >= want)) if np.any(before >= want) else N_CELLS
    return S


def owners(keys: np.ndarray, R: int):
    cell = (keys >> np.uint64(KEY_SHIFT)).astype(np.int64)
    S = splitters(np.bincount(cell, minlength=N_CELLS), R)
    return (np.searchsorted(S, cell, side="right") - 1).astype(np.int32), S


def top_level(r_cut: float, L: float) -> int:
    """R52: the level whose boxes make the export filter exact."""
    return 2 if r_cut <= 0.05 * L else 1


def top_boxes(tree: "oracle.Tree", level: int = 2):
    """R52: tight AABBs (lo, hi) of the tree's nodes at `level`, and of leaves above it."""
    sel = (tree.level == level) | ((tree.level < level) & (tree.n_child == 0))
    return tree.lo[sel].astype(np.float64), tree.hi[sel].astype(np.float64)


def within_reach(x: np.ndarray, lo: np.ndarray, hi: np.ndarray, r_cut: float, L: float) -> np.ndarray:
    """R52 for targets x [n][3] against boxes [nb]: nearest-image distance from the point to the box <= r_cut."""
    mid, half = 0.5 * (lo + hi), 0.5 * (hi - lo)
    out = np.zeros(x.shape[0], bool)
    for b in range(lo.shape[0]):
        d = x.astype(np.float64) - mid[b]
        d -= L * np.round(d / L)
        e = np.maximum(np.abs(d) - half[b], 0.0)
        out |= (e * e).sum(1) <= r_cut * r_cut
    return out


def let_walk(pos, mass, eps, params, R: int, active_idx=None, a_old=None, export_all: bool = False, level=None):
    """R49..R53 -> (acc f64[n_t][3], pot f64[n_t], info dict) in active order.  `level` overrides R52's choice of the
    top-cell level (tests use it to show that level 2 is not exact for r_cut > 0.05 L)."""
    pos = np.ascontiguousarray(pos, np.float32)
    mass = np.ascontiguousarray(mass, np.float32)
    eps = np.ascontiguousarray(eps, np.float32)
    n = pos.shape[0]
    L = float(params.L)
    r_cut = float(params.rcut_over_rs) * float(params.r_s)
    act = np.arange(n, dtype=np.uint32) if active_idx is None else np.ascontiguousarray(active_idx, np.uint32)
    nt = act.shape[0]
    own, S = owners(oracle.keys(pos, L), R)
    members = [np.flatnonzero(own == d) for d in range(R)]
    trees = [oracle.build_tree(pos[m], mass[m], eps[m], params) if m.size else None for m in members]
    th = oracle.particle_h(eps)
    acc = np.zeros((nt, 3))
    pot = np.zeros(nt)
    t_own = own[act]
    n_exported = np.zeros((R, R), np.int64)
    for d in range(R):                                   # primary: home domain, self excluded by slot
        k = np.flatnonzero(t_own == d)
        if k.size == 0:
            continue
        local_index = np.full(n, -1, np.int64)
        local_index[members[d]] = np.arange(members[d].size)
        a, p, _ = oracle.walk(trees[d], local_index[act[k]].astype(np.uint32), None if a_old is None else a_old[k],
                              want_counters=False)
        acc[k] += a
        pot[k] += p
    for q in range(R):                                   # secondary: domains ascending
        if trees[q] is None:
            continue
        lo, hi = top_boxes(trees[q], top_level(r_cut, L) if level is None else level)
        k = np.flatnonzero(t_own != q)
        if not export_all:
            k = k[within_reach(pos[act[k]], lo, hi, r_cut, L)]
        if k.size == 0:
            continue
        for d in range(R):
            n_exported[d, q] = int((t_own[k] == d).sum())
        a, p, _ = oracle.walk_ext(trees[q], pos[act[k]], th[act[k]], None if a_old is None else a_old[k])
        acc[k] += a
        pot[k] += p
    return acc, pot, {"owner": own, "splitters": S, "n_exported": n_exported,
                      "n_local": np.array([m.size for m in members])}
