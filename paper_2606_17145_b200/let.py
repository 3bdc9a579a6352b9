"""Row f4: host layer of the domain-decomposed short-range force -- one tree per domain (GPU),
targets exported to the domains within r_cut, partial results summed (PAPER.md:59 primary / secondary phases, :80).
Readings R49..R53, DESIGN.md Sec. 13.  Every arithmetic step runs in the library's kernels (binding.py); this module
only orders the calls, packs buffers and exchanges them: NCCL all-to-all / all-gather through torch.distributed
(`DistExchange`, one process per GPU), or -- for the single-GPU parity tests -- the same calls for every domain one
after the other with the exchange done by list transposition (`LocalExchange`: no rank ever waits on another).
Nothing here imports oracle/.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np
import torch

N_CELLS = 1 << 15       # level-5 cells = the top 15 bits of the 63-bit Morton key


def splitters(cell_hist, n_domains: int) -> np.ndarray:
    """R49: S[0..R]; domain d owns the level-5 cells [S[d], S[d+1]): S[d] = the first cell with at least
    ceil(d N / R) particles in the cells before it.  Integer work on the (all-reduced) histogram, on the host."""
    h = np.asarray(cell_hist, np.int64)
    before = np.cumsum(h) - h
    n = int(h.sum())
    S = np.empty(n_domains + 1, np.int64)
    S[0], S[n_domains] = 0, N_CELLS
    for d in range(1, n_domains):
        want = (d * n + n_domains - 1) // n_domains
        k = int(np.searchsorted(before, want, side="left"))     # `before` is non-decreasing
        S[d] = k if k < N_CELLS else N_CELLS
    return S


class LocalExchange:
    """All domains live in this process; a 'collective' is a transposition of Python lists."""

    def __init__(self, n_domains: int):
        self.R = n_domains
        self.ranks = list(range(n_domains))

    def allreduce_sum(self, per_rank):
        return sum(per_rank[r].to(torch.int64) for r in self.ranks)

    def allgather(self, per_rank):
        return [per_rank[r] for r in range(self.R)]

    def alltoall(self, send):
        """send[r][q] = rows rank r sends to rank q  ->  recv[r][q] = rows rank r receives from rank q."""
        return {r: [send[q][r] for q in range(self.R)] for r in self.ranks}


class DistExchange:
    """One process per GPU; torch.distributed (NCCL on GPUs, gloo in the CPU tests of the plumbing)."""

    def __init__(self, group=None):
        import torch.distributed as dist
        self.dist, self.group = dist, group
        self.R = dist.get_world_size(group)
        self.me = dist.get_rank(group)
        self.ranks = [self.me]

    def allreduce_sum(self, per_rank):
        t = per_rank[self.me].to(torch.int64).clone()
        self.dist.all_reduce(t, group=self.group)
        return t

    def allgather(self, per_rank):
        """Tensors [m_r, C] with different m_r: sizes first, then padded rows."""
        t = per_rank[self.me]
        m = torch.tensor([t.shape[0]], dtype=torch.int64, device=t.device)
        ms = [torch.empty_like(m) for _ in range(self.R)]
        self.dist.all_gather(ms, m, group=self.group)
        ms = [int(x.item()) for x in ms]
        cap = max(max(ms), 1)
        pad = torch.zeros((cap,) + tuple(t.shape[1:]), dtype=t.dtype, device=t.device)
        pad[:t.shape[0]] = t
        out = [torch.empty_like(pad) for _ in range(self.R)]
        self.dist.all_gather(out, pad, group=self.group)
        return [o[:k] for o, k in zip(out, ms)]

    def alltoall(self, send):
        rows = send[self.me]
        dev, dt, tail = rows[0].device, rows[0].dtype, tuple(rows[0].shape[1:])
        cnt = torch.tensor([x.shape[0] for x in rows], dtype=torch.int64, device=dev)
        rcnt = torch.empty_like(cnt)
        self.dist.all_to_all_single(rcnt, cnt, group=self.group)
        ins, outs = cnt.tolist(), rcnt.tolist()
        buf = torch.cat(rows, 0).contiguous()
        out = torch.empty((sum(outs),) + tail, dtype=dt, device=dev)
        self.dist.all_to_all_single(out, buf, output_split_sizes=outs, input_split_sizes=ins, group=self.group)
        return {self.me: list(torch.split(out, outs, 0))}


@dataclass
class Domain:
    """The particles one rank holds: f32 pos [n][3], mass [n], eps [n]; gid int64 [n] (global index, carried along);
    active: int32 local indices of the targets (any order), a_old f32 [n_active] in that order or None."""
    pos: torch.Tensor
    mass: torch.Tensor
    eps: torch.Tensor
    gid: torch.Tensor
    active: torch.Tensor | None = None
    a_old: torch.Tensor | None = None
    extra: dict = field(default_factory=dict)


def decompose(B, parts: dict, ex, box: float):
    """R49: every rank's particles (dict rank -> Domain with arbitrary contents; `active` as a bool mask over the
    particles and `a_old` per PARTICLE here) are moved to the rank that owns their level-5 cell.  Returns
    (dict rank -> Domain in ascending gid order with `active` = local indices, `a_old` in active order; splitters)."""
    hist = {r: B.og_domain_cell_hist(parts[r].pos, box) for r in ex.ranks}
    S = splitters(ex.allreduce_sum(hist).cpu().numpy(), ex.R)
    send = {}
    for r in ex.ranks:
        p = parts[r]
        dev = p.pos.device
        own = B.og_domain_owner(p.pos, box, torch.from_numpy(S.astype(np.int32)).to(dev))
        act = torch.zeros(p.pos.shape[0], device=dev) if p.active is None else p.active.to(torch.float32)
        ao = torch.zeros(p.pos.shape[0], device=dev) if p.a_old is None else p.a_old
        # one row per particle: x, y, z, m, eps, active, a_old, gid (two fp32 halves: exact below 2^48)
        g = p.gid.to(torch.int64)
        row = torch.cat([p.pos, p.mass[:, None], p.eps[:, None], act[:, None], ao[:, None],
                         (g >> 24).to(torch.float32)[:, None], (g & 0xFFFFFF).to(torch.float32)[:, None]], 1)
        send[r] = _split_by_owner(B, row, own, ex.R)
    recv = ex.alltoall(send)
    out = {}
    for r in ex.ranks:
        row = torch.cat(recv[r], 0)
        gid = (row[:, 7].to(torch.int64) << 24) | row[:, 8].to(torch.int64)
        gid, order = _sort_by_key(B, gid)
        row = row[order]
        act = torch.nonzero(row[:, 5] > 0).flatten().to(torch.int32)
        has_aold = any(parts[q].a_old is not None for q in ex.ranks)
        out[r] = Domain(row[:, 0:3].contiguous(), row[:, 3].contiguous(), row[:, 4].contiguous(), gid, act,
                        row[:, 6][act.long()].contiguous() if has_aold else None)
    return out, S


def _sort_by_key(B, key: torch.Tensor):
    """Ascending order of int64 keys >= 0 -> (sorted keys, order as int64 indices): the library's radix sort on the device
    (row a2), torch.sort for the CPU tensors of the plumbing tests."""
    n = int(key.shape[0])
    if n == 0 or not key.is_cuda or not hasattr(B, "og_radix_sort_pairs"):
        ks, order = torch.sort(key, stable=True)
        return ks, order
    bits = max(1, int(key.max().item()).bit_length())
    ks, vs = B.og_radix_sort_pairs(key.clone(), torch.arange(n, dtype=torch.int32, device=key.device), 0, bits)
    return ks, vs.long()


def _split_by_owner(B, row: torch.Tensor, own: torch.Tensor, n_domains: int):
    """rows grouped by owner (one stable sort on the owner + one gather) -> list over the destinations."""
    _, order = _sort_by_key(B, own.to(torch.int64))
    cnt = torch.bincount(own.long(), minlength=n_domains).tolist()
    return [x.contiguous() for x in torch.split(row[order], cnt, 0)]


def top_boxes(B, tree, level: int = 2) -> torch.Tensor:
    """R52: tight AABBs [nb][6] of the tree's nodes at `level` and of the leaves above it."""
    lv = B.og_tree_get(tree, B.OG_F_NODE_LEVEL)
    nc = B.og_tree_get(tree, B.OG_F_NODE_NCHILD)
    sel = (lv == level) | ((lv < level) & (nc == 0))
    lo = B.og_tree_get(tree, B.OG_F_NODE_LO)[sel][:, :3]
    hi = B.og_tree_get(tree, B.OG_F_NODE_HI)[sel][:, :3]
    return torch.cat([lo, hi], 1).contiguous()


def let_forces(B, doms: dict, ex, box: float, prm, geometric: bool = False, want_pot: bool = True, timings: dict | None = None):
    """R50..R53 for the domains this process holds.  -> dict rank -> (acc [n_active][3], pot [n_active] | None) in the
    order of Domain.active; `info` with the export counts."""
    r_cut = float(prm.rcut_over_rs) * float(prm.r_s)
    marks = []

    def mark(name):                                           # optional per-phase device times (ms) -> timings[name]
        if timings is not None:
            e = torch.cuda.Event(enable_timing=True)
            e.record()
            marks.append((name, e))

    mark("start")
    trees, boxes, acc, pot, tpos, teps, info = {}, {}, {}, {}, {}, {}, {"n_exported": {}}
    for r in ex.ranks:                                        # R50 + primary walk (home domain, self excluded)
        d = doms[r]
        dev = d.pos.device
        na = 0 if d.active is None else int(d.active.shape[0])
        if d.pos.shape[0] == 0:                               # an empty domain owns no tree: nothing is exported to it
            trees[r] = None
            boxes[r] = torch.empty((0, 6), dtype=torch.float32, device=dev)
            acc[r] = torch.zeros((0, 3), dtype=torch.float32, device=dev)
            pot[r] = torch.zeros(0, dtype=torch.float32, device=dev) if want_pot else None
            tpos[r] = torch.empty((0, 3), dtype=torch.float32, device=dev)
            teps[r] = torch.empty(0, dtype=torch.float32, device=dev)
            continue
        trees[r] = B.og_tree_build(d.pos, d.mass, d.eps, box, prm)
        mark("build")
        # R52: level-2 boxes are an exact filter only while an accepted level-1 node (target >= 0.05 box away from
        # its cell, outside the guard box) cannot reach inside r_cut; coarser meshes take the level-1 boxes
        boxes[r] = top_boxes(B, trees[r], 2 if r_cut <= 0.05 * float(box) else 1)
        a_old = None if geometric else d.a_old
        if na:
            acc[r], pot[r] = B.og_shortrange_accel(trees[r], d.active, a_old, want_pot=want_pot)
        else:
            acc[r] = torch.zeros((0, 3), dtype=torch.float32, device=dev)
            pot[r] = torch.zeros(0, dtype=torch.float32, device=dev) if want_pot else None
        mark("primary_walk")
        al = d.active.long()
        tpos[r], teps[r] = d.pos[al].contiguous(), d.eps[al].contiguous()
    all_boxes = ex.allgather(boxes)
    send, lists = {}, {}
    for r in ex.ranks:                                        # R52: who needs which other domain
        d = doms[r]
        ao = torch.zeros(tpos[r].shape[0], device=tpos[r].device) if (geometric or d.a_old is None) else d.a_old
        lists[r], send[r] = [], []
        for q in range(ex.R):
            if q == r or all_boxes[q].shape[0] == 0 or tpos[r].shape[0] == 0:
                lst = torch.empty(0, dtype=torch.int32, device=tpos[r].device)
            else:
                lst = B.og_let_export_list(tpos[r], all_boxes[q].to(tpos[r].device), r_cut, box)
            lists[r].append(lst)
            ll = lst.long()
            send[r].append(torch.cat([tpos[r][ll], teps[r][ll][:, None], ao[ll][:, None]], 1).contiguous())
            info["n_exported"][(r, q)] = int(lst.shape[0])
    mark("export_lists")
    recv = ex.alltoall(send)
    mark("exchange")
    back = {}
    for r in ex.ranks:                                        # secondary walk: all imported targets in one call
        cnt = [x.shape[0] for x in recv[r]]
        rows = torch.cat(recv[r], 0)
        if rows.shape[0] and trees[r] is not None:
            a, p = B.og_shortrange_accel_ext(trees[r], rows[:, 0:3].contiguous(), rows[:, 3].contiguous(),
                                             None if geometric else rows[:, 4].contiguous(), want_pot=want_pot)
            res = torch.cat([a, p[:, None] if want_pot else torch.zeros_like(a[:, :1])], 1)
        else:
            res = torch.empty((0, 4), dtype=torch.float32, device=rows.device)
        back[r] = [x.contiguous() for x in torch.split(res, cnt, 0)]
        mark("secondary_walk")
    got = ex.alltoall(back)
    mark("exchange")
    out = {}
    for r in ex.ranks:                                        # R51: home first, then the domains ascending
        for q in range(ex.R):
            part = got[r][q]
            if part.shape[0]:
                B.og_let_accumulate(acc[r], pot[r] if want_pot else None, lists[r][q], part[:, 0:3].contiguous(),
                                    part[:, 3].contiguous() if want_pot else None)
        out[r] = (acc[r], pot[r])
        if trees[r] is not None:
            if B.og_tree_status(trees[r]) != B.OG_OK:
                raise B.OgError(B.og_tree_status(trees[r]), B.og_last_error())
            B.og_tree_free(trees[r])
    mark("sum")
    if timings is not None:
        torch.cuda.synchronize()
        for (_, a), (name, b) in zip(marks[:-1], marks[1:]):
            timings[name] = timings.get(name, 0.0) + a.elapsed_time(b)
    return out, info
