"""Test-side stand-in for paper_2606_17145_b200.binding on CPU tensors, made of oracle/ calls: lets the -m "not gpu"
tests run the HOST layer of row f4 (paper_2606_17145_b200/let.py: packing, exchanges, ordering of the sums) across gloo
ranks without a GPU.  Test infrastructure only; the product never imports it."""
import numpy as np
import torch

import oracle
from oracle import let as olet

OG_OK = 0
OG_F_NODE_LEVEL, OG_F_NODE_NCHILD, OG_F_NODE_LO, OG_F_NODE_HI = 5, 9, 12, 13


class OgError(RuntimeError):
    pass


class _Tree:
    def __init__(self, t, prm):
        self.t, self.prm = t, prm


def _np(x, dt):
    return np.ascontiguousarray(x.detach().cpu().numpy(), dt)


def og_domain_cell_hist(pos, box):
    k = oracle.keys(_np(pos, np.float32), box)
    return torch.from_numpy(np.bincount((k >> np.uint64(48)).astype(np.int64), minlength=1 << 15).astype(np.int32))


def og_domain_owner(pos, box, splitters):
    k = oracle.keys(_np(pos, np.float32), box)
    cell = (k >> np.uint64(48)).astype(np.int64)
    return torch.from_numpy((np.searchsorted(_np(splitters, np.int64), cell, side="right") - 1).astype(np.int32))


def og_tree_build(pos, mass, eps, box, prm):
    return _Tree(oracle.build_tree(_np(pos, np.float32), _np(mass, np.float32), _np(eps, np.float32), prm), prm)


def og_tree_get(tree, field):
    t = tree.t
    if field == OG_F_NODE_LEVEL:
        return torch.from_numpy(t.level.copy())
    if field == OG_F_NODE_NCHILD:
        return torch.from_numpy(t.n_child.copy())
    a = t.lo if field == OG_F_NODE_LO else t.hi
    return torch.from_numpy(np.concatenate([a, np.zeros((a.shape[0], 1), np.float32)], 1))


def og_shortrange_accel(tree, active, a_old, want_pot=True):
    a, p, _ = oracle.walk(tree.t, _np(active, np.uint32), None if a_old is None else _np(a_old, np.float32),
                          want_counters=False)
    return torch.from_numpy(a.astype(np.float32)), torch.from_numpy(p.astype(np.float32))


def og_shortrange_accel_ext(tree, tpos, tsoft, a_old, want_pot=True):
    th = oracle.particle_h(_np(tsoft, np.float32))
    a, p, _ = oracle.walk_ext(tree.t, _np(tpos, np.float32), th, None if a_old is None else _np(a_old, np.float32))
    return torch.from_numpy(a.astype(np.float32)), torch.from_numpy(p.astype(np.float32))


def og_let_export_list(tpos, boxes, r_cut, box):
    b = _np(boxes, np.float64)
    m = olet.within_reach(_np(tpos, np.float32), b[:, :3], b[:, 3:], r_cut, box)
    return torch.from_numpy(np.flatnonzero(m).astype(np.int32))


def og_let_accumulate(acc, pot, idx, part_acc, part_pot):
    acc[idx.long()] += part_acc
    if pot is not None and part_pot is not None:
        pot[idx.long()] += part_pot


def og_tree_status(tree):
    return OG_OK


def og_last_error():
    return ""


def og_tree_free(tree):
    pass
