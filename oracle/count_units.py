"""TEST / MEASUREMENT INFRASTRUCTURE.  Counts the ALGORITHMIC work per target of the short-range
walk with the oracle's per-target counters, for bench.py's roofline line.

    python -m oracle.count_units [--config nfw256] [--sample 1048576] [--small]

Calls only oracle/ and the seeded generators.  Writes
paper_2606_17145_b200/algorithmic_units.json: per config, the mean per-target counters of the
relative-criterion walk (a_old from a geometric theta pass on the same targets, R23), the mean
algorithmic flops F_alg (decisions + interactions) and F_int (interactions only) with the frozen
weights of oracle.FLOP_WEIGHTS, and the node count (compulsory HBM bytes).
"""
from __future__ import annotations

import argparse
import json
import os
import time

import numpy as np

import oracle
from paper_2606_17145_b200 import workloads as W

OUT = os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "paper_2606_17145_b200",
                   "algorithmic_units.json")


def count(name: str, sample: int, small: bool, seed: int = 12345) -> dict:
    w = W.make(name, small=small)
    prm = oracle.make_params(w.L, w.r_s, G=w.G, rcut_over_rs=w.rcut_over_rs, alpha=w.alpha, theta=w.theta)
    t0 = time.time()
    t = oracle.build_tree(w.pos, w.mass, w.eps, prm)
    t_build = time.time() - t0
    act = np.arange(w.n, dtype=np.uint32) if w.active_idx is None else w.active_idx
    if sample and sample < act.shape[0]:
        rng = np.random.Generator(np.random.PCG64(seed))
        act = np.sort(rng.choice(act, sample, replace=False)).astype(np.uint32)
    t0 = time.time()
    a1, _, _ = oracle.walk(t, act, None, want_counters=False)
    a_old = np.linalg.norm(a1, axis=1).astype(np.float32)
    _, _, cnt = oracle.walk(t, act, a_old)
    t_walk2 = time.time() - t0
    F_alg, F_int = oracle.algorithmic_flops(cnt, with_pot=True)
    F_alg_np, F_int_np = oracle.algorithmic_flops(cnt, with_pot=False)
    mean = cnt.astype(np.float64).mean(axis=0)
    return {
        "config": w.name, "n": w.n, "n_active": w.n_active, "n_nodes": t.n_nodes,
        "targets_counted": int(act.shape[0]),
        "counters_per_target": {k: float(v) for k, v in zip(oracle.COUNTER_NAMES, mean)},
        "F_alg_per_target": float(F_alg.mean()), "F_int_per_target": float(F_int.mean()),
        "F_alg_per_target_nopot": float(F_alg_np.mean()), "F_int_per_target_nopot": float(F_int_np.mean()),
        "interactions_per_target": float(mean[2] + mean[4]),
        # every packed 48-byte walk record and every sorted particle (float4 + h) once; per active target: index 4,
        # a_old 4, gathered position 16, acc 12, pot 4
        "compulsory_hbm_bytes": int(t.n_nodes * 48 + w.n * 20 + w.n_active * 40),
        "weights": oracle.FLOP_WEIGHTS, "weights_nopot": oracle.FLOP_WEIGHTS_NOPOT,
        "oracle_build_s": t_build, "oracle_two_pass_walk_s": t_walk2, "oracle_threads": oracle.num_threads(),
    }


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", default="nfw256")
    ap.add_argument("--sample", type=int, default=1 << 20)
    ap.add_argument("--small", action="store_true")
    a = ap.parse_args()
    data = {}
    if os.path.exists(OUT):
        with open(OUT) as f:
            data = json.load(f)
    r = count(a.config, a.sample, a.small)
    data[r["config"]] = r
    with open(OUT, "w") as f:
        json.dump(data, f, indent=1, sort_keys=True)
    print(json.dumps(r, indent=1))


if __name__ == "__main__":
    main()
