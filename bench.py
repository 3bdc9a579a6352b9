#!/usr/bin/env python
"""bench.py -- one JSON line per run (contract in the task statement).

    python bench.py --gpus N --steps K --warmup W [--impl reference] [--workload nfw256]

A "step" is one pass of the whole hot path over one batch of
synthetic input: og_tree_build (Morton keys -> radix sort -> gather -> octree -> upward pass)
followed by og_shortrange_accel (relative opening criterion, alpha = 0.005, a_old from an untimed
geometric-theta pass) on all active targets.  Default workload: BASELINE.json configs[2], the
16.8M-particle clustered box the north_star's roofline target is quoted on ("nfw256").

value    = active particles per second over the whole step, inputs resident in HBM.
e2e      = the same through og_shortrange_accel_host with pinned HOST buffers (H2D + D2H inside).
roofline = the walk kernel (dominant): algorithmic flops (oracle-counted per-target figure of
           paper_2606_17145_b200/algorithmic_units.json x active targets) / its CUDA-event time,
           against the FP32 ALU peak SMs x 128 lanes x 2 flop x max SM clock ("bound": "alu").
cpu_baseline = the oracle (oracle/, untuned) on the host cores, bounded sample, rank 0, N = 1.

N > 1: one process per GPU (torchrun); every rank works on its own seeded box of the same config
(weak scaling, no data-path collective -- DESIGN.md Sec. 8); time = max over ranks.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_2606_17145_b200 import workloads as W  # noqa: E402

METRIC = "short-range tree-gravity particles/s (tree build + walk, 1 step) on B200"
UNIT = "particles/s"
SM_LANES = 128          # FP32 lanes per SM (B200)
KERNELS_PER_BUILD = 1 + (2 + 8) + 1 + 2   # keys, sort (digit histograms, their scan, 8 one-sweep passes), gather, octree + upward
KERNELS_PER_WALK_ALL = 1


def load_units(name):
    p = os.path.join(ROOT, "paper_2606_17145_b200", "algorithmic_units.json")
    if not os.path.exists(p):
        return None
    with open(p) as f:
        return json.load(f).get(name)


def ncu_traffic(name):
    """dram__bytes_read.sum + dram__bytes_write.sum of one k_walk_group launch on workload `name`, taken from the
    committed ncu --set full summary profiles/walk_traffic_<name>.txt (line "dram_bytes_per_launch <bytes>")."""
    p = os.path.join(ROOT, "profiles", f"walk_traffic_{name}.txt")
    if not os.path.exists(p):
        return None
    with open(p) as f:
        for line in f:
            tok = line.split()
            if len(tok) >= 2 and tok[0] == "dram_bytes_per_launch":
                return float(tok[1])
    return None


def fp32_probe(iters=100000):
    """Measured FP32 rates (TFLOP/s) of the scalar FFMA and the packed FFMA2 encoding, from the bench-side helper
    library libogprobe.so (csrc/probe.cu; not part of libogtree.so).  None if the helper is missing."""
    import ctypes as C
    path = os.path.join(ROOT, "paper_2606_17145_b200", "libogprobe.so")
    if not os.path.exists(path):
        return None
    lib = C.CDLL(path)
    lib.ogp_fp32_probe.restype = C.c_int
    lib.ogp_fp32_probe.argtypes = [C.c_int, C.c_uint64, C.POINTER(C.c_double), C.POINTER(C.c_double)]
    out = {}
    for mode, name in ((0, "ffma"), (1, "ffma2")):
        ms, fl = C.c_double(), C.c_double()
        if lib.ogp_fp32_probe(mode, iters, C.byref(ms), C.byref(fl)) != 0 or ms.value <= 0:
            return None
        out[name] = fl.value / (ms.value * 1e-3) / 1e12
    return out


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            return json.load(f), "measured"
    return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "sm_max_mhz": 1965.0}, "fallback"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), line.strip()))

    def stop(self, t0, t1):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        sm, smax, reasons = [], None, set()
        for ts, line in self.rows:
            f = [x.strip() for x in line.split(",")]
            if len(f) < 7:
                continue
            try:
                if t0 - 0.05 <= ts <= t1 + 0.15:
                    sm.append(float(f[0]))
                smax = float(f[1])
            except ValueError:
                continue
            if t0 - 0.05 <= ts <= t1 + 0.15:
                for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), f[3:7]):
                    if v.lower().startswith("active"):
                        reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": smax, "reasons": sorted(reasons),
                "samples": len(sm)}


def make_workload(name, rank):
    """BASELINE.json config by name; rank r > 0 draws an independent box with seed + 7919 r."""
    if rank == 0:
        return W.make(name)
    if name == "nfw256":
        return W.nfw_box(256, 2000, 100.0, W.SEED0 + 3000 + 7919 * rank)
    if name == "uniform32":
        return W.uniform_box(32, 1.0, W.SEED0 + 1000 + 7919 * rank)
    if name == "lattice128":
        return W.perturbed_lattice(128, 1.0, W.SEED0 + 2000 + 7919 * rank)
    if name == "zoom":
        return W.zoom(seed=W.SEED0 + 4000 + 7919 * rank)
    return W.make(name)


def aggregate(n_active_per_rank, ms_max):
    """value over all ranks: units all ranks processed / max-over-ranks time."""
    return float(sum(n_active_per_rank)) / (ms_max * 1e-3)


def dist_setup(n_gpus, backend):
    import torch.distributed as dist
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world > 1 and not dist.is_initialized():
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group(backend=backend)
    return world, rank, local


def all_max(x, device):
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return x
    t = torch.tensor([x], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def all_gather_int(x, device):
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return [x]
    t = torch.tensor([x], dtype=torch.int64, device=device)
    out = [torch.zeros_like(t) for _ in range(dist.get_world_size())]
    dist.all_gather(out, t)
    return [int(o.item()) for o in out]


def barrier():
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized():
        dist.barrier()


def cpu_baseline(w, sample=1 << 17, seed=4242):
    """The oracle as it stands on the host cores: full tree build (single thread) + relative-criterion walk
    of a seeded random sample of the active targets (all cores), walk time scaled to all active targets."""
    import oracle
    prm = oracle.make_params(w.L, w.r_s, G=w.G, rcut_over_rs=w.rcut_over_rs, alpha=w.alpha, theta=w.theta)
    t0 = time.perf_counter()
    t = oracle.build_tree(w.pos, w.mass, w.eps, prm)
    t_build = time.perf_counter() - t0
    act = np.arange(w.n, dtype=np.uint32) if w.active_idx is None else w.active_idx
    rng = np.random.Generator(np.random.PCG64(seed))
    ns = min(sample, act.shape[0])
    sub = np.sort(rng.choice(act, ns, replace=False)).astype(np.uint32)
    a1, _, _ = oracle.walk(t, sub, None, want_counters=False)          # a_old (untimed, as on the GPU)
    a_old = np.linalg.norm(a1, axis=1).astype(np.float32)
    t0 = time.perf_counter()
    oracle.walk(t, sub, a_old, want_counters=False)
    t_walk = time.perf_counter() - t0
    t_full = t_build + t_walk * (act.shape[0] / ns)
    return {"value": act.shape[0] / t_full, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
            "sample": f"full {w.n}-particle oracle tree build ({t_build:.1f} s, 1 thread) + relative-criterion walk of "
                      f"{ns} seeded random targets ({t_walk:.2f} s on {oracle.num_threads()} threads), walk time scaled "
                      f"by {act.shape[0]}/{ns}",
            "build_s": t_build, "walk_sample_s": t_walk, "walk_us_per_target_per_core":
            1e6 * t_walk * oracle.num_threads() / ns}, t


def run_reference(args):
    """--impl reference: the oracle, timed on the host cores (rank 0 only)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    import oracle
    w = W.make(args.workload)
    prm = oracle.make_params(w.L, w.r_s, G=w.G, rcut_over_rs=w.rcut_over_rs, alpha=w.alpha, theta=w.theta)
    t0 = time.perf_counter()
    t = oracle.build_tree(w.pos, w.mass, w.eps, prm)
    t_build = time.perf_counter() - t0
    act = np.arange(w.n, dtype=np.uint32) if w.active_idx is None else w.active_idx
    ns = min(args.ref_sample, act.shape[0])
    times = []
    for it in range(args.warmup + args.steps):
        rng = np.random.Generator(np.random.PCG64(977 + it))
        sub = np.sort(rng.choice(act, ns, replace=False)).astype(np.uint32)
        a1, _, _ = oracle.walk(t, sub, None, want_counters=False)
        a_old = np.linalg.norm(a1, axis=1).astype(np.float32)
        t0 = time.perf_counter()
        oracle.walk(t, sub, a_old, want_counters=False)
        dt = time.perf_counter() - t0
        if it >= args.warmup:
            times.append(dt)
    t_walk = float(np.mean(times))
    t_full = t_build + t_walk * (act.shape[0] / ns)
    value = act.shape[0] / t_full
    sample = (f"per step: relative-criterion oracle walk of {ns} seeded random targets, scaled by {act.shape[0]}/{ns}, "
              f"plus the full {w.n}-particle oracle tree build measured once ({t_build:.1f} s, 1 thread)")
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * t_full, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            # the keys of the repo arm's `config` (same workload, same canonical tree), so that the two lines compare
            "config": {"workload": w.name, "n": w.n, "n_active": w.n_active, "box": w.L, "r_s": w.r_s, "alpha": w.alpha,
                       "leaf_max": 8, "n_nodes": int(t.level.shape[0]), "max_level": int(t.level.max()),
                       "l2_policy": "inputs larger than L2 (no flush): particles + tree > 1.5 GB vs 126 MB L2",
                       "parallelism": f"oracle on {oracle.num_threads()} host cores (no GPU)"},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
                             "sample": sample},
            # ms_per_step is not a measured wall time: walk of `sample_targets` targets scaled to all active ones
            "extrapolated": True, "sample_targets": int(ns), "tree_build_s": t_build, "walk_sample_s": t_walk,
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))
    return 0


def run_ours(args):
    import torch
    from paper_2606_17145_b200 import binding as B

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the product path has no CPU fallback)")
    world, rank, local = dist_setup(args.gpus, "nccl")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    strong = args.scaling == "strong"
    w = make_workload(args.workload, 0 if strong else rank)   # strong: every rank holds the same box (and tree)
    n, na = w.n, w.n_active
    prm = B.make_params(w.r_s, G=w.G, rcut_over_rs=w.rcut_over_rs, alpha=w.alpha, theta=w.theta, leaf_max=8)
    prm.flags |= {"auto": 0, "32": B.OG_WALK_G32, "8": B.OG_WALK_G8}[args.walk_grouping]
    h_pos = torch.from_numpy(w.pos).pin_memory()
    h_mass = torch.from_numpy(w.mass).pin_memory()
    h_eps = torch.from_numpy(w.eps).pin_memory()
    h_act = None if w.active_idx is None else torch.from_numpy(w.active_idx.view(np.int32)).pin_memory()
    pos, mass, eps = h_pos.to(dev), h_mass.to(dev), h_eps.to(dev)
    act = None if h_act is None else h_act.to(dev)
    acc = torch.empty((na, 3), dtype=torch.float32, device=dev)
    pot = torch.empty((na,), dtype=torch.float32, device=dev)

    # a_old: |a| of a geometric-theta pass (R23), untimed
    tree = B.og_tree_build(pos, mass, eps, w.L, prm)
    B.og_shortrange_accel(tree, act, None, acc_out=acc, pot_out=pot)
    a_old = torch.linalg.vector_norm(acc, dim=1).contiguous()
    if B.og_tree_status(tree) != B.OG_OK:
        raise SystemExit("bench.py: tree status " + B.og_last_error())
    st_tree = B.og_tree_stats(tree)
    B.og_tree_free(tree)

    shard = None
    if strong:
        # SURVEY.md Sec. 8.5 / DESIGN.md Sec. 8: redundant tree per rank, contiguous Morton range of the active targets per
        # rank, balanced by the per-target work of an (untimed) counted pass; no data-path collective, no reduction
        from paper_2606_17145_b200 import sharding as S
        prm_c = B.make_params(w.r_s, G=w.G, rcut_over_rs=w.rcut_over_rs, alpha=w.alpha, theta=w.theta, leaf_max=8,
                              flags=B.OG_PERIODIC | B.OG_COUNT)
        tc = B.og_tree_build(pos, mass, eps, w.L, prm_c)
        B.og_shortrange_accel(tc, act, a_old, acc_out=acc, pot_out=pot)
        torch.cuda.synchronize()
        cost = B.og_tree_get(tc, B.OG_F_WALK_COST).cpu().numpy().view(np.uint32)[:na]
        inv_perm = B.og_tree_get(tc, B.OG_F_INV_PERM).cpu().numpy().view(np.uint32)
        # a rank's share is walked with the grouping the full list got (og.h: the bits of a sub-list equal the full
        # call's only under the same grouping, and the automatic choice looks at each list's own Morton span)
        tpw = B.og_tree_stats(tc)["walk_targets_per_warp"]
        B.og_tree_free(tc)
        if w.active_idx is not None:
            prm.flags |= B.OG_WALK_G8 if tpw == 8 else B.OG_WALK_G32
        slots = inv_perm if w.active_idx is None else inv_perm[w.active_idx]
        order = S.sorted_active_order(slots)
        bounds = S.partition_by_cost(cost[order], world)
        my_pos, my_idx = S.rank_sublist(w.active_idx, n, order, bounds, rank)
        full_acc, full_pot = acc.clone(), pot.clone()                 # the single-call result, for the bit check below
        my_pos_d = torch.from_numpy(my_pos.astype(np.int64)).to(dev)
        act = torch.from_numpy(my_idx.view(np.int32)).to(dev)
        a_old = a_old[my_pos_d].contiguous()
        na = int(my_idx.shape[0])
        acc = torch.empty((na, 3), dtype=torch.float32, device=dev)
        pot = torch.empty((na,), dtype=torch.float32, device=dev)
        shard = {"bounds": [int(x) for x in bounds], "cost_share_max_over_mean":
                 float(max(cost[order][bounds[r]:bounds[r + 1]].sum() for r in range(world)) * world / max(cost.sum(), 1))}

    def step(ev=None):
        if ev:
            ev[0].record()
        t = B.og_tree_build(pos, mass, eps, w.L, prm)
        if ev:
            ev[1].record()
        B.og_shortrange_accel(t, act, a_old, acc_out=acc, pot_out=pot)
        if ev:
            ev[2].record()
        B.og_tree_free(t)

    for _ in range(args.warmup):
        step()
    torch.cuda.synchronize()
    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(args.steps)]
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    sampler = ClockSampler(local)
    sampler.start()
    time.sleep(0.3)
    barrier()
    torch.cuda.synchronize()
    t0 = time.time()
    e0.record()
    for k in range(args.steps):
        step(evs[k])
    e1.record()
    torch.cuda.synchronize()
    barrier()
    t1 = time.time()
    ms_total = all_max(e0.elapsed_time(e1), dev)
    clocks = sampler.stop(t0, t1)
    ms_step = ms_total / args.steps
    ms_build = float(np.mean([e[0].elapsed_time(e[1]) for e in evs]))
    ms_walk = float(np.mean([e[1].elapsed_time(e[2]) for e in evs]))
    n_act_all = all_gather_int(na, dev)
    value = aggregate(n_act_all, ms_step)

    if strong:
        # every rank's share equals the single-call result bit for bit (whole warps of the same sorted order)
        ok = bool(torch.equal(acc, full_acc[my_pos_d]) and torch.equal(pot, full_pot[my_pos_d]))
        shard["bitwise_equal_to_single_call"] = bool(all_max(0.0 if ok else 1.0, dev) == 0.0)
        shard["targets_per_warp"] = int(tpw)
        if not shard["bitwise_equal_to_single_call"]:
            raise SystemExit("bench.py --scaling strong: a rank's share differs from the single-call result")
        h_act = torch.from_numpy(my_idx.view(np.int32)).pin_memory()
        del full_acc, full_pot
    # e2e through the HOST-buffer entry point (pinned inputs, H2D + build + walk + D2H inside)
    h_aold = a_old.cpu().pin_memory()
    h_acc = torch.empty((na, 3), dtype=torch.float32).pin_memory()
    h_pot = torch.empty((na,), dtype=torch.float32).pin_memory()
    e2e_steps = max(1, min(args.steps, 3))
    B.og_shortrange_accel_host(h_pos, h_mass, h_eps, w.L, prm, h_act, h_aold, acc_out=h_acc, pot_out=h_pot)
    barrier()
    torch.cuda.synchronize()
    f0, f1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    f0.record()
    for _ in range(e2e_steps):
        B.og_shortrange_accel_host(h_pos, h_mass, h_eps, w.L, prm, h_act, h_aold, acc_out=h_acc, pot_out=h_pot)
    f1.record()
    torch.cuda.synchronize()
    ms_e2e = all_max(f0.elapsed_time(f1), dev) / e2e_steps
    h2d = n * 20 + na * 4 + (0 if h_act is None else na * 4)
    d2h = na * 16

    if rank != 0:
        return 0
    # counters of one untimed counted walk (cross-check of the oracle-counted per-target figure)
    prm_c = B.make_params(w.r_s, G=w.G, rcut_over_rs=w.rcut_over_rs, alpha=w.alpha, theta=w.theta, leaf_max=8,
                          flags=B.OG_PERIODIC | B.OG_COUNT)
    tc = B.og_tree_build(pos, mass, eps, w.L, prm_c)
    B.og_shortrange_accel(tc, act, a_old, acc_out=acc, pot_out=pot)
    stc = B.og_tree_stats(tc)
    status = B.og_tree_status(tc)
    B.og_tree_free(tc)
    checksum = float(torch.linalg.vector_norm(acc.double(), dim=1).mean().item())

    peaks, peaks_src = measured_peaks()
    sms = torch.cuda.get_device_properties(dev).multi_processor_count
    fmax = float(peaks.get("sm_max_mhz", 1965.0)) * 1e6
    peak_tflops = sms * SM_LANES * 2 * fmax / 1e12
    units = load_units(w.name)
    Wt = {"V_cull": 6, "V_full": 16, "A_in": 21, "P_out": 11, "P_in": 32, "P_soft_extra": 13}
    F_gpu = (Wt["V_cull"] * stc["V_cull"] + Wt["V_full"] * stc["V_full"] + Wt["A_in"] * stc["A_in"] +
             Wt["P_out"] * stc["P_out"] + Wt["P_in"] * stc["P_in"] + Wt["P_soft_extra"] * stc["P_soft"])
    if units:
        F_alg = units["F_alg_per_target"] * na
        F_int = units["F_int_per_target"] * na
        inter = units["interactions_per_target"] * na
        units_src = "oracle-counted per-target figure (algorithmic_units.json) x active targets"
    else:
        # no oracle-counted figure for this workload: no algorithmic flops, hence no roofline fraction (the
        # kernel's own OG_COUNT counters are reported beside it but never grade the kernel)
        F_alg, F_int, inter = None, None, float(stc["A_in"] + stc["P_in"])
        units_src = "none: no oracle-counted figure in algorithmic_units.json for this workload (run oracle/count_units.py)"
    achieved = F_alg / (ms_walk * 1e-3) / 1e12 if F_alg else None
    probe = fp32_probe()
    t_hbm_ms = (units["compulsory_hbm_bytes"] if units else 0) / (float(peaks["hbm_gbs"]) * 1e9) * 1e3
    roofline = {
        "bound": "alu", "kernel": "k_walk_group", "achieved": achieved, "peak": peak_tflops, "unit": "TFLOP/s",
        "frac": achieved / peak_tflops if achieved else None, "traffic": ncu_traffic(w.name),
        "traffic_source": f"profiles/walk_traffic_{w.name}.txt (one committed ncu --set full capture; not measured in this run)",
        "peak_source": f"{sms} SMs x {SM_LANES} FP32 lanes x 2 flop x {fmax / 1e6:.0f} MHz (max SM clock, "
                       f"MEASURED_PEAKS.json {peaks_src}); DESIGN.md Sec. 7",
        "algorithmic_flops_per_launch": F_alg, "units": units_src,
        "frac_interactions_only": (F_int / (ms_walk * 1e-3) / 1e12 / peak_tflops) if F_int else None,
        "algorithmic_flops_gpu_counters": float(F_gpu),
        "ffma_probe_tflops": probe["ffma"] if probe else None,
        "ffma2_probe_tflops": probe["ffma2"] if probe else None,
        "hbm_bound_ms": t_hbm_ms, "alu_bound_ms": F_alg / (peak_tflops * 1e12) * 1e3 if F_alg else None,
        "kernel_ms": ms_walk, "kernel_share_of_step": ms_walk / (ms_build + ms_walk),
    }
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_step, "higher_is_better": True, "scaling": args.scaling, "vs_baseline": None, "dtype": "f32",
        "data": "synthetic",
        "config": {"workload": w.name, "n": n, "n_active": int(sum(n_act_all)) if strong else na, "box": w.L, "r_s": w.r_s, "alpha": w.alpha,
                   "leaf_max": 8, "n_nodes": st_tree["n_nodes"], "max_level": st_tree["max_level"],
                   "l2_policy": "inputs larger than L2 (no flush): particles + tree > 1.5 GB vs 126 MB L2",
                   "parallelism": ("1 GPU" if world == 1 else
                                   f"{world} GPUs, one box: tree built on every rank, Morton ranges of the active targets "
                                   f"balanced by last pass's per-target work" if strong else
                                   f"{world} independent boxes (one per GPU)")},
        "clocks": clocks,
        "e2e": {"value": aggregate(n_act_all, ms_e2e), "unit": UNIT, "h2d_bytes_per_step": h2d,
                "d2h_bytes_per_step": d2h, "ms_per_step": ms_e2e, "steps": e2e_steps},
        # with an explicit active list: slot keys, a radix sort (2 + ceil(log2 n / 8) one-sweep passes), slot unpack, and
        # the second instantiation of the walk kernel (the one the device-side decision does not pick returns at once)
        "gpu_launches": args.steps * (KERNELS_PER_BUILD + KERNELS_PER_WALK_ALL +
                                      (0 if act is None else 2 + 2 + ((max(1, (n - 1).bit_length()) + 7) // 8) + 1)),
        "roofline": roofline,
        "breakdown_ms": {"build_a1_a5": ms_build, "walk_a6_a7": ms_walk},
        "particles_per_s_walk_only": na / (ms_walk * 1e-3),
        "interactions_per_s_walk_only": inter / (ms_walk * 1e-3),
        "walk_counters": stc, "status": status, "checksum_mean_abs_acc": checksum,
    }
    if shard is not None:
        line["strong_sharding"] = shard
    if world == 1 and not args.no_cpu_baseline:
        cb, _ = cpu_baseline(w, sample=args.cpu_sample)
        line["cpu_baseline"] = cb
    print(json.dumps(line))
    return 0


def run_timesteps(args):
    """--timesteps K (row f2): K synchronisation steps of the hierarchical time-step shell on the
    workload (all particles, seeded small velocities): next tick -> drift ALL -> active list -> tree rebuild -> short-range
    walk of the active particles with their carried a_old -> kick + new bins.  Prints its own JSON line: per-step sizes
    of the active set and device times of each phase (the paper's small-bin regime)."""
    import torch
    from paper_2606_17145_b200 import binding as B
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the product path has no CPU fallback)")
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(0)
    w = W.make(args.workload)
    n, L = w.n, w.L
    prm = B.make_params(w.r_s, G=w.G, rcut_over_rs=w.rcut_over_rs, alpha=w.alpha, theta=w.theta, leaf_max=8)
    pos = torch.from_numpy(w.pos).to(dev)
    mass, eps = torch.from_numpy(w.mass).to(dev), torch.from_numpy(w.eps).to(dev)
    tree = B.og_tree_build(pos, mass, eps, L, prm)
    acc, _ = B.og_shortrange_accel(tree, None, None, want_pot=False)
    B.og_tree_free(tree)
    anorm = torch.linalg.vector_norm(acc, dim=1)
    a_med = float(anorm.median().item())
    eta, bmax = 0.025, 8
    dt_max = 4.0 * float(np.sqrt(2.0 * eta * float(w.eps.mean()) / a_med))     # the median particle sits two levels down
    g = torch.Generator(device=dev)
    g.manual_seed(W.SEED0 + 77)
    vel = (torch.randn((n, 3), generator=g, device=dev) * (0.05 * float(w.eps.mean()) / (dt_max / 2 ** bmax) / 16)).contiguous()
    bins = torch.zeros(n, dtype=torch.uint8, device=dev)
    a_old = torch.zeros(n, device=dev)
    act = torch.empty(n, dtype=torch.int32, device=dev)
    scratch = torch.empty(B.og_ts_scratch_bytes(n), dtype=torch.uint8, device=dev)
    B.og_ts_kick(vel, bins, a_old, None, n, acc, eps, eta, dt_max, bmax, 0, True)
    hist0 = torch.bincount(bins.long(), minlength=bmax + 1).cpu().tolist()
    ev = lambda: torch.cuda.Event(enable_timing=True)
    tick, rows = 0, []
    torch.cuda.synchronize()
    t_all0 = ev(); t_all1 = ev()
    t_all0.record()
    for _ in range(args.timesteps):
        e = [ev() for _ in range(6)]
        e[0].record()
        nxt = B.og_ts_next_tick(bins, tick, bmax, scratch)
        B.og_ts_drift(pos, vel, (nxt - tick) * dt_max / 2 ** bmax, L)
        tick = nxt
        e[1].record()
        na = B.og_ts_active_list(bins, tick, bmax, act, scratch)
        sub = act[:na]
        ao = a_old[sub.long()].contiguous()
        e[2].record()
        tree = B.og_tree_build(pos, mass, eps, L, prm)
        e[3].record()
        acc, _ = B.og_shortrange_accel(tree, sub, ao, want_pot=False)
        e[4].record()
        B.og_ts_kick(vel, bins, a_old, sub, na, acc, eps, eta, dt_max, bmax, tick, False)
        B.og_tree_free(tree)
        e[5].record()
        rows.append((tick, na, e))
    t_all1.record()
    torch.cuda.synchronize()
    per = [{"tick": t, "n_active": na, "ms_drift": e[0].elapsed_time(e[1]), "ms_active_list": e[1].elapsed_time(e[2]),
            "ms_build": e[2].elapsed_time(e[3]), "ms_walk": e[3].elapsed_time(e[4]), "ms_kick": e[4].elapsed_time(e[5])}
           for t, na, e in rows]
    total_ms = t_all0.elapsed_time(t_all1)
    updates = sum(p["n_active"] for p in per)
    line = {"mode": "timestep", "metric": "active-particle force updates/s over K hierarchical time steps (drift-all + tree "
            "rebuild + short-range walk + kick) on B200", "value": updates / (total_ms * 1e-3), "unit": "particle updates/s",
            "n_gpus": 1, "steps": args.timesteps, "ms_total": total_ms, "dtype": "f32", "data": "synthetic",
            "config": {"workload": w.name, "n": n, "eta": eta, "dt_max": dt_max, "bmax": bmax, "initial_bin_histogram": hist0},
            "per_step": per, "status": 0}
    print(json.dumps(line))
    return 0


def run_sph(args):
    """--sph N_DES (row f3): og_sph_density on the workload's particles (all of them targets), timed
    twice: cold (starting radius from the tree) and warm (h_guess = the previous answer, the regime of a running
    simulation).  Prints its own JSON line with the oracle (oracle/sph.py) timed on a bounded sample beside it."""
    import torch
    from paper_2606_17145_b200 import binding as B
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the product path has no CPU fallback)")
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(0)
    w = W.make(args.workload)
    n_des = float(args.sph)
    prm = B.make_params(w.r_s, G=w.G, rcut_over_rs=w.rcut_over_rs, alpha=w.alpha, theta=w.theta, leaf_max=8)
    pos, mass, eps = (torch.from_numpy(x).to(dev) for x in (w.pos, w.mass, w.eps))
    tree = B.og_tree_build(pos, mass, eps, w.L, prm)
    ev = lambda: torch.cuda.Event(enable_timing=True)

    def timed(guess):
        for _ in range(max(args.warmup, 1)):
            h, rho, nn = B.og_sph_density(tree, n_des, h_guess=guess)
        torch.cuda.synchronize()
        e0, e1 = ev(), ev()
        e0.record()
        for _ in range(args.steps):
            h, rho, nn = B.og_sph_density(tree, n_des, h_guess=guess)
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / args.steps, h, rho, nn

    ms_cold, h, rho, nn = timed(None)
    ms_warm, h2, _, _ = timed(h.clone())
    status = B.og_tree_status(tree)
    n_nodes = float(B.og_tree_stats(tree)["n_nodes"])
    line = {"mode": "sph_density", "metric": "SPH density + smoothing-length targets/s (neighbour walk + root of N(h) = n_des) on B200",
            "value": w.n / (ms_cold * 1e-3), "unit": "particles/s", "n_gpus": 1, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_cold, "ms_per_step_with_h_guess": ms_warm, "value_with_h_guess": w.n / (ms_warm * 1e-3),
            "higher_is_better": True, "dtype": "f32", "data": "synthetic",
            "config": {"workload": w.name, "n": w.n, "n_des": n_des, "tol_n": 0.0, "box": w.L},
            "roofline": {"bound": "hbm", "achieved": (w.n * 28.0 + n_nodes * 40.0) / (ms_cold * 1e-3) / 1e9,
                         "peak": measured_peaks()[0].get("hbm_gbs", 0.0), "unit": "GB/s",
                         "frac": (w.n * 28.0 + n_nodes * 40.0) / (ms_cold * 1e-3) / 1e9 / max(measured_peaks()[0].get("hbm_gbs", 1.0), 1.0),
                         "traffic": None, "note": "compulsory bytes only (every particle 16 B and every node's AABB + info 40 B "
                         "once, 12 B out per target; leaf_max 8): the kernel is a latency-bound walk, "
                         "one target per warp, far from either roofline (DESIGN.md Sec. 12)"},
            "checks": {"mean_N": float(nn.mean().item()), "max_abs_N_minus_n_des": float((nn - n_des).abs().max().item()),
                       "max_rel_h_warm_vs_cold": float(((h2 - h).abs() / h).max().item()), "mean_h": float(h.mean().item())},
            "status": status}
    if not args.no_cpu_baseline:
        import time
        from oracle import sph as osph
        rng = np.random.default_rng(4242)
        t = np.sort(rng.choice(w.n, size=args.sph_cpu_sample, replace=False))
        p64, m64 = w.pos.astype(np.float64), w.mass.astype(np.float64)
        t0 = time.perf_counter()
        ho, ro, no = osph.sph_density(p64, m64, w.L, n_des, targets=t)
        dt = time.perf_counter() - t0
        hg = h.cpu().numpy().astype(np.float64)[t]
        line["cpu_baseline"] = {"value": len(t) / dt, "unit": "particles/s", "cores": 1, "kind": "oracle",
                                "sample": f"oracle/sph.py on {len(t)} seeded random targets of the same workload (cKDTree build "
                                          f"included, {dt:.1f} s, 1 thread)",
                                "max_rel_h_vs_oracle_on_sample": float((np.abs(hg - ho) / ho).max())}
    B.og_tree_free(tree)
    print(json.dumps(line))
    return 0


def run_let(args):
    """--scaling let (row f4): ONE box split over the ranks by Morton ranges of whole level-5 cells;
    every step = domain decomposition (particles moved to their owners) + one tree per rank + primary walk + export of the
    targets within r_cut of another domain + secondary walk there + results sent back and summed.  Under torchrun the
    exchanges are NCCL all-to-all / all-gather (one process per GPU); with one process, --let-domains R runs the R domains
    one after the other on this GPU (no rank waits on another) and the time is the SUM over the domains: it measures the
    work the decomposition adds, not a speed-up."""
    import torch
    from paper_2606_17145_b200 import binding as B
    from paper_2606_17145_b200 import let
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the product path has no CPU fallback)")
    world, rank, local = dist_setup(args.gpus, "nccl")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    w = W.make(args.workload)
    if world > 1:
        ex, R, mine = let.DistExchange(), world, [rank]
    else:
        R = max(1, args.let_domains)
        ex, mine = let.LocalExchange(R), list(range(R))
    prm = B.make_params(w.r_s, G=w.G, rcut_over_rs=w.rcut_over_rs, alpha=w.alpha, theta=w.theta, leaf_max=8)
    prm.flags |= {"auto": 0, "32": B.OG_WALK_G32, "8": B.OG_WALK_G8}[args.walk_grouping]
    active = np.zeros(w.n, bool)
    active[np.arange(w.n) if w.active_idx is None else w.active_idx] = True

    def parts(a_old_pp):
        out = {}
        for r in mine:                                       # initial distribution: round robin over the ranks
            sel = np.arange(r, w.n, R)
            out[r] = let.Domain(*(torch.from_numpy(x[sel]).to(dev) for x in (w.pos, w.mass, w.eps)),
                                torch.from_numpy(sel.astype(np.int64)).to(dev), torch.from_numpy(active[sel]).to(dev),
                                None if a_old_pp is None else a_old_pp[torch.from_numpy(sel).to(dev)].contiguous())
        return out

    # a_old (R23 / R53): |a| of an untimed geometric pass of the same pipeline, scattered to a per-particle array
    doms, _ = let.decompose(B, parts(None), ex, w.L)
    res, _ = let.let_forces(B, doms, ex, w.L, prm, geometric=True, want_pot=False)
    a_pp = torch.zeros(w.n, device=dev)
    for r in mine:
        a_pp[doms[r].gid[doms[r].active.long()]] = torch.linalg.vector_norm(res[r][0], dim=1)
    if world > 1:
        import torch.distributed as dist
        dist.all_reduce(a_pp)
    start = parts(a_pp)
    ev = lambda: torch.cuda.Event(enable_timing=True)

    def step():
        d, _ = let.decompose(B, start, ex, w.L)
        out, info = let.let_forces(B, d, ex, w.L, prm)
        return d, out, info

    for _ in range(max(args.warmup, 1)):
        step()
    barrier(); torch.cuda.synchronize()
    e0, e1 = ev(), ev()
    e0.record()
    per_step = []
    for _ in range(args.steps):
        es = ev(); es.record()
        d, out, info = step()
        per_step.append(es)
    e1.record()
    torch.cuda.synchronize(); barrier()
    per_step = [a.elapsed_time(b) for a, b in zip(per_step, per_step[1:] + [e1])]
    ms = all_max(e0.elapsed_time(e1) / args.steps, dev)
    n_act = all_gather_int(sum(int(d[r].active.shape[0]) for r in mine), dev)
    n_loc = all_gather_int(sum(int(d[r].pos.shape[0]) for r in mine), dev)
    n_exp = all_gather_int(sum(v for (r, q), v in info["n_exported"].items() if r in mine), dev)
    chk = all_gather_int(int(sum(float(out[r][0].abs().sum().item()) for r in mine) * 1e3), dev)
    if rank == 0:
        line = {"mode": "let", "metric": "short-range tree-gravity particles/s, one box decomposed over the ranks (decomposition + "
                "tree per domain + primary walk + export / secondary walk + sum) on B200", "value": aggregate(n_act, ms),
                "unit": "particles/s", "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms,
                "higher_is_better": True, "scaling": "strong", "dtype": "f32", "data": "synthetic",
                "config": {"workload": w.name, "n": w.n, "n_active": int(active.sum()), "domains": R,
                           "walk_grouping": args.walk_grouping, "exchange": "nccl all-to-all, one process per GPU" if world > 1 else
                           f"{R} domains one after the other on one GPU (time = sum over the domains)"},
                "particles_per_domain": n_loc if world > 1 else [int(d[r].pos.shape[0]) for r in mine],
                "ms_each_step_rank0": per_step, "ms_median_step_rank0": sorted(per_step)[len(per_step) // 2], "exported_target_copies": int(sum(n_exp)), "checksum_sum_abs_acc_milli": int(sum(chk))}
        print(json.dumps(line))
    return 0


def run_pm(args):
    """--pm NG (row f1): og_pm_longrange on the workload (all particles sources and targets) with an
    NG^3 mesh and the workload's r_s.  HBM-bound: the line carries the achieved fraction of the measured copy bandwidth for
    the compulsory traffic (particles in, results out, every grid once per pass over it)."""
    import torch
    from paper_2606_17145_b200 import binding as B
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the product path has no CPU fallback)")
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(0)
    w = W.make(args.workload)
    ng = int(args.pm)
    pos, mass = torch.from_numpy(w.pos).to(dev), torch.from_numpy(w.mass).to(dev)
    pm = B.og_pm_create(ng, w.L, w.r_s, w.G)
    for _ in range(max(args.warmup, 1)):
        acc, pot = B.og_pm_longrange(pm, pos, mass)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(args.steps):
        acc, pot = B.og_pm_longrange(pm, pos, mass)
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / args.steps
    # the same particles in the tree's (Morton) order, as a code that keeps its particles along a space-filling curve
    # passes them: the mass assignment then sums the runs of particles that share a grid point inside the warp
    prm = B.make_params(w.r_s, G=w.G, rcut_over_rs=w.rcut_over_rs, alpha=w.alpha, theta=w.theta, leaf_max=8)
    tree = B.og_tree_build(pos, mass, torch.from_numpy(w.eps).to(dev), w.L, prm)
    perm = B.og_tree_get(tree, B.OG_F_PERM).long()
    pos_s, mass_s = pos[perm].contiguous(), mass[perm].contiguous()
    B.og_tree_free(tree)
    for _ in range(max(args.warmup, 1)):
        acc_s, pot_s = B.og_pm_longrange(pm, pos_s, mass_s)
    torch.cuda.synchronize()
    e0.record()
    for _ in range(args.steps):
        acc_s, pot_s = B.og_pm_longrange(pm, pos_s, mass_s)
    e1.record()
    torch.cuda.synchronize()
    ms_sorted = e0.elapsed_time(e1) / args.steps
    arms = float(torch.sqrt((acc * acc).sum(1).mean()).item())
    diff_sorted = float((acc_s - acc[perm]).abs().max().item()) / arms
    peaks, src = measured_peaks()
    g = float(ng) ** 3
    # deposit: 16 B in per particle + the mass grid written once; R2C + C2R: each grid read and written once per FFT
    # (two real grids of 4 B, one complex of ~4 B per point); Green: complex grid read + written; gradient: potential
    # read, float4 written; interpolation: 12 B position + 16 B out per target (the 8 x 16 B gathers hit L2)
    bytes_alg = w.n * 16.0 + g * 4.0 + 2.0 * (g * 4.0 + g * 4.0) + 2.0 * g * 4.0 + (g * 4.0 + g * 16.0) + w.n * 28.0
    hbm = peaks.get("hbm_gbs", 0.0)
    line = {"mode": "pm_longrange", "metric": "PM long-range force particles/s (CIC deposit + cuFFT + Green + gradient + CIC "
            "interpolation) on B200", "value": w.n / (ms * 1e-3), "unit": "particles/s", "n_gpus": 1, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms, "ms_per_step_morton_ordered_input": ms_sorted,
            "value_morton_ordered_input": w.n / (ms_sorted * 1e-3), "max_abs_acc_difference_between_the_orders_over_rms": diff_sorted,
            "higher_is_better": True, "dtype": "f32", "data": "synthetic",
            "config": {"workload": w.name, "n": w.n, "ng": ng, "r_s": w.r_s, "box": w.L},
            "roofline": {"bound": "hbm", "achieved": bytes_alg / (ms * 1e-3) / 1e9, "peak": hbm, "unit": "GB/s",
                         "frac": (bytes_alg / (ms * 1e-3) / 1e9 / hbm) if hbm else None, "traffic": None,
                         "frac_morton_ordered_input": (bytes_alg / (ms_sorted * 1e-3) / 1e9 / hbm) if hbm else None,
                         "algorithmic_bytes": bytes_alg, "peak_source": src},
            "checksum_mean_abs_acc": float(acc.abs().mean().item())}
    B.og_pm_free(pm)
    print(json.dumps(line))
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="nfw256", choices=list(W.CONFIG_NAMES))
    ap.add_argument("--cpu-sample", type=int, default=1 << 17)
    ap.add_argument("--ref-sample", type=int, default=1 << 15)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--walk-grouping", default="auto", choices=["auto", "32", "8"],
                    help="targets per warp of walks with an active list or external targets: chosen by the library (auto) "
                         "or fixed with OG_WALK_G32 / OG_WALK_G8 (standard step and --scaling let)")
    ap.add_argument("--let-domains", type=int, default=4, help="--scaling let with one process: number of domains emulated")
    ap.add_argument("--scaling", default="weak", choices=["weak", "strong", "let"],
                    help="weak (default): one independent box per GPU; strong: one box, every rank builds the tree and walks "
                         "a Morton range of the active targets (SURVEY.md Sec. 8.5)")
    ap.add_argument("--timesteps", type=int, default=0,
                    help="row f2: run this many synchronisation steps of the time-step shell instead of the standard step")
    ap.add_argument("--pm", type=int, default=0, help="row f1: time og_pm_longrange with an NG^3 mesh instead of the standard step")
    ap.add_argument("--sph", type=float, default=0.0,
                    help="row f3: time og_sph_density with this desired neighbour number instead of the standard step")
    ap.add_argument("--sph-cpu-sample", type=int, default=300)
    args = ap.parse_args()
    if args.timesteps > 0:
        return run_timesteps(args)
    if args.pm > 0:
        return run_pm(args)
    if args.sph > 0:
        return run_sph(args)
    if args.scaling == "let":
        return run_let(args)
    if args.warmup < 3:
        args.warmup = 3 if args.impl == "ours" else args.warmup
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
