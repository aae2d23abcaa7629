#!/usr/bin/env python
"""bench.py -- soft-force throughput of the B200 path (and of the CPU oracle beside it).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 3] [--impl ours|reference]

One "step" = one pass of the whole hot path (rows a1-a9 of DESIGN.md section 2) over one batch of
synthetic input: load -> bounding cube, Morton keys, radix sort, gather -> octree + groups ->
moments -> group walk + interactions -> neighbour CSR.  The default workload is BASELINE.json
configs[2] (the N = 1,048,576 Salpeter-mass Plummer sphere the metric is quoted on).

Timing: every step is bracketed by CUDA events on the stream the library launches on and ends with the
accelerations and potentials in the caller's device arrays (p3t_get_acc_pot, the "output in user order" half
of row a9); between steps the L2 is flushed by writing a 512 MiB buffer (the 16 MB input is far smaller
than the 126 MB L2) and the bodies are moved by one leapfrog step dt_soft with the returned forces (torch
ops, outside the event window), so that the walk's cost-ordered hand-out of the groups works from a
PREDICTION, as it does inside an integration; ms_per_step is the mean over the K timed steps; with N > 1
ranks each rank evaluates its own independent cluster (weak scaling, no data-path collective) and the
slowest rank's time is used.  Prints ONE JSON line on rank 0.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

FLOP_PP, FLOP_PC = 23, 65            # flops-per-interaction convention
N_SM_NOMINAL, FP32_LANES = 148, 128
METRIC = "soft-force particles/s (tree build + walk + neighbour lists, fp32)"
CLOCK_QUERY = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
               "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
               "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return dict(hbm_gbs=d["hbm_gbs"], sm_max_mhz=d.get("sm_max_mhz", 1965.0), source="measured")
    return dict(hbm_gbs=6650.0, sm_max_mhz=1965.0, source="fallback")


def algorithmic_bytes_tree(n, key_bits, n_cells, n_groups):
    """a1-a6 bytes the method must move (every array once per pass that reads or writes it)."""
    passes = 8 if key_bits == 63 else 4
    pack = 16 * n + 16 * n                        # a1: read mass+pos, write float4 bodies
    keys = 16 * n + 8 * n                         # a2: read bodies, write u64 key (the first pass makes idx = iota itself)
    sort = passes * 2 * 12 * n - 4 * n            # a3: each pass reads and writes (key, idx); pass 0 reads no idx
    gather = 4 * n + 16 * n + 16 * n + 8 * n + n  # a4: idx, body in, body out, keys -> common-prefix levels (1 B)
    build = 2 * n + 2 * n + 32 * n_cells + 4 * n_groups   # a5: c read twice, leaf level + cut flag written and read, topology, group starts
    moments = 16 * n + 88 * n_cells + 88 * n_cells  # a6: read bodies; write cells; parents re-read their children
    return dict(pack=pack, sort=keys + sort + gather, build=build, moments=moments)


class ClockSampler:
    def __init__(self, index):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        try:
            self.p = subprocess.Popen(["nvidia-smi", f"--query-gpu={CLOCK_QUERY}", "--format=csv,noheader,nounits",
                                       "-lms", "10", "-i", str(index)], stdout=self.f, stderr=subprocess.DEVNULL)
        except OSError:
            self.p = None

    def stop(self):
        out = dict(sm_mhz=None, sm_max_mhz=None, reasons=[], samples=0)
        if self.p is None:
            return out
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.p.kill()
        self.f.flush()
        rows = [r.split(",") for r in open(self.f.name).read().strip().splitlines() if r.count(",") >= 8]
        os.unlink(self.f.name)
        if not rows:
            return out
        sm = sorted(float(r[1]) for r in rows)
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [nm for k, nm in enumerate(names) if any("Active" == r[5 + k].strip() for r in rows)]
        power = max(float(r[3]) for r in rows)
        return dict(sm_mhz=sm[len(sm) // 2], sm_max_mhz=float(rows[0][2]), reasons=reasons, samples=len(rows), power_w_max=power)


def time_oracle(cfg, budget_particles):
    """The CPU oracle as it stands (O4: fp64 Barnes-Hut, same theta and acceptance rule), on a bounded sample."""
    from oracle import p3t_oracle as O

    m, q = cfg["mass"].astype(np.float64), cfg["pos"].astype(np.float64)
    n = cfg["n"]
    t0 = time.perf_counter()
    tree = O.Tree(m, q, nleaf=cfg["nleaf"], max_depth=21 if cfg["key_bits"] == 63 else 10)
    t_build = time.perf_counter() - t0
    ns = min(n, budget_particles)
    sub = np.sort(np.random.default_rng(7).choice(n, ns, replace=False)).astype(np.int64)
    t0 = time.perf_counter()
    r = tree.walk(cfg["eps"], cfg["theta"], cfg["r_in"], cfg["r_out"], cfg["r_search"], subset=sub)
    t_walk = time.perf_counter() - t0
    t_full = t_build + t_walk * n / ns
    # O2 (direct sum, the definition the tree approximates) on a small target subset, extrapolated to all N targets
    nd = min(n, max(16, int(2.5e8 // n)))
    subd = np.sort(np.random.default_rng(11).choice(n, nd, replace=False)).astype(np.int64)
    t0 = time.perf_counter()
    O.direct(m, q, cfg["eps"], cfg["r_in"], cfg["r_out"], subset=subd)
    t_direct = time.perf_counter() - t0
    direct = dict(pairs_per_s=nd * (n - 1) / t_direct, extrapolated_s_per_evaluation=t_direct * n / nd,
                  sample=f"O2 fp64 direct sum on {nd} seeded targets ({t_direct:.2f} s), scaled by N/{nd}: extrapolated")
    return dict(value=n / t_full, unit="particles/s", cores=O.num_threads(), kind="oracle",
                sample=f"O4 fp64 CPU Barnes-Hut (gcc -O2 -fopenmp): tree build over all {n} bodies ({t_build:.2f} s) + walk of "
                       f"{ns} seeded random targets ({t_walk:.2f} s), walk time scaled by N/{ns}",
                interactions_per_s=float((r["n_pp"].sum() + r["n_pc"].sum()) / t_walk), direct_sum=direct), t_build + t_walk


def run_reference(args):
    """--impl reference: the oracle timed on the host cores; rank 0 only."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    from paper_1506_04553_b200 import workloads

    cfg = workloads.config(args.config)
    times, last = [], None
    for it in range(args.warmup + args.steps):
        last, dt = time_oracle(cfg, args.ref_sample)
        if it >= args.warmup:
            times.append(cfg["n"] / last["value"])
    t = float(np.mean(times))
    value = cfg["n"] / t
    cb = dict(last); cb["value"] = value
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": "particles/s", "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * t, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": cfg["name"], "n": cfg["n"], "theta": cfg["theta"], "note": "each step = one bounded sample, extrapolated to N"},
        "cpu_baseline": cb,
        "e2e": {"value": value, "unit": "particles/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--config", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--ref-sample", type=int, default=131072, help="targets walked by the oracle per step")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--nleaf", type=int, default=None)
    ap.add_argument("--ngroup", type=int, default=None)
    ap.add_argument("--merge", type=int, default=None)
    ap.add_argument("--curve", default=None, choices=["morton", "hilbert"], help="p3t_set_key_curve (default: the library's, hilbert)")
    ap.add_argument("--sort-passes", type=int, default=0, help="p3t_set_sort_passes (default 0: the library's plan)")
    ap.add_argument("--shard", action="store_true",
                    help="strong scaling: ONE cluster, every rank walks every world-th i-group (p3t_set_shard) and the "
                         "accelerations and potentials are summed over the ranks (NCCL all-reduce inside the timed step)")
    ap.add_argument("--walk-mode", type=int, default=None, help="p3t_set_walk_mode: 0 auto, 1 warp per group, 2 CTA per group")
    ap.add_argument("--n", type=int, default=None, help="override the particle count (not a bench value)")
    ap.add_argument("--same-positions", action="store_true", help="do not move the bodies between steps (not the headline case)")
    ap.add_argument("--settle", type=float, default=1.2, help="seconds of untimed steps before the warm-up (clock sampler)")
    ap.add_argument("--dt-soft", type=float, default=None, help="soft step of the drift between timed steps (default: the config's, else 1/1024)")
    ap.add_argument("--refit", type=int, default=0, help="tree reuse: p3t_refit_tree with a rebuild every REFIT calls (not the headline case)")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    args.warmup = max(args.warmup, 3)

    import torch

    from paper_1506_04553_b200 import binding, workloads

    rank, world = int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the soft-force path has no CPU fallback")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local}"))

    from paper_1506_04553_b200 import multi

    shard = args.shard and world > 1
    # default: an independent cluster per rank (same recipe, another seed); --shard: the same cluster on every rank
    cfg = multi.rank_config(args.config, 0 if shard else rank, n=args.n)
    n = cfg["n"]
    nleaf, ngroup = args.nleaf or cfg["nleaf"], args.ngroup or cfg["ngroup"]
    dev = f"cuda:{local}"
    mass_d = torch.from_numpy(cfg["mass"]).to(dev)
    pos_d = torch.from_numpy(cfg["pos"]).to(dev)
    flush = torch.empty(512 << 20, dtype=torch.uint8, device=dev)

    ctx = binding.P3T(n, key_bits=cfg["key_bits"], nbr_capacity=max(n, 1 << 16), device=local)
    ctx.set_params(cfg["eps"], cfg["theta"], cfg["r_in"], cfg["r_out"], cfg["r_search"])
    ctx.set_tree_params(nleaf, ngroup)
    if args.curve is not None:
        ctx.set_key_curve(args.curve)
    if args.sort_passes:
        ctx.set_sort_passes(args.sort_passes)
    if args.merge is not None:
        ctx.set_group_merge_levels(args.merge)
    if args.walk_mode is not None:
        ctx.set_walk_mode(args.walk_mode)

    if shard:
        ctx.set_shard(rank, world)
    acc_d = torch.empty((n, 3), dtype=torch.float32, device=dev)
    pot_d = torch.empty(n, dtype=torch.float32, device=dev)
    rec_d = torch.empty((n, 5), dtype=torch.float32, device=dev) if shard else None
    if args.refit:
        ctx.set_tree_reuse(args.refit)

    def step():
        ctx.load_particles(mass_d, pos_d)
        if args.refit:
            ctx.refit_tree()           # rebuilds by itself every args.refit calls or when too many bodies have strayed
        else:
            ctx.build_tree()
        ctx.eval_soft()
        if shard:      # every rank ends the step with the accelerations and potentials of all particles: one all-reduce
            multi.allreduce_shard(dist, ctx, rec_d)
        else:
            ctx.get_acc_pot_into(acc_d, pot_d)   # a9: accelerations and potentials in user order, in the caller's arrays

    # Between steps the bodies move by one leapfrog step with the returned forces (BASELINE.json configs[1] asks for it
    # in so many words: "positions are drifted by a leapfrog step dt_soft using the returned forces"; for the other
    # configs it makes the timed case the one an integration sees).  Torch ops on the device, outside the event window.
    dt_soft = args.dt_soft or cfg.get("dt_soft") or 1.0 / 1024.0
    drift = not shard and not args.same_positions
    vel_l = torch.from_numpy(cfg["vel"]).to(dev)
    pos_d = pos_d.clone()

    def move():
        if drift:
            vel_l.add_(acc_d, alpha=dt_soft)
            pos_d.add_(vel_l, alpha=dt_soft)

    # The clock sampler (nvidia-smi every 10 ms; its first sample takes a few hundred ms) runs from here to the end of
    # the timed region.  Small configs finish W + K steps before it delivers ten samples, so the same step first runs
    # untimed until 1.2 s have passed (same load as the timed steps), then the W warm-up steps, then the K timed ones.
    sampler = ClockSampler(local) if rank == 0 else None
    settle_steps, t_settle = 0, time.perf_counter()
    while time.perf_counter() - t_settle < args.settle:
        step()
        ctx.synchronize()
        settle_steps += 1
    for _ in range(args.warmup):
        flush.zero_()
        step()
        move()
    ctx.synchronize()
    if dist:
        dist.barrier()
    torch.cuda.synchronize()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    phases = {k: [] for k in ("ms_pack", "ms_sort", "ms_build", "ms_moments", "ms_walk", "ms_nbr")}
    for a, b in ev:
        flush.zero_()
        a.record()
        step()
        b.record()
        st = ctx.get_stats()           # synchronises; per-phase times come from the library's own CUDA events
        for k in phases:
            phases[k].append(st[k])
        move()
    torch.cuda.synchronize()
    if dist:
        dist.barrier()
    clocks = sampler.stop() if sampler else None
    total_n, ms = multi.aggregate(dist, n, float(np.mean([a.elapsed_time(b) for a, b in ev])), device=dev)
    if shard:
        total_n = n      # one cluster, not one per rank
    st = ctx.get_stats()
    ph = {k: float(np.mean(v)) for k, v in phases.items()}
    # secondary key: the same step with the positions of the last timed step repeated (the group order is then a
    # perfect prediction: the favourable case round 1 quoted)
    same_ms = None
    if drift and rank == 0:
        ts = []
        for _ in range(1 + min(args.steps, 5)):
            flush.zero_()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(); step(); e1.record()
            torch.cuda.synchronize()
            ts.append((e0.elapsed_time(e1), ctx.get_stats()["ms_walk"]))
        same_ms = {"ms_per_step": float(np.mean([t[0] for t in ts[1:]])), "ms_walk": float(np.mean([t[1] for t in ts[1:]]))}
    ffma_scalar = ffma_packed = None
    nbr_hist = None
    if rank == 0:      # neighbour-list length histogram of the last step (BASELINE.json config 4 asks for it)
        cnt, _ = ctx.get_neighbour_counts()
        hh = np.bincount(np.minimum(cnt, 16), minlength=17)
        nbr_hist = {"length_0..15_and_16+": [int(x) for x in hh], "max": int(cnt.max()), "mean": float(cnt.mean())}
    tree_hist = None
    if rank == 0:      # depth / leaf-occupancy histograms of the last tree
        meta, lev = ctx.array("cell_meta"), ctx.array("cell_level")
        leaf = (meta[:, 1] & 0x80000000) != 0
        occ = (meta[leaf, 1] & 0x7fffffff).astype(np.int64)
        tree_hist = {"leaves_per_level": [int(x) for x in np.bincount(lev[leaf], minlength=st["depth"] + 1)],
                     "cells_per_level": [int(x) for x in np.bincount(lev, minlength=st["depth"] + 1)],
                     "leaf_occupancy_1..nleaf_and_above": [int(x) for x in np.bincount(np.minimum(occ, nleaf + 1), minlength=nleaf + 2)[1:]],
                     "bodies_per_leaf_level": [int(x) for x in np.bincount(lev[leaf], weights=occ, minlength=st["depth"] + 1)],
                     "mean_leaf_occupancy": float(occ.mean()), "max_leaf_occupancy": int(occ.max())}
    if rank == 0:      # pure-FFMA calibration kernel, outside the timed region
        ffma_scalar, ffma_packed = ctx.measure_fp32_peak(False)[0], ctx.measure_fp32_peak(True)[0]

    # ---- NEXT row, outside the timed region: hard force over the neighbour lists of the last step
    hard = None
    if rank == 0:
        vel_d = torch.from_numpy(cfg["vel"]).to(dev)
        ah = torch.empty((n, 3), dtype=torch.float64, device=dev); jh = torch.empty_like(ah)
        ph_ = torch.empty(n, dtype=torch.float64, device=dev)
        th = []
        for _ in range(5):
            flush.zero_()
            ctx.eval_hard(vel_d, ah, jh, ph_)
            th.append(ctx.get_stats()["ms_hard"])
        ms_h = float(np.median(th[1:]))
        hb = n * (16 + 12 + 8 + 56) + st["n_neighbours"] * (4 + 16 + 12)      # own body, velocity, offsets, outputs; per pair idx, body, velocity
        hard = {"kernel": "hard_kernel (p3t_eval_hard: acceleration, jerk, potential over the neighbour lists, fp64)", "ms": ms_h,
                "pairs": st["n_neighbours"], "bound": "hbm", "algorithmic_bytes": hb, "achieved": hb / (ms_h * 1e-3) / 1e9, "unit": "GB/s"}

    # ---- NEXT row (rank 2), outside the timed region: whole steps of the scheme on a device-resident fp64 state
    # (kick, Hermite part by neighbour cluster / drift, soft force at the new time, kick; p3t_step)
    whole = None
    if rank == 0 and not shard:
        dt_soft = cfg.get("dt_soft") or 1.0 / 1024.0
        a0 = 0.1 * float(cfg["mass"].mean()) / cfg["r_out"] ** 2           # Eq. 19, alpha = 0.1 (L160)
        q64 = torch.from_numpy(cfg["pos"].astype(np.float64)).to(dev)
        v64 = torch.from_numpy(cfg["vel"].astype(np.float64)).to(dev)
        ctx.load_particles(mass_d, torch.from_numpy(cfg["pos"]).to(dev)); ctx.build_tree(); ctx.eval_soft()
        tw, infos = [], []
        for _ in range(6):
            flush.zero_()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            infos.append(ctx.step(mass_d, q64, v64, dt_soft, log2_div=2, eta=0.1, eta_s=0.01, a0=a0))
            e1.record()
            torch.cuda.synchronize()
            tw.append(e0.elapsed_time(e1))
        ms_w = float(np.median(tw[1:]))
        last = infos[-1]
        whole = {"call": "p3t_step (device-resident fp64 state)", "dt_soft": dt_soft, "ms_per_step": ms_w,
                 "particles_per_s": n / (ms_w * 1e-3), "ms_hermite": float(np.median([i["ms"] for i in infos[1:]])),
                 "nonisolated": last["n_nonisolated"], "hermite_steps": last["n_steps"], "clusters": last["n_components"],
                 "largest_cluster": last["max_component"], "blocks_of_busiest_cluster": last["n_blocks"]}

    # ---- end to end through the C ABI with HOST buffers (pinned), copies inside the timed region
    e2e = None
    if not args.no_e2e:
        mass_h = torch.from_numpy(cfg["mass"]).pin_memory().numpy()
        pos_h = torch.from_numpy(cfg["pos"]).pin_memory().numpy()
        acc_h = torch.empty((n, 3), dtype=torch.float32).pin_memory().numpy()
        pot_h = torch.empty(n, dtype=torch.float32).pin_memory().numpy()
        off_h = torch.empty(n + 1, dtype=torch.uint64).pin_memory().numpy()
        nbr_h = torch.empty(ctx.nbr_capacity, dtype=torch.int32).pin_memory().numpy().view(np.uint32)
        ts, d2h = [], 0
        for it in range(2 + min(args.steps, 5)):
            flush.zero_()
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            ctx.load_particles(mass_h, pos_h)
            ctx.build_tree()
            ctx.eval_soft()
            ctx.get_acc_pot_into(acc_h, pot_h)
            total = ctx.get_neighbours_into(off_h, nbr_h)
            dt = time.perf_counter() - t0
            d2h = acc_h.nbytes + pot_h.nbytes + off_h.nbytes + 4 * total
            if it >= 2:
                ts.append(dt)
        _, te_ms = multi.aggregate(dist, n, 1e3 * float(np.mean(ts)), device=dev)
        te = 1e-3 * te_ms
        e2e = {"value": total_n / te, "unit": "particles/s", "h2d_bytes_per_step": int(mass_h.nbytes + pos_h.nbytes),
               "d2h_bytes_per_step": int(d2h), "ms_per_step": 1e3 * te}

    if rank != 0:
        if dist:
            dist.destroy_process_group()
        return

    peaks = measured_peaks()
    # DRAM traffic of the dominant kernel per launch: from the committed ncu --set full capture of this workload
    traffic, traffic_src = None, None
    tp = os.path.join(ROOT, "profiles", "walk_kernel_dram_r2.csv")
    if os.path.exists(tp):
        import csv
        for row in csv.DictReader(open(tp)):
            if row["workload"] == cfg["name"]:
                traffic = int(row["dram_bytes_read"]) + int(row["dram_bytes_write"])
                traffic_src = "profiles/walk_kernel_dram_r2.csv (ncu --set full, dram__bytes_read.sum + dram__bytes_write.sum, per launch)"
    n_sm = torch.cuda.get_device_properties(local).multi_processor_count
    fp32_peak = 2 * FP32_LANES * n_sm * peaks["sm_max_mhz"] * 1e6 / 1e12          # TFLOP/s at the max SM clock
    flops = FLOP_PP * st["n_pp"] + FLOP_PC * st["n_pc"]
    walk_tflops = flops / (ph["ms_walk"] * 1e-3) / 1e12
    ab = algorithmic_bytes_tree(n, cfg["key_bits"], st["n_cells"], st["n_groups"])
    hbm = {k: ab[k] / (ph["ms_" + k] * 1e-3) / 1e9 for k in ab}
    tree_ms = ph["ms_pack"] + ph["ms_sort"] + ph["ms_build"] + ph["ms_moments"]
    # pack | keys+hist, onesweep passes, gather | levels, emit | moments (leaves, internal) | group prediction + order, walk | neighbour CSR (6)
    launches = 1 + (1 + st["sort_passes"] + (2 if st["sort_passes"] < (8 if cfg["key_bits"] == 63 else 4) else 0) + 1) + 2 + 2 + 3 + 6 + (2 if shard else 1)      # ... group prediction, order, walk; a9; unpack (sharded: record + class kernels)
    launches += 1 if st["walk_parts"] > 1 else 0                                              # split walk: the combine kernel

    out = {
        "metric": METRIC, "value": multi.throughput(total_n, ms), "unit": "particles/s", "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "strong" if shard else "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic",
        "config": {"workload": cfg["name"], "n": n, "theta": cfg["theta"], "eps": cfg["eps"], "r_out": cfg["r_out"],
                   "r_search": cfg["r_search"], "key_bits": cfg["key_bits"], "nleaf": nleaf, "ngroup": ngroup,
                   "l2": "flushed between steps (512 MiB write)", "positions": f"drifted between steps (leapfrog with the returned forces, dt_soft = 1/{round(1 / dt_soft)})" if drift else "same every step",
                   "timed_region": "load_particles + build_tree + eval_soft + get_acc_pot (device arrays)", "clock_settle_steps": settle_steps, "parallelism": (f"one cluster sharded over {world} GPUs by i-groups, all-reduce of the results" if shard
                                   else f"{world} independent cluster(s), one per GPU")},
        "interactions_per_s": (st["n_pp"] + st["n_pc"]) / (ph["ms_walk"] * 1e-3),
        "walk_particles_per_s": n / (ph["ms_walk"] * 1e-3),
        "interactions": {"n_pp": st["n_pp"], "n_pc": st["n_pc"], "n_near": st["n_near"], "n_neighbours": st["n_neighbours"],
                         "pp_per_particle": st["n_pp"] / n, "pc_per_particle": st["n_pc"] / n},
        "walk_parts": st["walk_parts"], "sort_passes": st["sort_passes"], "sort_max_run": st["sort_max_run"], "tree": {"n_cells": st["n_cells"], "n_leaves": st["n_leaves"], "n_groups": st["n_groups"], "depth": st["depth"], "histograms": tree_hist},
        "same_positions": same_ms,
        "neighbour_lists": nbr_hist, "workspace_bytes": int(ctx.workspace.numel()),
        "phases_ms": ph,
        "roofline": {"bound": "alu", "kernel": "walk_kernel (a7+a8)", "achieved": walk_tflops, "peak": fp32_peak, "unit": "TFLOP/s",
                     "frac": walk_tflops / fp32_peak, "traffic": None, "traffic_committed_capture": traffic, "traffic_source": traffic_src,
                     "peak_source": f"2 flop x {FP32_LANES} lanes x {n_sm} SMs x {peaks['sm_max_mhz']:.0f} MHz ({peaks['source']} sm_max_mhz; DESIGN.md section 8)",
                     "convention": f"{FLOP_PP} flop per p-p, {FLOP_PC} flop per p-c",
                     "ffma_microbench_tflops": {"scalar": ffma_scalar, "packed": ffma_packed},
                     "frac_of_ffma_microbench": walk_tflops / max(ffma_scalar, ffma_packed)},
        "roofline_hbm": {"bound": "hbm", "passes": "a1-a6 (sort, build, moments)", "achieved": sum(ab.values()) / (tree_ms * 1e-3) / 1e9,
                         "peak": peaks["hbm_gbs"], "unit": "GB/s", "frac": sum(ab.values()) / (tree_ms * 1e-3) / 1e9 / peaks["hbm_gbs"],
                         "per_pass_gbs": hbm, "algorithmic_bytes": ab, "peak_source": peaks["source"],
                         # the byte count is SURVEY.md 8(d)'s (an LSD sort of all digits); the build sorts the upper digits by
                         # radix passes and finishes short runs in place (p3t_set_sort_passes), so it MOVES less than it is booked for
                         "radix_passes_booked": 8 if cfg["key_bits"] == 63 else 4, "radix_passes_run": st["sort_passes"],
                         "moved_gbs": (sum(ab.values()) - (((8 if cfg["key_bits"] == 63 else 4) - st["sort_passes"]) * 24 * n)) / (tree_ms * 1e-3) / 1e9},
        "tree_reuse": ({"max_refits": args.refit, "tree_refits_at_end": st["tree_refits"], "n_stray": st["n_stray"]} if args.refit else None),
        "clocks": clocks, "gpu_launches": launches * args.steps, "gpu_launches_per_step": launches,
    }
    if hard:
        hard["peak"] = peaks["hbm_gbs"]; hard["frac"] = hard["achieved"] / peaks["hbm_gbs"]
        out["next_rows"] = {"hard_force": hard}
        if whole:
            out["next_rows"]["p3t_step"] = whole
    if e2e:
        out["e2e"] = e2e
    if not args.no_cpu_baseline and world == 1:
        out["cpu_baseline"], _ = time_oracle(cfg, args.ref_sample)
    print(json.dumps(out))
    if dist:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
