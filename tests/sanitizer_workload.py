"""Workload that compute-sanitizer runs over.

    compute-sanitizer --tool memcheck|racecheck|synccheck|initcheck python tests/sanitizer_workload.py [case ...]

Every case goes through the C ABI at config-1 size (N = 4096 Plummer, plus a ragged size) so that one run under
the sanitizer takes minutes: the hot path a1-a9 with the workload radii and the stress radii, both key widths, i-groups
of 32 and 64, both walk modes, the brute-force entry, the hard force, the Hermite part in all three tiers, the whole
step of the scheme, and the tree refit.  No arithmetic is checked here (the parity tests do that); the script only has
to exercise every kernel.  Results are summarised in profiles/sanitizer_r2.md.
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_1506_04553_b200 import binding, workloads  # noqa: E402


def soft(n, key_bits, ngroup, mode, stress, nleaf=16):
    cfg = workloads.config(1, n=n)
    r_in, r_out, h = (0.01, 0.1, 0.12) if stress else (cfg["r_in"], cfg["r_out"], cfg["r_search"])
    with binding.P3T(n, key_bits=key_bits, nbr_capacity=max(64 * n, 1 << 16)) as ctx:
        ctx.set_params(cfg["eps"], cfg["theta"], r_in, r_out, h)
        ctx.set_tree_params(nleaf, ngroup)
        ctx.set_walk_mode(mode)
        for _ in range(2):                       # second call: the cost-ordered hand-out of the groups
            ctx.soft_force(cfg["mass"], cfg["pos"])
        ctx.get_acc_pot()
        ctx.get_neighbour_counts()
        off, nbr = ctx.get_neighbours()
        st = ctx.get_stats()
    return st["n_pp"], st["n_pc"], int(off[-1])


def direct_and_hard(n):
    cfg = workloads.config(1, n=n)
    with binding.P3T(n, key_bits=63, nbr_capacity=64 * n) as ctx:
        ctx.set_params(cfg["eps"], cfg["theta"], 0.01, 0.1, 0.12)
        ctx.load_particles(cfg["mass"], cfg["pos"])
        ctx.eval_direct()
        ctx.get_acc_pot()
        ctx.eval_direct(np.arange(0, n, 7, dtype=np.uint32))
        ctx.soft_force(cfg["mass"], cfg["pos"])
        a, j, p = ctx.eval_hard(cfg["vel"])
        ctx.get_neighbours()
    return float(np.abs(a).max())


def hermite(n, cluster_max, r_out):
    cfg = workloads.config(1, n=n)
    a0 = 0.1 * float(cfg["mass"].mean()) / r_out ** 2
    with binding.P3T(n, key_bits=63, nbr_capacity=256 * n) as ctx:
        ctx.set_params(cfg["eps"], cfg["theta"], 0.1 * r_out, r_out, 1.2 * r_out)
        ctx.soft_force(cfg["mass"], cfg["pos"])
        if cluster_max:
            ctx.set_hermite_cluster_max(cluster_max)
        q, v = cfg["pos"].astype(np.float64), cfg["vel"].astype(np.float64)
        info = ctx.hermite_step(q, v, 1.0 / 512, a0=a0)
    return info["n_components"], info["max_component"], info["n_steps"]


def whole_step(n):
    cfg = workloads.config(1, n=n)
    r_out = 0.05
    a0 = 0.1 * float(cfg["mass"].mean()) / r_out ** 2
    with binding.P3T(n, key_bits=63, nbr_capacity=64 * n) as ctx:
        ctx.set_params(cfg["eps"], cfg["theta"], 0.1 * r_out, r_out, 1.2 * r_out)
        ctx.soft_force(cfg["mass"], cfg["pos"])
        q, v = cfg["pos"].astype(np.float64), cfg["vel"].astype(np.float64)
        for _ in range(2):
            info = ctx.step(cfg["mass"], q, v, 1.0 / 512, a0=a0)
    return info["n_steps"]


def refit(n):
    if not hasattr(binding.P3T, "refit_tree"):
        return "not built"
    cfg = workloads.config(1, n=n)
    with binding.P3T(n, key_bits=63, nbr_capacity=64 * n) as ctx:
        ctx.set_params(cfg["eps"], cfg["theta"], 0.01, 0.1, 0.12)
        ctx.soft_force(cfg["mass"], cfg["pos"])
        pos = cfg["pos"] + np.float32(1.0 / 1024) * cfg["vel"]
        ctx.load_particles(cfg["mass"], pos)
        ctx.refit_tree()
        ctx.eval_soft()
        ctx.get_acc_pot()
        off, nbr = ctx.get_neighbours()
    return int(off[-1])


def classes(n):
    if not hasattr(binding.P3T, "set_pair_classes"):
        return "not built"
    cfg = workloads.config(6, n=n)
    with binding.P3T(cfg["n"], key_bits=63, nbr_capacity=64 * cfg["n"]) as ctx:
        ctx.set_params(cfg["eps"], cfg["theta"], cfg["r_in"], cfg["r_out"], cfg["r_search"])
        ctx.set_pair_classes(cfg["classes"], **cfg["class_params"])
        ctx.soft_force(cfg["mass"], cfg["pos"])
        ctx.get_acc_pot()
        off, nbr = ctx.get_neighbours()
        ctx.eval_hard(cfg["vel"])
        ctx.set_hermite_class_params(0.03, 0.003, 0.1 * 0.01 / cfg["class_params"]["r_out_bf"] ** 2)
        q, v = cfg["pos"].astype(np.float64), cfg["vel"].astype(np.float64)
        ctx.step(cfg["mass"], q, v, cfg["dt_soft"], a0=0.1 * float(cfg["mass"][0]) / cfg["r_out"] ** 2)
    return int(off[-1])


CASES = {
    "soft63_g64_warp": lambda: soft(4096, 63, 64, 1, False),
    "soft30_g32_warp": lambda: soft(4096, 30, 32, 1, False),
    "soft63_g64_coop_stress": lambda: soft(4096, 63, 64, 2, True),
    "soft30_g32_coop_stress": lambda: soft(4096, 30, 32, 2, True),
    "soft63_g32_warp_stress_ragged": lambda: soft(4099, 63, 32, 1, True, nleaf=8),
    "soft63_auto_tiny": lambda: soft(37, 63, 64, 0, True),
    "soft63_g64_split4_stress": lambda: soft(4096, 63, 64, 4, True),
    "soft30_g32_split2": lambda: soft(4099, 30, 32, 3, False),
    "direct_and_hard": lambda: direct_and_hard(4096),
    "hermite_warp": lambda: hermite(4096, None, 0.01),
    "hermite_cluster": lambda: hermite(4096, 4096, 0.08),
    "hermite_grid": lambda: hermite(4096, 100, 0.08),
    "whole_step": lambda: whole_step(4096),
    "refit": lambda: refit(4096),
    "classes": lambda: classes(4096),
}


if __name__ == "__main__":
    names = sys.argv[1:] or list(CASES)
    for name in names:
        print(name, CASES[name](), flush=True)
    print("sanitizer workload done:", len(names), "cases")
