"""GPU parity of the hard-force row (include/p3t.h p3t_eval_hard) against oracle O6.

The GPU sums over the neighbour lists it produced itself (s_ij < h), the oracle over all pairs: equal because
1 - K = 1 - W = 0 beyond r_out <= h (Eq. 7, Eq. 12, Eq. 16).  Both evaluate every pair in fp64 from the same
fp32 inputs.  Tolerance 1e-7 relative per particle: 1 - K and 1 - W are differences of O(1) numbers, so for a
pair just inside r_out (1 - K ~ 1e-8) the two evaluation orders (Horner on the GPU, term by term in the oracle)
differ by ~1e-16 / (1 - K); everywhere else the agreement is ~1e-13 (checked on the median).
"""
import numpy as np
import pytest

from paper_1506_04553_b200 import workloads

pytestmark = pytest.mark.gpu


def _binding():
    from paper_1506_04553_b200 import binding
    return binding


def _compare(oracle, cfg, radii, subset=None, on_device=False):
    b = _binding()
    r_in, r_out, h = (float(np.float32(r)) for r in radii)      # what the C ABI receives (fp32 parameters)
    n = cfg["n"]
    m, q, v = (cfg[k].astype(np.float64) for k in ("mass", "pos", "vel"))
    with b.P3T(n, key_bits=63, nbr_capacity=max(64 * n, 1 << 16)) as ctx:
        ctx.set_params(cfg["eps"], cfg["theta"], r_in, r_out, h)
        ctx.soft_force(cfg["mass"], cfg["pos"])
        if on_device:
            import torch
            vd = torch.from_numpy(cfg["vel"]).cuda()
            a = torch.empty((n, 3), dtype=torch.float64, device="cuda"); j = torch.empty_like(a)
            p = torch.empty(n, dtype=torch.float64, device="cuda")
            ctx.eval_hard(vd, a, j, p)
            ctx.synchronize()
            a, j, p = a.cpu().numpy(), j.cpu().numpy(), p.cpu().numpy()
        else:
            a, j, p = ctx.eval_hard(cfg["vel"])
        st = ctx.get_stats()
        off, nbr = ctx.get_neighbours()
    sub = np.arange(n) if subset is None else subset
    ao, jo, po = oracle.hard(m, q, v, cfg["eps"], r_in, r_out, subset=None if subset is None else sub)
    nz = np.linalg.norm(ao, axis=1) > 0
    assert nz.sum() > 0                                     # the case does exercise the hard part
    # scale: magnitudes are set by the closest pair of each particle; compare against the particle's own norm
    for g, o in ((a[sub], ao), (j[sub], jo)):
        num = np.linalg.norm(g - o, axis=1)
        den = np.linalg.norm(o, axis=1)
        assert np.all(num[~nz] == 0)
        # a particle whose only neighbours sit at the very edge of the cutoff (1 - K ~ 1e-14) has a hard force many
        # orders below the typical one, made of rounding: its error is measured against 1e-6 of the typical force
        den = np.maximum(den, 1e-6 * np.median(den[nz]))
        assert (num[nz] / den[nz]).max() <= 1e-7 and np.median(num[nz] / den[nz]) <= 1e-12, (num[nz] / den[nz]).max()
    pden = np.maximum(np.abs(po), 1e-6 * np.median(np.abs(po[nz])))
    assert np.all(p[sub][~nz] == 0) and (np.abs(p[sub] - po)[nz] / pden[nz]).max() <= 1e-7
    # particles without neighbours inside r_out feel no hard force at all
    cnt = np.diff(off.astype(np.int64))
    assert np.all(np.linalg.norm(a[cnt == 0], axis=1) == 0)
    return st


def test_hard_force_config1_stress_radii_all_particles(oracle):
    cfg = workloads.config(1)
    st = _compare(oracle, cfg, (0.01, 0.1, 0.12))           # mean list length ~6: thousands of pairs inside r_out
    assert st["ms_hard"] > 0


def test_hard_force_device_pointers_and_ragged_size(oracle):
    cfg = workloads.config(2, n=3001)
    _compare(oracle, cfg, (0.02, 0.2, 0.2), on_device=True)  # r_search = r_out: every listed pair is inside the cutoff


def test_hard_force_headline_workload_on_a_subset(oracle):
    cfg = workloads.config(3)
    sub = np.sort(np.random.default_rng(3).choice(cfg["n"], 4096, replace=False)).astype(np.int64)
    # the 4096 targets with the most massive close neighbours are not in a random subset: add the listed ones
    _compare(oracle, cfg, (cfg["r_in"], cfg["r_out"], cfg["r_search"]), subset=sub)


def test_hard_force_call_order_and_capacity():
    b = _binding()
    cfg = workloads.config(1, n=2048)
    with b.P3T(2048, key_bits=63, nbr_capacity=16) as ctx:
        ctx.set_params(cfg["eps"], cfg["theta"], 0.01, 0.1, 0.12)
        ctx.load_particles(cfg["mass"], cfg["pos"])
        with pytest.raises(b.P3TError) as e:
            ctx.eval_hard(cfg["vel"])
        assert e.value.status == b.ESTATE
        ctx.build_tree(); ctx.eval_soft()
        with pytest.raises(b.P3TError) as e:
            ctx.eval_hard(cfg["vel"])                       # lists need more than 16 entries
        assert e.value.status == b.ECAPACITY
        bad = cfg["vel"].copy(); bad[5, 0] = np.nan
        with pytest.raises(b.P3TError) as e:
            ctx.eval_hard(bad)
        assert e.value.status == b.EINVAL
        # device form: the call only enqueues; the overflow (nothing was computed) surfaces at the next synchronising call
        import torch
        vd = torch.from_numpy(cfg["vel"]).cuda()
        ad = torch.full((2048, 3), 7.0, dtype=torch.float64, device="cuda")
        ctx.eval_hard(vd, ad, None, None)
        with pytest.raises(b.P3TError) as e:
            ctx.synchronize()
        assert e.value.status == b.ECAPACITY
        assert float(ad.min()) == 7.0                       # untouched
        ctx.synchronize()                                   # reported once; the context stays usable
