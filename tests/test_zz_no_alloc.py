"""p3t_direct_static (include/p3t.h): the allocation-free brute-force entry point against the existing path.

Collected last on purpose (the name sorts behind every other test file): the suite runs with `pytest -x`, and a failure
here must not hide the tests of the hot path.

The existing path is p3t_eval_direct on a context (workspace in caller memory); the new one keeps its scratch in a static
device array of the library.  Both evaluate the same fp32 pair terms in the same order, so the results should agree to
rounding; the bound is the tolerance of the theta = 0 parity tests (1e-5 of the particle's force, floored by the typical
force).  Two calls in a row on the shared array, the second with fewer particles and other parameters: nothing of the
first call may leak into it.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def _case(seed, n):
    rng = np.random.default_rng(seed)
    u = rng.uniform(1e-6, 1.0 - 1e-6, n)
    r = 0.2 / np.sqrt(u ** (-2.0 / 3.0) - 1.0)                       # centrally concentrated: real neighbour lists
    d = rng.normal(size=(n, 3))
    pos = np.clip(r[:, None] * d / np.linalg.norm(d, axis=1)[:, None], -20.0, 20.0).astype(np.float32)
    mass = (rng.uniform(0.2, 1.8, n) / n).astype(np.float32)
    return np.ascontiguousarray(mass), np.ascontiguousarray(pos)


def _existing_path(mass, pos, eps, r_in, r_out, h):
    from paper_1506_04553_b200 import binding

    with binding.P3T(len(mass), key_bits=63, nbr_capacity=1 << 22) as ctx:
        ctx.set_params(eps, 0.4, r_in, r_out, h)
        ctx.load_particles(mass, pos)
        ctx.eval_direct()
        acc, pot = ctx.get_acc_pot()
        counts, total = ctx.get_neighbour_counts()
    return acc, pot, counts, total


def _static_path(mass, pos, eps, r_in, r_out, h):
    import torch

    from paper_1506_04553_b200 import binding

    n = len(mass)
    dev = "cuda:0"
    m, q = torch.from_numpy(mass).to(dev), torch.from_numpy(pos).to(dev)
    # outputs start as garbage: whatever comes back was written by the call
    acc = torch.full((n, 3), float("nan"), dtype=torch.float32, device=dev)
    pot = torch.full((n,), float("nan"), dtype=torch.float32, device=dev)
    cnt = torch.full((n,), -1, dtype=torch.int32, device=dev)
    info = torch.full((2,), -1, dtype=torch.int64, device=dev)
    binding.direct_static(m, q, eps, r_in, r_out, h, acc, pot, cnt, info)
    torch.cuda.synchronize()
    return acc.cpu().numpy(), pot.cpu().numpy(), cnt.cpu().numpy().astype(np.uint32), info.cpu().numpy()


def _compare(a, b, what):
    acc0, pot0, cnt0, total0 = a
    acc1, pot1, cnt1, info1 = b
    assert np.all(np.isfinite(acc1)) and np.all(np.isfinite(pot1)), what
    an = np.linalg.norm(acc0.astype(np.float64), axis=1)
    err = np.linalg.norm(acc1.astype(np.float64) - acc0, axis=1) / np.maximum(an, np.median(an))
    perr = np.abs(pot1.astype(np.float64) - pot0) / np.maximum(np.abs(pot0), np.median(np.abs(pot0)))
    assert err.max() <= 1e-5 and perr.max() <= 1e-5, (what, err.max(), perr.max())
    assert np.array_equal(cnt1, cnt0), what
    assert int(info1[0]) == int(total0) == int(cnt0.sum()) and int(info1[1]) == 0, (what, info1, total0)
    assert total0 > 0, "the case should have neighbours"


def test_static_scratch_entry_point_matches_the_context_path_on_two_calls_in_a_row():
    first = (_case(11, 6001), (1e-4, 2e-3, 2e-2, 2.5e-2))
    second = (_case(12, 2500), (3e-4, 0.0, 3e-2, 3e-2))        # fewer bodies, other radii: stale bodies and counters must not matter
    for k, ((mass, pos), prm) in enumerate((first, second)):
        got = _static_path(mass, pos, *prm)
        ref = _existing_path(mass, pos, *prm)
        _compare(ref, got, f"call {k + 1}")
    # and the first case again, straight after the smaller one
    (mass, pos), prm = first
    _compare(_existing_path(mass, pos, *prm), _static_path(mass, pos, *prm), "call 3")


def test_static_scratch_entry_point_rejects_what_it_cannot_hold():
    import torch

    from paper_1506_04553_b200 import binding

    n = binding.STATIC_MAX_N + 1
    z = torch.zeros(3 * n, dtype=torch.float32, device="cuda:0")
    with pytest.raises(binding.P3TError) as e:
        binding.direct_static(z[:n], z.view(n, 3), 1e-3, 0.0, 0.1, 0.1, torch.empty_like(z).view(n, 3), torch.empty_like(z[:n]))
    assert e.value.status == binding.ECAPACITY and "P3T_STATIC_MAX_N" in str(e.value)
    with pytest.raises(binding.P3TError) as e:        # r_in >= r_out
        binding.direct_static(z[:8], z[:24].view(8, 3), 1e-3, 0.2, 0.1, 0.1, torch.empty(8, 3, device="cuda:0"), torch.empty(8, device="cuda:0"))
    assert e.value.status == binding.EINVAL
    # the largest size it does hold runs
    n = binding.STATIC_MAX_N
    mass, pos = _case(13, n)
    m, q = torch.from_numpy(mass).cuda(), torch.from_numpy(pos).cuda()
    acc, pot = torch.empty(n, 3, device="cuda:0"), torch.empty(n, device="cuda:0")
    binding.direct_static(m, q, 1e-4, 1e-3, 1e-2, 1.2e-2, acc, pot)
    torch.cuda.synchronize()
    assert torch.isfinite(acc).all() and torch.isfinite(pot).all() and (pot < 0).all()
