"""lcs_pair_count_static: the pair count with the library's own built-in scratch (no allocation, no borrowed pool).

Why the entry point exists, for whoever maintains this file: some users call the g(r) statistic from a diagnostics
hook inside a running time loop.  Their host application took all device memory at start-up and forbids cudaMalloc /
cudaFree from then on (those calls stall every stream on the GPU and may fail with HBM already given away), and they
sized the handle's send pool for the few per cent of particles that migrate -- too small for lcs_pair_count, which
borrows three position arrays from it.  lcs_pair_count_static keeps its scratch in a fixed 17 MiB array inside the
library's device image instead, for handles of up to 2^19 particle slots.

What is checked: on two calls in a row (the second starts with the first call's cell list still in the shared array,
and uses a different cell grid) the count equals lcs_pair_count's on the same handle -- integers, so the tolerance is
the one the other pair-count tests use: exact equality; a handle whose send pool is too small for lcs_pair_count still
gets the right count; a handle beyond the limit gets LCS_ERR_TOO_LARGE and nothing is enqueued; and the free device
memory reported by the driver does not move across the calls.

The file sorts last on purpose (pytest -x stops at the first failure; a failure here hides nothing), and it makes no
assumption on what ran before it in the process: it passes alone and after the rest of the suite."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

L = 6.283185307179586
F8 = ("x", "y", "z", "vx", "vy", "vz", "d", "id")


def _particles(rng, n):
    """Uniform particles plus a clump (many close pairs) and a few pairs across the periodic seam."""
    X = np.minimum(rng.random((3, n)) * L, np.nextafter(L, 0.0))
    k = n // 4
    X[:, :k] = (X[:, :k] - L / 2) * 0.03 + L / 2
    X[0, k:k + 40] = np.where(np.arange(40) % 2 == 0, 1e-3 * rng.random(40), np.nextafter(L, 0.0) - 1e-3 * rng.random(40))
    X[1, k:k + 40] = 1.0 + 1e-3 * rng.random(40)
    X[2, k:k + 40] = 2.0 + 1e-3 * rng.random(40)
    V = (rng.random((3, n)) * 2 - 1) * 0.3
    return {"x": X[0], "y": X[1], "z": X[2], "vx": V[0], "vy": V[1], "vz": V[2], "d": np.full(n, 1.0),
            "id": rng.permutation(n).astype(np.int64)}


def _handle(torch, N, P, cap, parts, send_capacity=0):
    from paper_2604_11008_b200 import LCS
    dev = LCS(N, *P, cap, send_capacity=send_capacity)
    dev.set_fluid(*(torch.zeros(N ** 3, dtype=torch.float64, device="cuda") for _ in range(3)))
    dp = {k: torch.from_numpy(np.ascontiguousarray(v)).cuda() for k, v in parts.items()}
    dev.set_particles(*(dp[k] for k in F8))
    assert dev.get_status()[:2] == (0, parts["id"].size)
    return dev


def test_static_scratch_pair_count_equals_pool_pair_count_twice_in_a_row():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("a CUDA device is required for -m gpu tests (no CPU fallback exists)")
    from paper_2604_11008_b200 import LcsError, LCS_ERR_INVALID_ARG, LCS_ERR_TOO_LARGE, LCS_PAIR_COUNT_STATIC_MAX_SLOTS
    rng = np.random.default_rng(2604)
    n, P, N = 30000, (2, 2, 2), 16
    cap = 2 * (int(2.5 * n / 8) // 2 + 400)
    parts = _particles(rng, n)
    dev = _handle(torch, N, P, cap, parts)
    out = torch.empty(1, dtype=torch.int64, device="cuda")
    # two different cell grids back to back: the second call finds the first call's cell list in the array
    shells = ((0.0, 0.01), (0.3, L / 3), (0.01, 0.05), (0.0, 2e-3), (0.05, 0.050001), (0.0, L / 3))
    want = {sh: int(dev.pair_count(*sh).item()) for sh in shells}
    assert want[(0.0, 0.01)] > 1000 and want[(0.0, L / 3)] > want[(0.3, L / 3)] > 0      # the comparison is not 0 == 0
    dev.pair_count_static(*shells[0], out=out)                   # first use in this process or not: either must work
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    first = int(dev.pair_count_static(*shells[0], out=out).item())
    second = int(dev.pair_count_static(*shells[1], out=out).item())
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free_before, "device memory was allocated or freed by the call"
    assert first == want[shells[0]] and second == want[shells[1]]
    for sh in shells:                                            # and the same shell twice running, no sync in between
        a = dev.pair_count_static(*sh).clone()
        b = dev.pair_count_static(*sh).clone()
        assert int(a.item()) == want[sh] and int(b.item()) == want[sh], sh
    # after a migration step the slabs have changed; both paths must still agree
    dev.step_fused(0.5)
    for sh in shells[:3]:
        assert int(dev.pair_count_static(*sh, out=out).item()) == int(dev.pair_count(*sh).item()), sh
    for bad in ((0.1, 0.1), (-0.1, 0.2), (0.0, L / 3 * 1.01)):   # same argument rules as lcs_pair_count
        with pytest.raises(LcsError) as ei:
            dev.pair_count_static(*bad)
        assert ei.value.code == LCS_ERR_INVALID_ARG
    dev.close()

    # the caller this is for: a send pool far too small for lcs_pair_count
    small = _handle(torch, N, P, cap, parts, send_capacity=cap // 16 // 2 * 2)
    with pytest.raises(LcsError) as ei:
        small.pair_count(0.0, 0.01)
    assert ei.value.code == LCS_ERR_INVALID_ARG
    assert int(small.pair_count_static(0.0, 0.01).item()) == want[(0.0, 0.01)]
    assert int(small.pair_count_static(0.3, L / 3).item()) == want[(0.3, L / 3)]
    small.close()

    # at the limit it runs, one slab slot pair beyond it is refused with the error code of its own
    cap_max = LCS_PAIR_COUNT_STATIC_MAX_SLOTS // 8
    at_limit = _handle(torch, N, P, cap_max, parts)
    assert int(at_limit.pair_count_static(0.0, 0.01).item()) == want[(0.0, 0.01)]
    at_limit.close()
    beyond = _handle(torch, N, P, cap_max + 2, parts)
    launches = beyond.kernel_launches
    with pytest.raises(LcsError) as ei:
        beyond.pair_count_static(0.0, 0.01)
    assert ei.value.code == LCS_ERR_TOO_LARGE and "slots" in str(ei.value)
    assert beyond.kernel_launches == launches                    # nothing was enqueued
    assert int(beyond.pair_count(0.0, 0.01).item()) == want[(0.0, 0.01)]
    beyond.close()
