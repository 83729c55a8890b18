"""Pins of the oracle's pair count (the statistic behind g(r); DESIGN.md
R-26): hand-countable configurations, the periodic seam, the edges of the shell, and the uniform-random limit g = 1 --
never against the oracle itself."""
import math

import numpy as np
import pytest

L = 6.283185307179586


def make(oracle_lib, X, P=(1, 1, 1), N=12):
    X = np.asarray(X, dtype=np.float64).reshape(-1, 3)
    n = X.shape[0]
    o = oracle_lib.Oracle(N, *P, max(8, 2 * n))
    z = np.zeros(n)
    assert o.set_particles(X[:, 0], X[:, 1], X[:, 2], z, z, z, np.ones(n), np.arange(n, dtype=np.int64)) == 0
    return o


def test_simple_cubic_lattice_has_3n_nearest_neighbour_pairs(oracle_lib):
    """m^3 points on a periodic simple cubic lattice of spacing a = L/m: every point has 6 neighbours at distance a,
    12 at a*sqrt(2), 8 at a*sqrt(3): 3n, 6n and 4n unordered pairs (the seam pairs included)."""
    m = 5
    a = L / m
    g = (np.arange(m) + 0.25) * a
    X = np.array([(x, y, z) for x in g for y in g for z in g])
    n = m ** 3
    o = make(oracle_lib, X, P=(1, 1, 1), N=10)
    assert o.pair_count(0.9 * a, 1.1 * a) == 3 * n
    assert o.pair_count(1.3 * a, 1.5 * a) == 6 * n
    assert o.pair_count(1.6 * a, 1.8 * a) == 4 * n
    assert o.pair_count(0.0, 0.9 * a) == 0
    assert o.pair_count(0.0, 1.8 * a) == 13 * n
    o.close()


def test_pairs_across_the_periodic_seam_and_shell_edges(oracle_lib):
    e = 1e-3
    # two particles 2e apart across the x seam, two across the y and z seams together, one far away
    X = [(e, 1.0, 1.0), (L - e, 1.0, 1.0),
         (3.0, e, L - e), (3.0, L - e, e),
         (5.0, 5.0, 5.0)]
    o = make(oracle_lib, X)
    assert o.pair_count(0.0, 1.0) == 2
    assert o.pair_count(1.9 * e, 2.1 * e) == 1                               # the x pair: distance 2e
    d = math.sqrt(8.0) * e
    assert o.pair_count(0.99 * d, 1.01 * d) == 1                             # the (y,z) pair: 2e in y and in z
    o.close()
    # half-open shell [r_lo, r_hi): a pair at distance exactly r (representable: 0.5) is in [r, ..) and not in [.., r)
    o = make(oracle_lib, [(1.0, 2.0, 3.0), (1.5, 2.0, 3.0)])
    assert o.pair_count(0.5, 0.6) == 1 and o.pair_count(0.4, 0.5) == 0 and o.pair_count(0.0, 0.5) == 0
    o.close()
    # coincident particles are a pair at r = 0
    o = make(oracle_lib, [(1.0, 1.0, 1.0), (1.0, 1.0, 1.0), (1.0, 1.0, 1.0)])
    assert o.pair_count(0.0, 1e-9) == 3
    o.close()
    with pytest.raises(ValueError):
        make(oracle_lib, [(1.0, 1.0, 1.0)]).pair_count(0.2, 0.1)


def test_uniform_random_particles_give_g_equal_one(oracle_lib):
    """g = count / (n(n-1)/2 * V_shell / L^3) -> 1 for uniformly distributed particles ("unity indicates a uniform
    distribution"); 3 sigma of the Poisson error of the expected count."""
    rng = np.random.default_rng(12)
    n = 6000
    X = rng.random((n, 3)) * L
    o = make(oracle_lib, X, P=(2, 2, 2), N=8)
    for r_lo, r_hi in ((0.0, 0.3), (0.3, 0.5), (0.05, 0.1)):
        expect = 0.5 * n * (n - 1) * (4.0 / 3.0) * math.pi * (r_hi ** 3 - r_lo ** 3) / L ** 3
        got = o.pair_count(r_lo, r_hi)
        assert abs(got - expect) <= 3.0 * math.sqrt(expect) + 1, (r_lo, r_hi, got, expect)
    o.close()


def test_count_does_not_depend_on_the_decomposition_or_order(oracle_lib):
    rng = np.random.default_rng(4)
    n = 1500
    X = rng.random((n, 3)) * L
    X[: n // 3] = (X[: n // 3] - L / 2) * 0.05 + L / 2            # a clump: many close pairs
    ref = None
    for P, perm in (((1, 1, 1), None), ((3, 2, 1), None), ((2, 2, 2), rng.permutation(n))):
        o = make(oracle_lib, X if perm is None else X[perm], P=P, N=12)
        c = (o.pair_count(0.0, 0.02), o.pair_count(0.02, 0.2))
        o.close()
        ref = ref or c
        assert c == ref and c[0] > 100
    # and against a numpy statement of the same definition
    d = X[:, None, :] - X[None, :, :]
    d = np.where(d > L / 2, d - L, np.where(d < -L / 2, d + L, d))
    r2 = np.sum(d * d, axis=2)[np.triu_indices(n, 1)]
    assert abs(int(np.sum(r2 < 0.02 ** 2)) - ref[0]) <= 2        # (numpy sums the squares in another order: edge pairs)
