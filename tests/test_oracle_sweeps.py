"""Pins of the oracle's axis-by-axis exchange (R-24): x, then y, then z,
each sweep classifying along one axis from the current position.  Checked against an
independent global-sort definition of every sweep and against the direct 27-way migration's slab contents."""
import numpy as np
import pytest

from test_oracle_migrate import L, F7, random_state

W = (1, 3, 9)


def axis_delta(pos, s, P, N, axis):
    """Independent statement of the direction along `axis`: minimum-image difference of subdomain indices."""
    p = (s % P[0], (s // P[0]) % P[1], s // (P[0] * P[1]))[axis]
    n_a = N // P[axis]
    own = np.minimum(np.floor(pos * (N / L)).astype(np.int64), N - 1) // n_a
    d = own - p
    if P[axis] >= 3:
        d = np.where(d > 1, d - P[axis], d)
        d = np.where(d < -1, d + P[axis], d)
    return d


def sweep_by_global_sort(pre, P, N, axis):
    """Result of one sweep by definition: the particle goes to the neighbour slab along `axis`; a slab is its stayers in
    order, then the incoming ones by (source slab, code, source slot) -- one global sort, no counters."""
    counts = pre["counts"]
    nP = P[0] * P[1] * P[2]
    src = np.repeat(np.arange(nP), counts)
    slot = np.concatenate([np.arange(c) for c in counts]) if counts.sum() else np.zeros(0, np.int64)
    pos = pre["xyz"[axis]]
    d = np.zeros(src.size, np.int64)
    for s in range(nP):
        m = src == s
        d[m] = axis_delta(pos[m], s, P, N, axis)
    assert d.size == 0 or np.max(np.abs(d)) <= 1
    coord = [src % P[0], (src // P[0]) % P[1], src // (P[0] * P[1])]
    coord[axis] = (coord[axis] + d) % P[axis]
    r = coord[0] + P[0] * (coord[1] + P[1] * coord[2])
    code = 13 + d * W[axis]
    order = np.lexsort((slot, code, src, (d != 0).astype(np.int64), r))
    out = {k: pre[k][order] for k in F7 + ("id",)}
    out["counts"] = np.bincount(r, minlength=nP)
    return out, int(np.count_nonzero(d))


@pytest.mark.parametrize("P,N,n,vscale", [
    ((2, 2, 2), 16, 3000, 0.9), ((3, 3, 3), 24, 6000, 0.9), ((1, 2, 3), 12, 2000, 0.9), ((1, 1, 1), 8, 300, 0.9),
    ((4, 4, 4), 32, 20000, 0.4), ((4, 2, 1), 16, 1, 0.9), ((2, 2, 2), 16, 0, 0.9), ((5, 1, 3), 15, 4000, 0.9)])
def test_each_sweep_equals_its_global_sort_and_the_slabs_match_the_direct_migration(oracle_lib, P, N, n, vscale):
    nP = P[0] * P[1] * P[2]
    cap = max(8, 3 * n // nP + 64)
    o = random_state(oracle_lib, N, P, n, cap=cap, seed=n + 7 * P[0], vscale=vscale)
    o_direct = random_state(oracle_lib, N, P, n, cap=cap, seed=n + 7 * P[0], vscale=vscale)
    assert o.push(1.0) == 0 and o_direct.push(1.0) == 0
    assert o_direct.migrate() == 0
    state = o.get_particles()
    for axis in range(3):
        want, n_moved = sweep_by_global_sort(state, P, N, axis)
        assert o.classify_axis(axis) == 0
        codes = o.get_particles()["code"]
        assert set(np.unique(codes)) <= {13 - W[axis], 13, 13 + W[axis]}
        assert o.migrate() == 0
        assert o.n_migrated_last == n_moved
        state = o.get_particles()
        for k in F7 + ("id", "counts"):
            assert np.array_equal(state[k], want[k]), (axis, k)
    # after x, y, z every particle sits in the slab that contains it, exactly as after the direct 27-way migration:
    # same counts and the same id SET per slab (the order inside a slab is the sweeps' own, R-24)
    direct = o_direct.get_particles()
    assert np.array_equal(state["counts"], direct["counts"])
    off = np.concatenate([[0], np.cumsum(state["counts"])])
    for s in range(nP):
        assert np.array_equal(np.sort(state["id"][off[s]:off[s + 1]]), np.sort(direct["id"][off[s]:off[s + 1]]))
    cells = [np.minimum(np.floor(state[k] * (N / L)).astype(np.int64), N - 1) for k in "xyz"]
    owner = cells[0] // (N // P[0]) + P[0] * (cells[1] // (N // P[1]) + P[1] * (cells[2] // (N // P[2])))
    assert np.array_equal(owner, np.repeat(np.arange(nP), state["counts"]))
    # a fourth sweep finds nothing to move
    assert o.classify_axis(0) == 0 and o.migrate() == 0 and o.n_migrated_last == 0


def test_corner_mover_takes_three_hops_and_seam_directions(oracle_lib):
    """Hand-placed: a particle bound for the (+,+,+) corner neighbour moves once per sweep; across the periodic seam the
    direction is the minimum image (P = 3: index difference -2 means +1)."""
    N, P = 12, (3, 3, 3)
    o = oracle_lib.Oracle(N, *P, 16)
    z = np.zeros(N ** 3)
    o.set_fluid(z, z, z)
    Ls = L / 3
    # particle 0: in slab (2,2,2) near its upper corner, crosses the seam into (0,0,0); particle 1: stays; particle 2:
    # in slab (0,1,1), crosses the lower x seam into (2,1,1)
    x = np.array([3 * Ls - 0.01, 0.5 * Ls, 0.01])
    y = np.array([3 * Ls - 0.01, 0.5 * Ls, 1.5 * Ls])
    zc = np.array([3 * Ls - 0.01, 0.5 * Ls, 1.5 * Ls])
    v = np.array([0.05, 0.0, -0.05])
    o.set_particles(x, y, zc, v, np.array([0.05, 0, 0]), np.array([0.05, 0, 0]), np.full(3, 1.0), np.array([10, 11, 12]))
    assert o.push(1.0) == 0
    where = []
    for axis in range(3):
        assert o.classify_axis(axis) == 0 and o.migrate() == 0
        st = o.get_particles()
        slab = np.repeat(np.arange(27), st["counts"])
        where.append({int(i): int(s) for i, s in zip(st["id"], slab)})
    sid = lambda px, py, pz: px + 3 * (py + 3 * pz)
    assert [w[10] for w in where] == [sid(0, 2, 2), sid(0, 0, 2), sid(0, 0, 0)]
    assert [w[11] for w in where] == [sid(0, 0, 0)] * 3
    assert [w[12] for w in where] == [sid(2, 1, 1)] * 3
    assert o.migrate_sweeps() == (0, [0, 0, 0])


def test_two_subdomains_per_axis_and_one(oracle_lib):
    """P_a = 2: both neighbours are the same slab and the index difference is the direction; P_a = 1: nothing moves."""
    N, P = 8, (2, 1, 1)
    o = oracle_lib.Oracle(N, *P, 16)
    z = np.zeros(N ** 3)
    o.set_fluid(z, z, z)
    x = np.array([0.01, L / 2 - 0.01, L - 0.01])
    vx = np.array([-0.05, 0.05, 0.05])          # below 0 (wraps to the top slab), over the middle face, over the seam
    mid = np.full(3, 1.0)
    o.set_particles(x, mid, mid, vx, np.zeros(3), np.zeros(3), np.full(3, 1.0), np.array([1, 2, 3]))
    assert o.push(1.0) == 0
    assert o.classify_axis(0) == 0
    assert list(o.get_particles()["code"]) == [14, 14, 12]     # slab 0: ids 1, 2 go up (+1); slab 1: id 3 goes down (-1)
    assert o.migrate() == 0
    st = o.get_particles()
    assert list(st["counts"]) == [1, 2] and list(st["id"]) == [3, 1, 2]
    for axis in (1, 2):
        assert o.classify_axis(axis) == 0
        assert set(o.get_particles()["code"]) == {13}
        assert o.migrate() == 0 and o.n_migrated_last == 0
