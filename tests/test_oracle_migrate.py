"""Pins for the oracle's a5-a8 (count, scan, stable pack, compaction, ordered append).
PAPER.md:112 (sequential definition), :114-124 (mask / prefix-scan / pack and the worked example),
:175 (unpack + compaction); order of the result: north_star / DESIGN.md R-12."""
import os

import numpy as np
import pytest

L = 6.283185307179586
HERE = os.path.dirname(os.path.abspath(__file__))
F7 = ("x", "y", "z", "vx", "vy", "vz", "d")


def read_golden_scan():
    rows = {}
    for line in open(os.path.join(HERE, "golden", "scan_example.txt")):
        if line.startswith("#") or ":" not in line:
            continue
        k, v = line.split(":")
        rows[k.strip()] = v.split()
    return rows


def test_paper_worked_example(oracle_lib):
    """mask 0,1,0,1,0 -> scan 0,1,1,2,2 -> particle 2 in buffer[1], particle 4 in buffer[2]."""
    g = read_golden_scan()
    mask = [int(t) for t in g["mask"]]
    scan = [int(t) for t in g["scan"]]
    assert list(np.cumsum(mask)) == scan                      # the paper's scan is the inclusive sum
    want = [None if t == "-" else int(t) for t in g["buffer_slot_1based"]]
    # five particles in subdomain 0 of a 2x1x1 box; the masked ones cross the +x face
    N = 8
    o = oracle_lib.Oracle(N, 2, 1, 1, 16)
    z = np.zeros(N ** 3)
    o.set_fluid(z, z, z)
    n = 5
    x0 = np.full(n, L / 2 - 0.1)
    vx = np.array([0.2 if m else 0.0 for m in mask])
    mid = np.full(n, 1.0)
    o.set_particles(x0, mid, mid, vx, np.zeros(n), np.zeros(n), np.full(n, 1.0), np.arange(1, n + 1))
    assert o.push(1.0) == 0
    pre = o.get_particles()
    assert list((pre["code"] != 13).astype(int)) == mask       # stage 1: the mask
    assert o.migrate() == 0
    slots = o.last_send_slots(0, n)                            # stage 2+3: 0-based storage positions
    got = [None if s < 0 else int(s) + 1 for s in slots]
    assert got == want
    out = o.get_particles()
    assert list(out["counts"]) == [3, 2]
    assert list(out["id"]) == [1, 3, 5, 2, 4]                  # stayers in order, then the buffer in order


def random_state(oracle_lib, N, P, n, cap, seed, vscale):
    """Ballistic random particles (zero fluid, huge tau): displacement = v*dt, all codes possible."""
    rng = np.random.default_rng(seed)
    o = oracle_lib.Oracle(N, *P, cap)
    z = np.zeros(N ** 3)
    o.set_fluid(z, z, z)
    X = rng.random((3, n)) * L
    Ls = np.array([L / P[0], L / P[1], L / P[2]])
    V = (rng.random((3, n)) * 2 - 1) * (vscale * Ls[:, None])
    ids = rng.permutation(n).astype(np.int64) + 100
    assert o.set_particles(X[0], X[1], X[2], V[0], V[1], V[2], np.full(n, 1.0), ids) == 0
    return o


def brute_force_migrate(pre, P, N):
    """Independent definition of the result: slab r = all particles whose NEW position lies in r,
    sorted by (is_migrant, source subdomain, code, source slot) -- one global sort, no counters."""
    counts = pre["counts"]
    nP = P[0] * P[1] * P[2]
    src = np.repeat(np.arange(nP), counts)
    slot = np.concatenate([np.arange(c) for c in counts]) if counts.sum() else np.zeros(0, np.int64)
    n_a = [N // P[0], N // P[1], N // P[2]]
    cells = [np.minimum(np.floor(pre[k] * (N / L)).astype(np.int64), N - 1) for k in "xyz"]
    r = (cells[0] // n_a[0]) + P[0] * ((cells[1] // n_a[1]) + P[1] * (cells[2] // n_a[2]))
    mig = (pre["code"] != 13).astype(np.int64)
    order = np.lexsort((slot, pre["code"], src, mig, r))      # last key is primary
    out = {k: pre[k][order] for k in F7 + ("id",)}
    out["counts"] = np.bincount(r, minlength=nP)
    return out, r, src


@pytest.mark.parametrize("P,N,n,vscale", [
    ((2, 2, 2), 16, 3000, 0.9), ((3, 3, 3), 24, 6000, 0.9), ((1, 2, 3), 12, 2000, 0.9),
    ((1, 1, 1), 8, 500, 0.9), ((4, 4, 4), 32, 20000, 0.3), ((2, 1, 1), 8, 7, 0.9),
    ((4, 2, 1), 16, 1, 0.9), ((2, 2, 2), 16, 0, 0.9)])
def test_migrate_equals_global_sort(oracle_lib, P, N, n, vscale):
    o = random_state(oracle_lib, N, P, n, cap=max(8, 3 * n // (P[0] * P[1] * P[2]) + 64), seed=n + P[0], vscale=vscale)
    assert o.push(1.0) == 0
    pre = o.get_particles()
    if n >= 2000 and min(P) >= 3:
        assert len(np.unique(pre["code"])) == 27               # every destination present
    # classify pin on random inputs: the slab that contains the new position is receiver(s, code)
    want, r_new, src = brute_force_migrate(pre, P, N)
    recv = np.array([o.receiver(s, c) for s, c in zip(src, pre["code"])], dtype=np.int64)
    assert np.array_equal(recv, r_new)
    tab = o.cnt_table()
    for s in range(o.P):
        assert np.array_equal(tab[s], np.bincount(pre["code"][src == s], minlength=27))   # a4
    assert o.migrate() == 0
    got = o.get_particles()
    assert np.array_equal(got["counts"], want["counts"])
    for k in F7 + ("id",):
        assert np.array_equal(got[k], want[k]), k              # bit-exact, order included
    assert np.all(got["code"] == 13)
    assert o.n_migrated_last == int((pre["code"] != 13).sum())
    # conservation of the ID multiset
    assert np.array_equal(np.sort(got["id"]), np.sort(pre["id"]))
    # containment: every particle ends in the subdomain that contains its position
    slab = np.repeat(np.arange(o.P), got["counts"])
    own = np.array([o.owner(x, y, z) for x, y, z in zip(got["x"], got["y"], got["z"])], dtype=np.int64)
    assert np.array_equal(slab, own)
    # idempotence: a second migrate with all codes 13 changes nothing
    assert o.migrate() == 0
    again = o.get_particles()
    for k in F7 + ("id", "counts"):
        assert np.array_equal(again[k], got[k])


def test_stayers_keep_relative_order_and_zero_or_all_migrants(oracle_lib):
    N, P = 16, (2, 2, 2)
    # zero migrants
    o = random_state(oracle_lib, N, P, 1000, 400, seed=1, vscale=0.0)
    o.push(1.0)
    pre = o.get_particles()
    assert np.all(pre["code"] == 13)
    o.migrate()
    post = o.get_particles()
    assert all(np.array_equal(pre[k], post[k]) for k in F7 + ("id", "counts"))
    # every particle leaves: all move by exactly one subdomain in +x
    rng = np.random.default_rng(3)
    n = 800
    o = oracle_lib.Oracle(N, *P, 400)
    z = np.zeros(N ** 3)
    o.set_fluid(z, z, z)
    X = rng.random((3, n)) * L
    o.set_particles(X[0], X[1], X[2], np.full(n, L / 2), np.zeros(n), np.zeros(n), np.full(n, 1.0), np.arange(n))
    o.push(1.0)
    pre = o.get_particles()
    assert np.all(pre["code"] == 14)
    o.migrate()
    post = o.get_particles()
    assert o.n_migrated_last == n and post["counts"].sum() == n
    # receiver r gets source r^1 (x neighbour) in source order
    src = np.repeat(np.arange(8), pre["counts"])
    for r in range(8):
        lo = post["counts"][:r].sum()
        assert np.array_equal(post["id"][lo:lo + post["counts"][r]], pre["id"][src == (r ^ 1)])
    # mixed: stayers of each slab keep their relative order
    o = random_state(oracle_lib, N, P, 4000, 1200, seed=5, vscale=0.5)
    o.push(1.0)
    pre = o.get_particles()
    o.migrate()
    post = o.get_particles()
    src = np.repeat(np.arange(8), pre["counts"])
    for s in range(8):
        stay_ids = pre["id"][(src == s) & (pre["code"] == 13)]
        lo = post["counts"][:s].sum()
        assert np.array_equal(post["id"][lo:lo + len(stay_ids)], stay_ids)


def test_capacity_overflow_is_a_sticky_error(oracle_lib):
    N = 8
    o = oracle_lib.Oracle(N, 2, 1, 1, 6)
    z = np.zeros(N ** 3)
    o.set_fluid(z, z, z)
    n = 10     # 5 per slab; all of slab 0 moves to slab 1 -> 10 > 6
    x = np.concatenate([np.full(5, 1.0), np.full(5, 4.0)])
    vx = np.concatenate([np.full(5, 3.0), np.zeros(5)])
    mid = np.full(n, 1.0)
    assert o.set_particles(x, mid, mid, vx, 0 * mid, 0 * mid, mid, np.arange(n)) == 0
    assert o.push(1.0) == 0
    assert o.migrate() == oracle_lib.ERR_CAPACITY
    assert o.status == oracle_lib.ERR_CAPACITY
    o2 = oracle_lib.Oracle(N, 2, 1, 1, 4)
    assert o2.set_particles(np.full(5, 1.0), np.ones(5), np.ones(5), *(np.zeros(5),) * 3, np.ones(5),
                            np.arange(5)) == oracle_lib.ERR_CAPACITY


def test_load_packed_roundtrip_and_migrate_on_foreign_state(oracle_lib):
    """Protocol P1 needs the oracle's migrate to run on a state it did not produce itself."""
    N, P = 16, (2, 2, 2)
    o = random_state(oracle_lib, N, P, 3000, 900, seed=9, vscale=0.8)
    o.push(1.0)
    pre = o.get_particles()
    o2 = oracle_lib.Oracle(N, *P, 900)
    assert o2.load_packed(pre["counts"], *(pre[k] for k in F7), pre["id"], pre["code"]) == 0
    assert np.array_equal(o2.cnt_table(), o.cnt_table())
    o.migrate()
    o2.migrate()
    a, b = o.get_particles(), o2.get_particles()
    for k in F7 + ("id", "counts"):
        assert np.array_equal(a[k], b[k])


def test_tiny_config_multi_step_invariants(oracle_lib):
    from workloads import gen
    cfg = gen.get_config("Tiny")
    wl = gen.make_workload(cfg)
    o = oracle_lib.Oracle(cfg["N"], *cfg["P"], cfg["capacity"], g=cfg["g"])
    o.set_fluid(wl["u"].numpy(), wl["v"].numpy(), wl["w"].numpy())
    p = {k: v.numpy() for k, v in wl["particles"].items()}
    assert o.set_particles(*(p[k] for k in F7), p["id"]) == 0
    for _ in range(cfg["steps"]):
        assert o.step(cfg["dt"]) == 0
        out = o.get_particles()
        assert out["counts"].sum() == cfg["n"]
        assert np.array_equal(np.sort(out["id"]), np.arange(cfg["n"]))
        assert 0.02 < o.n_migrated_last / cfg["n"] < 0.09
        slab = np.repeat(np.arange(o.P), out["counts"])
        cells = [np.minimum(np.floor(out[k] * (cfg["N"] / L)).astype(np.int64), cfg["N"] - 1) for k in "xyz"]
        nx = cfg["N"] // 2
        own = cells[0] // nx + 2 * (cells[1] // nx + 2 * (cells[2] // nx))
        assert np.array_equal(own, slab)
        ids = np.argsort(out["id"])
        assert np.array_equal(out["d"][ids], p["d"])          # diameter rides along unchanged
