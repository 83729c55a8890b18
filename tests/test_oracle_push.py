"""Pins for the oracle's a1-a4 (gather, advance, classify, count) against what the paper and the
mathematics fix -- closed forms, invariants and independent brute force; never the oracle itself.
PAPER.md:47 (periodic cube), :51-57 (Eq. 5-6, tau_p), :64 (trilinear from cell centres), :116 (mask)."""
import math
import os

import numpy as np
import pytest

L = 6.283185307179586
HERE = os.path.dirname(os.path.abspath(__file__))


def ulp_diff(a, b):
    a = np.asarray(a, dtype=np.float64).view(np.int64)
    b = np.asarray(b, dtype=np.float64).view(np.int64)
    return np.abs(a - b)


# ------------------------------------------------------------------------------------------------
# exp_neg (R-3)
# ------------------------------------------------------------------------------------------------
def test_exp_neg_against_libm(oracle_lib):
    rng = np.random.default_rng(7)
    zs = np.concatenate([[0.0, 1e-300, 1e-17, 0.5 * math.log(2), math.log(2), 1.0, 707.9, 708.0],
                         rng.random(20000) * 708.0, 10.0 ** rng.uniform(-12, 2.85, 20000)])
    got = np.array([oracle_lib.exp_neg(z) for z in zs])
    want = np.exp(-zs)
    assert oracle_lib.exp_neg(0.0) == 1.0
    assert np.all(got > 0.0)
    assert ulp_diff(got, want).max() <= 2
    assert oracle_lib.exp_neg(708.0000001) == 0.0 and oracle_lib.exp_neg(1e308) == 0.0
    assert oracle_lib.exp_neg(float("inf")) == 0.0
    assert math.isnan(oracle_lib.exp_neg(float("nan")))


def test_exp_neg_monotone(oracle_lib):
    zs = np.linspace(0.0, 40.0, 40001)
    got = np.array([oracle_lib.exp_neg(z) for z in zs])
    assert np.all(np.diff(got) <= 0.0)


# ------------------------------------------------------------------------------------------------
# tau_p against hand-evaluated values
# ------------------------------------------------------------------------------------------------
def test_tau_p_values(oracle_lib):
    rows = [l.split() for l in open(os.path.join(HERE, "golden", "tau_p.txt")) if l.strip() and l[0] != "#"]
    assert len(rows) == 4
    for r, rho, tau in rows:
        o = oracle_lib.Oracle(8, 1, 1, 1, 4, nu=1.5e-5, rho_ratio=float(rho))
        assert o.tau(2.0 * float(r)) == pytest.approx(float(tau), rel=1e-14)


# ------------------------------------------------------------------------------------------------
# cell / owner (R-13, R-15): half-open cells, x-fastest numbering
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("N,P", [(32, (2, 2, 2)), (12, (1, 2, 3)), (48, (3, 4, 2))])
def test_cell_and_owner_at_faces(oracle_lib, N, P):
    o = oracle_lib.Oracle(N, *P, 4)
    dx = L / N
    # every cell face and its two neighbours in floating point
    for i in range(N + 1):
        f = min(i * dx, np.nextafter(L, 0.0))
        for a in (np.nextafter(f, -1.0), f, np.nextafter(f, 10.0)):
            if not (0.0 <= a < L):
                continue
            c = o.cell(a)
            # independent definition: the unique i with i <= a*N/L < i+1, found by linear search
            t = a * (N / L)
            want = next(j for j in range(N) if j <= t < j + 1 or (j == N - 1 and t >= j))
            assert c == want
    assert o.cell(0.0) == 0 and o.cell(np.nextafter(L, 0.0)) == N - 1
    # monotone
    xs = np.sort(np.random.default_rng(1).random(2000) * L)
    cs = [o.cell(a) for a in xs]
    assert all(b >= a for a, b in zip(cs, cs[1:]))
    # owner: linear search over [lo, hi) index intervals per axis
    rng = np.random.default_rng(2)
    pts = rng.random((500, 3)) * L
    n_a = [N // P[0], N // P[1], N // P[2]]
    for x, y, z in pts:
        idx = []
        for a, (v, na, Pa) in enumerate(zip((x, y, z), n_a, P)):
            ci = o.cell(v)
            idx.append(next(p for p in range(Pa) if p * na <= ci < (p + 1) * na))
        assert o.owner(x, y, z) == idx[0] + P[0] * (idx[1] + P[1] * idx[2])


def test_receiver_hand_table(oracle_lib):
    # 1 x 2 x 3 decomposition: s = px + 1*(py + 2*pz), hand-computed neighbours
    o = oracle_lib.Oracle(12, 1, 2, 3, 4)
    code = lambda dx, dy, dz: (dx + 1) + 3 * (dy + 1) + 9 * (dz + 1)
    assert code(0, 0, 0) == 13
    s = 0 + 1 * (1 + 2 * 2)          # (px,py,pz) = (0,1,2) -> 5
    assert s == 5
    assert o.receiver(s, code(0, 0, 0)) == 5
    assert o.receiver(s, code(1, 0, 0)) == 5          # Px = 1: the x neighbour is itself
    assert o.receiver(s, code(-1, 0, 0)) == 5
    assert o.receiver(s, code(0, 1, 0)) == 0 + 1 * (0 + 2 * 2)     # py 1 -> 0 (periodic) = 4
    assert o.receiver(s, code(0, -1, 0)) == 4                      # Py = 2: both neighbours coincide
    assert o.receiver(s, code(0, 0, 1)) == 0 + 1 * (1 + 2 * 0)     # pz 2 -> 0 = 1
    assert o.receiver(s, code(0, 0, -1)) == 0 + 1 * (1 + 2 * 1)    # pz 2 -> 1 = 3
    assert o.receiver(s, code(1, 1, 1)) == 0 + 1 * (0 + 2 * 0)     # = 0
    assert o.receiver(0, code(0, -1, -1)) == 0 + 1 * (1 + 2 * 2)   # (0,0,0) -> (0,1,2) = 5


# ------------------------------------------------------------------------------------------------
# a1 trilinear interpolation
# ------------------------------------------------------------------------------------------------
def centres(N):
    return (np.arange(N) + 0.5) * (L / N)


def grid_field(N, fn):
    """F[i + N*(j + N*k)] = fn(x_i, y_j, z_k) at cell centres (x fastest)."""
    c = centres(N)
    Z, Y, X = np.meshgrid(c, c, c, indexing="ij")     # array index [k, j, i]
    return np.ascontiguousarray(fn(X, Y, Z)).reshape(-1)


def test_interp_constant_and_nodal_bit_exact(oracle_lib):
    N = 16
    o = oracle_lib.Oracle(N, 2, 2, 2, 4)
    rng = np.random.default_rng(3)
    cu, cv, cw = 0.1234567890123, -7.25, 3.0e-7
    o.set_fluid(np.full(N ** 3, cu), np.full(N ** 3, cv), np.full(N ** 3, cw))
    p = rng.random((3, 4000)) * L
    u, v, w = o.interp(*p)
    assert np.all(u == cu) and np.all(v == cv) and np.all(w == cw)
    # nodal values at cell centres: three different random fields (catches component mix-ups)
    F = [rng.standard_normal(N ** 3) for _ in range(3)]
    o.set_fluid(*F)
    c = centres(N)
    ii, jj, kk = (rng.integers(0, N, 3000) for _ in range(3))
    u, v, w = o.interp(c[ii], c[jj], c[kk])
    flat = ii + N * (jj + N * kk)
    # the centre coordinate is itself rounded, so f is within a few ulp of 0: allow 1e-13 absolute
    for got, Fc in zip((u, v, w), F):
        assert np.max(np.abs(got - Fc[flat])) < 1e-12


def test_interp_axis_orientation(oracle_lib):
    # u depends on x only, v on y only, w on z only: a transposed index or swapped axis fails
    N = 8
    o = oracle_lib.Oracle(N, 1, 1, 1, 4)
    o.set_fluid(grid_field(N, lambda X, Y, Z: X), grid_field(N, lambda X, Y, Z: 10 + Y),
                grid_field(N, lambda X, Y, Z: 20 + Z))
    rng = np.random.default_rng(4)
    lo, hi = 0.5 * L / N, L - 0.5 * L / N
    p = lo + rng.random((3, 2000)) * (hi - lo)
    u, v, w = o.interp(*p)
    assert np.allclose(u, p[0], rtol=0, atol=1e-13)
    assert np.allclose(v, 10 + p[1], rtol=0, atol=1e-13)
    assert np.allclose(w, 20 + p[2], rtol=0, atol=1e-13)


def test_interp_reproduces_trilinear_polynomials(oracle_lib):
    N = 24
    o = oracle_lib.Oracle(N, 2, 2, 2, 4)
    rng = np.random.default_rng(5)
    co = rng.standard_normal((3, 8))
    poly = lambda c: (lambda X, Y, Z: c[0] + c[1] * X + c[2] * Y + c[3] * Z + c[4] * X * Y
                      + c[5] * Y * Z + c[6] * Z * X + c[7] * X * Y * Z)
    o.set_fluid(*(grid_field(N, poly(c)) for c in co))
    lo, hi = 0.5 * L / N, L - 0.5 * L / N      # stencil does not cross the periodic seam
    p = lo + rng.random((3, 5000)) * (hi - lo)
    got = o.interp(*p)
    for g, c in zip(got, co):
        want = poly(c)(*p)
        assert np.max(np.abs(g - want)) <= 1e-14 * np.max(np.abs(want)) * 40


def test_interp_second_order_convergence(oracle_lib):
    rng = np.random.default_rng(6)
    p = rng.random((3, 4000)) * L
    errs = []
    for N in (16, 32, 64):
        o = oracle_lib.Oracle(N, 1, 1, 1, 4)
        f = grid_field(N, lambda X, Y, Z: np.sin(X) * np.cos(2 * Y) + np.sin(Z))
        o.set_fluid(f, f, f)
        u, _, _ = o.interp(*p)
        errs.append(np.max(np.abs(u - (np.sin(p[0]) * np.cos(2 * p[1]) + np.sin(p[2])))))
    assert 3.3 < errs[0] / errs[1] < 4.7 and 3.3 < errs[1] / errs[2] < 4.7


def test_interp_periodic_seam_against_halo_definition(oracle_lib):
    # independent definition: pad the field with a one-cell periodic halo and interpolate without
    # any modulo, by direct weighted sum of the 8 corners (weights (1-f) and f).
    N = 12
    rng = np.random.default_rng(8)
    F = [rng.standard_normal((N, N, N)) for _ in range(3)]      # [k, j, i]
    o = oracle_lib.Oracle(N, 1, 1, 1, 4)
    o.set_fluid(*(f.reshape(-1) for f in F))
    dx = L / N
    # points within half a cell of the seam on at least one axis, both sides
    p = rng.random((3, 3000)) * L
    near = rng.integers(0, 3, 3000)
    side = rng.integers(0, 2, 3000)
    off = rng.random(3000) * 0.5 * dx
    for a in range(3):
        sel = near == a
        p[a, sel] = np.where(side[sel] == 0, off[sel], np.nextafter(L, 0) - off[sel])
    got = o.interp(*p)
    H = [np.pad(f, 1, mode="wrap") for f in F]                  # halo index = cell index + 1
    g = [p[a] / dx - 0.5 for a in range(3)]
    i0 = [np.floor(v).astype(np.int64) for v in g]              # -1 .. N-1
    fr = [v - np.floor(v) for v in g]
    for comp in range(3):
        acc = np.zeros(p.shape[1])
        for dk in (0, 1):
            for dj in (0, 1):
                for di in (0, 1):
                    wgt = ((fr[0] if di else 1 - fr[0]) * (fr[1] if dj else 1 - fr[1])
                           * (fr[2] if dk else 1 - fr[2]))
                    acc += wgt * H[comp][i0[2] + dk + 1, i0[1] + dj + 1, i0[0] + di + 1]
        assert np.max(np.abs(got[comp] - acc)) < 5e-14


# ------------------------------------------------------------------------------------------------
# a2 advance: closed-form drag relaxation (PAPER.md:51-57 with constant U; gravity per north_star)
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("ratio", [1e-3, 0.1, 1.0, 5.0, 45.0, 100.0])
@pytest.mark.parametrize("g", [(0.0, 0.0, 0.0), (0.3, -0.2, -9.81)])
def test_drag_relaxation_closed_form(oracle_lib, ratio, g):
    N = 8
    nu, rho = 1.5e-5, 1000.0
    o = oracle_lib.Oracle(N, 1, 1, 1, 64, nu=nu, rho_ratio=rho, g=g)
    U = np.array([0.7, -0.4, 0.25])
    o.set_fluid(*(np.full(N ** 3, c) for c in U))
    rng = np.random.default_rng(11)
    n = 16
    d = 2.0 * 10e-6 * np.exp(0.3 * rng.standard_normal(n))
    tau = rho * d * d / (18.0 * nu)
    dt = ratio * float(np.median(tau))
    X0 = rng.random((3, n)) * L
    V0 = rng.standard_normal((3, n))
    o.set_particles(X0[0], X0[1], X0[2], V0[0], V0[1], V0[2], d, np.arange(n))
    K = 7
    for _ in range(K):
        assert o.push(dt) in (0,)
        assert o.migrate() == 0
    out = o.get_particles()
    order = np.argsort(out["id"])
    t = K * dt
    for a, (xn, vn) in enumerate((("x", "vx"), ("y", "vy"), ("z", "vz"))):
        Vt = U[a] + tau * g[a]                       # terminal velocity U + tau_p g
        e = np.exp(-t / tau)
        Vk = Vt + (V0[a] - Vt) * e
        Xk = np.mod(X0[a] + Vt * t + (V0[a] - Vt) * tau * (1.0 - e), L)
        got_v = out[vn][order]
        got_x = out[xn][order]
        assert np.max(np.abs(got_v - Vk)) <= 1e-13 * max(1.0, np.max(np.abs(Vk))) * 10
        dxp = np.abs(got_x - Xk)
        dxp = np.minimum(dxp, L - dxp)
        assert np.max(dxp) <= 1e-13 * L * 10
    assert np.array_equal(out["d"][order], d)


def test_small_step_is_explicit_euler(oracle_lib):
    # dt/tau -> 0: one step equals explicit Euler of Eq. 6 to O((dt/tau)^2)
    N = 8
    nu, rho = 1.5e-5, 843.0
    o = oracle_lib.Oracle(N, 1, 1, 1, 8, nu=nu, rho_ratio=rho)
    U = 0.5
    o.set_fluid(*(np.full(N ** 3, U),) * 3)
    d = 2e-5
    tau = rho * d * d / (18 * nu)
    dt = 1e-3 * tau
    v0 = 2.0
    o.set_particles([1.0], [1.0], [1.0], [v0], [v0], [v0], [d], [0])
    o.push(dt)
    out = o.get_particles()
    euler_v = v0 - dt / tau * (v0 - U)
    assert abs(out["vx"][0] - euler_v) < 2 * (dt / tau) ** 2 * abs(v0 - U)
    assert abs(out["x"][0] - (1.0 + dt * v0)) < 2 * dt * (dt / tau) * abs(v0 - U)


# ------------------------------------------------------------------------------------------------
# a3/a4 classify + count: hand-placed particles (R-13/R-14)
# ------------------------------------------------------------------------------------------------
def ballistic_oracle(oracle_lib, N, P, cap):
    """Zero fluid and a huge tau: displacement = v*dt to ~1e-12 relative, so destinations are chosen by hand."""
    o = oracle_lib.Oracle(N, *P, cap, nu=1.5e-5, rho_ratio=1000.0)
    z = np.zeros(N ** 3)
    o.set_fluid(z, z, z)
    return o


BIG_D = 1.0   # tau = 1000/(18*1.5e-5) ~ 3.7e6 s


@pytest.mark.parametrize("P", [(3, 3, 3), (2, 2, 2), (1, 2, 3), (1, 1, 1), (4, 2, 1)])
def test_all_27_codes_hand_placed(oracle_lib, P):
    N = 24
    o = ballistic_oracle(oracle_lib, N, P, 64)
    Ls = [L / P[0], L / P[1], L / P[2]]
    dt = 1.0
    # one particle per (source subdomain, direction): start at the centre of s, move by d*L_sub
    X, V, want_code, src = [], [], [], []
    for s in range(P[0] * P[1] * P[2]):
        pc = (s % P[0], (s // P[0]) % P[1], s // (P[0] * P[1]))
        for c in range(27):
            dd = (c % 3 - 1, (c // 3) % 3 - 1, c // 9 - 1)
            X.append([(pc[a] + 0.5) * Ls[a] for a in range(3)])
            V.append([dd[a] * 0.75 * Ls[a] / dt for a in range(3)])
            want_code.append(c)
            src.append(s)
    X, V = np.array(X).T, np.array(V).T
    n = X.shape[1]
    o.set_particles(X[0], X[1], X[2], V[0], V[1], V[2], np.full(n, BIG_D), np.arange(n))
    assert o.push(dt) == 0
    out = o.get_particles()
    order = np.argsort(out["id"])
    assert np.array_equal(out["code"][order], np.array(want_code, dtype=np.uint8))
    tab = o.cnt_table()
    assert np.all(tab == 1)                     # a4: exactly one particle per (s, c)
    # positions are wrapped into the box
    for k in "xyz":
        assert np.all((out[k] >= 0) & (out[k] < L))
    # after migrate every particle sits in the subdomain that contains it (north_star invariant)
    assert o.migrate() == 0
    out2 = o.get_particles()
    slab = np.repeat(np.arange(o.P), out2["counts"])
    own = np.array([o.owner(x, y, z) for x, y, z in zip(out2["x"], out2["y"], out2["z"])])
    assert np.array_equal(slab, own)
    # receiver check against hand arithmetic
    for pid, s, c in zip(range(n), src, want_code):
        pc = (s % P[0], (s // P[0]) % P[1], s // (P[0] * P[1]))
        dd = (c % 3 - 1, (c // 3) % 3 - 1, c // 9 - 1)
        r = ((pc[0] + dd[0]) % P[0]) + P[0] * (((pc[1] + dd[1]) % P[1]) + P[1] * ((pc[2] + dd[2]) % P[2]))
        assert slab[np.nonzero(out2["id"] == pid)[0][0]] == r


def test_seam_wrap_and_face_rule(oracle_lib):
    N = 16
    o = ballistic_oracle(oracle_lib, N, (2, 2, 2), 16)
    eps = 1e-9
    face = L / 2
    Lb = np.nextafter(L, 0.0)
    #            x0          vx*dt      expected code dx, expected x'
    cases = [(eps, -2 * eps, -1, None),           # wraps below 0 -> top subdomain, code -1
             (Lb - eps, 3 * eps, +1, None),       # wraps above L -> bottom subdomain, code +1
             (face - eps, 2 * eps, +1, None),     # crosses the interior face upward
             (face + eps, -2 * eps, -1, None),    # crosses the interior face downward
             (face - eps, 0.5 * eps, 0, None),    # stays
             (1e-20, -2e-20, -1, Lb)]             # -tiny + L rounds to L -> clamped to L_below (R-19)
    n = len(cases)
    x0 = np.array([c[0] for c in cases])
    v = np.array([c[1] for c in cases])
    mid = np.full(n, 1.0)
    o.set_particles(x0, mid, mid, v, np.zeros(n), np.zeros(n), np.full(n, BIG_D), np.arange(n))
    assert o.push(1.0) == 0
    out = o.get_particles()
    order = np.argsort(out["id"])
    codes = out["code"][order].astype(int)
    assert list(codes % 3 - 1) == [c[2] for c in cases]
    assert np.all((codes // 3) % 3 == 1) and np.all(codes // 9 == 1)
    xs = out["x"][order]
    assert np.all((xs >= 0) & (xs < L))
    assert xs[5] == Lb
    # a particle exactly on a face belongs to the upper subdomain (half-open cells)
    assert o.owner(face, 1.0, 1.0) == 1 and o.owner(np.nextafter(face, 0), 1.0, 1.0) == 0


def test_jump_and_nonfinite_are_sticky_errors(oracle_lib):
    N = 16
    o = ballistic_oracle(oracle_lib, N, (4, 4, 4), 16)
    o.set_particles([1.0], [1.0], [1.0], [L / 4 * 1.6], [0.0], [0.0], [BIG_D], [0])
    assert o.push(1.0) == oracle_lib.ERR_JUMP
    assert o.status == oracle_lib.ERR_JUMP and o.migrate() == oracle_lib.ERR_JUMP
    o2 = ballistic_oracle(oracle_lib, N, (4, 4, 4), 16)
    o2.set_particles([1.0], [1.0], [1.0], [float("nan")], [0.0], [0.0], [BIG_D], [0])
    assert o2.push(1.0) == oracle_lib.ERR_JUMP
    o3 = ballistic_oracle(oracle_lib, N, (4, 4, 4), 16)
    assert o3.set_particles([L], [1.0], [1.0], [0.0], [0.0], [0.0], [BIG_D], [0]) == oracle_lib.ERR_RANGE
