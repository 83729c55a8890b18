"""Pins of the oracle's two-stage RK2 with per-stage migration (R-25;
PAPER.md:64, :150-164, :175-177).  Checked against the closed form of Heun's method on the linear drag equation, the
exact solution (order of convergence), and decomposition independence -- never against the oracle itself."""
import math

import numpy as np
import pytest

L = 6.283185307179586
NU, RHO = 1.5e-5, 1000.0
F8 = ("x", "y", "z", "vx", "vy", "vz", "d", "id")


def by_id(p):
    order = np.argsort(p["id"])
    return {k: p[k][order] for k in F8}


@pytest.mark.parametrize("z", [0.01, 0.2, 0.5])
def test_heun_amplification_factor_and_position_polynomial(oracle_lib, z):
    """Constant U and g: Heun on dV/dt = -(V - U)/tau + g gives V_k - Vt = (1 - z + z^2/2)^k (V_0 - Vt), z = dt/tau, and
    X_k = X_0 + sum_j dt/2 (V_j + V1_j) with V1_j = V_j + dt K1_j; both written out here in plain numpy."""
    N = 8
    g = (0.3, -0.2, -9.81)
    U = np.array([0.7, -0.4, 0.25])
    d = 300e-6
    tau = RHO * d * d / (18 * NU)
    dt = z * tau
    o = oracle_lib.Oracle(N, 1, 1, 1, 8, nu=NU, rho_ratio=RHO, g=g)
    o.set_fluid(*(np.full(N ** 3, c) for c in U))
    x0 = np.array([1.0, 2.0, 3.0])
    v0 = np.array([1.5, -0.5, 0.8])
    o.set_particles([x0[0]], [x0[1]], [x0[2]], [v0[0]], [v0[1]], [v0[2]], [d], [0])
    K = 9
    x, v = x0.copy(), v0.copy()
    vt = U + tau * np.array(g)
    for k in range(K):
        assert o.step_rk2(dt) == 0
        k1 = (U - v) / tau + np.array(g)
        v1 = v + dt * k1
        k2 = (U - v1) / tau + np.array(g)
        x = x + 0.5 * dt * (v + v1)
        v = v + 0.5 * dt * (k1 + k2)
    out = o.get_particles()
    amp = (1 - z + 0.5 * z * z) ** K
    for a, (xn, vn) in enumerate((("x", "vx"), ("y", "vy"), ("z", "vz"))):
        assert abs(out[vn][0] - (vt[a] + amp * (v0[a] - vt[a]))) <= 1e-12 * max(1.0, abs(vt[a]))
        assert abs(out[vn][0] - v[a]) <= 1e-12 * max(1.0, abs(v[a]))
        dx = abs(out[xn][0] - math.fmod(x[a] + 8 * L, L))
        assert min(dx, L - dx) <= 1e-12 * L
    o.close()


def test_second_order_convergence_to_the_exact_solution(oracle_lib):
    N = 8
    U = np.array([0.5, 0.0, -0.25])
    d = 300e-6
    tau = RHO * d * d / (18 * NU)
    T = 0.4 * tau
    errs = []
    for steps in (4, 8, 16, 32):
        o = oracle_lib.Oracle(N, 1, 1, 1, 8, nu=NU, rho_ratio=RHO)
        o.set_fluid(*(np.full(N ** 3, c) for c in U))
        o.set_particles([1.0], [1.0], [1.0], [2.0], [-1.0], [0.5], [d], [0])
        for _ in range(steps):
            assert o.step_rk2(T / steps) == 0
        out = o.get_particles()
        v_exact = U[0] + (2.0 - U[0]) * math.exp(-T / tau)
        x_exact = 1.0 + U[0] * T + (2.0 - U[0]) * tau * (1 - math.exp(-T / tau))
        errs.append((abs(out["vx"][0] - v_exact), abs(out["x"][0] - x_exact)))
        o.close()
    for (ev0, ex0), (ev1, ex1) in zip(errs, errs[1:]):
        assert 3.5 < ev0 / ev1 < 4.5          # global error O(dt^2): halving dt divides it by 4
        assert 3.5 < ex0 / ex1 < 4.6


def random_inertial(rng, n, d):
    X = rng.random((3, n)) * L
    V = rng.standard_normal((3, n)) * 1.5
    return {"x": X[0], "y": X[1], "z": X[2], "vx": V[0], "vy": V[1], "vz": V[2],
            "d": np.full(n, d) * np.exp(0.2 * rng.standard_normal(n)), "id": rng.permutation(n).astype(np.int64)}


@pytest.mark.parametrize("drag_model", [0, 1])
def test_result_does_not_depend_on_the_decomposition(oracle_lib, drag_model):
    """The same particles on 1x1x1, 2x2x2 and 3x2x1 subdomains, several RK2 steps in a non-uniform field: identical state
    per id, bit for bit.  Stage 2 reads X0, V0 and K1 of stage 1 after a migration, so this fails unless all 17 arrays
    travel with the particle (and unless the stage-2 classification is relative to the slab the particle sits in)."""
    N = 12
    rng = np.random.default_rng(3)
    c = (np.arange(N) + 0.5) * (L / N)
    Xc, Yc, Zc = np.meshgrid(c, c, c, indexing="ij")          # x fastest in memory: transpose below
    u = (np.sin(Xc) * np.cos(2 * Yc)).transpose(2, 1, 0).ravel()
    v = (np.cos(Xc) * np.sin(Zc)).transpose(2, 1, 0).ravel()
    w = (np.sin(Yc + Zc)).transpose(2, 1, 0).ravel()
    n = 4000
    parts = random_inertial(rng, n, 300e-6)
    dt = 0.12 if drag_model == 0 else 0.05        # f up to ~5 shortens tau_eff: keep dt/tau_eff well below 2
    results = []
    for P in ((1, 1, 1), (2, 2, 2), (3, 2, 1)):
        o = oracle_lib.Oracle(N, *P, 4 * n // (P[0] * P[1] * P[2]) + 64, nu=NU, rho_ratio=RHO, g=(0, 0, -9.81),
                              drag_model=drag_model)
        o.set_fluid(u, v, w)
        assert o.set_particles(*(parts[k] for k in F8)) == 0
        moved = 0
        for _ in range(5):
            assert o.rk2_stage1(dt) == 0 and o.migrate() == 0
            moved += o.n_migrated_last
            assert o.rk2_stage2(dt) == 0 and o.migrate() == 0
            moved += o.n_migrated_last
        out = o.get_particles()
        # containment after the second migration
        cells = [np.minimum(np.floor(out[k] * (N / L)).astype(np.int64), N - 1) for k in "xyz"]
        owner = cells[0] // (N // P[0]) + P[0] * (cells[1] // (N // P[1]) + P[1] * (cells[2] // (N // P[2])))
        assert np.array_equal(owner, np.repeat(np.arange(P[0] * P[1] * P[2]), out["counts"]))
        results.append((by_id(out), moved))
        o.close()
    assert results[0][1] == 0 and results[1][1] > n // 10       # nothing migrates on 1x1x1; a lot does on 2x2x2
    for other, _ in results[1:]:
        for k in F8:
            assert np.array_equal(results[0][0][k], other[k]), k


def test_stage2_needs_the_migration_of_stage1(oracle_lib):
    o = oracle_lib.Oracle(8, 2, 1, 1, 8)
    z = np.zeros(512)
    o.set_fluid(z, z, z)
    o.set_particles([1.0], [1.0], [1.0], [0.1], [0.0], [0.0], [3e-4], [0])
    assert o.rk2_stage1(0.1) == 0
    assert o.rk2_stage2(0.1) != 0            # ORC_ERR_STATE: the codes of stage 1 have not been migrated


@pytest.mark.parametrize("d,dt", [(300e-6, 0.02), (600e-6, 0.05)])
def test_heun_with_nonlinear_drag_reevaluates_f_per_stage(oracle_lib, d, dt):
    """drag_model = 1 inside the two-stage RK2 (f = 1 + 0.15 Re_p^0.687 is part of Eq. 6, and the
    integrator has two stages, so each stage evaluates f from ITS slip): one particle, uniform U, gravity on, Heun
    written out here with libm pow -- f1 from |V0 - U|, f2 from |V1 - U|.  The variant that reuses the slip of V0 in
    stage 2 (a plausible mistake the decomposition-independence pin cannot see) must be far outside the tolerance."""
    N = 8
    g = np.array([0.0, 0.0, -9.81])
    U = np.array([0.6, -0.3, 0.2])
    tau_p = RHO * d * d / (18 * NU)
    o = oracle_lib.Oracle(N, 1, 1, 1, 8, nu=NU, rho_ratio=RHO, g=tuple(g), drag_model=1)
    o.set_fluid(*(np.full(N ** 3, c) for c in U))
    x0 = np.array([1.0, 2.0, 3.0])
    v0 = np.array([2.5, -1.5, 1.0])
    o.set_particles([x0[0]], [x0[1]], [x0[2]], [v0[0]], [v0[1]], [v0[2]], [d], [0])

    def f_of(v):
        return 1.0 + 0.15 * (d * float(np.linalg.norm(v - U)) / NU) ** 0.687

    assert f_of(v0) > 1.5                      # Re_p = O(10..100): the correction matters
    assert dt * f_of(v0) / tau_p < 0.5         # the paper's regime for an explicit scheme
    x, v = x0.copy(), v0.copy()
    xw, vw = x0.copy(), v0.copy()              # the wrong variant: stage 2 with the f of stage 1
    K = 6
    for _ in range(K):
        assert o.step_rk2(dt) == 0
        k1 = (U - v) * (f_of(v) / tau_p) + g
        v1 = v + dt * k1
        k2 = (U - v1) * (f_of(v1) / tau_p) + g
        x = x + 0.5 * dt * (v + v1)
        v = v + 0.5 * dt * (k1 + k2)
        k1w = (U - vw) * (f_of(vw) / tau_p) + g
        v1w = vw + dt * k1w
        k2w = (U - v1w) * (f_of(vw) / tau_p) + g
        xw = xw + 0.5 * dt * (vw + v1w)
        vw = vw + 0.5 * dt * (k1w + k2w)
    out = o.get_particles()
    got_v = np.array([out["vx"][0], out["vy"][0], out["vz"][0]])
    got_x = np.array([out["x"][0], out["y"][0], out["z"][0]])
    assert np.all(np.abs(got_v - v) <= 1e-12 * np.maximum(1.0, np.abs(v)))
    dx = np.abs(got_x - np.mod(x, L))
    assert np.all(np.minimum(dx, L - dx) <= 1e-12 * L)
    assert np.max(np.abs(got_v - vw)) > 1e-6   # the pin discriminates: frozen-f Heun is not what the oracle computes
    o.close()
