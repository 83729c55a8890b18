"""Pins of the oracle's nonlinear drag (R-23): the drag factor
f = 1 + 0.15 Re_p^0.687, Re_p = d |V - U| / nu (Eq. 7-8), frozen at the start of the step.
Everything here is checked against libm / closed forms / root finding, never against the oracle itself."""
import math

import numpy as np
import pytest

L = 6.283185307179586
NU, RHO = 1.5e-5, 1000.0


def f_ref(d, w):
    return 1.0 + 0.15 * (d * w / NU) ** 0.687


def test_pow_0687_against_libm(oracle_lib):
    rng = np.random.default_rng(5)
    R = np.concatenate([10.0 ** rng.uniform(-8, 8, 4000), 2.0 ** np.arange(-40, 41, dtype=np.float64),
                        np.nextafter(2.0 ** np.arange(-5, 6, dtype=np.float64), 0.0),        # just below powers of two
                        np.array([1.4142135623730951, np.nextafter(1.4142135623730951, 2.0), 0.7071067811865476])])
    got = np.array([oracle_lib.pow_0687(r) for r in R])
    want = np.power(R, 0.687)
    assert np.max(np.abs(got - want) / want) <= 2e-14
    # the drag factor itself (what the step uses) is then good to a few ulp
    assert np.max(np.abs((1 + 0.15 * got) - (1 + 0.15 * want)) / (1 + 0.15 * want)) <= 1e-14


def test_pow_0687_special_values_and_monotone(oracle_lib):
    assert oracle_lib.pow_0687(0.0) == 0.0                      # no slip -> f = 1 exactly
    assert oracle_lib.pow_0687(1e-310) == 0.0                   # below the smallest normal number
    assert oracle_lib.pow_0687(1.0) == 1.0                      # f(Re = 1) = 1.15
    assert math.isnan(oracle_lib.pow_0687(float("nan")))
    assert oracle_lib.pow_0687(float("inf")) == float("inf")
    R = 10.0 ** np.linspace(-6, 6, 2001)
    v = np.array([oracle_lib.pow_0687(r) for r in R])
    assert np.all(np.diff(v) > 0)


def one_particle(oracle_lib, U, g, d, v0, drag_model, N=8):
    o = oracle_lib.Oracle(N, 1, 1, 1, 8, nu=NU, rho_ratio=RHO, g=g, drag_model=drag_model)
    o.set_fluid(*(np.full(N ** 3, c) for c in U))
    o.set_particles([1.0], [2.0], [3.0], [v0[0]], [v0[1]], [v0[2]], [d], [0])
    return o


@pytest.mark.parametrize("d,slip", [(20e-6, 0.5), (100e-6, 2.0), (400e-6, 5.0), (20e-6, 1e-9)])
def test_one_step_closed_form_with_frozen_f(oracle_lib, d, slip):
    """One step is the exact solution of dV/dt = -f (V - U)/tau_p + g with U and f frozen at the start of the step."""
    U = np.array([0.3, -0.2, 0.1])
    g = np.array([0.0, 0.4, -9.81])
    dirn = np.array([2.0, -1.0, 2.0]) / 3.0
    v0 = U + slip * dirn
    tau_p = RHO * d * d / (18 * NU)
    f = f_ref(d, slip)
    tau = tau_p / f
    for ratio in (0.05, 1.0, 20.0):
        dt = ratio * tau
        o = one_particle(oracle_lib, U, g, d, v0, 1)
        assert o.push(dt) == 0
        out = o.get_particles()
        e = math.exp(-dt / tau)
        for a, (xn, vn, x0) in enumerate((("x", "vx", 1.0), ("y", "vy", 2.0), ("z", "vz", 3.0))):
            vt = U[a] + tau * g[a]
            v1 = vt + (v0[a] - vt) * e
            x1 = math.fmod(x0 + vt * dt + (v0[a] - vt) * tau * (1 - e) + 4 * L, L)
            assert abs(out[vn][0] - v1) <= 1e-12 * max(1.0, abs(v1))
            dx = abs(out[xn][0] - x1)
            assert min(dx, L - dx) <= 1e-12 * L
        o.close()


def test_settling_speed_solves_w_f_equals_tau_g(oracle_lib):
    """Still fluid + gravity: the velocity converges to the root of w f(Re(w)) = tau_p g (the terminal speed under the
    nonlinear drag), found here by bisection with libm."""
    d, gz = 200e-6, -9.81
    tau_p = RHO * d * d / (18 * NU)
    o = one_particle(oracle_lib, (0.0, 0.0, 0.0), (0.0, 0.0, gz), d, (0.0, 0.0, 0.0), 1)
    dt = 0.2 * tau_p
    for _ in range(400):
        assert o.push(dt) == 0
        assert o.migrate() == 0
    w = -o.get_particles()["vz"][0]
    lo, hi = 0.0, tau_p * abs(gz)
    for _ in range(200):
        mid = 0.5 * (lo + hi)
        if mid * f_ref(d, mid) < tau_p * abs(gz):
            lo = mid
        else:
            hi = mid
    assert abs(w - lo) <= 1e-10 * lo
    assert w < 0.75 * tau_p * abs(gz)          # well below the Stokes settling speed: the correction matters here
    o.close()


def test_zero_slip_is_stokes_bit_for_bit_and_small_slip_tends_to_it(oracle_lib):
    U = (0.25, 0.5, -0.75)
    d = 30e-6
    dt = 3e-3
    a = one_particle(oracle_lib, U, (0.0, 0.0, -9.81), d, U, 0)
    b = one_particle(oracle_lib, U, (0.0, 0.0, -9.81), d, U, 1)
    a.push(dt); b.push(dt)
    pa, pb = a.get_particles(), b.get_particles()
    for k in ("x", "y", "z", "vx", "vy", "vz"):
        assert pa[k][0] == pb[k][0]            # V = U: Re = 0, f = 1 exactly
    v0 = (U[0] + 1e-7, U[1], U[2])
    a = one_particle(oracle_lib, U, (0.0, 0.0, 0.0), d, v0, 0)
    b = one_particle(oracle_lib, U, (0.0, 0.0, 0.0), d, v0, 1)
    a.push(dt); b.push(dt)
    # f - 1 = 0.15 Re^0.687 with Re = d 1e-7 / nu = 2e-7: a relative change of the slip decay of order 4e-6
    assert abs(a.get_particles()["vx"][0] - b.get_particles()["vx"][0]) <= 1e-5 * 1e-7


def test_drag_model_argument_is_checked(oracle_lib):
    with pytest.raises(ValueError):
        oracle_lib.Oracle(8, 1, 1, 1, 8, drag_model=2)
