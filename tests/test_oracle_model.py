"""Pins P5 (+ special cases) for the oracle's model functions: HH right-hand side and the RK4 increment.

Nothing here retypes the oracle's formula as the expected value: expectations come from special cases
with closed forms (Eq. 11-14 evaluated where tanh is 0 or saturated), from the order
of the integrator, from a fixed point, and from scipy's independent adaptive integrator.
"""
import numpy as np
from scipy.integrate import solve_ivp
from scipy.optimize import fsolve

import oracle
from workloads import HH_P_TRUE, MODEL_HH, MODEL_LINEAR, linear_matrix

P = HH_P_TRUE


def test_gate_kinetics_special_values():
    # At V = V_a: tanh = 0 => a_inf = 1/2, tau = tau0 + tau1 (Eq. 13-14 with Table 1 shifted -65 mV)
    for V, comp, tau in ((-40.0, 1, 0.5), (-60.0, 2, 8.0), (-55.0, 3, 6.0)):
        for a in (0.0, 0.3, 1.0):
            x = np.array([V, 0.2, 0.2, 0.2]); x[comp] = a
            F = oracle.rhs(MODEL_HH, x, P, 0.0)
            assert np.isclose(F[comp], (0.5 - a) / tau, rtol=1e-15, atol=1e-17)
    # Saturation: V -> +inf gives m_inf, n_inf -> 1, h_inf -> 0 (dV_h < 0), tau -> tau0
    F = oracle.rhs(MODEL_HH, [2000.0, 0.25, 0.25, 0.25], P, 0.0)
    assert np.allclose(F[1:], [(1 - 0.25) / 0.1, (0 - 0.25) / 1.0, (1 - 0.25) / 1.0], rtol=1e-14)
    F = oracle.rhs(MODEL_HH, [-2000.0, 0.25, 0.25, 0.25], P, 0.0)
    assert np.allclose(F[1:], [(0 - 0.25) / 0.1, (1 - 0.25) / 1.0, (0 - 0.25) / 1.0], rtol=1e-14)


def test_gate_kinetics_width_constants_from_table_1():
    # The special values above (tanh = 0 or +-1) do not see the MAGNITUDE of Delta-V_a.  One width away from the midpoint,
    # V = V_a + Delta-V_a, Eq. 13-14 give a_inf = (1 + tanh 1)/2 and tau = tau0 + tau1 (1 - tanh^2 1);
    # half a width away, tanh(1/2).  The numbers below are typed from Table 1 (n: 10, 30, 1.0, 5.0;
    # m: 25, 15, 0.1, 0.4; h: 5, -15, 1.0, 7.0) with V_a shifted by -65 mV (reading Delta-3), not read from the oracle.
    table1 = {1: (25.0 - 65.0, 15.0, 0.1, 0.4), 2: (5.0 - 65.0, -15.0, 1.0, 7.0), 3: (10.0 - 65.0, 30.0, 1.0, 5.0)}   # state order (V, m, h, n)
    for comp, (Va, dVa, tau0, tau1) in table1.items():
        for k in (1.0, 0.5, -1.0, 2.0):
            th = np.tanh(k)
            a_inf, tau = 0.5 + 0.5 * th, tau0 + tau1 * (1.0 - th * th)
            for a in (0.0, 0.35, 1.0):
                x = np.array([Va + k * dVa, 0.2, 0.2, 0.2]); x[comp] = a
                F = oracle.rhs(MODEL_HH, x, P, 0.0)
                assert np.isclose(F[comp], (a_inf - a) / tau, rtol=2e-14, atol=1e-16), (comp, k, a)
    # the three widths are different numbers: swapping any two of them must fail the loop above (guards the test itself)
    swapped = {1: table1[1][:1] + (30.0,) + table1[1][2:], 3: table1[3][:1] + (15.0,) + table1[3][2:]}
    for comp, (Va, dVa, tau0, tau1) in swapped.items():
        th = np.tanh(1.0)
        x = np.array([Va + dVa, 0.2, 0.2, 0.2]); x[comp] = 0.35
        F = oracle.rhs(MODEL_HH, x, P, 0.0)
        assert not np.isclose(F[comp], (0.5 + 0.5 * th - 0.35) / (tau0 + tau1 * (1 - th * th)), rtol=1e-3)


def test_voltage_equation_terms():
    # Eq. 11 in the (gNa,gK,gL,ENa,EK,EL,C) parametrisation: isolate each current.
    gNa, gK, gL, ENa, EK, EL, Cm = 100.0, 30.0, 0.5, 40.0, -80.0, -50.0, 2.0
    p = [gNa, gK, gL, ENa, EK, EL, Cm]
    V = -30.0
    assert np.isclose(oracle.rhs(MODEL_HH, [V, 0, 0, 0], p, 7.0)[0], (7.0 + gL * (EL - V)) / Cm, rtol=1e-15)
    assert np.isclose(oracle.rhs(MODEL_HH, [EL, 0, 0, 0], p, 3.0)[0], 3.0 / Cm, rtol=1e-15)
    # sodium only: V = EL kills the leak, n = 0 kills potassium; m^3 h
    assert np.isclose(oracle.rhs(MODEL_HH, [EL, 0.5, 0.4, 0], p, 0.0)[0], gNa * 0.125 * 0.4 * (ENa - EL) / Cm, rtol=1e-15)
    # potassium only: n^4
    assert np.isclose(oracle.rhs(MODEL_HH, [EL, 0, 0.4, 0.5], p, 0.0)[0], gK * 0.0625 * (EK - EL) / Cm, rtol=1e-15)
    # m and h enter asymmetrically (m cubed, h linear): swapping them changes the answer by 0.4^2/0.5^2... check ratio
    a = oracle.rhs(MODEL_HH, [EL, 0.5, 0.4, 0], p, 0.0)[0]
    b = oracle.rhs(MODEL_HH, [EL, 0.4, 0.5, 0], p, 0.0)[0]
    assert np.isclose(a / b, (0.125 * 0.4) / (0.064 * 0.5), rtol=1e-14)


def test_fixed_point_stays_at_rest():
    f = lambda x: oracle.rhs(MODEL_HH, x, P, 0.0)
    xs = fsolve(f, [-65.0, 0.05, 0.6, 0.3], xtol=1e-14)
    assert np.abs(f(xs)).max() < 1e-10 and -80 < xs[0] < -50
    g = oracle.step_increment(MODEL_HH, xs, P, 0.0, 0.0, 0.02)
    assert np.abs(g).max() < 1e-11


def test_rk4_is_fourth_order_and_matches_adaptive_integrator():
    x0 = np.array([-30.0, 0.4, 0.3, 0.5])     # on the upstroke: large derivatives
    I0, I1, T = 4.0, 9.0, 0.08

    def integrate(nsteps):
        x, h = x0.copy(), T / nsteps
        for k in range(nsteps):
            a, b = I0 + (I1 - I0) * k / nsteps, I0 + (I1 - I0) * (k + 1) / nsteps
            x = x + oracle.step_increment(MODEL_HH, x, P, a, b, h)
        return x

    # reference: scipy's adaptive integrator on the same ODE with linearly interpolated current
    sol = solve_ivp(lambda t, x: oracle.rhs(MODEL_HH, x, P, I0 + (I1 - I0) * t / T), (0, T), x0, rtol=1e-13, atol=1e-14,
                    method="DOP853")
    ref = sol.y[:, -1]
    xs = [integrate(n) for n in (16, 32, 64, 128, 256)]
    assert np.abs(xs[-1] - ref).max() < 1e-10
    # self-convergence: successive differences fall by 2^4 = 16 per halving once in the asymptotic regime
    d = [np.abs(xs[i] - xs[i + 1]).max() for i in range(4)]
    ratios = [d[i] / d[i + 1] for i in range(1, 3)]
    assert all(13.0 < r < 19.0 for r in ratios), (d, ratios)


def test_rk4_stage_weights_on_a_polynomial_rhs():
    # With all conductances 0 and C = 1: dV/dt = I(t), linear in t over the step, so one RK4 step is exact:
    # g_V = dt (I0 + I1)/2 -- pins the (1,2,2,1)/6 weights and the midpoint current (G5).
    p = [0, 0, 0, 0, 0, 0, 1.0]
    g = oracle.step_increment(MODEL_HH, [-65.0, 0.1, 0.2, 0.3], p, 2.0, 5.0, 0.04)
    assert np.isclose(g[0], 0.04 * 3.5, rtol=1e-15)
    # a gate at fixed V relaxes exponentially: a(dt) - a0 = (a_inf - a0)(1 - exp(-dt/tau)); RK4 reproduces the
    # Taylor polynomial 1 - z + z^2/2 - z^3/6 + z^4/24 of exp(-z) exactly (V is constant since dV/dt = 0).
    V, a0, dt = -55.0, 0.9, 0.3          # n gate at V = V_n: a_inf = 0.5, tau = 6
    g = oracle.step_increment(MODEL_HH, [V, 0.1, 0.2, a0], p, 0.0, 0.0, dt)
    z = dt / 6.0
    assert np.isclose(g[3], (0.5 - a0) * (z - z**2 / 2 + z**3 / 6 - z**4 / 24), rtol=1e-13)
    assert g[0] == 0.0


def test_linear_map_reproduces_A():
    for D in (1, 2, 3, 4):
        A = linear_matrix(D) if D <= 2 else np.arange(1.0, D * D + 1).reshape(D, D) / 10
        assert oracle.model_np(MODEL_LINEAR, D) == D * D
        for k in range(D):
            e = np.zeros(D); e[k] = 1.0
            g = oracle.step_increment(MODEL_LINEAR, e, A.ravel(), 0, 0, 1.0)
            assert np.allclose(g + e, A[:, k], rtol=0, atol=1e-16)
    assert oracle.model_np(MODEL_HH, 4) == 7
