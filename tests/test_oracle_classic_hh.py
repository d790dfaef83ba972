"""Pins for the classic Hodgkin-Huxley rate functions (model 2; BASELINE.json "standard HH").

The rate functions are the textbook ones (Hodgkin & Huxley 1952, rest shifted to -65 mV).  What fixes the oracle's
implementation: the textbook resting values of the gating variables and time constants, the removable singularities of
alpha_m and alpha_n, the asymptotic limits, finite-difference consistency across the singular points, the V equation
shared with model 1, RK4 convergence order, and the generic Delta-A pins run on this model."""
import numpy as np
import pytest

import oracle
from oracle import OracleChain
from workloads import MODEL_HH, MODEL_HH_CLASSIC, HH_P_TRUE, make_workload

P = HH_P_TRUE


def rates(V):
    """(alpha, beta) of m, h, n recovered from the oracle's right-hand side: F_a(a=0) = alpha, F_a(a=1) = -beta."""
    F0 = oracle.rhs(MODEL_HH_CLASSIC, [V, 0.0, 0.0, 0.0], P, 0.0)
    F1 = oracle.rhs(MODEL_HH_CLASSIC, [V, 1.0, 1.0, 1.0], P, 0.0)
    return F0[1:], -F1[1:]


def test_textbook_resting_values():
    al, be = rates(-65.0)
    inf = al / (al + be)
    tau = 1.0 / (al + be)
    # m_inf, h_inf, n_inf at rest: 0.0529, 0.5961, 0.3177 (every textbook table of the 1952 model)
    assert np.allclose(inf, [0.05293, 0.59612, 0.31768], atol=2e-5)
    # beta_m(rest) = 4, alpha_h(rest) = 0.07, beta_n(rest) = 0.125 exactly
    assert be[0] == pytest.approx(4.0, rel=1e-15) and al[1] == pytest.approx(0.07, rel=1e-15) and be[2] == pytest.approx(0.125, rel=1e-15)
    # time constants at rest: tau_m ~ 0.237 ms, tau_h ~ 8.5 ms, tau_n ~ 5.5 ms
    assert np.allclose(tau, [0.2367, 8.516, 5.458], rtol=2e-3)


def test_removable_singularities_and_limits():
    al, _ = rates(-40.0)
    assert al[0] == pytest.approx(1.0, rel=1e-15)            # alpha_m(-40) = 0.1 * 10
    al, _ = rates(-55.0)
    assert al[2] == pytest.approx(0.1, rel=1e-15)            # alpha_n(-55) = 0.01 * 10
    # continuity and slope across the singular points: u/(1-e^-u) = 1 + u/2 + u^2/12 - ...
    for V0, scale, k in ((-40.0, 1.0, 0), (-55.0, 0.1, 2)):
        for dV in (1e-9, 1e-6, 1e-3, -1e-9, -1e-6, -1e-3):
            u = dV / 10.0
            al, _ = rates(V0 + dV)
            assert al[k] == pytest.approx(scale * (1 + u / 2 + u * u / 12), rel=1e-13)
    # far limits: alpha_m ~ 0.1 (V+40) for large V, -> 0 for very negative V; beta_h -> 1, 0
    al, be = rates(200.0)
    assert al[0] == pytest.approx(24.0, rel=1e-9) and be[1] == pytest.approx(1.0, rel=1e-9)
    al, be = rates(-300.0)
    assert 0 <= al[0] < 1e-9 and 0 <= be[1] < 1e-11


def test_rates_match_the_formulas_on_a_grid_in_extended_precision():
    V = np.linspace(-120, 80, 401).astype(np.longdouble) + np.longdouble(0.0137)
    ld = np.longdouble
    am = ld(0.1) * (V + 40) / (1 - np.exp(-(V + 40) / 10)); bm = 4 * np.exp(-(V + 65) / 18)
    ah = ld(0.07) * np.exp(-(V + 65) / 20); bh = 1 / (1 + np.exp(-(V + 35) / 10))
    an = ld(0.01) * (V + 55) / (1 - np.exp(-(V + 55) / 10)); bn = ld(0.125) * np.exp(-(V + 65) / 80)
    for i, v in enumerate(V):
        al, be = rates(float(v))
        ref_a = np.array([am[i], ah[i], an[i]], dtype=np.float64); ref_b = np.array([bm[i], bh[i], bn[i]], dtype=np.float64)
        assert np.allclose(al, ref_a, rtol=2e-14, atol=0) and np.allclose(be, ref_b, rtol=2e-14, atol=0), float(v)


def test_voltage_equation_is_shared_and_rest_is_nearly_stationary():
    x = [-30.0, 0.4, 0.3, 0.6]
    assert oracle.rhs(MODEL_HH_CLASSIC, x, P, 3.0)[0] == oracle.rhs(MODEL_HH, x, P, 3.0)[0]
    al, be = rates(-65.0)
    rest = np.concatenate([[-65.0], al / (al + be)])
    F = oracle.rhs(MODEL_HH_CLASSIC, rest, P, 0.0)
    assert np.max(np.abs(F[1:])) < 1e-15                      # gates exactly at their steady state
    assert abs(F[0]) < 0.01                                   # -65 mV is the resting potential of these parameters to ~0.01 mV/ms


def test_rk4_increment_converges_at_fourth_order():
    x = np.array([-50.0, 0.2, 0.4, 0.45])
    def flow(dt, n):
        y = x.copy()
        for _ in range(n):
            y = y + oracle.step_increment(MODEL_HH_CLASSIC, y, P, 7.0, 7.0, dt)
        return y
    ref = flow(0.08 / 64, 64)
    e1 = np.abs(flow(0.08, 1) - ref).max(); e2 = np.abs(flow(0.04, 2) - ref).max(); e4 = np.abs(flow(0.02, 4) - ref).max()
    assert 10 < e1 / e2 < 24 and 10 < e2 / e4 < 24, (e1, e2, e4)


@pytest.mark.parametrize("disc", [0, 1])
def test_delta_A_brute_force_and_invariants_on_the_classic_model(disc):
    w = make_workload(2, M=16, kinetics="classic")
    assert w.model == MODEL_HH_CLASSIC
    o = OracleChain.from_workload(w); o.set_discretisation(disc)
    rng = np.random.default_rng(4)
    x, p = o.get_path()
    A0 = o.full_action()
    for n in range(o.M + 1):
        xp = x[n] + w.w_state * rng.normal(size=4)
        dA, S = o.site_delta_A(n, xp)
        X2 = x.copy(); X2[n] = xp
        assert abs(dA - float(o.full_action(X2) - A0)) <= 1e-15 * float(abs(A0)) * 20 + 1e-13 * S, n
    for l in range(7):
        pl = p[l] + w.w_param[l] * rng.normal()
        dA, S = o.param_delta_A(l, pl)
        p2 = p.copy(); p2[l] = pl
        assert abs(dA - float(o.full_action(None, p2) - A0)) <= 1e-15 * float(abs(A0)) * 20 + 1e-13 * S, l
    A_prev = o.full_action()
    for t in range(4):
        o.sweep(1, seed=3)
        tr = o.trace()
        acc_sum = tr["dA"][tr["acc"] == 1].sum() + np.nansum(np.where(tr["accp"] == 1, tr["dAp"], 0.0))
        A_now = o.full_action()
        assert abs(float(A_now - A_prev) - acc_sum) <= 1e-11 * float(abs(A_prev))
        A_prev = A_now


def test_classic_truth_spikes_under_the_config_current():
    # the classic model fires under the config current (1 spike in the 5 ms of M = 256 is not
    # guaranteed; use the M = 4096 window: several spikes, V within [-80, 45] mV)
    w = make_workload(2, M=4096, kinetics="classic")
    V = w.x_true[0, :, 0]
    spikes = np.sum((V[1:] > 0) & (V[:-1] <= 0))
    assert spikes >= 3 and V.min() > -85 and V.max() < 50, (spikes, V.min(), V.max())
