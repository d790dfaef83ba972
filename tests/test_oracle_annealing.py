"""Pins for the simulated annealing of the dynamics term (first half; Eq. 10):
beta multiplies A_d only, starts at beta0, grows by f_beta = (1/beta0)^(1/N_cool) per iteration until it is 1."""
import numpy as np
import pytest

from oracle import OracleChain
from workloads import make_workload


def test_schedule_is_eq10():
    w = make_workload(0, M=8)
    o = OracleChain.from_workload(w)
    o.sweep(3, seed=1)                                   # annealing starts at the sweep index of the call
    beta0, n_cool = 0.01, 50
    o.set_annealing(beta0, n_cool)
    f = (1.0 / beta0) ** (1.0 / n_cool)                  # Eq. 10
    beta = beta0
    for k in range(n_cool + 5):
        assert o.annealing_beta() == pytest.approx(min(beta, 1.0) if k < n_cool else 1.0, rel=1e-13), k
        o.sweep(1, seed=1)
        beta *= f
    assert o.annealing_beta() == 1.0


@pytest.mark.parametrize("disc", [0, 1])
def test_beta_multiplies_the_dynamics_term_only(disc):
    w = make_workload(2, M=12)
    o = OracleChain.from_workload(w); o.set_discretisation(disc)
    x, p = o.get_path()
    A1 = float(o.full_action())
    # measurement part alone: the action with the dynamics weight switched off is what beta -> 0 leaves
    o0 = OracleChain(w.model, 4, 1, 12, w.dt, w.Rm, np.zeros(4), w.p0[0]); o0.set_discretisation(disc)
    o0.set_data(w.y[0], w.I[0]); o0.set_proposal(w.w_state, w.w_param); o0.set_path(x)
    Ao = float(o0.full_action())
    o.set_annealing(0.25, 10)
    Ab = float(o.full_action())
    assert Ab == pytest.approx(Ao + 0.25 * (A1 - Ao), rel=1e-13)
    # local and parameter Delta-A are differences of THAT action
    rng = np.random.default_rng(0)
    for n in (0, 5, 12):
        xp = x[n] + w.w_state * rng.normal(size=4)
        dA, S = o.site_delta_A(n, xp)
        X2 = x.copy(); X2[n] = xp
        assert abs(dA - float(o.full_action(X2) - o.full_action())) <= 1e-13 * (abs(Ab) + S)
    dA, S = o.param_delta_A(0, p[0] * 1.001)
    p2 = p.copy(); p2[0] *= 1.001
    assert abs(dA - float(o.full_action(None, p2) - o.full_action())) <= 1e-13 * (abs(Ab) + S)


def test_annealed_chain_telescopes_and_ends_on_the_plain_chain_rule():
    w = make_workload(2, M=30)
    o = OracleChain.from_workload(w)
    o.set_annealing(0.05, 6)
    for t in range(9):
        beta = o.annealing_beta()
        A_before = float(o.full_action())                # at this sweep's beta
        o.sweep(1, seed=4)
        tr = o.trace()
        acc_sum = tr["dA"][tr["acc"] == 1].sum() + np.nansum(np.where(tr["accp"] == 1, tr["dAp"], 0.0))
        # re-evaluate the new path at the SAME beta the sweep used
        q = OracleChain.from_workload(w); q.set_path(o.get_path()[0]); q.set_params(o.get_path()[1])
        Aq1 = float(q.full_action())
        q0 = OracleChain(w.model, 4, 1, 30, w.dt, w.Rm, np.zeros(4), o.get_path()[1]); q0.set_data(w.y[0], w.I[0]); q0.set_path(o.get_path()[0])
        Aq0 = float(q0.full_action())
        A_after = Aq0 + beta * (Aq1 - Aq0)
        assert abs((A_after - A_before) - acc_sum) <= 1e-10 * abs(A_before), t
    assert o.annealing_beta() == 1.0
    # with beta back at 1 the chain continues exactly like an un-annealed chain started from the same state and sweep index
    ref = OracleChain.from_workload(w); ref.set_params(o.get_path()[1]); ref.set_path(o.get_path()[0]); ref.sweep_index = o.sweep_index
    o.sweep(3, seed=4); ref.sweep(3, seed=4)
    assert np.array_equal(o.get_path()[0], ref.get_path()[0])
