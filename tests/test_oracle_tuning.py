"""Pins for the step-size auto-tuning (second half):
    Delta_i <- Delta_i [1 + alpha (N_acc,i / N_skip - f_acc)]   every N_skip-th iteration, for every path component and
parameter, N_acc,i = accepted changes of component i over the past N_skip iterations."""
import numpy as np
import pytest

from oracle import OracleChain
from workloads import MODEL_LINEAR, make_workload, linear_truth


@pytest.mark.parametrize("mode", [0, 1])
def test_adjustment_rule_from_the_traced_decisions(mode):
    w = make_workload(2, M=40)
    o = OracleChain.from_workload(w); o.set_update_mode(mode)
    o.sweep(2, seed=3)
    n_skip, f_acc, alpha = 5, 0.23, 0.1
    o.set_tuning(True, n_skip, f_acc, alpha)
    ws, wp = o.get_widths()
    assert np.array_equal(ws, np.tile(w.w_state, (41, 1))) and np.array_equal(wp, w.w_param)
    for rnd in range(3):
        Ns, Np_ = np.zeros((41, 4)), np.zeros(7)
        for t in range(n_skip):
            if t:                                            # no adjustment inside the window
                assert np.array_equal(o.get_widths()[0], ws)
            o.sweep(1, seed=3)
            tr = o.trace()
            Ns += tr["acc"] if mode == 1 else tr["acc"][:, None]     # a joint move changes every component of its site
            Np_ += tr["accp"]
        ws = ws * (1.0 + alpha * (Ns / n_skip - f_acc))
        wp = wp * (1.0 + alpha * (Np_ / n_skip - f_acc))
        gs, gp = o.get_widths()
        assert np.array_equal(gs, ws) and np.array_equal(gp, wp), rnd
    o.set_tuning(False)
    o.sweep(7, seed=3)
    assert np.array_equal(o.get_widths()[0], ws)             # frozen after the initialisation phase


def test_untuned_chain_is_unchanged_and_frozen_parameters_stay_frozen():
    w = make_workload(0, M=30)                               # parameters frozen (width 0)
    a = OracleChain.from_workload(w); b = OracleChain.from_workload(w)
    b.set_tuning(True, 4, 0.23, 0.0)                         # alpha = 0: the rule is the identity
    a.sweep(12, seed=1); b.sweep(12, seed=1)
    assert np.array_equal(a.get_path()[0], b.get_path()[0])
    c = OracleChain.from_workload(w); c.set_tuning(True, 4, 0.23, 0.05); c.sweep(12, seed=1)
    assert np.all(c.get_widths()[1] == 0.0)
    assert not np.array_equal(c.get_widths()[0], a.get_widths()[0])


def test_tuning_drives_the_acceptance_to_the_target():
    rng = np.random.default_rng(3)
    M = 64
    A, xt, y = linear_truth(M, rng)
    o = OracleChain(MODEL_LINEAR, 2, 1, M, 1.0, 100.0, [100.0, 100.0], A.ravel())
    o.set_data(y); o.set_proposal([0.02, 0.5]); o.set_path(np.column_stack([y, np.zeros(M + 1)]))
    o.set_update_mode(1)
    o.set_tuning(True, 20, 0.23, 0.1)
    o.sweep(6000, seed=2)
    o.set_tuning(False)
    s0 = o.stats().astype(float)
    o.sweep(2000, seed=2)
    s1 = o.stats().astype(float)
    rate = (s1[0, :2] - s0[0, :2]) / (s1[1, :2] - s0[1, :2])
    assert np.all(np.abs(rate - 0.23) < 0.04), rate           # started from widths 10x too small / too large
    ws, _ = o.get_widths()
    assert ws[5:-5, 0].std() / ws[5:-5, 0].mean() < 0.5       # interior sites end up with similar step sizes
