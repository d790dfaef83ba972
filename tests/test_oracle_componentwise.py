"""Pins for component-wise updates (PAPER.md:226-230 keeps step sizes and acceptance counters
"per component of the path"): set_update_mode(1) proposes ONE component of x_n at a time, D decisions per site.

What fixes it: every single decision of a sweep replayed against brute-force differences of the full action; the draws
(same proposal per component as the joint move, accept uniform of block a); per-component counters; and the sampler's
stationary distribution on the linear-Gaussian model (replicas in the eigenbasis of the exact posterior, with power)."""
import numpy as np
import pytest

import oracle
from oracle import OracleChain
from workloads import MODEL_LINEAR, make_workload, linear_truth

from test_oracle_posterior import gaussian_posterior


@pytest.mark.parametrize("cfg,disc", [(2, 0), (2, 1), (1, 0)])
def test_every_decision_of_a_sweep_is_a_single_component_metropolis_step(cfg, disc):
    w = make_workload(cfg, M=12)
    o = OracleChain.from_workload(w); o.set_update_mode(1); o.set_discretisation(disc)
    D = o.D
    for sweep in range(3):
        X, p = o.get_path()
        X = X.copy()
        o.sweep(1, seed=11, do_params=False)
        tr = o.trace()
        assert tr["dA"].shape == (o.M + 1, D)
        for parity in (0, 1):                       # even sites first, then odd; components in index order inside a site
            for n in range(parity, o.M + 1, 2):
                for a in range(D):
                    X2 = X.copy(); X2[n, a] = tr["xprop"][n, a]
                    brute = float(o.full_action(X2, p) - o.full_action(X, p))
                    A0 = float(abs(o.full_action(X, p)))
                    assert abs(tr["dA"][n, a] - brute) <= 2e-14 * A0 + 1e-13 * tr["S"][n, a], (sweep, n, a)
                    assert bool(tr["acc"][n, a]) == bool(tr["logu"][n, a] < -tr["dA"][n, a])
                    if tr["acc"][n, a]:
                        X = X2
        assert np.array_equal(X, o.get_path()[0])    # the replay lands on the chain's path bit for bit


def test_draws_same_proposal_as_the_joint_move_and_one_uniform_per_component():
    w = make_workload(0, M=20)
    oj = OracleChain.from_workload(w)
    oc = OracleChain.from_workload(w); oc.set_update_mode(1)
    oj.sweep(1, seed=5); oc.sweep(1, seed=5)
    tj, tc = oj.trace(), oc.trace()
    even = np.arange(0, 21, 2)
    # even sites are visited first, from the same state in both chains: identical proposals component by component
    assert np.array_equal(tj["xprop"][even], tc["xprop"][even])
    # the joint move's accept uniform is block 0 of the accept stream = component 0's; the others are different draws
    assert np.array_equal(tj["logu"][even], tc["logu"][even, 0])
    for a in range(1, 4):
        assert not np.any(tc["logu"][:, a] == tc["logu"][:, 0])
    assert np.all(tc["logu"] < 0)


def test_counters_are_per_component_and_zero_width_components_always_accept():
    w = make_workload(0, M=30)
    o = OracleChain.from_workload(w); o.set_update_mode(1)
    o.set_proposal([0.5, 0.0, 0.02, 0.02])
    o.sweep(20, seed=2)
    st = o.stats()
    assert np.all(st[1, :4] == 20 * 31)
    assert st[0, 1] == 20 * 31                        # w = 0: x' = x, dA = 0, accepted
    assert len({int(st[0, 0]), int(st[0, 2]), int(st[0, 3])}) == 3 and np.all(st[0, [0, 2, 3]] < 20 * 31)


def _eigenmode_z(K=24, n_samples=1500, thin=10, seed=42, w=0.25, weight_bug=1.0):
    M, D = 6, 2
    rng = np.random.default_rng(seed)
    A, xt, y = linear_truth(M, rng)
    Rf, Rm = np.array([100.0, 100.0]), 100.0
    J, h = gaussian_posterior(A, Rf, Rm, y)
    mu = np.linalg.solve(J, h)
    lam, V = np.linalg.eigh(J)
    Lc = np.linalg.cholesky(J)
    m1, m2 = [], []
    for k in range(K):
        x0 = mu + np.linalg.solve(Lc.T, rng.normal(size=mu.size))
        o = OracleChain(MODEL_LINEAR, D, 1, M, 1.0, Rm, Rf * weight_bug, A.ravel(), chain_id=k)
        o.set_update_mode(1)
        o.set_data(y); o.set_proposal([w, w]); o.set_path(x0.reshape(M + 1, D))
        cs = np.empty((n_samples, mu.size))
        for t in range(n_samples):
            o.sweep(thin, seed=9)
            cs[t] = ((o.get_path()[0].ravel() - mu) @ V) * np.sqrt(lam)
        m1.append(cs.mean(0)); m2.append((cs**2).mean(0))
    m1, m2 = np.array(m1), np.array(m2)
    return m1.mean(0) / (m1.std(0, ddof=1) / np.sqrt(K)), (m2.mean(0) - 1.0) / (m2.std(0, ddof=1) / np.sqrt(K)), m2.mean(0)


def test_stationary_replicas_match_the_gaussian_posterior():
    z_mean, z_var, var = _eigenmode_z()
    z = np.concatenate([z_mean, z_var])
    assert np.abs(z).max() < 4.0 and np.sqrt(np.mean(z**2)) < 1.5, z
    assert np.all(np.abs(var[1:] - 1.0) < 0.03), var


def test_the_replica_test_has_power():
    z_mean, z_var, var = _eigenmode_z(K=12, n_samples=1500, weight_bug=1.05)
    assert np.abs(z_var).max() > 6.0, z_var


def test_config_widths_give_workable_acceptance_componentwise():
    # at the config-0 widths the joint move is accepted ~2 % of the time at equilibrium, the
    # component-wise moves 19-33 %: the widths were chosen for component-wise updates
    w = make_workload(0, M=256)
    rates = {}
    for mode in (0, 1):
        o = OracleChain.from_workload(w); o.set_update_mode(mode)
        o.sweep(600, seed=1)
        s0 = o.stats().astype(float)
        o.sweep(400, seed=1)
        s1 = o.stats().astype(float)
        rates[mode] = (s1[0, :4] - s0[0, :4]) / (s1[1, :4] - s0[1, :4])
    assert rates[0][0] < 0.08, rates
    assert np.all(rates[1] > 0.10) and np.all(rates[1] < 0.60), rates
