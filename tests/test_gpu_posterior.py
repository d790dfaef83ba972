"""The CUDA path AS A SAMPLER (north_star: "posterior means must agree with the oracle within 3 Monte
Carlo standard errors"), checked two ways that do not lean on decision-by-decision parity:

 1. against MATHEMATICS: on the linear-Gaussian model the target is the Gaussian N(J^-1 h, J^-1) assembled from the
    definition of the action (tests/test_oracle_posterior.py); K replica chains started from exact posterior samples must
    give unbiased time averages of the first and second moments, on both engines and both update modes;
 2. against the ORACLE with INDEPENDENT seeds: Hodgkin-Huxley config 0, K chains per side, ensemble posterior means per
    (site, component) compared in units of their combined across-replica standard error."""
import numpy as np
import pytest

from test_oracle_posterior import gaussian_posterior
from workloads import MODEL_LINEAR, Workload, linear_truth, make_workload

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def P():
    import torch
    import paper_1103_4887_b200 as P
    assert torch.cuda.is_available()
    P.lib()
    return P


def _linear_replicas(K, M, seed):
    rng = np.random.default_rng(seed)
    A, xt, y = linear_truth(M, rng)
    Rf, Rm = np.array([100.0, 100.0]), 100.0
    J, h = gaussian_posterior(A, Rf, Rm, y)
    mu = np.linalg.solve(J, h)
    Lc = np.linalg.cholesky(J)
    x0 = np.stack([(mu + np.linalg.solve(Lc.T, rng.normal(size=mu.size))).reshape(M + 1, 2) for _ in range(K)])   # exact posterior samples
    w = Workload(name="linear_replicas", model=MODEL_LINEAR, D=2, L=1, Np=4, M=M, dt=1.0, Rm=Rm, Rf=Rf, n_chains=K,
                 p0=np.tile(A.ravel(), (K, 1)), p_true=A.ravel(), lo=np.full((K, 4), -2.0), hi=np.full((K, 4), 2.0),
                 w_state=np.array([0.1, 0.1]), w_param=np.zeros(4), y=np.tile(y[None, :, None], (K, 1, 1)), I=None, x0=x0,
                 x_true=np.tile(xt[None], (K, 1, 1)), n_sweeps=0)
    return w, mu, np.diag(np.linalg.inv(J))


@pytest.mark.parametrize("engine,mode", [(1, 0), (2, 0), (2, 1), (1, 1)])
def test_stationary_replicas_match_the_exact_gaussian_posterior(P, engine, mode):
    K, M = 64, 192
    w, mu, sig2 = _linear_replicas(K, M, seed=17)
    h = P.Pimc.from_workload(w)
    h.set_update_mode(mode)
    h.set_engine(engine)
    assert h.get_engine()["engine"] == engine
    h.set_accum(True, 1); h.reset_moments()
    h.sweep(3000, seed=123)
    mx, _, n = h.moments()
    assert n == 3000
    mx = mx.cpu().numpy()                                  # (K, 2, M+1, D): mean, var of every chain's time series
    means = mx[:, 0].reshape(K, -1)
    sq = mx[:, 1].reshape(K, -1) + means**2
    z1 = (means.mean(0) - mu) / (means.std(0, ddof=1) / np.sqrt(K))
    z2 = (sq.mean(0) - (sig2 + mu**2)) / (sq.std(0, ddof=1) / np.sqrt(K))
    for z in (z1, z2):                                     # z's are correlated along the path: gross checks, as in the oracle's pin
        assert np.abs(z).max() < 5.0, np.abs(z).max()
        assert np.sqrt(np.mean(z**2)) < 1.5, np.sqrt(np.mean(z**2))
        assert np.mean(np.abs(z) > 3.0) < 0.03
    # power: the same statistic rejects a sampler whose target has a 10 % different model-error weight
    A = w.p_true.reshape(2, 2)
    Jb, hb = gaussian_posterior(A, w.Rf * 1.1, w.Rm, w.y[0, :, 0])
    mub, sig2b = np.linalg.solve(Jb, hb), np.diag(np.linalg.inv(Jb))
    z2b = (sq.mean(0) - (sig2b + mub**2)) / (sq.std(0, ddof=1) / np.sqrt(K))
    assert np.sqrt(np.mean(z2b**2)) > 2.5


def test_hh_posterior_means_agree_with_the_oracle_within_three_standard_errors(P):
    # independent Philox keys on the two sides: nothing but the target distribution is shared
    from oracle import OracleChain
    K, M, burn, n_s = 8, 128, 600, 1400
    w1 = make_workload(0, M=M)
    wk = make_workload(0, M=M, n_chains=K)
    for c in range(K):                                     # K replicas of the SAME data
        wk.y[c], wk.I[c], wk.x0[c] = w1.y[0], w1.I[0], w1.x0[0]
    h = P.Pimc.from_workload(wk, with_params=False)
    h.set_update_mode(P.UPDATE_COMPONENTWISE)              # the config's widths are component-wise widths
    h.sweep_states_only(burn, seed=1001)
    h.set_accum(True, 1); h.reset_moments()
    h.sweep_states_only(n_s, seed=1001)
    g = h.moments()[0].cpu().numpy()[:, 0]                 # (K, M+1, D) time-averaged means
    o_means = []
    for c in range(K):
        o = OracleChain.from_workload(w1, chain=0, with_params=False)
        o.set_update_mode(1)
        o.sweep(burn, seed=5000 + c, do_params=False)
        o.set_accum(True, 1); o.reset_moments()
        o.sweep(n_s, seed=5000 + c, do_params=False)
        o_means.append(o.moments()[0][0])
    o_means = np.array(o_means)
    se = np.sqrt(g.var(0, ddof=1) / K + o_means.var(0, ddof=1) / K)
    z = (g.mean(0) - o_means.mean(0)) / se
    print("HH posterior means, GPU vs oracle (independent seeds): rms z %.2f, max |z| %.2f, frac > 3: %.3f" %
          (np.sqrt(np.mean(z**2)), np.abs(z).max(), np.mean(np.abs(z) > 3)))
    # t-distributed with ~2(K-1) degrees of freedom and strongly correlated along the path
    assert np.sqrt(np.mean(z**2)) < 1.6 and np.mean(np.abs(z) > 3.0) < 0.05 and np.abs(z).max() < 7.0
