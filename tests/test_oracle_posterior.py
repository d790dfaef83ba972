"""Pins P1, P3(vi)-(vii), P6: the oracle AS A SAMPLER against closed forms.

PAPER.md:36: "Kalman filtering is the exact solution when the model is linear and the noise is Gaussian".
For the linear map the action is quadratic, A(X) = 1/2 X^T J X - h^T X + c, so the target is N(J^-1 h, J^-1).
J and h are assembled here from the DEFINITION of the action with dense matrices --
not from the oracle's site-local formulas -- and cross-checked by an independent Kalman filter + RTS
smoother with a diffuse prior on x_0 (P(x_0) uniform, dropped from A).
"""
import numpy as np
import pytest

from oracle import OracleChain
from workloads import MODEL_LINEAR, linear_matrix, linear_truth


def gaussian_posterior(A, Rf, Rm, y):
    """Dense J, h of the quadratic action for D-dim linear map, first component observed at n = 1..M."""
    M, D = len(y) - 1, A.shape[0]
    N = (M + 1) * D
    B = np.zeros((M * D, N))                         # residuals r_n = x_{n+1} - A x_n
    for n in range(M):
        B[n * D:(n + 1) * D, (n + 1) * D:(n + 2) * D] = np.eye(D)
        B[n * D:(n + 1) * D, n * D:(n + 1) * D] = -A
    W = np.kron(np.eye(M), np.diag(Rf))
    H = np.zeros((M, N))                             # measurements of component 0 at n = 1..M
    for n in range(1, M + 1):
        H[n - 1, n * D] = 1.0
    J = B.T @ W @ B + Rm * H.T @ H
    h = Rm * H.T @ y[1:]
    return J, h


def kalman_rts(A, Rf, Rm, y, P0=1e9):
    M, D = len(y) - 1, A.shape[0]
    Q, R = np.diag(1.0 / np.asarray(Rf)), 1.0 / Rm
    Hm = np.zeros((1, D)); Hm[0, 0] = 1.0
    mf, Pf, mp, Pp = [np.zeros(D)], [P0 * np.eye(D)], [None], [None]
    for n in range(1, M + 1):
        m_, P_ = A @ mf[-1], A @ Pf[-1] @ A.T + Q
        S = Hm @ P_ @ Hm.T + R
        K = P_ @ Hm.T / S
        mp.append(m_); Pp.append(P_)
        mf.append(m_ + (K * (y[n] - m_[0])).ravel())
        Pf.append(P_ - K @ Hm @ P_)
    ms, Ps = [None] * (M + 1), [None] * (M + 1)
    ms[M], Ps[M] = mf[M], Pf[M]
    for n in range(M - 1, -1, -1):
        G = Pf[n] @ A.T @ np.linalg.inv(Pp[n + 1])
        ms[n] = mf[n] + G @ (ms[n + 1] - mp[n + 1])
        Ps[n] = Pf[n] + G @ (Ps[n + 1] - Pp[n + 1]) @ G.T
    return np.array(ms), np.array(Ps)


def test_two_closed_forms_agree():
    # Same Gaussian two ways.  The Kalman recursion needs a proper prior N(0, P0 I) on x_0; that prior adds
    # I/P0 to the x_0 block of J exactly, so the two must agree to rounding for ANY P0; P0 -> inf is the
    # action's flat prior and changes the x_0 block by 1/P0 only.
    rng = np.random.default_rng(1)
    A, xt, y = linear_truth(60, rng)
    J, h = gaussian_posterior(A, [100.0, 100.0], 100.0, y)
    for P0 in (10.0, 1e4):
        Jp = J.copy(); Jp[0, 0] += 1 / P0; Jp[1, 1] += 1 / P0
        mu = np.linalg.solve(Jp, h).reshape(-1, 2)
        Sig = np.linalg.inv(Jp)
        ms, Ps = kalman_rts(A, [100.0, 100.0], 100.0, y, P0=P0)
        assert np.allclose(mu, ms, rtol=1e-8, atol=1e-9)
        for n in (0, 1, 30, 59, 60):
            assert np.allclose(Sig[2 * n:2 * n + 2, 2 * n:2 * n + 2], Ps[n], rtol=1e-6, atol=1e-10)
    # flat-prior limit: means of the diffuse J vs Kalman with a very wide prior
    mu_flat = np.linalg.solve(J, h).reshape(-1, 2)
    ms, _ = kalman_rts(A, [100.0, 100.0], 100.0, y, P0=1e8)
    assert np.allclose(mu_flat, ms, atol=5e-6)
    # and the numbers SURVEY.md Appendix A.3 quotes for config 1: posterior sd ~0.067 observed, ~0.32 hidden
    sd = np.sqrt(np.diag(np.linalg.inv(J))).reshape(-1, 2)
    assert abs(sd[30, 0] - 0.067) < 0.004 and abs(sd[30, 1] - 0.32) < 0.03


def _replica_z(M, K, n_burn, n_sweeps, seed, Rm=100.0, Rf=(100.0, 100.0), w=0.1, D=2, weight_bug=None):
    rng = np.random.default_rng(seed)
    A, xt, y = linear_truth(M, rng, D=D)
    Rf = np.asarray(Rf, float)
    J, h = gaussian_posterior(A, Rf, Rm, y)
    mu = np.linalg.solve(J, h)
    Lc = np.linalg.cholesky(J)
    sig2 = np.diag(np.linalg.inv(J))
    means, sq = [], []
    for k in range(K):
        x0 = mu + np.linalg.solve(Lc.T, rng.normal(size=mu.size))        # exact posterior sample
        o = OracleChain(MODEL_LINEAR, D, 1, M, 1.0, Rm, Rf if weight_bug is None else Rf * weight_bug, A.ravel(),
                        chain_id=k)
        o.set_data(y); o.set_proposal(np.full(D, w)); o.set_path(x0.reshape(M + 1, D))
        o.sweep(n_burn, seed=77)
        o.set_accum(True, 1); o.reset_moments(); o.sweep(n_sweeps, seed=77)
        mx, _, n = o.moments()
        assert n == n_sweeps
        means.append(mx[0].ravel()); sq.append(mx[1].ravel() + mx[0].ravel() ** 2)
    means, sq = np.array(means), np.array(sq)
    z1 = (means.mean(0) - mu) / (means.std(0, ddof=1) / np.sqrt(K))
    z2 = (sq.mean(0) - (sig2 + mu**2)) / (sq.std(0, ddof=1) / np.sqrt(K))
    return z1, z2, o


def _eigenmode_z(weight_bug=None, K=24, n_samples=2000, thin=10, seed=42, w=0.15):
    """Sharp stationarity test on a small problem (M = 6, D = 2: 14 dimensions) in the eigenbasis of J, where
    the whitened coordinates c_i = sqrt(lam_i) v_i.(x - mu) are independent N(0,1) under the exact posterior.
    K replica chains START from exact posterior samples, so time averages are unbiased and
    z = (ensemble mean - exact) / SE_across_replicas ~ t_{K-1} independently per mode."""
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
        o = OracleChain(MODEL_LINEAR, D, 1, M, 1.0, Rm, Rf if weight_bug is None else Rf * weight_bug, A.ravel(), chain_id=k)
        o.set_data(y); o.set_proposal([w, w]); o.set_path(x0.reshape(M + 1, D))
        cs = np.empty((n_samples, mu.size))
        for t in range(n_samples):
            o.sweep(thin, seed=9)
            cs[t] = ((o.get_path()[0].ravel() - mu) @ V) * np.sqrt(lam)
        m1.append(cs.mean(0)); m2.append((cs**2).mean(0))
    m1, m2 = np.array(m1), np.array(m2)
    z_mean = m1.mean(0) / (m1.std(0, ddof=1) / np.sqrt(K))
    z_var = (m2.mean(0) - 1.0) / (m2.std(0, ddof=1) / np.sqrt(K))
    return z_mean, z_var, m2.mean(0)


def test_stationary_replicas_match_gaussian_posterior_in_eigenbasis():
    z_mean, z_var, var = _eigenmode_z()
    z = np.concatenate([z_mean, z_var])
    assert np.abs(z).max() < 4.0, z
    assert np.sqrt(np.mean(z**2)) < 1.5, z
    assert np.all(np.abs(var[1:] - 1.0) < 0.03), var          # every well-mixed mode's variance within 3 %


def test_eigenbasis_test_has_power_against_wrong_weight_or_rule():
    # a sampler whose model-error weight is 5 % off must fail the same statistic by a wide margin
    z_mean, z_var, var = _eigenmode_z(weight_bug=1.05, K=12, n_samples=1500)
    assert np.abs(z_var).max() > 6.0, z_var


def test_replicas_match_gaussian_posterior_per_site_longer_path():
    # Same idea per (site, component) on a longer path (z's are strongly correlated along the path, so only
    # gross checks here): M = 96, K = 64 replicas.
    z1, z2, _ = _replica_z(M=96, K=64, n_burn=0, n_sweeps=200, seed=6)
    for z in (z1, z2):
        assert np.abs(z).max() < 5.0
        assert np.mean(np.abs(z) > 3.0) < 0.05


def test_interior_acceptance_rate_matches_conditional_gaussian_integral():
    # P3(vi): at stationarity the single-site acceptance of interior sites is
    # E_x E_d min(1, exp(-dA)) with x ~ N(0, K^-1), d ~ N(0, w^2 I), K = Rf (I + A^T A) + Rm e0 e0^T
    A = linear_matrix(2); Rf, Rm, w = 100.0, 100.0, 0.1
    K = Rf * (np.eye(2) + A.T @ A) + Rm * np.diag([1.0, 0.0])
    ev = np.linalg.eigvalsh(K)
    assert np.allclose(ev, [198.0, 298.0], atol=0.1)
    rng = np.random.default_rng(0)
    n = 2_000_000
    Lk = np.linalg.cholesky(np.linalg.inv(K))
    x = rng.normal(size=(n, 2)) @ Lk.T
    d = rng.normal(0, w, (n, 2))
    dA = 0.5 * np.einsum("ni,ij,nj->n", d, K, d) + np.einsum("ni,ij,nj->n", d, K, x)
    expect = np.minimum(1.0, np.exp(-dA)).mean()
    assert abs(expect - 0.383) < 0.003
    z1, z2, o = _replica_z(M=256, K=2, n_burn=0, n_sweeps=300, seed=8)
    # the last replica's counters: all sites incl. the two boundaries (which accept a bit more often)
    st = o.stats()
    rate = st[0, 0] / st[1, 0]
    assert abs(rate - expect) < 0.01, (rate, expect)


def test_equipartition_of_the_action():
    # P3(vii): for a Gaussian target <A> - A(mu) = (number of dimensions)/2, per-sample sd sqrt(dims/2)
    M, D = 200, 2
    rng = np.random.default_rng(3)
    A, xt, y = linear_truth(M, rng)
    J, h = gaussian_posterior(A, [100.0, 100.0], 100.0, y)
    mu = np.linalg.solve(J, h)
    Lc = np.linalg.cholesky(J)
    o = OracleChain(MODEL_LINEAR, D, 1, M, 1.0, 100.0, [100.0, 100.0], A.ravel())
    o.set_data(y); o.set_proposal([0.1, 0.1])
    Amu = float(o.full_action(mu.reshape(M + 1, D)))
    o.set_path((mu + np.linalg.solve(Lc.T, rng.normal(size=mu.size))).reshape(M + 1, D))
    vals = []
    for t in range(300):
        o.sweep(10, seed=5)
        vals.append(float(o.full_action()) - Amu)
    dims = D * (M + 1)
    vals = np.array(vals)
    # successive samples are correlated; allow 6 "independent-sample" standard errors
    assert abs(vals.mean() - dims / 2) < 6 * np.sqrt(dims / 2) / np.sqrt(len(vals)) * 3
    assert 0.6 * np.sqrt(dims / 2) < vals.std() < 1.5 * np.sqrt(dims / 2)


def test_textbook_one_site_gaussian():
    # P6: M = 1, D = 1, map x1 = a x0.  A = (Rm/2)(y1 - x1)^2 + (Rf/2)(x1 - a x0)^2 with x0 flat:
    # marginal of x1 is N(y1, 1/Rm); x1 - a x0 ~ N(0, 1/Rf) independent of x1.
    a, Rm, Rf, y1 = 0.9, 4.0, 25.0, 0.7
    K, n = 24, 4000
    m1, m2, r2 = [], [], []
    for k in range(K):
        o = OracleChain(MODEL_LINEAR, 1, 1, 1, 1.0, Rm, [Rf], [a], chain_id=k)
        o.set_data([123.0, y1]); o.set_proposal([0.5]); o.set_path([[y1 / a], [y1]])
        o.sweep(200, seed=1)
        xs = []
        for t in range(n // 10):
            o.sweep(10, seed=1); x, _ = o.get_path(); xs.append(x.ravel().copy())
        xs = np.array(xs)
        m1.append(xs[:, 1].mean()); m2.append(((xs[:, 1] - y1) ** 2).mean()); r2.append(((xs[:, 1] - a * xs[:, 0]) ** 2).mean())
    for vals, exact in ((m1, y1), (m2, 1 / Rm), (r2, 1 / Rf)):
        vals = np.array(vals)
        z = (vals.mean() - exact) / (vals.std(ddof=1) / np.sqrt(K))
        assert abs(z) < 4.0, (z, vals.mean(), exact)


def test_parameter_moves_sample_the_conditional_gaussian():
    # States frozen (w_state = 0): the parameter chain targets p(a | X) ~ exp(-(Rf/2) sum (x_{n+1} - a x_n)^2),
    # a Gaussian with mean Sxy/Sxx and precision Rf Sxx (bounds far away).
    rng = np.random.default_rng(4)
    M, Rf = 40, 50.0
    xs = np.cumsum(rng.normal(size=M + 1)) * 0.3 + 1.0
    Sxx, Sxy = np.sum(xs[:-1] ** 2), np.sum(xs[:-1] * xs[1:])
    mean, sd = Sxy / Sxx, 1 / np.sqrt(Rf * Sxx)
    K = 16
    ms, vs = [], []
    for k in range(K):
        o = OracleChain(MODEL_LINEAR, 1, 1, M, 1.0, 1.0, [Rf], [mean + sd], chain_id=k)
        o.set_data(np.zeros(M + 1)); o.set_proposal([0.0], [2.0 * sd]); o.set_bounds([-10.0], [10.0]); o.set_path(xs)
        o.sweep(200, seed=3)
        o.set_accum(True, 1); o.reset_moments(); o.sweep(6000, seed=3)
        _, mp, n = o.moments()
        ms.append(mp[0, 0]); vs.append(mp[1, 0] + (mp[0, 0] - mean) ** 2)
        assert np.array_equal(o.get_path()[0].ravel(), xs)
    ms, vs = np.array(ms), np.array(vs)
    assert abs(ms.mean() - mean) / (ms.std(ddof=1) / np.sqrt(K)) < 4.0
    assert abs(vs.mean() - sd**2) / (vs.std(ddof=1) / np.sqrt(K)) < 4.0
    # truncated prior: bounds [mean, +inf) => half-Gaussian, E[a] = mean + sd sqrt(2/pi)
    ms = []
    for k in range(K):
        o = OracleChain(MODEL_LINEAR, 1, 1, M, 1.0, 1.0, [Rf], [mean + sd], chain_id=100 + k)
        o.set_data(np.zeros(M + 1)); o.set_proposal([0.0], [2.0 * sd]); o.set_bounds([mean], [10.0]); o.set_path(xs)
        o.sweep(200, seed=3); o.set_accum(True, 1); o.reset_moments(); o.sweep(6000, seed=3)
        ms.append(o.moments()[1][0, 0])
    ms = np.array(ms)
    assert abs(ms.mean() - (mean + sd * np.sqrt(2 / np.pi))) / (ms.std(ddof=1) / np.sqrt(K)) < 4.0
