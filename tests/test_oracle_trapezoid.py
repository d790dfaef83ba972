"""Pins for the paper's own discretisation of the model-error term: the trapezoid rule
    eps_n = x_n - x_{n-1} - (dt/2) [F(x_n) + F(x_{n-1})]                                (Eq. 7)
    A = sum_{n=1..M} (R_o/2)(y_n - h(x_n))^2 + sum_{n=1..M} sum_a (R_d,a/2) eps_{n,a}^2
selected in the oracle with set_discretisation(1).  The oracle caches c_n = (dt/2) F(x_n) (the paper caches F_n,
PAPER.md:189, 242) and forms every residual as (x_{n+1} - x_n) - c_n - c_{n+1}.

What fixes it: the full action retyped here from Eq. 7 with the vector field taken from the oracle's stand-alone
right-hand side; the site-local and parameter Delta-A against brute-force differences of that action; the update
invariants; and, for a linear vector field, the Gaussian posterior assembled here from the definition, sampled by
stationary replica chains.
"""
import numpy as np
import pytest

import oracle
from oracle import OracleChain
from workloads import MODEL_HH, MODEL_LINEAR, make_workload, linear_matrix, linear_truth

TRAPEZOID = 1


def hh_chain(M=16, params=False, seed=5):
    w = make_workload(2 if params else 0, M=M, seed=seed)
    o = OracleChain.from_workload(w)
    o.set_discretisation(TRAPEZOID)
    return w, o


def linear_chain(M=16, D=2, seed=3):
    rng = np.random.default_rng(seed)
    A = linear_matrix(D) if D <= 2 else 0.5 * np.eye(D) + 0.1 * rng.normal(size=(D, D))
    Rf = np.array([100.0, 50.0, 70.0, 20.0])[:D]
    o = OracleChain(MODEL_LINEAR, D, 1, M, 1.0, 100.0, Rf, A.ravel())
    o.set_discretisation(TRAPEZOID)
    o.set_data(rng.normal(size=M + 1))
    o.set_proposal(np.full(D, 0.1), np.full(D * D, 0.01))
    o.set_path(rng.normal(size=(M + 1, D)))
    return o, A, Rf


def action_from_eq7(x, y, F, dt, Rm, Rf, L=1):
    """The action written out from PAPER.md:121, 135-137 in extended precision; F[n] = vector field at x_n."""
    ld = np.longdouble
    x, F = x.astype(ld), F.astype(ld)
    A = ld(0)
    for n in range(1, len(x)):
        eps = x[n] - x[n - 1] - ld(dt) / 2 * (F[n] + F[n - 1])
        A += np.sum(ld(0.5) * np.asarray(Rf, ld) * eps * eps)
        A += np.sum(ld(0.5) * ld(Rm) * (np.asarray(y[n], ld).reshape(-1)[:L] - x[n, :L]) ** 2)
    return A


def test_full_action_is_the_papers_eq7_hh():
    w, o = hh_chain(24)
    x, p = o.get_path()
    I = w.I[0]
    F = np.array([oracle.rhs(MODEL_HH, x[n], p, I[n]) for n in range(o.M + 1)])
    ref = action_from_eq7(x, w.y[0], F, w.dt, w.Rm, w.Rf)
    got = o.full_action()
    assert abs(float(got - ref)) <= 1e-13 * float(abs(ref)), (got, ref)
    # and it differs from the RK4-map action of the same path (a different discretisation, not a relabelling)
    o.set_discretisation(0)
    assert abs(float(o.full_action() - ref)) > 1e-6 * float(abs(ref))


def test_full_action_is_the_papers_eq7_linear():
    o, A, Rf = linear_chain(20, 2)
    x, p = o.get_path()
    F = x @ (A - np.eye(2)).T / 1.0                     # F(x) = (A x - x)/dt, dt = 1
    y = np.random.default_rng(3).normal(size=21)         # same draw as linear_chain's data
    ref = action_from_eq7(x, y, F, 1.0, 100.0, Rf)
    assert abs(float(o.full_action() - ref)) <= 1e-13 * float(abs(ref))


@pytest.mark.parametrize("which", ["hh", "lin1", "lin2", "lin3", "lin4"])
def test_site_delta_A_equals_brute_force_every_site(which):
    rng = np.random.default_rng(11)
    if which == "hh":
        w, o = hh_chain(16)
        widths = w.w_state
    else:
        o, _, _ = linear_chain(16, int(which[-1]))
        widths = np.full(o.D, 0.1)
    x, p = o.get_path()
    A0 = o.full_action()
    for n in range(o.M + 1):                      # n = 0 (no left term, no measurement) and n = M (no right term) included
        for rep in range(3):
            xp = x[n] + widths * rng.normal(size=o.D)
            dA, S = o.site_delta_A(n, xp)
            X2 = x.copy(); X2[n] = xp
            brute = float(o.full_action(X2) - A0)
            assert abs(dA - brute) <= 1e-15 * float(abs(A0)) * 20 + 1e-13 * S, (n, dA, brute)


def test_site_M_depends_on_its_own_vector_field():
    # in the trapezoid form the LAST site enters eps_M through F(x_M) as well: moving only a gate variable of x_M
    # (which the RK4-map action cannot see beyond the direct residual) changes eps_M's voltage component
    w, o = hh_chain(16)
    x, p = o.get_path()
    M = o.M
    xp = x[M].copy(); xp[1] += 0.05
    dA_trap, _ = o.site_delta_A(M, xp)
    F0, F1 = oracle.rhs(MODEL_HH, x[M], p, w.I[0][M]), oracle.rhs(MODEL_HH, xp, p, w.I[0][M])
    assert F0[0] != F1[0]
    Fm = oracle.rhs(MODEL_HH, x[M - 1], p, w.I[0][M - 1])
    e_old = x[M] - x[M - 1] - w.dt / 2 * (F0 + Fm)
    e_new = xp - x[M - 1] - w.dt / 2 * (F1 + Fm)
    ref = np.sum(0.5 * np.asarray(w.Rf) * (e_new**2 - e_old**2))
    assert abs(dA_trap - ref) <= 1e-12 * max(1.0, abs(ref))


@pytest.mark.parametrize("which", ["hh", "lin2"])
def test_param_delta_A_equals_brute_force(which):
    rng = np.random.default_rng(2)
    if which == "hh":
        w, o = hh_chain(16, params=True)
        steps = w.w_param
    else:
        o, _, _ = linear_chain(16, 2)
        steps = np.full(4, 0.01)
    x, p = o.get_path()
    A0 = o.full_action()
    for l in range(o.Np):
        pl = p[l] + steps[l] * rng.normal()
        dA, S = o.param_delta_A(l, pl)
        p2 = p.copy(); p2[l] = pl
        brute = float(o.full_action(None, p2) - A0)
        assert abs(dA - brute) <= 1e-15 * float(abs(A0)) * 20 + 1e-13 * S, (l, dA, brute)


def test_invariants_antisymmetry_telescoping_cache_order_split():
    w, o = hh_chain(40, params=True)
    x, p = o.get_path()
    rng = np.random.default_rng(0)
    # antisymmetry dA(x -> x') = -dA(x' -> x)
    for n in (0, 1, 17, 39, 40):
        xp = x[n] + w.w_state * rng.normal(size=4)
        d1, S = o.site_delta_A(n, xp)
        X2 = x.copy(); X2[n] = xp
        o2 = OracleChain.from_workload(w); o2.set_discretisation(TRAPEZOID); o2.set_path(X2)
        d2, _ = o2.site_delta_A(n, x[n])
        assert abs(d1 + d2) <= 1e-14 * S
    # telescoping over sweeps: sum of accepted dA (states and parameters) = A(after) - A(before)
    A_prev = o.full_action()
    for t in range(5):
        o.sweep(1, seed=4)
        tr = o.trace()
        acc_sum = tr["dA"][tr["acc"] == 1].sum() + np.nansum(np.where(tr["accp"] == 1, tr["dAp"], 0.0))
        A_now = o.full_action()
        assert abs(float(A_now - A_prev) - acc_sum) <= 1e-11 * float(abs(A_prev)), t
        A_prev = A_now
    # cache coherence: c_n == (dt/2) F(x_n, p; I_n) recomputed, n = 0..M
    x, p = o.get_path()
    c = o.get_cache()
    assert c.shape == (o.M + 1, 4)
    ref = np.array([0.5 * w.dt * oracle.rhs(MODEL_HH, x[n], p, w.I[0][n]) for n in range(o.M + 1)])
    assert np.max(np.abs(c - ref)) <= 1e-15 * np.max(np.abs(ref)) * 4
    # visiting order inside a half-sweep does not matter; sweep(a) + sweep(b) == sweep(a + b)
    outs = []
    for order in (0, 1, 2):
        q = OracleChain.from_workload(w); q.set_discretisation(TRAPEZOID)
        q.sweep(6, seed=4, order=order)
        outs.append(q.get_path())
    for xo, po in outs[1:]:
        assert np.array_equal(xo, outs[0][0]) and np.array_equal(po, outs[0][1])
    q = OracleChain.from_workload(w); q.set_discretisation(TRAPEZOID)
    q.sweep(2, seed=4); q.sweep(4, seed=4)
    assert np.array_equal(q.get_path()[0], outs[0][0])


def trapezoid_posterior(A, Rf, Rm, y, dt=1.0):
    """Dense J, h of the quadratic trapezoid action for F(x) = (A - I) x / dt, first component observed at n = 1..M:
    eps_n = P x_n - Q x_{n-1},  P = I - (dt/2) B,  Q = I + (dt/2) B,  B = (A - I)/dt."""
    M, D = len(y) - 1, A.shape[0]
    N = (M + 1) * D
    Bm = (A - np.eye(D)) / dt
    Pm, Qm = np.eye(D) - dt / 2 * Bm, np.eye(D) + dt / 2 * Bm
    E = np.zeros((M * D, N))
    for n in range(1, M + 1):
        E[(n - 1) * D:n * D, n * D:(n + 1) * D] = Pm
        E[(n - 1) * D:n * D, (n - 1) * D:n * D] = -Qm
    W = np.kron(np.eye(M), np.diag(Rf))
    H = np.zeros((M, N))
    for n in range(1, M + 1):
        H[n - 1, n * D] = 1.0
    return E.T @ W @ E + Rm * H.T @ H, Rm * H.T @ y[1:]


def _eigenmode_z(disc_of_sampler, K=24, n_samples=1500, thin=10, seed=42, w=0.15, weight_bug=1.0):
    M, D = 6, 2
    rng = np.random.default_rng(seed)
    A, xt, y = linear_truth(M, rng)
    Rf, Rm = np.array([100.0, 100.0]), 100.0
    J, h = trapezoid_posterior(A, Rf, Rm, y)
    mu = np.linalg.solve(J, h)
    lam, V = np.linalg.eigh(J)
    Lc = np.linalg.cholesky(J)
    m1, m2 = [], []
    for k in range(K):
        x0 = mu + np.linalg.solve(Lc.T, rng.normal(size=mu.size))        # exact posterior sample
        o = OracleChain(MODEL_LINEAR, D, 1, M, 1.0, Rm, Rf * weight_bug, A.ravel(), chain_id=k)
        o.set_discretisation(disc_of_sampler)
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


def test_quadratic_form_of_the_oracle_action_is_the_assembled_one():
    # A(X) = 1/2 X^T J X - h^T X + c exactly for the linear field: check J and h through the oracle's full action
    rng = np.random.default_rng(5)
    M, D = 5, 2
    A, xt, y = linear_truth(M, rng)
    Rf, Rm = np.array([100.0, 60.0]), 80.0
    J, h = trapezoid_posterior(A, Rf, Rm, y)
    o = OracleChain(MODEL_LINEAR, D, 1, M, 1.0, Rm, Rf, A.ravel())
    o.set_discretisation(TRAPEZOID); o.set_data(y); o.set_proposal([0.1, 0.1])
    o.set_path(np.zeros((M + 1, D)))
    c0 = float(o.full_action())
    for rep in range(6):
        X = rng.normal(size=(M + 1) * D)
        got = float(o.full_action(X.reshape(M + 1, D)))
        ref = 0.5 * X @ J @ X - h @ X + c0
        assert abs(got - ref) <= 1e-11 * max(1.0, abs(ref))


def test_stationary_replicas_match_the_trapezoid_gaussian_posterior():
    z_mean, z_var, var = _eigenmode_z(TRAPEZOID)
    z = np.concatenate([z_mean, z_var])
    assert np.abs(z).max() < 4.0, z
    assert np.sqrt(np.mean(z**2)) < 1.5, z
    assert np.all(np.abs(var[1:] - 1.0) < 0.03), var


def test_the_replica_test_has_power():
    # a sampler whose model-error weight is 5 % off must fail the same statistic by a wide margin
    z_mean, z_var, var = _eigenmode_z(TRAPEZOID, K=12, n_samples=1500, weight_bug=1.05)
    assert np.abs(z_var).max() > 6.0, z_var


# ------------------------------------------------------------------------------------------------------------
# The identity the tile engine's trapezoid parameter moves rest on: with Eq. 7 the parameters enter
# the action only through (dt/2) F_V = theta(p) . phi(x, I), seven monomials typed here from PAPER.md:256-260 Eq. 11, so
#   Delta-A(p -> p') = (Rf_V / 2) [ (theta' - theta)^T Q (theta' + theta) - 2 (theta' - theta) . b ]
# with Q = sum psi psi^T, b = sum d psi independent of p.  Checked against the oracle's direct sum over the path.
# ------------------------------------------------------------------------------------------------------------
def _theta(p):
    gNa, gK, gL, ENa, EK, EL, C = [np.longdouble(v) for v in p]
    return np.array([1, gNa, gNa * ENa, gK, gK * EK, gL, gL * EL], dtype=np.longdouble) / C


def _phi(x, I, dt):
    ld = np.longdouble
    V, m, h, n = [x[:, c].astype(ld) for c in range(4)]
    one = np.ones_like(V)
    return ld(dt) / 2 * np.stack([I.astype(ld), -m**3 * h * V, m**3 * h, -n**4 * V, n**4, -V, one], axis=1)


@pytest.mark.parametrize("kinetics", ["tanh", "classic"])
def test_parameter_moves_are_a_quadratic_form_in_seven_monomials(kinetics):
    w = make_workload(2, M=300, seed=9, kinetics=kinetics)
    o = OracleChain.from_workload(w)
    o.set_discretisation(TRAPEZOID)
    rng = np.random.default_rng(4)
    x, p = o.get_path()
    x = x + 0.3 * rng.normal(size=x.shape) * np.array([1.0, 0.02, 0.02, 0.02])      # off the initial path: residuals of every size
    o.set_path(x)
    phi = _phi(x, w.I[0], w.dt)
    psi = phi[:-1] + phi[1:]                                                        # terms n -> n+1, n = 0..M-1
    d = (x[1:, 0] - x[:-1, 0]).astype(np.longdouble)
    Q, b = psi.T @ psi, psi.T @ d
    th = _theta(p)
    # the cached V entries ARE theta . phi (the gate entries hold no parameter)
    c = o.get_cache()
    assert np.allclose(c[:, 0], np.asarray(phi @ th, dtype=np.float64), rtol=1e-13, atol=1e-15)
    worst = 0.0
    for l in range(7):
        for scale in (1.0, 30.0, -200.0):
            pl = p[l] + scale * w.w_param[l] * rng.normal()
            p2 = p.copy(); p2[l] = pl
            th2 = _theta(p2)
            formula = float(np.longdouble(w.Rf[0]) / 2 * ((th2 - th) @ Q @ (th2 + th) - 2 * (th2 - th) @ b))
            dA, S = o.param_delta_A(l, pl)
            assert abs(formula - dA) <= 1e-12 * max(abs(dA), S), (kinetics, l, scale, formula, dA, S)
            worst = max(worst, abs(formula - dA) / max(abs(dA), S))
    # power: a dropped monomial or a wrong sign does not survive (gL EL missing from theta . phi)
    bad = float(np.longdouble(w.Rf[0]) / 2 * ((th2 - th)[:6] @ Q[:6, :6] @ (th2 + th)[:6] - 2 * (th2 - th)[:6] @ b[:6]))
    assert abs(bad - dA) > 1e-6 * max(abs(dA), S)
    print("max |formula - oracle| / max(|dA|, S):", worst)
