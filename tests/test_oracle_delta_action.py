"""Pins P2 and P3: local Delta-A vs the brute-force difference of the full action
(dA = A(X') - A(X), and PAPER.md:135-137 for A), and the invariants of the update rule.
"""
import numpy as np
import pytest

import oracle
from oracle import OracleChain
from workloads import MODEL_HH, MODEL_LINEAR, make_workload, linear_matrix


def small_hh(M=16, seed=5, params=False):
    w = make_workload(2 if params else 0, M=M, seed=seed)
    return w, OracleChain.from_workload(w)


def small_linear(M=16, D=2, seed=3):
    rng = np.random.default_rng(seed)
    A = linear_matrix(D) if D <= 2 else 0.5 * np.eye(D) + 0.1 * rng.normal(size=(D, D))
    Rf = np.array([100.0, 50.0, 70.0, 20.0])[:D]
    o = OracleChain(MODEL_LINEAR, D, 1, M, 1.0, 100.0, Rf, A.ravel())
    o.set_data(rng.normal(size=M + 1))
    o.set_proposal(np.full(D, 0.1), np.full(D * D, 0.01))
    o.set_path(rng.normal(size=(M + 1, D)))
    return o


@pytest.mark.parametrize("which", ["hh", "lin1", "lin2", "lin3"])
def test_site_delta_A_equals_brute_force_every_site(which):
    rng = np.random.default_rng(11)
    if which == "hh":
        w, o = small_hh(16)
        widths = w.w_state
    else:
        o = small_linear(16, int(which[-1]))
        widths = np.full(o.D, 0.1)
    x, p = o.get_path()
    A0 = o.full_action()
    for n in range(o.M + 1):                      # includes the boundaries n = 0 (no n-1 term, no measurement) and n = M
        for rep in range(3):
            xp = x[n] + widths * rng.normal(size=o.D)
            dA, S = o.site_delta_A(n, xp)
            X2 = x.copy(); X2[n] = xp
            brute = float(o.full_action(X2) - A0)
            # cancellation in the full action limits the brute force to ~eps * A0
            assert abs(dA - brute) <= 1e-15 * float(abs(A0)) * 20 + 1e-13 * S, (n, dA, brute)


def test_site_0_has_no_measurement_and_site_M_no_forward_term():
    w, o = small_hh(16)
    x, p = o.get_path()
    M = o.M
    # changing y_0 must not change dA at any site (the action sums n = 1..M)
    xp0 = x[0] + [0.3, 0.01, -0.01, 0.02]
    d_before = o.site_delta_A(0, xp0)[0]
    y2 = w.y[0].copy(); y2[0] += 10.0
    o.set_data(y2, w.I[0])
    assert o.site_delta_A(0, xp0)[0] == d_before
    # but y_M matters
    xpM = x[M] + [0.3, 0.01, -0.01, 0.02]
    dM = o.site_delta_A(M, xpM)[0]
    y3 = w.y[0].copy(); y3[M] += 1.0
    o.set_data(y3, w.I[0])
    assert o.site_delta_A(M, xpM)[0] != dM
    # closed form of the measurement part at site M for a V-only change where hidden comps unchanged:
    o.set_data(w.y[0], w.I[0])
    xpV = x[M].copy(); xpV[0] += 0.7
    dA = o.site_delta_A(M, xpV)[0]
    g = o.get_cache()
    r_old = (x[M, 0] - x[M - 1, 0]) - g[M - 1, 0]
    expect = 0.5 * w.Rf[0] * ((r_old + 0.7) ** 2 - r_old**2) + 0.5 * w.Rm * ((w.y[0, M, 0] - xpV[0]) ** 2 - (w.y[0, M, 0] - x[M, 0]) ** 2)
    assert np.isclose(dA, expect, rtol=1e-12)


@pytest.mark.parametrize("which", ["hh", "lin2"])
def test_param_delta_A_equals_brute_force(which):
    rng = np.random.default_rng(12)
    if which == "hh":
        w, o = small_hh(16, params=True)
        wp = w.w_param * 10
    else:
        o = small_linear(16, 2); wp = np.full(4, 0.05)
    x, p = o.get_path()
    A0 = o.full_action()
    for l in range(o.Np):
        pl = p[l] + wp[l] * rng.normal()
        dA, S = o.param_delta_A(l, pl)
        p2 = p.copy(); p2[l] = pl
        brute = float(o.full_action(None, p2) - A0)
        assert abs(dA - brute) <= 20e-15 * float(abs(A0)) + 1e-13 * S, (l, dA, brute)


def test_param_delta_A_linear_closed_form():
    # D = 1: A_d = (Rf/2) sum (x_{n+1} - a x_n)^2 is quadratic in a:
    # dA(a -> a') = (Rf/2) [ (a'^2 - a^2) Sxx - 2 (a' - a) Sxy ]
    rng = np.random.default_rng(2)
    M = 12
    o = OracleChain(MODEL_LINEAR, 1, 1, M, 1.0, 3.0, [7.0], [0.8])
    xs = rng.normal(size=M + 1)
    o.set_data(rng.normal(size=M + 1)); o.set_proposal([0.1], [0.1]); o.set_path(xs)
    Sxx, Sxy = np.sum(xs[:-1] ** 2), np.sum(xs[:-1] * xs[1:])
    a, a2 = 0.8, 0.93
    expect = 0.5 * 7.0 * ((a2**2 - a**2) * Sxx - 2 * (a2 - a) * Sxy)
    assert np.isclose(o.param_delta_A(0, a2)[0], expect, rtol=1e-12)


def test_antisymmetry():
    # dA(x -> x') = -dA(x' -> x)  to rounding relative to the term scale S
    w, o = small_hh(32)
    rng = np.random.default_rng(4)
    x, _ = o.get_path()
    for n in (0, 1, 7, 16, 31, 32):
        xp = x[n] + w.w_state * rng.normal(size=4)
        d1, S1 = o.site_delta_A(n, xp)
        X2 = x.copy(); X2[n] = xp
        o.set_path(X2)
        d2, S2 = o.site_delta_A(n, x[n])
        o.set_path(x)
        assert abs(d1 + d2) <= 4e-15 * S1
        assert np.isclose(S1, S2, rtol=1e-12)


def test_telescoping_over_a_sweep():
    # sum of accepted dA over one sweep (states then parameters) = A(after) - A(before)
    for cfg, M in ((0, 64), (2, 64)):
        w = make_workload(cfg, M=M, seed=9)
        o = OracleChain.from_workload(w)
        for t in range(5):
            A0 = o.full_action()
            o.sweep(1, seed=17)
            tr = o.trace()
            tot = tr["dA"][tr["acc"] == 1].sum() + np.nansum(np.where(tr["accp"] == 1, tr["dAp"], 0.0))
            A1 = o.full_action()
            assert abs(tot - float(A1 - A0)) <= 1e-12 * max(1.0, float(abs(A0))), (cfg, t)
            assert tr["acc"].sum() > 0


def test_cache_coherence_after_runs():
    # (iii) after any run g[n] equals the increment recomputed from (x_n, p) -- including accepted parameter moves
    w = make_workload(2, M=48, seed=21)
    o = OracleChain.from_workload(w)
    o.sweep(40, seed=3)
    x, p = o.get_path()
    g = o.get_cache()
    st = o.stats()
    assert st[0, 4:].sum() > 0, "no parameter move was accepted; test is vacuous"
    for n in range(w.M):
        ref = oracle.step_increment(MODEL_HH, x[n], p, w.I[0, n], w.I[0, n + 1], w.dt)
        assert np.array_equal(g[n], ref)


def test_order_independence_within_half_sweep():
    # "each even n, and then each odd n can be updated independently, in any order or simultaneously"
    w = make_workload(2, M=65, seed=8)       # odd M: last site is odd
    res = []
    for order in (0, 1, 2):
        o = OracleChain.from_workload(w)
        o.sweep(6, seed=5, order=order)
        res.append(o.get_path())
    for x, p in res[1:]:
        assert np.array_equal(x, res[0][0]) and np.array_equal(p, res[0][1])


def test_even_sites_first_then_odd():
    # G2: even first.  After ONE even half-sweep-only... observable: the odd sites' dA are computed against the
    # already-updated even neighbours.  Recompute odd-site dA from the trace on the post-even path.
    w = make_workload(0, M=20, seed=2)
    o = OracleChain.from_workload(w)
    x0, _ = o.get_path()
    o.sweep(1, seed=1)
    tr = o.trace()
    # reconstruct the path after the even half-sweep
    xe = x0.copy()
    for n in range(0, w.M + 1, 2):
        if tr["acc"][n]:
            xe[n] = tr["xprop"][n]
    o2 = OracleChain.from_workload(w)
    o2.set_path(xe)
    for n in range(1, w.M + 1, 2):
        assert np.isclose(o2.site_delta_A(n, tr["xprop"][n])[0], tr["dA"][n], rtol=1e-13, atol=1e-13)
    # and even sites were evaluated against the ORIGINAL odd neighbours
    o3 = OracleChain.from_workload(w)
    for n in range(0, w.M + 1, 2):
        assert o3.site_delta_A(n, tr["xprop"][n])[0] == tr["dA"][n]


def test_accept_rule_limits():
    w = make_workload(0, M=40, seed=6)
    # (v) Rm = Rf = 0  => dA = 0 => always accepted (log u < 0 strictly)
    o = OracleChain(MODEL_HH, 4, 1, w.M, w.dt, 0.0, np.zeros(4), w.p0[0])
    o.set_data(w.y[0], w.I[0]); o.set_proposal(w.w_state); o.set_path(w.x0[0])
    o.sweep(3, seed=1)
    st = o.stats()
    assert np.all(st[0, :4] == st[1, :4]) and st[1, 0] == 3 * (w.M + 1)
    # zero widths => x' = x, dA = 0 exactly, accepted, path unchanged
    o = OracleChain.from_workload(w)
    o.set_proposal(np.zeros(4))
    o.sweep(2, seed=1)
    assert np.array_equal(o.get_path()[0], w.x0[0])
    tr = o.trace()
    assert np.all(tr["dA"] == 0.0) and np.all(tr["acc"] == 1)
    # huge precision => large positive dA => (almost) never accepted, path stays
    o = OracleChain(MODEL_HH, 4, 1, w.M, w.dt, 1e12, np.full(4, 1e14), w.p0[0])
    o.set_data(w.y[0], w.I[0]); o.set_proposal(w.w_state); o.set_path(w.x_true[0])
    o.sweep(2, seed=1)
    assert o.stats()[0, 0] < 0.5 * o.stats()[1, 0]
    # NaN dA rejects (G3): a NaN in the data poisons the measurement term at that site
    y = w.y[0].copy(); y[5] = np.nan
    o = OracleChain.from_workload(w); o.set_data(y, w.I[0])
    o.sweep(4, seed=2)
    assert np.array_equal(o.get_path()[0][5], w.x0[0][5])


def test_metropolis_rule_is_log_u_less_than_minus_dA():
    w = make_workload(2, M=50, seed=6)
    o = OracleChain.from_workload(w)
    for t in range(10):
        o.sweep(1, seed=4)
        tr = o.trace()
        assert np.array_equal(tr["acc"].astype(bool), tr["logu"] < -tr["dA"])
        ev = ~np.isnan(tr["dAp"])
        assert np.array_equal(tr["accp"][ev].astype(bool), tr["logup"][ev] < -tr["dAp"][ev])
        assert np.all(tr["logu"] < 0)
        # accept uniform is the stream-1 draw of (site, sweep): recompute one
        n = 7
        wd = oracle.draw_words(4, t, 0, n, 1, 0)
        assert tr["logu"][n] == np.log(oracle.u01_from_two_words(wd[0], wd[1]))


def test_out_of_bounds_parameter_never_accepted():
    w = make_workload(2, M=30, seed=6)
    o = OracleChain.from_workload(w)
    p0 = w.p0[0].copy()
    # bounds that exclude every proposal except an exact repeat
    o.set_bounds(p0, p0)
    o.set_proposal(w.w_state, w.w_param * 50)
    g0 = o.get_cache()
    o.set_proposal(np.zeros(4), w.w_param * 50)
    o.sweep(20, seed=3)
    x, p = o.get_path()
    assert np.array_equal(p, p0) and np.array_equal(o.get_cache(), g0)
    st = o.stats()
    assert np.all(st[0, 4:] == 0) and np.all(st[1, 4:] == 20)
    # frozen parameters (w = 0) are not even proposed
    o = OracleChain.from_workload(w)
    wp = w.w_param.copy(); wp[[1, 4]] = 0.0
    o.set_proposal(w.w_state, wp)
    o.sweep(5, seed=3)
    st = o.stats()
    assert st[1, 4 + 1] == 0 and st[1, 4 + 4] == 0 and st[1, 4 + 0] == 5


def test_sweep_split_equals_sweep_whole():
    # (viii) counter RNG + absolute sweep index: sweep(20) == sweep(8) + sweep(12), bit for bit
    w = make_workload(2, M=40, seed=13)
    a = OracleChain.from_workload(w); a.set_accum(True, 2); a.reset_moments(); a.sweep(20, seed=9)
    b = OracleChain.from_workload(w); b.set_accum(True, 2); b.reset_moments(); b.sweep(8, seed=9); b.sweep(12, seed=9)
    assert b.sweep_index == 20
    for u, v in zip(a.get_path(), b.get_path()):
        assert np.array_equal(u, v)
    ma, mb = a.moments(), b.moments()
    assert ma[2] == mb[2] == 10
    assert np.array_equal(ma[0], mb[0]) and np.array_equal(ma[1], mb[1])
    # resume from a checkpoint: (path, p, sweep index) is the whole state
    c = OracleChain.from_workload(w); c.sweep(8, seed=9)
    x, p = c.get_path()
    d = OracleChain.from_workload(w); d.set_params(p); d.set_path(x); d.sweep_index = 8; d.sweep(12, seed=9)
    e = OracleChain.from_workload(w); e.sweep(20, seed=9)
    assert np.array_equal(d.get_path()[0], e.get_path()[0]) and np.array_equal(d.get_path()[1], e.get_path()[1])


def test_moments_and_histograms_are_plain_sample_statistics():
    w = make_workload(2, M=24, seed=13)
    o = OracleChain.from_workload(w)
    o.sweep(5, seed=2)
    o.hist_config([3, -1, 24], [0, 6, 2], [-80.0, 0.7, 0.0], [-40.0, 0.9, 1.0], 8)
    o.set_accum(True, 1); o.reset_moments()
    xs, ps = [], []
    for t in range(30):
        o.sweep(1, seed=2)
        x, p = o.get_path(); xs.append(x); ps.append(p)
    xs, ps = np.array(xs), np.array(ps)
    mx, mp, n = o.moments()
    assert n == 30
    assert np.allclose(mx[0], xs.mean(0), rtol=1e-13, atol=1e-13) and np.allclose(mx[1], xs.var(0), rtol=1e-9, atol=1e-15)
    assert np.allclose(mp[0], ps.mean(0), rtol=1e-13) and np.allclose(mp[1], ps.var(0), rtol=1e-9, atol=1e-18)
    h = o.hist()
    for s, (vals, lo, hi) in enumerate(((xs[:, 3, 0], -80.0, -40.0), (ps[:, 6], 0.7, 0.9), (xs[:, 24, 2], 0.0, 1.0))):
        ref, _ = np.histogram(vals, bins=8, range=(lo, hi))
        under, over = np.sum(vals < lo), np.sum(vals >= hi)
        # numpy puts v == hi in the last bin; our convention sends it to overflow -- no such sample here
        assert h[s, 0] == under and h[s, -1] == over and np.array_equal(h[s, 1:-1], ref)
        assert h[s].sum() == 30
    # n_skip: every 3rd sweep
    o.set_accum(True, 3); o.reset_moments(); o.sweep(10, seed=2)
    assert o.moments()[2] == 4        # sweeps 0,3,6,9 after the reset
