"""Pins for the oracle's optional diagnostics: the per-sweep parameter record (Fig. 4) and the model / observation
errors eps_n, delta_n with their running statistics.  Expectations come from the DEFINITION of the action
(A = sum (R_o/2) delta^2 + sum (R_d/2) eps^2), from plain numpy statistics of values collected one sweep at
a time, and from the acceptance counters -- not from the routines under test."""
import numpy as np
import pytest

from oracle import OracleChain
from workloads import make_workload


@pytest.mark.parametrize("cfg,disc", [(2, 0), (2, 1), (1, 0), (1, 1)])
def test_residuals_reassemble_the_action(cfg, disc):
    w = make_workload(cfg, M=50)
    o = OracleChain.from_workload(w)
    if disc:
        o.set_discretisation(1)
    o.sweep(7, seed=5)
    eps, delta = o.residuals()
    assert eps.shape == (w.M, w.D) and delta.shape == (w.M + 1, w.L)
    assert np.all(delta[0] == 0.0)                                   # y_0 is not part of the action (n = 1..M)
    x, _ = o.get_path()
    assert np.array_equal(delta[1:, 0], np.asarray(w.y[0], float).reshape(w.M + 1, -1)[1:, 0] - x[1:, 0])
    A = 0.5 * w.Rm * np.sum(delta.astype(np.longdouble) ** 2) + np.sum(0.5 * np.asarray(w.Rf, np.longdouble) * eps.astype(np.longdouble) ** 2)
    ref = o.full_action()
    assert abs(A - ref) <= 1e-12 * abs(ref), (A, ref)
    # power: the residual of the OTHER discretisation does not reassemble it
    o.set_discretisation(1 - disc)
    e2, _ = o.residuals()
    A2 = 0.5 * w.Rm * np.sum(delta.astype(np.longdouble) ** 2) + np.sum(0.5 * np.asarray(w.Rf, np.longdouble) * e2.astype(np.longdouble) ** 2)
    assert abs(A2 - ref) > 1e-6 * abs(ref)


def test_parameter_record_is_the_chain_of_parameters():
    w = make_workload(2, M=60)
    o = OracleChain.from_workload(w)
    o.param_trace_enable(True)
    o.set_accum(True, 1); o.reset_moments()
    rec = []
    for _ in range(40):
        o.sweep(1, seed=9)
        rec.append(o.get_path()[1].copy())
    rec = np.asarray(rec)
    tr = o.param_trace()
    assert np.array_equal(tr, rec)
    # accepted parameter moves = changes of the recorded value (n_skip = 1), per parameter
    st = o.stats()
    changes = np.count_nonzero(np.diff(np.vstack([w.p0[0][None], tr]), axis=0), axis=0)
    assert np.array_equal(changes, st[0, w.D:].astype(int)) and changes.sum() > 10
    # the running moments are the plain statistics of the record
    _, mp, n = o.moments()
    assert n == 40 and np.allclose(mp[0], tr.mean(0), rtol=1e-13) and np.allclose(mp[1], tr.var(0), rtol=1e-9, atol=1e-18)
    # every n_skip-th sweep only; cleared by a reset; off = nothing kept
    o.set_accum(True, 4); o.reset_moments()
    assert o.param_trace().shape == (0, 7)
    o.sweep(21, seed=9)
    assert o.param_trace().shape == (6, 7) and np.array_equal(o.param_trace()[-1], o.get_path()[1])
    o.param_trace_enable(False)
    o.sweep(8, seed=9)
    assert o.param_trace().shape == (0, 7)


@pytest.mark.parametrize("disc", [0, 1])
def test_residual_statistics_are_plain_statistics_of_the_sampled_paths(disc):
    w = make_workload(2, M=40)
    o = OracleChain.from_workload(w)
    if disc:
        o.set_discretisation(1)
    o.residual_stats_enable(True)
    o.set_accum(True, 1); o.reset_moments()
    E, Dl = [], []
    for _ in range(25):
        o.sweep(1, seed=4)
        e, d = o.residuals()
        E.append(e); Dl.append(d)
    E, Dl = np.asarray(E), np.asarray(Dl)
    me, ve, md, vd, n = o.residual_stats()
    assert n == 25
    assert np.allclose(me, E.mean(0), rtol=1e-12, atol=1e-15) and np.allclose(ve, E.var(0), rtol=1e-8, atol=1e-15)
    assert np.allclose(md, Dl.mean(0), rtol=1e-12, atol=1e-15) and np.allclose(vd, Dl.var(0), rtol=1e-8, atol=1e-15)
    o.reset_moments()
    assert o.residual_stats()[4] == 0 and np.all(o.residual_stats()[0] == 0)
