"""GPU parity for the paper's trapezoid discretisation (PIMC_DISC_TRAPEZOID; Eq. 7)
against the oracle's set_discretisation(1): teacher-forced per-site and parameter Delta-A, free-running bit-identical
chains with uniform proposals, cache coherence (c_n = (dt/2) F(x_n), n = 0..M), batched chains, fp32, edge sizes."""
import numpy as np
import pytest

from helpers import TOL32, TOL64, gpu_handle, oracle_chains, teacher_forced
from workloads import make_workload

pytestmark = pytest.mark.gpu
TRAP = 1


@pytest.fixture(scope="module")
def P():
    import torch
    import paper_1103_4887_b200 as P
    assert torch.cuda.is_available()
    P.lib()
    return P


CASES = [
    # name, cfg, M, launch, with_params, n_sweeps, engine (0 automatic = tile-resident when it fits, 1 global-memory)
    ("cfg0_M256_auto", 0, 256, None, False, 40, 0),
    ("cfg0_M257_3ctas_global", 0, 257, (3, 32), False, 20, 1),
    ("cfg2_M600_auto", 2, 600, None, True, 40, 0),
    ("cfg2_M601_5ctas_global", 2, 601, (5, 64), True, 20, 1),
    ("cfg2_M601_5ctas_tile", 2, 601, (5, 192), True, 20, 2),
    ("cfg2_M333_1cta_global", 2, 333, (1, 96), True, 20, 1),
    ("cfg1_M999_7ctas_global", 1, 999, (7, 32), False, 20, 1),
    ("cfg1_M1000_auto", 1, 1000, None, False, 40, 0),
    ("cfg2_M1201_38tiles_tile", 2, 1201, None, True, 20, 2),
    ("cfg2_M4000_126tiles_of_64_tile", 2, 4000, (126, 64), True, 10, 2),
]


@pytest.mark.parametrize("name,cfg,M,launch,with_params,n_sweeps,engine", CASES, ids=[c[0] for c in CASES])
def test_teacher_forced_parity_trapezoid(P, name, cfg, M, launch, with_params, n_sweeps, engine):
    w = make_workload(cfg, M=M)
    h = gpu_handle(w, with_params=with_params, disc=TRAP)
    if engine:
        h.set_engine(engine)
    if launch:
        h.set_launch(*launch)
    if engine:
        assert h.get_engine()["engine"] == engine
    orcs = oracle_chains(w, with_params=with_params, disc=TRAP)
    rep = teacher_forced(w, h, orcs, n_sweeps, seed=20110347, do_params=with_params, disc=TRAP)
    print(name, h.get_launch(), rep)
    assert rep["sites"] == n_sweeps * (M + 1)
    assert rep["max_rel"] <= TOL64 and rep["mismatch_outside_window"] == 0 and rep["ties"] <= 2, rep
    assert rep["max_xprop_ulp"] <= 4.0 and rep["accepted"] > 0, rep
    if with_params:
        assert rep["param_moves"] > 0 and rep["max_param_rel"] <= TOL64, rep
    assert rep["max_path_diff"] <= 1e-12


@pytest.mark.parametrize("cfg,M,launch,engine", [(0, 256, None, 0), (2, 500, (4, 64), 1), (2, 500, (4, 192), 2), (1, 700, (3, 128), 1),
                                                 (3, 4001, None, 0), (3, 4001, None, 1),
                                                 # the sufficient-statistics parameter moves of the tile engine in the shapes its exchange distinguishes:
                                                 # 38 tiles of 64 threads (one statistic per reducer, fewer compute threads than statistics),
                                                 # 126 tiles of 64 threads (more tiles than threads), 9 tiles (several statistics per reducer), one tile
                                                 (2, 1201, None, 2), (2, 4000, (126, 64), 2), (2, 2000, (9, 256), 2), (2, 200, None, 2)])
def test_free_running_uniform_bit_identical_trapezoid(P, cfg, M, launch, engine):
    w = make_workload(cfg, M=M)
    h = gpu_handle(w, kind=1, disc=TRAP)
    if engine:
        h.set_engine(engine)
    if launch:
        h.set_launch(*launch)
    o = oracle_chains(w, kind=1, disc=TRAP)[0]
    h.set_accum(True, 2); o.set_accum(True, 2)
    h.reset_moments(); o.reset_moments()
    h.sweep(60, seed=5); o.sweep(60, seed=5)
    xg, pg = [a.cpu().numpy() for a in h.get_path()]
    xo, po = o.get_path()
    assert np.array_equal(xg[0], xo), np.abs(xg[0] - xo).max()
    assert np.array_equal(pg[0], po)
    assert np.array_equal(h.stats().cpu().numpy()[0].astype(np.uint64), o.stats())
    mx, mp, n = h.moments()
    ox, op, on = o.moments()
    assert n == on == 30
    assert np.allclose(mx.cpu().numpy()[0], ox, rtol=1e-13, atol=1e-13)
    # cache coherence on the device: c_n = (dt/2) F(x_n, p; I_n) for n = 0..M, against the oracle's recomputation
    g = h.get_cache().cpu().numpy()[0]
    og = o.get_cache()
    assert g.shape == og.shape == (M + 1, w.D)
    # (the gate rates (a_inf - a)/tau cancel, so the error is relative to the scale of the terms: (dt/2) x (100 mV/ms, 1/ms))
    scale = np.maximum(np.abs(og), 0.5 * w.dt * (np.array([100.0, 1.0, 1.0, 1.0]) if w.D == 4 else np.ones(w.D)))
    assert np.max(np.abs(g - og) / scale) < 1e-13


def test_batched_chains_and_fp32_trapezoid(P):
    w = make_workload(4, M=300, n_chains=5)
    h = gpu_handle(w, launch=(1, 64), disc=TRAP)
    rep = teacher_forced(w, h, oracle_chains(w, disc=TRAP), 15, seed=99, disc=TRAP)
    assert rep["max_rel"] <= TOL64 and rep["mismatch_outside_window"] == 0 and rep["max_param_rel"] <= TOL64, rep
    w = make_workload(2, M=600)
    h = gpu_handle(w, dtype=32, disc=TRAP)
    rep = teacher_forced(w, h, oracle_chains(w, state_dtype=32, disc=TRAP), 15, seed=3, tol=TOL32, state_dtype=32, disc=TRAP)
    assert rep["max_rel"] <= TOL32 and rep["mismatch_outside_window"] == 0, rep


def test_edge_sizes_switching_and_engine_rule_trapezoid(P):
    import paper_1103_4887_b200 as Pm
    for M in (1, 2, 5):
        w = make_workload(0, M=M)
        h = gpu_handle(w, with_params=False, disc=TRAP)
        rep = teacher_forced(w, h, oracle_chains(w, with_params=False, disc=TRAP), 10, seed=3, do_params=False, disc=TRAP)
        assert rep["max_rel"] <= TOL64 and rep["mismatch_outside_window"] == 0, (M, rep)
    # switching the discretisation on a live handle rebuilds the cache
    w = make_workload(2, M=300)
    h = gpu_handle(w)
    h.sweep(3, seed=1)
    h.set_discretisation(Pm.DISC_TRAPEZOID)
    assert h.get_cache().shape == (1, 301, 4)
    h.sweep(3, seed=1)
    h.set_discretisation(Pm.DISC_RK4MAP)
    assert h.get_cache().shape == (1, 300, 4)
    with pytest.raises(Pm.PimcError):
        h.set_discretisation(7)


@pytest.mark.parametrize("engine", ["tile", "global_one_cta_per_chain"])
def test_sufficient_statistics_parameter_moves_edge_cases(P, engine):
    # trapezoid rule: the parameter moves come from one reduction of path sums per sweep -- on the tile engine (several
    # chains with several tiles each, one reducer set per chain) and on the global-memory engine with one CTA per chain (block reduction).
    # Tight bounds (proposals outside are rejected unevaluated), a frozen parameter, the parameter record, both kinetics: chains
    # bit-identical to the oracle's
    import paper_1103_4887_b200 as Pm
    for kinetics in ("tanh", "classic"):
        w = make_workload(4, M=700, n_chains=3, kinetics=kinetics)
        wp = w.w_param.copy(); wp[2] = 0.0                       # gL frozen
        lo, hi = w.p0 - 1.5 * wp, w.p0 + 1.5 * wp                 # bounds 1.5 step sizes around the start: a good share of the proposals falls outside
        lo[:, 2], hi[:, 2] = w.lo[:, 2], w.hi[:, 2]
        h = gpu_handle(w, kind=1, disc=TRAP)
        h.set_proposal(w.w_state, wp, 1)
        h.set_bounds(lo, hi)
        if engine == "tile":
            h.set_engine(Pm.ENGINE_TILE)
            assert h.get_launch()["ctas_per_chain"] > 1
        else:
            h.set_engine(Pm.ENGINE_GLOBAL); h.set_launch(1, 160)
            assert h.get_launch()["ctas_per_chain"] == 1 and h.get_engine()["engine"] == Pm.ENGINE_GLOBAL
        h.set_accum(True, 1); h.reset_moments()
        rec = h.param_trace(25)
        h.sweep(25, seed=21)
        xg, pg = [a.cpu().numpy() for a in h.get_path()]
        st = h.stats().cpu().numpy().astype(np.uint64)
        for c, o in enumerate(oracle_chains(w, kind=1, disc=TRAP)):
            o.set_proposal(w.w_state, wp, 1)
            o.set_bounds(lo[c], hi[c])
            o.set_accum(True, 1); o.reset_moments(); o.param_trace_enable(True)
            o.sweep(25, seed=21)
            xo, po = o.get_path()
            assert np.array_equal(xg[c], xo) and np.array_equal(pg[c], po), (kinetics, c)
            assert np.array_equal(st[c], o.stats()), (kinetics, c, st[c], o.stats())
            assert np.array_equal(rec.cpu().numpy()[c], o.param_trace()), (kinetics, c)
            acc, prop = o.stats()[0][4:], o.stats()[1][4:]
            assert prop[2] == 0 and acc[2] == 0 and np.all(prop[[0, 1, 3, 4, 5, 6]] == 25)
            assert 0 < acc.sum() < prop.sum()                     # some accepted, some rejected (incl. out of bounds)
