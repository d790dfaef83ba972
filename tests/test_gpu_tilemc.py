"""Parity of the many-chain tile-resident engine (PIMC_ENGINE_TILE_MC, pimc_tilemc_kernel.cuh) with the oracle.

The engine has no debug trace, so the protocol is SURVEY.md §8(c) T2 (free-running): with UNIFORM proposals every chain must
stay bit-identical to the oracle's (path, parameters, counters, histograms; moments to rounding), through halo exchanges,
per-chain all-gathers, several waves of chains, partly filled waves, ragged last tiles; with Gaussian proposals the chains
agree to rounding as long as no decision falls into the near-tie window (checked against the trace-capable engines, which
are themselves compared with the oracle decision by decision)."""
import numpy as np
import pytest

from helpers import gpu_handle, oracle_chains
from workloads import make_workload

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def P():
    import torch
    import paper_1103_4887_b200 as P
    assert torch.cuda.is_available()
    P.lib()
    return P


def _mc_handle(P, w, launch=None, halo=-1, kind=1, dtype=64, with_params=True):
    h = gpu_handle(w, kind=kind, dtype=dtype, with_params=with_params)
    if launch:
        h.set_launch(*launch)
    h.set_engine(P.ENGINE_TILE_MC, halo)
    assert h.get_engine()["engine"] == P.ENGINE_TILE_MC
    return h


def _compare_free_running(P, w, h, n_sweeps, seed, chains=None, n_skip=1, hist=None, split=None):
    h.set_accum(True, n_skip); h.reset_moments()
    if hist:
        h.hist_config(*hist)
    for n in (split or [n_sweeps]):
        h.sweep(n, seed=seed)
    assert h.fault() == 0
    xg, pg = [a.cpu().numpy() for a in h.get_path()]
    st = h.stats().cpu().numpy().astype(np.uint64)
    mx, mp, n = h.moments()
    mx, mp = mx.cpu().numpy(), mp.cpu().numpy()
    hg = h.hist().cpu().numpy().astype(np.uint64) if hist else None
    g = h.get_cache().cpu().numpy()
    orcs = oracle_chains(w, kind=1)
    for c in (range(w.n_chains) if chains is None else chains):
        o = orcs[c]
        o.set_accum(True, n_skip); o.reset_moments()
        if hist:
            o.hist_config(*hist)
        o.sweep(n_sweeps, seed=seed)
        xo, po = o.get_path()
        assert np.array_equal(xg[c], xo), (c, np.abs(xg[c] - xo).max(), np.nonzero(np.any(xg[c] != xo, axis=1))[0][:10])
        assert np.array_equal(pg[c], po), c
        assert np.array_equal(st[c], o.stats()), (c, st[c], o.stats())
        ox, op, on = o.moments()
        assert n == on
        assert np.allclose(mx[c], ox, rtol=1e-13, atol=1e-13), c
        assert np.allclose(mp[c], op, rtol=1e-13, atol=1e-16), c
        if hist:
            assert np.array_equal(hg[c], o.hist()), c
        og = o.get_cache()
        assert np.max(np.abs(g[c] - og) / np.maximum(np.abs(og), 1e-3)) < 1e-12, c      # different elementary-function libraries


@pytest.mark.parametrize("M,n_chains,launch,halo", [
    (1000, 5, None, -1),          # 5 tiles per chain (last one ragged), 25 groups: one wave, one group per CTA
    (1000, 5, (0, 256), 4),       # two groups per CTA, exchange every 2 sweeps
    (777, 3, (0, 384), 16),       # three groups per CTA, odd M, deepest halo
    (200, 7, None, -1),           # whole chain in one group: no hand-off at all
    (3000, 50, None, 8),          # 13 tiles x 50 chains = 650 groups > 592 slots: two waves
])
def test_free_running_uniform_bit_identical(P, M, n_chains, launch, halo):
    w = make_workload(4, M=M, n_chains=n_chains)
    h = _mc_handle(P, w, launch=launch, halo=halo)
    sel = ([3, M, 10, -1], [0, 3, 1, 0], [-100.0, -1.0, -1.0, 50.0], [60.0, 2.0, 2.0, 200.0], 16)
    chains = None if n_chains <= 8 else [0, 1, 24, 25, 26, 49]
    _compare_free_running(P, w, h, 30, seed=5, chains=chains, n_skip=3, hist=sel)


def test_split_calls_states_only_params_only(P):
    w = make_workload(4, M=900, n_chains=4)
    h = _mc_handle(P, w)
    _compare_free_running(P, w, h, 21, seed=9, split=[8, 1, 12])
    # states-only + params-only == full sweep, sweep by sweep (the oracle has no parameters-only sweep)
    e = _mc_handle(P, w)
    for t in range(6):
        e.sweep_index = t; e.sweep_states_only(1, seed=3); e.sweep_index = t; e.sweep_params_only(1, seed=3)
    f = _mc_handle(P, w); f.sweep(6, seed=3)
    orcs = oracle_chains(w, kind=1)
    xe, pe = [a.cpu().numpy() for a in e.get_path()]
    xf, pf = [a.cpu().numpy() for a in f.get_path()]
    assert np.array_equal(xe, xf) and np.array_equal(pe, pf)
    for c, o in enumerate(orcs):
        o.sweep(6, seed=3)
        xo, po = o.get_path()
        assert np.array_equal(xf[c], xo) and np.array_equal(pf[c], po), c
    # states-only sweeps with accumulation against the oracle's
    g = _mc_handle(P, w); g.set_accum(True, 2); g.reset_moments(); g.sweep_states_only(9, seed=3)
    mx = g.moments()[0].cpu().numpy()
    for c, o in enumerate(oracle_chains(w, kind=1)):
        o.set_accum(True, 2); o.reset_moments(); o.sweep(9, seed=3, do_params=False)
        assert np.array_equal(g.get_path()[0].cpu().numpy()[c], o.get_path()[0]), c
        assert np.allclose(mx[c], o.moments()[0], rtol=1e-13, atol=1e-13), c


def test_cfg4_full_size_in_bench_launch(P):
    # config 4 as given: 128 chains x M = 8192; automatic engine = TILE_MC (35 tiles per chain, 16 chains per wave, 8 waves);
    # 12 sweeps in one call (three halo exchanges, 84 all-gathers per chain); 12 chains spread over the waves against the oracle
    w = make_workload(4)
    h = gpu_handle(w, kind=1)
    eng, shape = h.get_engine(), h.get_launch()
    print("cfg4 automatic:", eng, shape)
    assert eng["engine"] == P.ENGINE_TILE_MC, eng
    _compare_free_running(P, w, h, 12, seed=11, chains=[0, 15, 16, 17, 40, 63, 64, 77, 100, 111, 112, 127])


def test_gaussian_proposals_agree_with_the_global_engine(P):
    # Gaussian proposals are not bit-reproducible against libm, but the engines of this library share their arithmetic for the
    # proposals: same draws, same decisions => identical paths, unless a decision falls into the near-tie window of the
    # (differently ordered) parameter sums.  The GLOBAL engine is compared with the oracle decision by decision elsewhere.
    w = make_workload(4, M=1500, n_chains=6)
    a = _mc_handle(P, w, kind=0)
    b = gpu_handle(w, kind=0); b.set_engine(P.ENGINE_GLOBAL)
    a.sweep(40, seed=2); b.sweep(40, seed=2)
    xa, pa = [t.cpu().numpy() for t in a.get_path()]
    xb, pb = [t.cpu().numpy() for t in b.get_path()]
    assert np.array_equal(a.stats().cpu().numpy(), b.stats().cpu().numpy())
    assert np.allclose(xa, xb, rtol=0, atol=1e-10) and np.allclose(pa, pb, rtol=1e-12)


def test_fp32_and_classic_kinetics(P):
    w = make_workload(4, M=1200, n_chains=3)
    h = _mc_handle(P, w, dtype=32)
    orcs = oracle_chains(w, state_dtype=32, kind=1)
    h.sweep(15, seed=4)
    xg, pg = [a.cpu().numpy() for a in h.get_path()]
    for c, o in enumerate(orcs):
        o.sweep(15, seed=4)
        xo, po = o.get_path()
        # fp32 states: the two sides round the model step differently (fp32 kernels vs fp64 oracle on fp32 states), so a decision may
        # differ; uniform proposals keep unaffected sites bit-identical
        same = np.mean(np.all(xg[c] == xo.astype(np.float32), axis=1))
        assert same > 0.98, (c, same)
    wc = make_workload(4, M=1200, n_chains=3, kinetics="classic")
    h = _mc_handle(P, wc)
    _compare_free_running(P, wc, h, 15, seed=4)


def test_unsupported_settings_fall_back_or_refuse(P):
    w = make_workload(4, M=1000, n_chains=100)
    h = gpu_handle(w, kind=1)
    assert h.get_engine()["engine"] == P.ENGINE_TILE_MC           # automatic: more chains than the one-tile-per-SM engine can hold
    h.enable_trace()
    assert h.get_engine()["engine"] != P.ENGINE_TILE_MC           # the debug trace lives in the other engines
    h.disable_trace()
    h.set_discretisation(P.DISC_TRAPEZOID)
    assert h.get_engine()["engine"] != P.ENGINE_TILE_MC
    with pytest.raises(P.PimcError):
        h.set_engine(P.ENGINE_TILE_MC)
    w1 = make_workload(1, M=500)
    h1 = gpu_handle(w1, with_params=False)
    with pytest.raises(P.PimcError):
        h1.set_engine(P.ENGINE_TILE_MC)
