"""Parity at BASELINE.json's full sizes, in the launch configuration bench.py times, and the fp32 variant of config 3.

Full-size cases use what the oracle can still do in seconds: a few teacher-forced sweeps (every site compared), and
free-running sweeps with UNIFORM proposals, which are bit-reproducible, so path, parameters, counters and the traced
Delta-A of every site must agree."""
import numpy as np
import pytest

from helpers import TOL32, TOL64, gpu_handle, oracle_chains, teacher_forced
from workloads import make_workload

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def P():
    import torch
    import paper_1103_4887_b200 as P
    assert torch.cuda.is_available()
    P.lib()
    return P


def test_cfg3_full_size_teacher_forced_in_bench_launch(P):
    # config 3: HH, M = 32768, dt = 0.01, states + 7 parameters; automatic launch = the one bench.py times
    w = make_workload(3)
    h = gpu_handle(w)
    shape = h.get_launch()
    assert w.M == 32768 and shape["ctas_per_chain"] >= 100, shape      # spread over the SMs, tile-resident engine
    rep = teacher_forced(w, h, oracle_chains(w), 3, seed=20110347)
    print("cfg3 full size", shape, rep)
    assert rep["sites"] == 3 * (w.M + 1)
    assert rep["max_rel"] <= TOL64 and rep["mismatch_outside_window"] == 0 and rep["ties"] <= 1, rep
    assert rep["param_moves"] > 0 and rep["max_param_rel"] <= TOL64, rep
    assert rep["max_xprop_ulp"] <= 4.0 and rep["max_path_diff"] <= 1e-12, rep


def oracle_chains_one(w, c, with_params):
    from oracle import OracleChain
    o = OracleChain.from_workload(w, chain=c, with_params=with_params)
    o.set_proposal(w.w_state, w.w_param if with_params else None, 0)
    return o


def _free_running_uniform(P, w, n_sweeps, seed, chains=None, disc=0):
    h = gpu_handle(w, kind=1, disc=disc)
    tr = h.enable_trace()
    h.set_accum(True, 1); h.reset_moments()
    h.sweep(n_sweeps, seed=seed)
    xg, pg = [a.cpu().numpy() for a in h.get_path()]
    st = h.stats().cpu().numpy().astype(np.uint64)
    dA = tr["dA"].cpu().numpy(); acc = tr["acc"].cpu().numpy()
    mx, mp, n = h.moments()
    mx = mx.cpu().numpy()
    orcs = oracle_chains(w, kind=1, disc=disc)
    worst = 0.0
    for c in (range(w.n_chains) if chains is None else chains):
        o = orcs[c]
        o.set_accum(True, 1); o.reset_moments()
        o.sweep(n_sweeps, seed=seed)
        xo, po = o.get_path()
        assert np.array_equal(xg[c], xo), (c, np.abs(xg[c] - xo).max())
        assert np.array_equal(pg[c], po), c
        assert np.array_equal(st[c], o.stats()), c
        ot = o.trace()                                   # last sweep: same state on both sides, so every site compares
        assert np.array_equal(acc[c], ot["acc"]), c
        err = np.abs(dA[c] - ot["dA"]) / np.maximum(np.maximum(np.abs(ot["dA"]), ot["S"]), 1e-300)
        worst = max(worst, float(err.max()))
        ox, op, on = o.moments()
        assert n == on == n_sweeps
        assert np.allclose(mx[c], ox, rtol=1e-13, atol=1e-13)
    assert worst <= TOL64, worst
    return worst


def test_cfg3_full_size_free_running_bit_identical(P):
    w = make_workload(3)
    worst = _free_running_uniform(P, w, 24, seed=7)       # 24 sweeps: three halo exchanges of the tile engine
    print("cfg3 free-running, max dA error / scale:", worst)


def test_cfg3_full_size_production_variant_bit_identical(P):
    # The instantiation bench.py times: no debug trace, no annealing, no tuning (template flag TR = 0), stage-1 cache on,
    # automatic launch (148 CTAs x 256 threads), moments every sweep -- 40 sweeps in ONE launch, i.e. across five halo
    # exchanges and 280 grid-wide parameter all-reduces, then path, parameters, counters, histograms bit for bit and the
    # moments to 1e-13 against the oracle (uniform proposals: bit-reproducible draws).
    w = make_workload(3)
    n_sweeps, seed = 40, 20110348
    h = gpu_handle(w, kind=1)
    shape = h.get_launch()
    assert shape["ctas_per_chain"] >= 100 and shape["threads_per_cta"] == 256, shape
    sites = [0, 1, 221, 222, 16383, 32767, 32768, -1, -1]
    comps = [0, 1, 2, 3, 0, 1, 0, 0, 6]
    lo = [-100, 0, 0, 0, -100, 0, -100, 60, 0.5]
    hi = [60, 1, 1, 1, 60, 1, 60, 180, 1.5]
    h.hist_config(sites, comps, lo, hi, 16)
    h.set_accum(True, 1); h.reset_moments()
    n0 = h.launch_count
    h.sweep(n_sweeps, seed=seed)
    assert h.launch_count - n0 == 1
    assert h.fault() == 0
    xg, pg = [a.cpu().numpy() for a in h.get_path()]
    o = oracle_chains(w, kind=1)[0]
    o.hist_config(sites, comps, lo, hi, 16)
    o.set_accum(True, 1); o.reset_moments()
    o.sweep(n_sweeps, seed=seed)
    xo, po = o.get_path()
    assert np.array_equal(xg[0], xo), np.abs(xg[0] - xo).max()
    assert np.array_equal(pg[0], po)
    assert np.array_equal(h.stats().cpu().numpy().astype(np.uint64)[0], o.stats())
    assert np.array_equal(h.hist().cpu().numpy()[0], o.hist())
    mx, mp, n = h.moments()
    ox, op, on = o.moments()
    assert n == on == n_sweeps
    assert np.allclose(mx.cpu().numpy()[0], ox, rtol=1e-13, atol=1e-13) and np.allclose(mp.cpu().numpy()[0], op, rtol=1e-13, atol=1e-13)
    assert int(o.stats()[0, 4:].sum()) > 50          # parameter moves were accepted along the way (the caches flipped)


def test_cfg3_full_size_fp32_teacher_forced_in_bench_launch(P):
    # the fp32 variant of config 3 at the benchmarked size and launch: per-site Delta-A within 1e-5 (relative to max(|dA|, S))
    # of the fp64 oracle evaluated on the same fp32 states at the GPU's own fp32 proposals; proposals within a few FLOAT ulp
    w = make_workload(3)
    h = gpu_handle(w, dtype=32)
    shape = h.get_launch()
    assert shape["ctas_per_chain"] >= 100, shape
    rep = teacher_forced(w, h, oracle_chains(w, state_dtype=32), 2, seed=5, tol=TOL32, state_dtype=32)
    print("cfg3 fp32 full size", shape, rep)
    assert rep["sites"] == 2 * (w.M + 1)
    assert rep["max_rel"] <= TOL32 and rep["mismatch_outside_window"] == 0, rep
    assert rep["param_moves"] > 0 and rep["max_param_rel"] <= 10 * TOL32, rep
    assert rep["max_xprop_ulp"] <= 8.0 * 2.0**29, rep        # helpers.ulp_diff counts fp64 ulps: 8 float ulps of the operands' scale


def test_cfg3_full_size_trapezoid_bit_identical(P):
    # the paper's own discretisation (Eq. 7) at the benchmarked size, tile-resident engine, 148 CTAs
    w = make_workload(3)
    worst = _free_running_uniform(P, w, 20, seed=7, disc=1)
    print("cfg3 trapezoid free-running, max dA error / scale:", worst)


def test_cfg4_full_size_batched_chains_bit_identical(P):
    # config 4: 128 independent chains x M = 8192; every chain's path after 2 sweeps, 16 of them against the oracle
    w = make_workload(4)
    assert w.n_chains == 128 and w.M == 8192
    worst = _free_running_uniform(P, w, 2, seed=11, chains=list(range(0, 128, 8)))
    print("cfg4 free-running, max dA error / scale:", worst)


@pytest.mark.parametrize("cfg,M,launch,with_params", [(2, 600, None, True), (2, 601, (5, 64), True), (0, 256, None, False),
                                                      (1, 1000, None, False), (3, 4000, None, True)])
def test_fp32_teacher_forced_parity(P, cfg, M, launch, with_params):
    # config 3's fp32 variant: per-site Delta-A within 1e-5 of the fp64 oracle evaluated on the same fp32 states and the
    # GPU's own fp32 proposals (probe A.5)
    w = make_workload(cfg, M=M)
    h = gpu_handle(w, dtype=32, with_params=with_params, launch=launch)
    orcs = oracle_chains(w, state_dtype=32, with_params=with_params)
    rep = teacher_forced(w, h, orcs, 20, seed=3, tol=TOL32, do_params=with_params, state_dtype=32)
    print("fp32", cfg, M, h.get_launch(), rep)
    assert rep["max_rel"] <= TOL32, rep
    assert rep["mismatch_outside_window"] == 0, rep
    if with_params:
        assert rep["param_moves"] > 0 and rep["max_param_rel"] <= 10 * TOL32, rep
    assert rep["max_xprop_ulp"] <= 8.0 * 2.0**29, rep            # 8 float ulps (the helper counts fp64 ulps)


@pytest.mark.parametrize("cfg", [0, 1, 2, 3, 4])
def test_first_100_sweeps_of_every_config_identical_decisions(P, cfg):
    # north_star: "accept/reject decisions over the first 100 sweeps of each config must be identical except where
    # |dA + log u| < 1e-9, and the count of such cases is reported" -- the configs as given (Gaussian proposals, full size,
    # automatic launch); config 4 compares 4 of its 128 chains (the oracle needs 28 ms per chain and sweep)
    import torch
    w = make_workload(cfg)
    with_params = bool(np.any(w.w_param > 0))
    h = gpu_handle(w, with_params=with_params)
    chains = [0] if w.n_chains == 1 else [0, 41, 86, 127]
    orcs = {c: oracle_chains_one(w, c, with_params) for c in chains}
    tr = h.enable_trace()
    ties, decisions = 0, 0
    for t in range(100):
        h.sweep(1, seed=w.chain_seed)
        acc = tr["acc"].cpu().numpy(); accp = tr["accp"].cpu().numpy() if with_params else None
        resync = False
        for c, o in orcs.items():
            o.sweep(1, seed=w.chain_seed, do_params=with_params)
            ot = o.trace()
            bad = np.nonzero(acc[c] != ot["acc"])[0]
            for n in bad:
                assert abs(ot["dA"][n] + ot["logu"][n]) < 1e-9, (cfg, t, c, n)
            ties += len(bad)
            decisions += acc[c].size
            if with_params:
                badp = np.nonzero(accp[c] != ot["accp"])[0]
                for l in badp:
                    assert abs(ot["dAp"][l] + ot["logup"][l]) < 1e-9, (cfg, t, c, l)
                ties += len(badp)
                decisions += int(np.sum(~np.isnan(ot["dAp"])))
            resync = resync or len(bad) > 0 or (with_params and len(badp) > 0)
        if resync:            # protocol T2: record, verify the window, resync, continue
            xg, pg = [a.clone() for a in h.get_path()]
            for c, o in orcs.items():
                x, p = o.get_path()
                xg[c] = torch.as_tensor(x, device=xg.device); pg[c] = torch.as_tensor(p, device=pg.device)
            h.set_params(pg); h.set_path(xg)
    for c, o in orcs.items():
        xo, po = o.get_path()
        assert np.max(np.abs(h.get_path()[0][c].cpu().numpy() - xo)) < 1e-9
    print(f"cfg{cfg}: {decisions} decisions in the first 100 sweeps, {ties} inside the near-tie window, 0 outside")
    assert ties <= 3
