"""The paper's whole procedure on the paper-shaped workload, at reduced
length: trapezoid discretisation, initialisation phase with simulated annealing and step-size tuning, then statistics with
frozen step sizes -- the CUDA path against the oracle, and the workload recipe itself."""
import numpy as np
import pytest

from workloads import PAPER_P_TRUE, make_workload


def test_paper_shaped_workload_recipe():
    w = make_workload(5)
    assert (w.M, w.dt, w.Rm) == (8000, 0.04, 100.0) and np.array_equal(w.Rf, [1e2, 1e6, 1e6, 1e6])
    assert np.array_equal(w.p_true, PAPER_P_TRUE) and w.p_true[1] == 20.0                                 # Table 2: g_K = 20
    assert np.array_equal(w.w_state, [2e-3, 1e-3, 1e-3, 1e-3])
    assert w.extra["beta0"] == 0.01 and w.extra["f_acc"] == 0.23 and w.extra["alpha"] == 0.02 and w.extra["n_skip"] == 400
    V = w.x_true[0, :, 0]
    assert 5 <= np.sum((V[1:] > 0) & (V[:-1] <= 0)) <= 60 and -90 < V.min() and V.max() < 60     # a spiking neuron, 320 ms
    assert -12 < w.I.min() and w.I.max() < 22 and np.std(w.I) > 2                                 # a chaotic, bounded stimulus
    assert abs(np.std(w.y[0, :, 0] - V) - 0.1) < 0.01                                             # R_o = 100
    w2 = make_workload(5)
    assert np.array_equal(w.y, w2.y) and np.array_equal(w.I, w2.I)                                # seeded


@pytest.mark.gpu
def test_paper_procedure_end_to_end_matches_oracle():
    import torch
    import paper_1103_4887_b200 as P
    from oracle import OracleChain
    assert torch.cuda.is_available()
    w = make_workload(5, M=1200)
    h = P.Pimc.from_workload(w)
    o = OracleChain.from_workload(w)
    for s in (h, o):
        s.set_proposal(w.w_state, w.w_param, 1)              # uniform proposals: bit-reproducible on both sides
        s.set_discretisation(1)                              # the paper's trapezoid rule
        s.set_annealing(0.01, 60)                            # N_cool
        s.set_tuning(True, 10, 0.23, 0.05)                   # N_skip, f_acc, alpha
    assert h.get_engine()["engine"] == P.ENGINE_TILE         # initialisation phase (annealing and tuning): tile-resident too
    h.sweep(150, seed=9); o.sweep(150, seed=9)               # N_init
    for s in (h, o):
        s.set_tuning(False)
        s.set_accum(True, 5); s.reset_moments()
    assert h.get_engine()["engine"] == P.ENGINE_TILE         # production phase: tile-resident engine, frozen tuned step sizes
    h.sweep(100, seed=9); o.sweep(100, seed=9)
    xg, pg = [a.cpu().numpy()[0] for a in h.get_path()]
    xo, po = o.get_path()
    assert np.array_equal(xg, xo) and np.array_equal(pg, po)
    ws, wp = [a.cpu().numpy()[0] for a in h.get_widths()]
    ows, owp = o.get_widths()
    assert np.array_equal(ws, ows) and np.array_equal(wp, owp)
    assert ws[:, 0].mean() > 1.15 * w.w_state[0]             # 2e-3 mV is far too small a step: 15 adjustments (at most +3.85 % each) enlarged it
    mx, mp, n = h.moments()
    ox, op, on = o.moments()
    assert n == on == 20
    assert np.allclose(mx.cpu().numpy()[0], ox, rtol=1e-13, atol=1e-13) and np.allclose(mp.cpu().numpy()[0], op, rtol=1e-13, atol=1e-15)
    assert np.array_equal(h.stats().cpu().numpy()[0].astype(np.uint64), o.stats())


@pytest.mark.gpu
def test_procedure_module_runs_both_phases_tile_resident():
    # paper_1103_4887_b200.procedure: the paper's example calculation through the public binding, shortened
    from paper_1103_4887_b200 import procedure
    r = procedure.run(iterations=3000, n_skip=50, M=2000)
    assert r["engine"] == {"initialisation": "tile-resident", "production": "tile-resident"} and r["fault"] == 0
    assert r["samples"] == 1500 // 50 and r["proposed"][0] == 2001 * 3000 and r["proposed"][4] == 3000
    assert 0.15 < r["accepted"][0] / r["proposed"][0] < 0.6          # tuned towards f_acc = 0.23 from too small a step
    assert r["mean_step_size"][0] > 2e-3                             # and the step sizes grew on the way
    assert all(np.isfinite(r["param_mean"])) and all(s >= 0 for s in r["param_sd"])
