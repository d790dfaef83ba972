"""The optional diagnostics on the CUDA path against the oracle: the per-sweep parameter record (Fig. 4), the model
and observation errors eps_n, delta_n of a path and their running statistics.  Uniform proposals make the chains
bit-identical, so the record must be identical and the residuals agree to the rounding of the cached model step."""
import numpy as np
import pytest

from helpers import gpu_handle, oracle_chains
from workloads import make_workload

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("engine", ["tile", "global"])
def test_parameter_record_is_bit_identical_to_the_oracle(engine):
    import paper_1103_4887_b200 as P
    w = make_workload(4, M=700, n_chains=3)
    h = gpu_handle(w, kind=1)
    if engine == "global":
        h.set_engine(P.ENGINE_GLOBAL)
    assert h.get_engine()["engine"] == (P.ENGINE_TILE if engine == "tile" else P.ENGINE_GLOBAL)
    rec = h.param_trace(12)
    h.set_accum(True, 3); h.reset_moments()
    h.sweep(25, seed=5); h.sweep(14, seed=5)                 # 13 accumulated sweeps: the 13th does not fit and is dropped
    orcs = oracle_chains(w, kind=1)
    for c, o in enumerate(orcs):
        o.param_trace_enable(True)
        o.set_accum(True, 3); o.reset_moments()
        o.sweep(39, seed=5)
        ot = o.param_trace()
        assert ot.shape == (13, 7)
        assert np.array_equal(rec.cpu().numpy()[c], ot[:12]), c
        assert np.array_equal(h.get_path()[1].cpu().numpy()[c], o.get_path()[1])
    assert h.moments()[2] == 13
    h.reset_moments()                                        # restarts at record 0
    h.sweep(3, seed=5)
    for c, o in enumerate(orcs):
        o.reset_moments(); o.sweep(3, seed=5)
        assert np.array_equal(rec.cpu().numpy()[c, 0], o.param_trace()[0])
    h.param_trace(0)
    h.sweep(3, seed=5)


@pytest.mark.parametrize("disc,dtype", [(0, 64), (1, 64), (0, 32)])
def test_residuals_and_their_running_statistics(disc, dtype):
    w = make_workload(2, M=900)
    h = gpu_handle(w, kind=1, disc=disc, dtype=dtype)
    o = oracle_chains(w, kind=1, disc=disc, state_dtype=dtype)[0]
    h.set_residual_stats(True)
    o.residual_stats_enable(True)
    for q in (h, o):
        q.set_accum(True, 2); q.reset_moments()
    n0 = h.launch_count
    h.sweep(21, seed=8); o.sweep(21, seed=8)
    # one launch per accumulated sweep (11 of them) + one residual kernel each; the trailing sweeps ride in the last launch
    assert h.launch_count - n0 == 11 + 11
    if dtype == 64:
        assert np.array_equal(h.get_path()[0].cpu().numpy()[0], o.get_path()[0])
    eps, delta = [a.cpu().numpy()[0].astype(np.float64) for a in h.residuals()]
    oe, od = o.residuals()
    tol = 1e-12 if dtype == 64 else 2e-5
    if dtype == 64:
        assert np.array_equal(delta, od)
        assert np.max(np.abs(eps - oe)) <= tol * max(1.0, np.max(np.abs(oe)))
        me, ve, md, vd = [a.cpu().numpy()[0] for a in h.residual_stats()]
        ome, ove, omd, ovd, n = o.residual_stats()
        assert n == 11 == h.moments()[2]
        assert np.allclose(me, ome, rtol=0, atol=1e-12) and np.allclose(ve, ove, rtol=1e-9, atol=1e-12)
        assert np.array_equal(md, omd) and np.allclose(vd, ovd, rtol=1e-12, atol=1e-15)
        # the residuals reassemble the action (definition)
        A = 0.5 * w.Rm * np.sum(delta.astype(np.longdouble) ** 2) + np.sum(0.5 * np.asarray(w.Rf, np.longdouble) * eps.astype(np.longdouble) ** 2)
        ref = o.full_action()
        assert abs(A - ref) <= 1e-10 * abs(ref)
    else:
        # fp32 chains are not bit-identical to the oracle's (different libm): compare the definition on the GPU's own path
        x = h.get_path()[0].cpu().numpy()[0].astype(np.float64)
        y = np.asarray(w.y[0], np.float32).astype(np.float64).reshape(w.M + 1, -1)
        assert np.allclose(delta[1:, 0], y[1:, 0] - x[1:, 0], rtol=0, atol=1e-5) and np.all(delta[0] == 0)
        assert np.all(np.isfinite(eps)) and np.max(np.abs(eps[:, 0])) < 50
    h.set_residual_stats(False)
    n0 = h.launch_count
    h.sweep(10, seed=8)
    assert h.launch_count - n0 == 1
