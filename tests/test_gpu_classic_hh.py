"""GPU parity for the classic Hodgkin-Huxley rate functions (PIMC_MODEL_HH_CLASSIC) against the
oracle's model 2: the stand-alone step increment, teacher-forced sweeps on both engines and both discretisations,
free-running bit-identical chains, fp32."""
import numpy as np
import pytest

from helpers import TOL32, TOL64, gpu_handle, oracle_chains, teacher_forced
from workloads import HH_P_TRUE, MODEL_HH_CLASSIC, make_workload

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def P():
    import torch
    import paper_1103_4887_b200 as P
    assert torch.cuda.is_available()
    P.lib()
    return P


def test_step_increment_matches_oracle_classic(P):
    import torch
    import oracle
    rng = np.random.default_rng(5)
    n = 4000
    V = np.concatenate([rng.uniform(-90, 50, n - 8), [-40.0, -55.0, -40.0 + 1e-7, -55.0 - 1e-7, -40.0 + 1e-3, -55.0 + 1e-3, -65.0, 0.0]])
    x = np.column_stack([V, rng.uniform(-0.1, 1.1, n), rng.uniform(-0.1, 1.1, n), rng.uniform(-0.1, 1.1, n)])
    I0, I1 = rng.uniform(0, 15, n), rng.uniform(0, 15, n)
    p = HH_P_TRUE * (1 + 0.1 * rng.normal(size=7))
    for dt in (0.01, 0.02):
        g = P.step_selftest(MODEL_HH_CLASSIC, torch.from_numpy(x).cuda(), torch.from_numpy(p).cuda(), torch.from_numpy(I0).cuda(),
                            torch.from_numpy(I1).cuda(), dt).cpu().numpy()
        ref = np.array([oracle.step_increment(MODEL_HH_CLASSIC, x[i], p, I0[i], I1[i], dt) for i in range(n)])
        scale = np.maximum(np.abs(ref), dt * np.array([100.0, 4.0, 1.0, 1.0]))     # beta_m reaches ~4-30 /ms
        assert np.max(np.abs(g - ref) / scale) < 5e-14


CASES = [
    # name, M, launch, engine, disc, with_params
    ("M600_auto_rk4", 600, None, 0, 0, True),
    ("M601_5ctas_global_rk4", 601, (5, 64), 1, 0, True),
    ("M600_auto_trapezoid", 600, None, 0, 1, True),
    ("M333_1cta_global_trapezoid", 333, (1, 96), 1, 1, True),
    ("M256_states_only", 256, None, 0, 0, False),
]


@pytest.mark.parametrize("name,M,launch,engine,disc,with_params", CASES, ids=[c[0] for c in CASES])
def test_teacher_forced_parity_classic(P, name, M, launch, engine, disc, with_params):
    w = make_workload(2 if with_params else 0, M=M, kinetics="classic")
    h = gpu_handle(w, with_params=with_params, disc=disc)
    if engine:
        h.set_engine(engine)
    if launch:
        h.set_launch(*launch)
    orcs = oracle_chains(w, with_params=with_params, disc=disc)
    rep = teacher_forced(w, h, orcs, 30, seed=20110347, do_params=with_params, disc=disc)
    print(name, h.get_launch(), h.get_engine(), rep)
    assert rep["max_rel"] <= TOL64 and rep["mismatch_outside_window"] == 0 and rep["ties"] <= 2, rep
    assert rep["max_xprop_ulp"] <= 4.0 and rep["accepted"] > 0, rep
    if with_params:
        assert rep["param_moves"] > 0 and rep["max_param_rel"] <= TOL64, rep


def test_free_running_bit_identical_and_fp32_classic(P):
    w = make_workload(3, M=4000, kinetics="classic")
    h = gpu_handle(w, kind=1)
    o = oracle_chains(w, kind=1)[0]
    h.sweep(40, seed=5); o.sweep(40, seed=5)
    xg, pg = [a.cpu().numpy() for a in h.get_path()]
    xo, po = o.get_path()
    assert np.array_equal(xg[0], xo) and np.array_equal(pg[0], po)
    assert np.array_equal(h.stats().cpu().numpy()[0].astype(np.uint64), o.stats())
    w = make_workload(2, M=600, kinetics="classic")
    h = gpu_handle(w, dtype=32)
    rep = teacher_forced(w, h, oracle_chains(w, state_dtype=32), 15, seed=3, tol=TOL32, state_dtype=32)
    assert rep["max_rel"] <= TOL32 and rep["mismatch_outside_window"] == 0, rep
