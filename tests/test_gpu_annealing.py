"""GPU parity for the simulated annealing of the dynamics term (pimc_set_annealing; Eq. 10; SURVEY.md
§8(f) NEXT-4, first half) against the oracle: teacher-forced sweeps while beta rises, on both engines (automatic, forced global-memory, forced tile-resident) and discretisations,
and free-running bit-identical chains through the whole cooling schedule and beyond."""
import numpy as np
import pytest

from helpers import TOL64, gpu_handle, oracle_chains, teacher_forced
from workloads import make_workload

pytestmark = pytest.mark.gpu
ANNEAL = (0.01, 12)


@pytest.fixture(scope="module")
def P():
    import torch
    import paper_1103_4887_b200 as P
    assert torch.cuda.is_available()
    P.lib()
    return P


@pytest.mark.parametrize("M,launch,engine,disc", [(600, None, 0, 0), (601, (5, 64), 1, 0), (600, None, 0, 1), (333, (1, 96), 1, 1), (2500, None, 2, 0), (1201, None, 2, 1)])   # engine 0: automatic, 1: global-memory, 2: tile-resident
def test_teacher_forced_parity_while_annealing(P, M, launch, engine, disc):
    w = make_workload(2, M=M)
    h = gpu_handle(w, disc=disc)
    if engine:
        h.set_engine(engine)
    if launch:
        h.set_launch(*launch)
    h.set_annealing(*ANNEAL)
    orcs = oracle_chains(w, disc=disc)
    for o in orcs:
        o.set_annealing(*ANNEAL)
    rep = teacher_forced(w, h, orcs, 16, seed=77, disc=disc, anneal=ANNEAL)
    print(M, launch, engine, disc, rep)
    assert rep["max_rel"] <= TOL64 and rep["mismatch_outside_window"] == 0 and rep["ties"] <= 2, rep
    assert rep["param_moves"] > 0 and rep["max_param_rel"] <= TOL64 and rep["max_path_diff"] <= 1e-12, rep
    assert orcs[0].annealing_beta() == 1.0
    if engine != 1:                                  # the tile-resident engine carries the schedule (its general variant) and what follows
        assert h.get_engine()["engine"] == P.ENGINE_TILE


@pytest.mark.parametrize("cfg,M,launch,engine", [(2, 500, None, 0), (2, 500, (4, 64), 1), (3, 4001, None, 0), (3, 32768, None, 2)])
def test_free_running_through_the_cooling_schedule(P, cfg, M, launch, engine):
    w = make_workload(cfg, M=M)
    h = gpu_handle(w, kind=1)
    if engine:
        h.set_engine(engine)
    if launch:
        h.set_launch(*launch)
    o = oracle_chains(w, kind=1)[0]
    h.sweep(3, seed=5); o.sweep(3, seed=5)               # annealing starts at the sweep index of the call
    h.set_annealing(0.02, 20); o.set_annealing(0.02, 20)
    if engine != 1:                                  # while beta < 1 the automatic choice stays the tile-resident engine
        assert h.get_engine()["engine"] == P.ENGINE_TILE
    h.sweep(11, seed=5); h.sweep(19, seed=5); o.sweep(30, seed=5)     # two launches across the schedule and past its end
    xg, pg = [a.cpu().numpy() for a in h.get_path()]
    xo, po = o.get_path()
    assert np.array_equal(xg[0], xo) and np.array_equal(pg[0], po)
    assert np.array_equal(h.stats().cpu().numpy()[0].astype(np.uint64), o.stats())
    # annealing really changed the chain: the plain chain from the same start ends elsewhere
    q = oracle_chains(w, kind=1)[0]; q.sweep(33, seed=5)
    assert not np.array_equal(q.get_path()[0], xo)
    import paper_1103_4887_b200 as Pm
    with pytest.raises(Pm.PimcError):
        h.set_annealing(0.0, 10)
    with pytest.raises(Pm.PimcError):
        h.set_annealing(1.5, 10)


@pytest.mark.parametrize("disc,update", [(0, 1), (1, 0), (1, 1)])
def test_cooling_schedule_with_the_other_tile_kernels(P, disc, update):
    # the general variants of the trapezoid / component-wise tile kernels carry the schedule too: bit-identical chains
    w = make_workload(3, M=3001)
    h = gpu_handle(w, kind=1, disc=disc)
    h.set_engine(P.ENGINE_TILE)
    o = oracle_chains(w, kind=1, disc=disc)[0]
    h.set_update_mode(update); o.set_update_mode(update)
    h.set_annealing(0.05, 14); o.set_annealing(0.05, 14)
    h.sweep(9, seed=8); h.sweep(9, seed=8); o.sweep(18, seed=8)
    assert h.get_engine()["engine"] == P.ENGINE_TILE
    xg, pg = [a.cpu().numpy() for a in h.get_path()]
    xo, po = o.get_path()
    assert np.array_equal(xg[0], xo) and np.array_equal(pg[0], po)
    assert np.array_equal(h.stats().cpu().numpy()[0].astype(np.uint64), o.stats())
