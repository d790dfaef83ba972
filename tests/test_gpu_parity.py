"""GPU parity tests proper (-m gpu): the CUDA path, called through the C ABI (libpimc.so via the ctypes
binding), against the CPU oracle on the same seeded inputs.  Tolerances are BASELINE.json's north_star:
per-site Delta-A to 1e-12 (fp64) relative to max(|dA|, S), identical decisions
except inside the near-tie window |dA + log u| < 1e-9, integer work bit-exact."""
import os

import numpy as np
import pytest

import oracle
from oracle import OracleChain
from workloads import MODEL_HH, MODEL_LINEAR, make_workload, HH_P_TRUE, linear_matrix, Workload
from helpers import TOL64, gpu_handle, oracle_chains, teacher_forced, to_dev, ulp_diff

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def P():
    import paper_1103_4887_b200 as P
    P.lib()
    return P


# ------------------------------------------------------------------------------------------------------------
# A1: RNG
# ------------------------------------------------------------------------------------------------------------
def test_philox_words_and_uniforms_bit_exact(P):
    import torch
    rng = np.random.default_rng(3)
    n = 200_003                                   # ragged tail over the launch grid
    ctrs = rng.integers(0, 2**32, size=(n, 4), dtype=np.uint64).astype(np.uint32)
    ctrs[:4] = [[0, 0, 0, 0], [0xFFFFFFFF] * 4, [0x243F6A88, 0x85A308D3, 0x13198A2E, 0x03707344], [1, 2, 3, 4]]
    key = (0xA4093822, 0x299F31D0)
    out = P.rng_selftest(torch.from_numpy(ctrs.view(np.int32)).cuda(), key)
    words = out["words"].cpu().numpy().view(np.uint32)
    ref = oracle.philox_bulk(ctrs, key)
    assert np.array_equal(words, ref)
    assert [hex(v) for v in words[2]] == ["0xd16cfe09", "0x94fdcceb", "0x5001e420", "0x24126ea1"]   # published KAT
    u = out["u_prop"].cpu().numpy()
    assert np.array_equal(u, (ref.astype(np.float64) + 0.5) * 2.0**-32)
    ua = out["u_acc"].cpu().numpy()
    v = ((ref[:, 1].astype(np.uint64) << np.uint64(32)) | ref[:, 0].astype(np.uint64)) >> np.uint64(12)
    assert np.array_equal(ua, (v.astype(np.float64) + 0.5) * 2.0**-52)
    assert u.min() > 0 and u.max() < 1 and ua.min() > 0 and ua.max() < 1
    # normals: same Box-Muller, different math library: a few ulp of the radius at most
    z = out["z"].cpu().numpy()
    idx = rng.integers(0, n, 3000)
    for i in idx:
        zr = np.concatenate([oracle.box_muller(u[i, 0], u[i, 1]), oracle.box_muller(u[i, 2], u[i, 3])])
        scale = np.sqrt(-2 * np.log(u[i, [0, 0, 2, 2]]))
        assert np.all(np.abs(z[i] - zr) <= 8 * np.spacing(scale)), (i, z[i], zr)
    assert abs(z.mean()) < 5 / np.sqrt(z.size) and abs(z.var() - 1) < 5 * np.sqrt(2 / z.size)


def test_philox_vs_curand_device_black_box(P, tmp_path):
    """libpimc's device Philox words against cuRAND's own curand_Philox4x32_10 running on the same GPU (a library routine as a
    black box: tests/curand_philox_device.cu, compiled here with nvcc)."""
    import ctypes as C
    import shutil
    import subprocess
    import torch
    if shutil.which("nvcc") is None:
        pytest.skip("nvcc is not on PATH on this box")
    so = str(tmp_path / "libcurand_philox_device.so")
    subprocess.run(["nvcc", "-gencode", "arch=compute_100a,code=sm_100a", "-O2", "--shared", "-Xcompiler", "-fPIC", "-o", so,
                    os.path.join(os.path.dirname(os.path.abspath(__file__)), "curand_philox_device.cu")], check=True)
    L = C.CDLL(so)
    L.curand_philox_device.restype = C.c_int
    L.curand_philox_device.argtypes = [C.c_uint64, C.c_void_p, C.c_uint32, C.c_uint32, C.c_void_p]
    rng = np.random.default_rng(11)
    n = 100_003
    ctrs = rng.integers(0, 2**32, size=(n, 4), dtype=np.uint64).astype(np.uint32)
    ctrs[:3] = [[0, 0, 0, 0], [0xFFFFFFFF] * 4, [0x243F6A88, 0x85A308D3, 0x13198A2E, 0x03707344]]
    key = (0xA4093822, 0x299F31D0)
    d_ctrs = torch.from_numpy(ctrs.view(np.int32)).cuda()
    ours = P.rng_selftest(d_ctrs, key)["words"]
    theirs = torch.empty_like(ours)
    torch.cuda.synchronize()
    assert L.curand_philox_device(n, d_ctrs.data_ptr(), key[0], key[1], theirs.data_ptr()) == 0
    assert torch.equal(ours, theirs)
    assert [hex(v) for v in theirs[2].cpu().numpy().view(np.uint32)] == ["0xd16cfe09", "0x94fdcceb", "0x5001e420", "0x24126ea1"]


# ------------------------------------------------------------------------------------------------------------
# A0: model step
# ------------------------------------------------------------------------------------------------------------
def test_step_increment_matches_oracle(P):
    import torch
    rng = np.random.default_rng(5)
    n = 5000
    x = np.column_stack([rng.uniform(-90, 50, n), rng.uniform(-0.1, 1.1, n), rng.uniform(-0.1, 1.1, n), rng.uniform(-0.1, 1.1, n)])
    I0, I1 = rng.uniform(0, 15, n), rng.uniform(0, 15, n)
    p = HH_P_TRUE * (1 + 0.1 * rng.normal(size=7))
    for dt in (0.01, 0.02):
        g = P.step_selftest(MODEL_HH, torch.from_numpy(x).cuda(), torch.from_numpy(p).cuda(), torch.from_numpy(I0).cuda(),
                            torch.from_numpy(I1).cuda(), dt).cpu().numpy()
        ref = np.array([oracle.step_increment(MODEL_HH, x[i], p, I0[i], I1[i], dt) for i in range(n)])
        scale = np.maximum(np.abs(ref), dt * np.array([100.0, 1.0, 1.0, 1.0]))
        assert np.max(np.abs(g - ref) / scale) < 2e-14
    for D in (1, 2, 3, 4):
        A = rng.normal(size=(D, D))
        xs = rng.normal(size=(100, D))
        g = P.step_selftest(MODEL_LINEAR, torch.from_numpy(xs).cuda(), torch.from_numpy(A.ravel().copy()).cuda(), None, None, 1.0).cpu().numpy()
        ref = np.array([oracle.step_increment(MODEL_LINEAR, xs[i], A.ravel(), 0, 0, 1.0) for i in range(100)])
        assert np.allclose(g, ref, rtol=0, atol=1e-14)


# ------------------------------------------------------------------------------------------------------------
# A2-A4: teacher-forced parity (T1) on the configs, at sizes the oracle finishes in seconds, several tiles + ragged tail
# ------------------------------------------------------------------------------------------------------------
CASES = [
    # name, cfg, M, launch (ctas_per_chain, threads), with_params, n_sweeps
    ("cfg0_M256_auto", 0, 256, None, False, 100),
    ("cfg0_M257_3ctas", 0, 257, (3, 32), False, 30),
    ("cfg2_M600_auto", 2, 600, None, True, 100),
    ("cfg2_M601_5ctas", 2, 601, (5, 64), True, 40),
    ("cfg2_M333_1cta", 2, 333, (1, 96), True, 40),
    ("cfg1_M1000_auto", 1, 1000, None, False, 100),
    ("cfg1_M999_7ctas", 1, 999, (7, 32), False, 30),
]


@pytest.mark.parametrize("name,cfg,M,launch,with_params,n_sweeps", CASES, ids=[c[0] for c in CASES])
def test_teacher_forced_parity(P, name, cfg, M, launch, with_params, n_sweeps):
    w = make_workload(cfg, M=M)
    h = gpu_handle(w, with_params=with_params, launch=launch)
    orcs = oracle_chains(w, with_params=with_params)
    rep = teacher_forced(w, h, orcs, n_sweeps, seed=20110347, do_params=with_params)
    print(name, h.get_launch(), rep)
    assert rep["sites"] == n_sweeps * (M + 1)
    assert rep["max_rel"] <= TOL64, rep
    assert rep["mismatch_outside_window"] == 0, rep
    assert rep["ties"] <= 2, rep
    assert rep["max_xprop_ulp"] <= 4.0, rep
    assert rep["accepted"] > 0
    if with_params:
        assert rep["param_moves"] > 0 and rep["max_param_rel"] <= TOL64, rep
    assert rep["max_path_diff"] <= 1e-12


def test_teacher_forced_batched_chains(P):
    # cfg4 shape in miniature: several independent chains, distinct data and Philox streams, one CTA per chain
    w = make_workload(4, M=300, n_chains=5)
    h = gpu_handle(w, launch=(1, 64))
    orcs = oracle_chains(w)
    rep = teacher_forced(w, h, orcs, 25, seed=99)
    assert rep["max_rel"] <= TOL64 and rep["mismatch_outside_window"] == 0 and rep["max_param_rel"] <= TOL64, rep
    # and split over several CTAs per chain
    h2 = gpu_handle(w, launch=(4, 32))
    rep = teacher_forced(w, h2, oracle_chains(w), 10, seed=99)
    assert rep["max_rel"] <= TOL64 and rep["mismatch_outside_window"] == 0 and rep["max_param_rel"] <= TOL64, rep


# ------------------------------------------------------------------------------------------------------------
# T2: free-running, no resync.  With UNIFORM proposals x' = x + w(2u-1) is bit-reproducible, so as long as
# every decision agrees the two chains stay bit-identical; so do histograms and counters.
# ------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("cfg,M,launch", [(0, 256, None), (2, 500, (4, 64)), (1, 700, (3, 128))])
def test_free_running_uniform_proposals_bit_identical(P, cfg, M, launch):
    w = make_workload(cfg, M=M)
    h = gpu_handle(w, launch=launch, kind=1)
    o = oracle_chains(w, kind=1)[0]
    sel = ([3, M, 10], [0, w.D - 1, 1], [-100.0 if cfg != 1 else -3.0, -1.0, -1.0], [60.0 if cfg != 1 else 3.0, 2.0, 2.0])
    if w.w_param.any():
        sel = tuple(list(a) + [b] for a, b in zip(sel, (-1, 0, 50.0, 200.0)))
    h.hist_config(*sel, 16); o.hist_config(*sel, 16)
    h.set_accum(True, 3); o.set_accum(True, 3)
    h.reset_moments(); o.reset_moments()
    h.sweep(100, seed=5); o.sweep(100, seed=5)
    xg, pg = [a.cpu().numpy() for a in h.get_path()]
    xo, po = o.get_path()
    assert np.array_equal(xg[0], xo), np.abs(xg[0] - xo).max()
    assert np.array_equal(pg[0], po)
    assert np.array_equal(h.stats().cpu().numpy()[0].astype(np.uint64), o.stats())
    assert np.array_equal(h.hist().cpu().numpy()[0].astype(np.uint64), o.hist())
    mx, mp, n = h.moments()
    ox, op, on = o.moments()
    assert n == on == 34
    assert np.allclose(mx.cpu().numpy()[0], ox, rtol=1e-13, atol=1e-13)
    assert np.allclose(mp.cpu().numpy()[0], op, rtol=1e-13, atol=1e-16)
    # cache coherence on the device: g == increment recomputed by the oracle from the final (x, p)
    g = h.get_cache().cpu().numpy()[0]
    og = o.get_cache()
    assert np.max(np.abs(g - og) / np.maximum(np.abs(og), 1e-3)) < 1e-13


def test_free_running_gaussian_first_100_sweeps(P):
    # north_star: decisions over the first 100 sweeps identical except near ties; paths agree to rounding
    w = make_workload(2, M=400)
    h = gpu_handle(w)
    o = oracle_chains(w)[0]
    tr = h.enable_trace()
    mism = 0
    for t in range(100):
        h.sweep(1, seed=8); o.sweep(1, seed=8)
        ot = o.trace()
        ga = tr["acc"].cpu().numpy()[0]
        bad = np.nonzero(ga != ot["acc"])[0]
        for n in bad:
            assert abs(ot["dA"][n] + ot["logu"][n]) < 1e-9
            mism += 1
        assert np.array_equal(tr["accp"].cpu().numpy()[0], ot["accp"])
        if len(bad):      # resync (protocol T2)
            x, p = o.get_path(); h.set_params(to_dev(p[None], h)); h.set_path(to_dev(x[None], h))
    xg, pg = [a.cpu().numpy()[0] for a in h.get_path()]
    xo, po = o.get_path()
    print("near-tie mismatches in 100 sweeps:", mism)
    assert mism <= 1
    assert np.max(np.abs(xg - xo)) < 1e-10 and np.max(np.abs(pg - po)) < 1e-12


# ------------------------------------------------------------------------------------------------------------
# launch-shape independence, split sweeps, checkpoint/resume
# ------------------------------------------------------------------------------------------------------------
def test_results_do_not_depend_on_launch_shape(P):
    w = make_workload(0, M=515)
    ref = None
    for launch in ((1, 32), (1, 512), (2, 128), (5, 64), (9, 32), (0, 0)):
        h = gpu_handle(w, with_params=False, launch=launch)
        h.sweep_states_only(30, seed=4)
        x = h.get_path()[0].cpu().numpy()
        st = h.stats().cpu().numpy()
        if ref is None:
            ref = (x, st)
        assert np.array_equal(x, ref[0]) and np.array_equal(st, ref[1]), launch
    # with parameter moves the reduction tree depends on the shape: totals agree to rounding, decisions the same
    w = make_workload(2, M=515)
    outs = []
    for launch in ((1, 64), (4, 64), (7, 32)):
        h = gpu_handle(w, launch=launch)
        h.sweep(30, seed=4)
        outs.append([a.cpu().numpy() for a in h.get_path()])
    for x, p in outs[1:]:
        assert np.allclose(x, outs[0][0], rtol=0, atol=1e-11) and np.allclose(p, outs[0][1], rtol=1e-13)
    # run-to-run bit reproducibility at a fixed shape
    a = gpu_handle(w, launch=(4, 64)); a.sweep(30, seed=4)
    assert np.array_equal(a.get_path()[0].cpu().numpy(), outs[1][0])


def test_split_sweeps_and_resume_bit_identical(P):
    import torch
    w = make_workload(2, M=300)
    a = gpu_handle(w, launch=(3, 64)); a.set_accum(True, 2); a.reset_moments(); a.sweep(20, seed=9)
    b = gpu_handle(w, launch=(3, 64)); b.set_accum(True, 2); b.reset_moments(); b.sweep(8, seed=9); b.sweep(12, seed=9)
    assert a.sweep_index == b.sweep_index == 20
    for u, v in zip(a.get_path(), b.get_path()):
        assert torch.equal(u, v)
    ma, mb = a.moments(), b.moments()
    assert ma[2] == mb[2] == 10 and torch.equal(ma[0], mb[0]) and torch.equal(ma[1], mb[1])
    # resume from (path, p, sweep index)
    c = gpu_handle(w, launch=(3, 64)); c.sweep(8, seed=9)
    x, p = c.get_path()
    d = gpu_handle(w, launch=(3, 64)); d.set_params(p); d.set_path(x); d.sweep_index = 8; d.sweep(12, seed=9)
    assert torch.equal(d.get_path()[0], a.get_path()[0]) and torch.equal(d.get_path()[1], a.get_path()[1])
    # states-only + params-only == full sweep, sweep by sweep (same counters)
    e = gpu_handle(w, launch=(3, 64))
    for t in range(5):
        e.sweep_index = t; e.sweep_states_only(1, seed=9); e.sweep_index = t; e.sweep_params_only(1, seed=9)
    f = gpu_handle(w, launch=(3, 64)); f.sweep(5, seed=9)
    assert torch.equal(e.get_path()[0], f.get_path()[0]) and torch.equal(e.get_path()[1], f.get_path()[1])


# ------------------------------------------------------------------------------------------------------------
# edge cases
# ------------------------------------------------------------------------------------------------------------
def test_edge_cases_tiny_paths_and_degenerate_settings(P):
    # M = 1 and M = 2 (every site is a boundary), D = 1..4 linear
    for D in (1, 2, 3, 4):
        for M in (1, 2, 5):
            rng = np.random.default_rng(10 * D + M)
            A = 0.5 * np.eye(D) + 0.1 * rng.normal(size=(D, D))
            w = Workload(name="tiny", model=MODEL_LINEAR, D=D, L=min(1, D), Np=D * D, M=M, dt=1.0, Rm=3.0, Rf=np.linspace(5, 9, D),
                         n_chains=2, p0=np.tile(A.ravel(), (2, 1)), p_true=A.ravel(), lo=np.full((2, D * D), -5.0),
                         hi=np.full((2, D * D), 5.0), w_state=np.full(D, 0.3), w_param=np.full(D * D, 0.05),
                         y=rng.normal(size=(2, M + 1, 1)), I=None, x0=rng.normal(size=(2, M + 1, D)), x_true=np.zeros((2, M + 1, D)),
                         n_sweeps=10)
            h = gpu_handle(w)
            rep = teacher_forced(w, h, oracle_chains(w), 10, seed=3)
            assert rep["max_rel"] <= TOL64 and rep["mismatch_outside_window"] == 0 and rep["max_param_rel"] <= TOL64, (D, M, rep)
    w = make_workload(2, M=64)
    # zero widths: x' = x, dA = 0, accepted, path unchanged
    h = gpu_handle(w); h.set_proposal(np.zeros(4), None)
    h.sweep(3, seed=1)
    assert np.array_equal(h.get_path()[0].cpu().numpy(), w.x0)
    st = h.stats().cpu().numpy()[0]
    assert np.all(st[0, :4] == 3 * 65) and np.all(st[1, :4] == 3 * 65) and np.all(st[:, 4:] == 0)
    # Rm = Rf = 0: everything accepted
    w0 = make_workload(0, M=64); w0.Rm = 0.0; w0.Rf = np.zeros(4)
    h = gpu_handle(w0, with_params=False); h.sweep(4, seed=1)
    st = h.stats().cpu().numpy()[0]
    assert np.all(st[0, :4] == st[1, :4]) and st[1, 0] == 4 * 65
    # bounds that admit nothing: parameters and cache never change, proposals counted
    w = make_workload(2, M=64); w.lo = w.p0.copy(); w.hi = w.p0.copy(); w.w_param = w.w_param * 50
    h = gpu_handle(w); h.set_proposal(np.zeros(4), w.w_param)
    g0 = h.get_cache().clone()
    h.sweep(10, seed=2)
    assert np.array_equal(h.get_path()[1].cpu().numpy(), w.p0)
    import torch
    assert torch.equal(h.get_cache(), g0)
    st = h.stats().cpu().numpy()[0]
    assert np.all(st[0, 4:] == 0) and np.all(st[1, 4:] == 10)
    # NaN in the data rejects at that site (comparison false), neighbours unaffected
    w = make_workload(0, M=64); w.y[0, 5, 0] = np.nan
    h = gpu_handle(w, with_params=False); h.sweep(5, seed=2)
    x = h.get_path()[0].cpu().numpy()[0]
    assert np.array_equal(x[5], w.x0[0, 5]) and not np.array_equal(x[4], w.x0[0, 4])


def test_c_abi_argument_errors_on_device(P):
    import ctypes as C
    import torch
    w = make_workload(0, M=32)
    h = gpu_handle(w)
    L = P.lib()
    assert L.pimc_set_accum(h._h, 1, 0) == -1                    # n_skip < 1
    assert L.pimc_set_launch(h._h, 1, 33) == -1                  # threads not a multiple of 32
    assert L.pimc_set_launch(h._h, 5000, 512) == -1              # out of range
    assert L.pimc_sweep(h._h, -1, 0) == -1
    neg = (C.c_double * 4)(-1.0, 0, 0, 0)
    assert L.pimc_set_proposal(h._h, neg, None, 0) == -1
    assert b"w_state" in L.pimc_last_error(h._h) or len(L.pimc_last_error(h._h)) > 0
    # sweeping before a path is set is a state error
    h2 = P.Pimc(w.model, w.D, w.L, w.M, w.dt, w.Rm, w.Rf, w.p0)
    assert L.pimc_sweep(h2._h, 1, 0) == -2
    # misaligned / too small workspace
    ws = torch.empty(1 << 20, dtype=torch.uint8, device="cuda")
    hh = C.c_void_p()
    rf = (C.c_double * 4)(*w.Rf); p0 = (C.c_double * 7)(*w.p0[0])
    assert L.pimc_init(C.byref(hh), 1, 4, 1, 32, 0.02, 1.0, rf, p0, 1, 64, C.c_void_p(ws.data_ptr() + 8), 1 << 19, None) == -1
    assert L.pimc_init(C.byref(hh), 1, 4, 1, 32, 0.02, 1.0, rf, p0, 1, 64, C.c_void_p(ws.data_ptr()), 1024, None) == -1
    assert L.pimc_init(C.byref(hh), 1, 3, 1, 32, 0.02, 1.0, rf, p0, 1, 64, C.c_void_p(ws.data_ptr()), 1 << 20, None) == -4


def test_boundary_robustness_alignment_schedules_and_fault_path(P):
    import ctypes as C
    import torch
    w = make_workload(2, M=200)
    h = gpu_handle(w)
    L = P.lib()
    # caller arrays must be 32-byte aligned (SURVEY.md 8(b) conventions): a view that starts 8 bytes in is refused
    x = torch.zeros((w.M + 1) * w.D + 4, dtype=torch.float64, device="cuda")
    assert x.data_ptr() % 32 == 0
    assert L.pimc_set_path(h._h, C.c_void_p(x.data_ptr() + 8)) == -1 and b"aligned" in L.pimc_last_error(h._h)
    assert L.pimc_get_path(h._h, C.c_void_p(x.data_ptr() + 8), None) == -1
    assert L.pimc_set_data(h._h, C.c_void_p(x.data_ptr() + 16), C.c_void_p(x.data_ptr())) == -1
    assert L.pimc_moments(h._h, C.c_void_p(x.data_ptr() + 8), None) == -1
    assert L.pimc_debug_trace(h._h, C.c_void_p(x.data_ptr() + 24), None, None, None, None, None) == -1
    # the error string is the LATEST failure's, not the first one's
    assert L.pimc_set_accum(h._h, 1, 0) == -1 and b"n_skip" in L.pimc_last_error(h._h)
    assert L.pimc_sweep(h._h, -1, 0) == -1 and b"n_sweeps" in L.pimc_last_error(h._h)
    # schedules count sweeps from the index at which they were switched on: the index may not be moved below it
    h.sweep(5, seed=1)
    h.set_accum(True, 2); h.reset_moments()
    assert h.sweep_index == 5
    assert L.pimc_set_sweep_index(h._h, 3) == -2
    h.sweep_index = 9                                   # forward is fine
    h.set_accum(False, 1)
    h.sweep_index = 3                                   # and backwards once nothing counts from an origin
    # step-size tuning needs full sweeps
    h.set_tuning(True, 5, 0.23, 0.02)
    assert L.pimc_sweep_states_only(h._h, 1, 1) == -2 and L.pimc_sweep_params_only(h._h, 1, 1) == -2
    assert b"tuning" in L.pimc_last_error(h._h)
    h.sweep(10, seed=1, check_fault=True)               # the checked path: synchronises and raises on a lost hand-off
    h.set_tuning(False)
    h.sweep_states_only(1, seed=1)
    # exchange knob: results do not depend on it
    h1, h2 = gpu_handle(w, kind=1), gpu_handle(w, kind=1)
    h2.set_exchange(0)
    assert L.pimc_set_exchange(h2._h, -1) == -1
    h1.sweep(12, seed=3); h2.sweep(12, seed=3)
    assert torch.equal(h1.get_path()[0], h2.get_path()[0]) and torch.equal(h1.get_path()[1], h2.get_path()[1])


def test_run_host_with_caller_scratch(P):
    w = make_workload(2, M=200)
    scratch = P.run_host_scratch(w)
    a = P.run_host(w, n_burn=5, n_sweeps=20, seed=6, want_path=True)
    b = P.run_host(w, n_burn=5, n_sweeps=20, seed=6, want_path=True, scratch=scratch)
    c = P.run_host(w, n_burn=5, n_sweeps=20, seed=6, want_path=True, scratch=scratch)      # reuse
    for k in ("mean_x", "var_x", "mean_p", "var_p", "x", "p"):
        assert np.array_equal(a[k], b[k]) and np.array_equal(a[k], c[k]), k
    import ctypes as C
    import torch
    small = torch.empty(1024, dtype=torch.uint8, device="cuda")
    with pytest.raises(P.PimcError):
        P.run_host(w, n_burn=0, n_sweeps=1, seed=6, scratch=small)
    assert P.lib().pimc_run_host_workspace_bytes(w.model, w.D, w.L, w.M, 1, 64) > P.lib().pimc_workspace_bytes(w.model, w.D, w.L, w.M, 1, 64)
    assert P.lib().pimc_run_host_workspace_bytes(9, 4, 1, 10, 1, 64) == 0


def test_run_host_end_to_end_matches_device_api(P):
    w = make_workload(2, M=200)
    out = P.run_host(w, n_burn=10, n_sweeps=40, seed=6, want_path=True)
    h = gpu_handle(w); h.sweep(10, seed=6); h.set_accum(True, 1); h.reset_moments(); h.sweep(40, seed=6)
    mx, mp, n = h.moments()
    assert n == 40
    assert np.array_equal(out["mean_x"], mx.cpu().numpy()[:, 0]) and np.array_equal(out["var_x"], mx.cpu().numpy()[:, 1])
    assert np.array_equal(out["x"], h.get_path()[0].cpu().numpy()) and np.array_equal(out["p"], h.get_path()[1].cpu().numpy())
    assert out["h2d_bytes"] > 0 and out["d2h_bytes"] > 0


def test_several_observed_components_run_on_the_global_engine(P):
    # the tile-resident engine is compiled for one observed component (every BASELINE config); L >= 2 falls back
    import paper_1103_4887_b200 as Pm
    for D, L in ((3, 2), (4, 4), (2, 2)):
        rng = np.random.default_rng(100 * D + L)
        A = 0.6 * np.eye(D) + 0.1 * rng.normal(size=(D, D))
        M = 300
        w = Workload(name="multi_obs", model=MODEL_LINEAR, D=D, L=L, Np=D * D, M=M, dt=1.0, Rm=7.0, Rf=np.linspace(5, 9, D),
                     n_chains=1, p0=A.ravel()[None].copy(), p_true=A.ravel(), lo=np.full((1, D * D), -5.0), hi=np.full((1, D * D), 5.0),
                     w_state=np.full(D, 0.3), w_param=np.full(D * D, 0.02), y=rng.normal(size=(1, M + 1, max(L, 1))), I=None,
                     x0=rng.normal(size=(1, M + 1, D)), x_true=np.zeros((1, M + 1, D)), n_sweeps=10)
        h = gpu_handle(w)
        assert h.get_engine()["engine"] == Pm.ENGINE_GLOBAL
        rep = teacher_forced(w, h, oracle_chains(w), 8, seed=3)
        assert rep["max_rel"] <= TOL64 and rep["mismatch_outside_window"] == 0 and rep["max_param_rel"] <= TOL64, (D, L, rep)
        with pytest.raises(Pm.PimcError):
            h.set_engine(Pm.ENGINE_TILE)
