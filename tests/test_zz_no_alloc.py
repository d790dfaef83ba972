"""The no-allocation entry point pimc_run_host_static (include/pimc.h): all device memory of the call comes from one static
device array inside libpimc.so.  Collected LAST on purpose (file name): the suite runs with pytest -x.

GPU test: its results must equal those of the existing path (pimc_run_host_ws with a caller-provided scratch buffer: the same
kernels in the same launch shape, which are run-to-run bit-reproducible) on calls in a row that reuse the shared array with
different shapes, i.e. on stale contents."""
import numpy as np
import pytest

from workloads import make_workload


def _same(a, b):
    assert np.array_equal(a["x"], b["x"]) and np.array_equal(a["p"], b["p"])              # final path and parameters: bit-identical
    for k in ("mean_x", "var_x", "mean_p", "var_p"):
        assert np.allclose(a[k], b[k], rtol=1e-13, atol=1e-13), k                          # the moment tolerance of the parity tests
        assert np.all(np.isfinite(a[k]))


def test_static_scratch_limit_is_stated_and_enforced_without_a_device():
    # no compute call: the size check comes before anything touches CUDA, so this runs in the CPU suite as well
    import paper_1103_4887_b200 as P
    cap = P.static_scratch_bytes()
    assert cap == 32 << 20
    L = P.lib()
    w3, w4 = make_workload(3, M=32768), make_workload(4, M=8192, n_chains=16)
    assert L.pimc_run_host_workspace_bytes(w3.model, w3.D, w3.L, w3.M, 1, 64) <= cap          # the headline workload fits
    assert L.pimc_run_host_workspace_bytes(w4.model, w4.D, w4.L, w4.M, 16, 64) > cap
    with pytest.raises(P.PimcError) as ei:
        P.run_host(w4, 0, 1, 1, static=True)
    assert "static array holds" in str(ei.value) and str(cap) in str(ei.value), str(ei.value)


@pytest.mark.gpu
def test_run_host_static_matches_the_caller_scratch_path_on_calls_in_a_row():
    import torch
    import paper_1103_4887_b200 as P
    assert torch.cuda.is_available()
    calls = [(make_workload(2, M=4096), 5, 30, 11, 1),      # tile-resident engine, 7 parameters, uniform proposals
             (make_workload(0, M=256), 3, 40, 12, 0),       # much smaller shape right after: the array holds the previous call's bytes
             (make_workload(2, M=4096), 5, 30, 11, 1),      # the first call again: same result as before
             (make_workload(3), 0, 12, 13, 0)]              # config 3 at full size: 28.1 of the 32 MiB
    first = None
    for i, (w, n_burn, n_sweeps, seed, kind) in enumerate(calls):
        ref = P.run_host(w, n_burn, n_sweeps, seed, kind=kind, want_path=True, scratch=P.run_host_scratch(w))
        out = P.run_host(w, n_burn, n_sweeps, seed, kind=kind, want_path=True, static=True)
        _same(out, ref)
        if i == 0:
            first = out
        if i == 2:
            _same(out, first)
    # fp32 through the same array
    w = make_workload(2, M=1000)
    _same(P.run_host(w, 2, 10, 5, dtype=32, kind=1, want_path=True, static=True),
          P.run_host(w, 2, 10, 5, dtype=32, kind=1, want_path=True, scratch=P.run_host_scratch(w, dtype=32)))
