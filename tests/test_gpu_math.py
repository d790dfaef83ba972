"""The kernels' own branch-free elementary functions (pimc_math.cuh) against the host libm (numpy), through the
pimc_math_selftest entry of the C ABI.  They must stay within a few ulp so that proposals and log-uniforms agree
with the oracle to rounding."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def ulps(a, ref):
    return np.abs(a - ref) / np.spacing(np.abs(ref))


def test_elementary_functions_within_a_few_ulp():
    import torch
    import paper_1103_4887_b200 as P
    rng = np.random.default_rng(1)
    x = np.concatenate([rng.uniform(-700, 700, 100000), rng.uniform(-1, 1, 100000), rng.uniform(0, 7.9, 100000),
                        (rng.integers(0, 2**32, 100000) + 0.5) * 2.0**-32, 2.0 ** rng.uniform(-40, 40, 50000),
                        [0.5, 1.0, 2.0, np.pi / 2, np.pi, 3 * np.pi / 2, 2 * np.pi, 1e-9, 2.0**-33, 1 - 2.0**-33, 45.7]])
    out = P.math_selftest(torch.from_numpy(x).cuda()).cpu().numpy()
    ax = np.abs(x)
    ok = np.abs(x) <= 700
    assert ulps(out[ok, 0], np.exp(x[ok])).max() <= 2.0
    # log: relative accuracy, except right at 1 where the result is tiny: there the absolute error is bounded by ulp(1)
    ref = np.log(ax)
    err = np.abs(out[:, 1] - ref)
    assert np.all((err <= 2.0 * np.spacing(np.abs(ref))) | (err <= 2.0**-52)), ulps(out[:, 1], ref).max()
    assert ulps(out[:, 2], np.sqrt(ax)).max() <= 1.0
    a = np.minimum(ax, 7.9)
    assert np.max(np.abs(out[:, 3] - np.sin(a))) <= 2.0**-52 and np.max(np.abs(out[:, 4] - np.cos(a))) <= 2.0**-52
    big = np.abs(np.sin(a)) > 0.1
    assert ulps(out[big, 3], np.sin(a[big])).max() <= 4.0
    assert ulps(out[:, 5], 1.0 / ax).max() <= 2.0
    # the shared-exponential form of the three HH gate rates against the tanh definition (Table 1 shifted by
    # -65 mV) in long double, over the whole finite range (saturation included)
    sel = np.abs(x) < 700
    V = x[sel].astype(np.longdouble)
    for col, (Va, dVa, tau0, tau1) in enumerate(((-40, 15, 0.1, 0.4), (-60, -15, 1.0, 7.0), (-55, 30, 1.0, 5.0))):
        th = np.tanh((V - Va) / np.longdouble(dVa))
        ref = ((0.5 + 0.5 * th) - np.longdouble(0.3)) / (np.longdouble(tau0) + np.longdouble(tau1) * (1 - th * th))
        got = out[sel, 6 + col]
        ref = ref.astype(np.float64)
        # the rate is O(1/tau) <= 10; where a_inf ~ a it cancels, so the bound is absolute + relative
        assert np.all(np.abs(got - ref) <= 1e-14 + 6e-15 * np.abs(ref)), (col, np.max(np.abs(got - ref)))
