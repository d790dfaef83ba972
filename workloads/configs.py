"""Workload recipes (BASELINE.json `configs`).

Stand-ins for the paper's Lorenz-driven Hodgkin-Huxley series,
which is not available.  Everything is drawn from ``numpy.random.default_rng``
with data seed = 11034887 + config index (+ 1000*chain for batched chains).
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

MODEL_LINEAR = 0
MODEL_HH = 1
MODEL_HH_CLASSIC = 2          # classic alpha/beta rate functions
N_CONFIGS = 5
DATA_SEED0 = 11034887

# (gNa, gK, gL, ENa, EK, EL, C)  -- BASELINE.json config 0 "standard HH" values
HH_P_TRUE = np.array([120.0, 36.0, 0.3, 50.0, -77.0, -54.4, 1.0])

# tanh kinetics of PAPER.md:268-270 (Eq. 13-14) with Table 1
# shifted by -65 mV: (V_a, dV_a, tau_a0, tau_a1)
_KIN = {"m": (-40.0, 15.0, 0.1, 0.4), "h": (-60.0, -15.0, 1.0, 7.0), "n": (-55.0, 30.0, 1.0, 5.0)}


def _classic_rates(V):
    """Data-synthesis only: classic Hodgkin-Huxley alpha/beta at rest = -65 mV."""
    def vtrap(u):
        u = np.where(np.abs(u) < 1e-9, 1e-9, u)
        return u / -np.expm1(-u)
    am, bm = vtrap((V + 40.0) / 10.0), 4.0 * np.exp(-(V + 65.0) / 18.0)
    ah, bh = 0.07 * np.exp(-(V + 65.0) / 20.0), 1.0 / (1.0 + np.exp(-(V + 35.0) / 10.0))
    an, bn = 0.1 * vtrap((V + 55.0) / 10.0), 0.125 * np.exp(-(V + 65.0) / 80.0)
    return (am, bm), (ah, bh), (an, bn)


def _hh_rhs_batch(x, I, p, kinetics="tanh"):
    """Data-synthesis only.  x: (..., 4) = (V, m, h, n); I: (...,); p: (7,)."""
    V, m, h, n = x[..., 0], x[..., 1], x[..., 2], x[..., 3]
    gNa, gK, gL, ENa, EK, EL, C = p
    out = np.empty_like(x)
    out[..., 0] = (I + gNa * m**3 * h * (ENa - V) + gK * n**4 * (EK - V) + gL * (EL - V)) / C
    if kinetics == "classic":
        for j, (al, be) in enumerate(_classic_rates(V), start=1):
            out[..., j] = al * (1.0 - x[..., j]) - be * x[..., j]
        return out
    for j, key in ((1, "m"), (2, "h"), (3, "n")):
        Va, dVa, t0, t1 = _KIN[key]
        th = np.tanh((V - Va) / dVa)
        out[..., j] = (0.5 + 0.5 * th - x[..., j]) / (t0 + t1 * (1.0 - th * th))
    return out


def lorenz_current(M: int, dt: float, rng: np.random.Generator, n_chains: int = 1, ms_per_unit: float = 20.0,
                   offset: float = 5.0, gain: float = 0.7):
    """Chaotic stimulus for the paper-shaped workload ("a chaotic stimulus current generated from one of the
    variables of the Lorenz model").  The paper's series is not available and its scaling is not stated: the x variable of
    the Lorenz-63 system (sigma = 10, rho = 28, beta = 8/3), one Lorenz time unit = ms_per_unit ms, I = offset + gain * x
    uA/cm2 (about -9 .. 19), started from a seeded point after a transient.  Returns I (C, M+1)."""
    h = dt / ms_per_unit
    sub = max(1, int(np.ceil(h / 0.002)))
    hs = h / sub

    def f(u):
        return np.stack([10.0 * (u[:, 1] - u[:, 0]), u[:, 0] * (28.0 - u[:, 2]) - u[:, 1], u[:, 0] * u[:, 1] - (8.0 / 3.0) * u[:, 2]], axis=1)

    def step(u):
        k1 = f(u); k2 = f(u + 0.5 * hs * k1); k3 = f(u + 0.5 * hs * k2); k4 = f(u + hs * k3)
        return u + (hs / 6.0) * (k1 + 2 * k2 + 2 * k3 + k4)

    u = np.array([1.0, 1.0, 20.0])[None, :] + rng.normal(size=(n_chains, 3))
    for _ in range(int(20.0 / hs)):                      # transient onto the attractor
        u = step(u)
    I = np.empty((n_chains, M + 1))
    for k in range(M + 1):
        I[:, k] = offset + gain * u[:, 0]
        for _ in range(sub):
            u = step(u)
    return I


def hh_truth(M: int, dt: float, rng: np.random.Generator, n_chains: int = 1, kinetics: str = "tanh", I=None, p=None,
             noise_sd: float = 1.0):
    """Twin-experiment data: returns I (C,M+1), x_true (C,M+1,4), y (C,M+1).

    Step current: 5 ms segments, segment k covers steps [k*5/dt, (k+1)*5/dt), amplitude U(0,15) uA/cm2.
    Truth: RK4 at dt with midpoint current 0.5*(I_n + I_{n+1}); x(0) = rest at -65 mV.
    Observation: V + N(0, 1 mV).
    """
    if I is None:
        seg = int(round(5.0 / dt))
        nseg = M // seg + 2
        amp = rng.uniform(0.0, 15.0, size=(n_chains, nseg))
        idx = np.arange(M + 1) // seg
        I = amp[:, idx]
    x = np.empty((n_chains, M + 1, 4))
    V0 = -65.0
    x[:, 0, 0] = V0
    for j, key in ((1, "m"), (2, "h"), (3, "n")):
        Va, dVa, _, _ = _KIN[key]
        x[:, 0, j] = 0.5 + 0.5 * np.tanh((V0 - Va) / dVa)
    if kinetics == "classic":
        for j, (al, be) in enumerate(_classic_rates(np.float64(V0)), start=1):
            x[:, 0, j] = al / (al + be)
    p = HH_P_TRUE if p is None else p
    for k in range(M):
        xn = x[:, k]
        I0, I1 = I[:, k], I[:, k + 1]
        Ih = 0.5 * (I0 + I1)
        k1 = _hh_rhs_batch(xn, I0, p, kinetics)
        k2 = _hh_rhs_batch(xn + 0.5 * dt * k1, Ih, p, kinetics)
        k3 = _hh_rhs_batch(xn + 0.5 * dt * k2, Ih, p, kinetics)
        k4 = _hh_rhs_batch(xn + dt * k3, I1, p, kinetics)
        x[:, k + 1] = xn + (dt / 6.0) * (k1 + 2 * k2 + 2 * k3 + k4)
    y = x[:, :, 0] + rng.normal(0.0, noise_sd, size=(n_chains, M + 1))
    return I, x, y


def linear_matrix(D: int = 2, rho: float = 0.99, theta: float = 0.05) -> np.ndarray:
    """Config 1 map matrix A = 0.99 * R(0.05 rad) (row-major D*D; D=1 gives [[rho]])."""
    if D == 1:
        return np.array([[rho]])
    A = np.eye(D)
    c, s = np.cos(theta), np.sin(theta)
    A[0, 0], A[0, 1], A[1, 0], A[1, 1] = c, -s, s, c
    return rho * A


def linear_truth(M: int, rng: np.random.Generator, D: int = 2, q_sd: float = 0.1, r_sd: float = 0.1):
    """x_{n+1} = A x_n + N(0, q_sd^2 I), x_0 ~ N(0, I); y_n = x_{n,0} + N(0, r_sd^2)."""
    A = linear_matrix(D)
    x = np.empty((M + 1, D))
    x[0] = rng.normal(size=D)
    for k in range(M):
        x[k + 1] = A @ x[k] + q_sd * rng.normal(size=D)
    y = x[:, 0] + r_sd * rng.normal(size=M + 1)
    return A, x, y


@dataclass
class Workload:
    """Everything pimc_init / pimc_set_* need, as plain numpy arrays (fp64)."""
    name: str
    model: int
    D: int
    L: int
    Np: int
    M: int
    dt: float
    Rm: float
    Rf: np.ndarray            # (D,)
    n_chains: int
    p0: np.ndarray            # (C, Np)
    p_true: np.ndarray        # (Np,)
    lo: np.ndarray            # (C, Np)
    hi: np.ndarray            # (C, Np)
    w_state: np.ndarray       # (D,)
    w_param: np.ndarray       # (Np,)  0 = frozen
    y: np.ndarray             # (C, M+1, L)
    I: np.ndarray | None      # (C, M+1) or None
    x0: np.ndarray            # (C, M+1, D) initial path
    x_true: np.ndarray        # (C, M+1, D)
    n_sweeps: int
    chain_seed: int = 1       # Philox key; chain index goes in the counter
    extra: dict = field(default_factory=dict)


_WP_CFG2 = np.array([0.10, 0.03, 0.008, 0.025, 0.035, 0.5, 0.004])
_WP_CFG3 = np.array([0.07, 0.02, 0.005, 0.018, 0.025, 0.4, 0.0026])


def _hh_workload(name, cfg, M, dt, n_chains, w_param, n_sweeps, estimate, seed=None, kinetics="tanh"):
    rng = np.random.default_rng(DATA_SEED0 + cfg if seed is None else seed)
    I, xt, y = hh_truth(M, dt, rng, n_chains, kinetics)
    x0 = np.empty((n_chains, M + 1, 4))
    x0[:, :, 0] = y
    x0[:, :, 1:] = 0.5
    pt = HH_P_TRUE
    if estimate:
        s = np.where(rng.random((n_chains, 7)) < 0.5, -1.0, 1.0)      # G8: +-20 % off truth
        p0 = pt[None, :] * (1.0 + 0.2 * s)
        wp = np.asarray(w_param, float)
    else:
        p0 = np.tile(pt, (n_chains, 1))
        wp = np.zeros(7)
    lo = np.tile(pt - 0.5 * np.abs(pt), (n_chains, 1))
    hi = np.tile(pt + 0.5 * np.abs(pt), (n_chains, 1))
    return Workload(name=name + ("_classic" if kinetics == "classic" else ""), model=MODEL_HH_CLASSIC if kinetics == "classic" else MODEL_HH, D=4, L=1, Np=7, M=M, dt=dt, Rm=1.0,
                    Rf=np.array([1e2, 1e4, 1e4, 1e4]), n_chains=n_chains, p0=p0, p_true=pt.copy(),
                    lo=lo, hi=hi, w_state=np.array([0.5, 0.02, 0.02, 0.02]), w_param=wp,
                    y=y[:, :, None].copy(), I=I, x0=x0, x_true=xt, n_sweeps=n_sweeps)


def make_workload(cfg: int, *, M: int | None = None, n_chains: int | None = None,
                  seed: int | None = None, kinetics: str = "tanh") -> Workload:
    """BASELINE.json `configs[cfg]`; M / n_chains may be overridden to make small parity cases.
    kinetics = "classic" generates the Hodgkin-Huxley configs with the classic alpha/beta rate functions (model 2)."""
    if cfg == 0:
        return _hh_workload("cfg0_hh_M256", 0, M or 256, 0.02, n_chains or 1, None, 2000, False, seed, kinetics)
    if cfg == 1:
        M = M or 4096
        rng = np.random.default_rng(DATA_SEED0 + 1 if seed is None else seed)
        A, xt, y = linear_truth(M, rng)
        x0 = np.zeros((1, M + 1, 2))
        x0[0, :, 0] = y
        return Workload(name="cfg1_linear_M4096", model=MODEL_LINEAR, D=2, L=1, Np=4, M=M, dt=1.0,
                        Rm=100.0, Rf=np.array([100.0, 100.0]), n_chains=1, p0=A.reshape(1, 4).copy(),
                        p_true=A.reshape(4).copy(), lo=np.full((1, 4), -2.0), hi=np.full((1, 4), 2.0),
                        w_state=np.array([0.1, 0.1]), w_param=np.zeros(4), y=y[None, :, None].copy(),
                        I=None, x0=x0, x_true=xt[None], n_sweeps=5000)
    if cfg == 2:
        return _hh_workload("cfg2_hh_M4096_params", 2, M or 4096, 0.02, n_chains or 1, _WP_CFG2, 20000, True, seed, kinetics)
    if cfg == 3:
        return _hh_workload("cfg3_hh_M32768_params", 3, M or 32768, 0.01, n_chains or 1, _WP_CFG3, 10000, True, seed, kinetics)
    if cfg == 4:
        return _hh_workload("cfg4_hh_128x8192_params", 4, M or 8192, 0.02, n_chains or 128,
                            _WP_CFG2 / np.sqrt(2.0), 5000, True, seed, kinetics)
    if cfg == 5:
        return _paper_workload(M or 8000, n_chains or 1, seed, kinetics)
    raise ValueError(f"no config {cfg}")


# PAPER.md:282-284, Table 2, in this build's conventions: rest at -65 mV instead of 0 (E_Na = 115 - 65,
# E_K = -12 - 65, E_L = 10.6 - 65) and physical parameters (gNa, gK, gL, ENa, EK, EL, C) instead of (p_1..p_7).
PAPER_P_TRUE = np.array([120.0, 20.0, 0.3, 50.0, -77.0, -54.4, 1.0])


def _paper_workload(M, n_chains, seed, kinetics):
    """The paper's own experiment shape: M = 8000 steps of dt = 0.04 ms (25 kHz,
    320 ms), Lorenz-driven current, R_d = diag(100, 1e6, 1e6, 1e6), R_o = 100, gK = 20, initial step sizes 2e-3 (V) and 1e-3
    (gates), to be tuned.  Synthetic regeneration: the original series is not available.  Meant for the trapezoid
    discretisation with annealing (beta0 = 0.01) and step-size tuning (f_acc = 0.23, alpha = 0.02, N_skip = 400)."""
    dt = 0.04
    rng = np.random.default_rng(DATA_SEED0 + 5 if seed is None else seed)
    I = lorenz_current(M, dt, rng, n_chains)
    pt = PAPER_P_TRUE
    I, xt, y = hh_truth(M, dt, rng, n_chains, kinetics, I=I, p=pt, noise_sd=0.1)     # R_o = 100 <=> sd 0.1 mV
    x0 = np.empty((n_chains, M + 1, 4))
    x0[:, :, 0] = y
    x0[:, :, 1:] = 0.5
    sgn = np.where(rng.random((n_chains, 7)) < 0.5, -1.0, 1.0)
    p0 = pt[None, :] * (1.0 + 0.2 * sgn)
    lo = np.tile(pt - 0.5 * np.abs(pt), (n_chains, 1))
    hi = np.tile(pt + 0.5 * np.abs(pt), (n_chains, 1))
    return Workload(name="cfg5_paper_shape_M8000" + ("_classic" if kinetics == "classic" else ""),
                    model=MODEL_HH_CLASSIC if kinetics == "classic" else MODEL_HH, D=4, L=1, Np=7, M=M, dt=dt, Rm=100.0,
                    Rf=np.array([1e2, 1e6, 1e6, 1e6]), n_chains=n_chains, p0=p0, p_true=pt.copy(), lo=lo, hi=hi,
                    w_state=np.array([2e-3, 1e-3, 1e-3, 1e-3]), w_param=1e-3 * np.abs(pt), y=y[:, :, None].copy(), I=I, x0=x0,
                    x_true=xt, n_sweeps=1000000,
                    extra=dict(n_init=500000, n_cool=100000, beta0=0.01, f_acc=0.23, alpha=0.02, n_skip=400, disc="trapezoid"))
