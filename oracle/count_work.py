"""Operation count of the oracle's arithmetic: the ALGORITHMIC work per unit that bench.py's roofline credits
("Fix W_site and W_eval once (from the oracle's operation count)").

    python -m oracle.count_work            # prints the table and rewrites oracle/work_constants.json

Test infrastructure, like everything under oracle/.  It restates, operation by operation and in the oracle's own order,
what pimc_oracle.cpp does for (i) one joint site update (proposal draw, RK4 increment at the proposal, local Delta-A,
accept uniform) and (ii) one parameter-move model evaluation (RK4 increment with the proposed parameters, one term of the
Delta-A sum), on a number type that counts.  The restatement is VALIDATED against the compiled oracle bit for bit (the
oracle is built with -ffp-contract=off, so IEEE double operations in the same order give the same bits; a missing or
reordered operation would not): step increment, site Delta-A and parameter Delta-A of random states must be identical.

Counting rules (one "slot" = one FP64-pipe lane operation = one add, multiply or fused multiply-add):
  * every + - * counts one slot; a product that is consumed once by an add/subtract counts zero (the pair is one FMA);
  * library calls are costed by LIBM_SLOTS: FP64-pipe instruction counts of branch-free double-precision routines of the
    usual construction (range reduction + polynomial; reciprocal seed + Newton / series steps; the seed itself runs on another
    pipe), counted by hand from the routines the CUDA kernels use.  A cost table only: this module never imports
    paper_1103_4887_b200 and shares no code with it;
  * the oracle-only diagnostics are not work of the method and are not counted: the scale S = sum |terms| it returns for
    the test tolerances, and the Neumaier compensation of its parameter sum (counted as the one add a plain sum needs);
  * integer work (Philox, the 2^k scaling inside exp) is not FP64-pipe work.
"""
from __future__ import annotations

import json
import math
import os

import numpy as np

LIBM_SLOTS = {"div": 6, "exp": 19, "tanh": 27, "log": 23, "sqrt": 10, "sincos": 20, "u2f": 1}
HERE = os.path.dirname(os.path.abspath(__file__))
OUT = os.path.join(HERE, "work_constants.json")


class Tally:
    def __init__(self):
        self.slots = 0          # with mul+add fusion
        self.ops = 0            # every + - * counted
        self.calls = {}

    def call(self, name, n=1):
        self.calls[name] = self.calls.get(name, 0) + n
        self.slots += LIBM_SLOTS[name] * n
        self.ops += LIBM_SLOTS[name] * n


class C:
    """A double that counts.  `prod` marks a product not yet consumed: its first use in an add/subtract is free (FMA)."""
    __slots__ = ("v", "t", "prod")

    def __init__(self, v, t, prod=False):
        self.v, self.t, self.prod = float(v), t, prod

    @staticmethod
    def _val(o):
        return o.v if isinstance(o, C) else float(o)

    def _addsub(self, o, sign, swap=False):
        a, b = (C._val(o), self.v) if swap else (self.v, C._val(o))
        r = a + b if sign > 0 else a - b
        self.t.ops += 1
        fused = False
        for q in (self, o):
            if isinstance(q, C) and q.prod and not fused:
                q.prod = False
                fused = True
        if not fused:
            self.t.slots += 1
        return C(r, self.t)

    def __add__(self, o): return self._addsub(o, +1)
    def __radd__(self, o): return self._addsub(o, +1, swap=True)
    def __sub__(self, o): return self._addsub(o, -1)
    def __rsub__(self, o): return self._addsub(o, -1, swap=True)

    def __mul__(self, o):
        self.t.ops += 1
        self.t.slots += 1
        return C(self.v * C._val(o), self.t, prod=True)
    __rmul__ = __mul__

    def __truediv__(self, o):
        self.t.call("div")
        return C(self.v / C._val(o), self.t)

    def __rtruediv__(self, o):
        self.t.call("div")
        return C(C._val(o) / self.v, self.t)

    def __neg__(self):
        return C(-self.v, self.t, self.prod)      # sign flip: not an FP64-pipe operation


def tanh(x): x.t.call("tanh"); return C(math.tanh(x.v), x.t)
def log(x): x.t.call("log"); return C(math.log(x.v), x.t)
def sqrt(x): x.t.call("sqrt"); return C(math.sqrt(x.v), x.t)
def sincos(x): x.t.call("sincos"); return C(math.sin(x.v), x.t), C(math.cos(x.v), x.t)


# ---- the oracle's arithmetic, restated (pimc_oracle.cpp: gate_rate, hh_rhs, step_increment, site_delta_A, ...) ----------
KIN = {"m": (-40.0, 15.0, 0.1, 0.4), "h": (-60.0, -15.0, 1.0, 7.0), "n": (-55.0, 30.0, 1.0, 5.0)}


def gate_rate(k, V, a):
    Va, dVa, tau0, tau1 = k
    th = tanh((V - Va) / dVa)
    a_inf = 0.5 + 0.5 * th
    tau = tau0 + tau1 * (1.0 - th * th)
    return (a_inf - a) / tau


def hh_rhs(x, p, I):
    V, m, h, n = x
    gNa, gK, gL, ENa, EK, EL, Cm = p
    F0 = (I + gNa * (m * m * m) * h * (ENa - V) + gK * (n * n * n * n) * (EK - V) + gL * (EL - V)) / Cm
    return [F0, gate_rate(KIN["m"], V, m), gate_rate(KIN["h"], V, h), gate_rate(KIN["n"], V, n)]


def step_increment(x, p, I0, I1, dt):
    Ih = 0.5 * (I0 + I1)                               # plain floats: the midpoint current is one add + one multiply per site
    x[0].t.ops += 2; x[0].t.slots += 2
    k1 = hh_rhs(x, p, I0)
    xs = [x[a] + 0.5 * dt * k1[a] for a in range(4)]
    k2 = hh_rhs(xs, p, Ih)
    xs = [x[a] + 0.5 * dt * k2[a] for a in range(4)]
    k3 = hh_rhs(xs, p, Ih)
    xs = [x[a] + dt * k3[a] for a in range(4)]
    k4 = hh_rhs(xs, p, I1)
    return [(dt / 6.0) * (k1[a] + 2.0 * k2[a] + 2.0 * k3[a] + k4[a]) for a in range(4)]


def terms(Rf_a, r_new, r_old):
    t_new, t_old = 0.5 * Rf_a * r_new * r_new, 0.5 * Rf_a * r_old * r_old
    return t_new - t_old


def site_delta_A(t, xn, xp, xm, gm, xq, gn, y, p, I0, I1, dt, Rm, Rf):
    """Interior site (1 <= n <= M-1), RK4 map, L = 1: the three terms of row A2."""
    dA = C(0.0, t)
    for a in range(4):
        dA = dA + terms(Rf[a], (xp[a] - xm[a]) - gm[a], (xn[a] - xm[a]) - gm[a])
    dA = dA + terms(Rm, y - xp[0], y - xn[0])
    gp = step_increment(xp, p, I0, I1, dt)
    for a in range(4):
        dA = dA + terms(Rf[a], (xq[a] - xp[a]) - gp[a], (xq[a] - xn[a]) - gn[a])
    return dA, gp


def propose_and_accept_draws(t, xn, w):
    """Gaussian proposal of D = 4 components (two Box-Muller pairs) and log u of the accept test (pimc_oracle.cpp:
    u01_from_word, box_muller, propose_site, accept_log_u_state) on fixed uniforms: the count does not depend on them."""
    xp = []
    for pair in range(2):
        u1, u2 = C(0.3 + 0.1 * pair, t), C(0.6 - 0.2 * pair, t)
        t.call("u2f", 2); t.slots += 4; t.ops += 4            # (double)w + 0.5, * 2^-32, twice
        r = sqrt(-2.0 * log(u1))
        s, c = sincos(6.283185307179586 * u2)
        z = (r * c, r * s)
        for j in range(2):
            a = 2 * pair + j
            xp.append(xn[a] + w[a] * z[j])
    t.call("u2f", 1); t.slots += 2; t.ops += 2                # the 52-bit accept uniform
    logu = log(C(0.37, t))
    return xp, logu


def param_eval(t, xn, xq, gn, pp, I0, I1, dt, Rf):
    """One site's share of a parameter move (row A4): increment with the proposed parameters and its Delta-A term."""
    gp = step_increment(xn, pp, I0, I1, dt)
    part = C(0.0, t)
    for a in range(4):
        d = xq[a] - xn[a]
        part = part + terms(Rf[a], d - gp[a], d - gn[a])
    return part, gp


# ---- validation against the compiled oracle + the counts ---------------------------------------------------------------
def _validate_and_count():
    import sys
    sys.path.insert(0, os.path.dirname(HERE))
    import oracle
    from oracle import OracleChain
    from workloads import MODEL_HH, make_workload
    w = make_workload(2, M=64)
    o = OracleChain.from_workload(w)
    o.sweep(5, seed=3)                                            # a path that is not the initial one
    x, p = o.get_path()
    g = o.get_cache()
    I, y, dt = np.asarray(w.I[0], float), np.asarray(w.y[0], float).reshape(-1), float(w.dt)
    rng = np.random.default_rng(0)
    site = eval_ = None
    for n in (1, 17, 40, 63):
        # (i) step increment and site Delta-A at a random proposal
        xp_v = x[n] + np.asarray(w.w_state) * rng.normal(size=4)
        t = Tally()
        cx = lambda v: [C(q, t) for q in v]
        dA, gp = site_delta_A(t, cx(x[n]), cx(xp_v), cx(x[n - 1]), cx(g[n - 1]), cx(x[n + 1]), cx(g[n]), C(y[n], t), cx(p),
                              float(I[n]), float(I[n + 1]), dt, float(w.Rm), [float(v) for v in w.Rf])
        ref_g = oracle.step_increment(MODEL_HH, xp_v, p, I[n], I[n + 1], dt)
        ref_dA, _ = o.site_delta_A(n, xp_v)
        assert [q.v for q in gp] == list(ref_g), "restated RK4 increment is not the oracle's"
        assert dA.v == ref_dA, "restated site Delta-A is not the oracle's"
        propose_and_accept_draws(t, cx(x[n]), [float(v) for v in w.w_state])
        site = t
        # (ii) parameter-move evaluation: the sum of the per-site terms must be the oracle's Delta-A of the move
    l, pl = 1, p[1] * 1.001
    pp = p.copy(); pp[l] = pl
    ref, _ = o.param_delta_A(l, pl)
    tot = 0.0
    comp = 0.0
    for n in range(w.M):
        t = Tally()
        cx = lambda v: [C(q, t) for q in v]
        part, _ = param_eval(t, cx(x[n]), cx(x[n + 1]), cx(g[n]), cx(pp), float(I[n]), float(I[n + 1]), dt, [float(v) for v in w.Rf])
        eval_ = t
        tot += part.v
    assert abs(tot - ref) <= 1e-12 * max(abs(ref), 1.0), (tot, ref)     # plain vs Neumaier sum of identical terms
    return site, eval_


def main():
    site, ev = _validate_and_count()
    out = {
        "slots_per_site_update": site.slots, "ops_per_site_update_unfused": site.ops, "calls_per_site_update": site.calls,
        "slots_per_param_eval": ev.slots, "ops_per_param_eval_unfused": ev.ops, "calls_per_param_eval": ev.calls,
        "libm_slots": LIBM_SLOTS,
        "rule": "one slot per add/sub/mul, a product consumed once by an add is free (FMA); libm calls by libm_slots; "
                "oracle diagnostics (S, Neumaier compensation) and integer work not counted; interior site, HH tanh kinetics, "
                "RK4 map, D = 4, L = 1, Gaussian proposals",
    }
    print(json.dumps(out, indent=1))
    with open(OUT, "w") as f:
        json.dump(out, f, indent=1)
        f.write("\n")


if __name__ == "__main__":
    main()
