"""Shared helpers for the GPU parity tests: build both sides from the same workload, teacher-forced comparison."""
from __future__ import annotations

import numpy as np

from oracle import OracleChain

TOL64 = 1e-12      # north_star: per-site Delta-A relative tolerance in fp64 (relative to max(|dA|, S))
TOL32 = 1e-5       # fp32
TIE64 = 1e-9       # near-tie window |dA + log u|


def gpu_handle(w, dtype=64, with_params=True, launch=None, kind=0, disc=0):
    import paper_1103_4887_b200 as P
    h = P.Pimc.from_workload(w, dtype=dtype, with_params=with_params)
    if disc:
        h.set_discretisation(disc)
    h.set_proposal(w.w_state, w.w_param if with_params else None, kind)
    if launch:
        h.set_launch(*launch)
    return h


def oracle_chains(w, state_dtype=64, with_params=True, kind=0, disc=0):
    out = []
    for c in range(w.n_chains):
        o = OracleChain.from_workload(w, chain=c, state_dtype=state_dtype, with_params=with_params)
        if disc:
            o.set_discretisation(disc)
        o.set_proposal(w.w_state, w.w_param if with_params else None, kind)
        out.append(o)
    return out


def to_dev(a, h):
    import torch
    return torch.as_tensor(np.ascontiguousarray(a), dtype=h.tdtype).to(h.device).contiguous()


def ulp_diff(a, b):
    a = np.asarray(a, dtype=np.float64); b = np.asarray(b, dtype=np.float64)
    return np.abs(a - b) / np.maximum(np.spacing(np.maximum(np.abs(a), np.abs(b))), 1e-300)


def teacher_forced(w, h, orcs, n_sweeps, seed, tol=TOL64, tie=TIE64, do_params=True, state_dtype=64, disc=0, anneal=None):
    """SURVEY.md §8(c) T1.  For every sweep: force the GPU to the oracle's state, run one sweep on both with the
    trace on, and compare per-site Delta-A (evaluated by the oracle AT THE GPU's proposals, on the path as it stood
    when the site was visited), decisions, parameter moves and the resulting path.  Returns a report dict."""
    C, M, D, Np = w.n_chains, w.M, w.D, h.Np
    tr = h.enable_trace()
    rep = dict(sites=0, max_rel=0.0, ties=0, mismatch_outside_window=0, max_xprop_ulp=0.0, max_param_rel=0.0, param_ties=0,
               param_moves=0, max_path_diff=0.0, accepted=0)
    helper = [OracleChain.from_workload(w, chain=c, state_dtype=state_dtype, with_params=do_params) for c in range(C)]
    for hc in helper:
        if disc:
            hc.set_discretisation(disc)
        if anneal:
            hc.set_annealing(*anneal)
    for t in range(n_sweeps):
        X = np.stack([o.get_path()[0] for o in orcs]); Pp = np.stack([o.get_path()[1] for o in orcs])
        h.set_params(to_dev(Pp, h)); h.set_path(to_dev(X, h))
        h.sweep_index = orcs[0].sweep_index
        for hc in helper:
            hc.sweep_index = orcs[0].sweep_index          # same annealing multiplier as the sweep under test
        if do_params:
            h.sweep(1, seed)
        else:
            h.sweep_states_only(1, seed)
        g = {k: (v.cpu().numpy().astype(np.float64) if v is not None and v.dtype != h.torch.uint8 else (None if v is None else v.cpu().numpy()))
             for k, v in tr.items()}
        xg, pg = [a.cpu().numpy().astype(np.float64) for a in h.get_path()]
        for c, o in enumerate(orcs):
            o.sweep(1, seed, do_params=do_params)
            ot = o.trace()
            # --- state updates: oracle dA at the GPU's proposals, two stages (even sites on X, odd on X after even) ---
            hc = helper[c]
            hc.set_params(Pp[c]); hc.set_path(X[c])
            stage = X[c].copy()
            for parity in (0, 1):
                sites = range(parity, M + 1, 2)
                for n in sites:
                    dA_ref, S = hc.site_delta_A(n, g["xprop"][c, n])
                    err = abs(g["dA"][c, n] - dA_ref) / max(abs(dA_ref), S, 1e-300)
                    rep["max_rel"] = max(rep["max_rel"], err)
                    near = abs(dA_ref + ot["logu"][n]) < tie * max(1.0, S if state_dtype == 32 else 1.0)
                    expect = ot["logu"][n] < -dA_ref
                    if bool(g["acc"][c, n]) != bool(expect):
                        if near:
                            rep["ties"] += 1
                        else:
                            rep["mismatch_outside_window"] += 1
                    rep["sites"] += 1
                    if g["acc"][c, n]:
                        stage[n] = g["xprop"][c, n]; rep["accepted"] += 1
                hc.set_path(stage)
            # proposals: same draw, different math library for log/sqrt/sincos -> a few ulp of the operands' scale
            scale = np.maximum(np.maximum(np.abs(X[c]), np.abs(ot["xprop"])), 4.0 * np.asarray(w.w_state)[None, :])
            rep["max_xprop_ulp"] = max(rep["max_xprop_ulp"], float((np.abs(g["xprop"][c] - ot["xprop"]) / np.spacing(scale)).max()))
            # --- parameter moves ---
            if do_params:
                for l in range(Np):
                    if np.isnan(ot["dAp"][l]):
                        assert np.isnan(g["dAp"][c, l]) and g["accp"][c, l] == 0, (t, c, l)
                        continue
                    rep["param_moves"] += 1
                    err = abs(g["dAp"][c, l] - ot["dAp"][l]) / max(abs(ot["dAp"][l]), ot["Sp"][l], 1e-300)
                    rep["max_param_rel"] = max(rep["max_param_rel"], err)
                    if bool(g["accp"][c, l]) != bool(ot["accp"][l]):
                        assert abs(ot["dAp"][l] + ot["logup"][l]) < tie * max(1.0, ot["Sp"][l] * tol / tie), (t, c, l)
                        rep["param_ties"] += 1
            xo, po = o.get_path()
            same = (g["acc"][c] == ot["acc"])
            if same.all() and (not do_params or np.array_equal(g["accp"][c], ot["accp"])):
                rep["max_path_diff"] = max(rep["max_path_diff"], float(np.abs(xg[c] - xo).max()))
    h.disable_trace()
    return rep
