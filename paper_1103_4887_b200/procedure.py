"""The paper's example calculation, start to finish, through the public binding:

    initialisation phase   N_init iterations: simulated annealing of the dynamics term over the first N_cool of them
                           (beta_0 -> 1, Eq. 10) and step-size tuning every N_skip iterations towards the
                           acceptance rate f_acc; nothing is recorded
    production phase       N - N_init iterations with the step sizes frozen, the path and the parameters recorded every
                           N_skip-th iteration, means and standard deviations read out at the end

on the synthetic stand-in for the paper's experiment (`make_workload(5)`: M = 8000, dt = 0.04 ms, Lorenz-driven current,
trapezoid rule).  Every iteration runs in libpimc's kernels; this module only sequences the calls.

    python -m paper_1103_4887_b200.procedure                      # the paper's 10^6 iterations (about a quarter of a minute on a B200)
    python -m paper_1103_4887_b200.procedure --iterations 20000   # a short run

prints one JSON line: seconds per phase (wall clock around a device synchronize), iterations/s, the engine each phase ran on,
the estimated parameters with their standard deviations next to the values the data were generated with.
"""
from __future__ import annotations

import argparse
import json
import time


def run(iterations=1_000_000, n_init=None, n_cool=None, n_skip=400, beta0=0.01, f_acc=0.23, alpha=0.02, seed=1103, dtype=64,
        M=None, chunk=20_000, workload=None):
    """workload: any object with the fields of workloads.Workload (the caller's own data); None = the synthetic stand-in for the
    paper's experiment from the repository's `workloads` module (needs the repository root on sys.path)."""
    import torch
    from . import binding as B
    if workload is None:
        try:
            from workloads import make_workload
        except ImportError as e:
            raise ImportError("procedure.run() without `workload=` uses the repository's synthetic workload generator: put the "
                              "repository root on sys.path or pass your own workload object") from e

    if not torch.cuda.is_available():
        raise RuntimeError("paper_1103_4887_b200.procedure needs a CUDA device (libpimc has no CPU path)")
    n_init = iterations // 2 if n_init is None else n_init            # the first half is excluded
    n_cool = iterations // 10 if n_cool is None else n_cool           # N_cool = 10^5 of 10^6
    w = workload if workload is not None else (make_workload(5) if M is None else make_workload(5, M=M))
    h = B.Pimc.from_workload(w, dtype=dtype)
    h.set_discretisation(B.DISC_TRAPEZOID)
    h.set_proposal(w.w_state, w.w_param)                              # PAPER.md:282 initial step sizes
    if n_cool > 0:
        h.set_annealing(beta0, n_cool)
    h.set_tuning(True, n_skip, f_acc, alpha)

    def sweeps(n):
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        done = 0
        while done < n:                                               # bounded launches: a call returns within seconds
            k = min(chunk, n - done)
            h.sweep(k, seed)
            done += k
        torch.cuda.synchronize()
        return time.perf_counter() - t0

    engine_init = h.get_engine()["engine"]
    t_init = sweeps(n_init)
    h.set_tuning(False)                                               # step sizes stay as tuned
    h.set_accum(True, n_skip)
    h.reset_moments()
    engine_prod = h.get_engine()["engine"]
    n_prod = iterations - n_init
    t_prod = sweeps(n_prod)

    mx, mp, n_samples = h.moments()
    st = h.stats().cpu().numpy()[0]
    ws, wp = [a.cpu().numpy()[0] for a in h.get_widths()]
    mp = mp.cpu().numpy()[0]                                          # (2, Np): mean, variance
    names = {B.ENGINE_GLOBAL: "global-memory", B.ENGINE_TILE: "tile-resident"}
    out = {
        "workload": w.name, "M": int(w.M), "dtype": f"f{dtype}", "iterations": int(iterations), "n_init": int(n_init),
        "n_cool": int(n_cool), "n_skip": int(n_skip), "beta0": beta0, "f_acc": f_acc, "alpha": alpha,
        "seconds": {"initialisation": t_init, "production": t_prod, "total": t_init + t_prod},
        "iterations_per_s": {"initialisation": n_init / t_init if t_init > 0 else None, "production": n_prod / t_prod if t_prod > 0 else None,
                             "total": iterations / (t_init + t_prod)},
        "engine": {"initialisation": names.get(engine_init), "production": names.get(engine_prod)},
        "samples": int(n_samples), "gpu_launches": int(h.launch_count), "fault": int(h.fault()),
        "mean_step_size": [float(v) for v in ws.mean(axis=0)],
        "param_mean": [float(v) for v in mp[0]], "param_sd": [float(max(v, 0.0)) ** 0.5 for v in mp[1]],
        "param_true": [float(v) for v in w.p_true] if getattr(w, "p_true", None) is not None else None,
        "param_start": [float(v) for v in w.p0[0]],
        "accepted": [int(v) for v in st[0]], "proposed": [int(v) for v in st[1]],
    }
    h.close()
    return out


def main(argv=None):
    ap = argparse.ArgumentParser(description=__doc__.split("\n")[0])
    ap.add_argument("--iterations", type=int, default=1_000_000)
    ap.add_argument("--n-init", type=int, default=None)
    ap.add_argument("--n-cool", type=int, default=None)
    ap.add_argument("--n-skip", type=int, default=400)
    ap.add_argument("--dtype", type=int, default=64, choices=(64, 32))
    ap.add_argument("--M", type=int, default=None)
    ap.add_argument("--seed", type=int, default=1103)
    a = ap.parse_args(argv)
    print(json.dumps(run(a.iterations, a.n_init, a.n_cool, a.n_skip, seed=a.seed, dtype=a.dtype, M=a.M)))


if __name__ == "__main__":
    main()
