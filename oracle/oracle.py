"""ctypes wrapper around oracle/pimc_oracle.cpp -- TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
import this.  It never imports the CUDA package.
"""
from __future__ import annotations

import ctypes as C

import numpy as np

from . import build as _build

_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build.build())
        dp, u32p, u64p, u8p, ip = (C.POINTER(C.c_double), C.POINTER(C.c_uint32), C.POINTER(C.c_uint64),
                                   C.POINTER(C.c_uint8), C.POINTER(C.c_int))
        sig = {
            "orc_philox4x32_10": (None, [u32p, u32p, u32p]),
            "orc_philox_bulk": (None, [C.c_uint64, u32p, u32p, u32p]),
            "orc_draw_words": (None, [C.c_uint64, C.c_uint64, C.c_uint32, C.c_uint32, C.c_uint32, C.c_uint32, u32p]),
            "orc_u01_from_word": (C.c_double, [C.c_uint32]),
            "orc_u01_from_two_words": (C.c_double, [C.c_uint32, C.c_uint32]),
            "orc_u01f_from_word": (C.c_float, [C.c_uint32]),
            "orc_box_muller": (None, [C.c_double, C.c_double, dp]),
            "orc_model_np": (C.c_int, [C.c_int, C.c_int]),
            "orc_rhs": (None, [C.c_int, dp, dp, C.c_double, dp]),
            "orc_step_increment": (None, [C.c_int, C.c_int, dp, dp, C.c_double, C.c_double, C.c_double, dp]),
            "orc_create": (C.c_void_p, [C.c_int, C.c_int, C.c_int, C.c_int, C.c_double, C.c_double, dp, dp, C.c_int, C.c_uint32]),
            "orc_destroy": (None, [C.c_void_p]),
            "orc_set_data": (None, [C.c_void_p, dp, dp]),
            "orc_set_path": (None, [C.c_void_p, dp]),
            "orc_set_params": (None, [C.c_void_p, dp]),
            "orc_get_path": (None, [C.c_void_p, dp, dp]),
            "orc_get_cache": (None, [C.c_void_p, dp]),
            "orc_set_proposal": (None, [C.c_void_p, dp, dp, C.c_int]),
            "orc_set_bounds": (None, [C.c_void_p, dp, dp]),
            "orc_set_accum": (None, [C.c_void_p, C.c_int, C.c_uint64]),
            "orc_reset_moments": (None, [C.c_void_p]),
            "orc_sweep_index": (C.c_uint64, [C.c_void_p]),
            "orc_set_sweep_index": (None, [C.c_void_p, C.c_uint64]),
            "orc_hist_config": (C.c_int, [C.c_void_p, C.c_int, ip, ip, dp, dp, C.c_int]),
            "orc_hist": (None, [C.c_void_p, u64p]),
            "orc_sweep": (C.c_int, [C.c_void_p, C.c_uint64, C.c_uint64, C.c_int, C.c_int]),
            "orc_moments": (C.c_uint64, [C.c_void_p, dp]),
            "orc_stats": (None, [C.c_void_p, u64p]),
            "orc_trace": (None, [C.c_void_p, dp, dp, dp, u8p, dp, dp, dp, dp, u8p, dp]),
            "orc_site_delta_A": (C.c_double, [C.c_void_p, C.c_int, dp, dp]),
            "orc_param_delta_A": (C.c_double, [C.c_void_p, C.c_int, C.c_double, dp]),
            "orc_full_action": (None, [C.c_void_p, dp, dp, dp, dp]),
            "orc_cache_len": (C.c_int, [C.c_void_p]),
            "orc_set_update_mode": (C.c_int, [C.c_void_p, C.c_int]),
            "orc_set_annealing": (C.c_int, [C.c_void_p, C.c_double, C.c_uint64]),
            "orc_set_tuning": (C.c_int, [C.c_void_p, C.c_int, C.c_uint64, C.c_double, C.c_double]),
            "orc_get_widths": (None, [C.c_void_p, dp, dp]),
            "orc_annealing_beta": (C.c_double, [C.c_void_p]),
            "orc_set_discretisation": (C.c_int, [C.c_void_p, C.c_int]),
            "orc_param_trace_enable": (None, [C.c_void_p, C.c_int]),
            "orc_param_trace": (C.c_uint64, [C.c_void_p, dp, C.c_uint64]),
            "orc_residuals": (None, [C.c_void_p, dp, dp]),
            "orc_residual_stats_enable": (None, [C.c_void_p, C.c_int]),
            "orc_residual_stats": (C.c_uint64, [C.c_void_p, dp]),
            "orc_half_rhs": (None, [C.c_int, C.c_int, dp, dp, C.c_double, C.c_double, dp]),
        }
        for name, (res, args) in sig.items():
            f = getattr(L, name)
            f.restype, f.argtypes = res, args
        _lib = L
    return _lib


def _dp(a):
    return None if a is None else a.ctypes.data_as(C.POINTER(C.c_double))


def _f64(a):
    return None if a is None else np.ascontiguousarray(a, dtype=np.float64)


def philox4x32_10(ctr, key):
    c = np.ascontiguousarray(ctr, dtype=np.uint32)
    k = np.ascontiguousarray(key, dtype=np.uint32)
    o = np.empty(4, np.uint32)
    u32p = C.POINTER(C.c_uint32)
    lib().orc_philox4x32_10(c.ctypes.data_as(u32p), k.ctypes.data_as(u32p), o.ctypes.data_as(u32p))
    return o


def philox_bulk(ctrs, key):
    c = np.ascontiguousarray(ctrs, dtype=np.uint32).reshape(-1, 4)
    k = np.ascontiguousarray(key, dtype=np.uint32)
    o = np.empty_like(c)
    u32p = C.POINTER(C.c_uint32)
    lib().orc_philox_bulk(c.shape[0], c.ctypes.data_as(u32p), k.ctypes.data_as(u32p), o.ctypes.data_as(u32p))
    return o


def draw_words(seed, t, chain, index, stream, block=0):
    o = np.empty(4, np.uint32)
    lib().orc_draw_words(seed, t, chain, index, stream, block, o.ctypes.data_as(C.POINTER(C.c_uint32)))
    return o


def u01_from_word(w):
    return lib().orc_u01_from_word(int(w))


def u01_from_two_words(w0, w1):
    return lib().orc_u01_from_two_words(int(w0), int(w1))


def u01f_from_word(w):
    return lib().orc_u01f_from_word(int(w))


def box_muller(u1, u2):
    z = np.empty(2)
    lib().orc_box_muller(u1, u2, _dp(z))
    return z


def model_np(model, D):
    return lib().orc_model_np(model, D)


def rhs(model, x, p, I):
    x, p = _f64(x), _f64(p)
    F = np.empty_like(x)
    lib().orc_rhs(model, _dp(x), _dp(p), float(I), _dp(F))
    return F


def step_increment(model, x, p, I0, I1, dt):
    x, p = _f64(x), _f64(p)
    g = np.empty_like(x)
    lib().orc_step_increment(model, x.size, _dp(x), _dp(p), float(I0), float(I1), float(dt), _dp(g))
    return g


class OracleChain:
    """One Markov chain of the oracle (serial, fp64)."""

    def __init__(self, model, D, L, M, dt, Rm, Rf, p0, state_dtype=64, chain_id=0):
        self.model, self.D, self.L, self.M = model, D, L, M
        self.Np = model_np(model, D)
        Rf, p0 = _f64(Rf), _f64(p0).reshape(-1)
        assert Rf.size == D and p0.size == self.Np
        self._h = lib().orc_create(model, D, L, M, dt, Rm, _dp(Rf), _dp(p0), state_dtype, chain_id)
        if not self._h:
            raise ValueError("orc_create rejected the arguments")

    @classmethod
    def from_workload(cls, w, chain=0, state_dtype=64, with_params=True):
        o = cls(w.model, w.D, w.L, w.M, w.dt, w.Rm, w.Rf, w.p0[chain], state_dtype, chain)
        o.set_data(w.y[chain], None if w.I is None else w.I[chain])
        o.set_proposal(w.w_state, w.w_param if with_params else None)
        o.set_bounds(w.lo[chain], w.hi[chain])
        o.set_path(w.x0[chain])
        return o

    def __del__(self):
        if getattr(self, "_h", None):
            lib().orc_destroy(self._h)
            self._h = None

    def set_data(self, y, I=None):
        y, I = _f64(y).reshape(-1), (None if I is None else _f64(I).reshape(-1))
        assert y.size == (self.M + 1) * self.L and (I is None or I.size == self.M + 1)
        lib().orc_set_data(self._h, _dp(y), _dp(I))

    def set_path(self, x):
        x = _f64(x).reshape(-1)
        assert x.size == (self.M + 1) * self.D
        lib().orc_set_path(self._h, _dp(x))

    def set_params(self, p):
        p = _f64(p).reshape(-1)
        assert p.size == self.Np
        lib().orc_set_params(self._h, _dp(p))

    def get_path(self):
        x, p = np.empty((self.M + 1, self.D)), np.empty(self.Np)
        lib().orc_get_path(self._h, _dp(x), _dp(p))
        return x, p

    def get_cache(self):
        g = np.empty((lib().orc_cache_len(self._h), self.D))     # M rows (RK4 map) or M + 1 (trapezoid)
        lib().orc_get_cache(self._h, _dp(g))
        return g

    def set_tuning(self, enabled, n_skip=1, f_acc=0.23, alpha=0.02):
        """Step-size auto-tuning from the current sweep on; enabled=False freezes the step sizes."""
        assert lib().orc_set_tuning(self._h, int(bool(enabled)), int(n_skip), float(f_acc), float(alpha)) == 0

    def get_widths(self):
        ws, wp = np.empty((self.M + 1, self.D)), np.empty(self.Np)
        lib().orc_get_widths(self._h, _dp(ws), _dp(wp))
        return ws, wp

    def set_annealing(self, beta0, n_cool):
        """Simulated annealing of the dynamics term from the current sweep on (Eq. 10); n_cool = 0 = off."""
        assert lib().orc_set_annealing(self._h, float(beta0), int(n_cool)) == 0

    def annealing_beta(self):
        return lib().orc_annealing_beta(self._h)

    def set_update_mode(self, mode):
        """0 = joint D-vector proposal per site (default), 1 = component-wise (D decisions per site)."""
        assert lib().orc_set_update_mode(self._h, int(mode)) == 0
        self.update_mode = int(mode)

    def set_discretisation(self, disc):
        """0 = explicit RK4 map (default), 1 = the paper's trapezoid rule (Eq. 7)."""
        assert lib().orc_set_discretisation(self._h, int(disc)) == 0

    def set_proposal(self, w_state, w_param=None, kind=0):
        ws = _f64(w_state).reshape(-1)
        wp = None if w_param is None else _f64(w_param).reshape(-1)
        assert ws.size == self.D and (wp is None or wp.size == self.Np)
        lib().orc_set_proposal(self._h, _dp(ws), _dp(wp), kind)

    def set_bounds(self, lo, hi):
        lo, hi = _f64(lo).reshape(-1), _f64(hi).reshape(-1)
        assert lo.size == self.Np and hi.size == self.Np
        lib().orc_set_bounds(self._h, _dp(lo), _dp(hi))

    def set_accum(self, enabled, n_skip=1):
        lib().orc_set_accum(self._h, int(enabled), n_skip)

    def reset_moments(self):
        lib().orc_reset_moments(self._h)

    @property
    def sweep_index(self):
        return lib().orc_sweep_index(self._h)

    @sweep_index.setter
    def sweep_index(self, t):
        lib().orc_set_sweep_index(self._h, int(t))

    def hist_config(self, site, comp, lo, hi, nbins):
        site = np.ascontiguousarray(site, dtype=np.int32)
        comp = np.ascontiguousarray(comp, dtype=np.int32)
        lo, hi = _f64(lo), _f64(hi)
        ip = C.POINTER(C.c_int)
        self._hist_shape = (site.size, nbins + 2)
        lib().orc_hist_config(self._h, site.size, site.ctypes.data_as(ip), comp.ctypes.data_as(ip), _dp(lo), _dp(hi), nbins)

    def hist(self):
        out = np.zeros(self._hist_shape, np.uint64)
        lib().orc_hist(self._h, out.ctypes.data_as(C.POINTER(C.c_uint64)))
        return out

    def sweep(self, n_sweeps, seed, order=0, do_params=True):
        rc = lib().orc_sweep(self._h, int(n_sweeps), int(seed), order, int(do_params))
        if rc != 0:
            raise RuntimeError(f"orc_sweep failed: {rc}")

    def moments(self):
        nx = (self.M + 1) * self.D
        out = np.empty(2 * nx + 2 * self.Np)
        n = lib().orc_moments(self._h, _dp(out))
        mx = out[: 2 * nx].reshape(2, self.M + 1, self.D)
        mp = out[2 * nx:].reshape(2, self.Np)
        return mx, mp, n

    def param_trace_enable(self, on=True):
        """Record the parameters at every accumulated sweep (Fig. 4); cleared by reset_moments()."""
        lib().orc_param_trace_enable(self._h, int(bool(on)))

    def param_trace(self):
        n = lib().orc_param_trace(self._h, None, 0)
        out = np.empty((n, self.Np))
        lib().orc_param_trace(self._h, _dp(out), n)
        return out

    def residuals(self):
        """Model errors eps (M, D) and observation errors delta (M+1, L) of the current path."""
        eps, delta = np.empty((self.M, self.D)), np.empty((self.M + 1, max(self.L, 1)))[:, : self.L].copy()
        lib().orc_residuals(self._h, _dp(eps), _dp(delta))
        return eps, delta

    def residual_stats_enable(self, on=True):
        lib().orc_residual_stats_enable(self._h, int(bool(on)))

    def residual_stats(self):
        """(mean eps, var eps) (M, D) each, (mean delta, var delta) (M+1, L) each, sample count."""
        ne, nd = self.M * self.D, (self.M + 1) * self.L
        out = np.empty(2 * ne + 2 * nd)
        n = lib().orc_residual_stats(self._h, _dp(out))
        return (out[:ne].reshape(self.M, self.D), out[ne:2 * ne].reshape(self.M, self.D),
                out[2 * ne:2 * ne + nd].reshape(self.M + 1, self.L), out[2 * ne + nd:].reshape(self.M + 1, self.L), n)

    def stats(self):
        out = np.zeros((2, self.D + self.Np), np.uint64)
        lib().orc_stats(self._h, out.ctypes.data_as(C.POINTER(C.c_uint64)))
        return out

    def trace(self):
        M, D, Np = self.M, self.D, self.Np
        sh = (M + 1, D) if getattr(self, "update_mode", 0) == 1 else (M + 1,)       # per (site, component) or per site
        t = dict(dA=np.empty(sh), S=np.empty(sh), logu=np.empty(sh), acc=np.empty(sh, np.uint8),
                 xprop=np.empty((M + 1, D)), dAp=np.empty(Np), Sp=np.empty(Np), logup=np.empty(Np),
                 accp=np.empty(Np, np.uint8), pprop=np.empty(Np))
        u8 = C.POINTER(C.c_uint8)
        lib().orc_trace(self._h, _dp(t["dA"]), _dp(t["S"]), _dp(t["logu"]), t["acc"].ctypes.data_as(u8), _dp(t["xprop"]),
                        _dp(t["dAp"]), _dp(t["Sp"]), _dp(t["logup"]), t["accp"].ctypes.data_as(u8), _dp(t["pprop"]))
        return t

    def site_delta_A(self, n, xp):
        xp = _f64(xp).reshape(-1)
        S = C.c_double()
        dA = lib().orc_site_delta_A(self._h, int(n), _dp(xp), C.cast(C.byref(S), C.POINTER(C.c_double)))
        return dA, S.value

    def param_delta_A(self, l, pl):
        S = C.c_double()
        dA = lib().orc_param_delta_A(self._h, int(l), float(pl), C.cast(C.byref(S), C.POINTER(C.c_double)))
        return dA, S.value

    def full_action(self, x=None, p=None):
        """Full action in long double, returned as (hi, lo) doubles; sum them in np.longdouble."""
        x = None if x is None else _f64(x).reshape(-1)
        p = None if p is None else _f64(p).reshape(-1)
        hi, lo = C.c_double(), C.c_double()
        dpt = C.POINTER(C.c_double)
        lib().orc_full_action(self._h, _dp(x), _dp(p), C.cast(C.byref(hi), dpt), C.cast(C.byref(lo), dpt))
        return np.longdouble(hi.value) + np.longdouble(lo.value)
