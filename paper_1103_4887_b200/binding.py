"""Thin ctypes binding over libpimc.so -- argument marshalling only; every step of the path runs in the
CUDA kernels behind the C ABI of include/pimc.h.  PyTorch supplies device memory and the stream."""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

MODEL_LINEAR, MODEL_HH, MODEL_HH_CLASSIC = 0, 1, 2
PROPOSAL_GAUSSIAN, PROPOSAL_UNIFORM = 0, 1
ENGINE_AUTO, ENGINE_GLOBAL, ENGINE_TILE, ENGINE_TILE_MC = 0, 1, 2, 3
DISC_RK4MAP, DISC_TRAPEZOID = 0, 1
UPDATE_JOINT, UPDATE_COMPONENTWISE = 0, 1

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libpimc.so")
_lib = None

_vp, _dp, _u64p, _u8p, _ip, _u32p = (C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_uint64), C.c_void_p,
                                     C.POINTER(C.c_int), C.c_void_p)
_SIGNATURES = {
    "pimc_model_np": (C.c_int, [C.c_int, C.c_int]),
    "pimc_workspace_bytes": (C.c_size_t, [C.c_int] * 6),
    "pimc_init": (C.c_int, [C.POINTER(C.c_void_p), C.c_int, C.c_int, C.c_int, C.c_int, C.c_double, C.c_double, _dp, _dp,
                            C.c_int, C.c_int, _vp, C.c_size_t, _vp]),
    "pimc_set_data": (C.c_int, [_vp, _vp, _vp]),
    "pimc_set_path": (C.c_int, [_vp, _vp]),
    "pimc_set_params": (C.c_int, [_vp, _vp]),
    "pimc_get_path": (C.c_int, [_vp, _vp, _vp]),
    "pimc_get_cache": (C.c_int, [_vp, _vp]),
    "pimc_set_proposal": (C.c_int, [_vp, _dp, _dp, C.c_int]),
    "pimc_set_bounds": (C.c_int, [_vp, _dp, _dp]),
    "pimc_set_accum": (C.c_int, [_vp, C.c_int, C.c_longlong]),
    "pimc_reset_moments": (C.c_int, [_vp]),
    "pimc_sweep": (C.c_int, [_vp, C.c_longlong, C.c_ulonglong]),
    "pimc_sweep_states_only": (C.c_int, [_vp, C.c_longlong, C.c_ulonglong]),
    "pimc_sweep_params_only": (C.c_int, [_vp, C.c_longlong, C.c_ulonglong]),
    "pimc_moments": (C.c_int, [_vp, _vp, _u64p]),
    "pimc_stats": (C.c_int, [_vp, _vp]),
    "pimc_hist_config": (C.c_int, [_vp, C.c_int, _ip, _ip, _dp, _dp, C.c_int]),
    "pimc_hist": (C.c_int, [_vp, _vp]),
    "pimc_debug_trace": (C.c_int, [_vp, _vp, _vp, _vp, _vp, _vp, _vp]),
    "pimc_set_launch": (C.c_int, [_vp, C.c_int, C.c_int]),
    "pimc_get_launch": (C.c_int, [_vp, _ip, _ip, _ip, _ip]),
    "pimc_set_engine": (C.c_int, [_vp, C.c_int, C.c_int]),
    "pimc_set_discretisation": (C.c_int, [_vp, C.c_int]),
    "pimc_set_update_mode": (C.c_int, [_vp, C.c_int]),
    "pimc_set_annealing": (C.c_int, [_vp, C.c_double, C.c_longlong]),
    "pimc_set_tuning": (C.c_int, [_vp, C.c_int, C.c_longlong, C.c_double, C.c_double]),
    "pimc_get_widths": (C.c_int, [_vp, _vp, _vp]),
    "pimc_get_engine": (C.c_int, [_vp, _ip, _ip]),
    "pimc_set_exchange": (C.c_int, [_vp, C.c_int]),
    "pimc_param_trace": (C.c_int, [_vp, _vp, C.c_longlong]),
    "pimc_residuals": (C.c_int, [_vp, _vp, _vp]),
    "pimc_set_residual_stats": (C.c_int, [_vp, _vp]),
    "pimc_residual_stats": (C.c_int, [_vp, _vp]),
    "pimc_fault": (C.c_int, [_vp, _ip]),
    "pimc_sweep_index": (C.c_ulonglong, [_vp]),
    "pimc_set_sweep_index": (C.c_int, [_vp, C.c_ulonglong]),
    "pimc_launch_count": (C.c_ulonglong, [_vp]),
    "pimc_run_host": (C.c_int, [C.c_int, C.c_int, C.c_int, C.c_int, C.c_double, C.c_double, _dp, C.c_int, C.c_int, _vp, _vp, _vp,
                                _vp, _dp, _dp, _dp, _dp, C.c_int, C.c_longlong, C.c_longlong, C.c_ulonglong, _dp, _vp, _vp]),
    "pimc_run_host_workspace_bytes": (C.c_size_t, [C.c_int] * 6),
    "pimc_run_host_ws": (C.c_int, [C.c_int, C.c_int, C.c_int, C.c_int, C.c_double, C.c_double, _dp, C.c_int, C.c_int, _vp, _vp, _vp,
                                   _vp, _dp, _dp, _dp, _dp, C.c_int, C.c_longlong, C.c_longlong, C.c_ulonglong, _dp, _vp, _vp, _vp, C.c_size_t]),
    "pimc_latency_selftest": (C.c_int, [C.c_int, C.c_int, _dp, C.c_int]),
    "pimc_static_scratch_bytes": (C.c_size_t, []),
    "pimc_run_host_static": (C.c_int, [C.c_int, C.c_int, C.c_int, C.c_int, C.c_double, C.c_double, _dp, C.c_int, C.c_int, _vp, _vp, _vp,
                                       _vp, _dp, _dp, _dp, _dp, C.c_int, C.c_longlong, C.c_longlong, C.c_ulonglong, _dp, _vp, _vp]),
    "pimc_rng_selftest": (C.c_int, [_vp, C.c_ulonglong, C.c_uint, C.c_uint, _vp, _vp, _vp, _vp, _vp]),
    "pimc_step_selftest": (C.c_int, [C.c_int, C.c_int, C.c_int, _vp, _vp, _vp, _vp, C.c_double, C.c_ulonglong, _vp, _vp]),
    "pimc_math_selftest": (C.c_int, [_vp, C.c_ulonglong, _vp, _vp]),
    "pimc_fp64_peak_selftest": (C.c_int, [C.c_int, _dp]),
    "pimc_exchange_selftest": (C.c_int, [C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, _dp, _dp, _ip]),
    "pimc_last_error": (C.c_char_p, [_vp]),
    "pimc_destroy": (C.c_int, [_vp]),
}


class PimcError(RuntimeError):
    pass


def library_path() -> str:
    return _LIB_PATH


def exported_symbols():
    return sorted(_SIGNATURES)


def lib():
    """Load libpimc.so (built in-tree by paper_1103_4887_b200.build).  Fails loudly if it is missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(_LIB_PATH):
            raise PimcError(f"{_LIB_PATH} is missing: run `python -m paper_1103_4887_b200.build` (there is no fallback path)")
        L = C.CDLL(_LIB_PATH)
        for name, (res, args) in _SIGNATURES.items():
            f = getattr(L, name)
            f.restype, f.argtypes = res, args
        _lib = L
    return _lib


def model_np(model: int, D: int) -> int:
    return lib().pimc_model_np(model, D)


def _hd(a):
    """host double array -> ctypes pointer (keeps a reference on the returned tuple)."""
    if a is None:
        return None, None
    arr = np.ascontiguousarray(a, dtype=np.float64)
    return arr, arr.ctypes.data_as(_dp)


def _check(rc, h=None):
    if rc != 0:
        msg = lib().pimc_last_error(h)
        raise PimcError(f"libpimc error {rc}: {msg.decode() if msg else ''}")


def _ptr(t):
    return None if t is None else C.c_void_p(t.data_ptr())


class Pimc:
    """One handle = n_chains independent Markov chains of the same shape, resident on the current CUDA device.

    Stream contract: the handle is bound for life to ONE stream -- `stream` if given, else the torch stream that is current
    when the handle is created (include/pimc.h "Conventions").  Every call of this class enqueues on that stream, whatever
    torch stream is current at the time; tensors produced or consumed under another stream must be ordered against it by the
    caller (`handle.stream.wait_stream(other)` / `other.wait_stream(handle.stream)`)."""

    def __init__(self, model, D, L, M, dt, Rm, Rf, p0, n_chains=1, dtype=64, stream=None):
        import torch
        if not torch.cuda.is_available():
            raise PimcError("no CUDA device: libpimc has no CPU fallback")
        self.torch = torch
        self.model, self.D, self.L, self.M, self.C, self.dtype = model, D, L, M, n_chains, dtype
        self.Np = model_np(model, D)
        self.tdtype = torch.float64 if dtype == 64 else torch.float32
        self.device = torch.device("cuda", torch.cuda.current_device())
        nbytes = lib().pimc_workspace_bytes(model, D, L, M, n_chains, dtype)
        if nbytes == 0:
            raise PimcError("bad or unsupported problem shape")
        self._ws = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
        off = (-self._ws.data_ptr()) % 256
        self._stream = stream if stream is not None else torch.cuda.current_stream()
        _rf, rf = _hd(Rf)
        _p0, pp = _hd(np.asarray(p0, dtype=np.float64).reshape(-1))
        assert _rf.size == D and _p0.size == n_chains * self.Np
        h = C.c_void_p()
        _check(lib().pimc_init(C.byref(h), model, D, L, M, float(dt), float(Rm), rf, pp, n_chains, dtype,
                               C.c_void_p(self._ws.data_ptr() + off), nbytes, C.c_void_p(self._stream.cuda_stream)))
        self._h = h
        self._keep = {}

    @property
    def stream(self):
        """The torch stream all of this handle's work is enqueued on."""
        return self._stream

    @classmethod
    def from_workload(cls, w, dtype=64, with_params=True, device_arrays=None):
        """Build a handle from a workloads.Workload and load its data, widths, bounds and initial path."""
        import torch
        o = cls(w.model, w.D, w.L, w.M, w.dt, w.Rm, w.Rf, w.p0, n_chains=w.n_chains, dtype=dtype)
        td = o.tdtype
        y = torch.as_tensor(np.ascontiguousarray(w.y), dtype=td).to(o.device).contiguous()
        I = None if w.I is None else torch.as_tensor(np.ascontiguousarray(w.I), dtype=td).to(o.device).contiguous()
        x0 = torch.as_tensor(np.ascontiguousarray(w.x0), dtype=td).to(o.device).contiguous()
        o.set_data(y, I)
        o.set_proposal(w.w_state, w.w_param if with_params else None)
        o.set_bounds(w.lo, w.hi)
        o.set_path(x0)
        return o

    def close(self):
        if getattr(self, "_h", None):
            lib().pimc_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- setters ----
    def _dev(self, t, shape):
        assert t.is_cuda and t.dtype == self.tdtype and t.is_contiguous(), "need a contiguous CUDA tensor of the handle's dtype"
        assert t.numel() == int(np.prod(shape)), (tuple(t.shape), shape)
        return t

    def set_data(self, y, I=None):
        y = self._dev(y, (self.C, self.M + 1, self.L))
        if I is not None:
            I = self._dev(I, (self.C, self.M + 1))
        _check(lib().pimc_set_data(self._h, _ptr(y), _ptr(I)), self._h)

    def set_path(self, x):
        _check(lib().pimc_set_path(self._h, _ptr(self._dev(x, (self.C, self.M + 1, self.D)))), self._h)

    def set_params(self, p):
        _check(lib().pimc_set_params(self._h, _ptr(self._dev(p, (self.C, self.Np)))), self._h)

    def set_proposal(self, w_state, w_param=None, kind=PROPOSAL_GAUSSIAN):
        a, pa = _hd(w_state)
        b, pb = _hd(w_param)
        assert a.size == self.D and (b is None or b.size == self.Np)
        _check(lib().pimc_set_proposal(self._h, pa, pb, kind), self._h)

    def set_bounds(self, lo, hi):
        a, pa = _hd(lo)
        b, pb = _hd(hi)
        assert a.size == self.C * self.Np and b.size == self.C * self.Np
        _check(lib().pimc_set_bounds(self._h, pa, pb), self._h)

    def set_accum(self, enabled, n_skip=1):
        _check(lib().pimc_set_accum(self._h, int(enabled), int(n_skip)), self._h)

    def reset_moments(self):
        _check(lib().pimc_reset_moments(self._h), self._h)

    def set_launch(self, ctas_per_chain=0, threads_per_cta=0):
        _check(lib().pimc_set_launch(self._h, ctas_per_chain, threads_per_cta), self._h)

    def get_launch(self):
        v = [C.c_int() for _ in range(4)]
        _check(lib().pimc_get_launch(self._h, *[C.byref(q) for q in v]), self._h)
        return dict(ctas_per_chain=v[0].value, threads_per_cta=v[1].value, tile_sites=v[2].value, smem_bytes=v[3].value)

    def set_engine(self, engine=ENGINE_AUTO, halo=-1):
        _check(lib().pimc_set_engine(self._h, int(engine), int(halo)), self._h)

    def get_engine(self):
        e, hh = C.c_int(), C.c_int()
        _check(lib().pimc_get_engine(self._h, C.byref(e), C.byref(hh)), self._h)
        return dict(engine=e.value, halo=hh.value)

    def param_trace(self, capacity):
        """Record the parameters at every accumulated sweep (Fig. 4) -> device tensor (C, capacity, Np); 0 = off."""
        if not capacity:
            _check(lib().pimc_param_trace(self._h, None, 0), self._h)
            self._keep.pop("ptrace", None)
            return None
        buf = self.torch.full((self.C, int(capacity), self.Np), float("nan"), dtype=self.tdtype, device=self.device)
        self.torch.cuda.current_stream().synchronize()
        _check(lib().pimc_param_trace(self._h, _ptr(buf), int(capacity)), self._h)
        self._keep["ptrace"] = buf
        return buf

    def residuals(self):
        """Model errors eps (C, M, D) and observation errors delta (C, M+1, L) of the current path."""
        eps = self.torch.empty((self.C, self.M, self.D), dtype=self.tdtype, device=self.device)
        delta = self.torch.empty((self.C, self.M + 1, self.L), dtype=self.tdtype, device=self.device)
        _check(lib().pimc_residuals(self._h, _ptr(eps), _ptr(delta)), self._h)
        return eps, delta

    def set_residual_stats(self, enabled=True):
        if not enabled:
            _check(lib().pimc_set_residual_stats(self._h, None), self._h)
            self._keep.pop("resid", None)
            return
        n = 2 * self.M * self.D + 2 * (self.M + 1) * self.L
        buf = self.torch.zeros((self.C, n), dtype=self.torch.float64, device=self.device)
        self.torch.cuda.current_stream().synchronize()
        _check(lib().pimc_set_residual_stats(self._h, _ptr(buf)), self._h)
        self._keep["resid"] = buf

    def residual_stats(self):
        """(mean eps, var eps) (C, M, D), (mean delta, var delta) (C, M+1, L) over the accumulated sweeps."""
        ne, nd = self.M * self.D, (self.M + 1) * self.L
        out = self.torch.empty((self.C, 2 * ne + 2 * nd), dtype=self.torch.float64, device=self.device)
        _check(lib().pimc_residual_stats(self._h, _ptr(out)), self._h)
        sh_e, sh_d = (self.C, self.M, self.D), (self.C, self.M + 1, self.L)
        return (out[:, :ne].reshape(sh_e), out[:, ne:2 * ne].reshape(sh_e), out[:, 2 * ne:2 * ne + nd].reshape(sh_d), out[:, 2 * ne + nd:].reshape(sh_d))

    def set_exchange(self, first_poll_hold_cycles=450):
        _check(lib().pimc_set_exchange(self._h, int(first_poll_hold_cycles)), self._h)

    def fault(self):
        """Synchronise the stream; raises PimcError if an inter-CTA hand-off was lost."""
        f = C.c_int()
        _check(lib().pimc_fault(self._h, C.byref(f)), self._h)
        return f.value

    # ---- the hot path ----
    def sweep(self, n_sweeps, seed, check_fault=False):
        """n_sweeps full sweeps (asynchronous on the handle's stream).  check_fault=True synchronises the stream afterwards and
        raises PimcError if an inter-CTA hand-off was lost (pimc_fault): use it where a hung or torn launch must not pass."""
        _check(lib().pimc_sweep(self._h, int(n_sweeps), int(seed)), self._h)
        if check_fault:
            self.fault()

    def sweep_states_only(self, n_sweeps, seed):
        _check(lib().pimc_sweep_states_only(self._h, int(n_sweeps), int(seed)), self._h)

    def sweep_params_only(self, n_sweeps, seed):
        _check(lib().pimc_sweep_params_only(self._h, int(n_sweeps), int(seed)), self._h)

    # ---- getters (device tensors) ----
    def get_path(self):
        x = self.torch.empty((self.C, self.M + 1, self.D), dtype=self.tdtype, device=self.device)
        p = self.torch.empty((self.C, self.Np), dtype=self.tdtype, device=self.device)
        _check(lib().pimc_get_path(self._h, _ptr(x), _ptr(p)), self._h)
        return x, p

    def get_cache(self):
        rows = self.M + 1 if getattr(self, "disc", DISC_RK4MAP) == DISC_TRAPEZOID else self.M
        g = self.torch.empty((self.C, rows, self.D), dtype=self.tdtype, device=self.device)
        _check(lib().pimc_get_cache(self._h, _ptr(g)), self._h)
        return g

    def set_tuning(self, enabled, n_skip=1, f_acc=0.23, alpha=0.02):
        """Step-size auto-tuning from the current sweep on (both engines); enabled=False freezes the step sizes."""
        _check(lib().pimc_set_tuning(self._h, int(bool(enabled)), int(n_skip), float(f_acc), float(alpha)), self._h)

    def get_widths(self):
        t = self.torch
        ws = t.empty((self.C, self.M + 1, self.D), dtype=t.float64, device=self.device)
        wp = t.empty((self.C, max(self.Np, 1)), dtype=t.float64, device=self.device)
        _check(lib().pimc_get_widths(self._h, _ptr(ws), _ptr(wp) if self.Np else None), self._h)
        return ws, wp[:, :self.Np]

    def set_annealing(self, beta0, n_cool):
        """Anneal the dynamics term from the current sweep on (Eq. 10); n_cool = 0 switches it off."""
        _check(lib().pimc_set_annealing(self._h, float(beta0), int(n_cool)), self._h)

    def set_update_mode(self, mode):
        """UPDATE_JOINT (default) or UPDATE_COMPONENTWISE (D decisions per site; both engines).  Re-enable the trace afterwards:
        its dA / acc buffers are per (site, component) in component-wise mode."""
        _check(lib().pimc_set_update_mode(self._h, int(mode)), self._h)
        self.update_mode = int(mode)

    def set_discretisation(self, disc):
        """DISC_RK4MAP (default) or DISC_TRAPEZOID (the paper's rule, Eq. 7; both engines)."""
        _check(lib().pimc_set_discretisation(self._h, int(disc)), self._h)
        self.disc = int(disc)

    def moments(self):
        """-> (mean_x, var_x) each (C, M+1, D); (mean_p, var_p) each (C, Np); n_samples."""
        nx = (self.M + 1) * self.D
        out = self.torch.empty((self.C, 2 * nx + 2 * self.Np), dtype=self.torch.float64, device=self.device)
        n = C.c_uint64()
        _check(lib().pimc_moments(self._h, _ptr(out), C.byref(n)), self._h)
        mx = out[:, : 2 * nx].reshape(self.C, 2, self.M + 1, self.D)
        mp = out[:, 2 * nx:].reshape(self.C, 2, self.Np)
        return mx, mp, n.value

    def stats(self):
        out = self.torch.zeros((self.C, 2, self.D + self.Np), dtype=self.torch.int64, device=self.device)
        _check(lib().pimc_stats(self._h, _ptr(out)), self._h)
        return out

    def hist_config(self, site, comp, lo, hi, nbins):
        s = np.ascontiguousarray(site, dtype=np.int32)
        c = np.ascontiguousarray(comp, dtype=np.int32)
        a, pa = _hd(lo)
        b, pb = _hd(hi)
        self._hist_shape = (self.C, s.size, nbins + 2)
        _check(lib().pimc_hist_config(self._h, s.size, s.ctypes.data_as(_ip), c.ctypes.data_as(_ip), pa, pb, nbins), self._h)

    def hist(self):
        out = self.torch.zeros(self._hist_shape, dtype=self.torch.int64, device=self.device)
        _check(lib().pimc_hist(self._h, _ptr(out)), self._h)
        return out

    def enable_trace(self, params=True, xprop=True):
        t = self.torch
        sh = (self.C, self.M + 1, self.D) if getattr(self, "update_mode", UPDATE_JOINT) == UPDATE_COMPONENTWISE else (self.C, self.M + 1)
        tr = dict(dA=t.zeros(sh, dtype=self.tdtype, device=self.device),
                  acc=t.zeros(sh, dtype=t.uint8, device=self.device),
                  xprop=t.zeros((self.C, self.M + 1, self.D), dtype=self.tdtype, device=self.device) if xprop else None,
                  dAp=t.zeros((self.C, self.Np), dtype=self.tdtype, device=self.device) if params else None,
                  accp=t.zeros((self.C, self.Np), dtype=t.uint8, device=self.device) if params else None,
                  pprop=t.zeros((self.C, self.Np), dtype=self.tdtype, device=self.device) if params else None)
        self._keep["trace"] = tr
        _check(lib().pimc_debug_trace(self._h, _ptr(tr["dA"]), _ptr(tr["acc"]), _ptr(tr["xprop"]), _ptr(tr["dAp"]), _ptr(tr["accp"]),
                                      _ptr(tr["pprop"])), self._h)
        return tr

    def disable_trace(self):
        self._keep.pop("trace", None)
        _check(lib().pimc_debug_trace(self._h, None, None, None, None, None, None), self._h)

    @property
    def sweep_index(self):
        return lib().pimc_sweep_index(self._h)

    @sweep_index.setter
    def sweep_index(self, t):
        _check(lib().pimc_set_sweep_index(self._h, int(t)), self._h)

    @property
    def launch_count(self):
        return lib().pimc_launch_count(self._h)


def rng_selftest(ctrs, key):
    """ctrs: CUDA int32/uint32-compatible tensor (n,4) holding the counter words -> dict of device tensors."""
    import torch
    assert ctrs.is_cuda and ctrs.dtype == torch.int32 and ctrs.is_contiguous() and ctrs.shape[1] == 4
    n = ctrs.shape[0]
    out = torch.empty((n, 4), dtype=torch.int32, device=ctrs.device)
    u_prop = torch.empty((n, 4), dtype=torch.float64, device=ctrs.device)
    u_acc = torch.empty((n,), dtype=torch.float64, device=ctrs.device)
    z = torch.empty((n, 4), dtype=torch.float64, device=ctrs.device)
    _check(lib().pimc_rng_selftest(_ptr(ctrs), n, int(key[0]), int(key[1]), _ptr(out), _ptr(u_prop), _ptr(u_acc), _ptr(z),
                                   C.c_void_p(torch.cuda.current_stream().cuda_stream)))
    return dict(words=out, u_prop=u_prop, u_acc=u_acc, z=z)


def step_selftest(model, x, p, I0, I1, dt):
    import torch
    assert x.is_cuda and x.is_contiguous() and p.is_cuda
    dtype = 64 if x.dtype == torch.float64 else 32
    n, D = x.shape
    g = torch.empty_like(x)
    _check(lib().pimc_step_selftest(model, D, dtype, _ptr(x), _ptr(p), _ptr(I0), _ptr(I1), float(dt), n, _ptr(g),
                                    C.c_void_p(torch.cuda.current_stream().cuda_stream)))
    return g


def math_selftest(x):
    """x: CUDA float64 tensor (n,) -> (n,9): exp, log|x|, sqrt|x|, sin, cos, 1/|x|, HH gate rates m, h, n (kernel math)."""
    import torch
    assert x.is_cuda and x.dtype == torch.float64 and x.is_contiguous()
    out = torch.empty((x.numel(), 9), dtype=torch.float64, device=x.device)
    _check(lib().pimc_math_selftest(_ptr(x), x.numel(), _ptr(out), C.c_void_p(torch.cuda.current_stream().cuda_stream)))
    return out


def fp64_peak(millis=200):
    """Measured sustained FP64 FMA rate of this device in lane-FMA/s (roofline denominator probe)."""
    v = C.c_double()
    _check(lib().pimc_fp64_peak_selftest(int(millis), C.byref(v)))
    return v.value


def exchange_selftest(mode, n_ctas=0, threads=256, rounds=2000, work=0):
    """Grid-wide all-reduce probe (pimc_exchange_selftest) -> dict(cycles_per_round, max_abs_err, n_distinct)."""
    cyc, err, nd = C.c_double(), C.c_double(), C.c_int()
    _check(lib().pimc_exchange_selftest(int(mode), int(n_ctas), int(threads), int(rounds), int(work), C.byref(cyc), C.byref(err), C.byref(nd)))
    return dict(cycles_per_round=cyc.value, max_abs_err=err.value, n_distinct=nd.value)


def latency_selftest(what, arg=0):
    """pimc_latency_selftest: what = 0 -> dict of the L2-hit map (near / far ticks, SM groups); 1..5 -> one-way ticks of a packet;
    6 -> one-way ticks over many line addresses for a same-die and a cross-die pair of CTAs."""
    out = (C.c_double * 5)()
    _check(lib().pimc_latency_selftest(int(what), int(arg), out, 5))
    if what == 0:
        return dict(near=out[0], far=out[1], group_a=int(out[2]), group_b=int(out[3]), frac_near=out[4])
    if what == 6:
        return dict(same_min=out[0], same_max=out[1], cross_min=out[2], cross_max=out[3], frac_fast=out[4])
    return out[0]


def run_host_scratch(w, dtype=64):
    """A device scratch tensor for run_host(..., scratch=...) (pimc_run_host_workspace_bytes), so repeated calls skip cudaMalloc."""
    import torch
    n = lib().pimc_run_host_workspace_bytes(w.model, w.D, w.L, w.M, w.n_chains, dtype)
    t = torch.empty(n + 256, dtype=torch.uint8, device="cuda")
    return t


def static_scratch_bytes():
    """Size of the library's static device scratch array (pimc_static_scratch_bytes): the limit of run_host(..., static=True)."""
    return int(lib().pimc_static_scratch_bytes())


def run_host(w, n_burn, n_sweeps, seed, dtype=64, kind=PROPOSAL_GAUSSIAN, want_path=False, scratch=None, static=False):
    """End-to-end call on HOST numpy buffers (pimc_run_host / pimc_run_host_ws): H2D, sweeps, moments, D2H inside the call.
    static=True: pimc_run_host_static -- all device memory from the library's static array, no cudaMalloc anywhere."""
    npd = np.float64 if dtype == 64 else np.float32
    y = np.ascontiguousarray(w.y, dtype=npd)
    I = None if w.I is None else np.ascontiguousarray(w.I, dtype=npd)
    x0 = np.ascontiguousarray(w.x0, dtype=npd)
    p0 = np.ascontiguousarray(w.p0, dtype=npd)
    _rf, rf = _hd(w.Rf)
    _ws, ws = _hd(w.w_state)
    _wp, wp = _hd(w.w_param)
    _lo, lo = _hd(w.lo)
    _hi, hi = _hd(w.hi)
    nx = (w.M + 1) * w.D
    mom = np.empty((w.n_chains, 2 * nx + 2 * w.Np), dtype=np.float64)
    xo = np.empty_like(x0) if want_path else None
    po = np.empty_like(p0) if want_path else None
    vp = lambda a: None if a is None else C.c_void_p(a.ctypes.data)
    sp, sn = None, 0
    if scratch is not None:
        off = (-scratch.data_ptr()) % 256
        sp, sn = C.c_void_p(scratch.data_ptr() + off), scratch.numel() - off
    if static:
        _check(lib().pimc_run_host_static(w.model, w.D, w.L, w.M, float(w.dt), float(w.Rm), rf, w.n_chains, dtype, vp(y), vp(I), vp(x0), vp(p0),
                                          ws, wp, lo, hi, kind, int(n_burn), int(n_sweeps), int(seed), mom.ctypes.data_as(_dp), vp(xo), vp(po)))
    else:
        _check(lib().pimc_run_host_ws(w.model, w.D, w.L, w.M, float(w.dt), float(w.Rm), rf, w.n_chains, dtype, vp(y), vp(I), vp(x0), vp(p0),
                                      ws, wp, lo, hi, kind, int(n_burn), int(n_sweeps), int(seed), mom.ctypes.data_as(_dp), vp(xo), vp(po),
                                      sp, sn))
    mx = mom[:, : 2 * nx].reshape(w.n_chains, 2, w.M + 1, w.D)
    mp = mom[:, 2 * nx:].reshape(w.n_chains, 2, w.Np)
    bytes_in = y.nbytes + (0 if I is None else I.nbytes) + x0.nbytes + p0.nbytes
    bytes_out = mom.nbytes + (0 if xo is None else xo.nbytes + po.nbytes)
    return dict(mean_x=mx[:, 0], var_x=mx[:, 1], mean_p=mp[:, 0], var_p=mp[:, 1], x=xo, p=po, h2d_bytes=bytes_in, d2h_bytes=bytes_out)
