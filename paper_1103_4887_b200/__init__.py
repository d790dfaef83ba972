"""pimc-b200: B200-native (sm_100a) path-integral Monte Carlo data assimilation (arXiv 1103.4887).

The product is ``libpimc.so`` (C ABI in ``include/pimc.h``); this package is the thin Python binding.
There is no CPU fallback: every compute entry point runs CUDA kernels or raises.
"""
from .binding import (  # noqa: F401
    MODEL_LINEAR, MODEL_HH, MODEL_HH_CLASSIC, PROPOSAL_GAUSSIAN, PROPOSAL_UNIFORM, ENGINE_AUTO, ENGINE_GLOBAL, ENGINE_TILE, ENGINE_TILE_MC, DISC_RK4MAP, DISC_TRAPEZOID, UPDATE_JOINT, UPDATE_COMPONENTWISE, PimcError, Pimc, lib, library_path,
    model_np, rng_selftest, step_selftest, run_host, exported_symbols, fp64_peak, math_selftest, exchange_selftest, run_host_scratch, static_scratch_bytes, latency_selftest,
)
