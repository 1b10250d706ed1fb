"""B200-native monodomain + TP06 time step (arXiv 2112.12854, section 3.2) behind the C-ABI of include/ep.h.

The Python side only marshals arguments: every step of the path runs in the sm_100a kernels of csrc/.
There is no CPU fallback; importing works without a GPU (so the symbol table can be checked), computing does not.
"""
from .binding import (EP_MODEL_CRN98, EP_MODEL_STEWART, EP_MODEL_TP06, host_stencil_tri, shard_plan, halo_exchange_local, EpError, Sim, host_stencil, lib, math_eval, model_n_states, fp64_rate, weighted_mean_noalloc, NOALLOC_MAX_N)  # noqa: F401

__all__ = ["Sim", "EpError", "host_stencil", "lib", "math_eval", "model_n_states", "fp64_rate", "EP_MODEL_TP06", "EP_MODEL_CRN98", "EP_MODEL_STEWART", "host_stencil_tri", "shard_plan", "halo_exchange_local", "weighted_mean_noalloc", "NOALLOC_MAX_N"]
