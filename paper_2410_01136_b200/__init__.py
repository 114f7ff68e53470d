"""synax-b200: line-of-sight synchrotron I/Q/U + Faraday rotation and its VJP, hand-written CUDA for
NVIDIA B200 (sm_100a) behind the C ABI of include/synax.h.  This package is the thin Python binding
(argument marshalling only).  There is no CPU fallback: using any operation without the built CUDA
library or without a CUDA device raises."""
from .binding import (Plan, Model, SynaxError, forward, vjp, forward_f64, vjp_f64, vjp_f64_noalloc, loglike_vjp, adam_step, forward_host, vjp_host, load_library,  # noqa: F401
                      exported_symbols, STATUS)

__all__ = ["Plan", "Model", "SynaxError", "forward", "vjp", "forward_f64", "vjp_f64", "vjp_f64_noalloc", "loglike_vjp", "adam_step", "forward_host", "vjp_host", "load_library",
           "exported_symbols", "STATUS"]
