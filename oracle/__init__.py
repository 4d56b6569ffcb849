"""float64 CPU oracle (TEST INFRASTRUCTURE, not the product).

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It shares nothing with the CUDA
path in ``paper_1903_10088_b200/`` and never imports it.

The arithmetic lives in ``osiv_oracle.c`` (plain C, float64); this module only builds
it with gcc and marshals numpy arrays through ctypes.
"""
from .oracle import (  # noqa: F401
    Geometry, Params, build, lib, num_threads, set_num_threads, dgamma, ray, weight, candidate_K,
    forward, forward_brute, backward, backward_brute, tv_value, tv_grad, loglik, residual, tau,
    reconstruct, tv3_value, tv3_grad, reconstruct_stack,
)
