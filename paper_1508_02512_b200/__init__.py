"""B200-native hot path of arXiv:1508.02512: shifted rank-1 lattice QMC over sector-decomposed Feynman integrands.

    tables = qmc_prepare(workload)                 # graph, kinematics, eps_order -> sector tables   (host C++)
    result = qmc_integrate(tables, N, m, seed)     # -> Laurent coefficients +- errors               (sm_100a CUDA)

The Python layer only marshals arguments into the C-ABI library libqmcfeyn.so (include/qmc_feynman.h); it is
imported lazily so that `import paper_1508_02512_b200` works on a box where the library has not been built yet,
while any call fails loudly there (no CPU fallback).
"""
from . import binding
from .binding import (QmcError, Result, Tables, lib, qmc_flop_model, qmc_fp64_peak, qmc_cbc_vector, qmc_generating_vector, qmc_generating_vector_noalloc, qmc_embedded_vector, qmc_integrate_embedded, qmc_integrate_allocated,
                      qmc_integrate, qmc_integrate_async, qmc_prefactor_series, qmc_prepare, qmc_prepare_batch, qmc_result_device_totals, qmc_result_fetch,
                      qmc_shifts, qmc_statistics, strerror, LIB_PATH)

__all__ = ["QmcError", "Result", "Tables", "lib", "qmc_flop_model", "qmc_fp64_peak", "qmc_cbc_vector", "qmc_generating_vector", "qmc_generating_vector_noalloc", "qmc_embedded_vector", "qmc_integrate_embedded", "qmc_integrate_allocated",
           "qmc_integrate", "qmc_integrate_async", "qmc_prefactor_series", "qmc_prepare", "qmc_prepare_batch", "qmc_result_device_totals", "qmc_result_fetch",
           "qmc_shifts", "qmc_statistics", "strerror", "LIB_PATH", "binding"]
