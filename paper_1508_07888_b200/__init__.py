"""B200-native (sm_100a) radiative-transfer + thermo-chemistry hot path of EMMA (arXiv 1508.07888).

The product is the CUDA C-ABI library `libemma_rt.so` (include/emma_rt.h); this package is a thin ctypes binding
with the same entry-point names.  PyTorch is used only for device memory and streams.  There is no CPU fallback:
without the built library or without a CUDA device the binding raises.
"""
from .binding import (EmmaRT, EmmaRTError, emma_rt_arena_bytes, emma_rt_init, emma_rt_set_sources, emma_rt_step,  # noqa: F401
                      emma_rt_read, emma_rt_write, emma_rt_free, emma_rt_dt_cfl, lib, lib_path, Config, Diag,
                      emma_rt_photons_total_noalloc, NOALLOC_MAX_CELLGROUPS,
                      FIELD_U, FIELD_N, FIELD_F, FIELD_X, FIELD_T, FIELD_E, FIELD_N0, FIELD_SUBCYCLES, FIELD_XNEUTRAL,
                      OK, EINVAL, ENOMEM, ECUDA, ENONFINITE, ESTATE, ECFL, ESUBCYCLE, EXPORTED_SYMBOLS,
                      FLUX_GLF, FLUX_HLL, BC_PERIODIC, BC_TRANSMISSIVE, BC_REFLECTIVE, BC_INFLOW)
