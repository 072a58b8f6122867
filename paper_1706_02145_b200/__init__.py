"""B200-native hot path of the CELES multi-sphere T-matrix method (arxiv 1706.02145).

The product is libceles.so (hand-written sm_100a CUDA behind the C ABI of include/celes.h); this package is its
thin binding plus the host-side input preparation (Mie coefficients, plane-wave coefficients, seeded workloads).
"""
from .binding import (CELES_ECUDA, CELES_EINVAL, CELES_ELIMIT, CELES_ENOCONV, CELES_ENOMEM, CELES_OK, CelesError, Context,  # noqa: F401
                      CELES_FAR_FIELD_NOALLOC_MAX_DIR, celes_far_field_noalloc,
                      celes_coupling_matvec, celes_coupling_matvec_host, celes_coupling_matvec_rows, celes_destroy, celes_far_field, celes_fp32_peak_probe, celes_gaussian_beam,
                      celes_launch_config, celes_nmax, celes_partition, celes_plan_work, celes_plane_wave, celes_precond_apply, celes_precond_setup, celes_range_info, celes_scattered_field,
                      celes_setup, celes_solve, celes_system_matvec, celes_system_matvec_rows, celes_work_partition,
                      celes_system_matvec_host, celes_translation_table)
