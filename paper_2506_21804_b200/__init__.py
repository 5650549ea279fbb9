"""B200-native lattice Boltzmann hot path of arxiv 2506.21804 (BGK / HRR + Smagorinsky LES + HLBM).

Thin Python binding over the C ABI in include/lbm.h (library: liblbm_b200.so, CUDA sm_100a).
The binding only marshals arguments; every step of the path runs in the library's kernels.
There is no CPU fallback: loading fails loudly if the library is missing, and lbm_create fails if
no CUDA device is usable.
"""
from .binding import (LBM, LbmError, LbmParams, lbm_create, lbm_destroy, lbm_get_populations, lbm_init_equilibrium,
                      lbm_last_error, lbm_moments, lbm_query, lbm_set_fields, lbm_set_geometry, lbm_set_option,
                      lbm_set_stream, lbm_step, lbm_synchronize, lbm_totals, library_path, load_library, lbm_set_inflow,
                      lbm_set_vortices, lbm_get_inflow, lbm_set_porosity, lbm_set_body_velocity, lbm_get_populations_box,
                      lbm_set_populations_box, lbm_set_halo, lbm_step_halo, lbm_halo_pack, lbm_halo_unpack, lbm_totals_static)

__all__ = ["LBM", "LbmError", "LbmParams", "lbm_create", "lbm_destroy", "lbm_get_populations", "lbm_init_equilibrium",
           "lbm_last_error", "lbm_moments", "lbm_query", "lbm_set_fields", "lbm_set_geometry", "lbm_set_option",
           "lbm_set_stream", "lbm_step", "lbm_synchronize", "lbm_totals", "library_path", "load_library", "lbm_set_inflow",
           "lbm_set_vortices", "lbm_get_inflow", "lbm_set_porosity", "lbm_set_body_velocity", "lbm_get_populations_box",
           "lbm_set_populations_box", "lbm_set_halo", "lbm_step_halo", "lbm_halo_pack", "lbm_halo_unpack", "lbm_totals_static"]
