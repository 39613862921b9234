"""B200-native hot path of invDFT (arXiv 2510.10529): FE Kohn-Sham operator apply and Chebyshev filter.

Thin ctypes binding of the C-ABI library (include/fe_cheb.h); every step of the path runs in the sm_100a
kernels of csrc/.  There is no CPU fallback: importing works without a GPU, calling does not.
"""
from .binding import (  # noqa: F401
    FEError, FEMesh, cheb_filter, cheb_filter_host, fe_add_subspace, fe_apply_H, fe_apply_H_chain, fe_apply_potential, fe_chfsi, fe_density, fe_diag_peak, fe_get_constraints, fe_get_dirichlet_mask, fe_get_l2g, fe_get_mass, fe_get_node_coords,
    fe_get_quad_coords, fe_gram, fe_gram_static, fe_lanczos_bounds, fe_last_error, fe_launch_count, fe_mesh_create, fe_mesh_create_general, fe_mesh_destroy, fe_num_all_nodes, fe_num_constraint_entries, fe_nodes_per_cell,
    fe_minres_shifted, fe_num_cells, fe_num_free, fe_num_nodes, fe_quad_per_cell, fe_rayleigh_ritz, fe_ritz_residuals, fe_set_potential, fe_set_variant, library_path,
    load_library,
)
