"""B200-native batched H|psi> for plane-wave Kohn-Sham DFT (the hot path of arxiv 2308.07277).

The product is the C-ABI library ``libqm_hpsi.so`` (include/qm_hpsi.h, csrc/); this package is
its thin ctypes binding.  Importing the package does not load the library; the first call does,
and fails loudly if it has not been built (``python __graft_entry__.py``).
"""
from .binding import (  # noqa: F401
    GSpace, MatrixElements, BatchPlan, QmError, EXPORTS, LIB_PATH, load_library,
    qm_version, qm_fft_size_supported,
    qm_gspace_create, qm_gspace_destroy, qm_gspace_num_k, qm_gspace_num_g, qm_gspace_num_sticks,
    qm_gspace_get_index_map, qm_gspace_get_miller, qm_gspace_get_g2, qm_gspace_alias_free,
    qm_set_vloc, qm_set_nonlocal, qm_apply_h, qm_subspace, qm_subspace_static, qm_taylor_propagate, qm_density_reset, qm_density_accumulate, qm_density_get, qm_apply_h_host, qm_apply_h_host_async, qm_host_synchronize, qm_debug_g2r, qm_debug_r2g,
    qm_reserve, qm_batch_plan_create, qm_batch_plan_launch, qm_batch_plan_destroy, qm_split_operator_set, qm_split_operator_propagate,
    qm_mtxel_create, qm_mtxel_destroy, qm_mtxel_num_g, qm_mtxel_get_miller, qm_mtxel_get_index_map, qm_matrix_elements,
    qm_get_launch_count, qm_probe_fp64_tensor_peak,
    qm_profile_enable, qm_profile_reset, qm_profile_read, qm_kernel_name,
)
