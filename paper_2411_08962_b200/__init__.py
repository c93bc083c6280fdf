"""B200-native determinant-form Wick contraction (arXiv 2411.08962): Python binding of the C-ABI
library libwick_b200.so (include/wick.h).  See DESIGN.md."""
from .binding import (  # noqa: F401
    BUILD_IDENTITY_TEST, BUILD_ISOSPIN, CONTRACT_FORCE_FLAT, CONTRACT_NO_STAGED, CONTRACT_COMPLEX_COEFFS, CONTRACT_NO_REG_MINORS, CONTRACT_JACOBI, CONTRACT_JACOBI_UNFUSED, EXPORTED_SYMBOLS, OP_DEUTERON_EQ20, OP_HELIUM3_EQ21, Operator, Terms, WickError,
    block_tensor, build_block_terms, build_terms_matrix, combine_two_clusters, contract_many, operator_product, two_cluster_correlator, operator_from_nucleons, operator_from_raw, operator_paper,
    build_terms, build_terms_from_list, contract, contract_host, contract_workspace_bytes,
    launch_count, library_path, load_library, measure_fp64_peak, minor_dets, minor_dets_static, minor_table, static_scratch_bytes, profile_enable, profile_read, release_cached_buffers,
)
