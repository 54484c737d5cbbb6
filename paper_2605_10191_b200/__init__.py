"""polfed-b200: the POLFED hot path (Clenshaw-evaluated Chebyshev filter on a sparse
many-body Hamiltonian) as hand-written sm_100a kernels behind a C ABI (include/polfed.h).

The functions re-exported here are thin ctypes wrappers with the names of the C entry points.
"""
from .binding import (  # noqa: F401
    Basis, Ham, PolfedError, EXPORTS, LIB_PATH, TERM_KINDS, FORMAT_CSR, FORMAT_TILED, FORMAT_FLIP, FORMAT_SECTOR,
    lib, polfed_last_error, polfed_version, polfed_release_scratch,
    polfed_build_basis, polfed_basis_dim, polfed_basis_states, polfed_basis_rank,
    polfed_build_hamiltonian, polfed_ham_from_csr, polfed_ham_from_csr_ex, polfed_ham_csr, HAM_NO_SNAPSHOT,
    polfed_fused_step, polfed_filter_workspace_bytes, polfed_filter_workspace_bytes_ham,
    polfed_filter_apply,
    polfed_filter_apply_host, polfed_filter_coeffs,
    polfed_spectrum_bounds, polfed_block_lanczos_eigs,
    polfed_kpm_workspace_bytes, polfed_kpm_moments, polfed_kpm_dos,
    polfed_block_gram, polfed_block_update, polfed_block_gram_static, STATIC_GRAM_DOUBLES,
)
