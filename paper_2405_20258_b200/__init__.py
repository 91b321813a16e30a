"""B200-native static-subspace RPA correlation energy (arxiv 2405.20258) -- thin Python binding over the C-ABI
library `librpa_b200.so` (include/rpa_b200.h).  Argument marshalling only: every step of the hot path runs in
the library's CUDA kernels.  PyTorch supplies device memory and the CUDA stream, nothing else."""
from .binding import (RpaContext, RpaError, load_library, library_path, EXPORTED_SYMBOLS,
                      rpa_create, rpa_destroy, rpa_workspace_bytes, rpa_energy_workspace_bytes, rpa_set_workspace,
                      rpa_mtxel, rpa_chi0_static, rpa_subspace_basis, rpa_chi_subspace_freq,
                      rpa_correlation_energy, rpa_energy_device, rpa_energy_host, rpa_fp64_peak, rpa_launch_count,
                      rpa_profile_begin, rpa_profile_end, PROFILE_CLASSES,
                      rpa_chi0_static_occ, rpa_chi_subspace_freq_occ,
                      rpa_epsilon_inverse, rpa_epsilon_inverse_workspace_bytes, rpa_basis_info, rpa_basis_quality,
                      rpa_pass_begin, rpa_pass1_chi0, rpa_pass_basis, rpa_pass2_chis, rpa_pass_energy, rpa_pass_end,
                      rpa_noalloc_max_pairs, rpa_noalloc_setup, rpa_chi0_static_noalloc)

from .sharded import shard_range, Comm, rpa_energy_sharded

__all__ = ["shard_range", "Comm", "rpa_energy_sharded", "RpaContext", "RpaError", "load_library", "library_path", "EXPORTED_SYMBOLS",
           "rpa_create", "rpa_destroy", "rpa_workspace_bytes", "rpa_energy_workspace_bytes", "rpa_set_workspace",
           "rpa_mtxel", "rpa_chi0_static", "rpa_subspace_basis", "rpa_chi_subspace_freq",
           "rpa_correlation_energy", "rpa_energy_device", "rpa_energy_host", "rpa_fp64_peak", "rpa_launch_count",
           "rpa_profile_begin", "rpa_profile_end", "PROFILE_CLASSES",
           "rpa_chi0_static_occ", "rpa_chi_subspace_freq_occ",
           "rpa_epsilon_inverse", "rpa_epsilon_inverse_workspace_bytes", "rpa_basis_info", "rpa_basis_quality",
           "rpa_pass_begin", "rpa_pass1_chi0", "rpa_pass_basis", "rpa_pass2_chis", "rpa_pass_energy", "rpa_pass_end",
           "rpa_noalloc_max_pairs", "rpa_noalloc_setup", "rpa_chi0_static_noalloc"]
