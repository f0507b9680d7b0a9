"""B200-native implicit-filter hot path (arXiv 2404.07398): C-ABI CUDA library + thin Python binding.

    from paper_2404_07398_b200 import if_prepare, if_filter, if_spectrum
    h = if_prepare(coords, tri, period)           # once per mesh ("preparation")
    spec = if_spectrum(h, fields, ells, order_n)   # many fields x scales ("solving")

Build first: python -m paper_2404_07398_b200.build   (sm_100a; no CPU fallback).
"""
from .binding import (EXPORTS, IF_FLAG_HIGHPASS, IF_FLAG_KEEP_CSR, IF_FLAG_MULTIGRID, IF_FLAG_PAIRS, IF_FLAG_TRUE_RESIDUAL, IF_FLAG_VECTOR, Handle, ImplicitFilterError, if_apply, if_destroy, if_energy_noalloc, if_filter,
                      if_launch_count, if_load, if_mesh_export_csr, if_mesh_export_perm, if_mesh_multigrid_info, if_prepare, if_save, if_spectrum, if_spectrum_host,
                      if_workspace_bytes, load_library, strerror)

__all__ = ["EXPORTS", "IF_FLAG_HIGHPASS", "IF_FLAG_KEEP_CSR", "IF_FLAG_MULTIGRID", "IF_FLAG_PAIRS", "IF_FLAG_TRUE_RESIDUAL", "IF_FLAG_VECTOR", "Handle", "ImplicitFilterError", "if_apply", "if_destroy", "if_energy_noalloc", "if_filter",
           "if_launch_count", "if_load", "if_mesh_export_csr", "if_mesh_export_perm", "if_mesh_multigrid_info", "if_prepare", "if_save", "if_spectrum", "if_spectrum_host",
           "if_workspace_bytes", "load_library", "strerror"]
