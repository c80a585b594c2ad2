"""B200-native temporal non-local means (TNLM) enhancement hot path of arxiv/paper_1201_2450.

The product is ``libtnlm.so`` (hand-written sm_100a CUDA kernels behind the C ABI of
``include/tnlm.h``).  This package is the thin Python binding: argument marshalling only.
There is no CPU fallback: importing works without a GPU (so the ABI can be checked), but every
compute call requires the compiled library and CUDA tensors and fails loudly otherwise.
"""
from .binding import (TnlmParams, TnlmError, lib, library_path, workspace_bytes, weights_bytes,
                      host_workspace_bytes, tnlm_weights, tnlm_jacobi_step, tnlm_enhance, tnlm_enhance_host,
                      tnlm_jacobi_step_slab, tnlm_tv_diff, tnlm_srr, tnlm_srr_static, tnlm_cnr, kernel_name, launches_per_sweep, z_tile, probe_fp32, strerror,
                      VARIANT_AUTO, VARIANT_GENERIC, VARIANT_TILED, VARIANT_PAIRED, VARIANT_PAIRED_TMEM, EXPORTS,
                      TnlmrGeometry, tnlmr_workspace_bytes, tnlmr_project, tnlmr_backproject, tnlmr_cgls, tnlmr_reconstruct)

__all__ = ["TnlmParams", "TnlmError", "lib", "library_path", "workspace_bytes", "weights_bytes",
           "host_workspace_bytes", "tnlm_weights", "tnlm_jacobi_step", "tnlm_enhance", "tnlm_enhance_host",
           "tnlm_jacobi_step_slab", "tnlm_tv_diff", "tnlm_srr", "tnlm_srr_static", "tnlm_cnr", "kernel_name", "launches_per_sweep", "z_tile", "probe_fp32", "strerror",
           "VARIANT_AUTO", "VARIANT_GENERIC", "VARIANT_TILED", "VARIANT_PAIRED", "VARIANT_PAIRED_TMEM", "EXPORTS",
           "TnlmrGeometry", "tnlmr_workspace_bytes", "tnlmr_project", "tnlmr_backproject", "tnlmr_cgls", "tnlmr_reconstruct"]
