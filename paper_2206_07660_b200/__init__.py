"""paper_2206_07660_b200 — thin Python binding of libgw_b200 (include/gw.h).

Argument marshalling only: every step of the hot path (Eq. 22, 28a, 28b, 29, 30, 31; Algorithm 1)
runs in the CUDA kernels under csrc/.  PyTorch is used for device memory and streams, nothing else.
There is no CPU fallback: if the shared library is missing or the device is not sm_100 the calls raise.
"""
import ctypes
import os

from .binding import (GWProblem, GWError, GW_SYM_TR, GW_V_FULL, GW_V_QSLAB, gw_sigma_iteration_stream, gw_phi_gw, gw_complex_mma_probe, gw_fp64_subcore_probe, lib, lib_path, gw_polarization, gw_screened_interaction, gw_screened_interaction_phi, gw_transform,
                      gw_selfenergy, gw_exchange, gw_workspace_bytes, gw_sigma_iteration, gw_sigma_iteration_host,
                      gw_executed_flops, gw_launch_count, gw_fp64_peak, gw_fp64_peak_dfma, gw_strerror, gw_version,
                      gw_hartree, gw_hartree_static, gw_static_max_naux, gw_dyson_update, gw_electron_count, gw_find_mu, gw_axpby, gw_scgw_iteration)

__all__ = ["GWProblem", "GWError", "GW_SYM_TR", "GW_V_FULL", "GW_V_QSLAB", "gw_sigma_iteration_stream", "gw_phi_gw", "gw_complex_mma_probe", "gw_fp64_subcore_probe", "lib", "lib_path", "gw_polarization", "gw_screened_interaction", "gw_screened_interaction_phi", "gw_transform", "gw_selfenergy",
           "gw_exchange", "gw_workspace_bytes", "gw_sigma_iteration", "gw_sigma_iteration_host", "gw_executed_flops",
           "gw_launch_count", "gw_fp64_peak", "gw_fp64_peak_dfma", "gw_strerror", "gw_version",
           "gw_hartree", "gw_hartree_static", "gw_static_max_naux", "gw_dyson_update", "gw_electron_count", "gw_find_mu", "gw_axpby", "gw_scgw_iteration"]
