"""Seeded synthetic inputs for the GW self-energy hot path (SURVEY.md §8d recipe).

This package is the ONLY code shared by the CPU oracle (`oracle/`) and the CUDA
path (`paper_2206_07660_b200/`).  It holds none of the method's arithmetic
(no Eq. 22/28-31 of PAPER.md): it only builds the *inputs* of those equations

  * the Γ-centred k-mesh index tables k±q, −k
  * a time-reversal symmetric Fock spectrum → G(k,τ), γ(k)
  * the three-index tensor V[k1][k2][Q][i][j]            (Eq. 6-7)
  * the τ grid, the bosonic Matsubara set and the transform matrices
    T_wt (Eq. 28a) / T_tw (Eq. 30), which are *inputs* of the C-ABI.

They stand in for the paper's PySCF/IRBASIS data, which is
not available offline; see DESIGN.md "Input recipe".
"""
from .configs import CONFIGS, GWConfig, get_config
from .mesh import KMesh
from .grids import make_grids, make_fermionic_transform, make_fermionic_grids
from .fock import make_fock, greens_function, density_matrix, make_h0_s
from .vgen import make_V, make_V_block, to_qslab, make_V_qslab
from .problem import make_problem, make_spin_channels, rotate_spin_channels, Problem

__all__ = ["CONFIGS", "GWConfig", "get_config", "KMesh", "make_grids", "make_fermionic_transform", "make_fermionic_grids", "make_h0_s", "make_fock",
           "greens_function", "density_matrix", "make_V", "make_V_block",
           "make_problem", "make_spin_channels", "rotate_spin_channels", "to_qslab", "make_V_qslab", "Problem"]
