"""Assemble one synthetic problem instance: grids, transform matrices, G(k,τ), γ(k), V, k-mesh tables."""
from dataclasses import dataclass, field
import numpy as np

from .configs import GWConfig, get_config
from .mesh import KMesh
from .grids import make_grids
from .fock import make_fock, greens_function, density_matrix
from .vgen import make_V


@dataclass
class Problem:
    cfg: GWConfig
    mesh: KMesh
    tau: np.ndarray
    nbos: np.ndarray
    T_wt: np.ndarray          # [nw][ntau] complex128 (Eq. 28a)
    T_tw: np.ndarray          # [ntau][nw] complex128 (Eq. 30)
    eps: np.ndarray           # [nk][nao]  Fock eigenvalues (tests only: Lindhard pin)
    U: np.ndarray             # [nk][nao][nao] eigenvectors (tests only)
    G: np.ndarray             # [ntau][nk][nao][nao]
    gamma: np.ndarray         # [nk][nao][nao]
    V: object = None          # torch complex128 [nk][nk][naux][nao][nao] on v_device, or None
    extras: dict = field(default_factory=dict)


def make_problem(cfg, v_device="cpu", with_V=True) -> Problem:
    if not isinstance(cfg, GWConfig):
        cfg = get_config(cfg)
    mesh = KMesh(cfg.mesh)
    gr = make_grids(cfg.ntau, cfg.nw, cfg.beta)
    eps, U = make_fock(cfg, mesh)
    G = greens_function(eps, U, gr["tau"], cfg.beta)
    gamma = density_matrix(eps, U, cfg.beta)
    V = make_V(cfg, mesh, device=v_device) if with_V else None
    return Problem(cfg, mesh, gr["tau"], gr["nbos"], gr["T_wt"], gr["T_tw"], eps, U, G, gamma, V)
