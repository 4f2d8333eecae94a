"""Assemble one synthetic problem instance: grids, transform matrices, G(k,τ), γ(k), V, k-mesh tables."""
from dataclasses import dataclass, field
import numpy as np

from .configs import GWConfig, get_config
from .mesh import KMesh
from .grids import make_grids
from .fock import make_fock, greens_function, density_matrix
from .vgen import make_V, to_qslab


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


def make_spin_channels(p, ns=2):
    """Spin-polarised inputs for ns collinear channels (include/gw.h "Spin channels"; the paper's AFM MnO case):
    channel 0 is the problem's own G / gamma, the other channels get an independent seeded spectrum (a raw problem: independent
    seeded non-Hermitian matrices).  Returns (G [ns][ntau][nk][nao][nao], gamma [ns][nk][nao][nao])."""
    cfg, mesh = p.cfg, p.mesh
    Gs, gs = [p.G], [p.gamma]
    for ch in range(1, ns):
        if "W" in p.extras:             # raw problem
            rng = np.random.default_rng([cfg.seed, 7, ch])
            cplx = lambda shape, sc: (rng.normal(size=shape) + 1j * rng.normal(size=shape)) * sc
            scale = np.exp(-6.0 * np.minimum(p.tau, cfg.beta - p.tau) / cfg.beta).reshape(-1, 1, 1, 1)
            Gs.append(cplx(p.G.shape, 1.0 / np.sqrt(cfg.nao)) * scale)
            gs.append(cplx(p.gamma.shape, 1.0 / np.sqrt(cfg.nao)))
        else:
            eps, U = make_fock(cfg, mesh, channel=ch)
            Gs.append(greens_function(eps, U, p.tau, cfg.beta))
            gs.append(density_matrix(eps, U, cfg.beta))
    return np.ascontiguousarray(np.stack(Gs)), np.ascontiguousarray(np.stack(gs))


def rotate_spin_channels(Gs, gs, seed=0):
    """Two-component inputs from two collinear channels by ONE global spin rotation R in SU(2) (seeded): block (s, s') of the result is
    sum_c R[s][c] X^c conj(R[s'][c]), blocks in the order uu, ud, du, dd (include/gw.h "Spin blocks").  Off-diagonal blocks are non-zero,
    as with spin-orbit coupling; spin traces (P0, J) are those of the collinear channels, which is what the pins use."""
    rng = np.random.default_rng([220607660, 11, int(seed)])
    th, ph, ps = rng.uniform(0.3, 1.2), rng.uniform(0, 2 * np.pi), rng.uniform(0, 2 * np.pi)
    R = np.array([[np.cos(th) * np.exp(1j * ph), np.sin(th) * np.exp(1j * ps)],
                  [-np.sin(th) * np.exp(-1j * ps), np.cos(th) * np.exp(-1j * ph)]])
    rot = lambda X: np.ascontiguousarray(np.stack([sum(R[s, c] * X[c] * np.conj(R[sp, c]) for c in range(2)) for s in range(2) for sp in range(2)]))
    return rot(Gs), rot(gs), R


def make_problem(cfg, v_device="cpu", with_V=True, raw=False) -> Problem:
    """raw=False: the BASELINE.json inputs (time-reversal symmetric Fock-built G, group-averaged V).
    raw=True : inputs with NO symmetry at all — V blocks are independent draws (V[k1][k2] unrelated to V[k2][k1] or
               V[-k1][-k2]), G[t][k] and gamma[k] are seeded non-Hermitian complex matrices, extras["W"] is a seeded
               non-Hermitian [ntau][nk][naux][naux] array to stand in for Wt.  They tell the printed index patterns of
               Eq. 22 / 28b / 31 apart from their symmetric twins (transposed or conjugated operands); stage 2 (Cholesky)
               is not defined on them."""
    if not isinstance(cfg, GWConfig):
        cfg = get_config(cfg)
    mesh = KMesh(cfg.mesh)
    gr = make_grids(cfg.ntau, cfg.nw, cfg.beta)
    eps, U = make_fock(cfg, mesh)
    extras = {}
    if raw:
        rng = np.random.default_rng([cfg.seed, 7])
        cplx = lambda shape, sc: np.ascontiguousarray((rng.normal(size=shape) + 1j * rng.normal(size=shape)) * sc)
        # a tau-dependent scale keeps the decades-wide dynamic range of a physical G(tau)
        scale = np.exp(-6.0 * np.minimum(gr["tau"], cfg.beta - gr["tau"]) / cfg.beta).reshape(-1, 1, 1, 1)
        G = cplx((cfg.ntau, mesh.nk, cfg.nao, cfg.nao), 1.0 / np.sqrt(cfg.nao)) * scale
        gamma = cplx((mesh.nk, cfg.nao, cfg.nao), 1.0 / np.sqrt(cfg.nao))
        extras["W"] = cplx((cfg.ntau, mesh.nk, cfg.naux, cfg.naux), 1.0 / np.sqrt(cfg.naux))
    else:
        G = greens_function(eps, U, gr["tau"], cfg.beta)
        gamma = density_matrix(eps, U, cfg.beta)
    V = make_V(cfg, mesh, device=v_device, raw=raw) if with_V else None
    return Problem(cfg, mesh, gr["tau"], gr["nbos"], gr["T_wt"], gr["T_tw"], eps, U, G, gamma, V, extras)
