"""Time-reversal symmetric synthetic Fock spectrum → G(k,τ) and γ(k)   (inputs of Eq. 22, 28b, 31).

G^k(τ) = U diag(g(ε,τ)) U†,  g = −e^{−ετ}/(1+e^{−βε})   (single-particle form of PAPER.md Eq. 11 for a quadratic H, μ=0)
γ^k    = U diag(f(ε)) U†,    f = 1/(1+e^{βε})            (γ = −G(β⁻))
ε_{−k} = ε_k, U_{−k} = conj U_k.
"""
import numpy as np


def make_fock(cfg, mesh, channel=0):
    """channel: spin channel of a spin-polarised problem (an independent spectrum per channel; channel 0 is the closed-shell one)."""
    rng = np.random.default_rng([cfg.seed, 1] if channel == 0 else [cfg.seed, 1, int(channel)])
    nk, nao = mesh.nk, cfg.nao
    neg = mesh.neg()
    nocc = nao // 2
    eps = np.zeros((nk, nao))
    U = np.zeros((nk, nao, nao), dtype=np.complex128)
    for k in range(nk):
        if k > neg[k]:
            continue
        lo_hi = np.concatenate([rng.uniform(cfg.elo, -cfg.gap / 2, nocc),
                                rng.uniform(cfg.gap / 2, cfg.ehi, nao - nocc)])
        if k == 0 and cfg.gap > 0 and nocc >= 1 and nao - nocc >= 1:
            lo_hi[nocc - 1] = -cfg.gap / 2      # pin one eigenvalue at each gap edge at Γ
            lo_hi[nocc] = cfg.gap / 2
        e = np.sort(lo_hi)
        A = rng.normal(size=(nao, nao))
        if neg[k] != k:
            A = A + 1j * rng.normal(size=(nao, nao))
        Q, _ = np.linalg.qr(A)
        U[k] = Q
        eps[k] = e
        U[neg[k]] = Q.conj()
        eps[neg[k]] = e
    return eps, U


def _g_weights(eps, tau, beta):
    """g(ε,τ) in the overflow-safe form; |g| < 1e-300 flushed to exactly 0."""
    e = eps[None, ...]
    tt = tau.reshape((-1,) + (1,) * eps.ndim)
    with np.errstate(over="ignore", under="ignore"):
        pos = -np.exp(-np.abs(e) * tt) / (1.0 + np.exp(-beta * np.abs(e)))
        negv = -np.exp(-(beta - tt) * np.abs(e)) / (1.0 + np.exp(-beta * np.abs(e)))
    g = np.where(e >= 0, pos, negv)
    g[np.abs(g) < 1e-300] = 0.0
    return g


def greens_function(eps, U, tau, beta):
    """G[t][k][i][j] complex128."""
    g = _g_weights(eps, np.asarray(tau), beta)              # [t][k][n]
    return np.ascontiguousarray(np.einsum("kin,tkn,kjn->tkij", U, g, U.conj()))


def fermi(eps, beta):
    with np.errstate(over="ignore", under="ignore"):
        x = np.exp(-beta * np.abs(eps))
    return np.where(eps >= 0, x / (1.0 + x), 1.0 / (1.0 + x))


def density_matrix(eps, U, beta):
    """γ[k][i][j] complex128."""
    f = fermi(eps, beta)
    return np.ascontiguousarray(np.einsum("kin,kn,kjn->kij", U, f, U.conj()))


def make_h0_s(cfg, mesh, eps, U):
    """One-electron Hamiltonian H0[k] and overlap S[k] for the loop closure (Eq. 15-16): the paper takes them from
    PySCF; here H0[k] = U diag(eps) U^+ (the Fock spectrum that also built G) and S[k] = Q diag(s) Q^+ with seeded
    s in [0.6, 1.4] (a non-orthogonal basis, Hermitian positive definite), both time-reversal symmetric: X[-k] = conj X[k]."""
    rng = np.random.default_rng([cfg.seed, 3])
    nk, nao = mesh.nk, cfg.nao
    neg = mesh.neg()
    H0 = np.einsum("kin,kn,kjn->kij", U, eps, U.conj())
    S = np.zeros((nk, nao, nao), dtype=np.complex128)
    for k in range(nk):
        if k > neg[k]:
            continue
        A = rng.normal(size=(nao, nao))
        if neg[k] != k:
            A = A + 1j * rng.normal(size=(nao, nao))
        Q, _ = np.linalg.qr(A)
        sv = rng.uniform(0.6, 1.4, nao)
        Sk = (Q * sv[None, :]) @ Q.conj().T
        S[k] = 0.5 * (Sk + Sk.conj().T)
        S[neg[k]] = S[k].conj()
    return np.ascontiguousarray(H0), np.ascontiguousarray(S)
