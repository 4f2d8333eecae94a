"""τ grid, bosonic Matsubara set and the transform matrices T_wt / T_tw (inputs of Eq. 28a / Eq. 30).

The paper uses the IR basis with sparse sampling from IRBASIS and prints no formulas;
irbasis / sparse_ir are not installed here.  BASELINE.json says "Chebyshev τ-nodes on [0,β]" and "transform
matrices generated analytically from the grids".  Recipe = SURVEY.md §8c A7:

  nodes     x_t = −cos(π(2t+1)/2N), τ_t = β(1+x_t)/2            (Chebyshev–Gauss roots, mirror symmetric)
  bosonic   N non-negative indices: 0..⌊N/3⌋−1 dense, then geometrically spaced up to 4N
  basis     even Chebyshev polynomials T_{2j}, j < N/2  (bosonic functions on this path are τ ↔ β−τ symmetric)
  T_wt = Î·C          Î[a][j] = (β/2)∫ T_{2j}(x) cos(π n_a (x+1)) dx   (Gauss–Legendre), C = Chebyshev analysis
  T_tw = T_even(x_t)ᵀ · pinv(Î)                                  (least squares)

Both are real, stored as complex128.  These are *inputs*; kernels and oracle only apply them.
"""
import numpy as np


def bosonic_set(N):
    nd = N // 3
    need = N - nd
    sel = list(np.unique(np.round(np.geomspace(max(nd, 1), 4 * N, need)).astype(int)))
    pool = [i for i in np.unique(np.round(np.geomspace(max(nd, 1), 4 * N, 40 * N)).astype(int))
            if i not in sel and i >= nd]
    while len(sel) < need:
        sel.append(pool.pop(0))
    S = sorted(set(list(range(nd)) + sorted(sel)[:need]))
    extra = nd
    while len(S) < N:            # top up with the smallest unused integers
        if extra not in S:
            S.append(extra)
        extra += 1
    return np.array(sorted(S), dtype=np.int64)


def make_grids(ntau, nw, beta):
    """Returns dict(tau[ntau], nbos[nw], T_wt[nw][ntau], T_tw[ntau][nw]) (complex128 matrices, zero imaginary part)."""
    if nw != ntau:
        raise ValueError("this recipe uses nw == ntau (PAPER.md:347: N_tau equals N_omega)")
    N = ntau
    t = np.arange(N)
    half = -np.cos(np.pi * (2 * t[: (N + 1) // 2] + 1) / (2 * N))
    x = np.empty(N)
    x[: (N + 1) // 2] = half
    x[N - 1 - np.arange(N // 2)] = -half[: N // 2]      # exact mirror symmetry: x[N-1-t] = -x[t]
    if N % 2 == 1:
        x[N // 2] = 0.0
    tau = beta * (1.0 + x) / 2.0
    tau[N - 1 - np.arange(N // 2)] = beta - tau[: N // 2]
    S = bosonic_set(N)
    L = N // 2
    le = 2 * np.arange(L)
    M = 2 * N + 2 * int(S.max()) + 300
    xg, wg = np.polynomial.legendre.leggauss(M)
    Tg = np.cos(np.outer(le, np.arccos(xg)))
    Ie = np.array([(beta / 2) * (Tg * (wg * np.cos(np.pi * m * (xg + 1)))).sum(1) for m in S])
    Tt = np.cos(np.outer(le, np.arccos(x)))
    C = Tt * (2.0 / N)
    C[0] *= 0.5
    T_wt = Ie @ C
    T_tw = Tt.T @ np.linalg.pinv(Ie)
    cond = np.linalg.cond(Ie)
    if not cond < 1e3:
        raise RuntimeError(f"ill-conditioned sampling set: cond={cond:.3e}")
    return {"tau": tau, "nbos": S, "T_wt": np.ascontiguousarray(T_wt.astype(np.complex128)),
            "T_tw": np.ascontiguousarray(T_tw.astype(np.complex128)), "cond": cond}


def make_fermionic_transform(ntau, beta, nw=None):
    """tau -> i omega_n matrix for FERMIONIC functions on the same Chebyshev-Gauss tau nodes (Eq. 13, PAPER.md:110-116:
    G(i omega_n) = int_0^beta G(tau) e^{i omega_n tau} dtau, omega_n = (2n+1) pi / beta): an *input* of gw_transform, the
    next step of the workflow after the hot path (Sigma(tau) -> Sigma(i omega_n), Fig. 4 / PAPER.md:320).

    All N Chebyshev polynomials are used (fermionic functions have no tau <-> beta - tau symmetry):
      T_f = I_f . C,  C[j][t] = (2 - delta_j0)/N T_j(x_t),  I_f[n][j] = (beta/2) int_-1^1 T_j(x) e^{i omega_n beta (1+x)/2} dx
    (Gauss-Legendre).  Returns dict(nfer[nw], T_wt_f[nw][ntau] complex128)."""
    N = ntau
    nw = N if nw is None else nw
    S = bosonic_set(N)[:nw]                       # the same index pattern, read as fermionic indices n >= 0
    t = np.arange(N)
    x = -np.cos(np.pi * (2 * t + 1) / (2 * N))
    j = np.arange(N)
    Tt = np.cos(np.outer(j, np.arccos(x)))
    C = Tt * (2.0 / N)
    C[0] *= 0.5
    M = 2 * N + 2 * int(S.max()) + 300
    xg, wg = np.polynomial.legendre.leggauss(M)
    Tg = np.cos(np.outer(j, np.arccos(xg)))
    om = (2 * S + 1) * np.pi / beta
    If = np.array([(beta / 2) * (Tg * (wg * np.exp(1j * w * beta * (1.0 + xg) / 2))).sum(1) for w in om])
    return {"nfer": S, "omega": om, "T_wt_f": np.ascontiguousarray((If @ C).astype(np.complex128))}


def make_fermionic_grids(ntau, beta):
    """Fermionic companions of make_grids on the SAME Chebyshev-Gauss tau nodes, for the loop closure (Eq. 13-16, PAPER.md:110-129;
    Fig. 4 steps 3-4).  All four are *inputs* of the C ABI (gw_fermi_grid); kernels and oracle only apply them.

      nfer[nwf]      nwf = 2*(ntau//2) Matsubara indices, symmetric under n <-> -n-1 (omega_n <-> -omega_n): the non-negative half
                     is bosonic_set(ntau//2) read as fermionic indices
      omega[nwf]     omega_n = (2n+1) pi / beta
      T_wt_f[nwf][ntau]  tau -> i omega_n (Eq. 13): Chebyshev analysis with all ntau polynomials, then the exact integrals
                         I_f[n][j] = (beta/2) int_-1^1 T_j(x) e^{i omega_n beta (1+x)/2} dx  (Gauss-Legendre)
      T_tw_f[ntau][nwf]  i omega_n -> tau (Eq. 14) by least squares on the first L = 2*ntau//3 polynomials: T_L(x_t)^T pinv(I_f[:, :L]).
                         The integrals carry the 1/(i omega_n) tail of a fermionic function exactly (boundary terms of a polynomial),
                         so no separate tail treatment is needed.
      t_beta[nwf]        G(tau = beta^-) = sum_n t_beta[n] G(i omega_n)   (the same fit evaluated at x = +1; gamma = -G(beta^-))
      e_beta[ntau]       G(tau = beta^-) = sum_t e_beta[t] G(tau_t)       (Chebyshev interpolation from the nodes to x = +1)
    """
    N = ntau
    half = max(N // 2, 1)
    pos = bosonic_set(half)[:half] if half >= 3 else np.arange(half, dtype=np.int64)
    S = np.concatenate([-(pos[::-1]) - 1, pos]).astype(np.int64)
    L = max((2 * N) // 3, 1)
    t = np.arange(N)
    x = -np.cos(np.pi * (2 * t + 1) / (2 * N))
    j = np.arange(N)
    Tt = np.cos(np.outer(j, np.arccos(x)))
    C = Tt * (2.0 / N)
    C[0] *= 0.5
    M = 2 * N + 2 * int(np.abs(S).max()) + 300
    xg, wg = np.polynomial.legendre.leggauss(M)
    Tg = np.cos(np.outer(j, np.arccos(xg)))
    om = (2 * S + 1) * np.pi / beta
    If = np.array([(beta / 2) * (Tg * (wg * np.exp(1j * w * beta * (1.0 + xg) / 2))).sum(1) for w in om])
    pin = np.linalg.pinv(If[:, :L])
    cond = np.linalg.cond(If[:, :L])
    if not cond < 1e6:
        raise RuntimeError(f"ill-conditioned fermionic sampling set: cond={cond:.3e}")
    cc = lambda a: np.ascontiguousarray(np.asarray(a).astype(np.complex128))
    return {"nfer": S, "omega": np.ascontiguousarray(om.astype(np.float64)), "T_wt_f": cc(If @ C), "T_tw_f": cc(Tt[:L].T @ pin),
            "t_beta": cc(np.ones(L) @ pin), "e_beta": cc(C.sum(axis=0)), "cond": cond}
