"""ctypes front-end of the CPU oracle (oracle/gwref.c).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this.
It never imports the CUDA package and shares no code with it.  See gwref.c for the equations it follows
(Eq. 22, 28a, 28b, 29, 30, 31; Algorithm 1) and tests/test_oracle_pins.py for what pins it.
"""
import ctypes
import os
import subprocess
import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libgwref.so")
_lib = None


def build(force=False):
    """Compile gwref.c with gcc (-O2, OpenMP over the outermost independent loop only)."""
    src = os.path.join(_HERE, "gwref.c")
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(src):
        subprocess.check_call(["gcc", "-O2", "-std=c11", "-fopenmp", "-fPIC", "-shared", "-o", _SO, src, "-lm"])
    return _SO


class Dims(ctypes.Structure):
    _fields_ = [("nk1", ctypes.c_int32), ("nk2", ctypes.c_int32), ("nk3", ctypes.c_int32),
                ("nao", ctypes.c_int32), ("naux", ctypes.c_int32), ("ntau", ctypes.c_int32),
                ("nw", ctypes.c_int32), ("spin_deg", ctypes.c_int32), ("beta", ctypes.c_double)]


def lib():
    global _lib
    if _lib is None:
        build()
        _lib = ctypes.CDLL(_SO)
        _lib.gwref_num_threads.restype = ctypes.c_int
        for name in ("gwref_kadd", "gwref_ksub", "gwref_p0t_slice", "gwref_polarization", "gwref_dyson",
                     "gwref_screened_interaction_q", "gwref_screened_interaction", "gwref_sigma_slice",
                     "gwref_selfenergy", "gwref_exchange_slice", "gwref_exchange", "gwref_sigma_slice_qrange",
                     "gwref_exchange_slice_qrange", "gwref_hartree", "gwref_dyson_update_one", "gwref_dyson_update", "gwref_find_mu"):
            getattr(_lib, name).restype = ctypes.c_int
        _lib.gwref_transform.restype = None
        _lib.gwref_electron_count.restype = ctypes.c_double
        _lib.gwref_axpby.restype = None
    return _lib


def num_threads():
    return int(lib().gwref_num_threads())


def _dims(cfg):
    return Dims(cfg.mesh[0], cfg.mesh[1], cfg.mesh[2], cfg.nao, cfg.naux, cfg.ntau, cfg.nw, cfg.spin_deg, cfg.beta)


def _p(a):
    assert a.dtype == np.complex128 and a.flags["C_CONTIGUOUS"]
    return a.ctypes.data_as(ctypes.c_void_p)


class VBlocks:
    """Table of nk*nk block pointers.  `blocks` is either the full array V[k1][k2][Q][i][j] or a dict
    {(k1,k2): ndarray[naux][nao][nao]} holding only the resident blocks (big configs, sampled slices)."""

    def __init__(self, cfg, blocks):
        nk = cfg.nk
        self.keep = blocks
        self.table = (ctypes.c_void_p * (nk * nk))()
        if isinstance(blocks, dict):
            for (k1, k2), b in blocks.items():
                assert b.shape == (cfg.naux, cfg.nao, cfg.nao)
                self.table[k1 * nk + k2] = _p(b)
        else:
            assert blocks.shape == (nk, nk, cfg.naux, cfg.nao, cfg.nao)
            base = blocks.ctypes.data
            step = cfg.naux * cfg.nao * cfg.nao * 16
            for i in range(nk * nk):
                self.table[i] = base + i * step


def kadd(cfg, k, q):
    d = _dims(cfg)
    return lib().gwref_kadd(ctypes.byref(d), int(k), int(q))


def ksub(cfg, k, q):
    d = _dims(cfg)
    return lib().gwref_ksub(ctypes.byref(d), int(k), int(q))


def p0t_slice(cfg, vb, G_t, G_tbar, q):
    """Eq. 28b for one (q, tau_t).  G_t = G[t], G_tbar = G[ntau-1-t], each [nk][nao][nao]."""
    out = np.empty((cfg.naux, cfg.naux), np.complex128)
    d = _dims(cfg)
    rc = lib().gwref_p0t_slice(ctypes.byref(d), vb.table, _p(G_t), _p(G_tbar), int(q), _p(out))
    if rc:
        raise RuntimeError("oracle: a needed V block is not resident")
    return out


def polarization(cfg, vb, G):
    out = np.empty((cfg.ntau, cfg.nk, cfg.naux, cfg.naux), np.complex128)
    d = _dims(cfg)
    if lib().gwref_polarization(ctypes.byref(d), vb.table, _p(G), _p(out)):
        raise RuntimeError("oracle: a needed V block is not resident")
    return out


def dyson(P):
    """Eq. 29 for one matrix: (I - P)^-1 P."""
    n = P.shape[0]
    X = np.empty_like(P)
    if lib().gwref_dyson(n, _p(np.ascontiguousarray(P)), _p(X)):
        raise RuntimeError("oracle: zero pivot")
    return X


def transform(T, X):
    """Eq. 13 / 28a / 30 as a plain matrix application along the leading axis: Y[o][...] = sum_i T[o][i] X[i][...]."""
    T = np.ascontiguousarray(T, dtype=np.complex128); X = np.ascontiguousarray(X, dtype=np.complex128)
    n_out, n_in = T.shape
    assert X.shape[0] == n_in
    ln = int(np.prod(X.shape[1:]))
    Y = np.empty((n_out,) + X.shape[1:], np.complex128)
    lib().gwref_transform(ctypes.c_int(n_out), ctypes.c_int(n_in), _p(T), _p(X), ctypes.c_size_t(ln), _p(Y), ctypes.c_size_t(ln),
                          ctypes.c_size_t(ln))
    return Y


def phi(P):
    """Summand of Eq. 37 for one matrix: tr{ln[I - P] + P}."""
    n = P.shape[0]
    out = ctypes.c_double(0.0)
    if lib().gwref_phi(n, _p(np.ascontiguousarray(P, dtype=np.complex128)), ctypes.byref(out)):
        raise RuntimeError("oracle: zero pivot")
    return out.value


def screened_interaction_q(cfg, T_wt, T_tw, P0t_q, want_freq=False):
    """Stage 2 for one q.  P0t_q: packed [ntau][naux][naux]."""
    ps = cfg.naux * cfg.naux
    Wt_q = np.empty((cfg.ntau, cfg.naux, cfg.naux), np.complex128)
    P0w = np.empty((cfg.nw, cfg.naux, cfg.naux), np.complex128)
    Ww = np.empty((cfg.nw, cfg.naux, cfg.naux), np.complex128)
    d = _dims(cfg)
    rc = lib().gwref_screened_interaction_q(ctypes.byref(d), _p(T_wt), _p(T_tw), _p(np.ascontiguousarray(P0t_q)),
                                            ctypes.c_size_t(ps), _p(Wt_q), ctypes.c_size_t(ps), _p(P0w), _p(Ww))
    if rc:
        raise RuntimeError("oracle: zero pivot")
    return (Wt_q, P0w, Ww) if want_freq else Wt_q


def screened_interaction(cfg, T_wt, T_tw, P0t, want_freq=False):
    Wt = np.empty_like(P0t)
    P0w = np.empty((cfg.nw, cfg.nk, cfg.naux, cfg.naux), np.complex128) if want_freq else None
    Ww = np.empty((cfg.nw, cfg.nk, cfg.naux, cfg.naux), np.complex128) if want_freq else None
    d = _dims(cfg)
    rc = lib().gwref_screened_interaction(ctypes.byref(d), _p(T_wt), _p(T_tw), _p(P0t), _p(Wt),
                                          _p(P0w) if want_freq else None, _p(Ww) if want_freq else None)
    if rc:
        raise RuntimeError("oracle: zero pivot")
    return (Wt, P0w, Ww) if want_freq else Wt


def sigma_slice(cfg, vb, G_t, Wt_t, k, q_begin=0, q_end=None):
    """Eq. 31 for one (k, tau_t).  G_t: [nk][nao][nao], Wt_t: [nk][naux][naux] (indexed by the global q).
    q_begin/q_end restrict the q sum (one rank's partial sum)."""
    out = np.empty((cfg.nao, cfg.nao), np.complex128)
    d = _dims(cfg)
    q_end = cfg.nk if q_end is None else q_end
    if lib().gwref_sigma_slice_qrange(ctypes.byref(d), vb.table, _p(G_t), _p(Wt_t), int(k), int(q_begin), int(q_end), _p(out)):
        raise RuntimeError("oracle: a needed V block is not resident")
    return out


def selfenergy(cfg, vb, G, Wt):
    out = np.empty((cfg.ntau, cfg.nk, cfg.nao, cfg.nao), np.complex128)
    d = _dims(cfg)
    if lib().gwref_selfenergy(ctypes.byref(d), vb.table, _p(G), _p(Wt), _p(out)):
        raise RuntimeError("oracle: a needed V block is not resident")
    return out


def exchange_slice(cfg, vb, gamma, k, q_begin=0, q_end=None):
    out = np.empty((cfg.nao, cfg.nao), np.complex128)
    d = _dims(cfg)
    q_end = cfg.nk if q_end is None else q_end
    if lib().gwref_exchange_slice_qrange(ctypes.byref(d), vb.table, _p(gamma), int(k), int(q_begin), int(q_end), _p(out)):
        raise RuntimeError("oracle: a needed V block is not resident")
    return out


def exchange(cfg, vb, gamma):
    out = np.empty((cfg.nk, cfg.nao, cfg.nao), np.complex128)
    d = _dims(cfg)
    if lib().gwref_exchange(ctypes.byref(d), vb.table, _p(gamma), _p(out)):
        raise RuntimeError("oracle: a needed V block is not resident")
    return out


# ---------------------------------------------------------------------------------------------------------------------
# loop closure (Fig. 4, Eq. 15, 16, 20)
# ---------------------------------------------------------------------------------------------------------------------
def _pd(a):
    assert a.dtype == np.float64 and a.flags["C_CONTIGUOUS"]
    return a.ctypes.data_as(ctypes.c_void_p)


def hartree(cfg, vb, gamma):
    """Eq. 20: J[k][i][j]."""
    out = np.empty((cfg.nk, cfg.nao, cfg.nao), np.complex128)
    d = _dims(cfg)
    if lib().gwref_hartree(ctypes.byref(d), vb.table, _p(gamma), _p(out)):
        raise RuntimeError("oracle: a needed V block is not resident")
    return out


def dyson_update(cfg, omega, mu, S, F, Sigma_w=None):
    """Eq. 16 for all (n, k): G_w[n][k] = [(i omega_n + mu) S[k] - F[k] - Sigma_w[n][k]]^-1."""
    omega = np.ascontiguousarray(omega, dtype=np.float64)
    out = np.empty((len(omega), cfg.nk, cfg.nao, cfg.nao), np.complex128)
    d = _dims(cfg)
    if lib().gwref_dyson_update(ctypes.byref(d), len(omega), _pd(omega), ctypes.c_double(mu), _p(S), _p(F),
                                _p(Sigma_w) if Sigma_w is not None else None, _p(out)):
        raise RuntimeError("oracle: zero pivot")
    return out


def electron_count(cfg, t_beta, S, G_w):
    """Eq. 15 with gamma = -G(beta^-) = -sum_n t_beta[n] G_w[n]."""
    d = _dims(cfg)
    return float(lib().gwref_electron_count(ctypes.byref(d), G_w.shape[0], _p(t_beta), _p(S), _p(G_w)))


def find_mu(cfg, omega, t_beta, S, F, Sigma_w, n_target, mu_lo, mu_hi, mu_tol=1e-12):
    """Bisection for the chemical potential (Fig. 4 step 3).  Returns (mu, N_e(mu))."""
    omega = np.ascontiguousarray(omega, dtype=np.float64)
    scratch = np.empty((len(omega), cfg.nk, cfg.nao, cfg.nao), np.complex128)
    mu, ne = ctypes.c_double(0.0), ctypes.c_double(0.0)
    d = _dims(cfg)
    rc = lib().gwref_find_mu(ctypes.byref(d), len(omega), _pd(omega), _p(t_beta), _p(S), _p(F),
                             _p(Sigma_w) if Sigma_w is not None else None, ctypes.c_double(n_target), ctypes.c_double(mu_lo),
                             ctypes.c_double(mu_hi), ctypes.c_double(mu_tol), _p(scratch), ctypes.byref(mu), ctypes.byref(ne))
    if rc:
        raise RuntimeError(f"oracle: chemical-potential search failed (code {rc})")
    return mu.value, ne.value


def axpby(a, X, b, Y):
    """Y <- a X + b Y."""
    class C(ctypes.Structure):
        _fields_ = [("re", ctypes.c_double), ("im", ctypes.c_double)]
    assert X.shape == Y.shape
    lib().gwref_axpby.argtypes = [ctypes.c_size_t, C, ctypes.c_void_p, C, ctypes.c_void_p]
    lib().gwref_axpby(X.size, C(complex(a).real, complex(a).imag), _p(X), C(complex(b).real, complex(b).imag), _p(Y))
    return Y


def scgw_iteration(cfg, vb, T_wt, T_tw, fg, H0, S, G, n_target, mu_lo, mu_hi, alpha=1.0, mu_tol=1e-12):
    """One scGW iteration in the order of Fig. 4: G(tau) -> Sigma_inf (Eq. 20, 22), Sigma~(tau) (Alg. 1) ->
    Sigma~(i omega_n) (Eq. 13) -> mu (Eq. 15) -> G(i omega_n) (Eq. 16) -> G(tau) (Eq. 14) -> damping.  fg = gwgen.make_fermionic_grids(...).
    Every step is one of the oracle's C routines; this function only sequences them."""
    Gb = transform(fg["e_beta"].reshape(1, -1), G)[0]                         # G(beta^-)
    gamma = axpby(-1.0, Gb, 0.0, np.zeros_like(Gb))                            # gamma = -G(beta^-)
    J = hartree(cfg, vb, gamma)
    K = exchange(cfg, vb, gamma)
    P0t = polarization(cfg, vb, G)
    Wt = screened_interaction(cfg, T_wt, T_tw, P0t)
    Sigma_t = selfenergy(cfg, vb, G, Wt)
    Sigma_w = transform(fg["T_wt_f"], Sigma_t)
    F = axpby(1.0, J, 1.0, axpby(1.0, K, 1.0, H0.copy()))                      # F = H0 + K + J  (Eq. 17-18)
    mu, ne = find_mu(cfg, fg["omega"], fg["t_beta"], S, F, Sigma_w, n_target, mu_lo, mu_hi, mu_tol)
    G_w = dyson_update(cfg, fg["omega"], mu, S, F, Sigma_w)
    G_new = transform(fg["T_tw_f"], G_w)
    G_mix = axpby(alpha, G_new, 1.0 - alpha, G.copy())
    return dict(gamma=gamma, J=J, K=K, P0t=P0t, Wt=Wt, Sigma_t=Sigma_t, Sigma_w=Sigma_w, F=F, mu=mu, ne=ne, G_w=G_w, G_new=G_new, G=G_mix)


# ---------------------------------------------------------------------------------------------------------------------
# collinear spin channels (PAPER.md:41 spin-orbital indices, Eq. 28b's sum over sigma sigma')
# With no spin-orbit coupling G is block diagonal in spin, G^{sigma sigma'} = delta_{sigma sigma'} G^sigma, so Eq. 28b's double
# spin sum keeps the terms sigma = sigma' only: P0 = sum_sigma P0[G^sigma]; Eq. 31 and Eq. 22 hold per channel with the common W;
# Eq. 20's sum over sigma_1 adds the channels' density matrices.  Each term is one call of the single-channel routine with
# spin_deg = 1 (the literal sum, written out).
# ---------------------------------------------------------------------------------------------------------------------
def _one_channel(cfg):
    import dataclasses
    return dataclasses.replace(cfg, spin_deg=1)


def polarization_spin(cfg, vb, Gs):
    """Eq. 28b for ns collinear channels.  Gs: [ns][ntau][nk][nao][nao]; the prefactor is cfg.spin_deg (pass 1 for ns = 2)."""
    c1 = _one_channel(cfg)
    out = None
    for sg in range(Gs.shape[0]):
        term = polarization(c1, vb, np.ascontiguousarray(Gs[sg]))
        out = term if out is None else out + term
    return cfg.spin_deg * out


def p0t_slice_spin(cfg, vb, Gs_t, Gs_tbar, q):
    c1 = _one_channel(cfg)
    return cfg.spin_deg * sum(p0t_slice(c1, vb, np.ascontiguousarray(Gs_t[sg]), np.ascontiguousarray(Gs_tbar[sg]), q) for sg in range(Gs_t.shape[0]))


def selfenergy_spin(cfg, vb, Gs, Wt):
    """Eq. 31 per channel with the common Wt."""
    return np.stack([selfenergy(cfg, vb, np.ascontiguousarray(Gs[sg]), Wt) for sg in range(Gs.shape[0])])


def exchange_spin(cfg, vb, gammas):
    """Eq. 22 per channel."""
    return np.stack([exchange(cfg, vb, np.ascontiguousarray(gammas[sg])) for sg in range(gammas.shape[0])])


def hartree_spin(cfg, vb, gammas):
    """Eq. 20: the sum over sigma_1 runs over the channels (times cfg.spin_deg)."""
    c1 = _one_channel(cfg)
    return cfg.spin_deg * sum(hartree(c1, vb, np.ascontiguousarray(gammas[sg])) for sg in range(gammas.shape[0]))


def phi_gw(nk, beta, w, phi):
    """Eq. 37 with quadrature weights w[n]: (1/(2 N_k beta)) sum_q sum_n w[n] phi[n][q]."""
    w = np.ascontiguousarray(w, dtype=np.float64); phi = np.ascontiguousarray(phi, dtype=np.float64)
    lib().gwref_phi_gw.restype = ctypes.c_double
    lib().gwref_phi_gw.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_double, ctypes.c_void_p, ctypes.c_void_p]
    return float(lib().gwref_phi_gw(int(nk), int(phi.shape[1]), int(phi.shape[0]), float(beta), _pd(w), _pd(phi)))


# two-component spin blocks (spin-orbit coupling gives G off-diagonal spin components).  Blocks in the order uu, ud, du, dd.
def polarization_blocks(cfg, vb, Gb):
    """Eq. 28b as printed: P0 = -(s/N_k) sum_{sigma sigma'} sum_k V G^{sigma sigma'}(k+q, tau) V G^{sigma' sigma}(k, -tau).
    Gb: [4][ntau][nk][nao][nao].  Every (sigma, sigma') term is one call of the single-block slice routine with G^{sigma sigma'} in the
    k+q slot and G^{sigma' sigma} in the k slot."""
    c1 = _one_channel(cfg)
    N = cfg.ntau
    out = np.zeros((N, cfg.nk, cfg.naux, cfg.naux), np.complex128)
    for t in range(N):
        for q in range(cfg.nk):
            for s in range(2):
                for sp in range(2):
                    out[t, q] += p0t_slice(c1, vb, np.ascontiguousarray(Gb[2 * s + sp][t]), np.ascontiguousarray(Gb[2 * sp + s][N - 1 - t]), q)
    return cfg.spin_deg * out


def hartree_blocks(cfg, vb, gb):
    """Eq. 20: sigma_1 runs over the spin-diagonal blocks uu and dd."""
    c1 = _one_channel(cfg)
    return cfg.spin_deg * (hartree(c1, vb, np.ascontiguousarray(gb[0])) + hartree(c1, vb, np.ascontiguousarray(gb[3])))
