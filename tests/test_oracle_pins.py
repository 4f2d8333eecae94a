"""Pins of the CPU oracle against things that are NOT the oracle.

Each test is chosen so that a plausible mistake in oracle/gwref.c (dropped term, wrong sign, wrong index,
transposed operand, wrong k±q table, wrong normalisation) fails at least one of them.
"""
import numpy as np
import pytest

import torch

import gwgen
from gwgen.configs import GWConfig
from gwgen.fock import fermi


def relerr(a, b):
    return np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300)


# ----------------------------------------------------------------------------------------------------------------
# P1: scalar closed form (north_star: "closed form for nk=1, nao=1, naux=1").
#   G(tau) = -e^{-eps tau}/(1+e^{-beta eps}); V = v real.  G(tau) G(beta-tau) = f(1-f) is tau independent, so
#   P0t = -s v^2 f(1-f);  P0w = p delta_{n0}, p = -s v^2 beta f(1-f);  Ww = p/(1-p) delta_{n0};
#   Wt = p/(beta(1-p));  Sigma(tau) = -v^2 G(tau) p/(beta(1-p));  K = -v^2 f.       (Eq. 22, 28-31 with 1x1 matrices)
# ----------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("s", [1, 2])
@pytest.mark.parametrize("eps,v,beta", [(0.37, 0.8, 10.0), (-0.11, 1.3, 25.0)])
def test_P1_scalar_closed_form(oracle_lib, s, eps, v, beta):
    N = 32
    cfg = GWConfig("P1", (1, 1, 1), 1, 1, N, N, beta, -1, 1, 0.0, 1, spin_deg=s)
    gr = gwgen.make_grids(N, N, beta)
    tau = gr["tau"]
    f = 1.0 / (1.0 + np.exp(beta * eps))
    g = -np.exp(-eps * tau) / (1.0 + np.exp(-beta * eps))
    G = g.reshape(N, 1, 1, 1).astype(np.complex128)
    V = np.full((1, 1, 1, 1, 1), v, np.complex128)
    vb = oracle_lib.VBlocks(cfg, V)
    P0t = oracle_lib.polarization(cfg, vb, G)
    assert np.allclose(P0t.ravel(), -s * v * v * f * (1 - f), rtol=1e-13, atol=0)
    Wt, P0w, Ww = oracle_lib.screened_interaction(cfg, gr["T_wt"], gr["T_tw"], P0t, want_freq=True)
    p = -s * v * v * beta * f * (1 - f)
    expect_w = np.where(gr["nbos"] == 0, p, 0.0)
    assert np.max(np.abs(P0w.ravel() - expect_w)) < 1e-11 * abs(p)
    assert np.max(np.abs(Ww.ravel() - np.where(gr["nbos"] == 0, p / (1 - p), 0.0))) < 1e-11 * max(1.0, abs(p))
    assert np.max(np.abs(Wt.ravel() - p / (beta * (1 - p)))) < 1e-10 * abs(p / (beta * (1 - p)))
    Sg = oracle_lib.selfenergy(cfg, vb, G, Wt)
    assert relerr(Sg.ravel(), -v * v * g * p / (beta * (1 - p))) < 1e-10
    K = oracle_lib.exchange(cfg, vb, np.full((1, 1, 1), f, np.complex128))
    assert abs(K.ravel()[0] - (-v * v * f)) < 1e-14


# ----------------------------------------------------------------------------------------------------------------
# P2: Lindhard closed form for a Fock-built G (textbook non-interacting polarisation in the eigenbasis):
#   Vt^Q = U_k^+ V^Q(k,k+q) U_{k+q}
#   P0(q,tau)  = -(s/Nk) sum_k sum_ca Vt^Q_ca conj(Vt^Q'_ca) f_c (1-f_a) e^{-(e_a-e_c) tau}
#   P0(q,iOm)  = -(s/Nk) sum_k sum_ca Vt^Q_ca conj(Vt^Q'_ca) (f_c-f_a)/(e_a-e_c-iOm)      (beta f_c(1-f_a) at n=0 if e_a=e_c)
# A different contraction order in a different basis; uses the generator's eps, U, and mesh tables (not the oracle's).
# ----------------------------------------------------------------------------------------------------------------
def lindhard_tau(p, q, t):
    cfg, mesh = p.cfg, p.mesh
    add = mesh.add_table()
    V = p.V.numpy()
    beta = cfg.beta
    out = np.zeros((cfg.naux, cfg.naux), complex)
    logf = lambda e: -np.logaddexp(0.0, beta * e)
    for k in range(cfg.nk):
        kq = add[k][q]
        Vt = np.einsum("dc,Qda,ab->Qcb", p.U[k].conj(), V[k, kq], p.U[kq])
        de = p.eps[kq][None, :] - p.eps[k][:, None]                       # [c][a]
        w = np.exp(logf(p.eps[k])[:, None] + logf(-p.eps[kq])[None, :] - de * p.tau[t])
        out += np.einsum("Qca,ca,Pca->QP", Vt, w, Vt.conj())
    return -cfg.spin_deg / cfg.nk * out


def lindhard_omega(p, q, ns):
    cfg, mesh = p.cfg, p.mesh
    add = mesh.add_table()
    V = p.V.numpy()
    beta = cfg.beta
    ns = np.asarray(ns)
    Om = 2 * np.pi * ns / beta
    out = np.zeros((len(ns), cfg.naux, cfg.naux), complex)
    f = fermi(p.eps, beta)
    for k in range(cfg.nk):
        kq = add[k][q]
        Vt = np.einsum("dc,Qda,ab->Qcb", p.U[k].conj(), V[k, kq], p.U[kq]).reshape(cfg.naux, -1)
        de = (p.eps[kq][None, :] - p.eps[k][:, None]).ravel()
        df = (f[k][:, None] - f[kq][None, :]).ravel()
        deg = np.abs(de) < 1e-13
        w = np.where(deg[None, :], 0.0, df[None, :] / (np.where(deg, 1.0, de)[None, :] - 1j * Om[:, None]))
        wdeg = (beta * f[k][:, None] * (1 - f[kq][None, :])).ravel()
        w = w + np.where(deg[None, :] & (ns[:, None] == 0), wdeg[None, :], 0.0)
        M = (Vt[:, None, :] * Vt.conj()[None, :, :]).reshape(cfg.naux * cfg.naux, -1)   # [(QP)][(ca)]
        out += (w @ M.T).reshape(len(ns), cfg.naux, cfg.naux)
    return -cfg.spin_deg / cfg.nk * out


@pytest.mark.parametrize("name", ["T", "R", "0"])
def test_P2_lindhard_tau(problems, oracle_results, name):
    p = problems(name)
    P0t = oracle_results(name)["P0t"]
    rng = np.random.default_rng(5)
    for _ in range(6):
        q = int(rng.integers(p.cfg.nk)); t = int(rng.integers(p.cfg.ntau))
        assert relerr(P0t[t, q], lindhard_tau(p, q, t)) < 1e-12


def test_P2_lindhard_omega(problems, oracle_results):
    # stage 2a to the accuracy of the grid: beta=10, N=32 gives ~1e-12
    p = problems("T")
    P0w = oracle_results("T")["P0w"]
    for q in range(p.cfg.nk):
        assert relerr(P0w[:, q], lindhard_omega(p, q, p.nbos)) < 1e-10


# ----------------------------------------------------------------------------------------------------------------
# P3: definiteness / Hermiticity end to end (sign reading R1 of DESIGN.md): P0t <= 0 Hermitian, I - P0w HPD with
# eigenvalues >= 1 (what the paper's *Cholesky* solver needs), Ww in (-1,0], -Sigma >= 0, -K >= 0.
# ----------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("name", ["T", "R"])
def test_P3_definiteness(problems, oracle_results, name):
    cfg = problems(name).cfg
    r = oracle_results(name)
    herm = lambda A: np.abs(A - np.conj(np.swapaxes(A, -1, -2))).max() / np.abs(A).max()
    for key in ("P0t", "P0w", "Ww", "Wt", "Sigma", "K"):
        assert herm(r[key]) < 1e-12, key
    tol = 1e-12
    assert max(np.linalg.eigvalsh(r["P0t"][t, q]).max() for t in range(cfg.ntau) for q in range(cfg.nk)) < tol
    I = np.eye(cfg.naux)
    assert min(np.linalg.eigvalsh(I - r["P0w"][n, q]).min() for n in range(cfg.nw) for q in range(cfg.nk)) > 1 - 1e-9
    ev = np.array([np.linalg.eigvalsh(r["Ww"][n, q]) for n in range(cfg.nw) for q in range(cfg.nk)])
    assert ev.max() < 1e-9 and ev.min() > -1.0
    assert max(np.linalg.eigvalsh(r["Sigma"][t, k]).max() for t in range(cfg.ntau) for k in range(cfg.nk)) < tol
    assert max(np.linalg.eigvalsh(r["K"][k]).max() for k in range(cfg.nk)) < tol


# ----------------------------------------------------------------------------------------------------------------
# P4: P0^{-q}_{Q'Q}(tau_t) = P0^{q}_{QQ'}(tau_{tbar}) (always); P0^q(tau_tbar) = P0^q(tau_t) under TR inputs.
# P5: north_star's checks: Sigma_ij(k,tau) = conj Sigma_ji(k,tau); Sigma(-k) = Sigma(k)^*.
# ----------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("name", ["T", "R"])
def test_P4_P5_symmetries(problems, oracle_results, name):
    p = problems(name)
    r = oracle_results(name)
    neg = p.mesh.neg()
    P0t, Sg, K = r["P0t"], r["Sigma"], r["K"]
    assert relerr(np.swapaxes(P0t[:, neg], -1, -2), P0t[::-1]) < 1e-13
    assert relerr(P0t[::-1], P0t) < 1e-13
    assert relerr(np.conj(np.swapaxes(Sg, -1, -2)), Sg) < 1e-13
    assert relerr(Sg[:, neg], np.conj(Sg)) < 1e-13
    assert relerr(K[neg], np.conj(K)) < 1e-13


def test_P4_mesh_tables_match_generator(problems, oracle_lib):
    # the oracle has its own k±q arithmetic; the generator another; they must agree (3x2x2 mesh: odd and even dims)
    p = problems("R")
    add, sub = p.mesh.add_table(), p.mesh.sub_table()
    for k in range(p.cfg.nk):
        for q in range(p.cfg.nk):
            assert oracle_lib.kadd(p.cfg, k, q) == add[k][q]
            assert oracle_lib.ksub(p.cfg, k, q) == sub[k][q]
    assert add[sub[5][3]][3] == 5


# ----------------------------------------------------------------------------------------------------------------
# P6: brute force on the tiny config T: exact P0(iOm_n) (Lindhard) for |n| <= 4e5 -> Dyson per n -> explicit
# Matsubara sum Wt(tau_t) = (1/beta) sum_n W(iOm_n) e^{-iOm_n tau_t} (Eq. 29, 30) -> compared with the oracle's
# sparse-grid pipeline (Eq. 28a matrix, LU, Eq. 30 matrix).  Pins the transform pair and Dyson as physics.
# ----------------------------------------------------------------------------------------------------------------
def test_P6_bruteforce_matsubara(problems, oracle_results):
    p = problems("T")
    cfg = p.cfg
    Wt = oracle_results("T")["Wt"]
    nb, chunk = 400000, 50000
    I = np.eye(cfg.naux)
    ref = np.zeros_like(Wt)
    for q in range(cfg.nk):
        acc = np.zeros((cfg.ntau, cfg.naux, cfg.naux), complex)
        for lo in range(-nb, nb + 1, chunk):
            nn = np.arange(lo, min(lo + chunk, nb + 1))
            Pn = lindhard_omega(p, q, nn)
            Wn = np.linalg.solve(I[None] - Pn, Pn)
            ph = np.exp(-1j * np.outer(p.tau, 2 * np.pi * nn / cfg.beta))
            acc += np.tensordot(ph, Wn, axes=(1, 0))
        ref[:, q] = acc / cfg.beta
    assert relerr(Wt, ref) < 1e-8


# ----------------------------------------------------------------------------------------------------------------
# P7: trace identity tying stage 3 to stage 1 (exact at every tau node, for arbitrary Wt):
#   sum_k tr[Sigma[t][k] G[tbar][k]] = (1/s) sum_q tr[Wt[t][q] P0t[tbar][q]]
# ----------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("name", ["T", "R", "0"])
def test_P7_trace_identity(problems, oracle_results, oracle_lib, name):
    p = problems(name)
    cfg = p.cfg
    r = oracle_results(name)
    rng = np.random.default_rng(11)
    # arbitrary (non-physical, non-Hermitian) W to make the identity bite on index order
    Wr = rng.normal(size=r["Wt"].shape) + 1j * rng.normal(size=r["Wt"].shape)
    vb = oracle_lib.VBlocks(cfg, p.V.numpy())
    for W, Sg in ((r["Wt"], r["Sigma"]), (Wr, oracle_lib.selfenergy(cfg, vb, p.G, Wr))):
        lhs = np.einsum("tkij,tkji->t", Sg, p.G[::-1])
        rhs = np.einsum("tqab,tqba->t", W, r["P0t"][::-1]) / cfg.spin_deg
        assert np.max(np.abs(lhs - rhs) / np.abs(rhs)) < 1e-12


# ----------------------------------------------------------------------------------------------------------------
# P8: residual of the solve, independent of the oracle's LU: (I - P0w) Ww = P0w and Ww = (I - P0w)^-1 - I (Eq. 29)
# ----------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("name", ["T", "R"])
def test_P8_dyson_residual(problems, oracle_results, name):
    cfg = problems(name).cfg
    r = oracle_results(name)
    I = np.eye(cfg.naux)
    for n in range(cfg.nw):
        for q in range(cfg.nk):
            P, W = r["P0w"][n, q], r["Ww"][n, q]
            assert np.linalg.norm((I - P) @ W - P) <= 1e-13 * max(np.linalg.norm(P), 1e-300) + 1e-300
            assert relerr(W, np.linalg.inv(I - P) - I) < 1e-10 or np.linalg.norm(W) < 1e-12


def test_P8_dyson_nonhermitian_pivoting(oracle_lib):
    # generic complex matrix that needs row exchanges
    rng = np.random.default_rng(3)
    P = rng.normal(size=(9, 9)) + 1j * rng.normal(size=(9, 9))
    P[0, 0] = 1.0   # makes (I-P)[0,0] exactly zero -> first pivot must be exchanged
    X = oracle_lib.dyson(P)
    assert relerr(X, np.linalg.solve(np.eye(9) - P, P)) < 1e-12


def test_transform_matches_definition(problems, oracle_results):
    # Eq. 28a / Eq. 30 as matrix applications (numpy tensordot = re-statement with a library routine on the same matrices)
    p = problems("R")
    r = oracle_results("R")
    assert relerr(r["P0w"], np.tensordot(p.T_wt, r["P0t"], axes=(1, 0))) < 1e-13
    assert relerr(r["Wt"], np.tensordot(p.T_tw, r["Ww"], axes=(1, 0))) < 1e-13


def test_transform_rows_integrate_constants(problems):
    # normalisation of Eq. 28a: sum_t T_wt[n][t] = beta delta_{n0}; Eq. 30 maps a constant in Omega_0 to 1/beta
    for name in ("0", "T", "1"):
        cfg = gwgen.get_config(name)
        gr = gwgen.make_grids(cfg.ntau, cfg.nw, cfg.beta)
        rs = gr["T_wt"].sum(axis=1)
        assert abs(rs[0] - cfg.beta) < 1e-12 * cfg.beta
        assert np.abs(rs[1:]).max() < 1e-11 * cfg.beta
        assert np.allclose(gr["tau"][::-1], cfg.beta - gr["tau"], rtol=0, atol=4e-16 * cfg.beta)
        e0 = np.zeros(cfg.nw); e0[0] = 1.0
        assert np.abs(gr["T_tw"] @ e0 - 1.0 / cfg.beta).max() < 1e-10 / cfg.beta


# ----------------------------------------------------------------------------------------------------------------
# P9: exchange limit cross-checks two entry points: Eq. 31 with G := -gamma and W := I equals -K of Eq. 22.
# ----------------------------------------------------------------------------------------------------------------
def test_P9_exchange_limit(problems, oracle_results, oracle_lib):
    p = problems("R")
    cfg = p.cfg
    vb = oracle_lib.VBlocks(cfg, p.V.numpy())
    I = np.ascontiguousarray(np.broadcast_to(np.eye(cfg.naux, dtype=complex), (cfg.nk, cfg.naux, cfg.naux)))
    for k in (0, 3, cfg.nk - 1):
        S = oracle_lib.sigma_slice(cfg, vb, np.ascontiguousarray(-p.gamma), I, k)
        assert relerr(S, -oracle_results("R")["K"][k]) < 1e-13


# ----------------------------------------------------------------------------------------------------------------
# P10: literal 4-index evaluation of Eq. 28b / 31 / 22 (no temporaries) with numpy einsum, using the generator's tables.
# ----------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("name", ["T", "0"])
def test_P10_literal_einsum(problems, oracle_results, name):
    p = problems(name)
    cfg = p.cfg
    r = oracle_results(name)
    V = p.V.numpy()
    add, sub = p.mesh.add_table(), p.mesh.sub_table()
    N, nk = cfg.ntau, cfg.nk
    S = np.zeros_like(r["Sigma"]); K = np.zeros_like(r["K"])
    for t in range(N):
        for k in range(nk):
            for q in range(nk):
                km = sub[k][q]
                S[t, k] += np.einsum("ab,Qia,QP,Pbj->ij", p.G[t, km], V[k, km], r["Wt"][t, q], V[km, k])
    S *= -1.0 / nk
    for k in range(nk):
        for kp in range(nk):
            K[k] += np.einsum("Qia,ab,Qbj->ij", V[k, kp], p.gamma[kp], V[kp, k])
    K *= -1.0 / nk
    assert relerr(r["Sigma"], S) < 1e-13
    assert relerr(r["K"], K) < 1e-13
    # Eq. 28b, reading R1 of DESIGN.md: the printed "-1/Nk" is the antiperiodicity sign of G(-tau) = -G(beta-tau),
    # so the array contracted is G[tbar] and P0t = -(s/Nk) sum_k V G^k[tbar] G^{k+q}[t] V  (index pattern exactly as printed).
    lit = np.zeros_like(r["P0t"])
    for t in range(N):
        for q in range(nk):
            for k in range(nk):
                kq = add[k][q]
                lit[t, q] += np.einsum("Qda,cd,ab,Pbc->QP", V[k, kq], p.G[N - 1 - t, k], p.G[t, kq], V[kq, k])
    lit *= -cfg.spin_deg / nk
    assert relerr(r["P0t"], lit) < 1e-13


# ---- P11: summand of Eq. 37, phi = tr{ln[I - P] + P} ----
def test_P11_phi_scalar_and_series(oracle_lib):
    """Closed form for a 1x1 matrix, and the paper's own expansion (first line of Eq. 37):
    tr{ln[I-P]+P} = -Σ_{m>=2} tr(P^m)/m, evaluated by explicit matrix powers for a small-norm Hermitian P."""
    for pval in (-3.7, -0.2, 0.5):
        got = oracle_lib.phi(np.array([[pval]], dtype=np.complex128))
        assert abs(got - (np.log(1.0 - pval) + pval)) <= 1e-14 * max(1.0, abs(pval))
    rng = np.random.default_rng(5)
    n = 9
    A = rng.normal(size=(n, n)) + 1j * rng.normal(size=(n, n))
    P = -(A @ A.conj().T)
    P *= 0.3 / np.linalg.norm(P, 2)                       # spectral radius 0.3: the series converges fast
    series, Pm = 0.0, P.copy()
    for m in range(2, 80):
        Pm = Pm @ P
        series -= np.trace(Pm).real / m
    assert abs(oracle_lib.phi(P) - series) <= 1e-13


def test_P11_phi_matches_eigenvalues(problems, oracle_results, oracle_lib):
    """On real stage-2 data (config T): tr ln[I-P0w] + tr P0w = Σ_i ln(1-λ_i) + λ_i over the eigenvalues of the
    Hermitian P0w (a different route than the oracle's LU pivots); the (I-P)^2 term of Eq. 36 bounds it from below."""
    P0w = oracle_results("T")["P0w"]
    for n in (0, 3, 17):
        for q in (0, 4):
            P = P0w[n, q]
            lam = np.linalg.eigvalsh(0.5 * (P + P.conj().T))
            ref = float(np.sum(np.log1p(-lam) + lam))
            got = oracle_lib.phi(P)
            assert abs(got - ref) <= 1e-12 * max(1.0, abs(ref))
            assert got <= 1e-14 and got >= -0.5 * np.sum(lam ** 2) - 1e-12     # ln(1-x)+x in [-x²/2, 0] for x <= 0


# ---- P12: fermionic tau -> i omega_n transform (Eq. 13), the step after the hot path ----
def test_P12_fermionic_transform_closed_form(oracle_lib):
    """G(tau) = -e^{-eps tau}/(1+e^{-beta eps}) transforms to 1/(i omega_n - eps): pins the generator's fermionic matrix and the
    oracle's transform routine (sign of the exponent, omega_n = (2n+1) pi / beta, the beta/2 Jacobian) against a closed form."""
    import gwgen
    beta, N = 10.0, 32
    g = gwgen.make_grids(N, N, beta)
    f = gwgen.make_fermionic_transform(N, beta)
    eps = np.array([0.7, -0.3, 0.05])
    G = (-np.exp(-np.outer(g["tau"], eps)) / (1.0 + np.exp(-beta * eps))).astype(np.complex128)    # [ntau][3]
    got = oracle_lib.transform(f["T_wt_f"], G)
    ref = 1.0 / (1j * f["omega"][:, None] - eps[None, :])
    assert np.max(np.abs(got - ref) / np.abs(ref)) < 1e-9
    assert np.allclose(got, np.tensordot(f["T_wt_f"], G, axes=(1, 0)), rtol=1e-13, atol=0)


# ----------------------------------------------------------------------------------------------------------------
# Raw-input pins (no symmetry in V, G, gamma, W): the printed index patterns of Eq. 22 / 28b / 31 are told apart from
# their symmetric twins.  On the BASELINE inputs V[k+q][k]_bc = conj V[k][k+q]_cb and G = G^+, so an oracle that read the
# conjugate-transposed block, or G^+ in place of G, would pass P2-P10 above; on raw inputs it fails by O(1).
# ----------------------------------------------------------------------------------------------------------------
def _raw_oracle(oracle_lib, p):
    cfg = p.cfg
    vb = oracle_lib.VBlocks(cfg, p.V.numpy())
    P0t = oracle_lib.polarization(cfg, vb, p.G)
    Sg = oracle_lib.selfenergy(cfg, vb, p.G, p.extras["W"])
    K = oracle_lib.exchange(cfg, vb, p.gamma)
    return vb, P0t, Sg, K


def test_raw_inputs_have_no_symmetry(raw_problems):
    p = raw_problems("T")
    V = p.V.numpy()
    neg = p.mesh.neg()
    assert relerr(V[1, 2], np.conj(np.swapaxes(V[2, 1], -1, -2))) > 0.5          # no pair symmetry
    assert relerr(V[neg[1], neg[2]], np.conj(V[1, 2])) > 0.5                      # no time reversal
    assert relerr(p.G, np.conj(np.swapaxes(p.G, -1, -2))) > 0.5                   # G not Hermitian
    assert relerr(p.extras["W"], np.conj(np.swapaxes(p.extras["W"], -1, -2))) > 0.5


def test_P10_literal_einsum_raw(raw_problems, oracle_lib):
    """Eq. 28b / 31 / 22 exactly as printed, 4-index einsum with the generator's tables,
    on symmetry-free inputs; and the symmetric twins are shown to differ, so the pin bites."""
    p = raw_problems("T")
    cfg = p.cfg
    vb, P0t, Sg, K = _raw_oracle(oracle_lib, p)
    V, G, W = p.V.numpy(), p.G, p.extras["W"]
    add, sub = p.mesh.add_table(), p.mesh.sub_table()
    N, nk = cfg.ntau, cfg.nk
    lit = np.zeros_like(P0t); twin_V = np.zeros_like(P0t); twin_G = np.zeros_like(P0t)
    for t in range(N):
        for q in range(nk):
            for k in range(nk):
                kq = add[k][q]
                lit[t, q] += np.einsum("Qda,cd,ab,Pbc->QP", V[k, kq], G[N - 1 - t, k], G[t, kq], V[kq, k])
                twin_V[t, q] += np.einsum("Qda,cd,ab,Pcb->QP", V[k, kq], G[N - 1 - t, k], G[t, kq], V[k, kq].conj())
                twin_G[t, q] += np.einsum("Qda,dc,ab,Pbc->QP", V[k, kq], G[N - 1 - t, k].conj(), G[t, kq], V[kq, k])
    pref = -cfg.spin_deg / nk
    assert relerr(P0t, pref * lit) < 1e-13
    assert relerr(P0t, pref * twin_V) > 0.5 and relerr(P0t, pref * twin_G) > 0.5
    S = np.zeros_like(Sg); S_twin = np.zeros_like(Sg); Kl = np.zeros_like(K); K_twin = np.zeros_like(K)
    for k in range(nk):
        for q in range(nk):
            km = sub[k][q]
            for t in range(N):
                S[t, k] += np.einsum("ab,Qia,QP,Pbj->ij", G[t, km], V[k, km], W[t, q], V[km, k])
                S_twin[t, k] += np.einsum("ab,Qia,PQ,Pbj->ij", G[t, km], V[k, km], W[t, q], V[km, k])     # W transposed
            Kl[k] += np.einsum("Qia,ab,Qbj->ij", V[k, km], p.gamma[km], V[km, k])
            K_twin[k] += np.einsum("Qia,ab,Qjb->ij", V[k, km], p.gamma[km], V[k, km].conj())            # V[k'][k] -> V[k][k']^+
    assert relerr(Sg, -S / nk) < 1e-13 and relerr(Sg, -S_twin / nk) > 0.5
    assert relerr(K, -Kl / nk) < 1e-13 and relerr(K, -K_twin / nk) > 0.5


@pytest.mark.parametrize("name", ["T", "R"])
def test_P7_P9_raw(raw_problems, oracle_lib, name):
    """Trace identity (P7) and exchange limit (P9) hold for ARBITRARY inputs: checked on the symmetry-free ones."""
    p = raw_problems(name)
    cfg = p.cfg
    vb, P0t, Sg, K = _raw_oracle(oracle_lib, p)
    lhs = np.einsum("tkij,tkji->t", Sg, p.G[::-1])
    rhs = np.einsum("tqab,tqba->t", p.extras["W"], P0t[::-1]) / cfg.spin_deg
    assert np.max(np.abs(lhs - rhs) / np.abs(rhs)) < 1e-11
    I = np.ascontiguousarray(np.broadcast_to(np.eye(cfg.naux, dtype=complex), (cfg.nk, cfg.naux, cfg.naux)))
    for k in (0, cfg.nk - 1):
        S = oracle_lib.sigma_slice(cfg, vb, np.ascontiguousarray(-p.gamma), I, k)
        assert relerr(S, -K[k]) < 1e-13


# ----------------------------------------------------------------------------------------------------------------
# Loop closure: Eq. 15, 16, 20 and the chemical-potential search.
# ----------------------------------------------------------------------------------------------------------------
def _closure_inputs(p):
    cfg = p.cfg
    H0, S = gwgen.make_h0_s(cfg, p.mesh, p.eps, p.U)
    fg = gwgen.make_fermionic_grids(cfg.ntau, cfg.beta)
    return H0, S, fg


def test_P13_dyson_noninteracting_closed_form(problems, oracle_lib):
    """Sigma = 0: G(i omega_n) = [(i omega_n + mu) S - H0]^-1 = C diag(1/(i omega_n + mu - e)) C^+ with the generalised eigenpairs
    H0 C = S C e, C^+ S C = 1 (scipy.linalg.eigh, another basis and a library routine), and with a self-energy: A G = 1."""
    import scipy.linalg as sla
    p = problems("R")
    cfg = p.cfg
    H0, S, fg = _closure_inputs(p)
    mu = 0.137
    G_w = oracle_lib.dyson_update(cfg, fg["omega"], mu, S, H0)
    for k in (0, 5, cfg.nk - 1):
        e, C = sla.eigh(H0[k], S[k])
        for n in (0, len(fg["omega"]) // 2, len(fg["omega"]) - 1):
            ref = (C / (1j * fg["omega"][n] + mu - e)[None, :]) @ C.conj().T
            assert relerr(G_w[n, k], ref) < 1e-12
    rng = np.random.default_rng(2)
    Sw = rng.normal(size=G_w.shape) + 1j * rng.normal(size=G_w.shape)          # arbitrary (non-Hermitian) Sigma~(i omega_n)
    G2 = oracle_lib.dyson_update(cfg, fg["omega"], mu, S, H0, Sw)
    for n in (0, 7):
        for k in (1, 4):
            A = (1j * fg["omega"][n] + mu) * S[k] - H0[k] - Sw[n, k]
            assert np.linalg.norm(A @ G2[n, k] - np.eye(cfg.nao)) < 1e-12 * np.linalg.norm(A) * np.linalg.norm(G2[n, k])


def test_P14_electron_count_and_mu(problems, oracle_lib):
    """Sigma = 0 (config T: beta = 10, 32 nodes, where the grid is accurate to ~1e-9): Eq. 15 gives N_e(mu) = (s/N_k) sum_k sum_i
    f(e_i^k - mu) with the generalised eigenvalues, and the chemical-potential search lands on the root of that closed form
    (scipy.optimize.brentq)."""
    import scipy.linalg as sla
    import scipy.optimize as sop
    p = problems("T")
    cfg = p.cfg
    H0, S, fg = _closure_inputs(p)
    ev = np.array([sla.eigh(H0[k], S[k], eigvals_only=True) for k in range(cfg.nk)])
    ne_ref = lambda mu: cfg.spin_deg / cfg.nk * float(np.sum(1.0 / (1.0 + np.exp(cfg.beta * (ev - mu)))))
    for mu in (-0.4, 0.0, 0.3):
        G_w = oracle_lib.dyson_update(cfg, fg["omega"], mu, S, H0)
        assert abs(oracle_lib.electron_count(cfg, fg["t_beta"], S, G_w) - ne_ref(mu)) < 1e-8
    target = cfg.spin_deg * 1.25                               # 2.5 electrons per cell: mu inside the band
    mu, ne = oracle_lib.find_mu(cfg, fg["omega"], fg["t_beta"], S, H0, None, target, -0.1, 0.1)      # bracket must be widened
    mu_ref = sop.brentq(lambda m: ne_ref(m) - target, -5.0, 5.0, xtol=1e-14)
    assert abs(ne - target) < 1e-9                             # the paper's threshold
    assert abs(mu - mu_ref) < 1e-7
    # gamma from G(tau) (e_beta) and from G(i omega_n) (t_beta) agree: the two evaluation vectors are consistent with the transform pair
    G_w = oracle_lib.dyson_update(cfg, fg["omega"], mu, S, H0)
    Gb_w = np.tensordot(fg["t_beta"], G_w, axes=(0, 0))
    Gb_t = np.tensordot(fg["e_beta"], oracle_lib.transform(fg["T_tw_f"], G_w), axes=(0, 0))
    assert relerr(Gb_t, Gb_w) < 1e-8


def test_P15_hartree_literal_einsum(problems, raw_problems, oracle_lib):
    """Eq. 20 as printed, numpy einsum over the diagonal blocks, on symmetric and on symmetry-free inputs."""
    for p in (problems("R"), raw_problems("T")):
        cfg = p.cfg
        V = p.V.numpy()
        Vd = np.stack([V[k, k] for k in range(cfg.nk)])                      # [k][Q][i][j]
        rho = np.einsum("kab,kQba->Q", p.gamma, Vd)
        ref = cfg.spin_deg / cfg.nk * np.einsum("kQij,Q->kij", Vd, rho)
        assert relerr(oracle_lib.hartree(cfg, oracle_lib.VBlocks(cfg, V), p.gamma), ref) < 1e-13


def test_P16_fermionic_back_transform_closed_form(oracle_lib):
    """1/(i omega_n - eps) -> -e^{-eps tau}/(1+e^{-beta eps}) (Eq. 14) and its value at beta^-; forward transform (Eq. 13) back again."""
    beta, N = 10.0, 32
    g = gwgen.make_grids(N, N, beta)
    fg = gwgen.make_fermionic_grids(N, beta)
    assert np.array_equal(fg["nfer"], -fg["nfer"][::-1] - 1)                 # symmetric under omega_n -> -omega_n
    assert np.allclose(fg["omega"], (2 * fg["nfer"] + 1) * np.pi / beta, rtol=1e-15)
    eps = np.array([0.7, -0.3, 0.05])
    Gw = np.ascontiguousarray(1.0 / (1j * fg["omega"][:, None] - eps[None, :]))
    ref = -np.exp(-np.outer(g["tau"], eps)) / (1.0 + np.exp(-beta * eps))
    assert np.max(np.abs(oracle_lib.transform(fg["T_tw_f"], Gw) - ref)) < 1e-9
    assert np.max(np.abs(oracle_lib.transform(fg["t_beta"].reshape(1, -1), Gw)[0] + 1.0 / (1.0 + np.exp(beta * eps)))) < 1e-9
    assert np.max(np.abs(oracle_lib.transform(fg["e_beta"].reshape(1, -1), ref.astype(complex))[0] + 1.0 / (1.0 + np.exp(beta * eps)))) < 1e-9
    assert np.max(np.abs(oracle_lib.transform(fg["T_wt_f"], ref.astype(complex)) - Gw)) < 1e-9


def test_P17_scgw_iteration_noninteracting_limit(problems, oracle_lib):
    """V = 0: one iteration of Fig. 4 returns the non-interacting Green's function of (H0, S) at the chemical potential of the
    Fermi-function count, whatever G went in: G(tau) = -C diag(e^{-(e-mu) tau}/(1+e^{-beta(e-mu)})) C^+."""
    import scipy.linalg as sla
    import scipy.optimize as sop
    p = problems("T")
    cfg = p.cfg
    H0, S, fg = _closure_inputs(p)
    V0 = np.zeros(tuple(p.V.shape), np.complex128)
    target = cfg.spin_deg * 1.5
    r = oracle_lib.scgw_iteration(cfg, oracle_lib.VBlocks(cfg, V0), p.T_wt, p.T_tw, fg, H0, S, p.G, target, -1.0, 1.0)
    ev = [sla.eigh(H0[k], S[k]) for k in range(cfg.nk)]
    mu_ref = sop.brentq(lambda m: cfg.spin_deg / cfg.nk * sum(np.sum(1.0 / (1.0 + np.exp(cfg.beta * (e - m)))) for e, _ in ev) - target, -5, 5, xtol=1e-14)
    assert abs(r["mu"] - mu_ref) < 1e-7
    assert np.abs(r["Sigma_t"]).max() == 0.0 and np.abs(r["J"]).max() == 0.0
    for k in range(cfg.nk):
        e, C = ev[k]
        x = e - mu_ref
        g = -np.exp(-np.outer(p.tau, x)) / (1.0 + np.exp(-cfg.beta * x))
        ref = np.einsum("in,tn,jn->tij", C, g, C.conj())
        assert np.max(np.abs(r["G_new"][:, k] - ref)) < 1e-7


# ----------------------------------------------------------------------------------------------------------------
# Collinear spin channels: the oracle's spin routines are the literal sum over sigma of the
# single-channel ones.  Pins: two identical channels == closed shell; two different channels == the Lindhard closed form summed
# over the channels' own spectra; Eq. 20's sigma_1 sum by einsum.
# ----------------------------------------------------------------------------------------------------------------
def test_P18_two_identical_channels_equal_closed_shell(problems, oracle_results, oracle_lib):
    import dataclasses
    p = problems("T")
    cfg1 = dataclasses.replace(p.cfg, spin_deg=1)
    vb = oracle_lib.VBlocks(p.cfg, p.V.numpy())
    ref = oracle_results("T")
    G2 = np.ascontiguousarray(np.stack([p.G, p.G])); g2 = np.ascontiguousarray(np.stack([p.gamma, p.gamma]))
    assert relerr(oracle_lib.polarization_spin(cfg1, vb, G2), ref["P0t"]) < 1e-15          # spin_deg = 2 of the closed shell
    S2 = oracle_lib.selfenergy_spin(cfg1, vb, G2, ref["Wt"])
    K2 = oracle_lib.exchange_spin(cfg1, vb, g2)
    for sg in range(2):
        assert np.array_equal(S2[sg], ref["Sigma"]) and np.array_equal(K2[sg], ref["K"])
    assert relerr(oracle_lib.hartree_spin(cfg1, vb, g2), oracle_lib.hartree(p.cfg, vb, p.gamma)) < 1e-15


def test_P19_spin_polarised_lindhard_and_hartree(problems, oracle_lib):
    import copy
    import dataclasses
    p = problems("T")
    cfg1 = dataclasses.replace(p.cfg, spin_deg=1)
    Gs, gs = gwgen.make_spin_channels(p, 2)
    assert relerr(Gs[1], Gs[0]) > 0.1                                                      # the channels really differ
    vb = oracle_lib.VBlocks(p.cfg, p.V.numpy())
    P0 = oracle_lib.polarization_spin(cfg1, vb, Gs)
    chans = []
    for ch in range(2):
        pc = copy.copy(p)
        pc.cfg = cfg1
        pc.eps, pc.U = gwgen.make_fock(p.cfg, p.mesh, channel=ch)
        chans.append(pc)
    rng = np.random.default_rng(8)
    for _ in range(4):
        q, t = int(rng.integers(p.cfg.nk)), int(rng.integers(p.cfg.ntau))
        ref = lindhard_tau(chans[0], q, t) + lindhard_tau(chans[1], q, t)
        assert relerr(P0[t, q], ref) < 1e-12
        assert relerr(oracle_lib.p0t_slice_spin(cfg1, vb, Gs[:, t], Gs[:, p.cfg.ntau - 1 - t], q), P0[t, q]) < 1e-15
    V = p.V.numpy()
    Vd = np.stack([V[k, k] for k in range(p.cfg.nk)])
    rho = np.einsum("skab,kQba->Q", gs, Vd)
    assert relerr(oracle_lib.hartree_spin(cfg1, vb, gs), np.einsum("kQij,Q->kij", Vd, rho) / p.cfg.nk) < 1e-13


def test_qslab_layout_is_a_pure_gather(problems):
    """gwgen.to_qslab (the GW_V_QSLAB layout of include/gw.h) only moves blocks: slot (q, k, 0) = V[k][k+q], slot (q, k, 1) = V[k+q][k]."""
    p = problems("R")
    add = p.mesh.add_table()
    S = gwgen.to_qslab(p.V, p.mesh, 3, 9)
    for q in (3, 5, 8):
        for k in (0, 4, p.cfg.nk - 1):
            kq = int(add[k][q])
            assert torch.equal(S[q - 3, k, 0], p.V[k, kq]) and torch.equal(S[q - 3, k, 1], p.V[kq, k])


def test_P20_phi_gw_scalar_closed_form_and_definition(oracle_lib):
    """Eq. 37 summed with quadrature weights.  Scalar model of P1 (nk = nao = naux = 1, single pole): P0(i Omega_n) = p delta_n0 with
    p = -s v^2 beta f (1 - f), so Phi~_GW = (1/(2 beta)) w_0 [ln(1 - p) + p]; and the plain double sum on random data."""
    beta, eps, v, s = 10.0, 0.3, 0.7, 2
    f = 1.0 / (1.0 + np.exp(beta * eps))
    p = -s * v * v * beta * f * (1.0 - f)
    nw = 5
    w = np.array([1.0, 2.0, 2.0, 2.0, 2.0])
    phi = np.zeros((nw, 1))
    for n in range(nw):
        phi[n, 0] = oracle_lib.phi(np.array([[p if n == 0 else 0.0]], dtype=np.complex128))
    assert abs(oracle_lib.phi_gw(1, beta, w, phi) - (np.log(1.0 - p) + p) / (2.0 * beta)) < 1e-15
    rng = np.random.default_rng(4)
    w = rng.uniform(0.5, 2.0, 7); phi = rng.normal(size=(7, 11))
    assert abs(oracle_lib.phi_gw(12, 3.0, w, phi) - np.einsum("n,nq->", w, phi) / (2 * 12 * 3.0)) < 1e-14


def test_P21_two_component_blocks_spin_rotation(problems, oracle_lib):
    """Two-component blocks (uu, ud, du, dd) built from two collinear channels by one global SU(2) rotation R: the spin trace of Eq. 28b
    is rotation invariant, so P0[blocks] = P0[collinear] (pinned by P19); Sigma and K are linear in G with a spin-independent W, so
    their blocks are the rotated per-channel results; J sees the spin trace of gamma only."""
    import dataclasses
    p = problems("T")
    cfg1 = dataclasses.replace(p.cfg, spin_deg=1)
    vb = oracle_lib.VBlocks(p.cfg, p.V.numpy())
    Gs, gs = gwgen.make_spin_channels(p, 2)
    Gb, gb, R = gwgen.rotate_spin_channels(Gs, gs)
    assert relerr(R @ R.conj().T, np.eye(2)) < 1e-15 and np.abs(Gb[1]).max() > 0.05 * np.abs(Gb[0]).max()      # unitary; off-diagonal blocks present
    P_col = oracle_lib.polarization_spin(cfg1, vb, Gs)
    assert relerr(oracle_lib.polarization_blocks(cfg1, vb, Gb), P_col) < 1e-13
    Wt = oracle_lib.screened_interaction(cfg1, p.T_wt, p.T_tw, P_col)
    S_col = oracle_lib.selfenergy_spin(cfg1, vb, Gs, Wt)
    S_blk = oracle_lib.selfenergy_spin(cfg1, vb, Gb, Wt)
    K_col, K_blk = oracle_lib.exchange_spin(cfg1, vb, gs), oracle_lib.exchange_spin(cfg1, vb, gb)
    for s in range(2):
        for sp in range(2):
            rot = lambda X: sum(R[s, c] * X[c] * np.conj(R[sp, c]) for c in range(2))
            assert relerr(S_blk[2 * s + sp], rot(S_col)) < 1e-13 and relerr(K_blk[2 * s + sp], rot(K_col)) < 1e-13
    assert relerr(oracle_lib.hartree_blocks(cfg1, vb, gb), oracle_lib.hartree_spin(cfg1, vb, gs)) < 1e-13
