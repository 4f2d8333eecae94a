"""GPU parity of the loop closure (Eq. 15, 16, 20 and Fig. 4): every C-ABI call against the oracle's
routine on the same seeded inputs, then one whole scGW iteration G -> Sigma -> G' on configs T and R."""
import numpy as np
import pytest
import torch

import gwgen
from parity import relerr, device_problem, report

pytestmark = pytest.mark.gpu
TOL = 1e-10


def _closure(p):
    cfg = p.cfg
    H0, S = gwgen.make_h0_s(cfg, p.mesh, p.eps, p.U)
    fg = gwgen.make_fermionic_grids(cfg.ntau, cfg.beta)
    dfg = {k: torch.from_numpy(np.ascontiguousarray(v)).cuda() for k, v in fg.items() if k in ("omega", "T_wt_f", "T_tw_f", "t_beta", "e_beta")}
    return H0, S, fg, dfg


@pytest.mark.parametrize("name,raw", [("T", False), ("R", False), ("L", False), ("T", True), ("R", True)])
def test_hartree_parity(problems, raw_problems, oracle_lib, name, raw):
    """Eq. 20 on symmetric and on symmetry-free inputs (nao = 3, 7, 52)."""
    import paper_2206_07660_b200 as gw
    p = raw_problems(name) if raw else problems(name)
    prob, _, gamma = device_problem(p)
    J = gw.gw_hartree(prob, gamma).cpu().numpy()
    ref = oracle_lib.hartree(p.cfg, oracle_lib.VBlocks(p.cfg, p.V.numpy()), p.gamma)
    assert report(name + ("-raw" if raw else ""), "J", J, ref) <= TOL


@pytest.mark.parametrize("name", ["T", "R", "S", "L", "N64"])
def test_dyson_update_parity(problems, oracle_lib, name):
    """Eq. 16 with an arbitrary non-Hermitian Sigma~(i omega_n) (nao = 3, 7, 26, 52 and the documented maximum 64), and with none."""
    import paper_2206_07660_b200 as gw
    if name == "N64":
        cfg = gwgen.GWConfig("cfgN64", (2, 1, 1), 64, 8, 12, 12, 20.0, -1.0, 1.0, 0.0, 220607660 + 64)
        mesh = gwgen.KMesh(cfg.mesh)
        eps, U = gwgen.make_fock(cfg, mesh)
        H0, S = gwgen.make_h0_s(cfg, mesh, eps, U)
        fg = gwgen.make_fermionic_grids(cfg.ntau, cfg.beta)
    else:
        p = problems(name)
        cfg = p.cfg
        H0, S, fg, _ = _closure(p)
    rng = np.random.default_rng(11)
    nwf = len(fg["omega"])
    Sw = np.ascontiguousarray(0.3 * (rng.normal(size=(nwf, cfg.nk, cfg.nao, cfg.nao)) + 1j * rng.normal(size=(nwf, cfg.nk, cfg.nao, cfg.nao))))
    om = torch.from_numpy(fg["omega"]).cuda()
    dS, dH = torch.from_numpy(S).cuda(), torch.from_numpy(H0).cuda()
    for sig in (None, Sw):
        G_w, info = gw.gw_dyson_update(om, 0.137, dS, dH, torch.from_numpy(sig).cuda() if sig is not None else None)
        ref = oracle_lib.dyson_update(cfg, fg["omega"], 0.137, S, H0, sig)
        assert info.cpu().tolist() == [-1, -1]
        assert report(name, "G_w" + ("" if sig is None else "+Sigma"), G_w.cpu().numpy(), ref) <= TOL
        worst = max(relerr(G_w[n, k].cpu().numpy(), ref[n, k]) for n in range(nwf) for k in range(cfg.nk))
        assert worst < 1e-9, worst


def test_dyson_update_reports_singular_matrix():
    """A = (i omega + mu) S - F with S = 0, F = 0 at one k: info = {n, k} of a singular matrix, no abort."""
    import paper_2206_07660_b200 as gw
    nk, nao, nwf = 3, 5, 4
    S = torch.eye(nao, dtype=torch.complex128, device="cuda").repeat(nk, 1, 1).contiguous()
    F = torch.zeros_like(S)
    S[1] = 0
    om = torch.tensor([0.3, 0.9, 1.5, 2.1], dtype=torch.float64, device="cuda")
    _, info = gw.gw_dyson_update(om, 0.0, S, F)
    assert info.cpu().tolist() == [0, 1]


@pytest.mark.parametrize("name", ["T", "R"])
def test_electron_count_and_mu_parity(problems, oracle_lib, name):
    """Eq. 15 and the bisection of Fig. 4 step 3: N_e(mu) to round-off, mu to the bisection tolerance, |N_e - N| < 1e-9."""
    import paper_2206_07660_b200 as gw
    p = problems(name)
    cfg = p.cfg
    H0, S, fg, dfg = _closure(p)
    dS, dH = torch.from_numpy(S).cuda(), torch.from_numpy(H0).cuda()
    for mu in (-0.4, 0.0, 0.3):
        G_w, _ = gw.gw_dyson_update(dfg["omega"], mu, dS, dH)
        ne = float(gw.gw_electron_count(dfg["t_beta"], dS, G_w, cfg.spin_deg).cpu())
        ref = oracle_lib.electron_count(cfg, fg["t_beta"], S, oracle_lib.dyson_update(cfg, fg["omega"], mu, S, H0))
        assert abs(ne - ref) <= 1e-12 * max(1.0, abs(ref)), (mu, ne, ref)
    target = cfg.spin_deg * (cfg.nao // 2 + 0.25)
    mu, ne, G_w, n_eval = gw.gw_find_mu(dfg["omega"], dfg["t_beta"], dS, dH, None, target, -0.1, 0.1, 1e-12, cfg.spin_deg)
    mu_ref, ne_ref = oracle_lib.find_mu(cfg, fg["omega"], fg["t_beta"], S, H0, None, target, -0.1, 0.1, 1e-12)
    print(f"find_mu {name}: mu {mu:.15f} (oracle {mu_ref:.15f}), N_e - N = {ne - target:.2e}, {n_eval} evaluations")
    assert abs(mu - mu_ref) < 1e-9 and abs(ne - ne_ref) < 1e-10 and abs(ne - target) < 1e-9
    assert relerr(G_w.cpu().numpy(), oracle_lib.dyson_update(cfg, fg["omega"], mu_ref, S, H0)) < 1e-8


def test_axpby_parity(oracle_lib):
    import paper_2206_07660_b200 as gw
    rng = np.random.default_rng(3)
    X = rng.normal(size=1000003) + 1j * rng.normal(size=1000003)
    Y = rng.normal(size=1000003) + 1j * rng.normal(size=1000003)
    a, b = 0.3 - 0.7j, -1.1 + 0.2j
    got = gw.gw_axpby(a, torch.from_numpy(X).cuda(), b, torch.from_numpy(Y).cuda()).cpu().numpy()
    assert relerr(got, oracle_lib.axpby(a, X, b, Y.copy())) < 1e-15
    nan = torch.full((5,), float("nan"), dtype=torch.complex128, device="cuda")
    assert torch.equal(gw.gw_axpby(2.0, torch.ones(5, dtype=torch.complex128, device="cuda"), 0.0, nan).cpu(), torch.full((5,), 2.0, dtype=torch.complex128))


@pytest.mark.parametrize("name", ["T", "R"])
def test_scgw_iteration_parity(problems, oracle_lib, name):
    """One full iteration of Fig. 4, G -> Sigma -> G', every step a C-ABI call, against the oracle's sequence of its own routines."""
    import paper_2206_07660_b200 as gw
    p = problems(name)
    cfg = p.cfg
    H0, S, fg, dfg = _closure(p)
    target = cfg.spin_deg * (cfg.nao // 2)
    ref = oracle_lib.scgw_iteration(cfg, oracle_lib.VBlocks(cfg, p.V.numpy()), p.T_wt, p.T_tw, fg, H0, S, p.G, target, -1.0, 1.0, alpha=0.7)
    prob, G, _ = device_problem(p)
    got = gw.gw_scgw_iteration(prob, dfg, torch.from_numpy(H0).cuda(), torch.from_numpy(S).cuda(), G, target, -1.0, 1.0, alpha=0.7)
    torch.cuda.synchronize()
    assert got["info"].cpu().tolist() == [-1, -1]
    for key in ("gamma", "J", "K", "Wt", "Sigma_t", "Sigma_w", "F", "G_w", "G_new", "G"):
        assert report(name, "scgw " + key, got[key].cpu().numpy(), ref[key]) <= (TOL if key not in ("G_w", "G_new", "G") else 1e-9), key
    print(f"scgw {name}: mu {got['mu']:.12f} (oracle {ref['mu']:.12f}), N_e {got['ne']:.12f}, {got['n_eval']} N_e evaluations")
    assert abs(got["mu"] - ref["mu"]) < 1e-9 and abs(got["ne"] - target) < 1e-9


def test_phi_gw_parity(problems, oracle_lib):
    """Eq. 37: the Matsubara / q sum of the summand returned by gw_screened_interaction_phi, with quadrature weights."""
    import paper_2206_07660_b200 as gw
    p = problems("R")
    cfg = p.cfg
    prob, G, _ = device_problem(p)
    P0t = gw.gw_polarization(prob, G)
    _, _, phi = gw.gw_screened_interaction_phi(prob, P0t)
    w = np.where(p.nbos == 0, 1.0, 2.0)                      # n >= 0 grid: mirror images n < 0 folded in
    got = float(gw.gw_phi_gw(prob, torch.from_numpy(w).cuda(), phi).cpu())
    ref = oracle_lib.phi_gw(cfg.nk, cfg.beta, w, phi.cpu().numpy())
    assert abs(got - ref) <= 1e-13 * abs(ref)
    P0 = oracle_lib.polarization(cfg, oracle_lib.VBlocks(cfg, p.V.numpy()), p.G)
    _, P0w, _ = oracle_lib.screened_interaction(cfg, p.T_wt, p.T_tw, P0, want_freq=True)
    phi_ref = np.array([[oracle_lib.phi(P0w[n, q]) for q in range(cfg.nk)] for n in range(cfg.nw)])
    assert abs(got - oracle_lib.phi_gw(cfg.nk, cfg.beta, w, phi_ref)) <= 1e-10 * abs(ref)


def test_find_mu_reports_missing_bracket(problems):
    """A target above the number of spin orbitals can never be bracketed: GW_ENOBRACKET (-6), not an abort and not a wrong mu."""
    import paper_2206_07660_b200 as gw
    p = problems("T")
    cfg = p.cfg
    H0, S, fg, dfg = _closure(p)
    with pytest.raises(gw.GWError, match="bracket"):
        gw.gw_find_mu(dfg["omega"], dfg["t_beta"], torch.from_numpy(S).cuda(), torch.from_numpy(H0).cuda(), None, cfg.spin_deg * cfg.nao + 1.0, -0.1, 0.1, 1e-12, cfg.spin_deg)
