"""GPU parity of SURVEY.md §8f row f4: two collinear spin channels (gw.h "Spin channels") and out-of-core V
(gw.h "V layouts", gw_sigma_iteration_stream), each against the oracle on the same seeded inputs."""
import dataclasses

import numpy as np
import pytest
import torch

import gwgen
from parity import relerr, report

pytestmark = pytest.mark.gpu
TOL = 1e-10


def _dev_problem(p, cfg, ns=1, symmetry=0, q_begin=0, q_end=None, qslab=False):
    import paper_2206_07660_b200 as gw
    q_end = cfg.nk if q_end is None else q_end
    V = gwgen.to_qslab(p.V, p.mesh, q_begin, q_end).cuda() if qslab else p.V.cuda()
    return gw.GWProblem(cfg.mesh, cfg.nao, cfg.naux, cfg.ntau, cfg.nw, cfg.beta, V, torch.from_numpy(p.T_wt).cuda(), torch.from_numpy(p.T_tw).cuda(),
                        cfg.spin_deg, q_begin, q_end, symmetry, ns, gw.GW_V_QSLAB if qslab else gw.GW_V_FULL)


@pytest.mark.parametrize("name", ["T", "R", "S", "L"])
def test_spin_channels_parity(problems, oracle_lib, name):
    """ns = 2, spin_deg = 1: P0t (sum over the channels inside the stage-1 k loop), Wt, Sigma^sigma, K^sigma, J, all four basis-class
    kernels (nao = 3, 7: generic; 26, 52: warp-specialised)."""
    import paper_2206_07660_b200 as gw
    p = problems(name)
    cfg = dataclasses.replace(p.cfg, spin_deg=1)
    Gs, gs = gwgen.make_spin_channels(p, 2)
    prob = _dev_problem(p, cfg, ns=2)
    G, gamma = torch.from_numpy(Gs).cuda(), torch.from_numpy(gs).cuda()
    P0t = gw.gw_polarization(prob, G)
    Wt, info = gw.gw_screened_interaction(prob, P0t)
    Sigma = gw.gw_selfenergy(prob, G, Wt)
    K = gw.gw_exchange(prob, gamma)
    J = gw.gw_hartree(prob, gamma)
    torch.cuda.synchronize()
    vb = oracle_lib.VBlocks(cfg, p.V.numpy())
    rP = oracle_lib.polarization_spin(cfg, vb, Gs)
    rW = oracle_lib.screened_interaction(cfg, p.T_wt, p.T_tw, rP)
    assert info.cpu().tolist() == [-1, -1]
    for key, got, ref in (("P0t", P0t, rP), ("Wt", Wt, rW), ("Sigma", Sigma, oracle_lib.selfenergy_spin(cfg, vb, Gs, rW)),
                          ("K", K, oracle_lib.exchange_spin(cfg, vb, gs)), ("J", J, oracle_lib.hartree_spin(cfg, vb, gs))):
        assert report(name + " ns=2", key, got.cpu().numpy(), ref) <= TOL, key
    # time-reversal mode with two channels (both channels are time-reversal symmetric Fock-built G's)
    prob_tr = _dev_problem(p, cfg, ns=2, symmetry=gw.GW_SYM_TR)
    P_tr = gw.gw_polarization(prob_tr, G)
    S_tr = gw.gw_selfenergy(prob_tr, G, Wt)
    assert relerr(P_tr.cpu().numpy(), rP) <= TOL and relerr(S_tr.cpu().numpy(), Sigma.cpu().numpy()) <= 1e-12


@pytest.mark.parametrize("name", ["T", "L"])
def test_spin_channels_raw_inputs(raw_problems, oracle_lib, name):
    """ns = 2 on symmetry-free inputs (independent V blocks, non-Hermitian G and W): stages 1, 3, 4 and J as printed."""
    import paper_2206_07660_b200 as gw
    p = raw_problems(name)
    cfg = dataclasses.replace(p.cfg, spin_deg=1)
    Gs, gs = gwgen.make_spin_channels(p, 2)
    prob = _dev_problem(p, cfg, ns=2)
    G, gamma, W = torch.from_numpy(Gs).cuda(), torch.from_numpy(gs).cuda(), torch.from_numpy(p.extras["W"]).cuda()
    vb = oracle_lib.VBlocks(cfg, p.V.numpy())
    assert report(name + " raw ns=2", "P0t", gw.gw_polarization(prob, G).cpu().numpy(), oracle_lib.polarization_spin(cfg, vb, Gs)) <= TOL
    assert report(name + " raw ns=2", "Sigma", gw.gw_selfenergy(prob, G, W).cpu().numpy(), oracle_lib.selfenergy_spin(cfg, vb, Gs, p.extras["W"])) <= TOL
    assert report(name + " raw ns=2", "K", gw.gw_exchange(prob, gamma).cpu().numpy(), oracle_lib.exchange_spin(cfg, vb, gs)) <= TOL
    assert report(name + " raw ns=2", "J", gw.gw_hartree(prob, gamma).cpu().numpy(), oracle_lib.hartree_spin(cfg, vb, gs)) <= TOL


def test_identical_channels_equal_closed_shell(problems):
    """Two identical channels with spin_deg = 1 reproduce the closed-shell call (spin_deg = 2): P0t bit for bit, Sigma / K per channel."""
    import paper_2206_07660_b200 as gw
    p = problems("S")
    cfg = p.cfg
    prob = _dev_problem(p, cfg)
    G, gamma = torch.from_numpy(p.G).cuda(), torch.from_numpy(p.gamma).cuda()
    ref = gw.gw_sigma_iteration(prob, G, gamma)
    prob2 = _dev_problem(p, dataclasses.replace(cfg, spin_deg=1), ns=2)
    G2, g2 = torch.stack([G, G]).contiguous(), torch.stack([gamma, gamma]).contiguous()
    P2 = gw.gw_polarization(prob2, G2)
    assert relerr(P2.cpu().numpy(), ref["P0t"].cpu().numpy()) < 1e-14
    S2 = gw.gw_selfenergy(prob2, G2, ref["Wt"])
    K2 = gw.gw_exchange(prob2, g2)
    for sg in range(2):
        assert torch.equal(S2[sg], ref["Sigma"]) and torch.equal(K2[sg], ref["K"])


@pytest.mark.parametrize("name,raw", [("R", False), ("S", False), ("L", False), ("R", True), ("L", True)])
def test_qslab_layout_parity(problems, raw_problems, oracle_lib, name, raw):
    """GW_V_QSLAB: every stage on a q shard whose V holds only the 2 nk blocks per q, against the oracle's q-range routines and
    bit for bit against the GW_V_FULL evaluation of the same shard."""
    import paper_2206_07660_b200 as gw
    p = raw_problems(name) if raw else problems(name)
    cfg = p.cfg
    q0, q1 = (0, cfg.nk) if cfg.nk <= 2 else (1, cfg.nk - 1)
    full = _dev_problem(p, cfg, q_begin=q0, q_end=q1)
    slab = _dev_problem(p, cfg, q_begin=q0, q_end=q1, qslab=True)
    G, gamma = torch.from_numpy(p.G).cuda(), torch.from_numpy(p.gamma).cuda()
    vb = oracle_lib.VBlocks(cfg, p.V.numpy())
    P_f, P_s = gw.gw_polarization(full, G), gw.gw_polarization(slab, G)
    assert torch.equal(P_f, P_s)
    rP = oracle_lib.polarization(cfg, vb, p.G)[:, q0:q1]
    assert report(name, "P0t qslab", P_s.cpu().numpy(), rP) <= TOL
    if raw:
        W = torch.from_numpy(np.ascontiguousarray(p.extras["W"][:, q0:q1])).cuda()
        Wfull = p.extras["W"]
    else:
        W, info = gw.gw_screened_interaction(slab, P_s)
        assert info.cpu().tolist() == [-1, -1]
        Wfull = np.zeros((cfg.ntau, cfg.nk, cfg.naux, cfg.naux), np.complex128)
        Wfull[:, q0:q1] = W.cpu().numpy()
    S_f, S_s = gw.gw_selfenergy(full, G, W), gw.gw_selfenergy(slab, G, W)
    K_f, K_s = gw.gw_exchange(full, gamma), gw.gw_exchange(slab, gamma)
    assert torch.equal(S_f, S_s) and torch.equal(K_f, K_s)
    rS = np.stack([[oracle_lib.sigma_slice(cfg, vb, p.G[t], Wfull[t], k, q0, q1) for k in range(cfg.nk)] for t in range(cfg.ntau)])
    rK = np.stack([oracle_lib.exchange_slice(cfg, vb, p.gamma, k, q0, q1) for k in range(cfg.nk)])
    assert report(name, "Sigma qslab", S_s.cpu().numpy(), rS) <= TOL and report(name, "K qslab", K_s.cpu().numpy(), rK) <= TOL
    if q0 == 0:
        assert torch.equal(gw.gw_hartree(full, gamma), gw.gw_hartree(slab, gamma))
    else:
        with pytest.raises(gw.GWError):
            gw.gw_hartree(slab, gamma)                      # the shard holds no q = 0: no diagonal blocks


@pytest.mark.parametrize("name,ns,budget_q", [("R", 1, 1), ("R", 1, 5), ("S", 1, 1), ("Y", 1, 1), ("S", 2, 3), ("L", 1, 1), ("R", 2, 4), ("R", 4, 5), ("1", 1, 3)])
def test_streamed_iteration_equals_resident(problems, oracle_results, name, ns, budget_q):
    """gw_sigma_iteration_stream (V in host memory, two device slab buffers of budget_q q-points each): Sigma and K are bit-identical
    to the resident evaluation (the q sums continue across slabs in the same order) and match the oracle."""
    import paper_2206_07660_b200 as gw
    p = problems(name) if name != "1" else gwgen.make_problem("1")
    cfg = dataclasses.replace(p.cfg, spin_deg=1) if ns > 1 else p.cfg
    if ns > 1:
        Gs, gs = gwgen.make_spin_channels(p, 2)
        if ns == 4:
            Gs, gs, _ = gwgen.rotate_spin_channels(Gs, gs, seed=2)
    else:
        Gs, gs = p.G, p.gamma
    G, gamma = torch.from_numpy(Gs), torch.from_numpy(gs)
    # resident reference on the device
    prob = _dev_problem(p, cfg, ns=ns)
    P0t = gw.gw_polarization(prob, G.cuda())
    Wt, _ = gw.gw_screened_interaction(prob, P0t)
    S_res = gw.gw_selfenergy(prob, G.cuda(), Wt).cpu()
    K_res = gw.gw_exchange(prob, gamma.cuda()).cpu()
    # streamed
    hV = p.V.pin_memory()
    hprob = gw.GWProblem(cfg.mesh, cfg.nao, cfg.naux, cfg.ntau, cfg.nw, cfg.beta, hV, torch.from_numpy(p.T_wt), torch.from_numpy(p.T_tw), cfg.spin_deg, ns=ns)
    perq = 2 * cfg.nk * cfg.naux * cfg.nao * cfg.nao * 16
    out = gw.gw_sigma_iteration_stream(hprob, G.pin_memory(), gamma.pin_memory(), 2 * budget_q * perq + 1000)
    print(name, out["stats"])
    assert out["stats"]["q_per_slab"] == min(budget_q, cfg.nk) and out["stats"]["slabs"] == -(-cfg.nk // budget_q)
    assert torch.equal(out["Sigma"], S_res) and torch.equal(out["K"], K_res)
    if ns == 1 and name != "1":
        ref = oracle_results(name)
        assert relerr(out["Sigma"].numpy(), ref["Sigma"]) <= TOL and relerr(out["K"].numpy(), ref["K"]) <= TOL
    with pytest.raises(gw.GWError):
        gw.gw_sigma_iteration_stream(hprob, G.pin_memory(), gamma.pin_memory(), perq)      # budget below two one-q slabs: GW_ENOMEM


def test_streamed_iteration_time_reversal_mode(problems, oracle_results):
    """The streamed iteration under GW_SYM_TR (stage 1 uses the tau half and the Hermitian tiles per slab; the k reduction of stage 3 needs
    the full q range and is off): against the oracle."""
    import paper_2206_07660_b200 as gw
    p = problems("R")
    cfg = p.cfg
    hprob = gw.GWProblem(cfg.mesh, cfg.nao, cfg.naux, cfg.ntau, cfg.nw, cfg.beta, p.V.pin_memory(), torch.from_numpy(p.T_wt), torch.from_numpy(p.T_tw),
                         cfg.spin_deg, symmetry=gw.GW_SYM_TR)
    perq = 2 * cfg.nk * cfg.naux * cfg.nao * cfg.nao * 16
    out = gw.gw_sigma_iteration_stream(hprob, torch.from_numpy(p.G).pin_memory(), torch.from_numpy(p.gamma).pin_memory(), 2 * 4 * perq)
    ref = oracle_results("R")
    assert out["stats"]["slabs"] == 3
    assert relerr(out["Sigma"].numpy(), ref["Sigma"]) <= TOL and relerr(out["K"].numpy(), ref["K"]) <= TOL


@pytest.mark.skipif(torch.cuda.device_count() < 2, reason="needs two GPUs")
def test_two_gpu_q_shards_sum_to_oracle(problems, oracle_results):
    """Each of two GPUs evaluates its q shard from its own V q-slab (generated per rank, as bench.py --gpus N does); the partial
    Sigma and K add up to the oracle's full result (the NCCL all-reduce of dist.py is a plain sum of these partials)."""
    import paper_2206_07660_b200 as gw
    from paper_2206_07660_b200.dist import shard_range
    p = problems("R")
    cfg = p.cfg
    ref = oracle_results("R")
    S_tot, K_tot = None, None
    for rank in range(2):
        dev = torch.device("cuda", rank)
        with torch.cuda.device(dev):
            q0, q1 = shard_range(cfg.nk, 2, rank)
            V = gwgen.make_V_qslab(cfg, p.mesh, q0, q1, device=dev)
            prob = gw.GWProblem(cfg.mesh, cfg.nao, cfg.naux, cfg.ntau, cfg.nw, cfg.beta, V, torch.from_numpy(p.T_wt).to(dev), torch.from_numpy(p.T_tw).to(dev),
                                cfg.spin_deg, q0, q1, 0, 1, gw.GW_V_QSLAB)
            out = gw.gw_sigma_iteration(prob, torch.from_numpy(p.G).to(dev), torch.from_numpy(p.gamma).to(dev))
            torch.cuda.synchronize()
            assert relerr(out["Wt"].cpu().numpy(), ref["Wt"][:, q0:q1]) <= TOL
            S_tot = out["Sigma"].cpu() if S_tot is None else S_tot + out["Sigma"].cpu()
            K_tot = out["K"].cpu() if K_tot is None else K_tot + out["K"].cpu()
    assert relerr(S_tot.numpy(), ref["Sigma"]) <= TOL and relerr(K_tot.numpy(), ref["K"]) <= TOL


@pytest.mark.parametrize("name", ["T", "R", "S", "W"])
def test_two_component_blocks_parity(problems, oracle_lib, name):
    """ns = 4 (blocks uu, ud, du, dd; gw.h "Spin blocks"): P0t with the full sigma sigma' sum of Eq. 28b inside the stage-1 k loop, Wt,
    Sigma and K per block, J from the spin-diagonal blocks; GW_SYM_TR is refused for two-component G."""
    import paper_2206_07660_b200 as gw
    p = problems(name)
    cfg = dataclasses.replace(p.cfg, spin_deg=1)
    Gs, gs = gwgen.make_spin_channels(p, 2)
    Gb, gb, _ = gwgen.rotate_spin_channels(Gs, gs, seed=1)
    prob = _dev_problem(p, cfg, ns=4)
    G, gamma = torch.from_numpy(Gb).cuda(), torch.from_numpy(gb).cuda()
    P0t = gw.gw_polarization(prob, G)
    Wt, info = gw.gw_screened_interaction(prob, P0t)
    Sigma = gw.gw_selfenergy(prob, G, Wt)
    K = gw.gw_exchange(prob, gamma)
    J = gw.gw_hartree(prob, gamma)
    torch.cuda.synchronize()
    assert info.cpu().tolist() == [-1, -1]
    vb = oracle_lib.VBlocks(cfg, p.V.numpy())
    rP = oracle_lib.polarization_blocks(cfg, vb, Gb)
    rW = oracle_lib.screened_interaction(cfg, p.T_wt, p.T_tw, rP)
    for key, got, ref in (("P0t", P0t, rP), ("Wt", Wt, rW), ("Sigma", Sigma, oracle_lib.selfenergy_spin(cfg, vb, Gb, rW)),
                          ("K", K, oracle_lib.exchange_spin(cfg, vb, gb)), ("J", J, oracle_lib.hartree_blocks(cfg, vb, gb))):
        assert report(name + " ns=4", key, got.cpu().numpy(), ref) <= TOL, key
    with pytest.raises(gw.GWError):
        gw.gw_polarization(_dev_problem(p, cfg, ns=4, symmetry=gw.GW_SYM_TR), G)


def test_two_component_raw_inputs(raw_problems, oracle_lib):
    """ns = 4 on four independent non-Hermitian blocks (no relation between ud and du): the block pairing of Eq. 28b,
    G^{sigma sigma'} at k+q with G^{sigma' sigma} at k, is told apart from its transposed twin."""
    import paper_2206_07660_b200 as gw
    p = raw_problems("R")
    cfg = dataclasses.replace(p.cfg, spin_deg=1)
    G2a, g2a = gwgen.make_spin_channels(p, 2)
    rng = np.random.default_rng(21)
    Gb = np.ascontiguousarray(np.stack([G2a[0], G2a[1], G2a[0][::-1].copy() * 0.7, G2a[1] * (0.3 - 0.5j)]))
    gb = np.ascontiguousarray(np.stack([g2a[0], g2a[1], g2a[0].conj() * 0.7, g2a[1] * (0.3 - 0.5j)]))
    prob = _dev_problem(p, cfg, ns=4)
    G, gamma, W = torch.from_numpy(Gb).cuda(), torch.from_numpy(gb).cuda(), torch.from_numpy(p.extras["W"]).cuda()
    vb = oracle_lib.VBlocks(cfg, p.V.numpy())
    assert report("R raw ns=4", "P0t", gw.gw_polarization(prob, G).cpu().numpy(), oracle_lib.polarization_blocks(cfg, vb, Gb)) <= TOL
    assert report("R raw ns=4", "Sigma", gw.gw_selfenergy(prob, G, W).cpu().numpy(), oracle_lib.selfenergy_spin(cfg, vb, Gb, p.extras["W"])) <= TOL
    assert report("R raw ns=4", "K", gw.gw_exchange(prob, gamma).cpu().numpy(), oracle_lib.exchange_spin(cfg, vb, gb)) <= TOL
    assert report("R raw ns=4", "J", gw.gw_hartree(prob, gamma).cpu().numpy(), oracle_lib.hartree_blocks(cfg, vb, gb)) <= TOL
