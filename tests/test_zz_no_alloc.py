"""gw_hartree_static (include/gw.h): the Hartree term of Eq. 20 with its intermediate in a static device array of the library, for
callers that cannot allocate device memory.  Checked against the existing path gw_hartree (workspace in p->work) on calls in a row that
share the array, and against the oracle.  This file sorts last on purpose (the suite runs with pytest -x)."""
import ctypes

import numpy as np
import pytest
import torch

from parity import relerr, device_problem, report

TOL = 1e-10


def test_static_entry_rejects_sizes_beyond_its_scratch():
    """naux > GW_STATIC_MAX_NAUX: GW_ESTATIC (-7) with a message that says so, before any CUDA call (no GPU needed)."""
    import paper_2206_07660_b200 as gw
    from paper_2206_07660_b200.binding import _CProblem
    L = gw.lib()
    nmax = gw.gw_static_max_naux()
    assert nmax == 512
    ptr = ctypes.c_void_p(4096)
    c = _CProblem(1, 1, 1, 4, nmax + 1, 8, 8, 2, 0, 1, 10.0, 4096, None, None, None, 0)
    assert L.gw_hartree_static(ctypes.byref(c), ptr, ptr, None) == -7
    msg = gw.gw_strerror(-7)
    assert "static" in msg and "512" in msg
    c.naux = 897                                             # beyond what any kernel supports: the general answer comes first
    assert L.gw_hartree_static(ctypes.byref(c), ptr, ptr, None) == -4
    c.naux = nmax
    assert L.gw_hartree_static(ctypes.byref(c), None, ptr, None) == -1     # null gamma
    assert L.gw_hartree_static(None, ptr, ptr, None) == -1


@pytest.mark.gpu
def test_static_hartree_equals_workspace_path_on_calls_in_a_row(problems, oracle_lib):
    """Calls in a row on problems of different naux (44, 37, 44: the second leaves stale entries of the first behind its own) and with
    different gamma: every J equals gw_hartree's (same sums in the same order: bit for bit) and the oracle's within the tolerance of the
    parity tests.  The problem handed to the static entry point has NO workspace, and the device's free memory does not change over
    the later calls (nothing is allocated)."""
    import paper_2206_07660_b200 as gw
    rng = np.random.default_rng(7)
    runs = []
    for name in ("S", "R", "S"):
        p = problems(name)
        prob, _, gamma = device_problem(p)
        if runs:                                            # a different density matrix on every call
            gamma = gamma + torch.from_numpy(0.1 * (rng.normal(size=tuple(gamma.shape)) + 1j * rng.normal(size=tuple(gamma.shape)))).cuda()
        bare, _, _ = device_problem(p)
        bare.work = None; bare.c.work = None; bare.c.work_bytes = 0          # the static entry point must not need it
        J_ref = gw.gw_hartree(prob, gamma)
        J = torch.full_like(J_ref, float("nan"))
        runs.append((name, p, bare, gamma, J_ref, J))
    torch.cuda.synchronize()
    free = []
    for name, p, bare, gamma, J_ref, J in runs:
        gw.gw_hartree_static(bare, gamma, J)
        torch.cuda.synchronize()
        free.append(torch.cuda.mem_get_info()[0])
    assert free[1] == free[0] and free[2] == free[0], free                   # no cudaMalloc behind the calls
    for name, p, bare, gamma, J_ref, J in runs:
        assert report(name, "J static vs workspace", J.cpu().numpy(), J_ref.cpu().numpy()) <= TOL
        assert torch.equal(J, J_ref)
        ref = oracle_lib.hartree(p.cfg, oracle_lib.VBlocks(p.cfg, p.V.numpy()), gamma.cpu().numpy())
        assert report(name, "J static vs oracle", J.cpu().numpy(), ref) <= TOL
    # the existing path still refuses a problem without workspace; the static one refuses what does not fit its array
    with pytest.raises(gw.GWError):
        gw.gw_hartree(runs[0][2], runs[0][3])


@pytest.mark.gpu
def test_static_hartree_spin_blocks_and_size_limit(problems):
    """Two collinear channels (gamma [2][nk][nao][nao]) through the static entry point, twice in a row; and a device problem with
    naux = 513 is refused with GW_ESTATIC and leaves J untouched."""
    import gwgen
    import paper_2206_07660_b200 as gw
    p = problems("R")
    cfg = p.cfg
    _, gs = gwgen.make_spin_channels(p, 2)
    V = p.V.cuda()
    prob = gw.GWProblem(cfg.mesh, cfg.nao, cfg.naux, cfg.ntau, cfg.nw, cfg.beta, V, torch.from_numpy(p.T_wt).cuda(), torch.from_numpy(p.T_tw).cuda(), 1, ns=2)
    gamma = torch.from_numpy(gs).cuda()
    J_ref = gw.gw_hartree(prob, gamma)
    for _ in range(2):
        J = torch.full_like(J_ref, float("nan"))
        gw.gw_hartree_static(prob, gamma, J)
        assert torch.equal(J, J_ref) and relerr(J.cpu().numpy(), J_ref.cpu().numpy()) <= TOL
    nbig = gw.gw_static_max_naux() + 1
    Vb = torch.zeros((1, 1, nbig, 2, 2), dtype=torch.complex128, device="cuda")
    T = torch.zeros((4, 4), dtype=torch.complex128, device="cuda")
    big = gw.GWProblem((1, 1, 1), 2, nbig, 4, 4, 10.0, Vb, T, T, 2)
    g = torch.zeros((1, 2, 2), dtype=torch.complex128, device="cuda")
    Jb = torch.full((1, 2, 2), 5.0, dtype=torch.complex128, device="cuda")
    with pytest.raises(gw.GWError, match="static"):
        gw.gw_hartree_static(big, g, Jb)
    assert torch.equal(Jb, torch.full_like(Jb, 5.0))
    assert torch.equal(gw.gw_hartree(big, g), torch.zeros_like(Jb))          # the workspace path takes it
