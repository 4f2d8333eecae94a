"""GPU parity: the CUDA path, called through the C ABI, against the CPU oracle, element by element.

Gate (north_star): relative Frobenius error <= 1e-10 for P0t, Wt, Sigma (and K).  Integer outputs (info) bit-exact.
"""
import numpy as np
import pytest
import torch

from parity import relerr, worst_slice, device_problem

pytestmark = pytest.mark.gpu
TOL = 1e-10


def run_gpu(p, **kw):
    import paper_2206_07660_b200 as gw
    prob, G, gamma = device_problem(p, **kw)
    out = gw.gw_sigma_iteration(prob, G, gamma)
    torch.cuda.synchronize()
    return {k: v.cpu().numpy() for k, v in out.items()}


@pytest.mark.parametrize("name", ["0", "T", "R"])
def test_full_parity_small(problems, oracle_results, name):
    p = problems(name)
    ref = oracle_results(name)
    got = run_gpu(p)
    assert tuple(got["info"]) == (-1, -1)
    for key in ("P0t", "Wt", "Sigma", "K"):
        e = relerr(got[key], ref[key])
        assert e <= TOL, f"{name} {key}: rel Frobenius {e:.3e}"
    assert worst_slice(got["P0t"], ref["P0t"]) < 1e-8
    assert worst_slice(got["Sigma"], ref["Sigma"]) < 1e-8
