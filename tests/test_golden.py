"""Stored oracle values (tests/golden/cfgT_oracle.json, written by tests/golden/make_golden.py from oracle/ only)."""
import json
import os
import re

import numpy as np
import pytest

GOLD = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "cfgT_oracle.json")


def _entries(arrs, gold):
    for key, (re_, im_) in gold["entries"].items():
        name, idx = key.split("[", 1)
        idx = tuple(int(x) for x in re.findall(r"\d+", idx))
        yield key, complex(arrs[name][idx]), complex(re_, im_)


def test_oracle_reproduces_golden(oracle_results, oracle_lib):
    gold = json.load(open(GOLD))
    ref = oracle_results("T")
    for name, nrm in gold["norms"].items():
        assert abs(np.linalg.norm(ref[name]) - nrm) <= 1e-13 * nrm, name
    for key, got, want in _entries(ref, gold):
        assert abs(got - want) <= 1e-13 * max(abs(want), 1e-3), key
    for row, n in zip(gold["phi_n0_n1_n7"], (0, 1, 7)):
        for q, want in enumerate(row):
            assert abs(oracle_lib.phi(ref["P0w"][n, q]) - want) <= 1e-13 * max(1.0, abs(want))


@pytest.mark.gpu
def test_gpu_hits_golden(problems):
    import torch
    import paper_2206_07660_b200 as gw
    from parity import device_problem
    gold = json.load(open(GOLD))
    p = problems("T")
    prob, G, gamma = device_problem(p)
    out = gw.gw_sigma_iteration(prob, G, gamma)
    torch.cuda.synchronize()
    got = {k: v.cpu().numpy() for k, v in out.items()}
    for name, nrm in gold["norms"].items():
        assert abs(np.linalg.norm(got[name]) - nrm) <= 1e-10 * nrm, name
    for key, g, want in _entries(got, gold):
        assert abs(g - want) <= 1e-10 * gold["norms"][key.split("[")[0]], key
