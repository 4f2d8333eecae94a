#!/usr/bin/env python
"""Writes tests/golden/cfgT_oracle.json: a few entries and norms of the ORACLE's outputs on config T.

Calls only gwgen (seeded inputs) and oracle/ (never the CUDA path).  The paper prints no worked numerical example for this path
(PAPER.md has equations and scaling figures only), so these stored values are the oracle's own, pinned elsewhere by
tests/test_oracle_pins.py (closed forms, Lindhard function, invariants, brute-force Matsubara sum); the file guards against silent
changes of the generator or the oracle, and gives the GPU tests fixed numbers to hit.
Regenerate with:  python tests/golden/make_golden.py
"""
import json
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)


def main():
    import gwgen
    import oracle
    oracle.build()
    p = gwgen.make_problem("T")
    cfg = p.cfg
    vb = oracle.VBlocks(cfg, p.V.numpy())
    P0t = oracle.polarization(cfg, vb, p.G)
    Wt, P0w, Ww = oracle.screened_interaction(cfg, p.T_wt, p.T_tw, P0t, want_freq=True)
    Sg = oracle.selfenergy(cfg, vb, p.G, Wt)
    K = oracle.exchange(cfg, vb, p.gamma)
    phi = [[oracle.phi(P0w[n, q]) for q in range(cfg.nk)] for n in (0, 1, 7)]

    def pick(A, idx):
        z = complex(A[idx])
        return [z.real, z.imag]
    out = {"config": "T", "citation": "oracle/gwref.c on gwgen config T (Eq. 28b, 28a, 29, 30, 31, 22, 37 summand; PAPER.md:155-256)",
           "norms": {k: float(np.linalg.norm(v)) for k, v in (("P0t", P0t), ("Wt", Wt), ("Sigma", Sg), ("K", K))},
           "entries": {"P0t[3][2][1][4]": pick(P0t, (3, 2, 1, 4)), "P0t[30][5][0][0]": pick(P0t, (30, 5, 0, 0)),
                       "Wt[0][0][2][2]": pick(Wt, (0, 0, 2, 2)), "Wt[17][4][3][1]": pick(Wt, (17, 4, 3, 1)),
                       "Sigma[5][1][0][2]": pick(Sg, (5, 1, 0, 2)), "Sigma[31][3][2][2]": pick(Sg, (31, 3, 2, 2)),
                       "K[2][1][0]": pick(K, (2, 1, 0))},
           "phi_n0_n1_n7": phi}
    with open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "cfgT_oracle.json"), "w") as f:
        json.dump(out, f, indent=1)
    print("wrote cfgT_oracle.json")


if __name__ == "__main__":
    main()
