"""Shared helpers of the GPU parity tests: upload a gwgen problem, run the C-ABI path, compare with the oracle."""
import numpy as np
import torch


def relerr(a, b):
    a = np.asarray(a); b = np.asarray(b)
    return float(np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300))


def worst_slice(a, b, lead=2):
    """worst relative Frobenius error over the leading `lead` axes (per (t,q) / (t,k) slice)."""
    a = np.asarray(a).reshape((-1,) + a.shape[lead:]); b = np.asarray(b).reshape((-1,) + b.shape[lead:])
    num = np.sqrt((np.abs(a - b) ** 2).reshape(a.shape[0], -1).sum(1))
    den = np.sqrt((np.abs(b) ** 2).reshape(b.shape[0], -1).sum(1))
    return float(np.max(num / np.maximum(den, 1e-300)))


def max_elem(a, b):
    """largest element-wise |a - b| relative to the largest |b| of the array (reported next to the Frobenius numbers so that a
    regression confined to one tile is visible; not gated)."""
    a = np.asarray(a); b = np.asarray(b)
    return float(np.max(np.abs(a - b)) / max(float(np.max(np.abs(b))), 1e-300))


def report(tag, key, got, ref):
    """relative Frobenius error (the gated number), printed with the worst element."""
    e = relerr(got, ref)
    print(f"parity {tag} {key}: rel Frobenius {e:.2e}, max element |d|/max|ref| {max_elem(got, ref):.2e}")
    return e


def device_problem(p, q_begin=0, q_end=None, device="cuda", symmetry=0):
    import paper_2206_07660_b200 as gw
    cfg = p.cfg
    V = p.V.to(device) if isinstance(p.V, torch.Tensor) else torch.from_numpy(p.V).to(device)
    prob = gw.GWProblem(cfg.mesh, cfg.nao, cfg.naux, cfg.ntau, cfg.nw, cfg.beta, V,
                        torch.from_numpy(p.T_wt).to(device), torch.from_numpy(p.T_tw).to(device),
                        cfg.spin_deg, q_begin, q_end, symmetry)
    G = torch.from_numpy(p.G).to(device)
    gamma = torch.from_numpy(p.gamma).to(device)
    return prob, G, gamma
