"""Synthetic three-index tensor V[k1][k2][Q][i][j] (stands in for the GDF integrals of PAPER.md Eq. 6-7).

Raw R[k1][k2][Q][i][j]: real and imaginary parts i.i.d. N(0, 0.1²), an independent draw per (k1,k2) block,
from a counter-based generator that is a pure function of (seed, flat element index) — so any block can be
produced on its own, on the host or on the GPU, without materialising R.  Then the group average

    V[k1][k2]_ij = ½ ( R[k1][k2]_ij + conj R[k2][k1]_ji + conj R[−k1][−k2]_ij + R[−k2][−k1]_ji )

which gives exactly   V(k1,k2)_ij = conj V(k2,k1)_ji   (BASELINE.json "symmetrized")
and time reversal     V(−k1,−k2) = conj V(k1,k2).

Written with torch tensor ops so that the same code fills blocks on `cpu` or `cuda` (the generator is not
part of the timed path, and torch is plumbing here).  Host and device transcendental functions may differ
in the last bit, therefore parity tests always hand the *same bytes* to the oracle and to the CUDA path.
"""
import numpy as np
import torch

_M64 = (1 << 64) - 1


def _i64(x):
    """Python int (mod 2^64) -> value representable as torch.int64 (two's complement)."""
    x &= _M64
    return x - (1 << 64) if x >= (1 << 63) else x


_C1 = _i64(0x9E3779B97F4A7C15)
_C2 = _i64(0xBF58476D1CE4E5B9)
_C3 = _i64(0x94D049BB133111EB)


def _lsr(x, n):
    """logical shift right on int64 tensors"""
    return (x >> n) & ((1 << (64 - n)) - 1)


def _splitmix(x):
    z = x + _C1
    z = (z ^ _lsr(z, 30)) * _C2
    z = (z ^ _lsr(z, 27)) * _C3
    return z ^ _lsr(z, 31)


def _raw_block(seed, blk_index, n_per_block, device):
    """R block as complex128 [n_per_block]: Box-Muller on two splitmix64 streams keyed by the flat index."""
    idx = torch.arange(n_per_block, dtype=torch.int64, device=device) + blk_index * n_per_block
    key = _i64(seed * 0x2545F4914F6CDD1D)
    h1 = _splitmix(idx * 2 + key)
    h2 = _splitmix(idx * 2 + 1 + key)
    u1 = (_lsr(h1, 11).to(torch.float64) + 1.0) * (1.0 / 9007199254740992.0)     # (0,1]
    u2 = _lsr(h2, 11).to(torch.float64) * (1.0 / 9007199254740992.0)             # [0,1)
    r = torch.sqrt(-2.0 * torch.log(u1)) * 0.1
    ang = (2.0 * np.pi) * u2
    return torch.complex(r * torch.cos(ang), r * torch.sin(ang))


def make_V_block(cfg, mesh, k1, k2, device="cpu", neg=None, raw=False):
    """V[k1][k2] as a torch complex128 tensor [naux][nao][nao] on `device`.
    raw=True: the i.i.d. block R[k1][k2] itself, with none of the symmetries (tests of the literal, symmetry-free path)."""
    nk, nao, naux = mesh.nk, cfg.nao, cfg.naux
    if neg is None:
        neg = mesh.neg()
    n = naux * nao * nao
    seed = cfg.seed * 4 + 2

    def R(a, b):
        return _raw_block(seed, int(a) * nk + int(b), n, device).view(naux, nao, nao)

    if raw:
        return R(k1, k2).contiguous()

    m1, m2 = int(neg[k1]), int(neg[k2])
    v = R(k1, k2) + R(k2, k1).conj().transpose(1, 2) + R(m1, m2).conj() + R(m2, m1).transpose(1, 2)
    return (0.5 * v).resolve_conj().contiguous()


def make_V(cfg, mesh, device="cpu", out=None, raw=False):
    """Full V[k1][k2][Q][i][j] on `device` (torch complex128).  Fills one orbit of the symmetry group per
    generated block, so every block is generated once.  raw=True: every block is its own i.i.d. draw (no symmetry)."""
    nk, nao, naux = mesh.nk, cfg.nao, cfg.naux
    neg = mesh.neg()
    if out is None:
        out = torch.empty((nk, nk, naux, nao, nao), dtype=torch.complex128, device=device)
    if raw:
        for k1 in range(nk):
            for k2 in range(nk):
                out[k1, k2] = make_V_block(cfg, mesh, k1, k2, device, neg, raw=True)
        return out
    done = np.zeros((nk, nk), dtype=bool)
    for k1 in range(nk):
        for k2 in range(nk):
            if done[k1, k2]:
                continue
            v = make_V_block(cfg, mesh, k1, k2, device, neg)
            m1, m2 = int(neg[k1]), int(neg[k2])
            out[k1, k2] = v
            done[k1, k2] = True
            if not done[k2, k1]:
                out[k2, k1] = v.conj().transpose(1, 2)
                done[k2, k1] = True
            if not done[m1, m2]:
                out[m1, m2] = v.conj()
                done[m1, m2] = True
            if not done[m2, m1]:
                out[m2, m1] = v.transpose(1, 2)
                done[m2, m1] = True
    return out


def to_qslab(V, mesh, q_begin, q_end):
    """Layout conversion only: the q-slab view of V for the shard [q_begin, q_end) (include/gw.h "V layouts"):
    out[q - q_begin][k][0] = V[k][k+q], out[q - q_begin][k][1] = V[k+q][k]."""
    add = mesh.add_table()
    nk = mesh.nk
    out = torch.empty((q_end - q_begin, nk, 2) + tuple(V.shape[2:]), dtype=V.dtype, device=V.device)
    for q in range(q_begin, q_end):
        for k in range(nk):
            kq = int(add[k][q])
            out[q - q_begin, k, 0] = V[k, kq]
            out[q - q_begin, k, 1] = V[kq, k]
    return out


def make_V_qslab(cfg, mesh, q_begin, q_end, device="cpu", raw=False):
    """The q-slab of V for the shard [q_begin, q_end) generated directly (only the 2 nk blocks per q a rank needs, SURVEY.md §8e:
    "V slice {V[k][k+q] : q mine}"): out[q - q_begin][k][0] = V[k][k+q], out[q - q_begin][k][1] = V[k+q][k].  Same values as
    to_qslab(make_V(...)) up to the rounding order of the four-term group average (every block is a pure function of (seed, k1, k2))."""
    add = mesh.add_table()
    neg = mesh.neg()
    nk = mesh.nk
    out = torch.empty((q_end - q_begin, nk, 2, cfg.naux, cfg.nao, cfg.nao), dtype=torch.complex128, device=device)
    for q in range(q_begin, q_end):
        for k in range(nk):
            kq = int(add[k][q])
            out[q - q_begin, k, 0] = make_V_block(cfg, mesh, k, kq, device, neg, raw)
            out[q - q_begin, k, 1] = make_V_block(cfg, mesh, kq, k, device, neg, raw)
    return out
