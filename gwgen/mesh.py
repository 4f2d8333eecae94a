"""Γ-centred k-mesh index arithmetic (PAPER.md:41 momentum conservation, :87 q = k_j − k_i, :488 Γ-centred mesh).

k = (i1*nk2 + i2)*nk3 + i3 ; k±q and −k are component-wise modular.
"""
import numpy as np


class KMesh:
    def __init__(self, mesh):
        self.mesh = tuple(int(m) for m in mesh)
        n1, n2, n3 = self.mesh
        self.nk = n1 * n2 * n3
        idx = np.arange(self.nk)
        self.coords = np.stack([idx // (n2 * n3), (idx // n3) % n2, idx % n3], axis=1)

    def index(self, c):
        n1, n2, n3 = self.mesh
        c = np.asarray(c)
        return ((c[..., 0] % n1) * n2 + (c[..., 1] % n2)) * n3 + (c[..., 2] % n3)

    def neg(self):
        return self.index(-self.coords).astype(np.int32)

    def add_table(self):
        """add[k][q] = index of k+q."""
        return self.index(self.coords[:, None, :] + self.coords[None, :, :]).astype(np.int32)

    def sub_table(self):
        """sub[k][q] = index of k−q."""
        return self.index(self.coords[:, None, :] - self.coords[None, :, :]).astype(np.int32)
