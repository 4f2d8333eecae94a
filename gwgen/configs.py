"""The five BASELINE.json configs plus the tiny self-test config "T"."""
from dataclasses import dataclass

BASE_SEED = 220607660


@dataclass(frozen=True)
class GWConfig:
    name: str
    mesh: tuple          # (nk1, nk2, nk3), Γ-centred
    nao: int             # N_orb
    naux: int            # N_aux
    ntau: int            # N_τ
    nw: int              # N_ω (bosonic points used on this path)
    beta: float          # inverse temperature, Ha^-1 (β=700)
    elo: float           # Fock eigenvalue window [elo, ehi], μ = 0
    ehi: float
    gap: float           # gap at μ
    seed: int
    spin_deg: int = 2    # closed shell: Σ_σσ' of Eq. 28b

    @property
    def nk(self):
        return self.mesh[0] * self.mesh[1] * self.mesh[2]

    def bytes_V(self):
        return self.nk ** 2 * self.naux * self.nao ** 2 * 16

    def flops_nominal(self):
        """Algorithm 1 taken literally, 8 flops per complex multiply-add."""
        nk, nao, naux, nt, nw = self.nk, self.nao, self.naux, self.ntau, self.nw
        per = 8.0 * (naux * naux * nao * nao + 2 * naux * nao ** 3)
        s1 = nt * nk * nk * per
        s3 = s1
        tr = 2 * 8.0 * nw * nt * nk * naux * naux
        sol = nw * nk * (28.0 / 3.0) * naux ** 3
        s4 = nk * nk * 8.0 * 2 * naux * nao ** 3
        return {"stage1": s1, "stage2_transforms": tr, "stage2_solve": sol,
                "stage3": s3, "stage4": s4, "total": s1 + s3 + tr + sol + s4}


CONFIGS = {
    "0": GWConfig("cfg0", (1, 1, 1), 4, 16, 32, 32, 100.0, -1.0, 1.0, 0.0, BASE_SEED + 0),
    "1": GWConfig("cfg1", (2, 2, 2), 26, 100, 104, 104, 700.0, -2.0, 3.0, 0.04, BASE_SEED + 1),
    "2": GWConfig("cfg2", (4, 4, 4), 26, 200, 104, 104, 700.0, -2.0, 3.0, 0.04, BASE_SEED + 2),
    "3": GWConfig("cfg3", (5, 5, 5), 26, 200, 104, 104, 700.0, -2.0, 3.0, 0.04, BASE_SEED + 3),
    "4": GWConfig("cfg4", (4, 4, 4), 52, 400, 120, 120, 1000.0, -3.0, 5.0, 0.04, BASE_SEED + 4),
    # tiny self-test config: odd and even mesh dims, -k != k, small beta so the grid is physically accurate
    "T": GWConfig("cfgT", (3, 2, 1), 3, 5, 32, 32, 10.0, -1.0, 1.0, 0.0, BASE_SEED + 99),
    # config-2-shaped problem with a short tau grid: same per-CTA behaviour, 13x less work (ncu captures)
    "P": GWConfig("cfgP", (4, 4, 4), 26, 200, 8, 8, 700.0, -2.0, 3.0, 0.04, BASE_SEED + 97),
    # mid-size ragged config for parity tests: sizes that are not multiples of any tile
    "R": GWConfig("cfgR", (3, 2, 2), 7, 37, 18, 18, 30.0, -1.5, 2.0, 0.04, BASE_SEED + 98),
    # small problem with the production basis size (nao=26: the straight-line / warp-specialised kernel variants), ragged naux
    "S": GWConfig("cfgS", (2, 1, 2), 26, 44, 8, 8, 40.0, -2.0, 3.0, 0.04, BASE_SEED + 94),
    # odd sizes inside the compile-time k-step classes (nao = 25..28 -> 7 steps, 49..52 -> 13 steps), naux = one panel + 1 row
    "U": GWConfig("cfgU", (1, 2, 1), 27, 33, 6, 6, 20.0, -2.0, 3.0, 0.04, BASE_SEED + 93),
    "W": GWConfig("cfgW", (2, 1, 1), 49, 17, 6, 6, 20.0, -2.0, 3.0, 0.04, BASE_SEED + 92),
    # nao = 25: ONE valid line in the last 8-wide tile (the FMA tail of the pass GEMMs and the FMA strips of stage 3's final contraction
    # with a single column / row), naux = one panel + 9 rows, four k points (four one-q slabs in the streamed call)
    "Y": GWConfig("cfgY", (2, 1, 2), 25, 41, 6, 6, 20.0, -2.0, 3.0, 0.04, BASE_SEED + 89),
    # config-4-shaped problem with a short tau grid (same per-CTA behaviour, 15x less work)
    "Q": GWConfig("cfgQ", (4, 4, 4), 52, 400, 8, 8, 1000.0, -3.0, 5.0, 0.04, BASE_SEED + 95),
    # config-4-shaped basis (nao=52, naux > 224: the wide-panel / split-K kernel variants) at a size the oracle does in full
    "L": GWConfig("cfgL", (2, 1, 1), 52, 230, 8, 8, 50.0, -3.0, 5.0, 0.04, BASE_SEED + 96),
    # config 4's exact kernel launch shape (nao=52, naux=400: 25 n-tiles per CTA of the stage-1 cluster, 13 Q panels, split-K
    # final jobs) on a 2-point mesh with 6 tau nodes, small enough for the oracle to do in full
    "M": GWConfig("cfgM", (2, 1, 1), 52, 400, 6, 6, 50.0, -3.0, 5.0, 0.04, BASE_SEED + 91),
    # naux beyond one cluster's 448 panel columns (stage 1 runs two column passes), small basis
    "X": GWConfig("cfgX", (2, 1, 1), 6, 460, 6, 6, 20.0, -1.5, 2.0, 0.04, BASE_SEED + 90),
}


def get_config(name) -> GWConfig:
    return CONFIGS[str(name)]
