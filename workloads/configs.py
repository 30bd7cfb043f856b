"""The five BASELINE.json configurations (synthetic Si-like cells).

Recipe: SURVEY.md section 8(d) "Synthetic inputs" and DESIGN.md section 4.
The paper's own workloads are Si supercells with SG15 ONCV pseudopotentials
(Appendix E); those files are not available, so these
cells stand in for them with the same shapes.
"""
from __future__ import annotations

from dataclasses import dataclass
import numpy as np

ALAT = 10.26  # bohr, BASELINE.json configs


@dataclass(frozen=True)
class Config:
    name: str
    cell: str            # "fcc" (2 atoms) or "sc" (8*s^3 atoms)
    supercell: int       # s (1 for fcc)
    ecutwfc_ry: float
    grid: tuple
    nbands: int
    nk: int              # 1 => Gamma only, else seeded random k
    call_batch: int      # bands per qm_apply_h call
    dense_d: bool        # per-atom dense 4x4 D blocks (cfg 5) or diag(1,.5,.5,.5)

    @property
    def natoms(self) -> int:
        return 2 if self.cell == "fcc" else 8 * self.supercell ** 3

    @property
    def nproj(self) -> int:
        return 4 * self.natoms


CONFIGS = {
    "cfg1": Config("cfg1", "fcc", 1, 25.0, (24, 24, 24), 8, 1, 8, False),
    "cfg2": Config("cfg2", "fcc", 1, 30.0, (32, 32, 32), 16, 10, 16, False),
    "cfg3": Config("cfg3", "sc", 1, 30.0, (48, 48, 48), 64, 1, 64, False),
    "cfg4": Config("cfg4", "sc", 2, 30.0, (96, 96, 96), 256, 1, 32, False),
    "cfg5": Config("cfg5", "sc", 3, 30.0, (144, 144, 144), 512, 1, 16, True),
}


def get_config(name: str) -> Config:
    return CONFIGS[name]


def cell_for(cfg: Config):
    """Return (lattice[3,3] rows a_i in bohr, atom positions[natoms,3] Cartesian bohr).

    fcc axes follow the convention printed in the paper's examples
    (SURVEY A7): (a/2)(-1,0,1), (a/2)(0,1,1), (a/2)(-1,1,0).
    Atom order defines projector order 4*atom + {s, px, py, pz}.
    """
    a = ALAT
    if cfg.cell == "fcc":
        lat = 0.5 * a * np.array([[-1.0, 0.0, 1.0], [0.0, 1.0, 1.0], [-1.0, 1.0, 0.0]])
        pos = np.array([[0.0, 0.0, 0.0], [0.25 * a, 0.25 * a, 0.25 * a]])
        return lat, pos
    s = cfg.supercell
    lat = np.eye(3) * (a * s)
    fcc_sites = np.array([[0, 0, 0], [0, .5, .5], [.5, 0, .5], [.5, .5, 0]], dtype=np.float64)
    pos = []
    for i in range(s):
        for j in range(s):
            for k in range(s):
                origin = np.array([i, j, k], dtype=np.float64)
                for site in fcc_sites:
                    pos.append((origin + site) * a)
                    pos.append((origin + site + 0.25) * a)
    return lat, np.array(pos)
