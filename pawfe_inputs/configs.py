"""Workload shapes and seeded input data.  No FE / PAW operator arithmetic lives here.

Citations: BASELINE.json ``configs`` (the five shapes); SURVEY.md section 8(d) "Synthetic inputs";
PAPER.md:L470 (Table 2: (p, h) pairs), PAPER.md:L585 (up to two partial waves per l).
"""
from __future__ import annotations

import dataclasses
import math
from dataclasses import dataclass
from typing import Optional, Tuple

import numpy as np


@dataclass(frozen=True)
class Config:
    name: str
    ncells: Tuple[int, int, int]
    p: int                      # FE polynomial order, n_p = p + 1 GLL nodes per direction
    box: Tuple[float, float, float]   # bohr
    bc: str                     # "periodic" | "dirichlet"
    kfrac: Optional[Tuple[float, float, float]]  # k = kfrac * 2*pi/L per direction, None = real
    natoms: int
    Z: float                    # depth of the Gaussian well  -Z exp(-r^2 / 2 sigmaV^2)
    sigmaV: float
    nproj: int                  # 4 = {s,p}; 9 = {s,p,d}; 13 = {s,s',p,p',d}
    rc: float                   # projector cutoff radius (bohr)
    nvec: int                   # N
    block: int                  # B
    degree: int                 # Chebyshev degree m
    outer: int                  # outer ChFSI iterations for the full-loop test
    seed: int
    precisions: Tuple[str, ...]
    min_sep: float = 2.0
    wall_margin: float = 0.0    # Dirichlet: atoms placed in [margin, L - margin)

    @property
    def complex(self) -> bool:
        return self.kfrac is not None

    @property
    def nodes_per_dir(self) -> Tuple[int, int, int]:
        extra = 1 if self.bc == "dirichlet" else 0
        return tuple(n * self.p + extra for n in self.ncells)

    @property
    def ndofs_stored(self) -> int:
        nx, ny, nz = self.nodes_per_dir
        return nx * ny * nz

    @property
    def kpoint(self) -> Optional[np.ndarray]:
        if self.kfrac is None:
            return None
        return np.array([f * 2.0 * math.pi / L for f, L in zip(self.kfrac, self.box)])


def _cube(nc, p, h, **kw) -> dict:
    return dict(ncells=(nc, nc, nc), p=p, box=(nc * h, nc * h, nc * h), **kw)


_BASE_SEED = 26037 * 10

CONFIGS = {
    # BASELINE.json configs[0]: tiny periodic cube, side 8 bohr, 2^3 cells, p=4, real FP64
    0: Config(name="cfg0_tiny_p4", **_cube(2, 4, 4.0), bc="periodic", kfrac=None, natoms=2, Z=4.0,
              sigmaV=0.8, nproj=4, rc=3.0, nvec=16, block=16, degree=10, outer=30,
              seed=_BASE_SEED + 0, precisions=("fp64", "fp32", "tf32")),
    # configs[1]: 16^3 cells, p=6, h=2.0, 64 atoms, 9 projectors, 400 vec / B=200, m=20
    1: Config(name="cfg1_16c_p6", **_cube(16, 6, 2.0), bc="periodic", kfrac=None, natoms=64, Z=6.0,
              sigmaV=0.8, nproj=9, rc=3.0, nvec=400, block=200, degree=20, outer=1,
              seed=_BASE_SEED + 1, precisions=("fp32", "tf32")),
    # configs[2]: 24^3 cells, p=7, h=1.9, 256 atoms, 13 projectors, 1500 vec / B=250, m=24
    2: Config(name="cfg2_24c_p7", **_cube(24, 7, 1.9), bc="periodic", kfrac=None, natoms=256, Z=8.0,
              sigmaV=0.8, nproj=13, rc=3.0, nvec=1500, block=250, degree=24, outer=1,
              seed=_BASE_SEED + 2, precisions=("tf32",)),
    # configs[3]: complex single k-point, 20^3 cells, p=6, 128 atoms, 9 projectors, 800 / 200, m=20
    3: Config(name="cfg3_20c_p6_k", **_cube(20, 6, 2.0), bc="periodic", kfrac=(0.25, 0.25, 0.25),
              natoms=128, Z=6.0, sigmaV=0.8, nproj=9, rc=3.0, nvec=800, block=200, degree=20,
              outer=1, seed=_BASE_SEED + 3, precisions=("fp32", "tf32")),
    # configs[4]: 32^3 cells, p=6, Dirichlet, 1000 atoms, 13 projectors, 5000 / 256, m=30
    4: Config(name="cfg4_32c_p6_dirichlet", **_cube(32, 6, 2.0), bc="dirichlet", kfrac=None,
              natoms=1000, Z=10.0, sigmaV=0.8, nproj=13, rc=3.0, nvec=5000, block=256, degree=30,
              outer=1, seed=_BASE_SEED + 4, precisions=("tf32",), wall_margin=4.0),
}


def get_config(i: int) -> Config:
    return CONFIGS[i]


def twin(cfg: Config, nc: int = 4, natoms: Optional[int] = None, nvec: Optional[int] = None,
         block: Optional[int] = None, degree: Optional[int] = None, outer: Optional[int] = None) -> Config:
    """Reduced-cell twin: same p, h, potential, projector set, BC and k; fewer cells/atoms/vectors.

    Used where the oracle must finish in seconds.
    """
    h = cfg.box[0] / cfg.ncells[0]
    if natoms is None:
        natoms = max(2, round(cfg.natoms * nc ** 3 / (cfg.ncells[0] * cfg.ncells[1] * cfg.ncells[2])))
    margin = min(cfg.wall_margin, 0.25 * nc * h)
    return dataclasses.replace(
        cfg, name=f"{cfg.name}_twin{nc}", ncells=(nc, nc, nc), box=(nc * h, nc * h, nc * h),
        natoms=natoms, nvec=nvec or min(cfg.nvec, 24), block=block or min(cfg.block, 24),
        degree=degree or cfg.degree, outer=outer or cfg.outer, wall_margin=margin)


# ----------------------------------------------------------------------------------------------
# projector channel table ("dataset")
# ----------------------------------------------------------------------------------------------

_CHANNELS = {
    4: [(0, 0.7), (1, 0.7)],
    9: [(0, 0.7), (1, 0.7), (2, 0.7)],
    13: [(0, 0.7), (0, 0.5), (1, 0.7), (1, 0.5), (2, 0.7)],
}


def _radial_norm(l: int, sigma: float, rc: float) -> float:
    """int_0^rc [r^l exp(-r^2/2 sigma^2) (1-(r/rc)^2)^2]^2 r^2 dr by 200-point Gauss-Legendre."""
    x, w = np.polynomial.legendre.leggauss(200)
    r = 0.5 * rc * (x + 1.0)
    f = r ** l * np.exp(-r * r / (2.0 * sigma * sigma)) * (1.0 - (r / rc) ** 2) ** 2
    return float(0.5 * rc * np.sum(w * f * f * r * r))


def projector_table(nproj: int, rc: float):
    """Return (l, m, sigma, amp) arrays of length nproj.

    Projector alpha is  amp * r^l exp(-r^2 / 2 sigma^2) (1 - (r/rc)^2)^2 Y_lm(rhat)  for r < rc, else 0
    (real orthonormal spherical harmonics; order m = -l..l).  amp makes the L2 norm 1.
    """
    ls, ms, sg, amp = [], [], [], []
    for (l, s) in _CHANNELS[nproj]:
        a = 1.0 / math.sqrt(_radial_norm(l, s, rc))
        for m in range(-l, l + 1):
            ls.append(l); ms.append(m); sg.append(s); amp.append(a)
    assert len(ls) == nproj
    return (np.array(ls, dtype=np.int32), np.array(ms, dtype=np.int32),
            np.array(sg, dtype=np.float64), np.array(amp, dtype=np.float64))


def _max_channels_per_l(nproj: int) -> int:
    counts = {}
    for (l, _) in _CHANNELS[nproj]:
        counts[l] = counts.get(l, 0) + 1
    return max(counts.values())


# ----------------------------------------------------------------------------------------------
# seeded system
# ----------------------------------------------------------------------------------------------

@dataclass
class System:
    cfg: Config
    pos: np.ndarray        # (natoms, 3) float64
    Z: np.ndarray          # (natoms,)
    sigmaV: np.ndarray     # (natoms,)
    proj_l: np.ndarray     # (nproj,) int32
    proj_m: np.ndarray     # (nproj,) int32
    proj_sigma: np.ndarray  # (nproj,)
    proj_amp: np.ndarray   # (nproj,)
    rc: float
    D: np.ndarray          # (natoms, nproj, nproj) real symmetric  (Delta_H)
    dS: np.ndarray         # (natoms, nproj, nproj) real symmetric  (Delta_S)


def _place_atoms(rng, cfg: Config) -> np.ndarray:
    L = np.array(cfg.box)
    lo = np.full(3, cfg.wall_margin)
    hi = L - cfg.wall_margin
    pos = []
    tries = 0
    while len(pos) < cfg.natoms:
        tries += 1
        if tries > 200000:
            raise RuntimeError("atom placement failed")
        x = lo + (hi - lo) * rng.random(3)
        ok = True
        for y in pos:
            d = x - y
            if cfg.bc == "periodic":
                d -= L * np.round(d / L)
            if d @ d < cfg.min_sep ** 2:
                ok = False
                break
        if ok:
            pos.append(x)
    return np.array(pos)


def make_system(cfg: Config) -> System:
    """One rng stream; order: positions, D, dS."""
    rng = np.random.default_rng(cfg.seed)
    pos = _place_atoms(rng, cfg)
    npj = cfg.nproj

    def sym():
        a = rng.uniform(-0.1, 0.1, size=(cfg.natoms, npj, npj))
        iu = np.triu_indices(npj, 1)
        a[:, iu[1], iu[0]] = a[:, iu[0], iu[1]]
        return a

    D = sym()
    dS = sym()
    # "Delta_S scaled so S stays SPD" (BASELINE.json configs[0]); reading R11: an
    # input-only guard  ||dS^a||_2 <= 0.8 / (max channels per l), because unit-norm projectors of one
    # (l, m) have a Gram matrix with lambda_max <= number of channels.
    cap = 0.8 / _max_channels_per_l(npj)
    for a in range(cfg.natoms):
        rho = np.max(np.abs(np.linalg.eigvalsh(dS[a])))
        if rho > cap:
            dS[a] *= cap / rho
    l, m, sg, amp = projector_table(npj, cfg.rc)
    return System(cfg=cfg, pos=pos, Z=np.full(cfg.natoms, cfg.Z), sigmaV=np.full(cfg.natoms, cfg.sigmaV),
                  proj_l=l, proj_m=m, proj_sigma=sg, proj_amp=amp, rc=cfg.rc, D=D, dS=dS)


def random_block(cfg: Config, ncols: int, stream: int = 0) -> np.ndarray:
    """Seeded block (ndofs_stored x ncols), entries U[-0.5, 0.5] (complex: both parts)."""
    rng = np.random.default_rng([cfg.seed, 1000 + stream])
    M = cfg.ndofs_stored
    x = rng.uniform(-0.5, 0.5, size=(M, ncols))
    if cfg.complex:
        x = x + 1j * rng.uniform(-0.5, 0.5, size=(M, ncols))
    return x
