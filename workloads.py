"""Seeded synthetic inputs for the NEP hot path (shared by the oracle tests and the CUDA path).

This module holds NO arithmetic of the method (no basis functions, descriptors, network, forces):
only lattices, displacements, species, random parameters and Maxwell-Boltzmann velocities, so that
the fp64 oracle (oracle/) and the CUDA library (paper_2205_10046_b200/) can be fed identical arrays
without sharing any code of their own.

The five configurations are the ones listed in BASELINE.json `configs`; the readings of the
under-specified items are restated in DESIGN.md:
  * "n_max=4 from 8 basis functions" -> n_max=4 (n=0..4), N_bas=8 (k=0..8).
  * parameters U(-0.5,0.5)/sqrt(fan_in): w0,b0 fan_in=N_des; w1,b1 fan_in=N_neu; c^R fan_in=N_bas^R+1;
    c^A fan_in=N_bas^A+1; drawn in fp64, rounded to fp32; the fp32 values are THE parameters.
  * velocities: Maxwell-Boltzmann at T, centre-of-mass motion removed, rescaled to exactly T (3N dof).
Units: eV, Angstrom, amu, fs, K.
"""
from __future__ import annotations

from dataclasses import dataclass, field, replace
from typing import Optional, Tuple

import numpy as np

KB_EV_PER_K = 8.617333262e-5          # Boltzmann constant, eV/K
ACC_CONV = 9.648533212e-3             # (eV/Angstrom/amu) -> Angstrom/fs^2


@dataclass(frozen=True)
class Hyper:
    """NEP3 hyper-parameters in the paper's notation."""
    n_types: int
    rc_radial: float
    rc_angular: float
    n_max_radial: int      # n = 0..n_max^R
    n_max_angular: int     # n = 0..n_max^A
    basis_radial: int      # k = 0..N_bas^R
    basis_angular: int     # k = 0..N_bas^A
    n_neurons: int
    l_max_3b: int = 4
    l_max_4b: int = 2      # 0 = no 4-body block
    l_max_5b: int = 1      # 0 = no 5-body block

    @property
    def NR(self) -> int: return self.n_max_radial + 1
    @property
    def KR(self) -> int: return self.basis_radial + 1
    @property
    def NA(self) -> int: return self.n_max_angular + 1
    @property
    def KA(self) -> int: return self.basis_angular + 1
    @property
    def n_blocks(self) -> int:
        return self.l_max_3b + (1 if self.l_max_4b >= 2 else 0) + (1 if self.l_max_5b >= 1 else 0)
    @property
    def n_des(self) -> int:
        """Eq. (20), PAPER.md:192-197 (a counting formula, not arithmetic of the method)."""
        return self.NR + self.NA * self.n_blocks


@dataclass
class Params:
    """fp32 model parameters; layouts as in include/nep.h."""
    c_radial: np.ndarray    # [T][T][NR][KR]  index (t_i, t_j, n, k)
    c_angular: np.ndarray   # [T][T][NA][KA]
    w0: np.ndarray          # [H][D] row-major as Listing 1
    b0: np.ndarray          # [H]
    w1: np.ndarray          # [H]
    b1: np.ndarray          # [1]


@dataclass
class Config:
    name: str
    index: int
    lattice: str                       # diamond | rocksalt | fcc | bcc
    a: float
    cells: Tuple[int, int, int]
    sigma: float
    masses: Tuple[float, ...]
    species_rule: str                  # single | sublattice | random
    hyper: Hyper
    temperature: float
    dt_fs: float
    n_steps: int
    skin: float
    rebuild_every: int


_BASIS = {
    "diamond": np.array([[0, 0, 0], [0, .5, .5], [.5, 0, .5], [.5, .5, 0],
                         [.25, .25, .25], [.25, .75, .75], [.75, .25, .75], [.75, .75, .25]]),
    # rock salt: first four sites = fcc sublattice of species 0, last four = species 1
    "rocksalt": np.array([[0, 0, 0], [0, .5, .5], [.5, 0, .5], [.5, .5, 0],
                          [.5, 0, 0], [0, .5, 0], [0, 0, .5], [.5, .5, .5]]),
    "fcc": np.array([[0, 0, 0], [0, .5, .5], [.5, 0, .5], [.5, .5, 0]]),
    "bcc": np.array([[0, 0, 0], [.5, .5, .5]]),
}

_H_SMALL = dict(rc_radial=5.0, rc_angular=4.0, n_max_radial=4, n_max_angular=4,
                basis_radial=8, basis_angular=8, n_neurons=30)

CONFIGS = [
    Config("cfg0_diamond_256", 0, "diamond", 5.43, (4, 4, 2), 0.05, (28.0,), "single",
           Hyper(n_types=1, **_H_SMALL), 300.0, 1.0, 10, 0.0, 1),
    Config("cfg1_diamond_64k", 1, "diamond", 5.43, (20, 20, 20), 0.1, (28.0,), "single",
           Hyper(n_types=1, **_H_SMALL), 300.0, 1.0, 1000, 1.0, 10),
    Config("cfg2_rocksalt_110k", 2, "rocksalt", 6.46, (24, 24, 24), 0.1, (207.0, 128.0), "sublattice",
           Hyper(n_types=2, rc_radial=6.0, rc_angular=4.0, n_max_radial=6, n_max_angular=4,
                 basis_radial=10, basis_angular=8, n_neurons=50), 700.0, 1.0, 1000, 1.0, 10),
    Config("cfg3_fcc_alloy_1M", 3, "fcc", 3.6, (63, 63, 63), 0.1, (56.0, 59.0, 52.0, 55.0, 63.0), "random",
           Hyper(n_types=5, **_H_SMALL), 300.0, 1.0, 500, 1.0, 10),
    Config("cfg4_bcc_8M", 4, "bcc", 3.16, (160, 160, 160), 0.3, (184.0,), "single",
           Hyper(n_types=1, rc_radial=6.0, rc_angular=5.0, n_max_radial=6, n_max_angular=6,
                 basis_radial=10, basis_angular=10, n_neurons=50), 300.0, 1.0, 200, 1.0, 10),
]


def get_config(index: int, cells: Optional[Tuple[int, int, int]] = None) -> Config:
    """Config `index` of BASELINE.json; `cells` overrides the replica count (scaled-down test cases)."""
    cfg = CONFIGS[index]
    return replace(cfg, cells=tuple(cells)) if cells is not None else cfg


def _streams(cfg_index: int):
    """Independent child streams {displacements, species, parameters, velocities}."""
    ss = np.random.SeedSequence([2205, 10046, cfg_index])
    return [np.random.default_rng(s) for s in ss.spawn(4)]


@dataclass
class System:
    pos: np.ndarray        # [N][3] fp64, wrapped into [0, L)
    types: np.ndarray      # [N] int32
    box: np.ndarray        # [3] fp64 orthorhombic edge lengths
    masses: np.ndarray     # [T] fp64 amu
    vel: np.ndarray        # [N][3] fp64 Angstrom/fs


def make_system(cfg: Config) -> System:
    """Positions: conventional-cell-major, basis-minor order; Gaussian displacement; wrapped."""
    r_disp, r_spec, _, r_vel = _streams(cfg.index)
    basis = _BASIS[cfg.lattice]
    nx, ny, nz = cfg.cells
    nb = len(basis)
    ix, iy, iz = np.meshgrid(np.arange(nx), np.arange(ny), np.arange(nz), indexing="ij")
    origin = np.stack([ix.ravel(), iy.ravel(), iz.ravel()], axis=1).astype(np.float64)   # [cells][3]
    frac = origin[:, None, :] + basis[None, :, :]                                         # [cells][nb][3]
    pos = (frac.reshape(-1, 3) * cfg.a)
    n = pos.shape[0]
    box = np.array([nx, ny, nz], dtype=np.float64) * cfg.a
    pos = pos + r_disp.normal(0.0, cfg.sigma, size=(n, 3))
    pos -= box * np.floor(pos / box)
    pos = np.where(pos >= box, pos - box, pos)      # guard the fp edge case x == L after the wrap

    if cfg.species_rule == "single":
        types = np.zeros(n, dtype=np.int32)
    elif cfg.species_rule == "sublattice":
        types = np.tile((np.arange(nb) >= nb // 2).astype(np.int32), nx * ny * nz)
    elif cfg.species_rule == "random":
        types = r_spec.integers(0, cfg.hyper.n_types, size=n).astype(np.int32)
    else:
        raise ValueError(cfg.species_rule)

    masses = np.asarray(cfg.masses, dtype=np.float64)
    vel = maxwell_boltzmann(r_vel, masses[types], cfg.temperature)
    return System(np.ascontiguousarray(pos), types, box, masses, vel)


def maxwell_boltzmann(rng: np.random.Generator, m_per_atom: np.ndarray, temperature: float) -> np.ndarray:
    """v_a ~ N(0, k_B T / m), COM velocity removed, rescaled to exactly T with 3N degrees of freedom."""
    n = m_per_atom.shape[0]
    if temperature <= 0.0:
        return np.zeros((n, 3))
    sig = np.sqrt(KB_EV_PER_K * temperature / m_per_atom * ACC_CONV)
    v = rng.normal(size=(n, 3)) * sig[:, None]
    v -= (m_per_atom[:, None] * v).sum(axis=0) / m_per_atom.sum()
    t_now = (m_per_atom[:, None] * v * v).sum() / ACC_CONV / (3.0 * n * KB_EV_PER_K)
    return v * np.sqrt(temperature / t_now)


def make_params(cfg: Config, kind: str = "baseline") -> Params:
    """kind='baseline': U(-0.5,0.5)/sqrt(fan_in) (BASELINE.json).
    kind='stress': c ~ U(0,1)/sqrt(K), w0 x4 -- makes the 4-/5-body terms O(0.1-1) so that a wrong
    many-body term cannot hide under the absolute tolerances (SURVEY.md section 7 'weak signal')."""
    rng = _streams(cfg.index)[2]
    h = cfg.hyper
    T, D, H = h.n_types, h.n_des, h.n_neurons

    def u(shape, fan_in):
        return rng.uniform(-0.5, 0.5, size=shape) / np.sqrt(fan_in)

    c_r = u((T, T, h.NR, h.KR), h.KR)
    c_a = u((T, T, h.NA, h.KA), h.KA)
    w0 = u((H, D), D)
    b0 = u((H,), D)
    w1 = u((H,), H)
    b1 = u((1,), H)
    if kind == "stress":
        c_r = (c_r * np.sqrt(h.KR) + 0.5) / np.sqrt(h.KR)
        c_a = (c_a * np.sqrt(h.KA) + 0.5) / np.sqrt(h.KA)
        w0 = w0 * 4.0
    elif kind != "baseline":
        raise ValueError(kind)
    f32 = lambda a: np.ascontiguousarray(a.astype(np.float32))
    return Params(f32(c_r), f32(c_a), f32(w0), f32(b0), f32(w1), f32(b1))


def random_cluster(seed: int, n: int, n_types: int, extent: float, min_dist: float = 1.2):
    """Open (non-periodic) random cluster for the invariance / finite-difference pins: n points in a
    cube of edge `extent`, rejection-sampled so that no two are closer than `min_dist`."""
    rng = np.random.default_rng(np.random.SeedSequence([2205, 10046, 900, seed]))
    pts = []
    while len(pts) < n:
        p = rng.uniform(0.0, extent, size=3)
        if all(np.linalg.norm(p - q) >= min_dist for q in pts):
            pts.append(p)
    types = rng.integers(0, n_types, size=n).astype(np.int32)
    return np.array(pts), types


def sheared(system: "System", xy: float, xz: float, yz: float):
    """A genuinely triclinic copy of an orthorhombic system: positions and cell mapped by r' = r F with
    F = [[1,0,0],[xy,1,0],[xz,yz,1]] (row vectors).  Returns (pos', box'[3][3]) with rows a', b', c'."""
    F = np.array([[1.0, 0.0, 0.0], [xy, 1.0, 0.0], [xz, yz, 1.0]])
    return np.ascontiguousarray(system.pos @ F), np.diag(system.box) @ F


def perpendicular_widths(box33) -> np.ndarray:
    """Distances between opposite faces of the cell with rows a, b, c."""
    H = np.asarray(box33, dtype=np.float64).reshape(3, 3)
    vol = abs(np.linalg.det(H))
    a, b, c = H
    return np.array([vol / np.linalg.norm(np.cross(b, c)), vol / np.linalg.norm(np.cross(c, a)),
                     vol / np.linalg.norm(np.cross(a, b))])


def make_batch(idx: int, specs):
    """A batch of small structures for the training-evaluation path: specs =
    [(cells, tilt or None, seed)], each a replica of config `idx`'s lattice and species rule with its own seeded
    displacements (sigma 0.05 A), optionally sheared by the lower-triangular tilt (xy, xz, yz), positions shifted by
    random lattice vectors (unwrapped input).  Returns [(pos [n][3], types [n], cell rows [3][3])].  They stand in
    for the paper's DFT training structures, which are not available."""
    structs = []
    for k, (cells, tilt, seed) in enumerate(specs):
        cfg = get_config(idx, cells)
        s = make_system(cfg)
        rng = np.random.default_rng(np.random.SeedSequence([2205, 10046, 930, idx, k, seed]))
        pos = s.pos + rng.normal(0.0, 0.05, size=s.pos.shape)               # every structure its own displacements
        H = np.diag(s.box)
        if tilt is not None:
            F = np.array([[1.0, 0.0, 0.0], [tilt[0], 1.0, 0.0], [tilt[1], tilt[2], 1.0]])
            pos, H = pos @ F, H @ F
        pos = pos + rng.integers(-1, 2, size=pos.shape).astype(np.float64) @ H   # unwrapped input
        structs.append((np.ascontiguousarray(pos), s.types.copy(), H))
    return structs


def make_population(cfg: Config, n_pop: int, sigma: float = 0.1, kind: str = "stress"):
    """A seeded population of parameter sets around make_params(cfg, kind), as an evolution strategy draws
    them: member m = mean + sigma * N(0, 1) per parameter, rounded to fp32.  Member 0 is the
    mean itself.  With nep2=True-like patterns see nep2_pattern()."""
    mean = make_params(cfg, kind)
    rng = np.random.default_rng(np.random.SeedSequence([2205, 10046, 905, cfg.index, n_pop]))
    members = [mean]
    for _ in range(1, n_pop):
        members.append(Params(*[np.ascontiguousarray((a.astype(np.float64) + sigma * rng.normal(size=a.shape) * np.abs(a).mean()).astype(np.float32))
                                for a in (mean.c_radial, mean.c_angular, mean.w0, mean.b0, mean.w1, mean.b1)]))
    return members


def nep2_pattern(params: Params) -> Params:
    """The NEP2 special case of the NEP3 radial functions: c_nk^{ij} = delta_nk c_n^{ij}, i.e.
    g_n = c_n^{ij} f_n -- every coefficient with k != n set to zero (needs N_bas >= n_max)."""
    out = []
    for c in (params.c_radial, params.c_angular):
        z = np.zeros_like(c)
        for n_ in range(min(c.shape[2], c.shape[3])):
            z[:, :, n_, n_] = c[:, :, n_, n_]
        out.append(z)
    return Params(out[0], out[1], params.w0, params.b0, params.w1, params.b1)
