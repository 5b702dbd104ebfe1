"""Seeded synthetic inputs for the Allegro energy+force hot path (BASELINE.json configs 0-4).

This module holds NO arithmetic of the method (no basis functions, no network, no neighbour search):
only the recipes for positions, species, masses, velocities, hyper-parameter dictionaries and the
random weight blob.  It is the one module that both the fp64 oracle (``oracle/``) and the CUDA path
(``paper_2502_06073_b200.binding``) are allowed to share.  The shapes of the weight tensors are NOT
known here: whoever wants a blob passes the tensor layout it derived itself (the oracle from its own
plan, the CUDA library through ``allegro_weight_layout``).

The paper's own workloads (tobermorite T11, the 6,326-atom C-S-H nanoparticle box of PAPER.md:116,
MPtrj/OFF23 structures) and its trained weights are not available; these seeded systems take their
shape (species mix, density, cutoff, network size) and stand in for them.  Recipes: SURVEY.md §8d
table, readings A21 (velocities) and A24 (weights).
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

AMU_PER_A3_PER_GCC = 1.0 / 1.66053906660  # 1 g/cm^3 in amu/A^3
KB_EV = 8.617333262e-5                     # eV/K             (A20)
ACC_CONV = 9.648533212e-3                  # (eV/A/amu) -> A/fs^2  (A20)

# standard atomic weights (amu) for the species that occur in the configs, by atomic number
ATOMIC_WEIGHT = {1: 1.008, 8: 15.999, 11: 22.98976928, 12: 24.305, 13: 26.9815385, 14: 28.085,
                 20: 40.078, 26: 55.845}

# tensor kinds in a weight layout (must match include/allegro.h ALLEGRO_WK_*)
WK_MATRIX, WK_RESIDUAL, WK_SIGMA, WK_MU = 0, 1, 2, 3


@dataclass
class Workload:
    name: str
    pos: np.ndarray            # [N,3] fp64, Angstrom, unwrapped
    species: np.ndarray        # [N] int32 index into the species embedding
    mass: np.ndarray           # [N] fp64 amu
    cell: np.ndarray           # [3,3] fp64, rows = lattice vectors
    hp: dict                   # network hyper-parameters (keys mirror allegro_hparams)
    skin: float
    dt_fs: float
    n_steps: int
    temperature: float = 300.0
    pos_seed: int = 0
    weight_seed: int = 0
    vel_seed: int = 0
    notes: str = ""
    extra: dict = field(default_factory=dict)

    @property
    def n_atoms(self) -> int:
        return int(self.pos.shape[0])


def hparams(n_species, lmax, n_layers, n_channels, two_body, latent, edge, r_cut, avg_nn,
            n_bessel=8, poly_p=6, full_o3=1) -> dict:
    return dict(n_species=n_species, n_bessel=n_bessel, poly_p=poly_p, lmax=lmax, n_layers=n_layers,
                n_channels=n_channels, full_o3=full_o3, two_body_dims=list(two_body),
                latent_dims=list(latent), edge_dims=list(edge), r_cut=float(r_cut),
                avg_num_neighbors=float(avg_nn))


# ----------------------------------------------------------------------------------------------
# velocities and weights
# ----------------------------------------------------------------------------------------------
def maxwell_boltzmann(mass: np.ndarray, temperature: float, seed: int) -> np.ndarray:
    """A21: per component N(0, sqrt(kB T * 9.648533212e-3 / m)) A/fs, then remove COM velocity."""
    rng = np.random.default_rng(seed)
    v = rng.standard_normal((mass.shape[0], 3))
    v *= np.sqrt(KB_EV * temperature * ACC_CONV / mass)[:, None]
    v -= (mass[:, None] * v).sum(0) / mass.sum()
    return v


def _frac(x: float) -> float:
    return x - math.floor(x)


def make_weights(layout, hp: dict, seed: int) -> np.ndarray:
    """A24: tensors drawn in blob order as standard_normal(shape, fp64)/sqrt(fan_in) -> fp32.

    ``layout`` is a list of (kind, rows, cols).  kind WK_MATRIX: N(0,1/cols) matrix [rows, cols];
    WK_RESIDUAL: the two scalars (c_old, c_new) = 1/sqrt(2); WK_SIGMA / WK_MU: per-species scale
    and shift, sigma_s = (0.9+0.2 frac(0.618034 (s+1)))/sqrt(avg_num_neighbors),
    mu_s = -(1+4 frac(0.381966 (s+1))) eV.
    """
    rng = np.random.default_rng(seed)
    out = []
    for kind, rows, cols in layout:
        if kind == WK_MATRIX:
            w = rng.standard_normal((rows, cols)) / math.sqrt(cols)
            out.append(w.astype(np.float32).ravel())
        elif kind == WK_RESIDUAL:
            out.append(np.full(rows * cols, 1.0 / math.sqrt(2.0), np.float32))
        elif kind == WK_SIGMA:
            s = np.array([(0.9 + 0.2 * _frac(0.618034 * (k + 1))) for k in range(rows * cols)])
            out.append((s / math.sqrt(hp["avg_num_neighbors"])).astype(np.float32))
        elif kind == WK_MU:
            m = np.array([-(1.0 + 4.0 * _frac(0.381966 * (k + 1))) for k in range(rows * cols)])
            out.append(m.astype(np.float32))
        else:
            raise ValueError(f"unknown weight kind {kind}")
    return np.concatenate(out)


# ----------------------------------------------------------------------------------------------
# position recipes
# ----------------------------------------------------------------------------------------------
def _cubic(L: float) -> np.ndarray:
    return np.diag([L, L, L]).astype(np.float64)


def _box_from_density(total_mass_amu: float, rho_gcc: float) -> float:
    return (total_mass_amu / (rho_gcc * AMU_PER_A3_PER_GCC)) ** (1.0 / 3.0)


def _rsa_positions(n: int, L: float, dmin: float, rng) -> np.ndarray:
    """Random sequential addition under periodic boundaries: uniform trial points, rejected when
    closer than dmin to an accepted one (hash grid of side >= dmin for the lookups)."""
    nc = max(1, int(L // dmin))
    h = L / nc
    grid: dict = {}
    pts = np.empty((n, 3))
    k = 0
    d2min = dmin * dmin
    while k < n:
        trial = rng.random((4 * (n - k) + 16, 3)) * L
        for p in trial:
            c = np.minimum((p / h).astype(np.int64), nc - 1)
            ok = True
            for dx in (-1, 0, 1):
                for dy in (-1, 0, 1):
                    for dz in (-1, 0, 1):
                        key = ((c[0] + dx) % nc, (c[1] + dy) % nc, (c[2] + dz) % nc)
                        for q in grid.get(key, ()):
                            d = pts[q] - p
                            d -= L * np.round(d / L)
                            if d @ d < d2min:
                                ok = False
                                break
                        if not ok:
                            break
                    if not ok:
                        break
                if not ok:
                    break
            if ok:
                pts[k] = p
                grid.setdefault((int(c[0]), int(c[1]), int(c[2])), []).append(k)
                k += 1
                if k == n:
                    break
    return pts


def config0() -> Workload:
    rng = np.random.default_rng(0)
    g = np.arange(4)
    ii, jj, kk = np.meshgrid(g, g, g, indexing="ij")
    sites = np.stack([ii, jj, kk], -1).reshape(-1, 3)
    pos = (sites + 0.5) * 2.0 + rng.uniform(-0.3, 0.3, (64, 3))
    species = (sites.sum(1) % 2).astype(np.int32)
    mass = np.where(species == 0, 28.0, 16.0)
    hp = hparams(2, 1, 1, 8, [32, 32], [32, 32], [16], 4.0, 29.4)
    return Workload("cfg0_tiny", pos, species, mass, _cubic(8.0), hp, skin=0.0, dt_fs=0.5, n_steps=10,
                    pos_seed=0, weight_seed=0, vel_seed=1,
                    notes="64-atom jittered SC lattice, 2 species (BASELINE.json configs[0])")


_CFG1_CACHE: dict = {}


def _config1_cell():
    if "c" not in _CFG1_CACHE:
        n_si, n_o = 1365, 2731
        total = n_si * ATOMIC_WEIGHT[14] + n_o * ATOMIC_WEIGHT[8]
        L = _box_from_density(total, 2.2)
        rng = np.random.default_rng(2)
        pos = _rsa_positions(n_si + n_o, L, 1.4, rng)
        species = np.concatenate([np.zeros(n_si, np.int32), np.ones(n_o, np.int32)])
        species = species[rng.permutation(n_si + n_o)]
        _CFG1_CACHE["c"] = (pos, species, L)
    pos, species, L = _CFG1_CACHE["c"]
    return pos.copy(), species.copy(), L


def _cfg1_hp():
    return hparams(2, 2, 2, 16, [128, 64], [128, 64], [64], 5.0, 34.0)


def config1() -> Workload:
    pos, species, L = _config1_cell()
    mass = np.where(species == 0, ATOMIC_WEIGHT[14], ATOMIC_WEIGHT[8])
    return Workload("cfg1_sio2_4096", pos, species, mass, _cubic(L), _cfg1_hp(), skin=0.5, dt_fs=1.0,
                    n_steps=100, pos_seed=2, weight_seed=3, vel_seed=1002,
                    notes="amorphous SiO2-like RSA box, 2.2 g/cc (BASELINE.json configs[1])")


def _random_rotations(n: int, rng) -> np.ndarray:
    q = rng.standard_normal((n, 4))
    q /= np.linalg.norm(q, axis=1, keepdims=True)
    w, x, y, z = q.T
    R = np.empty((n, 3, 3))
    R[:, 0, 0] = 1 - 2 * (y * y + z * z); R[:, 0, 1] = 2 * (x * y - z * w); R[:, 0, 2] = 2 * (x * z + y * w)
    R[:, 1, 0] = 2 * (x * y + z * w); R[:, 1, 1] = 1 - 2 * (x * x + z * z); R[:, 1, 2] = 2 * (y * z - x * w)
    R[:, 2, 0] = 2 * (x * z - y * w); R[:, 2, 1] = 2 * (y * z + x * w); R[:, 2, 2] = 1 - 2 * (x * x + y * y)
    return R


def config2() -> Workload:
    n_mol, n_extra, g = 10922, 2, 23
    total = n_mol * (ATOMIC_WEIGHT[8] + 2 * ATOMIC_WEIGHT[1]) + n_extra * ATOMIC_WEIGHT[8]
    L = _box_from_density(total, 1.0)
    rng = np.random.default_rng(4)
    perm = rng.permutation(g ** 3)
    sites = np.stack(np.unravel_index(perm[: n_mol + n_extra], (g, g, g)), -1).astype(np.float64)
    centres = (sites + 0.5) * (L / g) + rng.uniform(-0.3, 0.3, (n_mol + n_extra, 3))
    R = _random_rotations(n_mol, rng)
    half = math.radians(104.5) / 2.0
    h1 = 0.96 * np.array([math.sin(half), 0.0, math.cos(half)])
    h2 = 0.96 * np.array([-math.sin(half), 0.0, math.cos(half)])
    mol = np.empty((n_mol, 3, 3))
    mol[:, 0] = centres[:n_mol]
    mol[:, 1] = centres[:n_mol] + R @ h1
    mol[:, 2] = centres[:n_mol] + R @ h2
    pos = np.concatenate([mol.reshape(-1, 3), centres[n_mol:]])
    species = np.concatenate([np.tile(np.array([1, 0, 0], np.int32), n_mol), np.ones(n_extra, np.int32)])
    mass = np.where(species == 0, ATOMIC_WEIGHT[1], ATOMIC_WEIGHT[8])  # species 0 = H, 1 = O
    hp = hparams(2, 2, 2, 32, [256, 128], [256, 128], [128], 6.0, 86.0)
    return Workload("cfg2_water_32768", pos, species, mass, _cubic(L), hp, skin=0.5, dt_fs=0.5,
                    n_steps=1000, pos_seed=4, weight_seed=5, vel_seed=1004,
                    notes="water-like box, 1.0 g/cc (BASELINE.json configs[2])")


def config3() -> Workload:
    Z = np.array([20, 14, 8, 1, 13, 11, 12, 26])          # Ca Si O H Al Na Mg Fe
    counts = np.array([27594, 27594, 124176, 55188, 6898, 6898, 6898, 6898])
    n = int(counts.sum())
    assert n == 262144
    total = float(sum(c * ATOMIC_WEIGHT[int(z)] for c, z in zip(counts, Z)))
    L = _box_from_density(total, 2.5)
    rng = np.random.default_rng(6)
    a, c = L / 32, L / 64
    ii, jj, kk = np.meshgrid(np.arange(32), np.arange(32), np.arange(64), indexing="ij")
    corner = np.stack([ii * a, jj * a, kk * c], -1).reshape(-1, 1, 3)
    basis = np.array([[0, 0, 0], [0.5 * a, 0.5 * a, 0], [0.5 * a, 0, 0.5 * c], [0, 0.5 * a, 0.5 * c]])
    pos = (corner + basis[None]).reshape(-1, 3) + rng.uniform(-0.4, 0.4, (n, 3))
    species = np.repeat((Z - 1).astype(np.int32), counts)[rng.permutation(n)]
    weight_of = np.zeros(89)
    for z in Z:
        weight_of[z - 1] = ATOMIC_WEIGHT[int(z)]
    mass = weight_of[species]
    hp = hparams(89, 3, 3, 64, [128, 256, 512], [512, 512, 512], [128], 6.0, 73.4)
    return Workload("cfg3_fm_262144", pos, species, mass, _cubic(L), hp, skin=0.5, dt_fs=0.5, n_steps=100,
                    pos_seed=6, weight_seed=7, vel_seed=1006,
                    notes="FM-sized network, 8 of 89 species, jittered FCT lattice (BASELINE.json configs[3])")


_CFG4_TILINGS = {15: (2, 2, 2), 17: (4, 4, 2), 19: (8, 4, 4), 21: (8, 8, 8), 23: (16, 16, 8), 26: (32, 32, 16),
                 25: (32, 16, 16), 27: (32, 32, 32)}


def config4(log2_n: int = 15) -> Workload:
    tx, ty, tz = _CFG4_TILINGS[log2_n]
    pos0, sp0, L = _config1_cell()
    rng = np.random.default_rng(8)
    offs = np.stack(np.meshgrid(np.arange(tx), np.arange(ty), np.arange(tz), indexing="ij"), -1).reshape(-1, 3)
    pos = (pos0[None] + offs[:, None, :] * L).reshape(-1, 3)
    pos = pos + rng.uniform(-0.05, 0.05, pos.shape)
    species = np.tile(sp0, offs.shape[0])
    mass = np.where(species == 0, ATOMIC_WEIGHT[14], ATOMIC_WEIGHT[8])
    cell = np.diag([tx * L, ty * L, tz * L]).astype(np.float64)
    n_steps = 100 if log2_n <= 21 else 10
    return Workload(f"cfg4_sio2_2^{log2_n}", pos, species, mass, cell, _cfg1_hp(), skin=0.5, dt_fs=1.0,
                    n_steps=n_steps, pos_seed=8, weight_seed=3, vel_seed=1008,
                    notes="cfg-1 cell tiled %dx%dx%d with +-0.05 A jitter (BASELINE.json configs[4])" % (tx, ty, tz))


def cluster(n_atoms: int = 7, n_species: int = 2, seed: int = 11, spread: float = 2.2, box: float = 40.0):
    """Small open cluster in a big periodic box (for the oracle's invariance / torque pins)."""
    rng = np.random.default_rng(seed)
    pos = box / 2 + rng.uniform(-spread, spread, (n_atoms, 3))
    species = rng.integers(0, n_species, n_atoms).astype(np.int32)
    return pos, species, _cubic(box)


def small_periodic(n_side: int = 3, spacing: float = 2.3, jitter: float = 0.35, n_species: int = 2, seed: int = 12):
    """Small jittered periodic lattice (box = n_side*spacing) for FD / supercell / skin pins."""
    rng = np.random.default_rng(seed)
    g = np.arange(n_side)
    sites = np.stack(np.meshgrid(g, g, g, indexing="ij"), -1).reshape(-1, 3)
    pos = (sites + 0.5) * spacing + rng.uniform(-jitter, jitter, (sites.shape[0], 3))
    species = rng.integers(0, n_species, sites.shape[0]).astype(np.int32)
    return pos, species, _cubic(n_side * spacing)


def get(cfg: int, **kw) -> Workload:
    return {0: config0, 1: config1, 2: config2, 3: config3, 4: config4}[cfg](**kw)
