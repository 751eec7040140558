"""Seeded synthetic inputs shared by the oracle tests and the CUDA path.

This module holds NO arithmetic of the method (no neighbour search, no features, no
network evaluation). It only draws random numbers: atom positions, species, vacancies,
molecule orientations and the fp32 weight blob, following the recipes of DESIGN.md
"Input recipe"; the inputs stand in for the paper's Li3PO4 / Si-O /
Pt-TiO2 workloads (Table 2), which are not available here.

Both `oracle/` and `paper_2509_21694_b200/` consumers receive the same arrays; neither of
them imports the other.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

FCC_BASIS = np.array(
    [[0.0, 0.0, 0.0], [0.5, 0.5, 0.0], [0.5, 0.0, 0.5], [0.0, 0.5, 0.5]], dtype=np.float64
)


@dataclass
class ModelSpec:
    """Shape of the MPNN (BASELINE.json configs); mirrors `mlip_model_header` in include/mlip.h."""

    n_species: int
    d: int
    n_rbf: int
    L_max: int
    r_cut: float
    agg_scale: float  # alpha = 1/sqrt(nominal mean degree), reading R7
    r_cut3: float = 0.0  # > 0: three-body variant (header flags bit 0): per layer G[16,d], g[16], W3[d,16] follow c2

    def n_weights(self) -> int:
        S, d, k = self.n_species, self.d, self.n_rbf
        per_layer = d * (2 * d + k) + d + d * d + d + d * 2 * d + d + d * d + d
        if self.r_cut3 > 0.0:
            per_layer += 16 * d + 16 + d * 16
        return S * d + S + self.L_max * per_layer + d * d + d + d + 1


@dataclass
class System:
    pos: np.ndarray  # [N,3] float64, unwrapped (jitter may leave the box)
    cell: np.ndarray  # [3,3] float64, rows a1,a2,a3
    species: np.ndarray  # [N] int32
    name: str = ""


@dataclass
class Config:
    """One benchmark configuration (BASELINE.json `configs[c-1]`)."""

    number: int
    system: System
    model: ModelSpec
    L: int
    precision: str  # "fp32" | "bf16"
    grid: tuple = (1, 1, 1)  # spatial sub-domains
    halo: float = 0.0
    weights: np.ndarray = field(default=None, repr=False)  # fp32 blob


def fcc_box(n_cells: int, a: float = 3.6) -> tuple[np.ndarray, np.ndarray]:
    """fcc sites for (ix,iy,iz) in C order times the 4-atom basis; cubic cell n_cells*a."""
    idx = np.indices((n_cells, n_cells, n_cells)).reshape(3, -1).T.astype(np.float64)  # C order
    sites = (idx[:, None, :] + FCC_BASIS[None, :, :]).reshape(-1, 3) * a
    cell = np.eye(3, dtype=np.float64) * (n_cells * a)
    return sites, cell


def make_fcc_system(n_cells: int, sigma: float, seed_pos: int, seed_species: int,
                    n_species: int = 4, vacancy_fraction: float = 0.0, seed_vac: int = 0,
                    a: float = 3.6, name: str = "") -> System:
    sites, cell = fcc_box(n_cells, a)
    rng = np.random.default_rng(seed_pos)
    pos = sites + rng.normal(0.0, sigma, size=sites.shape) if sigma > 0 else sites.copy()
    if vacancy_fraction > 0.0:
        keep = np.random.default_rng(seed_vac).uniform(0.0, 1.0, size=len(pos)) >= vacancy_fraction
        pos = pos[keep]
    species = np.random.default_rng(seed_species).integers(0, n_species, size=len(pos)).astype(np.int32)
    return System(np.ascontiguousarray(pos), cell, species, name)


def make_water_system(n_grid: int = 32, density: float = 0.033, sigma: float = 0.1,
                      seed_pos: int = 1005, seed_orient: int = 3005, name: str = "water") -> System:
    """Water-like box of BASELINE.json config 5: O on a jittered cubic grid, two H at 0.96 A and
    104.5 deg in a uniformly random orientation. Atom order: all O, all first H, all second H."""
    spacing = (1.0 / density) ** (1.0 / 3.0)
    idx = np.indices((n_grid, n_grid, n_grid)).reshape(3, -1).T.astype(np.float64)
    rng = np.random.default_rng(seed_pos)
    o = idx * spacing + rng.normal(0.0, sigma, size=idx.shape)
    q = np.random.default_rng(seed_orient).normal(size=(len(o), 4))
    q /= np.linalg.norm(q, axis=1, keepdims=True)
    w, x, y, z = q.T
    rot = np.stack([
        np.stack([1 - 2 * (y * y + z * z), 2 * (x * y - z * w), 2 * (x * z + y * w)], -1),
        np.stack([2 * (x * y + z * w), 1 - 2 * (x * x + z * z), 2 * (y * z - x * w)], -1),
        np.stack([2 * (x * z - y * w), 2 * (y * z + x * w), 1 - 2 * (x * x + y * y)], -1)], 1)
    half = np.deg2rad(104.5 / 2.0)
    h1 = 0.96 * np.array([np.sin(half), 0.0, np.cos(half)])
    h2 = 0.96 * np.array([-np.sin(half), 0.0, np.cos(half)])
    pos = np.concatenate([o, o + rot @ h1, o + rot @ h2], axis=0)
    species = np.concatenate([np.zeros(len(o)), np.ones(2 * len(o))]).astype(np.int32)
    cell = np.eye(3) * (n_grid * spacing)
    return System(np.ascontiguousarray(pos), cell, species, name)


def make_weights(spec: ModelSpec, seed: int) -> np.ndarray:
    """fp32 weight blob in the order of include/mlip.h (reading R9): matrices N(0,1/fan_in),
    biases N(0,0.1^2), T and E0 N(0,1), w_o N(0,1/d). Row-major [out,in]."""
    rng = np.random.default_rng(seed)
    S, d, k = spec.n_species, spec.d, spec.n_rbf
    parts = []

    def mat(out, inn):
        parts.append(rng.normal(0.0, 1.0 / np.sqrt(inn), size=(out, inn)))

    def bias(n):
        parts.append(rng.normal(0.0, 0.1, size=(n,)))

    parts.append(rng.normal(0.0, 1.0, size=(S, d)))  # T
    parts.append(rng.normal(0.0, 1.0, size=(S,)))  # E0
    for _ in range(spec.L_max):
        mat(d, 2 * d + k); bias(d)  # W1, b1
        mat(d, d); bias(d)  # W2, b2
        mat(d, 2 * d); bias(d)  # V1, c1
        mat(d, d); bias(d)  # V2, c2
        if spec.r_cut3 > 0.0:
            mat(16, d); bias(16)  # G, g (gates of the third atom)
            mat(d, 16)  # W3
    mat(d, d); bias(d)  # Wo, bo
    parts.append(rng.normal(0.0, 1.0 / np.sqrt(d), size=(d,)))  # wo
    bias(1)  # b_E
    blob = np.concatenate([p.ravel() for p in parts]).astype(np.float32)
    assert blob.size == spec.n_weights()
    return blob


def small_system(n_cells=3, sigma=0.05, seed=0, n_species=4, a=3.6, vacancy_fraction=0.0) -> System:
    """Generic small jittered fcc box for tests."""
    return make_fcc_system(n_cells, sigma, 1000 + seed, 2000 + seed, n_species,
                           vacancy_fraction, 3000 + seed, a, name=f"fcc{n_cells}")


def make_config(c: int, with_weights: bool = True, n_cells_override: int | None = None) -> Config:
    """BASELINE.json configs 1..5 (seeds 1000+c / 2000+c / 3000+c / 4000+c).

    `n_cells_override` shrinks the fcc box of configs 2-4 for tests (same recipe otherwise)."""
    if c == 1:
        sysm = make_fcc_system(n_cells_override or 3, 0.05, 1001, 2001, name="cfg1-fcc3")
        spec = ModelSpec(4, 64, 8, 2, 5.0, 1.0 / np.sqrt(43.0)); L, prec = 2, "fp32"
        grid, halo = (1, 1, 1), 0.0
    elif c in (2, 3):
        sysm = make_fcc_system(n_cells_override or 15, 0.1, 1002, 2002,
                               vacancy_fraction=0.03, seed_vac=3002, name="cfg2-fcc15-vac")
        spec = ModelSpec(4, 256, 16, 15, 6.0, 1.0 / np.sqrt(76.0))
        L, prec = (5 if c == 2 else 15), "bf16"
        grid, halo = (1, 1, 1), 0.0
    elif c == 4:
        sysm = make_fcc_system(n_cells_override or 64, 0.1, 1004, 2004, name="cfg4-fcc64")
        spec = ModelSpec(4, 256, 16, 4, 5.0, 1.0 / np.sqrt(45.0)); L, prec = 4, "bf16"
        grid, halo = (8, 1, 1), 20.0
    elif c == 5:
        sysm = make_water_system(n_cells_override or 32)
        spec = ModelSpec(2, 128, 16, 4, 5.0, 1.0 / np.sqrt(53.0), r_cut3=4.0); L, prec = 4, "fp32"
        grid, halo = (4, 1, 1), 20.0
    else:
        raise ValueError(f"unknown config {c}")
    seed_w = 4002 if c in (2, 3) else 4000 + c  # configs 2 and 3 share system and weights
    w = make_weights(spec, seed_w) if with_weights else None
    return Config(c, sysm, spec, L, prec, grid, halo, w)
