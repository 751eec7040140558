"""Writes the stored float64-oracle references for the FULL-SIZE BASELINE.json configurations.

    python tests/golden/make_full_size_refs.py [config2] [config3] [config4_balls] [config4_edges]

The float64 oracle needs minutes per configuration at these sizes, more than the GPU test run may spend, so its
results are computed once by THIS script -- which imports nothing but `oracle/` and the seeded input generators of
`synth_inputs/` -- and stored next to it. No value in these files comes from the CUDA path.

  config2_L5_oracle.npz     E, E_i [N], F [N,3] of BASELINE config 2 (13,125 atoms, L = 5 of 15, d = 256)
  config3_L15_oracle.npz    the same system with the unpruned L = 15 (pruned versus unpruned)
  config4_sampled_oracle.npz  config 4 (1,048,576 atoms, L = 4): E_i and F_i of the atoms around three sample points
                            (on a slab face, at the periodic corner of the box where three faces of the wrap meet, in
                            the middle of a slab). A per-atom energy depends on the atoms within L r_c only and a force
                            on those within 2 L r_c (the K-hop neighbourhood), so the oracle evaluated
                            on the ball of radius 2 L r_c + R around a point gives the EXACT F_k of every atom within R
                            of it and the exact E_i of every atom within L r_c + R.
  config4_edge_hash.npz     config 4: per-atom in-degree and an order-dependent 64-bit hash of the canonical edge list
                            (i, j, n) of the oracle's k-d tree neighbour list, folded over blocks of 256 receivers
                            (the list itself is 47.19 M rows; tests/test_gpu_full_size.py hashes the exported CUDA list
                            the same way).
"""
from __future__ import annotations

import os
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from oracle import mlip_oracle as O  # noqa: E402
from synth_inputs import make_config  # noqa: E402

# sample points of config 4 (box 230.4 A, 8 slabs of 28.8 A along x) and the radii of the sampled sets
CFG4_POINTS = {"slab_face": (57.6, 115.2, 115.2),      # the face between slabs 1 and 2
               "box_corner": (0.0, 0.0, 0.0),          # slab 7 | slab 0 through the periodic wrap, wrap in y and z too
               "mid_slab": (100.8, 60.0, 170.0)}       # interior of slab 3
CFG4_R_FORCE = 6.0    # forces exact within this distance of a sample point (about 77 atoms each)
CFG4_R_ENERGY = 9.0   # per-atom energies stored within this distance (about 260 atoms each)
HASH_BLOCK = 256


def _oracle_model(cfg):
    m = cfg.model
    return O.parse_weights(m.n_species, m.d, m.n_rbf, m.L_max, m.r_cut, m.agg_scale, cfg.weights)


def full_config(c: int, out_name: str):
    cfg = make_config(c)
    s = cfg.system
    t0 = time.perf_counter()
    E, E_i, F = O.energy_forces(_oracle_model(cfg), cfg.L, s.pos, s.cell, s.species)
    dt = time.perf_counter() - t0
    np.savez_compressed(os.path.join(HERE, out_name), E=np.float64(E), E_i=E_i, F=F, n_atoms=len(s.pos), L=cfg.L,
                        oracle_seconds=dt, cores=len(os.sched_getaffinity(0)))
    print(f"config {c}: N={len(s.pos)} L={cfg.L} E={E:.6f} oracle {dt:.1f} s", flush=True)


def ball(system, centre, radius):
    """Atoms within `radius` of `centre` under the minimum image of the (orthorhombic) box, re-centred in an open cell
    large enough that no periodic image of the cluster is within r_cut of it. Returns (pos, cell, global indices, distance)."""
    box = np.diag(system.cell)
    d = system.pos - np.asarray(centre, np.float64)
    d -= np.round(d / box) * box
    r = np.linalg.norm(d, axis=1)
    keep = np.nonzero(r <= radius)[0]
    side = 2.0 * radius + 20.0
    return d[keep] + 0.5 * side, np.eye(3) * side, keep, r[keep]


def config4_balls():
    cfg = make_config(4)
    s, m = cfg.system, cfg.model
    om = _oracle_model(cfg)
    reach = cfg.L * m.r_cut
    out = {}
    for name, centre in CFG4_POINTS.items():
        t0 = time.perf_counter()
        pos, cell, idx, r = ball(s, centre, 2.0 * reach + CFG4_R_FORCE + 0.5)
        _, E_i, F = O.energy_forces(om, cfg.L, pos, cell, s.species[idx])
        fsel = r <= CFG4_R_FORCE
        esel = r <= CFG4_R_ENERGY
        out[name + "_force_idx"] = idx[fsel].astype(np.int64)
        out[name + "_F"] = F[fsel]
        out[name + "_energy_idx"] = idx[esel].astype(np.int64)
        out[name + "_E_i"] = E_i[esel]
        print(f"config 4 {name}: ball {len(idx)} atoms, {fsel.sum()} forces, {esel.sum()} energies, "
              f"{time.perf_counter() - t0:.1f} s", flush=True)
    np.savez_compressed(os.path.join(HERE, "config4_sampled_oracle.npz"), points=np.array(list(CFG4_POINTS.values())),
                        names=np.array(list(CFG4_POINTS.keys())), **out)


def edge_hash(recv, send, shift, n_atoms):
    """Order-dependent 64-bit hash of a canonical edge list, folded over blocks of HASH_BLOCK receivers:
    h_e = mix(i, j, n); block hash = sum over its edges of (position of e in its row + 1) * h_e (mod 2^64).
    Also returns the per-atom in-degree. Test infrastructure: no arithmetic of the method."""
    recv = np.asarray(recv, np.int64)
    deg = np.bincount(recv, minlength=n_atoms).astype(np.int64)
    rowptr = np.concatenate([[0], np.cumsum(deg)])
    k = (np.arange(len(recv), dtype=np.int64) - rowptr[recv] + 1).astype(np.uint64)
    sh = np.asarray(shift, np.int64)
    packed = ((sh[:, 0] + 128) << 16) | ((sh[:, 1] + 128) << 8) | (sh[:, 2] + 128)
    with np.errstate(over="ignore"):
        h = (recv.astype(np.uint64) * np.uint64(0x9E3779B97F4A7C15)) ^ (np.asarray(send, np.int64).astype(np.uint64) * np.uint64(0xC2B2AE3D27D4EB4F)) \
            ^ (packed.astype(np.uint64) * np.uint64(0x165667B19E3779F9))
        h ^= h >> np.uint64(31)
        h *= np.uint64(0xBF58476D1CE4E5B9)
        h ^= h >> np.uint64(29)
        h *= k
        n_blocks = (n_atoms + HASH_BLOCK - 1) // HASH_BLOCK
        # uint64 sums per block (np.add.at wraps modulo 2^64)
        blocks = np.zeros(n_blocks, np.uint64)
        np.add.at(blocks, recv // HASH_BLOCK, h)
    return deg, blocks


def config4_edges():
    cfg = make_config(4, with_weights=False)
    s = cfg.system
    t0 = time.perf_counter()
    recv, send, shift = O.neighbor_list(s.pos, s.cell, cfg.model.r_cut)
    dt = time.perf_counter() - t0
    deg, blocks = edge_hash(recv, send, shift, len(s.pos))
    np.savez_compressed(os.path.join(HERE, "config4_edge_hash.npz"), n_edges=np.int64(len(recv)), degree=deg.astype(np.uint8),
                        block_hash=blocks, hash_block=HASH_BLOCK)
    print(f"config 4 edge list: {len(recv)} edges, oracle neighbour list {dt:.1f} s", flush=True)


if __name__ == "__main__":
    what = sys.argv[1:] or ["config2", "config4_balls", "config4_edges", "config3"]
    for w in what:
        if w == "config2":
            full_config(2, "config2_L5_oracle.npz")
        elif w == "config3":
            full_config(3, "config3_L15_oracle.npz")
        elif w == "config4_balls":
            config4_balls()
        elif w == "config4_edges":
            config4_edges()
        else:
            raise SystemExit(f"unknown target {w}")
