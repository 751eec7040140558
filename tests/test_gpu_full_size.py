"""-m gpu: parity at BASELINE.json's FULL size in the launch configuration bench.py times (config 4: 1,048,576 atoms,
L = 4, d = 256, bf16 tensor-core path, 8 slabs with a 20 A halo, K-hop halo and per-layer active sets on).

The oracle cannot evaluate a million atoms, but a per-atom energy E_i only depends on the atoms within L r_c of atom i
and a force F_i only on those within 2 L r_c (the K-hop neighbourhood), so SAMPLED outputs are computed
one by one by the float64 oracle on the ball cut out of the box around the sampled atom. Properties that hold at any
size cover the rest: total force zero, partitioned == unpartitioned on the GPU, every atom owned exactly once."""
import numpy as np
import pytest

from oracle import mlip_oracle as O
from synth_inputs import make_config
from tests.gpu_util import gpu_energy_forces, gpu_graph, gpu_setup, oracle_model, rms

pytestmark = pytest.mark.gpu


def _ball(system, i, radius):
    """Atoms within `radius` of atom i under the minimum image, re-centred in a cell large enough that no periodic image
    of the cluster is within r_cut of it. Returns (pos, cell, species, index of i in the cluster, distances)."""
    box = np.diag(system.cell)
    d = system.pos - system.pos[i]
    d -= np.round(d / box) * box
    r = np.linalg.norm(d, axis=1)
    keep = np.nonzero(r <= radius)[0]
    side = 2.0 * radius + 20.0
    return d[keep] + 0.5 * side, np.eye(3) * side, system.species[keep], int(np.nonzero(keep == i)[0][0]), r[keep]


@pytest.fixture(scope="module")
def full():
    cfg = make_config(4)
    mlip, ctx, model = gpu_setup(cfg.model, cfg.weights)
    g = gpu_graph(mlip, ctx, cfg.system, cfg.model.r_cut)
    part = mlip.Partition(ctx, g, cfg.halo, grid=cfg.grid)
    E, F, Ei = gpu_energy_forces(mlip, ctx, model, cfg.L, g, part, 1)
    info = part.info()
    layers = part.layer_info(cfg.L)
    del part
    return dict(cfg=cfg, mlip=mlip, ctx=ctx, model=model, g=g, E=E, F=F, Ei=Ei, info=info, layers=layers)


def test_full_size_properties(full):
    cfg, F, Ei, E = full["cfg"], full["F"], full["Ei"], full["E"]
    N = len(cfg.system.pos)
    assert N == 1048576 and len(full["info"]) == 8
    assert sum(i["n_owned"] for i in full["info"]) == N                      # every atom is a root atom exactly once
    assert all(rows[-1]["n_recv"] == i["n_owned"] for rows, i in zip(full["layers"], full["info"]))
    assert np.all(np.isfinite(F)) and np.all(np.isfinite(Ei))
    assert abs(Ei.sum() - E) <= 1e-6 * np.abs(Ei).sum()                      # E is the sum of the root energies
    # Newton's third law survives the partition: the sub-domain gradients are summed over ALL their atoms (reading R1)
    assert np.abs(F.sum(0)).max() <= 1e-3 * rms(F)
    # unpartitioned evaluation of the same box on the same GPU (fits the 180 GB of HBM)
    E1, F1, Ei1 = gpu_energy_forces(full["mlip"], full["ctx"], full["model"], cfg.L, full["g"], None, 1)
    assert rms(F - F1) <= 2e-2 * rms(F1)
    assert abs(E - E1) <= 1e-5 * np.abs(Ei1).sum()
    assert np.abs(Ei - Ei1).max() <= 2e-2 * rms(Ei1 - Ei1.mean())


def test_full_size_sampled_atom_energies_match_oracle(full):
    """E_i of sampled atoms (next to a slab face, mid-slab, the last atom) against the float64 oracle on the L r_c ball."""
    cfg, Ei = full["cfg"], full["Ei"]
    s, m = cfg.system, cfg.model
    om = oracle_model(m, cfg.weights)
    x = s.pos[:, 0] % 230.4
    near_face = int(np.argmin(np.abs(x - 28.8)))       # slab boundary of the 8 x 28.8 A partition
    mid_slab = int(np.argmin(np.abs(x - 100.8) + np.abs(s.pos[:, 1] - 115.0) + np.abs(s.pos[:, 2] - 115.0)))
    spread = rms(Ei - Ei.mean())
    for i in (near_face, mid_slab, len(s.pos) - 1):
        pos, cell, sp, k, r = _ball(s, i, cfg.L * m.r_cut + 0.5)
        E_ref = O.energy_forces(om, cfg.L, pos, cell, sp)[1][k]
        assert abs(Ei[i] - E_ref) <= 2e-2 * spread, (i, Ei[i], E_ref, spread)


def test_full_size_sampled_atom_force_matches_oracle(full):
    """F_i of one sampled atom next to a slab face: gradient of the energies of the atoms within L r_c of it, each
    evaluated on its own complete neighbourhood, i.e. the oracle on the 2 L r_c ball with omega = 1 inside L r_c."""
    cfg, F = full["cfg"], full["F"]
    s, m = cfg.system, cfg.model
    om = oracle_model(m, cfg.weights)
    x = s.pos[:, 0] % 230.4
    i = int(np.argmin(np.abs(x - 57.6) + 1e-3 * np.abs(s.pos[:, 1] - 60.0)))
    pos, cell, sp, k, r = _ball(s, i, 2 * cfg.L * m.r_cut + 0.5)
    omega = (r <= cfg.L * m.r_cut + 0.25).astype(np.float64)
    F_ref = O.energy_forces(om, cfg.L, pos, cell, sp, omega=omega)[2][k]
    assert np.abs(F[i] - F_ref).max() <= 5e-2 * rms(F), (F[i], F_ref, rms(F))
