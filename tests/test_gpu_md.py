"""-m gpu: the on-device MD driver mlip_md_run against the oracle's integrators on the same
start: Langevin (BAOAB + Philox4x32-10, reading R20) trajectories, the thermostat's temperature, and -- with a Verlet
skin -- graph / partition reuse and CUDA-graph replay against the rebuild-every-step run."""
import numpy as np
import pytest

from oracle import mlip_oracle as O
from synth_inputs import ModelSpec, make_weights, small_system
from tests.gpu_util import gpu_setup, oracle_model

pytestmark = pytest.mark.gpu


def _start(n_cells=6, seed=61, T0=0.004):
    spec = ModelSpec(4, 64, 8, 2, 3.0, 1.0 / np.sqrt(12.0))
    blob = make_weights(spec, 35)
    s = small_system(n_cells, 0.08, seed=seed)
    rng = np.random.default_rng(7)
    masses = rng.uniform(10.0, 60.0, len(s.pos))
    vel0 = rng.normal(0, T0, s.pos.shape); vel0 -= vel0.mean(0)
    return spec, blob, s, masses, vel0


def _gpu_md(spec, blob, s, masses, vel0, dt, n_steps, **kw):
    import torch
    mlip, ctx, model = gpu_setup(spec, blob)
    pos = torch.tensor(s.pos, dtype=torch.float64, device="cuda:0").contiguous()
    vel = torch.tensor(vel0, dtype=torch.float64, device="cuda:0").contiguous()
    mass = torch.tensor(masses, dtype=torch.float64, device="cuda:0")
    species = torch.tensor(s.species, dtype=torch.int32, device="cuda:0")
    e, stats = mlip.md_run(ctx, model, 2, pos, vel, mass, s.cell, species, dt, n_steps, **kw)
    return e, pos.cpu().numpy(), vel.cpu().numpy(), stats


@pytest.mark.parametrize("grid,halo", [((1, 1, 1), 0.0), ((2, 1, 1), 6.0)])
def test_langevin_matches_oracle_trajectory(grid, halo):
    import paper_2509_21694_b200 as mlip
    spec, blob, s, masses, vel0 = _start()
    n_steps, dt, T, fr, seed = 20, 2.0, 600.0, 0.01, 20260101
    e_ref, pos_ref, vel_ref = O.langevin_baoab(oracle_model(spec, blob), 2, s.pos, s.cell, s.species, masses, vel0, dt, n_steps,
                                               temperature=T, friction=fr, seed=seed)
    e, pos, vel, stats = _gpu_md(spec, blob, s, masses, vel0, dt, n_steps, grid=grid, halo=halo,
                                 thermostat=mlip.MLIP_MD_LANGEVIN, temperature=T, friction=fr, seed=seed)
    kin0 = 0.5 * np.sum(masses[:, None] * vel0 ** 2) / O.ACC_UNIT
    assert np.abs(e - e_ref).max() <= 1e-4 * kin0
    assert np.abs(pos - pos_ref).max() <= 1e-5
    assert np.abs(vel - vel_ref).max() <= 1e-5 * np.abs(vel_ref).max() + 1e-8
    # the thermostat acted: the trajectory differs from the NVE one by far more than the tolerance
    _, pos_nve, _ = O.nve_velocity_verlet(oracle_model(spec, blob), 2, s.pos, s.cell, s.species, masses, vel0, dt, n_steps,
                                          return_state=True)
    assert np.abs(pos_ref - pos_nve).max() > 1e-3
    assert stats["n_rebuilds"] == n_steps + 1


def test_langevin_zero_friction_is_nve_and_thermostat_sets_temperature():
    import paper_2509_21694_b200 as mlip
    spec, blob, s, masses, vel0 = _start()
    e_nve, p_nve, v_nve, _ = _gpu_md(spec, blob, s, masses, vel0, 2.0, 10)
    e_l0, p_l0, v_l0, _ = _gpu_md(spec, blob, s, masses, vel0, 2.0, 10, thermostat=mlip.MLIP_MD_LANGEVIN, temperature=300.0,
                                  friction=0.0, seed=5)
    assert np.array_equal(p_nve, p_l0) and np.array_equal(v_nve, v_l0)
    # strong coupling from a cold start: after 150 steps the kinetic temperature is the bath's (864 atoms: +-4 % 1 sigma)
    T = 900.0
    e, pos, vel, _ = _gpu_md(spec, blob, s, masses, np.zeros_like(vel0), 2.0, 150, thermostat=mlip.MLIP_MD_LANGEVIN,
                             temperature=T, friction=0.05, seed=99)
    T_kin = np.sum(masses[:, None] * vel ** 2) / O.ACC_UNIT / (3 * len(masses) * O.KB_EV)
    assert abs(T_kin / T - 1.0) < 0.15, T_kin


@pytest.mark.parametrize("grid,halo,graph", [((1, 1, 1), 0.0, False), ((2, 1, 1), 6.0, False), ((1, 1, 1), 0.0, True),
                                             ((2, 1, 1), 6.0, True)])
def test_verlet_skin_reuse_matches_rebuild_every_step(grid, halo, graph):
    """skin > 0: graph and partition are kept until an atom has moved skin/2; every step the candidate list is filtered
    with the canonical predicate, so the edge set of every step is the one a rebuild gives and the trajectory agrees
    with the rebuild-every-step run and with the oracle to fp32 accuracy; with cuda_graph the steps between rebuilds are
    replays of one captured CUDA graph."""
    spec, blob, s, masses, vel0 = _start(T0=0.006)
    n_steps, dt = 30, 2.0
    e0, p0, v0, st0 = _gpu_md(spec, blob, s, masses, vel0, dt, n_steps, grid=grid, halo=halo)
    e1, p1, v1, st1 = _gpu_md(spec, blob, s, masses, vel0, dt, n_steps, grid=grid, halo=halo, skin=0.4, cuda_graph=graph)
    kin0 = 0.5 * np.sum(masses[:, None] * vel0 ** 2) / O.ACC_UNIT
    assert st0["n_rebuilds"] == n_steps + 1
    assert 1 < st1["n_rebuilds"] < n_steps / 2, st1          # rebuilt when needed (atoms move ~0.7 A), not every step
    assert np.abs(e1 - e0).max() <= 1e-4 * kin0
    assert np.abs(p1 - p0).max() <= 1e-5 and np.abs(v1 - v0).max() <= 1e-5 * np.abs(v0).max() + 1e-8
    if graph:
        assert st1["n_graph_replays"] == n_steps + 1, st1
    e_ref, pos_ref, _ = O.nve_velocity_verlet(oracle_model(spec, blob), 2, s.pos, s.cell, s.species, masses, vel0, dt, n_steps,
                                              return_state=True)
    assert np.abs(e1 - e_ref).max() <= 1e-4 * kin0 and np.abs(p1 - pos_ref).max() <= 1e-5


def test_verlet_skin_bf16_partitioned_langevin():
    import paper_2509_21694_b200 as mlip
    spec = ModelSpec(4, 128, 16, 2, 3.0, 1.0 / np.sqrt(12.0))
    blob = make_weights(spec, 36)
    s = small_system(8, 0.08, seed=62)
    rng = np.random.default_rng(8)
    masses = rng.uniform(10.0, 60.0, len(s.pos))
    vel0 = rng.normal(0, 0.005, s.pos.shape); vel0 -= vel0.mean(0)
    kw = dict(grid=(2, 2, 1), halo=6.0, precision=mlip.MLIP_BF16, thermostat=mlip.MLIP_MD_LANGEVIN, temperature=500.0,
              friction=0.01, seed=3)
    e0, p0, v0, _ = _gpu_md(spec, blob, s, masses, vel0, 2.0, 20, **kw)
    e1, p1, v1, st = _gpu_md(spec, blob, s, masses, vel0, 2.0, 20, skin=0.5, cuda_graph=True, **kw)
    assert st["n_graph_replays"] == 21 and st["n_rebuilds"] < 10
    assert np.abs(p1 - p0).max() <= 2e-3      # 16-bit forces, different tile boundaries: agreement to bf16-path accuracy


def test_md_three_body_skin_and_graph():
    """The three-body variant (config-5 recipe, fp32) through the MD driver: Verlet-skin reuse + CUDA-graph replay give the
    trajectory of the rebuild-every-step run (the per-edge vector gradients and triplet lists follow the filtered graph)."""
    from synth_inputs import make_water_system
    spec = ModelSpec(2, 64, 8, 2, 5.0, 1.0 / np.sqrt(53.0), r_cut3=4.0)
    blob = make_weights(spec, 37)
    s = make_water_system(4)
    rng = np.random.default_rng(9)
    masses = np.where(s.species == 0, 16.0, 1.0)
    vel0 = rng.normal(0, 0.002, s.pos.shape); vel0 -= vel0.mean(0)
    e0, p0, v0, _ = _gpu_md(spec, blob, s, masses, vel0, 0.5, 20)
    e1, p1, v1, st = _gpu_md(spec, blob, s, masses, vel0, 0.5, 20, skin=0.4, cuda_graph=True)
    assert st["n_graph_replays"] == 21
    assert np.abs(p1 - p0).max() <= 1e-5 and np.abs(e1 - e0).max() <= 1e-7 * np.abs(e0).max() + 1e-5   # fp32 energy sums
    e_ref, pos_ref, _ = O.nve_velocity_verlet(oracle_model(spec, blob), 2, s.pos, s.cell, s.species, masses, vel0, 0.5, 20,
                                              return_state=True)
    assert np.abs(p1 - pos_ref).max() <= 1e-5


def test_md_degenerate_calls():
    """Zero steps (one evaluation, the initial total energy only), an empty system, and argument errors."""
    import torch
    import paper_2509_21694_b200 as mlip
    spec, blob, s, masses, vel0 = _start(n_cells=3)
    e, pos, vel, st = _gpu_md(spec, blob, s, masses, vel0, 2.0, 0, skin=0.3)
    assert e.shape == (1,) and np.isfinite(e[0]) and np.array_equal(pos, s.pos) and st["n_rebuilds"] == 1
    mlipm, ctx, model = gpu_setup(spec, blob)
    z3 = torch.zeros((0, 3), dtype=torch.float64, device="cuda:0")
    z1 = torch.zeros(0, dtype=torch.float64, device="cuda:0")
    zi = torch.zeros(0, dtype=torch.int32, device="cuda:0")
    for skin in (0.0, 0.3):
        e, st = mlip.md_run(ctx, model, 2, z3, z3.clone(), z1, s.cell, zi, 2.0, 3, skin=skin)
        assert np.all(e == 0.0)
    pos = torch.tensor(s.pos, dtype=torch.float64, device="cuda:0")
    vel = torch.zeros_like(pos)
    mass = torch.tensor(masses, dtype=torch.float64, device="cuda:0")
    sp = torch.tensor(s.species, dtype=torch.int32, device="cuda:0")
    with pytest.raises(mlip.MlipError) as ei:      # CUDA-graph replay needs fixed launch dimensions, i.e. a skin
        mlip.md_run(ctx, model, 2, pos, vel, mass, s.cell, sp, 2.0, 2, cuda_graph=True)
    assert ei.value.code == -1
    with pytest.raises(mlip.MlipError) as ei:      # halo < L r_cut is refused in skin mode too
        mlip.md_run(ctx, model, 2, pos, vel, mass, s.cell, sp, 2.0, 2, grid=(2, 1, 1), halo=3.0, skin=0.3)
    assert ei.value.code == -3
