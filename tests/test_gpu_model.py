"""-m gpu: energies and forces of the CUDA path (through the C ABI) against the float64 oracle on
the same seeded inputs. Tolerances are those of north_star / reading R14:
fp32 path  eps_E <= 1e-5, max|dF| <= 1e-4 RMS(F);  bf16 path  RMS(dF)/RMS(F) <= 2e-2;
partitioned vs unpartitioned GPU forces within 1e-5 RMS(F) in fp32."""
import numpy as np
import pytest

from oracle import mlip_oracle as O
from synth_inputs import ModelSpec, make_config, make_weights, small_system
from tests.gpu_util import errors, gpu_energy_forces, gpu_graph, gpu_setup, oracle_model, rms

pytestmark = pytest.mark.gpu

FP32_EPS_E, FP32_MAX_F = 1e-5, 1e-4
FP32_REL_EI = 1e-5   # per-atom energy relative error (north_star; denominator max(|E_i,ref|, RMS E_ref), reading R14)
BF16_RMS_F = 2e-2


def _run(spec, blob, system, L, precision=0, grid=None, halo=0.0):
    mlip, ctx, model = gpu_setup(spec, blob)
    g = gpu_graph(mlip, ctx, system, spec.r_cut)
    part = mlip.Partition(ctx, g, halo, grid=grid) if grid is not None else None
    return gpu_energy_forces(mlip, ctx, model, L, g, part, precision)


def test_config1_fp32_parity():
    cfg = make_config(1)
    s = cfg.system
    ref = O.energy_forces(oracle_model(cfg.model, cfg.weights), cfg.L, s.pos, s.cell, s.species)
    E, F, Ei = _run(cfg.model, cfg.weights, s, cfg.L)
    err = errors(E, F, Ei, ref[0], ref[2], ref[1])
    print(err)
    assert err["eps_E"] <= FP32_EPS_E and err["max_F"] <= FP32_MAX_F and err["rel_Ei"] <= FP32_REL_EI


@pytest.mark.parametrize("d,L,n_cells,r_cut,nbar", [(64, 3, 4, 5.0, 43.0), (128, 4, 4, 5.0, 43.0), (256, 2, 4, 6.0, 76.0),
                                                   (128, 0, 3, 5.0, 43.0), (64, 1, 2, 5.0, 43.0)])
def test_fp32_parity_shapes(d, L, n_cells, r_cut, nbar):
    spec = ModelSpec(4, d, 16 if d > 64 else 8, max(L, 1), r_cut, 1.0 / np.sqrt(nbar))
    blob = make_weights(spec, 77 + d)
    s = small_system(n_cells, 0.1, seed=d + L, vacancy_fraction=0.03)
    ref = O.energy_forces(oracle_model(spec, blob), L, s.pos, s.cell, s.species)
    E, F, Ei = _run(spec, blob, s, L)
    err = errors(E, F, Ei, ref[0], ref[2], ref[1])
    print(d, L, err)
    assert err["eps_E"] <= FP32_EPS_E and err["rel_Ei"] <= FP32_REL_EI
    if L > 0:
        assert err["max_F"] <= FP32_MAX_F
    else:
        assert np.all(F == 0)


def test_fp32_partitioned_equals_unpartitioned_and_oracle():
    spec = ModelSpec(4, 64, 8, 2, 3.0, 1.0 / np.sqrt(12.0))
    blob = make_weights(spec, 5)
    s = small_system(8, 0.08, seed=31)  # 28.8 A box, 2048 atoms; L r_cut = 6
    ref = O.energy_forces(oracle_model(spec, blob), 2, s.pos, s.cell, s.species)
    E0, F0, Ei0 = _run(spec, blob, s, 2)
    for grid in [(2, 1, 1), (3, 1, 1), (2, 2, 1), (1, 1, 4)]:
        E, F, Ei = _run(spec, blob, s, 2, grid=grid, halo=6.0)
        assert np.abs(F - F0).max() <= 1e-5 * rms(F0)
        assert abs(E - E0) <= 1e-5 * np.abs(Ei0).sum()
        err = errors(E, F, Ei, ref[0], ref[2], ref[1])
        assert err["eps_E"] <= FP32_EPS_E and err["max_F"] <= FP32_MAX_F and err["rel_Ei"] <= FP32_REL_EI
    # negative control: a halo of (L-1) r_cut is refused, not silently wrong
    mlip, ctx, model = gpu_setup(spec, blob)
    g = gpu_graph(mlip, ctx, s, spec.r_cut)
    part = mlip.Partition(ctx, g, 3.0, grid=(3, 1, 1))
    with pytest.raises(mlip.MlipError) as ei:
        mlip.energy_forces(ctx, model, 2, g, part, 0)
    assert ei.value.code == -3


def test_run_to_run_bitwise_and_order_independent():
    """No floating-point atomics: repeated evaluations are bitwise identical."""
    cfg = make_config(1)
    a = _run(cfg.model, cfg.weights, cfg.system, cfg.L)
    b = _run(cfg.model, cfg.weights, cfg.system, cfg.L)
    assert a[0] == b[0] and np.array_equal(a[1], b[1]) and np.array_equal(a[2], b[2])


def test_mpdp_L_argument():
    """the first L of L_max layers; L is a run-time argument."""
    spec = ModelSpec(4, 64, 8, 3, 5.0, 1.0 / np.sqrt(43.0))
    blob = make_weights(spec, 9)
    s = small_system(3, 0.05, seed=2)
    om = oracle_model(spec, blob)
    for L in (1, 2, 3):
        ref = O.energy_forces(om, L, s.pos, s.cell, s.species)
        E, F, Ei = _run(spec, blob, s, L)
        err = errors(E, F, Ei, ref[0], ref[2], ref[1])
        assert err["eps_E"] <= FP32_EPS_E and err["max_F"] <= FP32_MAX_F and err["rel_Ei"] <= FP32_REL_EI
    mlip, ctx, model = gpu_setup(spec, blob)
    g = gpu_graph(mlip, ctx, s, spec.r_cut)
    with pytest.raises(mlip.MlipError):
        mlip.energy_forces(ctx, model, 4, g, None, 0)


def test_step_host_matches_device_path():
    cfg = make_config(1)
    mlip, ctx, model = gpu_setup(cfg.model, cfg.weights)
    s = cfg.system
    E1, F1, _ = _run(cfg.model, cfg.weights, s, cfg.L)
    E2, F2 = mlip.step_host(ctx, model, cfg.L, s.pos, s.cell, s.species)
    assert E1 == E2 and np.array_equal(F1.astype(np.float32), F2)
    E3, F3 = mlip.step_host(ctx, model, cfg.L, s.pos, s.cell, s.species, grid=(1, 1, 1), halo=0.0)
    assert E3 == E2


# ---- MLIP_BF16: bf16 tensor-core contractions (tcgen05), fp32 accumulation ------------------------
@pytest.mark.parametrize("d,L,n_cells,r_cut,nbar", [(256, 0, 3, 5.0, 43.0), (256, 1, 3, 5.0, 43.0), (256, 2, 4, 6.0, 76.0),
                                                   (128, 2, 4, 5.0, 43.0), (256, 5, 5, 6.0, 76.0)])
def test_bf16_parity_shapes(d, L, n_cells, r_cut, nbar):
    """Reference = oracle with the UNROUNDED fp32 weights (reading R15). Sizes span several 128-edge
    tiles with a ragged last tile and segments that straddle tiles."""
    spec = ModelSpec(4, d, 16, max(L, 1), r_cut, 1.0 / np.sqrt(nbar))
    blob = make_weights(spec, 77 + d)
    s = small_system(n_cells, 0.1, seed=d + L, vacancy_fraction=0.03)
    ref = O.energy_forces(oracle_model(spec, blob), L, s.pos, s.cell, s.species)
    E, F, Ei = _run(spec, blob, s, L, precision=1)
    err = errors(E, F, Ei, ref[0], ref[2], ref[1])
    print(d, L, err)
    assert np.isfinite(F).all() and np.isfinite(E)
    assert err["eps_E"] <= 5e-3  # not a north_star bound; catches gross errors of the forward pass
    if L > 0:
        assert err["rms_F"] <= BF16_RMS_F
    else:
        assert np.all(F == 0)


def test_bf16_config2_shape_pruned_vs_unpruned():
    """BASELINE.json configs 2/3 on a shrunk box (fcc 6^3 with vacancies): L=5 of L_max=15 (MPDP,
    PAPER.md:151) and the unpruned L=15, bf16 GEMM inputs, force RMS error <= 2e-2."""
    cfg = make_config(3, n_cells_override=6)
    s = cfg.system
    om = oracle_model(cfg.model, cfg.weights)
    for L in (5, 15):
        ref = O.energy_forces(om, L, s.pos, s.cell, s.species)
        E, F, Ei = _run(cfg.model, cfg.weights, s, L, precision=1)
        err = errors(E, F, Ei, ref[0], ref[2], ref[1])
        print(L, err)
        assert err["rms_F"] <= BF16_RMS_F


def test_bf16_partitioned_matches_unpartitioned():
    spec = ModelSpec(4, 256, 16, 2, 3.0, 1.0 / np.sqrt(12.0))
    blob = make_weights(spec, 6)
    s = small_system(8, 0.08, seed=32)
    ref = O.energy_forces(oracle_model(spec, blob), 2, s.pos, s.cell, s.species)
    E0, F0, Ei0 = _run(spec, blob, s, 2, precision=1)
    for grid in [(2, 1, 1), (1, 3, 1)]:
        E, F, Ei = _run(spec, blob, s, 2, precision=1, grid=grid, halo=6.0)
        err = errors(E, F, Ei, ref[0], ref[2], ref[1])
        assert err["rms_F"] <= BF16_RMS_F
        # each owned atom sees the same neighbourhood in its sub-domain, but tile boundaries differ,
        # so the bf16 roundings of partial sums differ: equal only to bf16-path accuracy
        assert rms(F - F0) <= BF16_RMS_F * rms(F0)


def test_bf16_run_to_run_bitwise():
    spec = ModelSpec(4, 256, 16, 2, 5.0, 1.0 / np.sqrt(43.0))
    blob = make_weights(spec, 8)
    s = small_system(4, 0.1, seed=3)
    a = _run(spec, blob, s, 2, precision=1)
    b = _run(spec, blob, s, 2, precision=1)
    assert a[0] == b[0] and np.array_equal(a[1], b[1]) and np.array_equal(a[2], b[2])


def test_bf16_rejects_d64():
    cfg = make_config(1)
    mlip, ctx, model = gpu_setup(cfg.model, cfg.weights)
    g = gpu_graph(mlip, ctx, cfg.system, cfg.model.r_cut)
    with pytest.raises(mlip.MlipError) as ei:
        mlip.energy_forces(ctx, model, cfg.L, g, None, 1)
    assert ei.value.code == -2


# ---------------------------------------------------------------- per-layer active sets
def _run_part(spec, blob, system, L, precision, grid, halo, active=True, n_sub=None, khop=True):
    mlip, ctx, model = gpu_setup(spec, blob)
    ctx.set_active_sets(active)
    ctx.set_khop_halo(khop)
    g = gpu_graph(mlip, ctx, system, spec.r_cut)
    part = mlip.Partition(ctx, g, halo, n_sub=n_sub) if n_sub else mlip.Partition(ctx, g, halo, grid=grid)
    return gpu_energy_forces(mlip, ctx, model, L, g, part, precision), part.layer_info(L), part.info()


@pytest.mark.parametrize("khop", [False, True])
def test_active_set_sizes_match_oracle_classes(khop):
    """mlip_part_layer_info against the oracle's depth classes (geometric shells or K-hop counts): layer l
    runs on receivers of class <= L-1-l, senders of class <= L-l, and the induced edges whose receiver is
    in the first set."""
    import paper_2509_21694_b200 as mlip
    ctx = mlip.Context(0)
    ctx.set_khop_halo(khop)
    r_cut, L = 3.0, 3
    s = small_system(12, 0.08, seed=17)   # 43.2 A box
    g = gpu_graph(mlip, ctx, s, r_cut)
    graph = O.neighbor_list(s.pos, s.cell, r_cut)
    for grid, halo in [((4, 1, 1), 9.0), ((2, 2, 1), 9.0), ((1, 3, 1), 7.5), ((2, 1, 1), 12.0)]:
        part = mlip.Partition(ctx, g, halo, grid=grid)
        info = part.layer_info(L)
        if khop:
            both = O.partition_grid_khop(s.pos, s.cell, grid, halo, r_cut, graph)
            parts, classes = [(o, e) for o, e, _ in both], [h for _, _, h in both]
        else:
            parts = O.partition_grid(s.pos, s.cell, grid, halo)
            classes = O.halo_depth_classes(s.pos, s.cell, grid, halo, r_cut)
        for rows, (owned, ext), cls in zip(info, parts, classes):
            lr, ls, _ = O.induced_subgraph(graph, ext, len(s.pos))
            top = max(1, int(np.ceil(halo / r_cut - 1e-9)))
            for l, row in enumerate(rows):
                cr, cs = min(L - 1 - l, top), min(L - l, top)
                assert row["n_recv"] == int((cls <= cr).sum())
                assert row["n_send"] == int((cls <= cs).sum())
                assert row["n_edges"] == int((cls[lr] <= cr).sum())
            assert rows[L - 1]["n_recv"] == len(owned)
        ctx.set_active_sets(False)
        off = part.layer_info(L)
        ctx.set_active_sets(True)
        for rows, (owned, ext) in zip(off, parts):
            assert all(r["n_recv"] == len(ext) and r["n_send"] == len(ext) for r in rows)


@pytest.mark.parametrize("grid,n_sub,L,halo", [((4, 1, 1), None, 3, 9.0), ((2, 2, 2), None, 2, 6.0),
                                                 (None, 3, 3, 9.0), ((3, 1, 1), None, 1, 9.0),
                                                 ((2, 1, 1), None, 3, 10.5)])
def test_fp32_active_sets_equal_full_subgraphs_and_oracle(grid, n_sub, L, halo):
    """Skipping the layers' inactive atoms changes nothing: equal to evaluating every layer on the whole
    extended sub-graph (the skipped adjoints are exact zeros), to the unpartitioned GPU result within
    1e-5 RMS(F), and to the oracle's unpartitioned definition within the fp32 tolerances."""
    spec = ModelSpec(4, 64, 8, 3, 3.0, 1.0 / np.sqrt(12.0))
    blob = make_weights(spec, 15)
    s = small_system(12, 0.08, seed=41)   # 43.2 A box, 6912 atoms
    ref = O.energy_forces(oracle_model(spec, blob), L, s.pos, s.cell, s.species)
    E0, F0, Ei0 = _run(spec, blob, s, L)
    (E, F, Ei), layers, info = _run_part(spec, blob, s, L, 0, grid, halo, active=True, n_sub=n_sub)
    (Ef, Ff, Eif), layers_off, _ = _run_part(spec, blob, s, L, 0, grid, halo, active=False, n_sub=n_sub)
    (Eg, Fg, Eig), layers_geo, _ = _run_part(spec, blob, s, L, 0, grid, halo, active=True, n_sub=n_sub, khop=False)
    n_ev = lambda lay: sum(r["n_edges"] for rows in lay for r in rows)
    assert n_ev(layers) <= n_ev(layers_geo) < n_ev(layers_off) or L == 1
    assert E == Ef and np.array_equal(Ei, Eif)
    assert np.abs(F - Ff).max() <= 1e-6 * rms(F0)
    assert abs(Eg - E) <= 1e-6 * np.abs(Ei0).sum() and np.abs(Fg - F).max() <= 1e-5 * rms(F0)
    assert np.abs(F - F0).max() <= 1e-5 * rms(F0)
    assert abs(E - E0) <= 1e-5 * np.abs(Ei0).sum()
    err = errors(E, F, Ei, ref[0], ref[2], ref[1])
    assert err["eps_E"] <= FP32_EPS_E and err["max_F"] <= FP32_MAX_F and err["rel_Ei"] <= FP32_REL_EI


def test_bf16_active_sets_match_oracle():
    spec = ModelSpec(4, 256, 16, 3, 3.0, 1.0 / np.sqrt(12.0))
    blob = make_weights(spec, 16)
    s = small_system(12, 0.08, seed=42)
    ref = O.energy_forces(oracle_model(spec, blob), 3, s.pos, s.cell, s.species)
    for grid in [(4, 1, 1), (2, 2, 1)]:
        (E, F, Ei), layers, info = _run_part(spec, blob, s, 3, 1, grid, 9.0, active=True)
        (Ef, Ff, Eif), _, _ = _run_part(spec, blob, s, 3, 1, grid, 9.0, active=False)
        err = errors(E, F, Ei, ref[0], ref[2], ref[1])
        assert err["rms_F"] <= BF16_RMS_F
        # same tiles of the same edge prefix, exact zeros skipped: the two evaluations agree far below bf16 accuracy
        assert rms(F - Ff) <= 1e-3 * rms(Ff)


# ---------------------------------------------------------------- stress
def _gpu_stress(spec, blob, system, L, precision=0, grid=None, halo=0.0, shards=1):
    import torch
    mlip, ctx, model = gpu_setup(spec, blob)
    g = gpu_graph(mlip, ctx, system, spec.r_cut)
    part = mlip.Partition(ctx, g, halo, grid=grid) if grid is not None else None
    tot = None
    for k in range(shards):
        E, F, Ei, S = mlip.energy_forces_stress(ctx, model, L, g, part, precision, shard=k, n_shards=shards)
        torch.cuda.synchronize()
        out = [float(E.item()), F.cpu().numpy().astype(np.float64), S.cpu().numpy()]
        tot = out if tot is None else [a + b for a, b in zip(tot, out)]
    return tot


def test_fp32_stress_matches_oracle_unpartitioned_and_partitioned():
    """sigma = (1/V) dE/d(strain) against the oracle (itself pinned by strain finite differences):
    1e-4 of the largest component in fp32, identical decomposition over sub-domains and over shards."""
    spec = ModelSpec(4, 64, 8, 2, 3.0, 1.0 / np.sqrt(12.0))
    blob = make_weights(spec, 25)
    s = small_system(8, 0.08, seed=51)
    E_ref, Ei_ref, F_ref, sig_ref = O.energy_forces_stress(oracle_model(spec, blob), 2, s.pos, s.cell, s.species)
    scale = np.abs(sig_ref).max()
    E0, F0, S0 = _gpu_stress(spec, blob, s, 2)
    assert np.abs(S0 - sig_ref).max() <= 1e-4 * scale and np.array_equal(S0, S0.T)
    assert np.abs(F0 - F_ref).max() <= FP32_MAX_F * rms(F_ref)
    for grid, shards in [((3, 1, 1), 1), ((2, 2, 1), 1), ((4, 1, 1), 2)]:
        E, F, S = _gpu_stress(spec, blob, s, 2, grid=grid, halo=6.0, shards=shards)
        assert np.abs(S - sig_ref).max() <= 1e-4 * scale
        assert np.abs(S - S0).max() <= 1e-5 * scale
        assert np.abs(F - F0).max() <= 1e-5 * rms(F0) and abs(E - E0) <= 1e-5 * np.abs(Ei_ref).sum()
    cfg = make_config(1)
    ref = O.energy_forces_stress(oracle_model(cfg.model, cfg.weights), cfg.L, cfg.system.pos, cfg.system.cell, cfg.system.species)
    E, F, S = _gpu_stress(cfg.model, cfg.weights, cfg.system, cfg.L)
    assert np.abs(S - ref[3]).max() <= 1e-4 * np.abs(ref[3]).max()


def test_bf16_stress_matches_oracle():
    spec = ModelSpec(4, 256, 16, 2, 3.0, 1.0 / np.sqrt(12.0))
    blob = make_weights(spec, 26)
    s = small_system(8, 0.08, seed=52)
    sig_ref = O.energy_forces_stress(oracle_model(spec, blob), 2, s.pos, s.cell, s.species)[3]
    for grid in [None, (2, 1, 1)]:
        E, F, S = _gpu_stress(spec, blob, s, 2, precision=1, grid=grid, halo=6.0)
        assert np.abs(S - sig_ref).max() <= BF16_RMS_F * np.abs(sig_ref).max()


# ---------------------------------------------------------------- on-device MD
@pytest.mark.parametrize("grid,halo", [((1, 1, 1), 0.0), ((2, 1, 1), 6.0)])
def test_md_nve_matches_oracle_trajectory(grid, halo):
    """mlip_md_nve against the oracle's velocity-Verlet (pinned by its second-order energy error) on the same
    start: total energy per step, final positions and velocities. fp32 forces perturb a 20-step trajectory far
    below the tolerances; atoms cross the periodic box unwrapped, which the graph builder supports."""
    import torch
    spec = ModelSpec(4, 64, 8, 2, 3.0, 1.0 / np.sqrt(12.0))
    blob = make_weights(spec, 35)
    s = small_system(6, 0.08, seed=61)   # 21.6 A box, 864 atoms
    rng = np.random.default_rng(7)
    masses = rng.uniform(10.0, 60.0, len(s.pos))
    vel0 = rng.normal(0, 0.004, s.pos.shape); vel0 -= vel0.mean(0)
    n_steps, dt = 20, 2.0
    e_ref, pos_ref, vel_ref = O.nve_velocity_verlet(oracle_model(spec, blob), 2, s.pos, s.cell, s.species, masses,
                                                    vel0, dt, n_steps, return_state=True)
    mlip, ctx, model = gpu_setup(spec, blob)
    pos = torch.tensor(s.pos, dtype=torch.float64, device="cuda:0").contiguous()
    vel = torch.tensor(vel0, dtype=torch.float64, device="cuda:0").contiguous()
    mass = torch.tensor(masses, dtype=torch.float64, device="cuda:0")
    species = torch.tensor(s.species, dtype=torch.int32, device="cuda:0")
    e = mlip.md_nve(ctx, model, 2, pos, vel, mass, s.cell, species, dt, n_steps, grid=grid, halo=halo)
    kin0 = 0.5 * np.sum(masses[:, None] * vel0 ** 2) / O.ACC_UNIT
    assert np.abs(e - e_ref).max() <= 1e-4 * kin0
    assert np.abs(pos.cpu().numpy() - pos_ref).max() <= 1e-5          # Angstrom, after 40 fs
    assert np.abs(vel.cpu().numpy() - vel_ref).max() <= 1e-5 * np.abs(vel_ref).max() + 1e-8
    assert np.abs(pos_ref - s.pos).max() > 0.05                       # the atoms did move


# ---------------------------------------------------------------- triclinic cells (reading R12)
def test_fp32_triclinic_cell_matches_oracle_and_partitions():
    """General (non-orthorhombic) lattice, unwrapped positions: energies, forces and stress against the oracle, and a
    partitioned evaluation (bins on the scaled coordinates, halo against the perpendicular widths) against both."""
    from synth_inputs import System
    rng = np.random.default_rng(11)
    cell = np.array([[26.0, 0.0, 0.0], [5.0, 23.0, 0.0], [-4.0, 3.0, 21.0]])
    n = 1400
    pos = rng.uniform(0, 1, (n, 3)) @ cell
    # keep atoms apart (random points can sit on top of each other): reject pairs closer than 1.6 A
    g0 = O.neighbor_list(pos, cell, 1.6)
    keep = np.ones(n, bool); keep[np.maximum(g0[0], g0[1])] = False
    pos = pos[keep] + rng.integers(-1, 2, (int(keep.sum()), 3)).astype(float) @ cell
    s = System(pos, cell, rng.integers(0, 4, len(pos)).astype(np.int32))
    spec = ModelSpec(4, 64, 8, 2, 3.5, 1.0 / np.sqrt(14.0))
    blob = make_weights(spec, 55)
    E_ref, Ei_ref, F_ref, sig_ref = O.energy_forces_stress(oracle_model(spec, blob), 2, s.pos, s.cell, s.species)
    E0, F0, S0 = _gpu_stress(spec, blob, s, 2)
    assert abs(E0 - E_ref) <= FP32_EPS_E * np.abs(Ei_ref).sum()
    assert np.abs(F0 - F_ref).max() <= FP32_MAX_F * rms(F_ref)
    assert np.abs(S0 - sig_ref).max() <= 1e-4 * np.abs(sig_ref).max()
    for grid in [(2, 1, 1), (1, 2, 1), (1, 1, 2)]:
        E, F, S = _gpu_stress(spec, blob, s, 2, grid=grid, halo=7.0)
        assert np.abs(F - F0).max() <= 1e-5 * rms(F0) and abs(E - E0) <= 1e-5 * np.abs(Ei_ref).sum()
        assert np.abs(S - S0).max() <= 1e-5 * np.abs(sig_ref).max()


# ---------------------------------------------------------------- degenerate inputs
@pytest.mark.parametrize("precision,d", [(0, 64), (1, 128)])
def test_degenerate_systems(precision, d):
    """Empty box, atoms without neighbours, a sub-domain without atoms, two coincident atoms (r = 0 edges, reading R13)
    and a box smaller than r_cut (self images): finite results equal to the oracle's."""
    import torch
    from synth_inputs import System
    spec = ModelSpec(4, d, 8, 2, 3.0, 1.0 / np.sqrt(12.0))
    blob = make_weights(spec, 65)
    om = oracle_model(spec, blob)
    tolF = FP32_MAX_F if precision == 0 else 5e-2
    tolE = FP32_EPS_E if precision == 0 else 3e-3   # a handful of atoms: no averaging of the bf16 operand rounding
    # empty system
    mlip, ctx, model = gpu_setup(spec, blob)
    s0 = System(np.zeros((0, 3)), np.eye(3) * 10.0, np.zeros(0, np.int32))
    g = gpu_graph(mlip, ctx, s0, spec.r_cut)
    E, F, Ei = gpu_energy_forces(mlip, ctx, model, 2, g, None, precision)
    assert E == 0.0 and F.shape == (0, 3)
    part = mlip.Partition(ctx, g, 6.0, grid=(2, 1, 1))
    E, F, Ei = gpu_energy_forces(mlip, ctx, model, 2, g, part, precision)
    assert E == 0.0
    # three isolated atoms + one bonded pair, in a box cut so that some bins are empty
    pos = np.array([[1.0, 1.0, 1.0], [12.0, 1.0, 1.0], [1.0, 14.0, 9.0], [20.0, 20.0, 20.0], [21.9, 20.3, 19.8]])
    s1 = System(pos, np.eye(3) * 40.0, np.array([0, 1, 2, 3, 1], np.int32))
    ref = O.energy_forces(om, 2, s1.pos, s1.cell, s1.species)
    for grid in [None, (4, 1, 1), (2, 2, 2)]:
        E, F, Ei = _run(spec, blob, s1, 2, precision, grid=grid, halo=6.0)
        assert abs(E - ref[0]) <= tolE * np.abs(ref[1]).sum()
        assert np.abs(F - ref[2]).max() <= tolF * max(rms(ref[2]), 1e-6) + 1e-6
        assert np.all(F[:3] == 0.0)
    # two coincident atoms: the r = 0 edges are kept, their direction is defined as zero
    s2 = small_system(3, 0.05, seed=9)
    pos2 = s2.pos.copy(); pos2[5] = pos2[17]
    s2 = System(pos2, s2.cell, s2.species)
    ref = O.energy_forces(om, 2, s2.pos, s2.cell, s2.species)
    E, F, Ei = _run(spec, blob, s2, 2, precision)
    assert np.all(np.isfinite(F)) and abs(E - ref[0]) <= tolE * np.abs(ref[1]).sum()
    assert np.abs(F - ref[2]).max() <= tolF * rms(ref[2])
    # box smaller than r_cut: an atom is its own neighbour through the periodic images
    s3 = System(np.array([[0.3, 0.2, 0.1], [1.4, 1.2, 1.1]]), np.eye(3) * 2.6, np.array([0, 2], np.int32))
    ref = O.energy_forces(om, 2, s3.pos, s3.cell, s3.species)
    E, F, Ei = _run(spec, blob, s3, 2, precision)
    assert abs(E - ref[0]) <= tolE * np.abs(ref[1]).sum()
    # the net force is what is left of much larger image contributions that cancel: the bf16 path is held to an absolute bound
    assert np.abs(F - ref[2]).max() <= tolF * max(rms(ref[2]), 1e-6) + (1e-6 if precision == 0 else 1e-4)


def test_sharded_partition_builds_only_its_sub_domains_and_sums_to_the_full_result():
    """mlip_partition_grid_shard (one rank, its sub-domains only): the sub-domains of other shards are empty
    handles, the partial results of all shards sum to the result of the full partition, and a handle is refused by an
    evaluation with another (shard, n_shards)."""
    import torch
    import paper_2509_21694_b200 as mlip
    spec = ModelSpec(4, 64, 8, 2, 3.0, 1.0 / np.sqrt(12.0))
    blob = make_weights(spec, 91)
    s = small_system(8, 0.08, seed=17)
    m, ctx, model = gpu_setup(spec, blob)
    g = gpu_graph(m, ctx, s, spec.r_cut)
    grid, halo, n_shards = (2, 2, 1), 6.0, 3
    full = mlip.Partition(ctx, g, halo, grid=grid)
    E0, F0, Ei0 = gpu_energy_forces(m, ctx, model, 2, g, full, 0)
    info0 = full.info()
    E, F, Ei = 0.0, 0.0, 0.0
    for k in range(n_shards):
        part = mlip.Partition(ctx, g, halo, grid=grid, shard=k, n_shards=n_shards)
        info = part.info()
        assert len(info) == 4
        for j in range(4):
            assert info[j] == (info0[j] if j % n_shards == k else dict(n_owned=0, n_ext=0, n_edges=0))
        e, f, ei = mlip.energy_forces_shard(ctx, model, 2, g, part, k, n_shards, 0, want_atom_energy=True)
        ctx.status()
        E += float(e.item()); F = F + f.double().cpu().numpy(); Ei = Ei + ei.double().cpu().numpy()
        with pytest.raises(mlip.MlipError) as err:
            mlip.energy_forces_shard(ctx, model, 2, g, part, (k + 1) % n_shards, n_shards, 0)
        assert err.value.code == -1
        with pytest.raises(mlip.MlipError) as err:
            mlip.energy_forces(ctx, model, 2, g, part, 0)
        assert err.value.code == -1
    assert abs(E - E0) <= 1e-6 * np.abs(Ei0).sum() and np.abs(F - F0).max() <= 1e-6 * rms(F0) and np.array_equal(Ei, Ei0)
    with pytest.raises(mlip.MlipError):
        mlip.Partition(ctx, g, halo, grid=grid, shard=3, n_shards=3)

