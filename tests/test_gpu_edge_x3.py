"""-m gpu: edge cases of the fp32 tensor-core edge kernels (csrc/edge_x3.cu: MLIP_FP32 at d = 128, every contraction as six
bf16 MMAs over 3-term operand splits) against the float64 oracle at the fp32 tolerances of north_star
(per-atom energy 1e-5, max force error 1e-4 RMS F): sparse graphs whose 128-edge tiles hold more receivers than the
selector MMA of the segmented sum takes, fewer radial functions than the padded K of G1, one ragged tile, isolated atoms,
weights far outside the IEEE-half range (the split keeps the fp32 exponent), bitwise reproducibility, partitions, and the
device-side edge count of the Verlet-skin MD driver."""
import numpy as np
import pytest

from oracle import mlip_oracle as O
from synth_inputs import ModelSpec, System, make_water_system, make_weights, small_system
from tests.gpu_util import errors, gpu_energy_forces, gpu_graph, gpu_setup, oracle_model, rms

pytestmark = pytest.mark.gpu
FP32_EPS_E, FP32_MAX_F, FP32_REL_EI = 1e-5, 1e-4, 1e-5


def _run(spec, blob, system, L, grid=None, halo=0.0):
    mlip, ctx, model = gpu_setup(spec, blob)
    g = gpu_graph(mlip, ctx, system, spec.r_cut)
    part = mlip.Partition(ctx, g, halo, grid=grid) if grid is not None else None
    return gpu_energy_forces(mlip, ctx, model, L, g, part, 0)


def _check(out, ref):
    err = errors(out[0], out[1], out[2], ref[0], ref[2], ref[1])
    assert err["eps_E"] <= FP32_EPS_E and err["rel_Ei"] <= FP32_REL_EI and err["max_F"] <= FP32_MAX_F, err
    return err


@pytest.mark.parametrize("vacancy,min_recv_per_tile", [(0.55, 16), (0.15, 8)])
def test_x3_sparse_graph_many_receivers_per_tile(vacancy, min_recv_per_tile):
    """Mean in-degree 5 / 10: tiles with more than 16 receivers take the shared-memory loop of the segmented sum instead of
    the selector MMA, in both passes; isolated atoms are part of the first case."""
    r_cut, L = 3.0, 3
    s = small_system(10, 0.08, seed=int(100 * vacancy) + 128, vacancy_fraction=vacancy)
    recv = O.neighbor_list(s.pos, s.cell, r_cut)[0]
    deg = np.bincount(recv, minlength=len(s.pos))
    n_tiles = -(-len(recv) // 128)
    assert int((deg > 0).sum()) > min_recv_per_tile * n_tiles     # pigeonhole: some tile holds more receivers than that
    spec = ModelSpec(4, 128, 16, L, r_cut, 1.0 / np.sqrt(max(deg.mean(), 1.0)))
    blob = make_weights(spec, 428)
    ref = O.energy_forces(oracle_model(spec, blob), L, s.pos, s.cell, s.species)
    for grid in [None, (2, 1, 1), (2, 2, 1)]:
        err = _check(_run(spec, blob, s, L, grid=grid, halo=L * r_cut), ref)
        print(vacancy, grid, err)


@pytest.mark.parametrize("n_rbf", [2, 8, 13])
def test_x3_fewer_radial_functions_than_padded_k(n_rbf):
    spec = ModelSpec(4, 128, n_rbf, 2, 5.0, 1.0 / np.sqrt(43.0))
    blob = make_weights(spec, 430 + n_rbf)
    s = small_system(4, 0.08, seed=31)
    _check(_run(spec, blob, s, 2), O.energy_forces(oracle_model(spec, blob), 2, s.pos, s.cell, s.species))


def test_x3_single_ragged_tile_pair_and_isolated_atoms():
    """3 atoms in a big box: one bonded pair (2 edges: one tile, 126 empty rows) and an atom without neighbours."""
    spec = ModelSpec(2, 128, 16, 2, 3.0, 1.0)
    blob = make_weights(spec, 440)
    s = System(np.array([[5.0, 5.0, 5.0], [6.9, 5.3, 4.8], [15.0, 15.0, 15.0]]), np.eye(3) * 30.0, np.array([0, 1, 1], dtype=np.int32))
    ref = O.energy_forces(oracle_model(spec, blob), 2, s.pos, s.cell, s.species)
    out = _run(spec, blob, s, 2)
    _check(out, ref)
    assert np.all(out[1][2] == 0.0)                               # the isolated atom feels nothing


def test_x3_weights_outside_the_half_range_and_reproducible():
    """All weights x 30: the 16-bit path reports MLIP_ERR_NUMERIC for this model (tests/test_gpu_parity_gaps.py); the 3-term
    split has the exponent range of fp32. Forces of 1e14 eV/A: the problem is ill-conditioned in fp32 whatever evaluates it
    (edge vectors are stored in fp32) -- the CUDA-core kernels have the same largest force error, 2.6e-4 of RMS F at the same
    atom -- so the force bound here is 1e-3; the energies keep the north_star bounds. Two evaluations agree bit for bit (the
    only reduction instruction adds one term per edge and launch)."""
    spec = ModelSpec(4, 128, 16, 2, 5.0, 1.0 / np.sqrt(43.0))
    blob = (make_weights(spec, 441) * np.float32(30.0)).astype(np.float32)
    s = small_system(4, 0.1, seed=5)
    ref = O.energy_forces(oracle_model(spec, blob), 2, s.pos, s.cell, s.species)
    a = _run(spec, blob, s, 2, grid=(2, 1, 1), halo=10.0)
    b = _run(spec, blob, s, 2, grid=(2, 1, 1), halo=10.0)
    err = errors(a[0], a[1], a[2], ref[0], ref[2], ref[1])
    assert np.isfinite(a[1]).all() and err["eps_E"] <= FP32_EPS_E and err["rel_Ei"] <= FP32_REL_EI and err["max_F"] <= 1e-3, err
    assert a[0] == b[0] and np.array_equal(a[1], b[1]) and np.array_equal(a[2], b[2])


def test_x3_three_body_partitioned_water():
    """Angle terms through K = 32 of G1 and N = 32 of G4, 3 slabs: equals the unpartitioned result and the oracle."""
    spec = ModelSpec(2, 128, 16, 3, 5.0, 1.0 / np.sqrt(53.0), r_cut3=4.0)
    blob = make_weights(spec, 442)
    s = make_water_system(6, seed_pos=1142, seed_orient=3142)     # 648 atoms, box 18.7 A
    ref = O.energy_forces(oracle_model(spec, blob), 3, s.pos, s.cell, s.species)
    one = _run(spec, blob, s, 3)
    _check(one, ref)
    part = _run(spec, blob, s, 3, grid=(3, 1, 1), halo=15.0)
    _check(part, ref)
    assert np.abs(part[1] - one[1]).max() <= 1e-5 * rms(one[1])


def test_x3_md_skin_device_side_edge_count():
    """MLIP_FP32 at d = 128 through mlip_md_run with a Verlet skin and CUDA-graph replay: the edge kernels read their edge
    count from the device (EdgeArgs::E_dyn), CTAs beyond the filtered list have no tile."""
    import torch
    import paper_2509_21694_b200 as mlip
    spec = ModelSpec(4, 128, 16, 2, 3.0, 1.0 / np.sqrt(12.0))
    blob = make_weights(spec, 443)
    s = small_system(6, 0.08, seed=63)
    rng = np.random.default_rng(10)
    masses = rng.uniform(10.0, 60.0, len(s.pos))
    vel0 = rng.normal(0, 0.005, s.pos.shape); vel0 -= vel0.mean(0)

    def run(**kw):
        m, ctx, model = gpu_setup(spec, blob)
        pos = torch.tensor(s.pos, dtype=torch.float64, device="cuda:0").contiguous()
        vel = torch.tensor(vel0, dtype=torch.float64, device="cuda:0").contiguous()
        mass = torch.tensor(masses, dtype=torch.float64, device="cuda:0")
        species = torch.tensor(s.species, dtype=torch.int32, device="cuda:0")
        e, st = m.md_run(ctx, model, 2, pos, vel, mass, s.cell, species, 2.0, 20, **kw)
        return e, pos.cpu().numpy(), st

    e0, p0, _ = run()
    e1, p1, st = run(skin=0.5, cuda_graph=True, grid=(2, 1, 1), halo=6.0)
    assert st["n_graph_replays"] == 21
    # positions: fp32 forces, different tile boundaries (2 slabs against none). Energies: fp32 per-atom energies of 864 atoms
    # summed in a different order, 1e-5 eV measured
    assert np.abs(p1 - p0).max() <= 1e-5 and np.abs(e1 - e0).max() <= 5e-5
    e_ref, pos_ref, _ = O.nve_velocity_verlet(oracle_model(spec, blob), 2, s.pos, s.cell, s.species, masses, vel0, 2.0, 20,
                                              return_state=True)
    assert np.abs(p1 - pos_ref).max() <= 1e-5
