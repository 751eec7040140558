"""-m gpu: the CUDA cell-list graph (mlip_build_graph / mlip_graph_export_edges) must equal the
oracle's edge list BIT-EXACTLY in canonical order (north_star), incl. boxes smaller than
2 r_cut, a single cell, triclinic cells and unwrapped positions; partition sizes are checked
against the oracle's partition (O6)."""
import numpy as np
import pytest

from oracle import mlip_oracle as O
from synth_inputs import System, make_config, small_system

pytestmark = pytest.mark.gpu


def _ctx():
    import paper_2509_21694_b200 as mlip
    return mlip, mlip.Context(0)


def _compare(system, r_cut):
    from tests.gpu_util import gpu_graph
    mlip, ctx = _ctx()
    g = gpu_graph(mlip, ctx, system, r_cut)
    recv, send, shift = [t.cpu().numpy() for t in g.export_edges()]
    o_recv, o_send, o_shift = O.neighbor_list(system.pos, system.cell, r_cut)
    assert g.num_edges == len(o_recv)
    assert np.array_equal(recv, o_recv) and np.array_equal(send, o_send) and np.array_equal(shift, o_shift)
    return g.num_edges


@pytest.mark.parametrize("n_cells,r_cut", [(3, 5.0), (2, 5.0), (2, 3.0), (1, 5.0), (6, 6.0), (7, 5.0)])
def test_edge_list_bit_exact_fcc(n_cells, r_cut):
    s = small_system(n_cells, 0.08, seed=n_cells, vacancy_fraction=0.03 if n_cells >= 6 else 0.0)
    assert _compare(s, r_cut) > 0


def test_edge_list_config1():
    cfg = make_config(1)
    assert _compare(cfg.system, cfg.model.r_cut) > 4000


def test_edge_list_triclinic_unwrapped():
    rng = np.random.default_rng(7)
    cell = np.array([[19.0, 0.0, 0.0], [4.5, 17.0, 0.0], [-3.5, 2.0, 15.5]])
    pos = rng.uniform(0, 1, (600, 3)) @ cell
    pos += rng.integers(-2, 3, (600, 3)).astype(float) @ cell
    s = System(pos, cell, rng.integers(0, 4, 600).astype(np.int32))
    assert _compare(s, 4.0) > 1000


def test_edge_list_degenerate_inputs():
    s = System(np.array([[1.0, 2.0, 3.0]]), np.eye(3) * 4.0, np.zeros(1, np.int32))
    assert _compare(s, 5.0) == len(O.neighbor_list_bruteforce(s.pos, s.cell, 5.0)[0])  # self images only
    s2 = System(np.array([[0.0, 0, 0], [9.0, 9, 9]]), np.eye(3) * 30.0, np.zeros(2, np.int32))
    mlip, ctx = _ctx()
    from tests.gpu_util import gpu_graph
    assert gpu_graph(mlip, ctx, s2, 5.0).num_edges == 0
    s0 = System(np.zeros((0, 3)), np.eye(3) * 10.0, np.zeros(0, np.int32))
    assert gpu_graph(mlip, ctx, s0, 5.0).num_edges == 0


def test_edge_list_medium_box_cfg2_recipe():
    cfg = make_config(2, with_weights=False, n_cells_override=9)  # 2.8k atoms, r_cut 6, vacancies
    assert _compare(cfg.system, 6.0) > 200000


def test_partition_sizes_match_oracle():
    from tests.gpu_util import gpu_graph
    mlip, ctx = _ctx()
    s = small_system(10, 0.1, seed=4)  # 36 A box, 4000 atoms
    g = gpu_graph(mlip, ctx, s, 5.0)
    graph = O.neighbor_list(s.pos, s.cell, 5.0)
    # geometric halo (reading R2): the whole box of atoms within `halo` of the bin along every axis
    ctx.set_khop_halo(False)
    for grid, halo in [((3, 1, 1), 5.0), ((2, 2, 1), 4.0), ((1, 1, 4), 2.0)]:
        part = mlip.Partition(ctx, g, halo, grid=grid)
        info = part.info()
        oparts = O.partition_grid(s.pos, s.cell, grid, halo)
        assert sum(i["n_owned"] for i in info) == len(s.pos)
        for i, (owned, ext) in zip(info, oparts):
            assert i["n_owned"] == len(owned) and i["n_ext"] == len(ext)
            assert i["n_edges"] == len(O.induced_subgraph(graph, ext, len(s.pos))[0])
    slab = mlip.Partition(ctx, g, 5.0, n_sub=3).info()
    assert [i["n_owned"] for i in slab] == [len(p[0]) for p in O.partition_slabs(s.pos, s.cell, 3, 5.0)]
    # K-hop halo (the default): breadth-first search from the root atoms inside that box
    ctx.set_khop_halo(True)
    for grid, halo in [((3, 1, 1), 5.0), ((2, 2, 1), 4.0), ((1, 1, 4), 2.0), ((2, 1, 1), 10.0), ((1, 2, 1), 9.0)]:
        info = mlip.Partition(ctx, g, halo, grid=grid).info()
        oparts = O.partition_grid_khop(s.pos, s.cell, grid, halo, 5.0, graph)
        assert sum(i["n_owned"] for i in info) == len(s.pos)
        for i, (owned, ext, hops) in zip(info, oparts):
            assert i["n_owned"] == len(owned) and i["n_ext"] == len(ext)
            assert i["n_edges"] == len(O.induced_subgraph(graph, ext, len(s.pos))[0])


def test_edge_list_clustered_atoms_overflow_fallback():
    """A dense cluster in a large, mostly empty box: the per-atom scratch rows of the one-pass neighbour search are sized
    from the MEAN density and overflow here, so the builder must fall back to count + fill -- same bit-exact list."""
    rng = np.random.default_rng(23)
    pts = rng.normal(0.0, 2.5, (400, 3)) + 30.0
    far = rng.uniform(0, 60.0, (50, 3))
    s = System(np.concatenate([pts, far]), np.eye(3) * 60.0, rng.integers(0, 4, 450).astype(np.int32))
    n = _compare(s, 5.0)
    assert n > 450 * 60   # mean degree far above the scratch capacity of 1.5 * (4/3 pi r^3 N / V) + 32 ~ 33
