"""Pins for the oracle's radius graph (O1): brute force, closed forms, a library
k-d tree with periodic box, symmetry and lattice-translation invariance."""
import os

import numpy as np
import pytest
from scipy.spatial import cKDTree

from oracle import mlip_oracle as O
from synth_inputs import fcc_box, small_system

HERE = os.path.dirname(__file__)


def _same(g1, g2):
    return all(np.array_equal(a, b) for a, b in zip(g1, g2))


@pytest.mark.parametrize("n_cells,r_cut", [(3, 5.0), (2, 5.0), (2, 3.0), (1, 5.0)])
def test_cells_equals_bruteforce(n_cells, r_cut):
    # n_cells=2: box 7.2 A < 2 r_cut (several images of the same pair); n_cells=1: box < r_cut
    s = small_system(n_cells, 0.05, seed=n_cells)
    gb = O.neighbor_list_bruteforce(s.pos, s.cell, r_cut)
    gc = O.neighbor_list(s.pos, s.cell, r_cut)
    assert len(gb[0]) > 0 and _same(gb, gc)


def test_triclinic_and_unwrapped_equals_bruteforce():
    rng = np.random.default_rng(7)
    cell = np.array([[9.0, 0.0, 0.0], [2.5, 8.0, 0.0], [-1.5, 2.0, 7.5]])
    pos = rng.uniform(0, 1, (40, 3)) @ cell
    pos += rng.integers(-2, 3, (40, 3)).astype(float) @ cell  # unwrapped by lattice vectors
    gb = O.neighbor_list_bruteforce(pos, cell, 4.0)
    gc = O.neighbor_list(pos, cell, 4.0)
    assert len(gb[0]) > 100 and _same(gb, gc)


def test_fcc_shell_counts_closed_form():
    shells = np.loadtxt(os.path.join(HERE, "golden", "fcc_shells.txt"), dtype=int)
    a = 3.6
    sites, cell = fcc_box(6, a)  # 864 atoms
    for r_cut in (5.0, 6.0):
        expected = sum(c for n, c in shells if a * np.sqrt(n / 2.0) < r_cut)
        recv, send, shift = O.neighbor_list(sites, cell, r_cut)
        deg = np.bincount(recv, minlength=len(sites))
        assert np.all(deg == expected)
    assert sum(c for n, c in shells if a * np.sqrt(n / 2.0) < 5.0) == 42
    assert sum(c for n, c in shells if a * np.sqrt(n / 2.0) < 6.0) == 78
    # shell radii: sorted distinct distances of atom 0 match a*sqrt(n/2)
    _, r = O.edge_vectors(sites, cell, recv, send, shift)
    r0 = np.unique(np.round(r[recv == 0], 9))
    assert np.allclose(r0, [a * np.sqrt(n / 2.0) for n in range(1, 6)])


def test_against_kdtree_periodic_library():
    s = small_system(4, 0.1, seed=3)  # 14.4 A box >= 2 r_cut
    r_cut = 6.0
    recv, send, shift = O.neighbor_list(s.pos, s.cell, r_cut)
    box = np.diag(s.cell)
    wrapped = np.mod(s.pos, box)
    pairs = cKDTree(wrapped, boxsize=box).query_pairs(r_cut, output_type="ndarray")
    assert len(recv) == 2 * len(pairs)
    mine = set(zip(recv.tolist(), send.tolist()))
    lib = set(map(tuple, pairs.tolist())) | set(map(tuple, pairs[:, ::-1].tolist()))
    assert mine == lib


def test_symmetric_sorted_strict():
    s = small_system(3, 0.05, seed=1)
    recv, send, shift = O.neighbor_list(s.pos, s.cell, 5.0)
    fwd = set(zip(recv.tolist(), send.tolist(), map(tuple, shift.tolist())))
    rev = set(zip(send.tolist(), recv.tolist(), map(tuple, (-shift).tolist())))
    assert fwd == rev
    key = np.stack([recv, send, shift[:, 0], shift[:, 1], shift[:, 2]], 1)
    assert all(tuple(key[i]) < tuple(key[i + 1]) for i in range(len(key) - 1))
    _, r = O.edge_vectors(s.pos, s.cell, recv, send, shift)
    assert r.max() < 5.0 and r.min() > 0
    # strictness: a pair exactly at the cutoff is excluded
    pos = np.array([[0.0, 0, 0], [3.0, 0, 0]]); cell = np.eye(3) * 20
    assert len(O.neighbor_list(pos, cell, 3.0)[0]) == 0
    assert len(O.neighbor_list(pos, cell, np.nextafter(3.0, 4.0))[0]) == 2


def test_lattice_translation_of_one_atom():
    s = small_system(3, 0.05, seed=2)
    g1 = O.neighbor_list(s.pos, s.cell, 5.0)
    pos2 = s.pos.copy(); pos2[17] += 2 * s.cell[0] - s.cell[2]
    g2 = O.neighbor_list(pos2, s.cell, 5.0)
    assert np.array_equal(g1[0], g2[0]) and np.array_equal(g1[1], g2[1])
    r1 = np.sort(O.edge_vectors(s.pos, s.cell, *g1)[1]); r2 = np.sort(O.edge_vectors(pos2, s.cell, *g2)[1])
    assert np.allclose(r1, r2, rtol=0, atol=1e-12)
    # shifts of edges touching atom 17 changed by exactly the lattice vector
    touched = (g1[0] == 17) ^ (g1[1] == 17)
    dn = g2[2] - g1[2]
    assert np.all(dn[~touched] == 0)
    assert np.all(dn[g1[0] == 17][g1[1][g1[0] == 17] != 17] == np.array([2, 0, -1]))
