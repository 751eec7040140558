"""Pins for the oracle's model, forces and partitioned assembly (O2-O6): closed forms, finite
differences, an independent torch.float64 autograd re-derivation, invariances, the paper's
partition-exactness statement with its negative control, the receptive
field r_eff = M r_c, MPDP truncation, and NVE conservation order."""
import numpy as np
import pytest
import torch

from oracle import mlip_oracle as O
from synth_inputs import ModelSpec, fcc_box, make_weights, small_system


def make_model(d=16, n_rbf=8, L_max=2, r_cut=5.0, n_species=4, seed=11, nbar=43.0):
    spec = ModelSpec(n_species, d, n_rbf, L_max, r_cut, 1.0 / np.sqrt(nbar))
    blob = make_weights(spec, seed)
    return spec, blob, O.parse_weights(n_species, d, n_rbf, L_max, r_cut, spec.agg_scale, blob)


def rms(x):
    return float(np.sqrt(np.mean(np.square(x))))


# ---------------------------------------------------------------- features (O2)
def test_feature_closed_forms():
    rc = 5.0
    u, du = O.envelope(np.array([0.0, rc, rc / 2]), rc)
    assert u[0] == 1.0 and abs(u[1]) < 1e-16 and abs(du[1]) < 1e-15 and abs(u[2] - 0.5) < 1e-16
    mu = np.arange(8) * rc / 7
    g, dg = O.rbf(mu, rc, 8)
    assert np.allclose(np.diag(g), 1.0) and np.allclose(np.diag(dg), 0.0)
    # neighbouring centre: exp(-1/2)
    assert np.allclose(np.diag(g, 1), np.exp(-0.5))
    # derivatives by central differences
    r = np.linspace(0.3, 4.9, 9); h = 1e-6
    assert np.allclose((O.envelope(r + h, rc)[0] - O.envelope(r - h, rc)[0]) / (2 * h), O.envelope(r, rc)[1], atol=1e-9)
    assert np.allclose((O.rbf(r + h, rc, 8)[0] - O.rbf(r - h, rc, 8)[0]) / (2 * h), O.rbf(r, rc, 8)[1], atol=1e-8)
    x = np.linspace(-6, 6, 25)
    assert np.allclose(O.silu(x), x / (1 + np.exp(-x)))
    assert np.allclose((O.silu(x + h) - O.silu(x - h)) / (2 * h), O.dsilu(x), atol=1e-9)


# ---------------------------------------------------------------- energies (O3, O4)
def test_L0_closed_form_and_blob_order():
    spec, blob, m = make_model()
    s = small_system(3, 0.05, seed=4)
    E, E_i, F = O.energy_forces(m, 0, s.pos, s.cell, s.species)
    # independent unpacking of the tail of the blob: Wo, bo, wo, bE are the last d*d+2d+1 values
    d = spec.d; b = blob.astype(np.float64)
    Wo = b[-(d * d + 2 * d + 1):-(2 * d + 1)].reshape(d, d); bo = b[-(2 * d + 1):-(d + 1)]
    wo = b[-(d + 1):-1]; bE = b[-1]
    T = b[:spec.n_species * d].reshape(-1, d); E0 = b[spec.n_species * d:spec.n_species * d + spec.n_species]
    o = T @ Wo.T + bo
    e_species = (o / (1 + np.exp(-o))) @ wo + bE + E0
    assert np.allclose(E_i, e_species[s.species], rtol=1e-13)
    assert abs(E - e_species[s.species].sum()) < 1e-10 and np.all(F == 0)


def test_dimer_constant_beyond_cutoff_and_C1():
    spec, blob, m = make_model(L_max=2)
    cell = np.eye(3) * 40.0; species = np.array([0, 1])

    def E(r):
        return O.energy_forces(m, 2, np.array([[5.0, 5, 5], [5.0 + r, 5, 5]]), cell, species)[0]

    e_far = E(7.0)
    assert E(5.0) == e_far and E(6.3) == e_far            # no edge: exactly the isolated-atom sum
    assert abs(E(4.0) - e_far) > 1e-6                     # interacting inside the cutoff
    eps = 1e-3
    assert abs(E(5.0 - eps) - e_far) < 50 * eps ** 2      # value and slope vanish at r_cut (C1)
    F = O.energy_forces(m, 2, np.array([[5.0, 5, 5], [5.0 + 5.0 - 1e-7, 5, 5]]), cell, species)[2]
    assert np.abs(F).max() < 1e-5


def test_perfect_lattice_and_supercell():
    spec, blob, m = make_model(n_species=1)
    sites, cell = fcc_box(3, 3.6)
    z = np.zeros(len(sites), np.int32)
    E, E_i, F = O.energy_forces(m, 2, sites, cell, z)
    assert np.ptp(E_i) < 1e-12 and np.abs(F).max() < 1e-12
    s = small_system(2, 0.05, seed=5)
    spec4, _, m4 = make_model()
    E1, Ei1, F1 = O.energy_forces(m4, 2, s.pos, s.cell, s.species)
    reps = [np.array([a, b, c], float) for a in range(2) for b in range(2) for c in range(2)]
    pos8 = np.concatenate([s.pos + r @ s.cell for r in reps]); z8 = np.tile(s.species, 8)
    E8, Ei8, F8 = O.energy_forces(m4, 2, pos8, 2 * s.cell, z8)
    assert abs(E8 - 8 * E1) < 1e-10 * abs(E1) and np.allclose(F8, np.tile(F1, (8, 1)), atol=1e-12)


def test_invariances_and_zero_total_force():
    spec, blob, m = make_model()
    s = small_system(3, 0.05, seed=6)
    E, E_i, F = O.energy_forces(m, 2, s.pos, s.cell, s.species)
    assert np.abs(F.sum(0)).max() < 1e-13
    Et, _, Ft = O.energy_forces(m, 2, s.pos + np.array([0.37, -1.2, 5.5]), s.cell, s.species)
    assert abs(Et - E) < 1e-10 and np.allclose(Ft, F, atol=1e-11)
    q, _ = np.linalg.qr(np.random.default_rng(0).normal(size=(3, 3)))
    q *= np.sign(np.linalg.det(q))
    Er, _, Fr = O.energy_forces(m, 2, s.pos @ q.T, s.cell @ q.T, s.species)
    assert abs(Er - E) < 1e-10 and np.allclose(Fr, F @ q.T, atol=1e-11)
    perm = np.random.default_rng(1).permutation(len(s.pos))
    Ep, Eip, Fp = O.energy_forces(m, 2, s.pos[perm], s.cell, s.species[perm])
    assert abs(Ep - E) < 1e-10 and np.allclose(Fp, F[perm], atol=1e-11) and np.allclose(Eip, E_i[perm], atol=1e-11)


def test_mpdp_truncation_uses_first_layers():
    """keep the first K layers, feed layer-K features to the head."""
    spec, blob, m = make_model(L_max=3)
    s = small_system(2, 0.05, seed=8)
    E1 = O.energy_forces(m, 1, s.pos, s.cell, s.species)[0]
    E3 = O.energy_forces(m, 3, s.pos, s.cell, s.species)[0]
    # a 1-layer model built from the same first layer + the same head
    d, k, S = spec.d, spec.n_rbf, spec.n_species
    per_layer = d * (2 * d + k) + d + d * d + d + 2 * d * d + d + d * d + d
    head = S * d + S
    blob1 = np.concatenate([blob[:head + per_layer], blob[head + 3 * per_layer:]])
    m1 = O.parse_weights(S, d, k, 1, spec.r_cut, spec.agg_scale, blob1)
    assert O.energy_forces(m1, 1, s.pos, s.cell, s.species)[0] == E1 and abs(E3 - E1) > 1e-8


def test_receptive_field():
    """r_eff = M r_c: an atom farther than L r_cut from atom i cannot change E_i."""
    spec, blob, m = make_model(r_cut=3.0, nbar=12.0)
    s = small_system(6, 0.05, seed=9)  # 21.6 A box
    L = 2
    _, E_i, _ = O.energy_forces(m, L, s.pos, s.cell, s.species)
    k = 100
    pos2 = s.pos.copy(); pos2[k] += np.array([0.2, -0.15, 0.1])
    _, E_i2, _ = O.energy_forces(m, L, pos2, s.cell, s.species)
    box = np.diag(s.cell)
    dmin = np.minimum(np.linalg.norm((s.pos - s.pos[k] + box / 2) % box - box / 2, axis=1),
                      np.linalg.norm((s.pos - pos2[k] + box / 2) % box - box / 2, axis=1))
    far = dmin > L * 3.0
    assert far.sum() > 50 and np.all(E_i2[far] == E_i[far])
    near = dmin < 3.0
    assert np.abs(E_i2[near] - E_i[near]).max() > 1e-8


# ---------------------------------------------------------------- forces (O5)
def test_forces_finite_differences():
    spec, blob, m = make_model()
    s = small_system(2, 0.08, seed=10)
    E, _, F = O.energy_forces(m, 2, s.pos, s.cell, s.species)
    h = 1e-4
    rng = np.random.default_rng(3)
    for k, a in zip(rng.integers(0, len(s.pos), 8), rng.integers(0, 3, 8)):
        p = s.pos.copy(); p[k, a] += h; Ep = O.energy_forces(m, 2, p, s.cell, s.species)[0]
        p[k, a] -= 2 * h; Em = O.energy_forces(m, 2, p, s.cell, s.species)[0]
        assert abs(-(Ep - Em) / (2 * h) - F[k, a]) < 1e-6 * rms(F)


def _torch_energy(blob, spec, L, pos, cell, species, recv, send, shift, omega=None):
    """Independent restatement of O1-O4 in torch (float64); forces come from autograd."""
    w = torch.tensor(blob, dtype=torch.float64)
    S, d, k = spec.n_species, spec.d, spec.n_rbf
    off = 0

    def take(*shape):
        nonlocal off
        n = int(np.prod(shape)); t = w[off:off + n].reshape(shape); off += n
        return t

    T = take(S, d); E0 = take(S)
    layers = [[take(d, 2 * d + k), take(d), take(d, d), take(d), take(d, 2 * d), take(d), take(d, d), take(d)]
              for _ in range(spec.L_max)]
    Wo = take(d, d); bo = take(d); wo = take(d); bE = take(1)
    x = torch.tensor(pos, dtype=torch.float64, requires_grad=True)
    C = torch.tensor(cell, dtype=torch.float64)
    ri = torch.tensor(recv, dtype=torch.long); si = torch.tensor(send, dtype=torch.long)
    z = torch.tensor(species, dtype=torch.long)
    rv = x[si] - x[ri] + torch.tensor(shift, dtype=torch.float64) @ C
    r = rv.norm(dim=1)
    u = 0.5 * (torch.cos(torch.pi * r / spec.r_cut) + 1)
    delta = spec.r_cut / (k - 1)
    g = torch.exp(-(r[:, None] - torch.arange(k, dtype=torch.float64) * delta) ** 2 / (2 * delta ** 2))
    h = T[z]
    act = torch.nn.functional.silu
    for W1, b1, W2, b2, V1, c1, V2, c2 in layers[:L]:
        a = torch.cat([h[ri], h[si], u[:, None] * g], 1) @ W1.T + b1
        phi = act(act(a) @ W2.T + b2)
        mm = torch.zeros_like(h).index_add(0, ri, spec.agg_scale * u[:, None] * phi)
        h = h + act(torch.cat([h, mm], 1) @ V1.T + c1) @ V2.T + c2
    E_i = act(h @ Wo.T + bo) @ wo + bE + E0[z]
    om = torch.ones_like(E_i) if omega is None else torch.tensor(omega, dtype=torch.float64)
    E = (om * E_i).sum()
    E.backward()
    return E.item(), E_i.detach().numpy(), -x.grad.numpy()


def test_forces_against_torch_autograd():
    spec, blob, m = make_model(L_max=3)
    s = small_system(3, 0.05, seed=12)
    g = O.neighbor_list(s.pos, s.cell, spec.r_cut)
    E, E_i, F = O.energy_forces(m, 3, s.pos, s.cell, s.species, g)
    Et, Eit, Ft = _torch_energy(blob, spec, 3, s.pos, s.cell, s.species, *g)
    assert abs(E - Et) < 1e-11 * np.abs(E_i).sum()
    assert np.allclose(E_i, Eit, rtol=0, atol=1e-11)
    assert np.abs(F - Ft).max() < 1e-11 * max(rms(F), 1e-3)
    # weighted (owned-mask) objective, as used per sub-domain
    om = (np.arange(len(s.pos)) % 3 == 0).astype(float)
    Ew, _, Fw = O.energy_forces(m, 3, s.pos, s.cell, s.species, g, omega=om)
    Etw, _, Ftw = _torch_energy(blob, spec, 3, s.pos, s.cell, s.species, *g, omega=om)
    assert abs(Ew - Etw) < 1e-10 and np.abs(Fw - Ftw).max() < 1e-11 * max(rms(Fw), 1e-3)


# ---------------------------------------------------------------- partition (O6)
@pytest.mark.parametrize("grid", [(2, 1, 1), (3, 1, 1), (1, 2, 2), (2, 2, 1)])
def test_partitioned_equals_unpartitioned(grid):
    """every root node keeps exactly its K-hop neighbourhood; PAPER.md:169-171:
    sum root energies, sum gradients of root energies over sub-graphs."""
    spec, blob, m = make_model(r_cut=3.0, nbar=12.0)
    rng = np.random.default_rng(21)
    n = (10, 4, 4) if grid[0] > 1 else (4, 8, 8)   # long axis is the one that is cut
    idx = np.indices(n).reshape(3, -1).T.astype(float)
    basis = np.array([[0, 0, 0], [.5, .5, 0], [.5, 0, .5], [0, .5, .5]])
    pos = (idx[:, None, :] + basis[None]).reshape(-1, 3) * 3.6
    cell = np.diag(np.array(n) * 3.6)
    pos = pos + rng.normal(0, 0.05, pos.shape)
    species = rng.integers(0, 4, len(pos)).astype(np.int32)
    L = 2
    g = O.neighbor_list(pos, cell, spec.r_cut)
    E, E_i, F = O.energy_forces(m, L, pos, cell, species, g)
    parts = O.partition_grid(pos, cell, grid, L * spec.r_cut)
    owned_all = np.concatenate([p[0] for p in parts])
    assert np.array_equal(np.sort(owned_all), np.arange(len(pos)))  # each atom owned exactly once
    Ep, Eip, Fp, stats = O.energy_forces_partitioned(m, L, pos, cell, species, parts, g)
    assert abs(Ep - E) < 1e-12 * np.abs(E_i).sum()
    assert np.allclose(Eip, E_i, rtol=0, atol=1e-12)
    assert np.abs(Fp - F).max() < 1e-12 * rms(F)
    if grid == (3, 1, 1):
        assert max(s["n_ext"] for s in stats) < len(pos)  # the halo does not cover the box
        # negative control: halo (L-1) r_cut is too small and visibly breaks forces and energy
        bad = O.partition_grid(pos, cell, grid, (L - 1) * spec.r_cut)
        Eb, _, Fb, _ = O.energy_forces_partitioned(m, L, pos, cell, species, bad, g)
        assert np.abs(Fb - F).max() > 1e-4 * rms(F)
        assert abs(Eb - E) > 1e-7 * np.abs(E_i).sum()
        # owned-only forces (north_star wording, reading R1) would be wrong at any halo
        Fo = np.zeros_like(F)
        for owned, ext in parts:
            lg = O.induced_subgraph(g, ext, len(pos))
            om = np.isin(ext, owned).astype(float)
            Fs = O.energy_forces(m, L, pos[ext], cell, species[ext], lg, om)[2]
            Fo[owned] += Fs[om > 0]
        assert np.abs(Fo - F).max() > 1e-2 * rms(F)


def test_halo_growth_factor_uniform_box():
    """H = halo atoms / root atoms; uniform density => (w + 2 halo)/w - 1."""
    sites, cell = fcc_box(10, 3.6)
    parts = O.partition_slabs(sites + 0.01, cell, 2, 3.6 * 1.0)
    H = O.halo_growth_factor(parts)
    assert np.allclose(H, (18.0 + 2 * 3.6) / 18.0 - 1.0, atol=0.06)
    assert O.slab_axis(np.diag([10.0, 30.0, 20.0])) == 1 and O.slab_axis(np.eye(3) * 5) == 0


# ---------------------------------------------------------------- dynamics
def test_nve_energy_error_is_second_order():
    spec, blob, m = make_model(d=8, r_cut=4.0, nbar=20.0)
    s = small_system(2, 0.05, seed=13)
    masses = np.full(len(s.pos), 20.0)
    vel = np.random.default_rng(5).normal(0, 0.004, s.pos.shape)
    vel -= vel.mean(0)
    e1 = O.nve_velocity_verlet(m, 2, s.pos, s.cell, s.species, masses, vel, 4.0, 20)
    e2 = O.nve_velocity_verlet(m, 2, s.pos, s.cell, s.species, masses, vel, 2.0, 40)
    f1 = np.abs(e1 - e1[0]).max(); f2 = np.abs(e2 - e2[0]).max()
    assert f1 > 0 and 2.5 < f1 / f2 < 6.0


# ---------------------------------------------------------------- per-layer active sets
@pytest.mark.parametrize("grid,L", [((4, 1, 1), 3), ((2, 2, 1), 2), ((1, 1, 3), 2)])
def test_depth_class_never_exceeds_khop_distance(grid, L):
    """The geometric depth class must be a LOWER bound of the breadth-first hop distance to the root
    atoms (PAPER.md:165 Stage 2), otherwise an atom a root energy depends on through layer l could
    be left out of that layer's active set. Pinned against a plain BFS over the radius graph."""
    r_cut = 3.0
    s = small_system(12 if max(grid) == 4 else 8, 0.08, seed=17)   # 43.2 / 28.8 A box
    g = O.neighbor_list(s.pos, s.cell, r_cut)
    halo = L * r_cut
    parts = O.partition_grid(s.pos, s.cell, grid, halo)
    classes = O.halo_depth_classes(s.pos, s.cell, grid, halo, r_cut)
    some_halo_shell_is_populated = False
    for (owned, ext), cls in zip(parts, classes):
        hops = O.khop_distance(g, owned, len(s.pos), L + 2)[ext]
        assert np.array_equal(cls == 0, np.isin(ext, owned))
        assert np.all(cls <= hops)                    # class k  =>  at least k hops away
        assert cls.max() <= L
        # every edge changes the class by at most one (what makes the per-layer sets prefixes)
        lr, ls, _ = O.induced_subgraph(g, ext, len(s.pos))
        assert np.all(np.abs(cls[lr] - cls[ls]) <= 1)
        some_halo_shell_is_populated |= bool(np.any(cls == L))
        # the K-hop set of the paper is inside the geometric halo (reading R2)
        assert np.all(np.isin(np.nonzero(O.khop_distance(g, owned, len(s.pos), L) <= L)[0], ext))
    assert some_halo_shell_is_populated


def test_outermost_shell_never_receives():
    """With halo = L r_cut the atoms of class L only ever act as senders of layer 0: deleting every edge
    they RECEIVE leaves the root energies and the gradient of their sum unchanged (to rounding), while
    deleting the edges they SEND does not."""
    spec, blob, m = make_model(r_cut=3.7, nbar=18.0)   # second fcc shell (a = 3.6) is inside: a hop spans ~r_cut
    L = 2
    s = small_system(8, 0.08, seed=23)
    g = O.neighbor_list(s.pos, s.cell, spec.r_cut)
    grid = (3, 1, 1)
    parts = O.partition_grid(s.pos, s.cell, grid, L * spec.r_cut)
    classes = O.halo_depth_classes(s.pos, s.cell, grid, L * spec.r_cut, spec.r_cut)
    owned, ext = parts[1]
    cls = classes[1]
    lr, ls, lsh = O.induced_subgraph(g, ext, len(s.pos))
    om = (cls == 0).astype(float)
    E0, Ei0, F0 = O.energy_forces(m, L, s.pos[ext], s.cell, s.species[ext], (lr, ls, lsh), om)
    keep = cls[lr] < L
    assert 0 < keep.sum() < len(lr)
    E1, Ei1, F1 = O.energy_forces(m, L, s.pos[ext], s.cell, s.species[ext], (lr[keep], ls[keep], lsh[keep]), om)
    assert abs(E1 - E0) <= 1e-12 * np.abs(Ei0[om > 0]).sum()
    assert np.abs(F1 - F0).max() <= 1e-12 * rms(F0)
    keep2 = cls[ls] < L
    E2, _, F2 = O.energy_forces(m, L, s.pos[ext], s.cell, s.species[ext], (lr[keep2], ls[keep2], lsh[keep2]), om)
    assert np.abs(F2 - F0).max() > 1e-6 * rms(F0)


@pytest.mark.parametrize("grid", [(3, 1, 1), (2, 2, 1)])
def test_khop_partition_equals_unpartitioned(grid):
    """PAPER.md:165 as stated: extending every bin by the K-hop neighbourhood of its root atoms (K = number
    of layers kept) reproduces the unpartitioned energies and forces; K-1 hops do not. The K-hop set is
    a subset of the geometric box and, on this lattice (a hop advances < r_cut along an axis), a proper one."""
    spec, blob, m = make_model(r_cut=3.0, nbar=12.0)
    L = 2
    s = small_system(8, 0.08, seed=29)
    g = O.neighbor_list(s.pos, s.cell, spec.r_cut)
    E, E_i, F = O.energy_forces(m, L, s.pos, s.cell, s.species, g)
    kh = O.partition_grid_khop(s.pos, s.cell, grid, L * spec.r_cut, spec.r_cut, g)
    geo = O.partition_grid(s.pos, s.cell, grid, L * spec.r_cut)
    assert all(np.all(np.isin(ext, gext)) for (_, ext, _), (_, gext) in zip(kh, geo))
    assert sum(len(p[1]) for p in kh) < sum(len(p[1]) for p in geo)
    assert all(h.max() == L and np.array_equal(h == 0, np.isin(ext, owned)) for owned, ext, h in kh)
    Ep, Eip, Fp, _ = O.energy_forces_partitioned(m, L, s.pos, s.cell, s.species, [(o, e) for o, e, _ in kh], g)
    assert abs(Ep - E) < 1e-12 * np.abs(E_i).sum()
    assert np.allclose(Eip, E_i, rtol=0, atol=1e-12)
    assert np.abs(Fp - F).max() < 1e-12 * rms(F)
    bad = [(o, e[h <= L - 1]) for o, e, h in kh]
    Eb, _, Fb, _ = O.energy_forces_partitioned(m, L, s.pos, s.cell, s.species, bad, g)
    assert np.abs(Fb - F).max() > 1e-4 * rms(F)


# ---------------------------------------------------------------- stress
def test_stress_equals_strain_finite_difference_and_is_symmetric():
    """sigma_ab = (1/V) dE/d eps_ab, pinned by central differences of E under the homogeneous strain
    x -> (1 + eps) x, C -> C (1 + eps)^T with the edge list (and its image shifts) held fixed."""
    spec, blob, m = make_model(d=8, r_cut=4.0, nbar=20.0)
    s = small_system(2, 0.15, seed=19)
    g = O.neighbor_list(s.pos, s.cell, spec.r_cut)
    E, E_i, F, sig = O.energy_forces_stress(m, 2, s.pos, s.cell, s.species, g)
    assert np.allclose(sig, sig.T, rtol=0, atol=1e-14 * np.abs(sig).max())
    V = abs(np.linalg.det(s.cell))
    h = 1e-6
    fd = np.zeros((3, 3))
    for a in range(3):
        for b in range(3):
            eps = np.zeros((3, 3)); eps[a, b] = h
            Ep = O.energy_forces(m, 2, s.pos @ (np.eye(3) + eps).T, s.cell @ (np.eye(3) + eps).T, s.species, g)[0]
            Em = O.energy_forces(m, 2, s.pos @ (np.eye(3) - eps).T, s.cell @ (np.eye(3) - eps).T, s.species, g)[0]
            fd[a, b] = (Ep - Em) / (2 * h) / V
    assert np.abs(fd - sig).max() < 1e-6 * np.abs(sig).max()
    # rigid rotation costs no energy: the antisymmetric part of dE/d eps vanishes
    assert np.abs(fd - fd.T).max() < 1e-6 * np.abs(sig).max()


def test_stress_dimer_closed_form_and_cubic_lattice_isotropy():
    spec, blob, m = make_model(d=8, r_cut=4.0, nbar=20.0)
    # dimer along x: two directed edges, sigma_xx = 2 rbar r / V, everything else zero
    cell = np.diag([30.0, 30.0, 30.0])
    pos = np.array([[5.0, 5.0, 5.0], [7.5, 5.0, 5.0]])
    sp = np.array([0, 1], np.int32)
    E, E_i, F, ex = O.energy_forces(m, 2, pos, cell, sp, return_extra=True)
    sig = O.stress_from_rbar(cell, ex["rvec"], ex["r"], ex["rbar"])
    assert len(ex["r"]) == 2
    expect = np.zeros((3, 3)); expect[0, 0] = float(np.sum(ex["rbar"]) * 2.5 / 27000.0)
    assert np.allclose(sig, expect, rtol=1e-12, atol=1e-18)
    # virial theorem for a pair: sigma_xx V = -F_x(atom 1) * (x_1 - x_0)
    assert np.isclose(sig[0, 0] * 27000.0, -F[1, 0] * 2.5, rtol=1e-10)
    # perfect single-species fcc: cubic symmetry => isotropic stress
    sites, cell = fcc_box(3, 3.6)
    sig = O.energy_forces_stress(m, 2, sites, cell, np.zeros(len(sites), np.int32))[3]
    assert np.abs(sig - np.eye(3) * sig[0, 0]).max() < 1e-12 * abs(sig[0, 0])


def test_stress_partitioned_equals_unpartitioned():
    spec, blob, m = make_model(r_cut=3.0, nbar=12.0)
    L = 2
    s = small_system(8, 0.08, seed=33)
    g = O.neighbor_list(s.pos, s.cell, spec.r_cut)
    sig = O.energy_forces_stress(m, L, s.pos, s.cell, s.species, g)[3]
    for parts in (O.partition_grid(s.pos, s.cell, (3, 1, 1), L * spec.r_cut),
                  [(o, e) for o, e, _ in O.partition_grid_khop(s.pos, s.cell, (2, 2, 1), L * spec.r_cut, spec.r_cut, g)]):
        sp_ = O.stress_partitioned(m, L, s.pos, s.cell, s.species, parts, g)
        assert np.abs(sp_ - sig).max() < 1e-12 * np.abs(sig).max()
