"""Pins for the oracle's three-body (angle) variant O7 (BASELINE.json config 5; the paper names
the model family -- MatterSim, an M3GNet-type network, PAPER.md:91,119,131 -- but gives no equations, reading R17):
textbook values of the angle basis, a brute-force triplet loop on tiny inputs, the two-body limit W3 = 0, finite
differences, an independently written torch.float64 autograd restatement, invariances (incl. rotation: the term depends on
directions), C1 continuity at the three-body cutoff, partition equality with halo L r_cut, strain finite differences."""
import numpy as np
import pytest
import torch

from oracle import mlip_oracle as O
from synth_inputs import ModelSpec, fcc_box, make_config, make_weights, small_system, make_water_system


def rms(x):
    return float(np.sqrt(np.mean(np.square(x))))


def make_model(d=16, n_rbf=8, L_max=2, r_cut=5.0, r_cut3=4.0, n_species=2, seed=21, nbar=43.0):
    spec = ModelSpec(n_species, d, n_rbf, L_max, r_cut, 1.0 / np.sqrt(nbar), r_cut3=r_cut3)
    blob = make_weights(spec, seed)
    return spec, blob, O.parse_weights(n_species, d, n_rbf, L_max, r_cut, spec.agg_scale, blob, r_cut3=r_cut3)


def water_box(n_grid=3, seed=0):
    """27 molecules of the config-5 recipe (jittered cubic O grid, random orientations)."""
    return make_water_system(n_grid, seed_pos=1005 + seed, seed_orient=3005 + seed)


# ---------------------------------------------------------------- basis functions
def test_angle_basis_textbook_values():
    c = np.array([1.0, 0.0, -1.0, 0.3])
    Y, dY = O.y_l0(c)
    # Y_l^0(theta = 0) = sqrt((2l+1)/4pi); Y_2^0(pi/2) = -1/2 sqrt(5/4pi); parity (-1)^l
    assert np.allclose(Y[0], np.sqrt((2 * np.arange(4) + 1) / (4 * np.pi)), rtol=1e-15)
    assert np.allclose(Y[0], [0.28209479177387814, 0.4886025119029199, 0.6307831305050401, 0.7463526651802308])
    assert abs(Y[1, 2] + 0.5 * 0.6307831305050401) < 1e-15 and abs(Y[1, 1]) < 1e-16 and abs(Y[1, 3]) < 1e-16
    assert np.allclose(Y[2], Y[0] * np.array([1, -1, 1, -1]))
    # orthonormality on the sphere: 2 pi int_{-1}^{1} Y_l Y_l' dc = delta (Gauss-Legendre, exact for degree <= 6)
    x, w = np.polynomial.legendre.leggauss(8)
    Yq, _ = O.y_l0(x)
    assert np.allclose(2 * np.pi * (Yq * w[:, None]).T @ Yq, np.eye(4), atol=1e-14)
    h = 1e-6
    assert np.allclose((O.y_l0(c + h)[0] - O.y_l0(c - h)[0]) / (2 * h), dY, atol=1e-9)
    r3 = 4.0
    u, du = O.envelope3(np.array([0.0, 2.0, r3, 4.5]), r3)
    assert u[0] == 1.0 and abs(u[1] - 0.5) < 1e-16 and u[2] == 0.0 and u[3] == 0.0 and du[2] == 0.0 and du[3] == 0.0
    g, dg = O.rbf3(np.arange(4) * r3 / 3, r3)
    assert np.allclose(np.diag(g), 1.0) and np.allclose(np.diag(g, 1), np.exp(-0.5)) and np.allclose(np.diag(dg), 0.0)
    r = np.linspace(0.4, 3.9, 8)
    assert np.allclose((O.envelope3(r + h, r3)[0] - O.envelope3(r - h, r3)[0]) / (2 * h), O.envelope3(r, r3)[1], atol=1e-9)
    assert np.allclose((O.rbf3(r + h, r3)[0] - O.rbf3(r - h, r3)[0]) / (2 * h), O.rbf3(r, r3)[1], atol=1e-8)


def test_triplet_enumeration_counts():
    """Perfect fcc, a = 3.6, r3 = 3: 12 first-shell neighbours -> 12 * 11 ordered pairs per atom; the pairs of a
    receiver never contain e == e'; a neighbour seen through two images counts as two edges."""
    sites, cell = fcc_box(3, 3.6)
    recv, send, shift = O.neighbor_list(sites, cell, 5.0)
    _, r = O.edge_vectors(sites, cell, recv, send, shift)
    te, tp = map(np.concatenate, zip(*O.triplet_chunks(recv, r < 3.0, len(sites))))
    assert len(te) == len(sites) * 12 * 11
    assert np.all(recv[te] == recv[tp]) and np.all(te != tp) and np.all(r[te] < 3.0) and np.all(r[tp] < 3.0)
    assert len(np.unique(te * len(recv) + tp)) == len(te)
    # small chunks give the same set
    old = O.TRIPLET_CHUNK
    try:
        O.TRIPLET_CHUNK = 500
        te2, tp2 = map(np.concatenate, zip(*O.triplet_chunks(recv, r < 3.0, len(sites))))
    finally:
        O.TRIPLET_CHUNK = old
    assert np.array_equal(np.sort(te * len(recv) + tp), np.sort(te2 * len(recv) + tp2))
    # one atom in a box smaller than r3: its own images are distinct edges and pair with each other
    p = np.array([[0.1, 0.2, 0.3]]); c1 = np.eye(3) * 2.5
    g1 = O.neighbor_list(p, c1, 3.0)
    _, r1 = O.edge_vectors(p, c1, *g1)
    n_short = int((r1 < 2.9).sum())
    assert n_short == 6 and sum(len(a) for a, _ in O.triplet_chunks(g1[0], r1 < 2.9, 1)) == 6 * 5


def _brute_force_t(model, lay, h, pos, cell, graph):
    """t_e by plain Python loops over receivers and ordered neighbour pairs (tiny inputs only)."""
    recv, send, shift = graph
    rvec, r = O.edge_vectors(pos, cell, recv, send, shift)
    r3 = model.r_cut3
    t = np.zeros((len(recv), 16))
    for e in range(len(recv)):
        if r[e] >= r3:
            continue
        for p in range(len(recv)):
            if p == e or recv[p] != recv[e] or r[p] >= r3:
                continue
            c = float(np.dot(rvec[e], rvec[p]) / (r[e] * r[p]))
            P = [1.0, c, 0.5 * (3 * c * c - 1), 0.5 * (5 * c ** 3 - 3 * c)]
            zk = 1.0 / (1.0 + np.exp(-(lay["G"] @ h[send[p]] + lay["g"])))
            up = 0.5 * (np.cos(np.pi * r[p] / r3) + 1)
            for l in range(4):
                for n in range(4):
                    gn = np.exp(-0.5 * ((r[p] - n * r3 / 3) / (r3 / 3)) ** 2)
                    t[e, 4 * l + n] += up * np.sqrt((2 * l + 1) / (4 * np.pi)) * P[l] * gn * zk[4 * l + n]
        t[e] *= 0.5 * (np.cos(np.pi * r[e] / r3) + 1)
    return t


def test_three_body_terms_against_brute_force_loops():
    spec, blob, m = make_model()
    s = water_box(2)   # 24 atoms, box 6.2 A < 2 r_cut: multiple images
    g = O.neighbor_list(s.pos, s.cell, spec.r_cut)
    rvec, r = O.edge_vectors(s.pos, s.cell, *g)
    h = m.T[s.species] + 0.1 * np.random.default_rng(0).normal(size=(len(s.pos), spec.d))
    t, S, z = O.three_body_terms(m, m.layers[0], h, g[0], g[1], rvec, r)
    t_ref = _brute_force_t(m, m.layers[0], h, s.pos, s.cell, g)
    assert np.abs(t_ref).max() > 0.05 and np.allclose(t, t_ref, rtol=1e-12, atol=1e-14)
    assert np.all(t[r >= spec.r_cut3] == 0.0)


def test_W3_zero_is_the_two_body_model_bit_for_bit():
    spec, blob, m = make_model(L_max=2)
    s = water_box(3)
    for lay in m.layers:
        lay["W3"] = np.zeros_like(lay["W3"])
    # the two-body model with the same remaining weights
    spec2 = ModelSpec(spec.n_species, spec.d, spec.n_rbf, spec.L_max, spec.r_cut, spec.agg_scale)
    d, k, S = spec.d, spec.n_rbf, spec.n_species
    two = d * (2 * d + k) + d + d * d + d + 2 * d * d + d + d * d + d
    extra = 16 * d + 16 + 16 * d
    head = S * d + S
    parts = [blob[:head]] + [blob[head + l * (two + extra): head + l * (two + extra) + two] for l in range(spec.L_max)]
    parts.append(blob[head + spec.L_max * (two + extra):])
    m2 = O.parse_weights(S, d, k, spec.L_max, spec.r_cut, spec.agg_scale, np.concatenate(parts))
    a = O.energy_forces(m, 2, s.pos, s.cell, s.species)
    b = O.energy_forces(m2, 2, s.pos, s.cell, s.species)
    assert a[0] == b[0] and np.array_equal(a[1], b[1]) and np.array_equal(a[2], b[2])
    # and with W3 != 0 the angle term matters
    spec, blob, m = make_model(L_max=2)
    c = O.energy_forces(m, 2, s.pos, s.cell, s.species)
    assert abs(c[0] - b[0]) > 1e-3 and rms(c[2] - b[2]) > 1e-2 * rms(b[2])


def test_three_body_forces_finite_differences():
    spec, blob, m = make_model()
    s = water_box(3)
    E, _, F = O.energy_forces(m, 2, s.pos, s.cell, s.species)
    h = 1e-4
    rng = np.random.default_rng(3)
    for k, a in zip(rng.integers(0, len(s.pos), 10), rng.integers(0, 3, 10)):
        p = s.pos.copy(); p[k, a] += h; Ep = O.energy_forces(m, 2, p, s.cell, s.species)[0]
        p[k, a] -= 2 * h; Em = O.energy_forces(m, 2, p, s.cell, s.species)[0]
        assert abs(-(Ep - Em) / (2 * h) - F[k, a]) < 1e-6 * rms(F)


def _torch_energy_three_body(blob, spec, L, pos, cell, species, recv, send, shift, omega=None):
    """Independent restatement in torch.float64 (autograd forces): its own blob unpacking, its own triplet list from
    plain loops, its own basis."""
    w = torch.tensor(blob, dtype=torch.float64)
    S, d, k, r3 = spec.n_species, spec.d, spec.n_rbf, spec.r_cut3
    off = 0

    def take(*shape):
        nonlocal off
        n = int(np.prod(shape)); t = w[off:off + n].reshape(shape); off += n
        return t

    T = take(S, d); E0 = take(S)
    layers = [[take(d, 2 * d + k), take(d), take(d, d), take(d), take(d, 2 * d), take(d), take(d, d), take(d),
               take(16, d), take(16), take(d, 16)] for _ in range(spec.L_max)]
    Wo = take(d, d); bo = take(d); wo = take(d); bE = take(1)
    assert off == len(w)
    x = torch.tensor(pos, dtype=torch.float64, requires_grad=True)
    C = torch.tensor(cell, dtype=torch.float64)
    ri = torch.tensor(recv, dtype=torch.long); si = torch.tensor(send, dtype=torch.long)
    z = torch.tensor(species, dtype=torch.long)
    rv = x[si] - x[ri] + torch.tensor(shift, dtype=torch.float64) @ C
    r = rv.norm(dim=1)
    rn = r.detach().numpy()
    by_recv = {}
    for e in range(len(recv)):
        if rn[e] < r3:
            by_recv.setdefault(int(recv[e]), []).append(e)
    te = [e for es in by_recv.values() for e in es for p in es if p != e]
    tp = [p for es in by_recv.values() for e in es for p in es if p != e]
    te = torch.tensor(te, dtype=torch.long); tp = torch.tensor(tp, dtype=torch.long)
    u = 0.5 * (torch.cos(torch.pi * r / spec.r_cut) + 1)
    delta = spec.r_cut / (k - 1)
    g = torch.exp(-(r[:, None] - torch.arange(k, dtype=torch.float64) * delta) ** 2 / (2 * delta ** 2))
    u3 = torch.where(r < r3, 0.5 * (torch.cos(torch.pi * r / r3) + 1), torch.zeros_like(r))
    cosang = (rv[te] * rv[tp]).sum(1) / (r[te] * r[tp])
    leg = torch.stack([torch.ones_like(cosang), cosang, 1.5 * cosang ** 2 - 0.5, 2.5 * cosang ** 3 - 1.5 * cosang], 1)
    leg = leg * torch.sqrt((2 * torch.arange(4, dtype=torch.float64) + 1) / (4 * torch.pi))
    g3 = torch.exp(-(r[tp][:, None] - torch.arange(4, dtype=torch.float64) * r3 / 3) ** 2 / (2 * (r3 / 3) ** 2))
    basis = (leg[:, :, None] * g3[:, None, :]).reshape(-1, 16)      # index 4 l + n
    h = T[z]
    act = torch.nn.functional.silu
    for W1, b1, W2, b2, V1, c1, V2, c2, G, gb, W3 in layers[:L]:
        gate = torch.sigmoid(h @ G.T + gb)
        t = torch.zeros(len(recv), 16, dtype=torch.float64).index_add(0, te, u3[tp][:, None] * basis * gate[si[tp]])
        t = u3[:, None] * t
        a = torch.cat([h[ri], h[si], u[:, None] * g], 1) @ W1.T + b1 + t @ W3.T
        phi = act(act(a) @ W2.T + b2)
        mm = torch.zeros_like(h).index_add(0, ri, spec.agg_scale * u[:, None] * phi)
        h = h + act(torch.cat([h, mm], 1) @ V1.T + c1) @ V2.T + c2
    E_i = act(h @ Wo.T + bo) @ wo + bE + E0[z]
    om = torch.ones_like(E_i) if omega is None else torch.tensor(omega, dtype=torch.float64)
    E = (om * E_i).sum()
    E.backward()
    return E.item(), E_i.detach().numpy(), -x.grad.numpy()


def test_three_body_against_torch_autograd():
    spec, blob, m = make_model(L_max=3)
    s = water_box(3)
    g = O.neighbor_list(s.pos, s.cell, spec.r_cut)
    E, E_i, F = O.energy_forces(m, 3, s.pos, s.cell, s.species, g)
    Et, Eit, Ft = _torch_energy_three_body(blob, spec, 3, s.pos, s.cell, s.species, *g)
    assert abs(E - Et) < 1e-11 * np.abs(E_i).sum()
    assert np.allclose(E_i, Eit, rtol=0, atol=1e-11)
    assert np.abs(F - Ft).max() < 1e-11 * max(rms(F), 1e-3)
    om = (np.arange(len(s.pos)) % 3 == 0).astype(float)
    Ew, _, Fw = O.energy_forces(m, 3, s.pos, s.cell, s.species, g, omega=om)
    Etw, _, Ftw = _torch_energy_three_body(blob, spec, 3, s.pos, s.cell, s.species, *g, omega=om)
    assert abs(Ew - Etw) < 1e-10 and np.abs(Fw - Ftw).max() < 1e-11 * max(rms(Fw), 1e-3)


def test_three_body_invariances_and_zero_total_force():
    spec, blob, m = make_model()
    s = water_box(3)
    E, E_i, F = O.energy_forces(m, 2, s.pos, s.cell, s.species)
    assert np.abs(F.sum(0)).max() < 1e-12
    Et, _, Ft = O.energy_forces(m, 2, s.pos + np.array([0.37, -1.2, 5.5]), s.cell, s.species)
    assert abs(Et - E) < 1e-10 and np.allclose(Ft, F, atol=1e-11)
    q, _ = np.linalg.qr(np.random.default_rng(0).normal(size=(3, 3)))
    q *= np.sign(np.linalg.det(q))
    Er, _, Fr = O.energy_forces(m, 2, s.pos @ q.T, s.cell @ q.T, s.species)
    assert abs(Er - E) < 1e-10 and np.allclose(Fr, F @ q.T, atol=1e-11)
    perm = np.random.default_rng(1).permutation(len(s.pos))
    Ep, Eip, Fp = O.energy_forces(m, 2, s.pos[perm], s.cell, s.species[perm])
    assert abs(Ep - E) < 1e-10 and np.allclose(Fp, F[perm], atol=1e-11) and np.allclose(Eip, E_i[perm], atol=1e-11)


def test_three_body_energy_is_C1_at_the_three_body_cutoff():
    """Trimer: atom 2 moves through r3 from atom 0 while atom 1 stays inside: value and slope of the angle term vanish at
    r3 (both envelopes), so E has no kink there."""
    spec, blob, m = make_model(L_max=1)
    cell = np.eye(3) * 40.0
    species = np.array([0, 1, 1])

    def E(x):
        return O.energy_forces(m, 1, np.array([[10.0, 10, 10], [10.9, 10.3, 10], [10.0 + x, 10, 10.0]]), cell, species)[0]

    r3, eps = spec.r_cut3, 1e-3
    slope_in = (E(r3 - eps) - E(r3 - 2 * eps)) / eps
    slope_out = (E(r3 + 2 * eps) - E(r3 + eps)) / eps
    assert abs(slope_in - slope_out) < 20 * eps * max(1.0, abs(slope_in))
    assert abs(E(r3 - eps) + E(r3 + eps) - 2 * E(r3)) < 50 * eps ** 2
    # the angle term is live inside r3: moving atom 2 on a circle around atom 0 (|r| fixed) changes the energy
    def E_ang(th):
        return O.energy_forces(m, 1, np.array([[10.0, 10, 10], [10.9, 10.3, 10], [10 + 3 * np.cos(th), 10, 10 + 3 * np.sin(th)]]), cell, species)[0]
    spec0 = ModelSpec(spec.n_species, spec.d, spec.n_rbf, 1, spec.r_cut, spec.agg_scale, r_cut3=spec.r_cut3)
    assert abs(E_ang(0.3) - E_ang(1.9)) > 1e-5


@pytest.mark.parametrize("grid", [(2, 1, 1), (3, 1, 1), (1, 2, 2)])
def test_three_body_partitioned_equals_unpartitioned(grid):
    """r3 <= r_cut, so the halo stays L r_cut: the triplets of every atom that matters are complete."""
    spec, blob, m = make_model(r_cut=3.0, r_cut3=2.6, nbar=12.0)
    n = (10, 4, 4) if grid[0] > 1 else (4, 8, 8)
    idx = np.indices(n).reshape(3, -1).T.astype(float)
    basis = np.array([[0, 0, 0], [.5, .5, 0], [.5, 0, .5], [0, .5, .5]])
    rng = np.random.default_rng(31)
    pos = (idx[:, None, :] + basis[None]).reshape(-1, 3) * 3.6 + rng.normal(0, 0.08, (int(np.prod(n)) * 4, 3))
    cell = np.diag(np.array(n) * 3.6)
    species = rng.integers(0, 2, len(pos)).astype(np.int32)
    L = 2
    g = O.neighbor_list(pos, cell, spec.r_cut)
    E, E_i, F = O.energy_forces(m, L, pos, cell, species, g)
    parts = O.partition_grid(pos, cell, grid, L * spec.r_cut)
    Ep, Eip, Fp, _ = O.energy_forces_partitioned(m, L, pos, cell, species, parts, g)
    assert abs(Ep - E) < 1e-11 * np.abs(E_i).sum() and np.abs(Eip - E_i).max() < 1e-11
    assert np.abs(Fp - F).max() < 1e-11 * rms(F)
    kparts = [(o, e) for o, e, _ in O.partition_grid_khop(pos, cell, grid, L * spec.r_cut, spec.r_cut, g)]
    Ek, _, Fk, _ = O.energy_forces_partitioned(m, L, pos, cell, species, kparts, g)
    assert abs(Ek - E) < 1e-11 * np.abs(E_i).sum() and np.abs(Fk - F).max() < 1e-11 * rms(F)
    # negative control: a halo of (L-1) r_cut is not enough
    bad = O.partition_grid(pos, cell, grid, (L - 1) * spec.r_cut)
    Fb = O.energy_forces_partitioned(m, L, pos, cell, species, bad, g)[2]
    assert np.abs(Fb - F).max() > 1e-4 * rms(F)


def test_three_body_stress_equals_strain_finite_difference():
    spec, blob, m = make_model()
    s = water_box(3)
    E, _, F, sig = O.energy_forces_stress(m, 2, s.pos, s.cell, s.species)
    assert np.allclose(sig, sig.T, atol=1e-12 * np.abs(sig).max())
    V = abs(np.linalg.det(s.cell)); h = 1e-5
    for a, b in [(0, 0), (1, 2), (2, 0), (1, 1)]:
        eps = np.zeros((3, 3)); eps[a, b] += 0.5 * h; eps[b, a] += 0.5 * h
        Ep = O.energy_forces(m, 2, s.pos @ (np.eye(3) + eps).T, s.cell @ (np.eye(3) + eps).T, s.species)[0]
        Em = O.energy_forces(m, 2, s.pos @ (np.eye(3) - eps).T, s.cell @ (np.eye(3) - eps).T, s.species)[0]
        assert abs((Ep - Em) / (2 * h) / V - sig[a, b]) < 1e-6 * np.abs(sig).max()


def test_config5_recipe_statistics():
    """98,304 atoms, 5.26 M directed edges at 5 A, 2.55 M at 4 A, 63.9 M ordered triplets."""
    cfg = make_config(5, with_weights=False)
    s = cfg.system
    assert len(s.pos) == 98304 and cfg.model.r_cut3 == 4.0 and cfg.grid == (4, 1, 1) and cfg.halo == 20.0
    recv, send, shift = O.neighbor_list(s.pos, s.cell, 5.0)
    _, r = O.edge_vectors(s.pos, s.cell, recv, send, shift)
    m = np.bincount(recv[r < 4.0], minlength=len(s.pos)).astype(np.int64)
    assert abs(len(recv) - 5.26e6) < 0.03e6 and abs((r < 4.0).sum() - 2.55e6) < 0.03e6
    assert abs((m * (m - 1)).sum() - 63.9e6) < 0.6e6
    assert r.min() > 0.7
