"""float64 CPU ORACLE for the energy-and-force hot path (TEST INFRASTRUCTURE ONLY).

Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s cpu_baseline / `--impl reference`
legs may import this module. It shares no code with `paper_2509_21694_b200/` and never
imports it. It is deliberately plain and slow: NumPy float64, no blocking, fusion or
re-ordering beyond what the definitions below state (edges are only processed in chunks
to bound memory; a chunk boundary changes nothing but the order of independent rows).

What it computes (citations are PAPER.md lines; O1..O6 / R1..R19 are the readings listed
in DESIGN.md, taken from SURVEY.md 8(c), because the paper treats the network as a black
box):

  O1  radius graph under periodic boundaries with local cutoff r_c
  O2  Gaussian RBF x cosine envelope edge features                       BASELINE.json configs
  O3  L message-passing layers, first L of L_max kept (MPDP)
  O4  per-atom energy readout, E = sum_i E_i
  O5  forces F = -grad E (hand-derived reverse mode)
  O6  partition into spatial bins + halo; sum ROOT-node energies, sum the
      gradients of root energies w.r.t. ALL sub-graph atoms

  O7  three-body (angle) variant of the layers, BASELINE.json config 5: the paper's workhorse model MatterSim is an
      M3GNet-type network but the paper gives no equations; the definition is the proposal of
      SURVEY.md 8(f) NEXT-1 (reading R17), written out at `three_body_terms`.

The method (prune + partition + halo) reaches exactly the unpartitioned result
(PAPER.md:165), so `energy_forces` IS the definition and `energy_forces_partitioned`
restates the assembly rule. Pins (tests/test_oracle_*.py): brute-force O(N^2) neighbour
lists, fcc shell counts, scipy cKDTree, finite differences, torch.float64 autograd,
L=0 closed form, dimer closed form, invariances, partition equality + negative control,
NVE energy conservation order. Nothing here is "parity unpinned".
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np
import scipy.sparse as sp
from scipy.spatial import cKDTree
from scipy.special import expit

EDGE_CHUNK = 1 << 18


# --------------------------------------------------------------------------------------
# weights
# --------------------------------------------------------------------------------------
@dataclass
class Model:
    n_species: int
    d: int
    n_rbf: int
    L_max: int
    r_cut: float
    agg_scale: float
    T: np.ndarray
    E0: np.ndarray
    layers: list  # dicts W1,b1,W2,b2,V1,c1,V2,c2
    Wo: np.ndarray
    bo: np.ndarray
    wo: np.ndarray
    bE: float
    r_cut3: float = 0.0   # > 0: three-body variant (O7); layers then also hold G[16,d], g[16], W3[d,16]


N_ANGLE = 16  # (l_max + 1) * n_rbf3 = 4 * 4 angle-basis functions of the three-body variant, index 4 l + n


def parse_weights(n_species, d, n_rbf, L_max, r_cut, agg_scale, blob, r_cut3=0.0) -> Model:
    """Blob order of include/mlip.h: T[S,d], E0[S], per layer W1[d,2d+k] (columns: receiver h_i,
    sender h_j, e_hat), b1, W2[d,d], b2, V1[d,2d] (columns: h, m), c1, V2[d,d], c2 (and, three-body variant
    r_cut3 > 0, G[16,d], g[16], W3[d,16]); then Wo[d,d], bo, wo, b_E. fp32 values are promoted to float64
    unrounded (reading R15)."""
    w = np.asarray(blob, dtype=np.float64)
    pos = 0

    def take(*shape):
        nonlocal pos
        n = int(np.prod(shape))
        out = w[pos:pos + n].reshape(shape)
        pos += n
        return out

    T = take(n_species, d)
    E0 = take(n_species)
    layers = []
    for _ in range(L_max):
        layers.append(dict(W1=take(d, 2 * d + n_rbf), b1=take(d), W2=take(d, d), b2=take(d),
                           V1=take(d, 2 * d), c1=take(d), V2=take(d, d), c2=take(d)))
        if r_cut3 > 0.0:
            layers[-1].update(G=take(N_ANGLE, d), g=take(N_ANGLE), W3=take(d, N_ANGLE))
    Wo = take(d, d); bo = take(d); wo = take(d); bE = float(take(1)[0])
    assert pos == w.size, "weight blob size does not match the header"
    assert 0.0 <= r_cut3 <= r_cut, "three-body cutoff must not exceed the two-body one (halo stays L r_cut)"
    return Model(n_species, d, n_rbf, L_max, float(r_cut), float(agg_scale), T, E0, layers, Wo, bo, wo, bE, float(r_cut3))


# --------------------------------------------------------------------------------------
# O1 graph
# --------------------------------------------------------------------------------------
def perpendicular_widths(cell):
    """w_k = V / |a_i x a_j|: distance between the two faces of the cell normal to axis k."""
    a1, a2, a3 = cell
    vol = abs(np.dot(a1, np.cross(a2, a3)))
    return np.array([vol / np.linalg.norm(np.cross(a2, a3)),
                     vol / np.linalg.norm(np.cross(a3, a1)),
                     vol / np.linalg.norm(np.cross(a1, a2))])


def _canonical_d2(pos, cell, i, j, n):
    """d^2 of the canonical predicate, in this operation order (reading R10):
    t = (nx*a1 + ny*a2) + nz*a3 ; r = (x_j - x_i) + t ; d2 = (rx*rx + ry*ry) + rz*rz."""
    nf = n.astype(np.float64)
    t = (nf[:, 0:1] * cell[0][None, :] + nf[:, 1:2] * cell[1][None, :]) + nf[:, 2:3] * cell[2][None, :]
    r = (pos[j] - pos[i]) + t
    d2 = (r[:, 0] * r[:, 0] + r[:, 1] * r[:, 1]) + r[:, 2] * r[:, 2]
    return r, d2


def _canonical_sort(i, j, n):
    order = np.lexsort((n[:, 2], n[:, 1], n[:, 0], j, i))
    return i[order].astype(np.int32), j[order].astype(np.int32), n[order].astype(np.int32)


def neighbor_list_bruteforce(pos, cell, r_cut):
    """All directed edges (i <- j, n): d2 < r_cut^2 (strict), not (i == j and n == 0).
    O(N^2 * images). Positions are used as given (unwrapped), n is relative to them."""
    pos = np.asarray(pos, np.float64); cell = np.asarray(cell, np.float64)
    N = len(pos)
    wk = perpendicular_widths(cell)
    frac = pos @ np.linalg.inv(cell)
    spread = np.ceil(frac.max(0) - frac.min(0)).astype(int) + 1 if N else np.zeros(3, int)
    R = np.ceil(r_cut / wk).astype(int) + spread
    ii, jj = np.meshgrid(np.arange(N), np.arange(N), indexing="ij")
    ii = ii.ravel(); jj = jj.ravel()
    out_i, out_j, out_n = [], [], []
    rc2 = r_cut * r_cut
    for nx in range(-R[0], R[0] + 1):
        for ny in range(-R[1], R[1] + 1):
            for nz in range(-R[2], R[2] + 1):
                n = np.broadcast_to(np.array([nx, ny, nz]), (len(ii), 3))
                _, d2 = _canonical_d2(pos, cell, ii, jj, n)
                keep = d2 < rc2
                if nx == 0 and ny == 0 and nz == 0:
                    keep &= ii != jj
                out_i.append(ii[keep]); out_j.append(jj[keep]); out_n.append(n[keep])
    if not out_i:
        return (np.zeros(0, np.int32),) * 2 + (np.zeros((0, 3), np.int32),)
    return _canonical_sort(np.concatenate(out_i), np.concatenate(out_j), np.concatenate(out_n))


def neighbor_list(pos, cell, r_cut):
    """Same edge set as `neighbor_list_bruteforce`, found by a spatial search.

    Candidates: wrap atoms into the cell, add every periodic image that lies within r_cut of
    the cell, and ask a k-d tree (library routine) for all pairs within r_cut*(1+1e-9).
    Acceptance: the canonical float64 predicate on the ORIGINAL positions, so the result does
    not depend on how candidates were produced."""
    pos = np.asarray(pos, np.float64); cell = np.asarray(cell, np.float64)
    N = len(pos)
    if N == 0:
        return (np.zeros(0, np.int32),) * 2 + (np.zeros((0, 3), np.int32),)
    inv = np.linalg.inv(cell)
    frac = pos @ inv
    wrap = np.floor(frac).astype(np.int64)
    fw = frac - wrap
    wk = perpendicular_widths(cell)
    margin = r_cut * (1.0 + 1e-6) / wk  # fractional thickness of the image shell
    R = np.ceil(margin).astype(int)
    img_j, img_n, img_x = [], [], []
    base = fw @ cell
    for nx in range(-R[0], R[0] + 1):
        for ny in range(-R[1], R[1] + 1):
            for nz in range(-R[2], R[2] + 1):
                f = fw + np.array([nx, ny, nz], np.float64)
                inside = np.all((f >= -margin) & (f <= 1.0 + margin), axis=1)
                idx = np.nonzero(inside)[0]
                if idx.size:
                    img_j.append(idx)
                    img_n.append(np.broadcast_to(np.array([nx, ny, nz]), (idx.size, 3)))
                    img_x.append(base[idx] + np.array([nx, ny, nz], np.float64) @ cell)
    img_j = np.concatenate(img_j); img_n = np.concatenate(img_n); img_x = np.concatenate(img_x)
    tree_img = cKDTree(img_x)
    tree_own = cKDTree(base)
    coo = tree_own.sparse_distance_matrix(tree_img, r_cut * (1.0 + 1e-9), output_type="coo_matrix")
    i = coo.row.astype(np.int64)
    j = img_j[coo.col]
    n = img_n[coo.col] - wrap[j] + wrap[i]  # shift relative to the unwrapped input positions
    _, d2 = _canonical_d2(pos, cell, i, j, n)
    keep = (d2 < r_cut * r_cut) & ~((i == j) & np.all(n == 0, axis=1))
    return _canonical_sort(i[keep], j[keep], n[keep])


def edge_vectors(pos, cell, recv, send, shift):
    """r_e = (x_j - x_i) + n.C and its length, canonical operation order (O1)."""
    r, d2 = _canonical_d2(np.asarray(pos, np.float64), np.asarray(cell, np.float64), recv, send, shift)
    return r, np.sqrt(d2)


# --------------------------------------------------------------------------------------
# O2 features
# --------------------------------------------------------------------------------------
def envelope(r, r_cut):
    """u(r) = (cos(pi r / r_cut) + 1) / 2 and u'(r)."""
    x = np.pi * r / r_cut
    return 0.5 * (np.cos(x) + 1.0), -(0.5 * np.pi / r_cut) * np.sin(x)


def rbf(r, r_cut, n_rbf):
    """g_k(r) = exp(-gamma (r - mu_k)^2), mu_k = k r_cut/(n_rbf-1), gamma = 1/(2 Delta^2),
    Delta = r_cut/(n_rbf-1) (reading R8); returns g [E,k] and g' [E,k]."""
    delta = r_cut / (n_rbf - 1)
    mu = np.arange(n_rbf, dtype=np.float64) * delta
    gamma = 0.5 / (delta * delta)
    diff = r[:, None] - mu[None, :]
    g = np.exp(-gamma * diff * diff)
    return g, -2.0 * gamma * diff * g


def silu(x):
    return x * expit(x)


def dsilu(x):
    s = expit(x)
    return s * (1.0 + x * (1.0 - s))


# --------------------------------------------------------------------------------------
# O7 three-body (angle) term, SURVEY.md 8(f) NEXT-1 (reading R17; PAPER.md:91,119,131 name the model family only)
# --------------------------------------------------------------------------------------
def envelope3(r, r3):
    """u3(r) = (cos(pi r / r3) + 1)/2 for r < r3, else 0; and u3'(r)."""
    x = np.pi * r / r3
    inside = r < r3
    return np.where(inside, 0.5 * (np.cos(x) + 1.0), 0.0), np.where(inside, -(0.5 * np.pi / r3) * np.sin(x), 0.0)


def rbf3(r, r3):
    """g3_n(r) = exp(-gamma3 (r - n r3/3)^2), n = 0..3, gamma3 = 1/(2 (r3/3)^2); returns g [T,4], g' [T,4]."""
    delta = r3 / 3.0
    gamma = 0.5 / (delta * delta)
    diff = r[:, None] - (np.arange(4, dtype=np.float64) * delta)[None, :]
    g = np.exp(-gamma * diff * diff)
    return g, -2.0 * gamma * diff * g


def y_l0(c):
    """Y_l^0(c) = sqrt((2l+1)/(4 pi)) P_l(c), l = 0..3 (P0 = 1, P1 = c, P2 = (3c^2-1)/2, P3 = (5c^3-3c)/2) and
    d/dc; returns [T,4], [T,4]."""
    norm = np.sqrt((2.0 * np.arange(4) + 1.0) / (4.0 * np.pi))
    P = np.stack([np.ones_like(c), c, 0.5 * (3.0 * c * c - 1.0), 0.5 * (5.0 * c ** 3 - 3.0 * c)], axis=1)
    dP = np.stack([np.zeros_like(c), np.ones_like(c), 3.0 * c, 0.5 * (15.0 * c * c - 3.0)], axis=1)
    return P * norm, dP * norm


TRIPLET_CHUNK = 1 << 21


def triplet_chunks(recv, short, n_atoms):
    """Ordered pairs (e, e') of DISTINCT in-edges of the same receiver, both shorter than r3 (`short`), yielded in
    chunks of whole receivers. e != e' as edges: the same neighbour through two different images counts twice."""
    se = np.nonzero(short)[0]
    se = se[np.argsort(recv[se], kind="stable")]
    rc = recv[se]
    counts = np.bincount(rc, minlength=n_atoms)
    start = np.cumsum(counts) - counts           # position in `se` of the first short edge of every receiver
    per_recv = counts * counts
    lo = 0
    while lo < n_atoms:
        hi, tot = lo, 0
        while hi < n_atoms and (tot == 0 or tot + per_recv[hi] <= TRIPLET_CHUNK):
            tot += per_recv[hi]
            hi += 1
        a, b = start[lo], (start[hi - 1] + counts[hi - 1])
        if b > a:
            m = counts[rc[a:b]]
            pos_e = np.repeat(np.arange(a, b), m)
            off = np.arange(len(pos_e)) - np.repeat(np.cumsum(m) - m, m)
            pos_p = np.repeat(start[rc[a:b]], m) + off
            keep = pos_p != pos_e
            yield se[pos_e[keep]], se[pos_p[keep]]
        lo = hi


def _unit_vectors(rvec, r):
    with np.errstate(divide="ignore", invalid="ignore"):
        return np.where(r[:, None] > 0.0, rvec / r[:, None], 0.0)   # rhat := 0 at r = 0 (reading R13)


def _angle_basis(model, te, tp, rhat, r):
    """Per triplet (e, e'): c = rhat_e . rhat_e', the 16 basis values Y_l(c) g3_n(r_e') at index 4 l + n and the
    pieces their derivatives are assembled from."""
    c = np.einsum("ta,ta->t", rhat[te], rhat[tp])
    Y, dY = y_l0(c)
    g3, dg3 = rbf3(r[tp], model.r_cut3)
    Y16, dY16 = np.repeat(Y, 4, axis=1), np.repeat(dY, 4, axis=1)
    g16, dg16 = np.tile(g3, (1, 4)), np.tile(dg3, (1, 4))
    return c, Y16, dY16, g16, dg16


def three_body_terms(model, lay, h, recv, send, rvec, r):
    """t_e = u3(r_e) S_e,  S_e = sum over in-edges e' = (i <- k) != e of the same receiver with r_e' < r3 of
           u3(r_e') [Y_l^0(cos theta_ee') g3_n(r_e')]_{4l+n} * sigma(G h_k + g)          (16 components),
    zero for edges with r_e >= r3; cos theta_ee' = rhat_e . rhat_e' is the angle at the receiver. The term enters the
    first edge linear as W3 t_e. Returns t [E,16], S [E,16], z [N,16]."""
    N = len(h)
    z = expit(h @ lay["G"].T + lay["g"])
    u3, _ = envelope3(r, model.r_cut3)
    rhat = _unit_vectors(rvec, r)
    S = np.zeros((len(recv), N_ANGLE))
    for te, tp in triplet_chunks(recv, r < model.r_cut3, N):
        _, Y16, _, g16, _ = _angle_basis(model, te, tp, rhat, r)
        S += _scatter_matrix(te, len(recv)) @ (u3[tp, None] * Y16 * g16 * z[send[tp]])
    return u3[:, None] * S, S, z


def three_body_backward(model, lay, h, recv, send, rvec, r, tbar, S, z):
    """Reverse mode of three_body_terms given tbar = d(.)/d t_e [E,16]: returns the contributions to rbar [E] (through
    u3(r_e), u3(r_e') and g3_n(r_e')), to the per-edge VECTOR gradient gvec [E,3] (through cos theta, with
    d c / d r_e = (rhat_e' - c rhat_e) / r_e) and to hbar [N,d] (through the gates sigma(G h_k + g))."""
    N, E = len(h), len(recv)
    u3, du3 = envelope3(r, model.r_cut3)
    rhat = _unit_vectors(rvec, r)
    with np.errstate(divide="ignore"):
        inv_r = np.where(r > 0.0, 1.0 / r, 0.0)
    rbar = du3 * np.sum(tbar * S, axis=1)
    tau = tbar * u3[:, None]                       # adjoint of S_e
    gvec = np.zeros((E, 3))
    zbar = np.zeros((N, N_ANGLE))
    for te, tp in triplet_chunks(recv, r < model.r_cut3, N):
        c, Y16, dY16, g16, dg16 = _angle_basis(model, te, tp, rhat, r)
        tz = tau[te] * z[send[tp]]
        rbar += _scatter_matrix(tp, E) @ np.sum(tz * Y16 * (du3[tp, None] * g16 + u3[tp, None] * dg16), axis=1)
        cbar = u3[tp] * np.sum(tz * dY16 * g16, axis=1)
        gvec += _scatter_matrix(te, E) @ ((cbar * inv_r[te])[:, None] * (rhat[tp] - c[:, None] * rhat[te]))
        gvec += _scatter_matrix(tp, E) @ ((cbar * inv_r[tp])[:, None] * (rhat[te] - c[:, None] * rhat[tp]))
        zbar += _scatter_matrix(send[tp], N) @ (tau[te] * Y16 * g16 * u3[tp, None])
    hbar = (zbar * z * (1.0 - z)) @ lay["G"]
    return rbar, gvec, hbar


# --------------------------------------------------------------------------------------
# O3-O5 model
# --------------------------------------------------------------------------------------
def _scatter_matrix(index, n_rows, weights=None):
    """Sparse [n_rows, len(index)] matrix S with S[index[e], e] = weights[e]; S @ X sums rows of
    X into their targets (the scatter-sum of message passing as a library sparse product)."""
    e = len(index)
    data = np.ones(e) if weights is None else weights
    return sp.csr_matrix((data, (index, np.arange(e))), shape=(n_rows, e))


def _edge_layer_forward(model, lay, h, recv, send, r, t=None):
    """m_i = alpha sum_{e in in(i)} u(r_e) phi_e with
    a_e = W1 [h_i || h_j || e_hat_e] + b1 (+ W3 t_e, three-body variant) ; s = SiLU(a) ; p = W2 s + b2 ; phi = SiLU(p)."""
    N, d = h.shape
    m = np.zeros((N, d))
    for lo in range(0, len(recv), EDGE_CHUNK):
        sl = slice(lo, lo + EDGE_CHUNK)
        u, _ = envelope(r[sl], model.r_cut)
        g, _ = rbf(r[sl], model.r_cut, model.n_rbf)
        x = np.concatenate([h[recv[sl]], h[send[sl]], u[:, None] * g], axis=1)
        a = x @ lay["W1"].T + lay["b1"]
        if t is not None:
            a = a + t[sl] @ lay["W3"].T
        p = silu(a) @ lay["W2"].T + lay["b2"]
        phi = silu(p)
        m += _scatter_matrix(recv[sl], N, model.agg_scale * u) @ phi
    return m


def forward(model, L, species, recv, send, r, rvec=None):
    """h^0 = T[z]; L layers (O3); E_i = wo . SiLU(Wo h^L + bo) + b_E + E0[z] (O4).
    Returns E_i and the per-layer node states needed by the reverse pass. `rvec` (edge vectors) is needed by the
    three-body variant only."""
    assert 0 <= L <= model.L_max
    h = model.T[species].copy()
    hs, ms, cs = [], [], []
    for l in range(L):
        lay = model.layers[l]
        t = three_body_terms(model, lay, h, recv, send, rvec, r)[0] if model.r_cut3 > 0.0 else None
        m = _edge_layer_forward(model, lay, h, recv, send, r, t)
        c = np.concatenate([h, m], axis=1) @ lay["V1"].T + lay["c1"]
        hs.append(h); ms.append(m); cs.append(c)
        h = h + silu(c) @ lay["V2"].T + lay["c2"]
    o = h @ model.Wo.T + model.bo
    E_i = silu(o) @ model.wo + model.bE + model.E0[species]
    return E_i, dict(hs=hs, ms=ms, cs=cs, hL=h, o=o)


def backward_rbar(model, L, species, recv, send, r, cache, omega, rvec=None, return_gvec=False):
    """Reverse mode of sum_i omega_i E_i down to the per-edge scalar rbar_e = d(.)/d r_e (O5). The three-body variant
    also depends on the edge DIRECTIONS; with return_gvec the per-edge vector gradient gvec_e = d(.)/d rvec_e at fixed
    |r_e| contributions excluded from rbar (zeros for the two-body model) is returned as well."""
    N = len(species)
    d = model.d
    three = model.r_cut3 > 0.0
    hbar = omega[:, None] * ((model.wo * dsilu(cache["o"])) @ model.Wo)
    rbar = np.zeros(len(recv))
    gvec = np.zeros((len(recv), 3))
    for l in range(L - 1, -1, -1):
        lay = model.layers[l]
        h, c = cache["hs"][l], cache["cs"][l]
        if three:
            t, S3, z3 = three_body_terms(model, lay, h, recv, send, rvec, r)
            tbar = np.zeros((len(recv), N_ANGLE))
        cbar = (hbar @ lay["V2"]) * dsilu(c)
        hm = cbar @ lay["V1"]
        hbar = hbar + hm[:, :d]
        mbar = hm[:, d:]
        hadd = np.zeros((N, d))
        for lo in range(0, len(recv), EDGE_CHUNK):
            sl = slice(lo, lo + EDGE_CHUNK)
            ri, si = recv[sl], send[sl]
            u, du = envelope(r[sl], model.r_cut)
            g, dg = rbf(r[sl], model.r_cut, model.n_rbf)
            x = np.concatenate([h[ri], h[si], u[:, None] * g], axis=1)
            a = x @ lay["W1"].T + lay["b1"]
            if three:
                a = a + t[sl] @ lay["W3"].T
            p = silu(a) @ lay["W2"].T + lay["b2"]
            phi = silu(p)
            mb = mbar[ri]
            phibar = model.agg_scale * u[:, None] * mb
            ubar = model.agg_scale * np.sum(mb * phi, axis=1)
            pbar = phibar * dsilu(p)
            sbar = pbar @ lay["W2"]
            abar = sbar * dsilu(a)
            if three:
                tbar[sl] = abar @ lay["W3"]
            xbar = abar @ lay["W1"]
            hadd += _scatter_matrix(ri, N) @ xbar[:, :d]
            hadd += _scatter_matrix(si, N) @ xbar[:, d:2 * d]
            ebar = xbar[:, 2 * d:]
            ubar = ubar + np.sum(ebar * g, axis=1)
            rbar[sl] += ubar * du + np.sum(u[:, None] * ebar * dg, axis=1)
        hbar = hbar + hadd
        if three:
            rb3, gv3, hb3 = three_body_backward(model, lay, h, recv, send, rvec, r, tbar, S3, z3)
            rbar += rb3
            gvec += gv3
            hbar = hbar + hb3
    if return_gvec:
        return rbar, gvec
    return rbar


def forces_from_rbar(n_atoms, recv, send, rvec, r, rbar, gvec=None):
    """F_k = sum_{e in in(k)} rbar_e rhat_e - sum_{e in out(k)} rbar_e rhat_e, rhat := 0 at r = 0
    (reading R13), because d r_e / d x_send = rhat_e and d r_e / d x_recv = -rhat_e. With the three-body variant the
    gradient with respect to the edge VECTOR is rbar_e rhat_e + gvec_e and d rvec_e / d x_send = 1 = -d rvec_e / d x_recv."""
    with np.errstate(divide="ignore", invalid="ignore"):
        rhat = np.where(r[:, None] > 0.0, rvec / r[:, None], 0.0)
    f_edge = rbar[:, None] * rhat
    if gvec is not None:
        f_edge = f_edge + gvec
    return _scatter_matrix(recv, n_atoms) @ f_edge - _scatter_matrix(send, n_atoms) @ f_edge


def energy_forces(model, L, pos, cell, species, graph=None, omega=None, return_extra=False):
    """E, E_i and F = -dE/dx of the unpartitioned model (the plain definition).
    `omega` (default all ones) weights the per-atom energies in the differentiated sum."""
    pos = np.asarray(pos, np.float64); cell = np.asarray(cell, np.float64)
    species = np.asarray(species)
    if graph is None:
        graph = neighbor_list(pos, cell, model.r_cut)
    recv, send, shift = graph
    rvec, r = edge_vectors(pos, cell, recv, send, shift)
    E_i, cache = forward(model, L, species, recv, send, r, rvec)
    if omega is None:
        omega = np.ones(len(species))
    rbar, gvec = backward_rbar(model, L, species, recv, send, r, cache, np.asarray(omega, np.float64), rvec, return_gvec=True)
    F = forces_from_rbar(len(species), recv, send, rvec, r, rbar, gvec if model.r_cut3 > 0.0 else None)
    E = float(np.sum(omega * E_i))
    if return_extra:
        return E, E_i, F, dict(rbar=rbar, gvec=gvec, r=r, rvec=rvec, cache=cache, graph=graph)
    return E, E_i, F


def stress_from_rbar(cell, rvec, r, rbar, gvec=None):
    """Stress sigma = (1/V) dE/d(strain) (PAPER.md:173 lists stress beside energy and forces as a model
    output). Under a homogeneous strain x -> (1 + eps) x, C -> C (1 + eps)^T every edge vector transforms as
    r_e -> (1 + eps) r_e, so d r_e / d eps_ab = r_a r_b / r and
        sigma_ab = (1/V) sum_e rbar_e r_ea r_eb / r_e      (sum over DIRECTED edges, rbar_e = dE/dr_e;
    edges with r = 0 contribute nothing, reading R13). Symmetric by construction; eV / A^3."""
    V = abs(np.linalg.det(np.asarray(cell, np.float64)))
    with np.errstate(divide="ignore", invalid="ignore"):
        w = np.where(r > 0.0, rbar / r, 0.0)
    sigma = np.einsum("e,ea,eb->ab", w, rvec, rvec) / V
    if gvec is not None:   # three-body variant: d rvec_e / d eps_ab = delta_.a r_eb, the gradient w.r.t. rvec_e has gvec_e on top
        sigma = sigma + np.einsum("ea,eb->ab", gvec, rvec) / V
    return sigma


def energy_forces_stress(model, L, pos, cell, species, graph=None, omega=None):
    """E, E_i, F and the stress tensor [3,3] of the unpartitioned model."""
    E, E_i, F, ex = energy_forces(model, L, pos, cell, species, graph, omega, return_extra=True)
    return E, E_i, F, stress_from_rbar(cell, ex["rvec"], ex["r"], ex["rbar"], ex["gvec"] if model.r_cut3 > 0.0 else None)


# --------------------------------------------------------------------------------------
# O6 partitioned evaluation
# --------------------------------------------------------------------------------------
def slab_axis(cell):
    """Axis with the largest perpendicular width, ties -> lowest index (reading R3)."""
    return int(np.argmax(perpendicular_widths(cell)))


def partition_grid(pos, cell, grid, halo):
    """Stage 1: uniform grid of P = gx*gy*gz bins on the unit cube; atom -> bin
    by its wrapped scaled position, bin index min(floor(f*g), g-1) per axis.
    Stage 2 (reading R2): extended set = atoms whose periodic distance to the bin interval is
    <= halo along every axis (a superset of the K-hop BFS set of PAPER.md:165 when
    halo >= K*r_cut). Returns a list of (owned_idx, ext_idx) with owned a subset of ext."""
    pos = np.asarray(pos, np.float64); cell = np.asarray(cell, np.float64)
    frac = pos @ np.linalg.inv(cell)
    f = frac - np.floor(frac)
    wk = perpendicular_widths(cell)
    g = np.asarray(grid, int)
    bins = np.minimum(np.floor(f * g).astype(int), g - 1)
    parts = []
    for bx in range(g[0]):
        for by in range(g[1]):
            for bz in range(g[2]):
                b = np.array([bx, by, bz])
                owned = np.all(bins == b, axis=1)
                ext = np.ones(len(pos), bool)
                for k in range(3):
                    lo, hi = b[k] / g[k], (b[k] + 1) / g[k]
                    inside = (f[:, k] >= lo) & (f[:, k] < hi)
                    below = np.mod(lo - f[:, k], 1.0)
                    above = np.mod(f[:, k] - hi, 1.0)
                    dist = np.where(inside, 0.0, np.minimum(below, above)) * wk[k]
                    ext &= dist <= halo
                ext |= owned
                parts.append((np.nonzero(owned)[0], np.nonzero(ext)[0]))
    return parts


def partition_slabs(pos, cell, n_sub, halo):
    g = [1, 1, 1]
    g[slab_axis(cell)] = n_sub
    return partition_grid(pos, cell, g, halo)


def induced_subgraph(graph, ext_idx, n_atoms):
    """Sub-graph of the GLOBAL graph induced on ext (edges keep their shifts)."""
    recv, send, shift = graph
    local = -np.ones(n_atoms, np.int64)
    local[ext_idx] = np.arange(len(ext_idx))
    keep = (local[recv] >= 0) & (local[send] >= 0)
    return local[recv[keep]], local[send[keep]], shift[keep]


def energy_forces_partitioned(model, L, pos, cell, species, parts, graph=None):
    """E = sum_s sum_{i in own(s)} E_i^(s);  F = sum_s scatter_{k in ext(s)} of
    -d( sum_{i in own(s)} E_i^(s) ) / d x_k   (reading R1)."""
    pos = np.asarray(pos, np.float64); cell = np.asarray(cell, np.float64)
    species = np.asarray(species)
    N = len(pos)
    if graph is None:
        graph = neighbor_list(pos, cell, model.r_cut)
    E = 0.0
    E_i = np.zeros(N)
    F = np.zeros((N, 3))
    stats = []
    for owned, ext in parts:
        lrecv, lsend, lshift = induced_subgraph(graph, ext, N)
        omega = np.isin(ext, owned).astype(np.float64)
        Es, Eis, Fs = energy_forces(model, L, pos[ext], cell, species[ext], (lrecv, lsend, lshift), omega)
        E += Es
        E_i[owned] += Eis[omega > 0]
        F[ext] += Fs
        stats.append(dict(n_owned=len(owned), n_ext=len(ext), n_edges=len(lrecv)))
    return E, E_i, F, stats


def khop_distance(graph, owned_idx, n_atoms, max_hops):
    """Stage 2 of PAPER.md:165 as stated: breadth-first search over the radius graph from the root atoms
    of a bin. Returns hops[n_atoms] = number of edges on the shortest path to the nearest root atom
    (0 for root atoms, max_hops + 1 for atoms farther than max_hops)."""
    recv, send, _ = graph
    hops = np.full(n_atoms, max_hops + 1, np.int64)
    hops[owned_idx] = 0
    frontier = np.zeros(n_atoms, bool)
    frontier[owned_idx] = True
    for k in range(1, max_hops + 1):
        reached = np.zeros(n_atoms, bool)
        reached[send[frontier[recv]]] = True          # senders of edges into the frontier
        new = reached & (hops > k)
        hops[new] = k
        frontier = new
    return hops


def partition_grid_khop(pos, cell, grid, halo, r_cut, graph=None):
    """Stage 2 as the paper states it: the extended set of a bin is the K-hop
    neighbourhood of its root atoms, K = ceil(halo / r_cut), found by breadth-first search over the
    radius graph -- searched inside the geometric box of partition_grid (which contains every atom
    within K hops whenever halo >= K r_cut, so the restriction then changes nothing).
    Returns a list of (owned_idx, ext_idx, hops) with hops aligned with ext_idx (0 for root atoms)."""
    pos = np.asarray(pos, np.float64); cell = np.asarray(cell, np.float64)
    N = len(pos)
    if graph is None:
        graph = neighbor_list(pos, cell, r_cut)
    recv, send, shift = graph
    K = max(1, int(np.ceil(halo / r_cut - 1e-9)))
    out = []
    for owned, box in partition_grid(pos, cell, grid, halo):
        inside = np.zeros(N, bool)
        inside[box] = True
        keep = inside[recv] & inside[send]
        hops = khop_distance((recv[keep], send[keep], shift[keep]), owned, N, K)
        ext = np.nonzero(inside & (hops <= K))[0]
        out.append((owned, ext, hops[ext]))
    return out


def halo_depth_classes(pos, cell, grid, halo, r_cut):
    """Depth class of every atom of every extended set (same bins, same order as partition_grid):
    0 for root atoms, else ceil(D / r_cut) clipped to [1, ceil(halo / r_cut)], D = the largest per-axis
    periodic distance to the bin interval. An edge is shorter than r_cut, so a class-k atom is at least k
    hops from the nearest root atom (pinned against khop_distance in tests/test_oracle_graph.py): layer l
    of L (0-based) matters for the root energies of PAPER.md:169 only on receivers of class <= L-1-l.
    Returns a list of int arrays aligned with the ext_idx of partition_grid."""
    pos = np.asarray(pos, np.float64); cell = np.asarray(cell, np.float64)
    frac = pos @ np.linalg.inv(cell)
    f = frac - np.floor(frac)
    wk = perpendicular_widths(cell)
    g = np.asarray(grid, int)
    n_cls = max(2, 1 + int(np.ceil(halo / r_cut - 1e-9)))
    out = []
    for (owned, ext), b in zip(partition_grid(pos, cell, grid, halo), np.ndindex(*g)):
        D = np.zeros(len(pos))
        for k in range(3):
            lo, hi = b[k] / g[k], (b[k] + 1) / g[k]
            inside = (f[:, k] >= lo) & (f[:, k] < hi)
            below = np.mod(lo - f[:, k], 1.0)
            above = np.mod(f[:, k] - hi, 1.0)
            D = np.maximum(D, np.where(inside, 0.0, np.minimum(below, above)) * wk[k])
        cls = np.clip(np.ceil(D / r_cut - 1e-9).astype(np.int64), 1, n_cls - 1)
        cls[owned] = 0
        out.append(cls[ext])
    return out


def stress_partitioned(model, L, pos, cell, species, parts, graph=None):
    """"a similar decomposition applies" -- the strain derivative is linear in the energy,
    so sigma = sum_s (1/V) d( sum_{i in own(s)} E_i^(s) ) / d eps, each term over the edges of sub-graph s."""
    pos = np.asarray(pos, np.float64); cell = np.asarray(cell, np.float64)
    species = np.asarray(species)
    N = len(pos)
    if graph is None:
        graph = neighbor_list(pos, cell, model.r_cut)
    sigma = np.zeros((3, 3))
    for owned, ext in parts:
        lg = induced_subgraph(graph, ext, N)
        omega = np.isin(ext, owned).astype(np.float64)
        sigma += energy_forces_stress(model, L, pos[ext], cell, species[ext], lg, omega)[3]
    return sigma


def halo_growth_factor(parts):
    """H = (# atoms added by the halo) / (# root atoms), PAPER.md:289 (S1)."""
    return [(len(ext) - len(owned)) / max(len(owned), 1) for owned, ext in parts]


# --------------------------------------------------------------------------------------
# short NVE run (pin only)
# --------------------------------------------------------------------------------------
ACC_UNIT = 9.648533e-3  # (eV/A)/amu -> A/fs^2


def nve_velocity_verlet(model, L, pos, cell, species, masses, vel, dt, n_steps, return_state=False):
    """Velocity-Verlet; returns total energy (potential + kinetic, eV) per step
    (and the final positions and velocities when return_state is set)."""
    pos = np.array(pos, np.float64); vel = np.array(vel, np.float64)
    E, _, F = energy_forces(model, L, pos, cell, species)
    out = []
    for _ in range(n_steps):
        kin = 0.5 * np.sum(masses[:, None] * vel * vel) / ACC_UNIT
        out.append(E + kin)
        vel += 0.5 * dt * ACC_UNIT * F / masses[:, None]
        pos += dt * vel
        E, _, F = energy_forces(model, L, pos, cell, species)
        vel += 0.5 * dt * ACC_UNIT * F / masses[:, None]
    kin = 0.5 * np.sum(masses[:, None] * vel * vel) / ACC_UNIT
    out.append(E + kin)
    if return_state:
        return np.array(out), pos, vel
    return np.array(out)


# --------------------------------------------------------------------------------------
# Langevin dynamics (the integrator of every MD result of the paper: ASE Langevin)
# --------------------------------------------------------------------------------------
KB_EV = 8.617333262e-5  # Boltzmann constant, eV/K

_PHILOX_M0, _PHILOX_M1 = 0xD2511F53, 0xCD9E8D57
_PHILOX_W0, _PHILOX_W1 = 0x9E3779B9, 0xBB67AE85


def philox4x32(counter, key, rounds=10):
    """Philox4x32-10 counter-based generator (Salmon, Moraes, Dror, Shaw, SC'11), vectorised over the leading axis:
    counter uint32 [n,4], key uint32 [n,2] -> uint32 [n,4]. Random numbers the method draws are a pure function of
    (seed, step, atom), so the CUDA path restates the same generator instead of sharing code."""
    c = np.array(counter, dtype=np.uint64).reshape(-1, 4)
    k = np.array(key, dtype=np.uint64).reshape(-1, 2)
    c0, c1, c2, c3 = c[:, 0].copy(), c[:, 1].copy(), c[:, 2].copy(), c[:, 3].copy()
    k0, k1 = k[:, 0].copy(), k[:, 1].copy()
    mask = np.uint64(0xFFFFFFFF)
    for _ in range(rounds):
        p0 = np.uint64(_PHILOX_M0) * c0
        p1 = np.uint64(_PHILOX_M1) * c2
        hi0, lo0 = p0 >> np.uint64(32), p0 & mask
        hi1, lo1 = p1 >> np.uint64(32), p1 & mask
        c0, c1, c2, c3 = (hi1 ^ c1 ^ k0) & mask, lo1, (hi0 ^ c3 ^ k1) & mask, lo0
        k0 = (k0 + np.uint64(_PHILOX_W0)) & mask
        k1 = (k1 + np.uint64(_PHILOX_W1)) & mask
    return np.stack([c0, c1, c2, c3], axis=1).astype(np.uint32)


def langevin_normals(seed, step, n_atoms):
    """Three standard normal numbers per atom for the O step of time step `step`: Philox4x32-10 with
    counter = (atom, step, 0, 0), key = (seed low, seed high); the four 32-bit outputs x0..x3 give
    u1 = (x0 + 0.5) 2^-32, u2 = (x1 + 0.5) 2^-32, u3 = (x2 + 0.5) 2^-32, u4 = (x3 + 0.5) 2^-32 and, by Box-Muller,
    xi_x = sqrt(-2 ln u1) cos(2 pi u2), xi_y = sqrt(-2 ln u1) sin(2 pi u2), xi_z = sqrt(-2 ln u3) cos(2 pi u4)."""
    ctr = np.zeros((n_atoms, 4), np.uint32)
    ctr[:, 0] = np.arange(n_atoms, dtype=np.uint32)
    ctr[:, 1] = np.uint32(step)
    key = np.tile(np.array([[seed & 0xFFFFFFFF, (seed >> 32) & 0xFFFFFFFF]], dtype=np.uint32), (n_atoms, 1))
    x = philox4x32(ctr, key).astype(np.float64)
    u = (x + 0.5) * 2.0 ** -32
    ra, rb = np.sqrt(-2.0 * np.log(u[:, 0])), np.sqrt(-2.0 * np.log(u[:, 2]))
    return np.stack([ra * np.cos(2 * np.pi * u[:, 1]), ra * np.sin(2 * np.pi * u[:, 1]), rb * np.cos(2 * np.pi * u[:, 3])], axis=1)


def langevin_baoab_generic(force_fn, pos, masses, vel, dt, n_steps, temperature, friction, seed):
    """BAOAB splitting of Langevin dynamics (Leimkuhler & Matthews 2013; the paper runs ASE's Langevin integrator and
    does not print its update rule -- reading R20): per step
        B  v += (dt/2) a(x)          A  x += (dt/2) v
        O  v = c1 v + c2 sqrt(kB T / m) xi,  c1 = exp(-friction dt), c2 = sqrt(1 - c1^2)
        A  x += (dt/2) v             B  v += (dt/2) a(x)      (one force evaluation per step)
    with a = ACC_UNIT F / m, xi from `langevin_normals(seed, step, N)`. friction = 0 is velocity Verlet exactly.
    force_fn(pos) -> (E, F). Returns (total energy before every step and after the last, pos, vel)."""
    pos = np.array(pos, np.float64); vel = np.array(vel, np.float64)
    c1 = np.exp(-friction * dt)
    c2 = np.sqrt(1.0 - c1 * c1)
    sig = np.sqrt(KB_EV * temperature * ACC_UNIT / masses)[:, None]   # sqrt(kB T / m) in A/fs
    E, F = force_fn(pos)
    out = []
    for step in range(n_steps):
        out.append(E + 0.5 * np.sum(masses[:, None] * vel * vel) / ACC_UNIT)
        vel += 0.5 * dt * ACC_UNIT * F / masses[:, None]
        pos += 0.5 * dt * vel
        if friction > 0.0:
            vel = c1 * vel + c2 * sig * langevin_normals(seed, step, len(pos))
        pos += 0.5 * dt * vel
        E, F = force_fn(pos)
        vel += 0.5 * dt * ACC_UNIT * F / masses[:, None]
    out.append(E + 0.5 * np.sum(masses[:, None] * vel * vel) / ACC_UNIT)
    return np.array(out), pos, vel


def langevin_baoab(model, L, pos, cell, species, masses, vel, dt, n_steps, temperature, friction, seed):
    """Langevin dynamics of the model potential (see langevin_baoab_generic)."""
    def force_fn(x):
        E, _, F = energy_forces(model, L, x, cell, species)
        return E, F
    return langevin_baoab_generic(force_fn, pos, masses, vel, dt, n_steps, temperature, friction, seed)
