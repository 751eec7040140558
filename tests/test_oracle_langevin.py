"""Pins for the oracle's Langevin integrator (every MD result of the paper is ASE Langevin dynamics;
reading R20: BAOAB splitting, Philox4x32-10 normals): the generator against its published known-answer vectors, the normal
numbers against their moments, the friction -> 0 limit against velocity Verlet, and the fluctuation-dissipation
temperature and the configurational variance kB T / k of a harmonic bath."""
import os

import numpy as np

from oracle import mlip_oracle as O
from synth_inputs import ModelSpec, make_weights, small_system

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def test_philox_known_answers():
    rows = [l.split() for l in open(os.path.join(GOLDEN, "philox4x32_10_kat.txt")) if l.strip() and not l.startswith("#")]
    assert len(rows) == 3
    for row in rows:
        v = [int(x, 16) for x in row]
        out = O.philox4x32(np.array([v[0:4]], np.uint32), np.array([v[4:6]], np.uint32))[0]
        assert [int(x) for x in out] == v[6:10]
    # vectorised over rows = row by row
    ctr = np.array([[int(x, 16) for x in r[0:4]] for r in rows], np.uint32)
    key = np.array([[int(x, 16) for x in r[4:6]] for r in rows], np.uint32)
    assert np.array_equal(O.philox4x32(ctr, key), np.array([[int(x, 16) for x in r[6:10]] for r in rows], np.uint32))


def test_langevin_normals_moments_and_streams():
    n = 200000
    a = O.langevin_normals(seed=12345, step=0, n_atoms=n)
    assert a.shape == (n, 3) and np.isfinite(a).all()
    assert np.abs(a.mean(0)).max() < 4.0 / np.sqrt(n)
    assert np.abs(a.var(0) - 1.0).max() < 4.0 * np.sqrt(2.0 / n)
    assert np.abs(np.mean(a ** 4, 0) - 3.0).max() < 0.1                        # kurtosis of a normal
    c = np.corrcoef(a.T)
    assert np.abs(c - np.eye(3)).max() < 4.0 / np.sqrt(n)
    b = O.langevin_normals(seed=12345, step=1, n_atoms=n)
    assert np.abs(np.mean(a * b, 0)).max() < 4.0 / np.sqrt(n)                  # steps are independent streams
    assert np.array_equal(a, O.langevin_normals(12345, 0, n))                  # pure function of (seed, step, atom)
    assert not np.array_equal(a, O.langevin_normals(12346, 0, n))
    assert np.array_equal(a[:100], O.langevin_normals(12345, 0, 100))          # atom i does not depend on N


def test_zero_friction_is_velocity_verlet():
    spec = ModelSpec(4, 16, 8, 2, 3.0, 1.0 / np.sqrt(12.0))
    m = O.parse_weights(4, 16, 8, 2, 3.0, spec.agg_scale, make_weights(spec, 3))
    s = small_system(3, 0.08, seed=2)
    rng = np.random.default_rng(1)
    masses = rng.uniform(10, 60, len(s.pos)); vel = rng.normal(0, 0.004, s.pos.shape)
    e1, p1, v1 = O.nve_velocity_verlet(m, 2, s.pos, s.cell, s.species, masses, vel, 2.0, 8, return_state=True)
    e2, p2, v2 = O.langevin_baoab(m, 2, s.pos, s.cell, s.species, masses, vel, 2.0, 8, temperature=300.0, friction=0.0, seed=1)
    assert np.abs(e1 - e2).max() < 1e-11 and np.abs(p1 - p2).max() < 1e-12 and np.abs(v1 - v2).max() < 1e-13


def test_harmonic_bath_temperature_and_variance():
    """Independent 3-D oscillators F = -k x: the stationary state has <m v^2> = kB T per component (fluctuation-dissipation)
    and <x^2> = kB T / k; BAOAB reproduces the configurational variance of a harmonic well at any stable dt."""
    n, k_spring, T = 4000, 2.0, 450.0
    masses = np.full(n, 28.0)
    rng = np.random.default_rng(0)
    pos = rng.normal(0, 0.05, (n, 3)); vel = np.zeros((n, 3))

    def force_fn(x):
        return 0.5 * k_spring * float(np.sum(x * x)), -k_spring * x

    # equilibrate, then sample every step of a second run
    _, pos, vel = O.langevin_baoab_generic(force_fn, pos, masses, vel, 2.0, 600, T, 0.02, seed=7)
    kin, var = [], []
    for block in range(10):
        _, pos, vel = O.langevin_baoab_generic(force_fn, pos, masses, vel, 2.0, 40, T, 0.02, seed=100 + block)
        kin.append(np.mean(masses[:, None] * vel * vel) / O.ACC_UNIT)
        var.append(np.mean(pos * pos))
    kT = O.KB_EV * T
    assert abs(np.mean(kin) / kT - 1.0) < 0.03        # 4000 x 3 x 10 samples, BAOAB kinetic bias O(dt^2) ~ 1 %
    assert abs(np.mean(var) * k_spring / kT - 1.0) < 0.03
    # the thermostat is what sets it: at friction 0 the cold start stays cold
    _, p0, v0 = O.langevin_baoab_generic(force_fn, rng.normal(0, 0.01, (n, 3)), masses, np.zeros((n, 3)), 2.0, 200, T, 0.0, seed=7)
    assert np.mean(masses[:, None] * v0 * v0) / O.ACC_UNIT < 0.05 * kT
