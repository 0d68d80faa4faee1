"""Physics pins of the fp64 oracle (CPU only): what the mathematics fixes about forces, virials and
the integrator, independent of any implementation.

  * F_i = -dE/dr_i by central finite differences, periodic 5-species system with asymmetric c^{ij}
    (reading A5) and an open cluster                                   (Eqs. 21-23)
  * sum_i F_i = 0 (Newton's third law)
  * E invariant under translation, rigid rotation, same-species permutation
  * sum_i W_i = -dE/d(eps) for 6 independent strains; total virial symmetric (Eq. 24; reading A7/A9)
  * per-atom virial definition on a dimer                              (Eq. 24)
  * velocity-Verlet: unit constant from CODATA, time reversibility, energy error ~ dt^2
"""
import math

import numpy as np
import pytest
from scipy import constants as sc

import workloads as W


def small_periodic(cfg_index=3, cells=(3, 3, 3), kind="stress"):
    cfg = W.get_config(cfg_index, cells=cells)
    return cfg, W.make_system(cfg), W.make_params(cfg, kind)


def total_energy(oracle, hyper, params, pos, types, box, pbc=(1, 1, 1)):
    return oracle.compute(hyper, params, pos, types, box, pbc=pbc)[0].sum()


# ------------------------------------------------------------------ forces
def test_force_is_minus_energy_gradient_periodic(oracle_mod):
    cfg, s, p = small_periodic()           # fcc 3x3x3 = 108 atoms, box 10.8 >= 2 rc, 5 species
    e, f, w = oracle_mod.compute(cfg.hyper, p, s.pos, s.types, s.box)
    assert np.abs(f).max() > 1e-2          # the stress set gives forces far above round-off
    h = 1e-4
    rng = np.random.default_rng(0)
    for i in rng.choice(len(s.pos), 4, replace=False):
        for a in range(3):
            pp, pm = s.pos.copy(), s.pos.copy()
            pp[i, a] += h; pm[i, a] -= h
            fd = -(total_energy(oracle_mod, cfg.hyper, p, pp, s.types, s.box)
                   - total_energy(oracle_mod, cfg.hyper, p, pm, s.types, s.box)) / (2 * h)
            assert f[i, a] == pytest.approx(fd, rel=2e-6, abs=1e-8)
    np.testing.assert_allclose(f.sum(axis=0), 0.0, atol=1e-12)


def test_force_is_minus_energy_gradient_cluster_each_block(oracle_mod):
    """Open cluster; the network is replaced by one that looks at ONE descriptor block at a time, so
    a wrong derivative in any single block (radial, l=1..4, 4-body, 5-body) cannot hide behind the
    others."""
    cfg = W.get_config(2)
    hyper = cfg.hyper
    p = W.make_params(cfg, "stress")
    pos, types = W.random_cluster(1, 14, hyper.n_types, 5.5, min_dist=1.6)
    box = np.array([50.0, 50.0, 50.0])
    blocks = [(0, hyper.NR)] + [(hyper.NR + b * hyper.NA, hyper.NR + (b + 1) * hyper.NA) for b in range(6)]
    h = 1e-4
    for lo, hi in blocks:
        pb = W.Params(p.c_radial, p.c_angular, np.zeros_like(p.w0), p.b0, p.w1, p.b1)
        pb.w0[:, lo:hi] = 3.0 * p.w0[:, lo:hi]
        e, f, w = oracle_mod.compute(hyper, pb, pos, types, box, pbc=(0, 0, 0))
        scale = np.abs(f).max()
        assert scale > 1e-6
        for i in (0, 5):
            for a in range(3):
                pp, pm = pos.copy(), pos.copy()
                pp[i, a] += h; pm[i, a] -= h
                fd = -(total_energy(oracle_mod, hyper, pb, pp, types, box, (0, 0, 0))
                       - total_energy(oracle_mod, hyper, pb, pm, types, box, (0, 0, 0))) / (2 * h)
                assert f[i, a] == pytest.approx(fd, rel=5e-6, abs=2e-7 * scale)
        np.testing.assert_allclose(f.sum(axis=0), 0.0, atol=1e-12 * max(1.0, scale))


# ------------------------------------------------------------------ invariances
def test_energy_invariances(oracle_mod):
    cfg = W.get_config(3)
    hyper, p = cfg.hyper, W.make_params(cfg, "stress")
    pos, types = W.random_cluster(2, 16, hyper.n_types, 6.0, min_dist=1.5)
    box = np.array([60.0, 60.0, 60.0])
    e0, f0, w0 = oracle_mod.compute(hyper, p, pos, types, box, pbc=(0, 0, 0))
    # translation
    e1, f1, _ = oracle_mod.compute(hyper, p, pos + np.array([3.1, -2.2, 0.7]), types, box, pbc=(0, 0, 0))
    np.testing.assert_allclose(e1, e0, rtol=1e-12, atol=1e-14)
    # rigid rotation: per-atom energies invariant, forces co-rotate, virial transforms as a tensor
    rng = np.random.default_rng(4)
    Q, _ = np.linalg.qr(rng.normal(size=(3, 3)))
    if np.linalg.det(Q) < 0:
        Q[:, 0] = -Q[:, 0]
    e2, f2, w2 = oracle_mod.compute(hyper, p, pos @ Q.T, types, box, pbc=(0, 0, 0))
    np.testing.assert_allclose(e2, e0, rtol=1e-11, atol=1e-14)
    np.testing.assert_allclose(f2, f0 @ Q.T, rtol=1e-9, atol=1e-12)
    np.testing.assert_allclose(w2.reshape(-1, 3, 3), np.einsum("ab,nbc,dc->nad", Q, w0.reshape(-1, 3, 3), Q),
                               rtol=1e-9, atol=1e-12)
    # permutation of atoms (relabelling): outputs permute with the atoms
    perm = rng.permutation(len(pos))
    e3, f3, _ = oracle_mod.compute(hyper, p, pos[perm], types[perm], box, pbc=(0, 0, 0))
    np.testing.assert_allclose(e3, e0[perm], rtol=1e-12, atol=1e-14)
    np.testing.assert_allclose(f3, f0[perm], rtol=1e-10, atol=1e-13)
    # periodic: translation by an arbitrary vector and by a lattice vector
    cfgp, s, pp = small_periodic()
    ea = oracle_mod.compute(cfgp.hyper, pp, s.pos, s.types, s.box)[0]
    eb = oracle_mod.compute(cfgp.hyper, pp, s.pos + np.array([0.3, 7.7, -15.2]), s.types, s.box)[0]
    np.testing.assert_allclose(eb, ea, rtol=1e-11, atol=1e-14)


# ------------------------------------------------------------------ virial
def test_total_virial_is_minus_strain_derivative(oracle_mod):
    cfg, s, p = small_periodic(cells=(3, 3, 3))
    e, f, w = oracle_mod.compute(cfg.hyper, p, s.pos, s.types, s.box)
    wtot = w.sum(axis=0).reshape(3, 3)
    np.testing.assert_allclose(wtot, wtot.T, rtol=1e-9, atol=1e-10)      # reading A9: total is symmetric
    h = 1e-5
    # diagonal strains: scale one box edge and that coordinate
    for a in range(3):
        ep = []
        for sgn in (+1, -1):
            sc_ = np.ones(3); sc_[a] = 1.0 + sgn * h
            ep.append(total_energy(oracle_mod, cfg.hyper, p, s.pos * sc_, s.types, s.box * sc_))
        dE = (ep[0] - ep[1]) / (2 * h)
        assert wtot[a, a] == pytest.approx(-dE, rel=2e-6)
    # shear strains need a non-orthorhombic cell; use an open cluster instead (same identity)
    hyper = cfg.hyper
    pos, types = W.random_cluster(3, 15, hyper.n_types, 5.5, min_dist=1.5)
    box = np.array([60.0, 60.0, 60.0])
    e, f, w = oracle_mod.compute(hyper, p, pos, types, box, pbc=(0, 0, 0))
    wtot = w.sum(axis=0).reshape(3, 3)
    for a, b in [(0, 1), (0, 2), (1, 2), (1, 0), (0, 0)]:
        eps = np.zeros((3, 3)); eps[a, b] = h
        Ep = total_energy(oracle_mod, hyper, p, pos @ (np.eye(3) + eps).T, types, box, (0, 0, 0))
        Em = total_energy(oracle_mod, hyper, p, pos @ (np.eye(3) - eps).T, types, box, (0, 0, 0))
        assert wtot[a, b] == pytest.approx(-(Ep - Em) / (2 * h), rel=5e-6, abs=1e-9)


def test_per_atom_virial_dimer_definition(oracle_mod):
    """Two atoms: W_0 = r_01 (x) dU_1/dr_10 (Eq. 24).  dU_1/dr_10 is obtained independently as the
    finite-difference gradient of atom 1's OWN site energy with respect to atom 0's position."""
    cfg = W.get_config(2)
    hyper, p = cfg.hyper, W.make_params(cfg, "stress")
    pos = np.array([[0.0, 0.0, 0.0], [1.1, 1.7, -0.9]])
    types = np.array([0, 1], dtype=np.int32)
    box = np.array([40.0, 40.0, 40.0])
    e, f, w = oracle_mod.compute(hyper, p, pos, types, box, pbc=(0, 0, 0))
    h = 1e-5
    dU1 = np.zeros(3)
    for a in range(3):
        pp, pm = pos.copy(), pos.copy()
        pp[0, a] += h; pm[0, a] -= h
        dU1[a] = (oracle_mod.compute(hyper, p, pp, types, box, pbc=(0, 0, 0))[0][1]
                  - oracle_mod.compute(hyper, p, pm, types, box, pbc=(0, 0, 0))[0][1]) / (2 * h)
    r01 = pos[1] - pos[0]
    np.testing.assert_allclose(w[0].reshape(3, 3), np.outer(r01, dU1), rtol=1e-6, atol=1e-10)
    # and the asymmetric c^{ij}: U_0 != U_1 for a 0-1 dimer
    assert abs(e[0] - e[1]) > 1e-6


# ------------------------------------------------------------------ integrator
def test_unit_constants_from_codata():
    conv = sc.e / sc.physical_constants["atomic mass constant"][0] * 1e-10      # (eV/A/amu) -> A/fs^2: e/amu [m/s^2 per N/kg] * 1e10 (eV/A->N) * 1e-20 (m/s^2 -> A/fs^2)
    assert W.ACC_CONV == pytest.approx(conv, rel=2e-9)
    assert W.KB_EV_PER_K == pytest.approx(sc.k / sc.e, rel=1e-9)
    cfg = W.get_config(0)
    s = W.make_system(cfg)
    m = s.masses[s.types]
    t_kin = (m[:, None] * s.vel ** 2).sum() / conv / (3 * len(m) * sc.k / sc.e)
    assert t_kin == pytest.approx(cfg.temperature, rel=5e-9)
    np.testing.assert_allclose((m[:, None] * s.vel).sum(axis=0), 0.0, atol=1e-10)


def test_velocity_verlet_first_step_units(oracle_mod):
    """One step from rest-frame data: r1 = r0 + dt v0 + dt^2/2 * F0/m * conv with conv from CODATA and
    F0 from oracle.compute -- pins the unit constant and the kick-drift-kick order."""
    cfg, s, p = small_periodic(cells=(3, 3, 3))
    conv = sc.e / sc.physical_constants["atomic mass constant"][0] * 1e-10
    e0, f0, _ = oracle_mod.compute(cfg.hyper, p, s.pos, s.types, s.box)
    dt = 2.0
    pos1, vel1, ep, ek = oracle_mod.md(cfg.hyper, p, s.pos, s.vel, s.types, s.masses, s.box, dt, 1)
    m = s.masses[s.types][:, None]
    np.testing.assert_allclose(pos1, s.pos + dt * s.vel + 0.5 * dt * dt * f0 / m * conv, rtol=0, atol=1e-13)
    e1, f1, _ = oracle_mod.compute(cfg.hyper, p, pos1, s.types, s.box)
    np.testing.assert_allclose(vel1, s.vel + 0.5 * dt * (f0 + f1) / m * conv, rtol=0, atol=1e-12)  # CODATA-2018 vs -2022 constant: 1e-9 rel
    assert ep[0] == pytest.approx(e0.sum(), rel=1e-13) and ep[1] == pytest.approx(e1.sum(), rel=1e-13)
    assert ek[0] == pytest.approx(0.5 * (m * s.vel ** 2).sum() / conv, rel=5e-9)


def test_velocity_verlet_reversible_and_second_order(oracle_mod):
    cfg, s, p = small_periodic(cells=(3, 3, 3))
    args = (cfg.hyper, p)
    n = 8
    pos1, vel1, ep, ek = oracle_mod.md(*args, s.pos, s.vel, s.types, s.masses, s.box, 2.0, n)
    pos2, vel2, _, _ = oracle_mod.md(*args, pos1, -vel1, s.types, s.masses, s.box, 2.0, n)
    np.testing.assert_allclose(pos2, s.pos, rtol=0, atol=1e-11)
    np.testing.assert_allclose(-vel2, s.vel, rtol=0, atol=1e-13)
    # energy error scales as dt^2: halving dt over the same time span cuts the fluctuation ~4x
    etot = ep + ek
    _, _, ep_h, ek_h = oracle_mod.md(*args, s.pos, s.vel, s.types, s.masses, s.box, 1.0, 2 * n)
    err = np.abs(etot - etot[0]).max()
    err_h = np.abs((ep_h + ek_h) - (ep_h + ek_h)[0]).max()
    assert err > 0 and err_h > 0
    assert 2.5 < err / err_h < 6.0
    assert err < 1e-3 * abs(ek[0])
