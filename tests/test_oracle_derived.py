"""Pins of the oracle's derived outputs (CPU only): the latent-space vector and the heat
current (Eqs. 25-26).  Each is checked against something other than its own formula:

  * latent: a hand case; sum_mu latent_mu - b1 = U_i with U_i from the C network of Listing 1 (another
    code path); tanh bounds |latent_mu| <= |w1_mu|; the latent vector of the full pipeline reproduces the
    site energies the oracle's compute() returns
  * heat current: Eq. (25)'s second form on a dimer with dU_1/dr_10 from finite differences of atom 1's
    own site energy; rigid translation v_i = v0: J = (sum_i W_i) v0 = -(dE/d eps) v0 with the strain
    derivative by finite differences; J is linear in v and invariant to the order of atoms
"""
import numpy as np
import pytest

import workloads as W


def test_latent_hand_case(oracle_mod):
    class P:
        w0 = np.array([[0.5, -1.0], [2.0, 0.25]]); b0 = np.array([0.1, -0.2]); w1 = np.array([3.0, -0.5]); b1 = np.array([0.7])
    q = np.array([[1.0, 2.0]])
    lat = oracle_mod.latent(P, q)
    # neuron 0: tanh(0.5 - 2.0 - 0.1) = tanh(-1.6); neuron 1: tanh(2.0 + 0.5 + 0.2) = tanh(2.7)
    assert lat[0, 0] == pytest.approx(3.0 * -0.9216685544064713, rel=1e-14)
    assert lat[0, 1] == pytest.approx(-0.5 * 0.9910074536781176, rel=1e-14)


def test_latent_sums_to_site_energy(oracle_mod):
    cfg = W.get_config(3, cells=(3, 3, 3))
    s, p = W.make_system(cfg), W.make_params(cfg, "stress")
    e, f, w, q, fp, S = oracle_mod.compute(cfg.hyper, p, s.pos, s.types, s.box, want_internals=True)
    lat = oracle_mod.latent(p, q)
    assert lat.shape == (len(s.pos), cfg.hyper.n_neurons)
    np.testing.assert_allclose(lat.sum(axis=1) - float(p.b1[0]), e, rtol=1e-12, atol=1e-13)
    assert (np.abs(lat) <= np.abs(np.asarray(p.w1, dtype=np.float64))[None, :] + 1e-15).all()
    # and against the C network of Listing 1, atom by atom
    for i in (0, 17, 53):
        ui, _ = oracle_mod.ann(p.w0, p.b0, p.w1, p.b1, q[i])
        assert lat[i].sum() - float(p.b1[0]) == pytest.approx(ui, rel=1e-12, abs=1e-13)


def test_heat_current_dimer_second_form_of_eq25(oracle_mod):
    """J_0 = r_01 (dU_1/dr_10 . v_0), Eq. (25) second line, with dU_1/dr_10 = dU_1/dr_0 by central
    differences of atom 1's own site energy -- no virial involved."""
    cfg = W.get_config(2)
    hyper, p = cfg.hyper, W.make_params(cfg, "stress")
    pos = np.array([[0.0, 0.0, 0.0], [1.1, 1.7, -0.9]])
    vel = np.array([[0.013, -0.004, 0.009], [-0.002, 0.011, 0.005]])
    types = np.array([0, 1], dtype=np.int32)
    box = np.array([40.0, 40.0, 40.0])
    e, f, w = oracle_mod.compute(hyper, p, pos, types, box, pbc=(0, 0, 0))
    ja, jt = oracle_mod.heat_current(w, vel)
    h = 1e-5
    dU = np.zeros((2, 3))          # dU[0] = dU_1/dr_0 = dU_1/dr_10 ; dU[1] = dU_0/dr_1 = dU_0/dr_01
    for a in range(3):
        for mover, owner in ((0, 1), (1, 0)):
            pp, pm = pos.copy(), pos.copy()
            pp[mover, a] += h; pm[mover, a] -= h
            dU[mover, a] = (oracle_mod.compute(hyper, p, pp, types, box, pbc=(0, 0, 0))[0][owner]
                            - oracle_mod.compute(hyper, p, pm, types, box, pbc=(0, 0, 0))[0][owner]) / (2 * h)
    r01 = pos[1] - pos[0]
    np.testing.assert_allclose(ja[0], r01 * np.dot(dU[0], vel[0]), rtol=1e-6, atol=1e-12)
    np.testing.assert_allclose(ja[1], -r01 * np.dot(dU[1], vel[1]), rtol=1e-6, atol=1e-12)
    np.testing.assert_allclose(jt, ja[0] + ja[1], rtol=1e-15)


def test_heat_current_rigid_translation_is_strain_derivative(oracle_mod):
    """v_i = v0 for all i: J = (sum_i W_i) v0, and sum_i W_i = -dE/d eps (reading A7), the latter by finite
    differences of the total energy under the six strains of an open cluster."""
    cfg = W.get_config(3, cells=(3, 3, 3))
    hyper, p = cfg.hyper, W.make_params(cfg, "stress")
    pos, types = W.random_cluster(5, 14, hyper.n_types, 5.5, min_dist=1.5)
    box = np.array([60.0, 60.0, 60.0])
    e, f, w = oracle_mod.compute(hyper, p, pos, types, box, pbc=(0, 0, 0))
    v0 = np.array([0.007, -0.012, 0.004])
    ja, jt = oracle_mod.heat_current(w, np.tile(v0, (len(pos), 1)))
    h = 1e-5
    dE = np.zeros((3, 3))
    for a in range(3):
        for b in range(3):
            eps = np.zeros((3, 3)); eps[a, b] = h
            Ep = oracle_mod.compute(hyper, p, pos @ (np.eye(3) + eps).T, types, box, pbc=(0, 0, 0))[0].sum()
            Em = oracle_mod.compute(hyper, p, pos @ (np.eye(3) - eps).T, types, box, pbc=(0, 0, 0))[0].sum()
            dE[a, b] = (Ep - Em) / (2 * h)
    np.testing.assert_allclose(jt, -dE @ v0, rtol=2e-5, atol=1e-10)


def test_heat_current_linear_and_order_independent(oracle_mod):
    rng = np.random.default_rng(7)
    w = rng.normal(size=(23, 9)); v1 = rng.normal(size=(23, 3)); v2 = rng.normal(size=(23, 3))
    j1, t1 = oracle_mod.heat_current(w, v1)
    j2, t2 = oracle_mod.heat_current(w, v2)
    j3, t3 = oracle_mod.heat_current(w, 2.0 * v1 - 3.0 * v2)
    np.testing.assert_allclose(j3, 2.0 * j1 - 3.0 * j2, rtol=1e-12, atol=1e-12)
    perm = rng.permutation(23)
    jp, tp = oracle_mod.heat_current(w[perm], v1[perm])
    np.testing.assert_allclose(jp, j1[perm], rtol=0, atol=0)
    np.testing.assert_allclose(tp, t1, rtol=1e-12, atol=1e-12)
    # a transposed virial must NOT give the same current (guards the W[3a+b] layout)
    jt_, _ = oracle_mod.heat_current(w.reshape(-1, 3, 3).transpose(0, 2, 1).reshape(-1, 9), v1)
    assert np.abs(jt_ - j1).max() > 1e-3


# ------------------------------------------------------------------ Berendsen NVT (reading A15)
def test_oracle_unit_constants_from_codata(oracle_mod):
    from scipy import constants as sc
    conv = sc.e / sc.physical_constants["atomic mass constant"][0] * 1e-10
    assert oracle_mod.ACC_CONV == pytest.approx(conv, rel=2e-9)
    assert oracle_mod.KB_EV_PER_K == pytest.approx(sc.k / sc.e, rel=1e-9)
    cfg = W.get_config(0)
    s = W.make_system(cfg)        # workloads draws exactly cfg.temperature with its own constants
    assert oracle_mod.kinetic_temperature(s.vel, s.masses[s.types]) == pytest.approx(cfg.temperature, rel=5e-9)


def _zero_model(cfg):
    """all parameters zero: U_i = 0, no forces -- free particles"""
    p = W.make_params(cfg)
    for name in ("c_radial", "c_angular", "w0", "b0", "w1", "b1"):
        getattr(p, name)[...] = 0.0
    return p


def test_berendsen_free_particles_closed_form(oracle_mod):
    """No forces: velocity-Verlet leaves T unchanged, so T_{k+1} = T_k + (dt/tau)(T0 - T_k) exactly, i.e.
    T_k = T0 + (T_init - T0) (1 - dt/tau)^k; positions advance with the velocity of each step."""
    cfg = W.get_config(0)
    s, p = W.make_system(cfg), _zero_model(cfg)
    dt, tau, T0, n = 2.0, 50.0, 450.0, 12
    pos, vel, tb, ta = oracle_mod.md_berendsen(cfg.hyper, p, s.pos, s.vel, s.types, s.masses, s.box, dt, n, T0, T0, tau)
    k = np.arange(1, n + 1)
    np.testing.assert_allclose(ta, T0 + (cfg.temperature - T0) * (1.0 - dt / tau) ** k, rtol=1e-12)
    np.testing.assert_allclose(tb[1:], ta[:-1], rtol=1e-13)
    lam = np.sqrt(np.concatenate([[cfg.temperature], ta[:-1]]) ** -1 * ta)          # per-step scale factors
    scale_before = np.concatenate([[1.0], np.cumprod(lam)[:-1]])                  # velocity used in step k's drift
    np.testing.assert_allclose(pos, s.pos + dt * s.vel * scale_before.sum(), rtol=0, atol=1e-11)
    np.testing.assert_allclose(vel, s.vel * np.prod(lam), rtol=1e-13, atol=0)


def test_berendsen_limits_and_one_step_identity(oracle_mod):
    cfg = W.get_config(3, cells=(3, 3, 3))
    s, p = W.make_system(cfg), W.make_params(cfg, "stress")
    args = (cfg.hyper, p, s.pos, s.vel, s.types, s.masses, s.box)
    m_atom = s.masses[s.types]
    # tau -> infinity: the NVE trajectory of the pinned integrator
    pos_n, vel_n, _, _ = oracle_mod.md(*args, 1.0, 6)
    pos_b, vel_b, tb, ta = oracle_mod.md_berendsen(*args, 1.0, 6, 900.0, 900.0, 1e30)
    np.testing.assert_allclose(pos_b, pos_n, rtol=0, atol=1e-12)
    np.testing.assert_allclose(vel_b, vel_n, rtol=0, atol=1e-14)
    # one step: T_after - T_before = (dt/tau)(T_target - T_before), T_before from the NVE step alone
    pos1, vel1, _, _ = oracle_mod.md(*args, 1.0, 1)
    t_nve = oracle_mod.kinetic_temperature(vel1, m_atom)
    _, vel_b1, tb1, ta1 = oracle_mod.md_berendsen(*args, 1.0, 1, 100.0, 900.0, 20.0)     # target of step 1 of 1 = t_stop
    assert tb1[0] == pytest.approx(t_nve, rel=1e-13)
    assert ta1[0] - tb1[0] == pytest.approx((1.0 / 20.0) * (900.0 - t_nve), rel=1e-10)
    np.testing.assert_allclose(vel_b1 / vel1, np.sqrt(ta1[0] / tb1[0]), rtol=1e-12)     # a pure rescale
    # tau = dt: the target is hit exactly; the ramp is linear in the step number
    _, _, tb2, ta2 = oracle_mod.md_berendsen(*args, 1.0, 4, 300.0, 700.0, 1.0)
    np.testing.assert_allclose(ta2, [400.0, 500.0, 600.0, 700.0], rtol=1e-12)


# ------------------------------------------------------------------ triclinic cells (reading A8t)
def _brute_force_images(pos, H, rc):
    """the plain definition: j is a neighbour of i iff some lattice image of j is closer than rc"""
    n = len(pos)
    shifts = np.array([[i, j, k] for i in (-2, -1, 0, 1, 2) for j in (-2, -1, 0, 1, 2) for k in (-2, -1, 0, 1, 2)], dtype=np.float64) @ H
    sets = []
    for i in range(n):
        d = pos[None, :, :] - pos[i][None, None, :] + shifts[:, None, :]
        close = ((d * d).sum(axis=2) < rc * rc).any(axis=0)
        close[i] = False
        sets.append(set(np.nonzero(close)[0].tolist()))
    return sets


def test_triclinic_neighbours_equal_lattice_image_search(oracle_mod):
    cfg = W.get_config(3, cells=(4, 4, 4))
    s = W.make_system(cfg)
    pos, H = W.sheared(s, 0.31, -0.17, 0.23)
    rc = 6.0
    assert W.perpendicular_widths(H).min() >= 2 * rc
    cnt, lst = oracle_mod.neighbors(pos, H, rc)
    want = _brute_force_images(pos, H, rc)
    assert sum(len(w) for w in want) > 50 * len(pos)
    for i in range(len(pos)):
        assert set(lst[i, :cnt[i]].tolist()) == want[i]
    # positions shifted by arbitrary lattice vectors: the same sets
    rng = np.random.default_rng(3)
    pos2 = pos + rng.integers(-3, 4, size=(len(pos), 3)).astype(np.float64) @ H
    cnt2, lst2 = oracle_mod.neighbors(pos2, H, rc)
    for i in range(len(pos)):
        assert set(lst2[i, :cnt2[i]].tolist()) == want[i]


def test_triclinic_description_of_an_orthorhombic_lattice(oracle_mod):
    """The cell (a, b + a, c - 2b) spans the same lattice as (a, b, c): the same periodic structure, so every
    per-atom energy, force and virial must equal the orthorhombic (pinned) result."""
    cfg = W.get_config(3, cells=(3, 3, 3))
    s, p = W.make_system(cfg), W.make_params(cfg, "stress")
    H0 = np.diag(s.box)
    H1 = np.array([H0[0], H0[1] + H0[0], H0[2] - 2 * H0[1]])
    hy = cfg.hyper
    # cutoffs within half the smallest perpendicular width of the skewed cell
    from dataclasses import replace
    w = W.perpendicular_widths(H1).min()
    hy = replace(hy, rc_radial=min(hy.rc_radial, 0.49 * w), rc_angular=min(hy.rc_angular, 0.4 * w))
    e0, f0, w0 = oracle_mod.compute(hy, p, s.pos, s.types, s.box)
    e1, f1, w1 = oracle_mod.compute(hy, p, s.pos, s.types, H1)
    np.testing.assert_allclose(e1, e0, rtol=1e-12, atol=1e-13)
    np.testing.assert_allclose(f1, f0, rtol=1e-10, atol=1e-12)
    np.testing.assert_allclose(w1, w0, rtol=1e-10, atol=1e-12)


def test_triclinic_forces_and_shear_virial_by_finite_differences(oracle_mod):
    cfg = W.get_config(3, cells=(3, 3, 3))
    s, p = W.make_system(cfg), W.make_params(cfg, "stress")
    pos, H = W.sheared(s, 0.12, -0.08, 0.1)
    from dataclasses import replace
    w = W.perpendicular_widths(H).min()
    hy = replace(cfg.hyper, rc_radial=min(cfg.hyper.rc_radial, 0.49 * w), rc_angular=min(cfg.hyper.rc_angular, 0.4 * w))
    E = lambda x, B: oracle_mod.compute(hy, p, x, s.types, B)[0].sum()
    e, f, wv = oracle_mod.compute(hy, p, pos, s.types, H)
    h = 1e-4
    for i, a in ((0, 0), (17, 1), (53, 2)):
        pp, pm = pos.copy(), pos.copy()
        pp[i, a] += h; pm[i, a] -= h
        assert f[i, a] == pytest.approx(-(E(pp, H) - E(pm, H)) / (2 * h), rel=2e-6, abs=1e-8)
    np.testing.assert_allclose(f.sum(axis=0), 0.0, atol=1e-10)
    wtot = wv.sum(axis=0).reshape(3, 3)
    h = 1e-5
    for a, b in ((0, 1), (1, 0), (0, 2), (2, 1), (1, 1)):      # periodic cell: shear strains included
        eps = np.zeros((3, 3)); eps[a, b] = h
        Fp, Fm = (np.eye(3) + eps).T, (np.eye(3) - eps).T
        dE = (E(pos @ Fp, H @ Fp) - E(pos @ Fm, H @ Fm)) / (2 * h)
        assert wtot[a, b] == pytest.approx(-dE, rel=5e-6, abs=1e-8)


# ------------------------------------------------------------------ Langevin NVT (reading A16)
def test_counter_normal_statistics_and_independence(oracle_mod):
    z = np.array([oracle_mod.counter_normal(20220510, c) for c in range(200000)])
    n = len(z)
    assert abs(z.mean()) < 4.0 / np.sqrt(n)
    assert abs(z.var() - 1.0) < 4.0 * np.sqrt(2.0 / n)
    assert abs((z ** 3).mean()) < 4.0 * np.sqrt(15.0 / n)
    assert abs((z ** 4).mean() - 3.0) < 4.0 * np.sqrt(96.0 / n)
    assert abs(np.mean(z[:-1] * z[1:])) < 4.0 / np.sqrt(n)                 # neighbouring counters uncorrelated
    assert abs(np.mean(z[:-3] * z[3:])) < 4.0 / np.sqrt(n)                 # ... and the 3 components of an atom
    # the Kolmogorov distance to the normal distribution
    from scipy import stats
    assert stats.kstest(z, "norm").statistic < 1.63 / np.sqrt(n) * 1.5
    z2 = np.array([oracle_mod.counter_normal(20220511, c) for c in range(50000)])
    assert abs(np.mean(z[:50000] * z2)) < 4.0 / np.sqrt(50000)             # another seed: another stream
    assert oracle_mod.counter_normal(7, 12345) == oracle_mod.counter_normal(7, 12345)


def test_langevin_limits_and_free_particle_relaxation(oracle_mod):
    cfg = W.get_config(3, cells=(3, 3, 3))
    s, p = W.make_system(cfg), W.make_params(cfg, "stress")
    args = (cfg.hyper, p, s.pos, s.vel, s.types, s.masses, s.box)
    m_atom = s.masses[s.types]
    # tau -> infinity: c1 = 1, c2 = 0: the pinned NVE trajectory
    pos_n, vel_n, _, _ = oracle_mod.md(*args, 1.0, 4)
    pos_l, vel_l, _ = oracle_mod.md_langevin(*args, 1.0, 4, 900.0, 900.0, 1e30, seed=5)
    np.testing.assert_allclose(pos_l, pos_n, rtol=0, atol=1e-12)
    np.testing.assert_allclose(vel_l, vel_n, rtol=0, atol=1e-14)
    # one half step: exactly c1 v + c2 sigma R with the documented counters
    c1 = 0.8
    v1 = oracle_mod.langevin_half_step(s.vel, m_atom, 500.0, c1, seed=9, draw=3)
    n = len(m_atom)
    for i, a in ((0, 0), (5, 2), (n - 1, 1)):
        sig = np.sqrt(oracle_mod.KB_EV_PER_K * 500.0 / m_atom[i] * oracle_mod.ACC_CONV)
        want = c1 * s.vel[i, a] + np.sqrt(1 - c1 * c1) * sig * oracle_mod.counter_normal(9, (3 * n + i) * 3 + a)
        assert v1[i, a] == pytest.approx(want, rel=1e-14)
    # free particles (zero model): E[T_{k+1}] = c1^4 T_k + (1 - c1^4) T0 per full step (two half steps);
    # the kinetic temperature of 3N independent components fluctuates by T sqrt(2 / 3N)
    cfg0 = W.get_config(1, cells=(5, 5, 5))
    s0, p0 = W.make_system(cfg0), _zero_model(cfg0)
    dt, tau, T0, nst = 2.0, 8.0, 900.0, 10
    _, _, temps = oracle_mod.md_langevin(cfg0.hyper, p0, s0.pos, s0.vel, s0.types, s0.masses, s0.box, dt, nst, T0, T0, tau, seed=1)
    c4 = np.exp(-dt / (2 * tau)) ** 4
    want = T0 + (cfg0.temperature - T0) * c4 ** np.arange(1, nst + 1)
    assert (np.abs(temps - want) < 5.0 * want * np.sqrt(2.0 / (3 * len(s0.pos)))).all()
    assert temps[-1] > 2.5 * cfg0.temperature


# ------------------------------------------------------------------ loss terms of Eq. (33) (reading A17)
def test_loss_terms_hand_case_and_zero(oracle_mod):
    e = np.array([1.0, 3.0]); f = np.array([[1.0, 0.0, 0.0], [0.0, 2.0, 0.0]])
    w = np.zeros((2, 9)); w[0, 0] = 2.0; w[1, 0] = 4.0; w[0, 1] = 1.0; w[1, 5] = -2.0; w[0, 6] = 6.0
    ft = np.zeros((2, 3)); wt = np.zeros(6)
    le, lf, lv = oracle_mod.loss_terms(e, f, w, 1.5, ft, wt)
    assert le == pytest.approx(0.5)                                     # |4/2 - 1.5|
    assert lf == pytest.approx(np.sqrt(5.0 / 6.0))                      # (1 + 4) / (3 * 2)
    # per-atom totals: xx 3, xy 0.5, yz -1, zx 3; yy = zz = 0
    assert lv == pytest.approx(np.sqrt((9.0 + 0.25 + 1.0 + 9.0) / 6.0))
    le, lf, lv = oracle_mod.loss_terms(e, f, w, 2.0, f, np.array([3.0, 0.0, 0.0, 0.5, -1.0, 3.0]))
    assert (le, lf, lv) == (0.0, 0.0, 0.0)
    # Eq. (30) parameter count and the two norms
    cfg = W.get_config(2)
    p = W.make_params(cfg)
    h = cfg.hyper
    npar = (h.n_des + 2) * h.n_neurons + 1 + h.n_types ** 2 * (h.NR * h.KR + h.NA * h.KA)
    z = np.concatenate([np.asarray(a, np.float64).ravel() for a in (p.c_radial, p.c_angular, p.w0, p.b0, p.w1, p.b1)])
    assert len(z) == npar
    l1, l2 = oracle_mod.regularisation_terms(p)
    assert 0.0 < l1 <= l2 + 1e-15                                        # mean |z| <= rms z (Cauchy-Schwarz)
    # hand case, Eq. (33) last two terms: the six arrays hold z = {3, -4 | 0 | 12 | -5 | 0 | 0},
    # N_par = 7: sum |z| / N_par = 24 / 7;  sqrt(sum z^2 / N_par) = sqrt((9 + 16 + 144 + 25) / 7) = sqrt(194 / 7)
    import types
    hand = types.SimpleNamespace(c_radial=np.array([3.0, -4.0], np.float32), c_angular=np.array([0.0], np.float32),
                                 w0=np.array([[12.0]], np.float32), b0=np.array([-5.0], np.float32),
                                 w1=np.array([0.0], np.float32), b1=np.array([0.0], np.float32))
    l1, l2 = oracle_mod.regularisation_terms(hand)
    assert l1 == pytest.approx(3.4285714285714284, rel=1e-15) and l2 == pytest.approx(5.264435935053794, rel=1e-15)
    # a sign flip of every parameter changes neither; scaling by 3 scales both by 3
    flip = types.SimpleNamespace(**{k: -3.0 * v for k, v in vars(hand).items()})
    l1f, l2f = oracle_mod.regularisation_terms(flip)
    assert l1f == pytest.approx(10.285714285714286, rel=1e-15) and l2f == pytest.approx(15.793307805161383, rel=1e-15)


# ------------------------------------------------------------------ cells of any size: lattice images (reading A18)
def _image_counts(pos, H, rc, reach=3):
    """the plain definition in numpy: ordered entries (j, N) != (i, 0) with |r_j + N H - r_i| < rc"""
    shifts = np.array([[a, b, c] for a in range(-reach, reach + 1) for b in range(-reach, reach + 1)
                       for c in range(-reach, reach + 1)], dtype=np.float64)
    sv = shifts @ H
    zero = int(np.flatnonzero((shifts == 0).all(axis=1))[0])
    out = np.zeros(len(pos), dtype=np.int64)
    for i in range(len(pos)):
        d = pos[None, :, :] - pos[i][None, None, :] + sv[:, None, :]
        close = (d * d).sum(axis=2) < rc * rc
        close[zero, i] = False
        out[i] = close.sum()
    return out


def _small_and_super(idx, cells, reps, tilt=None, kind="stress"):
    """a small periodic cell and the (rx, ry, rz) supercell of the SAME infinite structure"""
    cfg = W.get_config(idx, cells)
    s, p = W.make_system(cfg), W.make_params(cfg, kind)
    pos, H = (s.pos, np.diag(s.box)) if tilt is None else W.sheared(s, *tilt)
    rx, ry, rz = reps
    offs = np.array([[a, b, c] for a in range(rx) for b in range(ry) for c in range(rz)], dtype=np.float64) @ H
    big = (pos[None, :, :] + offs[:, None, :]).reshape(-1, 3)
    Hbig = H * np.array([[rx], [ry], [rz]], dtype=np.float64)
    return cfg, p, pos, s.types, H, big, np.tile(s.types, len(offs)), Hbig, len(offs)


@pytest.mark.parametrize("idx,cells,reps,tilt", [
    (3, (2, 2, 2), (2, 2, 2), None),                   # fcc alloy, 32 atoms, 7.2 A cell: rc_R = 5 > L/2
    (3, (1, 1, 1), (4, 3, 3), None),                   # 4 atoms in a 3.6 A cell: every atom sees images of itself
    (2, (1, 1, 2), (2, 2, 1), None),                   # rock salt, rc_R = 6, 6.46 x 6.46 x 12.92 A
    (3, (2, 2, 1), (2, 2, 4), (0.21, -0.13, 0.17)),    # sheared small cell
])
def test_image_sum_equals_the_supercell(oracle_mod, idx, cells, reps, tilt):
    """A cell thinner than 2 r_c evaluated with lattice images == the same crystal described by a supercell that
    the pinned minimum-image path can handle: every atom's U_i, F_i, W_i and q, Fp, S equal those of its copies."""
    cfg, p, pos, types, H, big, tbig, Hbig, ncopy = _small_and_super(idx, cells, reps, tilt)
    hy = cfg.hyper
    assert W.perpendicular_widths(H).min() < 2 * hy.rc_radial <= W.perpendicular_widths(Hbig).min()
    e, f, w, q, fp, S = oracle_mod.compute_images(hy, p, pos, types, H, want_internals=True)
    eb, fb, wb, qb, fpb, Sb = oracle_mod.compute(hy, p, big, tbig, Hbig, want_internals=True)
    n = len(pos)
    for c in range(ncopy):
        sl = slice(c * n, (c + 1) * n)
        np.testing.assert_allclose(eb[sl], e, rtol=1e-12, atol=1e-13)
        np.testing.assert_allclose(fb[sl], f, rtol=1e-10, atol=1e-12)
        np.testing.assert_allclose(wb[sl], w, rtol=1e-10, atol=1e-12)
        np.testing.assert_allclose(qb[sl], q, rtol=1e-12, atol=1e-14)
        np.testing.assert_allclose(Sb[sl], S, rtol=1e-11, atol=1e-13)
    assert np.abs(f).max() > 1e-3 and np.abs(w).max() > 1e-3
    # neighbour entries, images counted: the numpy definition
    for rc in (hy.rc_radial, hy.rc_angular):
        assert np.array_equal(oracle_mod.count_images(pos, H, rc), _image_counts(pos, H, rc))
    # a cell wide enough for the minimum image: both paths are the same function
    e2, f2, w2 = oracle_mod.compute_images(hy, p, big, tbig, Hbig)
    np.testing.assert_allclose(e2, eb, rtol=1e-13, atol=1e-14)
    np.testing.assert_allclose(f2, fb, rtol=1e-11, atol=1e-13)
    np.testing.assert_allclose(w2, wb, rtol=1e-11, atol=1e-13)


def test_image_sum_forces_and_virial_by_finite_differences(oracle_mod):
    """F = -dE/dr (moving an atom moves all its images) and sum_i W_i = -dE/d(strain) in a cell with self-images."""
    cfg = W.get_config(3, (1, 1, 2))
    s, p = W.make_system(cfg), W.make_params(cfg, "stress")
    pos, H = W.sheared(s, 0.12, -0.07, 0.05)
    hy = cfg.hyper
    etot = lambda x, h: oracle_mod.compute_images(hy, p, x, s.types, h)[0].sum()
    e, f, w = oracle_mod.compute_images(hy, p, pos, s.types, H)
    hstep = 1e-5
    for i, a in ((0, 0), (3, 1), (5, 2)):
        xp, xm = pos.copy(), pos.copy()
        xp[i, a] += hstep; xm[i, a] -= hstep
        assert f[i, a] == pytest.approx(-(etot(xp, H) - etot(xm, H)) / (2 * hstep), rel=2e-6, abs=1e-8)
    assert np.abs(f.sum(axis=0)).max() < 1e-10
    wsum = w.sum(axis=0).reshape(3, 3)
    for a, b in ((0, 0), (1, 1), (2, 2), (0, 1), (1, 2), (2, 0)):
        eps = np.zeros((3, 3)); eps[a, b] = hstep
        Fp_, Fm_ = np.eye(3) + eps, np.eye(3) - eps          # r -> r F (row vectors): r^b picks up eps * r^a
        de = (etot(pos @ Fp_, H @ Fp_) - etot(pos @ Fm_, H @ Fm_)) / (2 * hstep)
        assert wsum[a, b] == pytest.approx(-de, rel=2e-6, abs=1e-8)


def test_loss_terms_batch_hand_case(oracle_mod):
    """Eq. (33) with N_str = 2, numbers worked by hand."""
    e = [np.array([1.0, 3.0]), np.array([2.0, 2.0, 5.0])]                 # per-atom energies 2 and 3
    f = [np.array([[1.0, 0.0, 0.0], [0.0, 2.0, 0.0]]), np.array([[0.0, 0.0, 2.0], [0.0, 0.0, 0.0], [1.0, 1.0, 0.0]])]
    w = [np.zeros((2, 9)), np.zeros((3, 9))]
    w[0][0, 0] = 2.0; w[0][1, 0] = 4.0; w[0][0, 1] = 1.0            # structure 0 per atom: xx 3, xy 0.5
    w[1][0, 4] = 3.0; w[1][2, 5] = -6.0; w[1][1, 6] = 9.0           # structure 1 per atom: yy 1, yz -2, zx 3
    ft = [np.zeros((2, 3)), np.zeros((3, 3))]
    le, lf, lv = oracle_mod.loss_terms_batch(e, f, w, [1.5, 3.5], ft, [np.zeros(6), np.zeros(6)])
    assert le == pytest.approx(np.sqrt((0.25 + 0.25) / 2))                      # (2 - 1.5)^2, (3 - 3.5)^2
    assert lf == pytest.approx(np.sqrt((1 + 4 + 4 + 1 + 1) / (3 * 5)))          # N = 5 atoms
    assert lv == pytest.approx(np.sqrt((9 + 0.25 + 1 + 4 + 9) / (6 * 2)))
    # one structure: the N_str = 1 function (pinned above)
    one = oracle_mod.loss_terms(e[1], f[1], w[1], 3.5, ft[1], np.zeros(6))
    assert oracle_mod.loss_terms_batch(e[1:], f[1:], w[1:], [3.5], ft[1:], [np.zeros(6)]) == pytest.approx(one)
    # exact targets: zero
    tw = [np.array([3.0, 0, 0, 0.5, 0, 0]), np.array([0, 1.0, 0, 0, -2.0, 3.0])]
    assert oracle_mod.loss_terms_batch(e, f, w, [2.0, 3.0], f, tw) == (0.0, 0.0, 0.0)
