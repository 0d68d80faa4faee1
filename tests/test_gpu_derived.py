"""GPU-vs-oracle parity of the derived outputs, through the C ABI (-m gpu):
the latent-space vector (nep_get_latent) and the heat current (Eqs. 25-26, nep_heat_current).

Tolerances, derived from the arithmetic: a latent component is w1_mu tanh(a) with a an fp32 dot product of
D terms, so |d latent| <= |w1_mu| (|da| + eps) with |da| ~ D eps max|w0 q|: asserted as 2e-5 of the largest
|latent| component (the same block-relative bar the descriptors use).  The heat current is a contraction
of the fp32-accumulated virial (parity bar 1e-4 relative, reading A14) with fp64 velocities in fp64:
per atom ||dJ_i|| <= 1e-4 max(||W_i||, median ||W||) ||v_i||; the contraction itself must be exact fp64 on
the GPU's own virial (1e-14), the total equal to the fp64 sum of the GPU's J_i (1e-12), and within
1e-4 (sum_i ||J_i|| / sqrt(n) + ||J||) of the oracle's total (independent per-atom errors add in quadrature).
"""
from dataclasses import replace

import numpy as np
import pytest

import workloads as W

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def pkg():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2205_10046_b200 as p
    p.load_library()
    return p


CASES = [(0, None, 0.0), (2, (4, 4, 3), 1.0), (3, (7, 6, 5), 1.0), (4, (9, 8, 7), 1.0)]


@pytest.mark.parametrize("kind", ["baseline", "stress"])
@pytest.mark.parametrize("idx,cells,skin", CASES)
def test_latent_vector(pkg, oracle_mod, idx, cells, skin, kind):
    cfg = W.get_config(idx, cells) if cells else W.get_config(idx)
    s, p = W.make_system(cfg), W.make_params(cfg, kind)
    nep = pkg.NEP(cfg.hyper, p, s.masses, device=0)
    pos = torch.tensor(s.pos, device="cuda:0")
    nep.nep_neighbors(pos, torch.tensor(s.types, device="cuda:0"), s.box, skin)
    e, f, w = nep.nep_compute(pos)
    lat = nep.nep_get_latent().cpu().numpy().astype(np.float64)
    eo, fo, wo, qo, fpo, So = oracle_mod.compute(cfg.hyper, p, s.pos, s.types, s.box, want_internals=True)
    lo = oracle_mod.latent(p, qo)
    assert lat.shape == lo.shape == (len(s.pos), cfg.hyper.n_neurons)
    assert np.abs(lat - lo).max() <= 2e-5 * np.abs(lo).max()
    # the defining property, on the GPU's own numbers: sum_mu latent - b1 = U_i
    assert np.abs(lat.sum(axis=1) - float(p.b1[0]) - e.cpu().numpy()).max() <= 1e-5
    nep.close()


@pytest.mark.parametrize("kind", ["baseline", "stress"])
@pytest.mark.parametrize("idx,cells,skin", CASES)
def test_heat_current(pkg, oracle_mod, idx, cells, skin, kind):
    cfg = W.get_config(idx, cells) if cells else W.get_config(idx)
    s, p = W.make_system(cfg), W.make_params(cfg, kind)
    nep = pkg.NEP(cfg.hyper, p, s.masses, device=0)
    pos, vel = torch.tensor(s.pos, device="cuda:0"), torch.tensor(s.vel, device="cuda:0")
    nep.nep_neighbors(pos, torch.tensor(s.types, device="cuda:0"), s.box, skin)
    e, f, w = nep.nep_compute(pos)
    ja, jt = nep.nep_heat_current(vel)
    ja, jt, wg = ja.cpu().numpy(), jt.cpu().numpy(), w.cpu().numpy()
    eo, fo, wo = oracle_mod.compute(cfg.hyper, p, s.pos, s.types, s.box)
    jo, jto = oracle_mod.heat_current(wo, s.vel)
    wn = np.linalg.norm(wo, axis=1)
    vn = np.linalg.norm(s.vel, axis=1)
    bound = 1e-4 * np.maximum(wn, np.median(wn)) * vn
    assert (np.linalg.norm(ja - jo, axis=1) <= bound + 1e-18).all()
    # the contraction itself is exact fp64 on the GPU's own virial (same summation order as Eq. 25 written out)
    jself, _ = oracle_mod.heat_current(wg, s.vel)
    assert np.abs(ja - jself).max() <= 1e-14 * max(np.abs(jself).max(), 1e-300)
    # total: fixed-order fp64 reduction of the GPU's J_i; against the oracle within the virial bar
    assert np.abs(jt - ja.sum(axis=0)).max() <= 1e-12 * np.abs(ja).sum()
    assert np.linalg.norm(jt - jto) <= 1e-4 * np.linalg.norm(jo, axis=1).sum() / np.sqrt(len(jo)) + 1e-4 * np.linalg.norm(jto)
    nep.close()


def test_heat_current_after_md_and_reproducible(pkg, oracle_mod):
    """After md_step the virial belongs to the final positions and vel_dev holds the matching velocities;
    two calls give bitwise identical totals (fixed reduction order)."""
    cfg = W.get_config(3, (7, 6, 5))
    s, p = W.make_system(cfg), W.make_params(cfg, "stress")
    nep = pkg.NEP(cfg.hyper, p, s.masses, device=0)
    pos, vel = torch.tensor(s.pos, device="cuda:0"), torch.tensor(s.vel, device="cuda:0")
    nep.nep_neighbors(pos, torch.tensor(s.types, device="cuda:0"), s.box, 1.0)
    nep.md_step(pos, vel, cfg.dt_fs, 5, cfg.rebuild_every, 1.0)
    ja1, jt1 = nep.nep_heat_current(vel)
    ja2, jt2 = nep.nep_heat_current(vel)
    assert torch.equal(jt1, jt2) and torch.equal(ja1, ja2)
    eo, fo, wo = oracle_mod.compute(cfg.hyper, p, pos.cpu().numpy(), s.types, s.box)
    jo, jto = oracle_mod.heat_current(wo, vel.cpu().numpy())
    wn = np.linalg.norm(wo, axis=1)
    bound = 1e-4 * np.maximum(wn, np.median(wn)) * np.linalg.norm(vel.cpu().numpy(), axis=1)
    assert (np.linalg.norm(ja1.cpu().numpy() - jo, axis=1) <= bound + 1e-18).all()
    nep.close()


def test_derived_outputs_need_an_evaluation(pkg):
    cfg = W.get_config(0)
    s, p = W.make_system(cfg), W.make_params(cfg)
    nep = pkg.NEP(cfg.hyper, p, s.masses, device=0)
    pos = torch.tensor(s.pos, device="cuda:0")
    nep.nep_neighbors(pos, torch.tensor(s.types, device="cuda:0"), s.box, 0.0)
    with pytest.raises(pkg.NepError) as ei:
        nep.nep_get_latent()
    assert ei.value.status == -5
    with pytest.raises(pkg.NepError) as ei:
        nep.nep_heat_current(torch.tensor(s.vel, device="cuda:0"))
    assert ei.value.status == -5
    nep.close()


# ------------------------------------------------------------------ Berendsen NVT
@pytest.mark.parametrize("idx,cells,skin,kind", [(0, None, 0.0, "baseline"), (3, (7, 6, 5), 1.0, "stress"), (2, (4, 4, 3), 1.0, "stress")])
def test_berendsen_nvt_trajectory(pkg, oracle_mod, idx, cells, skin, kind):
    """10 thermostatted steps with a temperature ramp against the oracle's md_berendsen: fp64 state, fp32 forces.
    Tolerances as the NVE trajectory test (1e-7 A, 1e-9 A/fs) scaled by the stress set's stronger forces; the
    temperature before the last rescale and its lambda to 1e-9 relative (a fixed-order fp64 reduction)."""
    cfg = W.get_config(idx, cells) if cells else W.get_config(idx)
    s, p = W.make_system(cfg), W.make_params(cfg, kind)
    nep = pkg.NEP(cfg.hyper, p, s.masses, device=0)
    pos, vel = torch.tensor(s.pos, device="cuda:0"), torch.tensor(s.vel, device="cuda:0")
    nep.nep_neighbors(pos, torch.tensor(s.types, device="cuda:0"), s.box, skin)
    n_steps, t0, t1, tau = 10, 500.0, 800.0, 25.0
    nep.md_step_nvt_berendsen(pos, vel, cfg.dt_fs, n_steps, cfg.rebuild_every, skin, t0, t1, tau)
    po, vo, tb, ta = oracle_mod.md_berendsen(cfg.hyper, p, s.pos, s.vel, s.types, s.masses, s.box, cfg.dt_fs, n_steps, t0, t1, tau)
    tol = 1.0 if kind == "baseline" else 30.0
    assert np.abs(pos.cpu().numpy() - po).max() < 1e-7 * tol
    assert np.abs(vel.cpu().numpy() - vo).max() < 1e-9 * tol
    t_last, lam = nep.nep_last_temperature()
    assert t_last == pytest.approx(tb[-1], rel=1e-7)
    assert lam == pytest.approx(np.sqrt(ta[-1] / tb[-1]), rel=1e-8)
    m = s.masses[s.types]
    assert oracle_mod.kinetic_temperature(vel.cpu().numpy(), m) == pytest.approx(ta[-1], rel=1e-7)
    nep.close()


def test_berendsen_nvt_reaches_target_and_rejects_bad_arguments(pkg, oracle_mod):
    cfg = W.get_config(3, (7, 6, 5))
    s, p = W.make_system(cfg), W.make_params(cfg, "stress")
    nep = pkg.NEP(cfg.hyper, p, s.masses, device=0)
    pos, vel = torch.tensor(s.pos, device="cuda:0"), torch.tensor(s.vel, device="cuda:0")
    nep.nep_neighbors(pos, torch.tensor(s.types, device="cuda:0"), s.box, 1.0)
    with pytest.raises(pkg.NepError) as ei:
        nep.nep_last_temperature()
    assert ei.value.status == -5
    # tau < dt would overshoot the target (and lambda^2 could go negative): rejected
    for bad in ((300.0, 300.0, 0.0), (-1.0, 300.0, 10.0), (300.0, -5.0, 10.0), (300.0, 300.0, 0.5)):
        with pytest.raises(pkg.NepError) as ei:
            nep.md_step_nvt_berendsen(pos, vel, 1.0, 1, 10, 1.0, *bad)
        assert ei.value.status == -1
    # tau = dt: every step lands exactly on its target; 150 steps with tau = 20 fs hold 600 K within 10 % (the random model keeps exchanging kinetic and potential energy)
    nep.md_step_nvt_berendsen(pos, vel, 1.0, 3, 10, 1.0, 600.0, 600.0, 1.0)
    m = s.masses[s.types]
    assert oracle_mod.kinetic_temperature(vel.cpu().numpy(), m) == pytest.approx(600.0, rel=1e-10)
    nep.md_step_nvt_berendsen(pos, vel, 1.0, 150, 10, 1.0, 600.0, 600.0, 20.0)
    assert abs(oracle_mod.kinetic_temperature(vel.cpu().numpy(), m) - 600.0) < 60.0
    assert nep.nep_max_displacement() < 0.5
    nep.close()


# ------------------------------------------------------------------ triclinic cells
TRI_CASES = [
    (1, (5, 5, 4), 1.0, (0.21, -0.13, 0.17), "baseline"),      # diamond, 1 species
    (2, (4, 4, 4), 0.5, (-0.18, 0.11, 0.09), "stress"),        # rock salt, 2 species, rc 6/4
    (3, (8, 7, 7), 1.0, (0.25, 0.2, -0.22), "stress"),         # fcc alloy, 5 species
    (4, (10, 9, 9), 0.5, (0.15, -0.1, 0.12), "stress"),        # bcc, rc 6/5, two angular passes
]


def _tri_system(idx, cells, tilt):
    cfg = W.get_config(idx, cells)
    s = W.make_system(cfg)
    pos, H = W.sheared(s, *tilt)
    return cfg, s, pos, H


@pytest.mark.parametrize("idx,cells,skin,tilt,kind", TRI_CASES)
def test_triclinic_neighbours_and_efw(pkg, oracle_mod, idx, cells, skin, tilt, kind):
    """Sheared replicas of the configurations: neighbour sets bit-exact against the oracle's reading A8t,
    E / F / W within north_star's tolerances."""
    cfg, s, pos, H = _tri_system(idx, cells, tilt)
    assert W.perpendicular_widths(H).min() >= 2 * (cfg.hyper.rc_radial + skin)
    p = W.make_params(cfg, kind)
    nep = pkg.NEP(cfg.hyper, p, s.masses, device=0)
    dpos = torch.tensor(pos, device="cuda:0")
    nep.nep_neighbors(dpos, torch.tensor(s.types, device="cuda:0"), H, skin)
    for which, rc in ((0, cfg.hyper.rc_radial), (1, cfg.hyper.rc_angular)):
        cnt, lst = nep.nep_get_neighbors(which)
        ocnt, olst = oracle_mod.neighbors(pos, H, rc + skin)
        cnt, lst = cnt.cpu().numpy(), lst.cpu().numpy()
        assert np.array_equal(cnt, ocnt)
        for i in range(len(pos)):
            assert set(lst[i, :cnt[i]].tolist()) == set(olst[i, :ocnt[i]].tolist())
    e, f, w = nep.nep_compute(dpos)
    eo, fo, wo = oracle_mod.compute(cfg.hyper, p, pos, s.types, H)
    e, f, w = e.cpu().numpy(), f.cpu().numpy(), w.cpu().numpy()
    assert np.abs(e - eo).max() <= 1e-5
    fn = np.linalg.norm(fo, axis=1, keepdims=True)
    assert (np.abs(f - fo) <= np.maximum(1e-4, 1e-4 * fn)).all()
    assert np.abs(f - fo).max() <= 1e-4 * max(np.abs(fo).max(), 1e-6)
    wn = np.linalg.norm(wo, axis=1)
    assert (np.linalg.norm(w - wo, axis=1) <= 1e-4 * np.maximum(wn, np.median(wn))).all()
    assert np.linalg.norm(w.sum(axis=0) - wo.sum(axis=0)) <= 1e-4 * np.linalg.norm(wo.sum(axis=0))
    nep.close()


def test_triclinic_md_and_equivalent_cell(pkg, oracle_mod):
    """10 NVE steps in a sheared cell with list rebuilds follow the oracle; and the skewed description
    (a, b + a, c) of an orthorhombic crystal gives the orthorhombic forces (positions far outside [0,1)^3 in
    fractional coordinates included)."""
    cfg, s, pos, H = _tri_system(3, (8, 7, 7), (0.25, 0.2, -0.22))
    p = W.make_params(cfg, "stress")
    nep = pkg.NEP(cfg.hyper, p, s.masses, device=0)
    dpos, dvel = torch.tensor(pos, device="cuda:0"), torch.tensor(s.vel, device="cuda:0")
    nep.nep_neighbors(dpos, torch.tensor(s.types, device="cuda:0"), H, 1.0)
    nep.md_step(dpos, dvel, 1.0, 10, 3, 1.0)
    po, vo, ep, ek = oracle_mod.md(cfg.hyper, p, pos, s.vel, s.types, s.masses, H, 1.0, 10)
    assert np.abs(dpos.cpu().numpy() - po).max() < 3e-6
    assert np.abs(dvel.cpu().numpy() - vo).max() < 3e-8
    nep.close()

    cfg = W.get_config(3, (8, 8, 8))
    s = W.make_system(cfg)
    H0 = np.diag(s.box)
    H1 = np.array([H0[0], H0[1] + H0[0], H0[2]])
    assert W.perpendicular_widths(H1).min() >= 2 * (cfg.hyper.rc_radial + 0.5)
    rng = np.random.default_rng(11)
    pos1 = s.pos + rng.integers(-2, 3, size=s.pos.shape).astype(np.float64) @ H0      # any lattice shifts
    out = []
    for pp, HH in ((s.pos, s.box), (pos1, H1)):
        nep = pkg.NEP(cfg.hyper, p, s.masses, device=0)
        dp = torch.tensor(pp, device="cuda:0")
        nep.nep_neighbors(dp, torch.tensor(s.types, device="cuda:0"), HH, 0.5)
        e, f, w = nep.nep_compute(dp)
        out.append((e.cpu().numpy(), f.cpu().numpy(), w.cpu().numpy()))
        nep.close()
    assert np.abs(out[0][0] - out[1][0]).max() <= 2e-6
    assert np.abs(out[0][1] - out[1][1]).max() <= 2e-5 * np.abs(out[0][1]).max()
    assert np.abs(out[0][2] - out[1][2]).max() <= 2e-5 * np.abs(out[0][2]).max()


# ------------------------------------------------------------------ Langevin NVT (reading A16)
@pytest.mark.parametrize("idx,cells,skin,kind", [(0, None, 0.0, "baseline"), (3, (7, 6, 5), 1.0, "stress")])
def test_langevin_nvt_trajectory(pkg, oracle_mod, idx, cells, skin, kind):
    """Same seed and counters on both sides: the thermostatted trajectories agree like the NVE ones (the
    normal deviates differ by fp64 round-off of log / cos only).  Splitting the run over two calls with
    first_step continues the same random stream."""
    cfg = W.get_config(idx, cells) if cells else W.get_config(idx)
    s, p = W.make_system(cfg), W.make_params(cfg, kind)
    n_steps, t0, t1, tau, seed = 8, 400.0, 700.0, 40.0, 20220510
    po, vo, temps = oracle_mod.md_langevin(cfg.hyper, p, s.pos, s.vel, s.types, s.masses, s.box, cfg.dt_fs, n_steps, t0, t1, tau, seed)
    tol = 1.0 if kind == "baseline" else 30.0
    nep = pkg.NEP(cfg.hyper, p, s.masses, device=0)
    pos, vel = torch.tensor(s.pos, device="cuda:0"), torch.tensor(s.vel, device="cuda:0")
    nep.nep_neighbors(pos, torch.tensor(s.types, device="cuda:0"), s.box, skin)
    nep.md_step_nvt_langevin(pos, vel, cfg.dt_fs, n_steps, cfg.rebuild_every, skin, t0, t1, tau, seed)
    assert np.abs(pos.cpu().numpy() - po).max() < 1e-7 * tol
    assert np.abs(vel.cpu().numpy() - vo).max() < 1e-9 * tol
    m = s.masses[s.types]
    assert oracle_mod.kinetic_temperature(vel.cpu().numpy(), m) == pytest.approx(temps[-1], rel=1e-6)
    nep.close()
    # two calls of 4 steps with a constant target == one call of 8 (first_step continues the counters)
    ref = oracle_mod.md_langevin(cfg.hyper, p, s.pos, s.vel, s.types, s.masses, s.box, cfg.dt_fs, 8, 500.0, 500.0, tau, seed)
    nep = pkg.NEP(cfg.hyper, p, s.masses, device=0)
    pos, vel = torch.tensor(s.pos, device="cuda:0"), torch.tensor(s.vel, device="cuda:0")
    nep.nep_neighbors(pos, torch.tensor(s.types, device="cuda:0"), s.box, skin)
    nep.md_step_nvt_langevin(pos, vel, cfg.dt_fs, 4, cfg.rebuild_every, skin, 500.0, 500.0, tau, seed, 0)
    nep.md_step_nvt_langevin(pos, vel, cfg.dt_fs, 4, cfg.rebuild_every, skin, 500.0, 500.0, tau, seed, 4)
    assert np.abs(pos.cpu().numpy() - ref[0]).max() < 1e-7 * tol
    assert np.abs(vel.cpu().numpy() - ref[1]).max() < 1e-9 * tol
    nep.close()


def test_langevin_normal_deviates_and_equilibrium(pkg, oracle_mod):
    """tau << dt resamples every velocity: v = sqrt(k_B T / m) R exactly, which exposes the device generator
    deviate by deviate against the oracle's; and a long run samples the target temperature."""
    cfg = W.get_config(3, (7, 6, 5))
    s, p = W.make_system(cfg), W.make_params(cfg, "stress")
    nep = pkg.NEP(cfg.hyper, p, s.masses, device=0)
    pos, vel = torch.tensor(s.pos, device="cuda:0"), torch.tensor(s.vel, device="cuda:0")
    nep.nep_neighbors(pos, torch.tensor(s.types, device="cuda:0"), s.box, 1.0)
    n, m = len(s.pos), s.masses[s.types]
    nep.md_step_nvt_langevin(pos, vel, 1.0, 1, 10, 1.0, 650.0, 650.0, 1e-3, 77, 5)     # c1 = exp(-500) = 0
    sig = np.sqrt(oracle_mod.KB_EV_PER_K * 650.0 / m * oracle_mod.ACC_CONV)
    z = vel.cpu().numpy() / sig[:, None]
    for i, a in ((0, 0), (1, 2), (417, 1), (n - 1, 2)):
        assert z[i, a] == pytest.approx(oracle_mod.counter_normal(77, ((2 * 5 + 1) * n + i) * 3 + a), rel=1e-12, abs=1e-14)
    assert abs(z.mean()) < 4.0 / np.sqrt(3 * n) and abs(z.var() - 1.0) < 4.0 * np.sqrt(2.0 / (3 * n))
    for bad in ((300.0, 300.0, 0.0, 1, 0), (-1.0, 300.0, 10.0, 1, 0), (300.0, 300.0, 10.0, 1, -1)):
        with pytest.raises(pkg.NepError) as ei:
            nep.md_step_nvt_langevin(pos, vel, 1.0, 1, 10, 1.0, *bad)
        assert ei.value.status == -1
    nep.md_step_nvt_langevin(pos, vel, 1.0, 200, 10, 1.0, 650.0, 650.0, 25.0, 78, 6)
    t_end = oracle_mod.kinetic_temperature(vel.cpu().numpy(), m)
    assert abs(t_end - 650.0) < 6.0 * 650.0 * np.sqrt(2.0 / (3 * n)) + 30.0
    nep.close()


# ------------------------------------------------------------------ parameter populations (one-structure slice)
@pytest.mark.parametrize("idx,cells,skin", [(0, None, 0.0), (3, (7, 6, 5), 1.0), (4, (9, 8, 7), 0.5)])
def test_population_of_parameter_sets(pkg, oracle_mod, idx, cells, skin):
    """Six parameter sets (an evolution-strategy population, one of them the NEP2 pattern c_nk = delta_nk c_n)
    evaluated at the same positions with one list filter: each member against the oracle; then
    nep_set_parameters + nep_compute reproduces a member bit for bit."""
    cfg = W.get_config(idx, cells) if cells else W.get_config(idx)
    s = W.make_system(cfg)
    members = W.make_population(cfg, 5, 0.15)
    members.append(W.nep2_pattern(members[0]))
    nep = pkg.NEP(cfg.hyper, members[3], s.masses, device=0)
    pos = torch.tensor(s.pos, device="cuda:0")
    nep.nep_neighbors(pos, torch.tensor(s.types, device="cuda:0"), s.box, skin)
    e, f, w = nep.nep_compute_population(pos, members)
    e, f, w = e.cpu().numpy(), f.cpu().numpy(), w.cpu().numpy()
    assert np.abs(e[0] - e[1]).max() > 1e-4                      # the members do differ
    for m, p in enumerate(members):
        eo, fo, wo = oracle_mod.compute(cfg.hyper, p, s.pos, s.types, s.box)
        assert np.abs(e[m] - eo).max() <= 1e-5
        fn = np.linalg.norm(fo, axis=1, keepdims=True)
        assert (np.abs(f[m] - fo) <= np.maximum(1e-4, 1e-4 * fn)).all()
        wn = np.linalg.norm(wo, axis=1)
        assert (np.linalg.norm(w[m] - wo, axis=1) <= 1e-4 * np.maximum(wn, np.median(wn))).all()
    nep.nep_set_parameters(members[2])
    e2, f2, w2 = nep.nep_compute(pos)
    assert np.array_equal(e2.cpu().numpy(), e[2]) and np.array_equal(f2.cpu().numpy(), f[2]) and np.array_equal(w2.cpu().numpy(), w[2])
    # and MD continues with the new model
    vel = torch.tensor(s.vel, device="cuda:0")
    nep.md_step(pos, vel, cfg.dt_fs, 2, cfg.rebuild_every, skin)
    po, vo, _, _ = oracle_mod.md(cfg.hyper, members[2], s.pos, s.vel, s.types, s.masses, s.box, cfg.dt_fs, 2)
    assert np.abs(pos.cpu().numpy() - po).max() < 3e-6
    nep.close()


def test_loss_terms_of_a_population(pkg, oracle_mod):
    """Eq. (33)'s data terms per member against synthetic targets (the oracle's E/F/W of the population mean
    plus noise): device reduction vs the oracle's loss_terms on the oracle's own E/F/W."""
    cfg = W.get_config(3, (7, 6, 5))
    s = W.make_system(cfg)
    members = W.make_population(cfg, 4, 0.15)
    rng = np.random.default_rng(5)
    e0, f0, w0 = oracle_mod.compute(cfg.hyper, members[0], s.pos, s.types, s.box)
    n = len(s.pos)
    u_t = e0.sum() / n + 0.003
    f_t = f0 + 0.05 * rng.normal(size=f0.shape)
    wt9 = w0.sum(axis=0) / n
    w_t = np.array([wt9[0], wt9[4], wt9[8], wt9[1], wt9[5], wt9[6]]) * 1.02 + 0.001
    nep = pkg.NEP(cfg.hyper, members[0], s.masses, device=0)
    pos = torch.tensor(s.pos, device="cuda:0")
    f_t_dev = torch.tensor(f_t, device="cuda:0")
    nep.nep_neighbors(pos, torch.tensor(s.types, device="cuda:0"), s.box, 1.0)
    with pytest.raises(pkg.NepError) as ei:
        nep.nep_loss_terms(u_t, f_t_dev, w_t)
    assert ei.value.status == -5
    for p in members:
        nep.nep_set_parameters(p)
        nep.nep_compute(pos)
        le, lf, lv = nep.nep_loss_terms(u_t, f_t_dev, w_t)
        eo, fo, wo = oracle_mod.compute(cfg.hyper, p, s.pos, s.types, s.box)
        oe, of, ov = oracle_mod.loss_terms(eo, fo, wo, u_t, f_t, w_t)
        assert le == pytest.approx(oe, abs=1e-6)          # per-atom energy: 1e-5 eV per atom at worst, averaged
        assert lf == pytest.approx(of, rel=1e-4)
        assert lv == pytest.approx(ov, rel=2e-3, abs=1e-6)
    nep.close()
