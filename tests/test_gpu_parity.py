"""GPU-vs-oracle parity through the C ABI (run with -m gpu on a B200).

Tolerances are BASELINE.json's north_star: neighbour lists bit-exact as sets; per-atom energy within
1e-5 eV absolute; each force component within max(1e-4 eV/A, 1e-4 |F|); virial within 1e-4 relative
(reading A14: per atom ||dW_i||_F <= 1e-4 max(||W_i||_F, median_i ||W_i||_F); total ||dW||_F <= 1e-4 ||W||_F).
Because the stated weight scale gives weak signals, the internals q, S, Fp are also compared
component-wise, relative to the largest component of their block (2e-5: DESIGN.md section 4 derives it from the fp32
sums of up to ~50 pair terms; SURVEY 8(c) had proposed 1e-5), and every case is repeated with
the amplified 'stress' parameter set where the 4-/5-body terms are O(0.1-1).
"""
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
    p.load_library()          # fails loudly if the extension is missing
    return p


# scaled-down replicas of the five configs: same lattice, species rule, hyper-parameters; sizes the
# oracle's O(N^2) search finishes in seconds, several thread blocks and a ragged tail (N % 128 != 0
# for most), box >= 2 (rc + skin)
CASES = [
    (0, None, 0.0),              # config 0 itself: 256 atoms, 21.72 x 21.72 x 10.86, skin 0
    (1, (5, 4, 3), 1.0),         # diamond 480 atoms, non-cubic box
    (2, (4, 4, 3), 1.0),         # rock salt 384 atoms, 2 species, rc 6/4
    (3, (7, 6, 5), 1.0),         # fcc alloy 840 atoms, 5 species
    (4, (9, 8, 7), 1.0),         # bcc 1008 atoms, sigma 0.3, rc 6/5, n_max 6/6
]


def make_nep(pkg, cfg, params, masses):
    return pkg.NEP(cfg.hyper, params, masses, device=0)


def to_dev(s):
    return (torch.tensor(s.pos, device="cuda:0"), torch.tensor(s.vel, device="cuda:0"),
            torch.tensor(s.types, device="cuda:0"))


def assert_sets_equal(cnt, lst, ocnt, olst):
    cnt, lst = cnt.cpu().numpy(), lst.cpu().numpy()
    assert np.array_equal(cnt, ocnt), "neighbour counts differ"
    a = np.sort(np.where(np.arange(lst.shape[1])[None, :] < cnt[:, None], lst, np.iinfo(np.int32).max), axis=1)
    b = np.sort(np.where(np.arange(olst.shape[1])[None, :] < ocnt[:, None], olst, np.iinfo(np.int32).max), axis=1)
    w = min(a.shape[1], b.shape[1])
    assert np.array_equal(a[:, :w], b[:, :w]), "neighbour sets differ"
    assert (a[:, w:] == np.iinfo(np.int32).max).all() and (b[:, w:] == np.iinfo(np.int32).max).all()


def check_efw(e, f, w, eo, fo, wo):
    e, f, w = e.cpu().numpy(), f.cpu().numpy(), w.cpu().numpy()
    assert np.abs(e - eo).max() <= 1e-5, f"energy: {np.abs(e - eo).max()}"
    fn = np.linalg.norm(fo, axis=1, keepdims=True)
    tol = np.maximum(1e-4, 1e-4 * fn)
    assert (np.abs(f - fo) <= tol).all(), f"force: max err {np.abs(f - fo).max()}"
    wn = np.linalg.norm(wo, axis=1)
    dw = np.linalg.norm(w - wo, axis=1)
    assert (dw <= 1e-4 * np.maximum(wn, np.median(wn))).all(), f"per-atom virial: worst ratio {(dw / np.maximum(wn, np.median(wn))).max()}"
    assert np.linalg.norm(w.sum(0) - wo.sum(0)) <= 1e-4 * np.linalg.norm(wo.sum(0)), "total virial"
    return np.abs(e - eo).max(), np.abs(f - fo).max()


def check_blocks(got, ref, blocks, rel, what):
    got = got.cpu().numpy().astype(np.float64)
    for lo, hi in blocks:
        scale = np.abs(ref[:, lo:hi]).max()
        err = np.abs(got[:, lo:hi] - ref[:, lo:hi]).max()
        assert err <= rel * scale, f"{what}[{lo}:{hi}]: err {err} vs scale {scale}"


@pytest.mark.parametrize("idx,cells,skin", CASES)
@pytest.mark.parametrize("kind", ["baseline", "stress"])
def test_parity_single_point(pkg, oracle_mod, idx, cells, skin, kind):
    cfg = W.get_config(idx, cells)
    s, p = W.make_system(cfg), W.make_params(cfg, kind)
    h = cfg.hyper
    nep = make_nep(pkg, cfg, p, s.masses)
    pos, vel, types = to_dev(s)
    nep.nep_neighbors(pos, types, s.box, skin)
    # (a1) neighbour sets, both cutoffs, bit-exact vs brute force
    for which, rc in ((0, h.rc_radial), (1, h.rc_angular)):
        cnt, lst = nep.nep_get_neighbors(which)
        ocnt, olst = oracle_mod.neighbors(s.pos, s.box, rc + skin)
        assert_sets_equal(cnt, lst, ocnt, olst)
    # (a2)-(a8)
    e, f, w = nep.nep_compute(pos)
    eo, fo, wo, qo, fpo, So = oracle_mod.compute(h, p, s.pos, s.types, s.box, want_internals=True)
    check_efw(e, f, w, eo, fo, wo)
    blocks = [(0, h.NR)] + [(h.NR + b * h.NA, h.NR + (b + 1) * h.NA) for b in range(h.n_blocks)]
    q, fp = nep.nep_get_descriptors()
    check_blocks(q, qo, blocks, 2e-5, "q")
    check_blocks(fp, fpo, blocks, 2e-5, "Fp")
    S = nep.nep_get_angular_sums().reshape(len(s.pos), -1)
    lblocks = [(n * 24 + a, n * 24 + b) for n in range(h.NA) for a, b in ((0, 3), (3, 8), (8, 15), (15, 24))]
    check_blocks(S, So.reshape(len(s.pos), -1), lblocks, 2e-5, "S")
    # scale-free checks, so that a wrong many-body term cannot hide under the absolute tolerances
    # whatever the force scale of the case is
    fe = np.abs(f.cpu().numpy() - fo).max()
    assert fe <= 1e-4 * np.abs(fo).max(), f"force error {fe} vs max |F| {np.abs(fo).max()}"
    ee = np.abs(e.cpu().numpy() - eo).max()
    assert ee <= 1e-5 * max(np.abs(eo).max(), 1e-3), f"energy error {ee} vs max |U| {np.abs(eo).max()}"
    nep.close()


def test_md_trajectory_config0(pkg, oracle_mod):
    """Config 0 as BASELINE.json states it: one evaluation + 10 NVE steps, dt = 1 fs, skin 0 (rebuild
    every step).  fp32-vs-fp64 trajectories stay together over 10 steps at this force scale."""
    cfg = W.get_config(0)
    s, p = W.make_system(cfg), W.make_params(cfg)
    nep = make_nep(pkg, cfg, p, s.masses)
    pos, vel, types = to_dev(s)
    nep.nep_neighbors(pos, types, s.box, cfg.skin)
    nep.md_step(pos, vel, cfg.dt_fs, cfg.n_steps, cfg.rebuild_every, cfg.skin)
    po, vo, ep, ek = oracle_mod.md(cfg.hyper, p, s.pos, s.vel, s.types, s.masses, s.box, cfg.dt_fs, cfg.n_steps)
    assert np.abs(pos.cpu().numpy() - po).max() < 1e-7
    assert np.abs(vel.cpu().numpy() - vo).max() < 1e-9
    e, f, w = nep.nep_get_last()
    eo, fo, wo = oracle_mod.compute(cfg.hyper, p, po, s.types, s.box)
    check_efw(e, f, w, eo, fo, wo)
    nep.close()


def test_md_energy_conservation_and_rebuilds(pkg):
    """Stress parameters (strong forces), skin 1, rebuild every 10 steps, 200 steps: total energy is
    conserved to the integrator's accuracy, the displacement bound holds, lists were rebuilt."""
    cfg = W.get_config(3, (7, 6, 5))
    s, p = W.make_system(cfg), W.make_params(cfg, "stress")
    nep = make_nep(pkg, cfg, p, s.masses)
    pos, vel, types = to_dev(s)
    m = torch.tensor(s.masses[s.types], device="cuda:0")[:, None]
    nep.nep_neighbors(pos, types, s.box, 1.0)

    def etot():
        e, _, _ = nep.nep_get_last()
        return float(e.sum() + 0.5 * (m * vel * vel).sum() / W.ACC_CONV)

    nep.nep_compute(pos)
    e0 = etot()
    ek0 = float(0.5 * (m * vel * vel).sum() / W.ACC_CONV)
    es = []
    for _ in range(20):
        nep.md_step(pos, vel, 1.0, 10, 10, 1.0)
        es.append(etot())
        assert nep.nep_max_displacement() < 0.5
    drift = max(abs(x - e0) for x in es)
    assert drift < 2e-3 * ek0, f"energy drift {drift} vs kinetic {ek0}"
    nep.close()


def test_errors(pkg):
    cfg = W.get_config(0)
    s, p = W.make_system(cfg), W.make_params(cfg)
    nep = make_nep(pkg, cfg, p, s.masses)
    pos, vel, types = to_dev(s)
    with pytest.raises(pkg.NepError) as ei:
        nep.n = len(s.pos)
        nep.nep_compute(pos)                                  # before nep_neighbors
    assert ei.value.status == -5
    with pytest.raises(pkg.NepError) as ei:
        nep.nep_neighbors(pos, types, s.box, 1.0)             # 10.86 < 2 (5 + 1)
    assert ei.value.status == -2
    box = np.diag(s.box).copy(); box[[0, 1]] = box[[1, 0]]              # left-handed cell: det < 0
    with pytest.raises(pkg.NepError) as ei:
        nep.nep_neighbors(pos, types, box, 0.0)
    assert ei.value.status == -3
    box = np.diag(s.box).copy(); box[1, 0] = 0.8 * box[0, 0]            # tilt that narrows a perpendicular width below 2 rc
    box[2, 1] = 2.0 * box[1, 1]
    with pytest.raises(pkg.NepError) as ei:
        nep.nep_neighbors(pos, types, box, 0.0)
    assert ei.value.status == -2
    nep.close()
