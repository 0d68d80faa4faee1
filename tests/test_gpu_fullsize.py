"""Full-size parity (BASELINE.json configs 1-4 as stated, in the launch configuration bench.py times).

The O(N^2) oracle cannot evaluate 64 k - 8.2 M atoms in a test, so the outputs are SAMPLED
(SURVEY.md section 8(c) "Large-N oracle practicality"):

  * neighbour sets (a1): brute force restricted to seeded sampled atoms (O(N) per atom,
    oracle.neighbors_of) for both cutoffs (+ skin), bit-exact as sets;
  * E / F / W (a2-a8): after md_step has advanced the system with list rebuilds at the stated cadence,
    the GPU's own snapshot is cut into windows -- an inner cube plus a halo of 2 rc_radial (F_i needs
    dU_j/dr_ji of every neighbour j, which needs j's whole environment) -- each evaluated by the oracle
    as an open cluster; inner atoms are compared with north_star's tolerances.  One window is centred on
    the box corner so that it straddles all three periodic boundaries;
  * properties that hold at any size: sum_i F_i = 0, finite state, displacement since the last build
    below skin / 2.
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
    p.load_library()
    return p


def cut_window(pos, box, centre, half_inner, halo):
    """Atoms within the cube |d|_inf < half_inner + halo of `centre` (minimum image), as open-cluster
    coordinates relative to the centre; returns (indices, coordinates, mask of the inner atoms)."""
    d = pos - centre
    d -= box * np.rint(d / box)
    sel = np.flatnonzero((np.abs(d) < half_inner + halo).all(axis=1))
    dc = d[sel]
    return sel, np.ascontiguousarray(dc), (np.abs(dc) < half_inner).all(axis=1)


def assert_efw_window(e, f, w, eo, fo, wo, wscale):
    assert np.abs(e - eo).max() <= 1e-5, f"energy: {np.abs(e - eo).max()}"
    fn = np.linalg.norm(fo, axis=1, keepdims=True)
    assert (np.abs(f - fo) <= np.maximum(1e-4, 1e-4 * fn)).all(), f"force: max err {np.abs(f - fo).max()}"
    assert np.abs(f - fo).max() <= 1e-4 * np.abs(fo).max(), "force error vs max |F| (scale-free)"
    wn = np.linalg.norm(wo, axis=1)
    dw = np.linalg.norm(w - wo, axis=1)
    assert (dw <= 1e-4 * np.maximum(wn, wscale)).all(), f"per-atom virial: worst {(dw / np.maximum(wn, wscale)).max()}"
    assert np.linalg.norm(w.sum(0) - wo.sum(0)) <= 1e-4 * np.linalg.norm(wo.sum(0)), "window virial sum"


# (config, sampled atoms for the set test, warm-up MD steps before the snapshot, inner half edge in A)
FULL = [(1, 2000, 20, 9.0), (2, 2000, 20, 9.0), (3, 1500, 20, 8.0), (4, 400, 10, 7.0)]


@pytest.mark.parametrize("idx,n_sample,n_md,half", FULL)
def test_full_size_sampled_parity(pkg, oracle_mod, idx, n_sample, n_md, half):
    cfg = W.get_config(idx)
    s, p = W.make_system(cfg), W.make_params(cfg)
    h = cfg.hyper
    n = len(s.pos)
    rng = np.random.default_rng(np.random.SeedSequence([2205, 10046, 700, idx]))
    nep = pkg.NEP(h, p, s.masses, device=0)
    pos = torch.tensor(s.pos, device="cuda:0")
    vel = torch.tensor(s.vel, device="cuda:0")
    types = torch.tensor(s.types, device="cuda:0")
    nep.nep_neighbors(pos, types, s.box, cfg.skin)

    # ---- (a1) neighbour sets of sampled atoms at full size, both cutoffs
    sel = np.sort(rng.choice(n, size=n_sample, replace=False))
    sel_dev = torch.tensor(sel, device="cuda:0")
    for which, rc in ((0, h.rc_radial), (1, h.rc_angular)):
        cnt, lst = nep.nep_get_neighbors(which)
        assert int(cnt.sum().item()) % 2 == 0                      # ordered pairs come in twos
        c = cnt[sel_dev].cpu().numpy()
        l = lst[sel_dev].cpu().numpy()
        del cnt, lst
        oc, ol = oracle_mod.neighbors_of(s.pos, s.box, rc + cfg.skin, sel)
        assert np.array_equal(c, oc), f"neighbour counts differ (which={which})"
        big = np.iinfo(np.int32).max
        a = np.sort(np.where(np.arange(l.shape[1])[None, :] < c[:, None], l, big), axis=1)
        b = np.sort(np.where(np.arange(ol.shape[1])[None, :] < oc[:, None], ol, big), axis=1)
        wd = min(a.shape[1], b.shape[1])
        assert np.array_equal(a[:, :wd], b[:, :wd]), f"neighbour sets differ (which={which})"

    # ---- the timed launch configuration: md_step with rebuilds every `rebuild_every` steps
    nep.md_step(pos, vel, cfg.dt_fs, n_md, cfg.rebuild_every, cfg.skin)
    assert nep.nep_max_displacement() < 0.5 * cfg.skin
    e, f, w = nep.nep_get_last()
    assert torch.isfinite(pos).all() and torch.isfinite(vel).all() and torch.isfinite(f).all()
    fsum = f.sum(0).abs().max().item()
    fabs = f.abs().sum(0).max().item()
    assert fsum <= 2e-6 * fabs, f"sum F = {fsum} vs sum |F| = {fabs}"
    snap = pos.cpu().numpy()
    e, f, w = e.cpu().numpy(), f.cpu().numpy(), w.cpu().numpy()
    wscale = np.median(np.linalg.norm(w[rng.choice(n, size=min(n, 20000), replace=False)], axis=1))

    # ---- (a2)-(a8) windows of the GPU's snapshot, evaluated by the oracle as open clusters
    centres = [np.zeros(3), 0.5 * s.box, rng.uniform(0.0, 1.0, 3) * s.box]
    n_inner = 0
    for centre in centres:
        isel, xyz, inner = cut_window(snap, s.box, centre, half, 2.0 * h.rc_radial)
        big_box = np.full(3, 1.0e4)
        eo, fo, wo = oracle_mod.compute(h, p, xyz, s.types[isel], big_box, pbc=(0, 0, 0))
        ii = isel[inner]
        assert_efw_window(e[ii], f[ii], w[ii], eo[inner], fo[inner], wo[inner], wscale)
        n_inner += int(inner.sum())
    assert n_inner >= 300
    nep.close()


def test_largest_atom_count_2_pow_24(pkg, oracle_mod):
    """n = 16,777,216 = 2^24 atoms, the limit include/nep.h states (config 1's diamond lattice and model at
    128^3 cells; ~65 GB of device memory).  List entries pack the neighbour's sorted index into the top 24
    bits of a 32-bit word: every index >= 2^23 used to come back negative (VERDICT r1 / ADVICE r1).  Sampled
    neighbour sets, and oracle windows in every octant -- the internal order is spatial, so the windows at high
    z hold atoms whose sorted indices are above 2^23."""
    cfg = W.get_config(1, (128, 128, 128))
    s, p = W.make_system(cfg), W.make_params(cfg)
    h = cfg.hyper
    n = len(s.pos)
    assert n == 1 << 24
    rng = np.random.default_rng(np.random.SeedSequence([2205, 10046, 701]))
    nep = pkg.NEP(h, p, s.masses, device=0)
    pos = torch.tensor(s.pos, device="cuda:0")
    vel = torch.tensor(s.vel, device="cuda:0")
    types = torch.tensor(s.types, device="cuda:0")
    nep.nep_neighbors(pos, types, s.box, cfg.skin)
    del types
    sel = np.sort(rng.choice(n, size=256, replace=False))
    sel_dev = torch.tensor(sel, device="cuda:0")
    for which, rc in ((0, h.rc_radial), (1, h.rc_angular)):
        cnt, lst = nep.nep_get_neighbors(which)
        c, l = cnt[sel_dev].cpu().numpy(), lst[sel_dev].cpu().numpy()
        assert int(lst.max().item()) >= (1 << 24) - 4096 and int(lst.min().item()) >= -1
        del cnt, lst
        torch.cuda.empty_cache()
        oc, ol = oracle_mod.neighbors_of(s.pos, s.box, rc + cfg.skin, sel)
        assert np.array_equal(c, oc)
        big = np.iinfo(np.int32).max
        a = np.sort(np.where(np.arange(l.shape[1])[None, :] < c[:, None], l, big), axis=1)
        b = np.sort(np.where(np.arange(ol.shape[1])[None, :] < oc[:, None], ol, big), axis=1)
        wd = min(a.shape[1], b.shape[1])
        assert np.array_equal(a[:, :wd], b[:, :wd])
    nep.md_step(pos, vel, cfg.dt_fs, 3, 2, cfg.skin)              # one rebuild inside
    e, f, w = nep.nep_get_last()
    assert torch.isfinite(pos).all() and torch.isfinite(f).all()
    fsum, fabs = f.sum(0).abs().max().item(), f.abs().sum(0).max().item()
    assert fsum <= 2e-6 * fabs
    snap = pos.cpu().numpy()
    e, f, w = e.cpu().numpy(), f.cpu().numpy(), w.cpu().numpy()
    wscale = np.median(np.linalg.norm(w[rng.choice(n, size=20000, replace=False)], axis=1))
    n_inner = 0
    for frac in ((0.0, 0.0, 0.0), (0.2, 0.3, 0.85), (0.9, 0.7, 0.6), (0.5, 0.5, 0.97)):
        isel, xyz, inner = cut_window(snap, s.box, np.array(frac) * s.box, 8.0, 2.0 * h.rc_radial)
        eo, fo, wo = oracle_mod.compute(h, p, xyz, s.types[isel], np.full(3, 1.0e4), pbc=(0, 0, 0))
        ii = isel[inner]
        assert_efw_window(e[ii], f[ii], w[ii], eo[inner], fo[inner], wo[inner], wscale)
        n_inner += int(inner.sum())
    assert n_inner >= 600
    nep.close()
