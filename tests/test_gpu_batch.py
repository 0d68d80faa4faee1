"""SURVEY.md section 8(f) row 4 on the GPU: a batch of small structures x a population of parameter sets
(nep_batch_neighbors / nep_batch_compute / nep_batch_loss) against the pinned oracle, structure by structure and
member by member.  The structures are the small cells a training set holds: thinner than 2 r_c (several lattice
images of a neighbour, images of the atom itself), different sizes, orthorhombic and sheared, plus one wide cell;
inputs are seeded replicas of the BASELINE.json lattices (workloads.py) -- they stand in for the paper's DFT
training structures, which are not available."""
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


make_batch = W.make_batch


BATCHES = [
    (3, [((2, 2, 2), None, 0), ((1, 1, 1), None, 1), ((2, 2, 1), (0.21, -0.13, 0.17), 2), ((3, 2, 2), None, 3), ((4, 4, 3), None, 4)]),
    (2, [((1, 1, 2), None, 0), ((2, 1, 1), (0.1, 0.05, -0.08), 1), ((2, 2, 2), None, 2)]),          # rc 6 / 4, two species, n_max 6
    (4, [((2, 2, 2), None, 0), ((3, 3, 2), (-0.12, 0.07, 0.1), 1), ((1, 2, 3), None, 2)]),          # rc 6 / 5, seven angular channels
    (0, [((2, 2, 1), None, 0), ((1, 1, 1), None, 1)]),                                              # diamond
]


def assert_member(e, f, w, eo, fo, wo):
    assert np.abs(e - eo).max() <= 1e-5
    fn = np.linalg.norm(fo, axis=1, keepdims=True)
    assert (np.abs(f - fo) <= np.maximum(1e-4, 1e-4 * fn)).all(), np.abs(f - fo).max()
    assert np.abs(f - fo).max() <= 1e-4 * max(np.abs(fo).max(), 1e-6)
    wn = np.linalg.norm(wo, axis=1)
    assert (np.linalg.norm(w - wo, axis=1) <= 1e-4 * np.maximum(wn, np.median(wn))).all()
    assert np.linalg.norm(w.sum(0) - wo.sum(0)) <= 1e-4 * np.linalg.norm(wo.sum(0))


@pytest.mark.parametrize("idx,specs", BATCHES)
def test_batch_of_small_structures_times_population(pkg, oracle_mod, idx, specs):
    cfg = W.get_config(idx)
    hy = cfg.hyper
    structs = make_batch(idx, specs)
    members = W.make_population(cfg, 4, sigma=0.3)                       # member 0 = the stress set, three drawn around it
    members.append(W.make_params(cfg, "baseline"))
    off = np.concatenate([[0], np.cumsum([len(p) for p, _, _ in structs])]).astype(np.int32)
    pos = torch.tensor(np.concatenate([p for p, _, _ in structs]), device="cuda:0")
    typ = torch.tensor(np.concatenate([t for _, t, _ in structs]), device="cuda:0")
    boxes = np.stack([H for _, _, H in structs])
    assert any(W.perpendicular_widths(H).min() < 2 * hy.rc_radial for _, _, H in structs)
    nep = pkg.NEP(hy, members[0], cfg.masses, device=0)
    nep.nep_batch_neighbors(off, pos, typ, boxes)
    e, f, w = nep.nep_batch_compute(members)
    e, f, w = e.cpu().numpy(), f.cpu().numpy(), w.cpu().numpy()
    eo_all, fo_all, wo_all = [], [], []
    for m, par in enumerate(members):
        eo_m, fo_m, wo_m = [], [], []
        for s, (p, t, H) in enumerate(structs):
            eo, fo, wo = oracle_mod.compute_images(hy, par, p, t, H)
            sl = slice(off[s], off[s + 1])
            assert_member(e[m, sl], f[m, sl], w[m, sl], eo, fo, wo)
            eo_m.append(eo); fo_m.append(fo); wo_m.append(wo)
        eo_all.append(eo_m); fo_all.append(fo_m); wo_all.append(wo_m)
    assert np.abs(f).max() > 1e-2                                        # not a comparison of zeros
    # ---- loss of Eq. (33): targets = member 0's oracle values shifted, so that no term vanishes
    n_str = len(structs)
    u_t = np.array([eo_all[0][s].mean() + 0.01 * (s + 1) for s in range(n_str)])
    f_t = np.concatenate([fo_all[0][s] + 0.02 for s in range(n_str)])
    six = [0, 4, 8, 1, 5, 6]
    w_t = np.stack([wo_all[0][s].sum(0)[six] / len(structs[s][0]) - 0.03 for s in range(n_str)])
    dev = lambda a: torch.tensor(np.ascontiguousarray(a), device="cuda:0")
    loss = nep.nep_batch_loss(dev(e), dev(f), dev(w), dev(u_t), dev(f_t), dev(w_t)).cpu().numpy()
    for m in range(len(members)):
        # the reduction itself (same E/F/W in, fp64): tight; and end to end against the oracle's own E/F/W
        ef = [e[m, off[s]:off[s + 1]] for s in range(n_str)]
        ff = [f[m, off[s]:off[s + 1]] for s in range(n_str)]
        wf = [w[m, off[s]:off[s + 1]] for s in range(n_str)]
        ft = [f_t[off[s]:off[s + 1]] for s in range(n_str)]
        want = oracle_mod.loss_terms_batch(ef, ff, wf, u_t, ft, w_t)
        np.testing.assert_allclose(loss[m], want, rtol=1e-12)
        full = oracle_mod.loss_terms_batch(eo_all[m], fo_all[m], wo_all[m], u_t, ft, w_t)
        np.testing.assert_allclose(loss[m], full, rtol=2e-4, atol=1e-7)
    # repeat: bitwise reproducible
    e2, f2, w2 = nep.nep_batch_compute(members)
    assert np.array_equal(e2.cpu().numpy(), e) and np.array_equal(f2.cpu().numpy(), f) and np.array_equal(w2.cpu().numpy(), w)
    nep.close()


def test_batch_equals_the_md_path_on_a_wide_cell_and_rejects_bad_input(pkg, oracle_mod):
    cfg = W.get_config(3, (4, 4, 3))
    s, p = W.make_system(cfg), W.make_params(cfg, "stress")
    nep = pkg.NEP(cfg.hyper, p, s.masses, device=0)
    pos, typ = torch.tensor(s.pos, device="cuda:0"), torch.tensor(s.types, device="cuda:0")
    with pytest.raises(pkg.NepError) as ei:
        nep.batch_n = len(s.pos)
        nep.nep_batch_compute([p])
    assert ei.value.status == -5
    nep.nep_neighbors(pos, typ, s.box, 0.0)
    e0, f0, w0 = nep.nep_compute(pos)
    nep.nep_batch_neighbors([0, len(s.pos)], pos, typ, [np.diag(s.box)])
    e, f, w = nep.nep_batch_compute([p])
    assert (e[0] - e0).abs().max().item() <= 2e-6
    assert (f[0] - f0).abs().max().item() <= 2e-5 * f0.abs().max().item()
    assert (w[0] - w0).abs().max().item() <= 2e-5 * w0.abs().max().item()
    for bad_off, bad_box, status in (([0, 0, len(s.pos)], [np.diag(s.box)] * 2, -1),            # empty structure
                                     ([0, len(s.pos)], [np.diag([0.7, 20.0, 20.0])], -2),       # thinner than rc / 6.5
                                     ([0, len(s.pos)], [-np.diag(s.box)], -3)):                 # left-handed
        with pytest.raises(pkg.NepError) as ei:
            nep.nep_batch_neighbors(bad_off, pos, typ, bad_box)
        assert ei.value.status == status
    t = s.types.copy(); t[3] = 7
    with pytest.raises(pkg.NepError) as ei:
        nep.nep_batch_neighbors([0, len(s.pos)], pos, torch.tensor(t, device="cuda:0"), [np.diag(s.box)])
    assert ei.value.status == -1
    nep.close()
