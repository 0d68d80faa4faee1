"""Edge and degenerate cases of the CUDA path against the oracle, through the C ABI (-m gpu).

Empty neighbourhoods (one atom; a dilute gas where most atoms see nobody), a dimer, ragged sizes that do
not fill a warp or a block, atoms exactly on the box faces and outside [0, L), a box of exactly the
minimum legal size, list overflow beyond the 256-slot limit, zero-step md_step, the host-buffer entry
points (nep_compute_host / md_run_host) against the device ones, model variants without the 4-/5-body
blocks and with the largest supported basis sizes, skin lists longer than 64 and 128 slots (multi-word
in-cutoff masks), more species than the register kernels take, and the shared-memory variants of the
radial kernels (NEP_RADIAL_SMEM).
"""
import os
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


def run_both(pkg, oracle_mod, hyper, params, masses, pos, types, box, skin=0.0):
    nep = pkg.NEP(hyper, params, masses, device=0)
    dpos = torch.tensor(pos, device="cuda:0")
    dtyp = torch.tensor(types, device="cuda:0")
    nep.nep_neighbors(dpos, dtyp, box, skin)
    for which, rc in ((0, hyper.rc_radial), (1, hyper.rc_angular)):
        cnt, lst = nep.nep_get_neighbors(which)
        ocnt, olst = oracle_mod.neighbors(pos, box, rc + skin)
        cnt, lst = cnt.cpu().numpy(), lst.cpu().numpy()
        assert np.array_equal(cnt, ocnt)
        for i in range(len(pos)):
            assert set(lst[i, :cnt[i]].tolist()) == set(olst[i, :ocnt[i]].tolist())
    e, f, w = nep.nep_compute(dpos)
    eo, fo, wo = oracle_mod.compute(hyper, params, pos, types, box)
    e, f, w = e.cpu().numpy(), f.cpu().numpy(), w.cpu().numpy()
    assert np.abs(e - eo).max() <= 1e-5
    fn = np.linalg.norm(fo, axis=1, keepdims=True)
    assert (np.abs(f - fo) <= np.maximum(1e-4, 1e-4 * fn)).all()
    assert np.abs(f - fo).max() <= 1e-4 * max(np.abs(fo).max(), 1e-6)
    wn = np.linalg.norm(wo, axis=1)
    # reading A14's floor is the median |W_i|; in a dilute gas the median is 0, so the mean stands in
    assert (np.linalg.norm(w - wo, axis=1) <= 1e-4 * np.maximum(wn, max(np.median(wn), wn.mean(), 1e-6))).all()
    nep.close()
    return e, f, w


def test_single_atom_has_no_neighbours(pkg, oracle_mod):
    """q = 0: U = sum_m w1_m tanh(-b0_m) - b1 (Eq. 1), F = 0, W = 0."""
    cfg = W.get_config(0)
    p = W.make_params(cfg, "stress")
    e, f, w = run_both(pkg, oracle_mod, cfg.hyper, p, [28.0], np.array([[3.0, 4.0, 5.0]]), np.zeros(1, np.int32),
                       np.array([30.0, 31.0, 32.0]))
    want = float((p.w1.astype(np.float64) * np.tanh(-p.b0.astype(np.float64))).sum() - p.b1[0])
    assert abs(e[0] - want) <= 1e-6
    assert np.all(f == 0.0) and np.all(w == 0.0)


@pytest.mark.parametrize("kind", ["baseline", "stress"])
def test_dimer_and_trimer(pkg, oracle_mod, kind):
    cfg = W.get_config(2)                                      # 2 species, rc 6/4
    p = W.make_params(cfg, kind)
    box = np.array([40.0, 41.0, 42.0])
    pos = np.array([[1.0, 1.0, 1.0], [3.1, 1.7, 0.2]])
    run_both(pkg, oracle_mod, cfg.hyper, p, cfg.masses, pos, np.array([0, 1], np.int32), box)
    pos = np.array([[39.5, 1.0, 1.0], [1.6, 1.7, 41.2], [0.3, 3.9, 0.7]])      # across the faces
    run_both(pkg, oracle_mod, cfg.hyper, p, cfg.masses, pos, np.array([1, 0, 1], np.int32), box)


@pytest.mark.parametrize("n", [31, 33, 129, 257])
def test_dilute_gas_ragged_sizes(pkg, oracle_mod, n):
    """Most atoms have empty angular lists, many have empty radial lists; n straddles warp/block sizes."""
    cfg = W.get_config(3)
    p = W.make_params(cfg, "stress")
    pos, types = W.random_cluster(n, n, cfg.hyper.n_types, 38.0, min_dist=1.6)
    run_both(pkg, oracle_mod, cfg.hyper, p, cfg.masses, pos, types, np.array([40.0, 40.0, 40.0]), skin=0.5)


def test_positions_on_faces_and_outside_the_box(pkg, oracle_mod):
    """Coordinates exactly 0, exactly L, negative and beyond L: the library never requires wrapped input."""
    cfg = W.get_config(1, (3, 3, 3))
    s, p = W.make_system(cfg), W.make_params(cfg, "stress")
    pos = s.pos.copy()
    pos[0] = [0.0, 0.0, 0.0]
    pos[1] = [s.box[0], 2.0, 2.5]                                  # x == L
    pos[5] += s.box * np.array([1.0, -1.0, 2.0])                   # other periodic images
    pos[9] -= 3.0 * s.box
    run_both(pkg, oracle_mod, cfg.hyper, p, s.masses, pos, s.types, s.box, skin=0.0)


def test_minimum_legal_box(pkg, oracle_mod):
    """Box edge exactly 2 (rc_radial + skin) is accepted (minimum image still unique); below is refused."""
    cfg = W.get_config(0)
    p = W.make_params(cfg)
    rng = np.random.default_rng(np.random.SeedSequence([2205, 10046, 901]))
    box = np.array([10.0, 10.0, 10.0])
    g = np.stack(np.meshgrid(*[np.arange(4)] * 3, indexing="ij"), -1).reshape(-1, 3) * 2.5
    pos = g + rng.normal(0.0, 0.1, g.shape)
    types = np.zeros(len(pos), np.int32)
    run_both(pkg, oracle_mod, cfg.hyper, p, [28.0], pos, types, box, skin=0.0)
    nep = pkg.NEP(cfg.hyper, p, [28.0], device=0)
    with pytest.raises(pkg.NepError) as ei:
        nep.nep_neighbors(torch.tensor(pos, device="cuda:0"), torch.tensor(types, device="cuda:0"), box * (1 - 1e-9), 0.0)
    assert ei.value.status == -2
    nep.close()


def test_overflow_beyond_256_angular_neighbours_is_an_error(pkg):
    cfg = W.get_config(0)
    p = W.make_params(cfg)
    rng = np.random.default_rng(np.random.SeedSequence([2205, 10046, 902]))
    pos = rng.uniform(0.0, 12.0, size=(3000, 3))                   # 1.7 atoms / A^3: ~470 inside 4 A
    nep = pkg.NEP(cfg.hyper, p, [28.0], device=0)
    with pytest.raises(pkg.NepError) as ei:
        nep.nep_neighbors(torch.tensor(pos, device="cuda:0"), torch.zeros(3000, dtype=torch.int32, device="cuda:0"),
                          np.array([12.0, 12.0, 12.0]), 0.0)
    assert ei.value.status == -4
    nep.close()


def test_dense_lists_regrow(pkg, oracle_mod):
    """Three times the density the first capacity guess is sized for in one corner: lists are regrown,
    never truncated."""
    cfg = W.get_config(0)
    p = W.make_params(cfg)
    pos, types = W.random_cluster(7, 150, 1, 9.0, min_dist=1.25)
    pos2, _ = W.random_cluster(8, 40, 1, 30.0, min_dist=2.0)
    pos = np.concatenate([pos, pos2 + 10.0])
    run_both(pkg, oracle_mod, cfg.hyper, p, [28.0], pos, np.zeros(len(pos), np.int32), np.array([42.0, 42.0, 42.0]), skin=1.0)


@pytest.mark.parametrize("l4,l5", [(0, 0), (2, 0), (0, 1)])
def test_models_without_many_body_blocks(pkg, oracle_mod, l4, l5):
    cfg = W.get_config(3, (4, 4, 3))
    cfg = replace(cfg, hyper=replace(cfg.hyper, l_max_4b=l4, l_max_5b=l5))
    s, p = W.make_system(cfg), W.make_params(cfg, "stress")
    run_both(pkg, oracle_mod, cfg.hyper, p, s.masses, s.pos, s.types, s.box, skin=0.3)


@pytest.mark.parametrize("nr,na,kr,ka,H,T", [(0, 0, 0, 0, 1, 1), (1, 7, 3, 15, 7, 3), (15, 15, 31, 31, 120, 2), (12, 8, 12, 8, 50, 3)])
def test_hyperparameter_extremes(pkg, oracle_mod, nr, na, kr, ka, H, T):
    """Smallest and largest supported basis / channel / neuron counts; (12,8,12,8,50,3) is the shape of
    the paper's MgAlCu model (nep.in)."""
    base = W.get_config(2, (3, 3, 3))
    hy = W.Hyper(n_types=T, rc_radial=6.0 if T != 3 else 6.0, rc_angular=3.5, n_max_radial=nr, n_max_angular=na,
                 basis_radial=kr, basis_angular=ka, n_neurons=H)
    cfg = replace(base, hyper=hy, masses=tuple([24.0, 27.0, 64.0][:T]), species_rule="random" if T > 1 else "single")
    s, p = W.make_system(cfg), W.make_params(cfg, "stress")
    run_both(pkg, oracle_mod, hy, p, s.masses, s.pos, s.types, s.box, skin=0.0)


def _dense_cubic(seed, cells, a, n_types):
    """simple-cubic lattice with Gaussian displacements: a dense periodic system (1 / a^3 atoms per A^3)"""
    rng = np.random.default_rng(np.random.SeedSequence([2205, 10046, 903, seed]))
    g = np.stack(np.meshgrid(*[np.arange(cells)] * 3, indexing="ij"), axis=-1).reshape(-1, 3).astype(np.float64)
    pos = (g + 0.5) * a + rng.normal(0.0, 0.08, size=g.shape)
    box = np.array([cells * a] * 3)
    return np.mod(pos, box), rng.integers(0, n_types, size=len(pos)).astype(np.int32), box


@pytest.mark.parametrize("a,expect_words", [(1.75, 2), (1.45, 3)])
def test_skin_lists_longer_than_one_mask_word(pkg, oracle_mod, a, expect_words):
    """More than 64 (a = 1.75 A) and more than 128 (a = 1.45 A) neighbours inside rc_angular + skin and in
    the shell up to rc_radial + skin: the in-cutoff masks take several 64-bit words and the delivery slot
    is a popcount across words."""
    cfg = W.get_config(3, (4, 4, 3))
    hy = replace(cfg.hyper, rc_radial=5.0, rc_angular=4.0)
    cells = int(np.ceil(12.2 / a))
    pos, types, box = _dense_cubic(1, cells, a, hy.n_types)
    p = W.make_params(replace(cfg, hyper=hy))
    nep = pkg.NEP(hy, p, cfg.masses, device=0)
    nep.nep_neighbors(torch.tensor(pos, device="cuda:0"), torch.tensor(types, device="cuda:0"), box, 1.0)
    assert (nep.nep_max_neighbors(1) + 63) // 64 >= expect_words
    nep.close()
    run_both(pkg, oracle_mod, hy, p, cfg.masses, pos, types, box, skin=1.0)


def test_more_species_than_the_register_kernels_take(pkg, oracle_mod):
    """Seven species: the radial kernels with per-type tables in shared memory."""
    base = W.get_config(2, (3, 3, 3))
    hy = W.Hyper(n_types=7, rc_radial=6.0, rc_angular=4.0, n_max_radial=4, n_max_angular=4, basis_radial=8,
                 basis_angular=8, n_neurons=20)
    cfg = replace(base, hyper=hy, masses=tuple(20.0 + 3.0 * t for t in range(7)), species_rule="random")
    s, p = W.make_system(cfg), W.make_params(cfg, "stress")
    run_both(pkg, oracle_mod, hy, p, s.masses, s.pos, s.types, s.box, skin=0.5)


def test_tables_too_large_for_shared_memory(pkg, oracle_mod):
    """Twelve species with 32 basis functions: the type-pair coefficient tables (148 / 152 KB) stay in global
    memory (k_angular / k_force_angular <4, false> in passes of four channels, the radial kernels' TAB_SM =
    false) and the per-thread radial tables force 32-thread blocks."""
    base = W.get_config(2, (3, 3, 3))
    hy = W.Hyper(n_types=12, rc_radial=6.0, rc_angular=4.0, n_max_radial=7, n_max_angular=5, basis_radial=31,
                 basis_angular=31, n_neurons=16)
    cfg = replace(base, hyper=hy, masses=tuple(20.0 + 3.0 * t for t in range(12)), species_rule="random")
    s, p = W.make_system(cfg), W.make_params(cfg, "stress")
    run_both(pkg, oracle_mod, hy, p, s.masses, s.pos, s.types, s.box, skin=0.5)


@pytest.mark.parametrize("seed", range(10))
def test_random_models_and_cells(pkg, oracle_mod, seed):
    """Seeded fuzz over the template space: species, channel and basis counts, neurons, many-body blocks,
    orthorhombic or sheared cell, skin."""
    rng = np.random.default_rng(np.random.SeedSequence([2205, 10046, 904, seed]))
    T = int(rng.integers(1, 7))
    hy = W.Hyper(n_types=T, rc_radial=float(rng.uniform(4.5, 6.0)), rc_angular=float(rng.uniform(3.0, 4.5)),
                 n_max_radial=int(rng.integers(0, 13)), n_max_angular=int(rng.integers(0, 11)),
                 basis_radial=int(rng.integers(0, 17)), basis_angular=int(rng.integers(0, 17)),
                 n_neurons=int(rng.integers(1, 70)), l_max_4b=int(rng.choice([0, 2])), l_max_5b=int(rng.choice([0, 1])))
    base = W.get_config(int(rng.choice([1, 2, 3])), tuple(int(c) for c in rng.integers(4, 6, size=3)))
    cfg = replace(base, hyper=hy, masses=tuple(float(m) for m in rng.uniform(10.0, 200.0, size=T)),
                  species_rule="random" if T > 1 else "single")
    s, p = W.make_system(cfg), W.make_params(cfg, "stress")
    skin = float(rng.choice([0.0, 0.4, 1.0]))
    if rng.random() < 0.5:
        pos, box = W.sheared(s, *rng.uniform(-0.25, 0.25, size=3))
    else:
        pos, box = s.pos, np.diag(s.box)
    if W.perpendicular_widths(box).min() < 2 * (hy.rc_radial + skin):
        skin = 0.0
    if W.perpendicular_widths(box).min() < 2 * hy.rc_radial:
        pytest.skip("cell too small for this draw")
    run_both(pkg, oracle_mod, hy, p, s.masses, pos, s.types, box, skin=skin)


@pytest.mark.parametrize("idx,cells", [(0, None), (2, (3, 3, 3)), (3, (4, 4, 3))])
def test_shared_memory_radial_variants(pkg, oracle_mod, idx, cells):
    """The configurations' species counts have register variants of the radial kernels; NEP_RADIAL_SMEM
    (read at nep_create) selects the shared-memory ones, which must agree with the oracle as well."""
    cfg = W.get_config(idx, cells) if cells else W.get_config(idx)
    s, p = W.make_system(cfg), W.make_params(cfg, "stress")
    os.environ["NEP_RADIAL_SMEM"] = "1"
    try:
        run_both(pkg, oracle_mod, cfg.hyper, p, s.masses, s.pos, s.types, s.box, skin=0.3 if cells else cfg.skin)
    finally:
        del os.environ["NEP_RADIAL_SMEM"]


@pytest.mark.parametrize("idx,cells", [(3, (4, 4, 3)), (4, (5, 5, 5))])
def test_network_kernel_variants_agree(pkg, oracle_mod, idx, cells):
    """The network runs on the tensor cores (3xTF32, k_ann_tc) where the shapes allow; NEP_ANN_FP32 (read at
    nep_create) selects the fp32-FMA kernel.  Both must meet the oracle, and each other to fp32 round-off."""
    cfg = W.get_config(idx, cells)
    s, p = W.make_system(cfg), W.make_params(cfg, "stress")
    out = {}
    for variant in ("tc", "fp32"):
        if variant == "fp32":
            os.environ["NEP_ANN_FP32"] = "1"
        try:
            nep = pkg.NEP(cfg.hyper, p, s.masses, device=0)
            dpos = torch.tensor(s.pos, device="cuda:0")
            nep.nep_neighbors(dpos, torch.tensor(s.types, device="cuda:0"), s.box, 0.3)
            e, f, w = nep.nep_compute(dpos)
            q, fp = nep.nep_get_descriptors()
            out[variant] = (e.cpu().numpy(), fp.cpu().numpy())
            nep.close()
        finally:
            os.environ.pop("NEP_ANN_FP32", None)
    eo, fo, wo, qo, fpo, So = oracle_mod.compute(cfg.hyper, p, s.pos, s.types, s.box, want_internals=True)
    for variant in out:
        e, fp = out[variant]
        assert np.abs(e - eo).max() <= 1e-5
        assert np.abs(fp - fpo).max() <= 2e-5 * np.abs(fpo).max()
    assert np.abs(out["tc"][0] - out["fp32"][0]).max() <= 2e-6
    assert np.abs(out["tc"][1] - out["fp32"][1]).max() <= 4e-6 * np.abs(fpo).max()


def test_wide_output_layer_takes_the_tanhf_kernel(pkg, oracle_mod):
    """k_ann_tc's tanh (MUFU.EX2 / MUFU.RCP) has an absolute error of ~1e-7 per neuron, i.e. sum_m |w1_m| x 1e-7 in
    U_i; nep_create / nep_set_parameters therefore send models with sum |w1| > 5 to the fp32 kernel with tanhf.
    200 neurons with |w1| in [3, 5] (sum ~ 800): the default handle must give bitwise what NEP_ANN_FP32 gives (the
    same kernel ran), and meet the oracle at the energy bar scaled with the output layer -- 1e-5 eV is north_star's
    bar for O(1) output weights (sum |w1| <= 5, where the dispatch switches); every error source of U_i (the fp32
    pre-activations, tanh, the fp32 sum) is linear in w1, so the bar is 1e-5 x sum |w1| / 5.  dU/dq likewise."""
    cfg = W.get_config(0)
    cfg = replace(cfg, hyper=replace(cfg.hyper, n_neurons=200))
    s, p = W.make_system(cfg), W.make_params(cfg, "stress")
    rng = np.random.default_rng(77)
    p = replace(p, w1=(rng.uniform(3.0, 5.0, 200) * rng.choice([-1.0, 1.0], 200)).astype(np.float32))
    out = {}
    for variant in ("default", "fp32"):
        if variant == "fp32":
            os.environ["NEP_ANN_FP32"] = "1"
        try:
            nep = pkg.NEP(cfg.hyper, p, s.masses, device=0)
            dpos = torch.tensor(s.pos, device="cuda:0")
            nep.nep_neighbors(dpos, torch.tensor(s.types, device="cuda:0"), s.box, 0.0)
            e, f, w = nep.nep_compute(dpos)
            q, fp = nep.nep_get_descriptors()
            out[variant] = (e.cpu().numpy(), fp.cpu().numpy(), f.cpu().numpy())
            nep.close()
        finally:
            os.environ.pop("NEP_ANN_FP32", None)
    assert np.array_equal(out["default"][0], out["fp32"][0]) and np.array_equal(out["default"][1], out["fp32"][1])
    eo, fo, wo, qo, fpo, So = oracle_mod.compute(cfg.hyper, p, s.pos, s.types, s.box, want_internals=True)
    scale = float(np.abs(p.w1).sum()) / 5.0
    assert scale > 100
    assert np.abs(out["default"][0] - eo).max() <= 1e-5 * scale
    assert np.abs(out["default"][1] - fpo).max() <= 2e-5 * np.abs(fpo).max()
    assert np.abs(out["default"][2] - fo).max() <= 1e-4 * np.abs(fo).max()


def test_packed_list_entry_round_trip_beyond_2_pow_23(pkg):
    """A list entry is (j << 8) | slot with j < 2^24: bit 31 is set for every j >= 2^23, and a signed shift would
    sign-extend it.  The device's own entry_pack / entry_j / slot mask, through nep_probe_entry_roundtrip -- the
    regular-run stand-in for the 65 GB test_largest_atom_count_2_pow_24."""
    cfg = W.get_config(0)
    s, p = W.make_system(cfg), W.make_params(cfg)
    nep = pkg.NEP(cfg.hyper, p, s.masses, device=0)
    js = np.array([0, 1, 255, 256, 2**23 - 1, 2**23, 2**23 + 1, 2**24 - 2, 2**24 - 1], dtype=np.int32)
    slots = np.array([0, 1, 63, 64, 127, 128, 255], dtype=np.int32)
    j = np.repeat(js, len(slots))
    slot = np.tile(slots, len(js))
    packed, j_out, slot_out = nep.nep_probe_entry_roundtrip(j, slot)
    assert np.array_equal(j_out, j) and np.array_equal(slot_out, slot)
    expect = ((j.astype(np.uint32) << np.uint32(8)) | slot.astype(np.uint32)).view(np.int32)
    assert np.array_equal(packed, expect)
    assert (packed[j >= 2**23] < 0).all(), "the cases must reach the sign bit"
    with pytest.raises(pkg.NepError):
        nep.nep_probe_entry_roundtrip(np.array([2**24], dtype=np.int32), np.array([0], dtype=np.int32))
    nep.close()


def test_md_step_zero_steps_and_state_errors(pkg):
    cfg = W.get_config(0)
    s, p = W.make_system(cfg), W.make_params(cfg)
    nep = pkg.NEP(cfg.hyper, p, s.masses, device=0)
    pos, vel, types = (torch.tensor(s.pos, device="cuda:0"), torch.tensor(s.vel, device="cuda:0"),
                       torch.tensor(s.types, device="cuda:0"))
    with pytest.raises(pkg.NepError) as ei:
        nep.n = len(s.pos)
        nep.md_step(pos, vel, 1.0, 1, 1, 0.0)
    assert ei.value.status == -5
    nep.nep_neighbors(pos, types, s.box, 0.0)
    p0, v0 = pos.clone(), vel.clone()
    nep.md_step(pos, vel, 1.0, 0, 1, 0.0)                         # evaluates, moves nothing
    assert torch.equal(pos, p0) and torch.equal(vel, v0)
    e, f, w = nep.nep_get_last()
    e2, f2, w2 = nep.nep_compute(pos)
    assert torch.equal(e, e2) and torch.equal(f, f2) and torch.equal(w, w2)     # deterministic, bit for bit
    with pytest.raises(pkg.NepError):
        nep.md_step(pos, vel, 1.0, 1, 0, 0.0)                     # rebuild_every < 1
    nep.close()


def test_host_buffer_entry_points_match_device_ones(pkg):
    cfg = W.get_config(3, (7, 6, 5))
    s, p = W.make_system(cfg), W.make_params(cfg, "stress")
    n = len(s.pos)
    nep = pkg.NEP(cfg.hyper, p, s.masses, device=0)
    pos, vel, types = (torch.tensor(s.pos, device="cuda:0"), torch.tensor(s.vel, device="cuda:0"),
                       torch.tensor(s.types, device="cuda:0"))
    nep.nep_neighbors(pos, types, s.box, 1.0)
    e, f, w = nep.nep_compute(pos)
    eh, fh, wh = np.zeros(n), np.zeros((n, 3)), np.zeros((n, 9))
    nep.nep_compute_host(s.pos, s.types, s.box, 1.0, eh, fh, wh)
    assert np.array_equal(eh, e.cpu().numpy()) and np.array_equal(fh, f.cpu().numpy()) and np.array_equal(wh, w.cpu().numpy())
    # 12 steps in one device call == 12 host calls of one step (same rebuild cadence), bit for bit
    nep.nep_neighbors(pos, types, s.box, 1.0)
    nep.md_step(pos, vel, 1.0, 12, 5, 1.0)
    ph, vh = s.pos.copy(), s.vel.copy()
    nep.md_run_host(ph, vh, s.types, s.box, 1.0, 1, 5, 1.0, eh, fh, wh)
    for _ in range(11):
        nep.md_run_host(ph, vh, None, None, 1.0, 1, 5, 1.0, eh, fh, wh)
    assert np.array_equal(ph, pos.cpu().numpy()) and np.array_equal(vh, vel.cpu().numpy())
    e, f, w = nep.nep_get_last()
    assert np.array_equal(fh, f.cpu().numpy())
    nep.close()


def test_skin_violation_is_reported_not_silent(pkg):
    """md_step used to rebuild on the fixed cadence only.  A run whose atoms move more than skin/2
    between two builds must fail with NEP_ERR_SKIN_EXCEEDED (-8), both at a scheduled rebuild and when the call
    ends; the same run with a cadence that keeps the bound passes."""
    cfg = W.get_config(3, (7, 6, 5))
    s, p = W.make_system(cfg), W.make_params(cfg)
    hot = s.vel * 12.0                                            # ~0.044 A/fs rms: 0.1 A in two or three steps
    for n_steps, every in ((12, 6), (4, 50)):                     # detected at the rebuild / at the end of the call
        nep = pkg.NEP(cfg.hyper, p, s.masses, device=0)
        pos, vel = torch.tensor(s.pos, device="cuda:0"), torch.tensor(hot, device="cuda:0")
        nep.nep_neighbors(pos, torch.tensor(s.types, device="cuda:0"), s.box, 0.2)
        with pytest.raises(pkg.NepError) as ei:
            nep.md_step(pos, vel, 1.0, n_steps, every, 0.2)
        assert ei.value.status == -8 and "skin/2" in str(ei.value)
        nep.close()
    nep = pkg.NEP(cfg.hyper, p, s.masses, device=0)
    pos, vel = torch.tensor(s.pos, device="cuda:0"), torch.tensor(hot, device="cuda:0")
    nep.nep_neighbors(pos, torch.tensor(s.types, device="cuda:0"), s.box, 0.5)
    nep.md_step(pos, vel, 1.0, 12, 1, 0.5)                        # rebuilt every step: displacement 0 at every evaluation
    assert nep.nep_max_displacement() == 0.0
    # skin = 0 needs a build per step: with a longer cadence any motion is a violation
    nep.nep_neighbors(pos, torch.tensor(s.types, device="cuda:0"), s.box, 0.0)
    with pytest.raises(pkg.NepError) as ei:
        nep.md_step(pos, vel, 1.0, 2, 5, 0.0)
    assert ei.value.status == -8
    nep.close()


def test_bad_types_and_host_array_dtypes_are_rejected(pkg):
    cfg = W.get_config(3, (7, 6, 5))
    s, p = W.make_system(cfg), W.make_params(cfg)
    n = len(s.pos)
    nep = pkg.NEP(cfg.hyper, p, s.masses, device=0)
    pos = torch.tensor(s.pos, device="cuda:0")
    for bad in (cfg.hyper.n_types, -1):
        t = s.types.copy(); t[n // 2] = bad
        with pytest.raises(pkg.NepError) as ei:
            nep.nep_neighbors(pos, torch.tensor(t, device="cuda:0"), s.box, 1.0)
        assert ei.value.status == -1 and "type" in str(ei.value)
        with pytest.raises(pkg.NepError) as ei:                   # the failed build left no usable lists behind
            nep.n = n
            nep.nep_compute(pos)
        assert ei.value.status == -5
    e, f, w = np.zeros(n), np.zeros((n, 3)), np.zeros((n, 9))
    with pytest.raises(TypeError):
        nep.nep_compute_host(s.pos.astype(np.float32), s.types, s.box, 1.0, e, f, w)
    with pytest.raises(TypeError):
        nep.nep_compute_host(s.pos, s.types.astype(np.int64), s.box, 1.0, e, f, w)
    with pytest.raises(ValueError):
        nep.nep_compute_host(s.pos, s.types, s.box, 1.0, e, np.zeros((n, 2)), w)
    with pytest.raises(TypeError):
        nep.md_run_host(s.pos.copy(), s.vel.astype(np.float32), s.types, s.box, 1.0, 1, 5, 1.0)
    nep.nep_compute_host(s.pos, s.types, s.box, 1.0, e, f, w)    # and the well-formed call still works
    assert np.isfinite(f).all() and np.abs(f).max() > 0.0
    nep.close()


def test_list_raggedness_and_batch_pair_counts(pkg, oracle_mod):
    """Measurement hooks: nep_list_raggedness = sum over warps of 32 x longest list / sum of lengths, recomputed here
    from the exported lists in the internal order is not possible (the order is internal), so it is bracketed: >= 1,
    = 1 when every atom has the same number of neighbours (perfect lattice), larger for a displaced one; and
    nep_batch_pair_counts = the oracle's lattice-image entry counts."""
    cfg = W.get_config(1, (6, 6, 6))
    s, p = W.make_system(cfg), W.make_params(cfg)
    nep = pkg.NEP(cfg.hyper, p, s.masses, device=0)
    pos, typ = torch.tensor(s.pos, device="cuda:0"), torch.tensor(s.types, device="cuda:0")
    with pytest.raises(pkg.NepError):
        nep.nep_list_raggedness()
    nep.nep_neighbors(pos, typ, s.box, cfg.skin)
    r_disp = nep.nep_list_raggedness()
    cnt, _ = nep.nep_get_neighbors(0)
    assert 1.0 <= r_disp <= float(cnt.max()) / float(cnt.float().mean()) + 1e-9
    lattice = (np.round(s.pos / (cfg.a / 4)) * (cfg.a / 4)) % s.box         # back onto the diamond sites
    nep.nep_neighbors(torch.tensor(lattice, device="cuda:0"), typ, s.box, 0.3)
    cnt, _ = nep.nep_get_neighbors(0)
    if int(cnt.min()) == int(cnt.max()):
        assert nep.nep_list_raggedness() == pytest.approx(1.0)
    assert nep.nep_list_raggedness() <= r_disp + 1e-9
    structs = W.make_batch(3, [((2, 2, 2), None, 0), ((2, 1, 1), (0.1, 0.05, -0.08), 1)])
    cfg3 = W.get_config(3)
    nep3 = pkg.NEP(cfg3.hyper, W.make_params(cfg3), cfg3.masses, device=0)
    off = np.concatenate([[0], np.cumsum([len(q) for q, _, _ in structs])]).astype(np.int32)
    nep3.nep_batch_neighbors(off, torch.tensor(np.concatenate([q for q, _, _ in structs]), device="cuda:0"),
                             torch.tensor(np.concatenate([t for _, t, _ in structs]), device="cuda:0"), np.stack([H for _, _, H in structs]))
    want_r = sum(int(oracle_mod.count_images(q, H, cfg3.hyper.rc_radial).sum()) for q, _, H in structs)
    want_a = sum(int(oracle_mod.count_images(q, H, cfg3.hyper.rc_angular).sum()) for q, _, H in structs)
    got_r, got_a = nep3.nep_batch_pair_counts()
    assert got_r == want_r
    assert abs(got_a - want_a) <= 2          # the angular split is the kernels' fp32 test r < rc_angular
    nep.close(); nep3.close()
