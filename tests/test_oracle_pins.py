"""Pins of the fp64 oracle against things OTHER than itself (CPU only).

Each test checks the oracle against a different definition from the paper or a textbook/library
routine, chosen so that a dropped term, wrong sign/index or a transposed operand fails at least one:
  * T_k recurrence            vs  cos(k arccos x)                      (Eq. 4)
  * f_c                       vs  closed values f_c(0)=1, f_c(rc/2)=1/2, f_c(rc)=0 (Eq. 5)
  * explicit S-forms (13)-(16) vs the Legendre double sum Eq. (6) with scipy's Legendre polynomials
  *                            vs |A_nlm|^2 of Eqs. (7)-(8) with scipy's spherical harmonics
  * q_n222 (Eq. 18)           vs  the Wigner-3j contraction Eq. (9) (sympy 3j, scipy Y_lm)
  * q_n1111 (Eq. 19)          vs  Eqs. (10)-(11), and the identity q_n1111 = (7/15) q_n1^2
  * q_n111 = q_n333 = 0 through the same contraction routine
  * N_des                     vs  the worked values 55 / 77 / 82
  * network                   vs  hand-evaluated one-neuron case and finite differences (Listing 1)
  * brute-force neighbours    vs  scipy cKDTree with periodic box
  * b_k gradients             vs  finite differences; all b_k harmonic
"""
import itertools
import math

import numpy as np
import pytest
from scipy.special import eval_legendre, sph_harm_y
from scipy.spatial import cKDTree
from sympy.physics.wigner import wigner_3j

import workloads as W

L_OF_K = [1] * 3 + [2] * 5 + [3] * 7 + [4] * 9


# ------------------------------------------------------------------ helpers independent of the oracle
def f_basis_closed_form(r, rc, nbas):
    """Eq. (4)-(5) through the trigonometric closed form T_k(x) = cos(k arccos x)."""
    x = 2.0 * (r / rc - 1.0) ** 2 - 1.0
    fc = 0.5 * (1.0 + math.cos(math.pi * r / rc)) if r <= rc else 0.0
    return np.array([0.5 * (math.cos(k * math.acos(max(-1.0, min(1.0, x)))) + 1.0) * fc for k in range(nbas + 1)])


def random_env(seed, m, rmin=1.0, rmax=3.9):
    rng = np.random.default_rng(seed)
    v = rng.normal(size=(m, 3))
    v /= np.linalg.norm(v, axis=1)[:, None]
    return v * rng.uniform(rmin, rmax, size=(m, 1))


def cluster_S_q(oracle, hyper, params, d_vecs, tj):
    """Run the oracle on an open cluster: atom 0 at the origin (type 0) + neighbours; return atom 0's
    internals."""
    pos = np.vstack([np.zeros((1, 3)), d_vecs])
    types = np.concatenate([[0], tj]).astype(np.int32)
    e, f, w, q, fp, S = oracle.compute(hyper, params, pos, types, np.array([100.0, 100.0, 100.0]),
                                       pbc=(0, 0, 0), want_internals=True)
    return q[0], S[0]


def g_angular(hyper, params, r, ti, tj):
    """g_n(r) of Eq. (3) for the angular channel from the closed-form basis (independent of oracle)."""
    f = f_basis_closed_form(r, hyper.rc_angular, hyper.basis_angular)
    return params.c_angular[ti, tj].astype(np.float64) @ f      # [NA]


def A_nlm(hyper, params, d_vecs, tj, l):
    """Eq. (8): A_nlm = sum_j g_n(r_ij) Y_lm(theta_ij, phi_ij), m = -l..l, complex, scipy Y_lm."""
    A = np.zeros((hyper.NA, 2 * l + 1), dtype=complex)
    for d, t in zip(d_vecs, tj):
        r = np.linalg.norm(d)
        if r >= hyper.rc_angular:
            continue
        theta, phi = math.acos(d[2] / r), math.atan2(d[1], d[0])
        g = g_angular(hyper, params, r, 0, t)
        for m in range(-l, l + 1):
            A[:, m + l] += g * sph_harm_y(l, m, theta, phi)
    return A


@pytest.fixture(scope="module")
def model():
    cfg = W.get_config(3)                      # 5 species, asymmetric c^{ij}
    return cfg.hyper, W.make_params(cfg, "stress")


# ------------------------------------------------------------------ basis functions
def test_chebyshev_basis_vs_trig_closed_form(oracle_mod):
    for rc, nbas in [(5.0, 8), (6.0, 10), (3.7, 12)]:
        for r in np.linspace(0.05, rc * 0.999, 37):
            f, _ = oracle_mod.fk(float(r), rc, nbas)
            np.testing.assert_allclose(f, f_basis_closed_form(r, rc, nbas), rtol=0, atol=2e-13)


def test_cutoff_closed_values(oracle_mod):
    rc = 4.2
    assert oracle_mod.fc(0.0, rc) == pytest.approx(1.0, abs=1e-15)
    assert oracle_mod.fc(rc / 2, rc) == pytest.approx(0.5, abs=1e-15)
    assert oracle_mod.fc(rc, rc) == pytest.approx(0.0, abs=1e-15)
    assert oracle_mod.fc(rc * 1.0001, rc) == 0.0
    f, df = oracle_mod.fk(rc, rc, 8)           # f_k(rc) = f_k'(rc) = 0: smooth at the cutoff
    assert np.abs(f).max() < 1e-15 and np.abs(df).max() < 1e-15


def test_basis_derivative_vs_finite_difference(oracle_mod):
    rc, nbas, h = 5.0, 8, 1e-6
    for r in [0.7, 1.9, 3.3, 4.6]:
        _, df = oracle_mod.fk(r, rc, nbas)
        fd = (oracle_mod.fk(r + h, rc, nbas)[0] - oracle_mod.fk(r - h, rc, nbas)[0]) / (2 * h)
        np.testing.assert_allclose(df, fd, rtol=0, atol=1e-8)


# ------------------------------------------------------------------ angular polynomials
def test_bk_gradient_vs_finite_difference_and_harmonic(oracle_mod):
    rng = np.random.default_rng(5)
    h = 1e-3
    for _ in range(5):
        d = rng.normal(size=3)
        g = oracle_mod.bk_grad(d)
        lap = np.zeros(24)
        for a in range(3):
            e = np.zeros(3); e[a] = h
            fd = (oracle_mod.bk(d + e) - oracle_mod.bk(d - e)) / (2 * h)
            # central differences are exact for degree<=2 and O(h^2) for cubic/quartic terms
            np.testing.assert_allclose(g[:, a], fd, rtol=0, atol=5e-5)
            # 4th-order second difference: exact for polynomials of degree <= 5
            lap += (-oracle_mod.bk(d + 2 * e) + 16 * oracle_mod.bk(d + e) - 30 * oracle_mod.bk(d)
                    + 16 * oracle_mod.bk(d - e) - oracle_mod.bk(d - 2 * e)) / (12 * h * h)
        assert np.abs(lap).max() < 1e-6           # Laplace's equation: all 24 are solid harmonics
        # homogeneity of degree l_k: b_k(2 d) = 2^l b_k(d)
        np.testing.assert_allclose(oracle_mod.bk(2 * d), oracle_mod.bk(d) * 2.0 ** np.array(L_OF_K), rtol=1e-12)


# ------------------------------------------------------------------ 3-body: three equivalent definitions
def test_3body_explicit_form_vs_legendre_double_sum(oracle_mod, model):
    """Eq. (6): q_nl = (2l+1)/(4 pi) sum_j sum_k g_n(r_ij) g_n(r_ik) P_l(cos theta_ijk),
    j = k terms included (reading A6)."""
    hyper, params = model
    d = random_env(11, 9)
    tj = np.array([0, 1, 2, 3, 4, 0, 1, 2, 3])
    q, _ = cluster_S_q(oracle_mod, hyper, params, d, tj)
    r = np.linalg.norm(d, axis=1)
    G = np.array([g_angular(hyper, params, r[j], 0, tj[j]) for j in range(len(d))])     # [j][n]
    cosm = (d @ d.T) / np.outer(r, r)
    for l in range(1, 5):
        P = eval_legendre(l, np.clip(cosm, -1.0, 1.0))
        ref = (2 * l + 1) / (4 * math.pi) * np.einsum("jn,kn,jk->n", G, G, P)
        got = q[hyper.NR + (l - 1) * hyper.NA: hyper.NR + l * hyper.NA]
        np.testing.assert_allclose(got, ref, rtol=1e-11, atol=1e-14)


def test_3body_explicit_form_vs_spherical_harmonics(oracle_mod, model):
    """Eqs. (7)-(8), PAPER.md:92-97 with (2 - delta_{0m}) (reading G2)."""
    hyper, params = model
    d = random_env(12, 7)
    tj = np.array([4, 3, 2, 1, 0, 2, 2])
    q, _ = cluster_S_q(oracle_mod, hyper, params, d, tj)
    for l in range(1, 5):
        A = A_nlm(hyper, params, d, tj, l)
        ref = sum((2 - (m == 0)) * np.abs(A[:, m + l]) ** 2 for m in range(0, l + 1))
        got = q[hyper.NR + (l - 1) * hyper.NA: hyper.NR + l * hyper.NA]
        np.testing.assert_allclose(got, ref, rtol=1e-11, atol=1e-14)


def test_S_sums_are_real_spherical_harmonic_moments(oracle_mod, model):
    """Eq. (12) with exponent l_k (reading G1): S_n,k of the l=1 block is (A_n10, Re A_n11, Im A_n11)
    up to the Y normalisation: Y_10 = sqrt(3/4pi) z, Y_11 = -sqrt(3/8pi)(x+iy)."""
    hyper, params = model
    d = random_env(13, 6)
    tj = np.array([0, 1, 2, 3, 4, 1])
    _, S = cluster_S_q(oracle_mod, hyper, params, d, tj)
    A = A_nlm(hyper, params, d, tj, 1)
    np.testing.assert_allclose(S[:, 0], A[:, 1].real / math.sqrt(3 / (4 * math.pi)), rtol=1e-11)
    np.testing.assert_allclose(S[:, 1], -A[:, 2].real / math.sqrt(3 / (8 * math.pi)), rtol=1e-11)
    np.testing.assert_allclose(S[:, 2], -A[:, 2].imag / math.sqrt(3 / (8 * math.pi)), rtol=1e-11)


# ------------------------------------------------------------------ 4-body and 5-body: Wigner-3j definitions
def contract3(A1, A2, A3, l1, l2, l3):
    """Eq. (9)."""
    tot = 0.0
    for m1, m2, m3 in itertools.product(range(-l1, l1 + 1), range(-l2, l2 + 1), range(-l3, l3 + 1)):
        if m1 + m2 + m3:
            continue
        tot += float(wigner_3j(l1, l2, l3, m1, m2, m3)) * A1[m1 + l1] * A2[m2 + l2] * A3[m3 + l3]
    return tot


def coupling4(l, m1, m2, m3, m4):
    """Eq. (11), PAPER.md:113-115 for l1=l2=l3=l4=l."""
    tot = 0.0
    for Lc in range(0, 2 * l + 1):
        for M in range(-Lc, Lc + 1):
            tot += (-1) ** M * float(wigner_3j(Lc, l, l, -M, m1, m2)) * float(wigner_3j(Lc, l, l, M, m3, m4))
    return tot


def test_4body_vs_wigner3j_contraction(oracle_mod, model):
    hyper, params = model
    d = random_env(21, 8)
    tj = np.array([0, 1, 2, 3, 4, 4, 3, 1])
    q, _ = cluster_S_q(oracle_mod, hyper, params, d, tj)
    A2 = A_nlm(hyper, params, d, tj, 2)
    blk4 = hyper.l_max_3b
    for n in range(hyper.NA):
        ref = contract3(A2[n], A2[n], A2[n], 2, 2, 2)
        assert abs(ref.imag) < 1e-14
        assert q[hyper.NR + blk4 * hyper.NA + n] == pytest.approx(ref.real, rel=1e-10, abs=1e-15)
    # q_n111 = q_n333 = 0 (checks the contraction routine used above)
    A1 = A_nlm(hyper, params, d, tj, 1)
    A3 = A_nlm(hyper, params, d, tj, 3)
    assert abs(contract3(A1[0], A1[0], A1[0], 1, 1, 1)) < 1e-14
    assert abs(contract3(A3[0], A3[0], A3[0], 3, 3, 3)) < 1e-14


def test_5body_vs_generalised_coupling_and_identity(oracle_mod, model):
    hyper, params = model
    d = random_env(22, 8)
    tj = np.array([1, 1, 2, 0, 4, 4, 3, 0])
    q, _ = cluster_S_q(oracle_mod, hyper, params, d, tj)
    A1 = A_nlm(hyper, params, d, tj, 1)
    blk5 = hyper.l_max_3b + 1
    coup = {ms: coupling4(1, *ms) for ms in itertools.product((-1, 0, 1), repeat=4)}
    for n in range(hyper.NA):
        ref = sum(c * A1[n][ms[0] + 1] * A1[n][ms[1] + 1] * A1[n][ms[2] + 1] * A1[n][ms[3] + 1]
                  for ms, c in coup.items() if c != 0.0)
        got = q[hyper.NR + blk5 * hyper.NA + n]
        assert abs(ref.imag) < 1e-14
        assert got == pytest.approx(ref.real, rel=1e-10, abs=1e-16)
        # closed-form identity implied by Eq. (19): q_n1111 = (7/15) q_n1^2
        assert got == pytest.approx(7.0 / 15.0 * q[hyper.NR + n] ** 2, rel=1e-11, abs=1e-16)


# ------------------------------------------------------------------ dimer: closed forms by hand
def test_dimer_along_z_closed_forms(oracle_mod, model):
    """One neighbour on the z axis: q_nl = (2l+1)/(4pi) g_n^2 (Eq. 6 with P_l(1)=1);
    q_n222 = 3j(222;000) (g Y_20)^3 = -sqrt(2/35) (g sqrt(5/4pi))^3; q_n1111 = 7/15 (g sqrt(3/4pi))^4;
    radial q_n = g_n^R(r)."""
    hyper, params = model
    r, tj = 2.3, 2
    q, _ = cluster_S_q(oracle_mod, hyper, params, np.array([[0.0, 0.0, r]]), np.array([tj]))
    g = g_angular(hyper, params, r, 0, tj)
    gR = params.c_radial[0, tj].astype(np.float64) @ f_basis_closed_form(r, hyper.rc_radial, hyper.basis_radial)
    NR, NA = hyper.NR, hyper.NA
    np.testing.assert_allclose(q[:NR], gR, rtol=1e-12)
    for l in range(1, 5):
        np.testing.assert_allclose(q[NR + (l - 1) * NA: NR + l * NA], (2 * l + 1) / (4 * math.pi) * g * g, rtol=1e-12)
    np.testing.assert_allclose(q[NR + 4 * NA: NR + 5 * NA],
                               -math.sqrt(2 / 35) * (g * math.sqrt(5 / (4 * math.pi))) ** 3, rtol=1e-12)
    np.testing.assert_allclose(q[NR + 5 * NA: NR + 6 * NA],
                               7 / 15 * (g * math.sqrt(3 / (4 * math.pi))) ** 4, rtol=1e-12)


# ------------------------------------------------------------------ counting formulas
def test_descriptor_length_worked_values(oracle_mod):
    """Eq. (20) and the values the paper prints (tests/golden/ndes_worked_values.txt, with citations)."""
    import os
    path = os.path.join(os.path.dirname(__file__), "golden", "ndes_worked_values.txt")
    rows = [list(map(int, ln.split())) for ln in open(path) if ln.strip() and not ln.startswith("#")]
    assert len(rows) == 3
    for nr, na, l3, l4, l5, ndes in rows:
        assert oracle_mod.num_descriptors(W.Hyper(1, 5.0, 4.0, nr, na, 8, 8, 30, l3, l4, l5)) == ndes
    for i, d in enumerate([35, 35, 37, 35, 49]):          # SURVEY.md section 8 size table
        assert oracle_mod.num_descriptors(W.CONFIGS[i].hyper) == d == W.CONFIGS[i].hyper.n_des


# ------------------------------------------------------------------ network (Listing 1)
def test_ann_hand_case_and_finite_differences(oracle_mod):
    # one neuron, one descriptor: U = w1 tanh(w0 q - b0) - b1 (Eq. 1: both biases are subtracted)
    e, fp = oracle_mod.ann([[0.7]], [0.2], [1.5], [0.3], [0.9])
    assert e == pytest.approx(1.5 * math.tanh(0.7 * 0.9 - 0.2) - 0.3, rel=1e-15)
    assert fp[0] == pytest.approx(1.5 * (1 - math.tanh(0.43) ** 2) * 0.7, rel=1e-14)
    # w0 is [neuron][descriptor] row-major: a transposed read would fail this non-square case
    rng = np.random.default_rng(3)
    H, D = 4, 6
    w0, b0, w1, b1, q = rng.normal(size=(H, D)), rng.normal(size=H), rng.normal(size=H), rng.normal(size=1), rng.normal(size=D)
    e, fp = oracle_mod.ann(w0, b0, w1, b1, q)
    assert e == pytest.approx(float(w1 @ np.tanh(w0 @ q - b0) - b1[0]), rel=1e-14)
    h = 1e-6
    for d in range(D):
        dq = np.zeros(D); dq[d] = h
        fd = (oracle_mod.ann(w0, b0, w1, b1, q + dq)[0] - oracle_mod.ann(w0, b0, w1, b1, q - dq)[0]) / (2 * h)
        assert fp[d] == pytest.approx(fd, abs=1e-8)


def test_descriptor_block_order_is_a_convention(oracle_mod, model):
    """Reading A2: permuting descriptor components together with the w0 columns leaves U unchanged --
    i.e. U depends on the order only through w0, nothing else in the oracle depends on it."""
    hyper, params = model
    d = random_env(31, 6)
    q, _ = cluster_S_q(oracle_mod, hyper, params, d, np.array([0, 1, 2, 3, 4, 0]))
    perm = np.random.default_rng(1).permutation(hyper.n_des)
    e0, _ = oracle_mod.ann(params.w0, params.b0, params.w1, params.b1, q)
    e1, _ = oracle_mod.ann(params.w0[:, perm], params.b0, params.w1, params.b1, q[perm])
    assert e0 == pytest.approx(e1, rel=1e-13)


# ------------------------------------------------------------------ neighbours
@pytest.mark.parametrize("seed", [0, 1])
def test_bruteforce_neighbours_vs_ckdtree(oracle_mod, seed):
    rng = np.random.default_rng(seed)
    box = np.array([13.0, 11.0, 12.5])
    pos = rng.uniform(0, 1, size=(400, 3)) * box
    rc = 5.0
    cnt, lst = oracle_mod.neighbors(pos, box, rc)
    tree = cKDTree(pos, boxsize=box)
    ref = tree.query_ball_point(pos, rc)
    for i in range(len(pos)):
        assert set(lst[i, :cnt[i]].tolist()) == set(ref[i]) - {i}


def _lattice_image_sets(pos, H, rc, sel):
    """the plain definition for the chosen atoms: j is a neighbour of i iff some lattice image of j is closer
    than rc (125 images; numpy, shares nothing with the C oracle)"""
    shifts = np.array([[a, b, c] for a in (-2, -1, 0, 1, 2) for b in (-2, -1, 0, 1, 2) for c in (-2, -1, 0, 1, 2)],
                      dtype=np.float64) @ H
    out = []
    for i in sel:
        d = pos[None, :, :] - pos[i][None, None, :] + shifts[:, None, :]
        close = ((d * d).sum(axis=2) < rc * rc).any(axis=0)
        close[i] = False
        out.append(set(np.nonzero(close)[0].tolist()))
    return out


@pytest.mark.parametrize("sheared", [False, True])
def test_neighbours_of_selected_atoms(oracle_mod, sheared):
    """onep_neighbors_of (the checker of the full-size neighbour-set parity tests) against the full brute force
    onep_neighbors, scipy's cKDTree (orthorhombic cell) and the lattice-image definition (sheared cell); a `cap`
    smaller than the longest list must be regrown, never truncate."""
    rng = np.random.default_rng(17)
    box = np.array([13.0, 11.0, 12.5])
    pos = rng.uniform(0, 1, size=(400, 3)) * box
    H = np.diag(box)
    if sheared:
        H = np.array([[13.0, 0.0, 0.0], [2.1, 11.0, 0.0], [-1.7, 1.3, 12.5]])
        pos = (pos / box) @ H
    pos = pos + rng.integers(-2, 3, size=pos.shape).astype(np.float64) @ H        # unwrapped input
    rc = 5.0
    sel = np.array([399, 0, 17, 17, 250, 3, 128], dtype=np.int64)                 # unordered, one repeated
    cnt_all, lst_all = oracle_mod.neighbors(pos, H if sheared else box, rc)
    for cap in (256, 4):                                                          # 4 << longest list (~45)
        cnt, lst = oracle_mod.neighbors_of(pos, H if sheared else box, rc, sel, cap=cap)
        assert cnt.shape == (len(sel),) and lst.shape[1] >= cnt.max() > 4
        for s_, i in enumerate(sel):
            assert cnt[s_] == cnt_all[i]
            assert lst[s_, :cnt[s_]].tolist() == lst_all[i, :cnt_all[i]].tolist()      # same order too
            assert (lst[s_, cnt[s_]:] == -1).all()
    frac = pos @ np.linalg.inv(H)
    wrapped = (frac - np.floor(frac)) @ H                  # same periodic structure; images within +-2 cells suffice
    want = _lattice_image_sets(wrapped, H, rc, sel)
    assert sum(len(w) for w in want) > 20 * len(sel)
    for s_, i in enumerate(sel):
        assert set(lst[s_, :cnt[s_]].tolist()) == want[s_]
    if not sheared:
        ref = cKDTree(wrapped, boxsize=box).query_ball_point(wrapped[sel], rc)
        for s_, i in enumerate(sel):
            assert set(lst[s_, :cnt[s_]].tolist()) == set(ref[s_]) - {int(i)}


def test_neighbour_predicate_is_strict_and_minimum_image(oracle_mod):
    box = np.array([12.0, 12.0, 12.0])
    pos = np.array([[0.5, 0.5, 0.5], [3.5, 4.5, 0.5],      # distance exactly 5.0 (3-4-5) -> excluded at rc=5
                    [11.5, 0.5, 0.5],                      # image distance 1.0 through the boundary
                    [6.5, 0.5, 0.5]])                      # distance 6.0 = L/2
    cnt, lst = oracle_mod.neighbors(pos, box, 5.0)
    assert set(lst[0, :cnt[0]].tolist()) == {2}
    cnt, lst = oracle_mod.neighbors(pos, box, 5.0 + 1e-12)
    assert set(lst[0, :cnt[0]].tolist()) == {1, 2}
    # unwrapped coordinates (an atom that left the box) give the same sets
    pos2 = pos.copy(); pos2[2, 0] -= 12.0; pos2[1] += np.array([24.0, -12.0, 12.0])
    cnt2, lst2 = oracle_mod.neighbors(pos2, box, 5.0 + 1e-12)
    assert set(lst2[0, :cnt2[0]].tolist()) == {1, 2}
