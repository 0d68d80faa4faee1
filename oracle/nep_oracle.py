"""ctypes loader for oracle/nep_oracle.c (fp64 CPU oracle -- test infrastructure, not the product).

Argument marshalling only; every number is computed by the C file.  The shared object is compiled
with gcc on first use (and by __graft_entry__.build()).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "nep_oracle.c")
_SO = os.path.join(_HERE, "libnep_oracle.so")
_lib = None


class OracleHyper(C.Structure):
    _fields_ = [("n_types", C.c_int32),
                ("rc_radial", C.c_double), ("rc_angular", C.c_double),
                ("n_max_radial", C.c_int32), ("n_max_angular", C.c_int32),
                ("basis_radial", C.c_int32), ("basis_angular", C.c_int32),
                ("l_max_3b", C.c_int32), ("l_max_4b", C.c_int32), ("l_max_5b", C.c_int32),
                ("n_neurons", C.c_int32)]

    @classmethod
    def from_hyper(cls, h) -> "OracleHyper":
        return cls(h.n_types, h.rc_radial, h.rc_angular, h.n_max_radial, h.n_max_angular,
                   h.basis_radial, h.basis_angular, h.l_max_3b, h.l_max_4b, h.l_max_5b, h.n_neurons)


def build(force: bool = False) -> str:
    """gcc -O2 -ffp-contract=off -fopenmp; rebuilt when the source is newer than the .so."""
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC", "-std=gnu11",
               _SRC, "-o", _SO, "-lm"]
        subprocess.run(cmd, check=True)
    return _SO


_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int32)
_lp = C.POINTER(C.c_int64)


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        L.onep_num_threads.restype = C.c_int
        L.onep_num_descriptors.restype = C.c_int
        L.onep_num_descriptors.argtypes = [C.POINTER(OracleHyper)]
        L.onep_fc.restype = C.c_double
        L.onep_fc.argtypes = [C.c_double, C.c_double]
        L.onep_dfc.restype = C.c_double
        L.onep_dfc.argtypes = [C.c_double, C.c_double]
        L.onep_fk.restype = None
        L.onep_fk.argtypes = [C.c_double, C.c_double, C.c_int, _dp, _dp]
        L.onep_bk.restype = None
        L.onep_bk.argtypes = [_dp, _dp]
        L.onep_bk_grad.restype = None
        L.onep_bk_grad.argtypes = [_dp, _dp]
        L.onep_constants.restype = None
        L.onep_constants.argtypes = [_dp, _dp, _dp]
        L.onep_q_from_S.restype = None
        L.onep_q_from_S.argtypes = [_dp, _dp, _dp]
        L.onep_ann.restype = None
        L.onep_ann.argtypes = [C.c_int, C.c_int, _dp, _dp, _dp, _dp, _dp, _dp, _dp]
        L.onep_last_timing.restype = None
        L.onep_last_timing.argtypes = [C.POINTER(C.c_double * 2)]
        L.onep_neighbors.restype = C.c_int64
        L.onep_neighbors.argtypes = [C.c_int64, _dp, _dp, _ip, C.c_double, _ip, _ip, C.c_int64]
        L.onep_neighbors_of.restype = C.c_int64
        L.onep_neighbors_of.argtypes = [C.c_int64, _dp, _dp, _ip, C.c_double, C.c_int64, _lp, _ip, _ip, C.c_int64]
        L.onep_compute.restype = C.c_int
        L.onep_compute.argtypes = [C.POINTER(OracleHyper), _dp, _dp, _dp, _dp, _dp, _dp,
                                   C.c_int64, _dp, _ip, _dp, _ip, _dp, _dp, _dp, _dp, _dp, _dp]
        L.onep_compute_images.restype = C.c_int
        L.onep_compute_images.argtypes = [C.POINTER(OracleHyper), _dp, _dp, _dp, _dp, _dp, _dp,
                                          C.c_int64, _dp, _ip, _dp, _dp, _dp, _dp, _dp, _dp, _dp]
        L.onep_count_images.restype = C.c_int
        L.onep_count_images.argtypes = [C.c_int64, _dp, _dp, C.c_double, _ip]
        L.onep_md.restype = C.c_int
        L.onep_md.argtypes = [C.POINTER(OracleHyper), _dp, _dp, _dp, _dp, _dp, _dp,
                              C.c_int64, _dp, _dp, _ip, _dp, _dp, _ip, C.c_double, C.c_int32, _dp, _dp]
        _lib = L
    return _lib


def _d(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.float64)


def _p(a: Optional[np.ndarray], t=_dp):
    return a.ctypes.data_as(t) if a is not None else None


def num_threads() -> int:
    return int(lib().onep_num_threads())


def num_descriptors(hyper) -> int:
    h = OracleHyper.from_hyper(hyper)
    return int(lib().onep_num_descriptors(C.byref(h)))


def fc(r: float, rc: float) -> float:
    return float(lib().onep_fc(r, rc))


def fk(r: float, rc: float, nbas: int):
    f = np.zeros(nbas + 1)
    df = np.zeros(nbas + 1)
    lib().onep_fk(r, rc, nbas, _p(f), _p(df))
    return f, df


def bk(d) -> np.ndarray:
    d = _d(d)
    out = np.zeros(24)
    lib().onep_bk(_p(d), _p(out))
    return out


def bk_grad(d) -> np.ndarray:
    d = _d(d)
    out = np.zeros((24, 3))
    lib().onep_bk_grad(_p(d), _p(out))
    return out


def constants():
    c3, c4, c5 = np.zeros(24), np.zeros(5), np.zeros(3)
    lib().onep_constants(_p(c3), _p(c4), _p(c5))
    return c3, c4, c5


def q_from_S(S):
    S = _d(S)
    out = np.zeros(6)
    dq = np.zeros((6, 24))
    lib().onep_q_from_S(_p(S), _p(out), _p(dq))
    return out, dq


def ann(w0, b0, w1, b1, q):
    w0, b0, w1, b1, q = map(_d, (w0, b0, w1, b1, q))
    H, D = w0.shape
    e = C.c_double(0.0)
    fp = np.zeros(D)
    lib().onep_ann(D, H, _p(w0), _p(b0), _p(w1), _p(b1), _p(q), C.byref(e), _p(fp))
    return e.value, fp


def _box9(box) -> np.ndarray:
    """The cell as 9 numbers, rows = lattice vectors a, b, c; three numbers mean an orthorhombic cell."""
    b = np.asarray(box, dtype=np.float64)
    if b.size == 3:
        b = np.diag(b.reshape(3))
    return np.ascontiguousarray(b.reshape(9))


def _pbc(pbc) -> np.ndarray:
    return np.ascontiguousarray(pbc, dtype=np.int32)


def neighbors(pos, box, rc: float, pbc=(1, 1, 1), cap: Optional[int] = None):
    """Brute-force neighbour sets: returns (count[n], list[n][cap]); grows cap until nothing is cut."""
    pos, box, pbc = _d(pos), _box9(box), _pbc(pbc)
    n = pos.shape[0]
    cap = cap or 64
    while True:
        count = np.zeros(n, dtype=np.int32)
        lst = np.full((n, cap), -1, dtype=np.int32)
        mx = lib().onep_neighbors(n, _p(pos), _p(box), _p(pbc, _ip), rc, _p(count, _ip), _p(lst, _ip), cap)
        if mx <= cap:
            return count, lst
        cap = int(mx)


def neighbors_of(pos, box, rc: float, sel, pbc=(1, 1, 1), cap: int = 256):
    pos, box, pbc = _d(pos), _box9(box), _pbc(pbc)
    sel = np.ascontiguousarray(sel, dtype=np.int64)
    n, ns = pos.shape[0], sel.shape[0]
    while True:
        count = np.zeros(ns, dtype=np.int32)
        lst = np.full((ns, cap), -1, dtype=np.int32)
        mx = lib().onep_neighbors_of(n, _p(pos), _p(box), _p(pbc, _ip), rc, ns, _p(sel, _lp),
                                     _p(count, _ip), _p(lst, _ip), cap)
        if mx <= cap:
            return count, lst
        cap = int(mx)


def compute(hyper, params, pos, types, box, pbc=(1, 1, 1), want_internals: bool = False):
    """Energy[n], force[n][3], virial[n][9] (+ q[n][D], fp[n][D], S[n][NA][24] if want_internals).
    `params` holds fp32 arrays; they are widened to fp64 here, unchanged in value."""
    h = OracleHyper.from_hyper(hyper)
    pos, box, pbc = _d(pos), _box9(box), _pbc(pbc)
    types = np.ascontiguousarray(types, dtype=np.int32)
    n = pos.shape[0]
    cr, ca, w0, b0, w1, b1 = map(_d, (params.c_radial, params.c_angular, params.w0, params.b0, params.w1, params.b1))
    D = int(lib().onep_num_descriptors(C.byref(h)))
    NA = hyper.n_max_angular + 1
    e = np.zeros(n)
    f = np.zeros((n, 3))
    w = np.zeros((n, 9))
    q = np.zeros((n, D)) if want_internals else None
    fp = np.zeros((n, D)) if want_internals else None
    S = np.zeros((n, NA, 24)) if want_internals else None
    rc = lib().onep_compute(C.byref(h), _p(cr), _p(ca), _p(w0), _p(b0), _p(w1), _p(b1),
                            n, _p(pos), _p(types, _ip), _p(box), _p(pbc, _ip),
                            _p(e), _p(f), _p(w), _p(q), _p(fp), _p(S))
    if rc != 0:
        raise MemoryError("oracle allocation failed")
    return (e, f, w, q, fp, S) if want_internals else (e, f, w)


def last_timing():
    """(seconds in the O(N^2) pair search, seconds in the evaluation given the lists) of the last compute /
    compute_images call -- wall clock only (bench.py's cpu_baseline)."""
    out = (C.c_double * 2)()
    lib().onep_last_timing(C.byref(out))
    return float(out[0]), float(out[1])


def compute_images(hyper, params, pos, types, box, want_internals: bool = False):
    """compute() for a fully periodic cell of ANY size (reading A18): the neighbours of an atom are all
    lattice images (j, N) within the cutoffs, (j, N) != (i, 0) -- what Eqs. (2), (12) mean for the small cells of a
    training set.  Same outputs as compute()."""
    h = OracleHyper.from_hyper(hyper)
    pos, box = _d(pos), _box9(box)
    types = np.ascontiguousarray(types, dtype=np.int32)
    n = pos.shape[0]
    cr, ca, w0, b0, w1, b1 = map(_d, (params.c_radial, params.c_angular, params.w0, params.b0, params.w1, params.b1))
    D = int(lib().onep_num_descriptors(C.byref(h)))
    NA = hyper.n_max_angular + 1
    e, f, w = np.zeros(n), np.zeros((n, 3)), np.zeros((n, 9))
    q = np.zeros((n, D)) if want_internals else None
    fp = np.zeros((n, D)) if want_internals else None
    S = np.zeros((n, NA, 24)) if want_internals else None
    rc = lib().onep_compute_images(C.byref(h), _p(cr), _p(ca), _p(w0), _p(b0), _p(w1), _p(b1),
                                   n, _p(pos), _p(types, _ip), _p(box), _p(e), _p(f), _p(w), _p(q), _p(fp), _p(S))
    if rc != 0:
        raise MemoryError("oracle allocation failed")
    return (e, f, w, q, fp, S) if want_internals else (e, f, w)


def count_images(pos, box, rc: float):
    """Ordered neighbour entries (j, N) within rc of each atom, lattice images counted separately."""
    pos, box = _d(pos), _box9(box)
    cnt = np.zeros(pos.shape[0], dtype=np.int32)
    if lib().onep_count_images(pos.shape[0], _p(pos), _p(box), rc, _p(cnt, _ip)) != 0:
        raise MemoryError("oracle allocation failed")
    return cnt


def md(hyper, params, pos, vel, types, masses, box, dt_fs: float, n_steps: int, pbc=(1, 1, 1)):
    """Velocity-Verlet NVE; returns (pos, vel, e_pot[n_steps+1], e_kin[n_steps+1]) (copies)."""
    h = OracleHyper.from_hyper(hyper)
    pos, vel = _d(pos).copy(), _d(vel).copy()
    box, pbc, masses = _box9(box), _pbc(pbc), _d(masses)
    types = np.ascontiguousarray(types, dtype=np.int32)
    cr, ca, w0, b0, w1, b1 = map(_d, (params.c_radial, params.c_angular, params.w0, params.b0, params.w1, params.b1))
    ep = np.zeros(n_steps + 1)
    ek = np.zeros(n_steps + 1)
    rc = lib().onep_md(C.byref(h), _p(cr), _p(ca), _p(w0), _p(b0), _p(w1), _p(b1),
                       pos.shape[0], _p(pos), _p(vel), _p(types, _ip), _p(masses), _p(box), _p(pbc, _ip),
                       dt_fs, n_steps, _p(ep), _p(ek))
    if rc != 0:
        raise MemoryError("oracle allocation failed")
    return pos, vel, ep, ek


# ---- outputs derived from what the path already computes --------------
def latent(params, q):
    """Latent-space vector of every atom: "an N_neu-dimensional space spanned by the vectors
    whose components are the product of the states of the hidden-layer neurons and the connection weights
    between them and the output layer":  latent[i][mu] = w1[mu] * tanh(sum_nu w0[mu][nu] q[i][nu] - b0[mu])
    with the hidden-layer state of Eq. (1).  q: [n][D] fp64 descriptors."""
    w0, b0, w1 = _d(params.w0), _d(params.b0), _d(params.w1)
    q = _d(q)
    n, H = q.shape[0], w0.shape[0]
    out = np.zeros((n, H))
    for i in range(n):
        for mu in range(H):
            out[i, mu] = w1[mu] * np.tanh(np.dot(w0[mu], q[i]) - b0[mu])
    return out


def heat_current(virial, vel):
    """Per-atom heat current J_i = W_i . v_i, Eq. (25), with the 9-component virial of
    Eq. (24) in the layout W[3a+b] (reading A9), i.e. J_i^a = sum_b W_i^{ab} v_i^b; and the total
    J = sum_i J_i, Eq. (26).  Returns (J_atom[n][3], J_total[3]); units eV * Angstrom / fs."""
    W, v = _d(virial), _d(vel)
    n = W.shape[0]
    ja = np.zeros((n, 3))
    for i in range(n):
        for a in range(3):
            ja[i, a] = W[i, 3 * a + 0] * v[i, 0] + W[i, 3 * a + 1] * v[i, 1] + W[i, 3 * a + 2] * v[i, 2]
    return ja, ja.sum(axis=0)


# ---- a second ensemble (NVT, Berendsen thermostat) ------------------------
# Unit constants of DESIGN.md reading A10 (CODATA; pinned against scipy.constants in tests/test_oracle_derived.py)
ACC_CONV = 9.648533212e-3      # (eV/Angstrom/amu) -> Angstrom/fs^2
KB_EV_PER_K = 8.617333262e-5


def kinetic_temperature(vel, masses_per_atom) -> float:
    """T = sum_i m_i v_i^2 / (3 N k_B) with 3N degrees of freedom (readings A10, A15)."""
    v, m = _d(vel), _d(masses_per_atom)
    return float((m[:, None] * v * v).sum() / ACC_CONV / (3.0 * len(m) * KB_EV_PER_K))


def md_berendsen(hyper, params, pos, vel, types, masses, box, dt_fs: float, n_steps: int,
                 t_start: float, t_stop: float, tau_fs: float, pbc=(1, 1, 1)):
    """NVT with the Berendsen thermostat (named PAPER.md:318, `nvt_ber` PAPER.md:602; Berendsen et al.,
    ref. 75 PAPER.md:1220; the paper prints no equation: DESIGN.md reading A15).  Each step is one
    velocity-Verlet step of md() above (kick-drift-kick, forces at the new positions), after which all
    velocities are scaled by  lambda = sqrt(1 + (dt / tau) (T_target / T - 1)),  T the kinetic temperature
    of the just-updated velocities; T_target of step s = 1..n_steps is t_start + (t_stop - t_start) s / n_steps.
    Returns (pos, vel, T_before[n_steps], T_after[n_steps]) -- temperatures before / after each rescale."""
    pos, vel = _d(pos).copy(), _d(vel).copy()
    m_atom = _d(masses)[np.ascontiguousarray(types, dtype=np.int32)]
    t_before = np.zeros(n_steps)
    t_after = np.zeros(n_steps)
    for s in range(1, n_steps + 1):
        pos, vel, _, _ = md(hyper, params, pos, vel, types, masses, box, dt_fs, 1, pbc=pbc)
        T = kinetic_temperature(vel, m_atom)
        t_target = t_start + (t_stop - t_start) * s / n_steps
        lam = np.sqrt(1.0 + (dt_fs / tau_fs) * (t_target / T - 1.0)) if T > 0.0 else 1.0
        vel = vel * lam
        t_before[s - 1] = T
        t_after[s - 1] = kinetic_temperature(vel, m_atom)
    return pos, vel, t_before, t_after


# ---- Langevin thermostat (reading A16) ---------------------------------------------------------
_M64 = (1 << 64) - 1


def counter_normal(seed: int, counter: int) -> float:
    """Standard normal deviate number `counter` of stream `seed` -- the counter-based generator both sides
    implement (reading A16): two SplitMix64 outputs x = mix(seed + (2 counter + h) * 0x9E3779B97F4A7C15),
    h = 0, 1 (mix = the SplitMix64 finaliser of Steele, Lea & Flood), uniforms u = ((x >> 11) + 0.5) 2^-53 in
    (0, 1), Box-Muller z = sqrt(-2 ln u_0) cos(2 pi u_1)."""
    u = []
    for h in (0, 1):
        z = (seed + (2 * counter + h) * 0x9E3779B97F4A7C15) & _M64
        z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & _M64
        z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & _M64
        z = z ^ (z >> 31)
        u.append(((z >> 11) + 0.5) * (1.0 / 9007199254740992.0))
    return float(np.sqrt(-2.0 * np.log(u[0])) * np.cos(2.0 * np.pi * u[1]))


def langevin_half_step(vel, masses_per_atom, t_target: float, c1: float, seed: int, draw: int):
    """v <- c1 v + sqrt(1 - c1^2) sqrt(k_B T / m) R for every component; R = counter_normal(seed,
    (draw * n + i) * 3 + a) for atom i (caller's order), component a, and `draw` the running number of
    the thermostat application (two per MD step)."""
    v, m = _d(vel).copy(), _d(masses_per_atom)
    n = len(m)
    c2 = np.sqrt(1.0 - c1 * c1)
    for i in range(n):
        sig = np.sqrt(KB_EV_PER_K * t_target / m[i] * ACC_CONV)
        for a in range(3):
            v[i, a] = c1 * v[i, a] + c2 * sig * counter_normal(seed, (draw * n + i) * 3 + a)
    return v


def md_langevin(hyper, params, pos, vel, types, masses, box, dt_fs: float, n_steps: int,
                t_start: float, t_stop: float, tau_fs: float, seed: int, first_step: int = 0, pbc=(1, 1, 1)):
    """NVT with the Langevin thermostat (named PAPER.md:318, `nvt_lan` PAPER.md:574-590; the paper cites
    Bussi & Parrinello, ref. 80 PAPER.md:1227, and prints no equation: DESIGN.md reading A16).  Step s =
    first_step .. first_step + n_steps - 1: thermostat half step (draw 2 s), one velocity-Verlet step of md(),
    thermostat half step (draw 2 s + 1); c1 = exp(-dt / (2 tau)); the target temperature of the (s - first_step
    + 1)-th step of the call ramps linearly like md_berendsen's.  Returns (pos, vel, T[n_steps]) with T after each step."""
    pos, vel = _d(pos).copy(), _d(vel).copy()
    m_atom = _d(masses)[np.ascontiguousarray(types, dtype=np.int32)]
    c1 = float(np.exp(-dt_fs / (2.0 * tau_fs)))
    temps = np.zeros(n_steps)
    for k in range(n_steps):
        s = first_step + k
        t_target = t_start + (t_stop - t_start) * (k + 1) / n_steps
        vel = langevin_half_step(vel, m_atom, t_target, c1, seed, 2 * s)
        pos, vel, _, _ = md(hyper, params, pos, vel, types, masses, box, dt_fs, 1, pbc=pbc)
        vel = langevin_half_step(vel, m_atom, t_target, c1, seed, 2 * s + 1)
        temps[k] = kinetic_temperature(vel, m_atom)
    return pos, vel, temps


# ---- loss of one structure under one parameter set: the data terms of Eq. (33), PAPER.md:266-283 ---------
def loss_terms(energy, force, virial, u_target: float, f_target, w_target6):
    """The three RMSE terms of Eq. (33) for N_str = 1 (reading A17): with N atoms,
      L_e = |sum_i U_i / N - u_target|                           (per-atom energy of the structure)
      L_f = sqrt( sum_i |F_i - F_i^tar|^2 / (3 N) )
      L_v = sqrt( sum_{mu nu in xx,yy,zz,xy,yz,zx} (sum_i W_i^{mu nu} / N - w_target[mu nu])^2 / 6 )
    Returns (L_e, L_f, L_v); the weighted sum and the regularisation terms of Eq. (33) are the caller's."""
    e, f, w = _d(energy), _d(force), _d(virial)
    ft, wt = _d(f_target), _d(w_target6)
    n = len(e)
    le = abs(e.sum() / n - u_target)
    lf = float(np.sqrt(((f - ft) ** 2).sum() / (3.0 * n)))
    wtot = w.sum(axis=0) / n
    six = np.array([wtot[0], wtot[4], wtot[8], wtot[1], wtot[5], wtot[6]])
    lv = float(np.sqrt(((six - wt) ** 2).sum() / 6.0))
    return float(le), lf, lv


def loss_terms_batch(energies, forces, virials, u_targets, f_targets, w_targets6):
    """The three RMSE terms of Eq. (33) for a batch of N_str structures; per structure s with
    N_s atoms: energies[s][N_s], forces[s][N_s][3], virials[s][N_s][9] (W[3a+b]), targets u_targets[s] (eV/atom),
    f_targets[s][N_s][3], w_targets6[s][6] (eV/atom; xx, yy, zz, xy, yz, zx).  With N = sum_s N_s:
      L_e = sqrt( 1/N_str sum_s (sum_i U_i / N_s - u_tar(s))^2 )
      L_f = sqrt( 1/(3N) sum_s sum_i |F_i - F_i^tar|^2 )
      L_v = sqrt( 1/(6 N_str) sum_s sum_{mu nu} (sum_i W_i^{mu nu} / N_s - w_tar(s)[mu nu])^2 )
    (U^NEP(n, z) and W^NEP(n, z) are per-atom energy and virial of structure n.)"""
    n_str = len(energies)
    se, sf, sv, n_tot = 0.0, 0.0, 0.0, 0
    for s in range(n_str):
        e, f, w = _d(energies[s]), _d(forces[s]), _d(virials[s])
        ns = len(e)
        n_tot += ns
        se += (e.sum() / ns - float(u_targets[s])) ** 2
        df = f - _d(f_targets[s])
        sf += float((df * df).sum())
        wt = w.sum(axis=0) / ns
        six = np.array([wt[0], wt[4], wt[8], wt[1], wt[5], wt[6]])
        dv = six - _d(w_targets6[s])
        sv += float((dv * dv).sum())
    return float(np.sqrt(se / n_str)), float(np.sqrt(sf / (3.0 * n_tot))), float(np.sqrt(sv / (6.0 * n_str)))


def regularisation_terms(params):
    """The last two terms of Eq. (33) without their weights: (sum |z_n| / N_par, sqrt(sum z_n^2 / N_par)) over
    all trainable parameters z (Eq. (30): c_radial, c_angular, w0, b0, w1, b1)."""
    z = np.concatenate([_d(a).reshape(-1) for a in (params.c_radial, params.c_angular, params.w0, params.b0, params.w1, params.b1)])
    return float(np.abs(z).sum() / len(z)), float(np.sqrt((z * z).sum() / len(z)))
