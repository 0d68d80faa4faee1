"""ctypes binding with the same names as include/nep.h -- argument marshalling only.

PyTorch is used for device memory and the CUDA stream; all arithmetic of the path happens inside
libnep_b200.so.  Functions raise NepError on any non-zero status.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.environ.get("NEP_B200_LIB") or os.path.join(_HERE, "libnep_b200.so")   # NEP_B200_LIB: another build of the same library (kernel experiments)
_lib = None

# every symbol include/nep.h declares
exported_symbols = (
    "nep_create", "nep_destroy", "nep_num_descriptors", "nep_neighbors", "nep_max_neighbors",
    "nep_get_neighbors", "nep_compute", "md_step", "nep_get_last", "nep_max_displacement", "nep_list_raggedness",
    "nep_compute_host", "md_run_host", "nep_get_descriptors", "nep_get_angular_sums", "nep_get_latent",
    "nep_heat_current", "nep_heat_current_static", "md_step_nvt_berendsen", "nep_last_temperature", "md_step_nvt_langevin", "nep_set_parameters",
    "nep_compute_population", "nep_loss_terms", "nep_batch_neighbors", "nep_batch_compute", "nep_batch_loss", "nep_batch_pair_counts",
    "nep_launch_count", "nep_pair_counts", "nep_device_bytes", "nep_profile", "nep_profile_num_kernels",
    "nep_profile_kernel_name", "nep_profile_read", "nep_probe_fp32", "nep_probe_entry_roundtrip", "nep_last_error", "nep_status_string",
)


class NepError(RuntimeError):
    def __init__(self, status: int, text: str):
        super().__init__(f"nep status {status}: {text}")
        self.status = status


class NepHyper(C.Structure):
    _fields_ = [("n_types", C.c_int32),
                ("rc_radial", C.c_double), ("rc_angular", C.c_double),
                ("n_max_radial", C.c_int32), ("n_max_angular", C.c_int32),
                ("basis_radial", C.c_int32), ("basis_angular", C.c_int32),
                ("l_max_3b", C.c_int32), ("l_max_4b", C.c_int32), ("l_max_5b", C.c_int32),
                ("n_neurons", C.c_int32)]

    @classmethod
    def from_hyper(cls, h) -> "NepHyper":
        return cls(h.n_types, h.rc_radial, h.rc_angular, h.n_max_radial, h.n_max_angular,
                   h.basis_radial, h.basis_angular, h.l_max_3b, h.l_max_4b, h.l_max_5b, h.n_neurons)


def lib_path() -> str:
    return _LIB_PATH


def lib_overridden() -> bool:
    """True when NEP_B200_LIB redirected the binding to a library other than the in-tree build."""
    return bool(os.environ.get("NEP_B200_LIB"))


def load_library():
    """Loads libnep_b200.so; fails loudly if it has not been built (no fallback of any kind)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_LIB_PATH):
        raise ImportError(f"{_LIB_PATH} is missing: build it with `python -m paper_2205_10046_b200.build` "
                          "(there is no CPU or PyTorch fallback for the NEP path)")
    if lib_overridden():
        import warnings
        warnings.warn(f"NEP_B200_LIB is set: loading {_LIB_PATH} instead of the in-tree libnep_b200.so; tests and "
                      "bench numbers of this process come from that build", RuntimeWarning, stacklevel=2)
    L = C.CDLL(_LIB_PATH)
    vp, i32, i64, dbl = C.c_void_p, C.c_int32, C.c_int64, C.c_double
    fp = C.POINTER(C.c_float)
    dp = C.POINTER(C.c_double)
    ip = C.POINTER(C.c_int32)
    L.nep_create.restype = C.c_int
    L.nep_create.argtypes = [C.POINTER(vp), C.POINTER(NepHyper), fp, fp, fp, fp, fp, fp, dp, C.c_int, vp]
    L.nep_destroy.restype = C.c_int
    L.nep_destroy.argtypes = [vp]
    L.nep_num_descriptors.restype = C.c_int
    L.nep_num_descriptors.argtypes = [C.POINTER(NepHyper)]
    L.nep_neighbors.restype = C.c_int
    L.nep_neighbors.argtypes = [vp, i64, vp, vp, dp, dbl]
    L.nep_max_neighbors.restype = C.c_int
    L.nep_max_neighbors.argtypes = [vp, C.c_int, ip]
    L.nep_get_neighbors.restype = C.c_int
    L.nep_get_neighbors.argtypes = [vp, C.c_int, vp, vp, i32]
    L.nep_compute.restype = C.c_int
    L.nep_compute.argtypes = [vp, vp, vp, vp, vp]
    L.md_step.restype = C.c_int
    L.md_step.argtypes = [vp, vp, vp, dbl, i32, i32, dbl]
    L.nep_get_last.restype = C.c_int
    L.nep_get_last.argtypes = [vp, vp, vp, vp]
    L.nep_max_displacement.restype = C.c_int
    L.nep_max_displacement.argtypes = [vp, dp]
    L.nep_list_raggedness.restype = C.c_int
    L.nep_list_raggedness.argtypes = [vp, dp]
    L.nep_compute_host.restype = C.c_int
    L.nep_compute_host.argtypes = [vp, i64, vp, vp, dp, dbl, vp, vp, vp]
    L.md_run_host.restype = C.c_int
    L.md_run_host.argtypes = [vp, i64, vp, vp, vp, dp, dbl, i32, i32, dbl, vp, vp, vp]
    L.nep_get_descriptors.restype = C.c_int
    L.nep_get_descriptors.argtypes = [vp, vp, vp]
    L.nep_get_angular_sums.restype = C.c_int
    L.nep_get_angular_sums.argtypes = [vp, vp]
    L.md_step_nvt_berendsen.restype = C.c_int
    L.md_step_nvt_berendsen.argtypes = [vp, vp, vp, dbl, i32, i32, dbl, dbl, dbl, dbl]
    L.md_step_nvt_langevin.restype = C.c_int
    L.md_step_nvt_langevin.argtypes = [vp, vp, vp, dbl, i32, i32, dbl, dbl, dbl, dbl, C.c_uint64, i64]
    L.nep_last_temperature.restype = C.c_int
    L.nep_last_temperature.argtypes = [vp, dp, dp]
    L.nep_set_parameters.restype = C.c_int
    L.nep_set_parameters.argtypes = [vp, vp, vp, vp, vp, vp, vp]
    L.nep_compute_population.restype = C.c_int
    L.nep_compute_population.argtypes = [vp, vp, i32, vp, vp, vp, vp, vp, vp, vp, vp, vp]
    L.nep_loss_terms.restype = C.c_int
    L.nep_loss_terms.argtypes = [vp, dbl, vp, dp, dp]
    L.nep_batch_neighbors.restype = C.c_int
    L.nep_batch_neighbors.argtypes = [vp, i32, ip, vp, vp, dp]
    L.nep_batch_compute.restype = C.c_int
    L.nep_batch_compute.argtypes = [vp, i32, vp, vp, vp, vp, vp, vp, vp, vp, vp]
    L.nep_batch_loss.restype = C.c_int
    L.nep_batch_loss.argtypes = [vp, i32, vp, vp, vp, vp, vp, vp, vp]
    L.nep_batch_pair_counts.restype = C.c_int
    L.nep_batch_pair_counts.argtypes = [vp, C.POINTER(i64), C.POINTER(i64)]
    L.nep_get_latent.restype = C.c_int
    L.nep_get_latent.argtypes = [vp, vp]
    L.nep_heat_current.restype = C.c_int
    L.nep_heat_current.argtypes = [vp, vp, vp, vp]
    L.nep_heat_current_static.restype = C.c_int
    L.nep_heat_current_static.argtypes = [vp, vp, vp, vp]
    L.nep_launch_count.restype = i64
    L.nep_launch_count.argtypes = [vp]
    L.nep_pair_counts.restype = C.c_int
    L.nep_pair_counts.argtypes = [vp, C.POINTER(i64), C.POINTER(i64)]
    L.nep_device_bytes.restype = i64
    L.nep_device_bytes.argtypes = [vp]
    L.nep_profile.restype = C.c_int
    L.nep_profile.argtypes = [vp, C.c_int]
    L.nep_profile_num_kernels.restype = C.c_int
    L.nep_profile_num_kernels.argtypes = []
    L.nep_profile_kernel_name.restype = C.c_char_p
    L.nep_profile_kernel_name.argtypes = [C.c_int]
    L.nep_profile_read.restype = C.c_int
    L.nep_profile_read.argtypes = [vp, dp, C.POINTER(i64)]
    L.nep_probe_fp32.restype = C.c_int
    L.nep_probe_fp32.argtypes = [C.c_int, vp, dp]
    L.nep_probe_entry_roundtrip.restype = C.c_int
    L.nep_probe_entry_roundtrip.argtypes = [C.c_int, i32, ip, ip, ip, ip, ip]
    L.nep_last_error.restype = C.c_char_p
    L.nep_last_error.argtypes = [vp]
    L.nep_status_string.restype = C.c_char_p
    L.nep_status_string.argtypes = [C.c_int]
    _lib = L
    return L


def _box9(box) -> np.ndarray:
    b = np.asarray(box, dtype=np.float64)
    if b.shape == (3,):
        b = np.diag(b)
    return np.ascontiguousarray(b.reshape(9))


def _f32(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.float32)


class NEP:
    """One model on one GPU/stream.  Methods mirror include/nep.h one to one."""

    def __init__(self, hyper, params, masses: Sequence[float], device: int = 0, stream: Optional[int] = None):
        import torch  # device memory + streams only
        if not torch.cuda.is_available():
            raise NepError(-6, "no CUDA device: the NEP path has no CPU fallback")
        self._torch = torch
        self._L = load_library()
        self.hyper = hyper
        self.device = device
        self._h = NepHyper.from_hyper(hyper)
        self.n_des = self._L.nep_num_descriptors(C.byref(self._h))
        if self.n_des < 0:
            raise NepError(self.n_des, self._L.nep_status_string(self.n_des).decode())
        torch.cuda.set_device(device)
        torch.cuda.init()
        if stream is None:
            stream = torch.cuda.current_stream(device).cuda_stream
        self.stream = stream
        fp = C.POINTER(C.c_float)
        arrs = [_f32(params.c_radial), _f32(params.c_angular), _f32(params.w0), _f32(params.b0),
                _f32(params.w1), _f32(params.b1)]
        m = np.ascontiguousarray(masses, dtype=np.float64)
        h = C.c_void_p()
        rc = self._L.nep_create(C.byref(h), C.byref(self._h), *[a.ctypes.data_as(fp) for a in arrs],
                                m.ctypes.data_as(C.POINTER(C.c_double)), device, C.c_void_p(stream))
        if rc != 0:
            raise NepError(rc, self._L.nep_status_string(rc).decode())
        self._h_ptr = h
        self.n = 0

    # ---- plumbing
    def _check(self, rc: int):
        if rc != 0:
            raise NepError(rc, self._L.nep_last_error(self._h_ptr).decode() or self._L.nep_status_string(rc).decode())

    def _dev(self, t, dtype, numel: Optional[int] = None):
        torch = self._torch
        if t is None:
            return None
        if not (t.is_cuda and t.dtype == dtype and t.is_contiguous()):
            raise ValueError(f"expected a contiguous CUDA tensor of dtype {dtype}")
        if numel is not None and t.numel() != numel:
            raise ValueError(f"expected {numel} elements, got {t.numel()}")
        return C.c_void_p(t.data_ptr())

    def close(self):
        if getattr(self, "_h_ptr", None) is not None and self._h_ptr.value:
            self._L.nep_destroy(self._h_ptr)
            self._h_ptr = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- include/nep.h
    def nep_neighbors(self, pos, types, box, skin: float):
        torch = self._torch
        n = pos.shape[0]
        b = _box9(box)
        self._check(self._L.nep_neighbors(self._h_ptr, n, self._dev(pos, torch.float64, 3 * n),
                                          self._dev(types, torch.int32, n),
                                          b.ctypes.data_as(C.POINTER(C.c_double)), float(skin)))
        self.n = n

    def nep_max_neighbors(self, which: int) -> int:
        v = C.c_int32(0)
        self._check(self._L.nep_max_neighbors(self._h_ptr, which, C.byref(v)))
        return v.value

    def nep_get_neighbors(self, which: int):
        torch = self._torch
        cap = max(1, self.nep_max_neighbors(which))
        count = torch.zeros(self.n, dtype=torch.int32, device=f"cuda:{self.device}")
        lst = torch.full((self.n, cap), -1, dtype=torch.int32, device=f"cuda:{self.device}")
        self._check(self._L.nep_get_neighbors(self._h_ptr, which, C.c_void_p(count.data_ptr()),
                                              C.c_void_p(lst.data_ptr()), cap))
        return count, lst

    def nep_compute(self, pos, energy=None, force=None, virial=None):
        torch = self._torch
        n = self.n
        dev = f"cuda:{self.device}"
        if energy is None:
            energy = torch.empty(n, dtype=torch.float64, device=dev)
        if force is None:
            force = torch.empty((n, 3), dtype=torch.float64, device=dev)
        if virial is None:
            virial = torch.empty((n, 9), dtype=torch.float64, device=dev)
        self._check(self._L.nep_compute(self._h_ptr, self._dev(pos, torch.float64, 3 * n),
                                        self._dev(energy, torch.float64, n), self._dev(force, torch.float64, 3 * n),
                                        self._dev(virial, torch.float64, 9 * n)))
        return energy, force, virial

    def md_step(self, pos, vel, dt_fs: float, n_steps: int, rebuild_every: int, skin: float):
        torch = self._torch
        n = self.n
        self._check(self._L.md_step(self._h_ptr, self._dev(pos, torch.float64, 3 * n),
                                    self._dev(vel, torch.float64, 3 * n), float(dt_fs), int(n_steps),
                                    int(rebuild_every), float(skin)))

    def md_step_nvt_berendsen(self, pos, vel, dt_fs: float, n_steps: int, rebuild_every: int, skin: float,
                              t_start: float, t_stop: float, tau_fs: float):
        torch = self._torch
        n = self.n
        self._check(self._L.md_step_nvt_berendsen(self._h_ptr, self._dev(pos, torch.float64, 3 * n),
                                                  self._dev(vel, torch.float64, 3 * n), float(dt_fs), int(n_steps),
                                                  int(rebuild_every), float(skin), float(t_start), float(t_stop),
                                                  float(tau_fs)))

    def md_step_nvt_langevin(self, pos, vel, dt_fs: float, n_steps: int, rebuild_every: int, skin: float,
                             t_start: float, t_stop: float, tau_fs: float, seed: int, first_step: int = 0):
        torch = self._torch
        n = self.n
        self._check(self._L.md_step_nvt_langevin(self._h_ptr, self._dev(pos, torch.float64, 3 * n),
                                                 self._dev(vel, torch.float64, 3 * n), float(dt_fs), int(n_steps),
                                                 int(rebuild_every), float(skin), float(t_start), float(t_stop),
                                                 float(tau_fs), int(seed), int(first_step)))

    def nep_last_temperature(self):
        """(T before the rescale, lambda) of the last thermostatted step."""
        t, lam = C.c_double(0.0), C.c_double(0.0)
        self._check(self._L.nep_last_temperature(self._h_ptr, C.byref(t), C.byref(lam)))
        return t.value, lam.value

    def nep_get_last(self):
        torch = self._torch
        n, dev = self.n, f"cuda:{self.device}"
        e = torch.empty(n, dtype=torch.float64, device=dev)
        f = torch.empty((n, 3), dtype=torch.float64, device=dev)
        w = torch.empty((n, 9), dtype=torch.float64, device=dev)
        self._check(self._L.nep_get_last(self._h_ptr, C.c_void_p(e.data_ptr()), C.c_void_p(f.data_ptr()),
                                         C.c_void_p(w.data_ptr())))
        return e, f, w

    def nep_list_raggedness(self) -> float:
        """Sum over warps of 32 x the longest skin list / sum of all list lengths, last build (1.0 = no idle lanes)."""
        v = C.c_double(0.0)
        self._check(self._L.nep_list_raggedness(self._h_ptr, C.byref(v)))
        return v.value

    def nep_max_displacement(self) -> float:
        v = C.c_double(0.0)
        self._check(self._L.nep_max_displacement(self._h_ptr, C.byref(v)))
        return v.value

    def nep_get_descriptors(self):
        torch = self._torch
        n, dev = self.n, f"cuda:{self.device}"
        q = torch.empty((n, self.n_des), dtype=torch.float32, device=dev)
        fp = torch.empty((n, self.n_des), dtype=torch.float32, device=dev)
        self._check(self._L.nep_get_descriptors(self._h_ptr, C.c_void_p(q.data_ptr()), C.c_void_p(fp.data_ptr())))
        return q, fp

    def nep_get_angular_sums(self):
        torch = self._torch
        S = torch.empty((self.n, self.hyper.n_max_angular + 1, 24), dtype=torch.float32, device=f"cuda:{self.device}")
        self._check(self._L.nep_get_angular_sums(self._h_ptr, C.c_void_p(S.data_ptr())))
        return S

    def nep_set_parameters(self, params):
        arrs = [_f32(a) for a in (params.c_radial, params.c_angular, params.w0, params.b0, params.w1, params.b1)]
        self._check(self._L.nep_set_parameters(self._h_ptr, *[C.c_void_p(a.ctypes.data) for a in arrs]))

    def nep_compute_population(self, pos, members):
        """E [n_pop][n], F [n_pop][n][3], W [n_pop][n][9] of a list of parameter sets at the same positions."""
        torch = self._torch
        n, dev, P = self.n, f"cuda:{self.device}", len(members)
        stack = [np.ascontiguousarray(np.stack([_f32(getattr(m, k)).reshape(-1) for m in members]))
                 for k in ("c_radial", "c_angular", "w0", "b0", "w1", "b1")]
        e = torch.empty((P, n), dtype=torch.float64, device=dev)
        f = torch.empty((P, n, 3), dtype=torch.float64, device=dev)
        w = torch.empty((P, n, 9), dtype=torch.float64, device=dev)
        self._check(self._L.nep_compute_population(self._h_ptr, self._dev(pos, torch.float64, 3 * n), P,
                                                   *[C.c_void_p(a.ctypes.data) for a in stack],
                                                   C.c_void_p(e.data_ptr()), C.c_void_p(f.data_ptr()), C.c_void_p(w.data_ptr())))
        return e, f, w

    def nep_loss_terms(self, u_target: float, f_target, w_target6):
        """(L_e, L_f, L_v) of Eq. (33) for the last evaluation."""
        torch = self._torch
        wt = (C.c_double * 6)(*[float(x) for x in w_target6])
        out = (C.c_double * 3)()
        self._check(self._L.nep_loss_terms(self._h_ptr, float(u_target), self._dev(f_target, torch.float64, 3 * self.n), wt, out))
        return out[0], out[1], out[2]

    # ---- batched evaluation for training (include/nep.h "batched evaluation")
    def nep_batch_neighbors(self, atom_offset, pos, types, boxes):
        """atom_offset: [n_str+1] ints (host); pos [N][3] f64 / types [N] i32 CUDA tensors; boxes [n_str][9] or [n_str][3][3] (host)."""
        torch = self._torch
        off = np.ascontiguousarray(atom_offset, dtype=np.int32)
        n_str, N = len(off) - 1, int(off[-1])
        bx = np.ascontiguousarray(np.asarray(boxes, dtype=np.float64).reshape(n_str, 9))
        self._check(self._L.nep_batch_neighbors(self._h_ptr, n_str, off.ctypes.data_as(C.POINTER(C.c_int32)),
                                                self._dev(pos, torch.float64, 3 * N), self._dev(types, torch.int32, N),
                                                bx.ctypes.data_as(C.POINTER(C.c_double))))
        self.batch_n, self.batch_n_str = N, n_str

    def nep_batch_compute(self, members, want_forces: bool = True):
        """E [n_pop][N], F [n_pop][N][3], W [n_pop][N][9] of a list of parameter sets on the whole batch."""
        torch = self._torch
        N, dev, P = self.batch_n, f"cuda:{self.device}", len(members)
        stack = [np.ascontiguousarray(np.stack([_f32(getattr(m, k)).reshape(-1) for m in members]))
                 for k in ("c_radial", "c_angular", "w0", "b0", "w1", "b1")]
        e = torch.empty((P, N), dtype=torch.float64, device=dev)
        f = torch.empty((P, N, 3), dtype=torch.float64, device=dev) if want_forces else None
        w = torch.empty((P, N, 9), dtype=torch.float64, device=dev) if want_forces else None
        self._check(self._L.nep_batch_compute(self._h_ptr, P, *[C.c_void_p(a.ctypes.data) for a in stack],
                                              C.c_void_p(e.data_ptr()), C.c_void_p(f.data_ptr()) if want_forces else None,
                                              C.c_void_p(w.data_ptr()) if want_forces else None))
        return e, f, w

    def nep_batch_pair_counts(self):
        """(entries inside rc_radial, entries inside rc_angular) of the whole batch, lattice images counted."""
        a, b = C.c_int64(0), C.c_int64(0)
        self._check(self._L.nep_batch_pair_counts(self._h_ptr, C.byref(a), C.byref(b)))
        return a.value, b.value

    def nep_batch_loss(self, e, f, w, u_target, f_target, w_target6):
        """[n_pop][3] = (L_e, L_f, L_v) of Eq. (33) per member; targets are CUDA f64 tensors [n_str], [N][3], [n_str][6]."""
        torch = self._torch
        P, N, S = e.shape[0], self.batch_n, self.batch_n_str
        out = torch.empty((P, 3), dtype=torch.float64, device=f"cuda:{self.device}")
        self._check(self._L.nep_batch_loss(self._h_ptr, P, self._dev(e, torch.float64, P * N), self._dev(f, torch.float64, 3 * P * N),
                                           self._dev(w, torch.float64, 9 * P * N), self._dev(u_target, torch.float64, S),
                                           self._dev(f_target, torch.float64, 3 * N), self._dev(w_target6, torch.float64, 6 * S),
                                           C.c_void_p(out.data_ptr())))
        return out

    def nep_get_latent(self):
        """[n][H] latent-space vectors of the last evaluation."""
        torch = self._torch
        lat = torch.empty((self.n, self.hyper.n_neurons), dtype=torch.float32, device=f"cuda:{self.device}")
        self._check(self._L.nep_get_latent(self._h_ptr, C.c_void_p(lat.data_ptr())))
        return lat

    def nep_heat_current(self, vel):
        """(J_atom [n][3], J_total [3]) of Eqs. (25)-(26) from the last evaluation's virial and `vel`."""
        torch = self._torch
        n, dev = self.n, f"cuda:{self.device}"
        ja = torch.empty((n, 3), dtype=torch.float64, device=dev)
        jt = torch.empty(3, dtype=torch.float64, device=dev)
        self._check(self._L.nep_heat_current(self._h_ptr, self._dev(vel, torch.float64, 3 * n),
                                             C.c_void_p(ja.data_ptr()), C.c_void_p(jt.data_ptr())))
        return ja, jt

    def nep_heat_current_static(self, vel, j_atom, j_total):
        """nep_heat_current for callers that must not allocate on the device: the block partials go to a
        fixed array inside the library (limit 4,194,304 atoms; NepError beyond it) instead of a cudaMalloc'ed
        buffer, and this wrapper allocates nothing either -- `j_atom` [n][3] and `j_total` [3] are fp64 CUDA
        tensors the caller made beforehand and are filled in place.  The array is shared by every call on a
        device: do not let two calls overlap on the GPU.  Make the first call on a device outside any stream
        capture (it looks the array's address up).  See include/nep.h."""
        torch = self._torch
        n = self.n
        self._check(self._L.nep_heat_current_static(self._h_ptr, self._dev(vel, torch.float64, 3 * n),
                                                    self._dev(j_atom, torch.float64, 3 * n),
                                                    self._dev(j_total, torch.float64, 3)))
        return j_atom, j_total

    def nep_launch_count(self) -> int:
        return int(self._L.nep_launch_count(self._h_ptr))

    def nep_pair_counts(self):
        """(ordered pairs inside rc_radial, inside rc_angular) at the last evaluation."""
        r, a = C.c_int64(0), C.c_int64(0)
        self._check(self._L.nep_pair_counts(self._h_ptr, C.byref(r), C.byref(a)))
        return r.value, a.value

    def nep_device_bytes(self) -> int:
        return int(self._L.nep_device_bytes(self._h_ptr))

    def nep_profile(self, enable: bool):
        self._check(self._L.nep_profile(self._h_ptr, 1 if enable else 0))

    def nep_profile_read(self):
        """{kernel name: (total ms, launches)} since the last nep_profile() call; synchronises."""
        k = self._L.nep_profile_num_kernels()
        ms = (C.c_double * k)()
        cnt = (C.c_int64 * k)()
        self._check(self._L.nep_profile_read(self._h_ptr, ms, cnt))
        return {self._L.nep_profile_kernel_name(i).decode(): (ms[i], cnt[i]) for i in range(k) if cnt[i] > 0}

    def nep_probe_fp32(self) -> float:
        v = C.c_double(0.0)
        rc = self._L.nep_probe_fp32(self.device, C.c_void_p(self.stream), C.byref(v))
        if rc != 0:
            raise NepError(rc, self._L.nep_status_string(rc).decode())
        return v.value

    def nep_probe_entry_roundtrip(self, j, slot):
        """(packed, j_out, slot_out) of the device's list-entry packing for int32 host arrays `j`, `slot`."""
        j = np.ascontiguousarray(j, dtype=np.int32)
        slot = np.ascontiguousarray(slot, dtype=np.int32)
        out = [np.empty_like(j) for _ in range(3)]
        ptr = lambda a: a.ctypes.data_as(C.POINTER(C.c_int32))
        rc = self._L.nep_probe_entry_roundtrip(self.device, len(j), ptr(j), ptr(slot), *(ptr(o) for o in out))
        if rc != 0:
            raise NepError(rc, self._L.nep_status_string(rc).decode())
        return tuple(out)

    # host-buffer entry points: numpy arrays or pinned CPU tensors (anything exposing a host pointer)
    @staticmethod
    def _host_ptr(a, kind: str = "f8", count: Optional[int] = None):
        """Pointer to a HOST array (numpy, or a CPU torch tensor, pinned or pageable) after checking what the C
        side assumes: element type `kind` ("f8" = float64, "i4" = int32), C-contiguous, `count` elements."""
        if a is None:
            return None
        if isinstance(a, np.ndarray):
            if a.dtype != np.dtype(kind):
                raise TypeError(f"host array has dtype {a.dtype}, the C ABI reads {np.dtype(kind)}")
            if not a.flags["C_CONTIGUOUS"]:
                raise ValueError("host arrays must be C-contiguous")
            if count is not None and a.size != count:
                raise ValueError(f"host array has {a.size} elements, expected {count}")
            return C.c_void_p(a.ctypes.data)
        name = str(a.dtype)
        if name != {"f8": "torch.float64", "i4": "torch.int32"}[kind]:
            raise TypeError(f"host tensor has dtype {name}, the C ABI reads {np.dtype(kind)}")
        if a.is_cuda:
            raise ValueError("the *_host calls take HOST memory")
        if not a.is_contiguous():
            raise ValueError("host tensors must be contiguous")
        if count is not None and a.numel() != count:
            raise ValueError(f"host tensor has {a.numel()} elements, expected {count}")
        return C.c_void_p(a.data_ptr())

    def nep_compute_host(self, pos, types, box, skin: float, energy=None, force=None, virial=None):
        n = pos.shape[0]
        b = _box9(box)
        hp = self._host_ptr
        self._check(self._L.nep_compute_host(self._h_ptr, n, hp(pos, "f8", 3 * n), hp(types, "i4", n),
                                             b.ctypes.data_as(C.POINTER(C.c_double)), float(skin),
                                             hp(energy, "f8", n), hp(force, "f8", 3 * n), hp(virial, "f8", 9 * n)))
        self.n = n

    def md_run_host(self, pos, vel, types, box, dt_fs: float, n_steps: int, rebuild_every: int, skin: float,
                    energy=None, force=None, virial=None):
        """types=None continues the run of the previous md_run_host call (see include/nep.h)."""
        n = pos.shape[0]
        b = _box9(box if box is not None else np.zeros(3))
        hp = self._host_ptr
        self._check(self._L.md_run_host(self._h_ptr, n, hp(pos, "f8", 3 * n), hp(vel, "f8", 3 * n),
                                        hp(types, "i4", n), b.ctypes.data_as(C.POINTER(C.c_double)),
                                        float(dt_fs), int(n_steps), int(rebuild_every), float(skin),
                                        hp(energy, "f8", n), hp(force, "f8", 3 * n), hp(virial, "f8", 9 * n)))
        self.n = n
