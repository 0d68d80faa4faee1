#!/usr/bin/env python
"""bench.py -- atom-step/s of the NEP3 hot path (BASELINE.json metric) on one B200 per rank.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config IDX] [--impl ours|reference]

A "step" is one pass of the whole hot path: one velocity-Verlet NVE
step = half kick + drift, [neighbour lists rebuilt every `rebuild_every` steps], energy / force /
virial evaluation, half kick -- everything inside the library's sm_100a kernels, through the C ABI
(include/nep.h).  The default workload is BASELINE.json configs[3] (1,000,188-atom five-species fcc
alloy), the configuration north_star's throughput target is quoted on.  Seeded synthetic inputs
(workloads.py); weights are the seeded random model, not a trained one.

Prints ONE JSON line (rank 0).  Keys beyond the base contract:
  roofline     the dominant kernel: algorithmic flops (or bytes) per launch / CUDA-event duration
  kernels      the same for every kernel of a step (events recorded by the library on its own stream,
               nep_profile_*, over the K steps that directly follow the timed region: the instrumentation itself
               costs 2.4 % of the step, so the timed region runs without it; --windows times and profiles together)
  cpu_baseline the fp64 oracle (oracle/, as it stands) timed on this box's host cores on a bounded sample
  e2e          the same metric through md_run_host() with pinned HOST buffers: every step uploads
               positions + velocities and downloads positions, velocities, energies and forces

Multi-GPU: the path has no sharding in north_star ("no multi-GPU sharding or collectives"), so --gpus N
runs N independent replicas ("replicas only"); torch.distributed is used for the barrier
and the max-over-ranks time only.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np

import workloads as W

METRIC = "atom-step/s (NEP force+MD step, 1 B200) and % of FP32/HBM roofline"
UNIT = "atom-step/s"
SM_COUNT, FP32_LANES, SM_MAX_MHZ_NOMINAL = 148, 128, 1965.0     # B200_PROFILING.md "Nominal figures"
L2_BYTES = 126e6
PER_BUILD_IDS = ("build_rev", "scan")          # kernel ids whose cost entry is per list build, not per launch


# ---------------------------------------------------------------------------------------------------
# Algorithmic cost model.  FMA = 2 flops.  Units are the
# ordered pairs inside the cutoffs at the timed evaluation (nep_pair_counts) and the atoms.
def kernel_costs(h: W.Hyper, n_atoms: int, pairs_r: int, pairs_a: int, list_r: int, list_a: int):
    """{kernel: (flops per launch, bytes per launch)} -- what the METHOD must compute / move, not what
    the kernels happen to execute.  list_r / list_a: entries of the skin lists (radial = all)."""
    NR, KR, NA, KA, D, H = h.NR, h.KR, h.NA, h.KA, h.n_des, h.n_neurons
    n = n_atoms
    out = {}
    # a2 radial descriptor: per pair r, f_c, x, T_k, f_k and the NR x KR contraction
    out["radial"] = (pairs_r * (35 + 4 * KR + 2 * NR * KR),
                     n * (16 + 4 * NR) + 4 * pairs_r)
    # a3+a4: g_n (NA x KA), 24 b_k, 24 NA accumulations; per atom the components from S
    out["angular"] = (pairs_a * (90 + 2 * NA * KA + 2 * 24 * NA) + n * 30 * NA,
                      n * (16 + 4 * 24 * NA + 4 * 6 * NA) + 4 * pairs_a)
    # a5: forward + backward of the network
    out["ann"] = (n * (4 * D * H + 10 * H), n * (8 * D + 4))
    # a7: g, g' (4 NA KA), A_k, B_k (4 x 24 NA), assembly of b_k / grad P_k (~500); per atom G_nk
    out["force_angular"] = (pairs_a * (4 * NA * KA + 4 * 24 * NA + 500) + n * 3 * 24 * NA,
                            n * (16 + 4 * 24 * NA + 4 * 6 * NA) + pairs_a * (4 + 12))
    # a6: radial partial forces.  SURVEY.md 8(d) counts 55 + 8 KR + 4 NR KR per ordered pair for BOTH
    # directions evaluated at atom i (Alg. 2); every direction is needed once only, so the method's
    # minimum is one direction per ordered pair: 55 + 4 KR + 2 NR KR.  Bytes: position, own Fp_R, list
    # entry, one 4-byte scalar delivered per pair, own sum.
    out["force_radial"] = (pairs_r * (55 + 4 * KR + 2 * NR * KR),
                           n * (16 + 4 * NR + 16 + 8) + pairs_r * (4 + 4))
    # a8: gather of the delivered partial forces into F_i, W_i (~30 flops per pair)
    out["final"] = (pairs_r * 30,
                    n * (16 + 16 + 4 + 8 * 13) + 4 * pairs_r + pairs_a * 16 + (pairs_r - pairs_a) * 4)
    # per-step filter of the skin lists to the in-cutoff lists (~12 flops per listed pair)
    out["filter"] = (list_r * 12, n * 32 + 4 * list_r + 4 * pairs_r)
    out["quantize"] = (n * 9, n * (24 + 4 + 4 + 16))
    # a1, per build (every rebuild_every steps).  SURVEY.md 8(d): ~100 B/atom binning/reorder + 4 B x (L_R + L_A)
    # list writes ~ 0.6 kB/atom and 300-500 candidate distance tests (~10 flops each) per atom.  The
    # candidate count is the stencil's: 125 cells of edge (rc_R + skin)/2 = 3.73 x the sphere's volume.
    cand = 3.73 * list_r
    out["cell_hist"] = (n * 12, n * (24 + 4 + 4 + 4))
    out["scatter"] = (0, n * (4 + 4 + 4 + 4))
    out["sort_cells"] = (0, n * 8)
    out["build_lists"] = (cand * 10, n * (16 + 8 + 4) + 4 * (list_r + list_a))
    # reverse index: every listed pair needs the slot of i in j's list (one byte), found from j's list row
    out["build_rev"] = (0, (4 + 1) * list_r)       # per build; divided by the launches of this id below
    out["kick_drift"] = (n * 3 * 5, n * (3 * 8 * 5 + 4))
    out["kick"] = (n * 3 * 3, n * (3 * 8 * 3 + 4))
    return out


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")
    NAMES = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")

    def __init__(self, gpu_index: int):
        self.idx, self.proc, self.lines = gpu_index, None, []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "50", "-i", str(self.idx)],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._pump, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _pump(self):
        for line in self.proc.stdout:
            self.lines.append(line)

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        time.sleep(0.06)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        self.thread.join(timeout=2)
        sm, mx, pw, reasons = [], [], [], set()
        for line in self.lines:
            f = [x.strip() for x in line.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1])); pw.append(float(f[2]))
            except ValueError:
                continue
            for name, val in zip(self.NAMES, f[3:7]):
                if val == "Active":
                    reasons.add(name)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        return {"sm_mhz": statistics.median(sm), "sm_max_mhz": max(mx), "reasons": sorted(reasons),
                "samples": len(sm), "power_w_max": max(pw)}


def measured_peaks():
    """HBM GB/s from MEASURED_PEAKS.json (driver-written), else the profiling guide's fallback."""
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
    except (OSError, KeyError, ValueError):
        return 6650.0, "fallback (B200_PROFILING.md)"


def measured_tf32_peak():
    """Dense TF32 tensor peak in TFLOP/s for the network kernel (k_ann_tc): the measured bf16 figure of
    MEASURED_PEAKS.json times the nominal TF32 : bf16 ratio 1/2 (B200_PROFILING.md), else half the guide's
    fallback (the kernel is timed inside a long step: the sustained figure)."""
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            return 0.5 * float(json.load(f)["bf16_tflops_sustained"]), "of measured: sustained bf16 x 1/2 (MEASURED_PEAKS.json)"
    except (OSError, KeyError, ValueError):
        return 0.5 * 1400.0, "of fallback: sustained bf16 1.4 PFLOP/s x 1/2 (B200_PROFILING.md)"


def ncu_traffic(workload: str):
    """DRAM bytes per launch from the committed ncu --set full capture, if one exists for this workload:
    profiles/traffic_<workload>.csv with lines `kernel,dram_bytes_per_launch`."""
    path = os.path.join(ROOT, "profiles", f"traffic_{workload}.csv")
    out = {}
    try:
        with open(path) as f:
            for line in f:
                k, _, v = line.strip().partition(",")
                try:
                    out[k] = float(v)
                except ValueError:
                    pass
    except OSError:
        pass
    return out


# ---------------------------------------------------------------------------------------------------
# The oracle on the host cores: cpu_baseline leg and --impl reference arm.
def oracle_sample_config(cfg: W.Config, n_target: int) -> W.Config:
    """A smaller replica of `cfg` (same lattice, species rule, model, sigma, temperature) with about
    n_target atoms, cubic cell count, box >= 2 (rc + skin)."""
    per_cell = len(W._BASIS[cfg.lattice])
    c = max(1, round((n_target / per_cell) ** (1.0 / 3.0)))
    c_min = int(np.ceil(2.0 * (cfg.hyper.rc_radial + cfg.skin) / cfg.a + 1e-9))
    return W.get_config(cfg.index, tuple(max(c_min, min(c, full)) for full in cfg.cells))


def run_oracle_steps(cfg: W.Config, n_steps: int):
    """Times oracle.md (initial evaluation + n_steps velocity-Verlet steps, fp64, brute-force
    neighbours every evaluation).  Returns (seconds, atoms, evaluations)."""
    import oracle
    s, p = W.make_system(cfg), W.make_params(cfg)
    oracle.lib()
    t0 = time.perf_counter()
    oracle.md(cfg.hyper, p, s.pos, s.vel, s.types, s.masses, s.box, cfg.dt_fs, n_steps)
    return time.perf_counter() - t0, len(s.pos), n_steps + 1


def cpu_baseline(cfg: W.Config):
    """The oracle on the host cores: its force evaluation GIVEN its neighbour lists, and
    the O(N^2) brute-force search reported separately (oracle.last_timing: wall clock of the two parts of one
    oracle.compute call).  cfg 0 and cfg 1 in full, cfg 2-4 on a 32,000-atom replica."""
    import oracle
    full = cfg.index in (0, 1)
    scfg = cfg if full else oracle_sample_config(cfg, 32000)
    s, p = W.make_system(scfg), W.make_params(scfg)
    n = len(s.pos)
    oracle.lib()
    reps = 50 if n < 5000 else 1
    t_search = t_eval = 0.0
    t0 = time.perf_counter()
    for _ in range(reps):
        oracle.compute(scfg.hyper, p, s.pos, s.types, s.box)
        a, b = oracle.last_timing()
        t_search += a / reps
        t_eval += b / reps
    t_cmp = (time.perf_counter() - t0) / reps
    what = (f"all {n} atoms of {cfg.name}" if full else
            f"{n}-atom replica ({'x'.join(map(str, scfg.cells))} cells) of {cfg.name}")
    return {"value": n / t_eval, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
            "sample": f"{what}: fp64 energy/force/virial evaluation given the neighbour lists, {t_eval:.3f} s of the "
                      f"{t_cmp:.3f} s of one oracle.compute call (mean of {reps}); the rest is its O(N^2) search",
            "search": {"seconds": t_search, "atoms_per_s": n / t_search,
                       "what": "O(N^2) brute-force pair search of the same call (radial + angular lists)"},
            "with_search_value": n / t_cmp}


def config_dict(cfg: W.Config, n_atoms: int, extra=None):
    h = cfg.hyper
    d = {"workload": cfg.name, "atoms": n_atoms, "species": h.n_types,
         "rc_radial_angular": [h.rc_radial, h.rc_angular], "n_max": [h.n_max_radial, h.n_max_angular],
         "basis": [h.basis_radial, h.basis_angular], "l_max": [h.l_max_3b, h.l_max_4b, h.l_max_5b],
         "neurons": h.n_neurons, "n_descriptors": h.n_des, "dt_fs": cfg.dt_fs, "skin": cfg.skin,
         "rebuild_every": cfg.rebuild_every, "temperature_K": cfg.temperature}
    if extra:
        d.update(extra)
    return d


def run_reference(args):
    """--impl reference: the oracle, as it stands, on the host cores; each step a bounded sample."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    import oracle
    cfg = W.get_config(args.config)
    budget_s = 150.0
    rate_guess = 600.0 * oracle.num_threads()             # atom-step/s of the oracle, order of magnitude
    n_target = int(min(32000, max(2000, rate_guess * budget_s / (args.steps + args.warmup + 1))))
    scfg = oracle_sample_config(cfg, n_target)
    if args.warmup > 0:
        run_oracle_steps(scfg, max(0, args.warmup - 1))
    secs, n, evals = run_oracle_steps(scfg, args.steps)
    value = n * args.steps / secs
    sample = (f"{n}-atom replica ({'x'.join(map(str, scfg.cells))} cells) of {cfg.name} per step; "
              f"{args.steps} NVE steps + initial evaluation timed together")
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": secs / args.steps * 1e3,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic (seeded lattice + random weights, workloads.py)",
            "config": config_dict(cfg, n, {"sample": sample}),
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
                             "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)
    return 0


# ---------------------------------------------------------------------------------------------------
def max_over_ranks(x: float, world: int, device: str = "cpu") -> float:
    """MAX all-reduce of one float over the ranks (the job's time is the slowest rank's)."""
    if world == 1:
        return float(x)
    import torch
    import torch.distributed as dist
    t = torch.tensor([x], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(world: int, atoms_per_rank: int, steps: int, ms_max: float) -> float:
    """Replicas only: every rank advances its own `atoms_per_rank` atoms by `steps` steps."""
    return world * atoms_per_rank * steps / (ms_max * 1e-3)


def launch_replicas(args) -> int:
    """`python bench.py --gpus N` with N > 1 and no torchrun environment: start N ranks of this same command, one
    replica per GPU, under torch.distributed.run on 127.0.0.1 (the launch line the driver uses).  Replicas only:
    the ranks share nothing but the barrier and the MAX-over-ranks time (north_star: no sharding, no collectives)."""
    import socket
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    return subprocess.run(cmd).returncode


def run_dry(args, rank: int, world: int) -> int:
    """--dry: the multi-rank entry path without any CUDA work (CPU boxes, tests): rendezvous over gloo, a barrier,
    a synthetic per-rank time through the same max_over_ranks / whole_job_value the timed arm uses, and rank 0's
    ONE line.  Not a measurement: "dry": true, value from the synthetic times."""
    import torch.distributed as dist
    cfg = W.get_config(args.config)
    n = int(np.prod(cfg.cells)) * len(W._BASIS[cfg.lattice])
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("gloo")
        dist.barrier()
    ms = max_over_ranks(10.0 + 5.0 * rank, world, "cpu")
    value = whole_job_value(world, n, args.steps, ms)
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    if rank == 0:
        print(json.dumps({"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                          "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True,
                          "scaling": "weak", "vs_baseline": None, "dtype": "f32", "dry": True,
                          "data": "none: --dry runs the launch path only (synthetic per-rank times, no CUDA work)",
                          "config": config_dict(cfg, n, {"parallelism": "replicas only" if world > 1 else "single GPU"}),
                          "gpu_launches": 0, "impl": "ours"}), flush=True)
    return 0


def run_ours(args):
    import torch
    import torch.distributed as dist
    import paper_2205_10046_b200 as pkg
    from paper_2205_10046_b200 import NEP          # raises if libnep_b200.so is missing: no fallback

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if args.dry:
        return run_dry(args, rank, world)
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the NEP path has no CPU fallback)")
    torch.cuda.set_device(local)
    dev = f"cuda:{local}"
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=torch.device(dev))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    cfg = W.get_config(args.config)
    s, p = W.make_system(cfg), W.make_params(cfg)
    n = len(s.pos)
    K, Wm = args.steps, args.warmup
    nep = NEP(cfg.hyper, p, s.masses, device=local)
    pos = torch.tensor(s.pos, device=dev)
    vel = torch.tensor(s.vel, device=dev)
    types = torch.tensor(s.types, device=dev)

    # ---- device-resident arm: inputs already in HBM when the timed region starts
    nep.nep_neighbors(pos, types, s.box, cfg.skin)
    nep.md_step(pos, vel, cfg.dt_fs, Wm, cfg.rebuild_every, cfg.skin)            # warm-up (untimed)
    barrier()
    sampler = ClockSampler(local)
    sampler.start()
    time.sleep(0.15)
    l0 = nep.nep_launch_count()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    windows = None
    profiled_ms = None
    if args.windows and args.windows > 1:
        nep.nep_profile(True)
        # --windows W: the K steps as W consecutive md_step calls, each bracketed by its own event pair and a
        # synchronize; between two windows the pair counts are read back (untimed).  ms = sum of the windows.
        # Shows how ms/step moves with the trajectory (the in-cutoff pair counts grow as the lattice disorders).
        windows, ms, prev = [], 0.0, {}
        edges = [round(K * w / args.windows) for w in range(args.windows + 1)]
        for w in range(args.windows):
            kw = edges[w + 1] - edges[w]
            if kw <= 0:
                continue
            barrier()
            ev0.record()
            nep.md_step(pos, vel, cfg.dt_fs, kw, cfg.rebuild_every, cfg.skin)
            ev1.record()
            barrier()
            ms_w = max_over_ranks(ev0.elapsed_time(ev1), world, dev)
            ms += ms_w
            pr, pa = nep.nep_pair_counts()
            cum = nep.nep_profile_read()                      # cumulative since nep_profile(True): difference = this window
            kus = {k: (v[0] - prev.get(k, (0.0, 0))[0]) / max(1, v[1] - prev.get(k, (0.0, 0))[1]) * 1e3
                   for k, v in cum.items() if v[1] > prev.get(k, (0.0, 0))[1]}
            prev = cum
            windows.append({"steps": [edges[w], edges[w + 1]], "ms_per_step": ms_w / kw,
                            "pairs_in_rc_per_atom": [pr / n, pa / n],
                            "longest_skin_lists": [nep.nep_max_neighbors(0), nep.nep_max_neighbors(1)],
                            "list_raggedness": nep.nep_list_raggedness(),
                            "kernel_avg_us": {k: round(v, 2) for k, v in kus.items()},
                            "force_angular_ns_per_pair": kus.get("force_angular", 0.0) * 1e3 / max(1, pa),
                            "force_radial_ns_per_pair": kus.get("force_radial", 0.0) * 1e3 / max(1, pr)})
    else:
        # the timed region runs WITHOUT the library's per-kernel events: an event pair around each of the ~13 launches
        # of a step costs 2.4 % of the step at 1M atoms (2.61 -> 2.67 ms).  The per-kernel durations behind `roofline`
        # and `kernels` are taken, still live and with CUDA events on the library's stream, over the K steps that
        # follow directly (same workload, same cadence; `profiled_ms_per_step` is that pass's own wall time).
        barrier()
        ev0.record()
        nep.md_step(pos, vel, cfg.dt_fs, K, cfg.rebuild_every, cfg.skin)
        ev1.record()
        barrier()
        ms = max_over_ranks(ev0.elapsed_time(ev1), world, dev)
    clocks = sampler.stop()
    launches = nep.nep_launch_count() - l0
    if windows is None:
        nep.nep_profile(True)
        barrier()
        ev0.record()
        nep.md_step(pos, vel, cfg.dt_fs, K, cfg.rebuild_every, cfg.skin)
        ev1.record()
        barrier()
        profiled_ms = ev0.elapsed_time(ev1)
    prof = nep.nep_profile_read()
    nep.nep_profile(False)
    pairs_r, pairs_a = nep.nep_pair_counts()
    cnt_r, _ = nep.nep_get_neighbors(0)
    cnt_a, _ = nep.nep_get_neighbors(1)
    list_r, list_a = int(cnt_r.sum().item()), int(cnt_a.sum().item())
    del cnt_r, cnt_a
    disp = nep.nep_max_displacement()
    dev_bytes = nep.nep_device_bytes()
    assert torch.isfinite(pos).all() and torch.isfinite(vel).all(), "non-finite state after the timed region"
    value = whole_job_value(world, n, K, ms)

    # ---- end-to-end arm: md_run_host with pinned host buffers, one call per step
    pos_h = torch.tensor(s.pos).pin_memory()
    vel_h = torch.tensor(s.vel).pin_memory()
    typ_h = torch.tensor(s.types).pin_memory()
    e_h = torch.empty(n, dtype=torch.float64).pin_memory()
    f_h = torch.empty((n, 3), dtype=torch.float64).pin_memory()
    nep.md_run_host(pos_h, vel_h, typ_h, s.box, cfg.dt_fs, 1, cfg.rebuild_every, cfg.skin, e_h, f_h)   # starts the run
    for _ in range(max(3, min(Wm, 10))):
        nep.md_run_host(pos_h, vel_h, None, None, cfg.dt_fs, 1, cfg.rebuild_every, cfg.skin, e_h, f_h)
    barrier()
    ev0.record()
    for _ in range(K):
        nep.md_run_host(pos_h, vel_h, None, None, cfg.dt_fs, 1, cfg.rebuild_every, cfg.skin, e_h, f_h)
    ev1.record()
    barrier()
    ms_e2e = max_over_ranks(ev0.elapsed_time(ev1), world, dev)
    h2d = pos_h.numel() * 8 + vel_h.numel() * 8
    d2h = h2d + e_h.numel() * 8 + f_h.numel() * 8
    e2e = {"value": whole_job_value(world, n, K, ms_e2e), "unit": UNIT, "h2d_bytes_per_step": h2d,
           "d2h_bytes_per_step": d2h, "ms_per_step": ms_e2e / K,
           "api": "md_run_host(n_steps=1) per step, pinned host pos/vel in, pos/vel/energy/force out"}

    # ---- rooflines
    fp32_probe = nep.nep_probe_fp32()
    hbm_peak, hbm_src = measured_peaks()
    alu_peak = SM_COUNT * FP32_LANES * 2 * SM_MAX_MHZ_NOMINAL * 1e6 / 1e12        # TFLOP/s, derived
    costs = kernel_costs(cfg.hyper, n, pairs_r, pairs_a, list_r, list_a)
    traffic = ncu_traffic(cfg.name)
    t_sum = sum(v[0] for v in prof.values())
    kernels = []
    builds = prof.get("build_lists", (0.0, 0))[1]
    for name, (tot_ms, cnt) in sorted(prof.items(), key=lambda kv: -kv[1][0]):
        avg_s = tot_ms / cnt * 1e-3
        entry = {"name": name, "launches": cnt, "avg_us": avg_s * 1e6, "share": tot_ms / t_sum}
        if name in costs and avg_s > 0:
            fl, by = costs[name]
            if name in PER_BUILD_IDS and builds > 0 and cnt != builds:
                # several launches share this id in one build: the cost stated is per build
                fl, by = fl * builds / cnt, by * builds / cnt
                costs[name] = (fl, by)
            entry.update({"tflops": fl / avg_s / 1e12, "alu_frac": fl / avg_s / 1e12 / alu_peak,
                          "gbs": by / avg_s / 1e9, "hbm_frac": by / avg_s / 1e9 / hbm_peak,
                          "flops_per_launch": fl, "bytes_per_launch": by})
        if name == "ann" and "tflops" in entry:
            # the network runs on the tensor cores (3xTF32 mma.sync): its contraction peak is the TF32 one;
            # algorithmic flops are counted once (the split issues three MMAs per product)
            tf32_peak, tf32_src = measured_tf32_peak()
            entry.update({"tensor_frac": entry["tflops"] / tf32_peak, "tensor_peak_tflops": tf32_peak,
                          "tensor_peak_source": tf32_src})
        kernels.append(entry)
    top = next((k for k in kernels if "tflops" in k), None)
    roofline = None
    if top is not None:
        if top["alu_frac"] >= top["hbm_frac"]:
            roofline = {"kernel": top["name"], "bound": "alu", "achieved": top["tflops"], "peak": alu_peak,
                        "unit": "TFLOP/s", "frac": top["alu_frac"],
                        "peak_source": "derived: 148 SMs x 128 FP32 lanes x 2 x 1.965 GHz (DESIGN.md)",
                        "peak_probe_tflops": fp32_probe, "frac_of_probe": top["tflops"] / fp32_probe}
        else:
            roofline = {"kernel": top["name"], "bound": "hbm", "achieved": top["gbs"], "peak": hbm_peak,
                        "unit": "GB/s", "frac": top["hbm_frac"], "peak_source": hbm_src}
        roofline["traffic"] = traffic.get(top["name"])
        roofline["avg_us"] = top["avg_us"]
        roofline["share_of_step"] = top["share"]
    step_flops = sum(costs[k["name"]][0] * k["launches"] for k in kernels if k["name"] in costs) / K
    step_bytes = sum(costs[k["name"]][1] * k["launches"] for k in kernels if k["name"] in costs) / K
    step = {"flops_per_atom": step_flops / n, "bytes_per_atom": step_bytes / n,
            "tflops": world * step_flops * K / (ms * 1e-3) / 1e12 / world,
            "alu_frac": step_flops * K / (ms * 1e-3) / 1e12 / alu_peak,
            "hbm_frac": step_bytes * K / (ms * 1e-3) / 1e9 / hbm_peak,
            "kernel_time_share_of_wall": t_sum / (profiled_ms if profiled_ms else ms) if world == 1 else None,
            "kernel_timing": ("CUDA-event pair per launch over the K steps after the timed region" if profiled_ms
                              else "CUDA-event pair per launch inside the timed windows"),
            "profiled_ms_per_step": profiled_ms / K if profiled_ms else None}

    nb_ids = ("cell_hist", "scan", "scatter", "sort_cells", "build_lists", "build_rev")
    nb_ms = sum(prof[k][0] for k in nb_ids if k in prof)
    neighbour_pass = None
    if builds > 0:
        nb_bytes = sum(costs[k][1] * prof[k][1] for k in nb_ids if k in prof and k in costs) / builds
        neighbour_pass = {"builds": builds, "us_per_build": nb_ms / builds * 1e3, "share_of_step": nb_ms / t_sum,
                          "bytes_per_build": nb_bytes, "gbs": nb_bytes / (nb_ms / builds * 1e-3) / 1e9,
                          "hbm_frac": nb_bytes / (nb_ms / builds * 1e-3) / 1e9 / hbm_peak,
                          "note": "plus one k_quantize per build (counted under quantize)"}

    cpu = cpu_baseline(cfg) if (rank == 0 and world == 1 and not args.no_cpu_baseline) else None

    if rank == 0:
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": Wm,
                "ms_per_step": ms / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                "dtype": "f32", "data": "synthetic (seeded lattice + random weights, workloads.py)",
                "config": config_dict(cfg, n, {
                    "parallelism": "replicas only" if world > 1 else "single GPU",
                    "library": pkg.lib_path(), "library_override_NEP_B200_LIB": pkg.lib_overridden(),
                    "l2_policy": f"inputs larger than L2: the handle's per-step working set is "
                                 f"{dev_bytes / 1e6:.0f} MB of device memory vs 126 MB of L2",
                    "pairs_in_rc_per_atom": [pairs_r / n, pairs_a / n],
                    "list_entries_per_atom": [list_r / n, list_a / n],
                    "max_displacement_since_build": disp,
                    "list_raggedness": nep.nep_list_raggedness()}),
                "clocks": clocks, "e2e": e2e, "gpu_launches": launches, "roofline": roofline,
                "kernels": kernels, "step": step, "neighbour_pass": neighbour_pass, "windows": windows,
                "fp32_probe_tflops": fp32_probe,
                "cpu_baseline": cpu, "impl": "ours"}
        print(json.dumps(line), flush=True)
    nep.close()
    if world > 1:
        dist.destroy_process_group()
    return 0


# ---------------------------------------------------------------------------------------------------
def run_batch(args):
    """--workload batch: SURVEY.md 8(f) row 4, one SNES generation's evaluation -- a population of parameter sets
    x a batch of small structures (nep_batch_compute) + the data terms of Eq. (33) per member (nep_batch_loss).
    Not BASELINE.json's metric (that is the MD step above): a second, separately named line for the widened row.
    A "step" = one generation: parameters uploaded from the host, E/F/W of every (member, atom), loss [n_pop][3]
    read back to the host.  Structures: seeded replicas of cfg 3's five-species fcc lattice, 16-108 atoms, a third
    of them sheared, most thinner than 2 r_c (lattice-image neighbours, reading A18)."""
    import torch
    import paper_2205_10046_b200 as pkg
    from paper_2205_10046_b200 import NEP
    if int(os.environ.get("RANK", "0")) != 0:
        return 0
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the NEP path has no CPU fallback)")
    cfg = W.get_config(3)
    shapes = [(2, 2, 2), (2, 2, 1), (3, 2, 2), (3, 3, 2), (3, 3, 3), (2, 1, 1)]
    tilts = [None, None, (0.21, -0.13, 0.17)]
    specs = [(shapes[k % len(shapes)], tilts[k % len(tilts)], k) for k in range(args.structures)]
    structs = W.make_batch(3, specs)
    members = W.make_population(cfg, args.pop, sigma=0.3)
    off = np.concatenate([[0], np.cumsum([len(p) for p, _, _ in structs])]).astype(np.int32)
    N, S, P = int(off[-1]), len(structs), len(members)
    pos = torch.tensor(np.concatenate([p for p, _, _ in structs]), device="cuda:0")
    typ = torch.tensor(np.concatenate([t for _, t, _ in structs]), device="cuda:0")
    boxes = np.stack([H for _, _, H in structs])
    nep = NEP(cfg.hyper, members[0], cfg.masses, device=0)
    nep.nep_batch_neighbors(off, pos, typ, boxes)
    rng = np.random.default_rng(7)
    u_t = torch.tensor(rng.normal(size=S), device="cuda:0")
    f_t = torch.tensor(rng.normal(size=(N, 3)) * 0.1, device="cuda:0")
    w_t = torch.tensor(rng.normal(size=(S, 6)) * 0.1, device="cuda:0")

    def generation():
        e, f, w = nep.nep_batch_compute(members)
        return nep.nep_batch_loss(e, f, w, u_t, f_t, w_t).cpu()

    for _ in range(max(3, args.warmup)):
        loss = generation()
    torch.cuda.synchronize()
    nep.nep_profile(True)                                   # per-kernel times of one extra, untimed generation
    generation()
    prof = nep.nep_profile_read()
    nep.nep_profile(False)
    ent_r, ent_a = nep.nep_batch_pair_counts()
    l0 = nep.nep_launch_count()
    sampler = ClockSampler(0)                               # SM clock and throttle reasons DURING the timed region
    sampler.start()
    time.sleep(0.15)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev0.record()
    for _ in range(args.steps):
        loss = generation()
    ev1.record()
    torch.cuda.synchronize()
    clocks = sampler.stop()
    ms = ev0.elapsed_time(ev1)
    assert torch.isfinite(loss).all()
    # a generation IS end to end: every step uploads the population's parameters from host arrays (nep_batch_compute
    # takes host pointers) and reads the loss back to the host; the structures are the fixed training set, resident
    par_bytes = int(sum(getattr(m_, k_).nbytes for m_ in members for k_ in ("c_radial", "c_angular", "w0", "b0", "w1", "b1")))
    e2e = {"value": N * P * args.steps / (ms * 1e-3), "unit": "atom-member evaluation/s",
           "h2d_bytes_per_step": par_bytes, "d2h_bytes_per_step": int(loss.numel() * loss.element_size()),
           "what": "same timed region: host parameter arrays in, loss [n_pop][3] back on the host, every generation"}
    launches = nep.nep_launch_count() - l0
    # oracle on the host cores: compute_images of a few structures with one member
    cpu = None
    if not args.no_cpu_baseline:
        import oracle
        # as cpu_baseline(): the evaluation GIVEN the lists is the value, the brute-force lattice-image pair
        # search of the same calls (oracle.last_timing) is reported beside it
        t0, na, t_search, t_eval = time.perf_counter(), 0, 0.0, 0.0
        for k in range(min(S, 12)):
            p_, t_, H_ = structs[k]
            oracle.compute_images(cfg.hyper, members[0], p_, t_, H_)
            a, b = oracle.last_timing()
            t_search += a
            t_eval += b
            na += len(p_)
        dt = time.perf_counter() - t0
        cpu = {"value": na / t_eval, "unit": "atom-member evaluation/s", "cores": oracle.num_threads(), "kind": "oracle",
               "sample": f"oracle.compute_images of the first {min(S, 12)} structures ({na} atoms), one member: fp64 "
                         f"evaluation given the lists, {t_eval:.3f} s of the {dt:.3f} s of those calls; the rest is the "
                         f"brute-force lattice-image search",
               "search": {"seconds": t_search, "atoms_per_s": na / max(t_search, 1e-12),
                          "what": "brute-force lattice-image pair search of the same calls"},
               "with_search_value": na / dt}
    line = {"metric": "atom-member evaluation/s (batched training evaluation, SURVEY.md 8(f) row 4)",
            "value": N * P * args.steps / (ms * 1e-3), "unit": "atom-member evaluation/s", "n_gpus": 1,
            "steps": args.steps, "warmup": max(3, args.warmup), "ms_per_step": ms / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f32",
            "data": "synthetic (seeded small structures + a seeded population, workloads.py)",
            "config": {"workload": "batch_cfg3_fcc_alloy_small_cells", "structures": S, "atoms": N, "population": P,
                       "library": pkg.lib_path(), "library_override_NEP_B200_LIB": pkg.lib_overridden(),
                       "atoms_per_structure": [int(np.diff(off).min()), int(np.diff(off).max())],
                       "neighbour_entries_per_atom": None,
                       "step": "host parameters -> nep_batch_compute (E, F, W of every member) -> nep_batch_loss -> host [n_pop][3]"},
            "gpu_launches": launches, "cpu_baseline": cpu, "impl": "ours", "clocks": clocks, "e2e": e2e,
            "kernels": [{"name": k, "launches": v[1], "avg_us": v[0] / v[1] * 1e3} for k, v in sorted(prof.items(), key=lambda kv: -kv[1][0])]}
    # roofline of the dominant kernel (kb_partial: Eq. (21) of every entry and member), algorithmic flops as in
    # kernel_costs (force_angular + force_radial per ordered pair), against the derived FP32 peak
    h = cfg.hyper
    fl = P * (ent_a * (4 * h.NA * h.KA + 4 * 24 * h.NA + 500) + N * 3 * 24 * h.NA + ent_r * (55 + 4 * h.KR + 2 * h.NR * h.KR))
    if "batch_partial" in prof:
        us = prof["batch_partial"][0] / prof["batch_partial"][1] * 1e3
        alu_peak = SM_COUNT * FP32_LANES * 2 * SM_MAX_MHZ_NOMINAL * 1e6 / 1e12
        line["roofline"] = {"kernel": "batch_partial", "bound": "alu", "achieved": fl / us / 1e6, "peak": alu_peak, "unit": "TFLOP/s",
                            "frac": fl / us / 1e6 / alu_peak, "avg_us": us,
                            "traffic": ncu_traffic("batch_cfg3_fcc_alloy_small_cells").get("batch_partial") if (S, P) == (600, 50) else None,
                            "peak_source": "derived: 148 SMs x 128 FP32 lanes x 2 x 1.965 GHz (DESIGN.md)"}
    line["config"]["neighbour_entries_per_atom"] = [ent_r / N, ent_a / N]
    print(json.dumps(line), flush=True)
    nep.close()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--config", type=int, default=3, help="index into BASELINE.json configs (default 3: 1M atoms)")
    ap.add_argument("--impl", choices=["ours", "reference"], default="ours")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--workload", choices=["md", "batch"], default="md",
                    help="md: BASELINE.json's metric (default); batch: the batched training evaluation of SURVEY 8(f) row 4")
    ap.add_argument("--structures", type=int, default=600, help="--workload batch: structures in the batch")
    ap.add_argument("--pop", type=int, default=50, help="--workload batch: parameter sets (PAPER.md:283: a population)")
    ap.add_argument("--windows", type=int, default=0,
                    help="time the K steps as this many consecutive windows (ms/step and pair counts per window)")
    ap.add_argument("--dry", action="store_true",
                    help="launch path only: ranks rendezvous over gloo and print the line from synthetic times (no CUDA)")
    args = ap.parse_args()
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ and args.workload == "md":
        return launch_replicas(args)                      # N replicas, one per GPU; this process only waits
    if args.warmup < 3:
        args.warmup = 3                                   # timing rule: at least 3 warm-up steps
    if args.impl == "reference":
        return run_reference(args)
    if args.workload == "batch":
        return run_batch(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
