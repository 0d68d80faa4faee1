"""CPU-only checks of the boundary and the harness: the C-ABI library loads and exports every symbol
include/nep.h declares (no compute calls), the Python binding lists the same names, bench.py's
replica aggregation works over a world_size-2 gloo group, and its cost model / sample selection are sane.
"""
import os
import re
import socket
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_functions():
    text = open(os.path.join(ROOT, "include", "nep.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b((?:nep|md)_[a-z0-9_]+)\s*\(", text)))


def test_library_exports_every_declared_symbol():
    from paper_2205_10046_b200 import build, binding
    build.build()                                   # nvcc cross-compiles without a GPU
    lib = binding.load_library()
    names = declared_functions()
    assert "nep_create" in names and "md_step" in names and "nep_neighbors" in names and "nep_compute" in names
    for name in names:
        assert hasattr(lib, name), f"{name} is declared in include/nep.h but not exported"
    assert sorted(binding.exported_symbols) == names


def test_host_only_entry_points():
    """The two entry points that are pure host arithmetic work without a GPU; nep_create fails loudly."""
    import ctypes as C
    import workloads as W
    from paper_2205_10046_b200 import binding
    lib = binding.load_library()
    for idx, want in ((0, 35), (2, 37), (4, 49)):             # SURVEY.md section 8 size table
        h = binding.NepHyper.from_hyper(W.get_config(idx).hyper)
        assert lib.nep_num_descriptors(C.byref(h)) == want
    bad = binding.NepHyper.from_hyper(W.get_config(0).hyper)
    bad.l_max_3b = 3
    assert lib.nep_num_descriptors(C.byref(bad)) == -1
    assert lib.nep_status_string(-4) == b"neighbour list overflow"
    assert lib.nep_profile_num_kernels() > 10
    import torch
    if not torch.cuda.is_available():
        with pytest.raises(binding.NepError):
            cfg = W.get_config(0)
            binding.NEP(cfg.hyper, W.make_params(cfg), [28.0])


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    import bench
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    ms = bench.max_over_ranks(10.0 + 5.0 * rank, world, "cpu")          # rank 1 is the slow one
    out[rank] = bench.whole_job_value(world, 1000, 7, ms)
    dist.barrier()
    dist.destroy_process_group()


def test_replica_aggregation_gloo_world2():
    import torch.multiprocessing as mp
    mgr = mp.Manager()
    out = mgr.dict()
    mp.spawn(_worker, args=(2, _free_port(), out), nprocs=2, join=True)
    want = 2 * 1000 * 7 / 15.0e-3
    assert out[0] == pytest.approx(want) and out[1] == pytest.approx(want)


def test_bench_gpus_2_starts_two_ranks_dry():
    """`python bench.py --gpus 2` must START two ranks (it used to run one and print n_gpus 1): the
    same entry path as the timed arm -- re-exec under torch.distributed.run on 127.0.0.1, rendezvous, barrier,
    MAX over ranks, one line from rank 0 -- with --dry standing in for the CUDA work (gloo, no GPU here)."""
    import json
    import subprocess
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "WORLD_SIZE", "LOCAL_RANK", "MASTER_PORT")}
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--dry", "--steps", "7", "--config", "1"],
                       capture_output=True, text=True, timeout=600, env=env, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1, r.stdout
    d = json.loads(lines[0])
    assert d["n_gpus"] == 2 and d["dry"] is True and d["scaling"] == "weak"
    assert d["config"]["parallelism"] == "replicas only" and d["config"]["atoms"] == 64000
    assert d["value"] == pytest.approx(2 * 64000 * 7 / 15.0e-3)      # the slow rank's 15 ms decides
    # N = 1: no launcher, no process group, same line shape
    r1 = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "1", "--dry", "--steps", "7", "--config", "1"],
                        capture_output=True, text=True, timeout=600, env=env, cwd=ROOT)
    d1 = json.loads([l for l in r1.stdout.splitlines() if l.startswith("{")][0])
    assert d1["n_gpus"] == 1 and d1["value"] == pytest.approx(64000 * 7 / 10.0e-3)


def test_cost_model_matches_survey_table():
    """cfg 0/1/3 radial pair 161 + 307 flops, angular pair 420 + 1,160 + 30.  The 307
    are BOTH directions of a pair evaluated at one atom (Alg. 2); every direction is needed once, so the
    model charges one direction per ordered pair, 55 + (307 - 55) / 2 = 181, and the 30-flop gather for
    every radial pair (an angular pair is one)."""
    sys.path.insert(0, ROOT)
    import bench
    import workloads as W
    h = W.get_config(3).hyper
    c = bench.kernel_costs(h, 0, 1, 0, 0, 0)
    assert c["radial"][0] == 161 and c["force_radial"][0] == 55 + (307 - 55) // 2 and c["final"][0] == 30
    c = bench.kernel_costs(h, 0, 1, 1, 0, 0)
    assert c["angular"][0] == 420 and c["force_angular"][0] == 1160 and c["final"][0] == 30


def test_oracle_sample_config_keeps_minimum_image():
    sys.path.insert(0, ROOT)
    import bench
    import workloads as W
    for idx in range(5):
        cfg = W.get_config(idx)
        s = bench.oracle_sample_config(cfg, 3000)
        assert all(c * cfg.a >= 2 * (cfg.hyper.rc_radial + cfg.skin) for c in s.cells)
        assert all(c <= full for c, full in zip(s.cells, cfg.cells))


def test_cpu_baseline_reports_the_evaluation_and_the_search_separately():
    """the oracle's force evaluation given its lists, the O(N^2) search beside it (the two
    parts of one oracle.compute call, oracle.last_timing); cfg 0 is timed in full."""
    sys.path.insert(0, ROOT)
    import bench
    import oracle
    import workloads as W
    cfg = W.get_config(0)
    c = bench.cpu_baseline(cfg)
    assert c["kind"] == "oracle" and c["cores"] == oracle.num_threads() and "all 256 atoms" in c["sample"]
    assert c["value"] > c["with_search_value"] > 0 and c["search"]["atoms_per_s"] > 0
    s, p = W.make_system(cfg), W.make_params(cfg)
    oracle.compute(cfg.hyper, p, s.pos, s.types, s.box)
    t_search, t_eval = oracle.last_timing()
    assert t_search > 0 and t_eval > 0


def test_neighbour_pass_has_cost_entries():
    """~0.6 kB/atom and 300-500 candidate tests per atom per build."""
    sys.path.insert(0, ROOT)
    import bench
    import workloads as W
    h = W.get_config(3).hyper
    n, lr, la = 1000, 78000, 45000
    c = bench.kernel_costs(h, n, 45000, 18000, lr, la)
    per_atom = sum(c[k][1] for k in ("cell_hist", "scatter", "sort_cells", "build_lists")) / n
    assert 500 <= per_atom <= 700
    assert 250 <= c["build_lists"][0] / 10 / n <= 500          # 3.73 x 78 = 291 candidate tests per atom
    assert c["build_rev"][1] == 5 * lr
