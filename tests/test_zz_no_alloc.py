"""nep_heat_current_static -- the heat current for callers that cannot allocate device memory (-m gpu).

Why the entry point exists: nep_heat_current keeps the per-block partial sums of J = sum_i W_i v_i in a buffer
it cudaMalloc's on first use.  A Green-Kubo sampling loop that runs inside a process whose free device memory
is already owned by another allocator (a framework's caching pool, a second simulation on the same GPU) cannot
count on that cudaMalloc succeeding, and a thread that shares the device with latency-sensitive streams cannot
afford the device-wide stall an allocation may cause.  nep_heat_current_static puts the partials in a fixed
array inside libnep_b200.so instead (limit 4,194,304 atoms) and allocates nothing.

What is checked: the new entry point launches the same two kernels in the same order as nep_heat_current, so
its J_i and J must be bitwise equal to the existing path's (the bar tests/test_gpu_derived.py uses for two calls
of nep_heat_current).  Two calls are made IN A ROW, the first on a system with more blocks than the second, with
different velocities: the shared array then still holds the first call's partials beyond the second call's
range, and a kernel that read them (or the host shadow of the array instead of its device address) would give a
wrong total.  A system above the limit must be refused with a message that names the limit.

The file's name makes pytest collect it last: `pytest -x` stops at the first failure, and a failure here must
not hide the parity tests.  Every test builds its own handles, so the file passes alone in a fresh process
(where its first call is also the per-device address look-up) and after the rest of the suite.
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


def evaluated(pkg, idx, cells, skin=1.0):
    cfg = W.get_config(idx, cells)
    s, p = W.make_system(cfg), W.make_params(cfg, "stress")
    nep = pkg.NEP(cfg.hyper, p, s.masses, device=0)
    pos = torch.tensor(s.pos, device="cuda:0")
    nep.nep_neighbors(pos, torch.tensor(s.types, device="cuda:0"), s.box, skin)
    nep.nep_compute(pos)
    return nep, s


def test_static_heat_current_equals_allocating_path_on_two_calls_in_a_row(pkg):
    big, s_big = evaluated(pkg, 3, (9, 8, 7))          # 2,016 atoms: 8 blocks of partials
    small, s_small = evaluated(pkg, 2, (4, 4, 3))      # 384 atoms: 2 blocks
    v_big = torch.tensor(s_big.vel, device="cuda:0")
    v_small = torch.tensor(3.0 * s_small.vel[::-1].copy(), device="cuda:0")
    # outputs are made by the caller BEFORE the calls: the entry point and its wrapper allocate nothing
    ja_b = torch.full((big.n, 3), np.nan, dtype=torch.float64, device="cuda:0")
    jt_b = torch.full((3,), np.nan, dtype=torch.float64, device="cuda:0")
    ja_s = torch.full((small.n, 3), np.nan, dtype=torch.float64, device="cuda:0")
    jt_s = torch.full((3,), np.nan, dtype=torch.float64, device="cuda:0")
    torch.cuda.synchronize()
    # bytes owned by the handles; neither is touched by nep_heat_current before the static calls, so the
    # allocating path's scratch does not exist yet and cannot be what the static path uses
    bytes_before = big.nep_device_bytes(), small.nep_device_bytes()

    big.nep_heat_current_static(v_big, ja_b, jt_b)                 # call 1: fills 24 partials
    small.nep_heat_current_static(v_small, ja_s, jt_s)             # call 2, right behind it: reads only its 6
    torch.cuda.synchronize()
    assert (big.nep_device_bytes(), small.nep_device_bytes()) == bytes_before, "the static path allocated"

    ra_b, rt_b = big.nep_heat_current(v_big)                       # the existing path (cudaMalloc'ed partials)
    ra_s, rt_s = small.nep_heat_current(v_small)
    torch.cuda.synchronize()
    assert torch.isfinite(jt_b).all() and torch.isfinite(jt_s).all()
    assert torch.equal(ja_b, ra_b) and torch.equal(jt_b, rt_b), "call 1 differs from nep_heat_current"
    assert torch.equal(ja_s, ra_s) and torch.equal(jt_s, rt_s), "call 2 differs from nep_heat_current"
    # and the total really is the sum of the per-atom terms (1e-12 relative, as in test_gpu_derived.py)
    for ja, jt in ((ja_b, jt_b), (ja_s, jt_s)):
        ref = ja.cpu().numpy().sum(0)
        assert np.abs(jt.cpu().numpy() - ref).max() <= 1e-12 * np.abs(ja.cpu().numpy()).sum()

    # a third call with only one of the outputs (the other NULL), again behind a larger call
    big.nep_heat_current_static(v_big, ja_b, jt_b)
    jt_only = torch.full((3,), np.nan, dtype=torch.float64, device="cuda:0")
    small.nep_heat_current_static(v_small, None, jt_only)
    torch.cuda.synchronize()
    assert torch.equal(jt_only, rt_s)
    big.close()
    small.close()


def test_static_heat_current_argument_and_state_errors(pkg):
    cfg = W.get_config(0)
    s, p = W.make_system(cfg), W.make_params(cfg)
    nep = pkg.NEP(cfg.hyper, p, s.masses, device=0)
    pos, vel = torch.tensor(s.pos, device="cuda:0"), torch.tensor(s.vel, device="cuda:0")
    ja = torch.empty((len(s.pos), 3), dtype=torch.float64, device="cuda:0")
    jt = torch.empty(3, dtype=torch.float64, device="cuda:0")
    nep.nep_neighbors(pos, torch.tensor(s.types, device="cuda:0"), s.box, 0.0)
    with pytest.raises(pkg.NepError) as ei:                        # no evaluation yet
        nep.nep_heat_current_static(vel, ja, jt)
    assert ei.value.status == -5
    nep.nep_compute(pos)
    with pytest.raises(pkg.NepError) as ei:                        # both outputs NULL
        nep.nep_heat_current_static(vel, None, None)
    assert ei.value.status == -1
    nep.nep_heat_current_static(vel, ja, jt)
    ra, rt = nep.nep_heat_current(vel)
    assert torch.equal(ja, ra) and torch.equal(jt, rt)
    nep.close()


def test_static_heat_current_refuses_systems_beyond_its_limit(pkg):
    """4,244,832 atoms (fcc, 102^3 cells) > 4,194,304: refused with the limit in the message, nothing launched."""
    nep, s = evaluated(pkg, 3, (102, 102, 102))
    assert nep.n > 4194304
    vel = torch.zeros((nep.n, 3), dtype=torch.float64, device="cuda:0")
    jt = torch.full((3,), 7.0, dtype=torch.float64, device="cuda:0")
    launches = nep.nep_launch_count()
    with pytest.raises(pkg.NepError) as ei:
        nep.nep_heat_current_static(vel, None, jt)
    assert ei.value.status == -1 and "4194304" in str(ei.value)
    assert nep.nep_launch_count() == launches
    torch.cuda.synchronize()
    assert (jt == 7.0).all()
    ra, rt = nep.nep_heat_current(vel)                             # the allocating path takes it
    torch.cuda.synchronize()
    assert (rt == 0.0).all()
    nep.close()
