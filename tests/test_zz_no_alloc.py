"""fs_scan_static: the switching scan for programs that cannot allocate device memory.

Some users of this library run it inside a process whose own memory pool already holds the card (a torch caching
allocator that was given the HBM, a solver that reserves it at start-up), or next to other busy streams that a
cudaMalloc / cudaFree would stall, since both synchronise the whole device.  For them the library has one entry point
that needs no handle and no workspace and allocates nothing: its per-CTA partial results sit in a fixed 65,792-byte
array inside the library image, which limits it to FS_SCAN_STATIC_MAX_N = 4,194,304 spins.

What is checked here: on two calls in a row (same stream, nothing in between, different field and thermal step, so a
value left in the shared array by the first call would show in the second) the entry point returns what the existing
path -- fs_create + fs_update_fields + fs_scan, whose scratch is the caller's workspace -- returns for the same state:
the count of switchable spins and the arg-max index bit for bit, the Eq. 5 left-hand side within 1e-12 relative (the
bar of tests/test_gpu_parity.py).  Then a smaller system right behind a larger one (stale partial results behind the
live ones), and the size limit.

This file sorts last on purpose (pytest -x stops at the first failure): it passes alone in a fresh process and behind
the rest of the suite.
"""
import ctypes

import numpy as np
import pytest


def test_scan_static_rejects_sizes_beyond_the_static_array():
    """Host logic only (runs without a GPU): N beyond the array's capacity is an argument error with the limit in the
    message, and nothing is launched."""
    from paper_2002_11401_b200.binding import load_library, FsParams, FS_ERR_ARG, SCAN_STATIC_MAX_N
    L = load_library()
    p = FsParams(0.001, 1, 1, 3, 3, 1.0)
    before = L.fs_kernel_launches()
    dummy = ctypes.c_void_p(256)                       # never dereferenced: the size check comes first
    rc = L.fs_scan_static(SCAN_STATIC_MAX_N + 1, dummy, dummy, dummy, dummy, ctypes.byref(p), 0.0, 0.0, 0.0, 0, 0, dummy, None)
    assert rc == FS_ERR_ARG
    msg = L.fs_last_error().decode()
    assert str(SCAN_STATIC_MAX_N) in msg and "FS_SCAN_STATIC_MAX_N" in msg
    assert L.fs_scan_static(0, dummy, dummy, dummy, dummy, ctypes.byref(p), 0.0, 0.0, 0.0, 0, 0, dummy, None) == FS_ERR_ARG
    assert L.fs_scan_static(10, None, dummy, dummy, dummy, ctypes.byref(p), 0.0, 0.0, 0.0, 0, 0, dummy, None) == FS_ERR_ARG
    assert L.fs_kernel_launches() == before


def _unpack(res):
    import torch
    r = res.cpu()
    return int(r[0]), int(r[1]), float(r[2:3].view(torch.float64)[0])


def _same(got, want):
    """count and arg-max index bit for bit; Eq. 5 left-hand side at the suite's 1e-12 (both -inf when nothing switches)"""
    assert got[:2] == want[:2], (got, want)
    if want[0] == 0:
        assert got[1] == -1 and got[2] == -np.inf and want[2] == -np.inf
    else:
        assert abs(got[2] - want[2]) <= 1e-12 * abs(want[2]), (got, want)


@pytest.mark.gpu
def test_scan_static_matches_fs_scan_on_two_calls_in_a_row():
    import torch
    from paper_2002_11401_b200 import workloads as W
    from paper_2002_11401_b200.binding import Sim, scan_static, FIELD_DIP

    assert torch.cuda.is_available()
    dev = torch.device("cuda:0")
    # config-4 recipe at 300 x 300: 180,600 spins = 176 full CTAs of 1024 spins + a ragged one of 376; thermal field on
    w = W.config("4", scale=300)
    spins = W.random_spins(w.N, seed=7)
    sim = Sim(w.pos, w.angle, w.hc, w.params, device="cuda:0")
    sim.set_spins(spins)
    sim.set_thermal(w.sigma_th, w.thermal_seed)
    sim.update_fields()
    hdip = sim.get_fields(FIELD_DIP).contiguous()
    ang = torch.as_tensor(np.ascontiguousarray(w.angle, np.float64)).to(dev)
    hc = torch.as_tensor(np.ascontiguousarray(w.hc, np.float64)).to(dev)
    s = torch.as_tensor(np.ascontiguousarray(spins, np.int8)).to(dev)

    # the existing path: two field values of the ramp (the first leaves ~half of the spins switchable, the second few)
    steps = [0, (2 * len(w.fields)) // 5]
    want = []
    for t in steps:
        hx, hy = w.fields[t]
        sim.set_field(hx, hy, t)
        want.append(sim.scan())
    assert want[0][0] > 0 and want[0] != want[1]

    # set-up call (looks up the array's address once per device), then the two calls under test, back to back
    res = [torch.empty(3, dtype=torch.int64, device=dev) for _ in range(3)]
    scan_static(ang, hc, s, hdip, w.params, *w.fields[steps[1]], w.sigma_th, w.thermal_seed, steps[1], result=res[2])
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    for k, t in enumerate(steps):
        hx, hy = w.fields[t]
        scan_static(ang, hc, s, hdip, w.params, hx, hy, w.sigma_th, w.thermal_seed, t, result=res[k])
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0           # nothing was taken from the device between the two reads
    for k in range(2):
        _same(_unpack(res[k]), want[k])
    _same(_unpack(res[2]), want[1])

    # a small system right behind the large one: the array still holds 176 stale partial results behind the 3 live ones
    n_small = 2 * 1024 + 100
    sub = Sim(w.pos[:n_small], w.angle[:n_small], w.hc[:n_small], w.params, device="cuda:0")
    sub.set_spins(spins[:n_small]); sub.set_thermal(w.sigma_th, w.thermal_seed)
    hx, hy = w.fields[steps[0]]
    sub.set_field(hx, hy, steps[0])
    want_small = sub.scan()
    hdip_small = sub.get_fields(FIELD_DIP).contiguous()
    scan_static(ang, hc, s, hdip, w.params, hx, hy, w.sigma_th, w.thermal_seed, steps[0], result=res[0])
    scan_static(ang[:n_small], hc[:n_small], s[:n_small], hdip_small, w.params, hx, hy, w.sigma_th, w.thermal_seed,
                steps[0], result=res[1])
    _same(_unpack(res[1]), want_small)
    _same(_unpack(res[0]), want[0])

    # nothing switchable: -1 and -inf, as fs_scan reports it
    sim.set_thermal(0.0, 0); sim.set_field(0.0, 0.0, 0)
    quiet = sim.scan()
    scan_static(ang, hc, s, hdip, w.params, 0.0, 0.0, 0.0, 0, 0, result=res[0])
    _same(_unpack(res[0]), quiet)
