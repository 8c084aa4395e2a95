"""gamer_hydro_run_uniform_noalloc: the multi-step driver for callers that cannot allocate device memory.

Who those callers are: a simulation code that gave all free device memory to its own pool at start-up (a later
cudaMalloc just fails), a time-step loop running beside other streams (an allocation or a free would stall them all),
a plug-in that must leave the host process's allocator alone.  gamer_hydro_run_uniform asks them for 4 + n_groups
floats of scratch that they cannot produce; the _noalloc entry point keeps that scratch in a fixed array inside the
library (good for gamer_hydro_noalloc_max_groups() groups per box) and takes only the state and the optional dt log.

What is checked: the new entry point runs the same kernels on the same inputs as gamer_hydro_run_uniform, so its
state, its interiors and its dt log must be bit-identical to the existing path's (the existing path is the one that
is compared with the oracle, in test_uniform_grid.py).  The array is shared by every call and keeps what the last
call left in it, so the calls here come in a row with DIFFERENT boxes, states and signal speeds: a stale speed
accumulator or a stale per-group speed would change the second call's time steps.

This file is named to be collected last: `pytest -x` stops at the first failure, and a failure here must not hide
the parity tests.  It passes alone in a fresh process (the first call then also does the per-device set-up) and after
all the other tests.
"""
import ctypes

import numpy as np
import pytest

from paper_0907_3390_b200 import hydro
from paper_0907_3390_b200 import workloads as W


def test_noalloc_rejects_boxes_beyond_the_built_in_scratch_without_a_device():
    """The size check comes before anything touches the device, so it can be tested here: one group too many is
    refused with GAMER_EINVAL and a message that names the limit and the way out."""
    L = hydro.lib()
    limit = hydro.gamer_hydro_noalloc_max_groups()
    assert limit == 65536
    buf = (ctypes.c_float * 64)()
    p = (ctypes.addressof(buf) + 15) & ~15
    # 257 x 256 x 1 = 65 792 groups > 65 536
    rc = L.gamer_hydro_run_uniform_noalloc(p, p + 64, 257, 256, 1, 0, 0, 0, 1, 0, 0.5, 1.0, 1.4, None, None)
    assert rc == hydro.GAMER_EINVAL
    msg = hydro.gamer_last_error()
    assert "65536" in msg and "gamer_hydro_run_uniform" in msg, msg
    # a bad box is still a bad box
    assert L.gamer_hydro_run_uniform_noalloc(p, p + 64, 0, 1, 1, 0, 0, 0, 1, 0, 0.5, 1.0, 1.4, None, None) == hydro.GAMER_EINVAL


def _boxes():
    """Three calls in a row: a fast 2x2x2 box, then a slower and smaller 1x1x2 box with a Dirichlet end (its true
    maximum speed is below what the first call left in the scratch), then the first one again."""
    c = W.config1()
    fast = c["inp"]                                            # 8 groups, periodic 2x2x2
    slow = c["inp"][:2].copy()
    slow[:, 1:4] *= 0.5                                        # half the momenta and a quarter of the energy:
    slow[:, 4] *= 0.25                                         # every velocity and sound speed halves, dt doubles
    return c, [(fast, (2, 2, 2), (0, 0, 0), 3, 0), (slow, (2, 1, 1), (1, 0, 0), 4, 1), (fast, (2, 2, 2), (0, 0, 0), 2, 1)]


def _run(entry, inp, box, bc, n_steps, order, c, with_work):
    import torch
    gx, gy, gz = box
    n = gx * gy * gz
    d_p = torch.from_numpy(inp).cuda()
    d_i = torch.full((n, 5, 16, 16, 16), float("nan"), dtype=torch.float32, device="cuda")
    d_log = torch.zeros(n_steps, dtype=torch.float32, device="cuda")
    if with_work:
        d_work = torch.full((4 + n,), 1e30, dtype=torch.float32, device="cuda")     # garbage: the call must clear it
        entry(d_p, d_i, gx, gy, gz, bc[0], bc[1], bc[2], n_steps, order, 0.4, c["dh"], c["gamma"], d_work, d_log)
    else:
        entry(d_p, d_i, gx, gy, gz, bc[0], bc[1], bc[2], n_steps, order, 0.4, c["dh"], c["gamma"], d_log)
    torch.cuda.synchronize()
    return d_p.cpu().numpy(), d_i.cpu().numpy(), d_log.cpu().numpy()


@pytest.mark.gpu
def test_noalloc_matches_run_uniform_bit_for_bit_on_calls_in_a_row():
    c, calls = _boxes()
    dts = []
    for k, (inp, box, bc, n_steps, order) in enumerate(calls):
        ref_p, ref_i, ref_dt = _run(hydro.gamer_hydro_run_uniform, inp, box, bc, n_steps, order, c, True)
        got_p, got_i, got_dt = _run(hydro.gamer_hydro_run_uniform_noalloc, inp, box, bc, n_steps, order, c, False)
        assert np.all(np.isfinite(ref_i)) and np.all(ref_dt > 0), "call %d: the existing path itself went wrong" % k
        assert np.array_equal(got_dt.view(np.int32), ref_dt.view(np.int32)), (k, got_dt, ref_dt)
        assert np.array_equal(got_i.view(np.int32), ref_i.view(np.int32)), k
        assert np.array_equal(got_p.view(np.int32), ref_p.view(np.int32)), k
        dts.append(ref_dt)
    # the scenario does what it is meant to: the second box is slower (larger dt) than what the first call left behind
    assert dts[1][0] > 1.5 * dts[0][-1], dts
    assert np.array_equal(dts[2][0], dts[0][0])


@pytest.mark.gpu
def test_noalloc_zero_steps_is_a_pure_set_up_call():
    """n_steps = 0 is the call to make at start-up: it does the per-device set-up and leaves the state alone."""
    import torch
    c = W.config1()
    d_p = torch.from_numpy(c["inp"]).cuda()
    d_i = torch.full((8, 5, 16, 16, 16), 7.0, dtype=torch.float32, device="cuda")
    hydro.gamer_hydro_run_uniform_noalloc(d_p, d_i, 2, 2, 2, 0, 0, 0, 0, 0, 0.4, c["dh"], c["gamma"])
    torch.cuda.synchronize()
    assert np.array_equal(d_p.cpu().numpy(), c["inp"]) and bool((d_i == 7.0).all())
