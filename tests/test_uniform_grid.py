"""NEXT-3: device-side ghost fill of a single-level tiling and the multi-step driver.

CPU part: the oracle's cell-by-cell ghost fill is pinned against an independent construction (np.pad of
the assembled box, workloads.box_to_groups) and against hand-picked cells.  GPU part (-m gpu): the CUDA ghost fill is
bit-exact against the oracle; gamer_hydro_run_uniform reproduces config 2 (Sod, 100 steps) without host round trips."""
import numpy as np
import pytest

import oracle
import riemann_exact
from paper_0907_3390_b200 import hydro
from paper_0907_3390_b200 import workloads as W


def random_interiors(grid, seed=7):
    gz, gy, gx = grid
    rng = np.random.default_rng(seed)
    return rng.standard_normal((gz * gy * gx, 5, 16, 16, 16)).astype(np.float32)


@pytest.mark.parametrize("grid", [(1, 1, 1), (2, 1, 3), (2, 3, 2)])
def test_oracle_ghost_fill_periodic_equals_padded_box(grid):
    a = random_interiors(grid)
    ref = W.box_to_groups(W.groups_to_box(a, grid))          # np.pad(mode="wrap") of the assembled box, then cut
    got = oracle.ghost_fill(a, grid)
    assert got.dtype == a.dtype and np.array_equal(got, ref)


@pytest.mark.parametrize("axis", [0, 1, 2])
def test_oracle_ghost_fill_keep_is_dirichlet(axis):
    grid = (2, 2, 2)
    a = random_interiors(grid, 11)
    lo = np.arange(1, 6, dtype=np.float32)
    hi = -np.arange(1, 6, dtype=np.float32)
    ref = W.box_to_groups(W.groups_to_box(a, grid), dirichlet_axis=axis, lo_state=lo, hi_state=hi)
    bc = [0, 0, 0]
    bc[axis] = 1
    # the caller's padded array holds the boundary states in the ghost cells beyond the box (anything elsewhere)
    pre = np.full_like(ref, 123.0)
    sl = [slice(None)] * 5
    sl[4 - axis] = slice(0, 3)
    pre[tuple(sl)] = lo.reshape(1, 5, 1, 1, 1)
    sl[4 - axis] = slice(19, 22)
    pre[tuple(sl)] = hi.reshape(1, 5, 1, 1, 1)
    got = oracle.ghost_fill(a, grid, tuple(bc), padded=pre)
    # interior groups' inner faces are neighbours' data; only the box ends keep the states
    assert np.array_equal(got, ref)


def test_oracle_ghost_fill_hand_picked_cells():
    grid = (1, 2, 3)                                          # gz, gy, gx
    a = random_interiors(grid, 3)
    p = oracle.ghost_fill(a, grid)
    g = lambda kz, ky, kx: (kz * 2 + ky) * 3 + kx
    # padded (z,y,x) = (3,3,0) of group (0,0,0): box cell x = -3 -> wraps to group kx=2, interior x = 13
    assert np.array_equal(p[g(0, 0, 0), :, 3, 3, 0], a[g(0, 0, 2), :, 0, 0, 13])
    # padded x = 21 of group kx=1: box cell x = 16+18 = 34 -> group kx=2, interior x = 2
    assert np.array_equal(p[g(0, 1, 1), :, 5, 4, 21], a[g(0, 1, 2), :, 2, 1, 2])
    # padded y = 1 of group ky=0: box cell y = -2 -> ky=1, interior y = 14; z ghost wraps onto the same group (gz = 1)
    assert np.array_equal(p[g(0, 0, 1), :, 0, 1, 10], a[g(0, 1, 1), :, 13, 14, 7])
    # interior is the group's own
    assert np.array_equal(p[:, :, 3:19, 3:19, 3:19], a)


def test_oracle_run_uniform_is_the_written_out_loop():
    c = W.config1()
    grid = (2, 2, 2)
    u = c["inp"].astype(np.float64)
    got, dts = oracle.run_uniform(u, grid, (0, 0, 0), 2, 0.5, c["dh"], c["gamma"])
    v = u.copy()
    for s in range(2):
        dt = 0.5 * c["dh"] / W.max_signal_speed(v, c["gamma"])        # workloads' own fp64 Eq.30
        assert abs(dt - dts[s]) <= 1e-13 * dt
        out = oracle.hydro_advance(v, dts[s], c["dh"], c["gamma"])
        v = W.box_to_groups(W.groups_to_box(out, grid))
    assert np.array_equal(got, v)


def test_oracle_run_uniform_strang_pairs_is_the_written_out_loop():
    """order = 1: forward pass, ghost refill, backward pass with the SAME dt, ghost refill; the next
    dt comes from the state after the backward sweep (:424)."""
    c = W.config1()
    grid = (2, 2, 2)
    u = c["inp"].astype(np.float64)
    got, dts = oracle.run_uniform(u, grid, (0, 0, 0), 2, 0.4, c["dh"], c["gamma"], order=1)
    v = u.copy()
    for s in range(2):
        dt = 0.4 * c["dh"] / W.max_signal_speed(v, c["gamma"])
        assert abs(dt - dts[s]) <= 1e-13 * dt
        out = oracle.hydro_advance(v, dts[s], c["dh"], c["gamma"])
        v = W.box_to_groups(W.groups_to_box(out, grid))
        out = oracle.hydro_advance(v, dts[s], c["dh"], c["gamma"], backward=1)
        v = W.box_to_groups(W.groups_to_box(out, grid))
    assert np.array_equal(got, v)
    fwd_only, _ = oracle.run_uniform(u, grid, (0, 0, 0), 2, 0.4, c["dh"], c["gamma"], order=0)
    assert not np.array_equal(got, fwd_only)


def diagonal_wave(n, shift, gamma=5.0 / 3.0, amp=1e-6, vb=0.3):
    """Sound wave along the box diagonal (the paper's K = (1,1,1)/sqrt 3) on a uniform diagonal flow, on
    an n^3 periodic unit box: rho0 = 1, P0 = 3/5 (c_s = 1).  `shift` = distance travelled along x + y + z."""
    c = (np.arange(n) + 0.5) / n
    Z, Y, X = np.meshgrid(c, c, c, indexing="ij")
    d = amp * np.sin(2 * np.pi * (X + Y + Z - shift))
    vc = vb + d / np.sqrt(3.0)
    return W.conserved(1.0 + d, vc, vc, vc, 0.6 * (1 + gamma * d), gamma)


DIAG_SPEED = np.sqrt(3.0) * (1.0 + np.sqrt(3.0) * 0.3)      # d(x+y+z)/dt of the wave: sqrt 3 (c_s + sqrt 3 v_b)


def test_oracle_run_uniform_is_second_order_with_strang_pairs():
    """The paper's accuracy test (:450-458) through the multi-step loop with forward+backward pairs (:176): one wave
    period, CFL 0.4, fp64, 16^3 and 32^3 cells, L1 error of the density against the analytic wave at the time actually
    reached.  (On this linear wave the three sweep operators nearly commute, so forward passes alone converge at the
    same rate: the test pins the loop's bookkeeping — same dt twice, 2 dt per step, ghost refill between — not the
    splitting order; the written-out-loop test above separates order 1 from order 0.)"""
    gamma, amp = 5.0 / 3.0, 1e-6

    def run(n, order):
        dh = 1.0 / n
        grid = (n // 16,) * 3
        dt = 0.4 * dh / (1.0 + 0.3)                            # Eq.30 on the unperturbed state, to size the run
        period = 1.0 / DIAG_SPEED
        n_steps = int(round(period / (dt * (2 if order else 1))))
        u, dts = oracle.run_uniform(W.box_to_groups(diagonal_wave(n, 0.0)), grid, (0, 0, 0), n_steps, 0.4, dh, gamma,
                                    n_threads=8, order=order)
        t = sum(dts) * (2 if order else 1)
        box = W.groups_to_box(u[:, :, 3:19, 3:19, 3:19], grid)
        return np.mean(np.abs(box[0] - diagonal_wave(n, DIAG_SPEED * t)[0])) / amp

    pair16, pair32 = run(16, 1), run(32, 1)
    slope_pair = np.log2(pair32 / pair16)
    assert -2.6 <= slope_pair <= -1.5, (pair16, pair32, slope_pair)


def test_ghost_fill_argument_validation_needs_no_device():
    import ctypes
    L = hydro.lib()
    buf = (ctypes.c_float * (53240 + 20480 + 64))()
    pad = (ctypes.addressof(buf) + 15) & ~15
    inter, work = pad + 53240 * 4, pad + (53240 + 20480) * 4
    assert L.gamer_hydro_ghost_fill(inter, pad, 0, 1, 1, 0, 0, 0, None) == hydro.GAMER_EINVAL
    assert L.gamer_hydro_ghost_fill(inter, pad, 1, 1, 1, 2, 0, 0, None) == hydro.GAMER_EINVAL
    assert L.gamer_hydro_ghost_fill(None, pad, 1, 1, 1, 0, 0, 0, None) == hydro.GAMER_EINVAL
    assert L.gamer_hydro_ghost_fill(inter, pad + 4, 1, 1, 1, 0, 0, 0, None) == hydro.GAMER_EINVAL
    ru = L.gamer_hydro_run_uniform
    assert ru(pad, inter, 1, 1, 1, 0, 0, 0, 1, 0, 0.5, 1.0, 1.4, None, None, None) == hydro.GAMER_EINVAL     # no d_work
    assert ru(pad, inter, 1, 1, 1, 0, 0, 0, 1, 0, 0.0, 1.0, 1.4, work, None, None) == hydro.GAMER_EINVAL     # cfl
    assert ru(pad, inter, 1, 1, 1, 0, 0, 0, -1, 0, 0.5, 1.0, 1.4, work, None, None) == hydro.GAMER_EINVAL    # n_steps
    assert ru(pad, inter, 1, 1, 1, 0, 0, 0, 1, 2, 0.5, 1.0, 1.4, work, None, None) == hydro.GAMER_EINVAL     # order
    assert "order" in hydro.gamer_last_error()


# ---------------------------------------------------------------------------------------------------------- GPU
@pytest.mark.gpu
@pytest.mark.parametrize("grid,bc", [((1, 1, 1), (0, 0, 0)), ((2, 3, 2), (0, 0, 0)), ((2, 2, 3), (1, 0, 0)),
                                     ((3, 2, 2), (0, 1, 1)), ((2, 2, 2), (1, 1, 1)),
                                     # thin boxes: the walk along x is cut into segments (one group each for gx = 8,
                                     # one or two groups each for gx = 70 with 5 strips on 148 SMs)
                                     ((1, 1, 8), (0, 0, 0)), ((1, 1, 8), (1, 0, 0)), ((1, 1, 70), (0, 0, 0)),
                                     ((1, 1, 70), (1, 0, 0)), ((1, 2, 45), (0, 1, 0))])
def test_gpu_ghost_fill_bit_exact(grid, bc):
    import torch
    gz, gy, gx = grid
    a = random_interiors(grid, 5)
    pre = np.random.default_rng(9).standard_normal((a.shape[0], 5, 22, 22, 22)).astype(np.float32)
    ref = oracle.ghost_fill(a, grid, bc, padded=pre)
    d_a = torch.from_numpy(a).cuda()
    d_p = torch.from_numpy(pre).cuda()
    hydro.gamer_hydro_ghost_fill(d_a, d_p, gx, gy, gz, *bc)
    torch.cuda.synchronize()
    assert np.array_equal(d_p.cpu().numpy(), ref)


@pytest.mark.gpu
@pytest.mark.parametrize("axis", [0, 1, 2])
def test_gpu_run_uniform_config2_sod(axis):
    """Config 2 on the device only: 100 steps of {Eq.30, forward pass, ghost fill} in one call.  Compared with the
    oracle's chain (same loop, fp32, <= 1e-3 as in DESIGN.md R16), with its dt sequence, and with the exact solution."""
    import torch
    gamma, dh, nsteps = 1.4, 1.0 / 128, 100
    U, left, right = W.config2_box(axis, gamma)
    grid = tuple(s // 16 for s in U.shape[1:])
    gz, gy, gx = grid
    l32, r32 = left.astype(np.float32), right.astype(np.float32)
    inp = W.box_to_groups(U.astype(np.float32), dirichlet_axis=axis, lo_state=l32, hi_state=r32)
    bc = [0, 0, 0]
    bc[axis] = 1
    d_p = torch.from_numpy(inp).cuda()
    d_i = torch.empty((inp.shape[0], 5, 16, 16, 16), dtype=torch.float32, device="cuda")
    d_work = torch.zeros(4 + d_i.shape[0], dtype=torch.float32, device="cuda")
    d_log = torch.zeros(nsteps, dtype=torch.float32, device="cuda")
    hydro.gamer_hydro_run_uniform(d_p, d_i, gx, gy, gz, bc[0], bc[1], bc[2], nsteps, 0, 0.5, dh, gamma, d_work, d_log)
    torch.cuda.synchronize()
    got, dts = d_p.cpu().numpy(), d_log.cpu().numpy().astype(np.float64)
    # the transverse sweeps are exact no-ops, so the oracle chain can run on one column of groups
    ref, ref_dts = oracle.run_uniform(inp, grid, tuple(bc), nsteps, 0.5, dh, gamma, n_threads=8)
    assert np.max(np.abs(dts - np.array(ref_dts)) / np.array(ref_dts)) <= 2e-6
    e = W.parity_error(got[:, :, 3:19, 3:19, 3:19], ref[:, :, 3:19, 3:19, 3:19], gamma)
    assert e["max_rel"] <= 1e-3, e
    assert np.array_equal(got[:, :, 3:19, 3:19, 3:19], d_i.cpu().numpy())
    box = W.groups_to_box(got[:, :, 3:19, 3:19, 3:19], grid)
    sel = [0, 0, 0]
    sel[2 - axis] = slice(None)
    rho = box[(0,) + tuple(sel)].astype(np.float64)
    x = (np.arange(128) + 0.5) * dh
    rho_e, _, _ = riemann_exact.sample((x - 0.5) / dts.sum(), 1, 0, 1, 0.125, 0, 0.1, gamma)
    assert np.mean(np.abs(rho - rho_e)) <= 1.0e-2


@pytest.mark.gpu
def test_gpu_run_uniform_one_step_equals_advance_plus_ghost_fill():
    """The driver's kernel reads dt from device memory and forms the dt-dependent constants itself: with the dt it
    logged, the plain entry points must give the same bits."""
    import torch
    c = W.config1()
    grid = (2, 2, 2)
    d_p = torch.from_numpy(c["inp"]).cuda()
    d_i = torch.empty((8, 5, 16, 16, 16), dtype=torch.float32, device="cuda")
    d_work = torch.zeros(4 + d_i.shape[0], dtype=torch.float32, device="cuda")
    d_log = torch.zeros(1, dtype=torch.float32, device="cuda")
    hydro.gamer_hydro_run_uniform(d_p, d_i, 2, 2, 2, 0, 0, 0, 1, 0, 0.5, c["dh"], c["gamma"], d_work, d_log)
    torch.cuda.synchronize()
    dt = float(d_log.cpu().numpy()[0])
    ref_speed = oracle.max_signal_speed(c["inp"], c["gamma"])
    assert abs(dt - 0.5 * c["dh"] / ref_speed) <= 2e-6 * dt
    d_in = torch.from_numpy(c["inp"]).cuda()
    d_out = torch.empty_like(d_i)
    hydro.gamer_hydro_advance(d_in, d_out, 8, 3, dt, c["dh"], c["gamma"])
    d_p2 = torch.full_like(d_p, float("nan"))
    hydro.gamer_hydro_ghost_fill(d_out, d_p2, 2, 2, 2)
    torch.cuda.synchronize()
    assert torch.equal(d_out.view(torch.int32), d_i.view(torch.int32))
    assert torch.equal(d_p2.view(torch.int32), d_p.view(torch.int32))
    assert np.array_equal(d_p.cpu().numpy(), oracle.ghost_fill(d_i.cpu().numpy(), grid))


@pytest.mark.gpu
def test_gpu_run_uniform_strang_pairs_match_the_oracle_chain():
    """order = 1: forward pass, ghost fill, backward pass with the SAME dt, ghost fill, on the device.
    Free-running against the oracle's chain over 3 steps (6 passes) on config 1 as a periodic 2x2x2 box: dt sequence to
    2e-6, state to 1e-4 (6 passes of <= 1e-5 each, metric R11); and one step must give the same bits as the plain
    entry points called with the logged dt (teacher-forced: each call <= 1e-5 against the oracle on the same input)."""
    import torch
    c = W.config1()
    grid, n_steps = (2, 2, 2), 3
    d_p = torch.from_numpy(c["inp"]).cuda()
    d_i = torch.empty((8, 5, 16, 16, 16), dtype=torch.float32, device="cuda")
    d_work = torch.zeros(4 + 8, dtype=torch.float32, device="cuda")
    d_log = torch.zeros(n_steps, dtype=torch.float32, device="cuda")
    hydro.gamer_hydro_run_uniform(d_p, d_i, 2, 2, 2, 0, 0, 0, n_steps, 1, 0.4, c["dh"], c["gamma"], d_work, d_log)
    torch.cuda.synchronize()
    got, dts = d_p.cpu().numpy(), d_log.cpu().numpy().astype(np.float64)
    ref, ref_dts = oracle.run_uniform(c["inp"], grid, (0, 0, 0), n_steps, 0.4, c["dh"], c["gamma"], n_threads=8, order=1)
    assert np.max(np.abs(dts - np.array(ref_dts)) / np.array(ref_dts)) <= 2e-6
    e = W.parity_error(got[:, :, 3:19, 3:19, 3:19], ref[:, :, 3:19, 3:19, 3:19], c["gamma"])
    assert e["max_rel"] <= 1e-4, e
    assert np.array_equal(got, oracle.ghost_fill(d_i.cpu().numpy(), grid))
    # one step, written out with the plain entry points and the dt the driver logged
    d_p1 = torch.from_numpy(c["inp"]).cuda()
    hydro.gamer_hydro_run_uniform(d_p1, d_i, 2, 2, 2, 0, 0, 0, 1, 1, 0.4, c["dh"], c["gamma"], d_work, d_log)
    torch.cuda.synchronize()
    dt = float(d_log.cpu().numpy()[0])
    d_in = torch.from_numpy(c["inp"]).cuda()
    d_out = torch.empty_like(d_i)
    d_pad = torch.full_like(d_in, float("nan"))
    hydro.gamer_hydro_advance(d_in, d_out, 8, 3, dt, c["dh"], c["gamma"])
    fwd = d_out.cpu().numpy()
    e = W.parity_error(fwd, oracle.hydro_advance(c["inp"], dt, c["dh"], c["gamma"]), c["gamma"])
    assert e["max_rel"] <= 1e-5, e
    hydro.gamer_hydro_ghost_fill(d_out, d_pad, 2, 2, 2)
    mid = d_pad.cpu().numpy()
    hydro.gamer_hydro_advance_ex(d_pad, d_out, 8, 3, dt, c["dh"], c["gamma"], backward=1)
    torch.cuda.synchronize()
    e = W.parity_error(d_out.cpu().numpy(), oracle.hydro_advance(mid, dt, c["dh"], c["gamma"], backward=1), c["gamma"])
    assert e["max_rel"] <= 1e-5, e
    assert torch.equal(d_out.view(torch.int32), d_i.view(torch.int32))


@pytest.mark.gpu
def test_gpu_run_uniform_diagonal_sound_wave_converges_with_strang_pairs():
    """The paper's accuracy test (:450-458) through the device-only driver with order = 1, in single precision: a sound
    wave of amplitude 1e-3 (well above fp32 round-off, still linear to 1e-3) along the box diagonal for one period on
    16^3 and 32^3 cells; the L1 error of the density falls faster than first order."""
    import torch
    gamma, amp = 5.0 / 3.0, 1e-3

    def run(n):
        dh = 1.0 / n
        g = n // 16
        inp = W.box_to_groups(diagonal_wave(n, 0.0, amp=amp)).astype(np.float32)
        dt0 = 0.4 * dh / 1.3
        n_steps = int(round((1.0 / DIAG_SPEED) / (2 * dt0)))
        d_p = torch.from_numpy(inp).cuda()
        d_i = torch.empty((g ** 3, 5, 16, 16, 16), dtype=torch.float32, device="cuda")
        d_work = torch.zeros(4 + g ** 3, dtype=torch.float32, device="cuda")
        d_log = torch.zeros(n_steps, dtype=torch.float32, device="cuda")
        hydro.gamer_hydro_run_uniform(d_p, d_i, g, g, g, 0, 0, 0, n_steps, 1, 0.4, dh, gamma, d_work, d_log)
        torch.cuda.synchronize()
        t = 2.0 * float(d_log.cpu().numpy().astype(np.float64).sum())
        box = W.groups_to_box(d_i.cpu().numpy().astype(np.float64), (g, g, g))
        return np.mean(np.abs(box[0] - diagonal_wave(n, DIAG_SPEED * t, amp=amp)[0])) / amp

    e16, e32 = run(16), run(32)
    slope = np.log2(e32 / e16)
    assert -2.6 <= slope <= -1.4, (e16, e32, slope)
