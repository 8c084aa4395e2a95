"""Parity of the CUDA path (through the C ABI) with the CPU oracle, element by element, on the five configs.

Bar (BASELINE.json north_star): per-cell max relative error <= 1e-5 against the fp32 oracle and <= 1e-4 against the
fp64 oracle, with the error metric of DESIGN.md reading R11 (workloads.parity_error); bit-exact where the method is
(uniform states, transverse no-ops)."""
import os

import numpy as np
import pytest

import oracle
import riemann_exact
from paper_0907_3390_b200 import hydro
from paper_0907_3390_b200 import workloads as W

pytestmark = pytest.mark.gpu

TOL32, TOL64 = 1e-5, 1e-4
NT = os.cpu_count() or 1


def torch_mod():
    import torch
    assert torch.cuda.is_available()
    return torch


def gpu_advance(inp, dt, dh, gamma, backward=0, face=False, speed=False, stream=None):
    torch = torch_mod()
    G = inp.shape[0]
    d_in = torch.from_numpy(np.ascontiguousarray(inp, np.float32)).cuda()
    d_out = torch.full((G, 5, 16, 16, 16), float("nan"), dtype=torch.float32, device="cuda")
    d_face = torch.full((G, 3, 3, 5, 16, 16), float("nan"), dtype=torch.float32, device="cuda") if face else None
    d_speed = torch.full((G,), float("nan"), dtype=torch.float32, device="cuda") if speed else None
    if backward or face or speed:
        hydro.gamer_hydro_advance_ex(d_in, d_out, G, 3, dt, dh, gamma, backward, d_face, d_speed, stream=stream)
    else:
        hydro.gamer_hydro_advance(d_in, d_out, G, 3, dt, dh, gamma, stream=stream)
    torch.cuda.synchronize()
    res = [d_out.cpu().numpy()]
    if face:
        res.append(d_face.cpu().numpy())
    if speed:
        res.append(d_speed.cpu().numpy())
    return res[0] if len(res) == 1 else tuple(res)


def check_parity(gpu, inp, dt, dh, gamma, backward=0):
    o32 = oracle.hydro_advance(inp, dt, dh, gamma, backward=backward, n_threads=NT)
    o64 = oracle.hydro_advance(inp, dt, dh, gamma, backward=backward, dtype=np.float64, n_threads=NT)
    e32 = W.parity_error(gpu, o32, gamma)
    e64 = W.parity_error(gpu, o64, gamma)
    assert e32["max_rel"] <= TOL32, ("vs fp32 oracle", e32)
    assert e64["max_rel"] <= TOL64, ("vs fp64 oracle", e64)
    return e32, e64


def face_flux_local_scale(inp, gamma):
    """Per-element scale of the face fluxes [G][3][3][5][16][16]: c * s_v on the two cells next to the interface,
    c = |v| + c_s, s_v = the R11 scale of variable v (rho, rho (|v| + c_s), e) — the size of |F^R| + |F^L| = c u there
    (Eq.8), taken from the padded input (interfaces 2|3, 10|11, 18|19 along d)."""
    u = np.asarray(inp, np.float64)
    rho, mx, my, mz, e = (u[:, i] for i in range(5))
    P = (gamma - 1.0) * (e - 0.5 * (mx * mx + my * my + mz * mz) / rho)
    c = np.sqrt(mx * mx + my * my + mz * mz) / rho + np.sqrt(gamma * P / rho)
    cell = np.stack([c * rho, c * c * rho, c * c * rho, c * c * rho, c * np.abs(e)], axis=1)      # [G][5][22][22][22]
    G = u.shape[0]
    scale = np.empty((G, 3, 3, 5, 16, 16))
    for d in range(3):
        ax = 4 - d                                            # numpy axis of x, y, z in [G][5][z][y][x]
        for p, n in enumerate((2, 10, 18)):
            pair = np.maximum(np.take(cell, n, axis=ax), np.take(cell, n + 1, axis=ax))        # [G][5][.][.] padded
            scale[:, d, p] = pair[:, :, 3:19, 3:19]
    return scale


def assert_face_flux_parity(face, o_face, inp, gamma, tol=1e-5):
    err = np.abs(face.astype(np.float64) - o_face) / face_flux_local_scale(inp, gamma)
    assert np.isfinite(face).all()
    assert err.max() <= tol, (err.max(), np.unravel_index(int(np.argmax(err)), err.shape))


def test_library_is_the_cuda_one():
    info = hydro.gamer_hydro_launch_info(1000)
    assert info["block"] == 512 and info["smem_bytes"] >= 212960 and info["grid"] >= 100
    assert info["regs_per_thread"] <= 128


@pytest.mark.parametrize("backward", [0, 1])
def test_config1(backward):
    c = W.config1()
    gpu = gpu_advance(c["inp"], c["dt"], c["dh"], c["gamma"], backward=backward)
    check_parity(gpu, c["inp"], c["dt"], c["dh"], c["gamma"], backward=backward)


@pytest.mark.parametrize("backward", [0, 1])
def test_uniform_state_bit_exact(backward):
    u = np.empty((3, 5, 22, 22, 22), np.float32)
    vals = np.array([[1.3, 0.4, -0.2, 0.7, 2.9], [0.01, 0.0, 0.0, 0.0, 5.0], [1000.0, 3e3, -2e3, 1e3, 1e5]], np.float32)
    for g in range(3):
        for i in range(5):
            u[g, i] = vals[g, i]
    out = gpu_advance(u, 0.002, 1 / 128, 5 / 3, backward=backward)
    for g in range(3):
        for i in range(5):
            assert (out[g, i] == vals[g, i]).all()


@pytest.mark.parametrize("n", [1, 2, 147, 148, 149, 300])
def test_ragged_group_counts(n):
    """Persistent grid = min(n, #SM): fewer groups than SMs, exactly one wave, one more than a wave, a ragged tail."""
    rng = np.random.default_rng(n)
    c = W.config1()
    idx = rng.integers(0, 8, n)
    inp = c["inp"][idx] * (1.0 + 0.01 * rng.uniform(-1, 1, (n, 1, 1, 1, 1))).astype(np.float32)
    gpu = gpu_advance(inp, c["dt"], c["dh"], c["gamma"])
    o32 = oracle.hydro_advance(inp, c["dt"], c["dh"], c["gamma"], n_threads=NT)
    assert W.parity_error(gpu, o32, c["gamma"])["max_rel"] <= TOL32


def test_zero_groups_is_a_noop():
    torch = torch_mod()
    d = torch.zeros(16, device="cuda")
    assert hydro.gamer_hydro_advance(d, d, 0, 3, 0.1, 1.0, 1.4) == 0
    assert hydro.gamer_hydro_advance(None, None, 0, 3, 0.1, 1.0, 1.4) == 0


def test_config3_all_groups():
    c = W.config3()
    gpu = gpu_advance(c["inp"], c["dt"], c["dh"], c["gamma"])
    check_parity(gpu, c["inp"], c["dt"], c["dh"], c["gamma"])


def test_config4_all_groups():
    c = W.config4()
    gpu = gpu_advance(c["inp"], c["dt"], c["dh"], c["gamma"])
    check_parity(gpu, c["inp"], c["dt"], c["dh"], c["gamma"])
    gpu_b = gpu_advance(c["inp"][:512], c["dt"], c["dh"], c["gamma"], backward=1)
    check_parity(gpu_b, c["inp"][:512], c["dt"], c["dh"], c["gamma"], backward=1)


@pytest.mark.parametrize("backward", [0, 1])
def test_config5_full_size_sampled(backward):
    """32 768 groups, filled on the device (6.98 GB in, 2.68 GB out), the launch configuration bench.py times (and the
    same with the backward sweep order, the other half of every step of the paper).  Every hot group and a sample of
    background groups are compared with the oracle one by one; every background group must come back bit-identical to
    its (uniform) input."""
    torch = torch_mod()
    n = W.CONFIG5["n_groups"]
    hot = W.config5_hot_groups(n)
    bg = torch.from_numpy(W.config5_group(False)).cuda()
    ht = torch.from_numpy(W.config5_group(True)).cuda()
    d_in = torch.empty((n, 5, 22, 22, 22), dtype=torch.float32, device="cuda")
    d_in[:] = bg
    d_in[torch.from_numpy(hot).cuda()] = ht
    d_out = torch.full((n, 5, 16, 16, 16), float("nan"), dtype=torch.float32, device="cuda")
    dt, dh, gamma = W.config5_dt(), W.CONFIG5["dh"], W.CONFIG5["gamma"]
    hydro.gamer_hydro_advance_ex(d_in, d_out, n, 3, dt, dh, gamma, backward, None, None)
    torch.cuda.synchronize()
    is_hot = torch.zeros(n, dtype=torch.bool, device="cuda")
    is_hot[torch.from_numpy(hot).cuda()] = True
    bg_out = d_out[~is_hot]
    assert bool((bg_out == bg[:, 3:19, 3:19, 3:19]).all())
    rng = np.random.default_rng(5)
    cold = rng.choice(np.setdiff1d(np.arange(n), hot), 64, replace=False)
    sample = np.sort(np.concatenate([hot, cold, [0, n - 1]]))
    sample = np.unique(sample)
    c = W.config5(sample, n)
    gpu = d_out[torch.from_numpy(sample).cuda()].cpu().numpy()
    check_parity(gpu, c["inp"], dt, dh, gamma, backward=backward)
    del d_in, d_out
    torch.cuda.empty_cache()


def test_face_flux_and_group_maxspeed():
    c = W.config1()
    for backward in (0, 1):
        out, face, speed = gpu_advance(c["inp"], c["dt"], c["dh"], c["gamma"], backward=backward, face=True, speed=True)
        o_out, o_face, o_speed = oracle.hydro_advance(c["inp"], c["dt"], c["dh"], c["gamma"], backward=backward,
                                                      want_face_flux=True, want_maxspeed=True)
        assert W.parity_error(out, o_out, c["gamma"])["max_rel"] <= TOL32
        np.testing.assert_allclose(speed, o_speed, rtol=2e-6)
        assert_face_flux_parity(face, o_face, c["inp"], c["gamma"])       # per element, at the cell's own scale


@pytest.mark.parametrize("backward", [0, 1])
def test_optional_outputs_over_several_groups_per_cta(backward):
    """350 different groups: every persistent CTA takes two or three in a row, so the per-group CFL reduction (slots
    that rotate with the iteration) and the face-flux addressing are exercised across group boundaries."""
    rng = np.random.default_rng(42 + backward)
    c = W.config3()
    idx = rng.permutation(c["inp"].shape[0])[:350]
    inp = np.ascontiguousarray(c["inp"][idx])
    out, face, speed = gpu_advance(inp, c["dt"], c["dh"], c["gamma"], backward=backward, face=True, speed=True)
    o_out, o_face, o_speed = oracle.hydro_advance(inp, c["dt"], c["dh"], c["gamma"], backward=backward,
                                                  want_face_flux=True, want_maxspeed=True, n_threads=NT)
    assert W.parity_error(out, o_out, c["gamma"])["max_rel"] <= TOL32
    np.testing.assert_allclose(speed, o_speed, rtol=2e-6)
    assert_face_flux_parity(face, o_face, inp, c["gamma"])
    # the optional outputs do not change the main one
    assert np.array_equal(out, gpu_advance(inp, c["dt"], c["dh"], c["gamma"], backward=backward))


@pytest.mark.parametrize("axis", [0, 1, 2])
def test_config2_sod_teacher_forced_and_free_running(axis):
    """Config 2 (128 groups, 128x64x64, gamma=1.4, 100 steps at CFL 0.5, readings R12-R16).
    Teacher-forced: at steps 1, 2, 10, 50, 100 the GPU is fed the oracle's state and compared after one call.
    Free-running: the GPU's own 100-step chain against the exact Riemann solution (same L1 bound as the oracle)
    and against the oracle chain (<= 1e-3)."""
    gamma, dh = 1.4, 1.0 / 128
    U, left, right = W.config2_box(axis, gamma)
    grid = tuple(s // 16 for s in U.shape[1:])
    Uo = U.astype(np.float32)
    Ug = Uo.copy()
    l32, r32 = left.astype(np.float32), right.astype(np.float32)
    t = 0.0
    for step in range(1, 101):
        inp_o = W.box_to_groups(Uo, dirichlet_axis=axis, lo_state=l32, hi_state=r32)
        dt = W.cfl_dt(inp_o, dh, gamma)
        out_o = oracle.hydro_advance(inp_o, dt, dh, gamma, n_threads=NT)
        if step in (1, 2, 10, 50, 100):
            forced = gpu_advance(inp_o, dt, dh, gamma)
            e = W.parity_error(forced, out_o, gamma)
            assert e["max_rel"] <= TOL32, (step, e)
        inp_g = W.box_to_groups(Ug, dirichlet_axis=axis, lo_state=l32, hi_state=r32)
        Ug = W.groups_to_box(gpu_advance(inp_g, dt, dh, gamma), grid)
        Uo = W.groups_to_box(out_o, grid)
        t += dt
    e = W.parity_error(Ug[None], Uo[None], gamma)
    assert e["max_rel"] <= 1e-3, e
    sel = [0, 0, 0]
    sel[2 - axis] = slice(None)
    rho = Ug[(0,) + tuple(sel)].astype(np.float64)
    x = (np.arange(128) + 0.5) * dh
    rho_e, _, _ = riemann_exact.sample((x - 0.5) / t, 1, 0, 1, 0.125, 0, 0.1, gamma)
    assert np.mean(np.abs(rho - rho_e)) <= 1.0e-2
    # transverse uniformity survives 100 steps exactly (the transverse sweeps are exact no-ops)
    shape = [1, 1, 1]
    shape[2 - axis] = 128
    assert (Ug[0] == Ug[(0,) + tuple(sel)].reshape(shape)).all()


def test_pipeline_matches_direct_call_with_ragged_chunks():
    """Secondary subsystem: pinned host buffers, chunks that leave a ragged tail, several streams."""
    torch = torch_mod()
    c = W.config3()
    n = 300
    inp = c["inp"][:n]
    direct = gpu_advance(inp, c["dt"], c["dh"], c["gamma"])
    h_in = torch.from_numpy(np.ascontiguousarray(inp)).pin_memory()
    for chunk, ns in ((64, 3), (7, 4), (300, 1), (1000, 2)):
        h_out = torch.full((n, 5, 16, 16, 16), float("nan"), dtype=torch.float32).pin_memory()
        hydro.gamer_hydro_pipeline_run(h_in, h_out, n, 3, c["dt"], c["dh"], c["gamma"], 0, chunk, ns)
        assert np.array_equal(h_out.numpy(), direct), (chunk, ns)
    # the staging buffers are kept between calls (grown above from 7 to 300 groups); release and run again
    before = torch.cuda.mem_get_info()[0]
    hydro.gamer_hydro_pipeline_release()
    assert torch.cuda.mem_get_info()[0] > before
    hydro.gamer_hydro_pipeline_release()          # a no-op when nothing is held
    h_out = torch.full((n, 5, 16, 16, 16), float("nan"), dtype=torch.float32).pin_memory()
    hydro.gamer_hydro_pipeline_run(h_in, h_out, n, 3, c["dt"], c["dh"], c["gamma"], 1, 50, 2)
    assert np.array_equal(h_out.numpy(), gpu_advance(inp, c["dt"], c["dh"], c["gamma"], backward=1))
    hydro.gamer_hydro_pipeline_release()


def test_runs_on_a_side_stream():
    torch = torch_mod()
    c = W.config1()
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        gpu = gpu_advance(c["inp"], c["dt"], c["dh"], c["gamma"], stream=s)
    o32 = oracle.hydro_advance(c["inp"], c["dt"], c["dh"], c["gamma"])
    assert W.parity_error(gpu, o32, c["gamma"])["max_rel"] <= TOL32


@pytest.mark.gpu
def test_issue_probe_reports_plausible_clock_counts():
    """The measurement aid behind DESIGN.md 7: a 3-register FMA costs more than one issue slot and less than two; a
    warp-march (about 2 700 instructions) costs between 2 700 and 4 500 clocks and gets cheaper per slot with more warps."""
    from paper_0907_3390_b200 import probes
    f3 = probes.gamer_probe_issue(0, 4)
    assert 1.2 <= f3 <= 2.0, f3
    for what in (1, 2, 3):
        c1, c4 = probes.gamer_probe_issue(what, 1), probes.gamer_probe_issue(what, 4)      # (fails if the state changed)
        assert 2700 <= c4 <= c1 <= 4500, (what, c1, c4)

