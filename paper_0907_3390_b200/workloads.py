"""Seeded synthetic inputs for the batched hydro update (the five configs of BASELINE.json).

This module serves BOTH the CPU oracle's tests and the CUDA path's tests / bench.  It holds none of the method's
arithmetic: it builds conserved-variable fields, cuts them into ghost-padded patch groups (the paper's CPU
"preparation step"), and picks dt from the CFL condition (Eq.30) in float64.
It imports neither the oracle nor the CUDA binding.  The recipe is stated in DESIGN.md §Inputs.

Layout of a batch: in[g][v][z][y][x], v = (rho, rho v_x, rho v_y, rho v_z, e), 22^3 padded cells per group,
interior at padded indices 3..18; groups of a box are ordered g = (gz*Gy + gy)*Gx + gx.
"""
import numpy as np

NCOMP, PS, NGHOST, NP = 5, 16, 3, 22
SEED_BASE = 9073390 * 10


def rng_for(config_index, stream=0):
    return np.random.default_rng(np.random.PCG64(SEED_BASE + config_index + 1000 * stream))


def conserved(rho, vx, vy, vz, P, gamma):
    """(rho, v, P) -> u[5][...] in float64; e = P/(gamma-1) + rho v^2/2 (Eqs.4-5)."""
    rho = np.asarray(rho, np.float64)
    u = np.empty((NCOMP,) + rho.shape, np.float64)
    u[0] = rho
    u[1] = rho * vx
    u[2] = rho * vy
    u[3] = rho * vz
    u[4] = P / (gamma - 1.0) + 0.5 * rho * (np.asarray(vx) ** 2 + np.asarray(vy) ** 2 + np.asarray(vz) ** 2)
    return u


def box_to_groups(U, dirichlet_axis=None, lo_state=None, hi_state=None):
    """Cut a box U[5][Nz][Ny][Nx] (extents multiples of 16) into ghost-padded groups [G][5][22][22][22].

    Ghost cells come from the periodic neighbours (sibling copy).  If `dirichlet_axis` (0:x,1:y,2:z)
    is given, ghosts beyond the two ends of that axis hold the constant states lo_state / hi_state (u[5]).
    """
    U = np.asarray(U)
    _, Nz, Ny, Nx = U.shape
    assert Nz % PS == 0 and Ny % PS == 0 and Nx % PS == 0
    g = NGHOST
    P = np.pad(U, ((0, 0), (g, g), (g, g), (g, g)), mode="wrap")
    if dirichlet_axis is not None:
        ax = 3 - dirichlet_axis          # numpy axis of P for x,y,z
        sl_lo = [slice(None)] * 4
        sl_hi = [slice(None)] * 4
        sl_lo[ax] = slice(0, g)
        sl_hi[ax] = slice(P.shape[ax] - g, P.shape[ax])
        P[tuple(sl_lo)] = np.asarray(lo_state).reshape(NCOMP, 1, 1, 1)
        P[tuple(sl_hi)] = np.asarray(hi_state).reshape(NCOMP, 1, 1, 1)
    Gz, Gy, Gx = Nz // PS, Ny // PS, Nx // PS
    out = np.empty((Gz * Gy * Gx, NCOMP, NP, NP, NP), U.dtype)
    for gz in range(Gz):
        for gy in range(Gy):
            for gx in range(Gx):
                out[(gz * Gy + gy) * Gx + gx] = P[:, gz * PS:gz * PS + NP, gy * PS:gy * PS + NP, gx * PS:gx * PS + NP]
    return out


def groups_to_box(out, grid):
    """Inverse of the interior part of box_to_groups: out[G][5][16][16][16], grid=(Gz,Gy,Gx) -> U[5][Nz][Ny][Nx]."""
    Gz, Gy, Gx = grid
    out = np.asarray(out)
    U = np.empty((NCOMP, Gz * PS, Gy * PS, Gx * PS), out.dtype)
    for gz in range(Gz):
        for gy in range(Gy):
            for gx in range(Gx):
                U[:, gz * PS:(gz + 1) * PS, gy * PS:(gy + 1) * PS, gx * PS:(gx + 1) * PS] = out[(gz * Gy + gy) * Gx + gx]
    return U


def max_signal_speed(u, gamma):
    """max over cells of c_s + max(|v_x|,|v_y|,|v_z|) in float64 (denominator of Eq.30)."""
    u = np.asarray(u, np.float64)
    if u.ndim == 5:      # [G][5][...]
        rho, mx, my, mz, e = (u[:, i] for i in range(5))
    else:                # [5][...]
        rho, mx, my, mz, e = (u[i] for i in range(5))
    P = (gamma - 1.0) * (e - 0.5 * (mx * mx + my * my + mz * mz) / rho)
    cs = np.sqrt(gamma * P / rho)
    vmax = np.maximum(np.maximum(np.abs(mx), np.abs(my)), np.abs(mz)) / rho
    return float((cs + vmax).max())


def cfl_dt(u, dh, gamma, cfl=0.5):
    """dt = cfl * dh / max speed over ALL cells given (padded cells included), float64, rounded once to float32."""
    return float(np.float32(cfl * dh / max_signal_speed(u, gamma)))


def gaussian_field(shape, slope, rng):
    """Real periodic Gaussian random field with 3-D power spectrum <|f_k|^2> ~ |k|^slope, k=0 mode zeroed, unit rms."""
    white = rng.standard_normal(shape)
    fk = np.fft.rfftn(white, axes=(0, 1, 2))
    kz = np.fft.fftfreq(shape[0])[:, None, None] * shape[0]
    ky = np.fft.fftfreq(shape[1])[None, :, None] * shape[1]
    kx = np.fft.rfftfreq(shape[2])[None, None, :] * shape[2]
    k2 = kz * kz + ky * ky + kx * kx
    k2[0, 0, 0] = 1.0
    amp = k2 ** (slope / 4.0)            # |k|^(slope/2) on the amplitude
    amp[0, 0, 0] = 0.0
    f = np.fft.irfftn(fk * amp, s=shape, axes=(0, 1, 2))
    return f / np.sqrt(np.mean(f * f))


# ---------------------------------------------------------------------------------------------------------------
# The five configs.  Each returns a dict: inp (float32 [G][5][22]^3), dt (float, already float32-rounded), dh, gamma,
# grid (Gz,Gy,Gx) and whatever the tests need to refill ghosts.
# ---------------------------------------------------------------------------------------------------------------

def config1(grid=(2, 2, 2)):
    """8 groups, rho=1+0.1 U(-1,1), v_i ~ N(0,0.1), P=1+0.1 U(-1,1) iid per cell, gamma=5/3, dh=1/128, CFL 0.5."""
    gamma, dh = 5.0 / 3.0, 1.0 / 128.0
    rng = rng_for(1)
    shp = (grid[0] * PS, grid[1] * PS, grid[2] * PS)
    rho = 1.0 + 0.1 * rng.uniform(-1, 1, shp)
    vx, vy, vz = (rng.normal(0.0, 0.1, shp) for _ in range(3))
    P = 1.0 + 0.1 * rng.uniform(-1, 1, shp)
    U = conserved(rho, vx, vy, vz, P, gamma)
    inp = box_to_groups(U).astype(np.float32)
    return dict(name="config1", inp=inp, dt=cfl_dt(inp, dh, gamma), dh=dh, gamma=gamma, grid=grid)


def sod_states(gamma=1.4):
    left = conserved(1.0, 0.0, 0.0, 0.0, 1.0, gamma)
    right = conserved(0.125, 0.0, 0.0, 0.0, 0.1, gamma)
    return left, right


def config2_box(axis=0, gamma=1.4, n_long=128, n_trans=64):
    """Sod shock tube along `axis` (0:x,1:y,2:z): box of n_long cells along the axis, n_trans across, float64 U[5]."""
    left, right = sod_states(gamma)
    shp = [n_trans, n_trans, n_trans]
    shp[2 - axis] = n_long              # numpy order (z,y,x)
    U = np.empty((NCOMP,) + tuple(shp), np.float64)
    coord = np.arange(n_long)
    is_left = coord < n_long // 2
    bshape = [1, 1, 1]
    bshape[2 - axis] = n_long
    m = is_left.reshape(bshape)
    for v in range(NCOMP):
        U[v] = np.where(m, left[v], right[v])
    return U, left, right


def config2(axis=0, gamma=1.4, n_long=128, n_trans=64):
    """128x64x64 box (128 groups, reading R12), Dirichlet ends along the tube, periodic across (R13)."""
    dh = 1.0 / 128.0
    U, left, right = config2_box(axis, gamma, n_long, n_trans)
    inp = box_to_groups(U, dirichlet_axis=axis, lo_state=left, hi_state=right).astype(np.float32)
    shp = U.shape[1:]
    grid = (shp[0] // PS, shp[1] // PS, shp[2] // PS)
    return dict(name="config2", inp=inp, dt=cfl_dt(inp, dh, gamma), dh=dh, gamma=gamma, grid=grid, axis=axis,
                left=left, right=right, n_steps=100)


def config3(grid=(8, 8, 8)):
    """512 groups: rho=1, P=1/gamma (c_s=1), v = Gaussian field with P(k)~k^-2, 3-D rms |v| = 1 (rms Mach 1)."""
    gamma, dh = 5.0 / 3.0, 1.0 / 128.0
    rng = rng_for(3)
    shp = (grid[0] * PS, grid[1] * PS, grid[2] * PS)
    v = [gaussian_field(shp, -2.0, rng) for _ in range(3)]
    norm = np.sqrt(np.mean(v[0] ** 2 + v[1] ** 2 + v[2] ** 2))
    v = [c / norm for c in v]
    U = conserved(np.ones(shp), v[0], v[1], v[2], np.full(shp, 1.0 / gamma), gamma)
    inp = box_to_groups(U).astype(np.float32)
    return dict(name="config3", inp=inp, dt=cfl_dt(inp, dh, gamma), dh=dh, gamma=gamma, grid=grid)


def _clumpy_gas(grid, slope, name):
    gamma, dh, alpha = 5.0 / 3.0, 1.0 / 256.0, 0.5
    rng = rng_for(4)
    shp = (grid[0] * PS, grid[1] * PS, grid[2] * PS)
    lnrho = 2.0 * gaussian_field(shp, slope, rng)
    lnrho -= lnrho.mean()
    rho = np.exp(lnrho)
    vel = []
    for ax in (2, 1, 0):                 # x, y, z <-> numpy axes 2, 1, 0
        grad = 0.5 * (np.roll(lnrho, -1, axis=ax) - np.roll(lnrho, 1, axis=ax))
        grad /= np.sqrt(np.mean(grad * grad))
        g = rng.standard_normal(shp)
        vel.append(0.5 * (np.sqrt(1.0 - alpha * alpha) * g + alpha * grad))
    U = conserved(rho, vel[0], vel[1], vel[2], rho ** gamma, gamma)
    inp = box_to_groups(U).astype(np.float32)
    return dict(name=name, inp=inp, dt=cfl_dt(inp, dh, gamma), dh=dh, gamma=gamma, grid=grid)


def config4(grid=(16, 16, 16)):
    """4096 groups: ln rho Gaussian, sigma=2, shell-integrated spectrum E(k) = 4 pi k^2 P(k) ~ k^-3 (3-D power
    P(k) ~ k^-5; reading R17: with 3-D power ~ k^-3 adjacent cells differ by a factor e^1.2 rms, up to
    e^6.6, and the floor-free scheme leaves the physical domain in both fp32 and fp64); P=rho^gamma;
    v = 0.5(sqrt(1-a^2) g + a grad ln rho / rms), g ~ N(0,1) iid, a = 0.5.  Every group stays physical: this is the
    config-4 input of the all-groups parity test and of the timing."""
    return _clumpy_gas(grid, -5.0, "config4")


def config4_literal(grid=(16, 16, 16)):
    """Config 4 exactly as BASELINE.json / SURVEY.md 8(c)#17 word it: the same recipe with the 3-D power spectrum of
    ln rho ~ |k|^-3.  The scheme has no floor (R7) and on this field part of the groups leave the physical
    domain (rho <= 0 or P <= 0 somewhere along the pass) on the CPU oracle in fp32 and in fp64 alike; the tests
    compare the CUDA path with the oracle on the groups that stay physical on both and state how many those are."""
    return _clumpy_gas(grid, -3.0, "config4_literal")


CONFIG5 = dict(n_groups=32768, grid=(32, 32, 32), gamma=5.0 / 3.0, dh=1.0 / 512.0, p_bg=1e-5, p_hot=1e3, frac=0.01)


def config5_hot_groups(n_groups=CONFIG5["n_groups"]):
    """Sorted indices of the round(0.01 n) groups that hold a hot 2^3 centre, chosen by a seeded permutation."""
    rng = rng_for(5)
    n_hot = int(round(CONFIG5["frac"] * n_groups))
    return np.sort(rng.permutation(n_groups)[:n_hot])


def config5_dt():
    c = CONFIG5
    return float(np.float32(0.5 * c["dh"] / np.sqrt(c["gamma"] * c["p_hot"] / 1.0)))


def config5_group(hot):
    """One padded group of config 5 in float32: rho=1, v=0, P=1e-5; if `hot`, padded cells 10..11 cubed have P=1e3.

    Hot cells sit >= 7 cells from every face, so every ghost shell is pure background and groups are consistent with
    any tiling of a periodic box."""
    c = CONFIG5
    P = np.full((NP, NP, NP), c["p_bg"], np.float64)
    if hot:
        P[10:12, 10:12, 10:12] = c["p_hot"]
    z = np.zeros((NP, NP, NP))
    return conserved(np.ones((NP, NP, NP)), z, z, z, P, c["gamma"]).astype(np.float32)


def config5(indices=None, n_groups=CONFIG5["n_groups"]):
    """Config 5 restricted to the group indices given (default: all — 7 GB, use the device-side fill instead)."""
    hot = set(config5_hot_groups(n_groups).tolist())
    if indices is None:
        indices = range(n_groups)
    indices = list(indices)
    bg, ht = config5_group(False), config5_group(True)
    inp = np.empty((len(indices), NCOMP, NP, NP, NP), np.float32)
    for i, g in enumerate(indices):
        inp[i] = ht if g in hot else bg
    c = CONFIG5
    return dict(name="config5", inp=inp, dt=config5_dt(), dh=c["dh"], gamma=c["gamma"], indices=indices)


# ---------------------------------------------------------------------------------------------------------------
# Parity metric (reading R11).  Comparison bookkeeping, not the method: err = |a-ref| / s per cell and
# variable with s = |ref| for rho and e, and s = rho_ref (|v|_ref + c_s,ref) for each momentum component (a raw
# relative error on a momentum component that is zero by chance is meaningless); err = 0 where a == ref bitwise.
# ---------------------------------------------------------------------------------------------------------------

def parity_error(a, ref, gamma):
    """a, ref: [G][5][...] conserved variables.  Returns dict(max_rel, per_var_rel[5], per_var_abs[5], argmax)."""
    a64 = np.asarray(a, np.float64)
    r64 = np.asarray(ref, np.float64)
    rho, mx, my, mz, e = (r64[:, i] for i in range(5))
    with np.errstate(invalid="ignore", divide="ignore"):
        P = (gamma - 1.0) * (e - 0.5 * (mx * mx + my * my + mz * mz) / rho)
        cs = np.sqrt(np.maximum(gamma * P / rho, 0.0))
        vmag = np.sqrt(mx * mx + my * my + mz * mz) / rho
    mscale = rho * (vmag + cs)
    scale = np.stack([np.abs(rho), mscale, mscale, mscale, np.abs(e)], axis=1)
    diff = np.abs(a64 - r64)
    with np.errstate(invalid="ignore", divide="ignore"):
        rel = np.where(diff == 0.0, 0.0, diff / scale)
    rel = np.where(np.isfinite(rel), rel, np.inf)
    bad_nan = ~np.isfinite(a64)
    rel = np.where(bad_nan, np.inf, rel)
    per_var_rel = [float(rel[:, i].max()) for i in range(5)]
    per_var_abs = [float(diff[:, i].max()) for i in range(5)]
    return dict(max_rel=float(rel.max()), per_var_rel=per_var_rel, per_var_abs=per_var_abs,
                argmax=tuple(int(i) for i in np.unravel_index(int(np.argmax(rel)), rel.shape)))
