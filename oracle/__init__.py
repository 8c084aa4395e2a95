"""ORACLE — test infrastructure, not the product.

ctypes wrapper around oracle/rtvd_oracle.cpp (plain CPU relaxing-TVD update written from PAPER.md §2.2/§3.1).
Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / `--impl reference` legs may import this.
It imports nothing from the CUDA package and the CUDA package imports nothing from here.
"""
import ctypes
import os

import numpy as np

from . import build as _build

NCOMP, PS, NGHOST, NP = 5, 16, 3, 22
IN_GROUP = NCOMP * NP ** 3      # 53 240 values per padded group
OUT_GROUP = NCOMP * PS ** 3     # 20 480 values per interior
FACE_GROUP = 3 * 3 * NCOMP * PS * PS

_lib = None


def lib():
    global _lib
    if _lib is None:
        path = _build.build()
        L = ctypes.CDLL(path)
        for sfx, ct in (("f32", ctypes.c_float), ("f64", ctypes.c_double)):
            p = ctypes.c_void_p
            getattr(L, "oracle_van_leer_" + sfx).restype = ct
            getattr(L, "oracle_van_leer_" + sfx).argtypes = [ct, ct]
            getattr(L, "oracle_cell_fluxes_" + sfx).restype = None
            getattr(L, "oracle_cell_fluxes_" + sfx).argtypes = [p, ct, ctypes.c_int, p, p, p]
            getattr(L, "oracle_row_update_" + sfx).restype = None
            getattr(L, "oracle_row_update_" + sfx).argtypes = [p, p, ctypes.c_int, ct, ct, ctypes.c_int, ctypes.c_int, p, p]
            getattr(L, "oracle_hydro_advance_" + sfx).restype = ctypes.c_longlong
            getattr(L, "oracle_hydro_advance_" + sfx).argtypes = [p, p, ctypes.c_longlong, ctypes.c_int, ct, ct, ct,
                                                                 ctypes.c_int, ctypes.c_int, p, p, ctypes.c_int]
            getattr(L, "oracle_hydro_advance_badmask_" + sfx).restype = ctypes.c_longlong
            getattr(L, "oracle_hydro_advance_badmask_" + sfx).argtypes = [p, p, ctypes.c_longlong, ctypes.c_int, ct, ct, ct,
                                                                         ctypes.c_int, ctypes.c_int, p, ctypes.c_int]
        L.oracle_count_ops.restype = None
        L.oracle_count_ops.argtypes = [ctypes.c_void_p]
        L.oracle_has_openmp.restype = ctypes.c_int
        _lib = L
    return _lib


def _sfx(dtype):
    dtype = np.dtype(dtype)
    if dtype == np.float32:
        return "f32"
    if dtype == np.float64:
        return "f64"
    raise TypeError("oracle computes in float32 or float64, got %s" % dtype)


def van_leer(a, b, dtype=np.float64):
    """Eq.11 on two scalars."""
    return getattr(lib(), "oracle_van_leer_" + _sfx(dtype))(float(a), float(b))


def cell_fluxes(u, gamma, dtype=np.float64, c_mode=0):
    """Cell-centred (F^R, F^L, c) of one cell, u = (rho, m_n, m_t1, m_t2, e) (Eq.8)."""
    dt = np.dtype(dtype)
    u = np.ascontiguousarray(u, dtype=dt)
    assert u.shape == (NCOMP,)
    FR, FL, c = np.empty(NCOMP, dt), np.empty(NCOMP, dt), np.empty(1, dt)
    getattr(lib(), "oracle_cell_fluxes_" + _sfx(dt))(u.ctypes.data, dt.type(gamma), c_mode, FR.ctypes.data,
                                                    FL.ctypes.data, c.ctypes.data)
    return FR, FL, c[0]


def row_update(u, k, gamma, dtype=None, c_mode=0, limiter_on=1, want_half=False, want_flux=False):
    """One 1-D relaxing-TVD update of a row.

    u: [5][N] row-local components (rho, m_n, m_t1, m_t2, e).  Returns unew [5][N] (cells 3..N-4 updated, the rest
    copied), plus optionally the midpoint state u^{t+dt/2} and the time-centred interface fluxes F_{n+1/2}.
    """
    dt = np.dtype(dtype if dtype is not None else u.dtype)
    u = np.ascontiguousarray(u, dtype=dt)
    assert u.ndim == 2 and u.shape[0] == NCOMP and u.shape[1] >= 7
    N = u.shape[1]
    unew = np.empty_like(u)
    uh = np.empty_like(u) if want_half else None
    fh = np.empty_like(u) if want_flux else None
    getattr(lib(), "oracle_row_update_" + _sfx(dt))(u.ctypes.data, unew.ctypes.data, N, dt.type(k), dt.type(gamma),
                                                   c_mode, limiter_on,
                                                   uh.ctypes.data if want_half else None,
                                                   fh.ctypes.data if want_flux else None)
    res = (unew,)
    if want_half:
        res += (uh,)
    if want_flux:
        res += (fh,)
    return res if len(res) > 1 else unew


def hydro_advance(inp, dt, dh, gamma, backward=0, dtype=None, ghost=NGHOST, c_mode=0, want_face_flux=False,
                  want_maxspeed=False, n_threads=1, return_bad=False):
    """One 3-sweep pass over a batch of patch groups.

    inp: [G][5][22][22][22].  Returns out [G][5][16][16][16] (+ face flux [G][3][3][5][16][16], + maxspeed [G]).
    Raises if any cell met on the way has rho <= 0 or P <= 0 unless return_bad=True (reading R7).
    """
    dtp = np.dtype(dtype if dtype is not None else inp.dtype)
    a = np.ascontiguousarray(inp, dtype=dtp)
    assert a.ndim == 5 and a.shape[1:] == (NCOMP, NP, NP, NP), a.shape
    G = a.shape[0]
    out = np.empty((G, NCOMP, PS, PS, PS), dtp)
    face = np.zeros((G, 3, 3, NCOMP, PS, PS), dtp) if want_face_flux else None
    ms = np.zeros((G,), dtp) if want_maxspeed else None
    bad = getattr(lib(), "oracle_hydro_advance_" + _sfx(dtp))(
        a.ctypes.data, out.ctypes.data, G, ghost, dtp.type(dt), dtp.type(dh), dtp.type(gamma), int(backward), c_mode,
        face.ctypes.data if want_face_flux else None, ms.ctypes.data if want_maxspeed else None, int(n_threads))
    if bad < 0:
        raise ValueError("oracle_hydro_advance: error %d" % bad)
    if bad > 0 and not return_bad:
        raise FloatingPointError("oracle met %d cells with rho<=0 or P<=0 (no floor is defined, DESIGN.md R7)" % bad)
    res = (out,)
    if want_face_flux:
        res += (face,)
    if want_maxspeed:
        res += (ms,)
    if return_bad:
        res += (bad,)
    return res if len(res) > 1 else out


def hydro_advance_badmask(inp, dt, dh, gamma, backward=0, dtype=None, c_mode=0, n_threads=1):
    """hydro_advance that also says WHERE the pass left the physical domain (reading R7/R17b).  Returns
    (out [G][5][16][16][16], badmask [G][22][22][22] uint8, count): bit 0 of badmask = the cell held five finite values
    with rho <= 0 or P <= 0 when some sweep read it; bit 1 = it held a non-finite value (what spreads from bit-0 cells,
    at most 3 cells along the axis of each later sweep).  Bookkeeping only: `out` is hydro_advance's."""
    dtp = np.dtype(dtype if dtype is not None else inp.dtype)
    a = np.ascontiguousarray(inp, dtype=dtp)
    assert a.ndim == 5 and a.shape[1:] == (NCOMP, NP, NP, NP), a.shape
    G = a.shape[0]
    out = np.empty((G, NCOMP, PS, PS, PS), dtp)
    mask = np.zeros((G, NP, NP, NP), np.uint8)
    bad = getattr(lib(), "oracle_hydro_advance_badmask_" + _sfx(dtp))(
        a.ctypes.data, out.ctypes.data, G, NGHOST, dtp.type(dt), dtp.type(dh), dtp.type(gamma), int(backward), c_mode,
        mask.ctypes.data, int(n_threads))
    if bad < 0:
        raise ValueError("oracle_hydro_advance_badmask: error %d" % bad)
    return out, mask, int(bad)


def count_ops():
    """Measured arithmetic of one patch-group pass: dict(add, mul, div, sqrt, cmp, abs)."""
    c = (ctypes.c_longlong * 6)()
    lib().oracle_count_ops(c)
    return dict(zip(("add", "mul", "div", "sqrt", "cmp", "abs"), [int(x) for x in c]))


def has_openmp():
    return bool(lib().oracle_has_openmp())


def ghost_fill(interior, grid, bc=(0, 0, 0), padded=None):
    """Preparation step on a single-level tiling, written out cell by cell (ghost zones of a patch group
    are copied from the sibling patches).  Pure data movement.

    interior: [G][5][16][16][16], G = gz*gy*gx groups tiling a box, grid = (gz, gy, gx), g = (kz*gy + ky)*gx + kx.
    bc = (bc_x, bc_y, bc_z): 0 periodic; 1 = ghost cells beyond that end of the box keep the value they have in
    `padded` (required then).  Returns [G][5][22][22][22].
    """
    a = np.asarray(interior)
    gz, gy, gx = grid
    assert a.shape == (gz * gy * gx, NCOMP, PS, PS, PS), a.shape
    out = np.array(padded, dtype=a.dtype, copy=True) if padded is not None else np.full(
        (a.shape[0], NCOMP, NP, NP, NP), np.nan, a.dtype)
    n = (gx * PS, gy * PS, gz * PS)
    for kz in range(gz):
        for ky in range(gy):
            for kx in range(gx):
                g = (kz * gy + ky) * gx + kx
                k = (kx, ky, kz)
                # per axis: source group coordinate and source interior index of each of the 22 padded positions
                src_grp, src_idx, ok = [], [], []
                for ax in range(3):
                    c = k[ax] * PS + np.arange(NP) - NGHOST          # cell coordinate in the box
                    inside = (c >= 0) & (c < n[ax])
                    c = np.mod(c, n[ax])
                    src_grp.append(c // PS)
                    src_idx.append(c % PS)
                    ok.append(inside | (bc[ax] == 0))
                # all 22^3 padded positions of this group at once (index arrays instead of three nested loops)
                Z, Y, X = np.meshgrid(np.arange(NP), np.arange(NP), np.arange(NP), indexing="ij")
                sg = (src_grp[2][Z] * gy + src_grp[1][Y]) * gx + src_grp[0][X]
                write = ok[2][Z] & ok[1][Y] & ok[0][X]
                vals = a[sg, :, src_idx[2][Z], src_idx[1][Y], src_idx[0][X]]        # [22][22][22][5]
                out[g][:, write] = vals[write].T
    return out


def max_signal_speed(padded, gamma):
    """max over all cells of c_s + max_i |v_i| (Eq.30), in the array's own precision."""
    u = np.asarray(padded)
    t = u.dtype.type
    rho = u[:, 0]
    v = np.abs(u[:, 1:4]) / rho[:, None]
    p = (t(gamma) - t(1)) * (u[:, 4] - t(0.5) * (u[:, 1] ** 2 + u[:, 2] ** 2 + u[:, 3] ** 2) / rho)
    return (np.sqrt(t(gamma) * p / rho) + v.max(axis=1)).max()


def run_uniform(padded, grid, bc, n_steps, cfl, dh, gamma, n_threads=1, order=0):
    """Multi-step loop on a single-level tiling (DESIGN.md NEXT-3).  Returns (padded state, list of dt).

    order = 0: each step is {dt from Eq.30 over all padded cells; one forward pass (x,y,z);
               ghost refill}.
    order = 1: the paper's full step: "a forward sweep in the order xyz, and follows a backward
               sweep in the order zyx.  The same time step must be employed by these two sweeps": each step is {dt
               from Eq.30; forward pass; ghost refill; backward pass (z,y,x) with the SAME dt; ghost refill} and
               advances the state by 2 dt.  The next dt is evaluated after the backward sweep (:424)."""
    assert order in (0, 1)
    u = np.array(padded, copy=True)
    t = u.dtype.type
    dts = []
    for _ in range(n_steps):
        dt = t(cfl) * t(dh) / max_signal_speed(u, gamma)
        out = hydro_advance(u, dt, dh, gamma, n_threads=n_threads)
        u = ghost_fill(out, grid, bc, padded=u)
        if order == 1:
            out = hydro_advance(u, dt, dh, gamma, backward=1, n_threads=n_threads)
            u = ghost_fill(out, grid, bc, padded=u)
        dts.append(float(dt))
    return u, dts
