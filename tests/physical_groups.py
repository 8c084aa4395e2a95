"""Which groups of a batch stay physical along one pass of the CPU oracle (test helper; uses oracle/, so tests only).

The scheme has no density or pressure floor (reading R7): a group is called physical when the oracle meets
no cell with rho <= 0 or P <= 0 on anything it reads, in fp32 AND in fp64, and both outputs are finite."""
from concurrent.futures import ThreadPoolExecutor

import numpy as np

import oracle


def physical_mask(inp, dt, dh, gamma, backward=0, n_threads=8):
    """Returns (mask[G] bool, out32[G][5][16]^3, out64[G][5][16]^3, bad32[G], bad64[G]); one oracle call per group
    (the oracle reports its count of non-physical cells per call)."""
    G = inp.shape[0]

    def one(args):
        g, dtype = args
        out, bad = oracle.hydro_advance(inp[g:g + 1], dt, dh, gamma, backward=backward, dtype=dtype, return_bad=True)
        return out[0], bad

    with ThreadPoolExecutor(n_threads) as ex:       # ctypes releases the GIL
        r32 = list(ex.map(one, [(g, np.float32) for g in range(G)]))
        r64 = list(ex.map(one, [(g, np.float64) for g in range(G)]))
    out32 = np.stack([r[0] for r in r32])
    out64 = np.stack([r[0] for r in r64])
    bad32 = np.array([r[1] for r in r32])
    bad64 = np.array([r[1] for r in r64])
    finite = np.isfinite(out32).all(axis=(1, 2, 3, 4)) & np.isfinite(out64).all(axis=(1, 2, 3, 4))
    return (bad32 == 0) & (bad64 == 0) & finite, out32, out64, bad32, bad64


def dilate3(mask):
    """mask [G][22][22][22] bool -> the same with every set cell grown by 3 cells along each axis (a 7^3 box, clipped at
    the edge of the padded group).  This is the domain of dependence of one pass (a sweep reaches 3 cells
    along its own axis, and the three sweeps of a pass act along x, y and z in turn): a cell that was non-physical when
    some sweep read it can change the pass's result at most inside this box, and nothing outside it."""
    d = np.asarray(mask, bool)
    for ax in (1, 2, 3):
        n = d.shape[ax]
        acc = d.copy()
        for sh in (1, 2, 3):
            to, fr = [slice(None)] * 4, [slice(None)] * 4
            to[ax], fr[ax] = slice(sh, n), slice(0, n - sh)
            acc[tuple(to)] |= d[tuple(fr)]
            to[ax], fr[ax] = slice(0, n - sh), slice(sh, n)
            acc[tuple(to)] |= d[tuple(fr)]
        d = acc
    return d


def outside(keep, a, dummy):
    """a [G][5][16][16][16] with the cells where keep [G][16][16][16] is False replaced by the physical state `dummy`
    (5 values), so that a whole-array comparison runs over the kept cells only."""
    return np.where(keep[:, None], a, np.asarray(dummy, a.dtype).reshape(1, 5, 1, 1, 1))
