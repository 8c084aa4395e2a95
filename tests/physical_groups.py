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
