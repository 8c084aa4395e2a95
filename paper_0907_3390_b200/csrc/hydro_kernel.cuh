// hydro_kernel.cuh — the batched hydro kernel (sm_100a): one persistent CTA per SM, one patch group at a time.
//
// Per group (steps 1-10):
//   H0  the padded group (212 960 B, contiguous in HBM) is bulk-copied into shared memory with cp.async.bulk (TMA,
//       SASS UBLKCP) completing on mbarriers.  Forward pass: in three chunks of z-planes, each issued by a warp
//       without z rows as soon as the z sweep of the PREVIOUS group has read those planes (the load runs under the
//       z sweep).  Backward pass: six chunks; ghost planes under the y and x sweeps, interior planes after the x sweep.
//   H1-H7 three in-place sweeps, one thread per row (rtvd_march), rows shrinking 22x22 -> 16x22 -> 16x16
//   H9  the last sweep streams the 16^3 interior to HBM straight from the registers of the march (forward, z march:
//       64-byte segments per half-warp; backward, x march: a thread owns a row, four cells per 128-bit store)
#pragma once
#include <cstdint>
#include "rtvd_march.cuh"

namespace gamer {

#ifndef GAMER_BLOCK_THREADS
#define GAMER_BLOCK_THREADS 512
#endif
constexpr int BLOCK_THREADS = GAMER_BLOCK_THREADS;
constexpr int GROUP_IN_FLOATS = NCOMP * NP * NP * NP;     // 53 240
constexpr int GROUP_OUT_FLOATS = NCOMP * PS * PS * PS;    // 20 480
constexpr int GROUP_FACE_FLOATS = 3 * 3 * NCOMP * PS * PS;
constexpr int GROUP_IN_BYTES = GROUP_IN_FLOATS * 4;       // 212 960
constexpr int VAR_FLOATS = NP * NP * NP;                  // 10 648
constexpr int CTL_BYTES = 512;                            // mbarriers, counters, reduction scratch (struct Ctl)
constexpr int SMEM_BYTES = GROUP_IN_BYTES + CTL_BYTES;

// ---- mbarrier / bulk-copy PTX ---------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_LOOP:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra WAIT_DONE;\n"
        "bra WAIT_LOOP;\n"
        "WAIT_DONE:\n"
        "}\n" ::"r"(smem_u32(bar)),
        "r"(parity)
        : "memory");
}
__device__ __forceinline__ void bulk_g2s(void* dst_smem, const void* src_gmem, uint32_t bytes, uint64_t* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     smem_u32(dst_smem)),
                 "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}
__device__ __forceinline__ void bulk_prefetch_l2(const void* src_gmem, uint32_t bytes) {
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(src_gmem), "r"(bytes) : "memory");
}
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

// ---- sinks ------------------------------------------------------------------------------------------------------
// Writes the updated cells back into the row in shared memory (in place); optionally the face fluxes to HBM.
// Along x (STRIDE 1) an even cell is held back one step and stored together with its odd right neighbour as one
// 64-bit store (cells 3 and 18 have no partner and go out alone).
template <int STRIDE>
struct SmemSink {
    float* dst[NCOMP];       // row-local component order, cell 0 of the row
    float* fptr[NCOMP];      // &face_flux[g][d][0][var(q)][b][a], or unused
    bool face_row;
    float held[NCOMP];
    template <int P>
    __device__ __forceinline__ void cell(int j, const float (&u)[NCOMP]) {
        constexpr int ODD = P & 1;
        if (STRIDE == 1) {
            if (ODD) {
                if (j == NG) {
#pragma unroll
                    for (int k = 0; k < NCOMP; ++k) dst[k][j] = u[k];
                } else {
#pragma unroll
                    for (int k = 0; k < NCOMP; ++k)
                        *reinterpret_cast<float2*>(dst[k] + j - 1) = make_float2(held[k], u[k]);
                }
            } else {
                if (j == NG + PS - 1) {
#pragma unroll
                    for (int k = 0; k < NCOMP; ++k) dst[k][j] = u[k];
                } else {
#pragma unroll
                    for (int k = 0; k < NCOMP; ++k) held[k] = u[k];
                }
            }
        } else {
#pragma unroll
            for (int k = 0; k < NCOMP; ++k) dst[k][j * STRIDE] = u[k];
        }
    }
    __device__ __forceinline__ void face(int p, const float (&f)[NCOMP]) {
        if (face_row) {
#pragma unroll
            for (int k = 0; k < NCOMP; ++k) fptr[k][p * (NCOMP * PS * PS)] = f[k];
        }
    }
};

// Writes the updated cells of the LAST sweep.  TO_GLOBAL: straight to out[g][v][.][.][.] with element stride OSTRIDE
// along the row; else in place in shared memory.  Tracks the CFL speed of the updated cells if WANT_SPEED.
template <int STRIDE, int OSTRIDE, bool TO_GLOBAL, bool WANT_SPEED>
struct FinalSink {
    float* dst[NCOMP];       // TO_GLOBAL: &out[g][var(q)][..] at interior cell 0 of the row; else smem row (cell 0)
    float* fptr[NCOMP];
    bool face_row;
    float gm1, ggm1;
    float speed;             // running max of c_s + max|v_i|
    float held[NCOMP];
    float h1[TO_GLOBAL && STRIDE == 1 ? NCOMP : 1], h2[TO_GLOBAL && STRIDE == 1 ? NCOMP : 1];
    template <int P>
    __device__ __forceinline__ void cell(int j, const float (&u)[NCOMP]) {
        constexpr int ODD = P & 1;
        if (TO_GLOBAL && STRIDE == 1) {
            // backward pass, last sweep along x (PHASE4 march): a thread owns the 16 contiguous cells of its output row
            // (64 B, aligned) and sends them off four at a time, as 128-bit stores; P = position in the group of four
            if (P == 3) {
#pragma unroll
                for (int k = 0; k < NCOMP; ++k) held[k] = u[k];
            } else if (P == 0) {
#pragma unroll
                for (int k = 0; k < NCOMP; ++k) h1[k] = u[k];
            } else if (P == 1) {
#pragma unroll
                for (int k = 0; k < NCOMP; ++k) h2[k] = u[k];
            } else {
#pragma unroll
                for (int k = 0; k < NCOMP; ++k)
                    *reinterpret_cast<float4*>(dst[k] + (j - 3 - NG)) = make_float4(held[k], h1[k], h2[k], u[k]);
            }
        } else if (TO_GLOBAL) {
#pragma unroll
            for (int k = 0; k < NCOMP; ++k) dst[k][(j - NG) * OSTRIDE] = u[k];
        } else if (STRIDE == 1) {
            if (ODD) {
                if (j == NG) {
#pragma unroll
                    for (int k = 0; k < NCOMP; ++k) dst[k][j] = u[k];
                } else {
#pragma unroll
                    for (int k = 0; k < NCOMP; ++k)
                        *reinterpret_cast<float2*>(dst[k] + j - 1) = make_float2(held[k], u[k]);
                }
            } else {
                if (j == NG + PS - 1) {
#pragma unroll
                    for (int k = 0; k < NCOMP; ++k) dst[k][j] = u[k];
                } else {
#pragma unroll
                    for (int k = 0; k < NCOMP; ++k) held[k] = u[k];
                }
            }
        } else {
#pragma unroll
            for (int k = 0; k < NCOMP; ++k) dst[k][j * STRIDE] = u[k];
        }
        if (WANT_SPEED) {    // Eq.30 on the updated cell; approximate reciprocal / root (1-2 ulp)
            const float rinv = rcp_fast(u[0]);
            float q = u[2] * u[2];
            q = fmaf(u[3], u[3], q);
            q = fmaf(u[1], u[1], q);
            const float eint = fmaf(-q, 0.5f * rinv, u[4]);
            const float cs = sqrt_fast((ggm1 * eint) * rinv);
            const float vm = fmaxf(fmaxf(fabsf(u[1]), fabsf(u[2])), fabsf(u[3])) * rinv;
            speed = fmaxf(speed, cs + vm);
        }
    }
    __device__ __forceinline__ void face(int p, const float (&f)[NCOMP]) {
        if (face_row) {
#pragma unroll
            for (int k = 0; k < NCOMP; ++k) fptr[k][p * (NCOMP * PS * PS)] = f[k];
        }
    }
};

// Row-local component order (rho, m_n, m_t1, m_t2, e) -> variable index, for sweep axis d (0:x, 1:y, 2:z).
__device__ __forceinline__ int var_of(int d, int q) {
    return q == 0 ? 0 : (q == 4 ? 4 : 1 + (d + q - 1) % 3);
}

// One sweep along axis D over the rows that are still valid.  `smem` holds the group as [v][z][y][x].
//   LO_A/N_A, LO_B/N_B: the two transverse axes (A = lower axis number, fastest across threads), start and count.
//   t: index of this thread's row among the N_A * N_B rows (rows beyond are skipped).  gate: see RowMarch::pair.
template <int D, int LO_A, int N_A, int LO_B, int N_B, bool LAST, bool LAST_TO_GLOBAL, bool WANT_FACE, bool WANT_SPEED,
          class Gate>
__device__ __forceinline__ void sweep(float* smem, const GasConst& gc, float* __restrict__ out_g,
                                      float* __restrict__ face_g, float& speed, const int t, Gate& gate) {
    constexpr int STRIDE = D == 0 ? 1 : (D == 1 ? NP : NP * NP);
    constexpr int AX_A = D == 0 ? 1 : 0;                      // transverse axes: the two that are not D, ascending
    constexpr int AX_B = D == 2 ? 1 : 2;
    constexpr int STR_A = AX_A == 0 ? 1 : NP;
    constexpr int STR_B = AX_B == 1 ? NP : NP * NP;
    constexpr int OSTRIDE = D == 0 ? 1 : (D == 1 ? PS : PS * PS);
    constexpr int OSTR_A = AX_A == 0 ? 1 : PS;
    constexpr int OSTR_B = AX_B == 1 ? PS : PS * PS;
    if (t >= N_A * N_B) return;
    // padded transverse coordinates of this thread's row.  Where the fast axis is the 16 interior x cells, the two
    // half-warps are placed 16 banks apart (y sweep: z and z+4; z sweep: y and y+8) so that the 4-byte accesses of a
    // warp hit 32 different banks; rows along x are 8-byte accessed and conflict-free for consecutive rows.
    int a, b;
    if (D == 1 && N_A == PS && N_B == NP) {
        const int w = t >> 5, h = (t >> 4) & 1;
        a = LO_A + (t & 15);
        b = w < 10 ? 8 * (w >> 2) + (w & 3) + 4 * h : 18 + h;
    } else if (D == 1 && N_A == NP && N_B == PS) {
        // backward y sweep: 22 x columns x 16 planes.  x = 0..15 as above (the half-warps 4 planes = 16 banks apart);
        // x = 16..21: six columns of planes that are two apart (a plane is 4 banks on, 6 columns fit in the 8)
        if (t < PS * PS) {
            a = t & 15;
            b = LO_B + 8 * (t >> 7) + ((t >> 5) & 3) + 4 * ((t >> 4) & 1);
        } else {
            const int r = t - PS * PS, zi = r / 6;
            a = PS + r - 6 * zi;
            b = LO_B + 2 * (zi & 7) + (zi >> 3);
        }
    } else if (D == 2 && N_A == PS && N_B == PS) {
        a = LO_A + (t & 15);
        b = LO_B + (t >> 5) + 8 * ((t >> 4) & 1);
    } else {
        a = LO_A + t % N_A;
        b = LO_B + t / N_A;
    }
    const int base = a * STR_A + b * STR_B;
    const float* src[NCOMP];
#pragma unroll
    for (int q = 0; q < NCOMP; ++q) src[q] = smem + var_of(D, q) * VAR_FLOATS + base;
    const bool face_row = WANT_FACE && a >= NG && a < NG + PS && b >= NG && b < NG + PS;
    if (!LAST) {
        SmemSink<STRIDE> sink;
#pragma unroll
        for (int q = 0; q < NCOMP; ++q) {
            sink.dst[q] = const_cast<float*>(src[q]);
            sink.fptr[q] = WANT_FACE ? face_g + ((D * 3) * NCOMP + var_of(D, q)) * (PS * PS) + (b - NG) * PS + (a - NG)
                                     : nullptr;
        }
        sink.face_row = face_row;
        rtvd_march<STRIDE, WANT_FACE>(src, gc, sink, gate);
    } else {
        FinalSink<STRIDE, OSTRIDE, LAST_TO_GLOBAL, WANT_SPEED> sink;
#pragma unroll
        for (int q = 0; q < NCOMP; ++q) {
            sink.dst[q] = LAST_TO_GLOBAL
                              ? out_g + var_of(D, q) * (PS * PS * PS) + (a - NG) * OSTR_A + (b - NG) * OSTR_B
                              : const_cast<float*>(src[q]);
            sink.fptr[q] = WANT_FACE ? face_g + ((D * 3) * NCOMP + var_of(D, q)) * (PS * PS) + (b - NG) * PS + (a - NG)
                                     : nullptr;
        }
        sink.face_row = face_row;
        sink.gm1 = gc.gm1;
        sink.ggm1 = gc.ggm1;
        sink.speed = speed;
        rtvd_march<STRIDE, WANT_FACE, LAST_TO_GLOBAL && D == 0>(src, gc, sink, gate);
        speed = sink.speed;
    }
}

// ---- control block behind the group in shared memory -------------------------------------------------------------
constexpr int PLANE_FLOATS = NP * NP;             // 484: one z-plane of one variable, contiguous in HBM and in smem
constexpr int PLANE_BYTES = PLANE_FLOATS * 4;     // 1936 = 16 * 121
constexpr int N_ZPAIR = NP / 2;                   // 11 pairs of z-planes
constexpr int N_ZWARP = PS * PS / 32;             // 8 warps march along z

#ifndef GAMER_CHUNK_PAIRS
#define GAMER_CHUNK_PAIRS 4           /* z-plane pairs per load chunk: planes 0-7, 8-15, 16-21 */
#endif
constexpr int CHUNK_PAIRS = GAMER_CHUNK_PAIRS;
constexpr int N_CHUNK = (N_ZPAIR + CHUNK_PAIRS - 1) / CHUNK_PAIRS;
__host__ __device__ constexpr int chunk_of_plane(int z) { return (z >> 1) / CHUNK_PAIRS; }
__host__ __device__ constexpr int chunk_lo(int c) { return 2 * c * CHUNK_PAIRS; }                    // first plane
__host__ __device__ constexpr int chunk_hi(int c) {                                                  // one past last
    return 2 * (c + 1) * CHUNK_PAIRS < NP ? 2 * (c + 1) * CHUNK_PAIRS : NP;
}

struct Ctl {
    uint64_t full[N_ZPAIR];           // forward: load chunk c of the group has landed; backward: full[0] = whole group
    unsigned int red[4];              // CFL speed of the group (bit pattern), slot = iteration & 3
    unsigned int zfin[4];             // warps that have finished the group, slot = iteration & 3
};
static_assert(sizeof(Ctl) <= CTL_BYTES, "control block");

// Polls an mbarrier phase.  try_wait comes back after a few cycles whatever suspend-time hint it is given (measured:
// one poll per ~13 cycles), and a polling warp takes issue slots from the marching warps of its SM sub-partition — the
// z warps that shared one with pollers ran 30 % slower.  So only ONE warp ever polls (the loader); every other wait
// in the forward pass is a hardware named barrier (bar.sync blocks without issuing).
__device__ __forceinline__ void mbar_wait_poll(uint64_t* bar, uint32_t parity) {
    uint32_t ok;
    do {
        asm volatile(
            "{\n"
            ".reg .pred p;\n"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
            "selp.u32 %0, 1, 0, p;\n"
            "}\n"
            : "=r"(ok)
            : "r"(smem_u32(bar)), "r"(parity)
            : "memory");
    } while (!ok);
}
__device__ __forceinline__ void named_bar_sync(int id, int n_threads) {
    asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(n_threads) : "memory");
}
__device__ __forceinline__ void named_bar_arrive(int id, int n_threads) {
    asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(n_threads) : "memory");
}

// Named barriers of the forward pass (0 is __syncthreads).  LOADER_WARP has no z rows and only 4 x rows.
constexpr int LOADER_WARP = BLOCK_THREADS / 32 - 1;
static_assert(BLOCK_THREADS == 512, "16 warps: 16 x tasks (the last one 4 rows wide), 11 y tasks, 8 z tasks");
constexpr int BAR_ZFREE = 1;                      // + c: the 256 z threads arrive, the loader warp syncs
constexpr int BAR_FULL = 1 + N_CHUNK;             // + c: the loader warp arrives, the x warps that need chunk c sync
static_assert(BAR_FULL + N_CHUNK <= 16, "named barriers");
constexpr int ZFREE_THREADS = PS * PS + 32;
// first / last load chunk that the x task of warp w (rows 32w..32w+31 of the (z,y) rows) reads
__host__ __device__ constexpr int xtask_chunk_lo(int w) { return chunk_of_plane(32 * w / NP); }
__host__ __device__ constexpr int xtask_chunk_hi(int w) {
    return chunk_of_plane((32 * w + 31 < NP * NP ? 32 * w + 31 : NP * NP - 1) / NP);
}
__host__ __device__ constexpr int full_threads(int c) {       // participants of BAR_FULL + c
    int n = 32;                                               // the loader
    for (int w = 0; w < LOADER_WARP; ++w)
        if (xtask_chunk_lo(w) <= c && c <= xtask_chunk_hi(w)) n += 32;
    return n;
}

// Bulk copies (TMA) of load chunk c — z-planes chunk_lo(c)..chunk_hi(c)-1, contiguous per variable in HBM and in
// shared memory — of all five variables of one group; they complete on full[c].  One thread calls this.
__device__ __forceinline__ void load_chunk(float* smem, Ctl* ctl, const float* __restrict__ in_g, int c) {
    const int lo = chunk_lo(c), bytes = (chunk_hi(c) - lo) * PLANE_BYTES;
    mbar_expect_tx(&ctl->full[c], NCOMP * bytes);
#pragma unroll
    for (int v = 0; v < NCOMP; ++v)
        bulk_g2s(smem + v * VAR_FLOATS + lo * PLANE_FLOATS, in_g + v * VAR_FLOATS + lo * PLANE_FLOATS, bytes,
                 &ctl->full[c]);
}

// Backward pass (z,y,x): the z sweep comes first and needs the planes in order; after it the ghost planes 0-2 and 19-21
// are dead (the y and x sweeps only touch z = 3..18), so the same planes of the CTA's NEXT group are loaded into them
// under the y and x sweeps; the interior planes follow in four chunks once the x sweep has read them.
constexpr int BCHUNK_PLANES = 4;                                  // interior planes per load chunk
constexpr int N_BCHUNK = 2 + PS / BCHUNK_PLANES;                  // ghost planes below, interior chunks, ghost planes above
__host__ __device__ constexpr int bchunk_lo(int c) { return c == 0 ? 0 : NG + BCHUNK_PLANES * (c - 1); }   // 0, 3, 7, 11, 15, 19
__host__ __device__ constexpr int bchunk_hi(int c) {
    return c == 0 ? NG : (c == N_BCHUNK - 1 ? NP : NG + BCHUNK_PLANES * c);
}
static_assert(bchunk_hi(N_BCHUNK - 2) == NG + PS && bchunk_lo(N_BCHUNK - 1) == NG + PS, "backward load chunks");
// One thread calls this.
__device__ __forceinline__ void load_bchunk(float* smem, Ctl* ctl, const float* __restrict__ in_g, int c) {
    const int lo = bchunk_lo(c), bytes = (bchunk_hi(c) - lo) * PLANE_BYTES;
    mbar_expect_tx(&ctl->full[c], NCOMP * bytes);
#pragma unroll
    for (int v = 0; v < NCOMP; ++v)
        bulk_g2s(smem + v * VAR_FLOATS + lo * PLANE_FLOATS, in_g + v * VAR_FLOATS + lo * PLANE_FLOATS, bytes,
                 &ctl->full[c]);
}
// Gate of the forward z march (the last sweep; its results go straight to HBM): once a thread has the last planes of
// a load chunk in registers it never reads the chunk again and says so on BAR_ZFREE + c (bar.arrive: nothing in the
// march waits).  The loader warp syncs on these barriers and starts the bulk copies of the same planes of the CTA's
// NEXT group into the space, so that the load runs under the z sweep instead of in front of the x sweep.
struct ZPlaneGate {
    bool has_next;
    __device__ __forceinline__ void acquire(int) {}
    __device__ __forceinline__ void release(int n) {
        const int k = n >> 1;
        if (has_next && ((k + 1) % CHUNK_PAIRS == 0 || k == N_ZPAIR - 1))
            named_bar_arrive(BAR_ZFREE + k / CHUNK_PAIRS, ZFREE_THREADS);
    }
};

// Gate of the backward z march (the first sweep): wait for a load chunk when the march first reaches one of its planes.
// The march reads planes n, n+1 (n even): chunk 0 at n = 0, chunk c >= 1 (first plane 4 c - 1) at n = 4 c - 2.
struct ChunkWaitGate {
    Ctl* ctl;
    uint32_t parity;
    __device__ __forceinline__ void acquire(int n) {
        static_assert(BCHUNK_PLANES == 4, "gate arithmetic");
        if (n == 0) mbar_wait_poll(&ctl->full[0], parity);
        else if ((n & 3) == 2) mbar_wait_poll(&ctl->full[(n + 2) >> 2], parity);
    }
    __device__ __forceinline__ void release(int) {}
};

// The loader warp, during the z sweep of a group that has a successor.
__device__ __forceinline__ void load_next_group(float* smem, Ctl* ctl, const float* __restrict__ in_next) {
#pragma unroll
    for (int c = 0; c < N_CHUNK; ++c) {
        named_bar_sync(BAR_ZFREE + c, ZFREE_THREADS);
        if ((threadIdx.x & 31) == 0) {
            fence_proxy_async();
            load_chunk(smem, ctl, in_next, c);
        }
    }
}

// The loader warp, before the x sweep: tells the x warps which chunks have landed.
__device__ __forceinline__ void release_chunks(Ctl* ctl, uint32_t parity) {
#pragma unroll
    for (int c = 0; c < N_CHUNK; ++c) {
        mbar_wait_poll(&ctl->full[c], parity);
        named_bar_arrive(BAR_FULL + c, full_threads(c));
    }
}

// Per-group CFL speed: warp maximum, then a shared-memory maximum over the warps that hold final cells; the last of
// them writes group_maxspeed[g].  The slot (iteration & 3) keeps groups that overlap in time apart.
__device__ __forceinline__ void reduce_speed(Ctl* ctl, float speed, unsigned int it, int n_warps,
                                             float* __restrict__ dst) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) speed = fmaxf(speed, __shfl_xor_sync(0xffffffffu, speed, o));
    if ((threadIdx.x & 31) == 0) {
        const int slot = it & 3;
        atomicMax(&ctl->red[slot], __float_as_uint(speed));          // positive floats order like their bit patterns
        if (atomicAdd(&ctl->zfin[slot], 1u) == (unsigned int)(n_warps - 1)) {
            *dst = __uint_as_float(atomicExch(&ctl->red[slot], 0u));
            ctl->zfin[slot] = 0u;
        }
    }
}

// DEVICE_DT: the time step is read from *d_dt (written by an earlier kernel on the same stream, e.g. cfl_dt_kernel)
// and the dt-dependent constants are formed here exactly as make_const() forms them on the host.
template <bool BACKWARD, bool WANT_FACE, bool WANT_SPEED, bool DEVICE_DT = false>
__global__ void __launch_bounds__(BLOCK_THREADS, 1)
hydro_advance_kernel(const float* __restrict__ in, float* __restrict__ out, long long n_groups, GasConst gc_in,
                     float* __restrict__ face_flux, float* __restrict__ group_maxspeed,
                     const float* __restrict__ d_dt = nullptr) {
    GasConst gc = gc_in;
    if (DEVICE_DT) {
        const float k = __fdiv_rn(*d_dt, gc.dh);
        gc.kq = __fmul_rn(0.25f, k);
        gc.kh = __fmul_rn(0.5f, k);
        gc.kq_gm1 = __fmul_rn(gc.kq, gc.gm1);
        gc.kq_sg = __fmul_rn(gc.kq, gc.sg);
    }
    extern __shared__ __align__(128) unsigned char smem_raw[];
    float* smem = reinterpret_cast<float*>(smem_raw);
    Ctl* ctl = reinterpret_cast<Ctl*>(smem_raw + GROUP_IN_BYTES);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

    if (threadIdx.x == 0) {
        for (int k = 0; k < N_ZPAIR; ++k) mbar_init(&ctl->full[k], 1);
        for (int i = 0; i < 4; ++i) {
            ctl->red[i] = 0u;
            ctl->zfin[i] = 0u;
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        fence_proxy_async();          // the first group of this CTA, chunk by chunk
        const float* in_g = in + (long long)blockIdx.x * GROUP_IN_FLOATS;
        if (!BACKWARD) {
            for (int c = 0; c < N_CHUNK; ++c) load_chunk(smem, ctl, in_g, c);
        } else {
            for (int c = 0; c < N_BCHUNK; ++c) load_bchunk(smem, ctl, in_g, c);
        }
    }
    __syncthreads();

    NoGate nogate;
    unsigned int it = 0;
    for (long long g = blockIdx.x; g < n_groups; g += gridDim.x, ++it) {
        const uint32_t parity = it & 1u;
        float* out_g = out + g * (long long)GROUP_OUT_FLOATS;
        float* face_g = WANT_FACE ? face_flux + g * (long long)GROUP_FACE_FLOATS : nullptr;
        float speed = 0.f;
        if (!BACKWARD) {
            // x sweep: warp w takes the (z,y) rows 32w..32w+31 and starts as soon as their planes have landed.  Warps
            // 8..15 have no z rows and arrive here while the z sweep of the previous group is still running.
            // (Giving those warps the planes that are handed back first was measured: no gain.)
            const int row_lo = 32 * warp;
            if (warp == LOADER_WARP) {
                release_chunks(ctl, parity);
            } else {
                for (int c = xtask_chunk_lo(warp); c <= xtask_chunk_hi(warp); ++c)
                    named_bar_sync(BAR_FULL + c, full_threads(c));
            }
            sweep<0, 0, NP, 0, NP, false, false, WANT_FACE, false>(smem, gc, out_g, face_g, speed, row_lo + lane, nogate);
            __syncthreads();
            sweep<1, NG, PS, 0, NP, false, false, WANT_FACE, false>(smem, gc, out_g, face_g, speed, threadIdx.x, nogate);
            __syncthreads();
            const long long gn = g + gridDim.x;
            if (warp < N_ZWARP) {
                ZPlaneGate gate;
                gate.has_next = gn < n_groups;
                sweep<2, NG, PS, NG, PS, true, true, WANT_FACE, WANT_SPEED>(smem, gc, out_g, face_g, speed, threadIdx.x,
                                                                            gate);
                if (WANT_SPEED) reduce_speed(ctl, speed, it, N_ZWARP, group_maxspeed + g);
            } else if (warp == LOADER_WARP && gn < n_groups) {
                load_next_group(smem, ctl, in + gn * (long long)GROUP_IN_FLOATS);
            }
            // no CTA-wide barrier: a plane is overwritten only after all z threads have read it (BAR_ZFREE), and the
            // next group's x tasks wait for their planes (BAR_FULL)
        } else {
            // The group arrives in six chunks of z-planes (bchunk_lo/hi); the z march (first sweep) waits for a chunk
            // only when it reaches its first plane.  All chunks of this group were issued earlier: by the prologue
            // (first group of the CTA) or under / after the sweeps of the previous group.
            // (Measured and rejected: the x march storing to HBM itself with 64-bit stores, 9 % slower — uncoalesced;
            // a loader warp issuing the copies instead of thread 0, 2 % slower — every warp has z rows in the first
            // sweep and a bulk copy holds its issuer for about as long as the transfer takes.)
            const long long gn = g + gridDim.x;
            const bool has_next = gn < n_groups;
            const float* in_next = in + (has_next ? gn : g) * (long long)GROUP_IN_FLOATS;
            if (threadIdx.x == 0 && has_next) bulk_prefetch_l2(in_next, GROUP_IN_BYTES);
            ChunkWaitGate zgate;
            zgate.ctl = ctl;
            zgate.parity = parity;
            sweep<2, 0, NP, 0, NP, false, false, WANT_FACE, false>(smem, gc, out_g, face_g, speed, threadIdx.x, zgate);
            __syncthreads();
            // the ghost planes 0-2 and 19-21 are dead from here on: the next group's go in under the y and x sweeps
            if (threadIdx.x == BLOCK_THREADS - 1 && has_next) {      // a thread without y or x rows
                fence_proxy_async();
                load_bchunk(smem, ctl, in_next, 0);
                load_bchunk(smem, ctl, in_next, N_BCHUNK - 1);
            }
            sweep<1, 0, NP, NG, PS, false, false, WANT_FACE, false>(smem, gc, out_g, face_g, speed, threadIdx.x, nogate);
            __syncthreads();
            // last sweep: along x, every thread sends its row to HBM itself, four cells per 128-bit store (lanes 64 B
            // apart: half of every sector written per store, the other half by the next one), and all the interior planes
            // are handed to the next group's bulk copies at once.  (In place + a coalesced copy-out, chunk by chunk:
            // 115.3 against 114.7 ns/group; DESIGN.md 6 has this and the other variants.)
            sweep<0, NG, PS, NG, PS, true, true, WANT_FACE, WANT_SPEED>(smem, gc, out_g, face_g, speed, threadIdx.x,
                                                                        nogate);
            if (WANT_SPEED && warp < PS * PS / 32) reduce_speed(ctl, speed, it, PS * PS / 32, group_maxspeed + g);
            __syncthreads();
            if (threadIdx.x == 0 && has_next) {
                fence_proxy_async();
                for (int c = 1; c < N_BCHUNK - 1; ++c) load_bchunk(smem, ctl, in_next, c);
            }
        }
    }
}

}  // namespace gamer
