// hydro_kernel.cuh — the batched hydro kernel (sm_100a): one persistent CTA per SM, one patch group at a time.
//
// Per group (steps 1-10):
//   H0  one elected thread bulk-copies the padded group (212 960 B, contiguous in HBM) into shared memory with
//       cp.async.bulk (TMA, SASS UBLKCP) completing on an mbarrier; the next group is prefetched into L2 meanwhile
//   H1-H7 three in-place sweeps, one thread per row (rtvd_march), rows shrinking 22x22 -> 16x22 -> 16x16
//   H9  the last sweep streams the 16^3 interior to HBM (forward: straight from the registers of the z march,
//       64-byte segments; backward: in place, then a 128-bit coalesced copy-out)
#pragma once
#include <cstdint>
#ifdef GAMER_MARCH_V1
#include "rtvd_march.cuh"
#else
#include "rtvd_march2.cuh"
#endif

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
constexpr int SMEM_BYTES = GROUP_IN_BYTES + 64;           // + mbarrier and reduction scratch

#ifdef GAMER_PHASE_TIMERS
// debug builds only (never defined by build.py): per-CTA cycles spent waiting for the load / in each sweep
__device__ long long g_phase_cycles[1024 * 4];
#endif

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
    template <int ODD>
    __device__ __forceinline__ void cell(int j, const float (&u)[NCOMP]) {
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
    template <int ODD>
    __device__ __forceinline__ void cell(int j, const float (&u)[NCOMP]) {
        if (TO_GLOBAL) {
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
        if (WANT_SPEED) {    // Eq.30 on the updated cell
            const float rinv = 1.0f / u[0];
            float q = u[2] * u[2];
            q = fmaf(u[3], u[3], q);
            q = fmaf(u[1], u[1], q);
            const float eint = fmaf(-q, 0.5f * rinv, u[4]);
            const float cs = sqrtf((ggm1 * eint) * rinv);
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
template <int D, int LO_A, int N_A, int LO_B, int N_B, bool LAST, bool LAST_TO_GLOBAL, bool WANT_FACE, bool WANT_SPEED>
__device__ __forceinline__ void sweep(float* smem, const GasConst& gc, float* __restrict__ out_g,
                                      float* __restrict__ face_g, float& speed) {
    constexpr int STRIDE = D == 0 ? 1 : (D == 1 ? NP : NP * NP);
    constexpr int AX_A = D == 0 ? 1 : 0;                      // transverse axes: the two that are not D, ascending
    constexpr int AX_B = D == 2 ? 1 : 2;
    constexpr int STR_A = AX_A == 0 ? 1 : NP;
    constexpr int STR_B = AX_B == 1 ? NP : NP * NP;
    constexpr int OSTRIDE = D == 0 ? 1 : (D == 1 ? PS : PS * PS);
    constexpr int OSTR_A = AX_A == 0 ? 1 : PS;
    constexpr int OSTR_B = AX_B == 1 ? PS : PS * PS;
#ifdef GAMER_DUP_ROWS      // timing experiment only: surplus threads redo rows (results are garbage)
    const int t = threadIdx.x % (N_A * N_B);
#else
    const int t = threadIdx.x;
    if (t >= N_A * N_B) return;
#endif
    // padded transverse coordinates of this thread's row.  Where the fast axis is the 16 interior x cells, the two
    // half-warps are placed 16 banks apart (y sweep: z and z+4; z sweep: y and y+8) so that the 4-byte accesses of a
    // warp hit 32 different banks; rows along x are 8-byte accessed and conflict-free for consecutive rows.
    int a, b;
    if (D == 1 && N_A == PS && N_B == NP) {
        const int w = t >> 5, h = (t >> 4) & 1;
        a = LO_A + (t & 15);
        b = w < 10 ? 8 * (w >> 2) + (w & 3) + 4 * h : 18 + h;
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
        rtvd_march<STRIDE, WANT_FACE>(src, gc, sink);
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
        rtvd_march<STRIDE, WANT_FACE>(src, gc, sink);
        speed = sink.speed;
    }
}

template <bool BACKWARD, bool WANT_FACE, bool WANT_SPEED>
__global__ void __launch_bounds__(BLOCK_THREADS, 1)
hydro_advance_kernel(const float* __restrict__ in, float* __restrict__ out, long long n_groups, GasConst gc,
                     float* __restrict__ face_flux, float* __restrict__ group_maxspeed) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    float* smem = reinterpret_cast<float*>(smem_raw);
    uint64_t* bar = reinterpret_cast<uint64_t*>(smem_raw + GROUP_IN_BYTES);
    unsigned int* red = reinterpret_cast<unsigned int*>(smem_raw + GROUP_IN_BYTES + 16);

    if (threadIdx.x == 0) {
        mbar_init(bar, 1);
        *red = 0u;
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

#ifdef GAMER_PHASE_TIMERS
    long long tacc[5] = {0, 0, 0, 0, 0}, tt0, tt1;
#define PHASE_T0() tt0 = clock64()
#define PHASE_ACC(i) do { tt1 = clock64(); tacc[i] += tt1 - tt0; tt0 = tt1; } while (0)
#else
#define PHASE_T0()
#define PHASE_ACC(i)
#endif
    uint32_t parity = 0;
    for (long long g = blockIdx.x; g < n_groups; g += gridDim.x) {
        PHASE_T0();
        if (threadIdx.x == 0) {
            fence_proxy_async();      // generic-proxy accesses of the previous group are ordered before the async write
            mbar_expect_tx(bar, GROUP_IN_BYTES);
            bulk_g2s(smem, in + g * (long long)GROUP_IN_FLOATS, GROUP_IN_BYTES, bar);
            const long long gn = g + gridDim.x;
            if (gn < n_groups) bulk_prefetch_l2(in + gn * (long long)GROUP_IN_FLOATS, GROUP_IN_BYTES);
        }
        mbar_wait(bar, parity);
        parity ^= 1u;
        PHASE_ACC(0);

        float* out_g = out + g * (long long)GROUP_OUT_FLOATS;
        float* face_g = WANT_FACE ? face_flux + g * (long long)GROUP_FACE_FLOATS : nullptr;
        float speed = 0.f;
        if (!BACKWARD) {
            sweep<0, 0, NP, 0, NP, false, false, WANT_FACE, false>(smem, gc, out_g, face_g, speed);   // x: (y,z) all
            __syncthreads();
            PHASE_ACC(1);
            sweep<1, NG, PS, 0, NP, false, false, WANT_FACE, false>(smem, gc, out_g, face_g, speed);  // y: x int, z all
            __syncthreads();
            PHASE_ACC(2);
            sweep<2, NG, PS, NG, PS, true, true, WANT_FACE, WANT_SPEED>(smem, gc, out_g, face_g, speed);   // z
        } else {
            sweep<2, 0, NP, 0, NP, false, false, WANT_FACE, false>(smem, gc, out_g, face_g, speed);   // z: (x,y) all
            __syncthreads();
            sweep<1, 0, NP, NG, PS, false, false, WANT_FACE, false>(smem, gc, out_g, face_g, speed);  // y: x all, z int
            __syncthreads();
            sweep<0, NG, PS, NG, PS, true, false, WANT_FACE, WANT_SPEED>(smem, gc, out_g, face_g, speed);  // x in place
            __syncthreads();
            // coalesced 128-bit copy-out of the interior: 16 B = 4 cells of a 16-cell row (row start 3 is not 16-B
            // aligned in shared memory, so read scalars, write float4)
            for (int i = threadIdx.x; i < GROUP_OUT_FLOATS / 4; i += BLOCK_THREADS) {
                const int x4 = i & 3, y = (i >> 2) & 15, z = (i >> 6) & 15, v = i >> 10;
                const float* s = smem + v * VAR_FLOATS + (z + NG) * (NP * NP) + (y + NG) * NP + NG + 4 * x4;
                float4 val = make_float4(s[0], s[1], s[2], s[3]);
                reinterpret_cast<float4*>(out_g)[i] = val;
            }
        }
        if (WANT_SPEED) {
            // positive floats order like their bit patterns
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) speed = fmaxf(speed, __shfl_xor_sync(0xffffffffu, speed, o));
            if ((threadIdx.x & 31) == 0) atomicMax(red, __float_as_uint(speed));
            __syncthreads();
            if (threadIdx.x == 0) {
                group_maxspeed[g] = __uint_as_float(*red);
                *red = 0u;
            }
        }
        __syncthreads();     // every thread is done with the buffer before the next bulk copy overwrites it
        PHASE_ACC(3);
    }
#ifdef GAMER_PHASE_TIMERS
    if (threadIdx.x == 0)
        for (int i = 0; i < 4; ++i) g_phase_cycles[blockIdx.x * 4 + i] = tacc[i];
#endif
}

}  // namespace gamer
