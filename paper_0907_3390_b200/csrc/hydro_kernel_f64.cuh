// hydro_kernel_f64.cuh — double-precision variant of the forward pass (NEXT-4; "single precision is
// assumed unless ... explicitly stated", double precision for the convergence tests).
//
// Same row march as the fp32 kernel (rtvd_march.cuh, T = double).  A padded group in fp64 is 425 920 B and does not fit
// in shared memory, so the pass is cut where the method allows it: the x and y sweeps act inside one z-plane
// (PAPER.md:174-178), so they run on two halves of 11 planes (212 960 B each, bulk-copied by TMA); what the z sweep
// needs of their result — the 16 x 16 interior columns of all 22 planes, 225 280 B — goes through a per-CTA scratch
// block in device memory (L2-resident: 33 MB for 148 CTAs) and comes back as one shared-memory block for the z sweep,
// which writes the interior straight to HBM.  One persistent CTA per SM, 256 threads (up to 255 registers: the
// march state is twice as wide in fp64).  Traffic per group: 425 920 B in + 163 840 B out (+ 2 x 225 280 B of scratch
// that stays in L2).
#pragma once
#include <cstdint>

#include "hydro_kernel.cuh"

namespace gamer {

constexpr int F64_THREADS = 256;
constexpr int HALF_PLANES = NP / 2;                                  // 11
constexpr int HALF_VAR = HALF_PLANES * NP * NP;                      // 5324 doubles: one variable of a half
constexpr int ZBUF_VAR = NP * PS * PS;                               // 5632 doubles: one variable of the z-sweep block
constexpr int BWD_VAR = PS * NP * NP;                                // 7744 doubles: 16 z-swept planes of one variable
constexpr int BWD_SCRATCH_DOUBLES = NCOMP * BWD_VAR;                 // 38 720 per CTA (backward pass)
constexpr int BWD_CHUNK_PLANES = 8;                                  // planes per y/x stage of the backward pass
constexpr int BWD_CHUNK_VAR = BWD_CHUNK_PLANES * NP * NP;            // 3872
constexpr int FWD_SCRATCH_DOUBLES = NCOMP * ZBUF_VAR;                // 28 160 per CTA (forward pass)
constexpr int F64_SCRATCH_DOUBLES = BWD_SCRATCH_DOUBLES;             // what the caller provides per CTA
constexpr int F64_DATA_BYTES = FWD_SCRATCH_DOUBLES * 8;              // 225 280 (>= 5 * 5324 * 8 = 212 960)
constexpr int F64_SMEM_BYTES = F64_DATA_BYTES + 64;

template <int STRIDE>
struct SrcF64 {
    const double* src[NCOMP];
    __device__ __forceinline__ void load(int n, double (&ua)[NCOMP], double (&ub)[NCOMP]) const {
#pragma unroll
        for (int k = 0; k < NCOMP; ++k) {
            ua[k] = src[k][n * STRIDE];
            ub[k] = src[k][(n + 1) * STRIDE];
        }
    }
};

// Writes updated cell j to dst[k] + (j - J0) * STRIDE (in place in shared memory: J0 = 0; to `out`: J0 = NG).
template <int STRIDE, int J0>
struct SinkF64 {
    double* dst[NCOMP];
    template <int ODD>
    __device__ __forceinline__ void cell(int j, const double (&u)[NCOMP]) {
#pragma unroll
        for (int k = 0; k < NCOMP; ++k) dst[k][(j - J0) * STRIDE] = u[k];
    }
    __device__ __forceinline__ void face(int, const double (&)[NCOMP]) {}
};

template <int STRIDE, int J0>
__device__ __forceinline__ void march_f64(double* const (&row)[NCOMP], double* const (&dst)[NCOMP],
                                          const GasConstT<double>& gc) {
    SrcF64<STRIDE> src;
    SinkF64<STRIDE, J0> sink;
#pragma unroll
    for (int k = 0; k < NCOMP; ++k) {
        src.src[k] = row[k];
        sink.dst[k] = dst[k];
    }
    NoGate gate;
    RowMarch<false, decltype(sink), double> m;
    m.run(src, gc, sink, gate);
}

__global__ void __launch_bounds__(F64_THREADS, 1)
hydro_advance_f64_kernel(const double* __restrict__ in, double* __restrict__ out, long long n_groups,
                         GasConstT<double> gc, double* __restrict__ scratch) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    double* buf = reinterpret_cast<double*>(smem_raw);
    uint64_t* bar = reinterpret_cast<uint64_t*>(smem_raw + F64_DATA_BYTES);
    double* zblock = scratch + (long long)blockIdx.x * F64_SCRATCH_DOUBLES;
    const int t = threadIdx.x;
    if (t == 0) {
        mbar_init(bar, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    uint32_t parity = 0;
    for (long long g = blockIdx.x; g < n_groups; g += gridDim.x) {
        const double* in_g = in + g * (long long)GROUP_IN_FLOATS;
        for (int h = 0; h < 2; ++h) {
            // ---- planes 11h .. 11h+10 of all variables into shared memory --------------------------------------
            if (t == 0) {
                fence_proxy_async();
                mbar_expect_tx(bar, NCOMP * HALF_VAR * 8);
                for (int v = 0; v < NCOMP; ++v)
                    bulk_g2s(buf + v * HALF_VAR, in_g + v * VAR_FLOATS + h * HALF_VAR, HALF_VAR * 8, bar);
            }
            mbar_wait_poll(bar, parity);
            parity ^= 1u;
            // ---- x sweep: 11 x 22 rows (y,z), in place --------------------------------------------------------
            if (t < HALF_PLANES * NP) {
                double* row[NCOMP];
#pragma unroll
                for (int q = 0; q < NCOMP; ++q) row[q] = buf + var_of(0, q) * HALF_VAR + t * NP;
                march_f64<1, 0>(row, row, gc);
            }
            __syncthreads();
            // ---- y sweep: x = 3..18, 11 planes, in place -------------------------------------------------------
            if (t < HALF_PLANES * PS) {
                const int x = NG + (t & 15), z = t >> 4;
                double* row[NCOMP];
#pragma unroll
                for (int q = 0; q < NCOMP; ++q) row[q] = buf + var_of(1, q) * HALF_VAR + z * (NP * NP) + x;
                march_f64<NP, 0>(row, row, gc);
            }
            __syncthreads();
            // ---- the 16 x 16 interior columns of these planes -> scratch block [v][z][j][i] ---------------------
            for (int i = t; i < NCOMP * HALF_PLANES * PS * PS; i += F64_THREADS) {
                const int x = i & 15, y = (i >> 4) & 15, zv = i >> 8, z = zv % HALF_PLANES, v = zv / HALF_PLANES;
                zblock[v * ZBUF_VAR + (h * HALF_PLANES + z) * (PS * PS) + y * PS + x] =
                    buf[v * HALF_VAR + z * (NP * NP) + (y + NG) * NP + x + NG];
            }
            __syncthreads();
        }
        // ---- z sweep on the block (read back through the generic proxy: written by this CTA before the barrier) ----
        for (int i = t; i < FWD_SCRATCH_DOUBLES / 2; i += F64_THREADS)
            reinterpret_cast<double2*>(buf)[i] = reinterpret_cast<const double2*>(zblock)[i];
        __syncthreads();
        {
            const int x = t & 15, y = t >> 4;
            double* row[NCOMP];
            double* dst[NCOMP];
            double* out_g = out + g * (long long)GROUP_OUT_FLOATS;
#pragma unroll
            for (int q = 0; q < NCOMP; ++q) {
                row[q] = buf + var_of(2, q) * ZBUF_VAR + y * PS + x;
                dst[q] = out_g + var_of(2, q) * (PS * PS * PS) + y * PS + x;
            }
            march_f64<PS * PS, NG>(row, dst, gc);
        }
        __syncthreads();
    }
}

// Backward (z,y,x) order.  The z sweep comes first and couples all planes, but its rows are independent: it runs on
// two halves of 11 y rows (all x, all 22 planes: 212 960 B each); the 16 z-swept interior planes pass through the
// scratch block; the y and x sweeps act inside a plane and run on two chunks of 8 planes (154 880 B), the x sweep
// writing the interior to HBM.
__global__ void __launch_bounds__(F64_THREADS, 1)
hydro_advance_f64_backward_kernel(const double* __restrict__ in, double* __restrict__ out, long long n_groups,
                                  GasConstT<double> gc, double* __restrict__ scratch) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    double* buf = reinterpret_cast<double*>(smem_raw);
    double* zplanes = scratch + (long long)blockIdx.x * F64_SCRATCH_DOUBLES;     // [v][k = 0..15][y][x]
    const int t = threadIdx.x;
    constexpr int HROWS = HALF_PLANES * NP;          // 242 (y,x) positions of a half
    for (long long g = blockIdx.x; g < n_groups; g += gridDim.x) {
        const double* in_g = in + g * (long long)GROUP_IN_FLOATS;
        for (int h = 0; h < 2; ++h) {
            // ---- rows y = 11h .. 11h+10 of every plane: buf[v][z][yy][x] ---------------------------------------
            for (int i = t; i < NCOMP * NP * HROWS; i += F64_THREADS) {
                const int r = i % HROWS, vz = i / HROWS;                          // vz = v * 22 + z
                buf[i] = in_g[vz * (NP * NP) + h * HROWS + r];
            }
            __syncthreads();
            // ---- z sweep: 242 rows (y,x), stride 242, in place -------------------------------------------------
            if (t < HROWS) {
                double* row[NCOMP];
#pragma unroll
                for (int q = 0; q < NCOMP; ++q) row[q] = buf + var_of(2, q) * (NP * HROWS) + t;
                march_f64<HROWS, 0>(row, row, gc);
            }
            __syncthreads();
            // ---- the 16 interior planes of this half -> scratch -------------------------------------------------
            for (int i = t; i < NCOMP * PS * HROWS; i += F64_THREADS) {
                const int r = i % HROWS, vk = i / HROWS, k = vk % PS, v = vk / PS;
                zplanes[v * BWD_VAR + k * (NP * NP) + h * HROWS + r] = buf[(v * NP + k + NG) * HROWS + r];
            }
            __syncthreads();
        }
        for (int c = 0; c < PS / BWD_CHUNK_PLANES; ++c) {
            // ---- planes k = 8c .. 8c+7 back from scratch: buf[v][kk][y][x] --------------------------------------
            for (int i = t; i < NCOMP * BWD_CHUNK_VAR / 2; i += F64_THREADS) {
                const int v = i / (BWD_CHUNK_VAR / 2), r = i % (BWD_CHUNK_VAR / 2);
                reinterpret_cast<double2*>(buf)[i] =
                    reinterpret_cast<const double2*>(zplanes + v * BWD_VAR + c * BWD_CHUNK_VAR)[r];
            }
            __syncthreads();
            // ---- y sweep: all 22 x, 8 planes, in place ----------------------------------------------------------
            if (t < BWD_CHUNK_PLANES * NP) {
                const int x = t % NP, kk = t / NP;
                double* row[NCOMP];
#pragma unroll
                for (int q = 0; q < NCOMP; ++q) row[q] = buf + var_of(1, q) * BWD_CHUNK_VAR + kk * (NP * NP) + x;
                march_f64<NP, 0>(row, row, gc);
            }
            __syncthreads();
            // ---- x sweep: y = 3..18, 8 planes, results straight to HBM ------------------------------------------
            if (t < BWD_CHUNK_PLANES * PS) {
                const int y = NG + (t & 15), kk = t >> 4;
                double* row[NCOMP];
                double* dst[NCOMP];
                double* out_g = out + g * (long long)GROUP_OUT_FLOATS;
#pragma unroll
                for (int q = 0; q < NCOMP; ++q) {
                    row[q] = buf + var_of(0, q) * BWD_CHUNK_VAR + kk * (NP * NP) + y * NP;
                    dst[q] = out_g + var_of(0, q) * (PS * PS * PS) + (c * BWD_CHUNK_PLANES + kk) * (PS * PS) + (y - NG) * PS;
                }
                march_f64<1, NG>(row, dst, gc);
            }
            __syncthreads();
        }
    }
}

}  // namespace gamer
