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
constexpr int F64_SCRATCH_DOUBLES = NCOMP * ZBUF_VAR;                // 28 160 per CTA
constexpr int F64_DATA_BYTES = F64_SCRATCH_DOUBLES * 8;              // 225 280 (>= 5 * 5324 * 8 = 212 960)
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
        for (int i = t; i < F64_SCRATCH_DOUBLES / 2; i += F64_THREADS)
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

}  // namespace gamer
