// hydro_kernel_f64.cuh — double-precision variant of the forward pass (NEXT-4; "single precision is
// assumed unless ... explicitly stated", double precision for the convergence tests).
//
// Same row march as the fp32 kernel (rtvd_march.cuh, T = double).  A padded group in fp64 is 425 920 B and does not fit
// in shared memory, so the pass is cut where the method allows it: the x and y sweeps act inside one z-plane
// (PAPER.md:174-178), so they run on two halves of 11 planes (212 960 B each, bulk-copied by TMA); what the z sweep
// needs of their result — the 16 x 16 interior columns of all 22 planes, 225 280 B — is parked in TENSOR MEMORY: a z
// row (22 cells x 5 variables x 2 words = 220 words) belongs to one thread from the moment the y sweep has produced it,
// and tcgen05.ld/st move 32-bit words between a thread's registers and "its" TMEM lane (512 columns per lane, two z
// warps per lane quadrant: 2 x 220 columns).  After the y sweep of a half every z thread copies its 11 planes' cells
// from shared memory into its lane; the z march then reads its row from there and writes the interior straight to HBM.
// Shared memory is free during the z sweep, so the first half of the CTA's next group is loaded under it.  One
// persistent CTA per SM, 256 threads (up to 255 registers: the march state is twice as wide in fp64).  Traffic per
// group: 425 920 B in + 163 840 B out.  (Round 1 passed the z block through a scratch block in device memory and read
// it back: 403 ns/group.)
#pragma once
#include <cstdint>

#include "hydro_kernel.cuh"
#include "tmem_rows.cuh"

#ifndef GAMER_F64_PREFETCH
#define GAMER_F64_PREFETCH 1
#endif

namespace gamer {

constexpr int F64_THREADS = 256;
constexpr int HALF_PLANES = NP / 2;                                  // 11
constexpr int HALF_VAR = HALF_PLANES * NP * NP;                      // 5324 doubles: one variable of a half
constexpr int ZBUF_VAR = NP * PS * PS;                               // 5632 doubles: one variable of the z-sweep block
constexpr int F64_DATA_BYTES = NCOMP * ZBUF_VAR * 8;                 // 225 280 (>= 5 * 5324 * 8 = 212 960)
constexpr int F64_SMEM_BYTES = F64_DATA_BYTES + 128;     // + mbarrier, TMEM base address, 8 doubles of reduction scratch


constexpr int ZROW_WORDS_PER_PLANE = 2 * NCOMP;                      // 10 columns: one cell, five doubles
constexpr int ZROW_COLS = NP * ZROW_WORDS_PER_PLANE;                 // 220 columns per z row
constexpr int ZROW_COL_STRIDE = 256;                                 // second z warp of a lane quadrant

// Row source of the z march: this thread's row in tensor memory, [plane][row-local component][lo, hi].
struct TmemRowSrc {
    uint32_t taddr;                                                  // lane quadrant and first column of the row
    __device__ __forceinline__ void load(int n, double (&ua)[NCOMP], double (&ub)[NCOMP]) const {
        uint32_t a[16], b[4];
        tmem_ld16(taddr + n * ZROW_WORDS_PER_PLANE, a);
        tmem_ld4(taddr + n * ZROW_WORDS_PER_PLANE + 16, b);
        tmem_wait_ld();
#pragma unroll
        for (int k = 0; k < NCOMP; ++k) ua[k] = __hiloint2double((int)a[2 * k + 1], (int)a[2 * k]);
#pragma unroll
        for (int k = 0; k < 3; ++k) ub[k] = __hiloint2double((int)a[10 + 2 * k + 1], (int)a[10 + 2 * k]);
        ub[3] = __hiloint2double((int)b[1], (int)b[0]);
        ub[4] = __hiloint2double((int)b[3], (int)b[2]);
    }
};

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
// WANT_FACE: the time-centred fluxes through the three patch-boundary planes go to fptr[k] + p * 5 * 256 if this row is
// an interior one (the layout of gamer_hydro.h: face_flux[g][d][p][v][b][a]).  WANT_SPEED: Eq.30 on
// every updated cell of the last sweep, running maximum in `speed`.
template <int STRIDE, int J0, bool WANT_FACE = false, bool WANT_SPEED = false>
struct SinkF64 {
    double* dst[NCOMP];
    double* fptr[WANT_FACE ? NCOMP : 1];
    bool face_row;
    double ggm1, speed;
    template <int ODD>
    __device__ __forceinline__ void cell(int j, const double (&u)[NCOMP]) {
#pragma unroll
        for (int k = 0; k < NCOMP; ++k) dst[k][(j - J0) * STRIDE] = u[k];
        if (WANT_SPEED) {
            const double rinv = rcp_fast(u[0]);
            double q = u[2] * u[2];
            q = fma(u[3], u[3], q);
            q = fma(u[1], u[1], q);
            const double eint = fma(-q, 0.5 * rinv, u[4]);
            const double cs = sqrt_fast((ggm1 * eint) * rinv);
            const double vm = fmax(fmax(fabs(u[1]), fabs(u[2])), fabs(u[3])) * rinv;
            speed = fmax(speed, cs + vm);
        }
    }
    __device__ __forceinline__ void face(int p, const double (&f)[NCOMP]) {
        if (WANT_FACE && face_row) {
#pragma unroll
            for (int k = 0; k < NCOMP; ++k) fptr[WANT_FACE ? k : 0][p * (NCOMP * PS * PS)] = f[k];
        }
    }
};

// &face_flux[g][D][0][var(q)][b][a] for row-local component q of a sweep along D (b, a: interior transverse indices)
template <int D>
__device__ __forceinline__ double* face_ptr(double* face_g, int q, int b, int a) {
    return face_g + ((D * 3) * NCOMP + var_of(D, q)) * (PS * PS) + b * PS + a;
}

// In-place (or to `dst`) march of one row; D = sweep axis, (b, a) = interior transverse indices of the row for the face
// fluxes (any value if face_g is NULL or the row is not an interior one: face_row = false).
template <int STRIDE, int J0, int D, bool WANT_FACE>
__device__ __forceinline__ void march_f64(double* const (&row)[NCOMP], double* const (&dst)[NCOMP],
                                          const GasConstT<double>& gc, double* face_g, bool face_row, int b, int a) {
    SrcF64<STRIDE> src;
    SinkF64<STRIDE, J0, WANT_FACE, false> sink;
#pragma unroll
    for (int k = 0; k < NCOMP; ++k) {
        src.src[k] = row[k];
        sink.dst[k] = dst[k];
        if (WANT_FACE) sink.fptr[k] = face_ptr<D>(face_g, k, b, a);
    }
    sink.face_row = WANT_FACE && face_row && face_g != nullptr;
    NoGate gate;
    RowMarch<WANT_FACE, decltype(sink), double> m;
    m.run(src, gc, sink, gate);
}

// Block maximum of the per-thread CFL speeds -> *dst (one double per group).  `red`: 8 doubles of shared memory.
__device__ __forceinline__ void block_max_f64(double v, double* red, double* dst) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = v;
    __syncthreads();
    if (threadIdx.x == 0) {
        double m = red[0];
        for (int w = 1; w < F64_THREADS / 32; ++w) m = fmax(m, red[w]);
        *dst = m;
    }
}

// WANT_OPT: the optional outputs of gamer_hydro_advance_f64_ex (either pointer may still be NULL): face_flux
// [g][3][3][5][16][16] and group_maxspeed[g], as in the fp32 kernel.
template <bool WANT_OPT>
__global__ void __launch_bounds__(F64_THREADS, 1)
hydro_advance_f64_kernel(const double* __restrict__ in, double* __restrict__ out, long long n_groups,
                         GasConstT<double> gc, double* __restrict__ face_flux, double* __restrict__ group_maxspeed) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    double* buf = reinterpret_cast<double*>(smem_raw);
    uint64_t* bar = reinterpret_cast<uint64_t*>(smem_raw + F64_DATA_BYTES);
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(smem_raw + F64_DATA_BYTES + 16);
    const int t = threadIdx.x, warp = t >> 5;
    if (warp == 0) tmem_alloc_all(tmem_slot);
    if (t == 0) {
        mbar_init(bar, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        // first half of the first group
        fence_proxy_async();
        const double* in_g = in + (long long)blockIdx.x * GROUP_IN_FLOATS;
        mbar_expect_tx(bar, NCOMP * HALF_VAR * 8);
        for (int v = 0; v < NCOMP; ++v) bulk_g2s(buf + v * HALF_VAR, in_g + v * VAR_FLOATS, HALF_VAR * 8, bar);
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const uint32_t tmem_base = *tmem_slot;
    // this thread's z row (x = t & 15, y = t >> 4): lane quadrant warp % 4, lane = lane id, columns by warp / 4
    const uint32_t zrow = tmem_base + ((uint32_t)(32 * (warp & 3)) << 16) + (uint32_t)((warp >> 2) * ZROW_COL_STRIDE);
    uint32_t parity = 0;
    for (long long g = blockIdx.x; g < n_groups; g += gridDim.x) {
        const double* in_g = in + g * (long long)GROUP_IN_FLOATS;
        const long long gn = g + gridDim.x;
        double* face_g = WANT_OPT && face_flux != nullptr ? face_flux + g * (long long)GROUP_FACE_FLOATS : nullptr;
        for (int h = 0; h < 2; ++h) {
            // ---- planes 11h .. 11h+10 of all variables are on their way into shared memory (issued earlier) -------
#if GAMER_F64_PREFETCH
            if (t == F64_THREADS - 1 && h == 0)          // the other half into L2 meanwhile (a thread without x rows)
                for (int v = 0; v < NCOMP; ++v) bulk_prefetch_l2(in_g + v * VAR_FLOATS + HALF_VAR, HALF_VAR * 8);
#endif
            mbar_wait_poll(bar, parity);
            parity ^= 1u;
            // ---- x sweep: 11 x 22 rows (y,z), in place --------------------------------------------------------
            if (t < HALF_PLANES * NP) {
                double* row[NCOMP];
#pragma unroll
                for (int q = 0; q < NCOMP; ++q) row[q] = buf + var_of(0, q) * HALF_VAR + t * NP;
                const int y = t % NP, z = h * HALF_PLANES + t / NP;
                march_f64<1, 0, 0, WANT_OPT>(row, row, gc, face_g, y >= NG && y < NG + PS && z >= NG && z < NG + PS, z - NG,
                                             y - NG);
            }
            __syncthreads();
            // ---- y sweep: x = 3..18, 11 planes, in place -------------------------------------------------------
            if (t < HALF_PLANES * PS) {
                const int x = NG + (t & 15), z = t >> 4;
                double* row[NCOMP];
#pragma unroll
                for (int q = 0; q < NCOMP; ++q) row[q] = buf + var_of(1, q) * HALF_VAR + z * (NP * NP) + x;
                const int zz = h * HALF_PLANES + z;
                march_f64<NP, 0, 1, WANT_OPT>(row, row, gc, face_g, zz >= NG && zz < NG + PS, zz - NG, x - NG);
            }
            __syncthreads();
            // ---- every z thread parks the cells of its column in these planes in tensor memory -------------------
            {
                const int x = t & 15, y = t >> 4;
                const double* col = buf + (y + NG) * NP + x + NG;
                uint32_t w[HALF_PLANES * ZROW_WORDS_PER_PLANE];
#pragma unroll
                for (int z = 0; z < HALF_PLANES; ++z)
#pragma unroll
                    for (int q = 0; q < NCOMP; ++q) {
                        const double val = col[var_of(2, q) * HALF_VAR + z * (NP * NP)];
                        w[z * ZROW_WORDS_PER_PLANE + 2 * q] = (uint32_t)__double2loint(val);
                        w[z * ZROW_WORDS_PER_PLANE + 2 * q + 1] = (uint32_t)__double2hiint(val);
                    }
                tmem_st110(zrow + (uint32_t)(h * HALF_PLANES * ZROW_WORDS_PER_PLANE), w);
                tmem_wait_st();
            }
            __syncthreads();          // shared memory is free: the other half (or the next group's first half) may land
            if (t == 0) {
                const double* src = h == 0 ? in_g + HALF_VAR : (gn < n_groups ? in + gn * (long long)GROUP_IN_FLOATS : nullptr);
                if (src != nullptr) {
                    fence_proxy_async();
                    mbar_expect_tx(bar, NCOMP * HALF_VAR * 8);
                    for (int v = 0; v < NCOMP; ++v) bulk_g2s(buf + v * HALF_VAR, src + v * VAR_FLOATS, HALF_VAR * 8, bar);
                }
            }
        }
        // ---- z sweep from tensor memory, results straight to HBM (the next group's first half lands meanwhile) -----
        {
            const int x = t & 15, y = t >> 4;
            double* dst[NCOMP];
            double* out_g = out + g * (long long)GROUP_OUT_FLOATS;
#pragma unroll
            for (int q = 0; q < NCOMP; ++q) dst[q] = out_g + var_of(2, q) * (PS * PS * PS) + y * PS + x;
            TmemRowSrc src;
            src.taddr = zrow;
            SinkF64<PS * PS, NG, WANT_OPT, WANT_OPT> sink;
#pragma unroll
            for (int q = 0; q < NCOMP; ++q) {
                sink.dst[q] = dst[q];
                if (WANT_OPT) sink.fptr[q] = face_ptr<2>(face_g, q, y, x);
            }
            sink.face_row = face_g != nullptr;
            sink.ggm1 = gc.ggm1;
            sink.speed = 0.0;
            NoGate gate;
            RowMarch<WANT_OPT, decltype(sink), double> m;
            m.run(src, gc, sink, gate);
            if (WANT_OPT && group_maxspeed != nullptr) {
                block_max_f64(sink.speed, reinterpret_cast<double*>(smem_raw + F64_DATA_BYTES + 32) , group_maxspeed + g);
                __syncthreads();          // `red` is reused by the next group
            }
        }
        // no barrier: the next copy into tensor memory is by the same thread, after its own march
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (warp == 0) tmem_dealloc_all(tmem_base);
}

// Backward (z,y,x) order, the mirror image of the forward kernel with x and z exchanged.  The z and y sweeps do not
// couple different x, so they run on two SLABS of 11 x columns: the z march of a slab reads its rows straight from
// device memory (a warp reads runs of 11 consecutive doubles of a plane: the rows are independent and every plane is
// read exactly when the march gets there) and writes the 16 interior planes into shared memory, [v][k][y][xs]
// (154 880 B); the y sweep works there in place; then every x-row owner (y, k) parks the slab's 11 cells of its row in
// tensor memory (220 columns per row as in the forward kernel).  After both slabs the x march runs from tensor
// memory and writes the interior to HBM.  Thread 255, which has no row in the z sweep, prefetches the CTA's next group
// into L2.  (Before: strided loads of two y halves, a round trip of the z-swept planes through a scratch block in
// device memory, y and x sweeps on two chunks of 8 planes: 765 ns/group.)
constexpr int SLAB_X = NP / 2;                                       // 11 x columns per slab
constexpr int SLAB_PLANE = NP * SLAB_X;                              // 242 doubles: one z-swept plane of a slab
constexpr int SLAB_VAR = PS * SLAB_PLANE;                            // 3872 doubles: one variable of a slab

// Row source of the backward z march: this thread's column in device memory, plane stride NP * NP, fetched two pairs
// of cells ahead by cp.async (LDGSTS) into a private ring in shared memory — three slots of 2 cells x 5 variables per
// thread, 61 440 B behind the slab — so that the march never waits for device memory and needs no registers for it.
constexpr int XSTAGE_PITCH = PS + 1;                                 // 17
static_assert(NCOMP * PS * PS * XSTAGE_PITCH * 8 <= F64_DATA_BYTES, "x-sweep staging fits");
constexpr int RING_SLOTS = 3;
constexpr int RING_DOUBLES = RING_SLOTS * 2 * NCOMP * F64_THREADS;   // 7680
static_assert((NCOMP * SLAB_VAR + RING_DOUBLES) * 8 <= F64_DATA_BYTES, "slab + ring fit");
static_assert(SLAB_X * ZROW_WORDS_PER_PLANE == 110 && HALF_PLANES * ZROW_WORDS_PER_PLANE == 110, "tmem_st110");
struct RingColSrc {
    const double* src[NCOMP];
    double* ring;                                                    // &ring[0][0][0][t]
    __device__ __forceinline__ void fetch(int n) const {             // cells n, n+1 -> slot (n / 2) % 3
        double* slot = ring + ((n >> 1) % RING_SLOTS) * (2 * NCOMP * F64_THREADS);
#pragma unroll
        for (int c = 0; c < 2; ++c)
#pragma unroll
            for (int k = 0; k < NCOMP; ++k)
                asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(smem_u32(slot + (c * NCOMP + k) * F64_THREADS)),
                             "l"(src[k] + (n + c) * (NP * NP))
                             : "memory");
    }
    __device__ __forceinline__ void load(int n, double (&ua)[NCOMP], double (&ub)[NCOMP]) const {
        if (n == 0) {
            fetch(0);
            asm volatile("cp.async.commit_group;" ::: "memory");
            fetch(2);
            asm volatile("cp.async.commit_group;" ::: "memory");
        }
        if (n + 4 < NP) fetch(n + 4);
        asm volatile("cp.async.commit_group;" ::: "memory");         // possibly empty: keeps the group count uniform
        asm volatile("cp.async.wait_group 2;" ::: "memory");         // all but the two youngest groups: cells n, n+1 are here
        const double* slot = ring + ((n >> 1) % RING_SLOTS) * (2 * NCOMP * F64_THREADS);
#pragma unroll
        for (int k = 0; k < NCOMP; ++k) {
            ua[k] = slot[k * F64_THREADS];
            ub[k] = slot[(NCOMP + k) * F64_THREADS];
        }
    }
};

template <bool WANT_OPT>
__global__ void __launch_bounds__(F64_THREADS, 1)
hydro_advance_f64_backward_kernel(const double* __restrict__ in, double* __restrict__ out, long long n_groups,
                                  GasConstT<double> gc, double* __restrict__ face_flux,
                                  double* __restrict__ group_maxspeed) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    double* buf = reinterpret_cast<double*>(smem_raw);
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(smem_raw + F64_DATA_BYTES + 16);
    const int t = threadIdx.x, warp = t >> 5;
    if (warp == 0) tmem_alloc_all(tmem_slot);
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const uint32_t tmem_base = *tmem_slot;
    // this thread's x row (y = 3 + (t & 15), plane k = t >> 4): lane quadrant warp % 4, columns by warp / 4
    const uint32_t xrow = tmem_base + ((uint32_t)(32 * (warp & 3)) << 16) + (uint32_t)((warp >> 2) * ZROW_COL_STRIDE);
    for (long long g = blockIdx.x; g < n_groups; g += gridDim.x) {
        const double* in_g = in + g * (long long)GROUP_IN_FLOATS;
        const long long gn = g + gridDim.x;
        double* face_g = WANT_OPT && face_flux != nullptr ? face_flux + g * (long long)GROUP_FACE_FLOATS : nullptr;
        for (int s = 0; s < 2; ++s) {
            // ---- z sweep of the slab: 22 x 11 rows (y, xs), device memory -> shared memory (interior planes) ---------
            if (t < NP * SLAB_X) {
                const int y = t / SLAB_X, xs = t - y * SLAB_X;
                RingColSrc src;
                src.ring = buf + NCOMP * SLAB_VAR + t;
                SinkF64<SLAB_PLANE, NG, WANT_OPT, false> sink;
                const int x = s * SLAB_X + xs;
#pragma unroll
                for (int q = 0; q < NCOMP; ++q) {
                    src.src[q] = in_g + var_of(2, q) * VAR_FLOATS + y * NP + x;
                    sink.dst[q] = buf + var_of(2, q) * SLAB_VAR + t;
                    if (WANT_OPT) sink.fptr[q] = face_ptr<2>(face_g, q, y - NG, x - NG);
                }
                sink.face_row = face_g != nullptr && y >= NG && y < NG + PS && x >= NG && x < NG + PS;
                NoGate gate;
                RowMarch<WANT_OPT, decltype(sink), double> m;
                m.run(src, gc, sink, gate);
            } else if (t == F64_THREADS - 1 && s == 1 && gn < n_groups) {
                bulk_prefetch_l2(in + gn * (long long)GROUP_IN_FLOATS, GROUP_IN_FLOATS * 8);
            }
            __syncthreads();
            // ---- y sweep: 11 x columns x 16 planes, in place -------------------------------------------------------
            if (t < SLAB_X * PS) {
                const int k = t / SLAB_X, xs = t - k * SLAB_X;
                double* row[NCOMP];
#pragma unroll
                for (int q = 0; q < NCOMP; ++q) row[q] = buf + var_of(1, q) * SLAB_VAR + k * SLAB_PLANE + xs;
                const int x = s * SLAB_X + xs;
                march_f64<SLAB_X, 0, 1, WANT_OPT>(row, row, gc, face_g, x >= NG && x < NG + PS, k, x - NG);
            }
            __syncthreads();
            // ---- every x-row owner parks the slab's cells of its row in tensor memory ----------------------------------
            {
                const int yi = t & 15, k = t >> 4;
                const double* rowp = buf + k * SLAB_PLANE + (yi + NG) * SLAB_X;
                uint32_t w[SLAB_X * ZROW_WORDS_PER_PLANE];
#pragma unroll
                for (int xs = 0; xs < SLAB_X; ++xs)
#pragma unroll
                    for (int q = 0; q < NCOMP; ++q) {
                        const double val = rowp[var_of(0, q) * SLAB_VAR + xs];
                        w[xs * ZROW_WORDS_PER_PLANE + 2 * q] = (uint32_t)__double2loint(val);
                        w[xs * ZROW_WORDS_PER_PLANE + 2 * q + 1] = (uint32_t)__double2hiint(val);
                    }
                tmem_st110(xrow + (uint32_t)(s * SLAB_X * ZROW_WORDS_PER_PLANE), w);
                tmem_wait_st();
            }
            __syncthreads();          // the slab buffer is free again
        }
        // ---- x sweep from tensor memory.  A thread owns a whole output row, so stores straight from the march would
        // put the lanes of a warp 128 B apart (32 sectors per store: 20 k cycles of the SM's store path per group).  The
        // march writes into shared memory instead, transposed and padded — [v][k][i][y], pitch 17: conflict-free for the
        // writers (lanes = y) and for the readers (lanes = i) — and a coalesced copy-out follows.
        {
            const int yi = t & 15, k = t >> 4;
            TmemRowSrc src;
            src.taddr = xrow;
            SinkF64<XSTAGE_PITCH, NG, WANT_OPT, WANT_OPT> sink;
#pragma unroll
            for (int q = 0; q < NCOMP; ++q) {
                sink.dst[q] = buf + ((var_of(0, q) * PS + k) * PS) * XSTAGE_PITCH + yi;
                if (WANT_OPT) sink.fptr[q] = face_ptr<0>(face_g, q, k, yi);
            }
            sink.face_row = face_g != nullptr;
            sink.ggm1 = gc.ggm1;
            sink.speed = 0.0;
            NoGate gate;
            RowMarch<WANT_OPT, decltype(sink), double> m;
            m.run(src, gc, sink, gate);
            if (WANT_OPT && group_maxspeed != nullptr)
                block_max_f64(sink.speed, reinterpret_cast<double*>(smem_raw + F64_DATA_BYTES + 32), group_maxspeed + g);
        }
        __syncthreads();
        {
            double* out_g = out + g * (long long)GROUP_OUT_FLOATS;
#pragma unroll 8
            for (int idx = t; idx < GROUP_OUT_FLOATS; idx += F64_THREADS) {
                const int i = idx & 15, yi = (idx >> 4) & 15, vk = idx >> 8;
                out_g[idx] = buf[(vk * PS + i) * XSTAGE_PITCH + yi];
            }
        }
        __syncthreads();          // the next z sweep writes the same shared memory
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (warp == 0) tmem_dealloc_all(tmem_base);
}

}  // namespace gamer
