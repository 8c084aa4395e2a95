// uniform_grid.cuh — device-side "preparation step" for a single-level tiling of patch groups, and the CFL time step.
//
// PAPER.md:322 (§3.1): before a solver call the ghost zones of every patch group are filled, on a uniform level by
// copying from the sibling patches.  PAPER.md:430-432, :647 name this CPU step the bottleneck of the whole code; here
// it is one memory-bound kernel on the device, so that a multi-step run never leaves HBM.
// PAPER.md:418-426 (§3.4, Eq.30): dt = C dh / max (c_s + max_i |v_i|).
#pragma once
#include <cuda_runtime.h>

#include "hydro_kernel.cuh"

namespace gamer {

struct BoxGeom {
    int gx, gy, gz;          // groups along x, y, z; group index g = (kz * gy + ky) * gx + kx
    int bc[3];               // per axis x, y, z: 0 = periodic, 1 = leave the ghost cells beyond the box untouched
    int nseg;                // ghost fill only: segments the walk along x is cut into (ghost_fill_segments)
};

// One CTA per (strip of groups along x, variable): the CTA walks kx = 0 .. gx-1 and assembles the 22^3 padded cells of
// one group and variable at a time in shared memory, then hands the contiguous, 16-byte-aligned 42 592-byte block to one
// bulk store (TMA), so that the LSU pipe only sees the gather side.
//   * Every global read is a 128-bit load of an aligned quarter of a 16-cell interior row (thread = (padded row, quarter);
//     rows whose y or z lies beyond the box come from the y/z neighbours, periodic, or are re-read from the padded array
//     itself, "keep").
//   * The ghost cells x = 0..2 of group kx are cells 13..15 of the same rows of group kx-1 and x = 19..21 are cells 0..2
//     of group kx+1: the threads that loaded those quarters one step earlier / later write them, so no separate load
//     of the x neighbours exists (the first version spent a quarter of its time on those 12-byte reads).  The walk
//     therefore runs from kx = -1 (wrap: only remembered) to kx = gx (wrap: only its first quarters are used), and two
//     tiles are in flight: tile kx is being filled while tile kx-1 receives its last ghost cells and leaves.
//   * A thin box (few strips: a Sod column has gy = gz = 1, so 5 CTAs) would leave most SMs idle: the walk is then cut
//     into nseg segments [x0, x1) of the strip, one CTA each, until there are about two CTAs per SM.  A segment starts
//     one group early and ends one group late like the whole walk does, at the cost of one extra quarter-row load at
//     each segment end.
constexpr int GF_THREADS = 256;
constexpr int GF_BAND = 8;                                        // z layers per band of strips (CTA numbering)
constexpr int GF_ROWS = NP * NP;                                  // 484 padded (z,y) rows
constexpr int GF_ITEMS = (GF_ROWS * 4 + GF_THREADS - 1) / GF_THREADS;   // 8 quarter rows per thread (the last one partial)
constexpr int GF_SMEM_BYTES = 2 * VAR_FLOATS * 4 + 2 * NP * 8;    // two tiles + the y and z offset tables
// segments per strip: 1 when the strips alone give two CTAs per SM, else as many as that takes (at most gx)
inline int ghost_fill_segments(int gx, int gy, int gz, int sm_count) {
    const long long strips = (long long)gy * gz * NCOMP, want = 2ll * sm_count;
    if (strips >= want) return 1;
    const long long nseg = (want + strips - 1) / strips;
    return (int)(nseg < gx ? nseg : gx);
}
// number of CTAs that ghost_fill_kernel needs for a box of gx x gy x gz groups cut into nseg segments along x
inline long long ghost_fill_ctas(int gx, int gy, int gz, int nseg = 1) { (void)gx; return (long long)gy * gz * NCOMP * nseg; }

// SEGMENTED = false is the whole-strip walk (nseg == 1) with its bounds known at compile time: the code of round 2.
template <bool SEGMENTED>
__global__ void __launch_bounds__(GF_THREADS, 2)
ghost_fill_kernel(const float* __restrict__ interior, float* __restrict__ padded, BoxGeom geo) {
    extern __shared__ __align__(128) unsigned char gf_smem[];
    float* const tiles = reinterpret_cast<float*>(gf_smem);                       // [2][VAR_FLOATS]
    long long* const off_y = reinterpret_cast<long long*>(gf_smem + 2 * VAR_FLOATS * 4);
    long long* const off_z = off_y + NP;
    const int v = blockIdx.x % NCOMP;
    const int strips = geo.gy * geo.gz;
    const int strip = SEGMENTED ? (blockIdx.x / NCOMP) % strips : blockIdx.x / NCOMP;
    const int seg = SEGMENTED ? blockIdx.x / (NCOMP * strips) : 0;
    // Strips are numbered in bands of GF_BAND z layers, z fastest inside a band: the ~60 strips that are resident at
    // the same time (2 CTAs per SM, 5 variables per strip) then form a block of about 7 x 8 in (ky, kz) that walks
    // along x together, so that most y AND z neighbour rows a strip reads were just read by the strip that owns them
    // and come from L2 instead of DRAM.  (All bands before the last are full, so band = strip / (GF_BAND * gy).)
    const int band = strip / (GF_BAND * geo.gy), in_band = strip - band * (GF_BAND * geo.gy);
    const int band_h = min(GF_BAND, geo.gz - band * GF_BAND);
    const int ky = in_band / band_h, kz = band * GF_BAND + in_band % band_h;
    const int x0 = SEGMENTED ? (int)((long long)seg * geo.gx / geo.nseg) : 0;
    const int x1 = SEGMENTED ? (int)((long long)(seg + 1) * geo.gx / geo.nseg) : geo.gx;
    // Per padded y and z: offset (in floats) of the source row inside `interior`, or -1 = beyond a "keep" end.
    constexpr long long GS = (long long)NCOMP * PS * PS * PS;     // floats per group of `interior`
    if (threadIdx.x < 2 * NP) {
        const bool is_z = threadIdx.x >= NP;
        const int p = threadIdx.x - (is_z ? NP : 0);
        const int k = is_z ? kz : ky, nk = is_z ? geo.gz : geo.gy, keep_flag = is_z ? geo.bc[2] : geo.bc[1];
        int c = p - NG, sk = k;
        bool keep = false;
        if (c < 0) { c += PS; sk = k > 0 ? k - 1 : nk - 1; keep = (k == 0 && keep_flag); }
        else if (c >= PS) { c -= PS; sk = k < nk - 1 ? k + 1 : 0; keep = (k == nk - 1 && keep_flag); }
        const long long off = is_z ? ((long long)sk * geo.gy * geo.gx) * GS + c * (PS * PS)
                                   : ((long long)sk * geo.gx) * GS + c * PS;
        (is_z ? off_z : off_y)[p] = keep ? -1 : off;
    }
    __syncthreads();
    const int part = threadIdx.x & 3;                              // quarter of the 16-cell row, the same for all items
    const float* const src_v = interior + v * (PS * PS * PS) + 4 * part;
    long long row_off[GF_ITEMS];                                   // source offset of this thread's rows, -1 = keep
#pragma unroll
    for (int k = 0; k < GF_ITEMS; ++k) {
        const int row = (threadIdx.x >> 2) + (GF_THREADS / 4) * k;
        row_off[k] = -1;
        if (row < GF_ROWS) {
            const int z = row / NP, y = row - z * NP;
            const long long oy = off_y[y], oz = off_z[z];
            row_off[k] = (oy >= 0 && oz >= 0) ? oy + oz : -1;
        }
    }
    const long long g0 = ((long long)kz * geo.gy + ky) * geo.gx;  // group index of kx = 0 in this strip
    float4 prev[GF_ITEMS];                                         // the quarters loaded one step earlier (group kx-1)
    for (int kx = x0 - 1; kx <= x1; ++kx) {
        const int ks = kx < 0 ? geo.gx - 1 : (kx == geo.gx ? 0 : kx);          // group whose interior is read (wrap)
        const bool fill = kx >= x0 && kx < x1;                                   // tile kx exists (in this segment)
        const bool wrap_l = kx == 0 && geo.bc[0], wrap_r = kx == geo.gx && geo.bc[0];   // "keep" ends along x
        float* const tile = tiles + (kx & 1) * VAR_FLOATS;                      // tile of group kx
        float* const tprev = tiles + ((kx + 1) & 1) * VAR_FLOATS;               // tile of group kx-1
        float* const dst = padded + ((g0 + (fill ? kx : x0)) * NCOMP + v) * (long long)VAR_FLOATS;
        float* const dprev = padded + ((g0 + (kx > x0 ? kx - 1 : x0)) * NCOMP + v) * (long long)VAR_FLOATS;
        // the bulk store that last read `tile` (group kx-2) must have finished reading before anybody writes to it
        if (threadIdx.x == 0) asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
        __syncthreads();
        const float* const src = src_v + ks * GS;
        float4 q[GF_ITEMS];
        // only the quarters that are used are loaded: all of them for a tile, the first / last ones at the two wraps
        const bool need = fill || (kx < x0 && part == 3) || (kx == x1 && part == 0);
#pragma unroll
        for (int k = 0; k < GF_ITEMS; ++k) {
            const int row = (threadIdx.x >> 2) + (GF_THREADS / 4) * k;
            q[k] = make_float4(0.f, 0.f, 0.f, 0.f);
            if (row < GF_ROWS && need && row_off[k] >= 0) q[k] = __ldg(reinterpret_cast<const float4*>(src + row_off[k]));
        }
#pragma unroll
        for (int k = 0; k < GF_ITEMS; ++k) {
            const int row = (threadIdx.x >> 2) + (GF_THREADS / 4) * k;
            if (row < GF_ROWS) {
                const bool keep_row = row_off[k] < 0;              // y or z beyond a "keep" end: the whole row is kept
                if (fill) {
                    float* o = tile + row * NP + NG + 4 * part;
                    if (keep_row) {
                        const float* e = dst + row * NP + NG + 4 * part;
                        q[k] = make_float4(e[0], e[1], e[2], e[3]);
                    }
                    o[0] = q[k].x; o[1] = q[k].y; o[2] = q[k].z; o[3] = q[k].w;
                    if (part == 3) {                               // ghost cells x = 0..2: cells 13..15 of group kx-1
                        float* l = tile + row * NP;
                        if (keep_row || wrap_l) {
                            const float* e = dst + row * NP;
                            l[0] = e[0]; l[1] = e[1]; l[2] = e[2];
                        } else {
                            l[0] = prev[k].y; l[1] = prev[k].z; l[2] = prev[k].w;
                        }
                    }
                }
                if (kx > x0 && part == 0) {                        // ghost cells x = 19..21 of group kx-1: cells 0..2 here
                    float* r = tprev + row * NP + NG + PS;
                    if (keep_row || wrap_r) {
                        const float* e = dprev + row * NP + NG + PS;
                        r[0] = e[0]; r[1] = e[1]; r[2] = e[2];
                    } else {
                        r[0] = q[k].x; r[1] = q[k].y; r[2] = q[k].z;
                    }
                }
            }
            prev[k] = q[k];
        }
        // tile kx-1 is complete: make the generic-proxy writes visible to the async proxy and let it go
        fence_proxy_async();
        __syncthreads();
        if (threadIdx.x == 0 && kx > x0) {
            asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(dprev), "r"(smem_u32(tprev)),
                         "r"(VAR_FLOATS * 4)
                         : "memory");
            asm volatile("cp.async.bulk.commit_group;" ::: "memory");
        }
    }
    if (threadIdx.x == 0) asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");   // the tiles must outlive the reads
}

// max of c_s + max(|v_x|,|v_y|,|v_z|) (Eq.30) as the bit pattern of a non-negative float in *acc (atomicMax on
// unsigned: positive floats order like their bit patterns).  keep_only = 0: over ALL padded cells of all groups
// (reading R10); keep_only = 1: only over the ghost cells beyond a "keep" end of the box, which no ghost
// fill ever changes.
__global__ void __launch_bounds__(256)
max_speed_kernel(const float* __restrict__ padded, long long n_groups, float gamma, unsigned int* __restrict__ acc,
                 BoxGeom geo, int keep_only) {
    float best = 0.f;
    const float ggm1 = gamma * (gamma - 1.0f);
    for (long long g = blockIdx.x; g < n_groups; g += gridDim.x) {
        const float* u = padded + g * (long long)GROUP_IN_FLOATS;
        const int kx = (int)(g % geo.gx), ky = (int)((g / geo.gx) % geo.gy), kz = (int)(g / ((long long)geo.gx * geo.gy));
        // per axis: padded indices below lo or from hi on lie beyond a "keep" end (lo = 0, hi = NP: none)
        const int lox = geo.bc[0] && kx == 0 ? NG : 0, hix = geo.bc[0] && kx == geo.gx - 1 ? NG + PS : NP;
        const int loy = geo.bc[1] && ky == 0 ? NG : 0, hiy = geo.bc[1] && ky == geo.gy - 1 ? NG + PS : NP;
        const int loz = geo.bc[2] && kz == 0 ? NG : 0, hiz = geo.bc[2] && kz == geo.gz - 1 ? NG + PS : NP;
        if (keep_only && lox == 0 && hix == NP && loy == 0 && hiy == NP && loz == 0 && hiz == NP) continue;
        for (int i = threadIdx.x; i < VAR_FLOATS; i += blockDim.x) {
            if (keep_only) {
                const int x = i % NP, y = (i / NP) % NP, z = i / (NP * NP);
                if (x >= lox && x < hix && y >= loy && y < hiy && z >= loz && z < hiz) continue;
            }
            const float rho = u[i], mx = u[VAR_FLOATS + i], my = u[2 * VAR_FLOATS + i], mz = u[3 * VAR_FLOATS + i],
                        e = u[4 * VAR_FLOATS + i];
            const float rinv = 1.0f / rho;
            const float eint = e - 0.5f * (mx * mx + my * my + mz * mz) * rinv;
            const float cs = sqrtf(ggm1 * eint * rinv);
            const float vm = fmaxf(fmaxf(fabsf(mx), fabsf(my)), fabsf(mz)) * rinv;
            best = fmaxf(best, cs + vm);
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) best = fmaxf(best, __shfl_xor_sync(0xffffffffu, best, o));
    if ((threadIdx.x & 31) == 0) atomicMax(acc, __float_as_uint(best));
}

// max over the per-group CFL speeds that the hydro kernel wrote (its fused NEXT-1 output) into *acc.
__global__ void __launch_bounds__(256)
group_speed_max_kernel(const float* __restrict__ group_speed, long long n_groups, unsigned int* __restrict__ acc) {
    float best = 0.f;
    for (long long g = blockIdx.x * (long long)blockDim.x + threadIdx.x; g < n_groups; g += (long long)gridDim.x * blockDim.x)
        best = fmaxf(best, group_speed[g]);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) best = fmaxf(best, __shfl_xor_sync(0xffffffffu, best, o));
    if ((threadIdx.x & 31) == 0) atomicMax(acc, __float_as_uint(best));
}

// dt = cfl dh / speed.  work[0]: speed accumulator (bits), work[1]: dt, work[2]: speed of the kept ghost cells (bits),
// with which the accumulator starts the next step.
__global__ void cfl_dt_kernel(float* __restrict__ work, float cfl, float dh, float* __restrict__ dt_log) {
    unsigned int* w = reinterpret_cast<unsigned int*>(work);
    const float dt = cfl * dh / __uint_as_float(w[0]);
    work[1] = dt;
    if (dt_log) *dt_log = dt;
    w[0] = w[2];
}

}  // namespace gamer
