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
};

// One CTA per (group, variable).  The 22^3 padded cells of that variable are assembled in shared memory — per (z,y)
// row: the 16 interior cells as four 128-bit loads from the owning group's interior, 3 + 3 ghost cells from the x
// neighbours; rows whose y or z lies beyond the box come from the y/z neighbours (periodic) or are re-read from the
// padded array itself ("keep") — and then written out as one contiguous, 16-byte-aligned block with 128-bit stores.
constexpr int GF_THREADS = 256;
constexpr int GF_TILE = 4;
// number of CTAs that ghost_fill_kernel needs for a box of gx x gy x gz groups
inline long long ghost_fill_ctas(int gx, int gy, int gz) {
    auto up = [](int a) { return (long long)((a + GF_TILE - 1) / GF_TILE); };
    return up(gx) * up(gy) * up(gz) * GF_TILE * GF_TILE * GF_TILE * NCOMP;
}
__global__ void __launch_bounds__(GF_THREADS)
ghost_fill_kernel(const float* __restrict__ interior, float* __restrict__ padded, BoxGeom geo) {
    __shared__ __align__(16) float tile[VAR_FLOATS];
    // CTAs walk the box in 4 x 4 x 4 tiles of groups, so that the neighbours whose interiors a group reads are
    // handled close in time and the reads hit L2 (in plain group order the z neighbours are gx*gy groups apart)
    const int v = blockIdx.x % NCOMP;
    const long long q = blockIdx.x / NCOMP;
    const int ntx = (geo.gx + GF_TILE - 1) / GF_TILE, nty = (geo.gy + GF_TILE - 1) / GF_TILE;
    const long long tile_id = q / (GF_TILE * GF_TILE * GF_TILE);
    const int w = (int)(q % (GF_TILE * GF_TILE * GF_TILE));
    const int kx = (int)(tile_id % ntx) * GF_TILE + w % GF_TILE;
    const int ky = (int)((tile_id / ntx) % nty) * GF_TILE + (w / GF_TILE) % GF_TILE;
    const int kz = (int)(tile_id / ((long long)ntx * nty)) * GF_TILE + w / (GF_TILE * GF_TILE);
    if (kx >= geo.gx || ky >= geo.gy || kz >= geo.gz) return;
    const long long g = ((long long)kz * geo.gy + ky) * geo.gx + kx;
    float* dst = padded + (g * NCOMP + v) * (long long)VAR_FLOATS;
    // Per padded y and z: offset (in floats) of the source row inside `interior`, or -1 = beyond a "keep" end.  The
    // index arithmetic is done once per CTA here, not once per cell (the first version was bound by it).
    __shared__ long long off_y[NP], off_z[NP];
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
    // x: own group, left and right neighbour (or -1 = beyond a "keep" end)
    const int kxl = kx > 0 ? kx - 1 : (geo.bc[0] ? -1 : geo.gx - 1);
    const int kxr = kx < geo.gx - 1 ? kx + 1 : (geo.bc[0] ? -1 : 0);
    const float* const src_c = interior + kx * GS + v * (PS * PS * PS);
    const float* const src_l = kxl < 0 ? nullptr : interior + kxl * GS + v * (PS * PS * PS) + (PS - NG);
    const float* const src_r = kxr < 0 ? nullptr : interior + kxr * GS + v * (PS * PS * PS) - (PS + NG);
    // (1) the 16 cells x = 3..18 of every row: four 128-bit loads per row
#pragma unroll 4
    for (int t = threadIdx.x; t < NP * NP * 4; t += GF_THREADS) {
        const int row = t >> 2, part = t & 3;
        const int z = row / NP, y = row - z * NP;
        const long long oy = off_y[y], oz = off_z[z];
        float* trow = tile + row * NP + NG + 4 * part;
        float4 q;
        if (oy >= 0 && oz >= 0) {
            q = *reinterpret_cast<const float4*>(src_c + oz + oy + 4 * part);
        } else {
            const float* d = dst + row * NP + NG + 4 * part;
            q = make_float4(d[0], d[1], d[2], d[3]);
        }
        trow[0] = q.x; trow[1] = q.y; trow[2] = q.z; trow[3] = q.w;
    }
    // (2) the ghost cells x = 0..2 (left neighbour's cells 13..15) and x = 19..21 (right neighbour's cells 0..2)
#pragma unroll 2
    for (int t = threadIdx.x; t < NP * NP * 2 * NG; t += GF_THREADS) {
        const int row = t / (2 * NG), j = t - row * (2 * NG);
        const int z = row / NP, y = row - z * NP;
        const long long oy = off_y[y], oz = off_z[z];
        const int x = j < NG ? j : PS + j;                        // padded x: 0..2 or 19..21
        const float* sx = j < NG ? src_l : src_r;                 // sx[x] is the source cell of padded x
        tile[row * NP + x] = (oy >= 0 && oz >= 0 && sx != nullptr) ? sx[oz + oy + x] : dst[row * NP + x];
    }
    __syncthreads();
    for (int i = threadIdx.x; i < VAR_FLOATS / 4; i += GF_THREADS)
        reinterpret_cast<float4*>(dst)[i] = reinterpret_cast<const float4*>(tile)[i];
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
