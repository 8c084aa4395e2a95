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
__global__ void __launch_bounds__(GF_THREADS)
ghost_fill_kernel(const float* __restrict__ interior, float* __restrict__ padded, BoxGeom geo) {
    __shared__ __align__(16) float tile[VAR_FLOATS];
    const long long g = blockIdx.x / NCOMP;
    const int v = blockIdx.x % NCOMP;
    const int kx = (int)(g % geo.gx), ky = (int)((g / geo.gx) % geo.gy), kz = (int)(g / ((long long)geo.gx * geo.gy));
    float* dst = padded + (g * NCOMP + v) * (long long)VAR_FLOATS;
    // x neighbours (group coordinate, or -1 = beyond a "keep" end)
    const int kxl = kx > 0 ? kx - 1 : (geo.bc[0] ? -1 : geo.gx - 1);
    const int kxr = kx < geo.gx - 1 ? kx + 1 : (geo.bc[0] ? -1 : 0);
    for (int t = threadIdx.x; t < NP * NP * 8; t += GF_THREADS) {
        const int row = t >> 3, part = t & 7;          // parts 0..3: interior quarter; 4: left ghosts; 5: right ghosts
        if (part > 5) continue;
        const int y = row % NP, z = row / NP;
        // source group and interior index along y and z
        int ys = y - NG, zs = z - NG, sky = ky, skz = kz;
        bool keep = false;
        if (ys < 0) { ys += PS; sky = ky > 0 ? ky - 1 : geo.gy - 1; keep |= (ky == 0 && geo.bc[1]); }
        else if (ys >= PS) { ys -= PS; sky = ky < geo.gy - 1 ? ky + 1 : 0; keep |= (ky == geo.gy - 1 && geo.bc[1]); }
        if (zs < 0) { zs += PS; skz = kz > 0 ? kz - 1 : geo.gz - 1; keep |= (kz == 0 && geo.bc[2]); }
        else if (zs >= PS) { zs -= PS; skz = kz < geo.gz - 1 ? kz + 1 : 0; keep |= (kz == geo.gz - 1 && geo.bc[2]); }
        float* trow = tile + row * NP;
        const int skx = part < 4 ? kx : (part == 4 ? kxl : kxr);
        const int x0 = part < 4 ? NG + 4 * part : (part == 4 ? 0 : NG + PS);          // first padded x of this part
        const int n = part < 4 ? 4 : NG;
        if (keep || skx < 0) {
            for (int i = 0; i < n; ++i) trow[x0 + i] = dst[row * NP + x0 + i];
        } else {
            const float* src = interior + ((((long long)skz * geo.gy + sky) * geo.gx + skx) * NCOMP + v) * (long long)(PS * PS * PS) +
                               (zs * PS + ys) * PS;
            if (part < 4) {
                const float4 q = *reinterpret_cast<const float4*>(src + 4 * part);
                trow[x0] = q.x; trow[x0 + 1] = q.y; trow[x0 + 2] = q.z; trow[x0 + 3] = q.w;
            } else {
                const int xs = part == 4 ? PS - NG : 0;
                for (int i = 0; i < NG; ++i) trow[x0 + i] = src[xs + i];
            }
        }
    }
    __syncthreads();
    for (int i = threadIdx.x; i < VAR_FLOATS / 4; i += GF_THREADS)
        reinterpret_cast<float4*>(dst)[i] = reinterpret_cast<const float4*>(tile)[i];
}

// max over ALL padded cells of all groups of c_s + max(|v_x|,|v_y|,|v_z|) (reading R10), as the bit pattern
// of a non-negative float in *acc (atomicMax on unsigned: positive floats order like their bit patterns).
__global__ void __launch_bounds__(256)
max_speed_kernel(const float* __restrict__ padded, long long n_groups, float gamma, unsigned int* __restrict__ acc) {
    float best = 0.f;
    const float ggm1 = gamma * (gamma - 1.0f);
    for (long long g = blockIdx.x; g < n_groups; g += gridDim.x) {
        const float* u = padded + g * (long long)GROUP_IN_FLOATS;
        for (int i = threadIdx.x; i < VAR_FLOATS; i += blockDim.x) {
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

// dt = cfl dh / speed; resets the accumulator for the next step.  work[0]: accumulator, work[1]: dt.
__global__ void cfl_dt_kernel(float* __restrict__ work, float cfl, float dh, float* __restrict__ dt_log) {
    const float speed = __uint_as_float(reinterpret_cast<unsigned int*>(work)[0]);
    const float dt = cfl * dh / speed;
    work[1] = dt;
    if (dt_log) *dt_log = dt;
    reinterpret_cast<unsigned int*>(work)[0] = 0u;
}

}  // namespace gamer
