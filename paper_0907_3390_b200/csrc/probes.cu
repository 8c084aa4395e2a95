// probes.cu — measurement aids of bench.py (include/gamer_probes.h), built into their own library libgamer_probes.so so
// that the product library exports the hydro path and nothing else.  They reuse the production row march
// (rtvd_march.cuh, hydro_kernel.cuh) but share no state with libgamer_hydro.so.
#include <cuda_runtime.h>

#include <cstdarg>
#include <cstdio>
#include <vector>

#include "../../include/gamer_probes.h"
#include "hydro_kernel.cuh"

namespace {

thread_local char g_err[512] = "";

int fail(int code, const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
    return code;
}

// SM count of the current device; opt-in of `fn` to the dynamic shared memory of one resident group
int prepare(const void* fn, int* sm_count) {
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(sm_count, cudaDevAttrMultiProcessorCount, dev);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, gamer::SMEM_BYTES);
    if (e != cudaSuccess) { (void)cudaGetLastError(); return fail(GAMER_PROBE_ECUDA, "probe set-up: %s", cudaGetErrorString(e)); }
    return GAMER_PROBE_OK;
}

// FMA-only micro-benchmark of the FP32 pipe ("measures an FMA-only micro-benchmark, and states which
// number is used"): 16 independent FFMA chains per thread, nothing else in the loop but its counter.
constexpr int PEAK_CHAINS = 16, PEAK_ITERS = 2048, PEAK_THREADS = 512, PEAK_CTAS_PER_SM = 4;
__global__ void __launch_bounds__(PEAK_THREADS) fp32_peak_kernel(float* __restrict__ sink, float a, float b) {
    float x[PEAK_CHAINS];
#pragma unroll
    for (int i = 0; i < PEAK_CHAINS; ++i) x[i] = 1e-3f * (float)(threadIdx.x + i);
    const float m = a + 1e-9f * (float)(threadIdx.x & 1), c = b;      // per-thread values: stay in vector registers
#pragma unroll 8
    for (int it = 0; it < PEAK_ITERS; ++it) {
#pragma unroll
        for (int i = 0; i < PEAK_CHAINS; ++i) x[i] = fmaf(x[i], m, c);
    }
    float s = 0.f;
#pragma unroll
    for (int i = 0; i < PEAK_CHAINS; ++i) s += x[i];
    if (s == 123.456f) sink[0] = s;                                    // keeps the chains alive, never true in practice
}

// Issue-rate probes: what an SM sub-partition sustains on the instruction mix of this kernel.
//   ffma3_probe_kernel: fused multiply-adds whose three source operands are three different registers that no
//     neighbouring instruction shares (the register file delivers about two operands per clock to a sub-partition:
//     such an FMA costs 1.5 issue slots, one with two reused operands costs 1).
//   march_probe_kernel<D>: the production row march (rtvd_march.cuh, the sweep of hydro_kernel.cuh along axis D) back to
//     back on k warps per sub-partition, in place on one resident group, no loads, no barriers: cycles per warp-march.
constexpr int PROBE3_CHAINS = 16, PROBE3_ITERS = 2000;
__global__ void __launch_bounds__(512, 1) ffma3_probe_kernel(float* __restrict__ sink, long long* __restrict__ cyc) {
    float x[PROBE3_CHAINS], y[PROBE3_CHAINS], z[PROBE3_CHAINS];
#pragma unroll
    for (int i = 0; i < PROBE3_CHAINS; ++i) {
        x[i] = threadIdx.x * 1e-3f + i;
        y[i] = 1.0f + 1e-6f * (threadIdx.x + i);
        z[i] = 1e-7f * (threadIdx.x + 3 * i);
    }
    const long long t0 = clock64();
#pragma unroll 1
    for (int it = 0; it < PROBE3_ITERS; ++it) {
#pragma unroll
        for (int r = 0; r < 4; ++r)
#pragma unroll
            for (int i = 0; i < PROBE3_CHAINS; ++i) x[i] = fmaf(x[i], y[i], z[i]);
    }
    const long long t1 = clock64();
    float s = 0.f;
#pragma unroll
    for (int i = 0; i < PROBE3_CHAINS; ++i) s += x[i] + y[i] + z[i];
    if (s == 123.456f) sink[0] = s;
    if ((threadIdx.x & 31) == 0) atomicMax(reinterpret_cast<unsigned long long*>(&cyc[blockIdx.x]), (unsigned long long)(t1 - t0));
}

template <int D>
__global__ void __launch_bounds__(gamer::BLOCK_THREADS, 1)
march_probe_kernel(const float* __restrict__ in, gamer::GasConst gc, int k_per_smsp, int reps, long long* __restrict__ cyc,
                   float* __restrict__ sink, int* __restrict__ changed) {
    using namespace gamer;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    float* smem = reinterpret_cast<float*>(smem_raw);
    for (int i = threadIdx.x; i < GROUP_IN_FLOATS; i += blockDim.x) smem[i] = in[i];
    __syncthreads();
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    NoGate nogate;
    float speed = 0.f;
    const long long t0 = clock64();
    if (warp < 4 * k_per_smsp) {
#pragma unroll 1
        for (int r = 0; r < reps; ++r) {
            // A sweep has fewer rows than 512 threads (484, 352, 256), so several warps march the same rows in place,
            // unsynchronised.  The probe runs with dt = 0: every update is u - 0 * (flux difference) = u, the same
            // instruction stream as any other dt, so all warps read and write back the SAME bits in every repetition
            // and the state stays the physical input state (checked below).
            if (D == 0)
                sweep<0, 0, NP, 0, NP, false, false, false, false>(smem, gc, nullptr, nullptr, speed, (32 * warp + lane) % 480, nogate);
            else if (D == 1)
                sweep<1, NG, PS, 0, NP, false, false, false, false>(smem, gc, nullptr, nullptr, speed, ((threadIdx.x % 352) & ~31) | lane, nogate);
            else
                sweep<2, NG, PS, NG, PS, false, false, false, false>(smem, gc, nullptr, nullptr, speed, threadIdx.x % 256, nogate);
        }
    }
    const long long t1 = clock64();
    if (lane == 0) atomicMax(reinterpret_cast<unsigned long long*>(&cyc[blockIdx.x]), (unsigned long long)(t1 - t0));
    if (smem[12345] == 123.456f) sink[0] = smem[12345] + speed;
    // the marched state must still be the input state, bit for bit (dt = 0): anything else means the probe timed garbage
    __syncthreads();
    int diff = 0;
    for (int i = threadIdx.x; i < GROUP_IN_FLOATS; i += blockDim.x) diff |= (__float_as_uint(smem[i]) != __float_as_uint(in[i]));
    if (diff) atomicOr(changed, 1);
}

}  // namespace

extern "C" {

int gamer_probe_fp32_peak(int repeats, float* d_sink, double* tflops, double* lane_fma_per_clk_per_sm, double sm_mhz) {
    if (repeats < 1 || d_sink == nullptr || tflops == nullptr) return fail(GAMER_PROBE_EINVAL, "repeats >= 1, d_sink and tflops non-NULL");
    int dev = 0, sm = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&sm, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess) { (void)cudaGetLastError(); return fail(GAMER_PROBE_ECUDA, "no CUDA device: %s", cudaGetErrorString(e)); }
    cudaEvent_t e0, e1;
    if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) return fail(GAMER_PROBE_ECUDA, "cudaEventCreate");
    const int grid = sm * PEAK_CTAS_PER_SM;
    double best_ms = 1e30;
    for (int r = 0; r < repeats + 1 && e == cudaSuccess; ++r) {           // the first launch is a warm-up
        cudaEventRecord(e0, 0);
        fp32_peak_kernel<<<grid, PEAK_THREADS>>>(d_sink, 1.0000001f, 1e-7f);
        cudaEventRecord(e1, 0);
        e = cudaEventSynchronize(e1);
        float ms = 0.f;
        if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
        if (r > 0 && ms < best_ms) best_ms = ms;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    if (e != cudaSuccess) return fail(GAMER_PROBE_ECUDA, "fp32_peak: %s", cudaGetErrorString(e));
    const double fma = (double)grid * PEAK_THREADS * PEAK_CHAINS * PEAK_ITERS;
    *tflops = 2.0 * fma / (best_ms * 1e-3) / 1e12;
    if (lane_fma_per_clk_per_sm) *lane_fma_per_clk_per_sm = sm_mhz > 0 ? fma / (best_ms * 1e-3) / (sm_mhz * 1e6) / sm : 0.0;
    g_err[0] = '\0';
    return GAMER_PROBE_OK;
}

int gamer_probe_issue(int what, int warps_per_smsp, double* cycles) {
    if (cycles == nullptr || what < 0 || what > 3 || warps_per_smsp < 1 || warps_per_smsp > 4)
        return fail(GAMER_PROBE_EINVAL, "issue_probe: what in 0..3, warps_per_smsp in 1..4, cycles non-NULL");
    int sm_count = 0;
    int rc = prepare(reinterpret_cast<const void*>(march_probe_kernel<0>), &sm_count);
    if (rc == GAMER_PROBE_OK) rc = prepare(reinterpret_cast<const void*>(march_probe_kernel<1>), &sm_count);
    if (rc == GAMER_PROBE_OK) rc = prepare(reinterpret_cast<const void*>(march_probe_kernel<2>), &sm_count);
    if (rc != GAMER_PROBE_OK) return rc;
    // one group of a smooth, physical, non-uniform state; dt = 0 keeps it exactly so over the in-place repetitions
    std::vector<float> h(gamer::GROUP_IN_FLOATS);
    unsigned int seed = 12345u;
    for (int v = 0; v < gamer::NCOMP; ++v)
        for (int i = 0; i < gamer::VAR_FLOATS; ++i) {
            seed = seed * 1664525u + 1013904223u;
            const float r = (float)(seed >> 8) * (1.0f / 16777216.0f);
            h[(size_t)v * gamer::VAR_FLOATS + i] = v == 0 ? 1.f + 0.1f * r : (v == 4 ? 1.5f + 0.1f * r : 0.1f * (r - 0.5f));
        }
    float* d_in = nullptr;
    long long* d_cyc = nullptr;
    float* d_sink = nullptr;
    int* d_changed = nullptr;
    int changed = 0;
    cudaError_t e = cudaMalloc(&d_in, gamer::GROUP_IN_BYTES);
    if (e == cudaSuccess) e = cudaMalloc(&d_cyc, (size_t)sm_count * sizeof(long long));
    if (e == cudaSuccess) e = cudaMalloc(&d_sink, sizeof(float));
    if (e == cudaSuccess) e = cudaMalloc(&d_changed, sizeof(int));
    if (e == cudaSuccess) e = cudaMemset(d_changed, 0, sizeof(int));
    if (e == cudaSuccess) e = cudaMemcpy(d_in, h.data(), gamer::GROUP_IN_BYTES, cudaMemcpyHostToDevice);
    const int reps = 20;
    gamer::GasConst gc = gamer::make_const(0.0f, 1.0f, 5.0f / 3.0f);
    std::vector<long long> c(sm_count);
    for (int pass = 0; pass < 2 && e == cudaSuccess; ++pass) {          // the first pass is a warm-up
        e = cudaMemset(d_cyc, 0, (size_t)sm_count * sizeof(long long));
        if (e != cudaSuccess) break;
        if (what == 0) ffma3_probe_kernel<<<sm_count, 512>>>(d_sink, d_cyc);
        else if (what == 1) march_probe_kernel<0><<<sm_count, gamer::BLOCK_THREADS, gamer::SMEM_BYTES>>>(d_in, gc, warps_per_smsp, reps, d_cyc, d_sink, d_changed);
        else if (what == 2) march_probe_kernel<1><<<sm_count, gamer::BLOCK_THREADS, gamer::SMEM_BYTES>>>(d_in, gc, warps_per_smsp, reps, d_cyc, d_sink, d_changed);
        else march_probe_kernel<2><<<sm_count, gamer::BLOCK_THREADS, gamer::SMEM_BYTES>>>(d_in, gc, warps_per_smsp, reps, d_cyc, d_sink, d_changed);
        e = cudaDeviceSynchronize();
        if (e == cudaSuccess) e = cudaMemcpy(c.data(), d_cyc, (size_t)sm_count * sizeof(long long), cudaMemcpyDeviceToHost);
    }
    if (e == cudaSuccess) e = cudaMemcpy(&changed, d_changed, sizeof(int), cudaMemcpyDeviceToHost);
    cudaFree(d_in);
    cudaFree(d_cyc);
    cudaFree(d_sink);
    cudaFree(d_changed);
    if (e != cudaSuccess) { (void)cudaGetLastError(); return fail(GAMER_PROBE_ECUDA, "issue_probe: %s", cudaGetErrorString(e)); }
    if (changed) return fail(GAMER_PROBE_ECUDA, "issue_probe: the marched state no longer equals its input (dt = 0): timing not valid");
    double mean = 0.0;
    for (int i = 0; i < sm_count; ++i) mean += (double)c[i];
    mean /= sm_count;
    // what = 0: 4 warps per sub-partition (512 threads), cycles per warp instruction of one sub-partition;
    // what = 1..3: cycles per warp-march and sub-partition slot
    *cycles = what == 0 ? mean / (4.0 * PROBE3_ITERS * 4 * PROBE3_CHAINS) : mean / reps / warps_per_smsp;
    g_err[0] = '\0';
    return GAMER_PROBE_OK;
}

const char* gamer_probe_last_error(void) { return g_err; }

}  // extern "C"
