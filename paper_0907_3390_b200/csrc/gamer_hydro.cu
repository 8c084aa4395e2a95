// gamer_hydro.cu — the C ABI of include/gamer_hydro.h: argument validation, launch, and the stream pipeline.
#include <cuda_runtime.h>

#include <cmath>
#include <cstdarg>
#include <cstdint>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <vector>

#include "../../include/gamer_hydro.h"
#include "hydro_kernel.cuh"
#include "uniform_grid.cuh"
#include "hydro_kernel_f64.cuh"

namespace {

thread_local char g_err[512] = "";

int fail(int code, const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
    return code;
}

bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

// do [a, a + a_bytes) and [b, b + b_bytes) intersect?  (NULL or empty ranges never do)
bool ranges_overlap(const void* a, size_t a_bytes, const void* b, size_t b_bytes) {
    if (a == nullptr || b == nullptr || a_bytes == 0 || b_bytes == 0) return false;
    const uintptr_t a0 = reinterpret_cast<uintptr_t>(a), b0 = reinterpret_cast<uintptr_t>(b);
    return a0 < b0 + b_bytes && b0 < a0 + a_bytes;
}

using KernelFn = void (*)(const float*, float*, long long, gamer::GasConst, float*, float*, const float*);

KernelFn pick_kernel(bool backward, bool face, bool speed) {
    using namespace gamer;
    const int key = (backward ? 4 : 0) | (face ? 2 : 0) | (speed ? 1 : 0);
    switch (key) {
        case 0: return hydro_advance_kernel<false, false, false>;
        case 1: return hydro_advance_kernel<false, false, true>;
        case 2: return hydro_advance_kernel<false, true, false>;
        case 3: return hydro_advance_kernel<false, true, true>;
        case 4: return hydro_advance_kernel<true, false, false>;
        case 5: return hydro_advance_kernel<true, false, true>;
        case 6: return hydro_advance_kernel<true, true, false>;
        default: return hydro_advance_kernel<true, true, true>;
    }
}

struct DeviceInfo {
    bool ready = false;
    int sm_count = 0;
    int smem_optin = 0;          // dynamic shared memory a block may opt in to, bytes
    bool attr_set[32] = {};      // one flag per kernel key (prepare())
};
std::mutex g_mu;
DeviceInfo g_dev[64];

// Streams and device staging buffers of gamer_hydro_pipeline_run, per device, kept between calls.
struct Staging {
    cudaStream_t stream[16] = {};
    float* d_in[16] = {};
    float* d_out[16] = {};
    size_t in_bytes[16] = {};
    size_t out_bytes[16] = {};
};
std::mutex g_pipe_mu[64];      // one per device: calls on different devices do not serialise
Staging g_staging[64];

// SM count of the current device and the opt-in to 208 KB of dynamic shared memory, once per device and kernel.
int prepare(const void* fn, int key, int smem_bytes, int* sm_count) {
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return fail(GAMER_ECUDA, "cudaGetDevice: %s", cudaGetErrorString(e));
    if (dev < 0 || dev >= 64) return fail(GAMER_ECUDA, "device ordinal %d out of range", dev);
    std::lock_guard<std::mutex> lk(g_mu);
    DeviceInfo& di = g_dev[dev];
    if (!di.ready) {
        int major = 0, smem_optin = 0;      // (checked per kernel below: the fp64 kernels need more than the fp32 ones)
        e = cudaDeviceGetAttribute(&di.sm_count, cudaDevAttrMultiProcessorCount, dev);
        if (e == cudaSuccess) e = cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev);
        if (e == cudaSuccess) e = cudaDeviceGetAttribute(&smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
        if (e != cudaSuccess) return fail(GAMER_ECUDA, "cudaDeviceGetAttribute: %s", cudaGetErrorString(e));
        if (major != 10)
            return fail(GAMER_EUNSUPPORTED, "this library is built for sm_100a only; device %d has compute capability %d.x",
                        dev, major);
        if (smem_optin < gamer::SMEM_BYTES)
            return fail(GAMER_EUNSUPPORTED, "device offers %d B of shared memory per block, %d needed", smem_optin,
                        gamer::SMEM_BYTES);
        di.smem_optin = smem_optin;
        di.ready = true;
    }
    if (!di.attr_set[key]) {
        if (smem_bytes > di.smem_optin)
            return fail(GAMER_EUNSUPPORTED, "device %d offers %d B of shared memory per block, this kernel needs %d", dev,
                        di.smem_optin, smem_bytes);
        e = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_bytes);
        if (e != cudaSuccess) return fail(GAMER_ECUDA, "cudaFuncSetAttribute: %s", cudaGetErrorString(e));
        di.attr_set[key] = true;
    }
    *sm_count = di.sm_count;
    return GAMER_OK;
}

int validate(const void* in, const void* out, long long n_groups, int ghost, float dt, float dh, float gamma,
             int backward, const void* face, const void* speed) {
    if (ghost != gamer::NG)
        return fail(GAMER_EUNSUPPORTED, "ghost = %d: the 7-point stencil of the scheme fixes ghost = 3", ghost);
    if (n_groups < 0) return fail(GAMER_EINVAL, "n_groups = %lld < 0", n_groups);
    if (!(dh > 0.f)) return fail(GAMER_EINVAL, "dh must be > 0");
    if (!(dt >= 0.f)) return fail(GAMER_EINVAL, "dt must be >= 0");
    if (!(gamma > 1.f)) return fail(GAMER_EINVAL, "gamma must be > 1");
    if (backward != 0 && backward != 1) return fail(GAMER_EINVAL, "backward must be 0 or 1");
    if (n_groups > 0 && (in == nullptr || out == nullptr)) return fail(GAMER_EINVAL, "NULL input or output pointer");
    if (!aligned16(in) || !aligned16(out) || !aligned16(face) || !aligned16(speed))
        return fail(GAMER_EINVAL, "pointers must be 16-byte aligned");
    return GAMER_OK;
}

// The kernel streams results of finished groups to the outputs while later groups are still being read: an output
// that overlaps the input (or another output) would be corrupted silently.  bytes[i] = extent of ptr[i].
int check_disjoint(const void* const* ptr, const size_t* bytes, int n) {
    for (int i = 0; i < n; ++i)
        for (int j = i + 1; j < n; ++j)
            if (ranges_overlap(ptr[i], bytes[i], ptr[j], bytes[j]))
                return fail(GAMER_EINVAL, "input, output and scratch buffers must not overlap");
    return GAMER_OK;
}

using gamer::make_const;

int launch(const float* d_in, float* d_out, long long n_groups, float dt, float dh, float gamma, int backward,
           float* d_face, float* d_speed, cudaStream_t stream) {
    const int key = (backward ? 4 : 0) | (d_face ? 2 : 0) | (d_speed ? 1 : 0);
    int sm_count = 0;
    KernelFn fn = pick_kernel(backward != 0, d_face != nullptr, d_speed != nullptr);
    const int rc = prepare(reinterpret_cast<const void*>(fn), key, gamer::SMEM_BYTES, &sm_count);
    if (rc != GAMER_OK) return rc;
    const int grid = (int)(n_groups < (long long)sm_count ? n_groups : (long long)sm_count);
    fn<<<grid, gamer::BLOCK_THREADS, gamer::SMEM_BYTES, stream>>>(d_in, d_out, n_groups, make_const(dt, dh, gamma),
                                                                  d_face, d_speed, nullptr);
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(GAMER_ECUDA, "kernel launch: %s", cudaGetErrorString(e));
    return GAMER_OK;
}

}  // namespace

// Built-in scratch of gamer_hydro_run_uniform_noalloc (gamer_hydro.h): the d_work of gamer_hydro_run_uniform for callers
// that cannot allocate.  It lives in the library image: each GPU that loads this library holds it until the process exits.
// In HOST code the name g_noalloc_work is only a handle for the runtime (a host-side shadow), not a device address: a
// kernel must be given what cudaGetSymbolAddress returns for the current device, never the name itself.
static_assert(GAMER_NOALLOC_MAX_GROUPS >= 1 && GAMER_NOALLOC_MAX_GROUPS <= (1 << 20), "keep the built-in scratch modest");
static __device__ __align__(256) float g_noalloc_work[4 + GAMER_NOALLOC_MAX_GROUPS];

namespace {

float* g_noalloc_ptr[64] = {};      // device address of g_noalloc_work on each device, looked up once (under g_mu)

// Device address of the built-in scratch on the CURRENT device.  The first call per device does the look-up (and with
// it loads the library's code on that device if nothing else has yet); later calls only read the cached pointer.
int noalloc_scratch(float** out) {
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) { (void)cudaGetLastError(); return fail(GAMER_ECUDA, "cudaGetDevice: %s", cudaGetErrorString(e)); }
    if (dev < 0 || dev >= 64) return fail(GAMER_ECUDA, "device ordinal %d out of range", dev);
    std::lock_guard<std::mutex> lk(g_mu);
    if (g_noalloc_ptr[dev] == nullptr) {
        void* p = nullptr;
        e = cudaGetSymbolAddress(&p, g_noalloc_work);
        if (e != cudaSuccess || p == nullptr) {
            (void)cudaGetLastError();
            return fail(GAMER_ECUDA, "cudaGetSymbolAddress of the built-in scratch on device %d: %s", dev, cudaGetErrorString(e));
        }
        g_noalloc_ptr[dev] = static_cast<float*>(p);
    }
    *out = g_noalloc_ptr[dev];
    return GAMER_OK;
}

}  // namespace

extern "C" {

int gamer_hydro_advance_ex(const float* d_in, float* d_out, long long n_groups, int ghost, float dt, float dh,
                           float gamma, int backward, float* d_face_flux, float* d_group_maxspeed, void* stream) {
    int rc = validate(d_in, d_out, n_groups, ghost, dt, dh, gamma, backward, d_face_flux, d_group_maxspeed);
    if (rc != GAMER_OK) return rc;
    {
        const size_t n = (size_t)n_groups, fl = sizeof(float);
        const void* ptr[4] = {d_in, d_out, d_face_flux, d_group_maxspeed};
        const size_t bytes[4] = {n * gamer::GROUP_IN_FLOATS * fl, n * gamer::GROUP_OUT_FLOATS * fl,
                                 n * gamer::GROUP_FACE_FLOATS * fl, n * fl};
        rc = check_disjoint(ptr, bytes, 4);
        if (rc != GAMER_OK) return rc;
    }
    g_err[0] = '\0';
    if (n_groups == 0) return GAMER_OK;
    return launch(d_in, d_out, n_groups, dt, dh, gamma, backward, d_face_flux, d_group_maxspeed,
                  static_cast<cudaStream_t>(stream));
}

int gamer_hydro_advance(const float* d_in, float* d_out, long long n_groups, int ghost, float dt, float dh,
                        float gamma, void* stream) {
    return gamer_hydro_advance_ex(d_in, d_out, n_groups, ghost, dt, dh, gamma, 0, nullptr, nullptr, stream);
}

size_t gamer_hydro_in_floats(long long n_groups, int ghost) {
    if (n_groups < 0 || ghost < 0) return 0;
    const size_t n = (size_t)(gamer::PS + 2 * ghost);
    return (size_t)n_groups * gamer::NCOMP * n * n * n;
}
size_t gamer_hydro_out_floats(long long n_groups) {
    return n_groups < 0 ? 0 : (size_t)n_groups * gamer::GROUP_OUT_FLOATS;
}
size_t gamer_hydro_face_flux_floats(long long n_groups) {
    return n_groups < 0 ? 0 : (size_t)n_groups * gamer::GROUP_FACE_FLOATS;
}

int gamer_hydro_pipeline_run(const float* h_in, float* h_out, long long n_groups, int ghost, float dt, float dh,
                             float gamma, int backward, long long groups_per_chunk, int n_streams) {
    int rc = validate(h_in, h_out, n_groups, ghost, dt, dh, gamma, backward, nullptr, nullptr);
    if (rc != GAMER_OK) return rc;
    {
        const void* ptr[2] = {h_in, h_out};
        const size_t bytes[2] = {(size_t)n_groups * gamer::GROUP_IN_FLOATS * sizeof(float),
                                 (size_t)n_groups * gamer::GROUP_OUT_FLOATS * sizeof(float)};
        rc = check_disjoint(ptr, bytes, 2);
        if (rc != GAMER_OK) return rc;
    }
    if (n_streams < 1 || n_streams > 16) return fail(GAMER_EINVAL, "n_streams must be in 1..16");
    if (groups_per_chunk < 1) return fail(GAMER_EINVAL, "groups_per_chunk must be >= 1");
    g_err[0] = '\0';
    if (n_groups == 0) return GAMER_OK;
    if (groups_per_chunk > n_groups) groups_per_chunk = n_groups;
    const long long n_chunks = (n_groups + groups_per_chunk - 1) / groups_per_chunk;
    if (n_streams > n_chunks) n_streams = (int)n_chunks;

    const size_t in_bytes = (size_t)groups_per_chunk * gamer::GROUP_IN_FLOATS * sizeof(float);
    const size_t out_bytes = (size_t)groups_per_chunk * gamer::GROUP_OUT_FLOATS * sizeof(float);
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess || dev < 0 || dev >= 64) return fail(GAMER_ECUDA, "cudaGetDevice: %s", cudaGetErrorString(e));
    // The streams and staging buffers are kept between calls (allocating 3 x 150 MB costs ~10 % of a config-5 call)
    // and grown when a call needs more; gamer_hydro_pipeline_release() frees them.  Calls are serialised per device.
    std::lock_guard<std::mutex> lk(g_pipe_mu[dev]);
    Staging& st = g_staging[dev];
    int status = GAMER_OK;
    for (int s = 0; s < n_streams && status == GAMER_OK; ++s) {
        if (st.stream[s] == nullptr) {
            e = cudaStreamCreateWithFlags(&st.stream[s], cudaStreamNonBlocking);
            if (e != cudaSuccess) { status = fail(GAMER_ECUDA, "cudaStreamCreate: %s", cudaGetErrorString(e)); break; }
        }
        if (st.in_bytes[s] < in_bytes) {
            if (st.d_in[s]) cudaFree(st.d_in[s]);
            st.d_in[s] = nullptr;
            st.in_bytes[s] = 0;
            e = cudaMalloc(&st.d_in[s], in_bytes);
            if (e == cudaSuccess) st.in_bytes[s] = in_bytes;
        }
        if (e == cudaSuccess && st.out_bytes[s] < out_bytes) {
            if (st.d_out[s]) cudaFree(st.d_out[s]);
            st.d_out[s] = nullptr;
            st.out_bytes[s] = 0;
            e = cudaMalloc(&st.d_out[s], out_bytes);
            if (e == cudaSuccess) st.out_bytes[s] = out_bytes;
        }
        if (e != cudaSuccess) {
            status = fail(e == cudaErrorMemoryAllocation ? GAMER_ENOMEM : GAMER_ECUDA, "cudaMalloc of staging buffers: %s",
                          cudaGetErrorString(e));
            (void)cudaGetLastError();
        }
    }
    // Fig.5: chunk c goes to stream c mod N_s: copy in, kernel, copy out.  Stream order keeps a
    // staging buffer from being overwritten before its previous chunk has left it.
    for (long long c = 0; c < n_chunks && status == GAMER_OK; ++c) {
        const int s = (int)(c % n_streams);
        const long long g0 = c * groups_per_chunk;
        const long long ng = (n_groups - g0) < groups_per_chunk ? (n_groups - g0) : groups_per_chunk;
        e = cudaMemcpyAsync(st.d_in[s], h_in + g0 * gamer::GROUP_IN_FLOATS,
                            (size_t)ng * gamer::GROUP_IN_FLOATS * sizeof(float), cudaMemcpyHostToDevice, st.stream[s]);
        if (e != cudaSuccess) { status = fail(GAMER_ECUDA, "cudaMemcpyAsync H2D: %s", cudaGetErrorString(e)); break; }
        status = launch(st.d_in[s], st.d_out[s], ng, dt, dh, gamma, backward, nullptr, nullptr, st.stream[s]);
        if (status != GAMER_OK) break;
        e = cudaMemcpyAsync(h_out + g0 * gamer::GROUP_OUT_FLOATS, st.d_out[s],
                            (size_t)ng * gamer::GROUP_OUT_FLOATS * sizeof(float), cudaMemcpyDeviceToHost, st.stream[s]);
        if (e != cudaSuccess) { status = fail(GAMER_ECUDA, "cudaMemcpyAsync D2H: %s", cudaGetErrorString(e)); break; }
    }
    for (int s = 0; s < n_streams; ++s) {
        if (st.stream[s]) {
            e = cudaStreamSynchronize(st.stream[s]);
            if (e != cudaSuccess && status == GAMER_OK)
                status = fail(GAMER_ECUDA, "cudaStreamSynchronize: %s", cudaGetErrorString(e));
        }
    }
    return status;
}

int gamer_hydro_pipeline_release(void) {
    int dev = 0;
    const cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess || dev < 0 || dev >= 64) return fail(GAMER_ECUDA, "cudaGetDevice: %s", cudaGetErrorString(e));
    std::lock_guard<std::mutex> lk(g_pipe_mu[dev]);
    Staging& st = g_staging[dev];
    for (int s = 0; s < 16; ++s) {
        if (st.stream[s]) cudaStreamSynchronize(st.stream[s]);
        if (st.d_in[s]) cudaFree(st.d_in[s]);
        if (st.d_out[s]) cudaFree(st.d_out[s]);
        if (st.stream[s]) cudaStreamDestroy(st.stream[s]);
    }
    st = Staging();
    g_err[0] = '\0';
    return GAMER_OK;
}

// the ghost fill comes in two instantiations: the whole-strip walk, and the walk cut into segments for thin boxes
static int prepare_ghost_fill(int* sm_count) {
    int rc = prepare(reinterpret_cast<const void*>(gamer::ghost_fill_kernel<false>), 13, gamer::GF_SMEM_BYTES, sm_count);
    if (rc == GAMER_OK) rc = prepare(reinterpret_cast<const void*>(gamer::ghost_fill_kernel<true>), 14, gamer::GF_SMEM_BYTES, sm_count);
    return rc;
}
static void launch_ghost_fill(const float* d_interior, float* d_padded, const gamer::BoxGeom& geo, cudaStream_t stream) {
    const unsigned int grid = (unsigned int)gamer::ghost_fill_ctas(geo.gx, geo.gy, geo.gz, geo.nseg);
    if (geo.nseg > 1)
        gamer::ghost_fill_kernel<true><<<grid, gamer::GF_THREADS, gamer::GF_SMEM_BYTES, stream>>>(d_interior, d_padded, geo);
    else
        gamer::ghost_fill_kernel<false><<<grid, gamer::GF_THREADS, gamer::GF_SMEM_BYTES, stream>>>(d_interior, d_padded, geo);
}

static int check_box(int gx, int gy, int gz, int bc_x, int bc_y, int bc_z) {
    if (gx < 1 || gy < 1 || gz < 1) return fail(GAMER_EINVAL, "box of %d x %d x %d groups", gx, gy, gz);
    if ((long long)gx * gy * gz * gamer::NCOMP > (1ll << 31) - 1) return fail(GAMER_EINVAL, "too many groups for one launch");
    if ((bc_x | bc_y | bc_z) & ~1) return fail(GAMER_EINVAL, "boundary flags must be 0 (periodic) or 1 (keep)");
    return GAMER_OK;
}

int gamer_hydro_ghost_fill(const float* d_interior, float* d_padded, int gx, int gy, int gz, int bc_x, int bc_y,
                           int bc_z, void* stream) {
    int rc = check_box(gx, gy, gz, bc_x, bc_y, bc_z);
    if (rc != GAMER_OK) return rc;
    if (d_interior == nullptr || d_padded == nullptr) return fail(GAMER_EINVAL, "NULL pointer");
    if (!aligned16(d_interior) || !aligned16(d_padded)) return fail(GAMER_EINVAL, "pointers must be 16-byte aligned");
    g_err[0] = '\0';
    int sm_count = 0;
    rc = prepare_ghost_fill(&sm_count);
    if (rc != GAMER_OK) return rc;
    gamer::BoxGeom geo{gx, gy, gz, {bc_x, bc_y, bc_z}, gamer::ghost_fill_segments(gx, gy, gz, sm_count)};
    launch_ghost_fill(d_interior, d_padded, geo, static_cast<cudaStream_t>(stream));
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(GAMER_ECUDA, "ghost_fill launch: %s", cudaGetErrorString(e));
    return GAMER_OK;
}

int gamer_hydro_run_uniform(float* d_padded, float* d_interior, int gx, int gy, int gz, int bc_x, int bc_y, int bc_z,
                            int n_steps, int order, float cfl, float dh, float gamma, float* d_work, float* d_dt_log,
                            void* stream_) {
    int rc = check_box(gx, gy, gz, bc_x, bc_y, bc_z);
    if (rc != GAMER_OK) return rc;
    const long long n = (long long)gx * gy * gz;
    rc = validate(d_padded, d_interior, n, gamer::NG, 0.f, dh, gamma, 0, d_work, d_dt_log);
    if (rc != GAMER_OK) return rc;
    if (d_work == nullptr) return fail(GAMER_EINVAL, "d_work must point to 4 + n_groups floats of device memory");
    if (n_steps < 0 || !(cfl > 0.f)) return fail(GAMER_EINVAL, "n_steps must be >= 0 and cfl > 0");
    if (order != 0 && order != 1) return fail(GAMER_EINVAL, "order must be 0 (forward passes) or 1 (forward + backward pairs)");
    {
        const size_t fl = sizeof(float);
        const void* ptr[4] = {d_padded, d_interior, d_work, d_dt_log};
        const size_t bytes[4] = {(size_t)n * gamer::GROUP_IN_FLOATS * fl, (size_t)n * gamer::GROUP_OUT_FLOATS * fl,
                                 (size_t)(4 + n) * fl, (size_t)n_steps * fl};
        rc = check_disjoint(ptr, bytes, 4);
        if (rc != GAMER_OK) return rc;
    }
    g_err[0] = '\0';
    cudaStream_t stream = static_cast<cudaStream_t>(stream_);
    using namespace gamer;
    // dt is read from device memory by every pass; the per-group CFL speed comes out of the LAST pass of a step
    // ("we can calculate the CFL condition in GPU after the backward sweep")
    KernelFn fwd = order == 0 ? hydro_advance_kernel<false, false, true, true> : hydro_advance_kernel<false, false, false, true>;
    KernelFn bwd = hydro_advance_kernel<true, false, true, true>;
    int sm_count = 0;
    rc = prepare(reinterpret_cast<const void*>(fwd), order == 0 ? 8 : 11, SMEM_BYTES, &sm_count);
    if (rc == GAMER_OK && order == 1) rc = prepare(reinterpret_cast<const void*>(bwd), 12, SMEM_BYTES, &sm_count);
    if (rc == GAMER_OK) rc = prepare_ghost_fill(&sm_count);
    if (rc != GAMER_OK) return rc;
    const int grid = (int)(n < (long long)sm_count ? n : (long long)sm_count);
    const int red_grid = (int)(n < 4ll * sm_count ? n : 4ll * sm_count);
    const unsigned int gsm_grid = (unsigned int)((n + 255) / 256 < 1024 ? (n + 255) / 256 : 1024);
    BoxGeom geo{gx, gy, gz, {bc_x, bc_y, bc_z}, ghost_fill_segments(gx, gy, gz, sm_count)};
    unsigned int* acc = reinterpret_cast<unsigned int*>(d_work);
    float* d_speed = d_work + 4;
    // Eq.30 over ALL padded cells (reading R10) costs one pass over the initial state.  After that the padded state
    // is: updated interiors (their speed comes out of the hydro kernel, fused, per group), periodic ghost cells
    // (copies of interiors) and ghost cells beyond "keep" ends (never change: their maximum is taken once, work[2]).
    cudaError_t e = cudaMemsetAsync(d_work, 0, 4 * sizeof(float), stream);
    if (n_steps > 0 && e == cudaSuccess) {
        if (bc_x | bc_y | bc_z) max_speed_kernel<<<red_grid, 256, 0, stream>>>(d_padded, n, gamma, acc + 2, geo, 1);
        max_speed_kernel<<<red_grid, 256, 0, stream>>>(d_padded, n, gamma, acc, geo, 0);
    }
    const GasConst gc = make_const(0.f, dh, gamma);
    for (int s = 0; s < n_steps && e == cudaSuccess; ++s) {
        cfl_dt_kernel<<<1, 1, 0, stream>>>(d_work, cfl, dh, d_dt_log ? d_dt_log + s : nullptr);
        fwd<<<grid, BLOCK_THREADS, SMEM_BYTES, stream>>>(d_padded, d_interior, n, gc, nullptr,
                                                         order == 0 ? d_speed : nullptr, d_work + 1);
        if (order == 1) {       // the backward sweep z,y,x follows with the SAME time step
            launch_ghost_fill(d_interior, d_padded, geo, stream);
            bwd<<<grid, BLOCK_THREADS, SMEM_BYTES, stream>>>(d_padded, d_interior, n, gc, nullptr, d_speed, d_work + 1);
        }
        group_speed_max_kernel<<<gsm_grid, 256, 0, stream>>>(d_speed, n, acc);
        launch_ghost_fill(d_interior, d_padded, geo, stream);
        e = cudaGetLastError();
    }
    if (e != cudaSuccess) return fail(GAMER_ECUDA, "run_uniform: %s", cudaGetErrorString(e));
    return GAMER_OK;
}

long long gamer_hydro_noalloc_max_groups(void) { return GAMER_NOALLOC_MAX_GROUPS; }

// gamer_hydro_run_uniform with the library's own scratch: no cudaMalloc / cudaFree / allocating routine on this path.
// The size is checked before the device is touched; every other argument is checked by gamer_hydro_run_uniform, which
// also clears the accumulators (stream-ordered memset of the first 16 bytes) — the per-group speeds behind them are
// overwritten by each step's last pass before the reduction reads them, so stale contents of an earlier call are never
// used.
int gamer_hydro_run_uniform_noalloc(float* d_padded, float* d_interior, int gx, int gy, int gz, int bc_x, int bc_y,
                                    int bc_z, int n_steps, int order, float cfl, float dh, float gamma, float* d_dt_log,
                                    void* stream) {
    int rc = check_box(gx, gy, gz, bc_x, bc_y, bc_z);
    if (rc != GAMER_OK) return rc;
    const long long n = (long long)gx * gy * gz;
    if (n > GAMER_NOALLOC_MAX_GROUPS)
        return fail(GAMER_EINVAL,
                    "box of %d x %d x %d = %lld groups exceeds the built-in scratch of gamer_hydro_run_uniform_noalloc "
                    "(GAMER_NOALLOC_MAX_GROUPS = %d): call gamer_hydro_run_uniform with your own d_work",
                    gx, gy, gz, n, GAMER_NOALLOC_MAX_GROUPS);
    float* d_work = nullptr;
    rc = noalloc_scratch(&d_work);
    if (rc != GAMER_OK) return rc;
    return gamer_hydro_run_uniform(d_padded, d_interior, gx, gy, gz, bc_x, bc_y, bc_z, n_steps, order, cfl, dh, gamma,
                                   d_work, d_dt_log, stream);
}

int gamer_hydro_advance_f64_ex(const double* d_in, double* d_out, long long n_groups, int ghost, double dt, double dh,
                               double gamma, int backward, double* d_face_flux, double* d_group_maxspeed, void* stream) {
    if (ghost != gamer::NG)
        return fail(GAMER_EUNSUPPORTED, "ghost = %d: the 7-point stencil of the scheme fixes ghost = 3", ghost);
    if (n_groups < 0) return fail(GAMER_EINVAL, "n_groups = %lld < 0", n_groups);
    if (!(dh > 0.0) || !(dt >= 0.0) || !(gamma > 1.0)) return fail(GAMER_EINVAL, "need dh > 0, dt >= 0, gamma > 1");
    if (backward != 0 && backward != 1) return fail(GAMER_EINVAL, "backward must be 0 or 1");
    if (n_groups > 0 && (d_in == nullptr || d_out == nullptr)) return fail(GAMER_EINVAL, "NULL input or output pointer");
    if (!aligned16(d_in) || !aligned16(d_out) || !aligned16(d_face_flux) || !aligned16(d_group_maxspeed))
        return fail(GAMER_EINVAL, "pointers must be 16-byte aligned");
    {
        const size_t n = (size_t)n_groups, db = sizeof(double);
        const void* ptr[4] = {d_in, d_out, d_face_flux, d_group_maxspeed};
        const size_t bytes[4] = {n * gamer::GROUP_IN_FLOATS * db, n * gamer::GROUP_OUT_FLOATS * db,
                                 n * gamer::GROUP_FACE_FLOATS * db, n * db};
        const int rc0 = check_disjoint(ptr, bytes, 4);
        if (rc0 != GAMER_OK) return rc0;
    }
    g_err[0] = '\0';
    if (n_groups == 0) return GAMER_OK;
    int sm_count = 0;
    using F64Fn = void (*)(const double*, double*, long long, gamer::GasConstT<double>, double*, double*);
    const bool opt = d_face_flux != nullptr || d_group_maxspeed != nullptr;
    F64Fn fn = backward ? (opt ? gamer::hydro_advance_f64_backward_kernel<true> : gamer::hydro_advance_f64_backward_kernel<false>)
                        : (opt ? gamer::hydro_advance_f64_kernel<true> : gamer::hydro_advance_f64_kernel<false>);
    const int rc = prepare(reinterpret_cast<const void*>(fn), (backward ? 10 : 9) + (opt ? 11 : 0), gamer::F64_SMEM_BYTES, &sm_count);
    if (rc != GAMER_OK) return rc;
    gamer::GasConstT<double> gc;
    const double k = dt / dh;
    gc.gm1 = gamma - 1.0;
    gc.ggm1 = gamma * (gamma - 1.0);
    gc.kq = 0.25 * k;
    gc.kh = 0.5 * k;
    gc.dh = dh;
    gc.sg = sqrt(gc.ggm1);
    gc.kq_gm1 = gc.kq * gc.gm1;
    gc.kq_sg = gc.kq * gc.sg;
    const int grid = (int)(n_groups < (long long)sm_count ? n_groups : (long long)sm_count);
    fn<<<grid, gamer::F64_THREADS, gamer::F64_SMEM_BYTES, static_cast<cudaStream_t>(stream)>>>(d_in, d_out, n_groups, gc,
                                                                                            d_face_flux, d_group_maxspeed);
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(GAMER_ECUDA, "kernel launch: %s", cudaGetErrorString(e));
    return GAMER_OK;
}

int gamer_hydro_launch_info(long long n_groups, int* grid, int* block, int* smem_bytes, int* regs_per_thread) {
    const void* fn = reinterpret_cast<const void*>(pick_kernel(false, false, false));
    const int smem = gamer::SMEM_BYTES;
    int sm_count = 0;
    const int rc = prepare(fn, 0, smem, &sm_count);
    if (rc != GAMER_OK) return rc;
    cudaFuncAttributes fa;
    const cudaError_t e = cudaFuncGetAttributes(&fa, fn);
    if (e != cudaSuccess) return fail(GAMER_ECUDA, "cudaFuncGetAttributes: %s", cudaGetErrorString(e));
    if (n_groups < 0) n_groups = 0;
    if (grid) *grid = (int)(n_groups < (long long)sm_count ? n_groups : (long long)sm_count);
    if (block) *block = gamer::BLOCK_THREADS;
    if (smem_bytes) *smem_bytes = smem;
    if (regs_per_thread) *regs_per_thread = fa.numRegs;
    g_err[0] = '\0';
    return GAMER_OK;
}

const char* gamer_last_error(void) { return g_err; }
const char* gamer_version(void) { return "gamer-hydro-b200 0.3.0 (sm_100a)"; }
int gamer_hydro_abi_version(void) { return GAMER_HYDRO_ABI_VERSION; }

}  // extern "C"
