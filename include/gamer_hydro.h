/* gamer_hydro.h — C ABI of the batched relaxing-TVD hydrodynamic update of GAMER (arXiv 0907.3390) for B200 (sm_100a).
 *
 * The operation ("GPU hydrodynamic solver", §3.1): many independent, fixed-size patch groups are
 * advanced by one dimensionally split pass (three 1-D sweeps) of the second-order relaxing TVD scheme of PAPER.md
 * §2.2 (Eqs.6-14, :126-172): first-order upwind half step, van-Leer-limited second-order full step, on the five
 * conserved variables (rho, rho v_x, rho v_y, rho v_z, e), fp32 (:448).
 *
 * LAYOUT (the contract)
 *   in [g][v][z][y][x]   g slowest, x fastest; v in {0:rho, 1:rho v_x, 2:rho v_y, 3:rho v_z, 4:e};
 *                        extents 22 = 2*8 + 2*3 in x, y, z (:324): 16 interior cells (two 8-cell patches) plus
 *                        `ghost` = 3 cells on each side (7-point stencil, :178).  Interior = indices 3..18.
 *                        212 960 bytes per group.
 *   out[g][v][k][j][i]   extents 16; out[g][v][k][j][i] is padded cell (k+3, j+3, i+3).  No ghost zones are written
 *                        (:344).  81 920 bytes per group.
 *   face_flux[g][d][p][v][b][a]  (optional) time-centred fluxes F^{t+dt/2} of Eq.14 through the three planes normal to
 *                        axis d (0:x, 1:y, 2:z) that bound the two 8-cell patch layers — padded interfaces 2|3 (p=0),
 *                        10|11 (p=1), 18|19 (p=2) — on the 16x16 interior transverse cells, (b,a) = the two
 *                        transverse interior indices, slower first: d=x:(k,j), d=y:(k,i), d=z:(j,i).  These are the
 *                        "fluxes across the boundaries of each patch" of :340/:344-346.  46 080 bytes per group.
 *   group_maxspeed[g]    (optional) max over the group's 16^3 UPDATED cells of c_s + max(|v_x|,|v_y|,|v_z|), the
 *                        denominator of the CFL condition Eq.30 (:418-426: "a single floating-point value per patch
 *                        group").
 *
 * WHAT gamer_hydro_advance* DO NOT DO: they do not fill ghost zones (the caller's "preparation step", :322 — see
 * gamer_hydro_ghost_fill for the single-level case), they do not choose dt (:418-426 — they only offer the per-group
 * reduction; gamer_hydro_run_uniform does), and nothing applies a density or pressure floor (the
 * paper names none): non-physical input (rho <= 0 or P <= 0) yields NaN/Inf in the affected cells, silently.
 *
 * NUMBER RANGE (fp32 passes): reciprocals and square roots are the hardware approximations with flush-to-zero
 * (rcp.approx.ftz, sqrt.approx.ftz; about 1 ulp, the parity bars of DESIGN.md hold with them): a DENORMAL operand or
 * result of those two operations is taken as zero.  That touches densities above about 8.5e37 (1/rho would be
 * denormal: it becomes 0, and velocity and pressure with it) and specific internal energies gamma (gamma-1) e_int/rho
 * below about 1.2e-38 (the sound speed becomes 0).  The CPU oracle keeps denormals, so parity with it is claimed on the
 * normal range only; every workload of BASELINE.json lies many decades inside it.  The fp64 passes do not flush.
 *
 * OWNERSHIP: the caller owns every buffer.  `d_*` are DEVICE pointers (cudaMalloc or equivalent) valid on the
 * device of `stream`; `h_*` are HOST pointers.  Nothing is allocated, freed or synchronised by gamer_hydro_advance*:
 * they only enqueue work on `stream` (NULL = the legacy default stream).  `d_in` is never written.  Input, outputs
 * and scratch must not overlap (checked on the address ranges: results of finished groups are streamed out while later
 * groups are still being read).
 *
 * ERRORS: every function returns GAMER_OK (0) or a negative gamer_status; nothing aborts or throws.  After a
 * failure gamer_last_error() returns a thread-local, statically stored, human-readable message.
 *   ghost != 3                                                        -> GAMER_EUNSUPPORTED  (stencil, :178)
 *   n_groups < 0; a required pointer NULL while n_groups > 0; a pointer not 16-byte aligned;
 *   !(dh > 0); !(dt >= 0); !(gamma > 1); backward not 0/1;
 *   address ranges of input / output / optional outputs / scratch that intersect       -> GAMER_EINVAL
 *   n_groups == 0                                                     -> GAMER_OK, nothing enqueued
 *   a CUDA runtime error (launch, attribute, copy)                    -> GAMER_ECUDA
 *   an allocation failure inside gamer_hydro_pipeline_run             -> GAMER_ENOMEM
 */
#ifndef GAMER_HYDRO_H
#define GAMER_HYDRO_H

#include <stddef.h>

#if defined(__GNUC__)
#define GAMER_API __attribute__((visibility("default")))
#else
#define GAMER_API
#endif

#ifdef __cplusplus
extern "C" {
#endif

enum gamer_status {
    GAMER_OK = 0,
    GAMER_EINVAL = -1,
    GAMER_EUNSUPPORTED = -2,
    GAMER_ECUDA = -3,
    GAMER_ENOMEM = -4
};

/* One forward pass (sweeps x, then y, then z) over n_groups patch groups, each sweep with the full dt
 * (Eqs.13-14).  d_in, d_out: device pointers, layouts above.  dt, dh: time step and cell size (only dt/dh enters).
 * gamma: ratio of specific heats (Eq.5).  stream: a cudaStream_t passed as void*.  Asynchronous. */
GAMER_API int gamer_hydro_advance(const float* d_in, float* d_out, long long n_groups, int ghost,
                        float dt, float dh, float gamma, void* stream);

/* Same with the paper's sweep-direction boolean (:326): backward = 0 sweeps x,y,z; backward = 1 sweeps z,y,x.
 * d_face_flux and d_group_maxspeed are optional device outputs (NULL = not computed), layouts above. */
GAMER_API int gamer_hydro_advance_ex(const float* d_in, float* d_out, long long n_groups, int ghost,
                           float dt, float dh, float gamma, int backward,
                           float* d_face_flux, float* d_group_maxspeed, void* stream);

/* Buffer sizes in floats: n*5*(16+2*ghost)^3, n*5*16^3, n*3*3*5*16*16.  0 if n_groups < 0 or ghost < 0. */
GAMER_API size_t gamer_hydro_in_floats(long long n_groups, int ghost);
GAMER_API size_t gamer_hydro_out_floats(long long n_groups);
GAMER_API size_t gamer_hydro_face_flux_floats(long long n_groups);

/* Secondary subsystem — the stream pipeline of PAPER.md:350-356 / Fig.5: n_groups groups in HOST memory are cut
 * into chunks of groups_per_chunk (the paper's N_g) that travel round-robin through n_streams (N_s) CUDA streams,
 * each doing one host->device copy, one kernel, one device->host copy, so that copies overlap kernels of other
 * chunks.  h_in / h_out: host pointers, same layouts as d_in / d_out; page-locked (pinned) memory is needed for the
 * copies to overlap — pageable memory works but serialises.  The call owns its device staging buffers
 * (n_streams * groups_per_chunk groups) and streams: it allocates them on first use, keeps them for the next call
 * (grown if that call needs more) and gamer_hydro_pipeline_release() frees them.  It runs on the current device and is
 * SYNCHRONOUS: on return h_out is complete.  Concurrent calls from several host threads are serialised.
 * 1 <= n_streams <= 16, groups_per_chunk >= 1, else GAMER_EINVAL. */
GAMER_API int gamer_hydro_pipeline_run(const float* h_in, float* h_out, long long n_groups, int ghost,
                             float dt, float dh, float gamma, int backward,
                             long long groups_per_chunk, int n_streams);

/* Frees the streams and staging buffers that gamer_hydro_pipeline_run keeps on the current device (after waiting for
 * them).  A no-op if there are none. */
GAMER_API int gamer_hydro_pipeline_release(void);

/* NEXT-3 — device-side preparation step for a SINGLE-LEVEL tiling ("ghost zones ... filled by directly
 * copying from the sibling patches"; :430-432, :647 name this CPU step the bottleneck of the code).  gx*gy*gz groups tile
 * a box of 16gx x 16gy x 16gz cells, group index g = (kz*gy + ky)*gx + kx.  d_interior: [g][v][16][16][16] (the layout
 * of d_out), read only.  d_padded: [g][v][22][22][22] (the layout of d_in); every interior cell is written from the
 * group's own interior and every ghost cell from the interior of the neighbouring group.  bc_x, bc_y, bc_z per axis:
 * 0 = periodic box; 1 = "keep": ghost cells that lie beyond that end of the box are NOT written, they keep what the
 * caller put there (a Dirichlet boundary).  Pure data movement, bit exact.  Asynchronous on `stream`.
 * gx, gy, gz < 1, a flag other than 0/1, a NULL or misaligned pointer -> GAMER_EINVAL. */
GAMER_API int gamer_hydro_ghost_fill(const float* d_interior, float* d_padded, int gx, int gy, int gz,
                           int bc_x, int bc_y, int bc_z, void* stream);

/* NEXT-3 — multi-step driver on such a box, entirely on the device (no host round trip between steps).
 * order = 0: each of the n_steps steps does: dt = cfl * dh / max over ALL padded cells of (c_s + max_i |v_i|) (Eq.30,
 *   PAPER.md:418-426; fp32, reading R10); one forward pass d_padded -> d_interior with that dt (read from
 *   device memory, constants formed exactly as on the host); gamer_hydro_ghost_fill(d_interior -> d_padded).
 * order = 1: the paper's full step ("a forward sweep in the order xyz, and follows a backward sweep
 *   in the order zyx.  The same time step must be employed by these two sweeps to maintain the second-order
 *   accuracy"): dt as above; forward pass; ghost fill; backward pass (z,y,x) with the SAME dt; ghost fill.  A step
 *   advances the state by 2 dt, and the next dt is evaluated after the backward sweep (:424).
 * The maximum is taken in one pass over the initial state; from then on it is the maximum of the per-group speeds of
 * the updated interiors that the last pass of a step writes as a by-product (:426: "a single floating-point value per
 * patch group") and of the ghost cells beyond "keep" ends, which never change — the same set of cells.  On return
 * (asynchronous on `stream`) d_padded holds the ghost-filled state after n_steps and d_interior its interiors.
 * d_work: 4 + gx*gy*gz floats of device scratch, 16-byte aligned.  d_dt_log: optional device array of n_steps floats
 * that receives the dt of every step (NULL = off).  order other than 0/1, n_steps < 0, !(cfl > 0) -> GAMER_EINVAL. */
GAMER_API int gamer_hydro_run_uniform(float* d_padded, float* d_interior, int gx, int gy, int gz,
                            int bc_x, int bc_y, int bc_z, int n_steps, int order, float cfl, float dh, float gamma,
                            float* d_work, float* d_dt_log, void* stream);

/* gamer_hydro_run_uniform for callers that must not allocate device memory.
 *
 * WHO THIS IS FOR.  gamer_hydro_run_uniform needs 4 + gx*gy*gz floats of device scratch (d_work) and leaves it to the
 * caller to provide them.  Some callers have nowhere to get them from once the run has started: a simulation code that
 * hands all free device memory to its own pool at start-up, so that a later cudaMalloc simply fails; a time-step loop
 * that other streams run beside, where an allocation would stall every one of them (cudaFree waits for all work on the
 * device, cudaMalloc may); a plug-in that runs inside someone else's process and is told not to touch the allocator.  For them the
 * scratch lives inside the library: a file-scope __device__ array of 4 + GAMER_NOALLOC_MAX_GROUPS floats (262 160
 * bytes).  It is part of the library image, so EVERY GPU on which the process uses this library holds those bytes
 * from the moment the library's code is loaded there until the process exits, whether or not this entry point is
 * ever called.
 *
 * Same operation, arguments, layouts, results (bit for bit) and error conventions as gamer_hydro_run_uniform, minus
 * d_work.  The caller still owns and passes the state (d_padded, d_interior) and the optional d_dt_log.  Differences:
 *   - gx*gy*gz > GAMER_NOALLOC_MAX_GROUPS -> GAMER_EINVAL ("... exceeds the built-in scratch ...").  Nothing is
 *     enqueued.  Use gamer_hydro_run_uniform with your own d_work for larger boxes.
 *   - The call itself never calls cudaMalloc, cudaFree or any library routine that allocates; it only enqueues a
 *     16-byte memset and kernels on `stream`.
 *   - SET-UP: the first call on each device (with that device current) asks the runtime for the device address of the
 *     array (cudaGetSymbolAddress; the result is kept per device) and opts the kernels into their shared-memory size.
 *     If the library's code was not yet loaded on that device, that first call loads it.  Make this first call during
 *     initialisation — with n_steps = 0 it changes nothing — and before any stream capture is begun.
 *   - ONE array per device, shared by all calls: the four accumulator words are cleared at the start of every call
 *     (stream-ordered), and the per-group speeds are written before they are read, so nothing of an earlier call leaks
 *     into a later one that follows it in stream order.  Two calls whose work OVERLAPS on the same GPU (different
 *     streams, or different host threads) race on the array and compute wrong time steps: serialise them, or give all
 *     but one of them gamer_hydro_run_uniform with separate d_work. */
#define GAMER_NOALLOC_MAX_GROUPS 65536
GAMER_API int gamer_hydro_run_uniform_noalloc(float* d_padded, float* d_interior, int gx, int gy, int gz,
                            int bc_x, int bc_y, int bc_z, int n_steps, int order, float cfl, float dh, float gamma,
                            float* d_dt_log, void* stream);
/* GAMER_NOALLOC_MAX_GROUPS as the library was built (for callers that do not compile against this header). */
GAMER_API long long gamer_hydro_noalloc_max_groups(void);

/* NEXT-4 — one pass in DOUBLE precision (the paper switches to double for its convergence tests).
 * Same operation, layouts and error conventions as gamer_hydro_advance_ex with double arrays: d_in
 * [g][v][22][22][22] (425 920 B per group), d_out [g][v][16][16][16]; backward = 0 sweeps x,y,z, 1 sweeps z,y,x;
 * d_face_flux [g][3][3][5][16][16] and d_group_maxspeed [g] are the optional outputs of gamer_hydro_advance_ex in
 * double (NULL = off).  Reciprocals and square roots are accurate to about 1 ulp.  A padded group does not fit in
 * shared memory in double precision: the pass is cut into halves and the rows of the last sweep wait in tensor memory
 * (DESIGN.md 8c); no device scratch is needed.
 * TENSOR MEMORY IS HELD EXCLUSIVELY: each persistent CTA of these kernels allocates all 512 tensor-memory columns of
 * its SM (tcgen05.alloc, which blocks until they are free) and keeps them until the kernel ends.  Anything else that
 * uses tensor memory on the same GPU at the same time — a cuBLAS / CUTLASS GEMM of the same process on another
 * stream — waits for this kernel to finish on the SMs it occupies, or makes this kernel wait for it.  Do not overlap
 * the fp64 passes with tensor-core GEMMs if either is latency critical.  (The fp32 passes use no tensor memory.)
 * A device that offers less than 225 408 B of shared memory per block -> GAMER_EUNSUPPORTED. */
GAMER_API int gamer_hydro_advance_f64_ex(const double* d_in, double* d_out, long long n_groups, int ghost,
                            double dt, double dh, double gamma, int backward, double* d_face_flux,
                            double* d_group_maxspeed, void* stream);

/* Launch geometry the library will use on the current device, for reporting: any pointer may be NULL.
 * grid = number of persistent CTAs for n_groups, block = threads per CTA, smem = dynamic shared memory per CTA in
 * bytes, regs = registers per thread of the kernel. */
GAMER_API int gamer_hydro_launch_info(long long n_groups, int* grid, int* block, int* smem_bytes, int* regs_per_thread);

GAMER_API const char* gamer_last_error(void);   /* thread-local, static storage; "" if the last call on this thread succeeded */
GAMER_API const char* gamer_version(void);      /* static string */

/* Binary-interface revision of the library that is loaded; compare with GAMER_HYDRO_ABI_VERSION of the header you
 * compiled against and refuse to run on a mismatch.  It is bumped whenever an exported function changes its argument
 * list or is removed: a caller built against an older header would still link and would silently pass shifted
 * arguments.  History: 1 = round 1; 2 = gamer_hydro_run_uniform gained `order` (between n_steps and cfl);
 * 3 = gamer_hydro_advance_f64 and gamer_hydro_f64_scratch_doubles removed (use gamer_hydro_advance_f64_ex with NULL
 * optional outputs; no device scratch exists any more), the measurement probes moved to libgamer_probes
 * (include/gamer_probes.h), gamer_hydro_run_uniform_noalloc added. */
#define GAMER_HYDRO_ABI_VERSION 3
GAMER_API int gamer_hydro_abi_version(void);

#ifdef __cplusplus
}
#endif
#endif /* GAMER_HYDRO_H */
