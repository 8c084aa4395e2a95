/* gamer_probes.h — measurement aids for the roofline analysis of the hydro pass (bench.py).
 * NOT part of the hydro path and not part of the product library: they live in libgamer_probes.so
 * (paper_0907_3390_b200/csrc/probes.cu), which only bench.py and one test load.
 * All functions are SYNCHRONOUS, run on the current device's default stream, allocate and free a few hundred KB of
 * device memory themselves, and return 0 or a negative code (message: gamer_probe_last_error(), thread-local). */
#ifndef GAMER_PROBES_H
#define GAMER_PROBES_H

#if defined(__GNUC__)
#define GAMER_PROBE_API __attribute__((visibility("default")))
#else
#define GAMER_PROBE_API
#endif

#ifdef __cplusplus
extern "C" {
#endif

enum gamer_probe_status { GAMER_PROBE_OK = 0, GAMER_PROBE_EINVAL = -1, GAMER_PROBE_ECUDA = -3 };

/* FMA-only micro-benchmark of the FP32 pipe: 4 CTAs of 512 threads per SM, 16 independent fused
 * multiply-add chains per thread, 2048 steps each, launched repeats + 1 times (the first is a warm-up), timed with CUDA
 * events.  *tflops receives the best launch's 2 x FMA count / time in TFLOP/s; *lane_fma_per_clk_per_sm (optional) the
 * same as FMAs per clock per SM if sm_mhz (the SM clock the caller observed, MHz) is > 0 — 128 is the unit count of the
 * part.  d_sink: one float of device memory (never written in practice). */
GAMER_PROBE_API int gamer_probe_fp32_peak(int repeats, float* d_sink, double* tflops, double* lane_fma_per_clk_per_sm,
                                          double sm_mhz);

/* Issue-rate probes (why the pass is bound by instruction issue and register-file reads).
 *   what = 0: *cycles = clocks one SM sub-partition needs per warp-wide FMA whose three source operands are three
 *             different registers (an FMA with two reused operands takes 1.05), 4 warps per sub-partition;
 *   what = 1, 2, 3: *cycles = clocks per warp-march (one warp, 32 rows of 22 cells, the production row march along x, y,
 *             z) and sub-partition slot when warps_per_smsp = 1..4 warps per sub-partition run marches back to back
 *             on a resident group with no loads and no barriers — the steady-state cost a schedule can at best reach.
 *             The marches run with dt = 0, so that warps sharing rows rewrite identical bits and every repetition sees
 *             the same physical state; the call fails if the state changed.
 * Values are means over the SMs of the current device, read from clock64 inside the kernels. */
GAMER_PROBE_API int gamer_probe_issue(int what, int warps_per_smsp, double* cycles);

GAMER_PROBE_API const char* gamer_probe_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* GAMER_PROBES_H */
