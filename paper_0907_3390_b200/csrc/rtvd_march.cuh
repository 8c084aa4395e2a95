// rtvd_march.cuh — the 1-D relaxing-TVD row update as a register sliding window (device code, sm_100a).
//
// One thread owns one row of 22 cells along the sweep direction and marches along it once.  Everything that the
// paper's kernel keeps in shared memory for neighbour exchange (the cell-centred fluxes) lives in
// the registers of the marching thread instead: each cell's freezing speed and F^R/F^L are computed exactly once,
// each flux difference is shared by the two interfaces that use it, and no shuffle or shared-memory traffic is
// needed beyond loading the 5 conserved variables of a cell once (+ once more for the final update) and storing the
// 5 updated values.
//
// Arithmetic (§2.2, Eqs.6-14; steps (a)-(f) of DESIGN.md).  With G^R = c u + F = 2 F^R, G^L = c u - F = 2 F^L
// (Eq.8; the factors 1/2 are folded into dt/dh, which is exact in binary floating point):
//   first-order interface flux    2 F_{n+1/2}   = G^R_n - G^L_{n+1}                               (:143, :170)
//   half step (Eq.13)             u^h_n         = u_n - (k/4) (2F_{n+1/2} - 2F_{n-1/2})
//   limited fluxes (Eqs.9-12)     2 F^R_{n+1/2} = G^R_n     + a b/(a+b) if a b > 0,  a = G^R_n - G^R_{n-1}, b = G^R_{n+1} - G^R_n
//                                 2 F^L_{n+1/2} = G^L_{n+1} + a b/(a+b) if a b > 0,  a = G^L_{n+1} - G^L_{n+2}, b = G^L_n - G^L_{n+1}
//                                 (phi(a/4, b/4) = 2 (a/4)(b/4) / ((a+b)/4) = a b / (2 (a+b)); times 2 for the G scaling)
//   full step (Eq.14)             u'_n          = u_n - (k/2) (2F^h_{n+1/2} - 2F^h_{n-1/2})
// The limiter is a select on the sign of the product (reading R6): nothing computed from a+b is used
// unless a b > 0.
#pragma once
#include <cuda_runtime.h>

#ifndef GAMER_MARCH_UNROLL
#define GAMER_MARCH_UNROLL 2     /* pairs of cells per loop body */
#endif

namespace gamer {

constexpr int MARCH_UNROLL = GAMER_MARCH_UNROLL;
constexpr int NCOMP = 5;
constexpr int PS = 16;
constexpr int NG = 3;
constexpr int NP = PS + 2 * NG;   // 22

struct GasConst {
    float gm1;    // gamma - 1
    float ggm1;   // gamma (gamma - 1)
    float kq;     // (dt/dh) / 4
    float kh;     // (dt/dh) / 2
    float kq_gm1;   // kq (gamma - 1)
    float kq_sg;    // kq sqrt(gamma (gamma - 1))
};

__device__ __forceinline__ float rcp_fast(float x) {
    float r;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}
__device__ __forceinline__ float sqrt_fast(float x) {
    float r;
    asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}

// Cell-centred G^R = c u + F and G^L = c u - F of one cell; u = (rho, m_n, m_t1, m_t2, e), m_n normal to the sweep.
// c = |v_n| + c_s (reading R1), P from all three momenta (Eqs.4-5, reading R2).
// (Blackwell's packed FFMA2/FADD2/FMUL2 were tried for the 5-vector operations: fewer instructions, no gain — a packed
// instruction holds the issue port for two cycles on this part.)
__device__ __forceinline__ void cell_split_flux(const float (&u)[NCOMP], const GasConst& gc, float (&gr)[NCOMP],
                                                float (&gl)[NCOMP]) {
    const float rinv = rcp_fast(u[0]);
    const float v = __fmul_rn(u[1], rinv);
    float q = __fmul_rn(u[2], u[2]);
    q = fmaf(u[3], u[3], q);
    q = fmaf(u[1], u[1], q);
    const float hk = __fmul_rn(0.5f, rinv);
    const float eint = fmaf(-q, hk, u[4]);          // e - rho v^2 / 2
    const float P = __fmul_rn(gc.gm1, eint);
    const float cs = sqrt_fast(__fmul_rn(__fmul_rn(gc.ggm1, eint), rinv));
    const float c = __fadd_rn(fabsf(v), cs);
#ifdef GAMER_SPLIT_CUF
    float F[NCOMP];
    F[0] = u[1];
    F[1] = fmaf(u[1], v, P);
    F[2] = u[2] * v;
    F[3] = u[3] * v;
    F[4] = (u[4] + P) * v;
#pragma unroll
    for (int k = 0; k < NCOMP; ++k) {
        gr[k] = fmaf(c, u[k], F[k]);
        gl[k] = fmaf(c, u[k], -F[k]);
    }
#else
    // G^R = c u + F = u (c + v) + (0, P, 0, 0, P v),  G^L = c u - F = u (c - v) - (0, P, 0, 0, P v):  F = u v + (0, P, 0, 0, P v).
    // Two instructions fewer per cell than c u +- F, and every multiply shares the operand c +- v with its neighbours
    // (operand-reuse cache: the register file delivers two operands per clock, a 3-register FFMA takes 1.5).
    // Explicit intrinsics: no FMA contraction, so every cell is computed by the same operations wherever it sits in the
    // pipeline (a uniform state must come back bit-exactly).
    const float cp = __fadd_rn(c, v), cm = __fsub_rn(c, v);
    const float Pv = __fmul_rn(P, v);
    gr[0] = __fmul_rn(u[0], cp);
    gr[1] = fmaf(u[1], cp, P);
    gr[2] = __fmul_rn(u[2], cp);
    gr[3] = __fmul_rn(u[3], cp);
    gr[4] = fmaf(u[4], cp, Pv);
    gl[0] = __fmul_rn(u[0], cm);
    gl[1] = fmaf(u[1], cm, -P);
    gl[2] = __fmul_rn(u[2], cm);
    gl[3] = __fmul_rn(u[3], cm);
    gl[4] = fmaf(u[4], cm, -Pv);
#endif
}

// base + a b / (a + b) if a b > 0, else base     (sgn = +1)   |   base - a b / (a + b) ...   (sgn = -1)
// A select on the sign of the product, never a mask (reading R6).
template <int SGN>
__device__ __forceinline__ float limited(float base, float a, float b) {
    const float p = a * b;
    const float r = rcp_fast(a + b);
    const float x = fmaf(SGN > 0 ? p : -p, r, base);
    return p > 0.f ? x : base;
}

// Marches one row.  `src[q]` points to cell 0 of component q (row-local order), element n at src[q][n * STRIDE].
// Sink must provide:
//   template <int ODD> void cell(int j, const float (&u)[5])   updated cell j = 3..18 (ODD = j & 1, static),
//                                            row-local component order
//   void face(int p, const float (&f)[5])   true flux F^{t+dt/2} through interface 2|3 (p=0), 10|11 (1), 18|19 (2);
//                                            called only if WANT_FACE
// A Sink may overwrite the row in place at index j (the march never reads cell j again).
//
// The march is a software pipeline of depth 6: at step n it loads cell n, forms the first-order flux through (n-1|n),
// the midpoint state of cell m = n-1, the limited fluxes through (m-2|m-1) and the new value of cell m-2 = n-3.
// Steps 0..5 fill the pipeline (PH = n, statically pruned); steps 6..21 are identical and run as a rolled loop
// (PH = 6) so that the code of all three sweeps stays resident in the instruction cache.
template <int STRIDE, bool WANT_FACE, class Sink>
struct RowMarch {
    float u1[NCOMP], u2[NCOMP], u3[NCOMP];     // u_{n-1}, u_{n-2}, u_{n-3} (the originals, kept for Eqs.13-14)
    float gr1_prev[NCOMP];                     // G^R_{n-1} at time t
    float f_prev[NCOMP];                       // 2F through (n-2|n-1)
    float gr2_prev[NCOMP], gl2_prev[NCOMP];    // midpoint G^R, G^L of cell m-1
    float gr2_pp[NCOMP];                       // midpoint G^R of cell m-2
    float ar1[NCOMP], ar2[NCOMP], al1[NCOMP];  // ar1 = G^R_{m-1}-G^R_{m-2}, ar2 = G^R_{m-2}-G^R_{m-3}, al1 likewise for L
    float fh_prev[NCOMP];                      // 2F^h through the previous limited interface

    template <int PH>
    __device__ __forceinline__ void step(const float (&u)[NCOMP], int n, const GasConst& gc, Sink& sink) {
        float gr1[NCOMP], gl1[NCOMP];
        cell_split_flux(u, gc, gr1, gl1);                                   // (a)
        if (PH >= 1) {
            float f[NCOMP];
#pragma unroll
            for (int k = 0; k < NCOMP; ++k) f[k] = gr1_prev[k] - gl1[k];     // (b) interface (n-1 | n)
            if (PH >= 2) {                                                  // midpoint cell m = n-1
                float uh[NCOMP], gr2[NCOMP], gl2[NCOMP];
#pragma unroll
                for (int k = 0; k < NCOMP; ++k) uh[k] = fmaf(-gc.kq, f[k] - f_prev[k], u1[k]);   // (c)
                cell_split_flux(uh, gc, gr2, gl2);                          // (d)
                if (PH >= 3) {                                              // m >= 2
                    float ar0[NCOMP], al0[NCOMP];
#pragma unroll
                    for (int k = 0; k < NCOMP; ++k) {
                        ar0[k] = gr2[k] - gr2_prev[k];                      // G^R_m - G^R_{m-1}
                        al0[k] = gl2[k] - gl2_prev[k];                      // G^L_m - G^L_{m-1}
                    }
                    if (PH >= 5) {                                          // m >= 4: (e) interface (m-2 | m-1)
                        float fh[NCOMP];
#pragma unroll
                        for (int k = 0; k < NCOMP; ++k) {
                            const float xr = limited<+1>(gr2_pp[k], ar2[k], ar1[k]);
                            // a = G^L_{m-1}-G^L_m = -al0, b = G^L_{m-2}-G^L_{m-1} = -al1: a b = al0 al1, a+b = -(al0+al1)
                            const float xl = limited<-1>(gl2_prev[k], al0[k], al1[k]);
                            fh[k] = xr - xl;
                        }
                        if (WANT_FACE) {
                            const int i = n - 3;                            // interface (i | i+1), i = m-2
                            if (i == NG - 1 || i == NG + PS / 2 - 1 || i == NG + PS - 1) {
                                float ff[NCOMP];
#pragma unroll
                                for (int k = 0; k < NCOMP; ++k) ff[k] = 0.5f * fh[k];
                                sink.face(i == NG - 1 ? 0 : (i == NG + PS - 1 ? 2 : 1), ff);
                            }
                        }
                        if (PH >= 6) {                                      // m >= 5: (f) cell j = m-2 = n-3
                            float un[NCOMP];
#pragma unroll
                            for (int k = 0; k < NCOMP; ++k) un[k] = fmaf(-gc.kh, fh[k] - fh_prev[k], u3[k]);
                            sink.template cell<(PH + 1) & 1>(n - 3, un);      // parity of j = n-3 is static
                        }
#pragma unroll
                        for (int k = 0; k < NCOMP; ++k) fh_prev[k] = fh[k];
                    }
#pragma unroll
                    for (int k = 0; k < NCOMP; ++k) {
                        ar2[k] = ar1[k];
                        ar1[k] = ar0[k];
                        al1[k] = al0[k];
                    }
                }
#pragma unroll
                for (int k = 0; k < NCOMP; ++k) {
                    gr2_pp[k] = gr2_prev[k];
                    gr2_prev[k] = gr2[k];
                    gl2_prev[k] = gl2[k];
                }
            }
#pragma unroll
            for (int k = 0; k < NCOMP; ++k) f_prev[k] = f[k];
        }
#pragma unroll
        for (int k = 0; k < NCOMP; ++k) {
            if (PH >= 2) u3[k] = u2[k];
            if (PH >= 1) u2[k] = u1[k];
            u1[k] = u[k];
            gr1_prev[k] = gr1[k];
        }
    }

    // Cells are fetched two at a time (n even, n+1): a row along x is read with 64-bit shared-memory loads.
    template <int PH0, int PH1>
    __device__ __forceinline__ void pair(const float* const (&src)[NCOMP], int n, const GasConst& gc, Sink& sink) {
        float ua[NCOMP], ub[NCOMP];
        if (STRIDE == 1) {
#pragma unroll
            for (int k = 0; k < NCOMP; ++k) {
                const float2 t = *reinterpret_cast<const float2*>(src[k] + n);
                ua[k] = t.x;
                ub[k] = t.y;
            }
        } else {
#pragma unroll
            for (int k = 0; k < NCOMP; ++k) {
                ua[k] = src[k][n * STRIDE];
                ub[k] = src[k][(n + 1) * STRIDE];
            }
        }
        step<PH0>(ua, n, gc, sink);
        step<PH1>(ub, n + 1, gc, sink);
    }

    __device__ __forceinline__ void run(const float* const (&src)[NCOMP], const GasConst& gc, Sink& sink) {
        pair<0, 1>(src, 0, gc, sink);
        pair<2, 3>(src, 2, gc, sink);
        pair<4, 5>(src, 4, gc, sink);
#pragma unroll MARCH_UNROLL
        for (int n = 6; n < NP; n += 2) pair<6, 6>(src, n, gc, sink);
    }
};

template <int STRIDE, bool WANT_FACE, class Sink>
__device__ __forceinline__ void rtvd_march(const float* const (&src)[NCOMP], const GasConst& gc, Sink& sink) {
    RowMarch<STRIDE, WANT_FACE, Sink> m;
    m.run(src, gc, sink);
}

}  // namespace gamer
