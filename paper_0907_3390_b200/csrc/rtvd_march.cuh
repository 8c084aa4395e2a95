// rtvd_march.cuh — the 1-D relaxing-TVD row update (§2.2, Eqs.6-14) as a register sliding window (sm_100a).
//
// One thread owns one row of 22 cells along the sweep direction and marches along it once.  How much is computed and
// carried per cell:
//
//  * half step (Eqs.8 and 13, :138, :168).  With G^R = c u + F = u (c + v) + Pi, G^L = c u - F = u (c - v) - Pi,
//    Pi = (0, P, 0, 0, P v), and q = (dt/dh)/4, substituting the first-order fluxes 2F_{n+1/2} = G^R_n - G^L_{n+1} into
//    Eq.13 gives
//        u^h_n = u_n - q (G^R_n + G^L_n) + q G^L_{n+1} + q G^R_{n-1}
//              = (1 - 2 q c_n) u_n  +  q (c - v)_{n+1} u_{n+1}  +  q (c + v)_{n-1} u_{n-1}  +  q (Pi_{n-1} - Pi_{n+1}).
//    So the time-t split fluxes are never formed: each cell contributes three scalars (q(c+v), q(c-v), 1-2qc) and
//    the two non-zero entries of q Pi, and a midpoint component costs 3 FMA-pipe instructions (4 for m_n and e).
//  * limited fluxes (Eqs.9-12).  The right-moving flux through (m-1|m) only needs cells m-2..m, so it is formed one
//    step ahead of the left-moving flux through the same interface and carried; every window is then one or two deep.
//
// Every cell is computed by the same instruction sequence wherever it sits in the row, so a uniform state (and a
// transverse sweep of 1-D data) comes back bit-exactly: equal midpoint states give equal fluxes and Eq.14 subtracts 0.
#pragma once
#include <cuda_runtime.h>

#ifndef GAMER_MARCH_UNROLL
#define GAMER_MARCH_UNROLL 3     /* pairs of cells per loop body (measured: 1: 113.5, 2: 105.4, 3: 104.5, 4: 108.4 ns/group) */
#endif

#ifndef GAMER_MARCH_UNROLL_F64
#define GAMER_MARCH_UNROLL_F64 2       /* pairs per body in fp64 (measured: 1: 294, 2: 288, 3: 481 ns/group forward) */
#endif

namespace gamer {

constexpr int MARCH_UNROLL = GAMER_MARCH_UNROLL;
constexpr int NCOMP = 5;
constexpr int PS = 16;
constexpr int NG = 3;
constexpr int NP = PS + 2 * NG;   // 22

// T = float is the paper's precision and the hot path; T = double is the variant the paper switches to
// for its convergence tests (:452).  The arithmetic is written once, on the overloads below.
template <class T>
struct GasConstT {
    T gm1;      // gamma - 1
    T ggm1;     // gamma (gamma - 1)
    T kq;       // (dt/dh) / 4
    T kh;       // (dt/dh) / 2
    T kq_gm1;   // kq (gamma - 1)
    T kq_sg;    // kq sqrt(gamma (gamma - 1))
    T dh;       // cell size            } only read when the time step comes from device memory
    T sg;       // sqrt(gamma (gamma-1)) }
};
using GasConst = GasConstT<float>;

// the constants of one pass, formed on the host in fp32 (the kernels that read dt from device memory repeat exactly this)
inline GasConst make_const(float dt, float dh, float gamma) {
    GasConst gc;
    const float k = dt / dh;
    gc.gm1 = gamma - 1.0f;
    gc.ggm1 = gamma * (gamma - 1.0f);
    gc.kq = 0.25f * k;
    gc.kh = 0.5f * k;
    gc.dh = dh;
    gc.sg = sqrtf(gc.ggm1);
    gc.kq_gm1 = gc.kq * gc.gm1;
    gc.kq_sg = gc.kq * gc.sg;
    return gc;
}

// explicitly rounded (never contracted) operations and fused multiply-add, per precision
__device__ __forceinline__ float mul_rn(float a, float b) { return __fmul_rn(a, b); }
__device__ __forceinline__ float add_rn(float a, float b) { return __fadd_rn(a, b); }
__device__ __forceinline__ float sub_rn(float a, float b) { return __fsub_rn(a, b); }
__device__ __forceinline__ float fma_rn(float a, float b, float c) { return fmaf(a, b, c); }
__device__ __forceinline__ float abs_of(float a) { return fabsf(a); }
__device__ __forceinline__ double mul_rn(double a, double b) { return __dmul_rn(a, b); }
__device__ __forceinline__ double add_rn(double a, double b) { return __dadd_rn(a, b); }
__device__ __forceinline__ double sub_rn(double a, double b) { return __dsub_rn(a, b); }
__device__ __forceinline__ double fma_rn(double a, double b, double c) { return fma(a, b, c); }
__device__ __forceinline__ double abs_of(double a) { return fabs(a); }

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

// Double precision: hardware seed (relative error 2^-20) and one third-order step (reciprocal: error e^3 = 2^-60) or
// its counterpart for the square root (error 5/16 e^3) — about 1 ulp, a fifth of the instructions of an IEEE division or square root.
__device__ __forceinline__ double rcp_fast(double x) {
    double r;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
    const double e = fma(-x, r, 1.0);          // 1/x = r / (1 - e) = r (1 + e + e^2 + ...): third order, |e| <= 2^-20
    return fma(r, fma(e, e, e), r);
}
__device__ __forceinline__ double sqrt_fast(double x) {
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    // sqrt x = x y (1 - e)^(-1/2), e = 1 - x y^2: x y (1 + e/2 + 3 e^2/8), third order, |e| <= 2^-19  (x > 0: P > 0 is
    // the caller's duty)
    const double s = x * y;
    const double e = fma(-s, y, 1.0);
    return fma(s, fma(0.375, e, 0.5) * e, s);
}

// What a cell at time t contributes to the half step of its neighbours and of itself (all times q = (dt/dh)/4).
template <class T>
struct HalfCoefT {
    T cp;     // q (c + v)
    T cm;     // q (c - v)
    T sig;    // 1 - 2 q c
    T P;      // q P
    T Pv;     // q P v
};

// u = (rho, m_n, m_t1, m_t2, e), m_n normal to the sweep.  c = |v_n| + c_s (reading R1), P from all three
// momenta (Eqs.4-5, reading R2).
template <class T>
__device__ __forceinline__ HalfCoefT<T> half_coef(const T (&u)[NCOMP], const GasConstT<T>& gc) {
    HalfCoefT<T> h;
    const T rinv = rcp_fast(u[0]);
    const T v = mul_rn(u[1], rinv);
    T q = mul_rn(u[2], u[2]);
    q = fma_rn(u[3], u[3], q);
    q = fma_rn(u[1], u[1], q);
    const T hk = mul_rn(T(0.5), rinv);
    const T eint = fma_rn(-q, hk, u[4]);                          // e - rho v^2 / 2
    h.P = mul_rn(gc.kq_gm1, eint);
    const T s = sqrt_fast(mul_rn(eint, rinv));
    const T vq = mul_rn(gc.kq, v);
    const T c = add_rn(abs_of(vq), mul_rn(gc.kq_sg, s));   // q (|v| + c_s)
    h.cp = add_rn(c, vq);
    h.cm = sub_rn(c, vq);
    h.sig = fma_rn(T(-2), c, T(1));
    h.Pv = mul_rn(h.P, v);
    return h;
}

// Cell-centred G^R = c u + F = u (c + v) + (0, P, 0, 0, P v) and G^L = c u - F = u (c - v) - (0, P, 0, 0, P v) of the
// midpoint state (2 F^R and 2 F^L of Eq.8).  Explicit intrinsics: no FMA contraction across cells.
template <class T>
__device__ __forceinline__ void cell_split_flux(const T (&u)[NCOMP], const GasConstT<T>& gc, T (&gr)[NCOMP],
                                                T (&gl)[NCOMP]) {
    const T rinv = rcp_fast(u[0]);
    const T v = mul_rn(u[1], rinv);
    T q = mul_rn(u[2], u[2]);
    q = fma_rn(u[3], u[3], q);
    q = fma_rn(u[1], u[1], q);
    const T hk = mul_rn(T(0.5), rinv);
    const T eint = fma_rn(-q, hk, u[4]);
    const T P = mul_rn(gc.gm1, eint);
    const T cs = sqrt_fast(mul_rn(mul_rn(gc.ggm1, eint), rinv));
    const T c = add_rn(abs_of(v), cs);
    const T cp = add_rn(c, v), cm = sub_rn(c, v);
    const T Pv = mul_rn(P, v);
    gr[0] = mul_rn(u[0], cp);
    gr[1] = fma_rn(u[1], cp, P);
    gr[2] = mul_rn(u[2], cp);
    gr[3] = mul_rn(u[3], cp);
    gr[4] = fma_rn(u[4], cp, Pv);
    gl[0] = mul_rn(u[0], cm);
    gl[1] = fma_rn(u[1], cm, -P);
    gl[2] = mul_rn(u[2], cm);
    gl[3] = mul_rn(u[3], cm);
    gl[4] = fma_rn(u[4], cm, -Pv);
}

// base + a b / (a + b) if a b > 0, else base     (sgn = +1)   |   base - a b / (a + b) ...   (sgn = -1)
// A select on the sign of the product, never a mask (reading R6).
template <int SGN, class T>
__device__ __forceinline__ T limited(T base, T a, T b) {
    const T p = a * b;
    const T r = rcp_fast(a + b);
    const T x = fma_rn(SGN > 0 ? p : -p, r, base);
    return p > T(0) ? x : base;
}

// Marches one row.  Src::load(n, ua, ub) fetches cells n (even) and n+1 of the row, row-local component order.
// Sink must provide:
//   template <int ODD> void cell(int j, const T (&u)[5])   updated cell j = 3..18 (ODD = j & 1, static),
//                                            row-local component order
//   void face(int p, const T (&f)[5])   true flux F^{t+dt/2} through interface 2|3 (p=0), 10|11 (1), 18|19 (2);
//                                            called only if WANT_FACE
// A Sink may overwrite the row in place at index j (the march never reads cell j again).
// Gate: gate.acquire(n) is called before cells n, n+1 are read and gate.release(n) once they are in registers.
//
// The march is a software pipeline in two independent halves per step.  Step n loads cell n and
//   stage A: forms the half-step coefficients of cell n and the midpoint state of cell n-1, which it latches;
//   stage B: takes the midpoint state of cell m = n-2 latched by the PREVIOUS step and forms its G^R, G^L, the
//            right-moving limited flux through (m-1|m), the left-moving one through (m-2|m-1), the total flux through
//            (m-2|m-1) and the new value of cell m-2 = n-4.
// Without the latch one step is a single dependency chain (coefficients -> midpoint state -> split fluxes -> limited
// fluxes -> new value) and a warp that shares its SM sub-partition with only one or two others (y and z sweeps)
// cannot fill the issue slots: latching cost 5 registers and one drain step per row and gained 3.4 %.
// Steps 0..7 fill the pipeline (PH = n, statically pruned); steps 8..21 are identical and run as a rolled loop
// (PH = 7), so that the code stays resident in the instruction cache; a last half step drains cell 18.
// PHASE4: the steady loop is written out in bodies of two pairs and Sink::cell<P> receives P = (j - 4) mod 4 — the position
// of the cell in a group of four, for a sink that collects four cells into one 128-bit store; otherwise P = j mod 2.
template <bool WANT_FACE, class Sink, class T = float, bool PHASE4 = false>
struct RowMarch {
    T u1[NCOMP], u2[NCOMP], u3[NCOMP], u4[NCOMP];   // u_{n-1} .. u_{n-4} (the originals, kept for Eqs.13-14)
    T sig1, cp1, P1, Pv1;                  // 1 - 2 q c, q (c+v), q P, q P v of cell n-1
    T cp2, P2, Pv2;                        // ... of cell n-2
    T uhl[NCOMP];                          // midpoint state of cell m = n-2 (latched by the previous step)
    T gr2_prev[NCOMP], gl2_prev[NCOMP];    // midpoint G^R, G^L of cell m-1
    T ar1[NCOMP], al1[NCOMP];              // G^R_{m-1} - G^R_{m-2}, G^L_{m-1} - G^L_{m-2}
    T xr_prev[NCOMP];                      // 2 F^R through (m-2|m-1), limited
    T fh_prev[NCOMP];                      // 2 F^h through (m-3|m-2)

    // stage B of step n: everything that follows from the midpoint state of cell m = n-2; new value of cell j = n-4
    template <int PH, int ODD, int Q = 0>
    __device__ __forceinline__ void stage_b(int n, const GasConstT<T>& gc, Sink& sink) {
        if (PH >= 3) {
            T gr2[NCOMP], gl2[NCOMP];
            cell_split_flux(uhl, gc, gr2, gl2);                             // (d), cell m
            if (PH >= 4) {                                                  // m >= 2
                T ar0[NCOMP], al0[NCOMP];
#pragma unroll
                for (int k = 0; k < NCOMP; ++k) {
                    ar0[k] = gr2[k] - gr2_prev[k];
                    al0[k] = gl2[k] - gl2_prev[k];
                }
                T xr[NCOMP];
                if (PH >= 5) {                                              // m >= 3: (e) right-moving, (m-1|m)
#pragma unroll
                    for (int k = 0; k < NCOMP; ++k) xr[k] = limited<+1>(gr2_prev[k], ar1[k], ar0[k]);
                }
                if (PH >= 6) {                                              // m >= 4: (e) left-moving, (m-2|m-1)
                    T fh[NCOMP];
#pragma unroll
                    for (int k = 0; k < NCOMP; ++k) {
                        const T xl = limited<-1>(gl2_prev[k], al0[k], al1[k]);
                        fh[k] = xr_prev[k] - xl;
                    }
                    if (WANT_FACE) {
                        const int i = n - 4;                                // interface (i | i+1), i = m-2
                        if (i == NG - 1 || i == NG + PS / 2 - 1 || i == NG + PS - 1) {
                            T ff[NCOMP];
#pragma unroll
                            for (int k = 0; k < NCOMP; ++k) ff[k] = T(0.5) * fh[k];
                            sink.face(i == NG - 1 ? 0 : (i == NG + PS - 1 ? 2 : 1), ff);
                        }
                    }
                    if (PH >= 7) {                                          // m >= 5: (f) cell j = m-2 = n-4
                        T un[NCOMP];
#pragma unroll
                        for (int k = 0; k < NCOMP; ++k) un[k] = fma_rn(-gc.kh, fh[k] - fh_prev[k], u4[k]);
                        sink.template cell<2 * Q + ODD>(n - 4, un);
                    }
#pragma unroll
                    for (int k = 0; k < NCOMP; ++k) fh_prev[k] = fh[k];
                }
#pragma unroll
                for (int k = 0; k < NCOMP; ++k) {
                    if (PH >= 5) xr_prev[k] = xr[k];
                    ar1[k] = ar0[k];
                    al1[k] = al0[k];
                }
            }
#pragma unroll
            for (int k = 0; k < NCOMP; ++k) {
                gr2_prev[k] = gr2[k];
                gl2_prev[k] = gl2[k];
            }
        }
    }

    // stage A of step n: coefficients of cell n (a), midpoint state of cell n-1 (b)+(c) into the latch; window shift
    template <int PH>
    __device__ __forceinline__ void stage_a(const T (&u)[NCOMP], const GasConstT<T>& gc) {
        const HalfCoefT<T> h = half_coef(u, gc);
        if (PH >= 2) {
            const T dP = sub_rn(P2, h.P), dPv = sub_rn(Pv2, h.Pv);
#pragma unroll
            for (int k = 0; k < NCOMP; ++k) {
                T b = (k == 1) ? fma_rn(sig1, u1[k], dP) : ((k == 4) ? fma_rn(sig1, u1[k], dPv) : mul_rn(sig1, u1[k]));
                b = fma_rn(cp2, u2[k], b);
                uhl[k] = fma_rn(h.cm, u[k], b);
            }
        }
#pragma unroll
        for (int k = 0; k < NCOMP; ++k) {
            if (PH >= 3) u4[k] = u3[k];
            if (PH >= 2) u3[k] = u2[k];
            if (PH >= 1) u2[k] = u1[k];
            u1[k] = u[k];
        }
        if (PH >= 1) { cp2 = cp1; P2 = P1; Pv2 = Pv1; }
        cp1 = h.cp; P1 = h.P; Pv1 = h.Pv; sig1 = h.sig;
    }

    template <int PH0, int PH1, int Q = 0, class Src, class Gate>
    __device__ __forceinline__ void pair(Src& src, int n, const GasConstT<T>& gc, Sink& sink, Gate& gate) {
        T ua[NCOMP], ub[NCOMP];
        gate.acquire(n);
        src.load(n, ua, ub);
        gate.release(n);
        stage_b<PH0, 0, Q>(n, gc, sink);        // n is even: j = n-4 is even
        stage_a<PH0>(ua, gc);
        stage_b<PH1, 1, Q>(n + 1, gc, sink);
        stage_a<PH1>(ub, gc);
    }

    template <class Src, class Gate>
    __device__ __forceinline__ void run(Src& src, const GasConstT<T>& gc, Sink& sink, Gate& gate) {
        pair<0, 1>(src, 0, gc, sink, gate);
        pair<2, 3>(src, 2, gc, sink, gate);
        pair<4, 5>(src, 4, gc, sink, gate);
        if (PHASE4) {
            pair<6, 7, 1>(src, 6, gc, sink, gate);          // cell 3 at step 7: P = 3, the first of a group of four
#pragma unroll 1
            for (int n = 8; n < NP - 2; n += 4) {
                pair<7, 7, 0>(src, n, gc, sink, gate);      // cells n-4, n-3: P = 0, 1
                pair<7, 7, 1>(src, n + 2, gc, sink, gate);  // cells n-2, n-1: P = 2 (the group is complete), 3
            }
            pair<7, 7, 0>(src, NP - 2, gc, sink, gate);     // cells 16, 17
            stage_b<7, 0, 1>(NP, gc, sink);                 // drain: cell 18, P = 2
            return;
        }
        pair<6, 7>(src, 6, gc, sink, gate);
        // pairs of cells per loop body: the fp64 step is 2.5 x as long, so its body is kept shorter
        constexpr int UNROLL = sizeof(T) == 8 ? GAMER_MARCH_UNROLL_F64 : MARCH_UNROLL;
#pragma unroll UNROLL
        for (int n = 8; n < NP; n += 2) pair<7, 7>(src, n, gc, sink, gate);
        stage_b<7, 0>(NP, gc, sink);            // drain: cell j = 18
    }
};

// Row source with a compile-time element stride: src[q] points to cell 0 of row-local component q.
template <int STRIDE>
struct StrideSrc {
    const float* src[NCOMP];
    __device__ __forceinline__ void load(int n, float (&ua)[NCOMP], float (&ub)[NCOMP]) const {
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
    }
};

struct NoGate {
    __device__ __forceinline__ void acquire(int) {}
    __device__ __forceinline__ void release(int) {}
};

template <int STRIDE, bool WANT_FACE, bool PHASE4 = false, class Sink, class Gate>
__device__ __forceinline__ void rtvd_march(const float* const (&src)[NCOMP], const GasConst& gc, Sink& sink,
                                           Gate& gate) {
    RowMarch<WANT_FACE, Sink, float, PHASE4> m;
    StrideSrc<STRIDE> s;
#pragma unroll
    for (int k = 0; k < NCOMP; ++k) s.src[k] = src[k];
    m.run(s, gc, sink, gate);
}

}  // namespace gamer
