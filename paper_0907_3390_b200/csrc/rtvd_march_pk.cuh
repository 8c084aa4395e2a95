// rtvd_march_pk.cuh — the 1-D relaxing-TVD row update as a register sliding window, Blackwell packed-FP32 version.
//
// Same pipeline and arithmetic as documented in rtvd_march.cuh (§2.2, Eqs.6-14; DESIGN.md steps (a)-(f)),
// but the 5-vector operations are issued as two packed f32x2 instructions (FFMA2/FADD2/FMUL2, sm_100a) plus one scalar:
//     A = (m_n, e)   B = (m_t1, m_t2)   s = rho            (row-local components 1,4 | 2,3 | 0)
// A packed instruction occupies the FP32 pipe for two cycles but only one issue slot, so the other pipes (MUFU for
// the reciprocals and square roots, the predicate compares of the limiter, shared-memory loads/stores) issue in its
// shadow.  The split fluxes are formed as G^R = u (c + v) + (0, P, 0, 0, P v), G^L = u (c - v) - (0, P, 0, 0, P v),
// which is Eq.8 (times 2) with F = u v + (0, P, 0, 0, P v) substituted: two instructions fewer per cell than c u ± F.
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

// The five conserved variables (or fluxes) of one cell: two packed pairs and a scalar.
struct V5 {
    float2 A;   // (m_n, e)
    float2 B;   // (m_t1, m_t2)
    float s;    // rho
};
__device__ __forceinline__ float2 bc2(float x) { return make_float2(x, x); }
__device__ __forceinline__ float2 neg2(float2 a) { return make_float2(-a.x, -a.y); }
__device__ __forceinline__ V5 v5_sub(const V5& x, const V5& y) {
    V5 r;
    r.A = __fadd2_rn(x.A, neg2(y.A));
    r.B = __fadd2_rn(x.B, neg2(y.B));
    r.s = x.s - y.s;
    return r;
}
__device__ __forceinline__ V5 v5_add(const V5& x, const V5& y) {
    V5 r;
    r.A = __fadd2_rn(x.A, y.A);
    r.B = __fadd2_rn(x.B, y.B);
    r.s = x.s + y.s;
    return r;
}
__device__ __forceinline__ V5 v5_mul(const V5& x, const V5& y) {
    V5 r;
    r.A = __fmul2_rn(x.A, y.A);
    r.B = __fmul2_rn(x.B, y.B);
    r.s = x.s * y.s;
    return r;
}
// u - k d
__device__ __forceinline__ V5 v5_nfma(float k, const V5& d, const V5& u) {
    V5 r;
    r.A = __ffma2_rn(bc2(-k), d.A, u.A);
    r.B = __ffma2_rn(bc2(-k), d.B, u.B);
    r.s = fmaf(-k, d.s, u.s);
    return r;
}
__device__ __forceinline__ void v5_to_array(const V5& v, float (&u)[NCOMP]) {
    u[0] = v.s;
    u[1] = v.A.x;
    u[2] = v.B.x;
    u[3] = v.B.y;
    u[4] = v.A.y;
}

// Cell-centred G^R = c u + F = 2 F^R and G^L = c u - F = 2 F^L of one cell (Eq.8).
// c = |v_n| + c_s (reading R1), P from all three momenta (Eqs.4-5, reading R2).
__device__ __forceinline__ void cell_split_flux(const V5& u, const GasConst& gc, V5& gr, V5& gl) {
    const float rinv = rcp_fast(u.s);
    const float v = u.A.x * rinv;
    float q = u.B.x * u.B.x;
    q = fmaf(u.B.y, u.B.y, q);
    q = fmaf(u.A.x, u.A.x, q);
    const float hk = 0.5f * rinv;
    const float eint = fmaf(-q, hk, u.A.y);          // e - rho v^2 / 2
    const float P = gc.gm1 * eint;
    const float cs = sqrt_fast((gc.ggm1 * eint) * rinv);
    const float c = fabsf(v) + cs;
    const float cp = c + v, cm = c - v;
    const float2 PP = make_float2(P, P * v);         // the part of F that is not u v
    gr.A = __ffma2_rn(u.A, bc2(cp), PP);
    gr.B = __fmul2_rn(u.B, bc2(cp));
    gr.s = u.s * cp;
    gl.A = __ffma2_rn(u.A, bc2(cm), neg2(PP));
    gl.B = __fmul2_rn(u.B, bc2(cm));
    gl.s = u.s * cm;
}

// base + p / s if p > 0, else base   (SGN = +1)   |   base - p / s ...   (SGN = -1);  p = a b, s = a + b.
// A select on the sign of the product, never a mask (reading R6).
template <int SGN>
__device__ __forceinline__ float limited(float base, float p, float s) {
    const float r = rcp_fast(s);
    const float x = fmaf(SGN > 0 ? p : -p, r, base);
    return p > 0.f ? x : base;
}
template <int SGN>
__device__ __forceinline__ V5 v5_limited(const V5& base, const V5& a, const V5& b) {
    const V5 p = v5_mul(a, b), s = v5_add(a, b);
    V5 r;
    r.A.x = limited<SGN>(base.A.x, p.A.x, s.A.x);
    r.A.y = limited<SGN>(base.A.y, p.A.y, s.A.y);
    r.B.x = limited<SGN>(base.B.x, p.B.x, s.B.x);
    r.B.y = limited<SGN>(base.B.y, p.B.y, s.B.y);
    r.s = limited<SGN>(base.s, p.s, s.s);
    return r;
}

// Marches one row; interface as in rtvd_march.cuh (Sink::cell<ODD>(j, u[5]), Sink::face(p, f[5]), row-local order).
template <int STRIDE, bool WANT_FACE, class Sink>
struct RowMarch {
    V5 u1, u2, u3;            // u_{n-1}, u_{n-2}, u_{n-3} (the originals, kept for Eqs.13-14)
    V5 gr1_prev;              // G^R_{n-1} at time t
    V5 f_prev;                // 2F through (n-2|n-1)
    V5 gr2_prev, gl2_prev;    // midpoint G^R, G^L of cell m-1
    V5 gr2_pp;                // midpoint G^R of cell m-2
    V5 ar1, ar2, al1;         // ar1 = G^R_{m-1}-G^R_{m-2}, ar2 = G^R_{m-2}-G^R_{m-3}, al1 likewise for L
    V5 fh_prev;               // 2F^h through the previous limited interface

    template <int PH>
    __device__ __forceinline__ void step(const V5& u, int n, const GasConst& gc, Sink& sink) {
        V5 gr1, gl1;
        cell_split_flux(u, gc, gr1, gl1);                                   // (a)
        if (PH >= 1) {
            const V5 f = v5_sub(gr1_prev, gl1);                             // (b) interface (n-1 | n)
            if (PH >= 2) {                                                  // midpoint cell m = n-1
                const V5 uh = v5_nfma(gc.kq, v5_sub(f, f_prev), u1);        // (c)
                V5 gr2, gl2;
                cell_split_flux(uh, gc, gr2, gl2);                          // (d)
                if (PH >= 3) {                                              // m >= 2
                    const V5 ar0 = v5_sub(gr2, gr2_prev);                   // G^R_m - G^R_{m-1}
                    const V5 al0 = v5_sub(gl2, gl2_prev);                   // G^L_m - G^L_{m-1}
                    if (PH >= 5) {                                          // m >= 4: (e) interface (m-2 | m-1)
                        const V5 xr = v5_limited<+1>(gr2_pp, ar2, ar1);
                        // a = G^L_{m-1}-G^L_m = -al0, b = G^L_{m-2}-G^L_{m-1} = -al1: a b = al0 al1, a+b = -(al0+al1)
                        const V5 xl = v5_limited<-1>(gl2_prev, al0, al1);
                        const V5 fh = v5_sub(xr, xl);
                        if (WANT_FACE) {
                            const int i = n - 3;                            // interface (i | i+1), i = m-2
                            if (i == NG - 1 || i == NG + PS / 2 - 1 || i == NG + PS - 1) {
                                float ff[NCOMP];
                                v5_to_array(fh, ff);
#pragma unroll
                                for (int k = 0; k < NCOMP; ++k) ff[k] *= 0.5f;
                                sink.face(i == NG - 1 ? 0 : (i == NG + PS - 1 ? 2 : 1), ff);
                            }
                        }
                        if (PH >= 6) {                                      // m >= 5: (f) cell j = m-2 = n-3
                            const V5 un5 = v5_nfma(gc.kh, v5_sub(fh, fh_prev), u3);
                            float un[NCOMP];
                            v5_to_array(un5, un);
                            sink.template cell<(PH + 1) & 1>(n - 3, un);    // parity of j = n-3 is static
                        }
                        fh_prev = fh;
                    }
                    ar2 = ar1;
                    ar1 = ar0;
                    al1 = al0;
                }
                gr2_pp = gr2_prev;
                gr2_prev = gr2;
                gl2_prev = gl2;
            }
            f_prev = f;
        }
        if (PH >= 2) u3 = u2;
        if (PH >= 1) u2 = u1;
        u1 = u;
        gr1_prev = gr1;
    }

    __device__ __forceinline__ static V5 from_array(const float (&a)[NCOMP]) {
        V5 v;
        v.s = a[0];
        v.A = make_float2(a[1], a[4]);
        v.B = make_float2(a[2], a[3]);
        return v;
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
        step<PH0>(from_array(ua), n, gc, sink);
        step<PH1>(from_array(ub), n + 1, gc, sink);
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
