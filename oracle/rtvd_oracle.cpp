// ORACLE — TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// Plain, slow, single-file CPU implementation of the batched relaxing-TVD hydrodynamic update of
// GAMER (arXiv 0907.3390), written from /root/reference/PAPER.md only.  It exists so that the CUDA
// path (paper_0907_3390_b200/csrc) can be compared against something that a reader can check
// against the paper by eye.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
// --impl reference legs may call it.  It shares no code, header, table or helper with the CUDA
// path and neither includes the other.
//
// What it follows (PAPER.md line : section / equation):
//   :108-120  §2.2 Eqs.1-5    conserved variables u=(rho, rho v_x, rho v_y, rho v_z, e), P=(gamma-1)(e-rho v^2/2)
//   :126-130  §2.2 Eq.6       1-D flux F(u), freezing speed c=|v|+c_s, auxiliary vector w=F/c
//   :132-138  §2.2 Eqs.7-8    F^R = c(u+w)/2, F^L = c(u-w)/2
//   :143      §2.2            first-order upwind interface flux F^R_{n+1/2}=F^R_n (and F^L_{n+1/2}=F^L_{n+1})
//   :145-162  §2.2 Eqs.9-12   second-order correction with the van Leer limiter
//   :164-172  §2.2 Eqs.13-14  midpoint (RK2) time integration: half step with upwind fluxes, full step with TVD fluxes
//   :174-178  §2.2            dimensional splitting, forward xyz / backward zyx, 7-point stencil = 3 ghost zones
//   :318-344  §3.1            patch group = 22^3 padded cells in, 16^3 interior cells out, boolean sweep direction
//   :340,:344 §3.1            fluxes across the patch boundaries are part of the output
//   :418-426  §3.4 Eq.30      per-group maximum of c_s + max(|v_x|,|v_y|,|v_z|)
// Readings of the points where the paper is silent are listed in DESIGN.md ("Readings"); the ones
// that matter here: c uses the velocity component normal to the sweep (R1), the limiter acts per
// component (R5) and is a select, not a mask (R6), no floors (R7), F^L is the mirror image of F^R (R4).
//
// Everything is a loop in the paper's order.  No blocking, no fusion, no SIMD.  Compile with
// -O2 -ffp-contract=off so that no FMA contraction changes the rounding the source states.
// The only parallelism is an optional `omp parallel for` over independent patch groups (:77, :310).
//
// Parity status: every function below is pinned by tests/test_oracle_pins.py.

#include <cmath>
#include <cstddef>
#include <cstdint>
#include <vector>
#include <algorithm>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

// ------------------------------------------------------------------------------------------------
// A scalar type that counts the arithmetic it performs.  Used only by oracle_count_ops() to replace
// the hand count of SURVEY.md 8(d) by a measured one.  add/sub, mul, div, sqrt, compare are tallied.
// ------------------------------------------------------------------------------------------------
struct OpCount { long long add = 0, mul = 0, div = 0, sqrt_ = 0, cmp = 0, abs_ = 0; };
static thread_local OpCount g_ops;

struct Counted {
    double v;
    Counted() : v(0) {}
    Counted(double x) : v(x) {}
    explicit operator double() const { return v; }
};
inline Counted operator+(Counted a, Counted b) { g_ops.add++; return Counted(a.v + b.v); }
inline Counted operator-(Counted a, Counted b) { g_ops.add++; return Counted(a.v - b.v); }
inline Counted operator*(Counted a, Counted b) { g_ops.mul++; return Counted(a.v * b.v); }
inline Counted operator/(Counted a, Counted b) { g_ops.div++; return Counted(a.v / b.v); }
inline bool operator>(Counted a, Counted b) { g_ops.cmp++; return a.v > b.v; }
inline bool operator<=(Counted a, Counted b) { g_ops.cmp++; return a.v <= b.v; }
inline Counted sqrt_T(Counted a) { g_ops.sqrt_++; return Counted(std::sqrt(a.v)); }
inline Counted abs_T(Counted a) { g_ops.abs_++; return Counted(std::fabs(a.v)); }
inline float sqrt_T(float a) { return std::sqrt(a); }
inline double sqrt_T(double a) { return std::sqrt(a); }
inline float abs_T(float a) { return std::fabs(a); }
inline double abs_T(double a) { return std::fabs(a); }
inline double to_double(float a) { return (double)a; }
inline double to_double(double a) { return a; }
inline double to_double(Counted a) { return a.v; }

constexpr int NCOMP = 5;       // rho, m_n (normal momentum), m_t1, m_t2, e   -- row-local component order
constexpr int PS = 16;         // interior cells per side of a patch group (2 patches of 8, :318)
constexpr int NGHOST = 3;      // :178
constexpr int NP = PS + 2 * NGHOST;   // 22

// ------------------------------------------------------------------------------------------------
// van Leer limiter, Eq.11 (:152-157): harmonic average of the two corrections if they have the same
// sign, else 0.  A select (reading R6): nothing is evaluated when the product is not positive.
// ------------------------------------------------------------------------------------------------
template <typename T>
inline T van_leer(T dF1, T dF2) {
    if (dF1 * dF2 > T(0)) return (T(2) * dF1 * dF2) / (dF1 + dF2);
    return T(0);
}

// ------------------------------------------------------------------------------------------------
// Cell-centred quantities of one cell for a sweep whose normal momentum is u[1] (:126-138).
//   v   = m_n / rho
//   P   = (gamma-1) (e - (m_n^2 + (m_t1^2 + m_t2^2)) / (2 rho))            Eqs.4-5, all three momenta (R2)
//   c_s = sqrt(gamma P / rho),  c = |v| + c_s                               :130 (R1: normal component)
//   F   = (m_n, m_n v + P, m_t1 v, m_t2 v, (e + P) v)                       Eqs.1-3 restricted to one direction
//   w   = F / c,  F^R = c (u + w)/2,  F^L = c (u - w)/2                     :130, Eq.8
// `c_mode` = 0: c = |v_n| + c_s (default reading R1); 1: c = |v| (3-D speed) + c_s (the alternative).
// ------------------------------------------------------------------------------------------------
template <typename T>
inline void cell_fluxes(const T u[NCOMP], T gamma, int c_mode, T FR[NCOMP], T FL[NCOMP], T* c_out) {
    const T rho = u[0], mn = u[1], mt1 = u[2], mt2 = u[3], e = u[4];
    const T v = mn / rho;
    const T ek = (mn * mn + (mt1 * mt1 + mt2 * mt2)) / (T(2) * rho);
    const T P = (gamma - T(1)) * (e - ek);
    const T cs = sqrt_T(gamma * P / rho);
    T c;
    if (c_mode == 0) {
        c = abs_T(v) + cs;
    } else {
        const T vt1 = mt1 / rho, vt2 = mt2 / rho;
        c = sqrt_T(v * v + (vt1 * vt1 + vt2 * vt2)) + cs;
    }
    T F[NCOMP];
    F[0] = mn;
    F[1] = mn * v + P;
    F[2] = mt1 * v;
    F[3] = mt2 * v;
    F[4] = (e + P) * v;
    for (int q = 0; q < NCOMP; ++q) {
        const T w = F[q] / c;
        FR[q] = c * ((u[q] + w) / T(2));
        FL[q] = c * ((u[q] - w) / T(2));
    }
    if (c_out) *c_out = c;
}

// ------------------------------------------------------------------------------------------------
// One 1-D relaxing-TVD update of a row of N cells (:126-172, steps (a)-(f) of DESIGN.md §Path).
//   u     [NCOMP][N]  in : row-local components (rho, m_n, m_t1, m_t2, e), cell n = 0..N-1
//   unew  [NCOMP][N]  out: cells 3..N-4 hold u^{t+dt}; all other cells are copied from u
//   k = dt/dh
//   limiter_on = 0 forces phi = 0 (first-order fluxes at the midpoint; used by a pin only)
//   uhalf [NCOMP][N]  optional out: midpoint state u^{t+dt/2} on cells 1..N-2 (0 elsewhere)
//   fhalf [NCOMP][N]  optional out: fhalf[q][n] = time-centred interface flux F^{t+dt/2}_{n+1/2}, n = 2..N-4
// ------------------------------------------------------------------------------------------------
template <typename T>
void row_update(const T* u, T* unew, int N, T k, T gamma, int c_mode, int limiter_on, T* uhalf, T* fhalf) {
    std::vector<T> FR((size_t)NCOMP * N), FL((size_t)NCOMP * N), f((size_t)NCOMP * N), uh((size_t)NCOMP * N),
        fh((size_t)NCOMP * N);
    auto at = [N](int q, int n) { return (size_t)q * N + n; };
    T cell[NCOMP], r[NCOMP], l[NCOMP];

    // (a) cell-centred F^R_n, F^L_n at time t, n = 0..N-1
    for (int n = 0; n < N; ++n) {
        for (int q = 0; q < NCOMP; ++q) cell[q] = u[at(q, n)];
        cell_fluxes<T>(cell, gamma, c_mode, r, l, nullptr);
        for (int q = 0; q < NCOMP; ++q) { FR[at(q, n)] = r[q]; FL[at(q, n)] = l[q]; }
    }
    // (b) first-order upwind interface flux F_{n+1/2} = F^R_{n+1/2} - F^L_{n+1/2} = F^R_n - F^L_{n+1}  (:143, :170)
    for (int n = 0; n <= N - 2; ++n)
        for (int q = 0; q < NCOMP; ++q) f[at(q, n)] = FR[at(q, n)] - FL[at(q, n + 1)];
    // (c) half step, Eq.13: u^{t+dt/2}_n = u_n - (F_{n+1/2} - F_{n-1/2}) / dx * dt/2,  n = 1..N-2
    for (int q = 0; q < NCOMP; ++q)
        for (int n = 0; n < N; ++n) uh[at(q, n)] = T(0);
    for (int n = 1; n <= N - 2; ++n)
        for (int q = 0; q < NCOMP; ++q)
            uh[at(q, n)] = u[at(q, n)] - (f[at(q, n)] - f[at(q, n - 1)]) * (k / T(2));
    // (d) cell-centred F^R_n, F^L_n of the midpoint state, n = 1..N-2
    for (int n = 1; n <= N - 2; ++n) {
        for (int q = 0; q < NCOMP; ++q) cell[q] = uh[at(q, n)];
        cell_fluxes<T>(cell, gamma, c_mode, r, l, nullptr);
        for (int q = 0; q < NCOMP; ++q) { FR[at(q, n)] = r[q]; FL[at(q, n)] = l[q]; }
    }
    // (e) second-order TVD interface fluxes, Eqs.9-12, n = 2..N-4:
    //     F^R_{n+1/2} = F^R_n     + phi( (F^R_n - F^R_{n-1})/2 ,     (F^R_{n+1} - F^R_n)/2 )
    //     F^L_{n+1/2} = F^L_{n+1} + phi( (F^L_{n+1} - F^L_{n+2})/2 , (F^L_n - F^L_{n+1})/2 )   mirror image (R4)
    for (int n = 2; n <= N - 4; ++n)
        for (int q = 0; q < NCOMP; ++q) {
            T dR = T(0), dL = T(0);
            if (limiter_on) {
                dR = van_leer<T>((FR[at(q, n)] - FR[at(q, n - 1)]) / T(2), (FR[at(q, n + 1)] - FR[at(q, n)]) / T(2));
                dL = van_leer<T>((FL[at(q, n + 1)] - FL[at(q, n + 2)]) / T(2), (FL[at(q, n)] - FL[at(q, n + 1)]) / T(2));
            }
            const T FRh = FR[at(q, n)] + dR;
            const T FLh = FL[at(q, n + 1)] + dL;
            fh[at(q, n)] = FRh - FLh;
        }
    // (f) full step, Eq.14: u^{t+dt}_n = u_n - (F^{t+dt/2}_{n+1/2} - F^{t+dt/2}_{n-1/2}) / dx * dt,  n = 3..N-4
    for (int q = 0; q < NCOMP; ++q)
        for (int n = 0; n < N; ++n) unew[at(q, n)] = u[at(q, n)];
    for (int n = 3; n <= N - 4; ++n)
        for (int q = 0; q < NCOMP; ++q)
            unew[at(q, n)] = u[at(q, n)] - (fh[at(q, n)] - fh[at(q, n - 1)]) * k;

    if (uhalf) for (size_t i = 0; i < (size_t)NCOMP * N; ++i) uhalf[i] = uh[i];
    if (fhalf) {
        for (size_t i = 0; i < (size_t)NCOMP * N; ++i) fhalf[i] = T(0);
        for (int n = 2; n <= N - 4; ++n)
            for (int q = 0; q < NCOMP; ++q) fhalf[at(q, n)] = fh[at(q, n)];
    }
}

// ------------------------------------------------------------------------------------------------
// One patch group, one 3-sweep pass (:174-178, :326-342).
//   in   [5][22][22][22]   (v, z, y, x), x fastest; v = rho, m_x, m_y, m_z, e
//   out  [5][16][16][16]   interior only (:344)
//   face [3][3][5][16][16] optional: time-centred fluxes through the planes that bound the two 8-cell patch
//                          layers in each direction (padded interfaces 2|3, 10|11, 18|19), for flux correction
//                          (:340, :344-346).  face[d][p][v][b][a]: d = sweep axis (0:x,1:y,2:z); (b,a) = the two
//                          transverse interior indices, slower first: d=x:(k,j)  d=y:(k,i)  d=z:(j,i).
//   maxspeed               optional: max over the 16^3 updated cells of c_s + max(|v_x|,|v_y|,|v_z|), Eq.30 (:420-426)
//   returns the number of cells (over all sweeps, on cells that are read) with rho <= 0 or P <= 0  (reading R7)
//   badmask [22][22][22]   optional bookkeeping beside that counter (no arithmetic depends on it): WHERE such cells
//                          were met.  bit 0: the cell held five finite values with rho <= 0 or P <= 0 when a sweep read
//                          it (where the pass leaves the physical domain); bit 1: it held a non-finite value (what
//                          spreads from such a cell: at most 3 cells along the axis of each later sweep, :178).
// ------------------------------------------------------------------------------------------------
template <typename T>
long long advance_group(const T* in, T* out, T k, T gamma, int backward, int c_mode, T* face, T* maxspeed,
                        unsigned char* badmask = nullptr) {
    const size_t NV = (size_t)NP * NP * NP;
    std::vector<T> W(in, in + NCOMP * NV);
    auto idx = [](int v, int z, int y, int x) { return (((size_t)v * NP + z) * NP + y) * NP + x; };
    long long bad = 0;
    T row[NCOMP * NP], rnew[NCOMP * NP], fh[NCOMP * NP];

    for (int s = 0; s < 3; ++s) {
        const int d = backward ? 2 - s : s;   // forward x,y,z ; backward z,y,x (:174-176)
        // transverse extents still valid at this point of the pass (each earlier sweep shrank its own axis)
        int lo[3] = {0, 0, 0}, hi[3] = {NP - 1, NP - 1, NP - 1};
        for (int sp = 0; sp < s; ++sp) {
            const int dp = backward ? 2 - sp : sp;
            lo[dp] = NGHOST; hi[dp] = NP - 1 - NGHOST;
        }
        // row-local component order (rho, m_n, m_t1, m_t2, e) -> global variable index
        const int t1 = (d + 1) % 3, t2 = (d + 2) % 3;
        const int comp[NCOMP] = {0, 1 + d, 1 + t1, 1 + t2, 4};
        int a[3];   // a[0]=x, a[1]=y, a[2]=z
        for (a[t2] = lo[t2]; a[t2] <= hi[t2]; ++a[t2])
            for (a[t1] = lo[t1]; a[t1] <= hi[t1]; ++a[t1]) {
                for (int n = 0; n < NP; ++n) {
                    a[d] = n;
                    for (int q = 0; q < NCOMP; ++q) row[q * NP + n] = W[idx(comp[q], a[2], a[1], a[0])];
                    const T rho = row[0 * NP + n];
                    const T ek = (row[1 * NP + n] * row[1 * NP + n] +
                                  (row[2 * NP + n] * row[2 * NP + n] + row[3 * NP + n] * row[3 * NP + n])) / (T(2) * rho);
                    const T P = (gamma - T(1)) * (row[4 * NP + n] - ek);
                    if (!(rho > T(0)) || !(P > T(0))) {
                        ++bad;
                        if (badmask) {
                            bool finite = true;
                            for (int q = 0; q < NCOMP; ++q) {
                                const double val = to_double(row[q * NP + n]);
                                finite = finite && (val - val == 0.0);       // false for NaN and +-Inf
                            }
                            badmask[((size_t)a[2] * NP + a[1]) * NP + a[0]] |= finite ? 1 : 2;
                        }
                    }
                }
                row_update<T>(row, rnew, NP, k, gamma, c_mode, 1, nullptr, face ? fh : nullptr);
                for (int n = NGHOST; n < NP - NGHOST; ++n) {
                    a[d] = n;
                    for (int q = 0; q < NCOMP; ++q) W[idx(comp[q], a[2], a[1], a[0])] = rnew[q * NP + n];
                }
                if (face) {
                    const int i1 = a[t1] - NGHOST, i2 = a[t2] - NGHOST;
                    if (i1 >= 0 && i1 < PS && i2 >= 0 && i2 < PS) {
                        // (b,a) = transverse interior indices, slower first = the higher axis number first
                        const int hiax = t1 > t2 ? t1 : t2;
                        const int bb = (hiax == t1) ? i1 : i2, aa = (hiax == t1) ? i2 : i1;
                        const int planes[3] = {NGHOST - 1, NGHOST + PS / 2 - 1, NGHOST + PS - 1};   // n of F_{n+1/2}
                        for (int p = 0; p < 3; ++p)
                            for (int q = 0; q < NCOMP; ++q)
                                face[((((size_t)d * 3 + p) * NCOMP + comp[q]) * PS + bb) * PS + aa] = fh[q * NP + planes[p]];
                    }
                }
            }
    }
    T smax = T(0);
    for (int v = 0; v < NCOMP; ++v)
        for (int z = 0; z < PS; ++z)
            for (int y = 0; y < PS; ++y)
                for (int x = 0; x < PS; ++x)
                    out[(((size_t)v * PS + z) * PS + y) * PS + x] = W[idx(v, z + NGHOST, y + NGHOST, x + NGHOST)];
    if (maxspeed) {
        for (int z = NGHOST; z < NP - NGHOST; ++z)
            for (int y = NGHOST; y < NP - NGHOST; ++y)
                for (int x = NGHOST; x < NP - NGHOST; ++x) {
                    const T rho = W[idx(0, z, y, x)], mx = W[idx(1, z, y, x)], my = W[idx(2, z, y, x)],
                            mz = W[idx(3, z, y, x)], e = W[idx(4, z, y, x)];
                    const T ek = (mx * mx + (my * my + mz * mz)) / (T(2) * rho);
                    const T P = (gamma - T(1)) * (e - ek);
                    const T cs = sqrt_T(gamma * P / rho);
                    T vm = abs_T(mx / rho);
                    const T vy = abs_T(my / rho), vz = abs_T(mz / rho);
                    if (vy > vm) vm = vy;
                    if (vz > vm) vm = vz;
                    const T s = cs + vm;
                    if (s > smax) smax = s;
                }
        *maxspeed = smax;
    }
    return bad;
}

template <typename T>
long long advance_batch(const T* in, T* out, long long n_groups, int ghost, T dt, T dh, T gamma, int backward,
                        int c_mode, T* face, T* maxspeed, int n_threads, unsigned char* badmask = nullptr) {
    if (ghost != NGHOST) return -2;
    if (n_groups < 0) return -1;
    const T k = dt / dh;
    const size_t in_stride = (size_t)NCOMP * NP * NP * NP, out_stride = (size_t)NCOMP * PS * PS * PS;
    const size_t face_stride = (size_t)3 * 3 * NCOMP * PS * PS;
    long long bad = 0;
#ifdef _OPENMP
    if (n_threads < 1) n_threads = 1;
#pragma omp parallel for schedule(dynamic, 1) num_threads(n_threads) reduction(+ : bad)
#endif
    for (long long g = 0; g < n_groups; ++g)
        bad += advance_group<T>(in + g * in_stride, out + g * out_stride, k, gamma, backward, c_mode,
                                face ? face + g * face_stride : nullptr, maxspeed ? maxspeed + g : nullptr,
                                badmask ? badmask + g * (size_t)NP * NP * NP : nullptr);
    return bad;
}

}  // namespace

// ================================================================================================
// C entry points (ctypes).  All pointers are HOST pointers owned by the caller.
// ================================================================================================
extern "C" {

int oracle_has_openmp(void) {
#ifdef _OPENMP
    return 1;
#else
    return 0;
#endif
}

float oracle_van_leer_f32(float a, float b) { return van_leer<float>(a, b); }
double oracle_van_leer_f64(double a, double b) { return van_leer<double>(a, b); }

void oracle_cell_fluxes_f32(const float* u, float gamma, int c_mode, float* FR, float* FL, float* c) {
    cell_fluxes<float>(u, gamma, c_mode, FR, FL, c);
}
void oracle_cell_fluxes_f64(const double* u, double gamma, int c_mode, double* FR, double* FL, double* c) {
    cell_fluxes<double>(u, gamma, c_mode, FR, FL, c);
}

void oracle_row_update_f32(const float* u, float* unew, int N, float k, float gamma, int c_mode, int limiter_on,
                           float* uhalf, float* fhalf) {
    row_update<float>(u, unew, N, k, gamma, c_mode, limiter_on, uhalf, fhalf);
}
void oracle_row_update_f64(const double* u, double* unew, int N, double k, double gamma, int c_mode, int limiter_on,
                           double* uhalf, double* fhalf) {
    row_update<double>(u, unew, N, k, gamma, c_mode, limiter_on, uhalf, fhalf);
}

// returns the count of non-physical cells met (>= 0), or a negative error (-1 bad argument, -2 unsupported ghost)
long long oracle_hydro_advance_f32(const float* in, float* out, long long n_groups, int ghost, float dt, float dh,
                                   float gamma, int backward, int c_mode, float* face_flux, float* maxspeed,
                                   int n_threads) {
    return advance_batch<float>(in, out, n_groups, ghost, dt, dh, gamma, backward, c_mode, face_flux, maxspeed,
                                n_threads);
}
long long oracle_hydro_advance_f64(const double* in, double* out, long long n_groups, int ghost, double dt, double dh,
                                   double gamma, int backward, int c_mode, double* face_flux, double* maxspeed,
                                   int n_threads) {
    return advance_batch<double>(in, out, n_groups, ghost, dt, dh, gamma, backward, c_mode, face_flux, maxspeed,
                                 n_threads);
}

// The same pass; additionally badmask[g][22][22][22] (zeroed by the caller) receives where non-physical cells were met
// (bits as described at advance_group).  Bookkeeping only: the results are those of oracle_hydro_advance_*.
long long oracle_hydro_advance_badmask_f32(const float* in, float* out, long long n_groups, int ghost, float dt, float dh,
                                           float gamma, int backward, int c_mode, unsigned char* badmask, int n_threads) {
    return advance_batch<float>(in, out, n_groups, ghost, dt, dh, gamma, backward, c_mode, nullptr, nullptr, n_threads,
                                badmask);
}
long long oracle_hydro_advance_badmask_f64(const double* in, double* out, long long n_groups, int ghost, double dt,
                                           double dh, double gamma, int backward, int c_mode, unsigned char* badmask,
                                           int n_threads) {
    return advance_batch<double>(in, out, n_groups, ghost, dt, dh, gamma, backward, c_mode, nullptr, nullptr, n_threads,
                                 badmask);
}

// Measured operation count of one patch-group pass (replaces the hand count of SURVEY.md 8(d)).
// counts[0..5] = add/sub, mul, div, sqrt, compare, abs.  The input is a fixed smooth state; the count does not
// depend on the data except through the limiter select (a non-positive product skips 3 mul + 1 add + 1 div), so the
// input is chosen monotone along every axis to take the expensive branch everywhere.
void oracle_count_ops(long long* counts) {
    const size_t NV = (size_t)NP * NP * NP;
    std::vector<Counted> in(NCOMP * NV), out((size_t)NCOMP * PS * PS * PS);
    for (int z = 0; z < NP; ++z)
        for (int y = 0; y < NP; ++y)
            for (int x = 0; x < NP; ++x) {
                const size_t c = ((size_t)z * NP + y) * NP + x;
                const double s = 0.011 * x + 0.013 * y + 0.017 * z + 0.0003 * x * x + 0.0002 * y * y + 0.0001 * z * z;
                const double rho = 1.0 + s, vx = 0.1 + 0.3 * s, vy = 0.2 + 0.2 * s, vz = 0.15 + 0.25 * s, P = 1.0 + 0.5 * s;
                in[0 * NV + c] = Counted(rho);
                in[1 * NV + c] = Counted(rho * vx);
                in[2 * NV + c] = Counted(rho * vy);
                in[3 * NV + c] = Counted(rho * vz);
                in[4 * NV + c] = Counted(P / (5.0 / 3.0 - 1.0) + 0.5 * rho * (vx * vx + vy * vy + vz * vz));
            }
    g_ops = OpCount();
    // row_update only: the bad-cell scan and the CFL scan are bookkeeping, so count around a copy of the sweep loop
    // by calling advance_group without the optional outputs and subtracting the scan's known cost afterwards.
    advance_group<Counted>(in.data(), out.data(), Counted(0.1), Counted(5.0 / 3.0), 0, 0, nullptr, nullptr);
    // bad-cell scan per cell read: 3 mul + 2 add (m^2 sums) + 1 mul + 1 div (/(2 rho)) + 1 add + 1 mul (P) + 2 cmp
    const long long cells_read = (long long)NP * (NP * NP + PS * NP + PS * PS);
    counts[0] = g_ops.add - cells_read * 4;   // 2 (sum) + 1 (e-ek) + 1 (gamma-1)
    counts[1] = g_ops.mul - cells_read * 5;   // 3 squares + 2*rho + (gamma-1)*
    counts[2] = g_ops.div - cells_read * 1;
    counts[3] = g_ops.sqrt_;
    counts[4] = g_ops.cmp - cells_read * 2;
    counts[5] = g_ops.abs_;
}

}  // extern "C"
