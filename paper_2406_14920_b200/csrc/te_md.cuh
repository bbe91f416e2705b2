// te_md.cuh -- McMurchie-Davidson device primitives shared by the product kernels (sm_100a, FP64).
//
// Follows PAPER.md: E coefficients eq. 5-8, Boys function eq. 18, auxiliary integrals
// R eq. 20-25, four-centre integral eq. 30/31.  Nothing here is shared with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace te {

// ---------------------------------------------------------------------------------------- index helpers
__host__ __device__ constexpr int ncart(int l) { return (l + 1) * (l + 2) / 2; }
__host__ __device__ constexpr int nherm(int L) { return (L + 1) * (L + 2) * (L + 3) / 6; }

// Hermite index (t,u,v), t+u+v <= N, nested layout: t slowest, v fastest.
template <int N>
__host__ __device__ constexpr int tidx(int t, int u, int v) {
    const int a = N - t;
    return ((N + 1) * (N + 2) * (N + 3) - (a + 1) * (a + 2) * (a + 3)) / 6 + u * (a + 1) - u * (u - 1) / 2 + v;
}

// Cartesian component i of shell l, lexicographic with x^l first (te_jk.h): returns powers.
__host__ __device__ constexpr int cart_row(int i) { return i < 1 ? 0 : (i < 3 ? 1 : (i < 6 ? 2 : 3)); }
__host__ __device__ constexpr int cart_x(int l, int i) { return l - cart_row(i); }
__host__ __device__ constexpr int cart_z(int l, int i) { return i - cart_row(i) * (cart_row(i) + 1) / 2; }
__host__ __device__ constexpr int cart_y(int l, int i) { return cart_row(i) - cart_z(l, i); }

// class index of a primitive shell pair, la <= lb: SS SP SD SF PP PD PF DD DF FF
__host__ __device__ constexpr int pair_class(int la, int lb) { return (la == 0 ? 0 : la == 1 ? 4 : la == 2 ? 7 : 9) + (lb - la); }

// Classes that have an FP32 leg in the mixed-precision build (te_build_jk_mixed): the FP32 kernel is the uniform-ket kernel, so
// only classes it serves well take part (measured on config 5): not the lightest ones (L <= 2: no FP32 kernel), not the
// block-per-lane classes (their FP64 kernel is faster than the FP32 uniform-ket kernel) and not the heaviest bras.
__host__ __device__ constexpr bool jk_fp32_class(int la, int lb, int lc, int ld) {
    const int L = la + lb + lc + ld;
    const int outs = ncart(la) * ncart(lb) + (ncart(la) + ncart(lb)) * (ncart(lc) + ncart(ld));
    if (L <= 2) return false;
    if (L <= 4 && outs <= 48) return false;
    if (la + lb >= 5) return false;
    if (la == 2 && lb == 2 && lc + ld >= 5) return false;
    if (la == 1 && lb == 3 && lc == 3 && ld == 3) return false;
    return true;
}

// ------------------------------------------------------------------------------------------ Boys table
// F_m(T_i) on the grid T_i = i * BOYS_DT, i = 0..BOYS_NPTS-1, m = 0..BOYS_MROWS-1; used for T < BOYS_TMAX.
constexpr double BOYS_DT = 1.0 / 16.0;
constexpr double BOYS_TMAX = 36.0;
constexpr int BOYS_NPTS = 577;                 // 36 * 16 + 1
constexpr int BOYS_NTAYLOR = 8;                // terms k = 0..7
constexpr int BOYS_MROWS = 12 + BOYS_NTAYLOR;  // m = 0..19
constexpr int BOYS_STRIDE = BOYS_MROWS + 1;    // row of a grid point: F_0..F_19(T_i), then exp(-T_i)

// Boys function F_0..F_L(T) (eq. 18).  T < 36: 8-term Taylor expansion of F_L about the nearest grid point,
// F_L(T) = sum_k F_{L+k}(T_i) (T_i - T)^k / k!  (truncation < 3e-17 relative), then the stable downward
// recursion F_{m-1} = (2T F_m + exp(-T)) / (2m-1); exp(-T) = exp(-T_i) exp(T_i - T) with the tabulated exp(-T_i) and an
// 8-term series in |T_i - T| <= 1/32 (truncation 2e-17 relative), which costs 8 FMAs instead of a libm exp().
// T >= 36: erf(sqrt T) = 1 to double precision, so F_0 = sqrt(pi/T)/2, then upward
// F_{m+1} = ((2m+1) F_m - exp(-T)) / (2T)  (stable for T >> m).
template <int L>
__device__ __forceinline__ void boys(double T, const double* __restrict__ tab, double* __restrict__ F) {
    if (T < BOYS_TMAX) {
        const int i = __double2int_rn(T * (1.0 / BOYS_DT));
        const double d = (double)i * BOYS_DT - T;
        const double* row = tab + i * BOYS_STRIDE + L;
        double s = __ldg(row + 7) * (1.0 / 5040.0);
        s = fma(s, d, __ldg(row + 6) * (1.0 / 720.0));
        s = fma(s, d, __ldg(row + 5) * (1.0 / 120.0));
        s = fma(s, d, __ldg(row + 4) * (1.0 / 24.0));
        s = fma(s, d, __ldg(row + 3) * (1.0 / 6.0));
        s = fma(s, d, __ldg(row + 2) * 0.5);
        s = fma(s, d, __ldg(row + 1));
        s = fma(s, d, __ldg(row + 0));
        F[L] = s;
        if (L > 0) {
            double ed = 1.0 / 5040.0;
            ed = fma(ed, d, 1.0 / 720.0);
            ed = fma(ed, d, 1.0 / 120.0);
            ed = fma(ed, d, 1.0 / 24.0);
            ed = fma(ed, d, 1.0 / 6.0);
            ed = fma(ed, d, 0.5);
            ed = fma(ed, d, 1.0);
            ed = fma(ed, d, 1.0);
            const double eT = __ldg(row + (BOYS_MROWS - L)) * ed, T2 = 2.0 * T;
#pragma unroll
            for (int m = L; m > 0; --m) F[m - 1] = fma(T2, F[m], eT) * (1.0 / (2 * m - 1));
        }
    } else {
        const double rT = 1.0 / T;
        F[0] = 0.88622692545275801365 * sqrt(rT);   // sqrt(pi)/2 / sqrt(T)
        if (L > 0) {
            const double eT = exp(-T), h = 0.5 * rT;
#pragma unroll
            for (int m = 0; m < L; ++m) F[m + 1] = ((2 * m + 1) * F[m] - eT) * h;
        }
    }
}

// ------------------------------------------------------------------------------------------- pair data
struct PairD {
    double P[3];    // Gaussian product centre (eq. 3)
    double PA[3];   // P - A
    double PB[3];   // P - B
    double p;       // a + b
    double pref;    // c~_m c~_n exp(-ab/p |A-B|^2): eq. 7 prefactors of all three dimensions folded in
    double rp;      // 1 / p (the quartet prefactor is formed from rp, rq and one rsqrt(p + q), without a division)
};

// Exponent of the auxiliary integrals and prefactor of a primitive quartet: alpha = pq/(p+q), 2 pi^{5/2} / (p q sqrt(p+q))
// (eq. 30).  omega2 = omega^2 > 0 selects the long-range operator erf(omega r)/r of eq. 32-33:
// alpha -> pq omega^2 / (pq + (p+q) omega^2) = alpha omega^2 / (alpha + omega^2) and the prefactor gains omega / sqrt(alpha + omega^2).
__device__ __forceinline__ void eri_scale(double p, double rp, double q, double rq, double omega2, double& alpha, double& pref) {
    const double s = rsqrt(p + q);   // 1 / sqrt(p + q)
    alpha = p * q * (s * s);
    pref = 34.986836655249725693 * (rp * rq) * s;
    if (omega2 > 0.0) {
        const double w = omega2 / (alpha + omega2);
        alpha *= w;
        pref *= sqrt(w);
    }
}

// E coefficients of one dimension, eq. 5-8 with E^{00}_0 = 1 (the eq. 7 exponential lives in PairD::pref).
// E[i][j][t], zero for t > i+j.  SIGN: multiply by (-1)^t (the ket factor of eq. 30).
template <int LA, int LB, bool SIGN, class T>
__device__ __forceinline__ void etable(T PA, T PB, T h, T (&E)[LA + 1][LB + 1][LA + LB + 1]) {
#pragma unroll
    for (int i = 0; i <= LA; ++i)
#pragma unroll
        for (int j = 0; j <= LB; ++j)
#pragma unroll
            for (int t = 0; t <= LA + LB; ++t) E[i][j][t] = T(0);
    E[0][0][0] = T(1);
#pragma unroll
    for (int i = 0; i < LA; ++i)
#pragma unroll
        for (int t = 0; t <= i + 1; ++t) {
            T v = PA * E[i][0][t];
            if (t > 0) v = fma(h, E[i][0][t - 1], v);
            if (t + 1 <= i) v = fma(T(t + 1), E[i][0][t + 1], v);
            E[i + 1][0][t] = v;
        }
#pragma unroll
    for (int i = 0; i <= LA; ++i)
#pragma unroll
        for (int j = 0; j < LB; ++j)
#pragma unroll
            for (int t = 0; t <= i + j + 1; ++t) {
                T v = PB * E[i][j][t];
                if (t > 0) v = fma(h, E[i][j][t - 1], v);
                if (t + 1 <= i + j) v = fma(T(t + 1), E[i][j][t + 1], v);
                E[i][j + 1][t] = v;
            }
    if (SIGN) {
#pragma unroll
        for (int i = 0; i <= LA; ++i)
#pragma unroll
            for (int j = 0; j <= LB; ++j)
#pragma unroll
                for (int t = 1; t <= LA + LB; t += 2) E[i][j][t] = -E[i][j][t];
    }
}

// R^0_{tuv}(alpha, X), t+u+v <= L, eq. 21-25, built in place: level m is computed from level m+1 by
// sweeping the degree n = t+u+v downward, so only one array of nherm(L) values is live.
template <int L>
__device__ __forceinline__ void rtable(double alpha, double X, double Y, double Z, const double* __restrict__ F,
                                       double* __restrict__ R) {
    double fac[L + 1];
    fac[0] = 1.0;
#pragma unroll
    for (int m = 1; m <= L; ++m) fac[m] = fac[m - 1] * (-2.0 * alpha);
    R[0] = fac[L] * F[L];
#pragma unroll
    for (int m = L - 1; m >= 0; --m) {
#pragma unroll
        for (int n = L - m; n >= 1; --n) {
#pragma unroll
            for (int t = n; t >= 0; --t) {
#pragma unroll
                for (int u = n - t; u >= 0; --u) {
                    const int v = n - t - u;
                    double r;
                    if (t > 0) {
                        r = X * R[tidx<L>(t - 1, u, v)];
                        if (t > 1) r = fma((double)(t - 1), R[tidx<L>(t - 2, u, v)], r);
                    } else if (u > 0) {
                        r = Y * R[tidx<L>(t, u - 1, v)];
                        if (u > 1) r = fma((double)(u - 1), R[tidx<L>(t, u - 2, v)], r);
                    } else {
                        r = Z * R[tidx<L>(t, u, v - 1)];
                        if (v > 1) r = fma((double)(v - 1), R[tidx<L>(t, u, v - 2)], r);
                    }
                    R[tidx<L>(t, u, v)] = r;
                }
            }
        }
        R[0] = fac[m] * F[m];
    }
}

// Generic primitive shell-quartet integral block, eq. 30 in the bracketing of eq. 31:
//   g_P = sum_Q E_Q^{kl} (-1)^Q R_{P+Q}   for every bra Hermite index P and one ket component pair (k,l),
//   (ij|kl) = pref * sum_P E_P^{ij} g_P.
// emit.ket(k, l) is called before and emit.ket_done(k, l) after the (i,j) sweep of a ket component pair;
// emit(i, j, k, l, value) receives the integral WITHOUT the per-component normalisation factors.
// FULL = fully unrolled (all indices compile-time, arrays in registers); otherwise rolled loops.
template <int LA, int LB, int LC, int LD, bool FULL, class Emit>
__device__ __forceinline__ void md_quartet(const PairD& bra, const PairD& ket, const double* __restrict__ boys_tab,
                                           Emit& emit, double omega2 = 0.0) {
    constexpr int LAB = LA + LB, LCD = LC + LD, L = LAB + LCD;
    constexpr int NA = ncart(LA), NB = ncart(LB), NC = ncart(LC), ND = ncart(LD);
    constexpr int UN = FULL ? 64 : 1;
    const double p = bra.p, q = ket.p;
    double alpha, pref;
    eri_scale(p, bra.rp, q, ket.rp, omega2, alpha, pref);
    const double X = bra.P[0] - ket.P[0], Y = bra.P[1] - ket.P[1], Z = bra.P[2] - ket.P[2];
    double F[L + 1];
    boys<L>(alpha * (X * X + Y * Y + Z * Z), boys_tab, F);
    double R[nherm(L)];
    rtable<L>(alpha, X, Y, Z, F, R);
    pref *= bra.pref * ket.pref;   // eq. 30 prefactor times both pair prefactors

    double Eb[3][LA + 1][LB + 1][LAB + 1], Ek[3][LC + 1][LD + 1][LCD + 1];
    {
        const double hb = 0.5 / p, hk = 0.5 / q;
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            etable<LA, LB, false>(bra.PA[d], bra.PB[d], hb, Eb[d]);
            etable<LC, LD, true>(ket.PA[d], ket.PB[d], hk, Ek[d]);
        }
    }
    double g[nherm(LAB)];
#pragma unroll UN
    for (int k = 0; k < NC; ++k) {
        const int kx = cart_x(LC, k), ky = cart_y(LC, k), kz = cart_z(LC, k);
#pragma unroll UN
        for (int l = 0; l < ND; ++l) {
            const int lx = cart_x(LD, l), ly = cart_y(LD, l), lz = cart_z(LD, l);
            emit.ket(k, l);
            // g_P for all P in the bra tetrahedron
#pragma unroll UN
            for (int t = 0; t <= LAB; ++t)
#pragma unroll UN
                for (int u = 0; u <= LAB - t; ++u)
#pragma unroll UN
                    for (int v = 0; v <= LAB - t - u; ++v) {
                        double s = 0.0;
#pragma unroll UN
                        for (int t2 = 0; t2 <= kx + lx; ++t2) {
                            const double ex = Ek[0][kx][lx][t2];
#pragma unroll UN
                            for (int u2 = 0; u2 <= ky + ly; ++u2) {
                                const double exy = ex * Ek[1][ky][ly][u2];
#pragma unroll UN
                                for (int v2 = 0; v2 <= kz + lz; ++v2)
                                    s = fma(exy * Ek[2][kz][lz][v2], R[tidx<L>(t + t2, u + u2, v + v2)], s);
                            }
                        }
                        g[tidx<LAB>(t, u, v)] = s;
                    }
#pragma unroll UN
            for (int i = 0; i < NA; ++i) {
                const int ix = cart_x(LA, i), iy = cart_y(LA, i), iz = cart_z(LA, i);
#pragma unroll UN
                for (int j = 0; j < NB; ++j) {
                    const int jx = cart_x(LB, j), jy = cart_y(LB, j), jz = cart_z(LB, j);
                    double s = 0.0;
#pragma unroll UN
                    for (int t = 0; t <= ix + jx; ++t) {
                        const double ex = Eb[0][ix][jx][t];
#pragma unroll UN
                        for (int u = 0; u <= iy + jy; ++u) {
                            const double exy = ex * Eb[1][iy][jy][u];
#pragma unroll UN
                            for (int v = 0; v <= iz + jz; ++v)
                                s = fma(exy * Eb[2][iz][jz][v], g[tidx<LAB>(t, u, v)], s);
                        }
                    }
                    emit(i, j, k, l, pref * s);
                }
            }
            emit.ket_done(k, l);
        }
    }
}

// per-component normalisation factor f(i) = sqrt((2l-1)!! / ((2ix-1)!!(2iy-1)!!(2iz-1)!!))  (eq. 2)
__host__ __device__ inline double comp_factor(int l, int i) {
    // d: xx xy xz yy yz zz ; f: xxx xxy xxz xyy xyz xzz yyy yyz yzz zzz
    if (l < 2) return 1.0;
    if (l == 2) return (i == 0 || i == 3 || i == 5) ? 1.0 : 1.7320508075688772935;   // sqrt 3
    if (i == 0 || i == 6 || i == 9) return 1.0;
    if (i == 4) return 3.8729833462074168852;                                          // sqrt 15
    return 2.2360679774997896964;                                                      // sqrt 5
}

}  // namespace te
