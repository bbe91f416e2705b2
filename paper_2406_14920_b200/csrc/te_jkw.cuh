// te_jkw.cuh -- "uniform-ket" J/K kernel: one warp = one KET primitive pair (warp-uniform) x 32 BRA primitive pairs (one per
// lane).  Everything that depends only on the ket -- its Hermite expansion coefficients E_Q^{kl} (eq. 5-8), folded with the
// (-1)^{t'+u'+v'} of eq. 30 and the pair prefactor, and its density block -- is built once per task in shared memory and read by
// broadcast; every lane keeps its own R^0_{tuv} tensor (eq. 21-25) in a conflict-free shared-memory column and its bra
// quantities in registers.  Per ket component pair (k,l) the lane forms
//     Y_P  = sum_{Q in box(kl)} E~_Q^{kl} R_{P+Q}            (ket Hermite -> Cartesian, eq. 31 inner bracket)
//     I_ij = pref * sum_P E_P^{ij} Y_P                       (bra Hermite -> Cartesian)
// and digests I_ij into the two J and four K updates of the quartet (eq. 34, 36) with the per-term masks of eq. 47.
#pragma once
#include "te_kernels.cuh"

#include <utility>

namespace te {

// compile-time loop: f(std::integral_constant<int, 0>{}), ..., f(std::integral_constant<int, N-1>{}) -- unlike "#pragma unroll"
// it cannot be declined by the compiler, so every index derived from the counter is a constant
template <int... Is, class F>
__device__ __forceinline__ void static_for_impl(std::integer_sequence<int, Is...>, F&& f) { (f(std::integral_constant<int, Is>{}), ...); }
template <int N, class F>
__device__ __forceinline__ void static_for(F&& f) { static_for_impl(std::make_integer_sequence<int, N>{}, f); }

// ROW[L][t][u] = index of (t,u,0) in the nested tetrahedral layout tidx<L>; (t,u,v) sits v entries further.
struct RowTab {
    unsigned short v[13 * 13 * 13];
    constexpr RowTab() : v{} {
        for (int L = 0; L < 13; ++L)
            for (int t = 0; t < 13; ++t)
                for (int u = 0; u < 13; ++u) {
                    const int a = L - t;
                    v[(L * 13 + t) * 13 + u] = (t <= L && u <= a)
                        ? (unsigned short)(((L + 1) * (L + 2) * (L + 3) - (a + 1) * (a + 2) * (a + 3)) / 6 + u * (a + 1) - u * (u - 1) / 2)
                        : (unsigned short)0;
                }
    }
};
static __constant__ RowTab c_rowtab = RowTab();

constexpr int WARP = 32;

#ifndef TE_KBAT
#define TE_KBAT 1
#endif
template <int LA, int LB, int LC, int LD, class T = double>
struct WShape {
    static constexpr int LAB = LA + LB, LCD = LC + LD, L = LAB + LCD;
    static constexpr int NA = ncart(LA), NB = ncart(LB), NC = ncart(LC), ND = ncart(LD);
    static constexpr int NHB = nherm(LAB), NR = nherm(L);
    static constexpr int NNZK = nnz_e(LC, LD);
    static constexpr int NE1 = (LC + 1) * (LD + 1) * (LCD + 1);
    // K_?c accumulators / D_?c blocks of the smaller ket shell stay in registers for the whole quartet when small
    // UNR: the loops over the ket component pairs (k,l) and their Hermite boxes are fully unrolled, so every table offset and
    // accumulator index is a compile-time constant (no row-table lookups, no dynamically indexed register arrays)
    // Measured (ncu source page, round 2): above a few hundred FMAs the compiler either declines the unrolling (leaving run-time
    // box loops that spend 5 integer instructions per DFMA) or honours it and the straight-line code misses the instruction
    // cache (no_instruction stalls); the alternative is compile-time (t',u'[,v']) loops skipped by warp-uniform branches, whose
    // body is NHB x (LDS + DFMA) with immediate offsets.  Per-class choice from CUDA-event times on config 5: s-, sp- and sd-type
    // bras (NHB <= 10, at most 10 FMAs per box entry) are fastest with the "#pragma unroll" form while it stays under ~6000
    // FMAs, pp bras and the larger light-bra classes with compile-time (t',u',v'), sf / pd bras (NHB = 20) with compile-time
    // (t',u') and a run-time v' loop -- except against pd-sized kets (LCD <= 3), where compile-time v' also wins ((PD|PD)
    // 351 -> 281 ms); for larger kets it gains < 2 % and triples the compile time of the library.
    static constexpr int SIZE = NHB * NNZK + nnz_e(LA, LB) * NC * ND;
    // k-batched form (VAR 3, below): FP64 only, s / sp bras against kets up to df, sd / pp bras against kets up to LCD = 4 (for df
    // kets the 20 ket_batch instantiations per class cost 30 minutes of compile time per translation unit for a 20 % gain)
    static constexpr bool KBEL = TE_KBAT && sizeof(T) == 8 && NC >= 3 && (NHB <= 4 ? LCD <= 6 : (NHB <= 10 && LCD <= 4));
    static constexpr int VAR = KBEL ? 3
                             : LCD == 6 ? 1   // ff kets (FP32 leg / forced family only): the 84-entry compile-time box costs minutes of ptxas
                             : (LA == 1 && LB == 1) ? 2
                             : NHB <= 10 ? (SIZE <= 6000 ? 0 : 2)
                             : (LA == 0 && LB == 3 && LC == 0 && LD == 3) ? 0 : (LCD <= 3 ? 2 : 1);
    static constexpr bool UNR = VAR == 0;
    static constexpr bool V2CT = VAR == 2;
    // VAR 3, "k-batched" ket transform (light bras, NHB <= 10, kets up to df): for a fixed l the Hermite boxes of the ket components k
    // overlap, so one R element loaded from the lane's shared-memory column feeds the FMAs of every k of a batch whose box holds
    // that shift Q (1.6-3 FMAs per private load instead of 1), all offsets compile-time (ket_batch below).
    static constexpr bool KBAT = VAR == 3;
    static constexpr int KBN = !KBAT ? 1 : (NC * NHB <= 32 ? NC : (NC % 5 == 0 && 5 * NHB <= 32 ? 5 : (NC % 3 == 0 ? 3 : (NC % 2 == 0 ? 2 : 1))));   // components per batch
    static constexpr int NKB = NC / KBN;
    static constexpr int UNK = UNR ? 128 : 1;
    static constexpr bool KEEPC = (UNR || KBAT) && (NA + NB) * NC <= 24;
    // NL = lanes of the warp that hold a quartet (R column stride).  Measured on B200: narrowing the warp to 8 lanes for L >= 10
    // (4x more resident warps) made (DF|DF) 2.4x SLOWER -- these kernels are bound by per-warp instruction / local-memory
    // throughput, not by latency -- so every lane holds a quartet.
    static constexpr int NL = 32;
    // without KEEPC the K_?c accumulators of the quartet live in a lane-private shared-memory column ((NA + NB) * NC values per
    // lane): they are summed over l there and flushed ONCE per quartet instead of once per (k,l)
    static constexpr int NKC = KEEPC ? 0 : (NA + NB) * NC;
    static constexpr int smem_doubles = NR * NL + NNZK + 3 * NE1 + NC * ND + NKC * NL;
};

// Segmented reduction over runs of lanes + one atomic per run and value, for N values that share a live flag.  The shuffle
// rounds of the N values are independent, so their latencies overlap (one value at a time, the rounds of a reduction form a
// serial SHFL -> DADD chain of ~40 cycles each; measured: the per-value version was the largest single cost of this kernel).
template <int N, class T, class AddrFn>
__device__ __forceinline__ void flush_vec(bool runs, int maxdist, int dist, bool head, bool live, T (&v)[N], AddrFn addr) {
    constexpr unsigned FULLMASK = 0xffffffffu;
    if (runs) {
#pragma unroll
        for (int x = 0; x < N; ++x) v[x] = live ? v[x] : T(0);
        for (int o = 1; o < maxdist; o <<= 1) {
#pragma unroll
            for (int x = 0; x < N; ++x) {
                const T t = __shfl_down_sync(FULLMASK, v[x], o);
                if (o < dist) v[x] += t;
            }
        }
        if (head) {
#pragma unroll
            for (int x = 0; x < N; ++x)
                if (v[x] != T(0)) atomicAdd(addr(x), (double)v[x]);
        }
    } else if (live) {
#pragma unroll
        for (int x = 0; x < N; ++x) atomicAdd(addr(x), (double)v[x]);
    }
}

// Offset of the E~ entries of the ket component pair (k,l) in the kt table (built in loop order l, k, t', u', v').
template <int LC, int LD>
__host__ __device__ constexpr int kt_off(int l, int k) {
    int s = 0;
    for (int l2 = 0; l2 < ncart(LD); ++l2)
        for (int k2 = 0; k2 < ncart(LC); ++k2) {
            if (l2 == l && k2 == k) return s;
            s += (cart_x(LC, k2) + cart_x(LD, l2) + 1) * (cart_y(LC, k2) + cart_y(LD, l2) + 1) * (cart_z(LC, k2) + cart_z(LD, l2) + 1);
        }
    return s;
}
// largest power of component k in [K0, K0 + KN) along dimension d (0 x, 1 y, 2 z)
template <int LC>
__host__ __device__ constexpr int kmax_pow(int K0, int KN, int d) {
    int m = 0;
    for (int k = K0; k < K0 + KN; ++k) {
        const int v = d == 0 ? cart_x(LC, k) : (d == 1 ? cart_y(LC, k) : cart_z(LC, k));
        m = v > m ? v : m;
    }
    return m;
}
template <int LC, int LD>
__host__ __device__ constexpr bool in_box(int k, int l, int t2, int u2, int v2) {
    return t2 <= cart_x(LC, k) + cart_x(LD, l) && u2 <= cart_y(LC, k) + cart_y(LD, l) && v2 <= cart_z(LC, k) + cart_z(LD, l);
}
template <int LC, int LD>
__host__ __device__ constexpr bool in_any_box(int K0, int KN, int l, int t2, int u2, int v2) {
    for (int k = K0; k < K0 + KN; ++k)
        if (in_box<LC, LD>(k, l, t2, u2, v2)) return true;
    return false;
}

// Ket Hermite -> Cartesian for the components k = K0 .. K0+KN-1 at fixed l:  Y[kk][P] = sum_{Q in box(k,l)} E~_Q^{kl} R_{P+Q}.
// Walks the UNION of the boxes once; an R element is loaded once per shift Q and used by every k whose box holds Q.
template <class T, int LAB, int LC, int LD, int NL, int l, int K0, int KN>
__device__ __forceinline__ void ket_batch(const T* __restrict__ Rl, const T* __restrict__ kt, T (&Y)[KN * nherm(LAB)]) {
    constexpr int LCD = LC + LD, L = LAB + LCD, NHB = nherm(LAB);
    constexpr int lx = cart_x(LD, l), ly = cart_y(LD, l), lz = cart_z(LD, l);
    constexpr int MX = lx + kmax_pow<LC>(K0, KN, 0), MY = ly + kmax_pow<LC>(K0, KN, 1), MZ = lz + kmax_pow<LC>(K0, KN, 2);
#pragma unroll
    for (int x = 0; x < KN * NHB; ++x) Y[x] = T(0);
    static_for<MX + 1>([&](auto T2) {
        constexpr int t2 = decltype(T2)::value;
        static_for<MY + 1>([&](auto U2) {
            constexpr int u2 = decltype(U2)::value;
            static_for<MZ + 1>([&](auto V2) {
                constexpr int v2 = decltype(V2)::value;
                if constexpr (in_any_box<LC, LD>(K0, KN, l, t2, u2, v2)) {
                    T r[NHB];
#pragma unroll
                    for (int t = 0; t <= LAB; ++t)
#pragma unroll
                        for (int u = 0; u <= LAB - t; ++u)
#pragma unroll
                            for (int v = 0; v <= LAB - t - u; ++v) r[tidx<LAB>(t, u, v)] = Rl[(tidx<L>(t + t2, u + u2, 0) + v + v2) * NL];
                    static_for<KN>([&](auto KKc) {
                        constexpr int kk = decltype(KKc)::value, k = K0 + kk;
                        if constexpr (in_box<LC, LD>(k, l, t2, u2, v2)) {
                            constexpr int sy = cart_y(LC, k) + ly, sz = cart_z(LC, k) + lz;
                            const T e = kt[kt_off<LC, LD>(l, k) + (t2 * (sy + 1) + u2) * (sz + 1) + v2];
#pragma unroll
                            for (int P = 0; P < NHB; ++P) Y[kk * NHB + P] = fma(e, r[P], Y[kk * NHB + P]);
                        }
                    });
                }
            });
        });
    });
}

// R^0_{tuv} of eq. 21-25 built in place in a shared-memory column (element i at R[i * 32]); same sweep as rtable<L>.
template <int L, int RS, class T>
__device__ __forceinline__ void rtable_sm(T alpha, T X, T Y, T Z, const T* __restrict__ F, T* R) {
    T fac[L + 1];
    fac[0] = T(1);
#pragma unroll
    for (int m = 1; m <= L; ++m) fac[m] = fac[m - 1] * (T(-2) * alpha);
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
                    T r;
                    if (t > 0) {
                        r = X * R[tidx<L>(t - 1, u, v) * RS];
                        if (t > 1) r = fma(T(t - 1), R[tidx<L>(t - 2, u, v) * RS], r);
                    } else if (u > 0) {
                        r = Y * R[tidx<L>(t, u - 1, v) * RS];
                        if (u > 1) r = fma(T(u - 1), R[tidx<L>(t, u - 2, v) * RS], r);
                    } else {
                        r = Z * R[tidx<L>(t, u, v - 1) * RS];
                        if (v > 1) r = fma(T(v - 1), R[tidx<L>(t, u, v - 2) * RS], r);
                    }
                    R[tidx<L>(t, u, v) * RS] = r;
                }
            }
        }
        R[0] = fac[m] * F[m];
    }
}

// T = double: the FP64 path.  T = float: the FP32 leg of the mixed-precision build: pair data, Boys values and the
// prefactor are formed in FP64 and rounded once; R, the E tables, both transforms and the digestion run in FP32; every quartet's
// sums are added to the FP64 J / K accumulators.
template <class T, int LA, int LB, int LC, int LD>
__global__ void __launch_bounds__(WARP) jkw_kernel(JKArgs a) {
    using S = WShape<LA, LB, LC, LD, T>;
    constexpr int LAB = S::LAB, LCD = S::LCD, L = S::L;
    constexpr int NA = S::NA, NB = S::NB, NC = S::NC, ND = S::ND, NHB = S::NHB;
    constexpr bool KEEPC = S::KEEPC;
    constexpr bool UNR = S::UNR;
    constexpr int UNK = S::UNK;
    constexpr int NL = S::NL;
    constexpr unsigned FULLMASK = 0xffffffffu;
    extern __shared__ double sm_raw[];
    T* const Rsm = reinterpret_cast<T*>(sm_raw);
    T* const kt = Rsm + S::NR * NL;
    T* const e1 = kt + S::NNZK;
    T* const dcd = e1 + 3 * S::NE1;
    const int lane = threadIdx.x;
    T* const Rl = Rsm + (lane < NL ? lane : 0);   // lanes >= NL never hold a quartet
    T* const kcl = dcd + NC * ND + lane;          // K_?c accumulator column of this lane (only without KEEPC)
    constexpr bool F32 = sizeof(T) == 4;
    if (F32 != (a.prec_mode == 2)) return;        // the FP32 instantiation serves the FP32 leg and nothing else

    const unsigned long long ntasks = a.ctrl->ntiles[a.slot];
    const long long span = (long long)NL * a.ctrl->chunk[a.slot];
    const long long ns = a.nshells;
    const long long nbf = a.nbf;
    long long cached_j = -1;
    PairD kp;
    PairIds ik;
    double qk = 0.0;
    unsigned int nlive = 0, nvis = 0, nslot = 0;

    while (true) {
        unsigned int task = 0;
        if (lane == 0) task = atomicAdd(&a.ctrl->tile_counter[a.slot], 1u);
        task = __shfl_sync(FULLMASK, task, 0);
        if (task >= ntasks) break;
        long long lo = 0, hi = a.nk;   // last ket j with tile_start[j] <= task
        while (hi - lo > 1) { const long long mid = (lo + hi) >> 1; if ((unsigned long long)a.tile_start[mid] <= task) lo = mid; else hi = mid; }
        const long long j = lo;
        const long long b_lo = (a.same ? j : 0) + ((long long)task - a.tile_start[j]) * span;
        const long long b_hi = min((long long)a.task_hi[j], b_lo + span);

        if (j != cached_j) {
            // ---- ket-uniform tables: 1-D E coefficients (signed), their products per (k,l,Q) in loop order, density block
            __syncwarp();
            kp = a.pk[j]; ik = a.ik[j]; qk = a.qk[j];
            if (lane < 3) {
                double E[LC + 1][LD + 1][LCD + 1];
                const double PA = lane == 0 ? kp.PA[0] : (lane == 1 ? kp.PA[1] : kp.PA[2]);
                const double PB = lane == 0 ? kp.PB[0] : (lane == 1 ? kp.PB[1] : kp.PB[2]);
                etable<LC, LD, true>(PA, PB, 0.5 / kp.p, E);
#pragma unroll
                for (int i = 0; i <= LC; ++i)
#pragma unroll
                    for (int jj = 0; jj <= LD; ++jj)
#pragma unroll
                        for (int t = 0; t <= LCD; ++t) e1[lane * S::NE1 + (i * (LD + 1) + jj) * (LCD + 1) + t] = (T)E[i][jj][t];
            }
            __syncwarp();
            int e = 0;
            for (int l = 0; l < ND; ++l) {
                const int lx = cart_x(LD, l), ly = cart_y(LD, l), lz = cart_z(LD, l);
                for (int k = 0; k < NC; ++k) {
                    const int kx = cart_x(LC, k), ky = cart_y(LC, k), kz = cart_z(LC, k);
                    const T* ex = e1 + (kx * (LD + 1) + lx) * (LCD + 1);
                    const T* ey = e1 + S::NE1 + (ky * (LD + 1) + ly) * (LCD + 1);
                    const T* ez = e1 + 2 * S::NE1 + (kz * (LD + 1) + lz) * (LCD + 1);
                    for (int t2 = 0; t2 <= kx + lx; ++t2)
                        for (int u2 = 0; u2 <= ky + ly; ++u2)
                            for (int v2 = 0; v2 <= kz + lz; ++v2, ++e)
                                if ((e & 31) == lane) kt[e] = ex[t2] * ey[u2] * ez[v2] * (T)kp.pref;
                }
            }
            for (int cd = lane; cd < NC * ND; cd += WARP) dcd[cd] = (T)a.Ds[(ik.offA + cd / ND) * nbf + ik.offB + cd % ND];
            __syncwarp();
            cached_j = j;
        }

        for (long long b0 = b_lo; b0 < b_hi; b0 += NL) {
            const long long bi = b0 + lane;
            bool active = lane < NL && bi < b_hi;
            PairD bp;
            PairIds ib;
            bool live_jab = false, live_jcd = false, live_kac = false, live_kbc = false, live_kad = false, live_kbd = false;
            if (active) {
                ++nvis;
                ib = a.ib[bi];
                const double qq = a.qb[bi] * qk;
                const double d1 = a.Dm[ik.shA * ns + ik.shB], d2 = a.Dm[ib.shA * ns + ib.shB], d3 = a.Dm[ib.shB * ns + ik.shB];
                const double d4 = a.Dm[ib.shA * ns + ik.shB], d5 = a.Dm[ib.shB * ns + ik.shA], d6 = a.Dm[ib.shA * ns + ik.shA];
                live_jab = qq * d1 >= a.tau;
                live_jcd = qq * d2 >= a.tau;
                live_kac = qq * d3 >= a.tau;
                live_kbc = qq * d4 >= a.tau;
                live_kad = qq * d5 >= a.tau;
                live_kbd = qq * d6 >= a.tau;
                active = live_jab | live_jcd | live_kac | live_kbc | live_kad | live_kbd;
                // mixed precision: this launch evaluates either the FP64 or the FP32 quartets (rule: fp32_quartet in te_kernels.cuh)
                if (a.prec_mode && fp32_quartet(a, qq, fmax(fmax(fmax(d1, d2), fmax(d3, d4)), fmax(d5, d6)), kp.p) != F32) active = false;
            }
            if (!__any_sync(FULLMASK, active)) continue;
            ++nslot;
            const bool any_jcd = __any_sync(FULLMASK, live_jcd);
            // Runs of lanes whose bras are primitive pairs of ONE contracted shell pair (the lists are shell-pair-major) share every
            // bra-side output address: their contributions are summed by a segmented shuffle reduction and the run's first lane
            // issues the atomic.  dist = lanes from this one to the end of its run.
            const int key = (lane < NL && bi < b_hi) ? (int)(ib.shA * ns + ib.shB) : -1 - lane;
            const int prev = __shfl_up_sync(FULLMASK, key, 1);
            const bool head = lane == 0 || key != prev;
            const unsigned heads = __ballot_sync(FULLMASK, head);
            const unsigned above = lane == 31 ? 0u : (heads >> (lane + 1)) << (lane + 1);
            const int dist = (above ? __ffs(above) - 1 : 32) - lane;
            const int maxdist = __reduce_max_sync(FULLMASK, dist);
            const bool runs = maxdist > 1;   // warp-uniform: without runs every lane adds its own contribution directly
            double f = 1.0;
            T Ebx[LA + 1][LB + 1][LAB + 1], Eby[LA + 1][LB + 1][LAB + 1], Ebz[LA + 1][LB + 1][LAB + 1];
            T dab[NA * NB], jab[NA * NB];
            T dbc[KEEPC ? NB * NC : 1], dac[KEEPC ? NA * NC : 1], kac[KEEPC ? NA * NC : 1], kbc[KEEPC ? NB * NC : 1];
#pragma unroll
            for (int x = 0; x < NA * NB; ++x) jab[x] = 0.0;
            if (KEEPC) {
#pragma unroll
                for (int x = 0; x < NA * NC; ++x) kac[x] = 0.0;
#pragma unroll
                for (int x = 0; x < NB * NC; ++x) kbc[x] = 0.0;
            } else {
#pragma unroll
                for (int x = 0; x < S::NKC; ++x) kcl[x * NL] = 0.0;
            }
            // D is symmetric and K = Kt + Kt^T is formed at the end: bra-ket density elements are read, and K contributions added, at
            // [ket AO row][bra AO column] -- the ket is warp-uniform, so a warp touches a few rows instead of scattered ones
            const double* Da = nullptr;                                     // rows of the scaled density at the bra's first shell (D_ab)
            const double* const Dc = a.Ds + (long long)ik.offA * nbf;       // rows at the ket's AOs
            const double* const Dd = a.Ds + (long long)ik.offB * nbf;
            if (active) {
                ++nlive;
                bp = a.pb[bi];
                if (ib.m == ib.n) f *= 0.5;
                if (ik.m == ik.n) f *= 0.5;
                if (a.same && bi == j) f *= 0.5;
                const double p = bp.p, q = kp.p;
                double alpha, pref;
                eri_scale(p, bp.rp, q, kp.rp, a.omega2, alpha, pref);
                const double X = bp.P[0] - kp.P[0], Y = bp.P[1] - kp.P[1], Z = bp.P[2] - kp.P[2];
                double F[L + 1];
                boys<L>(alpha * (X * X + Y * Y + Z * Z), a.boys_tab, F);
                // 2 pi^{5/2} / (p q sqrt(p+q)) (eq. 30) x bra prefactor x symmetry factor, folded into the Boys values
                pref *= bp.pref * f;
#pragma unroll
                for (int m = 0; m <= L; ++m) F[m] *= pref;
                T Fv[L + 1];
#pragma unroll
                for (int m = 0; m <= L; ++m) Fv[m] = (T)F[m];
                rtable_sm<L, NL, T>((T)alpha, (T)X, (T)Y, (T)Z, Fv, Rl);
                const T hb = (T)(0.5 * bp.rp);
                etable<LA, LB, false>((T)bp.PA[0], (T)bp.PB[0], hb, Ebx);
                etable<LA, LB, false>((T)bp.PA[1], (T)bp.PB[1], hb, Eby);
                etable<LA, LB, false>((T)bp.PA[2], (T)bp.PB[2], hb, Ebz);
                Da = a.Ds + (long long)ib.offA * nbf;
#pragma unroll
                for (int i = 0; i < NA; ++i)
#pragma unroll
                    for (int jj = 0; jj < NB; ++jj) dab[i * NB + jj] = (T)Da[i * nbf + ib.offB + jj];
                if (KEEPC) {
#pragma unroll
                    for (int k = 0; k < NC; ++k) {
#pragma unroll
                        for (int i = 0; i < NA; ++i) dac[i * NC + k] = (T)Dc[k * nbf + ib.offA + i];
#pragma unroll
                        for (int jj = 0; jj < NB; ++jj) dbc[jj * NC + k] = (T)Dc[k * nbf + ib.offB + jj];
                    }
                }
            }
            int ptr = 0;
#pragma unroll UNK
            for (int l = 0; l < ND; ++l) {
                const int lx = cart_x(LD, l), ly = cart_y(LD, l), lz = cart_z(LD, l);
                T dal[NA], dbl[NB], kal[NA], kbl[NB];
#pragma unroll
                for (int i = 0; i < NA; ++i) kal[i] = 0.0;
#pragma unroll
                for (int jj = 0; jj < NB; ++jj) kbl[jj] = 0.0;
                if (active) {
#pragma unroll
                    for (int i = 0; i < NA; ++i) dal[i] = Dd[l * nbf + ib.offA + i];
#pragma unroll
                    for (int jj = 0; jj < NB; ++jj) dbl[jj] = Dd[l * nbf + ib.offB + jj];
                }
                T Yall[S::KBAT ? S::KBN * NHB : 1];
                // always_inline: called from NC sites in the k-batched form; an out-of-line lambda would push every captured array to the stack
                auto kbody = [&](const int k, auto KK) __attribute__((always_inline)) {   // KK: position of k in Yall (k-batched), -1 otherwise
                    constexpr int kk = decltype(KK)::value;
                    const int sx = cart_x(LC, k) + lx, sy = cart_y(LC, k) + ly, sz = cart_z(LC, k) + lz;
                    T jkl = 0.0;
                    T kak[KEEPC ? 1 : NA], kbk[KEEPC ? 1 : NB];
                    if (!KEEPC) {
#pragma unroll
                        for (int i = 0; i < NA; ++i) kak[i] = 0.0;
#pragma unroll
                        for (int jj = 0; jj < NB; ++jj) kbk[jj] = 0.0;
                    }
                    if (active) {
                        // ---- ket Hermite -> Cartesian for this (k,l): Y_P = sum_Q E~_Q R_{P+Q}
                        T Yv[NHB];
#pragma unroll
                        for (int P = 0; P < NHB; ++P) Yv[P] = 0.0;
                        const T* ktp = kt + ptr;
                        if constexpr (kk >= 0) {
#pragma unroll
                            for (int P = 0; P < NHB; ++P) Yv[P] = Yall[(kk >= 0 ? kk : 0) * NHB + P];
                        } else if constexpr (UNR) {
#pragma unroll
                            for (int t2 = 0; t2 <= sx; ++t2)
#pragma unroll
                                for (int u2 = 0; u2 <= sy; ++u2)
#pragma unroll
                                    for (int v2 = 0; v2 <= sz; ++v2) {
                                        const T e = *ktp++;
#pragma unroll
                                        for (int t = 0; t <= LAB; ++t)
#pragma unroll
                                            for (int u = 0; u <= LAB - t; ++u)
#pragma unroll
                                                for (int v = 0; v <= LAB - t - u; ++v)
                                                    Yv[tidx<LAB>(t, u, v)] = fma(e, Rl[(tidx<L>(t + t2, u + u2, 0) + v + v2) * NL], Yv[tidx<LAB>(t, u, v)]);
                                    }
                        } else {
                            // (t2,u2) run over the whole ket triangle at compile time and the (warp-uniform) box limits of this
                            // (k,l) skip the rest, so every R offset is an immediate: one running pointer per v2, no row table
                            static_for<LCD + 1>([&](auto T2) {
                                constexpr int t2 = decltype(T2)::value;
                                if (t2 <= sx) {
                                    static_for<LCD + 1 - t2>([&](auto U2) {
                                        constexpr int u2 = decltype(U2)::value;
                                        if constexpr (S::V2CT) {
                                            if (u2 <= sy) {
                                                static_for<LCD + 1 - t2 - u2>([&](auto V2) {
                                                    constexpr int v2 = decltype(V2)::value;
                                                    if (v2 <= sz) {
                                                        const T e = *ktp++;
#pragma unroll
                                                        for (int t = 0; t <= LAB; ++t)
#pragma unroll
                                                            for (int u = 0; u <= LAB - t; ++u)
#pragma unroll
                                                                for (int v = 0; v <= LAB - t - u; ++v)
                                                                    Yv[tidx<LAB>(t, u, v)] = fma(e, Rl[(tidx<L>(t + t2, u + u2, 0) + v + v2) * NL], Yv[tidx<LAB>(t, u, v)]);
                                                    }
                                                });
                                            }
                                        } else if (u2 <= sy) {
                                            const T* Rq = Rl;
#pragma unroll 1
                                            for (int v2 = 0; v2 <= sz; ++v2, Rq += NL) {
                                                const T e = *ktp++;
#pragma unroll
                                                for (int t = 0; t <= LAB; ++t)
#pragma unroll
                                                    for (int u = 0; u <= LAB - t; ++u)
#pragma unroll
                                                        for (int v = 0; v <= LAB - t - u; ++v)
                                                            Yv[tidx<LAB>(t, u, v)] = fma(e, Rq[(tidx<L>(t + t2, u + u2, 0) + v) * NL], Yv[tidx<LAB>(t, u, v)]);
                                            }
                                        }
                                    });
                                }
                            });
                        }
                        // ---- bra Hermite -> Cartesian and digestion
                        T dbk[KEEPC ? 1 : NB], dak[KEEPC ? 1 : NA];
                        if (!KEEPC) {
#pragma unroll
                            for (int i = 0; i < NA; ++i) dak[i] = Dc[k * nbf + ib.offA + i];
#pragma unroll
                            for (int jj = 0; jj < NB; ++jj) dbk[jj] = Dc[k * nbf + ib.offB + jj];
                        }
                        const T dkl = dcd[k * ND + l];
#pragma unroll
                        for (int i = 0; i < NA; ++i) {
                            const int ix = cart_x(LA, i), iy = cart_y(LA, i), iz = cart_z(LA, i);
#pragma unroll
                            for (int jj = 0; jj < NB; ++jj) {
                                const int jx = cart_x(LB, jj), jy = cart_y(LB, jj), jz = cart_z(LB, jj);
                                T s = 0.0;
#pragma unroll
                                for (int t = 0; t <= ix + jx; ++t) {
                                    T su = 0.0;
#pragma unroll
                                    for (int u = 0; u <= iy + jy; ++u) {
                                        T sv = 0.0;
#pragma unroll
                                        for (int v = 0; v <= iz + jz; ++v) sv = fma(Ebz[iz][jz][v], Yv[tidx<LAB>(t, u, v)], sv);
                                        su = fma(Eby[iy][jy][u], sv, su);
                                    }
                                    s = fma(Ebx[ix][jx][t], su, s);
                                }
                                // s = f (ij|kl) without the per-component factors
                                jab[i * NB + jj] = fma(s, dkl, jab[i * NB + jj]);
                                jkl = fma(s, dab[i * NB + jj], jkl);
                                if (KEEPC) {
                                    kac[i * NC + k] = fma(s, dbl[jj], kac[i * NC + k]);
                                    kbc[jj * NC + k] = fma(s, dal[i], kbc[jj * NC + k]);
                                    kal[i] = fma(s, dbc[jj * NC + k], kal[i]);
                                    kbl[jj] = fma(s, dac[i * NC + k], kbl[jj]);
                                } else {
                                    kak[i] = fma(s, dbl[jj], kak[i]);
                                    kbk[jj] = fma(s, dal[i], kbk[jj]);
                                    kal[i] = fma(s, dbk[jj], kal[i]);
                                    kbl[jj] = fma(s, dak[i], kbl[jj]);
                                }
                            }
                        }
                        if (!live_jcd) jkl = 0.0;
                    }
                    if (!KEEPC) {   // sum over l in the lane's shared-memory column (inactive lanes add zeros)
#pragma unroll
                        for (int i = 0; i < NA; ++i) kcl[(i * NC + k) * NL] += kak[i];
#pragma unroll
                        for (int jj = 0; jj < NB; ++jj) kcl[(NA * NC + jj * NC + k) * NL] += kbk[jj];
                    }
                    ptr += (sx + 1) * (sy + 1) * (sz + 1);
                    if (any_jcd) {
#pragma unroll
                        for (int o = 16; o > 0; o >>= 1) jkl += __shfl_xor_sync(FULLMASK, jkl, o);
                        if (lane == 0) atomicAdd(&a.Jt[(ik.offA + k) * nbf + ik.offB + l], 2.0 * jkl);
                    }
                };
                if constexpr (S::KBAT) {
                    static_for<S::NKB>([&](auto KBc) __attribute__((always_inline)) {
                        constexpr int kb = decltype(KBc)::value;
                        if (active) {
                            static_for<ND>([&](auto Lc) {
                                if (l == decltype(Lc)::value) ket_batch<T, LAB, LC, LD, NL, decltype(Lc)::value, kb * S::KBN, S::KBN>(Rl, kt, Yall);
                            });
                        }
                        static_for<S::KBN>([&](auto KK) __attribute__((always_inline)) { kbody(kb * S::KBN + decltype(KK)::value, KK); });
                    });
                } else {
#pragma unroll UNK
                    for (int k = 0; k < NC; ++k) kbody(k, std::integral_constant<int, -1>{});
                }
                flush_vec<NA>(runs, maxdist, dist, head, live_kad, kal, [&](int i) { return &a.Kt[(ik.offB + l) * nbf + ib.offA + i]; });
                flush_vec<NB>(runs, maxdist, dist, head, live_kbd, kbl, [&](int jj) { return &a.Kt[(ik.offB + l) * nbf + ib.offB + jj]; });
            }
#pragma unroll
            for (int x = 0; x < NA * NB; ++x) jab[x] *= 2.0;
            flush_vec<NA * NB>(runs, maxdist, dist, head, live_jab, jab, [&](int x) { return &a.Jt[(ib.offA + x / NB) * nbf + ib.offB + x % NB]; });
            if (KEEPC) {
                flush_vec<(KEEPC ? NA * NC : 1)>(runs, maxdist, dist, head, live_kac, kac, [&](int x) { return &a.Kt[(ik.offA + x % NC) * nbf + ib.offA + x / NC]; });
                flush_vec<(KEEPC ? NB * NC : 1)>(runs, maxdist, dist, head, live_kbc, kbc, [&](int x) { return &a.Kt[(ik.offA + x % NC) * nbf + ib.offB + x / NC]; });
            } else {
                // the quartet's K_ac / K_bc sums come back from the shared-memory column, NC values (one row of the block) at a time
#pragma unroll 1
                for (int r = 0; r < NA + NB; ++r) {
                    T row[NC];
#pragma unroll
                    for (int k = 0; k < NC; ++k) row[k] = kcl[(r * NC + k) * NL];
                    const long long o1 = (r < NA ? ib.offA + r : ib.offB + (r - NA));
                    flush_vec<NC>(runs, maxdist, dist, head, r < NA ? live_kac : live_kbc, row, [&](int k) { return &a.Kt[(ik.offA + k) * nbf + o1]; });
                }
            }
            __syncwarp();
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        nlive += __shfl_down_sync(FULLMASK, nlive, o); nvis += __shfl_down_sync(FULLMASK, nvis, o); nslot += __shfl_down_sync(FULLMASK, nslot, o);
    }
    if (lane == 0 && nvis) {
        atomicAdd(&a.ctrl->live[a.slot], (unsigned long long)nlive);
        atomicAdd(&a.ctrl->visited[a.slot], (unsigned long long)nvis);
        atomicAdd(&a.ctrl->slots[a.slot], (unsigned long long)nslot);
    }
}

// Task schedule of the uniform-ket kernel.  For ket j the live bras are a contiguous range of the (bound-sorted) bra list:
// [same ? j : 0, cut_j) with cut_j = first bra whose q_bra * q_ket[j] * max|D| < tau (eq. 47, loosest density bound); a task is
// (ket j, chunk of 32*chunk bras).  task_hi[j] = cut_j, tile_start = exclusive prefix sum of the chunk counts.
static __global__ void __launch_bounds__(1024) schedule_w_kernel(const double* __restrict__ qb, long long nb, const double* __restrict__ qk,
                                                          long long nk, int same, double tau, int target_warps, int lanes, int chunk_cap,
                                                          long long* __restrict__ tile_start, int* __restrict__ task_hi, JKControl* ctrl, int slot) {
    __shared__ long long part[1024];
    __shared__ int s_chunk;
    const long long per = (nk + blockDim.x - 1) / blockDim.x;
    const long long j0 = threadIdx.x * per, j1 = min(nk, j0 + per);
    const double dmax = ctrl->dmax;
    long long tot = 0;
    for (long long j = j0; j < j1; ++j) {
        long long cut;
        if (tau <= 0.0) cut = nb;
        else {
            const double w = qk[j] * dmax;
            if (!(w > 0.0)) cut = 0;
            else {
                const double thr = tau / w * (1.0 - 1e-12);
                long long lo = 0, hi = nb;   // first bra index with qb < thr
                while (lo < hi) { const long long mid = (lo + hi) >> 1; if (qb[mid] >= thr) lo = mid + 1; else hi = mid; }
                cut = lo;
            }
        }
        const long long lo_j = same ? j : 0;
        if (cut < lo_j) cut = lo_j;
        task_hi[j] = (int)cut;
        tot += cut - lo_j;
    }
    part[threadIdx.x] = tot;
    __syncthreads();
    for (int o = blockDim.x >> 1; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) part[threadIdx.x] += part[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        // chunk: 32*chunk bras per task, sized so every resident warp gets ~8 tasks; 1..chunk_cap (every task pays two binary
        // searches of dependent global loads, ~10^4 cycles of latency, which the light classes cannot hide behind 16 batches)
        long long c = part[0] / ((long long)lanes * target_warps * 8);
        s_chunk = (int)max(1LL, min((long long)chunk_cap, c));
        // the task counters of the kernels are 32 bit: widen the tasks until their number fits (never reached by the five configs)
        while (part[0] / ((long long)lanes * s_chunk) + nk >= 0xfffffff0LL) s_chunk *= 2;
        ctrl->chunk[slot] = s_chunk;
    }
    __syncthreads();
    const long long span = (long long)lanes * s_chunk;
    long long s = 0;
    for (long long j = j0; j < j1; ++j) s += ((long long)task_hi[j] - (same ? j : 0) + span - 1) / span;
    __syncthreads();
    part[threadIdx.x] = s;
    __syncthreads();
    for (int o = 1; o < 1024; o <<= 1) {
        long long v = ((int)threadIdx.x >= o) ? part[threadIdx.x - o] : 0;
        __syncthreads();
        part[threadIdx.x] += v;
        __syncthreads();
    }
    long long run = part[threadIdx.x] - s;
    for (long long j = j0; j < j1; ++j) { tile_start[j] = run; run += ((long long)task_hi[j] - (same ? j : 0) + span - 1) / span; }
    if (threadIdx.x == blockDim.x - 1) { tile_start[nk] = part[threadIdx.x]; ctrl->ntiles[slot] = (unsigned long long)part[threadIdx.x]; }
}

}  // namespace te
