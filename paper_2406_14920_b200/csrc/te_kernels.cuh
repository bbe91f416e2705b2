// te_kernels.cuh -- per-angular-class kernels: Schwarz bounds + pair data, the J/K build and integral blocks.
// One template instantiation per (la lb|lc ld) class; instantiated and dispatched in te_inst_*.cu.
#pragma once
#include "te_internal.h"

namespace te {

// Number of non-zero Hermite coefficients of a pair class: sum over components of prod (i_tau + j_tau + 1).
__host__ __device__ constexpr int nnz_e(int la, int lb) {
    int s = 0;
    for (int i = 0; i < ncart(la); ++i)
        for (int j = 0; j < ncart(lb); ++j)
            s += (cart_x(la, i) + cart_x(lb, j) + 1) * (cart_y(la, i) + cart_y(lb, j) + 1) * (cart_z(la, i) + cart_z(lb, j) + 1);
    return s;
}
// FMAs of the two Hermite->Cartesian transforms of one primitive quartet (SURVEY.md section 8d model).
__host__ __device__ constexpr int transform_fmas(int la, int lb, int lc, int ld) {
    return nherm(la + lb) * nnz_e(lc, ld) + nnz_e(la, lb) * ncart(lc) * ncart(ld);
}
// Fully unrolled, register-resident evaluation for cheap classes; rolled loops otherwise.
__host__ __device__ constexpr bool use_full_unroll(int la, int lb, int lc, int ld) {
    return (la + lb + lc + ld) <= 2;
}

// Pair data of primitive shells (m, n) (eq. 3).
struct BasisView {
    const double* exp_;
    const double* ct;
    const double* xyz;
    const int* shell;
    const int* off;
};

__device__ __forceinline__ void make_pair(const BasisView& bv, int m, int n, PairD& pd) {
    const double a = bv.exp_[m], b = bv.exp_[n];
    const double p = a + b, rp = 1.0 / p;
    double r2 = 0.0;
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        const double A = bv.xyz[3 * m + d], B = bv.xyz[3 * n + d];
        const double P = (a * A + b * B) * rp;
        pd.P[d] = P; pd.PA[d] = P - A; pd.PB[d] = P - B;
        r2 += (A - B) * (A - B);
    }
    pd.p = p;
    pd.rp = rp;
    pd.pref = bv.ct[m] * bv.ct[n] * exp(-a * b * rp * r2);
}

// Candidate index -> (m, n): class (la, lb) candidates are the na x nb grid of primitives (la < lb) or the
// lower triangle i <= j of the na x na grid (la == lb); by_l lists primitive ids of each l in ascending order,
// so (l_m, m) <= (l_n, n) holds by construction.
__device__ __forceinline__ void decode_candidate(long long idx, bool same, long long nb, const int* __restrict__ la_list,
                                                 const int* __restrict__ lb_list, int& m, int& n) {
    long long i, j;
    if (!same) {
        i = idx / nb; j = idx % nb;
    } else {   // idx = j*(j+1)/2 + i, i <= j
        j = (long long)((sqrt(8.0 * (double)idx + 1.0) - 1.0) * 0.5);
        while (j * (j + 1) / 2 > idx) --j;
        while ((j + 1) * (j + 2) / 2 <= idx) ++j;
        i = idx - j * (j + 1) / 2;
    }
    m = la_list[i]; n = lb_list[j];
}

// ---------------------------------------------------------------------------------- Schwarz bound, eq. 45
template <int LA, int LB>
struct DiagMaxEmit {
    double mx = 0.0;
    __device__ __forceinline__ void ket(int, int) {}
    __device__ __forceinline__ void ket_done(int, int) {}
    __device__ __forceinline__ void operator()(int i, int j, int k, int l, double v) {
        if (i == k && j == l) {
            const double f = comp_factor(LA, i) * comp_factor(LB, j);
            mx = fmax(mx, sqrt(fabs(v)) * f);
        }
    }
};

template <int LA, int LB>
__global__ void __launch_bounds__(64) schwarz_kernel(BasisView bv, const int* __restrict__ la_list, const int* __restrict__ lb_list,
                                                      long long nb, long long ncand, const double* __restrict__ boys_tab,
                                                      double* __restrict__ q, long long* __restrict__ idx_out) {
    const long long idx = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (idx >= ncand) return;
    int m, n;
    decode_candidate(idx, LA == LB, nb, la_list, lb_list, m, n);
    PairD pd;
    make_pair(bv, m, n, pd);
    DiagMaxEmit<LA, LB> em;
    md_quartet<LA, LB, LA, LB, use_full_unroll(LA, LB, LA, LB)>(pd, pd, boys_tab, em);
    q[idx] = em.mx;
    idx_out[idx] = idx;
}

template <int LA, int LB>
__global__ void pair_fill_kernel(BasisView bv, const int* __restrict__ la_list, const int* __restrict__ lb_list, long long nb,
                                 long long n, const long long* __restrict__ cand, PairD* __restrict__ pairs, PairIds* __restrict__ ids) {
    const long long x = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (x >= n) return;
    int m, nn;
    decode_candidate(cand[x], LA == LB, nb, la_list, lb_list, m, nn);
    PairD pd;
    make_pair(bv, m, nn, pd);
    pairs[x] = pd;
    PairIds id;
    id.m = m; id.n = nn; id.shA = bv.shell[m]; id.shB = bv.shell[nn]; id.offA = bv.off[m]; id.offB = bv.off[nn];
    ids[x] = id;
}

// ------------------------------------------------------------------------------------ J/K tile schedule
// Pair lists are sorted by bound, descending.  For bra tile bt (TB bras) the live kets are a prefix of the ket
// list: those with q_ket >= tau / (q_bra_max(bt) * max|D|) (eq. 47 with the loosest density bound); when bra and
// ket class coincide only kets <= bra are unique (eq. 46).  tile_start = exclusive prefix sum of ket-tile counts.
static __global__ void __launch_bounds__(1024) schedule_kernel(const double* __restrict__ qb, long long nb, const double* __restrict__ qk,
                                                        long long nk, int same, double tau, int TB, int TK,
                                                        long long* __restrict__ tile_start, JKControl* ctrl, int slot) {
    __shared__ long long part[1024];
    const long long nbt = (nb + TB - 1) / TB;
    const long long chunk = (nbt + blockDim.x - 1) / blockDim.x;
    const long long t0 = threadIdx.x * chunk, t1 = min(nbt, t0 + chunk);
    const double dmax = ctrl->dmax;
    auto ntk = [&](long long bt) -> long long {
        long long cut;
        if (tau <= 0.0) cut = nk;
        else {
            const double w = qb[bt * TB] * dmax;
            if (!(w > 0.0)) cut = 0;
            else {
                const double thr = tau / w * (1.0 - 1e-12);
                long long lo = 0, hi = nk;   // first index with qk < thr
                while (lo < hi) { const long long mid = (lo + hi) >> 1; if (qk[mid] >= thr) lo = mid + 1; else hi = mid; }
                cut = lo;
            }
        }
        if (same) cut = min(cut, min(nb, (bt + 1) * TB));
        return (cut + TK - 1) / TK;
    };
    long long s = 0;
    for (long long bt = t0; bt < t1; ++bt) s += ntk(bt);
    part[threadIdx.x] = s;
    __syncthreads();
    for (int o = 1; o < 1024; o <<= 1) {
        long long v = (threadIdx.x >= o) ? part[threadIdx.x - o] : 0;
        __syncthreads();
        part[threadIdx.x] += v;
        __syncthreads();
    }
    long long run = part[threadIdx.x] - s;
    for (long long bt = t0; bt < t1; ++bt) { tile_start[bt] = run; run += ntk(bt); }
    if (threadIdx.x == blockDim.x - 1) { tile_start[nbt] = part[threadIdx.x]; ctrl->ntiles[slot] = (unsigned long long)part[threadIdx.x]; }
}

// ----------------------------------------------------------------------------------------- J/K digestion
// One thread = one unique primitive quartet (mn|rs).  For each ket component pair (k,l) the integrals (ij|kl)
// stream through the emitter, which contracts them with the (component-scaled) density into
//   Jt[ab] += 2f (ij|kl) D[cd]     Jt[cd] += 2f (ij|kl) D[ab]
//   Kt[ac] += f (ij|kl) D[bd]      Kt[bc] += f (ij|kl) D[ad]      Kt[ad] += f (ij|kl) D[bc]      Kt[bd] += f (ij|kl) D[ac]
// (f = product of 1/2 for m==n, r==s, bra==ket: "halve the diagonal") with one masked flush per output
// element; J = Jt + Jt^T and K = Kt + Kt^T are formed by finish_kernel.
template <int LA, int LB, int LC, int LD>
struct JKEmit {
    static constexpr int NA = ncart(LA), NB = ncart(LB), NC = ncart(LC), ND = ncart(LD);
    const double* __restrict__ Ds;
    double* __restrict__ Jt;
    double* __restrict__ Kt;
    long long nbf;
    int oa, ob, oc, od;
    double f;
    bool live_jab, live_jcd, live_kac, live_kbc, live_kad, live_kbd;
    double dab[NA * NB], jab[NA * NB];
    double dkl, jkl;
    double dbl[NB], dbk[NB], dal[NA], dak[NA];
    double kik[NA], kil[NA], kjk[NB], kjl[NB];

    __device__ __forceinline__ void begin() {
#pragma unroll
        for (int i = 0; i < NA; ++i)
#pragma unroll
            for (int j = 0; j < NB; ++j) { dab[i * NB + j] = Ds[(oa + i) * nbf + ob + j]; jab[i * NB + j] = 0.0; }
    }
    __device__ __forceinline__ void ket(int k, int l) {
        dkl = Ds[(oc + k) * nbf + od + l]; jkl = 0.0;
#pragma unroll
        for (int j = 0; j < NB; ++j) { dbl[j] = Ds[(ob + j) * nbf + od + l]; dbk[j] = Ds[(ob + j) * nbf + oc + k]; kjk[j] = 0.0; kjl[j] = 0.0; }
#pragma unroll
        for (int i = 0; i < NA; ++i) { dal[i] = Ds[(oa + i) * nbf + od + l]; dak[i] = Ds[(oa + i) * nbf + oc + k]; kik[i] = 0.0; kil[i] = 0.0; }
    }
    __device__ __forceinline__ void operator()(int i, int j, int, int, double v) {
        jab[i * NB + j] = fma(v, dkl, jab[i * NB + j]);
        jkl = fma(v, dab[i * NB + j], jkl);
        kik[i] = fma(v, dbl[j], kik[i]);
        kil[i] = fma(v, dbk[j], kil[i]);
        kjk[j] = fma(v, dal[i], kjk[j]);
        kjl[j] = fma(v, dak[i], kjl[j]);
    }
    __device__ __forceinline__ void ket_done(int k, int l) {
        if (live_jcd) atomicAdd(&Jt[(oc + k) * nbf + od + l], 2.0 * f * jkl);
#pragma unroll
        for (int i = 0; i < NA; ++i) {
            if (live_kac) atomicAdd(&Kt[(oa + i) * nbf + oc + k], f * kik[i]);
            if (live_kad) atomicAdd(&Kt[(oa + i) * nbf + od + l], f * kil[i]);
        }
#pragma unroll
        for (int j = 0; j < NB; ++j) {
            if (live_kbc) atomicAdd(&Kt[(ob + j) * nbf + oc + k], f * kjk[j]);
            if (live_kbd) atomicAdd(&Kt[(ob + j) * nbf + od + l], f * kjl[j]);
        }
    }
    __device__ __forceinline__ void end() {
        if (live_jab) {
#pragma unroll
            for (int i = 0; i < NA; ++i)
#pragma unroll
                for (int j = 0; j < NB; ++j) atomicAdd(&Jt[(oa + i) * nbf + ob + j], 2.0 * f * jab[i * NB + j]);
        }
    }
};

struct JKArgs {
    const PairD* pb; const double* qb; const PairIds* ib; long long nb;
    const PairD* pk; const double* qk; const PairIds* ik; long long nk;
    const double* Ds; const double* Dm; double* Jt; double* Kt;
    const double* boys_tab;
    const int* bstart; int nblk;            // first pair of every contracted shell-pair block of the bra list, [nblk + 1]
    const double* DHb; const double* DHk;   // Hermite densities of the bra / ket pair lists (split-quartet kernel)
    double* JHb; double* JHk;               // Hermite J accumulators of the bra / ket pair lists
    const long long* tile_start;
    const int* task_hi;
    JKControl* ctrl;
    double tau;
    double omega2;                          // 0: 1/r (eq. 30); omega^2 > 0: erf(omega r)/r (eq. 32-33)
    double prec_thr, amax32;                // mixed precision: FP32 below this density-weighted bound / ket exponent limit
    int prec_mode;                          // 0: every quartet (FP64 build); 1: FP64 leg, 2: FP32 leg of te_build_jk_mixed
    int nbf, nshells, slot, same;
};

// Mixed precision ("integrals with a density weighted Schwartz upper bound above a threshold (1e-5 ...) are evaluated in
// double precision while the rest are evaluated in single precision").  Density-weighted bound of a quartet = q_bra q_ket times
// the largest of its six density bounds.  FP32 also needs (2 alpha)^L inside its range; alpha <= p_ket, so quartets whose ket
// exponent exceeds amax32 (set per class from L) stay in FP64.  Both legs evaluate this predicate with the same FP64 inputs.
__device__ __forceinline__ bool fp32_quartet(const JKArgs& a, double qq, double dmax6, double p_ket) {
    return qq * dmax6 < a.prec_thr && p_ket <= a.amax32;
}

template <int LA, int LB, int LC, int LD, int TB, int TK>
__global__ void __launch_bounds__(TB * TK, (TB * TK >= 256 ? 2 : 1)) jk_kernel(JKArgs a) {
    constexpr bool FULL = use_full_unroll(LA, LB, LC, LD);
    __shared__ unsigned int s_tile;
    const long long nbt = (a.nb + TB - 1) / TB;
    const unsigned long long ntiles = a.ctrl->ntiles[a.slot];
    unsigned int nlive = 0;
    while (true) {
        if (threadIdx.x == 0) s_tile = atomicAdd(&a.ctrl->tile_counter[a.slot], 1u);
        __syncthreads();
        const unsigned long long tile = s_tile;
        __syncthreads();
        if (tile >= ntiles) break;
        // bra tile: last bt with tile_start[bt] <= tile
        long long lo = 0, hi = nbt;
        while (hi - lo > 1) { const long long mid = (lo + hi) >> 1; if ((unsigned long long)a.tile_start[mid] <= tile) lo = mid; else hi = mid; }
        const long long bt = lo, kt = (long long)tile - a.tile_start[bt];
        const long long bi = bt * TB + threadIdx.x / TK, kj = kt * TK + threadIdx.x % TK;
        if (bi >= a.nb || kj >= a.nk || (a.same && kj > bi)) continue;
        const double qq = a.qb[bi] * a.qk[kj];
        const PairIds ib = a.ib[bi], ik = a.ik[kj];
        const long long ns = a.nshells;
        JKEmit<LA, LB, LC, LD> em;
        const double d1 = a.Dm[ik.shA * ns + ik.shB], d2 = a.Dm[ib.shA * ns + ib.shB], d3 = a.Dm[ib.shB * ns + ik.shB];
        const double d4 = a.Dm[ib.shA * ns + ik.shB], d5 = a.Dm[ib.shB * ns + ik.shA], d6 = a.Dm[ib.shA * ns + ik.shA];
        em.live_jab = qq * d1 >= a.tau;
        em.live_jcd = qq * d2 >= a.tau;
        em.live_kac = qq * d3 >= a.tau;
        em.live_kbc = qq * d4 >= a.tau;
        em.live_kad = qq * d5 >= a.tau;
        em.live_kbd = qq * d6 >= a.tau;
        if (!(em.live_jab | em.live_jcd | em.live_kac | em.live_kbc | em.live_kad | em.live_kbd)) continue;
        if (a.prec_mode == 1 && fp32_quartet(a, qq, fmax(fmax(fmax(d1, d2), fmax(d3, d4)), fmax(d5, d6)), a.pk[kj].p)) continue;
        ++nlive;
        double f = 1.0;
        if (ib.m == ib.n) f *= 0.5;
        if (ik.m == ik.n) f *= 0.5;
        if (a.same && bi == kj) f *= 0.5;
        em.f = f; em.Ds = a.Ds; em.Jt = a.Jt; em.Kt = a.Kt; em.nbf = a.nbf;
        em.oa = ib.offA; em.ob = ib.offB; em.oc = ik.offA; em.od = ik.offB;
        const PairD bra = a.pb[bi], ket = a.pk[kj];
        em.begin();
        md_quartet<LA, LB, LC, LD, FULL>(bra, ket, a.boys_tab, em, a.omega2);
        em.end();
    }
    for (int o = 16; o > 0; o >>= 1) nlive += __shfl_down_sync(0xffffffffu, nlive, o);
    if ((threadIdx.x & 31) == 0 && nlive) atomicAdd(&a.ctrl->live[a.slot], (unsigned long long)nlive);
}

// ------------------------------------------------------------------------ nuclear attraction, eq. 14-26
// One thread = one primitive shell pair, looping over all point charges.  The sum over the charges (eq. 16) is taken in
// Hermite space, VH_P = sum_C q_C R^0_P(p, P - C) (eq. 20-25 with alpha = p), and transformed once:
//   Vt[a_i][b_j] += f c~c~ K_ab (2 pi / p) sum_P E_P^{ij} VH_P     (eq. 26; f = 1/2 for m == n, V = (Vt + Vt^T) o ff^T afterwards,
// which is how an unordered pair stands for both ordered pairs).  The paper stores the results in pair order and scatters on the
// host; here the scatter is an FP64 atomic add on the device.
template <int LA, int LB>
__global__ void __launch_bounds__(64) nuclear_kernel(const PairD* __restrict__ pairs, const PairIds* __restrict__ ids, long long n,
                                                      int ncharge, const double4* __restrict__ chg, const double* __restrict__ boys_tab,
                                                      int nbf, double* __restrict__ Vt) {
    constexpr int LAB = LA + LB, NA = ncart(LA), NB = ncart(LB), NH = nherm(LAB);
    const long long x = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (x >= n) return;
    const PairD pd = pairs[x];
    const PairIds id = ids[x];
    double acc[NH];
#pragma unroll
    for (int P = 0; P < NH; ++P) acc[P] = 0.0;
    for (int c = 0; c < ncharge; ++c) {
        const double4 ch = chg[c];   // x, y, z, q_C: the same address for every thread
        const double X = pd.P[0] - ch.x, Y = pd.P[1] - ch.y, Z = pd.P[2] - ch.z;
        double F[LAB + 1], R[NH];
        boys<LAB>(pd.p * (X * X + Y * Y + Z * Z), boys_tab, F);
#pragma unroll
        for (int m = 0; m <= LAB; ++m) F[m] *= ch.w;
        rtable<LAB>(pd.p, X, Y, Z, F, R);
#pragma unroll
        for (int P = 0; P < NH; ++P) acc[P] += R[P];
    }
    double E[3][LA + 1][LB + 1][LAB + 1];
#pragma unroll
    for (int d = 0; d < 3; ++d) etable<LA, LB, false>(pd.PA[d], pd.PB[d], 0.5 * pd.rp, E[d]);
    const double pref = pd.pref * (6.28318530717958647692 * pd.rp) * (id.m == id.n ? 0.5 : 1.0);
    for (int i = 0; i < NA; ++i) {
        const int ix = cart_x(LA, i), iy = cart_y(LA, i), iz = cart_z(LA, i);
        for (int j = 0; j < NB; ++j) {
            const int jx = cart_x(LB, j), jy = cart_y(LB, j), jz = cart_z(LB, j);
            double s = 0.0;
            for (int t = 0; t <= ix + jx; ++t)
                for (int u = 0; u <= iy + jy; ++u) {
                    const double exy = E[0][ix][jx][t] * E[1][iy][jy][u];
                    for (int v = 0; v <= iz + jz; ++v) s = fma(exy * E[2][iz][jz][v], acc[tidx<LAB>(t, u, v)], s);
                }
            atomicAdd(&Vt[(long long)(id.offA + i) * nbf + id.offB + j], pref * s);
        }
    }
}

// ------------------------------------------------------------------------------- integral blocks (testing)
template <int LA, int LB, int LC, int LD>
struct StoreEmit {
    double* out;
    int si, sj, sk, sl;
    __device__ __forceinline__ void ket(int, int) {}
    __device__ __forceinline__ void ket_done(int, int) {}
    __device__ __forceinline__ void operator()(int i, int j, int k, int l, double v) {
        out[i * si + j * sj + k * sk + l * sl] += v * comp_factor(LA, i) * comp_factor(LB, j) * comp_factor(LC, k) * comp_factor(LD, l);
    }
};

template <int LA, int LB, int LC, int LD>
__global__ void __launch_bounds__(32) eri_block_kernel(BasisView bv, const int* __restrict__ shell_pstart, int n,
                                                        const EriTask* __restrict__ tasks, const double* __restrict__ boys_tab,
                                                        double* __restrict__ out) {
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    if (x >= n) return;
    const EriTask t = tasks[x];
    StoreEmit<LA, LB, LC, LD> em;
    em.out = out + t.out; em.si = t.stride[0]; em.sj = t.stride[1]; em.sk = t.stride[2]; em.sl = t.stride[3];
    for (int m = shell_pstart[t.sh[0]]; m < shell_pstart[t.sh[0] + 1]; ++m)
        for (int nn = shell_pstart[t.sh[1]]; nn < shell_pstart[t.sh[1] + 1]; ++nn) {
            PairD bra;
            make_pair(bv, m, nn, bra);
            for (int r = shell_pstart[t.sh[2]]; r < shell_pstart[t.sh[2] + 1]; ++r)
                for (int s = shell_pstart[t.sh[3]]; s < shell_pstart[t.sh[3] + 1]; ++s) {
                    PairD ket;
                    make_pair(bv, r, s, ket);
                    md_quartet<LA, LB, LC, LD, false>(bra, ket, boys_tab, em);
                }
        }
}

}  // namespace te
