// te_jkq.cuh -- "split-quartet" J/K kernel for the heavy angular classes.
//
// One primitive quartet (mn|rs) is worked on by G lanes of a warp (NQ = 32/G quartets per warp, W warps per block, all
// quartets of a block share the KET pair).  What a quartet owns -- its R^0_{tuv} tensor (eq. 21-25), the bra's 1-D Hermite
// expansion coefficients (eq. 5-8), four density blocks and the bra's Hermite density -- lives in shared memory once per
// quartet, not once per lane; what the ket owns (E~_Q^{kl} with the (-1)^{t'+u'+v'} of eq. 30 and the pair prefactor folded
// in, its Hermite density) lives once per block.  The G lanes of a quartet
//   * build R cooperatively, degree by degree (elements of equal t+u+v are independent),
//   * do the Coulomb part in Hermite space (eq. 35, the "J-engine" of P:243-248, 364-366):
//         JH_bra[P] += sum_Q (-1)^Q R_{P+Q} DH_ket[Q]        JH_ket[Q] += (-1)^Q sum_P R_{P+Q} DH_bra[P]
//     with P (resp. Q) dealt over the lanes; the Hermite <-> Cartesian transforms of D and J run once per pair per
//     build in hermite_density_kernel / hermite_j_kernel instead of on the CPU as in the paper,
//   * deal the ket component pairs (k,l) among themselves for the exchange part: per (k,l) a lane forms
//         Y_P = sum_{Q in box(kl)} E~_Q^{kl} R_{P+Q},     I_ij = sum_P E_P^{ij} Y_P        (eq. 31)
//     in registers and digests I_ij into the four K updates of the quartet (eq. 36) with the per-term masks of eq. 47.
#pragma once
#include "te_jkw.cuh"

namespace te {

// ------------------------------------------------------------------------------------------ class tables
// All compile-time, evaluated on the host, uploaded once per class and copied to shared memory by every block.
template <int LA, int LB, int LC, int LD>
struct QTab {
    static constexpr int LAB = LA + LB, LCD = LC + LD, L = LAB + LCD;
    static constexpr int NC = ncart(LC), ND = ncart(LD), NKL = NC * ND, NNZK = nnz_e(LC, LD);
    static constexpr int NHB = nherm(LAB), NHK = nherm(LCD), NR = nherm(L);
    // R recurrence recipe, elements ordered by degree n = t+u+v: R[e] = XYZ[dir] * R[s1] + c2 * R[s2]   (eq. 22-24);
    // rc[r] = {e, s1, s2, dir | c2 << 2}, read with one 8-byte load (first member: 8-byte aligned)
    unsigned short rc[NR][4];
    // ket component pairs in processing order (largest Hermite box first, so the lanes of a round do similar work)
    unsigned short kl_k[NKL], kl_l[NKL], kl_start[NKL + 1];
    unsigned short pk[NNZK];       // box entry -> t2 | u2 << 4 | v2 << 8
    unsigned short qkl[NNZK];      // box entry -> position of its (k,l) in the processing order
    unsigned short rowtab[13 * 13];   // (T,U) -> index of R_{T,U,0} in the tetrahedral layout of order L
    unsigned short hb[NHB], hk[NHK];  // Hermite index -> t | u << 4 | v << 8 (bra / ket tetrahedra)
    unsigned short deg_start[14];

    constexpr QTab() : rc{}, kl_k{}, kl_l{}, kl_start{}, pk{}, qkl{}, rowtab{}, hb{}, hk{}, deg_start{} {
        int order[NKL] = {}, size[NKL] = {};
        for (int k = 0; k < NC; ++k)
            for (int l = 0; l < ND; ++l) {
                const int x = k * ND + l;
                order[x] = x;
                size[x] = (cart_x(LC, k) + cart_x(LD, l) + 1) * (cart_y(LC, k) + cart_y(LD, l) + 1) * (cart_z(LC, k) + cart_z(LD, l) + 1);
            }
        for (int i = 1; i < NKL; ++i) {   // stable insertion sort, size descending
            const int o = order[i];
            int j = i - 1;
            while (j >= 0 && size[order[j]] < size[o]) { order[j + 1] = order[j]; --j; }
            order[j + 1] = o;
        }
        int pos = 0;
        for (int n = 0; n < NKL; ++n) {
            const int k = order[n] / ND, l = order[n] % ND;
            kl_k[n] = (unsigned short)k; kl_l[n] = (unsigned short)l; kl_start[n] = (unsigned short)pos;
            for (int t2 = 0; t2 <= cart_x(LC, k) + cart_x(LD, l); ++t2)
                for (int u2 = 0; u2 <= cart_y(LC, k) + cart_y(LD, l); ++u2)
                    for (int v2 = 0; v2 <= cart_z(LC, k) + cart_z(LD, l); ++v2) {
                        pk[pos] = (unsigned short)(t2 | (u2 << 4) | (v2 << 8));
                        qkl[pos] = (unsigned short)n;
                        ++pos;
                    }
        }
        kl_start[NKL] = (unsigned short)pos;
        for (int t = 0; t < 13; ++t)
            for (int u = 0; u < 13; ++u) rowtab[t * 13 + u] = (t + u <= L) ? (unsigned short)tidx<L>(t, u, 0) : (unsigned short)0;
        for (int t = 0; t <= LAB; ++t)
            for (int u = 0; u <= LAB - t; ++u)
                for (int v = 0; v <= LAB - t - u; ++v) hb[tidx<LAB>(t, u, v)] = (unsigned short)(t | (u << 4) | (v << 8));
        for (int t = 0; t <= LCD; ++t)
            for (int u = 0; u <= LCD - t; ++u)
                for (int v = 0; v <= LCD - t - u; ++v) hk[tidx<LCD>(t, u, v)] = (unsigned short)(t | (u << 4) | (v << 8));
        int r = 0;
        for (int n = 0; n <= L; ++n) {
            deg_start[n] = (unsigned short)r;
            for (int t = n; t >= 0; --t)
                for (int u = n - t; u >= 0; --u) {
                    const int v = n - t - u;
                    int dir = 0, s1 = 0, s2 = 0, c2 = 0;
                    if (n > 0) {
                        if (t > 0) { dir = 0; s1 = tidx<L>(t - 1, u, v); if (t > 1) { s2 = tidx<L>(t - 2, u, v); c2 = t - 1; } }
                        else if (u > 0) { dir = 1; s1 = tidx<L>(t, u - 1, v); if (u > 1) { s2 = tidx<L>(t, u - 2, v); c2 = u - 1; } }
                        else { dir = 2; s1 = tidx<L>(t, u, v - 1); if (v > 1) { s2 = tidx<L>(t, u, v - 2); c2 = v - 1; } }
                    }
                    rc[r][0] = (unsigned short)tidx<L>(t, u, v); rc[r][1] = (unsigned short)s1; rc[r][2] = (unsigned short)s2;
                    rc[r][3] = (unsigned short)(dir | (c2 << 2));
                    ++r;
                }
        }
        deg_start[L + 1] = (unsigned short)r;
    }
};

template <int LA, int LB, int LC, int LD, int G, int W>
struct QShape {
    using Tab = QTab<LA, LB, LC, LD>;
    static constexpr int LAB = LA + LB, LCD = LC + LD, L = LAB + LCD;
    static constexpr int NA = ncart(LA), NB = ncart(LB), NC = ncart(LC), ND = ncart(LD);
    static constexpr int NHB = nherm(LAB), NHK = nherm(LCD), NR = nherm(L), NKL = NC * ND, NNZK = nnz_e(LC, LD);
    static constexpr int NE1B = (LA + 1) * (LB + 1) * (LAB + 1), NE1K = (LC + 1) * (LD + 1) * (LCD + 1);
    static constexpr int NQ = 32 / G;
    static constexpr int NDB = NB * ND + NB * NC + NA * ND + NA * NC;
    static constexpr int slot_doubles = NR + 3 * NE1B + NDB + NHB;
    static constexpr int block_doubles = NNZK + NHK + 3 * NE1K;
    static constexpr int smem_bytes = 8 * (block_doubles + W * NQ * slot_doubles) + (int)((sizeof(Tab) + 7) / 8 * 8);
};

// lanes per quartet: enough ket component pairs per lane to keep the lanes busy, few enough quartets per warp that a block's
// shared memory fits the number of blocks per SM the registers allow
constexpr int jkq_smem(int la, int lb, int lc, int ld, int g, int w) {
    const int lab = la + lb, lcd = lc + ld, L = lab + lcd;
    const int ndb = ncart(lb) * ncart(ld) + ncart(lb) * ncart(lc) + ncart(la) * ncart(ld) + ncart(la) * ncart(lc);
    const int slot = nherm(L) + 3 * (la + 1) * (lb + 1) * (lab + 1) + ndb + nherm(lab);
    const int blk = nnz_e(lc, ld) + nherm(lcd) + 3 * (lc + 1) * (ld + 1) * (lcd + 1);
    return 8 * (blk + w * (32 / g) * slot) + 2 * (3 * nnz_e(lc, ld) + 2 * nherm(L) + 600);
}
constexpr int jkq_lanes(int la, int lb, int lc, int ld, int w) {
    const int nkl = ncart(lc) * ncart(ld);
    int g = nkl >= 100 ? 8 : nkl >= 30 ? 4 : 2;
    if (la + lb <= 3 && lc + ld <= 5) g = 2;   // measured: light bras gain 10 % from 16 quartets per warp ((PD|PF), (PD|DD))
    // blocks per SM are set by registers (launch bounds: 4 for light bras, 2 otherwise); shared memory may use the rest
    const int cap = nherm(la + lb) <= 10 ? 54 * 1024 : 110 * 1024;
    while (g < 32 && jkq_smem(la, lb, lc, ld, g, w) > cap) g *= 2;
    return g;
}

// classes for which the split-quartet kernel is instantiated, and those it handles by default.  Measured on B200 (configs 2,
// 3 and 5, per-class CUDA-event times): it wins for every FF ket, for DF kets against bras with la+lb >= 2, for d/f-heavy bras
// (la+lb >= 4) against kets with lc+ld >= 4, and for (SD|DD), (PD|PF), (PD|DD); one quartet per lane (uniform-ket kernel) wins
// elsewhere.  TE_JK_IMPL=3 forces it wherever it exists.
constexpr bool jkq_default(int la, int lb, int lc, int ld) {
    // round 2 (after the uniform-ket kernel stopped flushing per (k,l)): (SD|DF), (PP|DF) and (SD|DD) moved to the uniform-ket kernel
    if (lc == 2 && ld == 3 && ((la == 0 && lb == 2) || (la == 1 && lb == 1))) return false;
    // with the k-batched ket transform the uniform-ket kernel also wins for s / sp bras against ff kets ((SS|FF) 311 -> 135 ms, (SP|FF) 558 -> 413 ms)
    if (lc == 3 && ld == 3 && la == 0 && lb <= 1) return false;
    if (la == 0 && lb == 3 && lc == 2 && ld == 3) return false;   // (SF|DF): 497 -> 460 ms in the uniform-ket kernel
    return (lc + ld == 6) || (lc == 2 && ld == 3 && la + lb >= 2) || (la + lb >= 4 && lc + ld >= 4) ||
           (la == 1 && lb == 2 && lc + ld >= 4);
}
// instantiated exactly where it is the default (round 1 instantiated it for every class with L >= 3 so that family 3 could force it
// anywhere; that doubled the compile time of the library for kernels no build uses)
constexpr bool use_jkq(int la, int lb, int lc, int ld) { return jkq_default(la, lb, lc, ld); }

template <int LA, int LB, int LC, int LD, int G, int W>
__global__ void __launch_bounds__(32 * W, (nherm(LA + LB) <= 10 ? 4 : 2)) jkq_kernel(JKArgs a, const QTab<LA, LB, LC, LD>* __restrict__ gtab) {
    using S = QShape<LA, LB, LC, LD, G, W>;
    using Tab = QTab<LA, LB, LC, LD>;
    constexpr int LAB = S::LAB, LCD = S::LCD, L = S::L;
    constexpr int NA = S::NA, NB = S::NB, NC = S::NC, ND = S::ND, NHB = S::NHB, NHK = S::NHK, NR = S::NR;
    constexpr int NKL = S::NKL, NNZK = S::NNZK, NE1B = S::NE1B, NE1K = S::NE1K, NQ = S::NQ;
    constexpr int NJK = (NHK + G - 1) / G;   // ket Hermite-J accumulators per lane
    constexpr unsigned FULLMASK = 0xffffffffu;
    extern __shared__ double sm[];
    __shared__ unsigned int s_task;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int slot = lane % NQ, g = lane / NQ;
    double* const kt = sm;                        // [NNZK] E~ of the ket, processing order
    double* const sdhk = kt + NNZK;               // [NHK]  (-1)^Q * ket prefactor * Hermite density of the ket
    double* const e1 = sdhk + NHK;                // [3][NE1K] 1-D ket tables (scratch for kt)
    double* const wb = e1 + 3 * NE1K + warp * (NQ * S::slot_doubles);
    double* const Rs = wb + slot;                 // element e at Rs[e * NQ]
    double* const Eb = Rs + NR * NQ;              // [3][NE1B]
    double* const Dbd = Eb + 3 * NE1B * NQ;       // [NB][ND]
    double* const Dbc = Dbd + NB * ND * NQ;       // [NB][NC]
    double* const Dad = Dbc + NB * NC * NQ;       // [NA][ND]
    double* const Dac = Dad + NA * ND * NQ;       // [NA][NC]
    double* const dhb = Dac + NA * NC * NQ;       // [NHB] Hermite density of the bra (no prefactor)
    const Tab* const tab = reinterpret_cast<const Tab*>(sm + S::block_doubles + W * NQ * S::slot_doubles);
    {
        const unsigned short* src = reinterpret_cast<const unsigned short*>(gtab);
        unsigned short* dst = reinterpret_cast<unsigned short*>(sm + S::block_doubles + W * NQ * S::slot_doubles);
        for (int x = tid; x < (int)(sizeof(Tab) / 2); x += 32 * W) dst[x] = src[x];
    }
    __syncthreads();
    const unsigned short* const rt = tab->rowtab;

    const unsigned long long ntasks = a.ctrl->ntiles[a.slot];
    const long long span = (long long)NQ * W * a.ctrl->chunk[a.slot];
    const long long ns = a.nshells, nbf = a.nbf;
    long long cached_j = -1;
    PairD kp;
    PairIds ik;
    double qk = 0.0;
    unsigned int nlive = 0, nvis = 0, nslot = 0;

    while (true) {
        if (tid == 0) s_task = atomicAdd(&a.ctrl->tile_counter[a.slot], 1u);
        __syncthreads();
        const unsigned int task = s_task;
        __syncthreads();
        if (task >= ntasks) break;
        long long lo = 0, hi = a.nk;   // last ket j with tile_start[j] <= task
        while (hi - lo > 1) { const long long mid = (lo + hi) >> 1; if ((unsigned long long)a.tile_start[mid] <= task) lo = mid; else hi = mid; }
        const long long j = lo;
        const long long b_lo = (a.same ? j : 0) + ((long long)task - a.tile_start[j]) * span;
        const long long b_hi = min((long long)a.task_hi[j], b_lo + span);

        if (j != cached_j) {
            // ---- ket tables, once per block and ket: 1-D E coefficients (signed), E~ per box entry, Hermite density
            kp = a.pk[j]; ik = a.ik[j]; qk = a.qk[j];
            if (tid < 3) {
                double E[LC + 1][LD + 1][LCD + 1];
                const double PA = tid == 0 ? kp.PA[0] : (tid == 1 ? kp.PA[1] : kp.PA[2]);
                const double PB = tid == 0 ? kp.PB[0] : (tid == 1 ? kp.PB[1] : kp.PB[2]);
                etable<LC, LD, true>(PA, PB, 0.5 / kp.p, E);
#pragma unroll
                for (int i = 0; i <= LC; ++i)
#pragma unroll
                    for (int jj = 0; jj <= LD; ++jj)
#pragma unroll
                        for (int t = 0; t <= LCD; ++t) e1[tid * NE1K + (i * (LD + 1) + jj) * (LCD + 1) + t] = E[i][jj][t];
            }
            __syncthreads();
            for (int q = tid; q < NNZK; q += 32 * W) {
                const int n = tab->qkl[q], p = tab->pk[q];
                const int k = tab->kl_k[n], l = tab->kl_l[n];
                const int t2 = p & 15, u2 = (p >> 4) & 15, v2 = p >> 8;
                kt[q] = e1[(cart_x(LC, k) * (LD + 1) + cart_x(LD, l)) * (LCD + 1) + t2] *
                        e1[NE1K + (cart_y(LC, k) * (LD + 1) + cart_y(LD, l)) * (LCD + 1) + u2] *
                        e1[2 * NE1K + (cart_z(LC, k) * (LD + 1) + cart_z(LD, l)) * (LCD + 1) + v2] * kp.pref;
            }
            for (int Q = tid; Q < NHK; Q += 32 * W) {
                const int p = tab->hk[Q];
                const int par = ((p & 15) + ((p >> 4) & 15) + (p >> 8)) & 1;
                const double d = a.DHk[j * NHK + Q] * kp.pref;
                sdhk[Q] = par ? -d : d;
            }
            __syncthreads();
            cached_j = j;
        }

        double jhk[NJK];
#pragma unroll
        for (int x = 0; x < NJK; ++x) jhk[x] = 0.0;
        bool any_jcd_task = false;

        for (long long b0 = b_lo + (long long)warp * NQ; b0 < b_hi; b0 += (long long)W * NQ) {
            const long long bi = b0 + slot;
            bool active = bi < b_hi;
            PairIds ib;
            bool live_jab = false, live_jcd = false, live_kac = false, live_kbc = false, live_kad = false, live_kbd = false;
            if (active) {
                if (g == 0) ++nvis;
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
                // FP64 leg of a mixed-precision build: the FP32 quartets belong to the other launch
                if (a.prec_mode == 1 && fp32_quartet(a, qq, fmax(fmax(fmax(d1, d2), fmax(d3, d4)), fmax(d5, d6)), kp.p)) {
                    active = false; live_jab = live_jcd = live_kac = live_kbc = live_kad = live_kbd = false;
                }
            }
            if (!__any_sync(FULLMASK, active)) continue;
            if (g == 0) ++nslot;
            const bool any_jcd = __any_sync(FULLMASK, live_jcd);
            any_jcd_task |= any_jcd;
            const bool live_k = live_kac | live_kbc | live_kad | live_kbd;
            double X = 0.0, Y_ = 0.0, Z = 0.0, alpha = 0.0;
            double F[L + 1];
            if (active) {
                if (g == 0) ++nlive;
                const PairD bp = a.pb[bi];
                double f = 1.0;
                if (ib.m == ib.n) f *= 0.5;
                if (ik.m == ik.n) f *= 0.5;
                if (a.same && bi == j) f *= 0.5;
                const double p = bp.p, q = kp.p;
                double pref;
                eri_scale(p, bp.rp, q, kp.rp, a.omega2, alpha, pref);
                X = bp.P[0] - kp.P[0]; Y_ = bp.P[1] - kp.P[1]; Z = bp.P[2] - kp.P[2];
                boys<L>(alpha * (X * X + Y_ * Y_ + Z * Z), a.boys_tab, F);
                // 2 pi^{5/2} / (p q sqrt(p+q)) (eq. 30) x bra prefactor x symmetry factor, folded into the Boys values
                pref *= bp.pref * f;
#pragma unroll
                for (int m = 0; m <= L; ++m) F[m] *= pref;
                // bra 1-D E tables: one dimension per lane of the group
                for (int d = g; d < 3; d += G) {
                    double E[LA + 1][LB + 1][LAB + 1];
                    const double PA = d == 0 ? bp.PA[0] : (d == 1 ? bp.PA[1] : bp.PA[2]);
                    const double PB = d == 0 ? bp.PB[0] : (d == 1 ? bp.PB[1] : bp.PB[2]);
                    etable<LA, LB, false>(PA, PB, 0.5 * bp.rp, E);
#pragma unroll
                    for (int i = 0; i <= LA; ++i)
#pragma unroll
                        for (int jj = 0; jj <= LB; ++jj)
#pragma unroll
                            for (int t = 0; t <= LAB; ++t) Eb[(d * NE1B + (i * (LB + 1) + jj) * (LAB + 1) + t) * NQ] = E[i][jj][t];
                }
                // density blocks (scaled density) and the bra's Hermite density
                const double* Da = a.Ds + (long long)ib.offA * nbf;
                const double* Db = a.Ds + (long long)ib.offB * nbf;
                for (int x = g; x < NB * ND; x += G) Dbd[x * NQ] = Db[(x / ND) * nbf + ik.offB + x % ND];
                for (int x = g; x < NB * NC; x += G) Dbc[x * NQ] = Db[(x / NC) * nbf + ik.offA + x % NC];
                for (int x = g; x < NA * ND; x += G) Dad[x * NQ] = Da[(x / ND) * nbf + ik.offB + x % ND];
                for (int x = g; x < NA * NC; x += G) Dac[x * NQ] = Da[(x / NC) * nbf + ik.offA + x % NC];
                for (int P = g; P < NHB; P += G) dhb[P * NQ] = a.DHb[bi * NHB + P];
            }
            // ---- R^0_{tuv}, eq. 21-25, in place: level m from level m+1, degree n = t+u+v descending; the elements of one
            // degree are dealt over the G lanes of the quartet
            {
                double fac = 1.0;
#pragma unroll
                for (int m = 0; m < L; ++m) fac *= -2.0 * alpha;
                if (active && g == 0) Rs[0] = fac * F[L];
                __syncwarp();
                const double ra = (alpha != 0.0) ? -0.5 / alpha : 0.0;
#pragma unroll
                for (int m = L - 1; m >= 0; --m) {
                    fac *= ra;
                    for (int n = L - m; n >= 1; --n) {
                        const int s0 = tab->deg_start[n], cnt = tab->deg_start[n + 1] - s0;
                        if (active) {
                            for (int x = g; x < cnt; x += G) {
                                const uint2 rc = *reinterpret_cast<const uint2*>(&tab->rc[s0 + x][0]);
                                const int e = rc.x & 0xffff, s1 = rc.x >> 16, s2 = rc.y & 0xffff, dc = rc.y >> 16;
                                const int dir = dc & 3;
                                const double c = dir == 0 ? X : (dir == 1 ? Y_ : Z);
                                Rs[e * NQ] = fma((double)(dc >> 2), Rs[s2 * NQ], c * Rs[s1 * NQ]);
                            }
                        }
                        __syncwarp();
                    }
                    if (active && g == 0) Rs[0] = fac * F[m];
                    __syncwarp();
                }
            }
            // ---- Coulomb part in Hermite space
            if (live_jab) {
                for (int P = g; P < NHB; P += G) {
                    const int p = tab->hb[P];
                    const int t = p & 15, u = (p >> 4) & 15, v = p >> 8;
                    double s = 0.0;
                    const unsigned short* rtp = rt + t * 13 + u;
                    static_for<LCD + 1>([&](auto T2) {
                        constexpr int t2 = decltype(T2)::value;
                        static_for<LCD + 1 - t2>([&](auto U2) {
                            constexpr int u2 = decltype(U2)::value;
                            const double* Rrow = Rs + ((int)rtp[t2 * 13 + u2] + v) * NQ;
#pragma unroll
                            for (int v2 = 0; v2 <= LCD - t2 - u2; ++v2) s = fma(sdhk[tidx<LCD>(t2, u2, v2)], Rrow[v2 * NQ], s);
                        });
                    });
                    atomicAdd(&a.JHb[bi * NHB + P], 2.0 * s);
                }
            }
            if (any_jcd) {
#pragma unroll
                for (int x = 0; x < NJK; ++x) {
                    const int Q = g + x * G;
                    if (live_jcd && Q < NHK) {
                        const int p = tab->hk[Q];
                        const int t2 = p & 15, u2 = (p >> 4) & 15, v2 = p >> 8;
                        double s = 0.0;
                        const unsigned short* rtp = rt + t2 * 13 + u2;
                        static_for<LAB + 1>([&](auto T) {
                            constexpr int t = decltype(T)::value;
                            static_for<LAB + 1 - t>([&](auto U) {
                                constexpr int u = decltype(U)::value;
                                const double* Rrow = Rs + ((int)rtp[t * 13 + u] + v2) * NQ;
#pragma unroll
                                for (int v = 0; v <= LAB - t - u; ++v) s = fma(dhb[tidx<LAB>(t, u, v) * NQ], Rrow[v * NQ], s);
                            });
                        });
                        jhk[x] += s;
                    }
                }
            }
            // ---- exchange part: the ket component pairs (k,l) are dealt over the lanes of the quartet
            if (active && live_k) {
#pragma unroll 1
                for (int n = g; n < NKL; n += G) {
                    const int k = tab->kl_k[n], l = tab->kl_l[n];
                    const int q0 = tab->kl_start[n], q1 = tab->kl_start[n + 1];
                    double Yv[NHB];
#pragma unroll
                    for (int P = 0; P < NHB; ++P) Yv[P] = 0.0;
#pragma unroll 1
                    for (int q = q0; q < q1; ++q) {
                        const double e = kt[q];
                        const int p = tab->pk[q];
                        const int t2 = p & 15, u2 = (p >> 4) & 15, v2 = p >> 8;
                        const unsigned short* rq = rt + t2 * 13 + u2;
                        const double* Rq = Rs + v2 * NQ;
#pragma unroll
                        for (int t = 0; t <= LAB; ++t)
#pragma unroll
                            for (int u = 0; u <= LAB - t; ++u) {
                                const double* Rrow = Rq + (int)rq[t * 13 + u] * NQ;
#pragma unroll
                                for (int v = 0; v <= LAB - t - u; ++v)
                                    Yv[tidx<LAB>(t, u, v)] = fma(e, Rrow[v * NQ], Yv[tidx<LAB>(t, u, v)]);
                            }
                    }
                    // bra Hermite -> Cartesian and K digestion; the larger bra shell (b) is the outer loop so that only the
                    // 2 * NA accumulators of the smaller one stay live across it
                    double kac[NA], kad[NA];
#pragma unroll
                    for (int i = 0; i < NA; ++i) { kac[i] = 0.0; kad[i] = 0.0; }
                    static_for<NB>([&](auto J) {
                        constexpr int jj = decltype(J)::value;
                        constexpr int jx = cart_x(LB, jj), jy = cart_y(LB, jj), jz = cart_z(LB, jj);
                        double kbc = 0.0, kbd = 0.0;
                        const double dbl = Dbd[(jj * ND + l) * NQ], dbk = Dbc[(jj * NC + k) * NQ];
                        static_for<NA>([&](auto I) {
                            constexpr int i = decltype(I)::value;
                            constexpr int ix = cart_x(LA, i), iy = cart_y(LA, i), iz = cart_z(LA, i);
                            double s = 0.0;
#pragma unroll
                            for (int t = 0; t <= ix + jx; ++t) {
                                double su = 0.0;
#pragma unroll
                                for (int u = 0; u <= iy + jy; ++u) {
                                    double sv = 0.0;
#pragma unroll
                                    for (int v = 0; v <= iz + jz; ++v)
                                        sv = fma(Eb[(2 * NE1B + (iz * (LB + 1) + jz) * (LAB + 1) + v) * NQ], Yv[tidx<LAB>(t, u, v)], sv);
                                    su = fma(Eb[(NE1B + (iy * (LB + 1) + jy) * (LAB + 1) + u) * NQ], sv, su);
                                }
                                s = fma(Eb[((ix * (LB + 1) + jx) * (LAB + 1) + t) * NQ], su, s);
                            }
                            // s = f (ij|kl) without the per-component factors
                            kac[i] = fma(s, dbl, kac[i]);
                            kad[i] = fma(s, dbk, kad[i]);
                            kbc = fma(s, Dad[(i * ND + l) * NQ], kbc);
                            kbd = fma(s, Dac[(i * NC + k) * NQ], kbd);
                        });
                        if (live_kbc) atomicAdd(&a.Kt[(ib.offB + jj) * nbf + ik.offA + k], kbc);
                        if (live_kbd) atomicAdd(&a.Kt[(ib.offB + jj) * nbf + ik.offB + l], kbd);
                    });
#pragma unroll
                    for (int i = 0; i < NA; ++i) {
                        if (live_kac) atomicAdd(&a.Kt[(ib.offA + i) * nbf + ik.offA + k], kac[i]);
                        if (live_kad) atomicAdd(&a.Kt[(ib.offA + i) * nbf + ik.offB + l], kad[i]);
                    }
                }
            }
            __syncwarp();
        }
        // ---- ket Hermite J of this task: sum over the quartets of the warp, one atomic per Hermite index
        if (__any_sync(FULLMASK, any_jcd_task)) {
#pragma unroll
            for (int x = 0; x < NJK; ++x) {
                double v = jhk[x];
#pragma unroll
                for (int o = NQ / 2; o > 0; o >>= 1) v += __shfl_xor_sync(FULLMASK, v, o);
                const int Q = g + x * G;
                if (slot == 0 && Q < NHK && v != 0.0) {
                    const int p = tab->hk[Q];
                    const int par = ((p & 15) + ((p >> 4) & 15) + (p >> 8)) & 1;
                    atomicAdd(&a.JHk[j * NHK + Q], (par ? -2.0 : 2.0) * kp.pref * v);
                }
            }
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

// ------------------------------------------------------------------- Hermite density / Hermite J (eq. 35)
// DH[pair][P] = sum_ij E_P^{ij} Ds[a_i][b_j]   (no pair prefactor; Ds = component-scaled density), one thread per pair.
template <int LA, int LB>
__global__ void __launch_bounds__(128) hermite_density_kernel(const PairD* __restrict__ pairs, const PairIds* __restrict__ ids, long long n,
                                                              const double* __restrict__ Ds, int nbf, double* __restrict__ DH) {
    constexpr int LAB = LA + LB, NA = ncart(LA), NB = ncart(LB), NH = nherm(LAB);
    const long long x = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (x >= n) return;
    const PairD pd = pairs[x];
    const PairIds id = ids[x];
    double E[3][LA + 1][LB + 1][LAB + 1];
    for (int d = 0; d < 3; ++d) etable<LA, LB, false>(pd.PA[d], pd.PB[d], 0.5 / pd.p, E[d]);
    double acc[NH];
    for (int P = 0; P < NH; ++P) acc[P] = 0.0;
    for (int i = 0; i < NA; ++i) {
        const int ix = cart_x(LA, i), iy = cart_y(LA, i), iz = cart_z(LA, i);
        for (int j = 0; j < NB; ++j) {
            const int jx = cart_x(LB, j), jy = cart_y(LB, j), jz = cart_z(LB, j);
            const double d = Ds[(long long)(id.offA + i) * nbf + id.offB + j];
            for (int t = 0; t <= ix + jx; ++t)
                for (int u = 0; u <= iy + jy; ++u) {
                    const double exy = d * E[0][ix][jx][t] * E[1][iy][jy][u];
                    for (int v = 0; v <= iz + jz; ++v) acc[tidx<LAB>(t, u, v)] = fma(exy, E[2][iz][jz][v], acc[tidx<LAB>(t, u, v)]);
                }
        }
    }
    for (int P = 0; P < NH; ++P) DH[x * NH + P] = acc[P];
}

// Jt[a_i][b_j] += sum_P E_P^{ij} JH[pair][P], one thread per pair (JH already carries both pair prefactors and the factor 2).
template <int LA, int LB>
__global__ void __launch_bounds__(128) hermite_j_kernel(const PairD* __restrict__ pairs, const PairIds* __restrict__ ids, long long n,
                                                        const double* __restrict__ JH, int nbf, double* __restrict__ Jt) {
    constexpr int LAB = LA + LB, NA = ncart(LA), NB = ncart(LB), NH = nherm(LAB);
    const long long x = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (x >= n) return;
    double jh[NH];
    bool any = false;
    for (int P = 0; P < NH; ++P) { jh[P] = JH[x * NH + P]; any |= jh[P] != 0.0; }
    if (!any) return;
    const PairD pd = pairs[x];
    const PairIds id = ids[x];
    double E[3][LA + 1][LB + 1][LAB + 1];
    for (int d = 0; d < 3; ++d) etable<LA, LB, false>(pd.PA[d], pd.PB[d], 0.5 / pd.p, E[d]);
    for (int i = 0; i < NA; ++i) {
        const int ix = cart_x(LA, i), iy = cart_y(LA, i), iz = cart_z(LA, i);
        for (int j = 0; j < NB; ++j) {
            const int jx = cart_x(LB, j), jy = cart_y(LB, j), jz = cart_z(LB, j);
            double s = 0.0;
            for (int t = 0; t <= ix + jx; ++t)
                for (int u = 0; u <= iy + jy; ++u) {
                    const double exy = E[0][ix][jx][t] * E[1][iy][jy][u];
                    for (int v = 0; v <= iz + jz; ++v) s = fma(exy * E[2][iz][jz][v], jh[tidx<LAB>(t, u, v)], s);
                }
            atomicAdd(&Jt[(long long)(id.offA + i) * nbf + id.offB + j], s);
        }
    }
}

}  // namespace te
