// te_jeng.cuh -- the "J engine" (eq. 35) as a build of its own: Coulomb matrix only, every class.
//
//     J_mu,nu = sum_P E_P^{mu nu}  sum_Q R_PQ  sum_{lambda sigma} E_Q^{lambda sigma} D_lambda,sigma
//
// The paper runs the two outer transforms on the CPU and only the middle sum on the GPU; here the Hermite density
// (hermite_density_kernel) and the back-transform (hermite_j_kernel) are device kernels too, and this kernel is the middle sum:
// for every unique primitive quartet, in Hermite space only,
//     JH_bra[P] += 2 f sum_Q (-1)^Q R_{P+Q} DH_ket[Q]          iff  q_bra q_ket Dm_CD >= tau     (J_AB <- D_CD)
//     JH_ket[Q] += 2 f (-1)^Q sum_P R_{P+Q} DH_bra[P]          iff  q_bra q_ket Dm_AB >= tau     (J_CD <- D_AB)
// No Hermite -> Cartesian transform of the integrals is ever formed: 4 nH_bra nH_ket flops per quartet instead of the
// (2 nH_bra nnzE_ket + 2 nnzE_bra ncart_cd + 4 ncart_ab ncart_cd) of the explicit route.  The work depends on the pair classes only
// through LAB = la + lb and LCD = lc + ld.  Layout as in the uniform-ket J/K kernel: one warp = one ket pair (its signed,
// prefactor-scaled Hermite density in shared memory) x 32 bra pairs, each lane's R tensor in a conflict-free shared-memory column.
#pragma once
#include "te_jkw.cuh"

namespace te {

template <int LAB, int LCD>
struct JShape {
    static constexpr int L = LAB + LCD, NHB = nherm(LAB), NHK = nherm(LCD), NR = nherm(L);
    static constexpr int smem_doubles = NR * WARP + NHB * WARP + 2 * NHK;
};

template <int LAB, int LCD>
__global__ void __launch_bounds__(WARP) jeng_kernel(JKArgs a) {
    using S = JShape<LAB, LCD>;
    constexpr int L = S::L, NHB = S::NHB, NHK = S::NHK;
    constexpr unsigned FULLMASK = 0xffffffffu;
    extern __shared__ double sm[];
    const int lane = threadIdx.x;
    double* const Rl = sm + lane;                         // element e of this lane's R tensor at Rl[e * 32]
    double* const dl = sm + S::NR * WARP + lane;          // this lane's bra Hermite density, element P at dl[P * 32]
    double* const sdk = sm + S::NR * WARP + NHB * WARP;   // [NHK] (-1)^Q x ket prefactor x Hermite density of the ket
    double* const jk = sdk + NHK;                         // [NHK] Hermite J of the ket, summed over the task by lane 0
    const unsigned short* const row = c_rowtab.v + L * 13 * 13;   // row[T * 13 + U] = index of R_{T,U,0}

    const unsigned long long ntasks = a.ctrl->ntiles[a.slot];
    const long long span = (long long)WARP * a.ctrl->chunk[a.slot];
    const long long ns = a.nshells;
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
        const PairD kp = a.pk[j];
        const PairIds ik = a.ik[j];
        const double qk = a.qk[j];
        const double dm_cd = a.Dm[ik.shA * ns + ik.shB];
        __syncwarp();
        {   // signed, prefactor-scaled Hermite density of the ket; zero its Hermite J accumulator
            int Q = 0;
            for (int t2 = 0; t2 <= LCD; ++t2)
                for (int u2 = 0; u2 <= LCD - t2; ++u2)
                    for (int v2 = 0; v2 <= LCD - t2 - u2; ++v2, ++Q)
                        if ((Q & 31) == lane) {
                            const double d = a.DHk[j * NHK + Q] * kp.pref;
                            sdk[Q] = ((t2 + u2 + v2) & 1) ? -d : d;
                            jk[Q] = 0.0;
                        }
        }
        __syncwarp();
        bool any_jcd_task = false;

        for (long long b0 = b_lo; b0 < b_hi; b0 += WARP) {
            const long long bi = b0 + lane;
            bool active = bi < b_hi, live_jab = false, live_jcd = false;
            PairIds ib;
            if (active) {
                ++nvis;
                ib = a.ib[bi];
                const double qq = a.qb[bi] * qk;
                live_jab = qq * dm_cd >= a.tau;
                live_jcd = qq * a.Dm[ib.shA * ns + ib.shB] >= a.tau;
                active = live_jab | live_jcd;
            }
            if (!__any_sync(FULLMASK, active)) continue;
            ++nslot;
            const bool any_jcd = __any_sync(FULLMASK, live_jcd);
            any_jcd_task |= any_jcd;
            if (active) {
                ++nlive;
                const PairD bp = a.pb[bi];
                double f = 1.0;
                if (ib.m == ib.n) f *= 0.5;
                if (ik.m == ik.n) f *= 0.5;
                if (a.same && bi == j) f *= 0.5;
                double alpha, pref;
                eri_scale(bp.p, bp.rp, kp.p, kp.rp, a.omega2, alpha, pref);
                const double X = bp.P[0] - kp.P[0], Y = bp.P[1] - kp.P[1], Z = bp.P[2] - kp.P[2];
                double F[L + 1];
                boys<L>(alpha * (X * X + Y * Y + Z * Z), a.boys_tab, F);
                pref *= bp.pref * f;   // eq. 30 prefactor x bra prefactor x symmetry factor, folded into the Boys values
#pragma unroll
                for (int m = 0; m <= L; ++m) F[m] *= pref;
                rtable_sm<L, WARP, double>(alpha, X, Y, Z, F, Rl);
                for (int P = 0; P < NHB; ++P) dl[P * WARP] = live_jcd ? a.DHb[bi * NHB + P] : 0.0;
                // ---- J_AB <- D_CD in Hermite space: one atomic per bra Hermite index
                if (live_jab) {
                    int P = 0;
                    for (int t = 0; t <= LAB; ++t)
                        for (int u = 0; u <= LAB - t; ++u)
                            for (int v = 0; v <= LAB - t - u; ++v, ++P) {
                                double s = 0.0;
                                int Q = 0;
                                for (int t2 = 0; t2 <= LCD; ++t2)
                                    for (int u2 = 0; u2 <= LCD - t2; ++u2) {
                                        const double* Rrow = Rl + ((int)row[(t + t2) * 13 + u + u2] + v) * WARP;
                                        for (int v2 = 0; v2 <= LCD - t2 - u2; ++v2, ++Q) s = fma(sdk[Q], Rrow[v2 * WARP], s);
                                    }
                                atomicAdd(&a.JHb[bi * NHB + P], 2.0 * s);
                            }
                }
            }
            // ---- J_CD <- D_AB in Hermite space: the warp's 32 quartets are summed per ket Hermite index
            if (any_jcd) {
                int Q = 0;
                for (int t2 = 0; t2 <= LCD; ++t2)
                    for (int u2 = 0; u2 <= LCD - t2; ++u2)
                        for (int v2 = 0; v2 <= LCD - t2 - u2; ++v2, ++Q) {
                            double s = 0.0;
                            if (active && live_jcd) {
                                int P = 0;
                                for (int t = 0; t <= LAB; ++t)
                                    for (int u = 0; u <= LAB - t; ++u) {
                                        const double* Rrow = Rl + ((int)row[(t + t2) * 13 + u + u2] + v2) * WARP;
                                        for (int v = 0; v <= LAB - t - u; ++v, ++P) s = fma(dl[P * WARP], Rrow[v * WARP], s);
                                    }
                            }
#pragma unroll
                            for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(FULLMASK, s, o);
                            if (lane == 0) jk[Q] += s;
                        }
            }
            __syncwarp();
        }
        __syncwarp();
        if (any_jcd_task) {
            int Q = 0;
            for (int t2 = 0; t2 <= LCD; ++t2)
                for (int u2 = 0; u2 <= LCD - t2; ++u2)
                    for (int v2 = 0; v2 <= LCD - t2 - u2; ++v2, ++Q)
                        if ((Q & 31) == lane && jk[Q] != 0.0)
                            atomicAdd(&a.JHk[j * NHK + Q], (((t2 + u2 + v2) & 1) ? -2.0 : 2.0) * kp.pref * jk[Q]);
        }
    }
    for (int o = 16; o > 0; o >>= 1) {
        nlive += __shfl_down_sync(FULLMASK, nlive, o); nvis += __shfl_down_sync(FULLMASK, nvis, o); nslot += __shfl_down_sync(FULLMASK, nslot, o);
    }
    if (lane == 0 && nvis) {
        atomicAdd(&a.ctrl->live[a.slot], (unsigned long long)nlive);
        atomicAdd(&a.ctrl->visited[a.slot], (unsigned long long)nvis);
        atomicAdd(&a.ctrl->slots[a.slot], (unsigned long long)nslot);
    }
}

}  // namespace te
