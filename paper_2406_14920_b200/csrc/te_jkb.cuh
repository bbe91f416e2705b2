// te_jkb.cuh -- "block-per-lane" J/K kernel for the s/p-only classes (few outputs per quartet, deep contractions).
//
// The ket pair is uniform across the warp (its signed, prefactor-folded E~_Q^{kl} sit in shared memory, as in te_jkw.cuh), but a
// lane does not own one primitive bra pair: it owns a whole contracted shell-pair BLOCK of the (shell-pair-major) bra list and
// walks its primitive pairs one per iteration.  Everything that depends only on the shells -- the five density blocks, the six
// density bounds of eq. 47, the output addresses -- is fetched once per block, all J/K contributions of the block are summed in
// registers and flushed once, and J_cd is summed per lane over the whole task.  Blocks are handed to lanes dynamically (a lane
// that finishes its block takes the next one of the task), so blocks of 1 and of 36 primitive pairs mix without idle lanes.
// Inside a block the pairs are in descending bound order, so each of the six per-term tests can only switch from live to dead:
// when it does, the density block that feeds that update is zeroed in place for the rest of the block (no per-integral masks).
#pragma once
#include "te_jkw.cuh"

namespace te {

constexpr int jkb_outputs(int la, int lb, int lc, int ld) {
    return ncart(la) * ncart(lb) + (ncart(la) + ncart(lb)) * (ncart(lc) + ncart(ld));
}
// classes handled by the block-per-lane kernel: R (L <= 4: 35 values), the density blocks and all outputs of a quartet must fit
// in registers (up to 48 outputs a few of them spill, still faster than the shared-memory R column of the uniform-ket kernel;
// measured: (ss|ss) and (sd|sd) are faster with one primitive quartet per lane)
constexpr bool use_jkb(int la, int lb, int lc, int ld) {
    // round 2: (SP|SF) and (SD|PP) (spilling here: 5e9 local-memory instructions per config-5 launch) are 10-17 % faster in the
    // uniform-ket kernel since its k-batched ket transform and ket-row accesses
    if ((la == 0 && lb == 1 && lc == 0 && ld == 3) || (la == 0 && lb == 2 && lc == 1 && ld == 1)) return false;
    return la + lb + lc + ld >= 1 && la + lb + lc + ld <= 4 && jkb_outputs(la, lb, lc, ld) <= 48;
}

template <int LA, int LB, int LC, int LD>
struct BShape {
    static constexpr int LCD = LC + LD;
    static constexpr int NC = ncart(LC), ND = ncart(LD);
    static constexpr int NNZK = nnz_e(LC, LD);
    static constexpr int NE1 = (LC + 1) * (LD + 1) * (LCD + 1);
    static constexpr int smem_doubles = NNZK + 3 * NE1 + NC * ND;
};

template <int LA, int LB, int LC, int LD>
__global__ void __launch_bounds__(WARP) jkb_kernel(JKArgs a) {
    using S = BShape<LA, LB, LC, LD>;
    constexpr int LAB = LA + LB, LCD = LC + LD, L = LAB + LCD;
    constexpr int NA = ncart(LA), NB = ncart(LB), NC = ncart(LC), ND = ncart(LD), NHB = nherm(LAB);
    constexpr unsigned FULLMASK = 0xffffffffu;
    extern __shared__ double sm[];
    double* const kt = sm;
    double* const e1 = kt + S::NNZK;
    double* const dcd = e1 + 3 * S::NE1;
    const int lane = threadIdx.x;

    const unsigned long long ntasks = a.ctrl->ntiles[a.slot];
    const long long span = (long long)WARP * a.ctrl->chunk[a.slot];
    const long long ns = a.nshells, nbf = a.nbf;
    long long cached_j = -1;
    PairD kp;
    PairIds ik;
    double qk = 0.0, dm_jab = 0.0;
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
            __syncwarp();
            kp = a.pk[j]; ik = a.ik[j]; qk = a.qk[j];
            dm_jab = a.Dm[ik.shA * ns + ik.shB];
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
                        for (int t = 0; t <= LCD; ++t) e1[lane * S::NE1 + (i * (LD + 1) + jj) * (LCD + 1) + t] = E[i][jj][t];
            }
            __syncwarp();
            int e = 0;
            for (int l = 0; l < ND; ++l) {
                const int lx = cart_x(LD, l), ly = cart_y(LD, l), lz = cart_z(LD, l);
                for (int k = 0; k < NC; ++k) {
                    const int kx = cart_x(LC, k), ky = cart_y(LC, k), kz = cart_z(LC, k);
                    const double* ex = e1 + (kx * (LD + 1) + lx) * (LCD + 1);
                    const double* ey = e1 + S::NE1 + (ky * (LD + 1) + ly) * (LCD + 1);
                    const double* ez = e1 + 2 * S::NE1 + (kz * (LD + 1) + lz) * (LCD + 1);
                    for (int t2 = 0; t2 <= kx + lx; ++t2)
                        for (int u2 = 0; u2 <= ky + ly; ++u2)
                            for (int v2 = 0; v2 <= kz + lz; ++v2, ++e)
                                if ((e & 31) == lane) kt[e] = ex[t2] * ey[u2] * ez[v2] * kp.pref;
                }
            }
            for (int cd = lane; cd < NC * ND; cd += WARP) dcd[cd] = a.Ds[(ik.offA + cd / ND) * nbf + ik.offB + cd % ND];
            __syncwarp();
            cached_j = j;
        }

        // first block that overlaps [b_lo, b_hi): last block with bstart <= b_lo
        int nb;
        {
            int blo = 0, bhi = a.nblk;
            while (bhi - blo > 1) { const int mid = (blo + bhi) >> 1; if (a.bstart[mid] <= b_lo) blo = mid; else bhi = mid; }
            nb = blo;
        }
        long long cur = 0, end = 0;
        bool assigned = false;
        unsigned fl = 0;   // update types (J_ab, K_ac, K_bc, K_ad, K_bd) that were live for at least one primitive pair of the block
        int offA = 0, offB = 0;
        double dm_jcd = 0.0, dm_kac = 0.0, dm_kbc = 0.0, dm_kad = 0.0, dm_kbd = 0.0, mjab = 0.0;
        double dab[NA * NB], dbl[NB * ND], dal[NA * ND], dbk[NB * NC], dak[NA * NC];
        double jab[NA * NB], kac[NA * NC], kbc[NB * NC], kad[NA * ND], kbd[NB * ND];
        double jcd[NC * ND];
#pragma unroll
        for (int x = 0; x < NC * ND; ++x) jcd[x] = 0.0;

        while (true) {
            const bool need = cur >= end;
            if (need && assigned) {
                // ---- the block is finished: one flush of everything it produced.  One branch per update type (was it ever live in
                // this block?) instead of a compare-and-branch per element: the flush runs with partial masks on almost every
                // iteration of the warp, so its instruction count matters as much as the integral code's.
                if (fl & 1) {
#pragma unroll
                    for (int x = 0; x < NA * NB; ++x) atomicAdd(&a.Jt[(offA + x / NB) * nbf + offB + x % NB], 2.0 * jab[x]);
                }
                if (fl & 2) {
#pragma unroll
                    for (int x = 0; x < NA * NC; ++x) atomicAdd(&a.Kt[(ik.offA + x % NC) * nbf + offA + x / NC], kac[x]);
                }
                if (fl & 4) {
#pragma unroll
                    for (int x = 0; x < NB * NC; ++x) atomicAdd(&a.Kt[(ik.offA + x % NC) * nbf + offB + x / NC], kbc[x]);
                }
                if (fl & 8) {
#pragma unroll
                    for (int x = 0; x < NA * ND; ++x) atomicAdd(&a.Kt[(ik.offB + x % ND) * nbf + offA + x / ND], kad[x]);
                }
                if (fl & 16) {
#pragma unroll
                    for (int x = 0; x < NB * ND; ++x) atomicAdd(&a.Kt[(ik.offB + x % ND) * nbf + offB + x / ND], kbd[x]);
                }
                assigned = false;
            }
            // ---- hand the next blocks of the task to the lanes that need one
            const unsigned needm = __ballot_sync(FULLMASK, need);
            if (need) {
                const int blk = nb + __popc(needm & ((1u << lane) - 1u));
                long long s = 0, e = 0;
                if (blk < a.nblk) { s = max((long long)a.bstart[blk], b_lo); e = min((long long)a.bstart[blk + 1], b_hi); }
                if (s < e) {
                    cur = s; end = e; assigned = true; fl = 0;
                    const PairIds ib = a.ib[s];
                    offA = ib.offA; offB = ib.offB;
                    dm_jcd = a.Dm[ib.shA * ns + ib.shB];
                    dm_kac = a.Dm[ib.shB * ns + ik.shB];
                    dm_kbc = a.Dm[ib.shA * ns + ik.shB];
                    dm_kad = a.Dm[ib.shB * ns + ik.shA];
                    dm_kbd = a.Dm[ib.shA * ns + ik.shA];
                    mjab = 1.0;
                    // D is symmetric (te_jk.h), and K = Kt + Kt^T is formed at the end: every bra-ket density element is read, and every K
                    // contribution added, at [ket AO row][bra AO column].  The ket is uniform across the warp, so the lanes of a warp
                    // (and all warps on the same ket) touch a handful of rows instead of rows scattered over the whole matrix.
                    const double* Da = a.Ds + (long long)offA * nbf;
                    const double* Dc = a.Ds + (long long)ik.offA * nbf;
                    const double* Dd = a.Ds + (long long)ik.offB * nbf;
#pragma unroll
                    for (int i = 0; i < NA; ++i) {
#pragma unroll
                        for (int jj = 0; jj < NB; ++jj) { dab[i * NB + jj] = Da[i * nbf + offB + jj]; jab[i * NB + jj] = 0.0; }
#pragma unroll
                        for (int l = 0; l < ND; ++l) { dal[i * ND + l] = Dd[l * nbf + offA + i]; kad[i * ND + l] = 0.0; }
#pragma unroll
                        for (int k = 0; k < NC; ++k) { dak[i * NC + k] = Dc[k * nbf + offA + i]; kac[i * NC + k] = 0.0; }
                    }
#pragma unroll
                    for (int jj = 0; jj < NB; ++jj) {
#pragma unroll
                        for (int l = 0; l < ND; ++l) { dbl[jj * ND + l] = Dd[l * nbf + offB + jj]; kbd[jj * ND + l] = 0.0; }
#pragma unroll
                        for (int k = 0; k < NC; ++k) { dbk[jj * NC + k] = Dc[k * nbf + offB + jj]; kbc[jj * NC + k] = 0.0; }
                    }
                } else {
                    cur = 0; end = 0;
                }
            }
            nb += __popc(needm);
            const bool work = cur < end;
            if (!__any_sync(FULLMASK, work)) break;
            ++nslot;
            if (work) {
                ++nvis;
                const long long bi = cur++;
                if (cur < end) {   // the next primitive pair of this lane's block: pull its data into L1 while this one computes
                    asm volatile("prefetch.global.L1 [%0];" ::"l"(a.pb + cur));
                    asm volatile("prefetch.global.L1 [%0];" ::"l"(reinterpret_cast<const char*>(a.pb + cur) + 88));
                    asm volatile("prefetch.global.L1 [%0];" ::"l"(a.qb + cur));
                }
                const double qq = a.qb[bi] * qk;
                // the per-term tests of eq. 47; bounds fall along the block, so a dead term stays dead: zero its density block
                const bool live_jab = qq * dm_jab >= a.tau, live_jcd = qq * dm_jcd >= a.tau, live_kac = qq * dm_kac >= a.tau;
                const bool live_kbc = qq * dm_kbc >= a.tau, live_kad = qq * dm_kad >= a.tau, live_kbd = qq * dm_kbd >= a.tau;
                if (!live_jab) mjab = 0.0;
                if (!live_jcd) {
#pragma unroll
                    for (int x = 0; x < NA * NB; ++x) dab[x] = 0.0;
                }
                if (!live_kac) {   // K_ac <- D_bd
#pragma unroll
                    for (int x = 0; x < NB * ND; ++x) dbl[x] = 0.0;
                }
                if (!live_kbc) {   // K_bc <- D_ad
#pragma unroll
                    for (int x = 0; x < NA * ND; ++x) dal[x] = 0.0;
                }
                if (!live_kad) {   // K_ad <- D_bc
#pragma unroll
                    for (int x = 0; x < NB * NC; ++x) dbk[x] = 0.0;
                }
                if (!live_kbd) {   // K_bd <- D_ac
#pragma unroll
                    for (int x = 0; x < NA * NC; ++x) dak[x] = 0.0;
                }
                // FP64 leg of a mixed-precision build: once the density-weighted bound falls below the switch, the rest of the block
                // (bounds fall along it, the ket is fixed) belongs to the FP32 launch
                const bool to32 = a.prec_mode == 1 &&
                                  fp32_quartet(a, qq, fmax(fmax(fmax(dm_jab, dm_jcd), fmax(dm_kac, dm_kbc)), fmax(dm_kad, dm_kbd)), kp.p);
                if (!(live_jab | live_jcd | live_kac | live_kbc | live_kad | live_kbd) || to32) {
                    cur = end;   // bounds fall along the block: the rest of it is dead too
                } else {
                    ++nlive;
                    fl |= (live_jab ? 1u : 0u) | (live_kac ? 2u : 0u) | (live_kbc ? 4u : 0u) | (live_kad ? 8u : 0u) | (live_kbd ? 16u : 0u);
                    const PairD bp = a.pb[bi];
                    const PairIds ibp = a.ib[bi];
                    double f = 1.0;
                    if (ibp.m == ibp.n) f *= 0.5;
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
                    double R[nherm(L)];
                    rtable<L>(alpha, X, Y, Z, F, R);
                    double Ebx[LA + 1][LB + 1][LAB + 1], Eby[LA + 1][LB + 1][LAB + 1], Ebz[LA + 1][LB + 1][LAB + 1];
                    const double hb = 0.5 * bp.rp;
                    etable<LA, LB, false>(bp.PA[0], bp.PB[0], hb, Ebx);
                    etable<LA, LB, false>(bp.PA[1], bp.PB[1], hb, Eby);
                    etable<LA, LB, false>(bp.PA[2], bp.PB[2], hb, Ebz);
                    int ptr = 0;
                    static_for<ND>([&](auto Lc) {
                        constexpr int l = decltype(Lc)::value;
                        constexpr int lx = cart_x(LD, l), ly = cart_y(LD, l), lz = cart_z(LD, l);
                        static_for<NC>([&](auto Kc) {
                            constexpr int k = decltype(Kc)::value;
                            constexpr int sx = cart_x(LC, k) + lx, sy = cart_y(LC, k) + ly, sz = cart_z(LC, k) + lz;
                            // ---- ket Hermite -> Cartesian for this (k,l): Y_P = sum_Q E~_Q R_{P+Q}
                            double Yv[NHB];
#pragma unroll
                            for (int P = 0; P < NHB; ++P) Yv[P] = 0.0;
#pragma unroll
                            for (int t2 = 0; t2 <= sx; ++t2)
#pragma unroll
                                for (int u2 = 0; u2 <= sy; ++u2)
#pragma unroll
                                    for (int v2 = 0; v2 <= sz; ++v2) {
                                        const double e = kt[ptr++];
#pragma unroll
                                        for (int t = 0; t <= LAB; ++t)
#pragma unroll
                                            for (int u = 0; u <= LAB - t; ++u)
#pragma unroll
                                                for (int v = 0; v <= LAB - t - u; ++v)
                                                    Yv[tidx<LAB>(t, u, v)] = fma(e, R[tidx<L>(t + t2, u + u2, v + v2)], Yv[tidx<LAB>(t, u, v)]);
                                    }
                            const double dklm = dcd[k * ND + l] * mjab;
                            // ---- bra Hermite -> Cartesian and digestion (eq. 34, 36)
#pragma unroll
                            for (int i = 0; i < NA; ++i) {
                                const int ix = cart_x(LA, i), iy = cart_y(LA, i), iz = cart_z(LA, i);
#pragma unroll
                                for (int jj = 0; jj < NB; ++jj) {
                                    const int jx = cart_x(LB, jj), jy = cart_y(LB, jj), jz = cart_z(LB, jj);
                                    double s = 0.0;
#pragma unroll
                                    for (int t = 0; t <= ix + jx; ++t) {
                                        double su = 0.0;
#pragma unroll
                                        for (int u = 0; u <= iy + jy; ++u) {
                                            double sv = 0.0;
#pragma unroll
                                            for (int v = 0; v <= iz + jz; ++v) sv = fma(Ebz[iz][jz][v], Yv[tidx<LAB>(t, u, v)], sv);
                                            su = fma(Eby[iy][jy][u], sv, su);
                                        }
                                        s = fma(Ebx[ix][jx][t], su, s);
                                    }
                                    // s = f (ij|kl) without the per-component factors
                                    jab[i * NB + jj] = fma(s, dklm, jab[i * NB + jj]);
                                    jcd[k * ND + l] = fma(s, dab[i * NB + jj], jcd[k * ND + l]);
                                    kac[i * NC + k] = fma(s, dbl[jj * ND + l], kac[i * NC + k]);
                                    kbc[jj * NC + k] = fma(s, dal[i * ND + l], kbc[jj * NC + k]);
                                    kad[i * ND + l] = fma(s, dbk[jj * NC + k], kad[i * ND + l]);
                                    kbd[jj * ND + l] = fma(s, dak[i * NC + k], kbd[jj * ND + l]);
                                }
                            }
                        });
                    });
                }
            }
        }
        // ---- J_cd of this task: one warp reduction per ket component pair
#pragma unroll
        for (int cd = 0; cd < NC * ND; ++cd) {
            double v = jcd[cd];
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(FULLMASK, v, o);
            if (lane == 0 && v != 0.0) atomicAdd(&a.Jt[(ik.offA + cd / ND) * nbf + ik.offB + cd % ND], 2.0 * v);
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

}  // namespace te
