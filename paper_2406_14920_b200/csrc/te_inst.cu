// te_inst.cu -- instantiates every kernel whose BRA pair class is TE_CB (compiled 10 times, -DTE_CB=0..9, so the
// 55 (la lb|lc ld) classes build in parallel).  Exposes launch_*_cb<TE_CB> entry points used by te_dispatch.cu.
#include "te_jkq.cuh"
#include "te_jkb.cuh"
#include "te_jeng.cuh"

#include <cmath>
#include <mutex>

#ifndef TE_CB
#error "compile with -DTE_CB=<bra class 0..9>"
#endif

namespace te {

constexpr int CLS_LA[TE_NCLASS] = {0, 0, 0, 0, 1, 1, 1, 2, 2, 3};
constexpr int CLS_LB[TE_NCLASS] = {0, 1, 2, 3, 1, 2, 3, 2, 3, 3};
constexpr int LA = CLS_LA[TE_CB], LB = CLS_LB[TE_CB];

// largest task of a class kernel, in warp batches.  Measured on config 5 (caps 16 / 64 / 256 per family): 64 is the best for
// every family (a task pays two binary searches of dependent loads; above 64 the tail of a launch is less balanced).
static int chunk_cap() { return 64; }

static std::mutex g_cache_mutex;   // guards the per-device caches of this translation unit (class tables, occupancy)

static BasisView view(const te_basis* b) { return BasisView{b->d_exp, b->d_ct, b->d_xyz, b->d_shell, b->d_off}; }

#define TE_CAT2(a, b) a##b
#define TE_CAT(a, b) TE_CAT2(a, b)

int TE_CAT(launch_schwarz_cb, TE_CB)(const te_basis* b, long long ncand, double* d_q, long long* d_idx) {
    const long long nb = b->l_start[LB + 1] - b->l_start[LB];
    const unsigned grid = (unsigned)((ncand + 63) / 64);
    schwarz_kernel<LA, LB><<<grid, 64>>>(view(b), b->d_by_l + b->l_start[LA], b->d_by_l + b->l_start[LB], nb, ncand, b->d_boys, d_q, d_idx);
    TE_CUDA(cudaGetLastError());
    return TE_OK;
}

int TE_CAT(launch_pair_fill_cb, TE_CB)(const te_basis* b, long long n, const long long* d_idx, PairD* d_pair, PairIds* d_ids) {
    const long long nb = b->l_start[LB + 1] - b->l_start[LB];
    pair_fill_kernel<LA, LB><<<(unsigned)((n + 127) / 128), 128>>>(view(b), b->d_by_l + b->l_start[LA], b->d_by_l + b->l_start[LB], nb, n, d_idx, d_pair, d_ids);
    TE_CUDA(cudaGetLastError());
    return TE_OK;
}

// uniform-ket kernel in precision T: one warp per block, per-lane R tensor in shared memory
template <class T, int LC, int LD>
static int launch_w(te_pairs* P, JKArgs& a, double tau, int lane, int dev, int sms, cudaStream_t st) {
    using S = WShape<LA, LB, LC, LD, T>;
    constexpr int smem = S::smem_doubles * (int)sizeof(T);
    static int bps[TE_MAX_DEV] = {0};
    std::lock_guard<std::mutex> lock(g_cache_mutex);
    int& blocks_per_sm = bps[dev];
    if (!blocks_per_sm) {
        TE_CUDA(cudaFuncSetAttribute(jkw_kernel<T, LA, LB, LC, LD>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
        TE_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&blocks_per_sm, jkw_kernel<T, LA, LB, LC, LD>, WARP, smem));
        if (blocks_per_sm < 1) { set_error("jkw_kernel<%d,%d,%d,%d>: %d bytes of shared memory do not fit", LA, LB, LC, LD, smem); blocks_per_sm = 0; return TE_ERR_CUDA; }
    }
    const int warps = sms * blocks_per_sm;
    schedule_w_kernel<<<1, 1024, 0, st>>>(P->d_qmax[TE_CB], a.nb, a.qk, a.nk, a.same, tau, warps, S::NL, chunk_cap(), P->d_tile_start[lane], P->d_task_hi[lane], a.ctrl, a.slot);
    const long long max_tasks = a.nk * ((a.nb + S::NL - 1) / S::NL);
    const unsigned grid = (unsigned)std::min<long long>(max_tasks, (long long)warps);
    jkw_kernel<T, LA, LB, LC, LD><<<grid, WARP, smem, st>>>(a);
    TE_CUDA(cudaGetLastError());
    return TE_OK;
}

// prec: 0 = plain FP64 build; 1 / 2 = FP64 / FP32 leg of a mixed-precision build.  Only the classes jk_fp32_class
// names have an FP32 kernel; the driver runs the others with prec = 0.
template <int CK>
static int jk_launch(te_pairs* P, double tau, int lane, int prec, cudaStream_t st) {
    constexpr int LC = CLS_LA[CK], LD = CLS_LB[CK];
    constexpr bool light = use_full_unroll(LA, LB, LC, LD);
    constexpr int TB = light ? 16 : 8, TK = light ? 16 : 8;
    const te_basis* b = P->basis;
    const int slot = TE_CB * TE_NCLASS + CK;
    JKArgs a{};
    a.pb = P->d_pair[TE_CB]; a.qb = P->d_q[TE_CB]; a.ib = P->d_ids[TE_CB]; a.nb = P->count[TE_CB];
    a.pk = P->d_pair[CK]; a.qk = P->d_q[CK]; a.ik = P->d_ids[CK]; a.nk = P->count[CK];
    a.Ds = P->d_Ds; a.Dm = P->d_Dm; a.Jt = P->d_Jt; a.Kt = P->d_Kt; a.boys_tab = b->d_boys;
    a.tile_start = P->d_tile_start[lane]; a.ctrl = prec == 2 ? P->d_ctrl32 : P->d_ctrl; a.tau = tau; a.omega2 = P->omega2;
    a.nbf = b->nbf; a.nshells = b->nshells; a.slot = slot; a.same = (TE_CB == CK);
    a.task_hi = P->d_task_hi[lane];
    a.bstart = P->d_bstart[TE_CB]; a.nblk = P->nblk[TE_CB];
    a.prec_mode = prec; a.prec_thr = P->prec_thr;
    {   // FP32 keeps (2 alpha)^L below 1e30 (alpha <= p_ket): above that ket exponent the quartet stays in FP64
        constexpr int Lq = LA + LB + LC + LD;
        a.amax32 = Lq == 0 ? 1e300 : 0.5 * std::pow(1e30, 1.0 / Lq);
    }
    const int dev = b->device;   // checked against the current device by te_build_jk; the caches below are per device
    if (dev < 0 || dev >= TE_MAX_DEV) { set_error("launch_jk: device id %d out of range", dev); return TE_ERR_BAD_ARG; }
    int sms = 148;
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    // kernel family per class: 2 (default) = measured policy; te_jk_set_kernel_family forces 0: generic thread-per-quartet kernel,
    // 1: uniform-ket warp kernel wherever it exists, 3: split-quartet kernel wherever it exists (tests hold each to the same bar)
    const int impl = P->impl;
    if (prec == 2) {
        if constexpr (jk_fp32_class(LA, LB, LC, LD)) return launch_w<float, LC, LD>(P, a, tau, lane, dev, sms, st);
        set_error("launch_jk: class (%d%d|%d%d) has no FP32 kernel", LA, LB, LC, LD);
        return TE_ERR_BAD_ARG;
    }
    if constexpr (use_jkb(LA, LB, LC, LD)) {
        if (impl == 2) {
            // block-per-lane kernel for the s/p-only classes: one warp per block, ket tables in shared memory
            using S = BShape<LA, LB, LC, LD>;
            constexpr int smem = S::smem_doubles * (int)sizeof(double);
            static int bps[TE_MAX_DEV] = {0};
            std::lock_guard<std::mutex> lock(g_cache_mutex);
            int& blocks_per_sm = bps[dev];
            if (!blocks_per_sm) {
                TE_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&blocks_per_sm, jkb_kernel<LA, LB, LC, LD>, WARP, smem));
                if (blocks_per_sm < 1) { blocks_per_sm = 0; set_error("jkb_kernel<%d,%d,%d,%d> does not fit", LA, LB, LC, LD); return TE_ERR_CUDA; }
            }
            const int warps = sms * blocks_per_sm;
            schedule_w_kernel<<<1, 1024, 0, st>>>(P->d_qmax[TE_CB], a.nb, a.qk, a.nk, a.same, tau, warps, WARP, chunk_cap(), P->d_tile_start[lane], P->d_task_hi[lane], a.ctrl, slot);
            const long long max_tasks = a.nk * ((a.nb + WARP - 1) / WARP);
            const unsigned grid = (unsigned)std::min<long long>(max_tasks, (long long)warps);
            jkb_kernel<LA, LB, LC, LD><<<grid, WARP, smem, st>>>(a);
            TE_CUDA(cudaGetLastError());
            return TE_OK;
        }
    }
    if constexpr (use_jkq(LA, LB, LC, LD)) {
        if (impl == 3 || impl == 2) {
            constexpr int QW = 4, QG = jkq_lanes(LA, LB, LC, LD, QW);
            using S = QShape<LA, LB, LC, LD, QG, QW>;
            using Tab = QTab<LA, LB, LC, LD>;
            static Tab* tabs[TE_MAX_DEV] = {nullptr};
            static int bps[TE_MAX_DEV] = {0};
            std::lock_guard<std::mutex> lock(g_cache_mutex);
            Tab*& d_tab = tabs[dev];
            int& blocks_per_sm = bps[dev];
            if (!d_tab) {
                static const Tab h_tab;
                Tab* d = nullptr;
                TE_CUDA(cudaMalloc(&d, sizeof(Tab)));
                TE_CUDA(cudaMemcpy(d, &h_tab, sizeof(Tab), cudaMemcpyHostToDevice));
                TE_CUDA(cudaFuncSetAttribute(jkq_kernel<LA, LB, LC, LD, QG, QW>, cudaFuncAttributeMaxDynamicSharedMemorySize, S::smem_bytes));
                TE_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&blocks_per_sm, jkq_kernel<LA, LB, LC, LD, QG, QW>, 32 * QW, S::smem_bytes));
                if (blocks_per_sm < 1) { cudaFree(d); set_error("jkq_kernel<%d,%d,%d,%d>: %d bytes of shared memory do not fit", LA, LB, LC, LD, S::smem_bytes); return TE_ERR_CUDA; }
                d_tab = d;
            }
            a.DHb = P->d_DH[TE_CB]; a.DHk = P->d_DH[CK]; a.JHb = P->d_JH[TE_CB]; a.JHk = P->d_JH[CK];
            const int blocks = sms * blocks_per_sm;
            schedule_w_kernel<<<1, 1024, 0, st>>>(P->d_qmax[TE_CB], a.nb, a.qk, a.nk, a.same, tau, blocks, S::NQ * QW, chunk_cap(), P->d_tile_start[lane], P->d_task_hi[lane], a.ctrl, slot);
            const long long max_tasks = a.nk * ((a.nb + S::NQ * QW - 1) / (S::NQ * QW));
            const unsigned grid = (unsigned)std::min<long long>(max_tasks, (long long)blocks);
            jkq_kernel<LA, LB, LC, LD, QG, QW><<<grid, 32 * QW, S::smem_bytes, st>>>(a, d_tab);
            TE_CUDA(cudaGetLastError());
            return TE_OK;
        }
    }
    if ((light && impl < 2) || impl == 0) {
        schedule_kernel<<<1, 1024, 0, st>>>(P->d_qmax[TE_CB], a.nb, P->d_qmax[CK], a.nk, a.same, tau, TB, TK, P->d_tile_start[lane], a.ctrl, slot);
        const long long max_tiles = ((a.nb + TB - 1) / TB) * ((a.nk + TK - 1) / TK);
        const int per_sm = light ? 8 : 16;   // resident CTAs per SM worth of persistent blocks
        const unsigned grid = (unsigned)std::min<long long>(max_tiles, (long long)sms * per_sm);
        jk_kernel<LA, LB, LC, LD, TB, TK><<<grid, TB * TK, 0, st>>>(a);
    } else {
        return launch_w<double, LC, LD>(P, a, tau, lane, dev, sms, st);
    }
    TE_CUDA(cudaGetLastError());
    return TE_OK;
}

int TE_CAT(launch_nuclear_cb, TE_CB)(te_pairs* P, int ncharge, const double4* d_chg, double* d_Vt, cudaStream_t st) {
    const long long n = P->count[TE_CB];
    if (n == 0) return TE_OK;
    nuclear_kernel<LA, LB><<<(unsigned)((n + 63) / 64), 64, 0, st>>>(P->d_pair[TE_CB], P->d_ids[TE_CB], n, ncharge, d_chg, P->basis->d_boys,
                                                                   P->basis->nbf, d_Vt);
    TE_CUDA(cudaGetLastError());
    return TE_OK;
}

// J engine (Coulomb only, Hermite space): one instantiation per (la + lb, lc + ld)
template <int CK>
static int jeng_launch(te_pairs* P, double tau, cudaStream_t st) {
    constexpr int LC = CLS_LA[CK], LD = CLS_LB[CK], LAB = LA + LB, LCD = LC + LD;
    using S = JShape<LAB, LCD>;
    constexpr int smem = S::smem_doubles * (int)sizeof(double);
    const te_basis* b = P->basis;
    const int dev = b->device;
    if (dev < 0 || dev >= TE_MAX_DEV) { set_error("launch_jeng: device id %d out of range", dev); return TE_ERR_BAD_ARG; }
    int sms = 148;
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    JKArgs a{};
    a.pb = P->d_pair[TE_CB]; a.qb = P->d_q[TE_CB]; a.ib = P->d_ids[TE_CB]; a.nb = P->count[TE_CB];
    a.pk = P->d_pair[CK]; a.qk = P->d_q[CK]; a.ik = P->d_ids[CK]; a.nk = P->count[CK];
    a.Ds = P->d_Ds; a.Dm = P->d_Dm; a.Jt = P->d_Jt; a.Kt = P->d_Kt; a.boys_tab = b->d_boys;
    a.DHb = P->d_DH[TE_CB]; a.DHk = P->d_DH[CK]; a.JHb = P->d_JH[TE_CB]; a.JHk = P->d_JH[CK];
    a.tile_start = P->d_tile_start[0]; a.task_hi = P->d_task_hi[0]; a.ctrl = P->d_ctrl; a.tau = tau; a.omega2 = P->omega2;
    a.nbf = b->nbf; a.nshells = b->nshells; a.slot = TE_CB * TE_NCLASS + CK; a.same = (TE_CB == CK);
    static int bps[TE_MAX_DEV] = {0};
    std::lock_guard<std::mutex> lock(g_cache_mutex);
    int& blocks_per_sm = bps[dev];
    if (!blocks_per_sm) {
        TE_CUDA(cudaFuncSetAttribute(jeng_kernel<LAB, LCD>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
        TE_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&blocks_per_sm, jeng_kernel<LAB, LCD>, WARP, smem));
        if (blocks_per_sm < 1) { set_error("jeng_kernel<%d,%d>: %d bytes of shared memory do not fit", LAB, LCD, smem); blocks_per_sm = 0; return TE_ERR_CUDA; }
    }
    const int warps = sms * blocks_per_sm;
    schedule_w_kernel<<<1, 1024, 0, st>>>(P->d_qmax[TE_CB], a.nb, a.qk, a.nk, a.same, tau, warps, WARP, chunk_cap(), P->d_tile_start[0], P->d_task_hi[0], a.ctrl, a.slot);
    const long long max_tasks = a.nk * ((a.nb + WARP - 1) / WARP);
    const unsigned grid = (unsigned)std::min<long long>(max_tasks, (long long)warps);
    jeng_kernel<LAB, LCD><<<grid, WARP, smem, st>>>(a);
    TE_CUDA(cudaGetLastError());
    return TE_OK;
}

template <int CK>
static int jeng_dispatch(int ck, te_pairs* P, double tau, cudaStream_t st) {
    if (ck == CK) return jeng_launch<CK>(P, tau, st);
    if constexpr (CK + 1 < TE_NCLASS) return jeng_dispatch<CK + 1>(ck, P, tau, st);
    set_error("launch_jeng: bad ket class %d", ck);
    return TE_ERR_BAD_ARG;
}

int TE_CAT(launch_jeng_cb, TE_CB)(int ck, te_pairs* P, double tau, cudaStream_t st) { return jeng_dispatch<TE_CB>(ck, P, tau, st); }

int TE_CAT(launch_hermite_density_cb, TE_CB)(te_pairs* P, cudaStream_t st) {
    const long long n = P->count[TE_CB];
    if (n == 0) return TE_OK;
    hermite_density_kernel<LA, LB><<<(unsigned)((n + 127) / 128), 128, 0, st>>>(P->d_pair[TE_CB], P->d_ids[TE_CB], n, P->d_Ds, P->basis->nbf, P->d_DH[TE_CB]);
    TE_CUDA(cudaGetLastError());
    return TE_OK;
}

int TE_CAT(launch_hermite_j_cb, TE_CB)(te_pairs* P, cudaStream_t st) {
    const long long n = P->count[TE_CB];
    if (n == 0) return TE_OK;
    hermite_j_kernel<LA, LB><<<(unsigned)((n + 127) / 128), 128, 0, st>>>(P->d_pair[TE_CB], P->d_ids[TE_CB], n, P->d_JH[TE_CB], P->basis->nbf, P->d_Jt);
    TE_CUDA(cudaGetLastError());
    return TE_OK;
}

template <int CK>
static int eri_launch(const te_basis* b, int n, const EriTask* d_tasks, double* out_dev) {
    constexpr int LC = CLS_LA[CK], LD = CLS_LB[CK];
    eri_block_kernel<LA, LB, LC, LD><<<(n + 31) / 32, 32>>>(view(b), b->d_shell_pstart, n, d_tasks, b->d_boys, out_dev);
    TE_CUDA(cudaGetLastError());
    return TE_OK;
}

template <int CK>
static int jk_dispatch(int ck, te_pairs* P, double tau, int lane, int prec, cudaStream_t st) {
    if (ck == CK) return jk_launch<CK>(P, tau, lane, prec, st);
    if constexpr (CK + 1 < TE_NCLASS) return jk_dispatch<CK + 1>(ck, P, tau, lane, prec, st);
    set_error("launch_jk: bad ket class %d", ck);
    return TE_ERR_BAD_ARG;
}

template <int CK>
static int eri_dispatch(int ck, const te_basis* b, int n, const EriTask* d_tasks, double* out_dev) {
    if (ck == CK) return eri_launch<CK>(b, n, d_tasks, out_dev);
    if constexpr (CK + 1 < TE_NCLASS) return eri_dispatch<CK + 1>(ck, b, n, d_tasks, out_dev);
    set_error("launch_eri: bad ket class %d", ck);
    return TE_ERR_BAD_ARG;
}

int TE_CAT(launch_jk_cb, TE_CB)(int ck, te_pairs* P, double tau, int lane, int prec, cudaStream_t st) { return jk_dispatch<TE_CB>(ck, P, tau, lane, prec, st); }
int TE_CAT(launch_eri_cb, TE_CB)(int ck, const te_basis* b, int n, const EriTask* d_tasks, double* out_dev) {
    return eri_dispatch<TE_CB>(ck, b, n, d_tasks, out_dev);
}

}  // namespace te
