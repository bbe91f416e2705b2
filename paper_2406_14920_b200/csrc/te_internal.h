// te_internal.h -- handle layouts and launch prototypes shared by the translation units of libte_jk.so.
#pragma once
#include <cuda_runtime.h>

#include <vector>

#include "../../include/te_jk.h"
#include "te_md.cuh"

namespace te {

void set_error(const char* fmt, ...);

#define TE_CUDA(expr)                                                                      \
    do {                                                                                   \
        cudaError_t e__ = (expr);                                                          \
        if (e__ != cudaSuccess) {                                                          \
            te::set_error("%s:%d: %s: %s", __FILE__, __LINE__, #expr, cudaGetErrorString(e__)); \
            return TE_ERR_CUDA;                                                            \
        }                                                                                  \
    } while (0)

struct PairIds {
    int m, n;        // global primitive-shell ids, (l_m, m) <= (l_n, n)
    int shA, shB;    // contracted shell ids
    int offA, offB;  // first AO of each contracted shell
};

struct JKControl {
    double dmax;                                        // max |D| (set by density_bounds_kernel)
    unsigned long long live[TE_NCLASS * TE_NCLASS];     // unique live quartets per class pair
    unsigned long long visited[TE_NCLASS * TE_NCLASS];  // unique quartets whose eq. 47 tests were evaluated (inside the schedule's cut)
    unsigned long long slots[TE_NCLASS * TE_NCLASS];    // quartet slots of the warp batches that ran the integral code (lane occupancy = live / slots)
    unsigned long long ntiles[TE_NCLASS * TE_NCLASS];   // scheduled tiles per class pair
    unsigned int tile_counter[TE_NCLASS * TE_NCLASS];   // dynamic tile queue heads
    int chunk[TE_NCLASS * TE_NCLASS];                   // uniform-ket kernel: bras per task = 32 * chunk
};

struct EriTask {
    int sh[4];       // canonical order: la<=lb, lc<=ld, class(ab)<=class(cd)
    int stride[4];   // output stride of each canonical index
    long long out;   // offset of the block in out_dev
};

}  // namespace te

struct te_basis {
    int natoms = 0, nshells = 0, nprim = 0, nbf = 0;
    std::vector<int> shell_l, shell_off, shell_pstart, shell_nprim;
    std::vector<double> prim_exp, prim_ct, prim_xyz;
    std::vector<int> prim_l, prim_shell, prim_iprim, prim_off, prims_by_l;
    int l_start[5] = {0, 0, 0, 0, 0};
    // device copies
    double *d_exp = nullptr, *d_ct = nullptr, *d_xyz = nullptr, *d_aofac = nullptr;
    int *d_shell = nullptr, *d_off = nullptr, *d_by_l = nullptr, *d_shell_off = nullptr, *d_shell_pstart = nullptr;
    const double* d_boys = nullptr;
    int device = 0;   // CUDA device the handle (and every te_pairs built from it) lives on
};

struct te_pairs {
    const te_basis* basis = nullptr;
    double tau_pair = 0.0;
    long long count[TE_NCLASS] = {0};
    te::PairD* d_pair[TE_NCLASS] = {nullptr};
    double* d_q[TE_NCLASS] = {nullptr};      // Schwarz bound of every pair
    double* d_qmax[TE_NCLASS] = {nullptr};   // largest bound of the pair's contracted shell-pair block (non-increasing along the list)
    te::PairIds* d_ids[TE_NCLASS] = {nullptr};
    // Hermite density / Hermite J of every pair (eq. 35), [count][nherm(la+lb)], rebuilt / zeroed by every build
    int* d_bstart[TE_NCLASS] = {nullptr};   // first pair of every contracted shell-pair block, [nblk + 1]
    int nblk[TE_NCLASS] = {0};
    double* d_DH[TE_NCLASS] = {nullptr};
    double* d_JH[TE_NCLASS] = {nullptr};
    // per-build scratch
    double *d_Ds = nullptr, *d_Jt = nullptr, *d_Kt = nullptr, *d_Dm = nullptr;
    te::JKControl* d_ctrl = nullptr;
    te::JKControl* d_ctrl32 = nullptr;   // task queues / counters of the FP32 leg of a mixed-precision build
    double prec_thr = 0.0;               // density-weighted bound below which a quartet is evaluated in FP32 (0: FP64 build)
    int impl = 2;                        // kernel-family policy (te_jk_set_kernel_family): 2 = measured per-class default
    double omega2 = 0.0;                 // operator of the build in flight: 0 = 1/r, omega^2 = erf(omega r)/r
    // schedule scratch of the class kernel in flight (class kernels of a build run back to back on the caller's stream)
    static constexpr int NSTREAM = 1;
    cudaEvent_t ev_done = nullptr;   // end of the last build / one-electron call on this handle: the next one waits for it
    bool ev_done_valid = false;
    long long* d_tile_start[NSTREAM] = {nullptr};
    int* d_task_hi[NSTREAM] = {nullptr};
    long long tile_cap = 0;
    double *d_hD = nullptr, *d_hJ = nullptr, *d_hK = nullptr;   // staging for te_build_jk_host
    bool profiling = false;
    cudaStream_t last_stream = nullptr;
    cudaEvent_t ev0[TE_NCLASS * TE_NCLASS] = {nullptr}, ev1[TE_NCLASS * TE_NCLASS] = {nullptr};
    bool ev_valid[TE_NCLASS * TE_NCLASS] = {false};
};

namespace te {
// te_inst_*.cu
int launch_schwarz(int la, int lb, const te_basis* b, long long ncand, double* d_q, long long* d_idx);
int launch_pair_fill(int la, int lb, const te_basis* b, long long n, const long long* d_idx, PairD* d_pair, PairIds* d_ids);
// lane: which schedule scratch; prec: 0 plain FP64, 1 / 2 = FP64 / FP32 leg of a mixed-precision build
int launch_jk_class(int cb, int ck, te_pairs* P, double tau, int lane, int prec, cudaStream_t st);
int launch_eri_class(int cb, int ck, const te_basis* b, int n, const EriTask* d_tasks, double* out_dev);
int launch_hermite_density(int cls, te_pairs* P, cudaStream_t st);   // d_Ds -> d_DH[cls]
int launch_hermite_j(int cls, te_pairs* P, cudaStream_t st);         // d_JH[cls] -> d_Jt
int launch_nuclear(int cls, te_pairs* P, int ncharge, const double4* d_chg, double* d_Vt, cudaStream_t st);
int launch_jeng_class(int cb, int ck, te_pairs* P, double tau, cudaStream_t st);   // Coulomb only, Hermite space (eq. 35)
constexpr int TE_MAX_DEV = 64;   // per-device caches (Boys table, class tables, occupancy) are indexed by the CUDA device id
}  // namespace te
