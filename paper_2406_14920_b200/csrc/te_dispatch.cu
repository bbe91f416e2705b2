// te_dispatch.cu -- routes (bra class, ket class) to the per-bra-class translation units (te_inst.cu, -DTE_CB=n).
#include "te_internal.h"

namespace te {

#define TE_FOR_CLASSES(X) X(0) X(1) X(2) X(3) X(4) X(5) X(6) X(7) X(8) X(9)
#define TE_DECL(n)                                                                                         \
    int launch_schwarz_cb##n(const te_basis*, long long, double*, long long*);                             \
    int launch_pair_fill_cb##n(const te_basis*, long long, const long long*, PairD*, PairIds*);            \
    int launch_jk_cb##n(int, te_pairs*, double, int, int, cudaStream_t);                                        \
    int launch_eri_cb##n(int, const te_basis*, int, const EriTask*, double*);                              \
    int launch_hermite_density_cb##n(te_pairs*, cudaStream_t);                                             \
    int launch_hermite_j_cb##n(te_pairs*, cudaStream_t);                                                   \
    int launch_nuclear_cb##n(te_pairs*, int, const double4*, double*, cudaStream_t);                          \
    int launch_jeng_cb##n(int, te_pairs*, double, cudaStream_t);
TE_FOR_CLASSES(TE_DECL)

int launch_schwarz(int la, int lb, const te_basis* b, long long ncand, double* d_q, long long* d_idx) {
    switch (pair_class(la, lb)) {
#define TE_CASE(n) case n: return launch_schwarz_cb##n(b, ncand, d_q, d_idx);
        TE_FOR_CLASSES(TE_CASE)
#undef TE_CASE
    }
    return TE_ERR_BAD_ARG;
}

int launch_pair_fill(int la, int lb, const te_basis* b, long long n, const long long* d_idx, PairD* d_pair, PairIds* d_ids) {
    const long long n_ = n;
    switch (pair_class(la, lb)) {
#define TE_CASE(k) case k: return launch_pair_fill_cb##k(b, n_, d_idx, d_pair, d_ids);
        TE_FOR_CLASSES(TE_CASE)
#undef TE_CASE
    }
    return TE_ERR_BAD_ARG;
}

int launch_jk_class(int cb, int ck, te_pairs* P, double tau, int lane, int prec, cudaStream_t st) {
    switch (cb) {
#define TE_CASE(n) case n: return launch_jk_cb##n(ck, P, tau, lane, prec, st);
        TE_FOR_CLASSES(TE_CASE)
#undef TE_CASE
    }
    return TE_ERR_BAD_ARG;
}

int launch_eri_class(int cb, int ck, const te_basis* b, int n, const EriTask* d_tasks, double* out_dev) {
    switch (cb) {
#define TE_CASE(k) case k: return launch_eri_cb##k(ck, b, n, d_tasks, out_dev);
        TE_FOR_CLASSES(TE_CASE)
#undef TE_CASE
    }
    return TE_ERR_BAD_ARG;
}

int launch_hermite_density(int cls, te_pairs* P, cudaStream_t st) {
    switch (cls) {
#define TE_CASE(k) case k: return launch_hermite_density_cb##k(P, st);
        TE_FOR_CLASSES(TE_CASE)
#undef TE_CASE
    }
    return TE_ERR_BAD_ARG;
}

int launch_hermite_j(int cls, te_pairs* P, cudaStream_t st) {
    switch (cls) {
#define TE_CASE(k) case k: return launch_hermite_j_cb##k(P, st);
        TE_FOR_CLASSES(TE_CASE)
#undef TE_CASE
    }
    return TE_ERR_BAD_ARG;
}

int launch_jeng_class(int cb, int ck, te_pairs* P, double tau, cudaStream_t st) {
    switch (cb) {
#define TE_CASE(n) case n: return launch_jeng_cb##n(ck, P, tau, st);
        TE_FOR_CLASSES(TE_CASE)
#undef TE_CASE
    }
    return TE_ERR_BAD_ARG;
}

int launch_nuclear(int cls, te_pairs* P, int ncharge, const double4* d_chg, double* d_Vt, cudaStream_t st) {
    switch (cls) {
#define TE_CASE(k) case k: return launch_nuclear_cb##k(P, ncharge, d_chg, d_Vt, st);
        TE_FOR_CLASSES(TE_CASE)
#undef TE_CASE
    }
    return TE_ERR_BAD_ARG;
}

}  // namespace te
