// te_lib.cu -- host side of the C ABI (include/te_jk.h): basis, pair builder, J/K build driver, Boys /
// peak utilities.  Kernels for the per-class work live in te_kernels.cuh and are instantiated in te_inst_*.cu.
#include "te_internal.h"

#include <cub/cub.cuh>

#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <cstdlib>
#include <climits>
#include <mutex>
#include <new>
#include <vector>

namespace te {

thread_local char g_err[512] = "";

void set_error(const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
}

// ------------------------------------------------------------------------------------------ Boys table
// F_m(T_i) for the Taylor grid of te_md.cuh, generated on the host in long double: convergent series at the
// top m (all terms positive), then the downward recursion.
static double* g_boys_tab[TE_MAX_DEV] = {nullptr};   // device, [BOYS_NPTS][BOYS_STRIDE]; one per CUDA device, built on first use
static std::mutex g_boys_mutex;

int ensure_boys_table(const double** out) {
    int dev = -1;
    TE_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= TE_MAX_DEV) { set_error("device id %d out of range", dev); return TE_ERR_BAD_ARG; }
    std::lock_guard<std::mutex> lock(g_boys_mutex);
    if (!g_boys_tab[dev]) {
        std::vector<double> h((size_t)BOYS_NPTS * BOYS_STRIDE);
        const int mtop = BOYS_MROWS - 1;
        for (int i = 0; i < BOYS_NPTS; ++i) {
            const long double T = (long double)i * (long double)BOYS_DT;
            const long double eT = expl(-T);
            long double term = 1.0L / (2 * mtop + 1), sum = term;
            for (int k = 1; k < 2000; ++k) {
                term *= 2.0L * T / (2 * mtop + 2 * k + 1);
                sum += term;
                if (term < 1e-22L * sum) break;
            }
            long double F = eT * sum;
            h[(size_t)i * BOYS_STRIDE + BOYS_MROWS] = (double)eT;
            h[(size_t)i * BOYS_STRIDE + mtop] = (double)F;
            for (int m = mtop; m > 0; --m) {
                F = (2.0L * T * F + eT) / (2 * m - 1);
                h[(size_t)i * BOYS_STRIDE + m - 1] = (double)F;
            }
        }
        double* d = nullptr;
        TE_CUDA(cudaMalloc(&d, h.size() * sizeof(double)));
        TE_CUDA(cudaMemcpy(d, h.data(), h.size() * sizeof(double), cudaMemcpyHostToDevice));
        g_boys_tab[dev] = d;
    }
    *out = g_boys_tab[dev];
    return TE_OK;
}

template <class T>
static int upload(const std::vector<T>& h, T** d) {
    *d = nullptr;
    if (h.empty()) return TE_OK;
    TE_CUDA(cudaMalloc(d, h.size() * sizeof(T)));
    TE_CUDA(cudaMemcpy(*d, h.data(), h.size() * sizeof(T), cudaMemcpyHostToDevice));
    return TE_OK;
}

static const int CLS_LA_H[TE_NCLASS] = {0, 0, 0, 0, 1, 1, 1, 2, 2, 3};
static const int CLS_LB_H[TE_NCLASS] = {0, 1, 2, 3, 1, 2, 3, 2, 3, 3};

static double dfact(int n) { double r = 1.0; for (; n > 1; n -= 2) r *= n; return r; }

}  // namespace te

using namespace te;

// ================================================================================================ basis
extern "C" int te_basis_create(int natoms, const double* xyz, int nshells, const int* shell_atom, const int* shell_l,
                               const int* shell_nprim, const double* exponents, const double* coefficients,
                               te_basis** out) {
    if (!out) { set_error("te_basis_create: out is NULL"); return TE_ERR_BAD_ARG; }
    *out = nullptr;
    if (natoms <= 0 || nshells <= 0 || !xyz || !shell_atom || !shell_l || !shell_nprim || !exponents || !coefficients) {
        set_error("te_basis_create: empty basis or NULL argument");
        return TE_ERR_BAD_ARG;
    }
    te_basis* b = new (std::nothrow) te_basis();
    if (!b) { set_error("te_basis_create: out of host memory"); return TE_ERR_ALLOC; }
    b->natoms = natoms; b->nshells = nshells;
    int np = 0, nbf = 0;
    for (int s = 0; s < nshells; ++s) {
        if (shell_l[s] < 0 || shell_nprim[s] < 1 || shell_atom[s] < 0 || shell_atom[s] >= natoms) {
            set_error("te_basis_create: shell %d has bad l / nprim / atom", s); delete b; return TE_ERR_BAD_ARG;
        }
        if (shell_l[s] > 3) { set_error("te_basis_create: shell %d has l = %d > 3", s, shell_l[s]); delete b; return TE_ERR_UNSUPPORTED_L; }
        b->shell_l.push_back(shell_l[s]); b->shell_off.push_back(nbf); b->shell_pstart.push_back(np);
        b->shell_nprim.push_back(shell_nprim[s]);
        nbf += ncart(shell_l[s]); np += shell_nprim[s];
    }
    b->shell_off.push_back(nbf); b->shell_pstart.push_back(np);
    b->nbf = nbf; b->nprim = np;
    for (int i = 0; i < np; ++i)
        if (!(exponents[i] > 0.0) || !std::isfinite(exponents[i]) || !std::isfinite(coefficients[i])) {
            set_error("te_basis_create: primitive %d has a non-positive exponent or non-finite value", i); delete b; return TE_ERR_BAD_ARG;
        }
    // Normalisation (eq. 1-2): radial norm of the x^l primitive, N = (2a/pi)^{3/4} (4a)^{l/2} / sqrt((2l-1)!!);
    // contracted self overlap of the x^l component S = sum c_m N_m c_n N_n (pi/p)^{3/2} (2l-1)!!/(2p)^l; c~ = cN/sqrt(S).
    const double pi = 3.14159265358979323846;
    std::vector<double> pxyz(3 * (size_t)np);
    b->prim_exp.resize(np); b->prim_ct.resize(np); b->prim_l.resize(np); b->prim_shell.resize(np);
    b->prim_iprim.resize(np); b->prim_off.resize(np);
    for (int s = 0; s < nshells; ++s) {
        const int l = shell_l[s], p0 = b->shell_pstart[s], n = shell_nprim[s];
        std::vector<double> c(n);
        for (int m = 0; m < n; ++m) {
            const double a = exponents[p0 + m];
            c[m] = coefficients[p0 + m] * std::pow(2.0 * a / pi, 0.75) * std::pow(4.0 * a, 0.5 * l) / std::sqrt(dfact(2 * l - 1));
        }
        double S = 0.0;
        for (int m = 0; m < n; ++m)
            for (int k = 0; k < n; ++k) {
                const double p = exponents[p0 + m] + exponents[p0 + k];
                S += c[m] * c[k] * std::pow(pi / p, 1.5) * dfact(2 * l - 1) / std::pow(2.0 * p, (double)l);
            }
        if (!(S > 0.0)) { set_error("te_basis_create: shell %d has zero norm", s); delete b; return TE_ERR_BAD_ARG; }
        for (int m = 0; m < n; ++m) {
            const int g = p0 + m;
            b->prim_exp[g] = exponents[g]; b->prim_ct[g] = c[m] / std::sqrt(S); b->prim_l[g] = l;
            b->prim_shell[g] = s; b->prim_iprim[g] = m; b->prim_off[g] = b->shell_off[s];
            for (int d = 0; d < 3; ++d) pxyz[3 * (size_t)g + d] = xyz[3 * shell_atom[s] + d];
        }
    }
    b->prim_xyz = pxyz;
    // primitives grouped by l (the pair builder enumerates class candidates from these lists)
    for (int l = 0; l < 4; ++l) {
        b->l_start[l] = (int)b->prims_by_l.size();
        for (int g = 0; g < np; ++g) if (b->prim_l[g] == l) b->prims_by_l.push_back(g);
    }
    b->l_start[4] = (int)b->prims_by_l.size();
    std::vector<double> aofac(nbf);
    for (int s = 0; s < nshells; ++s)
        for (int i = 0; i < ncart(shell_l[s]); ++i) aofac[b->shell_off[s] + i] = comp_factor(shell_l[s], i);
    // arguments are valid: from here on the device is needed (there is no CPU path)
    if (cudaGetDevice(&b->device) != cudaSuccess) { set_error("te_basis_create: no CUDA device (the library has no CPU path)"); delete b; return TE_ERR_CUDA; }
    int rc;
    if ((rc = upload(b->prim_exp, &b->d_exp)) || (rc = upload(b->prim_ct, &b->d_ct)) || (rc = upload(b->prim_xyz, &b->d_xyz)) ||
        (rc = upload(b->prim_shell, &b->d_shell)) || (rc = upload(b->prim_off, &b->d_off)) ||
        (rc = upload(b->prims_by_l, &b->d_by_l)) || (rc = upload(aofac, &b->d_aofac)) ||
        (rc = upload(b->shell_off, &b->d_shell_off)) || (rc = upload(b->shell_pstart, &b->d_shell_pstart)) || (rc = ensure_boys_table(&b->d_boys))) {
        te_basis_destroy(b);
        return rc;
    }
    *out = b;
    return TE_OK;
}

extern "C" void te_basis_destroy(te_basis* b) {
    if (!b) return;
    cudaFree(b->d_exp); cudaFree(b->d_ct); cudaFree(b->d_xyz); cudaFree(b->d_shell); cudaFree(b->d_off);
    cudaFree(b->d_by_l); cudaFree(b->d_aofac); cudaFree(b->d_shell_off); cudaFree(b->d_shell_pstart);
    delete b;
}

extern "C" int te_basis_nbf(const te_basis* b) { return b ? b->nbf : TE_ERR_BAD_ARG; }
extern "C" int te_basis_nprim(const te_basis* b) { return b ? b->nprim : TE_ERR_BAD_ARG; }

extern "C" int te_basis_shell_offsets(const te_basis* b, int* offsets) {
    if (!b || !offsets) { set_error("te_basis_shell_offsets: NULL argument"); return TE_ERR_BAD_ARG; }
    std::memcpy(offsets, b->shell_off.data(), sizeof(int) * (b->nshells + 1));
    return TE_OK;
}

extern "C" int te_basis_norm_coefs(const te_basis* b, double* norm) {
    if (!b || !norm) { set_error("te_basis_norm_coefs: NULL argument"); return TE_ERR_BAD_ARG; }
    std::memcpy(norm, b->prim_ct.data(), sizeof(double) * b->nprim);
    return TE_OK;
}

// =========================================================================================== pair build
__global__ void count_kept_kernel(const double* __restrict__ q_sorted, long long n, double tau, unsigned long long* out) {
    // q_sorted is descending: count entries >= tau
    long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    unsigned long long c = 0;
    for (; i < n; i += (long long)gridDim.x * blockDim.x) c += (q_sorted[i] >= tau) ? 1ull : 0ull;
    for (int o = 16; o > 0; o >>= 1) c += __shfl_down_sync(0xffffffffu, c, o);
    if ((threadIdx.x & 31) == 0 && c) atomicAdd(out, c);
}

// Shell-pair-major order: primitive pairs of one contracted shell pair (A,B) share every J/K output address, so the J/K kernels
// reduce over runs of them before touching memory.  key = A * nshells + B; bmax[key] = max bound of the block.
__global__ void block_key_kernel(const PairIds* __restrict__ ids, const double* __restrict__ q, long long n, int nshells,
                                 unsigned int* __restrict__ key, unsigned int* __restrict__ perm, unsigned long long* __restrict__ bmax) {
    const long long x = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (x >= n) return;
    const unsigned int k = (unsigned int)ids[x].shA * (unsigned int)nshells + (unsigned int)ids[x].shB;
    key[x] = k; perm[x] = (unsigned int)x;
    atomicMax(&bmax[k], (unsigned long long)__double_as_longlong(q[x]));   // bounds are >= 0: the bit pattern orders like the value
}
__global__ void block_max_gather_kernel(const unsigned int* __restrict__ key, long long n, const unsigned long long* __restrict__ bmax,
                                        double* __restrict__ bm) {
    const long long x = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (x < n) bm[x] = __longlong_as_double((long long)bmax[key[x]]);
}
__global__ void permute_pairs_kernel(const unsigned int* __restrict__ perm, long long n, const PairD* __restrict__ pin, const PairIds* __restrict__ iin,
                                     const double* __restrict__ qin, PairD* __restrict__ pout, PairIds* __restrict__ iout, double* __restrict__ qout) {
    const long long x = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (x >= n) return;
    const unsigned int y = perm[x];
    pout[x] = pin[y]; iout[x] = iin[y]; qout[x] = qin[y];
}

extern "C" int te_shellpair_build(const te_basis* b, double tau_pair, te_pairs** out) {
    if (!out) { set_error("te_shellpair_build: out is NULL"); return TE_ERR_BAD_ARG; }
    *out = nullptr;
    if (!b || !(tau_pair >= 0.0)) { set_error("te_shellpair_build: NULL basis or negative threshold"); return TE_ERR_BAD_ARG; }
    te_pairs* P = new (std::nothrow) te_pairs();
    if (!P) { set_error("te_shellpair_build: out of host memory"); return TE_ERR_ALLOC; }
    P->basis = b; P->tau_pair = tau_pair;
    unsigned long long* d_cnt = nullptr;
    int rc = TE_OK;
    auto fail = [&](int code) { cudaFree(d_cnt); te_pairs_destroy(P); return code; };
    if (cudaMalloc(&d_cnt, sizeof(unsigned long long)) != cudaSuccess) { set_error("cudaMalloc failed"); return fail(TE_ERR_ALLOC); }
    for (int la = 0; la < 4; ++la)
        for (int lb = la; lb < 4; ++lb) {
            const int cls = pair_class(la, lb);
            const long long na = b->l_start[la + 1] - b->l_start[la], nb = b->l_start[lb + 1] - b->l_start[lb];
            const long long ncand = (la == lb) ? na * (na + 1) / 2 : na * nb;
            P->count[cls] = 0;
            if (ncand == 0) continue;
            if (ncand > (long long)INT_MAX) {   // cub's item counts and the int pair indices of the J/K kernels
                set_error("te_shellpair_build: class %d has %lld candidate pairs, more than INT_MAX", cls, ncand); return fail(TE_ERR_BAD_ARG);
            }
            double *d_q = nullptr, *d_qs = nullptr;
            long long *d_idx = nullptr, *d_idxs = nullptr;
            void* d_tmp = nullptr;
            auto cleanup = [&]() { cudaFree(d_q); cudaFree(d_qs); cudaFree(d_idx); cudaFree(d_idxs); cudaFree(d_tmp); };
            if (cudaMalloc(&d_q, ncand * sizeof(double)) != cudaSuccess || cudaMalloc(&d_qs, ncand * sizeof(double)) != cudaSuccess ||
                cudaMalloc(&d_idx, ncand * sizeof(long long)) != cudaSuccess || cudaMalloc(&d_idxs, ncand * sizeof(long long)) != cudaSuccess) {
                cleanup(); set_error("te_shellpair_build: device allocation of %lld candidates failed", ncand); return fail(TE_ERR_ALLOC);
            }
            // pass 1: Schwarz bound of every candidate (eq. 45), diagonal integral class (la lb|la lb)
            if ((rc = launch_schwarz(la, lb, b, ncand, d_q, d_idx)) != TE_OK) { cleanup(); return fail(rc); }
            // sort by bound, descending (radix sort: stable, so ties keep ascending candidate order)
            size_t tmp_bytes = 0;
            cub::DeviceRadixSort::SortPairsDescending(nullptr, tmp_bytes, d_q, d_qs, d_idx, d_idxs, (int)ncand);
            if (cudaMalloc(&d_tmp, tmp_bytes) != cudaSuccess) { cleanup(); set_error("cub temp alloc failed"); return fail(TE_ERR_ALLOC); }
            if (cub::DeviceRadixSort::SortPairsDescending(d_tmp, tmp_bytes, d_q, d_qs, d_idx, d_idxs, (int)ncand) != cudaSuccess) {
                cleanup(); set_error("te_shellpair_build: radix sort failed: %s", cudaGetErrorString(cudaGetLastError())); return fail(TE_ERR_CUDA);
            }
            cudaMemset(d_cnt, 0, sizeof(unsigned long long));
            count_kept_kernel<<<296, 256>>>(d_qs, ncand, tau_pair, d_cnt);
            unsigned long long nk = 0;
            if (cudaMemcpy(&nk, d_cnt, sizeof(nk), cudaMemcpyDeviceToHost) != cudaSuccess) {
                cleanup(); set_error("te_shellpair_build: %s", cudaGetErrorString(cudaGetLastError())); return fail(TE_ERR_CUDA);
            }
            P->count[cls] = (long long)nk;
            if (nk) {
                // pass 2: pair data of the survivors in sorted order
                if (cudaMalloc(&P->d_pair[cls], nk * sizeof(PairD)) != cudaSuccess || cudaMalloc(&P->d_q[cls], nk * sizeof(double)) != cudaSuccess ||
                    cudaMalloc(&P->d_ids[cls], nk * sizeof(PairIds)) != cudaSuccess) {
                    cleanup(); set_error("te_shellpair_build: pair allocation failed"); return fail(TE_ERR_ALLOC);
                }
                const size_t nh = (size_t)nk * nherm(la + lb) * sizeof(double);
                if (cudaMalloc(&P->d_DH[cls], nh) != cudaSuccess || cudaMalloc(&P->d_JH[cls], nh) != cudaSuccess ||
                    cudaMalloc(&P->d_qmax[cls], nk * sizeof(double)) != cudaSuccess) {
                    cleanup(); set_error("te_shellpair_build: Hermite buffer allocation failed"); return fail(TE_ERR_ALLOC);
                }
                // pass 2: pair data of the survivors in bound order, then the shell-pair-major permutation:
                // stable sort by shell pair, then stable sort by the block's largest bound (descending); inside a block
                // the pairs stay in bound order
                PairD* t_pair = nullptr; PairIds* t_ids = nullptr;
                unsigned int *k0 = nullptr, *k1 = nullptr, *p0 = nullptr, *p1 = nullptr, *p2 = nullptr;
                unsigned long long* bmax = nullptr; double *bm = nullptr; void* tmp2 = nullptr;
                const size_t ns2 = (size_t)b->nshells * b->nshells;
                auto cleanup2 = [&]() { cudaFree(t_pair); cudaFree(t_ids); cudaFree(k0); cudaFree(k1); cudaFree(p0); cudaFree(p1); cudaFree(p2);
                                        cudaFree(bmax); cudaFree(bm); cudaFree(tmp2); };
                if (cudaMalloc(&t_pair, nk * sizeof(PairD)) != cudaSuccess || cudaMalloc(&t_ids, nk * sizeof(PairIds)) != cudaSuccess ||
                    cudaMalloc(&k0, nk * 4) != cudaSuccess || cudaMalloc(&k1, nk * 4) != cudaSuccess || cudaMalloc(&p0, nk * 4) != cudaSuccess ||
                    cudaMalloc(&p1, nk * 4) != cudaSuccess || cudaMalloc(&p2, nk * 4) != cudaSuccess || cudaMalloc(&bmax, ns2 * 8) != cudaSuccess ||
                    cudaMalloc(&bm, nk * sizeof(double)) != cudaSuccess) {
                    cleanup2(); cleanup(); set_error("te_shellpair_build: ordering scratch allocation failed"); return fail(TE_ERR_ALLOC);
                }
                if ((rc = launch_pair_fill(la, lb, b, (long long)nk, d_idxs, t_pair, t_ids)) != TE_OK) { cleanup2(); cleanup(); return fail(rc); }
                cudaMemset(bmax, 0, ns2 * 8);
                const unsigned gr = (unsigned)((nk + 255) / 256);
                block_key_kernel<<<gr, 256>>>(t_ids, d_qs, (long long)nk, b->nshells, k0, p0, bmax);
                size_t tb1 = 0, tb2 = 0;
                cub::DeviceRadixSort::SortPairs(nullptr, tb1, k0, k1, p0, p1, (int)nk);
                cub::DeviceRadixSort::SortPairsDescending(nullptr, tb2, bm, d_q, p1, p2, (int)nk);
                if (cudaMalloc(&tmp2, std::max(tb1, tb2)) != cudaSuccess) { cleanup2(); cleanup(); set_error("cub temp alloc failed"); return fail(TE_ERR_ALLOC); }
                tb1 = tb2 = std::max(tb1, tb2);
                cudaError_t es = cub::DeviceRadixSort::SortPairs(tmp2, tb1, k0, k1, p0, p1, (int)nk);
                block_max_gather_kernel<<<gr, 256>>>(k1, (long long)nk, bmax, bm);
                if (es == cudaSuccess) es = cub::DeviceRadixSort::SortPairsDescending(tmp2, tb2, bm, P->d_qmax[cls], p1, p2, (int)nk);
                if (es != cudaSuccess) { cleanup2(); cleanup(); set_error("te_shellpair_build: radix sort failed: %s", cudaGetErrorString(es)); return fail(TE_ERR_CUDA); }
                permute_pairs_kernel<<<gr, 256>>>(p2, (long long)nk, t_pair, t_ids, d_qs, P->d_pair[cls], P->d_ids[cls], P->d_q[cls]);
                cudaError_t e2 = cudaDeviceSynchronize();
                if (e2 == cudaSuccess) {
                    // block directory: where a new contracted shell pair starts in the final order
                    std::vector<PairIds> hid(nk);
                    e2 = cudaMemcpy(hid.data(), P->d_ids[cls], nk * sizeof(PairIds), cudaMemcpyDeviceToHost);
                    std::vector<int> bs;
                    for (unsigned long long x = 0; x < nk; ++x)
                        if (x == 0 || hid[x].shA != hid[x - 1].shA || hid[x].shB != hid[x - 1].shB) bs.push_back((int)x);
                    P->nblk[cls] = (int)bs.size();
                    bs.push_back((int)nk);
                    if (e2 == cudaSuccess && upload(bs, &P->d_bstart[cls]) != TE_OK) e2 = cudaErrorMemoryAllocation;
                }
                cleanup2();
                if (e2 != cudaSuccess) { cleanup(); set_error("te_shellpair_build: %s", cudaGetErrorString(e2)); return fail(TE_ERR_CUDA); }
            }
            cudaError_t e = cudaDeviceSynchronize();
            cleanup();
            if (e != cudaSuccess) { set_error("te_shellpair_build: %s", cudaGetErrorString(e)); return fail(TE_ERR_CUDA); }
        }
    cudaFree(d_cnt);
    // per-build scratch
    const size_t n2 = (size_t)b->nbf * b->nbf, ns2 = (size_t)b->nshells * b->nshells;
    if (cudaMalloc(&P->d_Ds, n2 * sizeof(double)) != cudaSuccess || cudaMalloc(&P->d_Jt, n2 * sizeof(double)) != cudaSuccess ||
        cudaMalloc(&P->d_Kt, n2 * sizeof(double)) != cudaSuccess || cudaMalloc(&P->d_Dm, ns2 * sizeof(double)) != cudaSuccess ||
        cudaMalloc(&P->d_ctrl, sizeof(JKControl)) != cudaSuccess || cudaMalloc(&P->d_ctrl32, sizeof(JKControl)) != cudaSuccess) {
        set_error("te_shellpair_build: scratch allocation failed"); te_pairs_destroy(P); return TE_ERR_ALLOC;
    }
    long long maxtiles = 0;
    for (int c = 0; c < TE_NCLASS; ++c) maxtiles = std::max(maxtiles, P->count[c] + 2);
    for (int s = 0; s < te_pairs::NSTREAM; ++s) {
        if (cudaMalloc(&P->d_tile_start[s], (maxtiles + 1) * sizeof(long long)) != cudaSuccess ||
            cudaMalloc(&P->d_task_hi[s], (maxtiles + 1) * sizeof(int)) != cudaSuccess) {
            set_error("te_shellpair_build: scratch allocation failed"); te_pairs_destroy(P); return TE_ERR_ALLOC;
        }
    }
    if (cudaEventCreateWithFlags(&P->ev_done, cudaEventDisableTiming) != cudaSuccess) {
        set_error("te_shellpair_build: event creation failed"); te_pairs_destroy(P); return TE_ERR_ALLOC;
    }
    P->tile_cap = maxtiles;
    for (int i = 0; i < TE_NCLASS * TE_NCLASS; ++i) { cudaEventCreate(&P->ev0[i]); cudaEventCreate(&P->ev1[i]); }
    *out = P;
    return TE_OK;
}

extern "C" void te_pairs_destroy(te_pairs* P) {
    if (!P) return;
    for (int c = 0; c < TE_NCLASS; ++c) { cudaFree(P->d_pair[c]); cudaFree(P->d_q[c]); cudaFree(P->d_ids[c]); cudaFree(P->d_DH[c]); cudaFree(P->d_JH[c]); cudaFree(P->d_qmax[c]); cudaFree(P->d_bstart[c]); }
    cudaFree(P->d_Ds); cudaFree(P->d_Jt); cudaFree(P->d_Kt); cudaFree(P->d_Dm); cudaFree(P->d_ctrl); cudaFree(P->d_ctrl32);
    for (int s = 0; s < te_pairs::NSTREAM; ++s) {
        cudaFree(P->d_tile_start[s]); cudaFree(P->d_task_hi[s]);
    }
    if (P->ev_done) cudaEventDestroy(P->ev_done);
    cudaFree(P->d_hD); cudaFree(P->d_hJ); cudaFree(P->d_hK);
    for (int i = 0; i < TE_NCLASS * TE_NCLASS; ++i) { if (P->ev0[i]) cudaEventDestroy(P->ev0[i]); if (P->ev1[i]) cudaEventDestroy(P->ev1[i]); }
    delete P;
}

extern "C" int te_pairs_info(const te_pairs* P, long long class_count[TE_NCLASS], long long* nkept) {
    if (!P) { set_error("te_pairs_info: NULL handle"); return TE_ERR_BAD_ARG; }
    long long tot = 0;
    for (int c = 0; c < TE_NCLASS; ++c) { if (class_count) class_count[c] = P->count[c]; tot += P->count[c]; }
    if (nkept) *nkept = tot;
    return TE_OK;
}

// The lists live on the device in shell-pair-major order (see te_shellpair_build); the exports present them in the order the
// header promises: Schwarz bound descending (stable, so equal bounds keep their internal order).
static int bound_order(const te_pairs* P, int cls, std::vector<double>& q, std::vector<long long>& order) {
    const long long n = P->count[cls];
    q.resize(n); order.resize(n);
    TE_CUDA(cudaMemcpy(q.data(), P->d_q[cls], n * sizeof(double), cudaMemcpyDeviceToHost));
    for (long long i = 0; i < n; ++i) order[i] = i;
    std::stable_sort(order.begin(), order.end(), [&](long long x, long long y) { return q[x] > q[y]; });
    return TE_OK;
}

extern "C" int te_pairs_export(const te_pairs* P, int cls, int* shellA, int* shellB, int* primA, int* primB, double* bound) {
    if (!P || cls < 0 || cls >= TE_NCLASS) { set_error("te_pairs_export: bad handle or class"); return TE_ERR_BAD_ARG; }
    const long long n = P->count[cls];
    if (n == 0) return TE_OK;
    std::vector<PairIds> ids(n);
    TE_CUDA(cudaMemcpy(ids.data(), P->d_ids[cls], n * sizeof(PairIds), cudaMemcpyDeviceToHost));
    std::vector<double> q; std::vector<long long> order;
    int rc = bound_order(P, cls, q, order);
    if (rc != TE_OK) return rc;
    const te_basis* b = P->basis;
    for (long long i = 0; i < n; ++i) {
        const PairIds& id = ids[order[i]];
        if (shellA) shellA[i] = id.shA;
        if (shellB) shellB[i] = id.shB;
        if (primA) primA[i] = b->prim_iprim[id.m];
        if (primB) primB[i] = b->prim_iprim[id.n];
        if (bound) bound[i] = q[order[i]];
    }
    return TE_OK;
}

extern "C" int te_pairs_export_geom(const te_pairs* P, int cls, double* P_xyz, double* p_exp, double* prefactor) {
    if (!P || cls < 0 || cls >= TE_NCLASS) { set_error("te_pairs_export_geom: bad handle or class"); return TE_ERR_BAD_ARG; }
    const long long n = P->count[cls];
    if (n == 0) return TE_OK;
    std::vector<PairD> pd(n);
    TE_CUDA(cudaMemcpy(pd.data(), P->d_pair[cls], n * sizeof(PairD), cudaMemcpyDeviceToHost));
    std::vector<double> q; std::vector<long long> order;
    int rc = bound_order(P, cls, q, order);
    if (rc != TE_OK) return rc;
    for (long long i = 0; i < n; ++i) {
        const PairD& x = pd[order[i]];
        if (P_xyz) for (int d = 0; d < 3; ++d) P_xyz[3 * i + d] = x.P[d];
        if (p_exp) p_exp[i] = x.p;
        if (prefactor) prefactor[i] = x.pref;
    }
    return TE_OK;
}

// ============================================================================================= J/K build
// Per-AO scaling by the component normalisation factor f (folded out of the integral kernels):
// Ds = D o (f f^T) on input; J = (Jt + Jt^T) o (f f^T) on output (same for K).
__global__ void scale_density_kernel(const double* __restrict__ D, const double* __restrict__ f, int nbf, double* __restrict__ Ds) {
    const long long n2 = (long long)nbf * nbf;
    for (long long x = blockIdx.x * (long long)blockDim.x + threadIdx.x; x < n2; x += (long long)gridDim.x * blockDim.x) {
        const int i = (int)(x / nbf), j = (int)(x % nbf);
        Ds[x] = D[x] * f[i] * f[j];
    }
}

// Dm[X][Y] = max |D| over the block of contracted shells (X,Y); also the global maximum.
__global__ void density_bounds_kernel(const double* __restrict__ D, const int* __restrict__ shell_off, int nshells, int nbf,
                                      double* __restrict__ Dm, JKControl* ctrl) {
    const long long ns2 = (long long)nshells * nshells;
    double mx_all = 0.0;
    for (long long x = blockIdx.x * (long long)blockDim.x + threadIdx.x; x < ns2; x += (long long)gridDim.x * blockDim.x) {
        const int X = (int)(x / nshells), Y = (int)(x % nshells);
        double mx = 0.0;
        for (int i = shell_off[X]; i < shell_off[X + 1]; ++i)
            for (int j = shell_off[Y]; j < shell_off[Y + 1]; ++j) mx = fmax(mx, fabs(D[(long long)i * nbf + j]));
        Dm[x] = mx;
        mx_all = fmax(mx_all, mx);
    }
    for (int o = 16; o > 0; o >>= 1) mx_all = fmax(mx_all, __shfl_down_sync(0xffffffffu, mx_all, o));
    if ((threadIdx.x & 31) == 0) atomicMax(reinterpret_cast<unsigned long long*>(&ctrl->dmax), (unsigned long long)__double_as_longlong(mx_all));
}

__global__ void finish_kernel(const double* __restrict__ Jt, const double* __restrict__ Kt, const double* __restrict__ f, int nbf,
                              double* __restrict__ J, double* __restrict__ K) {
    const long long n2 = (long long)nbf * nbf;
    for (long long x = blockIdx.x * (long long)blockDim.x + threadIdx.x; x < n2; x += (long long)gridDim.x * blockDim.x) {
        const int i = (int)(x / nbf), j = (int)(x % nbf);
        const long long y = (long long)j * nbf + i;
        const double s = f[i] * f[j];
        J[x] = (Jt[x] + Jt[y]) * s;
        K[x] = (Kt[x] + Kt[y]) * s;
    }
}

__global__ void copy_dmax_kernel(const JKControl* from, JKControl* to) { to->dmax = from->dmax; }

__global__ void finish_one_kernel(const double* __restrict__ Vt, const double* __restrict__ f, int nbf, double* __restrict__ V) {
    const long long n2 = (long long)nbf * nbf;
    for (long long x = blockIdx.x * (long long)blockDim.x + threadIdx.x; x < n2; x += (long long)gridDim.x * blockDim.x) {
        const int i = (int)(x / nbf), j = (int)(x % nbf);
        V[x] = (Vt[x] + Vt[(long long)j * nbf + i]) * (f[i] * f[j]);
    }
}

// Common start of every build on a handle: right device, wait for the previous build on this handle (the per-build scratch
// lives in the handle, so a handle carries ONE build at a time, whatever streams the callers use), per-build preamble.
static int build_begin(te_pairs* P, const double* D, double omega2, double prec_thr, cudaStream_t st, bool with_k) {
    const te_basis* b = P->basis;
    const int nbf = b->nbf;
    const size_t n2 = (size_t)nbf * nbf;
    int dev = -1;
    TE_CUDA(cudaGetDevice(&dev));
    if (dev != b->device) { set_error("te_build_jk: current device %d is not the device %d the basis was created on", dev, b->device); return TE_ERR_BAD_ARG; }
    if (P->ev_done_valid) TE_CUDA(cudaStreamWaitEvent(st, P->ev_done, 0));
    P->last_stream = st;
    P->omega2 = omega2;
    P->prec_thr = prec_thr;
    TE_CUDA(cudaMemsetAsync(P->d_Jt, 0, n2 * sizeof(double), st));
    if (with_k) TE_CUDA(cudaMemsetAsync(P->d_Kt, 0, n2 * sizeof(double), st));
    TE_CUDA(cudaMemsetAsync(P->d_ctrl, 0, sizeof(JKControl), st));
    TE_CUDA(cudaMemsetAsync(P->d_ctrl32, 0, sizeof(JKControl), st));
    scale_density_kernel<<<592, 256, 0, st>>>(D, b->d_aofac, nbf, P->d_Ds);
    density_bounds_kernel<<<592, 256, 0, st>>>(D, b->d_shell_off, b->nshells, nbf, P->d_Dm, P->d_ctrl);
    if (prec_thr > 0.0) copy_dmax_kernel<<<1, 1, 0, st>>>(P->d_ctrl, P->d_ctrl32);
    // Hermite density of every pair and zeroed Hermite J (eq. 35): inputs / accumulators of the Hermite-space Coulomb parts
    int rc = TE_OK;
    for (int c = 0; c < TE_NCLASS; ++c) {
        if (P->count[c] == 0) continue;
        TE_CUDA(cudaMemsetAsync(P->d_JH[c], 0, (size_t)P->count[c] * nherm(CLS_LA_H[c] + CLS_LB_H[c]) * sizeof(double), st));
        if ((rc = launch_hermite_density(c, P, st)) != TE_OK) return rc;
    }
    for (int i = 0; i < TE_NCLASS * TE_NCLASS; ++i) P->ev_valid[i] = false;
    return TE_OK;
}

// One build (1/r when omega2 == 0, erf(omega r)/r otherwise; FP64, or FP64 / FP32 by density-weighted bound when prec_thr > 0).
static int build_jk_impl(te_pairs* P, const double* D, double* J, double* K, double tau, double omega2, double prec_thr, cudaStream_t st) {
    const te_basis* b = P->basis;
    int rc = build_begin(P, D, omega2, prec_thr, st, true);
    if (rc != TE_OK) return rc;
    // class pairs, most expensive first (pair counts x transform work of one quartet)
    struct Job { int cb, ck; double w; bool has32; };
    std::vector<Job> jobs;
    for (int cb = 0; cb < TE_NCLASS; ++cb)
        for (int ck = cb; ck < TE_NCLASS; ++ck) {
            if (P->count[cb] == 0 || P->count[ck] == 0) continue;
            const int la = CLS_LA_H[cb], lb = CLS_LB_H[cb], lc = CLS_LA_H[ck], ld = CLS_LB_H[ck];
            const double w = (double)P->count[cb] * (double)P->count[ck] *
                             (60.0 + nherm(la + lb) * (double)nherm(lc + ld) + 7.0 * ncart(la) * ncart(lb) * ncart(lc) * ncart(ld));
            // mixed precision: classes without an FP32 leg (jk_fp32_class) run as in the FP64 build (prec 0)
            jobs.push_back(Job{cb, ck, w, prec_thr > 0.0 && jk_fp32_class(la, lb, lc, ld)});
        }
    std::sort(jobs.begin(), jobs.end(), [](const Job& x, const Job& y) { return x.w > y.w; });
    // Class kernels run back to back on the caller's stream: every one is a persistent grid that fills the GPU, and running
    // them concurrently on several streams measured 4.6 % SLOWER on config 5 (17.54 s serial, 18.38 s on 8 streams) and equal on
    // config 2.  With profiling on, an event pair brackets every class pair.
    for (const Job& j : jobs) {
        const int slot = j.cb * TE_NCLASS + j.ck;
        if (P->profiling) cudaEventRecord(P->ev0[slot], st);
        if ((rc = launch_jk_class(j.cb, j.ck, P, tau, 0, j.has32 ? 1 : 0, st)) != TE_OK) return rc;
        if (j.has32 && (rc = launch_jk_class(j.cb, j.ck, P, tau, 0, 2, st)) != TE_OK) return rc;
        if (P->profiling) { cudaEventRecord(P->ev1[slot], st); P->ev_valid[slot] = true; }
    }
    // Hermite J -> Cartesian J of every pair (the paper's CPU post-processing step, on the device)
    for (int c = 0; c < TE_NCLASS; ++c)
        if (P->count[c] && (rc = launch_hermite_j(c, P, st)) != TE_OK) return rc;
    finish_kernel<<<592, 256, 0, st>>>(P->d_Jt, P->d_Kt, b->d_aofac, b->nbf, J, K);
    TE_CUDA(cudaGetLastError());
    TE_CUDA(cudaEventRecord(P->ev_done, st));
    P->ev_done_valid = true;
    return TE_OK;
}

extern "C" int te_build_jk(te_pairs* P, const double* D, double* J, double* K, double tau, void* stream_) {
    if (!P || !D || !J || !K || !(tau >= 0.0)) { set_error("te_build_jk: NULL argument or negative threshold"); return TE_ERR_BAD_ARG; }
    return build_jk_impl(P, D, J, K, tau, 0.0, 0.0, (cudaStream_t)stream_);
}

extern "C" int te_build_jk_lr(te_pairs* P, const double* D, double* J, double* K, double tau, double omega, void* stream_) {
    if (!P || !D || !J || !K || !(tau >= 0.0) || !(omega > 0.0) || !std::isfinite(omega)) {
        set_error("te_build_jk_lr: NULL argument, negative threshold or non-positive omega"); return TE_ERR_BAD_ARG;
    }
    return build_jk_impl(P, D, J, K, tau, omega * omega, 0.0, (cudaStream_t)stream_);
}

extern "C" int te_build_jk_mixed(te_pairs* P, const double* D, double* J, double* K, double tau, double fp32_below, void* stream_) {
    if (!P || !D || !J || !K || !(tau >= 0.0) || !(fp32_below >= 0.0) || !std::isfinite(fp32_below)) {
        set_error("te_build_jk_mixed: NULL argument or negative threshold"); return TE_ERR_BAD_ARG;
    }
    return build_jk_impl(P, D, J, K, tau, 0.0, fp32_below, (cudaStream_t)stream_);
}

// Coulomb matrix alone by the J-engine route of eq. 35: Hermite density -> Hermite J in the jeng kernels -> Cartesian J.
extern "C" int te_build_j(te_pairs* P, const double* D, double* J, double tau, void* stream_) {
    if (!P || !D || !J || !(tau >= 0.0)) { set_error("te_build_j: NULL argument or negative threshold"); return TE_ERR_BAD_ARG; }
    cudaStream_t st = (cudaStream_t)stream_;
    const te_basis* b = P->basis;
    int rc = build_begin(P, D, 0.0, 0.0, st, false);
    if (rc != TE_OK) return rc;
    for (int cb = 0; cb < TE_NCLASS; ++cb)
        for (int ck = cb; ck < TE_NCLASS; ++ck) {
            if (P->count[cb] == 0 || P->count[ck] == 0) continue;
            const int slot = cb * TE_NCLASS + ck;
            if (P->profiling) cudaEventRecord(P->ev0[slot], st);
            if ((rc = launch_jeng_class(cb, ck, P, tau, st)) != TE_OK) return rc;
            if (P->profiling) { cudaEventRecord(P->ev1[slot], st); P->ev_valid[slot] = true; }
        }
    for (int c = 0; c < TE_NCLASS; ++c)
        if (P->count[c] && (rc = launch_hermite_j(c, P, st)) != TE_OK) return rc;
    finish_one_kernel<<<592, 256, 0, st>>>(P->d_Jt, b->d_aofac, b->nbf, J);
    TE_CUDA(cudaGetLastError());
    TE_CUDA(cudaEventRecord(P->ev_done, st));
    P->ev_done_valid = true;
    return TE_OK;
}

// Nuclear attraction (eq. 14-26): see nuclear_kernel in te_kernels.cuh.
extern "C" int te_nuclear_attraction(te_pairs* P, int ncharge, const double* xyz, const double* q, double* V_dev, void* stream_) {
    if (!P || ncharge < 0 || (ncharge > 0 && (!xyz || !q)) || !V_dev) { set_error("te_nuclear_attraction: NULL argument or negative count"); return TE_ERR_BAD_ARG; }
    const te_basis* b = P->basis;
    int dev = -1;
    TE_CUDA(cudaGetDevice(&dev));
    if (dev != b->device) { set_error("te_nuclear_attraction: current device %d is not the device %d the basis was created on", dev, b->device); return TE_ERR_BAD_ARG; }
    cudaStream_t st = (cudaStream_t)stream_;
    const size_t n2 = (size_t)b->nbf * b->nbf;
    std::vector<double4> h((size_t)ncharge);
    for (int c = 0; c < ncharge; ++c) {
        if (!std::isfinite(xyz[3 * c]) || !std::isfinite(xyz[3 * c + 1]) || !std::isfinite(xyz[3 * c + 2]) || !std::isfinite(q[c])) {
            set_error("te_nuclear_attraction: point charge %d is not finite", c); return TE_ERR_BAD_ARG;
        }
        h[c] = make_double4(xyz[3 * c], xyz[3 * c + 1], xyz[3 * c + 2], q[c]);
    }
    double4* d_chg = nullptr;
    if (ncharge > 0) {
        if (cudaMalloc(&d_chg, h.size() * sizeof(double4)) != cudaSuccess) { set_error("te_nuclear_attraction: device allocation failed"); return TE_ERR_ALLOC; }
        if (cudaMemcpy(d_chg, h.data(), h.size() * sizeof(double4), cudaMemcpyHostToDevice) != cudaSuccess) { cudaFree(d_chg); set_error("te_nuclear_attraction: copy failed"); return TE_ERR_CUDA; }
    }
    int rc = TE_OK;
    cudaError_t e = cudaSuccess;
    if (P->ev_done_valid) e = cudaStreamWaitEvent(st, P->ev_done, 0);   // d_Jt is the scratch of the J/K builds too
    if (e == cudaSuccess) e = cudaMemsetAsync(P->d_Jt, 0, n2 * sizeof(double), st);
    for (int c = 0; c < TE_NCLASS && rc == TE_OK && e == cudaSuccess && ncharge > 0; ++c) rc = launch_nuclear(c, P, ncharge, d_chg, P->d_Jt, st);
    if (rc == TE_OK && e == cudaSuccess) {
        finish_one_kernel<<<592, 256, 0, st>>>(P->d_Jt, b->d_aofac, b->nbf, V_dev);
        e = cudaGetLastError();
        if (e == cudaSuccess) e = cudaEventRecord(P->ev_done, st);
        if (e == cudaSuccess) P->ev_done_valid = true;
    }
    const cudaError_t e2 = cudaStreamSynchronize(st);   // the charge buffer is freed below
    cudaFree(d_chg);
    if (rc != TE_OK) return rc;
    if (e != cudaSuccess || e2 != cudaSuccess) { set_error("te_nuclear_attraction: %s", cudaGetErrorString(e != cudaSuccess ? e : e2)); return TE_ERR_CUDA; }
    return TE_OK;
}

extern "C" int te_build_jk_host(te_pairs* P, const double* D, double* J, double* K, double tau) {
    if (!P || !D || !J || !K) { set_error("te_build_jk_host: NULL argument"); return TE_ERR_BAD_ARG; }
    const size_t bytes = (size_t)P->basis->nbf * P->basis->nbf * sizeof(double);
    if (!P->d_hD) {
        if (cudaMalloc(&P->d_hD, bytes) != cudaSuccess || cudaMalloc(&P->d_hJ, bytes) != cudaSuccess || cudaMalloc(&P->d_hK, bytes) != cudaSuccess) {
            set_error("te_build_jk_host: device allocation failed"); return TE_ERR_ALLOC;
        }
    }
    TE_CUDA(cudaMemcpyAsync(P->d_hD, D, bytes, cudaMemcpyHostToDevice, 0));
    int rc = te_build_jk(P, P->d_hD, P->d_hJ, P->d_hK, tau, nullptr);
    if (rc != TE_OK) return rc;
    TE_CUDA(cudaMemcpyAsync(J, P->d_hJ, bytes, cudaMemcpyDeviceToHost, 0));
    TE_CUDA(cudaMemcpyAsync(K, P->d_hK, bytes, cudaMemcpyDeviceToHost, 0));
    TE_CUDA(cudaStreamSynchronize(0));
    return TE_OK;
}

extern "C" int te_jk_set_kernel_family(te_pairs* P, int family) {
    if (!P || family < 0 || family > 3) { set_error("te_jk_set_kernel_family: NULL handle or family outside 0..3"); return TE_ERR_BAD_ARG; }
    P->impl = family;
    return TE_OK;
}

extern "C" int te_jk_set_profiling(te_pairs* P, int on) {
    if (!P) { set_error("te_jk_set_profiling: NULL handle"); return TE_ERR_BAD_ARG; }
    P->profiling = on != 0;
    return TE_OK;
}

extern "C" int te_jk_stats(const te_pairs* P, long long quartets[TE_NCLASS][TE_NCLASS], float ms[TE_NCLASS][TE_NCLASS]) {
    if (!P) { set_error("te_jk_stats: NULL handle"); return TE_ERR_BAD_ARG; }
    TE_CUDA(cudaStreamSynchronize(P->last_stream));
    JKControl h, h32;
    TE_CUDA(cudaMemcpy(&h, P->d_ctrl, sizeof(h), cudaMemcpyDeviceToHost));
    TE_CUDA(cudaMemcpy(&h32, P->d_ctrl32, sizeof(h32), cudaMemcpyDeviceToHost));
    for (int cb = 0; cb < TE_NCLASS; ++cb)
        for (int ck = 0; ck < TE_NCLASS; ++ck) {
            const int slot = cb * TE_NCLASS + ck;
            if (quartets) quartets[cb][ck] = (long long)(h.live[slot] + h32.live[slot]);
            if (ms) {
                float t = 0.f;
                if (P->ev_valid[slot]) cudaEventElapsedTime(&t, P->ev0[slot], P->ev1[slot]);
                ms[cb][ck] = t;
            }
        }
    return TE_OK;
}

extern "C" int te_jk_precision_stats(const te_pairs* P, long long fp64_quartets[TE_NCLASS][TE_NCLASS], long long fp32_quartets[TE_NCLASS][TE_NCLASS]) {
    if (!P) { set_error("te_jk_precision_stats: NULL handle"); return TE_ERR_BAD_ARG; }
    TE_CUDA(cudaStreamSynchronize(P->last_stream));
    JKControl h, h32;
    TE_CUDA(cudaMemcpy(&h, P->d_ctrl, sizeof(h), cudaMemcpyDeviceToHost));
    TE_CUDA(cudaMemcpy(&h32, P->d_ctrl32, sizeof(h32), cudaMemcpyDeviceToHost));
    for (int cb = 0; cb < TE_NCLASS; ++cb)
        for (int ck = 0; ck < TE_NCLASS; ++ck) {
            if (fp64_quartets) fp64_quartets[cb][ck] = (long long)h.live[cb * TE_NCLASS + ck];
            if (fp32_quartets) fp32_quartets[cb][ck] = (long long)h32.live[cb * TE_NCLASS + ck];
        }
    return TE_OK;
}

extern "C" int te_jk_screening_stats(const te_pairs* P, long long visited[TE_NCLASS][TE_NCLASS], long long slots[TE_NCLASS][TE_NCLASS]) {
    if (!P) { set_error("te_jk_screening_stats: NULL handle"); return TE_ERR_BAD_ARG; }
    TE_CUDA(cudaStreamSynchronize(P->last_stream));
    JKControl h;
    TE_CUDA(cudaMemcpy(&h, P->d_ctrl, sizeof(h), cudaMemcpyDeviceToHost));
    for (int cb = 0; cb < TE_NCLASS; ++cb)
        for (int ck = 0; ck < TE_NCLASS; ++ck) {
            if (visited) visited[cb][ck] = (long long)h.visited[cb * TE_NCLASS + ck];
            if (slots) slots[cb][ck] = (long long)h.slots[cb * TE_NCLASS + ck];
        }
    return TE_OK;
}

// ============================================================================================= utilities
extern "C" int te_eri_block(const te_basis* b, int nq, const int* quartets, const long long* offs, double* out_dev) {
    if (!b || nq < 0 || (nq > 0 && (!quartets || !offs || !out_dev))) { set_error("te_eri_block: NULL argument"); return TE_ERR_BAD_ARG; }
    if (nq == 0) return TE_OK;
    // canonicalise every quartet to la<=lb, lc<=ld, class(ab)<=class(cd); record output strides
    std::vector<EriTask> tasks[TE_NCLASS * TE_NCLASS];
    for (int x = 0; x < nq; ++x) {
        int s[4], stride[4];
        for (int k = 0; k < 4; ++k) {
            s[k] = quartets[4 * x + k];
            if (s[k] < 0 || s[k] >= b->nshells) { set_error("te_eri_block: quartet %d has shell id %d out of range", x, s[k]); return TE_ERR_BAD_ARG; }
        }
        const int n[4] = {ncart(b->shell_l[s[0]]), ncart(b->shell_l[s[1]]), ncart(b->shell_l[s[2]]), ncart(b->shell_l[s[3]])};
        stride[0] = n[1] * n[2] * n[3]; stride[1] = n[2] * n[3]; stride[2] = n[3]; stride[3] = 1;
        int o[4] = {0, 1, 2, 3};
        if (b->shell_l[s[o[0]]] > b->shell_l[s[o[1]]]) std::swap(o[0], o[1]);
        if (b->shell_l[s[o[2]]] > b->shell_l[s[o[3]]]) std::swap(o[2], o[3]);
        int cb = pair_class(b->shell_l[s[o[0]]], b->shell_l[s[o[1]]]), ck = pair_class(b->shell_l[s[o[2]]], b->shell_l[s[o[3]]]);
        if (cb > ck) { std::swap(o[0], o[2]); std::swap(o[1], o[3]); std::swap(cb, ck); }
        EriTask t;
        for (int k = 0; k < 4; ++k) { t.sh[k] = s[o[k]]; t.stride[k] = stride[o[k]]; }
        t.out = offs[x];
        if (offs[x + 1] - offs[x] != (long long)n[0] * n[1] * n[2] * n[3]) { set_error("te_eri_block: out_offsets of quartet %d do not match its size", x); return TE_ERR_BAD_ARG; }
        tasks[cb * TE_NCLASS + ck].push_back(t);
    }
    TE_CUDA(cudaMemset(out_dev, 0, (size_t)offs[nq] * sizeof(double)));
    for (int cb = 0; cb < TE_NCLASS; ++cb)
        for (int ck = cb; ck < TE_NCLASS; ++ck) {
            auto& v = tasks[cb * TE_NCLASS + ck];
            if (v.empty()) continue;
            EriTask* d = nullptr;
            int rc = upload(v, &d);
            if (rc == TE_OK) rc = launch_eri_class(cb, ck, b, (int)v.size(), d, out_dev);
            cudaError_t e = cudaDeviceSynchronize();
            cudaFree(d);
            if (rc != TE_OK) return rc;
            if (e != cudaSuccess) { set_error("te_eri_block: %s", cudaGetErrorString(e)); return TE_ERR_CUDA; }
        }
    return TE_OK;
}

template <int L>
__global__ void boys_kernel(int n, const double* __restrict__ T, const double* __restrict__ tab, double* __restrict__ F) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    double f[L + 1];
    boys<L>(T[i], tab, f);
#pragma unroll
    for (int m = 0; m <= L; ++m) F[(size_t)i * (L + 1) + m] = f[m];
}

template <int L>
static void boys_dispatch(int mmax, int n, const double* T, const double* tab, double* F) {
    if (mmax == L) boys_kernel<L><<<(n + 127) / 128, 128>>>(n, T, tab, F);
    else if constexpr (L > 0) boys_dispatch<L - 1>(mmax, n, T, tab, F);
}

extern "C" int te_boys(int n, const double* T_dev, int mmax, double* F_dev) {
    if (n < 0 || mmax < 0 || mmax > 12 || (n > 0 && (!T_dev || !F_dev))) { set_error("te_boys: bad argument"); return TE_ERR_BAD_ARG; }
    if (n == 0) return TE_OK;
    const double* tab;
    int rc = ensure_boys_table(&tab);
    if (rc) return rc;
    boys_dispatch<12>(mmax, n, T_dev, tab, F_dev);
    TE_CUDA(cudaDeviceSynchronize());
    return TE_OK;
}

// Register-resident DFMA chains: 8 independent accumulators per thread, every SM busy.
__global__ void __launch_bounds__(256) dfma_peak_kernel(double* out, int iters, double a, double b) {
    double x0 = threadIdx.x, x1 = x0 + 1, x2 = x0 + 2, x3 = x0 + 3, x4 = x0 + 4, x5 = x0 + 5, x6 = x0 + 6, x7 = x0 + 7;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int k = 0; k < 16; ++k) {
            x0 = fma(x0, a, b); x1 = fma(x1, a, b); x2 = fma(x2, a, b); x3 = fma(x3, a, b);
            x4 = fma(x4, a, b); x5 = fma(x5, a, b); x6 = fma(x6, a, b); x7 = fma(x7, a, b);
        }
    }
    out[blockIdx.x * blockDim.x + threadIdx.x] = x0 + x1 + x2 + x3 + x4 + x5 + x6 + x7;
}

extern "C" int te_measure_fp64_peak(double* tflops) {
    if (!tflops) { set_error("te_measure_fp64_peak: NULL argument"); return TE_ERR_BAD_ARG; }
    int dev = 0, sms = 0;
    TE_CUDA(cudaGetDevice(&dev));
    TE_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    const int blocks = sms * 8, threads = 256, iters = 4096;
    double* d = nullptr;
    TE_CUDA(cudaMalloc(&d, (size_t)blocks * threads * sizeof(double)));
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    double best = 0.0;
    for (int rep = 0; rep < 6; ++rep) {
        cudaEventRecord(e0);
        dfma_peak_kernel<<<blocks, threads>>>(d, iters, 0.999999, 1e-9);
        cudaEventRecord(e1);
        cudaEventSynchronize(e1);
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        const double fl = 2.0 * 8 * 16 * (double)iters * blocks * threads;
        if (rep > 0) best = std::max(best, fl / (ms * 1e-3) / 1e12);
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(d);
    TE_CUDA(cudaGetLastError());
    *tflops = best;
    return TE_OK;
}

// The Hermite -> Cartesian transform of the uniform-ket kernel as a roofline probe: per iteration 20 lane-private LDS.64 from a
// conflict-free shared-memory column (element e of lane x at R[e * 32 + x], the layout of the R tensor) feed 20 independent
// DFMAs, one warp per block, `warps_per_sm` resident warps.  The rate it reaches is the shared-memory ceiling of that transform.
__global__ void __launch_bounds__(32) lds_dfma_probe_kernel(double* out, int iters, double e) {
    extern __shared__ double sm[];
    double* R = sm + threadIdx.x;
    for (int i = 0; i < 192; ++i) R[i * 32] = i * 0.001 + threadIdx.x;
    double y[20];
#pragma unroll
    for (int i = 0; i < 20; ++i) y[i] = 0.0;
    for (int it = 0; it < iters; ++it) {
        const double* Rq = R + (it & 7) * (20 * 32);
#pragma unroll
        for (int i = 0; i < 20; ++i) y[i] = fma(e, Rq[i * 32], y[i]);
    }
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < 20; ++i) s += y[i];
    out[blockIdx.x * 32 + threadIdx.x] = s;
}

extern "C" int te_measure_smem_dfma_rate(int warps_per_sm, double* tflops) {
    if (!tflops || warps_per_sm < 1 || warps_per_sm > 32) { set_error("te_measure_smem_dfma_rate: bad argument"); return TE_ERR_BAD_ARG; }
    int dev = 0, sms = 0;
    TE_CUDA(cudaGetDevice(&dev));
    TE_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    const int blocks = sms * warps_per_sm, iters = 20000;
    double* d = nullptr;
    TE_CUDA(cudaMalloc(&d, (size_t)blocks * 32 * sizeof(double)));
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    double best = 0.0;
    for (int rep = 0; rep < 4; ++rep) {
        cudaEventRecord(e0);
        lds_dfma_probe_kernel<<<blocks, 32, 192 * 32 * sizeof(double)>>>(d, iters, 1.0000001);
        cudaEventRecord(e1);
        cudaEventSynchronize(e1);
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        if (rep > 0) best = std::max(best, 2.0 * 20 * (double)iters * blocks * 32 / (ms * 1e-3) / 1e12);
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(d);
    TE_CUDA(cudaGetLastError());
    *tflops = best;
    return TE_OK;
}

extern "C" const char* te_last_error(void) { return te::g_err; }
