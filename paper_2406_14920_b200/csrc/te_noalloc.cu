// te_noalloc.cu -- te_nuclear_attraction_noalloc: the nuclear-attraction matrix (eq. 14-26) for callers that cannot
// allocate (CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc).
//
// te_nuclear_attraction (te_lib.cu) uses two pieces of scratch: a device copy of the point charges (cudaMalloc / cudaFree per call)
// and an nbf x nbf accumulator Vt (the handle's J/K scratch).  This variant takes the charges as a DEVICE array from the caller and
// keeps Vt in a file-scope static __device__ array of fixed size, so the call allocates nothing, on the host or on the device:
// no cudaMalloc, cudaFree, std::vector or allocating library routine.  The price: nbf <= TE_NOALLOC_MAX_NBF, every GPU that loads
// the library holds the 2 MB array until exit, every call shares it (calls that overlap on the GPU race), and it keeps the last
// call's contents (so every call clears the part it uses first).
#include "te_kernels.cuh"

#include <mutex>

namespace te {

constexpr int NOALLOC_MAX_NBF = TE_NOALLOC_MAX_NBF;

// Vt accumulator of the no-alloc path.  In HOST code this name is a host-side stand-in, not a device address: the address the
// kernels get comes from cudaGetSymbolAddress below, once per device.
static __device__ __align__(256) double g_noalloc_vt[(size_t)NOALLOC_MAX_NBF * NOALLOC_MAX_NBF];

static std::mutex g_noalloc_mutex;
static double* g_noalloc_ptr[TE_MAX_DEV] = {nullptr};   // device address of g_noalloc_vt on each device

// Same arithmetic as nuclear_kernel (te_kernels.cuh): one thread = one primitive shell pair looping over all point charges,
// the charge sum taken in Hermite space, one Hermite -> Cartesian transform per pair (eq. 26).  Differences: the charges are read
// as 4 doubles (x, y, z, q) from a caller-owned device array with no alignment demand, and Vt is the static scratch.
template <int LA, int LB>
__global__ void __launch_bounds__(64) nuclear_noalloc_kernel(const PairD* __restrict__ pairs, const PairIds* __restrict__ ids, long long n,
                                                              int ncharge, const double* __restrict__ chg, const double* __restrict__ boys_tab,
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
        const double X = pd.P[0] - chg[4 * c], Y = pd.P[1] - chg[4 * c + 1], Z = pd.P[2] - chg[4 * c + 2], qc = chg[4 * c + 3];
        double F[LAB + 1], R[NH];
        boys<LAB>(pd.p * (X * X + Y * Y + Z * Z), boys_tab, F);
#pragma unroll
        for (int m = 0; m <= LAB; ++m) F[m] *= qc;
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

// V = (Vt + Vt^T) o (f f^T): the unordered pairs stand for both ordered pairs; f = per-component normalisation factors.
static __global__ void noalloc_finish_kernel(const double* __restrict__ Vt, const double* __restrict__ f, int nbf, double* __restrict__ V) {
    const long long n2 = (long long)nbf * nbf;
    for (long long x = blockIdx.x * (long long)blockDim.x + threadIdx.x; x < n2; x += (long long)gridDim.x * blockDim.x) {
        const int i = (int)(x / nbf), j = (int)(x % nbf);
        V[x] = (Vt[x] + Vt[(long long)j * nbf + i]) * (f[i] * f[j]);
    }
}

template <int LA, int LB>
static cudaError_t launch_one(const te_pairs* P, int cls, int ncharge, const double* chg, double* vt, cudaStream_t st) {
    const long long n = P->count[cls];
    if (n == 0) return cudaSuccess;
    nuclear_noalloc_kernel<LA, LB><<<(unsigned)((n + 63) / 64), 64, 0, st>>>(P->d_pair[cls], P->d_ids[cls], n, ncharge, chg, P->basis->d_boys,
                                                                           P->basis->nbf, vt);
    return cudaGetLastError();
}

}  // namespace te

using namespace te;

extern "C" int te_nuclear_attraction_noalloc(const te_pairs* P, int ncharge, const double* xyzq_dev, double* V_dev, void* stream_) {
    if (!P || ncharge < 0 || (ncharge > 0 && !xyzq_dev) || !V_dev) { set_error("te_nuclear_attraction_noalloc: NULL argument or negative count"); return TE_ERR_BAD_ARG; }
    const te_basis* b = P->basis;
    if (b->nbf > NOALLOC_MAX_NBF) {
        set_error("te_nuclear_attraction_noalloc: nbf = %d exceeds the static scratch (TE_NOALLOC_MAX_NBF = %d); use te_nuclear_attraction", b->nbf, NOALLOC_MAX_NBF);
        return TE_ERR_BAD_ARG;
    }
    int dev = -1;
    TE_CUDA(cudaGetDevice(&dev));
    if (dev != b->device || dev < 0 || dev >= TE_MAX_DEV) {
        set_error("te_nuclear_attraction_noalloc: current device %d is not the device %d the basis was created on", dev, b->device);
        return TE_ERR_BAD_ARG;
    }
    double* vt = nullptr;
    {   // once per device, with that device current: the device address of the static scratch
        std::lock_guard<std::mutex> lock(g_noalloc_mutex);
        if (!g_noalloc_ptr[dev]) {
            void* p = nullptr;
            TE_CUDA(cudaGetSymbolAddress(&p, g_noalloc_vt));
            g_noalloc_ptr[dev] = static_cast<double*>(p);
        }
        vt = g_noalloc_ptr[dev];
    }
    cudaStream_t st = (cudaStream_t)stream_;
    const size_t n2 = (size_t)b->nbf * b->nbf;
    TE_CUDA(cudaMemsetAsync(vt, 0, n2 * sizeof(double), st));   // the array keeps the last call's contents
    if (ncharge > 0) {
        cudaError_t e = cudaSuccess;
        if (e == cudaSuccess) e = launch_one<0, 0>(P, 0, ncharge, xyzq_dev, vt, st);
        if (e == cudaSuccess) e = launch_one<0, 1>(P, 1, ncharge, xyzq_dev, vt, st);
        if (e == cudaSuccess) e = launch_one<0, 2>(P, 2, ncharge, xyzq_dev, vt, st);
        if (e == cudaSuccess) e = launch_one<0, 3>(P, 3, ncharge, xyzq_dev, vt, st);
        if (e == cudaSuccess) e = launch_one<1, 1>(P, 4, ncharge, xyzq_dev, vt, st);
        if (e == cudaSuccess) e = launch_one<1, 2>(P, 5, ncharge, xyzq_dev, vt, st);
        if (e == cudaSuccess) e = launch_one<1, 3>(P, 6, ncharge, xyzq_dev, vt, st);
        if (e == cudaSuccess) e = launch_one<2, 2>(P, 7, ncharge, xyzq_dev, vt, st);
        if (e == cudaSuccess) e = launch_one<2, 3>(P, 8, ncharge, xyzq_dev, vt, st);
        if (e == cudaSuccess) e = launch_one<3, 3>(P, 9, ncharge, xyzq_dev, vt, st);
        if (e != cudaSuccess) { set_error("te_nuclear_attraction_noalloc: %s", cudaGetErrorString(e)); return TE_ERR_CUDA; }
    }
    noalloc_finish_kernel<<<592, 256, 0, st>>>(vt, b->d_aofac, b->nbf, V_dev);
    TE_CUDA(cudaGetLastError());
    return TE_OK;
}
