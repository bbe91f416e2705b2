/*
 * te_jk.h -- C ABI of the B200-native direct-SCF Coulomb/exchange (J/K) Fock build.
 *
 * Method: arXiv 2406.14920 (PAPER.md; "P:n" = line n).  Four-centre electron-repulsion integrals over
 * contracted Cartesian Gaussian shells l = 0..3 (eq. 27-31), McMurchie-Davidson scheme
 * (E eq. 5-8, Boys eq. 18, R eq. 20-25), contracted on the fly with a density matrix into
 *   J_mu,nu     = sum_{lambda,sigma} (mu nu|lambda sigma) D_lambda,sigma      (eq. 34)
 *   K_mu,lambda = sum_{nu,sigma}     (mu nu|lambda sigma) D_nu,sigma          (eq. 36)
 * over Schwarz-screened PRIMITIVE shell pairs (eq. 45) with the per-term density-weighted
 * test of eq. 47.  No factors of 2 or 1/2 are applied to J or K.
 *
 * Conventions
 *  - Every function returns TE_OK (0) or a negative TE_ERR_* code; te_last_error() gives a thread-local
 *    message.  No C++ exception and no exit() crosses this boundary.
 *  - "host" / "device" says where a pointer must live.  Handles (te_basis, te_pairs) are library-owned:
 *    create with te_*_create / te_shellpair_build, free with te_*_destroy.  All other buffers are
 *    caller-owned.
 *  - Lengths in bohr.  Matrices are row-major nbf x nbf FP64.  AO order = caller's shell order; inside a
 *    shell the Cartesian components are lexicographic with x^l first:
 *      p: x y z;  d: xx xy xz yy yz zz;  f: xxx xxy xxz xyy xyz xzz yyy yyz yzz zzz.
 *  - Every contracted Cartesian function is normalised to unit self-overlap (eq. 1-2); the
 *    caller passes RAW contraction coefficients.
 *  - There is no CPU fallback: every call that computes needs a CUDA device (sm_100a build).
 *  - Devices: a te_basis lives on the CUDA device that was current in te_basis_create, and so does every te_pairs
 *    built from it; calls that compute return TE_ERR_BAD_ARG when another device is current.  Several devices may be
 *    used from one process (the library's tables are kept per device).
 *  - Concurrency: the scratch of a build (accumulators, schedules, statistics) lives in the te_pairs handle, so a
 *    handle carries ONE build at a time.  Builds issued on different streams with the same handle are serialised by
 *    the library on the device (each waits for the previous one); calls on one handle from several host threads at
 *    once are not supported.  Use one te_pairs per concurrent build.
 *  - Size limits: a pair class may hold at most INT_MAX candidate pairs (TE_ERR_BAD_ARG beyond).
 */
#ifndef TE_JK_H
#define TE_JK_H

#ifdef __cplusplus
extern "C" {
#endif

#define TE_OK 0
#define TE_ERR_BAD_ARG (-1)
#define TE_ERR_UNSUPPORTED_L (-2)
#define TE_ERR_ALLOC (-3)
#define TE_ERR_CUDA (-4)

#define TE_NCLASS 10 /* primitive shell-pair classes SS SP SD SF PP PD PF DD DF FF */
#define TE_NOALLOC_MAX_NBF 512 /* largest nbf te_nuclear_attraction_noalloc accepts: 512^2 doubles = 2 MiB of static device scratch */

typedef struct te_basis te_basis; /* opaque */
typedef struct te_pairs te_pairs; /* opaque */

/* Basis (eq. 1-2).  All pointers HOST.  xyz_bohr[natoms][3]; shell_atom/shell_l/shell_nprim
 * [nshells]; exponents/coefficients concatenated over shells in shell order (sum of shell_nprim entries).
 * l > 3 -> TE_ERR_UNSUPPORTED_L.  Normalises, uploads to the current CUDA device, returns a handle. */
int te_basis_create(int natoms, const double *xyz_bohr, int nshells, const int *shell_atom,
                    const int *shell_l, const int *shell_nprim, const double *exponents,
                    const double *coefficients, te_basis **out);
void te_basis_destroy(te_basis *b);
/* Number of Cartesian basis functions, sum of (l+1)(l+2)/2. */
int te_basis_nbf(const te_basis *b);
/* Number of primitive shells, sum of shell_nprim. */
int te_basis_nprim(const te_basis *b);
/* offsets[nshells+1] HOST: first AO of every shell. */
int te_basis_shell_offsets(const te_basis *b, int *offsets);
/* norm[nprim] HOST: normalised primitive coefficient c~ (x^l component) of every primitive shell. */
int te_basis_norm_coefs(const te_basis *b, double *norm);

/* Primitive shell-pair lists (section 3.2): all unordered primitive shell pairs, Schwarz bound
 * q = max over components of sqrt|(mu nu|mu nu)| (eq. 45), pairs with q < pair_threshold (PQTHRE)
 * dropped, survivors binned into the 10 (la<=lb) classes and sorted by q descending inside each class.
 * Computed on the device.  pair_threshold = 0 keeps every pair. */
int te_shellpair_build(const te_basis *b, double pair_threshold, te_pairs **out);
void te_pairs_destroy(te_pairs *p);
/* class_count[10], *nkept: HOST outputs. */
int te_pairs_info(const te_pairs *p, long long class_count[TE_NCLASS], long long *nkept);
/* HOST copies of class `cls` in the library's sorted order (arrays of class_count[cls] entries; any pointer
 * may be NULL): contracted shell ids, primitive index inside each shell, Schwarz bound. */
int te_pairs_export(const te_pairs *p, int cls, int *shellA, int *shellB, int *primA, int *primB,
                    double *bound);
/* HOST copies: Gaussian product centre P [n][3], exponent p = a+b, and prefactor
 * c~_m c~_n exp(-ab/p |A-B|^2) (eq. 3). */
int te_pairs_export_geom(const te_pairs *p, int cls, double *P_xyz, double *p_exp, double *prefactor);

/* One J/K build (section 3.4).  D_dev, J_dev, K_dev: DEVICE, row-major nbf x nbf; D must be
 * symmetric (the kernels read D_xy or D_yx, whichever is closer in memory to what the warp already touches); J and K
 * are OVERWRITTEN (not accumulated) and returned symmetric.  threshold = THRECL of eq. 47; 0 means no screening.  A primitive quartet's contribution X <- D_YZ is included iff
 * q_bra * q_ket * max|D_YZ block| >= threshold, separately for each of its J and K updates.
 * Asynchronous on cuda_stream (a cudaStream_t, NULL = default stream). */
int te_build_jk(te_pairs *p, const double *D_dev, double *J_dev, double *K_dev, double threshold,
                void *cuda_stream);
/* Same build with HOST D, J, K (pinned or pageable): copies in, builds, copies out, synchronises. */
int te_build_jk_host(te_pairs *p, const double *D_host, double *J_host, double *K_host,
                     double threshold);
/* Long-range build for range-separated hybrids (eq. 32-33): the same J and K with the operator
 * erf(omega r)/r in place of 1/r.  Only the argument of the auxiliary integrals, pq omega^2 / (pq + (p+q) omega^2),
 * and the prefactor, 2 pi^{5/2} omega / (p q sqrt(pq + (p+q) omega^2)), change; the pair lists, their Schwarz bounds
 * (which also bound the attenuated integrals) and the per-term rule are those of te_build_jk.  omega > 0, in 1/bohr. */
int te_build_jk_lr(te_pairs *p, const double *D_dev, double *J_dev, double *K_dev, double threshold, double omega,
                   void *cuda_stream);
/* Coulomb matrix alone by the "J engine" of eq. 35, for every angular class: the density is
 * transformed to the Hermite basis of each ket pair, the quartets are contracted in Hermite space (R_PQ only, no
 * Hermite -> Cartesian transform of integrals), and the Hermite J of each bra pair is transformed back -- all three steps
 * on the device (the paper keeps the outer two on the CPU).  Same pair lists and the same per-term rule as the J updates
 * of te_build_jk (J_AB <- D_CD iff q q Dm_CD >= threshold, J_CD <- D_AB iff q q Dm_AB >= threshold), so J equals the J
 * of te_build_jk to rounding.  J_dev: DEVICE nbf x nbf, OVERWRITTEN.  Asynchronous on cuda_stream. */
int te_build_j(te_pairs *p, const double *D_dev, double *J_dev, double threshold, void *cuda_stream);
/* Mixed-precision build ("integrals with a density weighted Schwartz upper bound above a threshold (1e-5,
 * the default) are evaluated in double precision while the rest are evaluated in single precision").  A primitive
 * quartet whose density-weighted bound -- q_bra q_ket times the largest of its six density bounds -- is below
 * fp32_below is evaluated by FP32 kernels (R, E tables, both transforms, digestion), the others by the FP64 kernels of
 * te_build_jk; pair data, Boys values and prefactors are always FP64, and J / K are accumulated in FP64.  Same pair
 * lists and per-term rule as te_build_jk.  30 of the 55 classes have an FP32 leg (not those with l_a+l_b+l_c+l_d <= 2,
 * the lightest s/p classes and df / ff bras), and a quartet whose ket exponent would push (2 alpha)^L outside the FP32
 * range stays FP64.  fp32_below = 0 reproduces te_build_jk.  The result differs from te_build_jk by the FP32 rounding of
 * the small terms (measured error study); it is NOT held to the 1e-10 parity bar. */
int te_build_jk_mixed(te_pairs *p, const double *D_dev, double *J_dev, double *K_dev, double threshold,
                      double fp32_below, void *cuda_stream);
/* Live quartets of the LAST build per precision leg (te_build_jk: everything in fp64_quartets).  HOST outputs. */
int te_jk_precision_stats(const te_pairs *p, long long fp64_quartets[TE_NCLASS][TE_NCLASS],
                          long long fp32_quartets[TE_NCLASS][TE_NCLASS]);
/* Nuclear-attraction matrix (eq. 14-26): V_mu,nu = sum_C q_C (mu| 1/|r - C| |nu) over `ncharge` point
 * charges, summed over the kept primitive pairs of the handle (one thread per primitive pair looping over the charges,
 * P:356).  The sign is that of eq. 14: a nucleus of charge Z enters with q_C = -Z.  xyz_bohr[ncharge][3] and q[ncharge]:
 * HOST; V_dev: DEVICE, row-major nbf x nbf, OVERWRITTEN, symmetric.  Runs on cuda_stream and synchronises it before
 * returning. */
int te_nuclear_attraction(te_pairs *p, int ncharge, const double *xyz_bohr, const double *q, double *V_dev,
                          void *cuda_stream);
/* Statistics of the LAST te_build_jk on this handle (synchronises the build's stream).  HOST outputs,
 * indexed [bra class][ket class] (only bra class <= ket class is used): unique primitive quartets that
 * had at least one live update, and device milliseconds spent in that class pair's kernel. */
int te_jk_stats(const te_pairs *p, long long quartets[TE_NCLASS][TE_NCLASS], float ms[TE_NCLASS][TE_NCLASS]);
/* Screening statistics of the LAST te_build_jk on this handle (synchronises), same indexing: `visited` = unique
 * primitive quartets inside the schedule's cut whose per-term tests (eq. 47) were evaluated (the oracle's
 * "visited" counts every unique quartet of the kept lists; the cut of P:391 skips the rest), `slots` = quartet
 * slots of the warp batches that ran the integral code, so live / slots is the lane occupancy of the class kernel.
 * Either pointer may be NULL. */
int te_jk_screening_stats(const te_pairs *p, long long visited[TE_NCLASS][TE_NCLASS], long long slots[TE_NCLASS][TE_NCLASS]);
/* The same matrix for callers that cannot allocate (CUDA graph capture, serving loops, harnesses that forbid cudaMalloc):
 * this call performs NO allocation, on the host or on the device (no cudaMalloc / cudaFree, no allocating library routine) and
 * no synchronisation; it is asynchronous on cuda_stream.  Its nbf x nbf accumulator is a file-scope static device array of
 * TE_NOALLOC_MAX_NBF^2 doubles (2 MiB, held by every GPU that loads the library until the process exits), so
 * nbf > TE_NOALLOC_MAX_NBF is rejected with TE_ERR_BAD_ARG (use te_nuclear_attraction).  The charges are a DEVICE array
 * xyzq_dev[ncharge][4] = (x, y, z, q_C), caller-owned, 8-byte aligned.  V_dev: DEVICE nbf x nbf, OVERWRITTEN.  Every call on a
 * device shares the one array: calls that overlap on the GPU (different streams, or different handles) RACE -- serialise them.
 * The array keeps the last call's contents; each call clears what it uses before accumulating.  Does not touch the handle's
 * scratch, so it may overlap a J/K build on the same handle. */
int te_nuclear_attraction_noalloc(const te_pairs *p, int ncharge, const double *xyzq_dev, double *V_dev, void *cuda_stream);
/* Kernel family used by the builds on this handle: 2 (default) = the measured per-class choice; 0 = generic
 * thread-per-quartet kernel for every class, 1 = uniform-ket warp kernel wherever it exists, 3 = split-quartet kernel
 * wherever it exists.  Every family computes the same J and K (tests hold each to the parity bar). */
int te_jk_set_kernel_family(te_pairs *p, int family);
/* Enable (1) / disable (0) per-class CUDA-event timing for te_jk_stats (off by default). */
int te_jk_set_profiling(te_pairs *p, int on);

/* Contracted, normalised integral blocks for testing (eq. 30).  quartets[n][4] HOST shell ids (A,B,C,D);
 * out_offsets[n+1] HOST; out_dev DEVICE with out_offsets[n] doubles:
 *   out_dev[out_offsets[q] + ((i*nB + j)*nC + k)*nD + l] = (A_i B_j | C_k D_l).  No screening. */
int te_eri_block(const te_basis *b, int nquartets, const int *quartets, const long long *out_offsets,
                 double *out_dev);

/* Boys function F_0..F_mmax(T) (eq. 18) evaluated by the device routine the kernels use
 * (tabulated Taylor expansion + downward recursion; asymptotic form + upward recursion for large T).
 * T_dev[n] DEVICE in; F_dev[n][mmax+1] DEVICE out; mmax <= 12. */
int te_boys(int n, const double *T_dev, int mmax, double *F_dev);

/* Sustained FP64 FMA throughput of the device (register-resident DFMA chains), in TFLOP/s: the measured
 * denominator of the "alu" roofline. */
int te_measure_fp64_peak(double *tflops);

/* FP64 rate, in TFLOP/s, of a loop that feeds every DFMA with one lane-private 8-byte shared-memory load (the operand pattern
 * of the Hermite -> Cartesian transform of the uniform-ket kernel: R in a conflict-free shared-memory column), with
 * `warps_per_sm` (1..32) one-warp blocks resident per SM: the shared-memory ceiling of that transform. */
int te_measure_smem_dfma_rate(int warps_per_sm, double *tflops);

const char *te_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* TE_JK_H */
