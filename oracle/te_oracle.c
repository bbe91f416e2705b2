/*
 * te_oracle.c -- TEST INFRASTRUCTURE ONLY.  Plain, slow, CPU FP64 oracle for the direct-SCF J/K Fock
 * build of arXiv 2406.14920.  It shares NO code with the CUDA product path
 * (paper_2406_14920_b200/csrc): only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may load it.  Compile: gcc -O2 -fopenmp -ffp-contract=off -fno-fast-math.
 *
 * Every function cites the passage of PAPER.md ("P:line", equation) it transcribes.  McMurchie-Davidson
 * scheme exactly as printed: E coefficients by eq. 5-8, Boys function eq. 18, auxiliary integrals R by
 * eq. 21-25, four-centre integral by eq. 30 in the bracketing of eq. 31, J by eq. 34, K by eq. 36,
 * Schwarz bound eq. 45, per-term screening eq. 47.  Readings of garbled / silent places: DESIGN.md section 3.
 *
 * Pins (tests/test_oracle_*.py): Boys vs scipy/mpmath incomplete gamma; unit self-overlap; closed-form
 * (ss|ss) eq. 28; brute-force Gauss-Hermite/Legendre quadrature of primitive integrals for every l;
 * 8-fold symmetry eq. 46; Schwarz inequality; translation / rotation invariance of Tr(DJ), Tr(DK);
 * O2 (symmetry-unique loops) == O1 (definition); Schwarz bound eq. 45 against its definition written out in
 * numpy and the (ss|ss) closed form; density bounds against a numpy block maximum; the per-term rule against a
 * numpy transcription on a tiny basis; long-range integrals eq. 33 against the attenuated (ss|ss) closed form,
 * the omega -> infinity limit and quadrature of eq. 32; nuclear attraction eq. 26 against eq. 17, 1-D
 * quadrature and the tight-s-charge limit of the (pinned) ERI code.  "parity unpinned": only the SIZE of the
 * screening error (no bound is printed in the paper); it is measured, not asserted.
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define NL 4            /* l = 0..3 */
#define NT 7            /* t = 0..6 per pair */
#define NR 13           /* t+t' = 0..12 */
#define PI 3.14159265358979323846

/* ------------------------------------------------------------------------------------------ helpers */
static int ncart(int l) { return (l + 1) * (l + 2) / 2; }

/* Cartesian components in lexicographic order, x^l first (reading 4):
   p = x,y,z; d = xx,xy,xz,yy,yz,zz; f = xxx,xxy,xxz,xyy,xyz,xzz,yyy,yyz,yzz,zzz */
static void cart_comp(int l, int idx, int c[3]) {
    int n = 0;
    c[0] = c[1] = c[2] = 0;
    for (int ix = l; ix >= 0; --ix)
        for (int iy = l - ix; iy >= 0; --iy) {
            if (n == idx) { c[0] = ix; c[1] = iy; c[2] = l - ix - iy; return; }
            ++n;
        }
}

/* n!! with (-1)!! = 0!! = 1 */
static double dfact(int n) { double r = 1.0; for (; n > 1; n -= 2) r *= n; return r; }

/* ------------------------------------------------------------------------------------- Boys function
 * F_m(T) = int_0^1 t^{2m} exp(-T t^2) dt  (eq. 18).  The paper only says "interpolation and
 * downward recursion"; the oracle uses textbook closed forms instead (reading 5):
 *   T < 25 : convergent series at m = mmax,
 *            F_m(T) = exp(-T) sum_k (2T)^k / [(2m+1)(2m+3)...(2m+2k+1)],
 *            then downward  F_{m-1} = (2T F_m + exp(-T)) / (2m-1);
 *   T >= 25: F_0 = (1/2) sqrt(pi/T) erf(sqrt T), then upward F_{m+1} = ((2m+1) F_m - exp(-T)) / (2T).
 */
void orc_boys(int mmax, double T, double *F) {
    double eT = exp(-T);
    if (T < 25.0) {
        double term = 1.0 / (2 * mmax + 1), sum = term;
        for (int k = 1; k < 400; ++k) {
            term *= 2.0 * T / (2 * mmax + 2 * k + 1);
            sum += term;
            if (term < 1e-18 * sum) break;
        }
        F[mmax] = eT * sum;
        for (int m = mmax; m > 0; --m) F[m - 1] = (2.0 * T * F[m] + eT) / (2 * m - 1);
    } else {
        F[0] = 0.5 * sqrt(PI / T) * erf(sqrt(T));
        for (int m = 0; m < mmax; ++m) F[m + 1] = ((2 * m + 1) * F[m] - eT) / (2.0 * T);
    }
}

/* ---------------------------------------------------------------------------------------- the basis */
typedef struct {
    int shell;       /* contracted shell id */
    int iprim;       /* index within the shell */
    int l;
    double a;        /* exponent */
    double ct;       /* c~ = raw coefficient x radial normalisation / sqrt(self overlap)  (step 1) */
    double A[3];
} OPrim;

typedef struct {
    int m, n;        /* global primitive-shell indices, (l_m, m) <= (l_n, n) lexicographically */
    int cls;         /* 0..9: SS SP SD SF PP PD PF DD DF FF */
    double p, P[3];  /* eq. 3 */
    double cc;       /* c~_m c~_n */
    double Kab;      /* exp(-ab/p |A-B|^2) */
    double q;        /* Schwarz bound, eq. 45 */
    double *E;       /* E[dim][i][j][t], i<=la, j<=lb, t<=la+lb (eq. 5-8), includes eq. 7 prefactor per dim */
} OPair;

typedef struct {
    int natoms, nshells, nprim, nbf;
    int *shell_l, *shell_off, *shell_pstart, *shell_nprim;
    OPrim *prim;
    long npairs;     /* kept, canonical (unordered) */
    OPair *pairs;
    double compf[NL][10];  /* per-component normalisation factor f(i) (step 1) */
    double omega;          /* 0: full-range 1/r (eq. 30); > 0: long-range erf(omega r)/r (eq. 32-33) in the J/K builds */
} OrcCtx;

/* Step 1 (eq. 1-2; north_star "unit self-overlap"; reading 3).
   N(a,l) = (2a/pi)^{3/4} (4a)^{l/2} / sqrt((2l-1)!!) normalises the x^l primitive;
   S = sum_mn c_m N_m c_n N_n (pi/p)^{3/2} (2l-1)!! / (2p)^l is the x^l self overlap (eq. 11);
   c~_m = c_m N_m / sqrt(S).  f(i) = sqrt((2l-1)!! / ((2ix-1)!!(2iy-1)!!(2iz-1)!!)). */
static void normalise_shell(int l, int np, const double *ex, const double *co, double *ct) {
    double S = 0.0;
    for (int m = 0; m < np; ++m) ct[m] = co[m] * pow(2.0 * ex[m] / PI, 0.75) * pow(4.0 * ex[m], 0.5 * l) / sqrt(dfact(2 * l - 1));
    for (int m = 0; m < np; ++m)
        for (int n = 0; n < np; ++n) {
            double p = ex[m] + ex[n];
            S += ct[m] * ct[n] * pow(PI / p, 1.5) * dfact(2 * l - 1) / pow(2.0 * p, (double)l);
        }
    for (int m = 0; m < np; ++m) ct[m] /= sqrt(S);
}

OrcCtx *orc_create(int natoms, const double *xyz, int nshells, const int *shell_atom, const int *shell_l,
                   const int *shell_nprim, const double *ex, const double *co) {
    OrcCtx *c = (OrcCtx *)calloc(1, sizeof(OrcCtx));
    c->natoms = natoms; c->nshells = nshells;
    c->shell_l = (int *)malloc(sizeof(int) * nshells);
    c->shell_off = (int *)malloc(sizeof(int) * (nshells + 1));
    c->shell_pstart = (int *)malloc(sizeof(int) * (nshells + 1));
    c->shell_nprim = (int *)malloc(sizeof(int) * nshells);
    int np = 0, nbf = 0;
    for (int s = 0; s < nshells; ++s) {
        if (shell_l[s] < 0 || shell_l[s] >= NL || shell_nprim[s] < 1) { free(c); return NULL; }
        c->shell_l[s] = shell_l[s]; c->shell_off[s] = nbf; c->shell_pstart[s] = np; c->shell_nprim[s] = shell_nprim[s];
        nbf += ncart(shell_l[s]); np += shell_nprim[s];
    }
    c->shell_off[nshells] = nbf; c->shell_pstart[nshells] = np; c->nbf = nbf; c->nprim = np;
    c->prim = (OPrim *)malloc(sizeof(OPrim) * np);
    double ct[64];
    for (int s = 0; s < nshells; ++s) {
        int p0 = c->shell_pstart[s];
        normalise_shell(shell_l[s], shell_nprim[s], ex + p0, co + p0, ct);
        for (int k = 0; k < shell_nprim[s]; ++k) {
            OPrim *pr = &c->prim[p0 + k];
            pr->shell = s; pr->iprim = k; pr->l = shell_l[s]; pr->a = ex[p0 + k]; pr->ct = ct[k];
            for (int d = 0; d < 3; ++d) pr->A[d] = xyz[3 * shell_atom[s] + d];
        }
    }
    for (int l = 0; l < NL; ++l)
        for (int i = 0; i < ncart(l); ++i) {
            int ci[3]; cart_comp(l, i, ci);
            c->compf[l][i] = sqrt(dfact(2 * l - 1) / (dfact(2 * ci[0] - 1) * dfact(2 * ci[1] - 1) * dfact(2 * ci[2] - 1)));
        }
    return c;
}

static void free_pairs(OrcCtx *c) {
    for (long i = 0; i < c->npairs; ++i) free(c->pairs[i].E);
    free(c->pairs); c->pairs = NULL; c->npairs = 0;
}

void orc_destroy(OrcCtx *c) {
    if (!c) return;
    free_pairs(c);
    free(c->shell_l); free(c->shell_off); free(c->shell_pstart); free(c->shell_nprim); free(c->prim); free(c);
}

int orc_nbf(const OrcCtx *c) { return c->nbf; }
int orc_nprim(const OrcCtx *c) { return c->nprim; }
void orc_norm_coefs(const OrcCtx *c, double *ct) { for (int i = 0; i < c->nprim; ++i) ct[i] = c->prim[i].ct; }

/* ------------------------------------------------------------------------ E coefficients (eq. 5-8)
 * One Cartesian dimension.  E^{00}_0 = exp(-ab/p (A-B)^2) (eq. 7); raise i with eq. 5, j with
 * eq. 6; zero outside 0 <= t <= i+j (eq. 8).  Table layout E[i][j][t] with dims (la+1,lb+1,la+lb+1). */
static void e_table_1d(int la, int lb, double a, double b, double A, double B, double *E) {
    const int nt = la + lb + 1, nj = lb + 1;
    const double p = a + b, P = (a * A + b * B) / p, PA = P - A, PB = P - B, h = 1.0 / (2.0 * p);
#define EE(i, j, t) E[((i) * nj + (j)) * nt + (t)]
    for (int k = 0; k < (la + 1) * nj * nt; ++k) E[k] = 0.0;
    EE(0, 0, 0) = exp(-a * b / p * (A - B) * (A - B));
    for (int i = 0; i < la; ++i)            /* eq. 5 at j = 0 */
        for (int t = 0; t <= i + 1; ++t) {
            double v = PA * EE(i, 0, t);
            if (t > 0) v += h * EE(i, 0, t - 1);
            if (t + 1 <= i) v += (t + 1) * EE(i, 0, t + 1);
            EE(i + 1, 0, t) = v;
        }
    for (int i = 0; i <= la; ++i)           /* eq. 6 */
        for (int j = 0; j < lb; ++j)
            for (int t = 0; t <= i + j + 1; ++t) {
                double v = PB * EE(i, j, t);
                if (t > 0) v += h * EE(i, j, t - 1);
                if (t + 1 <= i + j) v += (t + 1) * EE(i, j, t + 1);
                EE(i, j + 1, t) = v;
            }
#undef EE
}

static int class_of(int la, int lb) {   /* la <= lb */
    static const int base[NL] = {0, 4, 7, 9};
    return base[la] + (lb - la);
}

/* Pair quantities (eq. 3) for the ORDERED primitive pair (m,n). */
static void make_pair(const OrcCtx *c, int m, int n, OPair *pr) {
    const OPrim *pm = &c->prim[m], *pn = &c->prim[n];
    const int la = pm->l, lb = pn->l;
    pr->m = m; pr->n = n;
    pr->cls = la <= lb ? class_of(la, lb) : class_of(lb, la);
    pr->p = pm->a + pn->a;
    double r2 = 0.0;
    for (int d = 0; d < 3; ++d) {
        pr->P[d] = (pm->a * pm->A[d] + pn->a * pn->A[d]) / pr->p;
        r2 += (pm->A[d] - pn->A[d]) * (pm->A[d] - pn->A[d]);
    }
    pr->cc = pm->ct * pn->ct;
    pr->Kab = exp(-pm->a * pn->a / pr->p * r2);
    pr->q = 0.0;
    const int sz = (la + 1) * (lb + 1) * (la + lb + 1);
    pr->E = (double *)malloc(sizeof(double) * 3 * sz);
    for (int d = 0; d < 3; ++d) e_table_1d(la, lb, pm->a, pn->a, pm->A[d], pn->A[d], pr->E + d * sz);
}

/* ----------------------------------------------------------------- R^m_{tuv} (eq. 20-25)
 * R^m_{000} = (-2 alpha)^m F_m(alpha |L|^2) (eq. 24); lower the first non-zero index with eq. 21/22/23;
 * negative index -> 0 (eq. 25).  Plain 4-index array, no in-place tricks. */
typedef double RTab[NR][NR][NR][NR];   /* [m][t][u][v] */

static void r_table(int L, double alpha, const double X[3], RTab *Rp) {
    double F[NR];
    const double T = alpha * (X[0] * X[0] + X[1] * X[1] + X[2] * X[2]);
    orc_boys(L, T, F);
#define RR(m, t, u, v) (*Rp)[m][t][u][v]
    double f = 1.0;
    for (int m = 0; m <= L; ++m) { RR(m, 0, 0, 0) = f * F[m]; f *= -2.0 * alpha; }
    for (int n = 1; n <= L; ++n)
        for (int m = 0; m <= L - n; ++m)
            for (int t = 0; t <= n; ++t)
                for (int u = 0; u <= n - t; ++u) {
                    int v = n - t - u;
                    double r;
                    if (t > 0)      r = (t > 1 ? (t - 1) * RR(m + 1, t - 2, u, v) : 0.0) + X[0] * RR(m + 1, t - 1, u, v);
                    else if (u > 0) r = (u > 1 ? (u - 1) * RR(m + 1, t, u - 2, v) : 0.0) + X[1] * RR(m + 1, t, u - 1, v);
                    else            r = (v > 1 ? (v - 1) * RR(m + 1, t, u, v - 2) : 0.0) + X[2] * RR(m + 1, t, u, v - 1);
                    RR(m, t, u, v) = r;
                }
#undef RR
}

/* --------------------------------------------------- primitive shell-quartet block (eq. 30 / eq. 31)
 * out[((i*nB + j)*nC + k)*nD + l] = (m_i n_j | r_k s_l), all coefficient factors included
 * (C_mu of P:51 = c~ x f(i)).  Bracketing of eq. 31: inner_P = sum_Q E_Q^{kl} (-1)^Q R_{P+Q},
 * then sum_P E_P^{ij} inner_P; the prefactor 2 pi^{5/2} / (p q sqrt(p+q)) of eq. 30.
 * Ket E's take the ket exponent q (eq. 29; reading 2).
 *
 * Long-range operator erf(omega r)/r (eq. 32-33): identical sums; only the argument of the
 * auxiliary integrals, alpha -> p q omega^2 / (p q + (p + q) omega^2), and the prefactor,
 * 2 pi^{5/2} omega / (p q sqrt(p q + (p + q) omega^2)), change.  omega <= 0 selects the full-range eq. 30. */
static void prim_block_op(const OrcCtx *c, const OPair *bra, const OPair *ket, double omega, double *out) {
    const int la = c->prim[bra->m].l, lb = c->prim[bra->n].l, lc = c->prim[ket->m].l, ld = c->prim[ket->n].l;
    const int nA = ncart(la), nB = ncart(lb), nC = ncart(lc), nD = ncart(ld);
    const int Lab = la + lb, Lcd = lc + ld, L = Lab + Lcd;
    const double p = bra->p, q = ket->p;
    double alpha = p * q / (p + q);
    double pref = 2.0 * pow(PI, 2.5) / (p * q * sqrt(p + q)) * bra->cc * ket->cc;
    if (omega > 0.0) {   /* eq. 33 */
        const double den = p * q + p * omega * omega + q * omega * omega;
        alpha = p * q * omega * omega / den;
        pref = 2.0 * pow(PI, 2.5) * omega / (p * q * sqrt(den)) * bra->cc * ket->cc;
    }
    double X[3] = {bra->P[0] - ket->P[0], bra->P[1] - ket->P[1], bra->P[2] - ket->P[2]};
    static __thread RTab Rbuf;
    RTab *Rp = &Rbuf;
    r_table(L, alpha, X, Rp);
    const int szb = (la + 1) * (lb + 1) * (Lab + 1), szk = (lc + 1) * (ld + 1) * (Lcd + 1);
#define EB(d, i, j, t) bra->E[(d) * szb + (((i) * (lb + 1) + (j)) * (Lab + 1)) + (t)]
#define EK(d, i, j, t) ket->E[(d) * szk + (((i) * (ld + 1) + (j)) * (Lcd + 1)) + (t)]
    double inner[NT][NT][NT];
    for (int k = 0; k < nC; ++k) {
        int ck[3]; cart_comp(lc, k, ck);
        for (int l = 0; l < nD; ++l) {
            int cl[3]; cart_comp(ld, l, cl);
            for (int t = 0; t <= Lab; ++t)
                for (int u = 0; u <= Lab - t; ++u)
                    for (int v = 0; v <= Lab - t - u; ++v) {
                        double s = 0.0;
                        for (int t2 = 0; t2 <= ck[0] + cl[0]; ++t2)
                            for (int u2 = 0; u2 <= ck[1] + cl[1]; ++u2)
                                for (int v2 = 0; v2 <= ck[2] + cl[2]; ++v2) {
                                    double e = EK(0, ck[0], cl[0], t2) * EK(1, ck[1], cl[1], u2) * EK(2, ck[2], cl[2], v2);
                                    double sg = ((t2 + u2 + v2) & 1) ? -1.0 : 1.0;
                                    s += sg * e * (*Rp)[0][t + t2][u + u2][v + v2];
                                }
                        inner[t][u][v] = s;
                    }
            for (int i = 0; i < nA; ++i) {
                int ci[3]; cart_comp(la, i, ci);
                for (int j = 0; j < nB; ++j) {
                    int cj[3]; cart_comp(lb, j, cj);
                    double s = 0.0;
                    for (int t = 0; t <= ci[0] + cj[0]; ++t)
                        for (int u = 0; u <= ci[1] + cj[1]; ++u)
                            for (int v = 0; v <= ci[2] + cj[2]; ++v)
                                s += EB(0, ci[0], cj[0], t) * EB(1, ci[1], cj[1], u) * EB(2, ci[2], cj[2], v) * inner[t][u][v];
                    out[((i * nB + j) * nC + k) * nD + l] =
                        pref * c->compf[la][i] * c->compf[lb][j] * c->compf[lc][k] * c->compf[ld][l] * s;
                }
            }
        }
    }
#undef EB
#undef EK
}

/* Full-range block (eq. 30): what the Schwarz bounds, the pair lists and the integral-block checks use. */
static void prim_block(const OrcCtx *c, const OPair *bra, const OPair *ket, double *out) { prim_block_op(c, bra, ket, 0.0, out); }

/* Operator used by the J/K builds (orc_jk_o1 / orc_jk_o2): 0 = 1/r (default), omega > 0 = erf(omega r)/r.
   Pair lists and Schwarz bounds stay those of the full-range operator (reading 20). */
void orc_set_omega(OrcCtx *c, double omega) { c->omega = omega > 0.0 ? omega : 0.0; }

/* Raw primitive integral block for pins: unit coefficients (C = 1), arbitrary centres / exponents;
   omega <= 0: eq. 30, omega > 0: eq. 33. */
void orc_prim_eri_raw_lr(int la, double a, const double *A, int lb, double b, const double *B,
                         int lc, double cexp, const double *C, int ld, double d, const double *Dc, double omega, double *out) {
    OrcCtx ctx; memset(&ctx, 0, sizeof(ctx));
    OPrim pr[4];
    const int ls[4] = {la, lb, lc, ld}; const double es[4] = {a, b, cexp, d}; const double *cs[4] = {A, B, C, Dc};
    for (int k = 0; k < 4; ++k) { pr[k].shell = k; pr[k].iprim = 0; pr[k].l = ls[k]; pr[k].a = es[k]; pr[k].ct = 1.0; for (int x = 0; x < 3; ++x) pr[k].A[x] = cs[k][x]; }
    ctx.prim = pr; ctx.nprim = 4;
    for (int l = 0; l < NL; ++l) for (int i = 0; i < 10; ++i) ctx.compf[l][i] = 1.0;
    OPair bra, ket; make_pair(&ctx, 0, 1, &bra); make_pair(&ctx, 2, 3, &ket);
    prim_block_op(&ctx, &bra, &ket, omega, out);
    free(bra.E); free(ket.E);
}

void orc_prim_eri_raw(int la, double a, const double *A, int lb, double b, const double *B,
                      int lc, double cexp, const double *C, int ld, double d, const double *Dc, double *out) {
    orc_prim_eri_raw_lr(la, a, A, lb, b, B, lc, cexp, C, ld, d, Dc, 0.0, out);
}

/* Overlap block of two contracted shells by eq. 11: S = C C E0x E0y E0z (pi/p)^{3/2}. */
void orc_overlap_shell(const OrcCtx *c, int A, int B, double *out) {
    const int la = c->shell_l[A], lb = c->shell_l[B], nA = ncart(la), nB = ncart(lb);
    for (int k = 0; k < nA * nB; ++k) out[k] = 0.0;
    for (int m = c->shell_pstart[A]; m < c->shell_pstart[A + 1]; ++m)
        for (int n = c->shell_pstart[B]; n < c->shell_pstart[B + 1]; ++n) {
            OPair pr; make_pair(c, m, n, &pr);
            const int sz = (la + 1) * (lb + 1) * (la + lb + 1);
            for (int i = 0; i < nA; ++i) {
                int ci[3]; cart_comp(la, i, ci);
                for (int j = 0; j < nB; ++j) {
                    int cj[3]; cart_comp(lb, j, cj);
                    double e = 1.0;
                    for (int d = 0; d < 3; ++d) e *= pr.E[d * sz + ((ci[d] * (lb + 1) + cj[d]) * (la + lb + 1))];
                    out[i * nB + j] += pr.cc * c->compf[la][i] * c->compf[lb][j] * e * pow(PI / pr.p, 1.5);
                }
            }
            free(pr.E);
        }
}

/* --------------------------------------------------- Schwarz bound of a primitive shell pair (eq. 45)
 * q_mn = max over components (i in m, j in n) of sqrt|(m_i n_j | m_i n_j)| (reading 7). */
static double schwarz_bound(const OrcCtx *c, const OPair *pr) {
    const int la = c->prim[pr->m].l, lb = c->prim[pr->n].l, nA = ncart(la), nB = ncart(lb);
    double *blk = (double *)malloc(sizeof(double) * nA * nB * nA * nB);
    prim_block(c, pr, pr, blk);
    double q = 0.0;
    for (int i = 0; i < nA; ++i)
        for (int j = 0; j < nB; ++j) {
            double v = sqrt(fabs(blk[((i * nB + j) * nA + i) * nB + j]));
            if (v > q) q = v;
        }
    free(blk);
    return q;
}

/* Canonical order of an unordered primitive pair: (l, index) of the first <= that of the second. */
static int canon_first(const OrcCtx *c, int m, int n) {
    if (c->prim[m].l != c->prim[n].l) return c->prim[m].l < c->prim[n].l;
    return m <= n;
}

/* Steps 7-8: all unordered primitive shell pairs, bound, keep q >= tau_pair.
   Kept list is in ascending canonical order (class, m, n).  Returns the number kept. */
long orc_build_pairs(OrcCtx *c, double tau_pair) {
    free_pairs(c);
    const long np = c->nprim, ncand = np * (np + 1) / 2;
    OPair *all = (OPair *)malloc(sizeof(OPair) * ncand);
    char *keep = (char *)calloc(ncand, 1);
#pragma omp parallel for schedule(dynamic, 64)
    for (long idx = 0; idx < ncand; ++idx) {
        /* idx -> (hi, lo), hi >= lo */
        long hi = (long)((sqrt(8.0 * (double)idx + 1.0) - 1.0) / 2.0);
        while (hi * (hi + 1) / 2 > idx) --hi;
        while ((hi + 1) * (hi + 2) / 2 <= idx) ++hi;
        long lo = idx - hi * (hi + 1) / 2;
        int m = (int)lo, n = (int)hi;
        if (!canon_first(c, m, n)) { int t = m; m = n; n = t; }
        OPair pr; make_pair(c, m, n, &pr);
        pr.q = schwarz_bound(c, &pr);
        if (pr.q >= tau_pair) { all[idx] = pr; keep[idx] = 1; } else free(pr.E);
    }
    long nk = 0;
    for (long i = 0; i < ncand; ++i) nk += keep[i];
    c->pairs = (OPair *)malloc(sizeof(OPair) * (nk > 0 ? nk : 1));
    long k = 0;
    for (int cls = 0; cls < 10; ++cls)          /* ascending (class, m, n) */
        for (int m = 0; m < np; ++m)
            for (int n = 0; n < np; ++n) {
                if (!canon_first(c, m, n)) continue;
                long hi = m > n ? m : n, lo = m > n ? n : m;
                long idx = hi * (hi + 1) / 2 + lo;
                if (keep[idx] && all[idx].cls == cls && all[idx].m == m && all[idx].n == n) c->pairs[k++] = all[idx];
            }
    c->npairs = k;
    free(all); free(keep);
    return k;
}

void orc_get_pairs(const OrcCtx *c, int *cls, int *shA, int *shB, int *pA, int *pB, double *q,
                   double *Pxyz, double *p, double *pref) {
    for (long i = 0; i < c->npairs; ++i) {
        const OPair *pr = &c->pairs[i];
        cls[i] = pr->cls; shA[i] = c->prim[pr->m].shell; shB[i] = c->prim[pr->n].shell;
        pA[i] = c->prim[pr->m].iprim; pB[i] = c->prim[pr->n].iprim; q[i] = pr->q;
        for (int d = 0; d < 3; ++d) Pxyz[3 * i + d] = pr->P[d];
        p[i] = pr->p; pref[i] = pr->cc * pr->Kab;
    }
}

/* Schwarz bounds of ALL candidate pairs (for the guard band of DESIGN.md reading 10): q[hi*(hi+1)/2+lo]. */
void orc_all_bounds(const OrcCtx *c, double *qall) {
    const long np = c->nprim, ncand = np * (np + 1) / 2;
#pragma omp parallel for schedule(dynamic, 64)
    for (long idx = 0; idx < ncand; ++idx) {
        long hi = (long)((sqrt(8.0 * (double)idx + 1.0) - 1.0) / 2.0);
        while (hi * (hi + 1) / 2 > idx) --hi;
        while ((hi + 1) * (hi + 2) / 2 <= idx) ++hi;
        long lo = idx - hi * (hi + 1) / 2;
        int m = (int)lo, n = (int)hi;
        if (!canon_first(c, m, n)) { int t = m; m = n; n = t; }
        OPair pr; make_pair(c, m, n, &pr);
        qall[idx] = schwarz_bound(c, &pr);
        free(pr.E);
    }
}

/* ---------------------------------------------------------------------------- density bounds
 * Dm[X][Y] = max |D| over the block of contracted shells (X,Y): "max absolute value of the set". */
static double *density_bounds(const OrcCtx *c, const double *D) {
    const int ns = c->nshells, nbf = c->nbf;
    double *Dm = (double *)malloc(sizeof(double) * ns * ns);
    for (int X = 0; X < ns; ++X)
        for (int Y = 0; Y < ns; ++Y) {
            double mx = 0.0;
            for (int i = c->shell_off[X]; i < c->shell_off[X + 1]; ++i)
                for (int j = c->shell_off[Y]; j < c->shell_off[Y + 1]; ++j) {
                    double v = fabs(D[(long)i * nbf + j]);
                    if (v > mx) mx = v;
                }
            Dm[X * ns + Y] = mx;
        }
    return Dm;
}

void orc_density_bounds(const OrcCtx *c, const double *D, double *Dm_out) {
    double *Dm = density_bounds(c, D);
    memcpy(Dm_out, Dm, sizeof(double) * (size_t)c->nshells * c->nshells);
    free(Dm);
}

/* ------------------------------------------------------------------- O1: J and K from the definition
 * Eq. 34 and eq. 36 over ORDERED primitive pairs of the kept set, no permutational
 * symmetry, with the per-term rule of eq. 47 (readings 6, 8):
 *   J[A_i,B_j] += [m_i n_j|r_k s_l] D[C_k,D_l]  iff  q_mn q_rs Dm[C,D] >= tau
 *   K[A_i,C_k] += [m_i n_j|r_k s_l] D[B_j,D_l]  iff  q_mn q_rs Dm[B,D] >= tau
 * braA/braB/ketC restrict the loops to blocks (negative = no restriction): used for sampled blocks. */
static void ordered_pairs(const OrcCtx *c, OPair **out, long *nout) {
    long n = 0;
    for (long i = 0; i < c->npairs; ++i) n += (c->pairs[i].m == c->pairs[i].n) ? 1 : 2;
    OPair *o = (OPair *)malloc(sizeof(OPair) * (n > 0 ? n : 1));
    long k = 0;
    for (long i = 0; i < c->npairs; ++i) {
        const OPair *pr = &c->pairs[i];
        make_pair(c, pr->m, pr->n, &o[k]); o[k].q = pr->q; ++k;
        if (pr->m != pr->n) { make_pair(c, pr->n, pr->m, &o[k]); o[k].q = pr->q; ++k; }
    }
    *out = o; *nout = n;
}

void orc_jk_o1(const OrcCtx *c, const double *D, double tau, double *J, double *K,
               int doJ, int doK, int braA, int braB, int ketC) {
    const int nbf = c->nbf, ns = c->nshells;
    double *Dm = density_bounds(c, D);
    OPair *op; long nop; ordered_pairs(c, &op, &nop);
    memset(J, 0, sizeof(double) * (size_t)nbf * nbf);
    memset(K, 0, sizeof(double) * (size_t)nbf * nbf);
#pragma omp parallel
    {
        double *blk = (double *)malloc(sizeof(double) * 10000);
        double *Jt = (double *)calloc((size_t)nbf * nbf, sizeof(double));
        double *Kt = (double *)calloc((size_t)nbf * nbf, sizeof(double));
#pragma omp for schedule(dynamic, 1)
        for (long I = 0; I < nop; ++I) {
            const OPair *bra = &op[I];
            const OPrim *pm = &c->prim[bra->m], *pn = &c->prim[bra->n];
            const int A = pm->shell, B = pn->shell;
            if (braA >= 0 && A != braA) continue;
            if (braB >= 0 && B != braB) continue;
            const int nA = ncart(pm->l), nB = ncart(pn->l), oA = c->shell_off[A], oB = c->shell_off[B];
            for (long Jx = 0; Jx < nop; ++Jx) {
                const OPair *ket = &op[Jx];
                const OPrim *pr = &c->prim[ket->m], *ps = &c->prim[ket->n];
                const int C = pr->shell, Dd = ps->shell;
                if (ketC >= 0 && C != ketC) continue;
                const double qq = bra->q * ket->q;
                const int liveJ = doJ && (qq * Dm[C * ns + Dd] >= tau);
                const int liveK = doK && (qq * Dm[B * ns + Dd] >= tau);
                if (!liveJ && !liveK) continue;
                const int nC = ncart(pr->l), nD = ncart(ps->l), oC = c->shell_off[C], oD = c->shell_off[Dd];
                prim_block_op(c, bra, ket, c->omega, blk);
                for (int i = 0; i < nA; ++i)
                    for (int j = 0; j < nB; ++j)
                        for (int k = 0; k < nC; ++k)
                            for (int l = 0; l < nD; ++l) {
                                const double v = blk[((i * nB + j) * nC + k) * nD + l];
                                if (liveJ) Jt[(long)(oA + i) * nbf + oB + j] += v * D[(long)(oC + k) * nbf + oD + l];
                                if (liveK) Kt[(long)(oA + i) * nbf + oC + k] += v * D[(long)(oB + j) * nbf + oD + l];
                            }
            }
        }
#pragma omp critical
        {
            for (long x = 0; x < (long)nbf * nbf; ++x) { J[x] += Jt[x]; K[x] += Kt[x]; }
        }
        free(blk); free(Jt); free(Kt);
    }
    for (long i = 0; i < nop; ++i) free(op[i].E);
    free(op); free(Dm);
}

/* ------------------------------------------------ O2: symmetry-unique primitive quartets (eq. 46)
 * Unique quartets I >= Jx over the kept (unordered) pair list; degeneracy factor f = 1/2 per
 * coincidence m==n, r==s, I==Jx ("halve the diagonal"); six independently masked updates
 * (reading 8), then J = Jt + Jt^T, K = Kt + Kt^T.
 * stats[0] = unique quartets with >= 1 live update, stats[1] = unique quartets visited,
 * stats[2] = decisions whose bound product is within 1e-9 relative of tau (reading 10). */
void orc_jk_o2(const OrcCtx *c, const double *D, double tau, double *J, double *K, long long *stats) {
    const int nbf = c->nbf, ns = c->nshells;
    const long npairs = c->npairs;
    double *Dm = density_bounds(c, D);
    int nth = 1;
#ifdef _OPENMP
    nth = omp_get_max_threads();
#endif
    double **Jt = (double **)calloc(nth, sizeof(double *)), **Kt = (double **)calloc(nth, sizeof(double *));   /* NULL = thread never ran */
    long long nlive = 0, nvis = 0, nborder = 0;
#pragma omp parallel reduction(+ : nlive, nvis, nborder)
    {
        int tid = 0;
#ifdef _OPENMP
        tid = omp_get_thread_num();
#endif
        double *blk = (double *)malloc(sizeof(double) * 10000);
        double *Jp = Jt[tid] = (double *)calloc((size_t)nbf * nbf, sizeof(double));
        double *Kp = Kt[tid] = (double *)calloc((size_t)nbf * nbf, sizeof(double));
#pragma omp for schedule(dynamic, 1)
        for (long Ir = 0; Ir < npairs; ++Ir) {
            const long I = npairs - 1 - Ir;     /* long rows first */
            const OPair *bra = &c->pairs[I];
            const OPrim *pm = &c->prim[bra->m], *pn = &c->prim[bra->n];
            const int A = pm->shell, B = pn->shell, nA = ncart(pm->l), nB = ncart(pn->l);
            const int oA = c->shell_off[A], oB = c->shell_off[B];
            for (long Jx = 0; Jx <= I; ++Jx) {
                const OPair *ket = &c->pairs[Jx];
                const OPrim *pr = &c->prim[ket->m], *ps = &c->prim[ket->n];
                const int C = pr->shell, Dd = ps->shell;
                const double qq = bra->q * ket->q;
                const double b[6] = {qq * Dm[C * ns + Dd], qq * Dm[A * ns + B], qq * Dm[B * ns + Dd],
                                     qq * Dm[A * ns + Dd], qq * Dm[B * ns + C], qq * Dm[A * ns + C]};
                int live[6], any = 0;
                for (int x = 0; x < 6; ++x) {
                    live[x] = b[x] >= tau; any |= live[x];
                    if (tau > 0.0 && fabs(b[x] - tau) <= 1e-9 * tau) ++nborder;
                }
                ++nvis;
                if (!any) continue;
                ++nlive;
                const int nC = ncart(pr->l), nD = ncart(ps->l), oC = c->shell_off[C], oD = c->shell_off[Dd];
                prim_block_op(c, bra, ket, c->omega, blk);
                double f = 1.0;
                if (bra->m == bra->n) f *= 0.5;
                if (ket->m == ket->n) f *= 0.5;
                if (I == Jx) f *= 0.5;
                for (int i = 0; i < nA; ++i)
                    for (int j = 0; j < nB; ++j)
                        for (int k = 0; k < nC; ++k)
                            for (int l = 0; l < nD; ++l) {
                                const double v = f * blk[((i * nB + j) * nC + k) * nD + l];
                                const long ai = oA + i, bj = oB + j, ck = oC + k, dl = oD + l;
                                if (live[0]) Jp[ai * nbf + bj] += 2.0 * v * D[ck * nbf + dl];
                                if (live[1]) Jp[ck * nbf + dl] += 2.0 * v * D[ai * nbf + bj];
                                if (live[2]) Kp[ai * nbf + ck] += v * D[bj * nbf + dl];
                                if (live[3]) Kp[bj * nbf + ck] += v * D[ai * nbf + dl];
                                if (live[4]) Kp[ai * nbf + dl] += v * D[bj * nbf + ck];
                                if (live[5]) Kp[bj * nbf + dl] += v * D[ai * nbf + ck];
                            }
            }
        }
        free(blk);
    }
    /* fixed-order reduction over threads, then symmetrise */
    double *Js = (double *)calloc((size_t)nbf * nbf, sizeof(double)), *Ks = (double *)calloc((size_t)nbf * nbf, sizeof(double));
    for (int t = 0; t < nth; ++t) {
        if (!Jt[t]) continue;
        for (long x = 0; x < (long)nbf * nbf; ++x) { Js[x] += Jt[t][x]; Ks[x] += Kt[t][x]; }
        free(Jt[t]); free(Kt[t]);
    }
    for (int i = 0; i < nbf; ++i)
        for (int j = 0; j < nbf; ++j) {
            J[(long)i * nbf + j] = Js[(long)i * nbf + j] + Js[(long)j * nbf + i];
            K[(long)i * nbf + j] = Ks[(long)i * nbf + j] + Ks[(long)j * nbf + i];
        }
    free(Js); free(Ks); free(Jt); free(Kt); free(Dm);
    if (stats) { stats[0] = nlive; stats[1] = nvis; stats[2] = nborder; }
}

/* Contracted shell-quartet integral block (A B | C D), unscreened: sum over all primitives. */
void orc_eri_shell_quartet(const OrcCtx *c, int A, int B, int C, int Dd, double *out) {
    const int n = ncart(c->shell_l[A]) * ncart(c->shell_l[B]) * ncart(c->shell_l[C]) * ncart(c->shell_l[Dd]);
    double *blk = (double *)malloc(sizeof(double) * n);
    for (int x = 0; x < n; ++x) out[x] = 0.0;
    for (int m = c->shell_pstart[A]; m < c->shell_pstart[A + 1]; ++m)
        for (int nn = c->shell_pstart[B]; nn < c->shell_pstart[B + 1]; ++nn) {
            OPair bra; make_pair(c, m, nn, &bra);
            for (int r = c->shell_pstart[C]; r < c->shell_pstart[C + 1]; ++r)
                for (int s = c->shell_pstart[Dd]; s < c->shell_pstart[Dd + 1]; ++s) {
                    OPair ket; make_pair(c, r, s, &ket);
                    prim_block(c, &bra, &ket, blk);
                    for (int x = 0; x < n; ++x) out[x] += blk[x];
                    free(ket.E);
                }
            free(bra.E);
        }
    free(blk);
}

/* ------------------------------------------------------------ nuclear attraction V_mu,nu (eq. 14-26)
 * V_mu,nu = sum_C V_mu,nu,C (eq. 16), V_mu,nu,C = q_C C_mu C_nu (2 pi / p) sum_tuv E_t E_u E_v R^0_tuv(p, P - C)
 * (eq. 26), over the KEPT primitive shell pairs ("one primitive shell pair to one GPU thread ...
 * every thread loop through all point charges"); the operator is + q_C / |r - C| as printed in eq. 14 (a nucleus
 * of charge Z enters with q_C = -Z).  V is nbf x nbf, symmetric, overwritten.  orc_build_pairs must have run. */
void orc_nuclear_attraction(const OrcCtx *c, int ncharge, const double *xyzC, const double *qC, double *V) {
    const int nbf = c->nbf;
    memset(V, 0, sizeof(double) * (size_t)nbf * nbf);
    RTab *Rp = (RTab *)malloc(sizeof(RTab));
    for (long I = 0; I < c->npairs; ++I) {
        const OPair *pr = &c->pairs[I];
        const OPrim *pm = &c->prim[pr->m], *pn = &c->prim[pr->n];
        const int la = pm->l, lb = pn->l, nA = ncart(la), nB = ncart(lb), Lab = la + lb;
        const int oA = c->shell_off[pm->shell], oB = c->shell_off[pn->shell];
        const int szb = (la + 1) * (lb + 1) * (Lab + 1);
        for (int C = 0; C < ncharge; ++C) {
            double X[3] = {pr->P[0] - xyzC[3 * C], pr->P[1] - xyzC[3 * C + 1], pr->P[2] - xyzC[3 * C + 2]};
            r_table(Lab, pr->p, X, Rp);
            for (int i = 0; i < nA; ++i) {
                int ci[3]; cart_comp(la, i, ci);
                for (int j = 0; j < nB; ++j) {
                    int cj[3]; cart_comp(lb, j, cj);
                    double s = 0.0;
                    for (int t = 0; t <= ci[0] + cj[0]; ++t)
                        for (int u = 0; u <= ci[1] + cj[1]; ++u)
                            for (int v = 0; v <= ci[2] + cj[2]; ++v)
                                s += pr->E[0 * szb + ((ci[0] * (lb + 1) + cj[0]) * (Lab + 1)) + t] *
                                     pr->E[1 * szb + ((ci[1] * (lb + 1) + cj[1]) * (Lab + 1)) + u] *
                                     pr->E[2 * szb + ((ci[2] * (lb + 1) + cj[2]) * (Lab + 1)) + v] * (*Rp)[0][t][u][v];
                    const double val = qC[C] * pr->cc * c->compf[la][i] * c->compf[lb][j] * (2.0 * PI / pr->p) * s;
                    V[(long)(oA + i) * nbf + oB + j] += val;
                    /* the unordered pair (m,n), m != n, stands for both ordered pairs: mirror element */
                    if (pr->m != pr->n) V[(long)(oB + j) * nbf + oA + i] += val;
                }
            }
        }
    }
    free(Rp);
}

int orc_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
