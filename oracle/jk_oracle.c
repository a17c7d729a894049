/* ORACLE -- TEST INFRASTRUCTURE ONLY.
 *
 * Plain, slow CPU implementation of what the J/K hot path computes: fp64 inputs and outputs, integral core
 * and accumulators in long double (>= fp64; R-12, R-19) so that the whole error budget is the GPU's.  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may call it.
 * It shares no code, tables or constants with the CUDA library (paper_2406_11185_b200/csrc).
 *
 * Definitions followed (Eq. 1;  PAPER.md:68-70, ERI;  PAPER.md:81-82, screening):
 *   J_mu,nu     = sum_{lambda sigma} D_lambda,sigma (mu nu|lambda sigma)
 *   K_mu,lambda = sum_{nu sigma}     D_nu,sigma     (mu nu|lambda sigma)
 *   Q_AB = sqrt( max_{mu in A, nu in B} |(mu nu|mu nu)| )                     (SURVEY R-10)
 *   a unique shell quartet is kept iff (Q_AB*Q_CD)*Dmax >= tau, Dmax = max|D|  (SURVEY R-6, R-7;
 *   "If S(AB|CD) < TOLERANCE -> there will not be dispatch")
 * The screened symmetric scheme (orc_jk) applies the 16 updates of SURVEY R-9 per integral and
 * accumulates J, K in long double (SURVEY R-12).  orc_jk_brute is Eq. 1 written out with no
 * symmetry and no screening; orc_jk_block evaluates single shell blocks of J and K from the
 * definition with the same screen (used where the full oracle is too slow: cfg 2-4).
 *
 * Pins (tests/test_oracle_*.py): P1 Boys, P2-P4 closed forms, P5/P5b contraction+normalisation+J/K,
 * P6 one-centre high-L closed form, P7 derivative identity, P8 axis permutations, P9 symmetry,
 * P10 Schwarz, P11 positivity, P12 brute force, P13 long-double rerun, P14 screening bounds,
 * P15 order independence of the recurrence centre (R-22: the integral core builds the recurrences on the
 * centre nearest to each primitive pair's product centre, eri_core.inc.c).
 * No function here is "parity unpinned".
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* Highest shell angular momentum.  liboracle.so is built with 3 (s, p, d, f: the configs of BASELINE.json);
 * liboracle_g.so is the same source with -DLMAX_SHELL=4 (g shells).  Nothing but the table
 * sizes below depends on it: the recurrences are written for any L. */
#ifndef LMAX_SHELL
#define LMAX_SHELL 3
#endif
#define NPC ((LMAX_SHELL + 1) * (LMAX_SHELL + 2) / 2)   /* pair classes (hi >= lo): 10, or 15 with g */
#define NQC (NPC * (NPC + 1) / 2)                       /* quartet classes: 55, or 120 with g */
#define MAXM (4 * LMAX_SHELL)                 /* highest Boys order: 12 for (ff|ff) */
#define NCUM(l) (((l) + 1) * ((l) + 2) * ((l) + 3) / 6)   /* # Cartesian comps of degree <= l; NCUM(-1)=0 */
#define NCART(l) (((l) + 1) * ((l) + 2) / 2)
#define NCUM_MAX NCUM(2 * LMAX_SHELL)         /* 84 (165 with g) */
#define NCUM_B NCUM(LMAX_SHELL)               /* 20 (35) */
#define NCART_MAX NCART(LMAX_SHELL)           /* 10 (15) */
#define NBLK (NCART_MAX * NCART_MAX * NCART_MAX * NCART_MAX)   /* integrals of one shell quartet */

typedef struct {
    int natoms, nshells;
    const double *xyz;      /* [natoms*3] bohr */
    const int32_t *atom, *l, *nprim, *off;
    const double *expo, *coef;   /* FINAL coefficients */
} basis_t;

/* Cartesian component tables: cumulative index over degrees 0..6; inside a degree the order is
 * lx descending, then ly descending (SURVEY R-3). */
static int cart_x[NCUM_MAX], cart_y[NCUM_MAX], cart_z[NCUM_MAX];
static int tables_ready = 0;
static int cidx(int x, int y, int z)
{
    int l = x + y + z, ii = l - x;
    return l * (l + 1) * (l + 2) / 6 + ii * (ii + 1) / 2 + z;
}
static void init_tables(void)
{
    if (tables_ready) return;
    for (int l = 0; l <= 2 * LMAX_SHELL; ++l)
        for (int x = l; x >= 0; --x)
            for (int y = l - x; y >= 0; --y) {
                int z = l - x - y, k = cidx(x, y, z);
                cart_x[k] = x; cart_y[k] = y; cart_z[k] = z;
            }
    tables_ready = 1;
}

#define REAL double
#define NAME(x) x##_d
#define R_EXP exp
#define R_SQRT sqrt
#define R_ERF erf
#include "eri_core.inc.c"
#undef REAL
#undef NAME
#undef R_EXP
#undef R_SQRT
#undef R_ERF

#define REAL long double
#define NAME(x) x##_ld
#define R_EXP expl
#define R_SQRT sqrtl
#define R_ERF erfl
#include "eri_core.inc.c"
#undef REAL
#undef NAME
#undef R_EXP
#undef R_SQRT
#undef R_ERF

static basis_t mk_basis(int natoms, const double *xyz, int nshells, const int32_t *atom, const int32_t *l,
                        const int32_t *nprim, const int32_t *off, const double *expo, const double *coef)
{
    basis_t b = { natoms, nshells, xyz, atom, l, nprim, off, expo, coef };
    init_tables();
    return b;
}
#define BASIS_ARGS int natoms, const double *xyz, int nshells, const int32_t *atom, const int32_t *l, \
                   const int32_t *nprim, const int32_t *off, const double *expo, const double *coef
#define BASIS_PASS natoms, xyz, nshells, atom, l, nprim, off, expo, coef

static int check_basis(const basis_t *b)
{
    for (int s = 0; s < b->nshells; ++s) {
        if (b->l[s] < 0 || b->l[s] > LMAX_SHELL) return -2;
        if (b->atom[s] < 0 || b->atom[s] >= b->natoms) return -1;
        if (b->nprim[s] < 1) return -1;
    }
    return 0;
}

/* ---- exported: Boys (pin P1) ---- */
void orc_boys(int mmax, double T, double *F) { boys_d(mmax, T, F); }
void orc_boys_ld(int mmax, long double T, long double *F) { boys_ld(mmax, T, F); }

/* ---- exported: normalisation (SURVEY R-1) ----
 * N_k = (2a/pi)^(3/4) (4a)^(L/2) / sqrt((2L-1)!!);  d_k = c_k N_k;  then d_k /= sqrt(S),
 * S = sum_ij d_i d_j (pi/(a_i+a_j))^(3/2) (2L-1)!! / (2(a_i+a_j))^L  (self-overlap of the (L,0,0) function). */
int orc_normalize(int nshells, const int32_t *l, const int32_t *nprim, const int32_t *off,
                  const double *expo, const double *coef_raw, double *coef_out)
{
    const double pi = 3.14159265358979323846;
    for (int s = 0; s < nshells; ++s) {
        int L = l[s];
        double df = 1.0;                              /* (2L-1)!! */
        for (int k = 2 * L - 1; k > 1; k -= 2) df *= k;
        for (int k = 0; k < nprim[s]; ++k) {
            double a = expo[off[s] + k];
            if (!(a > 0.0)) return -1;
            coef_out[off[s] + k] = coef_raw[off[s] + k] * pow(2 * a / pi, 0.75) * pow(4 * a, 0.5 * L) / sqrt(df);
        }
        double S = 0.0;
        for (int i = 0; i < nprim[s]; ++i)
            for (int j = 0; j < nprim[s]; ++j) {
                double p = expo[off[s] + i] + expo[off[s] + j];
                S += coef_out[off[s] + i] * coef_out[off[s] + j] * pow(pi / p, 1.5) * df / pow(2 * p, L);
            }
        for (int k = 0; k < nprim[s]; ++k) coef_out[off[s] + k] /= sqrt(S);
    }
    return 0;
}

/* ---- exported: one shell-quartet block (pins P2-P9, P13) ---- */
int orc_eri_block(BASIS_ARGS, int sA, int sB, int sC, int sD, double *out)
{
    basis_t b = mk_basis(BASIS_PASS);
    if (check_basis(&b)) return check_basis(&b);
    scratch_t_d s;
    if (scratch_alloc_d(&s)) return -3;
    shell_quartet_d(&b, sA, sB, sC, sD, &s, out);
    scratch_free_d(&s);
    return 0;
}
int orc_eri_block_ld(BASIS_ARGS, int sA, int sB, int sC, int sD, long double *out)
{
    basis_t b = mk_basis(BASIS_PASS);
    if (check_basis(&b)) return check_basis(&b);
    scratch_t_ld s;
    if (scratch_alloc_ld(&s)) return -3;
    shell_quartet_ld(&b, sA, sB, sC, sD, &s, out);
    scratch_free_ld(&s);
    return 0;
}

/* The oracle proper (Schwarz table, J/K, blocks) evaluates the integral core in long double and keeps the
 * integrals in long double through the J/K accumulation; only the outputs are fp64 (reading R-19).  Reason: in the oracle's fixed input shell order the plain
 * fp64 HRR, (a,b+1_i| = (a+1_i,b| + (A_i-B_i)(ab|, cancels badly when angular momentum is shifted from a distant
 * diffuse shell onto a tight high-l shell (measured: cfg 1 shells (35,23): Q_fp64 3.003293e-4, Q_long-double
 * 3.003267e-4).  The fp64 instantiation is kept for pin P13 and for orc_eri_block. */
#define CORE_REAL long double
#define core_scratch_t scratch_t_ld
#define core_scratch_alloc scratch_alloc_ld
#define core_scratch_free scratch_free_ld
#define core_shell_quartet shell_quartet_ld

/* ---- exported: Schwarz bounds Q[nshells*nshells] (SURVEY R-10) ---- */
int orc_schwarz(BASIS_ARGS, double *Q)
{
    basis_t b = mk_basis(BASIS_PASS);
    if (check_basis(&b)) return check_basis(&b);
    int err = 0;
#pragma omp parallel
    {
        core_scratch_t s;
        CORE_REAL *blk = (CORE_REAL *)malloc(sizeof(CORE_REAL) * NBLK);
        if (core_scratch_alloc(&s) || !blk) {
#pragma omp atomic write
            err = -3;
        } else {
#pragma omp for schedule(dynamic, 4)
            for (int A = 0; A < nshells; ++A)
                for (int B = 0; B <= A; ++B) {
                    int nA = NCART(l[A]), nB = NCART(l[B]);
                    core_shell_quartet(&b, A, B, A, B, &s, blk);
                    double mx = 0.0;
                    for (int i = 0; i < nA; ++i)
                        for (int j = 0; j < nB; ++j) {
                            double vdiag = fabs((double)blk[((i * nB + j) * nA + i) * nB + j]);
                            if (vdiag > mx) mx = vdiag;
                        }
                    Q[(size_t)A * nshells + B] = Q[(size_t)B * nshells + A] = sqrt(mx);
                }
        }
        core_scratch_free(&s); free(blk);
    }
    return err;
}

static double dmax_of(const double *D, size_t n2)
{
    double m = 0.0;
    for (size_t i = 0; i < n2; ++i) { double a = fabs(D[i]); if (a > m || a != a) m = a; }
    return m;
}
double orc_dmax(const double *D, int nbf) { return dmax_of(D, (size_t)nbf * nbf); }

static void bf_offsets(const basis_t *b, int *bo)
{
    bo[0] = 0;
    for (int s = 0; s < b->nshells; ++s) bo[s + 1] = bo[s] + NCART(b->l[s]);
}

/* Block-density screen (reading R-23; Haeser & Ahlrichs): the one global
 * Dmax of the rule above is replaced, per quartet, by the largest density element the quartet's integrals can meet in
 * the 16 updates of R-9,
 *   Dblk(AB|CD) = max( |D|_AB, |D|_CD, |D|_AC, |D|_AD, |D|_BC, |D|_BD ),  |D|_XY = max_{mu in X, nu in Y} max(|D_mu,nu|, |D_nu,mu|),
 * keep iff (Q_AB*Q_CD)*Dblk >= tau.  Dblk <= Dmax, so the kept set is a subset of the global rule's, and Dblk is
 * invariant under the 8 index permutations, so the per-block definition (orc_jk_block) uses the same rule.
 * Dsh[nshells*nshells] holds |D|_XY. */
static void shell_block_max(const basis_t *b, const int *bo, const double *D, int N, double *Dsh)
{
    const int ns = b->nshells;
    for (int X = 0; X < ns; ++X)
        for (int Y = 0; Y < ns; ++Y) {
            double m = 0.0;
            for (int i = bo[X]; i < bo[X + 1]; ++i)
                for (int j = bo[Y]; j < bo[Y + 1]; ++j) {
                    double a = fabs(D[(size_t)i * N + j]), c = fabs(D[(size_t)j * N + i]);
                    if (a > m) m = a;
                    if (c > m) m = c;
                }
            Dsh[(size_t)X * ns + Y] = m;
        }
}
static double screen_density(const double *Dsh, int ns, double Dmax, int A, int B, int C, int Dd)
{
    if (!Dsh) return Dmax;                      /* global rule (R-6) */
    double m = Dsh[(size_t)A * ns + B], v;
    v = Dsh[(size_t)C * ns + Dd]; if (v > m) m = v;
    v = Dsh[(size_t)A * ns + C];  if (v > m) m = v;
    v = Dsh[(size_t)A * ns + Dd]; if (v > m) m = v;
    v = Dsh[(size_t)B * ns + C];  if (v > m) m = v;
    v = Dsh[(size_t)B * ns + Dd]; if (v > m) m = v;
    return m;
}
/* ---- exported: |D|_XY table of the block-density screen ---- */
int orc_dshell(BASIS_ARGS, const double *D, double *Dsh)
{
    basis_t b = mk_basis(BASIS_PASS);
    if (check_basis(&b)) return check_basis(&b);
    int *bo = (int *)malloc(sizeof(int) * (nshells + 1));
    bf_offsets(&b, bo);
    shell_block_max(&b, bo, D, bo[nshells], Dsh);
    free(bo);
    return 0;
}

/* quartet class index (both sides define this independently): pair class pc = hi(hi+1)/2+lo with
 * hi >= lo the two angular momenta; quartet class X(X+1)/2+Y with X >= Y the two pair classes. */
static int qclass(int la, int lb, int lc, int ld)
{
    int h1 = la > lb ? la : lb, l1 = la > lb ? lb : la;
    int h2 = lc > ld ? lc : ld, l2 = lc > ld ? ld : lc;
    int p1 = h1 * (h1 + 1) / 2 + l1, p2 = h2 * (h2 + 1) / 2 + l2;
    int X = p1 > p2 ? p1 : p2, Y = p1 > p2 ? p2 : p1;
    return X * (X + 1) / 2 + Y;
}

/* The loop of orc_jk restricted to bra pairs pab in [pab_lo, pab_hi): long double partial sums Jt, Kt [nbf*nbf]
 * (overwritten) and the counts of that range.  Summing the partial results of disjoint ranges that cover
 * [0, npair) gives orc_jk's result; tests/golden/make_golden.py uses this to checkpoint the hours-long full runs. */
static int jk_range(BASIS_ARGS, const double *D, double tau, const double *Qin, int64_t pab_lo, int64_t pab_hi,
                    long double *Jt, long double *Kt, int64_t *counts, int64_t *class_counts, int block_density)
{
    basis_t b = mk_basis(BASIS_PASS);
    if (check_basis(&b)) return check_basis(&b);
    int *bo = (int *)malloc(sizeof(int) * (nshells + 1));
    bf_offsets(&b, bo);
    const int N = bo[nshells];
    double *Q = (double *)malloc(sizeof(double) * (size_t)nshells * nshells);
    if (Qin) memcpy(Q, Qin, sizeof(double) * (size_t)nshells * nshells);
    else { int e = orc_schwarz(BASIS_PASS, Q); if (e) return e; }
    const double Dmax = dmax_of(D, (size_t)N * N);
    double *Dsh = NULL;
    if (block_density) {
        Dsh = (double *)malloc(sizeof(double) * (size_t)nshells * nshells);
        shell_block_max(&b, bo, D, N, Dsh);
    }
    const int64_t npair = (int64_t)nshells * (nshells + 1) / 2;
    if (pab_lo < 0) pab_lo = 0;
    if (pab_hi > npair) pab_hi = npair;
    for (size_t i = 0; i < (size_t)N * N; ++i) Jt[i] = Kt[i] = 0;
    int64_t n_all = 0, n_kept = 0, n_prim = 0;
    int64_t cc[NQC]; memset(cc, 0, sizeof cc);
    int err = 0;
#pragma omp parallel
    {
        core_scratch_t s;
        CORE_REAL *blk = (CORE_REAL *)malloc(sizeof(CORE_REAL) * NBLK);
        long double *Jp = (long double *)calloc((size_t)N * N, sizeof(long double));
        long double *Kp = (long double *)calloc((size_t)N * N, sizeof(long double));
        int64_t my_all = 0, my_kept = 0, my_prim = 0, mycc[NQC];
        memset(mycc, 0, sizeof mycc);
        if (core_scratch_alloc(&s) || !blk || !Jp || !Kp) {
#pragma omp atomic write
            err = -3;
        } else {
#pragma omp for schedule(dynamic, 1)
            for (int64_t pab = pab_hi - 1; pab >= pab_lo; --pab) {
                /* decode pab = A(A+1)/2 + B */
                int A = (int)((sqrt(8.0 * (double)pab + 1.0) - 1.0) / 2.0);
                while ((int64_t)A * (A + 1) / 2 > pab) --A;
                while ((int64_t)(A + 1) * (A + 2) / 2 <= pab) ++A;
                int B = (int)(pab - (int64_t)A * (A + 1) / 2);
                for (int C = 0; C <= A; ++C)
                    for (int Dd = 0; Dd <= C; ++Dd) {
                        int64_t pcd = (int64_t)C * (C + 1) / 2 + Dd;
                        if (pcd > pab) continue;
                        ++my_all;
                        /* keep iff (Q_AB*Q_CD)*Dmax >= tau  (block-density mode: Dblk(AB|CD) in place of Dmax) */
                        double bound = (Q[(size_t)A * nshells + B] * Q[(size_t)C * nshells + Dd])
                                       * screen_density(Dsh, nshells, Dmax, A, B, C, Dd);
                        if (bound < tau) continue;
                        ++my_kept;
                        my_prim += (int64_t)nprim[A] * nprim[B] * nprim[C] * nprim[Dd];
                        ++mycc[qclass(l[A], l[B], l[C], l[Dd])];
                        core_shell_quartet(&b, A, B, C, Dd, &s, blk);
                        double f = (A == B ? 0.5 : 1.0) * (C == Dd ? 0.5 : 1.0) * (pab == pcd ? 0.5 : 1.0);
                        int nA = NCART(l[A]), nB = NCART(l[B]), nC = NCART(l[C]), nD = NCART(l[Dd]);
                        for (int ia = 0; ia < nA; ++ia)
                        for (int ib = 0; ib < nB; ++ib)
                        for (int ic = 0; ic < nC; ++ic)
                        for (int id = 0; id < nD; ++id) {
                            long double t = (long double)f * blk[((ia * nB + ib) * nC + ic) * nD + id];
                            size_t m = bo[A] + ia, n = bo[B] + ib, lam = bo[C] + ic, sg = bo[Dd] + id;
#define DD(i, j) ((long double)D[(i) * (size_t)N + (j)])
#define JJ(i, j) Jp[(i) * (size_t)N + (j)]
#define KK(i, j) Kp[(i) * (size_t)N + (j)]
                            /* the 16 updates of SURVEY R-9 */
                            JJ(m, n) += DD(lam, sg) * t;  JJ(n, m) += DD(lam, sg) * t;
                            JJ(m, n) += DD(sg, lam) * t;  JJ(n, m) += DD(sg, lam) * t;
                            JJ(lam, sg) += DD(m, n) * t;  JJ(sg, lam) += DD(m, n) * t;
                            JJ(lam, sg) += DD(n, m) * t;  JJ(sg, lam) += DD(n, m) * t;
                            KK(m, lam) += DD(n, sg) * t;  KK(n, lam) += DD(m, sg) * t;
                            KK(m, sg) += DD(n, lam) * t;  KK(n, sg) += DD(m, lam) * t;
                            KK(lam, m) += DD(sg, n) * t;  KK(sg, m) += DD(lam, n) * t;
                            KK(lam, n) += DD(sg, m) * t;  KK(sg, n) += DD(lam, m) * t;
                        }
                    }
            }
#pragma omp critical
            {
                for (size_t i = 0; i < (size_t)N * N; ++i) { Jt[i] += Jp[i]; Kt[i] += Kp[i]; }
                n_all += my_all; n_kept += my_kept; n_prim += my_prim;
                for (int i = 0; i < NQC; ++i) cc[i] += mycc[i];
            }
        }
        core_scratch_free(&s); free(blk); free(Jp); free(Kp);
    }
    if (counts) { counts[0] = n_all; counts[1] = n_kept; counts[2] = n_prim; }
    if (class_counts) memcpy(class_counts, cc, sizeof cc);
    free(Q); free(bo); free(Dsh);
    return err;
}

/* ---- exported: screened, 8-fold-symmetric J/K (the oracle proper) ----
 * Q may be NULL (computed here) or a caller-supplied table from orc_schwarz.
 * counts[0] = unique quartets before screening, counts[1] = kept, counts[2] = primitive quartets in kept;
 * class_counts[NQC] = kept per class (55 entries; 120 in the g build).  J, K: full symmetric [nbf*nbf], overwritten. */
static int jk_full(BASIS_ARGS, const double *D, double tau, const double *Qin, double *J, double *K,
                   int64_t *counts, int64_t *class_counts, int block_density)
{
    size_t N = 0;
    for (int s = 0; s < nshells; ++s) N += (l[s] >= 0 && l[s] <= LMAX_SHELL) ? NCART(l[s]) : 0;
    long double *Jt = (long double *)calloc(N * N + 1, sizeof(long double));
    long double *Kt = (long double *)calloc(N * N + 1, sizeof(long double));
    if (!Jt || !Kt) { free(Jt); free(Kt); return -3; }
    int err = jk_range(BASIS_PASS, D, tau, Qin, 0, (int64_t)nshells * (nshells + 1) / 2, Jt, Kt, counts, class_counts,
                       block_density);
    if (err == 0)
        for (size_t i = 0; i < N * N; ++i) { J[i] = (double)Jt[i]; K[i] = (double)Kt[i]; }
    free(Jt); free(Kt);
    return err;
}
int orc_jk(BASIS_ARGS, const double *D, double tau, const double *Qin, double *J, double *K,
           int64_t *counts, int64_t *class_counts)
{
    return jk_full(BASIS_PASS, D, tau, Qin, J, K, counts, class_counts, 0);
}
/* ---- exported: the same with the block-density screen (R-23) ---- */
int orc_jk_bd(BASIS_ARGS, const double *D, double tau, const double *Qin, double *J, double *K,
              int64_t *counts, int64_t *class_counts)
{
    return jk_full(BASIS_PASS, D, tau, Qin, J, K, counts, class_counts, 1);
}

/* ---- exported: orc_jk's loop over the bra pairs pab in [pab_lo, pab_hi) only, long double partial sums out ---- */
int orc_jk_range(BASIS_ARGS, const double *D, double tau, const double *Qin, int64_t pab_lo, int64_t pab_hi,
                 long double *Jpart, long double *Kpart, int64_t *counts, int64_t *class_counts)
{
    return jk_range(BASIS_PASS, D, tau, Qin, pab_lo, pab_hi, Jpart, Kpart, counts, class_counts, 0);
}

/* ---- exported: kept-quartet counts only (no integrals), same loop and rule as orc_jk ---- */
static int count_impl(int nshells, const int32_t *l, const int32_t *nprim, const double *Q, double Dmax, const double *Dsh,
                      double tau, int64_t *counts, int64_t *class_counts)
{
    int64_t n_all = 0, n_kept = 0, n_prim = 0, cc[NQC];
    memset(cc, 0, sizeof cc);
#pragma omp parallel for schedule(dynamic, 8) reduction(+ : n_all, n_kept, n_prim, cc[:NQC])
    for (int A = 0; A < nshells; ++A)
        for (int B = 0; B <= A; ++B) {
            int64_t pab = (int64_t)A * (A + 1) / 2 + B;
            for (int C = 0; C <= A; ++C)
                for (int Dd = 0; Dd <= C; ++Dd) {
                    int64_t pcd = (int64_t)C * (C + 1) / 2 + Dd;
                    if (pcd > pab) continue;
                    ++n_all;
                    double bound = (Q[(size_t)A * nshells + B] * Q[(size_t)C * nshells + Dd])
                                   * screen_density(Dsh, nshells, Dmax, A, B, C, Dd);
                    if (bound < tau) continue;
                    ++n_kept;
                    n_prim += (int64_t)nprim[A] * nprim[B] * nprim[C] * nprim[Dd];
                    ++cc[qclass(l[A], l[B], l[C], l[Dd])];
                }
        }
    counts[0] = n_all; counts[1] = n_kept; counts[2] = n_prim;
    memcpy(class_counts, cc, sizeof cc);
    return 0;
}
int orc_count(int nshells, const int32_t *l, const int32_t *nprim, const double *Q, double Dmax, double tau,
              int64_t *counts, int64_t *class_counts)
{
    return count_impl(nshells, l, nprim, Q, Dmax, NULL, tau, counts, class_counts);
}
/* block-density rule: Dsh = the |D|_XY table of orc_dshell */
int orc_count_bd(int nshells, const int32_t *l, const int32_t *nprim, const double *Q, const double *Dsh, double tau,
                 int64_t *counts, int64_t *class_counts)
{
    return count_impl(nshells, l, nprim, Q, 0.0, Dsh, tau, counts, class_counts);
}

/* ---- exported: Eq. 1 written out, no symmetry, no screening (pin P12) ---- */
int orc_jk_brute(BASIS_ARGS, const double *D, double *J, double *K)
{
    basis_t b = mk_basis(BASIS_PASS);
    if (check_basis(&b)) return check_basis(&b);
    int *bo = (int *)malloc(sizeof(int) * (nshells + 1));
    bf_offsets(&b, bo);
    const int N = bo[nshells];
    long double *Jt = (long double *)calloc((size_t)N * N, sizeof(long double));
    long double *Kt = (long double *)calloc((size_t)N * N, sizeof(long double));
    core_scratch_t s;
    CORE_REAL *blk = (CORE_REAL *)malloc(sizeof(CORE_REAL) * NBLK);
    if (core_scratch_alloc(&s)) return -3;
    for (int A = 0; A < nshells; ++A) for (int B = 0; B < nshells; ++B)
    for (int C = 0; C < nshells; ++C) for (int Dd = 0; Dd < nshells; ++Dd) {
        core_shell_quartet(&b, A, B, C, Dd, &s, blk);
        int nA = NCART(l[A]), nB = NCART(l[B]), nC = NCART(l[C]), nD = NCART(l[Dd]);
        for (int ia = 0; ia < nA; ++ia) for (int ib = 0; ib < nB; ++ib)
        for (int ic = 0; ic < nC; ++ic) for (int id = 0; id < nD; ++id) {
            long double I = blk[((ia * nB + ib) * nC + ic) * nD + id];
            size_t m = bo[A] + ia, n = bo[B] + ib, lam = bo[C] + ic, sg = bo[Dd] + id;
            Jt[m * N + n] += (long double)D[lam * N + sg] * I;     /* J_mn = sum D_ls (mn|ls) */
            Kt[m * N + lam] += (long double)D[n * N + sg] * I;     /* K_ml = sum D_ns (mn|ls) */
        }
    }
    for (size_t i = 0; i < (size_t)N * N; ++i) { J[i] = (double)Jt[i]; K[i] = (double)Kt[i]; }
    core_scratch_free(&s); free(blk); free(Jt); free(Kt); free(bo);
    return 0;
}

/* ---- exported: one shell block of J and of K from the definition, with the screen ----
 * Jblk[nA*nB]:  J_mn = sum_{C,D} [ (Q_AB*Q_CD)*Dmax >= tau ] sum_{l in C, s in D} D_ls (mn|ls)
 * Kblk[nA*nB]:  K_ml = sum_{C,D} [ (Q_AC*Q_BD)*Dmax >= tau ] sum_{n in C, s in D} D_ns (m n|l s), m in A, l in B
 * (the screen is symmetric under the 8 permutations, so this equals the block of orc_jk's result). */
static int jk_block_impl(BASIS_ARGS, const double *D, double tau, const double *Q, double Dmax, const double *Dsh,
                         int sA, int sB, double *Jblk, double *Kblk, int64_t *work)
{
    int64_t w_q = 0, w_p = 0;
    basis_t b = mk_basis(BASIS_PASS);
    if (check_basis(&b)) return check_basis(&b);
    int *bo = (int *)malloc(sizeof(int) * (nshells + 1));
    bf_offsets(&b, bo);
    const int N = bo[nshells];
    const int nA = NCART(l[sA]), nB = NCART(l[sB]);
    long double Jt[NCART_MAX * NCART_MAX], Kt[NCART_MAX * NCART_MAX];
    for (int i = 0; i < NCART_MAX * NCART_MAX; ++i) Jt[i] = Kt[i] = 0;
    int err = 0;
#pragma omp parallel
    {
        core_scratch_t s;
        CORE_REAL *blk = (CORE_REAL *)malloc(sizeof(CORE_REAL) * NBLK);
        long double Jp[NCART_MAX * NCART_MAX], Kp[NCART_MAX * NCART_MAX];
        for (int i = 0; i < NCART_MAX * NCART_MAX; ++i) Jp[i] = Kp[i] = 0;
        if (core_scratch_alloc(&s) || !blk) {
#pragma omp atomic write
            err = -3;
        } else {
#pragma omp for schedule(dynamic, 1)
            for (int C = 0; C < nshells; ++C)
                for (int Dd = 0; Dd < nshells; ++Dd) {
                    int nC = NCART(l[C]), nD = NCART(l[Dd]);
                    if (Jblk && (Q[(size_t)sA * nshells + sB] * Q[(size_t)C * nshells + Dd])
                                    * screen_density(Dsh, nshells, Dmax, sA, sB, C, Dd) >= tau) {
                        core_shell_quartet(&b, sA, sB, C, Dd, &s, blk);
#pragma omp atomic
                        w_q += 1;
#pragma omp atomic
                        w_p += (int64_t)nprim[sA] * nprim[sB] * nprim[C] * nprim[Dd];
                        for (int ia = 0; ia < nA; ++ia) for (int ib = 0; ib < nB; ++ib)
                        for (int ic = 0; ic < nC; ++ic) for (int id = 0; id < nD; ++id)
                            Jp[ia * nB + ib] += (long double)D[(size_t)(bo[C] + ic) * N + bo[Dd] + id]
                                                * blk[((ia * nB + ib) * nC + ic) * nD + id];
                    }
                    if (Kblk && (Q[(size_t)sA * nshells + C] * Q[(size_t)sB * nshells + Dd])
                                    * screen_density(Dsh, nshells, Dmax, sA, C, sB, Dd) >= tau) {
                        /* (A C | B D): mu in A, nu in C, lambda in B, sigma in D */
                        core_shell_quartet(&b, sA, C, sB, Dd, &s, blk);
#pragma omp atomic
                        w_q += 1;
#pragma omp atomic
                        w_p += (int64_t)nprim[sA] * nprim[C] * nprim[sB] * nprim[Dd];
                        for (int ia = 0; ia < nA; ++ia) for (int ic = 0; ic < nC; ++ic)
                        for (int ib = 0; ib < nB; ++ib) for (int id = 0; id < nD; ++id)
                            Kp[ia * nB + ib] += (long double)D[(size_t)(bo[C] + ic) * N + bo[Dd] + id]
                                                * blk[((ia * nC + ic) * nB + ib) * nD + id];
                    }
                }
#pragma omp critical
            for (int i = 0; i < nA * nB; ++i) { Jt[i] += Jp[i]; Kt[i] += Kp[i]; }
        }
        core_scratch_free(&s); free(blk);
    }
    for (int i = 0; i < nA * nB; ++i) { if (Jblk) Jblk[i] = (double)Jt[i]; if (Kblk) Kblk[i] = (double)Kt[i]; }
    if (work) { work[0] = w_q; work[1] = w_p; }
    free(bo);
    return err;
}
int orc_jk_block(BASIS_ARGS, const double *D, double tau, const double *Q, double Dmax,
                 int sA, int sB, double *Jblk, double *Kblk, int64_t *work /* [2]: shell quartets, primitive quartets evaluated; may be NULL */)
{
    return jk_block_impl(BASIS_PASS, D, tau, Q, Dmax, NULL, sA, sB, Jblk, Kblk, work);
}
/* the same with the block-density screen (R-23); Dsh = the |D|_XY table of orc_dshell */
int orc_jk_block_bd(BASIS_ARGS, const double *D, double tau, const double *Q, const double *Dsh,
                    int sA, int sB, double *Jblk, double *Kblk, int64_t *work)
{
    return jk_block_impl(BASIS_PASS, D, tau, Q, 0.0, Dsh, sA, sB, Jblk, Kblk, work);
}

int orc_lmax(void) { return LMAX_SHELL; }
int orc_nqclass(void) { return NQC; }

int orc_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
