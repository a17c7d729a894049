/* ORACLE (test infrastructure only) -- integral core, included twice by jk_oracle.c:
 * once with REAL = double (the oracle proper) and once with REAL = long double (pin P13,
 * separates rounding error from formula error).  Shares no code with the CUDA library.
 *
 * What it computes: the contracted Cartesian four-centre electron-repulsion integrals
 *   (mu nu|lambda sigma) = iint phi_mu(r) phi_nu(r) |r-r'|^-1 phi_lambda(r') phi_sigma(r') d3r d3r'
 * (the ERI definition) by the Obara-Saika recurrences in Head-Gordon-Pople
 * form, the method the paper says it redesigned (refs 47 at PAPER.md:552).
 * The paper gives no equations for the algorithm; the recurrences below are the textbook
 * ones restated in SURVEY.md section 8(c) and are followed step by step in that order:
 *   Boys -> base case [00|00]^(m) -> VRR on the bra -> VRR on the ket -> contraction -> HRR.
 * No primitive screening, no approximations.
 *
 * Macros expected: REAL, NAME(x), R_EXP, R_SQRT, R_ERF.
 */

/* Boys function F_m(T) = int_0^1 t^(2m) exp(-T t^2) dt, m = 0..mmax  (SURVEY 8(c) "Boys").
 * T < 35: convergent series at m = mmax, then downward recursion.
 * T >= 35: F_0 = 1/2 sqrt(pi/T) erf(sqrt T), then upward recursion (stable there). */
static void NAME(boys)(int mmax, REAL T, REAL *F)
{
    const REAL pi = (REAL)3.14159265358979323846264338327950288L;
    REAL eT = R_EXP(-T);
    if (T < (REAL)35) {
        REAL term = (REAL)1 / (REAL)(2 * mmax + 1);
        REAL sum = term;
        for (int k = 1; k < 2000; ++k) {
            term *= (2 * T) / (REAL)(2 * mmax + 2 * k + 1);
            sum += term;
            if (term < sum * (REAL)1e-22) break;
        }
        F[mmax] = eT * sum;
        for (int m = mmax; m >= 1; --m)
            F[m - 1] = (2 * T * F[m] + eT) / (REAL)(2 * m - 1);
    } else {
        F[0] = (REAL)0.5 * R_SQRT(pi / T) * R_ERF(R_SQRT(T));
        for (int m = 0; m < mmax; ++m)
            F[m + 1] = ((REAL)(2 * m + 1) * F[m] - eT) / (2 * T);
    }
}

#define V(m, a, c) v[((size_t)(m) * NCUM_MAX + (a)) * NCUM_MAX + (c)]

/* Primitive [a0|c0]^(m) for all deg(a) <= lab, deg(c) <= lcd, deg(a)+deg(c)+m <= lab+lcd.
 * pref already holds the product of contraction coefficients. */
static void NAME(prim_vrr)(int lab, int lcd, REAL za, REAL zb, REAL zc, REAL zd,
                           const REAL *A, const REAL *B, const REAL *C, const REAL *D,
                           REAL coef, REAL *v)
{
    const REAL pi = (REAL)3.14159265358979323846264338327950288L;
    const int L = lab + lcd;
    REAL zeta = za + zb, eta = zc + zd;
    REAL P[3], Q[3], W[3], PA[3], QC[3], WP[3], WQ[3];
    REAL AB2 = 0, CD2 = 0, PQ2 = 0;
    for (int i = 0; i < 3; ++i) {
        P[i] = (za * A[i] + zb * B[i]) / zeta;
        Q[i] = (zc * C[i] + zd * D[i]) / eta;
        W[i] = (zeta * P[i] + eta * Q[i]) / (zeta + eta);
        PA[i] = P[i] - A[i];  QC[i] = Q[i] - C[i];
        WP[i] = W[i] - P[i];  WQ[i] = W[i] - Q[i];
        AB2 += (A[i] - B[i]) * (A[i] - B[i]);
        CD2 += (C[i] - D[i]) * (C[i] - D[i]);
        PQ2 += (P[i] - Q[i]) * (P[i] - Q[i]);
    }
    REAL rho = zeta * eta / (zeta + eta);
    REAL T = rho * PQ2;
    REAL KAB = R_EXP(-za * zb * AB2 / zeta);
    REAL KCD = R_EXP(-zc * zd * CD2 / eta);
    /* base: [00|00]^(m) = 2 pi^(5/2) / (zeta eta sqrt(zeta+eta)) K_AB K_CD F_m(T) */
    REAL pref = 2 * pi * pi * R_SQRT(pi) / (zeta * eta * R_SQRT(zeta + eta)) * KAB * KCD * coef;
    REAL F[MAXM + 1];
    NAME(boys)(L, T, F);
    for (int m = 0; m <= L; ++m) V(m, 0, 0) = pref * F[m];

    /* VRR on the bra:
     * [a+1_i,0|00]^(m) = (P_i-A_i)[a|0]^(m) + (W_i-P_i)[a|0]^(m+1)
     *                    + a_i/(2 zeta) ( [a-1_i|0]^(m) - (rho/zeta)[a-1_i|0]^(m+1) ) */
    for (int deg = 1; deg <= lab; ++deg) {
        for (int a = NCUM(deg - 1); a < NCUM(deg); ++a) {
            int pw[3] = { cart_x[a], cart_y[a], cart_z[a] };
            int i = pw[0] > 0 ? 0 : (pw[1] > 0 ? 1 : 2);
            pw[i] -= 1;
            int am = cidx(pw[0], pw[1], pw[2]);
            int ai = pw[i];
            int amm = -1;
            if (ai > 0) { pw[i] -= 1; amm = cidx(pw[0], pw[1], pw[2]); }
            for (int m = 0; m <= L - deg; ++m) {
                REAL val = PA[i] * V(m, am, 0) + WP[i] * V(m + 1, am, 0);
                if (ai > 0)
                    val += (REAL)ai / (2 * zeta) * (V(m, amm, 0) - rho / zeta * V(m + 1, amm, 0));
                V(m, a, 0) = val;
            }
        }
    }
    /* VRR on the ket:
     * [a0|c+1_i,0]^(m) = (Q_i-C_i)[a|c]^(m) + (W_i-Q_i)[a|c]^(m+1)
     *                    + c_i/(2 eta) ( [a|c-1_i]^(m) - (rho/eta)[a|c-1_i]^(m+1) )
     *                    + a_i/(2(zeta+eta)) [a-1_i|c]^(m+1) */
    for (int degc = 1; degc <= lcd; ++degc) {
        for (int c = NCUM(degc - 1); c < NCUM(degc); ++c) {
            int pw[3] = { cart_x[c], cart_y[c], cart_z[c] };
            int i = pw[0] > 0 ? 0 : (pw[1] > 0 ? 1 : 2);
            pw[i] -= 1;
            int cm = cidx(pw[0], pw[1], pw[2]);
            int ci = pw[i];
            int cmm = -1;
            if (ci > 0) { pw[i] -= 1; cmm = cidx(pw[0], pw[1], pw[2]); }
            for (int dega = 0; dega <= lab; ++dega) {
                for (int a = NCUM(dega - 1); a < NCUM(dega); ++a) {
                    int pa[3] = { cart_x[a], cart_y[a], cart_z[a] };
                    int aiq = pa[i];
                    int am = -1;
                    if (aiq > 0) { pa[i] -= 1; am = cidx(pa[0], pa[1], pa[2]); }
                    for (int m = 0; m <= L - dega - degc; ++m) {
                        REAL val = QC[i] * V(m, a, cm) + WQ[i] * V(m + 1, a, cm);
                        if (ci > 0)
                            val += (REAL)ci / (2 * eta) * (V(m, a, cmm) - rho / eta * V(m + 1, a, cmm));
                        if (aiq > 0)
                            val += (REAL)aiq / (2 * (zeta + eta)) * V(m + 1, am, cm);
                        V(m, a, c) = val;
                    }
                }
            }
        }
    }
}

typedef struct {
    REAL *v;     /* VRR table  [MAXM+2][NCUM_MAX][NCUM_MAX] */
    REAL *acc;   /* contracted [e0|f0]   [NCUM_MAX][NCUM_MAX] */
    REAL *hb;    /* bra HRR   [NCUM_B][NCUM_MAX][NCUM_MAX] */
    REAL *g;     /* (ab|c0)   [nA*nB][NCUM_MAX] */
    REAL *hk;    /* ket HRR   [NCUM_B][NCUM_MAX] */
    REAL *part;  /* one orientation's contribution  [NCART_MAX^4] */
} NAME(scratch_t);

static int NAME(scratch_alloc)(NAME(scratch_t) *s)
{
    s->v = (REAL *)malloc(sizeof(REAL) * (size_t)(MAXM + 2) * NCUM_MAX * NCUM_MAX);
    s->acc = (REAL *)malloc(sizeof(REAL) * (size_t)NCUM_MAX * NCUM_MAX);
    s->hb = (REAL *)malloc(sizeof(REAL) * (size_t)NCUM_B * NCUM_MAX * NCUM_MAX);
    s->g = (REAL *)malloc(sizeof(REAL) * (size_t)NCART_MAX * NCART_MAX * NCUM_MAX);
    s->hk = (REAL *)malloc(sizeof(REAL) * (size_t)NCUM_B * NCUM_MAX);
    s->part = (REAL *)malloc(sizeof(REAL) * (size_t)NCART_MAX * NCART_MAX * NCART_MAX * NCART_MAX);
    return (s->v && s->acc && s->hb && s->g && s->hk && s->part) ? 0 : -1;
}
static void NAME(scratch_free)(NAME(scratch_t) *s)
{
    free(s->v); free(s->acc); free(s->hb); free(s->g); free(s->hk); free(s->part);
}

/* Contribution to the nA*nB*nC*nD contracted integrals of one shell quartet, out[((ia*nB+ib)*nC+ic)*nD+id], of the
 * primitive quartets selected by (tieAB, tieCD): the recurrences are built on sA and sC (VRR) and shifted onto sB and
 * sD (HRR), and a primitive pair (alpha on sA, beta on sB) takes part iff the Gaussian product centre
 * P = (alpha A + beta B)/(alpha+beta) is nearer to sA than to sB, i.e. alpha > beta, or alpha == beta when tieAB != 0;
 * likewise for (sC, sD) with tieCD  (reading R-22).  Returns the number of primitive quartets it summed.
 * Coefficients are FINAL contraction coefficients d_k (SURVEY R-1). */
static long NAME(shell_quartet_part)(const basis_t *bs, int sA, int sB, int sC, int sD, int tieAB, int tieCD,
                                     NAME(scratch_t) *s, REAL *out)
{
    long nsummed = 0;
    const int la = bs->l[sA], lb = bs->l[sB], lc = bs->l[sC], ld = bs->l[sD];
    const int lab = la + lb, lcd = lc + ld;
    REAL A[3], B[3], C[3], D[3];
    for (int i = 0; i < 3; ++i) {
        A[i] = bs->xyz[3 * bs->atom[sA] + i];  B[i] = bs->xyz[3 * bs->atom[sB] + i];
        C[i] = bs->xyz[3 * bs->atom[sC] + i];  D[i] = bs->xyz[3 * bs->atom[sD] + i];
    }
    REAL *v = s->v, *acc = s->acc;
    for (int a = NCUM(la - 1); a < NCUM(lab); ++a)
        for (int c = NCUM(lc - 1); c < NCUM(lcd); ++c) acc[a * NCUM_MAX + c] = 0;

    /* contraction: sum over primitive quartets of d_a d_b d_c d_d [e0|f0]^(0) */
    for (int ia = 0; ia < bs->nprim[sA]; ++ia)
    for (int ib = 0; ib < bs->nprim[sB]; ++ib)
    for (int ic = 0; ic < bs->nprim[sC]; ++ic)
    for (int id = 0; id < bs->nprim[sD]; ++id) {
        int oa = bs->off[sA] + ia, ob = bs->off[sB] + ib, oc = bs->off[sC] + ic, od = bs->off[sD] + id;
        if (!(bs->expo[oa] > bs->expo[ob] || (tieAB && bs->expo[oa] == bs->expo[ob]))) continue;
        if (!(bs->expo[oc] > bs->expo[od] || (tieCD && bs->expo[oc] == bs->expo[od]))) continue;
        ++nsummed;
        REAL coef = (REAL)bs->coef[oa] * (REAL)bs->coef[ob] * (REAL)bs->coef[oc] * (REAL)bs->coef[od];
        NAME(prim_vrr)(lab, lcd, bs->expo[oa], bs->expo[ob], bs->expo[oc], bs->expo[od], A, B, C, D, coef, v);
        for (int a = NCUM(la - 1); a < NCUM(lab); ++a)
            for (int c = NCUM(lc - 1); c < NCUM(lcd); ++c) acc[a * NCUM_MAX + c] += V(0, a, c);
    }
    if (nsummed == 0) return 0;

    /* HRR on the bra: (a, b+1_i| c) = (a+1_i, b| c) + (A_i - B_i)(a b| c) */
#define HB(b, a, c) s->hb[((size_t)(b) * NCUM_MAX + (a)) * NCUM_MAX + (c)]
    for (int a = NCUM(la - 1); a < NCUM(lab); ++a)
        for (int c = NCUM(lc - 1); c < NCUM(lcd); ++c) HB(0, a, c) = acc[a * NCUM_MAX + c];
    for (int degb = 1; degb <= lb; ++degb) {
        for (int b = NCUM(degb - 1); b < NCUM(degb); ++b) {
            int pb[3] = { cart_x[b], cart_y[b], cart_z[b] };
            int i = pb[0] > 0 ? 0 : (pb[1] > 0 ? 1 : 2);
            pb[i] -= 1;
            int bm = cidx(pb[0], pb[1], pb[2]);
            REAL ABi = A[i] - B[i];
            for (int a = NCUM(la - 1); a < NCUM(lab - degb); ++a) {
                int pa[3] = { cart_x[a], cart_y[a], cart_z[a] };
                pa[i] += 1;
                int ap = cidx(pa[0], pa[1], pa[2]);
                for (int c = NCUM(lc - 1); c < NCUM(lcd); ++c)
                    HB(b, a, c) = HB(bm, ap, c) + ABi * HB(bm, a, c);
            }
        }
    }
    const int nA = NCART(la), nB = NCART(lb), nC = NCART(lc), nD = NCART(ld);
    /* HRR on the ket, per (a,b): (ab| c, d+1_i) = (ab| c+1_i, d) + (C_i - D_i)(ab| c d) */
#define HK(d, c) s->hk[(size_t)(d) * NCUM_MAX + (c)]
    for (int ia = 0; ia < nA; ++ia)
    for (int ib = 0; ib < nB; ++ib) {
        int a = NCUM(la - 1) + ia, b = NCUM(lb - 1) + ib;
        for (int c = NCUM(lc - 1); c < NCUM(lcd); ++c) HK(0, c) = HB(b, a, c);
        for (int degd = 1; degd <= ld; ++degd) {
            for (int d = NCUM(degd - 1); d < NCUM(degd); ++d) {
                int pd[3] = { cart_x[d], cart_y[d], cart_z[d] };
                int i = pd[0] > 0 ? 0 : (pd[1] > 0 ? 1 : 2);
                pd[i] -= 1;
                int dm = cidx(pd[0], pd[1], pd[2]);
                REAL CDi = C[i] - D[i];
                for (int c = NCUM(lc - 1); c < NCUM(lcd - degd); ++c) {
                    int pc[3] = { cart_x[c], cart_y[c], cart_z[c] };
                    pc[i] += 1;
                    int cp = cidx(pc[0], pc[1], pc[2]);
                    HK(d, c) = HK(dm, cp) + CDi * HK(dm, c);
                }
            }
        }
        for (int ic = 0; ic < nC; ++ic)
            for (int id = 0; id < nD; ++id)
                out[((ia * nB + ib) * nC + ic) * nD + id] = HK(NCUM(ld - 1) + id, NCUM(lc - 1) + ic);
    }
#undef HB
#undef HK
    return nsummed;
}

/* All nA*nB*nC*nD contracted integrals of one shell quartet, out[((ia*nB+ib)*nC+ic)*nD+id]: the sum over primitive
 * quartets is split into the four groups {P nearer A | P nearer B} x {Q nearer C | Q nearer D}; each group is evaluated
 * with the recurrences built on the nearer centres (the bra or ket pair handed over in swapped order, which is the
 * identity (ab|cd) = (ba|cd) = (ab|dc) of the definition) and the four results are added.
 * Why: the horizontal recurrence (a,b+1_i| = (a+1_i,b| + (A_i-B_i)(ab| subtracts numbers of size |A-B|^lb when P sits
 * on B; built on the nearer centre the shifted factor (x-B_i) = (x-P_i) + (P_i-B_i) stays small.  R-22. */
static void NAME(shell_quartet)(const basis_t *bs, int sA, int sB, int sC, int sD,
                                NAME(scratch_t) *s, REAL *out)
{
    const int nA = NCART(bs->l[sA]), nB = NCART(bs->l[sB]), nC = NCART(bs->l[sC]), nD = NCART(bs->l[sD]);
    for (int q = 0; q < nA * nB * nC * nD; ++q) out[q] = 0;
    for (int swab = 0; swab < 2; ++swab)
    for (int swcd = 0; swcd < 2; ++swcd) {
        REAL *part = s->part;
        long n = NAME(shell_quartet_part)(bs, swab ? sB : sA, swab ? sA : sB, swcd ? sD : sC, swcd ? sC : sD,
                                          !swab, !swcd, s, part);
        if (n == 0) continue;
        const int n2 = swab ? nA : nB, n3 = swcd ? nD : nC, n4 = swcd ? nC : nD;
        for (int ia = 0; ia < nA; ++ia)
        for (int ib = 0; ib < nB; ++ib)
        for (int ic = 0; ic < nC; ++ic)
        for (int id = 0; id < nD; ++id) {
            const int i1 = swab ? ib : ia, i2 = swab ? ia : ib, i3 = swcd ? id : ic, i4 = swcd ? ic : id;
            out[((ia * nB + ib) * nC + ic) * nD + id] += part[((i1 * n2 + i2) * n3 + i3) * n4 + i4];
        }
    }
}
#undef V
