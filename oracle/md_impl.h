/* ORACLE — TEST INFRASTRUCTURE ONLY.  Never linked, imported or called by the product path.
 *
 * md_impl.h: body of the McMurchie–Davidson oracle, "templated" on the scalar type by textual
 * inclusion.  The includer defines
 *     REAL      scalar type (long double for parity, double for the timed CPU baseline)
 *     SFX(name) name-mangling macro (name##_ld / name##_d)
 *     R_EXP, R_SQRT, R_FABS   libm routines for REAL
 *
 * What it computes (Appendix A):
 *   [c|ab] = ∬ φ_c(r1) |r1−r2|⁻¹ φ_a(r2) φ_b(r2) dr1 dr2                       (eq. 12, Coulomb kernel l.455)
 *   φ_a(r) = (x−A_x)^{a_x}(y−A_y)^{a_y}(z−A_z)^{a_z} exp(−ζ_a|r−A|²)          (eq. 13, unnormalised)
 *   (X_c|a b) = Σ_k Σ_i Σ_j c_k c_i c_j [c|ab]_{kij}                           (contracted, l.453)
 * by the closed McMurchie–Davidson route (Hermite expansion; SURVEY.md §8(c) steps 1–5), which shares
 * nothing with the Obara–Saika/HGPA recurrences (eqs. 1–4) the CUDA path is built from.
 * No blocking, fusion or reordering beyond those five steps.
 */

/* ---------------------------------------------------------------------------------------------
 * Boys function  F_m(T) = ∫_0^1 y^{2m} exp(−T y²) dy        (eq. 19; reading G11)
 *   T = 0      : 1/(2m+1)
 *   T < 120    : F_M(T) = e^{−T} Σ_{i≥0} (2T)^i / [(2M+1)(2M+3)…(2M+2i+1)]  at M = mmax (all terms
 *                positive, no cancellation), then downward F_{m−1} = (2T F_m + e^{−T})/(2m−1)
 *   T ≥ 120    : F_0 = ½√(π/T), upward F_{m+1} = (2m+1) F_m /(2T)   (dropped e^{−T} term < 1e-29 rel.)
 * ------------------------------------------------------------------------------------------- */
static void SFX(boys)(int mmax, REAL T, REAL *F)
{
    const REAL PI = (REAL)3.14159265358979323846264338327950288419716939937510L;
    if (T == (REAL)0) {
        for (int m = 0; m <= mmax; ++m) F[m] = (REAL)1 / (REAL)(2 * m + 1);
        return;
    }
    if (T < (REAL)120) {
        const REAL eT = R_EXP(-T);
        REAL term = (REAL)1 / (REAL)(2 * mmax + 1);
        REAL sum = term;
        for (int i = 1; i < 2000; ++i) {
            term *= ((REAL)2 * T) / (REAL)(2 * mmax + 2 * i + 1);
            sum += term;
            if (term < (REAL)1e-22L * sum) break;
        }
        F[mmax] = eT * sum;
        for (int m = mmax; m >= 1; --m)
            F[m - 1] = ((REAL)2 * T * F[m] + eT) / (REAL)(2 * m - 1);
        return;
    }
    F[0] = (REAL)0.5 * R_SQRT(PI / T);
    for (int m = 0; m < mmax; ++m) F[m + 1] = (REAL)(2 * m + 1) * F[m] / ((REAL)2 * T);
}

/* Per-axis Hermite expansion coefficients of a two-centre product:
 *   E_0^{00} = exp(−μQ²),  Q = A−B (this axis), μ = ζaζb/p, p = ζa+ζb
 *   E_t^{i+1,j} = E_{t−1}^{ij}/(2p) − (ζb Q/p) E_t^{ij} + (t+1) E_{t+1}^{ij}
 *   E_t^{i,j+1} = E_{t−1}^{ij}/(2p) + (ζa Q/p) E_t^{ij} + (t+1) E_{t+1}^{ij}
 * E[i][j][t], zero for t<0 or t>i+j.  Dimension LXO_LD = LXO_LMAX+1 per index pair, 2*LXO_LMAX+1 for t. */
#define LXO_LMAX 6
#define LXO_LD (LXO_LMAX + 1)
#define LXO_TD (2 * LXO_LMAX + 2)

static void SFX(hermite_E2)(int la, int lb, REAL za, REAL zb, REAL Q, REAL E[LXO_LD][LXO_LD][LXO_TD])
{
    const REAL p = za + zb, mu = za * zb / p;
    for (int i = 0; i < LXO_LD; ++i)
        for (int j = 0; j < LXO_LD; ++j)
            for (int t = 0; t < LXO_TD; ++t) E[i][j][t] = (REAL)0;
    E[0][0][0] = R_EXP(-mu * Q * Q);
    for (int i = 0; i < la; ++i)          /* raise i at j = 0 */
        for (int t = 0; t <= i + 1; ++t) {
            REAL v = -(zb * Q / p) * E[i][0][t] + (REAL)(t + 1) * E[i][0][t + 1];
            if (t > 0) v += E[i][0][t - 1] / ((REAL)2 * p);
            E[i + 1][0][t] = v;
        }
    for (int i = 0; i <= la; ++i)         /* raise j at every i */
        for (int j = 0; j < lb; ++j)
            for (int t = 0; t <= i + j + 1; ++t) {
                REAL v = (za * Q / p) * E[i][j][t] + (REAL)(t + 1) * E[i][j][t + 1];
                if (t > 0) v += E[i][j][t - 1] / ((REAL)2 * p);
                E[i][j + 1][t] = v;
            }
}

/* One-centre coefficients (step 2):  E_0^0 = 1;  E_t^{n+1} = E_{t−1}^n/(2q) + (t+1) E_{t+1}^n. */
static void SFX(hermite_E1)(int l, REAL q, REAL E[LXO_LD][LXO_TD])
{
    for (int n = 0; n < LXO_LD; ++n)
        for (int t = 0; t < LXO_TD; ++t) E[n][t] = (REAL)0;
    E[0][0] = (REAL)1;
    for (int n = 0; n < l; ++n)
        for (int t = 0; t <= n + 1; ++t) {
            REAL v = (REAL)(t + 1) * E[n][t + 1];
            if (t > 0) v += E[n][t - 1] / ((REAL)2 * q);
            E[n + 1][t] = v;
        }
}

/* Hermite Coulomb integrals (step 3):  R^n_{000} = (−2α)^n F_n(α|R|²),
 *   R^n_{t+1,u,v} = t R^{n+1}_{t−1,u,v} + R_x R^{n+1}_{t,u,v}   (likewise u with R_y, v with R_z)
 * Returns R^0_{tuv} for t+u+v ≤ L in R0[(t*(L+1)+u)*(L+1)+v].  work holds (L+1)^4 REALs. */
static void SFX(hermite_R)(int L, REAL alpha, const REAL Rv[3], REAL *work, REAL *R0)
{
    const int n1 = L + 1;
    REAL F[4 * LXO_LMAX + 1];
    SFX(boys)(L, alpha * (Rv[0] * Rv[0] + Rv[1] * Rv[1] + Rv[2] * Rv[2]), F);
#define RW(n, t, u, v) work[(((n) * n1 + (t)) * n1 + (u)) * n1 + (v)]
    REAL pw = (REAL)1;
    for (int n = 0; n <= L; ++n) { RW(n, 0, 0, 0) = pw * F[n]; pw *= (REAL)(-2) * alpha; }
    for (int s = 1; s <= L; ++s)                 /* s = t+u+v of the entry being made */
        for (int n = 0; n <= L - s; ++n)
            for (int t = 0; t <= s; ++t)
                for (int u = 0; u <= s - t; ++u) {
                    const int v = s - t - u;
                    REAL val;
                    if (t > 0) {
                        val = Rv[0] * RW(n + 1, t - 1, u, v);
                        if (t > 1) val += (REAL)(t - 1) * RW(n + 1, t - 2, u, v);
                    } else if (u > 0) {
                        val = Rv[1] * RW(n + 1, t, u - 1, v);
                        if (u > 1) val += (REAL)(u - 1) * RW(n + 1, t, u - 2, v);
                    } else {
                        val = Rv[2] * RW(n + 1, t, u, v - 1);
                        if (v > 1) val += (REAL)(v - 1) * RW(n + 1, t, u, v - 2);
                    }
                    RW(n, t, u, v) = val;
                }
    for (int t = 0; t <= L; ++t)
        for (int u = 0; u <= L - t; ++u)
            for (int v = 0; v <= L - t - u; ++v) R0[(t * n1 + u) * n1 + v] = RW(0, t, u, v);
#undef RW
}

/* Cartesian components of a shell, reading G2: for lx = l..0, for ly = l−lx..0, lz = l−lx−ly. */
static int SFX(components)(int l, int comp[][3])
{
    int n = 0;
    for (int x = l; x >= 0; --x)
        for (int y = l - x; y >= 0; --y) { comp[n][0] = x; comp[n][1] = y; comp[n][2] = l - x - y; ++n; }
    return n;
}

#define LXO_NCMAX ((LXO_LMAX + 1) * (LXO_LMAX + 2) / 2)

/* One contracted shell-set (X|ab), written as out[cx][ca][cb] (dense, row-major), steps 1–5.
 * Shell = centre[3], nprim, zeta[], coef[] (coef already holds any normalisation; reading G3). */
static void SFX(eri3_set)(int lx, const double *C, int kx, const double *zx, const double *cx_,
                          int la, const double *A, int ka, const double *za, const double *ca_,
                          int lb, const double *B, int kb, const double *zb, const double *cb_,
                          REAL *work, REAL *out)
{
    const REAL PI = (REAL)3.14159265358979323846264338327950288419716939937510L;
    const int L = lx + la + lb, n1 = L + 1;
    int cX[LXO_NCMAX][3], cA[LXO_NCMAX][3], cB[LXO_NCMAX][3];
    const int nX = SFX(components)(lx, cX), nA = SFX(components)(la, cA), nB = SFX(components)(lb, cB);
    REAL *Rwork = work;                         /* (L+1)^4 */
    REAL *R0 = Rwork + n1 * n1 * n1 * n1;       /* (L+1)^3 */
    REAL *G = R0 + n1 * n1 * n1;                /* (L+1)^3 : G_c[tuv] */
    for (int i = 0; i < nX * nA * nB; ++i) out[i] = (REAL)0;

    REAL Eab[3][LXO_LD][LXO_LD][LXO_TD];
    REAL Ec[LXO_LD][LXO_TD];
    const int lab = la + lb;
    for (int k = 0; k < kx; ++k)
        for (int i = 0; i < ka; ++i)
            for (int j = 0; j < kb; ++j) {
                const REAL q = zx[k], zi = za[i], zj = zb[j];
                const REAL p = zi + zj;
                const REAL alpha = p * q / (p + q);
                REAL Rv[3];
                for (int d = 0; d < 3; ++d) {
                    const REAL Pd = (zi * (REAL)A[d] + zj * (REAL)B[d]) / p;     /* eq. 16 */
                    Rv[d] = Pd - (REAL)C[d];                                      /* eq. 18 */
                    SFX(hermite_E2)(la, lb, zi, zj, (REAL)A[d] - (REAL)B[d], Eab[d]);
                }
                SFX(hermite_E1)(lx, q, Ec);     /* same exponent on all three axes */
                SFX(hermite_R)(L, alpha, Rv, Rwork, R0);
                const REAL pref = (REAL)2 * PI * PI * R_SQRT(PI) / (p * q * R_SQRT(p + q));
                const REAL cc = pref * (REAL)cx_[k] * (REAL)ca_[i] * (REAL)cb_[j];
                for (int ix = 0; ix < nX; ++ix) {
                    /* (ii) G_c[tuv] = Σ_{τνφ} (−1)^{τ+ν+φ} E^c_τ E^c_ν E^c_φ R^0_{t+τ,u+ν,v+φ} */
                    for (int t = 0; t <= lab; ++t)
                        for (int u = 0; u <= lab - t; ++u)
                            for (int v = 0; v <= lab - t - u; ++v) {
                                REAL s = (REAL)0;
                                for (int tt = 0; tt <= cX[ix][0]; ++tt)
                                    for (int uu = 0; uu <= cX[ix][1]; ++uu)
                                        for (int vv = 0; vv <= cX[ix][2]; ++vv) {
                                            const REAL e = Ec[cX[ix][0]][tt] * Ec[cX[ix][1]][uu] * Ec[cX[ix][2]][vv];
                                            const REAL sg = ((tt + uu + vv) & 1) ? (REAL)(-1) : (REAL)1;
                                            s += sg * e * R0[((t + tt) * n1 + (u + uu)) * n1 + (v + vv)];
                                        }
                                G[(t * n1 + u) * n1 + v] = s;
                            }
                    /* (iii) one dot product with E^{ab} per (a,b) component pair */
                    for (int ia = 0; ia < nA; ++ia)
                        for (int ib = 0; ib < nB; ++ib) {
                            REAL s = (REAL)0;
                            for (int t = 0; t <= cA[ia][0] + cB[ib][0]; ++t)
                                for (int u = 0; u <= cA[ia][1] + cB[ib][1]; ++u)
                                    for (int v = 0; v <= cA[ia][2] + cB[ib][2]; ++v)
                                        s += Eab[0][cA[ia][0]][cB[ib][0]][t] * Eab[1][cA[ia][1]][cB[ib][1]][u] *
                                             Eab[2][cA[ia][2]][cB[ib][2]][v] * G[(t * n1 + u) * n1 + v];
                            out[(ix * nA + ia) * nB + ib] += cc * s;
                        }
                }
            }
}

static size_t SFX(work_len)(int L)
{
    const size_t n1 = (size_t)L + 1;
    return n1 * n1 * n1 * n1 + 2 * n1 * n1 * n1;
}

/* Schwarz factor of an aux shell: Q_X = sqrt(max_c (X_c|X_c)), 2-centre Coulomb integral by the same
 * MD machinery: α = q q'/(q+q'), R = 0 (SURVEY.md §8(c) "Schwarz factors"). */
__attribute__((unused)) static REAL SFX(schwarz_aux)(int lx, int kx, const double *zx, const double *cx_, REAL *work)
{
    const REAL PI = (REAL)3.14159265358979323846264338327950288419716939937510L;
    const int L = 2 * lx, n1 = L + 1;
    int cX[LXO_NCMAX][3];
    const int nX = SFX(components)(lx, cX);
    REAL *Rwork = work, *R0 = work + n1 * n1 * n1 * n1;
    REAL E1[LXO_LD][LXO_TD], E2[LXO_LD][LXO_TD];
    REAL diag[LXO_NCMAX];
    for (int i = 0; i < nX; ++i) diag[i] = (REAL)0;
    const REAL zero[3] = {0, 0, 0};
    for (int k = 0; k < kx; ++k)
        for (int k2 = 0; k2 < kx; ++k2) {
            const REAL q = zx[k], q2 = zx[k2];
            SFX(hermite_E1)(lx, q, E1);
            SFX(hermite_E1)(lx, q2, E2);
            SFX(hermite_R)(L, q * q2 / (q + q2), zero, Rwork, R0);
            const REAL cc = (REAL)2 * PI * PI * R_SQRT(PI) / (q * q2 * R_SQRT(q + q2)) * (REAL)cx_[k] * (REAL)cx_[k2];
            for (int ix = 0; ix < nX; ++ix) {
                REAL s = (REAL)0;
                for (int t = 0; t <= cX[ix][0]; ++t)
                    for (int u = 0; u <= cX[ix][1]; ++u)
                        for (int v = 0; v <= cX[ix][2]; ++v)
                            for (int tt = 0; tt <= cX[ix][0]; ++tt)
                                for (int uu = 0; uu <= cX[ix][1]; ++uu)
                                    for (int vv = 0; vv <= cX[ix][2]; ++vv) {
                                        const REAL sg = ((tt + uu + vv) & 1) ? (REAL)(-1) : (REAL)1;
                                        s += E1[cX[ix][0]][t] * E1[cX[ix][1]][u] * E1[cX[ix][2]][v] * sg *
                                             E2[cX[ix][0]][tt] * E2[cX[ix][1]][uu] * E2[cX[ix][2]][vv] *
                                             R0[((t + tt) * n1 + (u + uu)) * n1 + (v + vv)];
                                    }
                diag[ix] += cc * s;
            }
        }
    REAL mx = (REAL)0;
    for (int i = 0; i < nX; ++i) if (diag[i] > mx) mx = diag[i];
    return R_SQRT(mx);
}

/* Schwarz factor of a primary shell pair: Q_ab = sqrt(max_{a,b} (a b|a b)), 4-centre diagonal; both sides
 * use E^{ab}; sum over both primitive pairs; R = P − P'. */
__attribute__((unused)) static REAL SFX(schwarz_pair)(int la, const double *A, int ka, const double *za, const double *ca_,
                              int lb, const double *B, int kb, const double *zb, const double *cb_, REAL *work)
{
    const REAL PI = (REAL)3.14159265358979323846264338327950288419716939937510L;
    const int L = 2 * (la + lb), n1 = L + 1;
    int cA[LXO_NCMAX][3], cB[LXO_NCMAX][3];
    const int nA = SFX(components)(la, cA), nB = SFX(components)(lb, cB);
    REAL *Rwork = work, *R0 = work + n1 * n1 * n1 * n1;
    REAL E1[3][LXO_LD][LXO_LD][LXO_TD], E2[3][LXO_LD][LXO_LD][LXO_TD];
    REAL diag[LXO_NCMAX * LXO_NCMAX];
    for (int i = 0; i < nA * nB; ++i) diag[i] = (REAL)0;
    for (int i = 0; i < ka; ++i)
        for (int j = 0; j < kb; ++j)
            for (int i2 = 0; i2 < ka; ++i2)
                for (int j2 = 0; j2 < kb; ++j2) {
                    const REAL p = (REAL)za[i] + (REAL)zb[j], p2 = (REAL)za[i2] + (REAL)zb[j2];
                    REAL Rv[3];
                    for (int d = 0; d < 3; ++d) {
                        const REAL P1 = ((REAL)za[i] * (REAL)A[d] + (REAL)zb[j] * (REAL)B[d]) / p;
                        const REAL P2 = ((REAL)za[i2] * (REAL)A[d] + (REAL)zb[j2] * (REAL)B[d]) / p2;
                        Rv[d] = P1 - P2;
                        SFX(hermite_E2)(la, lb, za[i], zb[j], (REAL)A[d] - (REAL)B[d], E1[d]);
                        SFX(hermite_E2)(la, lb, za[i2], zb[j2], (REAL)A[d] - (REAL)B[d], E2[d]);
                    }
                    SFX(hermite_R)(L, p * p2 / (p + p2), Rv, Rwork, R0);
                    const REAL cc = (REAL)2 * PI * PI * R_SQRT(PI) / (p * p2 * R_SQRT(p + p2)) *
                                    (REAL)ca_[i] * (REAL)cb_[j] * (REAL)ca_[i2] * (REAL)cb_[j2];
                    for (int ia = 0; ia < nA; ++ia)
                        for (int ib = 0; ib < nB; ++ib) {
                            const int tx = cA[ia][0] + cB[ib][0], ty = cA[ia][1] + cB[ib][1], tz = cA[ia][2] + cB[ib][2];
                            REAL s = (REAL)0;
                            for (int t = 0; t <= tx; ++t)
                                for (int u = 0; u <= ty; ++u)
                                    for (int v = 0; v <= tz; ++v)
                                        for (int tt = 0; tt <= tx; ++tt)
                                            for (int uu = 0; uu <= ty; ++uu)
                                                for (int vv = 0; vv <= tz; ++vv) {
                                                    const REAL sg = ((tt + uu + vv) & 1) ? (REAL)(-1) : (REAL)1;
                                                    s += E1[0][cA[ia][0]][cB[ib][0]][t] * E1[1][cA[ia][1]][cB[ib][1]][u] *
                                                         E1[2][cA[ia][2]][cB[ib][2]][v] * sg *
                                                         E2[0][cA[ia][0]][cB[ib][0]][tt] * E2[1][cA[ia][1]][cB[ib][1]][uu] *
                                                         E2[2][cA[ia][2]][cB[ib][2]][vv] *
                                                         R0[((t + tt) * n1 + (u + uu)) * n1 + (v + vv)];
                                                }
                            diag[ia * nB + ib] += cc * s;
                        }
                }
    REAL mx = (REAL)0;
    for (int i = 0; i < nA * nB; ++i) if (diag[i] > mx) mx = diag[i];
    return R_SQRT(mx);
}
