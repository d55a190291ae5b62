/* ORACLE — TEST INFRASTRUCTURE ONLY.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may load this library.  It shares no code with the CUDA path.
 *
 * md_eri3.c: exported entry points of the McMurchie–Davidson CPU oracle for 3-centre Coulomb integrals
 * (X|ab) over contracted Cartesian Gaussian shells (Appendix A eqs. 12–19) and the
 * density-fitting contractions built on them:
 *     γ_X  = Σ_ab (X|ab) D_ab        J_ab = Σ_X (X|ab) d_X
 * Two instantiations of md_impl.h: `_ld` (long double, used for parity) and `_d` (double, used only for the
 * timed CPU baseline).  Inputs and outputs are double arrays; `_ld` rounds once, on output.
 *
 * Shell tables are SoA (same meaning as include/lx.h, restated here, not shared): L[n], prim_off[n+1],
 * center[3n], zeta[nprim], coef[nprim] (coef includes any normalisation), bf_off[n+1] for the DF calls.
 * Layouts: eri3 out[pair][x][cx][ca][cb]; component order lx = l..0, ly = l−lx..0 (reading G2).
 *
 * Parity pins: tests/test_oracle_*.py (closed forms, worked example, exact identities, brute-force
 * quadrature, symmetry, far field).  Nothing here is "parity unpinned".
 */
#include <math.h>
#include <stddef.h>
#include <stdint.h>
#include <stdlib.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define REAL long double
#define SFX(n) n##_ld
#define R_EXP expl
#define R_SQRT sqrtl
#define R_FABS fabsl
#include "md_impl.h"
#undef REAL
#undef SFX
#undef R_EXP
#undef R_SQRT
#undef R_FABS
#undef LXO_LMAX
#undef LXO_LD
#undef LXO_TD
#undef LXO_NCMAX

#define REAL double
#define SFX(n) n##_d
#define R_EXP exp
#define R_SQRT sqrt
#define R_FABS fabs
#include "md_impl.h"
#undef REAL
#undef SFX

static int nc(int l) { return (l + 1) * (l + 2) / 2; }

int lxo_max_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* F_m(T), m = 0..mmax, long double in and out (for the 25-digit pins). */
void lxo_boys_ld(int mmax, long double T, long double *F) { boys_ld(mmax, T, F); }
void lxo_boys_d(int mmax, double T, double *F) { boys_d(mmax, T, F); }

typedef struct {
    const int32_t *L, *prim_off;
    const double *center, *zeta, *coef;
} tab_t;

#define ERI3_BATCH(SUF, RT)                                                                                   \
    int lxo_eri3_batch_##SUF(int lx, int la, int lb, const int32_t *xL, const int32_t *xoff, const double *xc, \
                             const double *xz, const double *xco, const int32_t *pL, const int32_t *poff,      \
                             const double *pc, const double *pz, const double *pco, const int32_t *x_idx,      \
                             int nx, const int32_t *pair_idx, int npair, double *out)                         \
    {                                                                                                         \
        const int nint = nc(lx) * nc(la) * nc(lb);                                                            \
        int bad = 0;                                                                                          \
        _Pragma("omp parallel")                                                                               \
        {                                                                                                     \
            RT *work = (RT *)malloc(sizeof(RT) * work_len_##SUF(lx + la + lb));                               \
            RT *buf = (RT *)malloc(sizeof(RT) * (size_t)nint);                                                \
            _Pragma("omp for schedule(dynamic)")                                                              \
            for (int ip = 0; ip < npair; ++ip) {                                                              \
                const int a = pair_idx[2 * ip], b = pair_idx[2 * ip + 1];                                     \
                if (pL[a] != la || pL[b] != lb) { bad = 1; continue; }                                        \
                for (int ix = 0; ix < nx; ++ix) {                                                             \
                    const int x = x_idx[ix];                                                                  \
                    if (xL[x] != lx) { bad = 1; continue; }                                                   \
                    eri3_set_##SUF(lx, xc + 3 * x, xoff[x + 1] - xoff[x], xz + xoff[x], xco + xoff[x],        \
                                   la, pc + 3 * a, poff[a + 1] - poff[a], pz + poff[a], pco + poff[a],        \
                                   lb, pc + 3 * b, poff[b + 1] - poff[b], pz + poff[b], pco + poff[b],        \
                                   work, buf);                                                                \
                    double *o = out + ((size_t)ip * nx + ix) * nint;                                          \
                    for (int i = 0; i < nint; ++i) o[i] = (double)buf[i];                                     \
                }                                                                                             \
            }                                                                                                 \
            free(work); free(buf);                                                                            \
        }                                                                                                     \
        return bad ? -1 : 0;                                                                                  \
    }
ERI3_BATCH(ld, long double)
ERI3_BATCH(d, double)

/* Schwarz factors (long double inside, double out): q_aux[naux_shell], q_pair[npair]. */
void lxo_schwarz_aux(int n, const int32_t *xL, const int32_t *xoff, const double *xz, const double *xco, double *q)
{
#pragma omp parallel
    {
        long double *work = (long double *)malloc(sizeof(long double) * work_len_ld(4 * 6));
#pragma omp for schedule(dynamic)
        for (int x = 0; x < n; ++x)
            q[x] = (double)schwarz_aux_ld(xL[x], xoff[x + 1] - xoff[x], xz + xoff[x], xco + xoff[x], work);
        free(work);
    }
}

void lxo_schwarz_pair(const int32_t *pL, const int32_t *poff, const double *pc, const double *pz,
                      const double *pco, const int32_t *pair_idx, int npair, double *q)
{
#pragma omp parallel
    {
        long double *work = (long double *)malloc(sizeof(long double) * work_len_ld(4 * 6));
#pragma omp for schedule(dynamic)
        for (int ip = 0; ip < npair; ++ip) {
            const int a = pair_idx[2 * ip], b = pair_idx[2 * ip + 1];
            q[ip] = (double)schwarz_pair_ld(pL[a], pc + 3 * a, poff[a + 1] - poff[a], pz + poff[a], pco + poff[a],
                                            pL[b], pc + 3 * b, poff[b + 1] - poff[b], pz + poff[b], pco + poff[b], work);
        }
        free(work);
    }
}

/* Density-fitting contractions over unique shell pairs (reading G16): for every listed pair (a,b) and every
 * aux shell X with  q_aux[X]*q_pair[ip] >= tau  (evaluated in double; a skipped set contributes exactly 0):
 *   gamma[bf(X)+cx]        += f Σ_{ca,cb} (cx|ca cb) D[bf(a)+ca, bf(b)+cb],   f = 2 if a != b else 1
 *   J[bf(a)+ca, bf(b)+cb]  += Σ_{X,cx} (cx|ca cb) d[bf(X)+cx]                  and mirrored to (b,a)
 * gamma may be NULL or J may be NULL to skip that output.  x_sel (n_xsel) restricts the aux shells visited
 * (NULL = all); p_sel likewise for pairs — used for the sampled parity/timing runs of config 5.
 * n_sets_out counts the unscreened shell-sets, n_int_out the Cartesian integrals in them. */
#define DF_FUN(SUF, RT)                                                                                        \
    int lxo_df_##SUF(int nxs, const int32_t *xL, const int32_t *xoff, const double *xc, const double *xz,      \
                     const double *xco, const int32_t *xbf, const int32_t *pL, const int32_t *poff,            \
                     const double *pc, const double *pz, const double *pco, const int32_t *pbf,                \
                     const int32_t *pair_idx, int npair, const double *q_aux, const double *q_pair,           \
                     double tau, const double *D, int ldD, const double *dvec, double *gamma, double *J,       \
                     int ldJ, const int32_t *x_sel, int n_xsel, const int32_t *p_sel, int n_psel,              \
                     int64_t *n_sets_out, int64_t *n_int_out)                                                  \
    {                                                                                                          \
        const int naux_bf = xbf[nxs];                                                                          \
        const int NP = p_sel ? n_psel : npair;                                                                 \
        const int NX = x_sel ? n_xsel : nxs;                                                                   \
        int64_t nsets = 0, nints = 0;                                                                          \
        _Pragma("omp parallel reduction(+ : nsets, nints)")                                                    \
        {                                                                                                      \
            RT *work = (RT *)malloc(sizeof(RT) * work_len_##SUF(3 * 6));                                       \
            RT *buf = (RT *)malloc(sizeof(RT) * 28 * 28 * 28);                                                 \
            RT *gloc = gamma ? (RT *)calloc((size_t)naux_bf, sizeof(RT)) : NULL;                               \
            _Pragma("omp for schedule(dynamic)")                                                               \
            for (int jp = 0; jp < NP; ++jp) {                                                                  \
                const int ip = p_sel ? p_sel[jp] : jp;                                                         \
                const int a = pair_idx[2 * ip], b = pair_idx[2 * ip + 1];                                      \
                const int la = pL[a], lb = pL[b], na = nc(la), nb = nc(lb);                                    \
                const RT f = (a != b) ? (RT)2 : (RT)1;                                                         \
                RT Jblk[28 * 28];                                                                              \
                for (int i = 0; i < na * nb; ++i) Jblk[i] = (RT)0;                                             \
                for (int jx = 0; jx < NX; ++jx) {                                                              \
                    const int x = x_sel ? x_sel[jx] : jx;                                                      \
                    if (q_aux && q_pair && q_aux[x] * q_pair[ip] < tau) continue;                              \
                    const int lx = xL[x], nxc = nc(lx);                                                        \
                    eri3_set_##SUF(lx, xc + 3 * x, xoff[x + 1] - xoff[x], xz + xoff[x], xco + xoff[x],         \
                                   la, pc + 3 * a, poff[a + 1] - poff[a], pz + poff[a], pco + poff[a],         \
                                   lb, pc + 3 * b, poff[b + 1] - poff[b], pz + poff[b], pco + poff[b],         \
                                   work, buf);                                                                 \
                    nsets += 1; nints += (int64_t)nxc * na * nb;                                               \
                    for (int cx = 0; cx < nxc; ++cx)                                                           \
                        for (int ca = 0; ca < na; ++ca)                                                        \
                            for (int cb = 0; cb < nb; ++cb) {                                                  \
                                const RT v = buf[(cx * na + ca) * nb + cb];                                    \
                                if (gloc) gloc[xbf[x] + cx] += f * v * (RT)D[(size_t)(pbf[a] + ca) * ldD + pbf[b] + cb]; \
                                if (J) Jblk[ca * nb + cb] += v * (RT)dvec[xbf[x] + cx];                        \
                            }                                                                                  \
                }                                                                                              \
                if (J)                                                                                         \
                    for (int ca = 0; ca < na; ++ca)                                                            \
                        for (int cb = 0; cb < nb; ++cb) {                                                      \
                            J[(size_t)(pbf[a] + ca) * ldJ + pbf[b] + cb] = (double)Jblk[ca * nb + cb];         \
                            J[(size_t)(pbf[b] + cb) * ldJ + pbf[a] + ca] = (double)Jblk[ca * nb + cb];         \
                        }                                                                                      \
            }                                                                                                  \
            if (gloc) {                                                                                        \
                _Pragma("omp critical")                                                                        \
                for (int i = 0; i < naux_bf; ++i) gamma[i] += (double)gloc[i];                                 \
                free(gloc);                                                                                    \
            }                                                                                                  \
            free(work); free(buf);                                                                             \
        }                                                                                                      \
        if (n_sets_out) *n_sets_out = nsets;                                                                   \
        if (n_int_out) *n_int_out = nints;                                                                     \
        return 0;                                                                                              \
    }
DF_FUN(ld, long double)
DF_FUN(d, double)
