/* lx.h — C ABI of liblx: B200-native (sm_100a) 3-centre Coulomb integrals (X|ab) and integral-direct DF-J.
 *
 * Everything the hot path computes is defined by arxiv 2210.03192 (cited below as PAPER.md:<line>):
 *   (X_c|a b) = Σ_k Σ_i Σ_j c_k c_i c_j [c|ab]_{kij}                          contracted shell-set
 *   [c|ab]    = ∬ φ_c(r1) |r1−r2|⁻¹ φ_a(r2) φ_b(r2) dr1 dr2                   eq. 12, Coulomb :455
 *   φ_a(r)    = (x−A_x)^{a_x}(y−A_y)^{a_y}(z−A_z)^{a_z} exp(−ζ_a|r−A|²)      eq. 13, unnormalised
 * evaluated by the Obara–Saika/HGPA scheme of PAPER.md §2.5 (lines 104–124): Boys → [00|0]^(m) (eq. 4) → VRR1
 * (eq. 3) → VRR2 → contraction → HRR (eq. 1), and fused with the density-fitting contractions
 *   γ_X  = Σ_ab (X|ab) D_ab ,   J_ab = Σ_X (X|ab) d_X
 * through a "digestion" step that replaces the store, so the 3-centre tensor is never written.
 *
 * Conventions common to every entry point
 *   - Pointers are DEVICE pointers unless the name ends in _host.  The caller owns every buffer; the library never
 *     frees or keeps caller memory.  The only library-owned device memory is the Boys table made by lx_init().
 *   - Calls are asynchronous on `stream` (a cudaStream_t passed as void*; NULL = legacy default stream) and return
 *     before completion.  lx_shells_t structs themselves live on the HOST; their array members are device pointers
 *     (host pointers for the *_host arguments of lx_schedule_create).
 *   - Return value: LX_OK (0) or a negative LX_E* code.  Nothing throws, prints or exits.
 *   - Cartesian component order inside a shell of angular momentum l (reading G2 of DESIGN.md):
 *       for lx = l..0, for ly = l−lx..0, lz = l−lx−ly          (xx, xy, xz, yy, yz, zz for l = 2)
 *     nc(l) = (l+1)(l+2)/2.  The aux index X is Cartesian as well (reading G1).
 *   - `coef` already contains every normalisation factor; the library multiplies by coef only (reading G3,
 *     PAPER.md:439, 453).  Units: bohr / Hartree.
 *   - Compiled class range: 0 ≤ lx ≤ LX_MAX_L_AUX, 0 ≤ la, lb ≤ LX_MAX_L_PRIM; anything else → LX_EUNSUPPORTED.
 */
#ifndef LX_H
#define LX_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define LX_MAX_L_AUX 6
#define LX_MAX_L_PRIM 4

#define LX_OK 0
#define LX_EINVAL (-1)        /* null / negative / inconsistent argument                                       */
#define LX_EUNSUPPORTED (-2)  /* class outside the compiled range                                               */
#define LX_ENOMEM (-3)        /* workspace too small (see the *_workspace_bytes functions)                      */
#define LX_ECUDA (-4)         /* CUDA runtime error; text via lx_strerror(LX_ECUDA)                             */
#define LX_ENOTINIT (-5)      /* lx_init() has not been called on this device                                   */
#define LX_ELIMIT (-6)        /* problem larger than the fixed scratch of lx_eri3_batch_static                 */
#define LX_ENOTPD (-7)        /* lx_fit_solve: the metric is not (numerically) positive definite                */

/* Gaussian shell table, structure of arrays (a shell is a centre, exponents ζ, contraction
 * coefficients and l, over unnormalised primitives).  Immutable during a call. */
typedef struct {
    int32_t nshell;
    const int32_t *L;        /* [nshell]    angular momentum l                                                  */
    const int32_t *K;        /* [nshell]    contraction degree (= prim_off[i+1]-prim_off[i])                    */
    const int32_t *prim_off; /* [nshell+1]  offsets into zeta / coef                                            */
    const double *center;    /* [nshell*3]  x,y,z in bohr                                                       */
    const double *zeta;      /* [nprim]     exponents ζ                                                         */
    const double *coef;      /* [nprim]     coefficients including normalisation                                */
    const int32_t *bf_off;   /* [nshell+1]  first Cartesian basis-function index (DF calls only; may be NULL
                                            for lx_eri3_batch)                                                  */
} lx_shells_t;

/* Library state.  lx_init builds the Boys-function interpolation table (PAPER.md:132 and eq. 19:
 * F_m(x) = ∫_0^1 y^{2m} exp(−x y²) dy) on the host in long double and uploads it to `device`.  Idempotent for the same
 * device; a call with another device moves the library there (the old tables are freed; one device at a time per
 * process — the intended use is one process per GPU).  Kernel attributes (dynamic shared-memory limits) are set per
 * device at the first launch of each kernel.  lx_finalize frees the tables. */
int lx_init(int device);
int lx_finalize(void);
const char *lx_strerror(int status);
/* Version / build string of the library ("lx3 <n> sm_100a ..."), static storage. */
const char *lx_version(void);

/* lx_eri3_batch — PAPER.md §2.5 (lines 104–124), SURVEY.md §8(a) rows a1–a8.
 * Computes the full shell-sets (X|ab) for every listed primary shell pair × every listed aux shell of ONE class:
 *   out[((p*nx + x)*nc(lx) + cx)*nc(la)*nc(lb) + ca*nc(lb) + cb] = (X_cx | a_ca b_cb),
 *   a = pair_idx[2p], b = pair_idx[2p+1], X = x_idx[x];  dense, row-major, fully overwritten.
 * All aux shells listed must have L = lx and all pairs L = (la, lb): the caller's contract (not checked on the
 * device).  la < lb is legal: the library swaps the roles of the two shells internally and still writes [ca][cb] in
 * the caller's order.  No screening is applied (reading G13).  Degenerate geometry (A = B, P = C, all centres
 * equal, the same shell twice in a pair) is legal (reading G15).
 *   x_idx [nx], pair_idx [npair*2]: device int32.   out: device double, npair*nx*nc(lx)*nc(la)*nc(lb) elements.
 *   workspace: device scratch of at least lx_eri3_workspace_bytes(...) bytes (primitive-pair data, row a1).
 * nx == 0 or npair == 0 is a no-op returning LX_OK.
 * Errors: LX_EINVAL (null pointer with non-zero count, negative count), LX_EUNSUPPORTED, LX_ENOMEM, LX_ENOTINIT,
 * LX_ECUDA.
 * Workspace contract: the record stride of the primitive-pair data is workspace_bytes / npair, so the workspace must be
 * sized with kmax_pair >= max K_a*K_b over the listed pairs.  The lists live on the device, so the call itself cannot
 * see a violation without synchronising: if a listed pair has more primitive pairs than the stride, nothing is read
 * or written out of bounds, every integral of that pair comes back as NaN, and lx_async_status() reports LX_ENOMEM.
 * With LX_CHECK=1 in the environment (read by lx_init; debug aid) the call first validates on the device, and
 * synchronises: index range and class conformity of x_idx / pair_idx (LX_EINVAL) and the stride (LX_ENOMEM), and
 * launches nothing if the check fails. */
int lx_eri3_batch(int lx, int la, int lb, const lx_shells_t *aux, const lx_shells_t *prim,
                  const int32_t *x_idx, int nx, const int32_t *pair_idx, int npair, double *out,
                  void *workspace, size_t workspace_bytes, void *stream);

/* Status of the asynchronous work issued since the last call of this function: LX_OK, LX_ENOMEM (a pair exceeded the
 * workspace stride, see lx_eri3_batch) or LX_EINVAL (LX_CHECK=1 found an index out of range or a shell of the wrong
 * class).  Reads one word from the device (synchronises with the legacy stream; the caller synchronises its own
 * streams first) and clears it. */
int lx_async_status(void);

/* Workspace size for lx_eri3_batch: kmax_pair = max over listed pairs of K_a*K_b (contraction degrees). */
size_t lx_eri3_workspace_bytes(int lx, int la, int lb, int nx, int npair, int kmax_pair);

/* Schwarz factors on the GPU (SURVEY.md §8(c) "Schwarz factors", §8(f) NEXT-2; "identical screening"):
 *     q_aux[X]   = sqrt(max_c (X_c|X_c))        for every shell of `aux`            (2-centre Coulomb integrals)
 *     q_pair[k]  = sqrt(max_{a,b} (a b|a b))    for every listed primary shell pair  (diagonal 4-centre integrals)
 * so that |(X_c|a b)| <= q_aux[X] q_pair[k] for every component (Cauchy-Schwarz).  These are the arrays
 * lx_schedule_create takes.  HOST in, HOST out: every array member of the table, pair_idx [npair*2] and the result
 * are host pointers; the call uploads the table, evaluates the factors on the device (Hermite-Gaussian expansion of the
 * pair densities, one thread per shell / shell pair, FP64) and returns after the result is complete.  Run once per
 * basis; not part of the per-iteration path.  Accuracy: relative error <= 1e-12 against the long-double oracle
 * (tests/test_gpu_schwarz.py), so a screening decision q_aux*q_pair < tau can differ from one taken with exact factors
 * only for products within 1e-12 (relative) of tau.
 * Errors: LX_EINVAL, LX_EUNSUPPORTED (L outside the compiled range), LX_ENOTINIT, LX_ECUDA. */
int lx_schwarz_aux_host(const lx_shells_t *aux_host, double *q_aux_host);
int lx_schwarz_pair_host(const lx_shells_t *prim_host, const int32_t *pair_idx_host, int npair, double *q_pair_host);

/* The steps after gamma and before J (SURVEY.md §8(f) NEXT-2, second half; PAPER.md:21 "robust" fit, :365 the two passes
 * of density fitting):  V_XY = (X|Y) two-centre Coulomb metric of the aux basis,  d = V^-1 gamma  fit coefficients.
 *
 * lx_metric_2c:  V[(bf(X)+c)*ld + bf(Y)+c'] = (X_c|Y_c') = ∬ X_c(r1) Y_c'(r2) / r12  for every pair of aux shells, Cartesian
 *   components in the library's order, bf(X) = Σ_{X'<X} nc(L_X') (aux_host->bf_off, if given, must say the same).
 *   aux_host: HOST shell table (uploaded inside; L <= LX_MAX_L_AUX, any contraction degree).  V_dev: DEVICE, caller-owned,
 *   [naux_bf rows, leading dimension ld >= naux_bf]; every entry of the naux_bf x naux_bf block is written (nothing has to
 *   be cleared) and the result is exactly symmetric.  Evaluated by Hermite expansion of each shell about its own centre
 *   (one thread per shell pair; lx_schwarz.cu), the same route as the Schwarz factors.  Synchronous.
 *   Errors: LX_ENOTINIT, LX_EINVAL (null table / V_dev, ld too small, bf_off not Cartesian-cumulative, K inconsistent),
 *   LX_EUNSUPPORTED (L out of range), LX_ECUDA.
 *
 * lx_fit_solve:  rhs <- V^-1 rhs by Cholesky factorisation (V = L L^T) and two triangular solves.
 *   V_dev: DEVICE [n, ld], symmetric positive definite; OVERWRITTEN: one triangle holds the factor afterwards (the other
 *   keeps V).  With factored != 0 the array is taken to hold that factor already (an earlier call on the same V) and only
 *   the solves run — the usual case of one metric and a new gamma per SCF iteration.  rhs_dev: DEVICE, nrhs vectors of
 *   length n, each contiguous (vector r at rhs_dev + r*n), overwritten by the solutions; nrhs = 0 only factorises.
 *   The factorisation is cuSOLVER's potrf (a plain library routine, opened with dlopen at the first call); the triangular
 *   solves are kernels of this library (lx_fit.cu: blocked substitution, 2 n/64 launches per right-hand side, the factor
 *   read once each way).  Synchronous; allocates the factorisation workspace / about n + n/32 doubles for the duration of the
 *   call.
 *   Errors: LX_ENOTINIT, LX_EINVAL, LX_ENOTPD (a leading minor of V is not positive definite: linearly dependent aux
 *   functions), LX_EUNSUPPORTED (factorising call and cuSOLVER cannot be loaded), LX_ENOMEM, LX_ECUDA. */
int lx_metric_2c(const lx_shells_t *aux_host, double *V_dev, long long ld);
int lx_fit_solve(double *V_dev, long long ld, int n, double *rhs_dev, int nrhs, int factored);

/* Schedule — SURVEY.md §8(a) row a0; PAPER.md:54 (batches per class), :365 ("identical screening").
 * Built once per basis on the HOST from host copies of the shell tables.  Buckets aux shells by L and shell pairs
 * by (La, Lb) (pairs with La < Lb are stored swapped), orders every bucket by contraction degree and then by
 * Schwarz factor descending, so that for every pair the aux shells that survive
 *        q_aux[X] * q_pair[p] >= tau          (evaluated in double; a set with the product < tau is skipped)
 * form a prefix of the aux bucket; stores the prefix length per (pair, lx).  q_aux_host [aux.nshell] and q_pair_host
 * [npair] are Schwarz factors Q_X = sqrt(max (X|X)), Q_ab = sqrt(max (ab|ab)) supplied by the caller; if either is
 * NULL no screening is applied.  pair_idx_host [npair*2] lists the unique shell pairs (a,b) to visit; a pair with
 * a == b is weighted once, a != b stands for both (a,b) and (b,a) (reading G16).
 * The schedule owns small device copies of its index lists (freed by lx_schedule_destroy). */
typedef struct lx_schedule lx_schedule_t;
int lx_schedule_create(const lx_shells_t *aux_host, const lx_shells_t *prim_host, const double *q_aux_host,
                       const double *q_pair_host, const int32_t *pair_idx_host, int npair, double tau,
                       lx_schedule_t **out);
int lx_schedule_destroy(lx_schedule_t *s);
/* Number of unscreened shell-sets / Cartesian integrals one DF pass evaluates (reading G19). */
int64_t lx_schedule_num_sets(const lx_schedule_t *s);
int64_t lx_schedule_num_integrals(const lx_schedule_t *s);
/* Workspace (bytes) needed by lx_df_gamma / lx_df_J with this schedule. */
size_t lx_df_workspace_bytes(const lx_schedule_t *s);

/* lx_df_gamma — SURVEY.md §8(a) row a9 (PAPER.md:283 digestion callable, :365).
 *   gamma[bf(X)+cx] = Σ_{pairs p=(a,b)} f_p Σ_{ca,cb} (X_cx|a_ca b_cb) D[(bf(a)+ca)*ldD + bf(b)+cb],
 *   f_p = 2 if a != b else 1, over the unscreened sets of the schedule.  D (nbf×nbf, leading dimension ldD) is read
 *   as symmetric.  gamma [naux_bf] is overwritten.  FP64 atomics are used across thread blocks, so the last bits
 *   may differ from run to run (reading G14).
 * lx_df_J — row a10.
 *   J[(bf(a)+ca)*ldJ + bf(b)+cb] = Σ_{X,cx} (X_cx|a_ca b_cb) d[bf(X)+cx], mirrored to (b,a); J (nbf×nbf) is
 *   overwritten in full (blocks of unlisted or fully screened pairs become zero).
 * aux / prim: the same tables the schedule was built from, with DEVICE array members (bf_off required).
 * Stream semantics: the class launches of a pass are independent, so where they are small (fewer than 2 M shell-sets per
 * launch on average) the library spreads them over a few internal side
 * streams (environment LX_DF_STREAMS, read by lx_init, default 4 including `stream`; 1 = `stream` only) that are forked from
 * `stream` after the pre-pass and joined to it before the call returns: work queued on `stream` after the call sees the finished
 * result, as with a single stream.  The two DF calls are not re-entrant (one call at a time per process). */
int lx_df_gamma(const lx_schedule_t *s, const lx_shells_t *aux, const lx_shells_t *prim, const double *D, int ldD,
                double *gamma, void *workspace, size_t workspace_bytes, void *stream);
int lx_df_J(const lx_schedule_t *s, const lx_shells_t *aux, const lx_shells_t *prim, const double *d, double *J,
            int ldJ, void *workspace, size_t workspace_bytes, void *stream);

/* lx_eri3_batch_static — lx_eri3_batch for callers that must not allocate and have no workspace to pass (code under CUDA
 * graph capture, tight serving loops, harnesses that forbid cudaMalloc).  Same operation, same kernels, same result and
 * argument meaning as lx_eri3_batch, but the primitive-pair data (row a1: 48 bytes per primitive pair) lives in a fixed
 * array in device memory that the library itself holds: LX_STATIC_SCRATCH_BYTES = 4 MiB on EVERY GPU that loads the
 * library, from the first use of the library on that GPU until the process exits.
 *   limit:     npair * kmax_pair * 48 bytes <= LX_STATIC_SCRATCH_BYTES (87 381 primitive pairs, e.g. 9 709 shell pairs of
 *              K_a K_b = 9); beyond it the call returns LX_ELIMIT and launches nothing.  kmax_pair >= max K_a K_b over
 *              the listed pairs (explicit here; a pair above it comes back as NaN and lx_async_status() says LX_ENOMEM).
 *   allocates: nothing — no cudaMalloc / cudaFree / allocating library routine; lx_init(device), which must have been
 *              called, has looked up the array's device address.  The first launch of a class kernel in a process loads
 *              its code and sets its shared-memory attribute (CUDA lazy loading): run each class once before a capture.
 *   checks:    the LX_CHECK=1 validation pass of lx_eri3_batch (it synchronises) is not run here; lx_async_status() works as usual.
 *   sharing:   every call uses the SAME array and leaves its contents behind.  Nothing in it has to start at zero: a call
 *              rewrites every record it reads.  Calls that overlap on the GPU (different streams, or another process
 *              thread) RACE on it: issue them on one stream, or order them with events.  lx_eri3_batch with caller
 *              workspaces is the entry point for concurrent calls. */
#define LX_STATIC_SCRATCH_BYTES (4u << 20)
size_t lx_static_scratch_bytes(void);
int lx_eri3_batch_static(int lx, int la, int lb, const lx_shells_t *aux, const lx_shells_t *prim,
                         const int32_t *x_idx, int nx, const int32_t *pair_idx, int npair, int kmax_pair,
                         double *out, void *stream);

/* Host-buffer convenience path (used for the end-to-end measurement): same result as lx_eri3_batch but every
 * array member of aux/prim, x_idx, pair_idx and out are HOST pointers; the call allocates device scratch, copies
 * in, runs, copies out and synchronises.  Returns after `out_host` is complete. */
int lx_eri3_batch_host(int lx, int la, int lb, const lx_shells_t *aux_host, const lx_shells_t *prim_host,
                       const int32_t *x_idx_host, int nx, const int32_t *pair_idx_host, int npair,
                       double *out_host);

/* Boys function F_m(T), m = 0..mmax, for n values of T — the device routine the integral kernels use (row a2),
 * exported for the accuracy sweep.  T [n] and out [n*(mmax+1)] are device pointers; mmax <= 18. */
int lx_boys(const double *T, int n, int mmax, double *out, void *stream);

/* Measurement helper: sustained FP64 FMA rate of the device (TFLOP/s, FMA = 2 flops) from a register-resident chain
 * kernel (8 independent DFMA chains per thread, 8 blocks x 256 threads per SM, `iters` x 64 FMAs per thread), best of
 * 5 timed launches.  This is the measured denominator of the FP64-pipe roofline; synchronises. */
int lx_fp64_probe(int iters, double *tflops_host);

/* Row a6 of the path (HGPA step 5): Cartesian -> real solid-harmonic transform of the
 * auxiliary index of finished shell-sets,
 *     out[set][m][r] = sum_c S_l[m][c] in[set][c][r],   set < nsets, m = 0..2l, c < nc(l), r < nab,
 * i.e. `in` is the output of lx_eri3_batch viewed as [npair*nx][nc(lx)][nc(la)*nc(lb)] and `out` holds (X_m|ab) for the
 * pure functions S_lm, m = -l..l in this order (reading G1: the paper's aux functions are solid harmonics).  S_lm are the
 * real solid harmonics in Racah normalisation (S_l0 = r^l P_l(cos theta); S_20 = z^2 - x^2/2 - y^2/2), each a linear
 * combination of the Cartesian components of degree l (ABI order, reading G2).  Device pointers, `in != out`, the caller
 * owns both; asynchronous on `stream`.  LX_EUNSUPPORTED for l > LX_MAX_L_AUX, LX_EINVAL for null / aliased buffers. */
int lx_cart_to_pure(int lx, int64_t nsets, int nab, const double *in, double *out, void *stream);

/* (X_m|ab) for SOLID-HARMONIC auxiliary functions (the paper's own target (ab|c); SURVEY.md §8(f)
 * NEXT-1): same arguments as lx_eri3_batch plus kmax_pair (largest K_a*K_b of the listed pairs), and
 *     out[npair][nx][2lx+1][nc(la)][nc(lb)],  m = -lx..lx.
 * Classes served by the team and chain kernels with lx >= 2 run fused: for a pure ket eq. 2 is exact after
 * projection, so only the level-0 chain targets are evaluated and the solid-harmonic matrix is applied in the epilogue.
 * Other classes evaluate the Cartesian shell-sets into the workspace and apply lx_cart_to_pure.  The workspace must hold
 * lx_eri3_pure_workspace_bytes(...) bytes (LX_ENOMEM otherwise); everything else as for lx_eri3_batch. */
int lx_eri3_batch_pure(int lx, int la, int lb, const lx_shells_t *aux, const lx_shells_t *prim, const int32_t *x_idx,
                       int nx, const int32_t *pair_idx, int npair, int kmax_pair, double *out, void *workspace,
                       size_t workspace_bytes, void *stream);
size_t lx_eri3_pure_workspace_bytes(int lx, int la, int lb, int nx, int npair, int kmax_pair);

/* The matrix S_l used by lx_cart_to_pure, (2l+1) x nc(l) row-major, into HOST memory (no device needed). */
int lx_solid_matrix(int l, double *matrix_host);

/* Which kernel template serves a class: "team" (register-only chain form, lx_team.cuh), "chain" (warp-specialised
 * chain form, lx_chain_kernel.cuh), "owner" (one owner warp per ket component, lx_owner.cuh), "slab" (the same for La+Lb = 6
 * with slab-wise VRR1 and HRR, lx_slab.cuh), "lane" (bra component per lane, lx_lane.cuh) or "group" (shared-memory,
 * lx_group.cuh); "" if the class is outside the compiled range.  Static storage.  For reports only.
 * Some classes have two families and choose by the contraction degree of the launch ("K-aware
 * dispatch"): lx_kernel_family_k takes the bound K_a K_b K_x the caller knows for the launch (what lx_eri3_batch derives from
 * its K stride, the DF schedule from its buckets); kmax <= 0 = unknown.  lx_kernel_family(lx, la, lb) is the unknown case.
 * Builds with -DLX_TUNING read LX_FAMILY=team|chain|lane|owner once and force the named family where a class has it. */
const char *lx_kernel_family(int lx, int la, int lb);
const char *lx_kernel_family_k(int lx, int la, int lb, int kmax);

/* Number of kernel launches the library has issued since lx_init (for the bench's `gpu_launches` claim). */
int64_t lx_launch_count(void);

#ifdef __cplusplus
}
#endif
#endif /* LX_H */
