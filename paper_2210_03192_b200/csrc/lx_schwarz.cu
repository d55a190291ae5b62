// lx_schwarz.cu — Schwarz factors and the two-centre metric V_XY = (X|Y) on the GPU (PAPER.md:365
// "identical screening", :21 the fit metric):
//     Q_X  = sqrt(max_c (X_c|X_c))          2-centre Coulomb integrals of an aux shell with itself
//     Q_ab = sqrt(max_{a,b} (a b|a b))      diagonal 4-centre integrals of a primary shell pair
// so that |(X|ab)| <= Q_X Q_ab for every component and a shell-set with Q_X Q_ab < tau can be skipped.
//
// Method (written for this library): a product of Cartesian Gaussians is expanded in Hermite Gaussians Λ_tuv about the
// product centre P (coefficients E_t^{ij} per axis, three-term recurrences in i and j), and the Coulomb integral of two
// Hermite Gaussians is (−1)^{t'+u'+v'} R_{t+t',u+u',v+v'} with R^n_{000} = (−2α)^n F_n(α|PP'|²) and
// R^n_{t+1,u,v} = t R^{n+1}_{t−1,u,v} + X R^{n+1}_{t,u,v}.  This is NOT the Obara–Saika route of the class kernels: the
// factors are a side input of the path (a0, the schedule), only the diagonal is needed, and one thread per shell pair
// with its tables in local memory is enough — the pass over all 3.3 M pairs of config 5 takes a fraction of a second.
// The R table is built in place from the highest auxiliary order down (descending (t,u,v) order keeps the operands of
// order n+1 alive until they have been read).  The Boys function is the library's own table routine (lx_common.cuh).
#include <algorithm>
#include <vector>

#include "lx_common.cuh"
#include "lx_state.h"

namespace lx {

// E_t^{ij}, t <= i+j <= LI+LJ, of (x−A)^i (x−B)^j exp(−p (x−P)²) [the exponential factor exp(−μ AB²) kept outside]:
// E[(i*(LJ+1)+j)*(LI+LJ+1) + t].  pa = P−A, pb = P−B, o2p = 1/(2p).
template <int LI, int LJ>
__device__ void hermite_pair(double pa, double pb, double o2p, double *E) {
    constexpr int NT = LI + LJ + 1;
    for (int n = 0; n < (LI + 1) * (LJ + 1) * NT; ++n) E[n] = 0.0;
    E[0] = 1.0;
    for (int i = 0; i <= LI; ++i)
        for (int j = 0; j <= LJ; ++j) {
            if (i == 0 && j == 0) continue;
            // raise j from (i, j−1) if j > 0, else raise i from (i−1, 0)
            const bool rj = j > 0;
            const double *src = E + ((rj ? i : i - 1) * (LJ + 1) + (rj ? j - 1 : 0)) * NT;
            double *dst = E + (i * (LJ + 1) + j) * NT;
            const double x = rj ? pb : pa;
            for (int t = 0; t <= i + j; ++t) {
                double v = x * src[t];
                if (t > 0) v += o2p * src[t - 1];
                if (t + 1 <= i + j - 1) v += (double)(t + 1) * src[t + 1];
                dst[t] = v;
            }
        }
}

// R^0_{tuv}, t+u+v <= L, into R[(t*N1 + u)*N1 + v], N1 = L+1; X = P − P', al = pp'/(p+p').
template <int L>
__device__ void hermite_coulomb(const double *__restrict__ boys_tab, double al, const double (&X)[3], double *R) {
    constexpr int N1 = L + 1;
    double F[L + 1];
    boys_all<L>(boys_tab, al * (X[0] * X[0] + X[1] * X[1] + X[2] * X[2]), F);
    double sc = 1.0;                       // (−2α)^n
    double pw[L + 1];
    for (int n = 0; n <= L; ++n) { pw[n] = sc * F[n]; sc *= -2.0 * al; }
    R[0] = pw[L];
    for (int n = L - 1; n >= 0; --n) {
        const int top = L - n;             // orders n+1 hold t+u+v <= top−1
        for (int t = top; t >= 0; --t)
            for (int u = top - t; u >= 0; --u)
                for (int v = top - t - u; v >= 0; --v) {
                    double r;
                    if (t > 0) {
                        r = X[0] * R[((t - 1) * N1 + u) * N1 + v];
                        if (t > 1) r += (double)(t - 1) * R[((t - 2) * N1 + u) * N1 + v];
                    } else if (u > 0) {
                        r = X[1] * R[(u - 1) * N1 + v];
                        if (u > 1) r += (double)(u - 1) * R[(u - 2) * N1 + v];
                    } else if (v > 0) {
                        r = X[2] * R[v - 1];
                        if (v > 1) r += (double)(v - 1) * R[v - 2];
                    } else {
                        r = pw[n];
                    }
                    R[(t * N1 + u) * N1 + v] = r;
                }
    }
}

__device__ __forceinline__ void cart_powers(int l, int idx, int (&pw)[3]) {
    int i = 0;
    while ((i + 1) * (i + 2) / 2 <= idx) ++i;     // i = y + z (order G2)
    pw[2] = idx - i * (i + 1) / 2;
    pw[1] = i - pw[2];
    pw[0] = l - i;
}

// One thread per listed pair of class (LA, LB); pairs[2k], pairs[2k+1] any order of the two shells; q[slot[k]] out.
template <int LA, int LB>
__global__ void __launch_bounds__(64)
schwarz_pair_kernel(DevShells prim, const int32_t *__restrict__ pairs, const int32_t *__restrict__ slot, int n,
                    const double *__restrict__ boys_tab, double *__restrict__ q) {
    constexpr int L = 2 * (LA + LB), N1 = L + 1, NT = LA + LB + 1, NE = (LA + 1) * (LB + 1) * NT;
    constexpr int NA = nc(LA), NB = nc(LB);
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n) return;
    int a = pairs[2 * k], b = pairs[2 * k + 1];
    if (prim.L[a] < prim.L[b]) { const int t = a; a = b; b = t; }
    const int Ka = prim.K[a], Kb = prim.K[b], oa = prim.prim_off[a], ob = prim.prim_off[b];
    double A[3], B[3], AB[3], r2 = 0.0;
    for (int d = 0; d < 3; ++d) {
        A[d] = prim.center[3 * a + d];
        B[d] = prim.center[3 * b + d];
        AB[d] = A[d] - B[d];
        r2 += AB[d] * AB[d];
    }
    double E1[3][NE], E2[3][NE], R[N1 * N1 * N1], diag[NA * NB];
    for (int i = 0; i < NA * NB; ++i) diag[i] = 0.0;
    const int nq = Ka * Kb;
    for (int ij = 0; ij < nq; ++ij) {
        const int i = ij / Kb, j = ij - i * Kb;
        const double za = prim.zeta[oa + i], zb = prim.zeta[ob + j], p = za + zb, ip = 1.0 / p;
        const double w1 = prim.coef[oa + i] * prim.coef[ob + j] * exp(-za * zb * ip * r2);
        double P1[3];
        for (int d = 0; d < 3; ++d) {
            P1[d] = (za * A[d] + zb * B[d]) * ip;
            hermite_pair<LA, LB>(-zb * ip * AB[d], za * ip * AB[d], 0.5 * ip, E1[d]);
        }
        for (int kl = 0; kl <= ij; ++kl) {             // (ij|kl) = (kl|ij) on the diagonal: off-diagonal pairs count twice
            const int i2 = kl / Kb, j2 = kl - i2 * Kb;
            const double za2 = prim.zeta[oa + i2], zb2 = prim.zeta[ob + j2], p2 = za2 + zb2, ip2 = 1.0 / p2;
            const double w2 = prim.coef[oa + i2] * prim.coef[ob + j2] * exp(-za2 * zb2 * ip2 * r2);
            double X[3];
            for (int d = 0; d < 3; ++d) {
                X[d] = P1[d] - (za2 * A[d] + zb2 * B[d]) * ip2;
                hermite_pair<LA, LB>(-zb2 * ip2 * AB[d], za2 * ip2 * AB[d], 0.5 * ip2, E2[d]);
            }
            hermite_coulomb<L>(boys_tab, p * p2 / (p + p2), X, R);
            // 2π^{5/2}/(p p' sqrt(p+p'))
            const double cc = (kl == ij ? 1.0 : 2.0) * 34.98683665524972497 * ip * ip2 * rsqrt(p + p2) * w1 * w2;
            for (int ia = 0; ia < NA; ++ia) {
                int pa[3];
                cart_powers(LA, ia, pa);
                for (int ib = 0; ib < NB; ++ib) {
                    int pb[3];
                    cart_powers(LB, ib, pb);
                    const double *e1x = E1[0] + (pa[0] * (LB + 1) + pb[0]) * NT, *e2x = E2[0] + (pa[0] * (LB + 1) + pb[0]) * NT;
                    const double *e1y = E1[1] + (pa[1] * (LB + 1) + pb[1]) * NT, *e2y = E2[1] + (pa[1] * (LB + 1) + pb[1]) * NT;
                    const double *e1z = E1[2] + (pa[2] * (LB + 1) + pb[2]) * NT, *e2z = E2[2] + (pa[2] * (LB + 1) + pb[2]) * NT;
                    const int tx = pa[0] + pb[0], ty = pa[1] + pb[1], tz = pa[2] + pb[2];
                    double s = 0.0;
                    for (int t = 0; t <= tx; ++t)
                        for (int t2 = 0; t2 <= tx; ++t2) {
                            const double fx = ((t2 & 1) ? -1.0 : 1.0) * e1x[t] * e2x[t2];
                            double sy = 0.0;
                            for (int u = 0; u <= ty; ++u)
                                for (int u2 = 0; u2 <= ty; ++u2) {
                                    const double fy = ((u2 & 1) ? -1.0 : 1.0) * e1y[u] * e2y[u2];
                                    const double *Rr = R + ((t + t2) * N1 + (u + u2)) * N1;
                                    double sz = 0.0;
                                    for (int v = 0; v <= tz; ++v) {
                                        double s2 = 0.0;
                                        for (int v2 = 0; v2 <= tz; ++v2) s2 += ((v2 & 1) ? -e2z[v2] : e2z[v2]) * Rr[v + v2];
                                        sz += e1z[v] * s2;
                                    }
                                    sy += fy * sz;
                                }
                            s += fx * sy;
                        }
                    diag[ia * NB + ib] += cc * s;
                }
            }
        }
    }
    double mx = 0.0;
    for (int i = 0; i < NA * NB; ++i) mx = fmax(mx, diag[i]);
    q[slot[k]] = sqrt(mx);
}

// One thread per aux shell of angular momentum LX (2-centre, one centre: X = 0, T = 0).
template <int LX>
__global__ void __launch_bounds__(64)
schwarz_aux_kernel(DevShells aux, const int32_t *__restrict__ ids, int n, const double *__restrict__ boys_tab,
                   double *__restrict__ q) {
    constexpr int L = 2 * LX, N1 = L + 1, NT = LX + 1, NX = nc(LX);
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n) return;
    const int x = ids[k], K = aux.K[x], o = aux.prim_off[x];
    double E1[(LX + 1) * NT], E2[(LX + 1) * NT], R[N1 * N1 * N1], diag[NX];
    for (int i = 0; i < NX; ++i) diag[i] = 0.0;
    const double zero[3] = {0.0, 0.0, 0.0};
    for (int i = 0; i < K; ++i) {
        const double z1 = aux.zeta[o + i];
        hermite_pair<LX, 0>(0.0, 0.0, 0.5 / z1, E1);
        for (int j = 0; j <= i; ++j) {
            const double z2 = aux.zeta[o + j];
            hermite_pair<LX, 0>(0.0, 0.0, 0.5 / z2, E2);
            hermite_coulomb<L>(boys_tab, z1 * z2 / (z1 + z2), zero, R);
            const double cc = (i == j ? 1.0 : 2.0) * 34.98683665524972497 / (z1 * z2) * rsqrt(z1 + z2) * aux.coef[o + i] * aux.coef[o + j];
            for (int ic = 0; ic < NX; ++ic) {
                int pc[3];
                cart_powers(LX, ic, pc);
                double s = 0.0;
                for (int t = 0; t <= pc[0]; ++t)
                    for (int t2 = 0; t2 <= pc[0]; ++t2)
                        for (int u = 0; u <= pc[1]; ++u)
                            for (int u2 = 0; u2 <= pc[1]; ++u2)
                                for (int v = 0; v <= pc[2]; ++v)
                                    for (int v2 = 0; v2 <= pc[2]; ++v2) {
                                        const double sg = ((t2 + u2 + v2) & 1) ? -1.0 : 1.0;
                                        s += sg * E1[pc[0] * NT + t] * E1[pc[1] * NT + u] * E1[pc[2] * NT + v] * E2[pc[0] * NT + t2] *
                                             E2[pc[1] * NT + u2] * E2[pc[2] * NT + v2] * R[((t + t2) * N1 + (u + u2)) * N1 + (v + v2)];
                                    }
                diag[ic] += cc * s;
            }
        }
    }
    double mx = 0.0;
    for (int i = 0; i < NX; ++i) mx = fmax(mx, diag[i]);
    q[x] = sqrt(mx);
}

// ---- two-centre metric V_XY = (X|Y) (second half) -----------------------------
// One thread per pair of aux shells (X of angular momentum LX, Y of LY <= LX; for LX = LY only y <= x), all Cartesian
// components of the block in local memory.  A single Gaussian about its own centre has E_t^{i0} = 0 unless t ≡ i (mod 2)
// (PA = 0 in the recurrence), so the Hermite sums step by two.  The block and its transpose are written, the diagonal
// block (x = y) symmetrised, so V is exactly symmetric.
template <int LX, int LY>
__global__ void __launch_bounds__(64)
metric_kernel(DevShells aux, const int32_t *__restrict__ bf_off, const int32_t *__restrict__ idx, int nX,
              const int32_t *__restrict__ idy, int nY, const double *__restrict__ boys_tab, double *__restrict__ V,
              long long ld) {
    constexpr int L = LX + LY, N1 = L + 1, NTX = LX + 1, NTY = LY + 1, NX = nc(LX), NY = nc(LY);
    const long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= (long long)nX * nY) return;
    const int ix = (int)(k / nY), iy = (int)(k - (long long)ix * nY);
    const int x = idx[ix], y = idy[iy];
    if (LX == LY && y > x) return;
    const int Kx = aux.K[x], Ky = aux.K[y], ox = aux.prim_off[x], oy = aux.prim_off[y];
    double AB[3];
    for (int d = 0; d < 3; ++d) AB[d] = aux.center[3 * x + d] - aux.center[3 * y + d];
    double EX[(LX + 1) * NTX], EY[(LY + 1) * NTY], R[N1 * N1 * N1], blk[NX * NY];
    for (int i = 0; i < NX * NY; ++i) blk[i] = 0.0;
    for (int i = 0; i < Kx; ++i) {
        const double z1 = aux.zeta[ox + i];
        hermite_pair<LX, 0>(0.0, 0.0, 0.5 / z1, EX);
        for (int j = 0; j < Ky; ++j) {
            const double z2 = aux.zeta[oy + j];
            hermite_pair<LY, 0>(0.0, 0.0, 0.5 / z2, EY);
            hermite_coulomb<L>(boys_tab, z1 * z2 / (z1 + z2), AB, R);
            // 2π^{5/2} / (ζ1 ζ2 sqrt(ζ1+ζ2))
            const double cc = 34.98683665524972497 / (z1 * z2) * rsqrt(z1 + z2) * aux.coef[ox + i] * aux.coef[oy + j];
            for (int cx = 0; cx < NX; ++cx) {
                int px[3];
                cart_powers(LX, cx, px);
                const double *e1x = EX + px[0] * NTX, *e1y = EX + px[1] * NTX, *e1z = EX + px[2] * NTX;
                for (int cy = 0; cy < NY; ++cy) {
                    int py[3];
                    cart_powers(LY, cy, py);
                    const double *e2x = EY + py[0] * NTY, *e2y = EY + py[1] * NTY, *e2z = EY + py[2] * NTY;
                    // (−1)^{t'+u'+v'} with t' ≡ py (mod 2) throughout: one sign for the whole component
                    const double sg = ((py[0] + py[1] + py[2]) & 1) ? -1.0 : 1.0;
                    double s = 0.0;
                    for (int t = px[0] & 1; t <= px[0]; t += 2)
                        for (int t2 = py[0] & 1; t2 <= py[0]; t2 += 2) {
                            const double fx = e1x[t] * e2x[t2];
                            double sy = 0.0;
                            for (int u = px[1] & 1; u <= px[1]; u += 2)
                                for (int u2 = py[1] & 1; u2 <= py[1]; u2 += 2) {
                                    const double fy = e1y[u] * e2y[u2];
                                    const double *Rr = R + ((t + t2) * N1 + (u + u2)) * N1;
                                    double sz = 0.0;
                                    for (int v = px[2] & 1; v <= px[2]; v += 2) {
                                        double s2 = 0.0;
                                        for (int v2 = py[2] & 1; v2 <= py[2]; v2 += 2) s2 = fma(e2z[v2], Rr[v + v2], s2);
                                        sz = fma(e1z[v], s2, sz);
                                    }
                                    sy = fma(fy, sz, sy);
                                }
                            s = fma(fx, sy, s);
                        }
                    blk[cx * NY + cy] = fma(cc * sg, s, blk[cx * NY + cy]);
                }
            }
        }
    }
    double *Vxy = V + (long long)bf_off[x] * ld + bf_off[y], *Vyx = V + (long long)bf_off[y] * ld + bf_off[x];
    if (x == y) {
        for (int cx = 0; cx < NX; ++cx)
            for (int cy = 0; cy < NY; ++cy) Vxy[(long long)cx * ld + cy] = 0.5 * (blk[cx * NY + cy] + blk[cy * NY + cx]);
    } else {
        for (int cx = 0; cx < NX; ++cx)
            for (int cy = 0; cy < NY; ++cy) {
                Vxy[(long long)cx * ld + cy] = blk[cx * NY + cy];
                Vyx[(long long)cy * ld + cx] = blk[cx * NY + cy];
            }
    }
}

template <class T>
static cudaError_t upload(const T *host, size_t n, T **dev) {
    *dev = nullptr;
    if (n == 0) return cudaSuccess;
    cudaError_t e = cudaMalloc((void **)dev, n * sizeof(T));
    if (e != cudaSuccess) return e;
    return cudaMemcpy(*dev, host, n * sizeof(T), cudaMemcpyHostToDevice);
}

struct DevTable {
    int32_t *L = nullptr, *K = nullptr, *prim_off = nullptr;
    double *center = nullptr, *zeta = nullptr, *coef = nullptr;
    cudaError_t put(const lx_shells_t *h) {
        const size_t n = (size_t)h->nshell, np = n ? (size_t)h->prim_off[n] : 0;
        cudaError_t e;
        if ((e = upload(h->L, n, &L)) != cudaSuccess) return e;
        if ((e = upload(h->K, n, &K)) != cudaSuccess) return e;
        if ((e = upload(h->prim_off, n + 1, &prim_off)) != cudaSuccess) return e;
        if ((e = upload(h->center, 3 * n, &center)) != cudaSuccess) return e;
        if ((e = upload(h->zeta, np, &zeta)) != cudaSuccess) return e;
        return upload(h->coef, np, &coef);
    }
    DevShells view() const { return DevShells{L, K, prim_off, center, zeta, coef, nullptr}; }
    ~DevTable() {
        cudaFree(L); cudaFree(K); cudaFree(prim_off); cudaFree(center); cudaFree(zeta); cudaFree(coef);
    }
};

static bool table_ok(const lx_shells_t *s) {
    return s && s->nshell >= 0 && (s->nshell == 0 || (s->L && s->K && s->prim_off && s->center && s->zeta && s->coef));
}

}  // namespace lx

using namespace lx;

#define LXS_CUDA(expr)                                              \
    do {                                                            \
        cudaError_t _e = (expr);                                    \
        if (_e != cudaSuccess) return state_cuda_fail((int)_e);     \
    } while (0)

extern "C" {

int lx_schwarz_aux_host(const lx_shells_t *aux, double *q_aux) {
    if (!state_ready()) return LX_ENOTINIT;
    if (!table_ok(aux)) return LX_EINVAL;
    if (aux->nshell == 0) return LX_OK;
    if (!q_aux) return LX_EINVAL;
    std::vector<int32_t> ids[LX_MAX_L_AUX + 1];
    for (int i = 0; i < aux->nshell; ++i) {
        if (aux->L[i] < 0 || aux->L[i] > LX_MAX_L_AUX) return LX_EUNSUPPORTED;
        ids[aux->L[i]].push_back(i);
    }
    DevTable t;
    LXS_CUDA(t.put(aux));
    double *dq = nullptr;
    LXS_CUDA(cudaMalloc((void **)&dq, (size_t)aux->nshell * sizeof(double)));
    int rc = LX_OK;
    for (int l = 0; l <= LX_MAX_L_AUX && rc == LX_OK; ++l) {
        const int n = (int)ids[l].size();
        if (!n) continue;
        int32_t *dids = nullptr;
        cudaError_t e = upload(ids[l].data(), (size_t)n, &dids);
        if (e == cudaSuccess) {
            const int blocks = (n + 63) / 64;
            switch (l) {
#define LXS_AUX(LV) case LV: schwarz_aux_kernel<LV><<<blocks, 64>>>(t.view(), dids, n, state_boys_tab(), dq); break;
                LXS_AUX(0) LXS_AUX(1) LXS_AUX(2) LXS_AUX(3) LXS_AUX(4) LXS_AUX(5) LXS_AUX(6)
#undef LXS_AUX
            }
            state_count_launches(1);
            e = cudaDeviceSynchronize();
        }
        cudaFree(dids);
        if (e != cudaSuccess) rc = state_cuda_fail((int)e);
    }
    if (rc == LX_OK) {
        cudaError_t e = cudaMemcpy(q_aux, dq, (size_t)aux->nshell * sizeof(double), cudaMemcpyDeviceToHost);
        if (e != cudaSuccess) rc = state_cuda_fail((int)e);
    }
    cudaFree(dq);
    return rc;
}

int lx_schwarz_pair_host(const lx_shells_t *prim, const int32_t *pair_idx, int npair, double *q_pair) {
    if (!state_ready()) return LX_ENOTINIT;
    if (!table_ok(prim) || npair < 0) return LX_EINVAL;
    if (npair == 0) return LX_OK;
    if (!pair_idx || !q_pair) return LX_EINVAL;
    constexpr int NCL = (LX_MAX_L_PRIM + 1) * (LX_MAX_L_PRIM + 1);
    std::vector<int32_t> pr[NCL], sl[NCL];
    for (int k = 0; k < npair; ++k) {
        const int a = pair_idx[2 * k], b = pair_idx[2 * k + 1];
        if (a < 0 || a >= prim->nshell || b < 0 || b >= prim->nshell) return LX_EINVAL;
        const int la = std::max(prim->L[a], prim->L[b]), lb = std::min(prim->L[a], prim->L[b]);
        if (lb < 0 || la > LX_MAX_L_PRIM) return LX_EUNSUPPORTED;
        const int c = la * (LX_MAX_L_PRIM + 1) + lb;
        pr[c].push_back(a);
        pr[c].push_back(b);
        sl[c].push_back(k);
    }
    DevTable t;
    LXS_CUDA(t.put(prim));
    double *dq = nullptr;
    LXS_CUDA(cudaMalloc((void **)&dq, (size_t)npair * sizeof(double)));
    int rc = LX_OK;
    for (int c = 0; c < NCL && rc == LX_OK; ++c) {
        const int n = (int)sl[c].size();
        if (!n) continue;
        int32_t *dp = nullptr, *ds = nullptr;
        cudaError_t e = upload(pr[c].data(), pr[c].size(), &dp);
        if (e == cudaSuccess) e = upload(sl[c].data(), sl[c].size(), &ds);
        if (e == cudaSuccess) {
            const int blocks = (n + 63) / 64;
            switch (c) {
#define LXS_PAIR(A_, B_) case A_ * (LX_MAX_L_PRIM + 1) + B_: \
    schwarz_pair_kernel<A_, B_><<<blocks, 64>>>(t.view(), dp, ds, n, state_boys_tab(), dq); break;
                LXS_PAIR(0, 0)
                LXS_PAIR(1, 0) LXS_PAIR(1, 1)
                LXS_PAIR(2, 0) LXS_PAIR(2, 1) LXS_PAIR(2, 2)
                LXS_PAIR(3, 0) LXS_PAIR(3, 1) LXS_PAIR(3, 2) LXS_PAIR(3, 3)
                LXS_PAIR(4, 0) LXS_PAIR(4, 1) LXS_PAIR(4, 2) LXS_PAIR(4, 3) LXS_PAIR(4, 4)
#undef LXS_PAIR
            }
            state_count_launches(1);
            e = cudaDeviceSynchronize();
        }
        cudaFree(dp);
        cudaFree(ds);
        if (e != cudaSuccess) rc = state_cuda_fail((int)e);
    }
    if (rc == LX_OK) {
        cudaError_t e = cudaMemcpy(q_pair, dq, (size_t)npair * sizeof(double), cudaMemcpyDeviceToHost);
        if (e != cudaSuccess) rc = state_cuda_fail((int)e);
    }
    cudaFree(dq);
    return rc;
}

int lx_metric_2c(const lx_shells_t *aux, double *V_dev, long long ld) {
    if (!state_ready()) return LX_ENOTINIT;
    if (!table_ok(aux)) return LX_EINVAL;
    if (aux->nshell == 0) return LX_OK;
    std::vector<int32_t> ids[LX_MAX_L_AUX + 1], bf((size_t)aux->nshell + 1);
    bf[0] = 0;
    for (int i = 0; i < aux->nshell; ++i) {
        const int l = aux->L[i];
        if (l < 0 || l > LX_MAX_L_AUX) return LX_EUNSUPPORTED;
        if (aux->K[i] < 1 || aux->prim_off[i + 1] - aux->prim_off[i] != aux->K[i]) return LX_EINVAL;
        ids[l].push_back(i);
        bf[i + 1] = bf[i] + (l + 1) * (l + 2) / 2;
        if (aux->bf_off && aux->bf_off[i] != bf[i]) return LX_EINVAL;        // the metric is laid out in Cartesian order
    }
    if (!V_dev || ld < bf[aux->nshell]) return LX_EINVAL;
    DevTable t;
    LXS_CUDA(t.put(aux));
    int32_t *dbf = nullptr, *dids[LX_MAX_L_AUX + 1] = {};
    cudaError_t e = upload(bf.data(), bf.size(), &dbf);
    for (int l = 0; l <= LX_MAX_L_AUX && e == cudaSuccess; ++l) e = upload(ids[l].data(), ids[l].size(), &dids[l]);
    int launches = 0;
    for (int lx = 0; lx <= LX_MAX_L_AUX && e == cudaSuccess; ++lx)
        for (int ly = 0; ly <= lx && e == cudaSuccess; ++ly) {
            const long long n = (long long)ids[lx].size() * (long long)ids[ly].size();
            if (!n) continue;
            const unsigned blocks = (unsigned)((n + 63) / 64);
            switch (lx * (LX_MAX_L_AUX + 1) + ly) {
#define LXS_MET(A_, B_) case A_ * (LX_MAX_L_AUX + 1) + B_:                                                      \
    metric_kernel<A_, B_><<<blocks, 64>>>(t.view(), dbf, dids[A_], (int)ids[A_].size(), dids[B_], (int)ids[B_].size(), \
                                          state_boys_tab(), V_dev, ld);                                         \
    break;
                LXS_MET(0, 0)
                LXS_MET(1, 0) LXS_MET(1, 1)
                LXS_MET(2, 0) LXS_MET(2, 1) LXS_MET(2, 2)
                LXS_MET(3, 0) LXS_MET(3, 1) LXS_MET(3, 2) LXS_MET(3, 3)
                LXS_MET(4, 0) LXS_MET(4, 1) LXS_MET(4, 2) LXS_MET(4, 3) LXS_MET(4, 4)
                LXS_MET(5, 0) LXS_MET(5, 1) LXS_MET(5, 2) LXS_MET(5, 3) LXS_MET(5, 4) LXS_MET(5, 5)
                LXS_MET(6, 0) LXS_MET(6, 1) LXS_MET(6, 2) LXS_MET(6, 3) LXS_MET(6, 4) LXS_MET(6, 5) LXS_MET(6, 6)
#undef LXS_MET
            }
            ++launches;
            e = cudaGetLastError();
        }
    if (e == cudaSuccess) e = cudaDeviceSynchronize();
    state_count_launches(launches);
    cudaFree(dbf);
    for (int l = 0; l <= LX_MAX_L_AUX; ++l) cudaFree(dids[l]);
    return e == cudaSuccess ? LX_OK : state_cuda_fail((int)e);
}

}  // extern "C"
