// lx_api.cu — C-ABI entry points of liblx (include/lx.h): library state, Boys table, primitive-pair pre-pass,
// class dispatch, the Schwarz-screened schedule and the DF drivers.
#include <algorithm>
#include <atomic>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>
#include <string>
#include <vector>

#include "lx_common.cuh"
#include "lx_dispatch.h"
#include "lx_state.h"
#include "lx_owner.cuh"

namespace lx {

// ------------------------------------------------------------------------------------------------ library state
struct State {
    bool ready = false;
    int device = -1;
    int num_sms = 0;
    double *boys_tab = nullptr;      // [BOYS_NGRID][BOYS_MROWS]
    double *solid[LX_MAX_L_AUX + 1] = {};   // per l: (2l+1) x nc(l) Cartesian -> real solid harmonic matrix
    std::atomic<long long> launches{0};
    char cuda_msg[256] = "no CUDA error recorded";
    // grow-only device arena for the host-buffer convenience path
    void *arena = nullptr;
    size_t arena_bytes = 0;
    // asynchronous status word in device memory, OR-ed into by the kernels (lx_async_status)
    int *flag_dev = nullptr;
    int check = 0;                   // LX_CHECK=1 in the environment (read by lx_init)
    double *static_scratch = nullptr;   // device address of lx_static_scratch on the current device (lx_eri3_batch_static)
    // side streams of the DF drivers: the class launches of a pass are independent (they only add into gamma / J), so their
    // tails overlap when they are spread over a few streams (LX_DF_STREAMS, default 4; 1 = the caller's stream only)
    static constexpr int MAX_SIDE = 7;
    int n_side = 0;
    cudaStream_t side[MAX_SIDE] = {};
    cudaEvent_t side_ev[MAX_SIDE] = {};
    cudaEvent_t fork_ev = nullptr;
};
static State g;
static std::mutex g_mu;

static int cuda_fail(cudaError_t e) {
    snprintf(g.cuda_msg, sizeof(g.cuda_msg), "CUDA error %d: %s", (int)e, cudaGetErrorString(e));
    return LX_ECUDA;
}
#define LX_CUDA(expr)                                 \
    do {                                              \
        cudaError_t _e = (expr);                      \
        if (_e != cudaSuccess) return cuda_fail(_e);  \
    } while (0)

bool state_ready() { return g.ready; }
const double *state_boys_tab() { return g.boys_tab; }
int state_num_sms() { return g.num_sms; }
void state_count_launches(int n) { g.launches += n; }
int state_cuda_fail(int e) { return cuda_fail((cudaError_t)e); }

static const launch_fn k_launch[4][7] = {
    {launch_lx0_mode0, launch_lx1_mode0, launch_lx2_mode0, launch_lx3_mode0, launch_lx4_mode0, launch_lx5_mode0, launch_lx6_mode0},
    {launch_lx0_mode1, launch_lx1_mode1, launch_lx2_mode1, launch_lx3_mode1, launch_lx4_mode1, launch_lx5_mode1, launch_lx6_mode1},
    {launch_lx0_mode2, launch_lx1_mode2, launch_lx2_mode2, launch_lx3_mode2, launch_lx4_mode2, launch_lx5_mode2, launch_lx6_mode2},
    {launch_lx0_mode3, launch_lx1_mode3, launch_lx2_mode3, launch_lx3_mode3, launch_lx4_mode3, launch_lx5_mode3, launch_lx6_mode3},
};

// ------------------------------------------------------------------------------------------------ Boys table (host)
// F_m(T) = ∫_0^1 y^{2m} exp(−T y²) dy (eq. 19) on the grid T_i = i/16 in long double:
// positive-term series at the top order, then downward recursion.  Written for this library; shares nothing with
// the test oracle.
static void boys_table_host(std::vector<double> &tab) {
    tab.assign((size_t)BOYS_NGRID * BOYS_MROWS, 0.0);
    const int M = BOYS_MROWS - 1;
    std::vector<long double> F(BOYS_MROWS);
    for (int i = 0; i < BOYS_NGRID; ++i) {
        const long double T = (long double)i / (long double)BOYS_PER_UNIT;
        const long double eT = expl(-T);
        long double term = 1.0L / (long double)(2 * M + 1), sum = term;
        for (int n = 1; n < 4000; ++n) {
            term *= (2.0L * T) / (long double)(2 * M + 2 * n + 1);
            sum += term;
            if (term < 1e-24L * sum) break;
        }
        F[M] = eT * sum;
        for (int m = M; m >= 1; --m) F[m - 1] = (2.0L * T * F[m] + eT) / (long double)(2 * m - 1);
        for (int m = 0; m < BOYS_MROWS; ++m) tab[(size_t)i * BOYS_MROWS + m] = (double)F[m];
    }
}

// ------------------------------------------------------------------------------------------------ kernels
// a1: primitive-pair data, one thread per (pair, primitive pair).  P by eq. 16, γ by eq. 14, K_ij = c_i c_j
// exp(−ζaζb/γ |AB|²) (exponential factor of eq. 4).
constexpr int FLAG_KSTRIDE = 1, FLAG_AUX_CLASS = 2, FLAG_PAIR_CLASS = 4, FLAG_RANGE = 8;
__global__ void pair_data_kernel(DevShells prim, const int32_t *__restrict__ pair_list, int npair, int swapped,
                                 const long long *__restrict__ pd_off, int kstride, int kiter, double *__restrict__ pd,
                                 int *__restrict__ flag) {
    // flat index over pairs × kiter lanes; a lane walks ij = lane, lane+kiter, ... < K_a K_b
    const long long total = (long long)npair * kiter;
    for (long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x; t < total; t += (long long)gridDim.x * blockDim.x) {
        const long long p = t / kiter;
        const int lane = (int)(t - p * kiter);
        const int a = pair_list[2 * p + swapped], b = pair_list[2 * p + 1 - swapped];
        const int Ka = prim.K[a], Kb = prim.K[b];
        // a pair with more primitive pairs than the record stride: the class kernels clamp the same way (no read past
        // the record), the contraction is truncated and the status word says so (lx_async_status → LX_ENOMEM)
        if (Ka * Kb > kstride && lane == 0) atomicOr(flag, FLAG_KSTRIDE);
        const int Kab = min(Ka * Kb, kstride);
        const double Ax = prim.center[3 * a], Ay = prim.center[3 * a + 1], Az = prim.center[3 * a + 2];
        const double Bx = prim.center[3 * b], By = prim.center[3 * b + 1], Bz = prim.center[3 * b + 2];
        const double r2 = (Ax - Bx) * (Ax - Bx) + (Ay - By) * (Ay - By) + (Az - Bz) * (Az - Bz);
        for (int ij = lane; ij < Kab; ij += kiter) {
            const int i = ij / Kb, j = ij - i * Kb;
            const double za = prim.zeta[prim.prim_off[a] + i], zb = prim.zeta[prim.prim_off[b] + j];
            const double ca = prim.coef[prim.prim_off[a] + i], cb = prim.coef[prim.prim_off[b] + j];
            const double gam = za + zb, ig = 1.0 / gam;
            const long long o = ((pd_off ? pd_off[p] : p * (long long)kstride) + ij) * PD_STRIDE;
            pd[o + 0] = gam;
            pd[o + 1] = (za * Ax + zb * Bx) * ig;
            pd[o + 2] = (za * Ay + zb * By) * ig;
            pd[o + 3] = (za * Az + zb * Bz) * ig;
            // a truncated pair (see above) poisons its integrals: loud NaNs instead of a silently short contraction
            pd[o + 4] = (Ka * Kb > kstride) ? __longlong_as_double(0x7ff8000000000000LL) : ca * cb * exp(-za * zb * ig * r2);
            pd[o + 5] = 0.5 * ig;
        }
    }
}

// LX_CHECK=1: class conformity of the index lists (the caller's contract otherwise, lx.h)
__global__ void check_lists_kernel(DevShells aux, int naux, DevShells prim, int nprim, int lx_, int la, int lb,
                                   const int32_t *__restrict__ x_idx, int nx, const int32_t *__restrict__ pair_idx, int npair,
                                   int kstride, int *__restrict__ flag) {
    int f = 0;
    for (long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x; t < (long long)nx + npair; t += (long long)gridDim.x * blockDim.x) {
        if (t < nx) {
            const int x = x_idx[t];
            if (x < 0 || x >= naux) f |= FLAG_RANGE;
            else if (aux.L[x] != lx_) f |= FLAG_AUX_CLASS;
        } else {
            const int a = pair_idx[2 * (t - nx)], b = pair_idx[2 * (t - nx) + 1];
            if (a < 0 || a >= nprim || b < 0 || b >= nprim) f |= FLAG_RANGE;
            else {
                if (prim.L[a] != la || prim.L[b] != lb) f |= FLAG_PAIR_CLASS;
                if (prim.K[a] * prim.K[b] > kstride) f |= FLAG_KSTRIDE;
            }
        }
    }
    if (f) atomicOr(flag, f);
}

__global__ void boys_kernel(const double *__restrict__ tab, const double *__restrict__ T, int n, int mmax,
                            double *__restrict__ out) {
    const long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (t >= (long long)n * (mmax + 1)) return;
    const int i = (int)(t / (mmax + 1)), m = (int)(t - (long long)i * (mmax + 1));
    out[t] = boys_one(tab, m, T[i]);
}

// FP64 FMA throughput probe: 8 independent DFMA chains per thread (roofline denominator of the ALU-bound classes).
__global__ void __launch_bounds__(256) dfma_probe_kernel(int iters, double seed, double *__restrict__ sink) {
    double a0 = seed + threadIdx.x, a1 = a0 + 1, a2 = a0 + 2, a3 = a0 + 3, a4 = a0 + 4, a5 = a0 + 5, a6 = a0 + 6, a7 = a0 + 7;
    const double m = 0.999999, c = 1e-9;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            a0 = fma(a0, m, c); a1 = fma(a1, m, c); a2 = fma(a2, m, c); a3 = fma(a3, m, c);
            a4 = fma(a4, m, c); a5 = fma(a5, m, c); a6 = fma(a6, m, c); a7 = fma(a7, m, c);
        }
    }
    const double r = ((a0 + a1) + (a2 + a3)) + ((a4 + a5) + (a6 + a7));
    if (r == 123.456) sink[0] = r;
}

// ------------------------------------------------------------------------------------------------ solid harmonics (a6)
// Real solid harmonics S_lm as polynomials in (x, y, z), Racah normalisation, by the recurrences of the regular solid
// harmonics (Helgaker, Jorgensen, Olsen, "Molecular Electronic-Structure Theory", eqs. 6.4.70-6.4.73):
//   S_00 = 1
//   S_{l+1, l+1}  = sqrt(2^{d_l0} (2l+1)/(2l+2)) (x S_ll - (1 - d_l0) y S_{l,-l})
//   S_{l+1,-l-1}  = sqrt(2^{d_l0} (2l+1)/(2l+2)) (y S_ll + (1 - d_l0) x S_{l,-l})
//   S_{l+1, m}    = ((2l+1) z S_lm - sqrt((l+m)(l-m)) r^2 S_{l-1,m}) / sqrt((l+m+1)(l-m+1)),  |m| <= l
// Row m + l of the matrix holds the coefficients of S_lm over the Cartesian components in ABI order (reading G2).
// Written for this library; the test oracle uses the closed formula instead and shares nothing with this.
struct SolidPoly {
    double c[LX_MAX_L_AUX + 1][LX_MAX_L_AUX + 1][LX_MAX_L_AUX + 1];
    SolidPoly() { std::memset(c, 0, sizeof(c)); }
};
static void poly_axpy_shift(SolidPoly &dst, double f, const SolidPoly &src, int sx, int sy, int sz) {
    const int N = LX_MAX_L_AUX + 1;
    for (int x = 0; x + sx < N; ++x)
        for (int y = 0; y + sy < N; ++y)
            for (int z = 0; z + sz < N; ++z) dst.c[x + sx][y + sy][z + sz] += f * src.c[x][y][z];
}
static void solid_matrices_host(std::vector<std::vector<double>> &mats) {
    const int LM = LX_MAX_L_AUX;
    // S[l][m + l]
    std::vector<std::vector<SolidPoly>> S(LM + 1);
    S[0].resize(1);
    S[0][0].c[0][0][0] = 1.0;
    for (int l = 0; l < LM; ++l) {
        S[l + 1].resize(2 * l + 3);
        const double d0 = l == 0 ? 1.0 : 0.0;
        const double f = std::sqrt(std::pow(2.0, d0) * (2.0 * l + 1.0) / (2.0 * l + 2.0));
        const SolidPoly &pll = S[l][2 * l], &pml = S[l][0];          // S_{l,l}, S_{l,-l}
        SolidPoly &top = S[l + 1][2 * l + 2], &bot = S[l + 1][0];    // S_{l+1,l+1}, S_{l+1,-l-1}
        poly_axpy_shift(top, f, pll, 1, 0, 0);
        poly_axpy_shift(bot, f, pll, 0, 1, 0);
        if (l > 0) {
            poly_axpy_shift(top, -f, pml, 0, 1, 0);
            poly_axpy_shift(bot, f, pml, 1, 0, 0);
        }
        for (int m = -l; m <= l; ++m) {
            SolidPoly &t = S[l + 1][m + l + 1];
            const double den = std::sqrt((double)(l + m + 1) * (double)(l - m + 1));
            poly_axpy_shift(t, (2.0 * l + 1.0) / den, S[l][m + l], 0, 0, 1);
            if (l >= 1 && std::abs(m) <= l - 1) {
                const double g2 = -std::sqrt((double)(l + m) * (double)(l - m)) / den;
                const SolidPoly &q = S[l - 1][m + l - 1];
                poly_axpy_shift(t, g2, q, 2, 0, 0);
                poly_axpy_shift(t, g2, q, 0, 2, 0);
                poly_axpy_shift(t, g2, q, 0, 0, 2);
            }
        }
    }
    mats.assign(LM + 1, {});
    for (int l = 0; l <= LM; ++l) {
        mats[l].assign((size_t)(2 * l + 1) * nc(l), 0.0);
        for (int m = 0; m < 2 * l + 1; ++m) {
            int ci = 0;
            for (int x = l; x >= 0; --x)
                for (int y = l - x; y >= 0; --y, ++ci) mats[l][(size_t)m * nc(l) + ci] = S[l][m].c[x][y][l - x - y];
        }
    }
}

// out[set][m][r] = sum_c S[m][c] in[set][c][r]; one thread per (set, r): the nc(l) inputs are read once into
// registers (coalesced over r), the matrix sits in shared memory; HBM-bound (reads nc(l), writes 2l+1 doubles per thread)
template <int L>
__global__ void __launch_bounds__(256) cart_to_pure_kernel(const double *__restrict__ S, long long nsets, int nab,
                                                           const double *__restrict__ in, double *__restrict__ out) {
    constexpr int ncl = nc(L), npl = 2 * L + 1;
    __shared__ double sm[ncl * npl];
    for (int i = threadIdx.x; i < ncl * npl; i += blockDim.x) sm[i] = S[i];
    __syncthreads();
    const long long total = nsets * nab;
    for (long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x; t < total; t += (long long)gridDim.x * blockDim.x) {
        const long long set = t / nab;
        const int r = (int)(t - set * nab);
        const double *src = in + set * ncl * nab + r;
        double *dst = out + set * npl * nab + r;
        double v[ncl];
#pragma unroll
        for (int c = 0; c < ncl; ++c) v[c] = __ldg(src + (size_t)c * nab);
#pragma unroll
        for (int m = 0; m < npl; ++m) {
            double acc = 0.0;
#pragma unroll
            for (int c = 0; c < ncl; ++c) acc = fma(sm[m * ncl + c], v[c], acc);
            dst[(size_t)m * nab] = acc;
        }
    }
}

static int check_shells(const lx_shells_t *s, bool need_bf) {
    if (!s) return LX_EINVAL;
    if (s->nshell < 0) return LX_EINVAL;
    if (s->nshell > 0 && (!s->L || !s->K || !s->prim_off || !s->center || !s->zeta || !s->coef)) return LX_EINVAL;
    if (need_bf && s->nshell > 0 && !s->bf_off) return LX_EINVAL;
    return LX_OK;
}

static int class_supported(int lx_, int la, int lb) {
    return lx_ >= 0 && lx_ <= LX_MAX_L_AUX && la >= 0 && la <= LX_MAX_L_PRIM && lb >= 0 && lb <= LX_MAX_L_PRIM;
}

static int launch_pair_data(const DevShells &prim, const int32_t *pair_list, int npair, int swapped,
                            const long long *pd_off, int kstride, double *pd, cudaStream_t st) {
    if (npair == 0) return LX_OK;
    const int kiter = std::min(kstride, 32);
    const long long total = (long long)npair * kiter;
    const int threads = 256;
    long long blocks = (total + threads - 1) / threads;
    if (blocks > 148LL * 16) blocks = 148LL * 16;
    pair_data_kernel<<<(unsigned)blocks, threads, 0, st>>>(prim, pair_list, npair, swapped, pd_off, kstride, kiter, pd, g.flag_dev);
    g.launches++;
    LX_CUDA(cudaGetLastError());
    return LX_OK;
}

}  // namespace lx

using namespace lx;

// Scratch of the allocation-free entry point lx_eri3_batch_static (include/lx.h): the primitive-pair data (row a1) of ONE
// call.  File scope, fixed size: every GPU that loads the library holds these 4 MiB until the process exits.  In host code
// the name is only a stand-in for the symbol, not a device address: lx_init() asks cudaGetSymbolAddress for the address on
// the device it initialises and the entry point hands THAT to the kernels.
static __device__ __align__(256) double lx_static_scratch[LX_STATIC_SCRATCH_BYTES / sizeof(double)];

// ================================================================================================ C ABI
extern "C" {

const char *lx_version(void) { return "lx3 0.3 sm_100a (team/chain/owner/lane/group kernels, Lx<=6, La,Lb<=4)"; }

const char *lx_kernel_family_k(int lx_, int la, int lb, int kmax) {
    if (!(lx_ >= 0 && lx_ <= LX_MAX_L_AUX && la >= 0 && la <= LX_MAX_L_PRIM && lb >= 0 && lb <= LX_MAX_L_PRIM)) return "";
    static const char *names[] = {"team", "owner", "chain", "lane", "group", "slab"};
    return names[class_family(lx_, std::max(la, lb), std::min(la, lb), kmax)];
}
const char *lx_kernel_family(int lx_, int la, int lb) { return lx_kernel_family_k(lx_, la, lb, 0); }

const char *lx_strerror(int status) {
    switch (status) {
        case LX_OK: return "success";
        case LX_EINVAL: return "invalid argument";
        case LX_EUNSUPPORTED: return "class outside the compiled range (Lx<=6, La,Lb<=4)";
        case LX_ENOMEM: return "workspace too small";
        case LX_ECUDA: return g.cuda_msg;
        case LX_ENOTINIT: return "lx_init() has not been called";
        case LX_ELIMIT: return "npair * kmax_pair exceeds the fixed scratch of lx_eri3_batch_static (LX_STATIC_SCRATCH_BYTES = 4 MiB = 87381 primitive pairs): use lx_eri3_batch with a workspace";
        case LX_ENOTPD: return "lx_fit_solve: the metric is not positive definite (linearly dependent aux functions?)";
        default: return "unknown status";
    }
}

static void free_device_state() {
    if (g.boys_tab) cudaFree(g.boys_tab);
    if (g.arena) cudaFree(g.arena);
    if (g.flag_dev) cudaFree(g.flag_dev);
    for (int i = 0; i < g.n_side; ++i) {
        cudaStreamDestroy(g.side[i]);
        cudaEventDestroy(g.side_ev[i]);
    }
    if (g.fork_ev) cudaEventDestroy(g.fork_ev);
    g.n_side = 0;
    g.fork_ev = nullptr;
    for (int l = 0; l <= LX_MAX_L_AUX; ++l) {
        if (g.solid[l]) cudaFree(g.solid[l]);
        g.solid[l] = nullptr;
    }
    g.boys_tab = nullptr;
    g.arena = nullptr;
    g.arena_bytes = 0;
    g.flag_dev = nullptr;
    g.static_scratch = nullptr;
    g.ready = false;
}

int lx_init(int device) {
    std::lock_guard<std::mutex> lock(g_mu);
    if (g.ready && g.device == device) return LX_OK;
    if (g.ready) {                       // moving to another device: the old tables are freed under the old device
        cudaSetDevice(g.device);
        free_device_state();
    }
    LX_CUDA(cudaSetDevice(device));
    {
        const char *e = std::getenv("LX_CHECK");
        g.check = (e && e[0] == '1') ? 1 : 0;
    }
    LX_CUDA(cudaMalloc((void **)&g.flag_dev, sizeof(int)));
    LX_CUDA(cudaMemset(g.flag_dev, 0, sizeof(int)));
    {
        // device address of the static scratch array on THIS device (lx_eri3_batch_static); checked like every other call
        void *p = nullptr;
        LX_CUDA(cudaGetSymbolAddress(&p, lx_static_scratch));
        g.static_scratch = reinterpret_cast<double *>(p);
    }
    {
        const char *e = std::getenv("LX_DF_STREAMS");
        int n = e ? std::atoi(e) : 4;
        n = std::max(1, std::min(n, State::MAX_SIDE + 1)) - 1;
        LX_CUDA(cudaEventCreateWithFlags(&g.fork_ev, cudaEventDisableTiming));
        for (int i = 0; i < n; ++i) {
            LX_CUDA(cudaStreamCreateWithFlags(&g.side[i], cudaStreamNonBlocking));
            LX_CUDA(cudaEventCreateWithFlags(&g.side_ev[i], cudaEventDisableTiming));
            g.n_side = i + 1;
        }
    }
    cudaDeviceProp prop;
    LX_CUDA(cudaGetDeviceProperties(&prop, device));
    g.num_sms = prop.multiProcessorCount;
    std::vector<double> tab;
    boys_table_host(tab);
    LX_CUDA(cudaMalloc(&g.boys_tab, tab.size() * sizeof(double)));
    LX_CUDA(cudaMemcpy(g.boys_tab, tab.data(), tab.size() * sizeof(double), cudaMemcpyHostToDevice));
    std::vector<std::vector<double>> mats;
    solid_matrices_host(mats);
    for (int l = 0; l <= LX_MAX_L_AUX; ++l) {
        LX_CUDA(cudaMalloc(&g.solid[l], mats[l].size() * sizeof(double)));
        LX_CUDA(cudaMemcpy(g.solid[l], mats[l].data(), mats[l].size() * sizeof(double), cudaMemcpyHostToDevice));
    }
    g.device = device;
    g.ready = true;
    return LX_OK;
}

int lx_finalize(void) {
    std::lock_guard<std::mutex> lock(g_mu);
    if (g.ready) cudaSetDevice(g.device);
    free_device_state();
    return LX_OK;
}

int lx_async_status(void) {
    if (!g.ready) return LX_ENOTINIT;
    int f = 0;
    LX_CUDA(cudaMemcpy(&f, g.flag_dev, sizeof(int), cudaMemcpyDeviceToHost));
    if (f) LX_CUDA(cudaMemset(g.flag_dev, 0, sizeof(int)));
    if (f & (FLAG_RANGE | FLAG_AUX_CLASS | FLAG_PAIR_CLASS)) return LX_EINVAL;
    if (f & FLAG_KSTRIDE) return LX_ENOMEM;
    return LX_OK;
}

int64_t lx_launch_count(void) { return (int64_t)g.launches.load(); }

int lx_fp64_probe(int iters, double *tflops_host) {
    if (!g.ready) return LX_ENOTINIT;
    if (iters <= 0 || !tflops_host) return LX_EINVAL;
    double *sink = nullptr;
    LX_CUDA(cudaMalloc(&sink, 8));
    cudaEvent_t e0, e1;
    LX_CUDA(cudaEventCreate(&e0));
    LX_CUDA(cudaEventCreate(&e1));
    const int blocks = g.num_sms * 8, threads = 256;
    dfma_probe_kernel<<<blocks, threads>>>(iters / 8 + 1, 1.0, sink);  // warm-up
    double best = 0.0;
    for (int rep = 0; rep < 5; ++rep) {
        cudaEventRecord(e0);
        dfma_probe_kernel<<<blocks, threads>>>(iters, 1.0, sink);
        cudaEventRecord(e1);
        LX_CUDA(cudaEventSynchronize(e1));
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        const double fl = 2.0 * 64.0 * (double)iters * (double)blocks * threads;
        best = std::max(best, fl / (ms * 1e-3) * 1e-12);
    }
    g.launches += 6;
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(sink);
    *tflops_host = best;
    return LX_OK;
}

int lx_solid_matrix(int l, double *matrix_host) {
    if (l < 0 || l > LX_MAX_L_AUX || !matrix_host) return LX_EINVAL;
    std::vector<std::vector<double>> mats;
    solid_matrices_host(mats);
    std::memcpy(matrix_host, mats[l].data(), mats[l].size() * sizeof(double));
    return LX_OK;
}

int lx_cart_to_pure(int lx_, int64_t nsets, int nab, const double *in, double *out, void *stream) {
    if (!g.ready) return LX_ENOTINIT;
    if (lx_ < 0 || lx_ > LX_MAX_L_AUX) return LX_EUNSUPPORTED;
    if (nsets < 0 || nab < 0) return LX_EINVAL;
    if (nsets == 0 || nab == 0) return LX_OK;
    if (!in || !out || in == out) return LX_EINVAL;
    const long long total = (long long)nsets * nab;
    const int threads = 256;
    long long blocks = (total + threads - 1) / threads;
    if (blocks > (long long)g.num_sms * 16) blocks = (long long)g.num_sms * 16;
    cudaStream_t st = (cudaStream_t)stream;
    switch (lx_) {
#define LX_C2P(LV) case LV: cart_to_pure_kernel<LV><<<(unsigned)blocks, threads, 0, st>>>(g.solid[LV], nsets, nab, in, out); break;
        LX_C2P(0) LX_C2P(1) LX_C2P(2) LX_C2P(3) LX_C2P(4) LX_C2P(5) LX_C2P(6)
#undef LX_C2P
    }
    g.launches++;
    LX_CUDA(cudaGetLastError());
    return LX_OK;
}

int lx_boys(const double *T, int n, int mmax, double *out, void *stream) {
    if (!g.ready) return LX_ENOTINIT;
    if (n < 0 || mmax < 0 || mmax > BOYS_MMAX) return LX_EINVAL;
    if (n == 0) return LX_OK;
    if (!T || !out) return LX_EINVAL;
    const long long total = (long long)n * (mmax + 1);
    boys_kernel<<<(unsigned)((total + 255) / 256), 256, 0, (cudaStream_t)stream>>>(g.boys_tab, T, n, mmax, out);
    g.launches++;
    LX_CUDA(cudaGetLastError());
    return LX_OK;
}

size_t lx_eri3_workspace_bytes(int lx_, int la, int lb, int nx, int npair, int kmax_pair) {
    (void)lx_; (void)la; (void)lb; (void)nx;
    if (npair <= 0 || kmax_pair <= 0) return 256;
    return (size_t)npair * (size_t)kmax_pair * PD_STRIDE * sizeof(double) + 256;
}

int lx_eri3_batch(int lx_, int la, int lb, const lx_shells_t *aux, const lx_shells_t *prim, const int32_t *x_idx,
                  int nx, const int32_t *pair_idx, int npair, double *out, void *workspace, size_t workspace_bytes,
                  void *stream) {
    if (!g.ready) return LX_ENOTINIT;
    if (nx < 0 || npair < 0) return LX_EINVAL;
    if (!class_supported(lx_, la, lb)) return LX_EUNSUPPORTED;
    if (nx == 0 || npair == 0) return LX_OK;
    int rc;
    if ((rc = check_shells(aux, false)) != LX_OK) return rc;
    if ((rc = check_shells(prim, false)) != LX_OK) return rc;
    if (!x_idx || !pair_idx || !out || !workspace) return LX_EINVAL;
    // kmax_pair is not passed here: the workspace holds npair*kstride*PD_STRIDE doubles, so derive the stride from its size
    const size_t avail = workspace_bytes >= 256 ? workspace_bytes - 256 : 0;
    const long long kstride_ll = (long long)(avail / ((size_t)npair * PD_STRIDE * sizeof(double)));
    if (kstride_ll < 1) return LX_ENOMEM;
    const int kstride = (int)std::min<long long>(kstride_ll, 1 << 20);
    cudaStream_t st = (cudaStream_t)stream;
    const int swapped = la < lb ? 1 : 0;
    const int cla = swapped ? lb : la, clb = swapped ? la : lb;
    DevShells dprim = dev_view(prim), daux = dev_view(aux);
    double *pd = reinterpret_cast<double *>(workspace);
    // The stride must cover the largest K_a*K_b of the batch (contract: lx_eri3_workspace_bytes(kmax_pair)).  The index
    // lists live on the device, so a violation cannot be seen here without a synchronisation: the pre-pass records it in
    // the status word (lx_async_status → LX_ENOMEM) and every kernel clamps to the stride, so nothing is read out of
    // bounds.  LX_CHECK=1 validates stride and class conformity up front, synchronously.
    if (g.check) {
        if ((rc = lx_async_status()) != LX_OK) return rc;
        check_lists_kernel<<<64, 256, 0, st>>>(daux, aux->nshell, dprim, prim->nshell, lx_, la, lb, x_idx, nx, pair_idx, npair,
                                               kstride, g.flag_dev);
        g.launches++;
        LX_CUDA(cudaGetLastError());
        LX_CUDA(cudaStreamSynchronize(st));
        if ((rc = lx_async_status()) != LX_OK) return rc;
    }
    if ((rc = launch_pair_data(dprim, pair_idx, npair, swapped, nullptr, kstride, pd, st)) != LX_OK) return rc;
    // khint: the stride bounds K_a K_b; the aux contraction is not known on the host (aux shells are mostly uncontracted)
    SetMap map{(long long)npair * nx, nx, npair, x_idx, pair_idx, nullptr, kstride};
    PairData pdat{pd, nullptr, kstride};
    DfArgs df{nullptr, nullptr, 0};
    cudaError_t e = k_launch[0][lx_](cla, clb, map, daux, dprim, pdat, g.boys_tab, out, swapped, df, g.num_sms, st);
    g.launches++;
    if (e != cudaSuccess) return cuda_fail(e);
    return LX_OK;
}

size_t lx_static_scratch_bytes(void) { return (size_t)LX_STATIC_SCRATCH_BYTES; }

// Allocation-free variant of lx_eri3_batch (include/lx.h): pre-pass and class kernel as there, primitive-pair data in the
// library's static device array.  No cudaMalloc / cudaFree here or below: launch_pair_data and the class launchers only launch.
int lx_eri3_batch_static(int lx_, int la, int lb, const lx_shells_t *aux, const lx_shells_t *prim, const int32_t *x_idx,
                         int nx, const int32_t *pair_idx, int npair, int kmax_pair, double *out, void *stream) {
    if (!g.ready || !g.static_scratch) return LX_ENOTINIT;
    if (nx < 0 || npair < 0) return LX_EINVAL;
    if (!class_supported(lx_, la, lb)) return LX_EUNSUPPORTED;
    if (nx == 0 || npair == 0) return LX_OK;
    int rc;
    if ((rc = check_shells(aux, false)) != LX_OK) return rc;
    if ((rc = check_shells(prim, false)) != LX_OK) return rc;
    if (!x_idx || !pair_idx || !out || kmax_pair < 1) return LX_EINVAL;
    if ((unsigned long long)npair * (unsigned long long)kmax_pair * PD_STRIDE * sizeof(double) > (unsigned long long)LX_STATIC_SCRATCH_BYTES)
        return LX_ELIMIT;
    cudaStream_t st = (cudaStream_t)stream;
    const int swapped = la < lb ? 1 : 0;
    const int cla = swapped ? lb : la, clb = swapped ? la : lb;
    DevShells dprim = dev_view(prim), daux = dev_view(aux);
    double *pd = g.static_scratch;           // the looked-up device address, never the symbol's host-side name
    if ((rc = launch_pair_data(dprim, pair_idx, npair, swapped, nullptr, kmax_pair, pd, st)) != LX_OK) return rc;
    SetMap map{(long long)npair * nx, nx, npair, x_idx, pair_idx, nullptr, kmax_pair};
    PairData pdat{pd, nullptr, kmax_pair};
    DfArgs df{nullptr, nullptr, 0};
    cudaError_t e = k_launch[0][lx_](cla, clb, map, daux, dprim, pdat, g.boys_tab, out, swapped, df, g.num_sms, st);
    g.launches++;
    if (e != cudaSuccess) return cuda_fail(e);
    return LX_OK;
}

size_t lx_eri3_pure_workspace_bytes(int lx_, int la, int lb, int nx, int npair, int kmax_pair) {
    // pair data + (for classes without a fused kernel) the Cartesian shell-sets the transform reads
    const size_t base = lx_eri3_workspace_bytes(lx_, la, lb, nx, npair, kmax_pair);
    if (npair <= 0 || nx <= 0 || !class_supported(lx_, la, lb)) return base;
    return base + 256 + (size_t)npair * nx * nc(lx_) * nc(la) * nc(lb) * sizeof(double);
}

int lx_eri3_batch_pure(int lx_, int la, int lb, const lx_shells_t *aux, const lx_shells_t *prim, const int32_t *x_idx,
                       int nx, const int32_t *pair_idx, int npair, int kmax_pair, double *out, void *workspace,
                       size_t workspace_bytes, void *stream) {
    if (!g.ready) return LX_ENOTINIT;
    if (nx < 0 || npair < 0 || kmax_pair < 0) return LX_EINVAL;
    if (!class_supported(lx_, la, lb)) return LX_EUNSUPPORTED;
    if (nx == 0 || npair == 0) return LX_OK;
    int rc;
    if ((rc = check_shells(aux, false)) != LX_OK) return rc;
    if ((rc = check_shells(prim, false)) != LX_OK) return rc;
    if (!x_idx || !pair_idx || !out || !workspace || kmax_pair < 1) return LX_EINVAL;
    const size_t pd_bytes = lx_eri3_workspace_bytes(lx_, la, lb, nx, npair, kmax_pair);
    if (workspace_bytes < pd_bytes) return LX_ENOMEM;
    cudaStream_t st = (cudaStream_t)stream;
    const int swapped = la < lb ? 1 : 0;
    const int cla = swapped ? lb : la, clb = swapped ? la : lb;
    DevShells dprim = dev_view(prim), daux = dev_view(aux);
    double *pd = reinterpret_cast<double *>(workspace);
    // fused path: level-0 chain targets + solid-harmonic projection in the epilogue (team kernel classes, Lx >= 2)
    if ((rc = launch_pair_data(dprim, pair_idx, npair, swapped, nullptr, kmax_pair, pd, st)) != LX_OK) return rc;
    SetMap map{(long long)npair * nx, nx, npair, x_idx, pair_idx, nullptr, kmax_pair};
    PairData pdat{pd, nullptr, kmax_pair};
    DfArgs df{g.solid[lx_], nullptr, 0};
    cudaError_t e = k_launch[3][lx_](cla, clb, map, daux, dprim, pdat, g.boys_tab, out, swapped, df, g.num_sms, st);
    if (e == cudaSuccess) {
        g.launches++;
        return LX_OK;
    }
    if (e != cudaErrorNotSupported) return cuda_fail(e);
    // fallback: Cartesian shell-sets into the workspace, then row a6 as its own kernel
    const size_t cart_bytes = (size_t)npair * nx * nc(lx_) * nc(la) * nc(lb) * sizeof(double);
    const size_t coff = (pd_bytes + 255) & ~(size_t)255;
    if (workspace_bytes < coff + cart_bytes) return LX_ENOMEM;
    double *cart = reinterpret_cast<double *>(reinterpret_cast<char *>(workspace) + coff);
    if ((rc = lx_eri3_batch(lx_, la, lb, aux, prim, x_idx, nx, pair_idx, npair, cart, workspace, pd_bytes, stream)) != LX_OK) return rc;
    return lx_cart_to_pure(lx_, (int64_t)npair * nx, nc(la) * nc(lb), cart, out, stream);
}

// ------------------------------------------------------------------------------------------------ schedule (a0)
struct lx_schedule {
    struct AuxBucket {
        int L, K;
        std::vector<int32_t> ids;   // sorted by Q descending
        std::vector<double> q;
        int32_t *d_ids = nullptr;
    };
    struct PairBucket {
        int la, lb;                 // la >= lb (pairs stored swapped if needed)
        std::vector<int32_t> pairs; // [n][2]
        std::vector<double> q;
        std::vector<long long> pd_off;
        int kmax = 1;
        int32_t *d_pairs = nullptr;
        long long *d_pd_off = nullptr;
    };
    struct Launch {
        int ab, pb;                 // bucket indices
        long long nsets;
        long long *d_cum = nullptr;
    };
    std::vector<AuxBucket> aux_b;
    std::vector<PairBucket> pair_b;
    std::vector<Launch> launches;
    long long prim_pairs = 0, nsets = 0, nints = 0;
    int naux_bf = 0, nbf = 0;
};

int lx_schedule_destroy(lx_schedule_t *s) {
    if (!s) return LX_OK;
    for (auto &b : s->aux_b) if (b.d_ids) cudaFree(b.d_ids);
    for (auto &b : s->pair_b) {
        if (b.d_pairs) cudaFree(b.d_pairs);
        if (b.d_pd_off) cudaFree(b.d_pd_off);
    }
    for (auto &l : s->launches) if (l.d_cum) cudaFree(l.d_cum);
    delete s;
    return LX_OK;
}

int lx_schedule_create(const lx_shells_t *aux, const lx_shells_t *prim, const double *q_aux, const double *q_pair,
                       const int32_t *pair_idx, int npair, double tau, lx_schedule_t **out) {
    if (!g.ready) return LX_ENOTINIT;
    if (!out) return LX_EINVAL;
    *out = nullptr;
    int rc;
    if ((rc = check_shells(aux, true)) != LX_OK) return rc;
    if ((rc = check_shells(prim, true)) != LX_OK) return rc;
    if (npair < 0 || (npair > 0 && !pair_idx)) return LX_EINVAL;
    const bool screen = q_aux && q_pair;
    for (int i = 0; i < aux->nshell; ++i) if (aux->L[i] < 0 || aux->L[i] > LX_MAX_L_AUX) return LX_EUNSUPPORTED;
    for (int i = 0; i < prim->nshell; ++i) if (prim->L[i] < 0 || prim->L[i] > LX_MAX_L_PRIM) return LX_EUNSUPPORTED;
    for (int p = 0; p < npair; ++p)
        for (int k = 0; k < 2; ++k)
            if (pair_idx[2 * p + k] < 0 || pair_idx[2 * p + k] >= prim->nshell) return LX_EINVAL;

    lx_schedule *s = new (std::nothrow) lx_schedule();
    if (!s) return LX_ENOMEM;
    s->naux_bf = aux->nshell ? aux->bf_off[aux->nshell] : 0;
    s->nbf = prim->nshell ? prim->bf_off[prim->nshell] : 0;

    // aux buckets keyed by (L, K), each sorted by Q descending (ties by shell id → deterministic)
    {
        std::vector<int> order(aux->nshell);
        for (int i = 0; i < aux->nshell; ++i) order[i] = i;
        auto qa = [&](int i) { return screen ? q_aux[i] : 0.0; };
        std::sort(order.begin(), order.end(), [&](int x, int y) {
            if (aux->L[x] != aux->L[y]) return aux->L[x] < aux->L[y];
            if (aux->K[x] != aux->K[y]) return aux->K[x] < aux->K[y];
            if (qa(x) != qa(y)) return qa(x) > qa(y);
            return x < y;
        });
        for (int i : order) {
            if (s->aux_b.empty() || s->aux_b.back().L != aux->L[i] || s->aux_b.back().K != aux->K[i]) {
                s->aux_b.emplace_back();
                s->aux_b.back().L = aux->L[i];
                s->aux_b.back().K = aux->K[i];
            }
            s->aux_b.back().ids.push_back(i);
            s->aux_b.back().q.push_back(qa(i));
        }
    }
    // pair buckets keyed by (La, Lb) with La >= Lb, ordered by K_a K_b then Q descending
    {
        struct P { int a, b, kab; double q; };
        std::vector<P> ps(npair);
        for (int p = 0; p < npair; ++p) {
            int a = pair_idx[2 * p], b = pair_idx[2 * p + 1];
            if (prim->L[a] < prim->L[b]) std::swap(a, b);
            ps[p] = P{a, b, prim->K[a] * prim->K[b], screen ? q_pair[p] : 0.0};
        }
        std::sort(ps.begin(), ps.end(), [&](const P &x, const P &y) {
            const int lax = prim->L[x.a], lbx = prim->L[x.b], lay = prim->L[y.a], lby = prim->L[y.b];
            if (lax != lay) return lax < lay;
            if (lbx != lby) return lbx < lby;
            if (x.kab != y.kab) return x.kab < y.kab;
            if (x.q != y.q) return x.q > y.q;
            if (x.a != y.a) return x.a < y.a;
            return x.b < y.b;
        });
        long long po = 0;
        for (const P &p : ps) {
            const int la = prim->L[p.a], lb = prim->L[p.b];
            // one bucket per (La, Lb) and contraction class K_a K_b = 1 | 2 | 3-4 | 5-9 | >= 10: launches are nearly uniform in
            // K, and K-aware kernel choices (lx_inst.cu) see a tight bound
            auto kclass = [](int k) { return k <= 1 ? 0 : (k == 2 ? 1 : (k <= 4 ? 2 : (k <= 9 ? 3 : 4))); };
            if (s->pair_b.empty() || s->pair_b.back().la != la || s->pair_b.back().lb != lb ||
                kclass(s->pair_b.back().kmax) != kclass(p.kab)) {
                s->pair_b.emplace_back();
                s->pair_b.back().la = la;
                s->pair_b.back().lb = lb;
            }
            auto &b = s->pair_b.back();
            b.pairs.push_back(p.a);
            b.pairs.push_back(p.b);
            b.q.push_back(p.q);
            b.pd_off.push_back(po);
            b.kmax = std::max(b.kmax, p.kab);
            po += p.kab;
        }
        s->prim_pairs = po;
    }
    // per class: Schwarz prefix lengths → cumulative set counts
    for (size_t ib = 0; ib < s->pair_b.size(); ++ib) {
        auto &pb = s->pair_b[ib];
        const size_t np = pb.q.size();
        for (size_t ia = 0; ia < s->aux_b.size(); ++ia) {
            auto &ab = s->aux_b[ia];
            std::vector<long long> cum(np + 1, 0);
            for (size_t p = 0; p < np; ++p) {
                long long n = (long long)ab.ids.size();
                if (screen) {
                    // aux q sorted descending: survivors (q_x*q_p >= tau, the same double expression the oracle
                    // uses) are a prefix; binary search for its length
                    size_t lo = 0, hi = ab.ids.size();
                    while (lo < hi) {
                        const size_t mid = (lo + hi) / 2;
                        if (ab.q[mid] * pb.q[p] < tau) hi = mid; else lo = mid + 1;
                    }
                    n = (long long)lo;
                }
                cum[p + 1] = cum[p] + n;
            }
            if (cum[np] == 0) continue;
            lx_schedule::Launch l;
            l.ab = (int)ia;
            l.pb = (int)ib;
            l.nsets = cum[np];
            if (cudaMalloc(&l.d_cum, cum.size() * sizeof(long long)) != cudaSuccess ||
                cudaMemcpy(l.d_cum, cum.data(), cum.size() * sizeof(long long), cudaMemcpyHostToDevice) != cudaSuccess) {
                lx_schedule_destroy(s);
                return cuda_fail(cudaGetLastError());
            }
            s->launches.push_back(l);
            s->nsets += l.nsets;
            s->nints += l.nsets * nc(ab.L) * nc(pb.la) * nc(pb.lb);
        }
    }
    for (auto &b : s->aux_b) {
        if (cudaMalloc(&b.d_ids, b.ids.size() * sizeof(int32_t)) != cudaSuccess ||
            cudaMemcpy(b.d_ids, b.ids.data(), b.ids.size() * sizeof(int32_t), cudaMemcpyHostToDevice) != cudaSuccess) {
            lx_schedule_destroy(s);
            return cuda_fail(cudaGetLastError());
        }
    }
    for (auto &b : s->pair_b) {
        if (cudaMalloc(&b.d_pairs, b.pairs.size() * sizeof(int32_t)) != cudaSuccess ||
            cudaMemcpy(b.d_pairs, b.pairs.data(), b.pairs.size() * sizeof(int32_t), cudaMemcpyHostToDevice) != cudaSuccess ||
            cudaMalloc(&b.d_pd_off, b.pd_off.size() * sizeof(long long)) != cudaSuccess ||
            cudaMemcpy(b.d_pd_off, b.pd_off.data(), b.pd_off.size() * sizeof(long long), cudaMemcpyHostToDevice) != cudaSuccess) {
            lx_schedule_destroy(s);
            return cuda_fail(cudaGetLastError());
        }
    }
    *out = s;
    return LX_OK;
}

int64_t lx_schedule_num_sets(const lx_schedule_t *s) { return s ? s->nsets : 0; }
int64_t lx_schedule_num_integrals(const lx_schedule_t *s) { return s ? s->nints : 0; }
size_t lx_df_workspace_bytes(const lx_schedule_t *s) {
    return s ? (size_t)s->prim_pairs * PD_STRIDE * sizeof(double) + 256 : 256;
}

static int df_run(const lx_schedule_t *s, const lx_shells_t *aux, const lx_shells_t *prim, int mode, const DfArgs &df,
                  void *workspace, size_t workspace_bytes, cudaStream_t st) {
    if (workspace_bytes < lx_df_workspace_bytes(s)) return LX_ENOMEM;
    DevShells dprim = dev_view(prim), daux = dev_view(aux);
    double *pd = reinterpret_cast<double *>(workspace);
    int rc;
    for (const auto &pb : s->pair_b)
        if ((rc = launch_pair_data(dprim, pb.d_pairs, (int)pb.q.size(), 0, pb.d_pd_off, pb.kmax, pd, st)) != LX_OK) return rc;
    // fork: the side streams wait for the pre-pass (and for the caller's memset of the output); the launches go round the
    // streams; join: the caller's stream waits for every side stream.  Stream order is all the synchronisation the pass needs.
    // Only where the launches are small: measured (B200) config 4 (280 k sets per launch) 11.9 -> 10.4 ms with four streams, config 5
    // (10 M sets per launch) 2.23 -> 2.43 s — large launches fill the GPU by themselves and only disturb each other.
    const bool small_launches = !s->launches.empty() && s->nsets / (long long)s->launches.size() < 2000000LL;
    const int ns = small_launches ? g.n_side : 0;
    if (ns > 0) {
        LX_CUDA(cudaEventRecord(g.fork_ev, st));
        for (int i = 0; i < ns; ++i) LX_CUDA(cudaStreamWaitEvent(g.side[i], g.fork_ev, 0));
    }
    int turn = 0;
    for (const auto &l : s->launches) {
        const auto &ab = s->aux_b[l.ab];
        const auto &pb = s->pair_b[l.pb];
        SetMap map{l.nsets, (int)ab.ids.size(), (int)pb.q.size(), ab.d_ids, pb.d_pairs, l.d_cum, pb.kmax * ab.K};
        PairData pdat{pd, pb.d_pd_off, pb.kmax};
        cudaStream_t ls = turn == 0 ? st : g.side[turn - 1];
        turn = (turn + 1) % (ns + 1);
        cudaError_t e = k_launch[mode][ab.L](pb.la, pb.lb, map, daux, dprim, pdat, g.boys_tab, nullptr, 0, df, g.num_sms, ls);
        g.launches++;
        if (e != cudaSuccess) return cuda_fail(e);
    }
    for (int i = 0; i < ns; ++i) {
        LX_CUDA(cudaEventRecord(g.side_ev[i], g.side[i]));
        LX_CUDA(cudaStreamWaitEvent(st, g.side_ev[i], 0));
    }
    return LX_OK;
}

int lx_df_gamma(const lx_schedule_t *s, const lx_shells_t *aux, const lx_shells_t *prim, const double *D, int ldD,
                double *gamma, void *workspace, size_t workspace_bytes, void *stream) {
    if (!g.ready) return LX_ENOTINIT;
    if (!s || !D || !gamma || !workspace) return LX_EINVAL;
    int rc;
    if ((rc = check_shells(aux, true)) != LX_OK) return rc;
    if ((rc = check_shells(prim, true)) != LX_OK) return rc;
    if (ldD < s->nbf) return LX_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    LX_CUDA(cudaMemsetAsync(gamma, 0, (size_t)s->naux_bf * sizeof(double), st));
    DfArgs df{D, gamma, ldD};
    return df_run(s, aux, prim, 1, df, workspace, workspace_bytes, st);
}

int lx_df_J(const lx_schedule_t *s, const lx_shells_t *aux, const lx_shells_t *prim, const double *d, double *J,
            int ldJ, void *workspace, size_t workspace_bytes, void *stream) {
    if (!g.ready) return LX_ENOTINIT;
    if (!s || !d || !J || !workspace) return LX_EINVAL;
    int rc;
    if ((rc = check_shells(aux, true)) != LX_OK) return rc;
    if ((rc = check_shells(prim, true)) != LX_OK) return rc;
    if (ldJ < s->nbf) return LX_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    LX_CUDA(cudaMemsetAsync(J, 0, (size_t)s->nbf * (size_t)ldJ * sizeof(double), st));
    DfArgs df{d, J, ldJ};
    return df_run(s, aux, prim, 2, df, workspace, workspace_bytes, st);
}

// ------------------------------------------------------------------------------------------------ host-buffer path
static size_t align256(size_t x) { return (x + 255) & ~(size_t)255; }

int lx_eri3_batch_host(int lx_, int la, int lb, const lx_shells_t *aux, const lx_shells_t *prim,
                       const int32_t *x_idx, int nx, const int32_t *pair_idx, int npair, double *out) {
    if (!g.ready) return LX_ENOTINIT;
    if (nx < 0 || npair < 0) return LX_EINVAL;
    if (!class_supported(lx_, la, lb)) return LX_EUNSUPPORTED;
    if (nx == 0 || npair == 0) return LX_OK;
    int rc;
    if ((rc = check_shells(aux, false)) != LX_OK) return rc;
    if ((rc = check_shells(prim, false)) != LX_OK) return rc;
    if (!x_idx || !pair_idx || !out) return LX_EINVAL;
    int kmax = 1;
    for (int p = 0; p < npair; ++p) kmax = std::max(kmax, prim->K[pair_idx[2 * p]] * prim->K[pair_idx[2 * p + 1]]);
    const size_t nint = (size_t)npair * nx * nc(lx_) * nc(la) * nc(lb);
    const size_t ws = lx_eri3_workspace_bytes(lx_, la, lb, nx, npair, kmax);
    auto tab_bytes = [](const lx_shells_t *s, size_t *np) {
        *np = (size_t)s->prim_off[s->nshell];
        return 3 * align256((size_t)(s->nshell + 1) * 4) + align256((size_t)s->nshell * 24) + 2 * align256(*np * 8);
    };
    size_t npx, npp;
    const size_t in_bytes = tab_bytes(aux, &npx) + tab_bytes(prim, &npp) + align256((size_t)nx * 4) + align256((size_t)npair * 8);
    const size_t total = in_bytes + align256(ws) + align256(nint * 8);
    std::lock_guard<std::mutex> lock(g_mu);
    if (g.arena_bytes < total) {
        if (g.arena) cudaFree(g.arena);
        g.arena = nullptr;
        g.arena_bytes = 0;
        LX_CUDA(cudaMalloc(&g.arena, total));
        g.arena_bytes = total;
    }
    char *base = reinterpret_cast<char *>(g.arena);
    size_t o = 0;
    cudaStream_t st = 0;
    auto put = [&](const void *src, size_t bytes) -> void * {
        void *d = base + o;
        cudaMemcpyAsync(d, src, bytes, cudaMemcpyHostToDevice, st);
        o += align256(bytes);
        return d;
    };
    auto put_tab = [&](const lx_shells_t *s, size_t np, lx_shells_t *d) {
        d->nshell = s->nshell;
        d->L = (const int32_t *)put(s->L, (size_t)s->nshell * 4);
        d->K = (const int32_t *)put(s->K, (size_t)s->nshell * 4);
        d->prim_off = (const int32_t *)put(s->prim_off, (size_t)(s->nshell + 1) * 4);
        d->center = (const double *)put(s->center, (size_t)s->nshell * 24);
        d->zeta = (const double *)put(s->zeta, np * 8);
        d->coef = (const double *)put(s->coef, np * 8);
        d->bf_off = nullptr;
    };
    lx_shells_t daux, dprim;
    put_tab(aux, npx, &daux);
    put_tab(prim, npp, &dprim);
    const int32_t *dx = (const int32_t *)put(x_idx, (size_t)nx * 4);
    const int32_t *dp = (const int32_t *)put(pair_idx, (size_t)npair * 8);
    void *dws = base + o;
    o += align256(ws);
    double *dout = reinterpret_cast<double *>(base + o);
    LX_CUDA(cudaGetLastError());
    rc = lx_eri3_batch(lx_, la, lb, &daux, &dprim, dx, nx, dp, npair, dout, dws, ws, st);
    if (rc != LX_OK) return rc;
    LX_CUDA(cudaMemcpyAsync(out, dout, nint * 8, cudaMemcpyDeviceToHost, st));
    LX_CUDA(cudaStreamSynchronize(st));
    return LX_OK;
}

}  // extern "C"
