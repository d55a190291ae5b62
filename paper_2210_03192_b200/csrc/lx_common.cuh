// lx_common.cuh — shared device-side definitions of liblx (sm_100a only).
//
// Notation follows arxiv 2210.03192: a,b = primary (bra) Cartesian shells on centres A,B with exponents
// ζa, ζb; c = auxiliary (ket) shell X on centre C with exponent ζc; γ = ζa+ζb (eq. 14), ρ = γζc/(γ+ζc) (eq. 15),
// P (eq. 16), AB = A−B (eq. 17), PC = P−C (eq. 18); [e 0|c]^(m) auxiliary integrals of §2.5.1 (lines 104–124).
#pragma once
#include <atomic>
#include <cstdint>
#include <cuda_runtime.h>

#include "../../include/lx.h"

namespace lx {

// number of Cartesian components of a shell and of all shells of lower degree
__host__ __device__ constexpr int nc(int l) { return (l + 1) * (l + 2) / 2; }
__host__ __device__ constexpr int off(int l) { return l * (l + 1) * (l + 2) / 6; }
__host__ __device__ constexpr int cmax(int a, int b) { return a > b ? a : b; }
__host__ __device__ constexpr int cmin(int a, int b) { return a < b ? a : b; }

// ---- Boys table: F_m on a uniform grid T_i = i/16, rows m = 0..BOYS_MROWS-1,
// used by a degree-7 Taylor expansion in T around the nearest grid point; T >= BOYS_TMAX uses the asymptotic form.
constexpr int BOYS_MMAX = 18;                       // largest m any kernel may request
constexpr int BOYS_DEG = 7;
constexpr int BOYS_MROWS = BOYS_MMAX + BOYS_DEG + 1;  // 26
constexpr int BOYS_PER_UNIT = 16;
constexpr int BOYS_TMAX = 84;                       // Γ(m+½,T)/Γ(m+½) < 1e-17 for m <= 18, T >= 84
constexpr int BOYS_NGRID = BOYS_TMAX * BOYS_PER_UNIT + 2;

// Device views --------------------------------------------------------------------------------------------------
struct DevShells {
    const int32_t *L, *K, *prim_off;
    const double *center, *zeta, *coef;
    const int32_t *bf_off;
};
inline DevShells dev_view(const lx_shells_t *s) {
    return DevShells{s->L, s->K, s->prim_off, s->center, s->zeta, s->coef, s->bf_off};
}

// How a flat shell-set id maps onto (pair slot, aux slot).
//   dense  (cum == nullptr): sid = p * nx + x                      (lx_eri3_batch)
//   prefix (cum != nullptr): sets of pair p are x = 0 .. cum[p+1]-cum[p]-1 of x_list (Schwarz prefix, DF calls)
struct SetMap {
    long long nsets;
    int nx;
    int npair;
    const int32_t *x_list;     // aux shell ids
    const int32_t *pair_list;  // [npair][2] primary shell ids in CANONICAL order (L of first >= L of second)
    const long long *cum;      // [npair+1] or nullptr
    int khint;                 // host-side upper bound of K_a K_b K_x over the launch where known (0 = unknown): picks K-aware kernels
};

// Primitive-pair data: per primitive pair PD_STRIDE doubles {γ, Px, Py, Pz, K_ij, 1/(2γ)},
// K_ij = c_i c_j exp(−ζaζb/γ |AB|²)  (the exponential factor of eq. 4).
constexpr int PD_STRIDE = 6;
struct PairData {
    const double *pd;
    const long long *pd_off;  // per-pair offset in primitive pairs, or nullptr → p * kstride
    int kstride;
};

// What the digestion step needs.  mode: 0 = store, 1 = γ, 2 = J.
struct DfArgs {
    const double *D;   // γ: density (nbf × nbf, ld)        J: fit vector d [naux_bf]
    double *out;       // γ: gamma [naux_bf]                 J: J (nbf × nbf, ld)
    int ld;
};

// Function attributes are per device: raise the dynamic shared-memory limit of `kern` once per device of this process
// (`mask` = one bit per device ordinal, a static of the launcher instantiation).
template <class KernT>
inline cudaError_t ensure_dyn_smem(KernT kern, size_t smem, std::atomic<unsigned long long> &mask) {
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    const unsigned long long bit = 1ull << (dev & 63);
    if (mask.load(std::memory_order_acquire) & bit) return cudaSuccess;
    e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    mask.fetch_or(bit, std::memory_order_release);
    return cudaSuccess;
}

// Which shell of a pair carries the VRR (eq. 3 builds [e0|0] on centre A, eq. 1 then transfers onto b).  The transfer
// (x−B)^b = Σ_k C(b,k) AB^{b−k} (x−A)^k cancels by (|AB|/σ)^{Lb} when the product Gaussian sits near B (ζb >> ζa): the
// moments about A are then of size |AB|^e while the result is of size σ^e.  Building on the shell with the LARGER
// (most diffuse) exponent keeps P near A and the transfer free of cancellation; for La = Lb the two roles can be
// exchanged per shell pair at no cost (measured on config 3: 1e-12 -> 1e-14 of the batch maximum).
__device__ __forceinline__ double shell_min_zeta(const DevShells &s, int i) {
    const int o = s.prim_off[i], k = s.K[i];
    double m = s.zeta[o];
    for (int j = 1; j < k; ++j) m = fmin(m, s.zeta[o + j]);
    return m;
}

// F_m(T)·scale for one m (thread-per-(set,m) evaluation).
__device__ __forceinline__ double boys_one(const double *__restrict__ tab, int m, double T) {
    if (T < (double)BOYS_TMAX) {
        const int i = __double2int_rn(T * (double)BOYS_PER_UNIT);
        const double d = (double)i * (1.0 / BOYS_PER_UNIT) - T;  // −Δ
        const double *row = tab + (size_t)i * BOYS_MROWS + m;
        // F_m(T) = Σ_k F_{m+k}(T_i) (T_i − T)^k / k!   (dF_m/dT = −F_{m+1})
        double r = __ldg(row + 7) * (1.0 / 7.0);
        r = fma(r, d, __ldg(row + 6)) * (1.0 / 6.0);
        r = fma(r, d, __ldg(row + 5)) * (1.0 / 5.0);
        r = fma(r, d, __ldg(row + 4)) * (1.0 / 4.0);
        r = fma(r, d, __ldg(row + 3)) * (1.0 / 3.0);
        r = fma(r, d, __ldg(row + 2)) * (1.0 / 2.0);
        r = fma(r, d, __ldg(row + 1));
        r = fma(r, d, __ldg(row));
        return r;
    }
    // asymptotic: F_m(T) = (2m−1)!!/(2T)^m · ½ sqrt(π/T)   (the incomplete-gamma tail is < 1e-17 relative here)
    // (2T is exact, so its powers carry only rounding errors; the odd-integer product is exact up to 29!!)
    const double x = T + T;
    double pw = 1.0, odd = 1.0;
    for (int k = 0; k < m; ++k) {
        pw *= x;
        odd *= (double)(2 * k + 1);
    }
    return 0.5 * sqrt(3.14159265358979323846 / T) * (odd / pw);
}

// All of F_0..F_M(T) for one thread: top order by the table, then downward recursion
// F_{m−1} = (2T F_m + e^{−T})/(2m−1) (stable for every T); asymptotic branch upward without the e^{−T} term.
template <int M>
__device__ __forceinline__ void boys_all(const double *__restrict__ tab, double T, double (&F)[M + 1]) {
    if (T < (double)BOYS_TMAX) {
        F[M] = boys_one(tab, M, T);
        if constexpr (M > 0) {
            const double eT = exp(-T);
            const double T2 = T + T;
#pragma unroll
            for (int m = M; m >= 1; --m) F[m - 1] = fma(T2, F[m], eT) * (1.0 / (double)(2 * m - 1));
        }
    } else {
        F[0] = 0.5 * sqrt(3.14159265358979323846 / T);
        const double h = 0.5 / T;
#pragma unroll
        for (int m = 0; m < M; ++m) F[m + 1] = F[m] * ((double)(2 * m + 1) * h);
    }
}

// Cartesian component table, indexed by the cumulative component index g = off(l) + idx (order G2):
// packed byte 0..2 = (x,y,z) powers, byte 3 = recursion direction (the axis with the smallest positive power,
// so that the two-term form of the recurrences is used whenever the shell allows it).
constexpr int CART_LMAX = 2 * LX_MAX_L_PRIM;                 // bra shells reach la+lb
constexpr int CART_N = off(CART_LMAX + 1);                   // 165
__host__ __device__ constexpr uint32_t cart_entry(int g) {
    int l = 0;
    while (off(l + 1) <= g) ++l;
    int idx = g - off(l), i = 0;
    while ((i + 1) * (i + 2) / 2 <= idx) ++i;                // i = y+z
    const int z = idx - i * (i + 1) / 2, y = i - z, x = l - i;
    int dir = 0, best = 99;
    if (x > 0 && x < best) { best = x; dir = 0; }
    if (y > 0 && y < best) { best = y; dir = 1; }
    if (z > 0 && z < best) { best = z; dir = 2; }
    return (uint32_t)x | ((uint32_t)y << 8) | ((uint32_t)z << 16) | ((uint32_t)dir << 24);
}

// Index algebra in order G2: idx(a) = s(s+1)/2 + a_z with s = a_y + a_z, so lowering/raising one axis is
//   x: idx unchanged      y: idx ∓ s (−) / + s+1 (+)      z: idx − s − 1 (−) / + s + 2 (+)
__device__ __forceinline__ int idx_down1(int idx, int s, int dir) { return dir == 0 ? idx : (dir == 1 ? idx - s : idx - s - 1); }
__device__ __forceinline__ int idx_down2(int idx, int s, int dir) {
    return dir == 0 ? idx : (dir == 1 ? idx - 2 * s + 1 : idx - 2 * s - 1);
}
__device__ __forceinline__ int idx_up1(int idx, int s, int dir) { return dir == 0 ? idx : (dir == 1 ? idx + s + 1 : idx + s + 2); }

}  // namespace lx
