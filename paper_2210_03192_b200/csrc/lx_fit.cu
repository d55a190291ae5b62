// lx_fit.cu — the fit solve d = V⁻¹ γ of density fitting (second half):
// Cholesky factorisation V = L Lᵀ of the two-centre metric and two triangular solves per right-hand side.
//
// The factorisation is a dense LAPACK routine (potrf), not part of the integral path, and is taken from cuSOLVER as a
// plain library call (like a library GEMM would be).  cuSOLVER is opened at the first call with dlopen, so that liblx.so
// itself has no link-time dependency on it: where the library is missing, a factorising call returns LX_EUNSUPPORTED and
// every other entry point works as before.
//
// The two triangular solves — the part that runs every iteration — are kernels of this file: the library's potrs treats a
// single right-hand side as a matrix (trsm) and took 0.79 s at n = 39 680 where the factor is only read once each way
// (2 x 6.3 GB).  Layout: potrf(LOWER) on the column-major image of the symmetric array leaves, in ROW-major terms, the upper
// triangle U = Lᵀ (U[i][j], j >= i, rows contiguous), V = Uᵀ U.
//   forward   Uᵀ y = g : block column by block column (64 wide): every CTA solves the 64 x 64 diagonal block in shared
//             memory (redundantly: cheaper than a second launch), then subtracts the block's contribution from its 128
//             later entries of g — rows of U read along j, coalesced.
//   backward  U d = y  : block row by block row from the end: the dot product of each row with the part of d already known
//             is split over CTAs of 2 048 entries (the row is contiguous; 8 loads per thread, all in flight), the last CTA
//             to finish (ticket) sums the partial results in a fixed order and solves the diagonal block.
// 2 n/64 launches per right-hand side, each reading its rows of the factor exactly once.
#include <cusolverDn.h>
#include <dlfcn.h>

#include <mutex>

#include "../../include/lx.h"
#include "lx_state.h"

namespace {

struct Solver {
    bool tried = false, ok = false;
    void *so = nullptr;
    decltype(&cusolverDnCreate) create = nullptr;
    decltype(&cusolverDnDestroy) destroy = nullptr;
    decltype(&cusolverDnCreateParams) create_params = nullptr;
    decltype(&cusolverDnDestroyParams) destroy_params = nullptr;
    decltype(&cusolverDnXpotrf_bufferSize) potrf_size = nullptr;
    decltype(&cusolverDnXpotrf) potrf = nullptr;
    cusolverDnHandle_t handle = nullptr;      // made once per device, kept for the life of the process
    int handle_dev = -1;

    template <class F>
    bool sym(F &f, const char *name) {
        f = reinterpret_cast<F>(dlsym(so, name));
        return f != nullptr;
    }
    bool load() {
        if (tried) return ok;
        tried = true;
        for (const char *n : {"libcusolver.so.11", "libcusolver.so.12", "libcusolver.so"}) {
            so = dlopen(n, RTLD_NOW | RTLD_GLOBAL);
            if (so) break;
        }
        if (!so) return false;
        ok = sym(create, "cusolverDnCreate") && sym(destroy, "cusolverDnDestroy") &&
             sym(create_params, "cusolverDnCreateParams") && sym(destroy_params, "cusolverDnDestroyParams") &&
             sym(potrf_size, "cusolverDnXpotrf_bufferSize") && sym(potrf, "cusolverDnXpotrf");
        return ok;
    }
    // the handle belongs to the device that was current when it was made (lx_init may have moved the library since)
    bool ensure() {
        if (!load()) return false;
        int cur = -1;
        if (cudaGetDevice(&cur) != cudaSuccess) return false;
        if (handle && handle_dev != cur) {
            destroy(handle);
            handle = nullptr;
        }
        if (!handle) {
            if (create(&handle) != CUSOLVER_STATUS_SUCCESS) { handle = nullptr; return false; }
            handle_dev = cur;
        }
        return true;
    }
};

constexpr int TB = 64;       // block width of the triangular solves
constexpr int TT = 256;      // threads per CTA, backward step
constexpr int TF = 128;      // threads per CTA, forward step (64 loads are held in registers: 170 registers per thread)

// The 64 x 64 diagonal block in shared memory: upper triangle of U, unit diagonal in the padding of a ragged last block.
__device__ __forceinline__ void load_diag(double (*Us)[TB + 1], const double *__restrict__ U, long long ld, int j0, int m,
                                          int tid, int nthreads) {
    for (int e = tid; e < TB * TB; e += nthreads) {
        const int i = e / TB, j = e - i * TB;
        Us[i][j] = (j >= i && j < m) ? U[(long long)(j0 + i) * ld + j0 + j] : (i == j ? 1.0 : 0.0);
    }
}

// Diagonal solves by ONE warp, lane l holding entries l and l+32 in registers; the pivot value travels by shuffle, so a step
// of the serial chain is multiply (by the reciprocal pivot) - shuffle - fma, with no block barrier.
// forward: Uᵀ y = r  (y_i = r_i / U_ii, then r_j -= U_ij y_i for j > i)
__device__ __forceinline__ void diag_fwd(const double (*Us)[TB + 1], double r0, double r1, double *ys, int lane) {
    const double v0 = 1.0 / Us[lane][lane], v1 = 1.0 / Us[lane + 32][lane + 32];
#pragma unroll 8
    for (int i = 0; i < 32; ++i) {
        const double yi = __shfl_sync(0xffffffffu, r0 * v0, i);
        if (lane == i) ys[i] = yi;
        if (lane > i) r0 = fma(-Us[i][lane], yi, r0);
        r1 = fma(-Us[i][lane + 32], yi, r1);
    }
#pragma unroll 8
    for (int i = 32; i < 64; ++i) {
        const double yi = __shfl_sync(0xffffffffu, r1 * v1, i - 32);
        if (lane == i - 32) ys[i] = yi;
        if (lane + 32 > i) r1 = fma(-Us[i][lane + 32], yi, r1);
    }
}
// backward: U d = t  (d_c = t_c / U_cc, then t_k -= U_kc d_c for k < c)
__device__ __forceinline__ void diag_bwd(const double (*Us)[TB + 1], double t0, double t1, double *ds, int lane) {
    const double v0 = 1.0 / Us[lane][lane], v1 = 1.0 / Us[lane + 32][lane + 32];
#pragma unroll 8
    for (int c = 63; c >= 32; --c) {
        const double dc = __shfl_sync(0xffffffffu, t1 * v1, c - 32);
        if (lane == c - 32) ds[c] = dc;
        if (lane + 32 < c) t1 = fma(-Us[lane + 32][c], dc, t1);
        t0 = fma(-Us[lane][c], dc, t0);
    }
#pragma unroll 8
    for (int c = 31; c >= 0; --c) {
        const double dc = __shfl_sync(0xffffffffu, t0 * v0, c);
        if (lane == c) ds[c] = dc;
        if (lane < c) t0 = fma(-Us[lane][c], dc, t0);
    }
}

// forward step of block column j0: y[j0..j0+m) from r, then r[j] -= Σ_i U[j0+i][j] y[j0+i] for j >= j0+m.
__global__ void __launch_bounds__(TF)
tri_fwd_kernel(const double *__restrict__ U, long long ld, int n, int j0, double *__restrict__ r, double *__restrict__ y) {
    __shared__ double Us[TB][TB + 1];
    __shared__ double ys[TB];
    const int m = min(TB, n - j0), tid = threadIdx.x;
    load_diag(Us, U, ld, j0, m, tid, TF);
    const long long j = (long long)j0 + m + (long long)blockIdx.x * TF + tid;
    const double rj = j < n ? r[j] : 0.0;
    // the thread's 64 entries of the block row (8·ld bytes apart) are requested BEFORE the barrier and the diagonal solve:
    // they do not depend on y, the barrier keeps ptxas from sinking them, and their latency hides behind the solve
    const double *col = U + (long long)j0 * ld + (j < n ? j : (long long)j0);
    const bool full = m == TB;
    double v[TB];
    if (full) {
#pragma unroll
        for (int i = 0; i < TB; ++i) v[i] = __ldcs(col + (long long)i * ld);
    }
    __syncthreads();
    if (tid < 32) {                                  // r[j0..j0+m) is not written by this launch
        const double r0 = tid < m ? r[j0 + tid] : 0.0, r1 = tid + 32 < m ? r[j0 + tid + 32] : 0.0;
        diag_fwd(Us, r0, r1, ys, tid);
    }
    __syncthreads();
    if (blockIdx.x == 0 && tid < m) y[j0 + tid] = ys[tid];
    if (j < n) {
        double s0 = 0.0, s1 = 0.0, s2 = 0.0, s3 = 0.0;
        if (full) {
#pragma unroll
            for (int i = 0; i < TB; i += 4) {
                s0 = fma(v[i], ys[i], s0);
                s1 = fma(v[i + 1], ys[i + 1], s1);
                s2 = fma(v[i + 2], ys[i + 2], s2);
                s3 = fma(v[i + 3], ys[i + 3], s3);
            }
        } else {
            for (int i = 0; i < m; ++i) s0 = fma(col[(long long)i * ld], ys[i], s0);
        }
        r[j] = rj - ((s0 + s1) + (s2 + s3));
    }
}

// backward step of block row j0: CTA (i, c) takes chunk c (TC entries) of the dot product Σ_{j >= j0+m} U[j0+i][j] d[j] of row
// i into part[i][c]; the last CTA to finish (ticket) forms t_i = y_i − Σ_c part[i][c] (fixed order) and solves the diagonal
// block for d[j0..j0+m).  Every CTA loads the diagonal block up front (its latency hides behind the row loads; which CTA
// finishes last is not known before).
constexpr int TC = 8 * TT;   // entries of a row per CTA: 8 per thread, all requested at once

__global__ void __launch_bounds__(TT)
tri_bwd_kernel(const double *__restrict__ U, long long ld, int n, int j0, const double *__restrict__ y, double *d,
               double *part, int npart, unsigned *ticket) {
    __shared__ double Us[TB][TB + 1];
    __shared__ double ds[TB];
    __shared__ double red[TT / 32];
    __shared__ bool last;
    const int m = min(TB, n - j0), tid = threadIdx.x, i = blockIdx.x, c = blockIdx.y;
    load_diag(Us, U, ld, j0, m, tid, TT);
    const double *row = U + (long long)(j0 + i) * ld;
    const long long jb = (long long)j0 + m + (long long)c * TC + tid;
    double a[8], b[8];
#pragma unroll
    for (int k = 0; k < 8; ++k) {
        const long long j = jb + k * TT;
        a[k] = j < n ? __ldcs(row + j) : 0.0;
        b[k] = j < n ? d[j] : 0.0;
    }
    __syncthreads();                                 // scheduling fence: ptxas otherwise sinks the loads between the FMAs
    double s = 0.0;
#pragma unroll
    for (int k = 0; k < 8; ++k) s = fma(a[k], b[k], s);
    for (int o = 16; o; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if ((tid & 31) == 0) red[tid >> 5] = s;
    __syncthreads();
    if (tid == 0) {
        double acc = 0.0;
        for (int w = 0; w < TT / 32; ++w) acc += red[w];
        part[i * npart + c] = acc;
        __threadfence();
        last = atomicAdd(ticket, 1u) == (unsigned)(m * gridDim.y - 1);
    }
    __syncthreads();
    if (!last) return;
    __threadfence();
    if (tid == 0) *ticket = 0u;                      // ready for the next launch (stream order)
    if (tid < 32) {
        double t0 = tid < m ? y[j0 + tid] : 0.0, t1 = tid + 32 < m ? y[j0 + tid + 32] : 0.0;
        for (int q = 0; q < (int)gridDim.y; ++q) {
            if (tid < m) t0 -= __ldcg(part + tid * npart + q);
            if (tid + 32 < m) t1 -= __ldcg(part + (tid + 32) * npart + q);
        }
        diag_bwd(Us, t0, t1, ds, tid);
    }
    __syncthreads();
    if (tid < m) d[j0 + tid] = ds[tid];
}

Solver g_solver;
std::mutex g_mu;

}  // namespace

extern "C" int lx_fit_solve(double *V_dev, long long ld, int n, double *rhs_dev, int nrhs, int factored) {
    if (!lx::state_ready()) return LX_ENOTINIT;
    if (n < 0 || nrhs < 0 || ld < n) return LX_EINVAL;
    if (n == 0) return LX_OK;
    if (!V_dev || (nrhs > 0 && !rhs_dev)) return LX_EINVAL;
    std::lock_guard<std::mutex> lock(g_mu);
    int rc = LX_OK;
    void *dwork = nullptr, *hwork = nullptr;
    double *scratch = nullptr;
    int *dinfo = nullptr, info = 0;
    auto cuda_ok = [&](cudaError_t e) {
        if (e != cudaSuccess && rc == LX_OK) rc = lx::state_cuda_fail((int)e);
        return e == cudaSuccess;
    };
    do {
        if (!factored) {
            if (!g_solver.ensure()) { rc = LX_EUNSUPPORTED; break; }
            cusolverDnParams_t prm = nullptr;
            bool ok = g_solver.create_params(&prm) == CUSOLVER_STATUS_SUCCESS;
            // V is symmetric: its row-major image is its column-major image
            const cublasFillMode_t uplo = CUBLAS_FILL_MODE_LOWER;
            size_t dbytes = 0, hbytes = 0;
            ok = ok && g_solver.potrf_size(g_solver.handle, prm, uplo, n, CUDA_R_64F, V_dev, ld, CUDA_R_64F, &dbytes, &hbytes) ==
                           CUSOLVER_STATUS_SUCCESS;
            if (ok) ok = cuda_ok(cudaMalloc((void **)&dinfo, sizeof(int))) && (!dbytes || cuda_ok(cudaMalloc(&dwork, dbytes)));
            if (ok && hbytes && !(hwork = malloc(hbytes))) { rc = LX_ENOMEM; ok = false; }
            ok = ok && g_solver.potrf(g_solver.handle, prm, uplo, n, CUDA_R_64F, V_dev, ld, CUDA_R_64F, dwork, dbytes, hwork,
                                      hbytes, dinfo) == CUSOLVER_STATUS_SUCCESS;
            ok = ok && cuda_ok(cudaMemcpy(&info, dinfo, sizeof(int), cudaMemcpyDeviceToHost));
            if (prm) g_solver.destroy_params(prm);
            if (!ok) { if (rc == LX_OK) rc = lx::state_cuda_fail((int)cudaErrorUnknown); break; }
            if (info != 0) { rc = LX_ENOTPD; break; }                // a leading minor is not positive definite
        }
        if (nrhs > 0) {
            // y [n] | part [TB][npart] | ticket
            const int npart = (n + TC - 1) / TC;
            if (!cuda_ok(cudaMalloc((void **)&scratch, ((size_t)n + (size_t)TB * npart + 1) * sizeof(double)))) break;
            double *y = scratch, *part = scratch + n;
            unsigned *ticket = reinterpret_cast<unsigned *>(scratch + n + (size_t)TB * npart);
            if (!cuda_ok(cudaMemset(ticket, 0, sizeof(double)))) break;
            const int nb = (n + TB - 1) / TB;
            for (int r = 0; r < nrhs; ++r) {
                double *g = rhs_dev + (size_t)r * n;
                for (int b = 0; b < nb; ++b) {
                    const int j0 = b * TB, m = n - j0 < TB ? n - j0 : TB, rest = n - j0 - m;
                    tri_fwd_kernel<<<rest > 0 ? (rest + TF - 1) / TF : 1, TF>>>(V_dev, ld, n, j0, g, y);
                }
                for (int b = nb - 1; b >= 0; --b) {
                    const int j0 = b * TB, m = n - j0 < TB ? n - j0 : TB;
                    const int rest = n - j0 - m, chunks = rest > 0 ? (rest + TC - 1) / TC : 1;
                    tri_bwd_kernel<<<dim3(m, chunks), TT>>>(V_dev, ld, n, j0, y, g, part, npart, ticket);
                }
            }
            lx::state_count_launches(2 * nb * nrhs);
            if (!cuda_ok(cudaGetLastError())) break;
        }
        cuda_ok(cudaDeviceSynchronize());
    } while (false);
    cudaFree(dwork);
    cudaFree(dinfo);
    cudaFree(scratch);
    free(hwork);
    return rc;
}
