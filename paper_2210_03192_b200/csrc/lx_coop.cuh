// lx_coop.cuh — cooperative shared-memory kernel template, one instantiation per (Lx|La Lb) class (La >= Lb).
//
// A thread block evaluates NSLOT shell-sets at a time; every stage of the HGPA scheme (§2.5.1, lines
// 104–124) is a flat list of (slot, integral) work items strided over the block's threads, with the intermediates of
// one primitive triple in shared memory and the contracted (e0|c) accumulated there across the primitive loop
// ("early contraction").  Stages:
//   a2  Boys → [00|0]^(m)                      eq. 4, one thread per (set, m) as in PAPER.md:132
//   a3  VRR1  [e0|0]^(m), e = 1..La+Lb          eq. 3
//   a4  VRR2  [e0|c]^(m), |c| = 1..Lx           full Obara–Saika relation for a Cartesian ket (reading G4)
//   a5  contraction into (e0|c), La <= e <= La+Lb
//   a7  HRR   (X|a b) from (X|e 0)              eq. 1
//   a8–a10 store / γ digestion / J digestion
// Component index algebra replaces the paper's constant-memory index tables (lx_common.cuh).
#pragma once
#include "lx_common.cuh"

namespace lx {

template <int LX, int LA, int LB>
struct CoopCls {
    static_assert(LA >= LB, "canonical order");
    static constexpr int L = LX + LA + LB;
    static constexpr int E = LA + LB;
    static constexpr int NG = off(E + 1);                  // bra components of all shells e = 0..E
    static constexpr int NV1 = (L + 1) * NG;               // VRR1 work region [m][g]
    __host__ __device__ static constexpr int elo(int k) { return cmax(LA - (LX - k), 0); }
    __host__ __device__ static constexpr int base(int k) { return off(elo(k)); }
    __host__ __device__ static constexpr int NAk(int k) { return NG - base(k); }
    __host__ __device__ static constexpr int lvl(int k) { return (LX - k + 1) * nc(k) * NAk(k); }  // VRR2 level |c| = k
    __host__ __device__ static constexpr int nbuf_size() {
        int m = 0;
        for (int k = 1; k < LX; ++k) m = cmax(m, lvl(k));
        return m;
    }
    static constexpr int NBUF = nbuf_size();
    static constexpr int NBUFS = LX >= 2 ? cmin(3, LX - 1) : 0;
    static constexpr int NA_ACC = NG - off(LA);            // bra components e = LA..E
    static constexpr int NACC = nc(LX) * NA_ACC;           // contracted VRR2 targets (e0|c)
    __host__ __device__ static constexpr int NAH(int j) { return off(E - j + 1) - off(LA); }
    __host__ __device__ static constexpr int hrr(int j) { return nc(LX) * NAH(j) * nc(j); }
    static constexpr int NINT = nc(LX) * nc(LA) * nc(LB);
    __host__ __device__ static constexpr int nh_size(bool staged) {
        int m = 0;
        for (int j = 1; j < LB; ++j) m = cmax(m, hrr(j));
        if (staged && LB > 0) m = cmax(m, NINT);
        return m;
    }
    static constexpr int HDR = 20;
    __host__ __device__ static constexpr int slot_doubles(bool staged) {
        return HDR + NACC + cmax(NV1 + NBUFS * NBUF, 2 * nh_size(staged));
    }
    // slots per block: fill ~96 KB so that two blocks fit on an SM, never more than one set per thread
    __host__ __device__ static constexpr int nslot(bool staged, int nthreads) {
        const int bytes = slot_doubles(staged) * 8 + 24;
        int s = (96 * 1024) / bytes;
        if (s < 1) s = 1;
        if (s > nthreads) s = nthreads;
        return s;
    }
};

constexpr int COOP_THREADS = 256;

// header slots (doubles) -----------------------------------------------------------------------------------------
enum { H_PA = 0, H_WP = 3, H_WQ = 6, H_AB = 9, H_O2G = 12, H_MRG = 13, H_O2GZ = 14, H_O2Z = 15, H_MRZ = 16, H_T = 17, H_PREF = 18 };

template <int LX, int LA, int LB, int MODE>
__global__ void __launch_bounds__(COOP_THREADS)
coop_kernel(SetMap map, DevShells aux, DevShells prim, PairData pdat, const double *__restrict__ boys_tab,
            double *__restrict__ out, int swapped, DfArgs df) {
    using C = CoopCls<LX, LA, LB>;
    constexpr bool STAGED = (MODE != 0);
    constexpr int S = C::nslot(STAGED, COOP_THREADS);
    constexpr int SLOT = C::slot_doubles(STAGED);
    constexpr int NT = COOP_THREADS;
    constexpr int L = C::L, E = C::E, NG = C::NG;

    extern __shared__ double smem[];
    double *slots = smem;
    int *s_pair = reinterpret_cast<int *>(smem + (size_t)S * SLOT);  // pair slot (index into pair_list)
    int *s_x = s_pair + S;                                           // aux shell id
    int *s_K = s_x + S;                                              // primitive triples of the set (0 = inactive)
    int *s_Kab = s_K + S;
    int *s_kmax = s_Kab + S;
    uint32_t *cart = reinterpret_cast<uint32_t *>(s_kmax + 4);

    const int tid = threadIdx.x;
    for (int g = tid; g < CART_N; g += NT) cart[g] = cart_entry(g);

    for (long long sbase = (long long)blockIdx.x * S; sbase < map.nsets; sbase += (long long)gridDim.x * S) {
        if (tid == 0) *s_kmax = 0;
        __syncthreads();
        // ---- slot setup ---------------------------------------------------------------------------------------
        if (tid < S) {
            const long long sid = sbase + tid;
            int K = 0;
            if (sid < map.nsets) {
                int p, xs;
                if (map.cum == nullptr) {
                    p = (int)(sid / map.nx);
                    xs = (int)(sid - (long long)p * map.nx);
                } else {
                    int lo = 0, hi = map.npair;  // largest p with cum[p] <= sid
                    while (hi - lo > 1) {
                        const int mid = (lo + hi) >> 1;
                        if (map.cum[mid] <= sid) lo = mid; else hi = mid;
                    }
                    p = lo;
                    xs = (int)(sid - map.cum[p]);
                }
                const int a = map.pair_list[2 * p + swapped], b = map.pair_list[2 * p + 1 - swapped];
                const int x = map.x_list[xs];
                const int Kab = prim.K[a] * prim.K[b];
                K = Kab * aux.K[x];
                s_pair[tid] = p;
                s_x[tid] = x;
                s_Kab[tid] = Kab;
                double *h = slots + (size_t)tid * SLOT;
                h[H_AB + 0] = prim.center[3 * a + 0] - prim.center[3 * b + 0];
                h[H_AB + 1] = prim.center[3 * a + 1] - prim.center[3 * b + 1];
                h[H_AB + 2] = prim.center[3 * a + 2] - prim.center[3 * b + 2];
                atomicMax(s_kmax, K);
            }
            s_K[tid] = K;
        }
        for (int n = tid; n < S * C::NACC; n += NT) {
            const int s = n / C::NACC, r = n - s * C::NACC;
            slots[(size_t)s * SLOT + C::HDR + r] = 0.0;
        }
        __syncthreads();
        const int kmax = *s_kmax;

        // ---- primitive loop (contraction, a5) ---------------------------------------------------------------------
        for (int kt = 0; kt < kmax; ++kt) {
            if (tid < S && kt < s_K[tid]) {
                double *h = slots + (size_t)tid * SLOT;
                const int p = s_pair[tid], x = s_x[tid], Kab = s_Kab[tid];
                const int kx = kt / Kab, ij = kt - kx * Kab;
                const long long po = pdat.pd_off ? pdat.pd_off[p] : (long long)p * pdat.kstride;
                const double *q = pdat.pd + (po + ij) * 5;
                const double g = q[0], Px = q[1], Py = q[2], Pz = q[3], Kij = q[4];
                const int a = map.pair_list[2 * p + swapped];
                const int xo = aux.prim_off[x] + kx;
                const double zc = aux.zeta[xo], cx = aux.coef[xo];
                const double PCx = Px - aux.center[3 * x + 0], PCy = Py - aux.center[3 * x + 1], PCz = Pz - aux.center[3 * x + 2];
                const double igz = 1.0 / (g + zc);
                const double rho = g * zc * igz;
                h[H_PA + 0] = Px - prim.center[3 * a + 0];
                h[H_PA + 1] = Py - prim.center[3 * a + 1];
                h[H_PA + 2] = Pz - prim.center[3 * a + 2];
                const double rg = -zc * igz;                      // −ρ/γ
                const double rz = g * igz;                        //  ρ/ζc
                h[H_WP + 0] = rg * PCx; h[H_WP + 1] = rg * PCy; h[H_WP + 2] = rg * PCz;
                h[H_WQ + 0] = rz * PCx; h[H_WQ + 1] = rz * PCy; h[H_WQ + 2] = rz * PCz;
                h[H_O2G] = 0.5 / g;
                h[H_MRG] = rg;
                h[H_O2GZ] = 0.5 * igz;
                h[H_O2Z] = 0.5 / zc;
                h[H_MRZ] = -rz;
                h[H_T] = rho * (PCx * PCx + PCy * PCy + PCz * PCz);
                // 2π^{5/2} / (γ ζc sqrt(γ+ζc)) · K_ij · c_k      (eq. 4 prefactor with the contraction coefficients)
                h[H_PREF] = 34.98683665524972497 * Kij * cx * sqrt(igz) / (g * zc);
            }
            __syncthreads();
            // ---- a2: [00|0]^(m) = pref · F_m(T) ----------------------------------------------------------------------
            for (int n = tid; n < S * (L + 1); n += NT) {
                const int s = n / (L + 1), m = n - s * (L + 1);
                if (kt < s_K[s]) {
                    double *h = slots + (size_t)s * SLOT;
                    double *V1 = h + C::HDR + C::NACC;
                    V1[m * NG] = h[H_PREF] * boys_one(boys_tab, m, h[H_T]);
                }
            }
            __syncthreads();
            // ---- a3: VRR1 (eq. 3) ------------------------------------------------------------------------------------
#pragma unroll
            for (int e = 1; e <= E; ++e) {
                const int nm = L - e + 1, ne = nc(e), per = nm * ne;
                for (int n = tid; n < S * per; n += NT) {
                    const int s = n / per, r = n - s * per;
                    if (kt >= s_K[s]) continue;
                    const int m = r / ne, ci = r - m * ne;
                    const uint32_t ce = cart[off(e) + ci];
                    const int dir = ce >> 24;
                    const int ai = (ce >> (8 * dir)) & 0xff;
                    const int sy = ((ce >> 8) & 0xff) + ((ce >> 16) & 0xff);
                    double *h = slots + (size_t)s * SLOT;
                    double *V1 = h + C::HDR + C::NACC;
                    const int g1 = off(e - 1) + idx_down1(ci, sy, dir);
                    double v = h[H_PA + dir] * V1[m * NG + g1] + h[H_WP + dir] * V1[(m + 1) * NG + g1];
                    if (ai > 1) {
                        const int g2 = off(e - 2) + idx_down2(ci, sy, dir);
                        v += (double)(ai - 1) * h[H_O2G] * fma(h[H_MRG], V1[(m + 1) * NG + g2], V1[m * NG + g2]);
                    }
                    V1[m * NG + off(e) + ci] = v;
                }
                __syncthreads();
            }
            // ---- a4/a5: VRR2 levels |c| = 1..LX; the last level is accumulated into (e0|c) --------------------------------
            if constexpr (LX == 0) {
                for (int n = tid; n < S * C::NACC; n += NT) {
                    const int s = n / C::NACC, r = n - s * C::NACC;
                    if (kt >= s_K[s]) continue;
                    double *h = slots + (size_t)s * SLOT;
                    h[C::HDR + r] += h[C::HDR + C::NACC + off(LA) + r];
                }
            }
#pragma unroll
            for (int k = 1; k <= LX; ++k) {
                const int nk = nc(k), NAk = C::NAk(k), bk = C::base(k);
                const int nm = LX - k + 1, per = nm * nk * NAk;
                // source levels: k-1 (S1) and k-2 (S2); level 0 is the VRR1 region
                const int o1 = (k - 1 == 0) ? 0 : C::NV1 + ((k - 2) % 3) * C::NBUF;
                const int n1c = nc(k - 1), NA1 = (k == 1) ? NG : C::NAk(k - 1), b1 = (k == 1) ? 0 : C::base(k - 1);
                const int o2 = (k - 2 <= 0) ? 0 : C::NV1 + ((k - 3) % 3) * C::NBUF;
                const int n2c = k >= 2 ? nc(k - 2) : 1, NA2 = (k <= 2) ? NG : C::NAk(k - 2), b2 = (k <= 2) ? 0 : C::base(k - 2);
                const int ot = C::NV1 + ((k - 1) % 3) * C::NBUF;
                for (int n = tid; n < S * per; n += NT) {
                    const int s = n / per, r = n - s * per;
                    if (kt >= s_K[s]) continue;
                    const int gl = r % NAk, t = r / NAk;
                    const int cc = t % nk, m = t / nk;
                    double *h = slots + (size_t)s * SLOT;
                    double *W = h + C::HDR + C::NACC;
                    const uint32_t ck = cart[off(k) + cc];
                    const int dir = ck >> 24;
                    const int ci = (ck >> (8 * dir)) & 0xff;               // (c+1_i)_i
                    const int syc = ((ck >> 8) & 0xff) + ((ck >> 16) & 0xff);
                    const int c1 = idx_down1(cc, syc, dir);
                    const int ga = bk + gl;
                    const uint32_t ca = cart[ga];
                    const int ax = ca & 0xff, ay = (ca >> 8) & 0xff, az = (ca >> 16) & 0xff;
                    const int e = ax + ay + az;
                    const int ai = (ca >> (8 * dir)) & 0xff;
                    const double *S1 = W + o1 + ((m + 1) * n1c + c1) * NA1 - b1;
                    double v = h[H_WQ + dir] * S1[ga];
                    if (ai > 0) {
                        const int ga1 = off(e - 1) + idx_down1(ga - off(e), ay + az, dir);
                        v = fma((double)ai * h[H_O2GZ], S1[ga1], v);
                    }
                    if (ci > 1) {
                        const int c2 = idx_down2(cc, syc, dir);
                        const double *S2 = W + o2 + (m * n2c + c2) * NA2 - b2;
                        v = fma((double)(ci - 1) * h[H_O2Z], fma(h[H_MRZ], S2[n2c * NA2 + ga], S2[ga]), v);
                    }
                    if (k < LX) W[ot + (m * nk + cc) * NAk + gl] = v;
                    else h[C::HDR + cc * C::NA_ACC + gl] += v;
                }
                __syncthreads();
            }
            if constexpr (LX == 0) __syncthreads();
        }

        // ---- a7: HRR (eq. 1), level j builds |b| = j from |b| = j−1; H_0 = (e0|c) accumulators -------------------------
        // buffers alias the VRR work region (all primitives are done)
        constexpr int NH = C::nh_size(STAGED);
#pragma unroll
        for (int j = 1; j <= LB; ++j) {
            const int nbj = nc(j), NAj = C::NAH(j), per = nc(LX) * NAj * nbj;
            const int nb1 = nc(j - 1), NA1 = C::NAH(j - 1);
            const int osrc = (j == 1) ? C::HDR : C::HDR + C::NACC + ((j - 1) & 1) * NH;
            const int odst = C::HDR + C::NACC + (j & 1) * NH;
            const bool last = (j == LB);
            for (int n = tid; n < S * per; n += NT) {
                const int s = n / per, r = n - s * per;
                if (s_K[s] == 0) continue;
                double *h = slots + (size_t)s * SLOT;
                int bj, al, c;
                if (last && swapped) {           // enumerate in the caller's [c][b][a] order
                    al = r % NAj; const int t = r / NAj; bj = t % nbj; c = t / nbj;
                } else {
                    bj = r % nbj; const int t = r / nbj; al = t % NAj; c = t / NAj;
                }
                const uint32_t cb = cart[off(j) + bj];
                const int dir = cb >> 24;
                const int syb = ((cb >> 8) & 0xff) + ((cb >> 16) & 0xff);
                const int b1 = idx_down1(bj, syb, dir);
                const int ga = off(LA) + al;
                const uint32_t ca = cart[ga];
                const int ay = (ca >> 8) & 0xff, az = (ca >> 16) & 0xff;
                const int e = (ca & 0xff) + ay + az;
                const int alp = off(e + 1) + idx_up1(ga - off(e), ay + az, dir) - off(LA);
                const double *src = h + osrc + (size_t)c * NA1 * nb1;
                const double v = fma(h[H_AB + dir], src[al * nb1 + b1], src[alp * nb1 + b1]);
                if (!last) {
                    h[odst + (c * NAj + al) * nbj + bj] = v;
                } else if constexpr (!STAGED) {
                    out[(sbase + s) * C::NINT + r] = v;
                } else {
                    h[odst + (c * NAj + al) * nbj + bj] = v;   // staged in [c][a][b] order for the digestion
                }
            }
            __syncthreads();
        }
        if constexpr (LB == 0 && !STAGED) {
            for (int n = tid; n < S * C::NINT; n += NT) {
                const int s = n / C::NINT, r = n - s * C::NINT;
                if (s_K[s] == 0) continue;
                out[(sbase + s) * C::NINT + r] = slots[(size_t)s * SLOT + C::HDR + r];
            }
        }
        // ---- a9 / a10: digestion -------------------------------------------------------------------------
        if constexpr (STAGED) {
            constexpr int ofin = (LB == 0) ? C::HDR : C::HDR + C::NACC + (LB & 1) * NH;
            constexpr int NA = nc(LA), NB = nc(LB), NX = nc(LX);
            if constexpr (MODE == 1) {
                // γ[bf(X)+c] += f Σ_ab (c|ab) D[bf(a)+ia, bf(b)+ib]
                for (int n = tid; n < S * NX; n += NT) {
                    const int s = n / NX, c = n - s * NX;
                    if (s_K[s] == 0) continue;
                    const double *F = slots + (size_t)s * SLOT + ofin + c * NA * NB;
                    const int p = s_pair[s];
                    const int a = map.pair_list[2 * p], b = map.pair_list[2 * p + 1];
                    const double *Dab = df.D + (size_t)prim.bf_off[a] * df.ld + prim.bf_off[b];
                    double acc = 0.0;
                    for (int ia = 0; ia < NA; ++ia)
                        for (int ib = 0; ib < NB; ++ib) acc = fma(F[ia * NB + ib], __ldg(Dab + (size_t)ia * df.ld + ib), acc);
                    atomicAdd(df.out + aux.bf_off[s_x[s]] + c, (a != b) ? 2.0 * acc : acc);
                }
            } else {
                // J[bf(a)+ia, bf(b)+ib] += Σ_c (c|ab) d[bf(X)+c], mirrored
                for (int n = tid; n < S * NA * NB; n += NT) {
                    const int s = n / (NA * NB), r = n - s * (NA * NB);
                    if (s_K[s] == 0) continue;
                    const double *F = slots + (size_t)s * SLOT + ofin + r;
                    const double *dx = df.D + aux.bf_off[s_x[s]];
                    double acc = 0.0;
#pragma unroll
                    for (int c = 0; c < NX; ++c) acc = fma(F[c * NA * NB], __ldg(dx + c), acc);
                    const int p = s_pair[s];
                    const int a = map.pair_list[2 * p], b = map.pair_list[2 * p + 1];
                    const int ia = r / NB, ib = r - ia * NB;
                    const size_t ra = prim.bf_off[a] + ia, rb = prim.bf_off[b] + ib;
                    atomicAdd(df.out + ra * df.ld + rb, acc);
                    if (a != b) atomicAdd(df.out + rb * df.ld + ra, acc);
                }
            }
        }
        __syncthreads();
    }
}

template <int LX, int LA, int LB, int MODE>
cudaError_t coop_launch(const SetMap &map, const DevShells &aux, const DevShells &prim, const PairData &pdat,
                        const double *boys_tab, double *out, int swapped, const DfArgs &df, int num_sms,
                        cudaStream_t stream) {
    using C = CoopCls<LX, LA, LB>;
    constexpr bool STAGED = (MODE != 0);
    constexpr int S = C::nslot(STAGED, COOP_THREADS);
    constexpr size_t smem = (size_t)S * C::slot_doubles(STAGED) * 8 + (size_t)(4 * S + 4) * 4 + CART_N * 4;
    static_assert(smem <= 227 * 1024, "class does not fit in shared memory");
    static bool configured = false;
    auto kern = coop_kernel<LX, LA, LB, MODE>;
    if (!configured) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        configured = true;
    }
    if (map.nsets <= 0) return cudaSuccess;
    const int per_sm = cmax(1, cmin(8, (int)((227 * 1024) / (smem + 1024))));
    long long blocks = (map.nsets + S - 1) / S;
    const long long cap = (long long)num_sms * per_sm;
    if (blocks > cap) blocks = cap;
    kern<<<(unsigned)blocks, COOP_THREADS, smem, stream>>>(map, aux, prim, pdat, boys_tab, out, swapped, df);
    return cudaGetLastError();
}

}  // namespace lx
