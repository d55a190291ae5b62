// lx_group.cuh — the class kernel template: one instantiation per (Lx|La Lb) class (La >= Lb) and digestion mode.
//
// A GROUP of G threads (G = 1..32 lanes of a warp, or 64..256 threads = whole warps joined by a named barrier) owns one
// shell-set from the first primitive to the store; a block holds NTHREADS/G groups and walks the batch with a
// grid-stride loop.  The recurrence intermediates of one primitive triple and the contracted (e0|c) live in the group's
// slice of shared memory; everything that does not depend on the lane is resolved at compile time:
//   a2  Boys → [00|0]^(m)                    eq. 4, one lane per m
//   a3  VRR1 [e0|0]^(m), e = 1..La+Lb        eq. 3: lanes over the components of shell e, the
//                                            m loop runs in registers (each loaded value feeds two orders)
//   a4  VRR2 [e0|c]^(m), |c| = 1..Lx         full Obara–Saika ket relation (reading G4): lanes over the (m, bra
//                                            component) items of a level — decoded once per level into registers —
//                                            and the ket components c unrolled at compile time, so the recursion axis,
//                                            the c−1 / c−2 addresses and the integer factors are immediates
//   a5  contraction: the last VRR2 level accumulates into (e0|c), La <= e <= La+Lb ("early contraction")
//   a7  HRR (eq. 1): lanes over (c, bra component) items, the b components unrolled at compile time
//   a8–a10  the finished shell-set is staged in shared memory and stored coalesced, or digested into γ / J
//            without ever reaching global memory.
// Index algebra (lx_common.cuh) and small per-block tables replace the paper's constant-memory index maps.
#pragma once
#include <type_traits>

#include "lx_common.cuh"

namespace lx {

template <int I, int N, class F>
__device__ __forceinline__ void static_for(F &&f) {
    if constexpr (I < N) {
        f(std::integral_constant<int, I>{});
        static_for<I + 1, N>(f);
    }
}

__host__ __device__ constexpr int pow2ceil(int x) {
    int p = 1;
    while (p < x) p <<= 1;
    return p;
}

// Which auxiliary orders m of [·|c]^(m) are actually reachable from the targets [·|c]^(0), |c| = LX, when the ket is
// lowered along the axis with the smallest positive power (the DAG of reading G4): inclusive range lo..hi per ket
// component, hi < lo = never needed.  Evaluated at compile time; the kernel skips everything outside.
struct KetNeed {
    int lo[LX_MAX_L_AUX + 1][nc(LX_MAX_L_AUX)];
    int hi[LX_MAX_L_AUX + 1][nc(LX_MAX_L_AUX)];
};
constexpr KetNeed ket_need(int LX) {
    KetNeed t{};
    for (int k = 0; k <= LX_MAX_L_AUX; ++k)
        for (int c = 0; c < nc(LX_MAX_L_AUX); ++c) { t.lo[k][c] = 99; t.hi[k][c] = -1; }
    for (int c = 0; c < nc(LX); ++c) { t.lo[LX][c] = 0; t.hi[LX][c] = 0; }
    for (int k = LX; k >= 1; --k)
        for (int cc = 0; cc < nc(k); ++cc) {
            if (t.hi[k][cc] < t.lo[k][cc]) continue;
            const uint32_t ck = cart_entry(off(k) + cc);
            const int dir = ck >> 24, ci = (ck >> (8 * dir)) & 0xff;
            const int sc = ((ck >> 8) & 0xff) + ((ck >> 16) & 0xff);
            const int c1 = dir == 0 ? cc : (dir == 1 ? cc - sc : cc - sc - 1);
            t.lo[k - 1][c1] = cmin(t.lo[k - 1][c1], t.lo[k][cc] + 1);
            t.hi[k - 1][c1] = cmax(t.hi[k - 1][c1], t.hi[k][cc] + 1);
            if (ci > 1) {
                const int c2 = dir == 0 ? cc : (dir == 1 ? cc - 2 * sc + 1 : cc - 2 * sc - 1);
                t.lo[k - 2][c2] = cmin(t.lo[k - 2][c2], t.lo[k][cc]);
                t.hi[k - 2][c2] = cmax(t.hi[k - 2][c2], t.hi[k][cc] + 1);
            }
        }
    return t;
}
constexpr int ket_need_nm_max(const KetNeed &t, int k) {
    int m = 0;
    for (int c = 0; c < nc(k); ++c) m = cmax(m, t.hi[k][c] - t.lo[k][c] + 1);
    return m;
}

template <int LX, int LA, int LB>
struct GrpCls {
    static_assert(LA >= LB, "canonical order");
    static constexpr int L = LX + LA + LB;
    static constexpr int E = LA + LB;
    static constexpr int NG = off(E + 1);                  // bra components of all shells e = 0..E
    static constexpr int NV1 = (L + 1) * NG;               // VRR1 work region [m][g]
    __host__ __device__ static constexpr int elo(int k) { return k <= 0 ? 0 : cmax(LA - (LX - k), 0); }
    __host__ __device__ static constexpr int base(int k) { return off(elo(k)); }
    __host__ __device__ static constexpr int NAk(int k) { return NG - base(k); }
    __host__ __device__ static constexpr int lvl(int k) { return (LX - k + 1) * nc(k) * NAk(k); }  // [m][c][a], |c| = k
    // rotating buffers for levels 1..LX-1: level k lives at boff(k); three consecutive levels never overlap
    static constexpr int NBUF1 = []() constexpr { int m = 0; for (int k = 1; k < LX; ++k) m = cmax(m, lvl(k)); return m; }();
    static constexpr int NBUFS = LX >= 2 ? cmin(3, LX - 1) : 0;
    __host__ __device__ static constexpr int boff(int k) { return NV1 + ((k - 1) % 3) * NBUF1; }   // k = 1..LX-1
    static constexpr int NA_ACC = NG - off(LA);            // bra components e = LA..E
    static constexpr int NACC = nc(LX) * NA_ACC;           // contracted VRR2 targets (e0|c), layout [c][a]
    __host__ __device__ static constexpr int NAH(int j) { return off(E - j + 1) - off(LA); }
    __host__ __device__ static constexpr int hrr(int j) { return nc(LX) * NAH(j) * nc(j); }        // [c][a][b], |b| = j
    static constexpr int NINT = nc(LX) * nc(LA) * nc(LB);
    static constexpr int NH = []() constexpr { int m = 0; for (int j = 1; j <= LB; ++j) m = cmax(m, hrr(j)); return m; }();
    static constexpr int NWORK = cmax(NV1 + NBUFS * NBUF1, 2 * NH);
    static constexpr int SLOT = NACC + NWORK;              // doubles per shell-set
    // group size: enough threads per SM (~512) given how many sets fit in ~200 KB of shared memory
    static constexpr int G_AUTO = cmin(256, pow2ceil(cmax(1, (512 * SLOT * 8 + 200 * 1024 - 1) / (200 * 1024))));
};

// Tuning hook: group size per class (0 = automatic); specialisations in lx_tune.h.
template <int LX, int LA, int LB>
struct GrpTune { static constexpr int G = 0; };

}  // namespace lx
#include "lx_tune.h"
namespace lx {

template <int G>
__device__ __forceinline__ void group_sync(int group_in_block) {
    if constexpr (G <= 32) {
        __syncwarp();
    } else {
        asm volatile("bar.sync %0, %1;" ::"r"(group_in_block + 1), "r"(G) : "memory");
    }
}

// per-block tables (shared memory): cart[g] = (x,y,z,dir); dn[g] = cumulative index of a−1_x | a−1_y<<8 | a−1_z<<16
// (g itself where the power is zero); up[g] = cumulative index of a+1_x, a+1_y, a+1_z relative to g.
struct GrpTables {
    uint32_t cart[CART_N];
    uint32_t dn[CART_N];
    uint32_t up[CART_N];
};

__device__ __forceinline__ void build_tables(GrpTables *t, int tid, int nthreads) {
    for (int g = tid; g < CART_N; g += nthreads) {
        const uint32_t ce = cart_entry(g);
        const int x = ce & 0xff, y = (ce >> 8) & 0xff, z = (ce >> 16) & 0xff;
        const int e = x + y + z, s = y + z, idx = g - off(e);
        const int dx = x > 0 ? off(e - 1) + idx : g;
        const int dy = y > 0 ? off(e - 1) + idx - s : g;
        const int dz = z > 0 ? off(e - 1) + idx - s - 1 : g;
        t->cart[g] = ce;
        t->dn[g] = (uint32_t)dx | ((uint32_t)dy << 8) | ((uint32_t)dz << 16);
        const int ux = off(e + 1) + idx - g, uy = off(e + 1) + idx + s + 1 - g, uz = off(e + 1) + idx + s + 2 - g;
        t->up[g] = (uint32_t)ux | ((uint32_t)uy << 8) | ((uint32_t)uz << 16);
    }
}

#ifdef LX_FORCE_RC
constexpr int GRP_RC = LX_FORCE_RC;
#else
constexpr int GRP_RC = 4;  // items a lane keeps decoded in registers at a time
#endif

template <int LX, int LA, int LB, int MODE, int G, int NTHREADS, int MINB>
__global__ void __launch_bounds__(NTHREADS, MINB)
group_kernel(SetMap map, DevShells aux, DevShells prim, PairData pdat, const double *__restrict__ boys_tab,
             double *__restrict__ out, int swapped, DfArgs df) {
    using C = GrpCls<LX, LA, LB>;
    constexpr int L = C::L, E = C::E, NG = C::NG, SLOT = C::SLOT;
    constexpr int GPB = NTHREADS / G;                       // groups (shell-sets) per block
    constexpr int NXC = nc(LX), NA = nc(LA), NB = nc(LB);
    constexpr KetNeed NEED = ket_need(LX);
    constexpr int M0 = NEED.lo[0][0];                       // lowest order of [a0|0]^(m) any VRR2 path reads

    extern __shared__ double smem[];
    GrpTables *tabs = reinterpret_cast<GrpTables *>(smem + (size_t)GPB * SLOT);
    const int tid = threadIdx.x;
    const int grp = tid / G, lane = tid % G;
    double *slot = smem + (size_t)grp * SLOT;
    double *ACC = slot;
    double *W = slot + C::NACC;

    build_tables(tabs, tid, NTHREADS);
    for (int n = lane; n < SLOT; n += G) slot[n] = 0.0;     // never feed uninitialised shared memory to an FMA
    __syncthreads();
    const uint32_t *cart = tabs->cart, *dn = tabs->dn, *up = tabs->up;

    for (long long sbase = (long long)blockIdx.x * GPB; sbase < map.nsets; sbase += (long long)gridDim.x * GPB) {
        // ---- set this group works on -----------------------------------------------------------------------------
        const long long sid = sbase + grp;
        const bool live = sid < map.nsets;
        int p = 0, x = 0, a = 0, b = 0, Kab = 1, K = 0;
        bool tr = MODE == 0 && swapped != 0;                // caller's order is [c][b][a]: transposed store
        if (live) {
            int xs;
            if (map.cum == nullptr) {
                p = (int)(sid / map.nx);
                xs = (int)(sid - (long long)p * map.nx);
            } else {
                int lo = 0, hi = map.npair;                 // largest p with cum[p] <= sid
                while (hi - lo > 1) {
                    const int mid = (lo + hi) >> 1;
                    if (map.cum[mid] <= sid) lo = mid; else hi = mid;
                }
                p = lo;
                xs = (int)(sid - map.cum[p]);
            }
            a = map.pair_list[2 * p + swapped];
            b = map.pair_list[2 * p + 1 - swapped];
            x = map.x_list[xs];
            Kab = min(prim.K[a] * prim.K[b], pdat.kstride);   // never read past the pair's record (lx_api.cu: checked there)
            K = Kab * aux.K[x];
            if constexpr (LA == LB && LB > 0) {              // the VRR runs on the shell with the larger exponents (lx_common.cuh)
                if (shell_min_zeta(prim, b) > shell_min_zeta(prim, a)) {
                    const int t = a; a = b; b = t;
                    tr = !tr;
                }
            }
        }
        int kmax = K;
        if constexpr (G < 32) kmax = __reduce_max_sync(0xffffffffu, K);   // groups of one warp step together
        const double Ax = live ? prim.center[3 * a + 0] : 0.0, Ay = live ? prim.center[3 * a + 1] : 0.0,
                     Az = live ? prim.center[3 * a + 2] : 0.0;
        const double Cx = live ? aux.center[3 * x + 0] : 0.0, Cy = live ? aux.center[3 * x + 1] : 0.0,
                     Cz = live ? aux.center[3 * x + 2] : 0.0;
        const long long po = live ? (pdat.pd_off ? pdat.pd_off[p] : (long long)p * pdat.kstride) : 0;

        // ---- primitive loop (contraction, a5) -----------------------------------------------------------------------
        for (int kt = 0; kt < kmax; ++kt) {
            const bool on = kt < K;
            double PA[3], WP[3], WQ[3], o2g = 0, mrg = 0, o2gz = 0, o2z = 0, mrz = 0;
            if (on) {
                const int kx = kt / Kab, ij = kt - kx * Kab;
                const double *q = pdat.pd + (po + ij) * PD_STRIDE;
                const double g = q[0], Px = q[1], Py = q[2], Pz = q[3], Kij = q[4];
                const int xo = aux.prim_off[x] + kx;
                const double zc = aux.zeta[xo], cx = aux.coef[xo];
                const double PCx = Px - Cx, PCy = Py - Cy, PCz = Pz - Cz;
                const double igz = 1.0 / (g + zc);
                const double rg = -zc * igz;                  // −ρ/γ
                const double rz = g * igz;                    //  ρ/ζc
                PA[0] = Px - Ax; PA[1] = Py - Ay; PA[2] = Pz - Az;
                WP[0] = rg * PCx; WP[1] = rg * PCy; WP[2] = rg * PCz;
                WQ[0] = rz * PCx; WQ[1] = rz * PCy; WQ[2] = rz * PCz;
                o2g = 0.5 / g; mrg = rg; o2gz = 0.5 * igz; o2z = 0.5 / zc; mrz = -rz;
                const double T = g * zc * igz * (PCx * PCx + PCy * PCy + PCz * PCz);
                // eq. 4 prefactor 2π^{5/2}/(γ ζc sqrt(γ+ζc)) · K_ij · c_k, times F_m(T): one lane per m
                const double pref = 34.98683665524972497 * Kij * cx * sqrt(igz) / (g * zc);
                for (int m = M0 + lane; m <= L; m += G) W[m * NG] = pref * boys_one(boys_tab, m, T);
            } else {
                PA[0] = PA[1] = PA[2] = WP[0] = WP[1] = WP[2] = WQ[0] = WQ[1] = WQ[2] = 0.0;
            }
            group_sync<G>(grp);

            // ---- a3: VRR1 (eq. 3), lanes over the components of shell e, m in registers -----------------------------
            static_for<1, E + 1>([&](auto ie) {
                constexpr int e = decltype(ie)::value;
                constexpr int ne = nc(e), nm = L - e + 1 - M0;       // orders M0 .. L-e
                if (on) {
                    for (int ci = lane; ci < ne; ci += G) {
                        const int g0 = off(e) + ci;
                        const uint32_t ce = cart[g0];
                        const int dir = ce >> 24;
                        const int ai = (ce >> (8 * dir)) & 0xff;
                        const int g1 = (dn[g0] >> (8 * dir)) & 0xff;
                        const double pa = dir == 0 ? PA[0] : (dir == 1 ? PA[1] : PA[2]);
                        const double wp = dir == 0 ? WP[0] : (dir == 1 ? WP[1] : WP[2]);
                        // all loads of this component first, then the arithmetic, then the stores (the compiler
                        // cannot move a shared-memory load above an earlier store on its own)
                        double v1[nm + 1];
#pragma unroll
                        for (int m = 0; m <= nm; ++m) v1[m] = W[(M0 + m) * NG + g1];
                        if (ai > 1) {
                            const int g2 = (dn[g1] >> (8 * dir)) & 0xff;
                            const double c2 = (double)(ai - 1) * o2g;
                            double v2[nm + 1];
#pragma unroll
                            for (int m = 0; m <= nm; ++m) v2[m] = W[(M0 + m) * NG + g2];
#pragma unroll
                            for (int m = 0; m < nm; ++m) v1[m] = fma(c2, fma(mrg, v2[m + 1], v2[m]), fma(wp, v1[m + 1], pa * v1[m]));
                        } else {
#pragma unroll
                            for (int m = 0; m < nm; ++m) v1[m] = fma(wp, v1[m + 1], pa * v1[m]);
                        }
#pragma unroll
                        for (int m = 0; m < nm; ++m) W[(M0 + m) * NG + g0] = v1[m];
                    }
                }
                group_sync<G>(grp);
            });

            // ---- a4/a5: VRR2 levels |c| = 1..LX; the last level is accumulated into (e0|c) -------------------------------
            if constexpr (LX == 0) {
                if (on) {
                    if (kt == 0) for (int r = lane; r < C::NACC; r += G) ACC[r] = W[off(LA) + r];
                    else for (int r = lane; r < C::NACC; r += G) ACC[r] += W[off(LA) + r];
                }
                group_sync<G>(grp);
            }
            static_for<1, LX + 1>([&](auto ik) {
                constexpr int k = decltype(ik)::value;
                constexpr int nk = nc(k), NAk = C::NAk(k), bk = C::base(k);
                constexpr int nm = ket_need_nm_max(NEED, k);        // most orders any ket component of this level needs
                constexpr int NIT = nm * NAk;
                // source levels k-1 (S1) and k-2 (S2); level 0 is the VRR1 region [m][g]
                constexpr int o1 = (k == 1) ? 0 : C::boff(k - 1), n1c = nc(k - 1);
                constexpr int NA1 = (k == 1) ? NG : C::NAk(k - 1), b1 = (k == 1) ? 0 : C::base(k - 1);
                constexpr int o2 = (k <= 2) ? 0 : C::boff(k - 2), n2c = (k >= 2) ? nc(k - 2) : 1;
                constexpr int NA2 = (k <= 2) ? NG : C::NAk(k - 2), b2 = (k <= 2) ? 0 : C::base(k - 2);
                constexpr int ot = (k < LX) ? C::boff(k) : 0;
                if (on) {
                    for (int r0 = lane; r0 < NIT; r0 += G * GRP_RC) {
                        // decode up to GRP_RC (m, a) items of this lane once; reused for every ket component
                        int s1[GRP_RC], s1d[GRP_RC][3], s2[GRP_RC], dst[GRP_RC], mq[GRP_RC];
                        double fa[GRP_RC][3];
#pragma unroll
                        for (int j = 0; j < GRP_RC; ++j) {
                            const int r = r0 + j * G;
                            const bool ok = r < NIT;
                            const int rr = ok ? r : 0;
                            const int m = rr / NAk, gl = rr - m * NAk;
                            const int ga = bk + gl;
                            const uint32_t ca = cart[ga], da = dn[ga];
                            const int rowS1 = (m + 1) * n1c * NA1 - b1;
                            s1[j] = rowS1 + ga;
#pragma unroll
                            for (int d = 0; d < 3; ++d) {
                                s1d[j][d] = rowS1 + (int)((da >> (8 * d)) & 0xff);
                                fa[j][d] = (double)((ca >> (8 * d)) & 0xff) * o2gz;
                            }
                            s2[j] = m * n2c * NA2 - b2 + ga;
                            dst[j] = ok ? ((k < LX) ? m * nk * NAk + gl : gl) : -1;
                            mq[j] = ok ? m : 99;
                        }
                        static_for<0, nk>([&](auto icc) {
                            constexpr int cc = decltype(icc)::value;
                            constexpr uint32_t ck = cart_entry(off(k) + cc);
                            constexpr int dir = ck >> 24;
                            constexpr int ci = (ck >> (8 * dir)) & 0xff;
                            constexpr int cy = (ck >> 8) & 0xff, cz = (ck >> 16) & 0xff, sc = cy + cz;
                            constexpr int c1 = dir == 0 ? cc : (dir == 1 ? cc - sc : cc - sc - 1);
                            constexpr int c2 = dir == 0 ? cc : (dir == 1 ? cc - 2 * sc + 1 : cc - 2 * sc - 1);
                            constexpr int mlo = NEED.lo[k][cc], nmc = NEED.hi[k][cc] - NEED.lo[k][cc] + 1;
                            if constexpr (nmc > 0) {
                                const double f3 = (double)(ci - 1) * o2z;
                                // item order m' is relative to the first order this ket component needs
                                const double *S1 = W + o1 + c1 * NA1 + mlo * n1c * NA1;
                                const double *S2 = W + o2 + c2 * NA2 + mlo * n2c * NA2;
                                double v[GRP_RC];
                                bool act[GRP_RC];
#pragma unroll
                                for (int j = 0; j < GRP_RC; ++j) {
                                    act[j] = mq[j] < nmc;
                                    if (act[j]) {
                                        v[j] = WQ[dir] * S1[s1[j]];
                                        v[j] = fma(fa[j][dir], S1[s1d[j][dir]], v[j]);
                                        if constexpr (ci > 1) v[j] = fma(f3, fma(mrz, S2[s2[j] + n2c * NA2], S2[s2[j]]), v[j]);
                                    }
                                }
                                if constexpr (k < LX) {
#pragma unroll
                                    for (int j = 0; j < GRP_RC; ++j)
                                        if (act[j]) W[ot + cc * NAk + mlo * nk * NAk + dst[j]] = v[j];
                                } else {
                                    if (kt != 0) {
#pragma unroll
                                        for (int j = 0; j < GRP_RC; ++j)
                                            if (act[j]) v[j] += ACC[cc * C::NA_ACC + dst[j]];
                                    }
#pragma unroll
                                    for (int j = 0; j < GRP_RC; ++j)
                                        if (act[j]) ACC[cc * C::NA_ACC + dst[j]] = v[j];
                                }
                            }
                        });
                    }
                }
                group_sync<G>(grp);
            });
        }

        // ---- a7: HRR (eq. 1): level j builds |b| = j from |b| = j−1; H_0 = (e0|c); buffers alias the VRR region ---------
        constexpr int NH = C::NH;
        static_for<1, LB + 1>([&](auto ij) {
            constexpr int j = decltype(ij)::value;
            constexpr int nbj = nc(j), NAj = C::NAH(j), nb1 = nc(j - 1), NA1 = C::NAH(j - 1);
            constexpr int NIT = NXC * NAj;
            double *src = (j == 1) ? ACC : W + ((j - 1) & 1) * NH;
            double *dstb = W + (j & 1) * NH;
            if (K > 0) {
                double AB[3];
                AB[0] = Ax - prim.center[3 * b + 0];
                AB[1] = Ay - prim.center[3 * b + 1];
                AB[2] = Az - prim.center[3 * b + 2];
                for (int r0 = lane; r0 < NIT; r0 += G * GRP_RC) {
                    int s0[GRP_RC], sd[GRP_RC][3], dst[GRP_RC];
#pragma unroll
                    for (int q = 0; q < GRP_RC; ++q) {
                        const int r = r0 + q * G;
                        const bool ok = r < NIT;
                        const int rr = ok ? r : 0;
                        const int c = rr / NAj, al = rr - c * NAj;
                        const uint32_t ua = up[off(LA) + al];
                        s0[q] = (c * NA1 + al) * nb1;
#pragma unroll
                        for (int d = 0; d < 3; ++d) sd[q][d] = (c * NA1 + al + (int)((ua >> (8 * d)) & 0xff)) * nb1;
                        dst[q] = ok ? (c * NAj + al) * nbj : -1;
                    }
                    static_for<0, nbj>([&](auto ibj) {
                        constexpr int bj = decltype(ibj)::value;
                        constexpr uint32_t cb = cart_entry(off(j) + bj);
                        constexpr int dir = cb >> 24;
                        constexpr int by = (cb >> 8) & 0xff, bz = (cb >> 16) & 0xff, sb = by + bz;
                        constexpr int b1 = dir == 0 ? bj : (dir == 1 ? bj - sb : bj - sb - 1);
                        double v[GRP_RC];
#pragma unroll
                        for (int q = 0; q < GRP_RC; ++q) v[q] = fma(AB[dir], src[s0[q] + b1], src[sd[q][dir] + b1]);
#pragma unroll
                        for (int q = 0; q < GRP_RC; ++q)
                            if (dst[q] >= 0) dstb[dst[q] + bj] = v[q];
                    });
                }
            }
            group_sync<G>(grp);
        });
        const double *FIN = (LB == 0) ? ACC : W + (LB & 1) * NH;   // finished shell-set, layout [c][a][b]

        // ---- a8 / a9 / a10 -----------------------------------------------------------------------------------------------
        if (K > 0) {
            if constexpr (MODE == 0) {
                double *o = out + sid * C::NINT;
                if (!tr || LB == 0) {
                    for (int r = lane; r < C::NINT; r += G) o[r] = FIN[r];
                } else {                                          // caller's order is [c][b][a]
                    for (int r = lane; r < C::NINT; r += G) {
                        const int ia = r % NA, t = r / NA, ib = t % NB, c = t / NB;
                        o[r] = FIN[(c * NA + ia) * NB + ib];
                    }
                }
            } else if constexpr (MODE == 1) {
                // γ[bf(X)+c] += f Σ_ab (c|ab) D[bf(a)+ia, bf(b)+ib]
                const double *Dab = df.D + (size_t)prim.bf_off[a] * df.ld + prim.bf_off[b];
                const double f = (a != b) ? 2.0 : 1.0;
                for (int c = lane; c < NXC; c += G) {
                    const double *F = FIN + c * NA * NB;
                    double acc = 0.0;
                    for (int ia = 0; ia < NA; ++ia)
#pragma unroll
                        for (int ib = 0; ib < NB; ++ib) acc = fma(F[ia * NB + ib], __ldg(Dab + (size_t)ia * df.ld + ib), acc);
                    atomicAdd(df.out + aux.bf_off[x] + c, f * acc);
                }
            } else {
                // J[bf(a)+ia, bf(b)+ib] += Σ_c (c|ab) d[bf(X)+c], mirrored
                const double *dx = df.D + aux.bf_off[x];
                const size_t ra0 = prim.bf_off[a], rb0 = prim.bf_off[b];
                for (int r = lane; r < NA * NB; r += G) {
                    double acc = 0.0;
#pragma unroll
                    for (int c = 0; c < NXC; ++c) acc = fma(FIN[c * NA * NB + r], __ldg(dx + c), acc);
                    const int ia = r / NB, ib = r - ia * NB;
                    atomicAdd(df.out + (ra0 + ia) * df.ld + rb0 + ib, acc);
                    if (a != b) atomicAdd(df.out + (rb0 + ib) * df.ld + ra0 + ia, acc);
                }
            }
        }
        group_sync<G>(grp);
    }
}

// Block shape: how many groups share a block, chosen at compile time to maximise resident warps per SM under the
// shared-memory limit (227 KB per SM / per block).
struct BlockShape { int nthreads, gpb, blocks_per_sm; size_t smem; };
constexpr BlockShape pick_shape(int G, size_t slot_bytes) {
    const size_t limit = 227 * 1024, tab = sizeof(GrpTables) + 16;
    BlockShape best{0, 0, 0, 0};
    int best_warps = -1;
    for (int cand = 4; cand >= 1; --cand) {
        // G <= 32: cand = warps per block; G > 32: cand = groups per block
        const int nthreads = G <= 32 ? cand * 32 : cand * G;
        if (nthreads > 256 && cand > 1) continue;
        const int gpb = nthreads / G;
        const size_t smem = (size_t)gpb * slot_bytes + tab;
        if (smem > limit) continue;
        int bps = (int)(limit / (smem + 1024));
        if (bps > 2048 / nthreads) bps = 2048 / nthreads;
        if (bps > 32) bps = 32;
        if (bps < 1) bps = 1;
        const int warps = bps * nthreads / 32;
        if (warps > best_warps) { best_warps = warps; best = BlockShape{nthreads, gpb, bps, smem}; }
    }
    return best;
}

template <int LX, int LA, int LB, int MODE>
cudaError_t group_launch(const SetMap &map, const DevShells &aux, const DevShells &prim, const PairData &pdat,
                         const double *boys_tab, double *out, int swapped, const DfArgs &df, int num_sms,
                         cudaStream_t stream) {
    using C = GrpCls<LX, LA, LB>;
#ifdef LX_FORCE_G   // tuning builds only: one group size for every class that fits
    constexpr int G = (LX_FORCE_G <= 32 && (size_t)(32 / LX_FORCE_G) * C::SLOT * 8 > 220 * 1024) || (size_t)C::SLOT * 8 > 220 * 1024
                          ? C::G_AUTO : LX_FORCE_G;
#else
    constexpr int G = GrpTune<LX, LA, LB>::G > 0 ? GrpTune<LX, LA, LB>::G : C::G_AUTO;
#endif
    constexpr BlockShape shape = pick_shape(G, (size_t)C::SLOT * 8);
    static_assert(shape.nthreads > 0, "class does not fit in shared memory");
    constexpr int NT = shape.nthreads;
    // register cap: as many blocks per SM as shared memory allows, but never fewer than 96 registers per thread
    constexpr int MINB = cmax(1, cmin(shape.blocks_per_sm, 65536 / (NT * 96)));
    auto kern = group_kernel<LX, LA, LB, MODE, G, NT, MINB>;
    static std::atomic<unsigned long long> configured{0};
    if (cudaError_t e = ensure_dyn_smem(kern, shape.smem, configured); e != cudaSuccess) return e;
    if (map.nsets <= 0) return cudaSuccess;
    long long blocks = (map.nsets + shape.gpb - 1) / shape.gpb;
    const long long cap = (long long)num_sms * shape.blocks_per_sm;
    if (blocks > cap) blocks = cap;
    kern<<<(unsigned)blocks, NT, shape.smem, stream>>>(map, aux, prim, pdat, boys_tab, out, swapped, df);
    return cudaGetLastError();
}

}  // namespace lx
