// lx_lane.cuh — register-resident class kernel ("lane kernel") for classes whose bra components fit one warp.
//
// Ownership.  A LANE owns one bra Cartesian component a (any shell e = 0..La+Lb, cumulative index g) of one
// shell-set and keeps, for that a, the whole ket pyramid [a0|c]^(m), |c| = 0..Lx, in REGISTERS.  The ket recurrence
// (full Obara–Saika relation, reading G4)
//     [a0|c+1_i]^(m) = (ρ/ζc) PC_i [a0|c]^(m+1) + a_i/(2(γ+ζc)) [a−1_i 0|c]^(m+1)
//                      + c_i/(2ζc) ( [a0|c−1_i]^(m) − (ρ/ζc) [a0|c−1_i]^(m+1) )
// touches another bra component only through its second term, so the only cross-lane traffic is ONE warp shuffle
// per pyramid node (from the lane that owns a−1_i; the axis i is a compile-time property of the ket component).
// Everything else of VRR2 — ket component, order m, the m-range each ket component really needs (KetNeed), the
// register each node lives in — is resolved at compile time; after unrolling, the per-primitive VRR2 code is a
// straight line of DFMA + SHFL with no shared-memory access.  NG = off(La+Lb+1) lanes form a set; a warp carries
// SPW = 32/NG sets (32, 8, 3, 1 for La+Lb = 0..3).
//   a2  Boys → [00|0]^(m)              eq. 4: lanes over m; one lane per set if NG = 1
//   a3  VRR1 [e0|0]^(m)                eq. 3 in the warp's shared-memory slice, lanes over the
//                                      components of shell e, m in registers; then every lane loads its own column
//   a4  VRR2                           registers + shuffles (above)
//   a5  contraction                    (e0|c) accumulated in registers over the primitive loop
//   a7  HRR (eq. 1)      all 32 lanes over the (c, a) items of one set at a time, b unrolled
//   a8–a10                             coalesced store from shared memory, or γ / J digestion
// The paper's design keeps all of this in shared memory; on sm_100a shared-memory
// bandwidth (128 B/clk/SM = 16 doubles) against 64 DFMA/clk/SM is what bounds that design, hence
// registers + shuffles here.
#pragma once
#include "lx_group.cuh"

namespace lx {

// Register index of pyramid node (k, c, m): off[k][c] + (m − lo[k][c]).
struct KetPyr {
    int off[LX_MAX_L_AUX + 1][nc(LX_MAX_L_AUX)];
    int total;
};
constexpr KetPyr ket_pyr(const KetNeed &t, int LX) {
    KetPyr p{};
    int n = 0;
    for (int k = 0; k <= LX; ++k)
        for (int c = 0; c < nc(k); ++c) {
            p.off[k][c] = n;
            if (t.hi[k][c] >= t.lo[k][c]) n += t.hi[k][c] - t.lo[k][c] + 1;
        }
    p.total = n;
    return p;
}

// Per-set header in shared memory (written by the lane that owns component 0 of the set).
struct LaneHdr {
    double A[3], C[3];
    long long po;          // first primitive pair of the shell pair in the pair-data array
    int xo0, Kab, K, pad;  // first aux primitive; K_a K_b; K_a K_b K_x (0 = no set in this slot)
};

// The ket pyramid of one bra component for one primitive (a4), all in registers.  P holds level 0 on entry
// (orders NEED.lo[0][0] .. NEED.hi[0][0] of [a0|0]^(m)); the top level |c| = LX is accumulated into ACC (a5).
// How the a − 1_i term is fetched:
//   XL_NONE   the set has a single bra component (no such term)
//   XL_SHFL   from lane src[i] by shuffle
//   XL_FETCH  by shuffle, except lanes with from_pub set: they read what an earlier helper pass published,
//             pub[node * NPUB + pubidx[i]]  (pubidx[i] = index of a − 1_i among the published components)
//   XL_PUB    helper pass: shuffle, and lanes with from_pub set publish (slot pubidx[0]) every value a child node
//             asks its a − 1_i neighbour for; the top level is only published, not evaluated
enum { XL_NONE = 0, XL_SHFL = 1, XL_FETCH = 2, XL_PUB = 3 };
template <int LX, int XL, int NPUB>
__device__ __forceinline__ void ket_pyramid(double *P, double *ACC, const double (&WQ)[3], const double (&fa)[3],
                                            double o2z, double mrz, const int (&src)[3], bool on, bool from_pub,
                                            const int (&pubidx)[3], double *pub) {
    constexpr KetNeed NEED = ket_need(LX);
    constexpr KetPyr PYR = ket_pyr(NEED, LX);
    constexpr int N0 = NEED.hi[0][0] - NEED.lo[0][0] + 1;
    static_for<1, LX + 1>([&](auto ik) {
        constexpr int k = decltype(ik)::value;
        static_for<0, nc(k)>([&](auto icc) {
            constexpr int cc = decltype(icc)::value;
            constexpr uint32_t ck = cart_entry(off(k) + cc);
            constexpr int dir = ck >> 24;
            constexpr int ci = (ck >> (8 * dir)) & 0xff;
            constexpr int cy = (ck >> 8) & 0xff, cz = (ck >> 16) & 0xff, sc = cy + cz;
            constexpr int c1 = dir == 0 ? cc : (dir == 1 ? cc - sc : cc - sc - 1);
            constexpr int c2 = dir == 0 ? cc : (dir == 1 ? cc - 2 * sc + 1 : cc - 2 * sc - 1);
            constexpr int mlo = NEED.lo[k][cc], mhi = NEED.hi[k][cc];
            static_for<0, (mhi >= mlo ? mhi - mlo + 1 : 0)>([&](auto im) {
                constexpr int m = mlo + decltype(im)::value;
                constexpr int i1 = PYR.off[k - 1][c1] + (m + 1 - NEED.lo[k - 1][c1]);
                constexpr int node = PYR.off[k][cc] + (m - mlo) - N0;      // number of this node among levels 1..LX
                const double s1 = P[i1];
                if constexpr (XL == XL_PUB) {
                    if (from_pub) pub[node * NPUB + pubidx[0]] = s1;
                    if constexpr (k == LX) return;
                }
                double v = WQ[dir] * s1;
                if constexpr (XL == XL_SHFL || XL == XL_PUB) {
                    v = fma(fa[dir], __shfl_sync(0xffffffffu, s1, src[dir]), v);
                } else if constexpr (XL == XL_FETCH) {
                    double nb = __shfl_sync(0xffffffffu, s1, src[dir]);
                    if (from_pub) nb = pub[node * NPUB + pubidx[dir]];
                    v = fma(fa[dir], nb, v);
                }
                if constexpr (ci > 1) {
                    constexpr int i2 = PYR.off[k - 2][c2] + (m - NEED.lo[k - 2][c2]);
                    v = fma((double)(ci - 1) * o2z, fma(mrz, P[i2 + 1], P[i2]), v);
                }
                if constexpr (k < LX) P[PYR.off[k][cc] + (m - mlo)] = v;
                else if (on) ACC[cc] += v;
            });
        });
    });
    if constexpr (LX == 0) {
        if (on) ACC[0] += P[0];
    }
}

// Lane layout of a class.  ES = 0: all NG bra components of a set are lanes of one warp.  ES > 0 ("split"): the
// components of the shells e >= ES are the MAIN lanes of a set (NGM of them, SPW = 32/NGM sets per warp); the NHC
// components of the shells e < ES are evaluated first by a HELPER pass of the same warp, lanes = (primitive slice,
// set, helper component), which publishes the pyramid values of shell ES−1 to shared memory for the main lanes of
// shell ES.  ES = 2 turns the 35 components of La+Lb = 4 into 31 main lanes (measured: (4|22) 8.3 -> 3.5 ms, (3|22)
// 4.5 -> 2.2 ms against the shared-memory group kernel).  For La+Lb = 3 the split (2 x 16 main lanes) measured 12-15 %
// slower than 20 lanes of one set per warp, so it is used from La+Lb = 4 on only.
__host__ __device__ constexpr int lane_es(int E) { return E >= 4 ? 2 : 0; }
// does the class (La >= Lb) run on the lane kernel?  (otherwise: the shared-memory group kernel)
__host__ __device__ constexpr bool lane_fits(int LA, int LB) {
    return off(LA + LB + 1) - off(lane_es(LA + LB)) <= 32 && LA >= lane_es(LA + LB);
}

template <int LX, int LA, int LB>
struct LaneCls {
    using C = GrpCls<LX, LA, LB>;
    static constexpr int L = C::L, E = C::E, NG = C::NG;
    static constexpr int ES = lane_es(E);
    static constexpr int NHC = off(ES);                     // helper components (shells e < ES)
    static constexpr int NGM = NG - NHC;                    // main components
    static constexpr bool fits = lane_fits(LA, LB);
    static constexpr int SPW = fits ? 32 / NGM : 1;         // shell-sets per warp
    static constexpr int NSL = ES > 0 ? 32 / (SPW * NHC) : 1;   // primitive slices of the helper pass
    static constexpr int NPUB = ES > 0 ? nc(ES - 1) : 1;    // published components (shell ES−1)
    static constexpr KetNeed NEED = ket_need(LX);
    static constexpr KetPyr PYR = ket_pyr(NEED, LX);
    static constexpr int M0 = NEED.lo[0][0];                // lowest order of [a0|0]^(m) the ket pyramid reads
    static constexpr int N0 = NEED.hi[0][0] - NEED.lo[0][0] + 1;
    static constexpr int NCH = PYR.total - N0;              // pyramid nodes of the levels 1..LX
    static constexpr int NM0 = L + 1 - M0;                  // orders kept per bra component in the VRR1 region
    static constexpr int NPRM = 17;                         // per-primitive record (odd stride: no bank conflicts)
    static constexpr int V1S = NG > 1 ? ((NM0 * NG) | 1) : 0;   // VRR1 region [m − M0][g] of one primitive, odd stride
    static constexpr int PUBS = ES > 0 ? ((NCH * NPUB) | 1) : 0;   // published values of one primitive
    static constexpr int PPS = NPRM + V1S + PUBS;           // doubles staged per primitive
    static constexpr int HDR = (int)(sizeof(LaneHdr) / 8);
    static constexpr int NFIN = C::NACC + 2 * C::NH;        // (e0|c) + the two HRR buffers
    // primitives staged per chunk: as many as fit the warp's share of shared memory (1700 doubles = 13.6 KB for 16
    // resident warps per SM; 2266 = 18 KB for 12 warps where the published values need the room), at most 16
    static constexpr int BUDGET = ES > 0 ? 2266 : 1700;
    static constexpr int KB = NG > 1 ? cmax(1, cmin(16, (cmax(BUDGET, SPW * (HDR + NFIN)) / SPW - HDR) / PPS)) : 0;
    static constexpr int SLOT = HDR + cmax(KB * PPS, NFIN); // doubles of shared memory per set
};

// Prefactor record of one primitive triple (phase A → phases B, C, D).
enum { PR_PA = 0, PR_WP = 3, PR_WQ = 6, PR_O2G = 9, PR_MRG = 10, PR_O2GZ = 11, PR_O2Z = 12, PR_MRZ = 13, PR_PREF = 14, PR_T = 15 };

template <int LX, int LA, int LB, int MODE, int NWARPS, int MINB>
__global__ void __launch_bounds__(NWARPS * 32, MINB)
lane_kernel(SetMap map, DevShells aux, DevShells prim, PairData pdat, const double *__restrict__ boys_tab,
            double *__restrict__ out, int swapped, DfArgs df) {
    using C = GrpCls<LX, LA, LB>;
    using LC = LaneCls<LX, LA, LB>;
    constexpr int L = C::L, E = C::E, NG = C::NG, SPW = LC::SPW, SLOT = LC::SLOT;
    constexpr int ES = LC::ES, NHC = LC::NHC, NGM = LC::NGM, NSL = LC::NSL, NPUB = LC::NPUB;
    constexpr int NXC = nc(LX), NA = nc(LA), NB = nc(LB);
    constexpr KetPyr PYR = LC::PYR;
    constexpr int M0 = LC::M0, NM0 = LC::NM0, N0 = LC::N0;
    constexpr int NPRM = LC::NPRM, V1S = LC::V1S, PUBS = LC::PUBS, KB = LC::KB, HDR = LC::HDR;
    constexpr int O_V1 = HDR + KB * NPRM, O_PUB = O_V1 + KB * V1S;   // slot layout: header | records | VRR1 | published
    constexpr unsigned FULL = 0xffffffffu;

    extern __shared__ double smem[];
    GrpTables *tabs = reinterpret_cast<GrpTables *>(smem + (size_t)NWARPS * SPW * SLOT);
    const int tid = threadIdx.x;
    const int warp = tid >> 5, lane = tid & 31;
    // main lane → (set slot of the warp, bra component); lanes beyond SPW*NGM shadow slot 0 and never write
    const bool active = lane < SPW * NGM;
    const int slot = active ? lane / NGM : 0;
    const int g = NHC + (active ? lane - slot * NGM : 0);
    double *wbase = smem + (size_t)warp * SPW * SLOT;
    double *myslot = wbase + (size_t)slot * SLOT;

    build_tables(tabs, tid, NWARPS * 32);
    for (int n = lane; n < SPW * SLOT; n += 32) wbase[n] = 0.0;
    __syncthreads();
    const uint32_t *cart = tabs->cart, *dn = tabs->dn, *up = tabs->up;

    // per-lane constants of the owned (main) bra component
    const uint32_t ce_own = cart[g], dn_own = dn[g];
    const int a_own[3] = {(int)(ce_own & 0xff), (int)((ce_own >> 8) & 0xff), (int)((ce_own >> 16) & 0xff)};
    const int e_own = a_own[0] + a_own[1] + a_own[2];
    const bool fetch_pub = ES > 0 && e_own == ES;             // a − 1_i lives in the helper pass
    int src[3], pubidx[3];                                    // lane / published slot that owns a − 1_i
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        const int gd = (int)((dn_own >> (8 * d)) & 0xff);     // cumulative index of a − 1_d (g itself where a_d = 0)
        src[d] = (active && !fetch_pub) ? slot * NGM + gd - NHC : lane;
        pubidx[d] = (fetch_pub && gd != g) ? gd - off(ES > 0 ? ES - 1 : 0) : 0;
    }
    const double fa0[3] = {(double)a_own[0], (double)a_own[1], (double)a_own[2]};
    // helper lane → (primitive slice, set slot, helper component)
    const int h_sl = ES > 0 ? lane / (SPW * NHC) : 0;
    const int h_slot = ES > 0 ? (lane % (SPW * NHC)) / NHC : 0;
    const int h_g = ES > 0 ? lane % NHC : 0;
    const bool h_active = ES > 0 && lane < NSL * SPW * NHC;
    const uint32_t h_ce = cart[h_g], h_dn = dn[h_g];
    const bool h_pub = ES > 0 && h_active && h_g >= off(ES > 0 ? ES - 1 : 0);
    int h_src[3], h_pubidx[3];
    double h_fa0[3];
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        h_src[d] = h_active ? lane - h_g + (int)((h_dn >> (8 * d)) & 0xff) : lane;
        h_pubidx[d] = h_pub ? h_g - off(ES > 0 ? ES - 1 : 0) : 0;
        h_fa0[d] = (double)((h_ce >> (8 * d)) & 0xff);
    }

    const long long wstride = (long long)gridDim.x * NWARPS * SPW;
    for (long long sbase = ((long long)blockIdx.x * NWARPS + warp) * SPW; sbase < map.nsets; sbase += wstride) {
        // ---- set this lane works on ----------------------------------------------------------------------------
        const long long sid = sbase + slot;
        const bool live = sid < map.nsets;
        int p = 0, x = 0, a = 0, b = 0, Kab = 1, K = 0;
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
            Kab = min(prim.K[a] * prim.K[b], pdat.kstride);
            K = Kab * aux.K[x];
        }
        const int kmax = __reduce_max_sync(FULL, K);
        const double Ax = live ? prim.center[3 * a + 0] : 0.0, Ay = live ? prim.center[3 * a + 1] : 0.0,
                     Az = live ? prim.center[3 * a + 2] : 0.0;
        const double Cx = live ? aux.center[3 * x + 0] : 0.0, Cy = live ? aux.center[3 * x + 1] : 0.0,
                     Cz = live ? aux.center[3 * x + 2] : 0.0;
        double AB[3] = {0.0, 0.0, 0.0};
        if (live) {
            AB[0] = Ax - prim.center[3 * b + 0];
            AB[1] = Ay - prim.center[3 * b + 1];
            AB[2] = Az - prim.center[3 * b + 2];
        }
        const long long po = live ? (pdat.pd_off ? pdat.pd_off[p] : (long long)p * pdat.kstride) : 0;
        const int xo0 = live ? aux.prim_off[x] : 0;

        double ACC[NXC];
#pragma unroll
        for (int c = 0; c < NXC; ++c) ACC[c] = 0.0;

        if constexpr (NG == 1) {
            // ---- E = 0: a lane is a whole set; everything of a primitive stays in this lane's registers -------------
            int kx = 0, ij = 0;
            double zc = 1.0, cxc = 0.0, o2z = 0.5;
            for (int kt = 0; kt < kmax; ++kt) {
                const bool on = kt < K;
                double WQ[3] = {0, 0, 0}, mrz = 0, T = 0, pref = 0;
                if (on) {
                    if (ij == 0) {
                        zc = aux.zeta[xo0 + kx];
                        cxc = aux.coef[xo0 + kx];
                        o2z = 0.5 / zc;
                    }
                    const double *q = pdat.pd + (po + ij) * PD_STRIDE;
                    const double gm = q[0], PCx = q[1] - Cx, PCy = q[2] - Cy, PCz = q[3] - Cz, Kij = q[4], o2g = q[5];
                    const double s = rsqrt(gm + zc);              // (γ+ζc)^{-1/2}
                    const double igz = s * s;
                    const double rz = gm * igz;                   //  ρ/ζc
                    WQ[0] = rz * PCx; WQ[1] = rz * PCy; WQ[2] = rz * PCz;
                    mrz = -rz;
                    T = gm * zc * igz * (PCx * PCx + PCy * PCy + PCz * PCz);
                    // eq. 4: 2π^{5/2}/(γ ζc sqrt(γ+ζc)) K_ij c_k = 8π^{5/2} (1/2γ)(1/2ζc)(γ+ζc)^{-1/2} K_ij c_k
                    pref = 139.94734662099889988 * Kij * cxc * o2g * o2z * s;
                    if (++ij == Kab) { ij = 0; ++kx; }
                }
                double P[PYR.total];
                double F[L + 1];
                boys_all<L>(boys_tab, T, F);
#pragma unroll
                for (int i = 0; i < N0; ++i) P[PYR.off[0][0] + i] = pref * F[M0 + i];
                const double fa[3] = {0.0, 0.0, 0.0};
                ket_pyramid<LX, XL_NONE, 1>(P, ACC, WQ, fa, o2z, mrz, src, on, false, pubidx, nullptr);
            }
        } else {
            LaneHdr *hdr = reinterpret_cast<LaneHdr *>(myslot);
            if (active && g == NHC) {
                hdr->A[0] = Ax; hdr->A[1] = Ay; hdr->A[2] = Az;
                hdr->C[0] = Cx; hdr->C[1] = Cy; hdr->C[2] = Cz;
                hdr->po = po; hdr->xo0 = xo0; hdr->Kab = Kab; hdr->K = K;
            }
            __syncwarp();
            for (int k0 = 0; k0 < kmax; k0 += KB) {
                const int KBc = min(KB, kmax - k0);           // warp-uniform
                // ---- phase A: prefactors, lanes over (primitive, set) ----------------------------------------------
                for (int it = lane; it < KBc * SPW; it += 32) {
                    const int s = it % SPW, kk = it / SPW, kt = k0 + kk;
                    const LaneHdr *h = reinterpret_cast<const LaneHdr *>(wbase + (size_t)s * SLOT);
                    if (kt < h->K) {
                        const int hKab = h->Kab;
                        const int kx = kt / hKab, ij = kt - kx * hKab;
                        const double zc = aux.zeta[h->xo0 + kx], cxc = aux.coef[h->xo0 + kx];
                        const double *q = pdat.pd + (h->po + ij) * PD_STRIDE;
                        const double gm = q[0], Px = q[1], Py = q[2], Pz = q[3], Kij = q[4], o2g = q[5];
                        const double PCx = Px - h->C[0], PCy = Py - h->C[1], PCz = Pz - h->C[2];
                        const double o2z = 0.5 / zc;
                        const double sq = rsqrt(gm + zc);         // (γ+ζc)^{-1/2}
                        const double igz = sq * sq;
                        const double rg = -zc * igz;              // −ρ/γ
                        const double rz = gm * igz;               //  ρ/ζc
                        double *pr = wbase + (size_t)s * SLOT + HDR + kk * NPRM;
                        pr[PR_PA + 0] = Px - h->A[0]; pr[PR_PA + 1] = Py - h->A[1]; pr[PR_PA + 2] = Pz - h->A[2];
                        pr[PR_WP + 0] = rg * PCx; pr[PR_WP + 1] = rg * PCy; pr[PR_WP + 2] = rg * PCz;
                        pr[PR_WQ + 0] = rz * PCx; pr[PR_WQ + 1] = rz * PCy; pr[PR_WQ + 2] = rz * PCz;
                        pr[PR_O2G] = o2g; pr[PR_MRG] = rg; pr[PR_O2GZ] = 0.5 * igz; pr[PR_O2Z] = o2z; pr[PR_MRZ] = -rz;
                        // eq. 4: 2π^{5/2}/(γ ζc sqrt(γ+ζc)) K_ij c_k = 8π^{5/2} (1/2γ)(1/2ζc)(γ+ζc)^{-1/2} K_ij c_k
                        pr[PR_PREF] = 139.94734662099889988 * Kij * cxc * o2g * o2z * sq;
                        pr[PR_T] = gm * zc * igz * (PCx * PCx + PCy * PCy + PCz * PCz);
                    }
                }
                __syncwarp();
                // ---- phase B (a2): Boys → [00|0]^(m), lanes over (primitive, set, m) ------------------------
                for (int it = lane; it < KBc * SPW * NM0; it += 32) {
                    const int mi = it % NM0, t = it / NM0, s = t % SPW, kk = t / SPW;
                    double *sl = wbase + (size_t)s * SLOT;
                    if (k0 + kk < reinterpret_cast<const LaneHdr *>(sl)->K) {
                        const double *pr = sl + HDR + kk * NPRM;
                        sl[O_V1 + kk * V1S + mi * NG] = pr[PR_PREF] * boys_one(boys_tab, M0 + mi, pr[PR_T]);
                    }
                }
                __syncwarp();
                // ---- phase C (a3): VRR1 (eq. 3), lanes over (primitive, set, component of shell e), m in registers -------------
                static_for<1, E + 1>([&](auto ie) {
                    constexpr int e = decltype(ie)::value;
                    constexpr int ne = nc(e), nm = L - e + 1 - M0;       // orders M0 .. L-e
                    for (int it = lane; it < KBc * SPW * ne; it += 32) {
                        const int ci = it % ne, t = it / ne, s = t % SPW, kk = t / SPW;
                        double *sl = wbase + (size_t)s * SLOT;
                        if (k0 + kk < reinterpret_cast<const LaneHdr *>(sl)->K) {
                            const double *pr = sl + HDR + kk * NPRM;
                            double *Wk = sl + O_V1 + kk * V1S;
                            const int g0 = off(e) + ci;
                            const uint32_t ce = cart[g0];
                            const int dir = ce >> 24;
                            const int ai = (ce >> (8 * dir)) & 0xff;
                            const int g1 = (dn[g0] >> (8 * dir)) & 0xff;
                            const double pa = pr[PR_PA + dir], wp = pr[PR_WP + dir];
                            double v1[nm + 1];
#pragma unroll
                            for (int m = 0; m <= nm; ++m) v1[m] = Wk[m * NG + g1];
                            if (ai > 1) {
                                const int g2 = (dn[g1] >> (8 * dir)) & 0xff;
                                const double c2 = (double)(ai - 1) * pr[PR_O2G], mrg = pr[PR_MRG];
                                double v2[nm + 1];
#pragma unroll
                                for (int m = 0; m <= nm; ++m) v2[m] = Wk[m * NG + g2];
#pragma unroll
                                for (int m = 0; m < nm; ++m) v1[m] = fma(c2, fma(mrg, v2[m + 1], v2[m]), fma(wp, v1[m + 1], pa * v1[m]));
                            } else {
#pragma unroll
                                for (int m = 0; m < nm; ++m) v1[m] = fma(wp, v1[m + 1], pa * v1[m]);
                            }
#pragma unroll
                            for (int m = 0; m < nm; ++m) Wk[m * NG + g0] = v1[m];
                        }
                    }
                    __syncwarp();
                });
                // ---- phase D0 (a4): helper pass, shells e < ES; lanes over (primitive slice, set, component) -------------------
                if constexpr (ES > 0) {
                    double *hsl = wbase + (size_t)h_slot * SLOT;
                    const int hK = reinterpret_cast<const LaneHdr *>(hsl)->K;
                    for (int kb = 0; kb < KBc; kb += NSL) {   // warp-uniform trip count
                        const int kk = min(kb + h_sl, KB - 1);
                        const bool hon = h_active && kb + h_sl < KBc && k0 + kb + h_sl < hK;
                        const double *pr = hsl + HDR + kk * NPRM;
                        const double *Wk = hsl + O_V1 + kk * V1S;
                        double P[PYR.total];
#pragma unroll
                        for (int i = 0; i < N0; ++i) P[PYR.off[0][0] + i] = Wk[i * NG + h_g];
                        const double WQ[3] = {pr[PR_WQ], pr[PR_WQ + 1], pr[PR_WQ + 2]};
                        const double o2gz = pr[PR_O2GZ], o2z = pr[PR_O2Z], mrz = pr[PR_MRZ];
                        const double fa[3] = {h_fa0[0] * o2gz, h_fa0[1] * o2gz, h_fa0[2] * o2gz};
                        ket_pyramid<LX, XL_PUB, NPUB>(P, ACC, WQ, fa, o2z, mrz, h_src, false, h_pub && hon, h_pubidx,
                                                      hsl + O_PUB + kk * PUBS);
                    }
                    __syncwarp();
                }
                // ---- phase D (a4/a5): VRR2 in registers, one primitive after the other; no synchronisation inside ----------
                for (int kk = 0; kk < KBc; ++kk) {
                    const bool on = k0 + kk < K;
                    const double *pr = myslot + HDR + kk * NPRM;
                    const double *Wk = myslot + O_V1 + kk * V1S;
                    double P[PYR.total];
#pragma unroll
                    for (int i = 0; i < N0; ++i) P[PYR.off[0][0] + i] = Wk[i * NG + g];
                    const double WQ[3] = {pr[PR_WQ], pr[PR_WQ + 1], pr[PR_WQ + 2]};
                    const double o2gz = pr[PR_O2GZ], o2z = pr[PR_O2Z], mrz = pr[PR_MRZ];
                    const double fa[3] = {fa0[0] * o2gz, fa0[1] * o2gz, fa0[2] * o2gz};
                    ket_pyramid<LX, (ES > 0 ? XL_FETCH : XL_SHFL), NPUB>(P, ACC, WQ, fa, o2z, mrz, src, on, fetch_pub, pubidx,
                                                                       myslot + O_PUB + kk * PUBS);
                }
                __syncwarp();
            }
        }

        // ---- contracted (e0|c) → shared memory [c][a], e = LA..E -------------------------------------------------
        if (active && e_own >= LA) {
#pragma unroll
            for (int c = 0; c < NXC; ++c) myslot[HDR + c * C::NA_ACC + g - off(LA)] = ACC[c];
        }
        __syncwarp();

        // ---- a7–a10 per set of the warp, all 32 lanes ---------------------------------------------------------------
        constexpr int NH = C::NH;
        for (int s = 0; s < SPW; ++s) {
            if (sbase + s >= map.nsets) break;                    // warp-uniform
            double *SA = wbase + (size_t)s * SLOT + HDR;          // this set's (e0|c)
            double *SW = SA + C::NACC;
            double ABs[3];
#pragma unroll
            for (int d = 0; d < 3; ++d) ABs[d] = __shfl_sync(FULL, AB[d], s * NGM);
            static_for<1, LB + 1>([&](auto ij_) {
                constexpr int j = decltype(ij_)::value;
                constexpr int nbj = nc(j), NAj = C::NAH(j), nb1 = nc(j - 1), NA1 = C::NAH(j - 1);
                constexpr int NIT = NXC * NAj;
                double *srcb = (j == 1) ? SA : SW + ((j - 1) & 1) * NH;
                double *dstb = SW + (j & 1) * NH;
                for (int r0 = lane; r0 < NIT; r0 += 32 * GRP_RC) {
                    int s0[GRP_RC], sd[GRP_RC][3], dst[GRP_RC];
#pragma unroll
                    for (int q = 0; q < GRP_RC; ++q) {
                        const int r = r0 + q * 32;
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
                        for (int q = 0; q < GRP_RC; ++q) v[q] = fma(ABs[dir], srcb[s0[q] + b1], srcb[sd[q][dir] + b1]);
#pragma unroll
                        for (int q = 0; q < GRP_RC; ++q)
                            if (dst[q] >= 0) dstb[dst[q] + bj] = v[q];
                    });
                }
                __syncwarp();
            });
            const double *FIN = (LB == 0) ? SA : SW + (LB & 1) * NH;   // finished shell-set, layout [c][a][b]
            const long long sid_s = sbase + s;

            if constexpr (MODE == 0) {
                double *o = out + sid_s * C::NINT;
                if (!swapped || LB == 0) {
                    for (int r = lane; r < C::NINT; r += 32) o[r] = FIN[r];
                } else {                                          // caller's order is [c][b][a]
                    for (int r = lane; r < C::NINT; r += 32) {
                        const int ia = r % NA, t = r / NA, ib = t % NB, c = t / NB;
                        o[r] = FIN[(c * NA + ia) * NB + ib];
                    }
                }
            } else {
                const int as = __shfl_sync(FULL, a, s * NGM), bs = __shfl_sync(FULL, b, s * NGM),
                          xs_ = __shfl_sync(FULL, x, s * NGM);
                if constexpr (MODE == 1) {
                    // γ[bf(X)+c] += f Σ_ab (c|ab) D[bf(a)+ia, bf(b)+ib]
                    const double *Dab = df.D + (size_t)prim.bf_off[as] * df.ld + prim.bf_off[bs];
                    const double f = (as != bs) ? 2.0 : 1.0;
                    for (int c = lane; c < NXC; c += 32) {
                        const double *F = FIN + c * NA * NB;
                        double acc = 0.0;
                        for (int ia = 0; ia < NA; ++ia)
#pragma unroll
                            for (int ib = 0; ib < NB; ++ib) acc = fma(F[ia * NB + ib], __ldg(Dab + (size_t)ia * df.ld + ib), acc);
                        atomicAdd(df.out + aux.bf_off[xs_] + c, f * acc);
                    }
                } else {
                    // J[bf(a)+ia, bf(b)+ib] += Σ_c (c|ab) d[bf(X)+c], mirrored
                    const double *dx = df.D + aux.bf_off[xs_];
                    const size_t ra0 = prim.bf_off[as], rb0 = prim.bf_off[bs];
                    for (int r = lane; r < NA * NB; r += 32) {
                        double acc = 0.0;
#pragma unroll
                        for (int c = 0; c < NXC; ++c) acc = fma(FIN[c * NA * NB + r], __ldg(dx + c), acc);
                        const int ia = r / NB, ib = r - ia * NB;
                        atomicAdd(df.out + (ra0 + ia) * df.ld + rb0 + ib, acc);
                        if (as != bs) atomicAdd(df.out + (rb0 + ib) * df.ld + ra0 + ia, acc);
                    }
                }
            }
        }
        __syncwarp();
    }
}

template <int LX, int LA, int LB, int MODE>
cudaError_t lane_launch(const SetMap &map, const DevShells &aux, const DevShells &prim, const PairData &pdat,
                        const double *boys_tab, double *out, int swapped, const DfArgs &df, int num_sms,
                        cudaStream_t stream) {
    using LC = LaneCls<LX, LA, LB>;
    constexpr int NWARPS = 4;
    constexpr size_t smem = (size_t)NWARPS * LC::SPW * LC::SLOT * 8 + sizeof(GrpTables) + 16;
    static_assert(smem <= 227 * 1024, "class does not fit in shared memory");
    // resident blocks per SM: shared memory and a 128-register budget per thread
    constexpr int by_smem = (int)((227 * 1024) / (smem + 1024));
    constexpr int BPS = cmax(1, cmin(cmin(by_smem, 16), 65536 / (NWARPS * 32 * 128)));
    auto kern = lane_kernel<LX, LA, LB, MODE, NWARPS, BPS>;
    static std::atomic<unsigned long long> configured{0};
    if (cudaError_t e = ensure_dyn_smem(kern, smem, configured); e != cudaSuccess) return e;
    if (map.nsets <= 0) return cudaSuccess;
    const long long per_block = (long long)NWARPS * LC::SPW;
    long long blocks = (map.nsets + per_block - 1) / per_block;
    const long long cap = (long long)num_sms * BPS;
    if (blocks > cap) blocks = cap;
    kern<<<(unsigned)blocks, NWARPS * 32, smem, stream>>>(map, aux, prim, pdat, boys_tab, out, swapped, df);
    return cudaGetLastError();
}

}  // namespace lx
