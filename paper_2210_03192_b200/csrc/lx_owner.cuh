// lx_owner.cuh — "owner kernel": the chain form of lx_chain.cuh with ONE OWNER PER KET COMPONENT, for weakly contracted
// launches and for high aux angular momentum (which classes: owner_fits / owner_kmax below).
//
// The resummed ket recurrence (lx_chain.cuh header; eq. 2 of the paper, plus the c−1 terms of reading G4)
//
//     [a0|c]^(0) = Σ_{n <= c/2}  β(c,n) (2ζc)^{−|n|} (2(γ+ζc))^{−|c−2n|} ( Π_i B_i^{c_i − 2n_i} Y_{|n|} )[a]
//
// is evaluated here per ket component c: a warp (LANE = shell-set, 32 sets per batch) takes a component, runs the chains of
// ALL its partners n on the start vectors Y_p / a! in shared memory and sums them, weighted by the integers β, into one
// register accumulator — over the partners and over the primitives (a5, "early contraction").  Compared with
// the team / chain kernels (one chain per DISTINCT target (p, t), then a gather through shared memory) a level-p chain is run
// once per c that needs it (119 chains instead of 50 targets for Lx = 6), but nothing is staged: the finished (e0|c) of the 32
// sets is in the owner's registers, goes through the HRR (a7, eq. 1) right there and leaves through a private
// 32 × nc(La)nc(Lb) staging slot as a coalesced run (a8) or is digested (a9/a10).  Shared memory holds only the
// start vectors and the staging slots, so that Lx = 5, 6 fit where the (e0|c) region of the chain kernel (32 sets × nc(Lx) ×
// NACC doubles) does not, and the per-batch cost (no passes, no gather, no idle epilogue warps) is small enough for K ≈ 1.
// The kernel ("resident form") is owner2_kernel below.  A first form with dedicated producer warps, a double-buffered primitive
// loop and the start vectors of the next batch made ahead was slower on contracted launches ((5|22) K = 25: 22.5 against
// 19.6 ms) and, in the end, on K = 1 launches as well ((6|22): 1.75 against 1.54 ms); it was removed.
#pragma once
#include "lx_team.cuh"

namespace lx {

#ifndef LX_OWNER_MAXE
#define LX_OWNER_MAXE 5
#endif
// does the class (La >= Lb) have an owner kernel?  Lx = 5, 6: La+Lb = 2..4.  Lx = 2..4: the classes of the chain kernel (La+Lb =
// 3, 4 where the team kernel does not apply) and the two team classes where it measured faster, (3|21) and (4|11) — all of them
// for weakly contracted launches only (owner_kmax).
__host__ __device__ constexpr bool owner_over_team(int LX, int LA, int LB) {
    return (LX == 3 && LA == 2 && LB == 1) || (LX == 4 && LA == 1 && LB == 1);
}
__host__ __device__ constexpr bool owner_fits(int LX, int LA, int LB) {
    if (!(LX <= LX_MAX_L_AUX && LA + LB <= LX_OWNER_MAXE && LB <= 2 && LA >= LB)) return false;
    if (LA + LB == 5) return true;
    if (LX >= 5) return LA + LB >= 2;
    return (LX >= 2 && LA + LB >= 3) || owner_over_team(LX, LA, LB);
}
// largest contraction degree K_a K_b K_x (as known on the host, SetMap.khint) for which the owner kernel is chosen; measured on
// config 5 (K = 1..4: (3|31) 41 -> 17 ms, (4|31) 43 -> 20 ms, (3|22) 26 -> 14 ms, (2|31) 70 -> 36 ms against the chain kernel,
// (3|21) 99 -> 73 ms against the team kernel; the other team classes lose) and config 2 (K = 9:
// the chain / team kernels win for Lx <= 4, the owner kernel for Lx = 5, 6)
__host__ __device__ constexpr int owner_kmax(int LX, int LA, int LB) {
    return LX >= 5 || LA + LB >= 5 ? (LA + LB >= 3 ? (1 << 30) : 4) : 4;
}

template <int LX, int LA, int LB>
struct OwnCls {
    static constexpr int E = LA + LB, NG = off(E + 1), NACC = NG - off(LA);
    static constexpr int NXC = nc(LX), NA = nc(LA), NB = nc(LB), NAB = NA * NB, NINT = NXC * NAB;
    static constexpr int NLEV = LX / 2 + 1;                       // levels p = 0..Lx/2
    // warps per block from the register budget of a consumer (chain copy NG + accumulator NACC doubles, plus scalars)
    static constexpr int NW = E <= 2 ? 24 : (E == 3 ? 16 : (E == 4 ? 12 : 8));
    static constexpr int SP = NAB | 1;                            // staging stride of a set (odd: conflict-free both ways)
    static constexpr int UREC = NLEV * NG + 3 + NLEV;             // doubles per set of one start-vector buffer: u, r[3], ck[p]
};

// Batch header in shared memory (lane = set).
struct OwnHdr {
    double A[3][32], C[3][32], AB[3][32];
    long long po[32];
    int xo0[32], Kab[32], K[32], a[32], b[32], x[32], p[32];
    int tr[32];    // slab kernel: the set is stored transposed ([c][b][a]: mirrored class, or roles exchanged for La = Lb)
    int kmax;      // largest K of the batch (0: no live set)
    int ready;     // spare
    int next_c;    // next ket component of the batch to hand out (warps take components dynamically)
    int next_p;    // slab kernel: next producer work item
};

// Start vectors Y_p / a! (a3, eq. 3) of primitive q, level pw, for the 32 sets of the batch (one work item of a warp).
// Buffer layout [UREC][32]: u[p][g], r[3] = 2γ(P−C), ck[p] = (1/(2(γ+ζc)))^{Lx−2p} (1/(2ζc))^p.
template <int LX, int LA, int LB>
__device__ __forceinline__ void owner_produce(double *__restrict__ ub, const OwnHdr *hd, int q, int pw, int lane,
                                              const DevShells &aux, const PairData &pdat,
                                              const double *__restrict__ boys_tab) {
    using OC = OwnCls<LX, LA, LB>;
    constexpr int E = OC::E, NG = OC::NG, NLEV = OC::NLEV;
    const double A[3] = {hd->A[0][lane], hd->A[1][lane], hd->A[2][lane]};
    const double C[3] = {hd->C[0][lane], hd->C[1][lane], hd->C[2][lane]};
    const int Kab = hd->Kab[lane], K = hd->K[lane], xo0 = hd->xo0[lane];
    const bool on = q < K;
    const int qq = on ? q : 0;
    const int kx = qq / Kab, ij = qq - kx * Kab;
    const double zc = aux.zeta[xo0 + kx], cxc = on ? aux.coef[xo0 + kx] : 0.0;
    const PrimRec R = prim_rec(pdat.pd + (hd->po[lane] + ij) * PD_STRIDE, zc, cxc, A, C);
    static_for<0, NLEV>([&](auto ip) {
        constexpr int p = decltype(ip)::value;
        if (pw == p) {
            constexpr int MLO = LX - 2 * p, MHI = LX - p + E;
            double F[MHI - MLO + 1];
            boys_range<MLO, MHI>(boys_tab, R.T, F);
            double u[NG];
            vrr1_level<LX, E, p, MLO>(R, F, u);
            static_for<0, NG>([&](auto ig) { ub[(p * NG + decltype(ig)::value) * 32 + lane] = u[decltype(ig)::value]; });
            ub[(NLEV * NG + 3 + p) * 32 + lane] = level_scale<LX - 2 * p, p>(R);
            if constexpr (p == 0) {
#pragma unroll
                for (int d = 0; d < 3; ++d) ub[(NLEV * NG + d) * 32 + lane] = R.r[d];
            }
        }
    });
}


// One chain with RUN-TIME step counts (tx, ty, tz): the three step bodies are compile-time unrolled on the register
// copy z of the start vector, the loops around them are not.  Every ket component and every partner runs this one piece
// of code, so that the whole kernel stays resident in the instruction cache: with compile-time chains per component
// (≈ 400 KB of SASS for Lx = 6, each instruction executed once per batch of a K = 1 class) the warps stalled on
// instruction fetch most of the time (measured: "no instruction" 7.9 of 19 stall cycles per issue).
template <int LA, int E>
__device__ __forceinline__ void owner_chain(const double *__restrict__ zb, int lane, int tx, int ty, int tz, double rx,
                                            double ry, double rz, double ck, double (&acc)[off(E + 1) - off(LA)]) {
    constexpr int NG = off(E + 1), NACC = NG - off(LA);
    double z[NG];
    static_for<0, NG>([&](auto ig) { z[decltype(ig)::value] = zb[decltype(ig)::value * 32 + lane]; });
#pragma unroll 1
    for (int j = 0; j < tx; ++j) chain_step<0, 0, NG>(z, rx);
#pragma unroll 1
    for (int j = 0; j < ty; ++j) chain_step<1, 0, NG>(z, ry);
#pragma unroll 1
    for (int j = 0; j < tz; ++j) chain_step<2, 0, NG>(z, rz);
    static_for<0, NACC>([&](auto ii) { acc[decltype(ii)::value] = fma(ck, z[off(LA) + decltype(ii)::value], acc[decltype(ii)::value]); });
}

// All partners n <= c/2 of ket component c for one primitive, acc += Σ_n β(c,n) ck_|n| (Π_i B_i^{c_i−2n_i} u_|n|), with the
// partners that differ along the PRIMARY axis A summed in Horner form — the operators commute, so for fixed (n_B, n_C)
//     Σ_{n_A} w(n_A) B_A^{c_A − 2n_A} u_{p(n_A)} = B_A^{c_A − 2N} [ ... (B_A² (B_A² w(0) u_{p(0)} + w(1) u_{p(1)}) + w(2) u_{p(2)}) ... ],   N = ⌊c_A/2⌋,
// costs c_A steps along A instead of Σ (c_A − 2n_A), and the steps along the other two axes run once per (n_B, n_C) instead of
// once per partner ((6|22): 381 instead of 684 FP64 instructions for c = x⁶).  Each start vector is still read once per partner.
template <int LX, int LA, int LB, int A>
__device__ __forceinline__ void owner_partners_axis(int cA, int cB, int cC, const double *__restrict__ ub, int lane,
                                                    double (&acc)[OwnCls<LX, LA, LB>::NACC], double scale) {
    using OC = OwnCls<LX, LA, LB>;
    constexpr int NG = OC::NG, NACC = OC::NACC, NLEV = OC::NLEV;
    constexpr int B = (A + 1) % 3, C = (A + 2) % 3;
    const double rA = ub[(NLEV * NG + A) * 32 + lane], rB = ub[(NLEV * NG + B) * 32 + lane], rC = ub[(NLEV * NG + C) * 32 + lane];
    // β(c,n) = Π_i c_i!/(n_i!(c_i−2n_i)!2^{n_i}) grows along an axis by (c_i−2n_i)(c_i−2n_i−1)/(2(n_i+1)): kept as exact small
    // integers in double (no integer division in the loop)
    auto grow = [](int ci, int ni) { return (double)((ci - 2 * ni) * (ci - 2 * ni - 1)) * (ni == 0 ? 0.5 : (ni == 1 ? 0.25 : 1.0 / 6.0)); };
    const int NA_ = cA >> 1;
    double bB = scale;
#pragma unroll 1
    for (int nB = 0; 2 * nB <= cB; ++nB) {
        double bBC = bB;
#pragma unroll 1
        for (int nC = 0; 2 * nC <= cC; ++nC) {
            const int p0 = nB + nC;
            double z[NG];
            {
                const double w = ub[(NLEV * NG + 3 + p0) * 32 + lane];
                const double *u = ub + (size_t)p0 * NG * 32 + lane;
                static_for<0, NG>([&](auto ig) { z[decltype(ig)::value] = w * u[decltype(ig)::value * 32]; });
            }
            double bA = 1.0;
#pragma unroll 1
            for (int nA = 1; nA <= NA_; ++nA) {
                bA *= grow(cA, nA - 1);
                chain_step<A, 0, NG>(z, rA);
                chain_step<A, 0, NG>(z, rA);
                const double w = bA * ub[(NLEV * NG + 3 + p0 + nA) * 32 + lane];
                const double *u = ub + (size_t)(p0 + nA) * NG * 32 + lane;
                static_for<0, NG>([&](auto ig) { z[decltype(ig)::value] = fma(w, u[decltype(ig)::value * 32], z[decltype(ig)::value]); });
            }
            if (cA & 1) chain_step<A, 0, NG>(z, rA);
#pragma unroll 1
            for (int k = cB - 2 * nB; k > 0; --k) chain_step<B, 0, NG>(z, rB);
#pragma unroll 1
            for (int k = cC - 2 * nC; k > 0; --k) chain_step<C, 0, NG>(z, rC);
            static_for<0, NACC>([&](auto ii) { acc[decltype(ii)::value] = fma(bBC, z[off(LA) + decltype(ii)::value], acc[decltype(ii)::value]); });
            bBC *= grow(cC, nC);
        }
        bB *= grow(cB, nB);
    }
}

// ket component c (index within the shell, order G2).  HORNER: the primary axis is the one with the largest power.  Measured
// (B200): the Horner form wins for K = 1 batches ((6|22): 1.64 -> 1.55 ms) and loses 3-6 % inside a primitive loop ((5|22) K = 25:
// 19.6 -> 20.2 ms), where the plain form — one independent chain per partner — overlaps better; each path takes its own.
template <int LX, int LA, int LB, bool HORNER>
__device__ __forceinline__ void owner_partners(int c, const double *__restrict__ ub, int lane,
                                               double (&acc)[OwnCls<LX, LA, LB>::NACC], double scale = 1.0) {
    using OC = OwnCls<LX, LA, LB>;
    constexpr int E = OC::E, NG = OC::NG, NLEV = OC::NLEV;
    int s = 0;
    while ((s + 1) * (s + 2) / 2 <= c) ++s;                     // s = c_y + c_z
    const int cz = c - s * (s + 1) / 2, cy = s - cz, cx = LX - s;
    if constexpr (HORNER) {
        if (cx >= cy && cx >= cz) owner_partners_axis<LX, LA, LB, 0>(cx, cy, cz, ub, lane, acc, scale);
        else if (cy >= cz) owner_partners_axis<LX, LA, LB, 1>(cy, cz, cx, ub, lane, acc, scale);
        else owner_partners_axis<LX, LA, LB, 2>(cz, cx, cy, ub, lane, acc, scale);
    } else {
        const double rx = ub[(NLEV * NG + 0) * 32 + lane], ry = ub[(NLEV * NG + 1) * 32 + lane], rz = ub[(NLEV * NG + 2) * 32 + lane];
        auto grow = [](int ci, int ni) { return (double)((ci - 2 * ni) * (ci - 2 * ni - 1)) * (ni == 0 ? 0.5 : (ni == 1 ? 0.25 : 1.0 / 6.0)); };
        double bx = scale;
#pragma unroll 1
        for (int nx = 0; 2 * nx <= cx; ++nx) {
            double bxy = bx;
#pragma unroll 1
            for (int ny = 0; 2 * ny <= cy; ++ny) {
                double beta = bxy;
#pragma unroll 1
                for (int nz = 0; 2 * nz <= cz; ++nz) {
                    const int p = nx + ny + nz;
                    const double ck = beta * ub[(NLEV * NG + 3 + p) * 32 + lane];
                    owner_chain<LA, E>(ub + (size_t)p * NG * 32, lane, cx - 2 * nx, cy - 2 * ny, cz - 2 * nz, rx, ry, rz, ck, acc);
                    beta *= grow(cz, nz);
                }
                bxy *= grow(cy, ny);
            }
            bx *= grow(cx, nx);
        }
    }
}

// a7 + a8/a9/a10 of one finished ket component: HRR in registers (eq. 1), then the 32 sets leave through
// the warp's staging slot as one coalesced run per set (MODE 0) or are contracted with D into γ (MODE 1).  (The J digestion
// never comes here: it sums Σ_c d_c (e0|c) in the accumulator and transfers once per batch, owner2_kernel::j_reduce.)
template <int LX, int LA, int LB, int MODE>
__device__ __forceinline__ void owner_finish(int c, const double (&acc)[OwnCls<LX, LA, LB>::NACC], const OwnHdr *hd,
                                             double *__restrict__ stw, int lane, long long batch, const SetMap &map,
                                             const DevShells &aux, const DevShells &prim, double *__restrict__ out, bool tr,
                                             const DfArgs &df) {
    static_assert(MODE == 0 || MODE == 1, "store and gamma modes");
    using OC = OwnCls<LX, LA, LB>;
    constexpr int NACC = OC::NACC, NXC = OC::NXC, NA = OC::NA, NB = OC::NB, NAB = OC::NAB, SP = OC::SP;
    double H0[NACC];
    static_for<0, NACC>([&](auto ii) {
        constexpr int i = decltype(ii)::value;
        H0[i] = acc[i] * (double)cart_fact(off(LA) + i);        // back from the u = f / a! basis (lx_chain.cuh)
    });
    const double AB[3] = {hd->AB[0][lane], hd->AB[1][lane], hd->AB[2][lane]};
    if constexpr (MODE == 0) {
        hrr_store<LA, LB>(H0, AB, stw + (size_t)lane * SP, tr);
        __syncwarp();
        const int nlive = (int)min((long long)32, map.nsets - batch * 32);
        const int total = nlive * NAB;
        double *o = out + (batch * 32 * NXC + c) * NAB;
        for (int it = lane; it < total; it += 32) {
            const int s = it / NAB, i = it - s * NAB;
            o[(size_t)s * (NXC * NAB) + i] = stw[s * SP + i];
        }
        __syncwarp();
    } else {
        double fin[NAB];
        hrr_store<LA, LB>(H0, AB, fin, false);
        // γ[bf(X)+c] += f Σ_ab (c|ab) D[bf(a)+ia, bf(b)+ib]
        if (hd->p[lane] >= 0) {
            const int sa = hd->a[lane], sb = hd->b[lane];
            const double *Dab = df.D + (size_t)prim.bf_off[sa] * df.ld + prim.bf_off[sb];
            double sum = 0.0;
#pragma unroll
            for (int ia = 0; ia < NA; ++ia)
#pragma unroll
                for (int ib = 0; ib < NB; ++ib) sum = fma(fin[ia * NB + ib], __ldg(Dab + (size_t)ia * df.ld + ib), sum);
            atomicAdd(df.out + aux.bf_off[hd->x[lane]] + c, (sa != sb ? 2.0 : 1.0) * sum);
        }
    }
}

// ---- owner kernel, resident form ------------------------------------------------------------------------------------------
// For weakly contracted launches the start vectors of ALL primitives of a batch fit shared memory (NSLOT buffers), and
// usually those of several batches do.  A block then takes up to OWN2_MAXB batches per round: every warp helps to make the
// start vectors (work items (batch, primitive, level), handed out dynamically), and after one block barrier every warp owns
// ket components of "its" batch (warp mod number of batches) with the primitive loop INSIDE the partner sums — no pass
// structure, no barrier per primitive, no idle producer warps, and enough components per round for every warp even at
// Lx = 3, 4 (10 / 15 components per batch).  A batch with more primitives than buffers runs in chunks of NSLOT primitives.
constexpr int OWN2_MAXB = 4;
struct Own2Ctl { int nb, tot, next_p, pad; int slot0[OWN2_MAXB + 1]; };
template <int LX, int LA, int LB, int MODE>
struct Own2Cls {
    using OC = OwnCls<LX, LA, LB>;
    static constexpr int UB = OC::UREC * 32;                              // doubles per start-vector buffer
    static constexpr int SPG = OC::NACC | 1;                              // MODE 2: stride of a set's Σ_c d_c (e0|c)
    // per warp: staging slot (MODE 0); MODE 2: partial sums, then J rows — written after the round's chains are done, so the
    // slots ALIAS the start-vector buffers and cost no shared memory (more batches per round)
    static constexpr int STW = MODE == 1 ? 0 : 32 * OC::SP;
    static constexpr int fixed = (MODE == 0 ? OC::NW * STW * 8 : 0) + OWN2_MAXB * (int)sizeof(OwnHdr) + (int)sizeof(Own2Ctl) + 64;
    static constexpr int NSLOT = cmin(16, (222 * 1024 - fixed) / (UB * 8));
    static constexpr size_t smem = (size_t)fixed + (size_t)NSLOT * UB * 8;
    // A batch with more primitives than buffers runs in chunks; its warps work in lock-step there, so in the store mode the
    // staging slots (used only after the last chunk of a pass) lend their space to more buffers: fewer chunks, fewer barriers
    static constexpr int NSLOT_C = MODE == 0 ? cmin(16, (int)(((size_t)NSLOT * UB + (size_t)OC::NW * STW) / UB)) : NSLOT;
    static_assert(NSLOT >= 1, "owner kernel: no room for a start-vector buffer");
    static_assert(MODE != 2 || (size_t)NSLOT * UB >= (size_t)OC::NW * STW, "owner kernel: J slots do not fit the aliased buffers");
};

template <int LX, int LA, int LB, int MODE>
__global__ void __launch_bounds__(OwnCls<LX, LA, LB>::NW * 32, 1)
owner2_kernel(SetMap map, DevShells aux, DevShells prim, PairData pdat, const double *__restrict__ boys_tab,
              double *__restrict__ out, int swapped, DfArgs df) {
    using OC = OwnCls<LX, LA, LB>;
    using O2 = Own2Cls<LX, LA, LB, MODE>;
    constexpr int NACC = OC::NACC, NXC = OC::NXC, NB = OC::NB, NAB = OC::NAB, NLEV = OC::NLEV, NW = OC::NW, SP = OC::SP;
    constexpr int UB = O2::UB, NSLOT = O2::NSLOT, NSLOT_C = O2::NSLOT_C, STW = O2::STW;
    constexpr unsigned FULL = 0xffffffffu;

    extern __shared__ double smem[];
    double *U = smem;                                            // [NSLOT][UREC][32]
    double *ST = MODE == 2 ? U : U + (size_t)NSLOT * UB;         // [NW][STW] (MODE 2: aliases U)
    OwnHdr *hdr = reinterpret_cast<OwnHdr *>(U + (size_t)NSLOT * UB + (MODE == 0 ? (size_t)NW * STW : 0));
    Own2Ctl *ctl = reinterpret_cast<Own2Ctl *>(hdr + OWN2_MAXB);

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const long long nbatch = (map.nsets + 31) / 32, G = gridDim.x;
    const bool tr = MODE == 0 && swapped != 0;
    double *stw = ST + (size_t)warp * STW;

    auto decode = [&](long long bb, OwnHdr *h) {
        const SetId sid = decode_set(map, bb * 32 + lane, swapped);
        const int Kab = min(prim.K[sid.a] * prim.K[sid.b], pdat.kstride);
        const int K = sid.live ? Kab * aux.K[sid.x] : 0;
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            const double Ad = prim.center[3 * sid.a + d];
            h->A[d][lane] = Ad;
            h->C[d][lane] = aux.center[3 * sid.x + d];
            h->AB[d][lane] = Ad - prim.center[3 * sid.b + d];
        }
        h->po[lane] = pdat.pd_off ? pdat.pd_off[sid.p] : (long long)sid.p * pdat.kstride;
        h->xo0[lane] = aux.prim_off[sid.x];
        h->Kab[lane] = Kab;
        h->K[lane] = K;
        h->a[lane] = sid.a;
        h->b[lane] = sid.b;
        h->x[lane] = sid.x;
        h->p[lane] = sid.live ? sid.p : -1;
        const int km = __reduce_max_sync(FULL, K);
        if (lane == 0) { h->kmax = km; h->ready = 0; h->next_c = 0; h->next_p = 0; }
    };
    // a10 (MODE 2).  An owner folds d_c into the weights of its chains and keeps ONE accumulator over all the ket components it
    // takes: G = Σ_c d_c (e0|c) — the HRR is linear and does not depend on c, so it runs once per batch, not once per component
    // (the step before the HRR is where the paper's J-engine contracts as well).  The warps w = w0, w0 + dw, ..
    // worked on the batch of header h: the first of them sums their partial G and transfers it (eq. 1, lane = set) into its
    // slot; then its lanes take the elements (a, b) and walk the sets: one atomic per run of equal pairs and element (mirrored).
    auto j_reduce = [&](const OwnHdr *h, int w0, int dw) {
        constexpr int SPG = O2::SPG;
        if (warp != w0) return;                                  // one warp per batch: the tail of a round is short
        double H0[NACC];
#pragma unroll
        for (int i = 0; i < NACC; ++i) H0[i] = 0.0;
        for (int w = w0; w < NW; w += dw) {
            const double *g = ST + (size_t)w * STW + (size_t)lane * SPG;
            static_for<0, NACC>([&](auto ii) { H0[decltype(ii)::value] += g[decltype(ii)::value]; });
        }
        const double AB[3] = {h->AB[0][lane], h->AB[1][lane], h->AB[2][lane]};
        __syncwarp();
        hrr_store<LA, LB>(H0, AB, stw + (size_t)lane * SP, false);    // J contributions of the lane's set into the warp's own slot
        __syncwarp();
        // lanes over the elements (a, b); the sets of a batch are walked in order, runs of equal pairs are summed and flushed
        for (int r = lane; r < NAB; r += 32) {
            const int ia = r / NB, ib = r - ia * NB;
            int cur = -1, s0 = 0;
            double sum = 0.0;
            auto flush = [&]() {
                if (cur >= 0) {
                    const int sa = h->a[s0], sb = h->b[s0];
                    const size_t ra0 = prim.bf_off[sa], rb0 = prim.bf_off[sb];
                    atomicAdd(df.out + (ra0 + ia) * df.ld + rb0 + ib, sum);
                    if (sa != sb) atomicAdd(df.out + (rb0 + ib) * df.ld + ra0 + ia, sum);
                }
            };
#pragma unroll 1
            for (int ss = 0; ss < 32; ++ss) {
                const int ps = h->p[ss];
                if (ps < 0) continue;
                if (ps != cur) {
                    flush();
                    cur = ps;
                    s0 = ss;
                    sum = 0.0;
                }
                sum += stw[(size_t)ss * SP + r];
            }
            flush();
        }
    };
    // this warp's G (back from the u = f / a! basis) into its slot
    auto g_store = [&](const double (&acc)[NACC]) {
        constexpr int SPG = O2::SPG;
        static_for<0, NACC>([&](auto ii) {
            constexpr int i = decltype(ii)::value;
            stw[(size_t)lane * SPG + i] = acc[i] * (double)cart_fact(off(LA) + i);
        });
    };

    long long base = blockIdx.x;
    while (base < nbatch) {
        __syncthreads();                                         // the previous round is finished
        if (warp < OWN2_MAXB) decode(base + warp * G, hdr + warp);
        __syncthreads();
        if (tid == 0) {
            // plan of the round: as many of the next batches as have all their primitives resident
            int nb = 0, tot = 0;
            for (int i = 0; i < OWN2_MAXB; ++i) {
                const int k = hdr[i].kmax;
                if (k <= 0 || tot + k > NSLOT) break;
                ctl->slot0[i] = tot;
                tot += k;
                ++nb;
            }
            ctl->slot0[nb] = tot;
            ctl->nb = nb;
            ctl->tot = tot;
            ctl->next_p = 0;
        }
        __syncthreads();
        const int nb = ctl->nb;
        if (nb > 0) {
            // ---- start vectors: work items (slot = (batch, primitive), level) ---------------------------------------------------
            const int nitem = ctl->tot * NLEV;
            while (true) {
                int item = 0;
                if (lane == 0) item = atomicAdd(&ctl->next_p, 1);
                item = __shfl_sync(FULL, item, 0);
                if (item >= nitem) break;
                const int sq = item / NLEV, lev = item - sq * NLEV;
                int i = 0;
                while (i + 1 < nb && ctl->slot0[i + 1] <= sq) ++i;
                owner_produce<LX, LA, LB>(U + (size_t)sq * UB, hdr + i, sq - ctl->slot0[i], lev, lane, aux, pdat, boys_tab);
            }
            __syncthreads();
            // ---- ket components of this warp's batch ------------------------------------------------------------------------------
            const int ib_ = warp % nb;
            OwnHdr *hd = hdr + ib_;
            const int kq = hd->kmax;
            const double *ub0 = U + (size_t)ctl->slot0[ib_] * UB;
            const long long batch = base + ib_ * G;
            double acc[NACC];
#pragma unroll
            for (int i = 0; i < NACC; ++i) acc[i] = 0.0;
            const bool dlive = MODE == 2 && hd->p[lane] >= 0;
            const double *dvec = MODE == 2 ? df.D + aux.bf_off[hd->x[lane]] : nullptr;
            while (true) {
                int c = 0;
                if (lane == 0) c = atomicAdd(&hd->next_c, 1);
                c = __shfl_sync(FULL, c, 0);
                if (c >= NXC) break;
                double scale = 1.0;
                if constexpr (MODE == 2) scale = dlive ? __ldg(dvec + c) : 0.0;
                if (kq == 1) {
                    owner_partners<LX, LA, LB, true>(c, ub0, lane, acc, scale);
                } else {
#pragma unroll 1
                    for (int q = 0; q < kq; ++q) owner_partners<LX, LA, LB, false>(c, ub0 + (size_t)q * UB, lane, acc, scale);
                }
                if constexpr (MODE != 2) {
                    owner_finish<LX, LA, LB, MODE>(c, acc, hd, stw, lane, batch, map, aux, prim, out, tr, df);
#pragma unroll
                    for (int i = 0; i < NACC; ++i) acc[i] = 0.0;
                }
            }
            if constexpr (MODE == 2) {
                __syncthreads();                                 // every warp is done with the start vectors: their space takes the sums
                g_store(acc);
                __syncthreads();
                j_reduce(hd, ib_, nb);
            }
            base += (long long)nb * G;
        } else {
            // ---- one batch with more primitives than buffers: chunks of NSLOT primitives, one ket component per warp and pass ------
            OwnHdr *hd = hdr;
            const int kmax = hd->kmax;
            double acc[NACC];
#pragma unroll
            for (int i = 0; i < NACC; ++i) acc[i] = 0.0;
            const bool dlive = MODE == 2 && hd->p[lane] >= 0;
            const double *dvec = MODE == 2 ? df.D + aux.bf_off[hd->x[lane]] : nullptr;
#pragma unroll 1
            for (int c0 = 0; c0 < NXC; c0 += NW) {
                const int c = c0 + warp;
                double scale = 1.0;
                if constexpr (MODE == 2) scale = (dlive && c < NXC) ? __ldg(dvec + c) : 0.0;
#pragma unroll 1
                for (int q0 = 0; q0 < kmax; q0 += NSLOT_C) {
                    const int nq = min(NSLOT_C, kmax - q0);
                    __syncthreads();                             // the previous chunk is consumed (and the previous pass is stored)
#pragma unroll 1
                    for (int item = warp; item < nq * NLEV; item += NW) {
                        const int sq = item / NLEV, lev = item - sq * NLEV;
                        owner_produce<LX, LA, LB>(U + (size_t)sq * UB, hd, q0 + sq, lev, lane, aux, pdat, boys_tab);
                    }
                    __syncthreads();
                    if (c < NXC) {
#pragma unroll 1
                        for (int q = 0; q < nq; ++q) owner_partners<LX, LA, LB, false>(c, U + (size_t)q * UB, lane, acc, scale);
                    }
                }
                if constexpr (MODE == 0 && NSLOT_C > NSLOT) __syncthreads();   // the staging slots overlap the buffers of the last chunk
                if constexpr (MODE != 2) {
                    if (c < NXC) owner_finish<LX, LA, LB, MODE>(c, acc, hd, stw, lane, base, map, aux, prim, out, tr, df);
#pragma unroll
                    for (int i = 0; i < NACC; ++i) acc[i] = 0.0;
                }
            }
            if constexpr (MODE == 2) {
                __syncthreads();
                g_store(acc);
                __syncthreads();
                j_reduce(hd, 0, 1);
            }
            base += G;
        }
    }
}

template <int LX, int LA, int LB, int MODE>
cudaError_t owner_launch(const SetMap &map, const DevShells &aux, const DevShells &prim, const PairData &pdat,
                         const double *boys_tab, double *out, int swapped, const DfArgs &df, int num_sms,
                         cudaStream_t stream) {
    using OC = OwnCls<LX, LA, LB>;
    using O2 = Own2Cls<LX, LA, LB, MODE>;
    if (map.nsets <= 0) return cudaSuccess;
    long long blocks = (map.nsets + 31) / 32;
    if (blocks > (long long)num_sms) blocks = num_sms;
    static_assert(O2::smem <= 227 * 1024, "owner kernel: does not fit in shared memory");
    auto kern = owner2_kernel<LX, LA, LB, MODE>;
    static std::atomic<unsigned long long> configured{0};
    if (cudaError_t e = ensure_dyn_smem(kern, O2::smem, configured); e != cudaSuccess) return e;
    kern<<<(unsigned)blocks, OC::NW * 32, O2::smem, stream>>>(map, aux, prim, pdat, boys_tab, out, swapped, df);
    return cudaGetLastError();
}

// ---- kernel family of a class (La >= Lb), shared by the dispatcher (lx_inst.cu) and lx_kernel_family() ------------------
#ifndef LX_TEAM_WMAX
#define LX_TEAM_WMAX 2
#endif
#ifndef LX_TEAM_BUDGET
#define LX_TEAM_BUDGET 72
#endif
enum { FAM_TEAM = 0, FAM_OWNER = 1, FAM_CHAIN = 2, FAM_LANE = 3, FAM_GROUP = 4, FAM_SLAB = 5 };
// warps of the team kernel of a class, 0 = the class does not run on the team kernel.  Measured (B200): for Lx <= 4 the team
// kernel wins for La+Lb <= 2 and wherever one or two warps hold all targets ((3|21): three warps with 80 accumulator doubles
// per lane); for Lx = 5, 6 while at most three warps hold the targets.
__host__ __device__ constexpr int team_width(int LX, int LA, int LB) {
    if (LA + LB > 4) return 0;
    const bool wide = LX == 3 && LA == 2 && LB == 1;
    const int tw = team_size(LX, LA, LB, wide ? 80 : LX_TEAM_BUDGET);
    const bool ok = tw > 0 && (LX <= 4 ? (LA + LB <= 2 || tw <= (wide ? 3 : LX_TEAM_WMAX)) : (LA + LB >= 1 && tw <= 3));
    return ok ? tw : 0;
}
// khint: host-side bound of K_a K_b K_x of the launch, <= 0 = unknown (SetMap.khint)
__host__ __device__ constexpr int class_family(int LX, int LA, int LB, int khint) {
    if (owner_fits(LX, LA, LB) && (LX >= 5 || owner_over_team(LX, LA, LB) || team_width(LX, LA, LB) == 0) &&
        (owner_kmax(LX, LA, LB) == (1 << 30) || (khint > 0 && khint <= owner_kmax(LX, LA, LB))))
        return FAM_OWNER;
    if (team_width(LX, LA, LB) > 0) return FAM_TEAM;
    if (chain_fits(LX, LA, LB)) return FAM_CHAIN;
    if (lane_fits(LA, LB)) return FAM_LANE;
    return LX >= 3 && LA + LB >= 5 && LA + LB <= 6 ? FAM_SLAB : FAM_GROUP;   // slab kernel (lx_slab.cuh)
}

}  // namespace lx
