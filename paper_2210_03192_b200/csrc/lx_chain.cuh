// lx_chain.cuh — warp-specialised, register-resident class kernel ("chain kernel") for La+Lb <= 4.
//
// The ket recurrence in chain form.  With B_i = (ρ/ζc) PC_i + S_i/(2(γ+ζc)), (S_i f)[a] = a_i f[a−1_i], the two-term
// relation of the paper (eq. 2) is [·0|t+1_i]^(m) = B_i [·0|t]^(m+1) on the vector over all bra
// components a.  The operators B_i commute and ∂B_i/∂C_i/(2ζc) = −ρ/(2ζc²), so the terms eq. 2 drops for a Cartesian
// ket (reading G4: the c−1 terms of the full Obara–Saika relation) resum exactly into
//
//     [a0|c]^(0) = Σ_{n <= c/2}  β(c,n) (2ζc)^{−|n|}  ( Π_i B_i^{c_i − 2n_i}  Y_{|n|} )[a]
//     Y_p^{(·)}  = Δ^p Z^{(Lx−2p)},  (ΔZ)^{(m)} = Z^{(m)} − (ρ/ζc) Z^{(m+1)},  Z^{(m)}[a] = [a0|0]^(m)  (VRR1, eq. 3)
//     β(c,n)     = Π_i c_i! / (n_i! (c_i−2n_i)! 2^{n_i})                    (an integer: ways to pair off 2n_i of c_i)
//
// (checked against the CPU oracle by tests/test_gpu_parity.py; the closed n-quantal form of the paper, eq. 8 with
// reading G5, is the expansion of Π B_i^{t_i}).  Δ commutes with VRR1, so Y_p is obtained by running eq. 3 on the
// s-type values Σ_s C(p,s)(−ρ/ζc)^s [00|0]^(Lx−2p+s): every level p costs one plain VRR1 pyramid of orders 0..La+Lb.
// In the basis u[a] = f[a]/(a_x! a_y! a_z!) the operator is B_i u = (1/(2(γ+ζc))) (r_i u[a] + u[a−1_i]), r_i = 2γ PC_i:
// ONE FP64 instruction per bra component and step, no integer factors, the scalar 1/(2(γ+ζc))^{|t|} deferred.
//
// Mapping (sm_100a: 64 FP64 lanes and 128 B/clk of shared memory per SM; the register file is the only place where
// a recurrence costs nothing but DFMAs).  A block works on 32 shell-sets at a time, LANE = shell-set, so that every
// index below is a compile-time constant and every shared-memory access is lane-contiguous:
//   producer warps   per primitive triple: prefactors, Boys (a2), VRR1 in registers (a3) → the start vectors u = Y_p/a!
//                    of the levels of this pass, written to a ring of shared-memory buffers
//   consumer warps   one per chain target (p, t): load u, apply the |t| steps in place in registers (a4) and
//                    accumulate c^{|t|}(2ζc)^{−p}·(...) over the primitives in registers (a5)
//   hand-off         named barriers full[b] / empty[b] (producer bar.arrive ↔ consumer bar.sync and back)
// Classes with more targets than resident warps run several passes over the primitive loop.  After the passes the
// targets are combined with the integers β into (e0|c) in shared memory [set][c][a], the HRR (a7, eq. 1) runs in
// registers per (set, c) in place, and the finished shell-sets are stored coalesced or digested (a8–a10).
#pragma once
#include "lx_lane.cuh"

namespace lx {

// ---- compile-time component algebra (order G2) -------------------------------------------------------------------
__host__ __device__ constexpr int cart_pow(int g, int axis) { return (int)((cart_entry(g) >> (8 * axis)) & 0xff); }
__host__ __device__ constexpr int cart_shell(int g) { return cart_pow(g, 0) + cart_pow(g, 1) + cart_pow(g, 2); }
// cumulative index of the component with powers (x, y, z)
__host__ __device__ constexpr int cart_index(int x, int y, int z) {
    const int e = x + y + z, s = y + z;
    return off(e) + s * (s + 1) / 2 + z;
}
__host__ __device__ constexpr int cart_dn(int g, int axis) {   // a − 1_axis (power must be positive)
    return cart_index(cart_pow(g, 0) - (axis == 0), cart_pow(g, 1) - (axis == 1), cart_pow(g, 2) - (axis == 2));
}
__host__ __device__ constexpr int cart_up(int g, int axis) {   // a + 1_axis
    return cart_index(cart_pow(g, 0) + (axis == 0), cart_pow(g, 1) + (axis == 1), cart_pow(g, 2) + (axis == 2));
}
__host__ __device__ constexpr int ifact(int n) { int r = 1; for (int i = 2; i <= n; ++i) r *= i; return r; }
__host__ __device__ constexpr int cart_fact(int g) { return ifact(cart_pow(g, 0)) * ifact(cart_pow(g, 1)) * ifact(cart_pow(g, 2)); }
__host__ __device__ constexpr int ibinom(int n, int k) { return ifact(n) / (ifact(k) * ifact(n - k)); }
__host__ __device__ constexpr int ipow2(int n) { return 1 << n; }
// β(c,n) along one axis
__host__ __device__ constexpr int beta1(int c, int n) { return ifact(c) / (ifact(n) * ifact(c - 2 * n) * ipow2(n)); }

// ---- chain targets of a class: level p = 0..LX/2 holds the components t of degree LX − 2p ------------------------------
constexpr int CHAIN_MAXT = 50;                 // LX = 6: 28 + 15 + 6 + 1
struct ChainTargets {
    int n;
    int p[CHAIN_MAXT];      // level
    int g[CHAIN_MAXT];      // cumulative Cartesian index of t
};
constexpr ChainTargets chain_targets(int LX) {
    ChainTargets t{};
    t.n = 0;
    for (int p = 0; 2 * p <= LX; ++p)
        for (int ci = 0; ci < nc(LX - 2 * p); ++ci) {
            t.p[t.n] = p;
            t.g[t.n] = off(LX - 2 * p) + ci;
            ++t.n;
        }
    return t;
}

// VRR1 nodes of one level: shells e = 0..E at orders 0..E−e
__host__ __device__ constexpr int chain_nv1(int E) { int n = 0; for (int e = 0; e <= E; ++e) n += nc(e) * (E - e + 1); return n; }

constexpr int CHAIN_MAXPASS = 8;
struct ChainPlan {
    int npass;
    int t0[CHAIN_MAXPASS], t1[CHAIN_MAXPASS];       // target range of a pass
    int plo[CHAIN_MAXPASS], phi[CHAIN_MAXPASS];     // levels the pass needs
    int nprod[CHAIN_MAXPASS];                       // producer warps of the pass
    int nw;                                         // warps per block
    int nbuf;                                       // ring buffers (max producers + 1)
    int nlev;                                       // most levels any pass needs
};
// Consumer warps per pass are capped by the register budget (a consumer keeps NG + NA_ACC doubles live); producers
// per pass balance one VRR1 pyramid per level against the chain of the pass's first (longest) target.
constexpr ChainPlan chain_plan(int LX, int LA, int LB) {
    const int E = LA + LB, NG = off(E + 1), NACC = NG - off(LA);
    const ChainTargets T = chain_targets(LX);
    const int cap = E <= 2 ? 16 : (E == 3 ? 11 : 8);
    const int nwmax = E <= 2 ? 24 : (E == 3 ? 16 : 12);
    ChainPlan P{};
    P.npass = (T.n + cap - 1) / cap;
    const int ncw = (T.n + P.npass - 1) / P.npass;
    P.nw = 0; P.nbuf = 0; P.nlev = 0;
    for (int i = 0; i < P.npass; ++i) {
        P.t0[i] = i * ncw;
        P.t1[i] = cmin(T.n, (i + 1) * ncw);
        P.plo[i] = T.p[P.t0[i]];
        P.phi[i] = T.p[P.t1[i] - 1];
        const int nlev = P.phi[i] - P.plo[i] + 1;
        const int k0 = LX - 2 * P.plo[i];                              // steps of the longest chain of the pass
        const int cons = cmax(1, k0) * NG + 2 * NACC + 8;
        const int prod = nlev * (3 * chain_nv1(E) + NG + 60) + 70;
        int np = (prod + cons - 1) / cons;
        np = cmax(1, cmin(np, cmin(E >= 4 ? 3 : 4, nwmax - (P.t1[i] - P.t0[i]))));
        P.nprod[i] = np;
        P.nw = cmax(P.nw, P.t1[i] - P.t0[i] + np);
        P.nbuf = cmax(P.nbuf, np + 1);
        P.nlev = cmax(P.nlev, nlev);
    }
    return P;
}

template <int LX, int LA, int LB>
struct ChainCls {
    using C = GrpCls<LX, LA, LB>;
    static constexpr int E = C::E, L = C::L, NG = C::NG, NACC = C::NA_ACC;
    static constexpr int NXC = nc(LX), NA = nc(LA), NB = nc(LB), NAB = NA * NB, NINT = C::NINT;
    static constexpr int SLOTN = NINT | 1;                    // doubles per set in the (e0|c) / shell-set region
    static constexpr ChainTargets T = chain_targets(LX);
    static constexpr ChainPlan P = chain_plan(LX, LA, LB);
    static constexpr int NW = P.nw;
    static constexpr int ZREC = (P.nlev * NG + 3 + P.nlev) * 32;    // doubles per ring buffer
    static constexpr int HDRD = 9 * 32 + 32 + 6 * 16;         // header: 9 doubles + 1 int64 + 6 ints per set, in doubles
    static constexpr size_t smem = ((size_t)32 * SLOTN + (size_t)P.nbuf * ZREC + HDRD + 4) * 8;
    static constexpr bool fits = E <= 4 && LX <= 4 && smem <= 227 * 1024 && NW <= 32 && 2 * P.nbuf + 1 <= 16;
};
__host__ __device__ constexpr bool chain_fits(int LX, int LA, int LB) {
    if (LA + LB > 4 || LX > 4) return false;
    const ChainPlan P = chain_plan(LX, LA, LB);
    const int NG = off(LA + LB + 1);
    const size_t smem = ((size_t)32 * ((nc(LX) * nc(LA) * nc(LB)) | 1) + (size_t)P.nbuf * (P.nlev * NG + 3 + P.nlev) * 32 +
                         9 * 32 + 32 + 6 * 16 + 4) * 8;
    return smem <= 227 * 1024 && P.nw <= 32 && 2 * P.nbuf + 1 <= 16;
}

__device__ __forceinline__ void named_sync(int id, int count) {
    asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(count) : "memory");
}
__device__ __forceinline__ void named_arrive(int id, int count) {
    asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(count) : "memory");
}

// One step of a chain along AXIS on the shells >= LO, in place (descending g reads not-yet-updated lower shells).
template <int AXIS, int LO, int NG>
__device__ __forceinline__ void chain_step(double (&z)[NG], double r) {
    static_for<0, NG - off(LO)>([&](auto ii) {
        constexpr int g = NG - 1 - decltype(ii)::value;
        if constexpr (cart_pow(g, AXIS) > 0) z[g] = fma(r, z[g], z[cart_dn(g, AXIS)]);
        else z[g] = r * z[g];
    });
}
// Last step, fused with the contraction: acc[a] += ck (r z[a] + z[a−1_i]) on the shells >= LA.
template <int AXIS, int LA, int NG, int NACC>
__device__ __forceinline__ void chain_last(const double (&z)[NG], double r, double ck, double (&acc)[NACC]) {
    static_for<0, NACC>([&](auto ii) {
        constexpr int g = off(LA) + decltype(ii)::value;
        double v;
        if constexpr (cart_pow(g, AXIS) > 0) v = fma(r, z[g], z[cart_dn(g, AXIS)]);
        else v = r * z[g];
        acc[g - off(LA)] = fma(ck, v, acc[g - off(LA)]);
    });
}

// Consumer body for one primitive: target with powers (TX, TY, TZ); zb = start vector [g][32] of its level.
template <int LA, int E, int TX, int TY, int TZ>
__device__ __forceinline__ void chain_apply(const double *__restrict__ zb, int lane, double rx, double ry, double rz,
                                            double ck, double (&acc)[off(E + 1) - off(LA)]) {
    constexpr int NG = off(E + 1), NACC = NG - off(LA), N = TX + TY + TZ;
    constexpr int LO0 = cmax(0, LA - N);                      // lowest shell any step reads
    double z[NG];
    static_for<off(LO0), NG>([&](auto ig) { z[decltype(ig)::value] = zb[decltype(ig)::value * 32 + lane]; });
    if constexpr (N == 0) {
        static_for<0, NACC>([&](auto ii) { acc[decltype(ii)::value] = fma(ck, z[off(LA) + decltype(ii)::value], acc[decltype(ii)::value]); });
    } else {
        static_for<1, N>([&](auto ij) {
            constexpr int j = decltype(ij)::value;           // step j of N, not the last
            constexpr int axis = j <= TX ? 0 : (j <= TX + TY ? 1 : 2);
            constexpr int LO = cmax(0, LA - (N - j));
            chain_step<axis, LO, NG>(z, axis == 0 ? rx : (axis == 1 ? ry : rz));
        });
        constexpr int axis = N <= TX ? 0 : (N <= TX + TY ? 1 : 2);
        chain_last<axis, LA, NG, NACC>(z, axis == 0 ? rx : (axis == 1 ? ry : rz), ck, acc);
    }
}

// Register offset of VRR1 node (shell e, order m, component ci): shells packed one after the other.
__host__ __device__ constexpr int v1_off(int E, int e) { int n = 0; for (int q = 0; q < e; ++q) n += nc(q) * (E - q + 1); return n; }

template <int LX, int LA, int LB, int MODE, int NW, int MINB>
__global__ void __launch_bounds__(NW * 32, MINB)
chain_kernel(SetMap map, DevShells aux, DevShells prim, PairData pdat, const double *__restrict__ boys_tab,
             double *__restrict__ out, int swapped, DfArgs df) {
    using CC = ChainCls<LX, LA, LB>;
    constexpr int E = CC::E, NG = CC::NG, NACC = CC::NACC, NXC = CC::NXC, NA = CC::NA, NB = CC::NB, NAB = CC::NAB;
    constexpr int NINT = CC::NINT, SLOTN = CC::SLOTN, ZREC = CC::ZREC;
    constexpr ChainTargets T = CC::T;
    constexpr ChainPlan P = CC::P;
    constexpr unsigned FULL = 0xffffffffu;

    extern __shared__ double smem[];
    double *TC = smem;                                       // [set][c * NAB + ·]: (e0|c), then the finished shell-set
    double *ZB = TC + (size_t)32 * SLOTN;                    // ring of start-vector buffers
    double *hd = ZB + (size_t)P.nbuf * ZREC;                 // header doubles [9][32]: A, C, AB
    long long *hpo = reinterpret_cast<long long *>(hd + 9 * 32);
    int *hi = reinterpret_cast<int *>(hpo + 32);             // [6][32]: xo0, Kab, K, a, b, x
    int *s_kmax = hi + 6 * 32;

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const long long nbatch = (map.nsets + 31) / 32;

    for (long long batch = blockIdx.x; batch < nbatch; batch += gridDim.x) {
        // ---- set of each lane (warp 0 decodes, everybody reads the header) ---------------------------------------------
        if (warp == 0) {
            const long long sid = batch * 32 + lane;
            const bool live = sid < map.nsets;
            int p = 0, xs = 0;
            if (live) {
                if (map.cum == nullptr) {
                    p = (int)(sid / map.nx);
                    xs = (int)(sid - (long long)p * map.nx);
                } else {
                    int lo = 0, hi_ = map.npair;             // largest p with cum[p] <= sid
                    while (hi_ - lo > 1) {
                        const int mid = (lo + hi_) >> 1;
                        if (map.cum[mid] <= sid) lo = mid; else hi_ = mid;
                    }
                    p = lo;
                    xs = (int)(sid - map.cum[p]);
                }
            }
            const int a = map.pair_list[2 * p + swapped], b = map.pair_list[2 * p + 1 - swapped];
            const int x = map.x_list[xs];
            const int Kab = prim.K[a] * prim.K[b];
            const int K = live ? Kab * aux.K[x] : 0;
#pragma unroll
            for (int d = 0; d < 3; ++d) {
                const double Ad = prim.center[3 * a + d];
                hd[d * 32 + lane] = Ad;
                hd[(3 + d) * 32 + lane] = aux.center[3 * x + d];
                hd[(6 + d) * 32 + lane] = Ad - prim.center[3 * b + d];
            }
            hpo[lane] = pdat.pd_off ? pdat.pd_off[p] : (long long)p * pdat.kstride;
            hi[0 * 32 + lane] = aux.prim_off[x];
            hi[1 * 32 + lane] = Kab;
            hi[2 * 32 + lane] = K;
            hi[3 * 32 + lane] = a;
            hi[4 * 32 + lane] = b;
            hi[5 * 32 + lane] = x;
            const int km = __reduce_max_sync(FULL, K);
            if (lane == 0) *s_kmax = km;
        }
        __syncthreads();
        const int kmax = *s_kmax;

        // ---- passes over the primitive loop --------------------------------------------------------------------------------
        static_for<0, P.npass>([&](auto ipass) {
            constexpr int ip = decltype(ipass)::value;
            constexpr int T0 = P.t0[ip], NC = P.t1[ip] - P.t0[ip], PLO = P.plo[ip], NLV = P.phi[ip] - P.plo[ip] + 1;
            constexpr int NPROD = P.nprod[ip], NBUF = NPROD + 1;
            constexpr int BCOUNT = (NC + 1) * 32;            // threads on a full[] / empty[] barrier
            double acc[NACC];
#pragma unroll
            for (int i = 0; i < NACC; ++i) acc[i] = 0.0;

            if (warp >= NC && warp < NC + NPROD) {
                // ================= producer: primitives q = j, j + NPROD, ... =================================================
                const int j = warp - NC;
                const double Ax = hd[0 * 32 + lane], Ay = hd[1 * 32 + lane], Az = hd[2 * 32 + lane];
                const double Cx = hd[3 * 32 + lane], Cy = hd[4 * 32 + lane], Cz = hd[5 * 32 + lane];
                const long long po = hpo[lane];
                const int xo0 = hi[0 * 32 + lane], Kab = hi[1 * 32 + lane], K = hi[2 * 32 + lane];
                for (int q = j; q < kmax; q += NPROD) {
                    const int bsel = q % NBUF;
                    if (q >= NBUF) named_sync(1 + NBUF + bsel, BCOUNT);      // consumers are done with this buffer
                    double *zb = ZB + (size_t)bsel * ZREC;
                    const bool on = q < K;
                    const int qq = on ? q : 0;
                    const int kx = qq / Kab, ij = qq - kx * Kab;
                    const double zc = aux.zeta[xo0 + kx], cxc = on ? aux.coef[xo0 + kx] : 0.0;
                    const double *pq = pdat.pd + (po + ij) * PD_STRIDE;
                    const double gm = __ldg(pq), Px = __ldg(pq + 1), Py = __ldg(pq + 2), Pz = __ldg(pq + 3),
                                 Kij = __ldg(pq + 4), o2g = __ldg(pq + 5);
                    const double PCx = Px - Cx, PCy = Py - Cy, PCz = Pz - Cz;
                    const double o2z = 0.5 / zc;
                    const double sq = rsqrt(gm + zc);         // (γ+ζc)^{-1/2}
                    const double igz = sq * sq;
                    const double mrg = -zc * igz;             // −ρ/γ
                    const double mrz = -gm * igz;             // −ρ/ζc
                    const double PA[3] = {Px - Ax, Py - Ay, Pz - Az};
                    const double WP[3] = {mrg * PCx, mrg * PCy, mrg * PCz};
                    const double Tt = gm * zc * igz * (PCx * PCx + PCy * PCy + PCz * PCz);
                    // eq. 4: 2π^{5/2}/(γ ζc sqrt(γ+ζc)) K_ij c_k = 8π^{5/2} (1/2γ)(1/2ζc)(γ+ζc)^{-1/2} K_ij c_k
                    const double pref = 139.94734662099889988 * Kij * cxc * o2g * o2z * sq;
                    const double g2 = gm + gm;
                    const double cs = 0.5 * igz;              // 1/(2(γ+ζc))
                    double *rec = zb + (size_t)NLV * NG * 32;
                    rec[0 * 32 + lane] = g2 * PCx;
                    rec[1 * 32 + lane] = g2 * PCy;
                    rec[2 * 32 + lane] = g2 * PCz;
                    // Boys orders LX − 2p .. LX − p + E for the levels of this pass: one table evaluation at the top
                    constexpr int MLO = LX - 2 * (PLO + NLV - 1), MHI = LX - PLO + E;
                    double F[MHI - MLO + 1];
                    if (Tt < (double)BOYS_TMAX) {
                        F[MHI - MLO] = boys_one(boys_tab, MHI, Tt);
                        if constexpr (MHI > MLO) {
                            const double eT = exp(-Tt), T2 = Tt + Tt;
#pragma unroll
                            for (int m = MHI; m > MLO; --m) F[m - 1 - MLO] = fma(T2, F[m - MLO], eT) * (1.0 / (double)(2 * m - 1));
                        }
                    } else {
                        double f = 0.5 * sqrt(3.14159265358979323846 / Tt);
                        const double h = 0.5 / Tt;
#pragma unroll
                        for (int m = 0; m <= MHI; ++m) {
                            if (m >= MLO) F[m - MLO] = f;
                            f *= (double)(2 * m + 1) * h;
                        }
                    }
                    static_for<0, NLV>([&](auto ilv) {
                        constexpr int lv = decltype(ilv)::value, p = PLO + lv, k = LX - 2 * p;
                        // deferred scalar of the level: (1/(2(γ+ζc)))^k (1/(2ζc))^p
                        double ck = 1.0;
#pragma unroll
                        for (int i = 0; i < k; ++i) ck *= cs;
#pragma unroll
                        for (int i = 0; i < p; ++i) ck *= o2z;
                        rec[(3 + lv) * 32 + lane] = ck;
                        // a3: VRR1 (eq. 3) on W^(m) = pref Σ_s C(p,s) (−ρ/ζc)^s F_{k+m+s}, m = 0..E
                        constexpr int NV = chain_nv1(E);
                        double V[NV];
                        static_for<0, E + 1>([&](auto im) {
                            constexpr int m = decltype(im)::value;
                            double w = F[k + m + p - MLO];
                            static_for<0, p>([&](auto is) {
                                constexpr int s = p - 1 - decltype(is)::value;     // Horner in (−ρ/ζc)
                                w = fma(w, mrz, (double)ibinom(p, s) * F[k + m + s - MLO]);
                            });
                            V[m] = pref * w;
                        });
                        static_for<1, E + 1>([&](auto ie) {
                            constexpr int e = decltype(ie)::value;
                            static_for<0, nc(e)>([&](auto ici) {
                                constexpr int ci = decltype(ici)::value, g = off(e) + ci;
                                constexpr int dir = (int)(cart_entry(g) >> 24), ai = cart_pow(g, dir);
                                constexpr int g1 = cart_dn(g, dir), c1 = g1 - off(e - 1);
                                static_for<0, E - e + 1>([&](auto im) {
                                    constexpr int m = decltype(im)::value;
                                    constexpr int i1 = v1_off(E, e - 1) + m * nc(e - 1) + c1;
                                    double v = fma(WP[dir], V[i1 + nc(e - 1)], PA[dir] * V[i1]);
                                    if constexpr (ai > 1) {
                                        constexpr int c2 = cart_dn(g1, dir) - off(e - 2);
                                        constexpr int i2 = v1_off(E, e - 2) + m * nc(e - 2) + c2;
                                        v = fma((double)(ai - 1) * o2g, fma(mrg, V[i2 + nc(e - 2)], V[i2]), v);
                                    }
                                    V[v1_off(E, e) + m * nc(e) + ci] = v;
                                });
                            });
                        });
                        // start vector u[a] = Y_p[a] / a!
                        static_for<0, NG>([&](auto ig) {
                            constexpr int g = decltype(ig)::value, e = cart_shell(g);
                            constexpr double inv = 1.0 / (double)cart_fact(g);
                            zb[((size_t)lv * NG + g) * 32 + lane] = V[v1_off(E, e) + (g - off(e))] * inv;
                        });
                    });
                    __threadfence_block();
                    named_arrive(1 + bsel, BCOUNT);           // full[bsel]
                }
            } else if (warp < NC) {
                // ================= consumer: target T0 + warp ====================================================================
                for (int q = 0; q < kmax; ++q) {
                    const int bsel = q % NBUF;
                    named_sync(1 + bsel, BCOUNT);             // full[bsel]
                    const double *zb = ZB + (size_t)bsel * ZREC;
                    const double *rec = zb + (size_t)NLV * NG * 32;
                    const double rx = rec[0 * 32 + lane], ry = rec[1 * 32 + lane], rz = rec[2 * 32 + lane];
                    static_for<0, NC>([&](auto iw) {
                        constexpr int w = decltype(iw)::value, tg = T.g[T0 + w], lv = T.p[T0 + w] - PLO;
                        if (warp == w) {
                            const double ck = rec[(3 + lv) * 32 + lane];
                            chain_apply<LA, E, cart_pow(tg, 0), cart_pow(tg, 1), cart_pow(tg, 2)>(zb + (size_t)lv * NG * 32, lane, rx, ry, rz, ck, acc);
                        }
                    });
                    if (q + NBUF < kmax) named_arrive(1 + NBUF + bsel, BCOUNT);   // empty[bsel]
                }
            }
            __syncthreads();
            // ---- combine the targets into (e0|c): level 0 writes, higher levels add β·U one role after the other (deterministic) ----
            double *mine = TC + (size_t)lane * SLOTN;
            static_for<0, NC>([&](auto iw) {
                constexpr int w = decltype(iw)::value, tg = T.g[T0 + w], p = T.p[T0 + w];
                if constexpr (p == 0) {
                    if (warp == w) {
                        constexpr int cidx = tg - off(LX);
                        static_for<0, NACC>([&](auto ii) {
                            constexpr int i = decltype(ii)::value;
                            mine[cidx * NAB + i] = acc[i] * (double)cart_fact(off(LA) + i);
                        });
                    }
                }
            });
            static_for<0, NC>([&](auto iw) {
                constexpr int w = decltype(iw)::value, tg = T.g[T0 + w], p = T.p[T0 + w];
                if constexpr (p > 0) {
                    __syncthreads();
                    if (warp == w) {
                        constexpr int tx = cart_pow(tg, 0), ty = cart_pow(tg, 1), tz = cart_pow(tg, 2);
                        static_for<0, p + 1>([&](auto inx) {
                            constexpr int nx = decltype(inx)::value;
                            static_for<0, p - nx + 1>([&](auto iny) {
                                constexpr int ny = decltype(iny)::value, nz = p - nx - ny;
                                constexpr int cx = tx + 2 * nx, cy = ty + 2 * ny, cz = tz + 2 * nz;
                                constexpr int cidx = cart_index(cx, cy, cz) - off(LX);
                                constexpr double beta = (double)(beta1(cx, nx) * beta1(cy, ny) * beta1(cz, nz));
                                static_for<0, NACC>([&](auto ii) {
                                    constexpr int i = decltype(ii)::value;
                                    mine[cidx * NAB + i] += (beta * (double)cart_fact(off(LA) + i)) * acc[i];
                                });
                            });
                        });
                    }
                }
            });
            __syncthreads();
        });

        // ---- a7: HRR (eq. 1) in registers per (set = lane, c), in place in the set's region --------------------------------
        if constexpr (LB > 0) {
            const double AB[3] = {hd[6 * 32 + lane], hd[7 * 32 + lane], hd[8 * 32 + lane]};
            for (int c = warp; c < NXC; c += NW) {
                double *reg = TC + (size_t)lane * SLOTN + c * NAB;
                double H0[NACC];
                static_for<0, NACC>([&](auto ii) { H0[decltype(ii)::value] = reg[decltype(ii)::value]; });
                constexpr int NA1 = off(E) - off(LA);        // bra components of the shells LA..E−1
                double H1[NA1 * 3];
                static_for<0, NA1>([&](auto ial) {
                    constexpr int al = decltype(ial)::value, g = off(LA) + al;
                    static_for<0, 3>([&](auto id) {
                        constexpr int d = decltype(id)::value;
                        H1[al * 3 + d] = fma(AB[d], H0[al], H0[cart_up(g, d) - off(LA)]);
                    });
                });
                if constexpr (LB == 1) {
                    static_for<0, NA * 3>([&](auto ii) { reg[decltype(ii)::value] = H1[decltype(ii)::value]; });
                } else {
                    static_assert(LB <= 2, "chain kernel: HRR written for Lb <= 2");
                    static_for<0, NA>([&](auto ial) {
                        constexpr int al = decltype(ial)::value, g = off(LA) + al;
                        static_for<0, 6>([&](auto ib) {
                            constexpr int bj = decltype(ib)::value, gb = off(2) + bj;
                            constexpr int d = (int)(cart_entry(gb) >> 24);
                            constexpr int b1 = cart_dn(gb, d) - off(1);
                            reg[al * 6 + bj] = fma(AB[d], H1[al * 3 + b1], H1[(cart_up(g, d) - off(LA)) * 3 + b1]);
                        });
                    });
                }
            }
            __syncthreads();
        }

        // ---- a8 / a9 / a10: one warp per set -----------------------------------------------------------------------------------
        for (int s = warp; s < 32; s += NW) {
            const long long sid_s = batch * 32 + s;
            if (sid_s >= map.nsets) break;                    // warp-uniform
            const double *FIN = TC + (size_t)s * SLOTN;       // finished shell-set, layout [c][a][b]
            if constexpr (MODE == 0) {
                double *o = out + sid_s * NINT;
                if (!swapped || LB == 0) {
                    for (int r = lane; r < NINT; r += 32) o[r] = FIN[r];
                } else {                                      // caller's order is [c][b][a]
                    for (int r = lane; r < NINT; r += 32) {
                        const int ia = r % NA, t = r / NA, ib = t % NB, c = t / NB;
                        o[r] = FIN[(c * NA + ia) * NB + ib];
                    }
                }
            } else {
                const int as = hi[3 * 32 + s], bs = hi[4 * 32 + s], xs_ = hi[5 * 32 + s];
                if constexpr (MODE == 1) {
                    // γ[bf(X)+c] += f Σ_ab (c|ab) D[bf(a)+ia, bf(b)+ib]
                    const double *Dab = df.D + (size_t)prim.bf_off[as] * df.ld + prim.bf_off[bs];
                    const double f = (as != bs) ? 2.0 : 1.0;
                    for (int c = lane; c < NXC; c += 32) {
                        const double *Fc = FIN + c * NAB;
                        double sum = 0.0;
                        for (int ia = 0; ia < NA; ++ia)
#pragma unroll
                            for (int ib = 0; ib < NB; ++ib) sum = fma(Fc[ia * NB + ib], __ldg(Dab + (size_t)ia * df.ld + ib), sum);
                        atomicAdd(df.out + aux.bf_off[xs_] + c, f * sum);
                    }
                } else {
                    // J[bf(a)+ia, bf(b)+ib] += Σ_c (c|ab) d[bf(X)+c], mirrored
                    const double *dx = df.D + aux.bf_off[xs_];
                    const size_t ra0 = prim.bf_off[as], rb0 = prim.bf_off[bs];
                    for (int r = lane; r < NAB; r += 32) {
                        double sum = 0.0;
#pragma unroll
                        for (int c = 0; c < NXC; ++c) sum = fma(FIN[c * NAB + r], __ldg(dx + c), sum);
                        const int ia = r / NB, ib = r - ia * NB;
                        atomicAdd(df.out + (ra0 + ia) * df.ld + rb0 + ib, sum);
                        if (as != bs) atomicAdd(df.out + (rb0 + ib) * df.ld + ra0 + ia, sum);
                    }
                }
            }
        }
        __syncthreads();
    }
}

template <int LX, int LA, int LB, int MODE>
cudaError_t chain_launch(const SetMap &map, const DevShells &aux, const DevShells &prim, const PairData &pdat,
                         const double *boys_tab, double *out, int swapped, const DfArgs &df, int num_sms,
                         cudaStream_t stream) {
    using CC = ChainCls<LX, LA, LB>;
    constexpr int NW = CC::NW;
    constexpr size_t smem = CC::smem;
    // resident blocks per SM: shared memory, and registers (a consumer keeps NG + NACC doubles live)
    constexpr int by_smem = (int)((227 * 1024) / (smem + 1024));
    constexpr int regs = CC::E <= 2 ? 80 : (CC::E == 3 ? 128 : 168);
    constexpr int by_regs = 65536 / (NW * 32 * regs);
    constexpr int BPS = cmax(1, cmin(cmin(by_smem, by_regs), 8));
    auto kern = chain_kernel<LX, LA, LB, MODE, NW, BPS>;
    static bool configured = false;
    if (!configured) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        configured = true;
    }
    if (map.nsets <= 0) return cudaSuccess;
    long long blocks = (map.nsets + 31) / 32;
    const long long cap = (long long)num_sms * BPS;
    if (blocks > cap) blocks = cap;
    kern<<<(unsigned)blocks, NW * 32, smem, stream>>>(map, aux, prim, pdat, boys_tab, out, swapped, df);
    return cudaGetLastError();
}

}  // namespace lx
