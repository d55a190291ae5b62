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
    int ring;                                       // doubles of the ring (npx + 1 buffers of zrec doubles)
    int ncx, npx, zrec;                             // consumer / producer warps of the block, doubles per ring buffer
    bool ok;                                        // every target of a level p >= 1 sits in the last pass
};
// doubles of one ring buffer of a pass over nlev levels: start vectors [level][g][32], r[3][32], ck[level][32]
__host__ __device__ constexpr int chain_zrec(int nlev, int NG) { return (nlev * NG + 3 + nlev) * 32; }
// Consumer warps per pass are capped by the register budget (a consumer keeps NG + NA_ACC doubles live); producers
// per pass balance the VRR1 pyramids of the pass's levels against the chain of its first (longest) target.
constexpr ChainPlan chain_plan(int LX, int LA, int LB) {
    const int E = LA + LB, NG = off(E + 1), NACC = NG - off(LA);
    const ChainTargets T = chain_targets(LX);
    const int cap = E <= 2 ? 16 : (E == 3 ? 11 : 8);
    const int nwmax = E <= 2 ? 24 : (E == 3 ? 16 : 12);
    ChainPlan P{};
    P.npass = (T.n + cap - 1) / cap;
    const int ncw = (T.n + P.npass - 1) / P.npass;
    P.nw = 0; P.ring = 0; P.ok = true; P.ncx = 0; P.npx = 0;
    int nlevx = 0;
    for (int i = 0; i < P.npass; ++i) {
        // even split, except that the targets of the levels p >= 1 (index >= nc(LX)) all go to the last pass
        P.t0[i] = i == 0 ? 0 : P.t1[i - 1];
        P.t1[i] = i == P.npass - 1 ? T.n : cmin(nc(LX), (i + 1) * ncw);
        if (P.t1[i] - P.t0[i] > cap || P.t1[i] <= P.t0[i]) P.ok = false;
        P.plo[i] = T.p[P.t0[i]];
        P.phi[i] = T.p[P.t1[i] - 1];
        if (P.phi[i] > 0 && i != P.npass - 1) P.ok = false;
        const int nlev = P.phi[i] - P.plo[i] + 1;
        const int k0 = LX - 2 * P.plo[i];                              // steps of the longest chain of the pass
        const int cons = cmax(1, k0) * NG + 2 * NACC + NG + 10;       // instructions per primitive (measured shape)
        const int prod = nlev * (4 * chain_nv1(E) + 2 * NG + 60) + 130;
        int np = (prod + cons - 1) / cons;
        np = cmax(1, cmin(np, cmin(6, nwmax - (P.t1[i] - P.t0[i]))));
        P.nprod[i] = np;
        P.ncx = cmax(P.ncx, P.t1[i] - P.t0[i]);
        P.npx = cmax(P.npx, np);
        nlevx = cmax(nlevx, nlev);
    }
    // one ring for all passes; it shares 227 KB with the (e0|c) region of the 32 sets, the header and two small tables
    P.npx = cmin(P.npx, nwmax - P.ncx);
    P.zrec = chain_zrec(nlevx, NG);
    const int room = (227 * 1024) / 8 - 32 * ((nc(LX) * nc(LA) * nc(LB)) | 1) - 944 - 256;
    while (P.npx > 1 && (P.npx + 1) * P.zrec > room) --P.npx;
    P.nw = P.ncx + P.npx;
    P.ring = (P.npx + 1) * P.zrec;
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
    static constexpr int NUB = (T.n - NXC) * NACC * 32;       // staging of the contracted targets of the levels p >= 1
    static constexpr int ZBD = cmax(P.ring, NUB);             // the staging area aliases the ring
    static constexpr int HDR1 = 9 * 32 + 32 + 7 * 16 + 4;     // header: 9 doubles + 1 int64 + 7 ints per set + kmax, in doubles
    static constexpr int HDRD = 2 * HDR1;                     // double-buffered (the next batch is decoded ahead)
    static constexpr size_t smem = ((size_t)32 * SLOTN + (size_t)ZBD + HDRD + 4) * 8 + 2048;   // + partner table
    static constexpr bool fits = E <= 4 && LX <= 4 && P.ok && smem <= 227 * 1024 && NW <= 32;
};
__host__ __device__ constexpr bool chain_fits(int LX, int LA, int LB) {
    if (LA + LB > 4 || LX > 4) return false;
    const ChainPlan P = chain_plan(LX, LA, LB);
    const int NG = off(LA + LB + 1), NACC = NG - off(LA);
    int NT = 0;
    for (int p = 0; 2 * p <= LX; ++p) NT += nc(LX - 2 * p);
    const int nub = (NT - nc(LX)) * NACC * 32;
    const size_t smem = ((size_t)32 * ((nc(LX) * nc(LA) * nc(LB)) | 1) + (size_t)cmax(P.ring, nub) + 2 * (9 * 32 + 32 + 7 * 16 + 4) + 4) * 8 + 2048;
    return P.ok && smem <= 227 * 1024 && P.nw <= 32;
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

}  // namespace lx
