// lx_team.cuh — register-only class kernel ("team kernel"): the chain form of lx_chain.cuh without the producer /
// consumer hand-off.  LANE = shell-set as there; a block is a team of W warps that share one batch of 32 shell-sets and
// split the chain targets (p, t) between them.  Every warp evaluates, per primitive triple and entirely in its own
// registers: prefactors, Boys (a2), the VRR1 pyramid (a3, eq. 3) of each level it needs, the chains of its targets (a4)
// and their contraction (a5).  There is no shared-memory traffic and no barrier inside the primitive loop; with W = 1
// ("solo") nothing is computed twice, with W > 1 only the cheap VRR1 pyramids are.  Shared memory is touched once per
// batch: the contracted targets are dropped there, gathered with the integers β(c,n) into (e0|c), run through the HRR
// (a7, eq. 1) in registers per (set, c), and stored coalesced or digested (a8–a10).
// Used where the targets of a warp fit its registers (small La+Lb or small Lx); the warp-specialised chain kernel
// covers the rest.
#pragma once
#include "lx_chain.cuh"

namespace lx {

// Per-primitive scalars of one shell-set, lane-private.
struct PrimRec {
    double PA[3], WP[3], r[3];   // P−A;  −(ρ/γ)(P−C);  2γ(P−C)
    double o2g, mrg, mrz, o2z;   // 1/2γ;  −ρ/γ;  −ρ/ζc;  1/2ζc
    double cs;                   // 1/(2(γ+ζc))
    double pref, T;              // eq. 4 prefactor (with K_ij c_k; 0 for a padded primitive);  ρ|PC|²
};

__device__ __forceinline__ PrimRec prim_rec(const double *__restrict__ pq, double zc, double cxc, const double (&A)[3],
                                            const double (&C)[3]) {
    PrimRec R;
    const double gm = __ldg(pq), Px = __ldg(pq + 1), Py = __ldg(pq + 2), Pz = __ldg(pq + 3), Kij = __ldg(pq + 4);
    R.o2g = __ldg(pq + 5);
    const double PCx = Px - C[0], PCy = Py - C[1], PCz = Pz - C[2];
    R.o2z = 0.5 / zc;
    const double sq = rsqrt(gm + zc);         // (γ+ζc)^{-1/2}
    const double igz = sq * sq;
    R.mrg = -zc * igz;
    R.mrz = -gm * igz;
    R.PA[0] = Px - A[0]; R.PA[1] = Py - A[1]; R.PA[2] = Pz - A[2];
    R.WP[0] = R.mrg * PCx; R.WP[1] = R.mrg * PCy; R.WP[2] = R.mrg * PCz;
    const double g2 = gm + gm;
    R.r[0] = g2 * PCx; R.r[1] = g2 * PCy; R.r[2] = g2 * PCz;
    R.cs = 0.5 * igz;
    R.T = gm * zc * igz * (PCx * PCx + PCy * PCy + PCz * PCz);
    // eq. 4: 2π^{5/2}/(γ ζc sqrt(γ+ζc)) K_ij c_k = 8π^{5/2} (1/2γ)(1/2ζc)(γ+ζc)^{-1/2} K_ij c_k
    R.pref = 139.94734662099889988 * Kij * cxc * R.o2g * R.o2z * sq;
    return R;
}

// F_m(T) for m = MLO..MHI, branch-free so that the scheduler can interleave it with the chains of the previous primitive:
// the top order from the table (degree-7 Taylor around the nearest grid point, index clamped) or, for T >= BOYS_TMAX,
// from the asymptotic form (2M−1)!!/2^{M+1} sqrt(π) T^{−M−1/2}; then the downward recursion
// F_{m−1} = (2T F_m + e^{−T})/(2m−1), which is stable for every T.
template <int MLO, int MHI>
__device__ __forceinline__ void boys_range(const double *__restrict__ tab, double T, double (&F)[MHI - MLO + 1]) {
    const bool far = T >= (double)BOYS_TMAX;
    const double Tt = far ? (double)BOYS_TMAX - 0.03125 : T;
    const int i = __double2int_rn(Tt * (double)BOYS_PER_UNIT);
    const double d = (double)i * (1.0 / BOYS_PER_UNIT) - Tt;  // −Δ
    const double *row = tab + (size_t)i * BOYS_MROWS + MHI;
    double t = __ldg(row + 7) * (1.0 / 7.0);
    t = fma(t, d, __ldg(row + 6)) * (1.0 / 6.0);
    t = fma(t, d, __ldg(row + 5)) * (1.0 / 5.0);
    t = fma(t, d, __ldg(row + 4)) * (1.0 / 4.0);
    t = fma(t, d, __ldg(row + 3)) * (1.0 / 3.0);
    t = fma(t, d, __ldg(row + 2)) * (1.0 / 2.0);
    t = fma(t, d, __ldg(row + 1));
    t = fma(t, d, __ldg(row));
    const double rs = rsqrt(T), it = rs * rs;
    double a = 0.88622692545275801365 * rs;                  // sqrt(π)/2 · T^{−1/2}
#pragma unroll
    for (int k = 0; k < MHI; ++k) a *= ((double)(2 * k + 1) * 0.5) * it;
    F[MHI - MLO] = far ? a : t;
    if constexpr (MHI > MLO) {
        const double eT = exp(-T), T2 = T + T;
#pragma unroll
        for (int m = MHI; m > MLO; --m) F[m - 1 - MLO] = fma(T2, F[m - MLO], eT) * (1.0 / (double)(2 * m - 1));
    }
}

// Start vector of level p: u[a] = (Δ^p Z^{(LX−2p)})[a] / a!, a over the shells 0..E (lx_chain.cuh header).
// F holds the Boys values from order MLO on.
template <int LX, int E, int P_, int MLO, int NF>
__device__ __forceinline__ void vrr1_level(const PrimRec &R, const double (&F)[NF], double (&u)[off(E + 1)]) {
    constexpr int k = LX - 2 * P_, NV = chain_nv1(E), NG = off(E + 1);
    double V[NV];
    static_for<0, E + 1>([&](auto im) {
        constexpr int m = decltype(im)::value;
        double w = F[k + m + P_ - MLO];
        static_for<0, P_>([&](auto is) {
            constexpr int s = P_ - 1 - decltype(is)::value;     // Horner in (−ρ/ζc)
            w = fma(w, R.mrz, (double)ibinom(P_, s) * F[k + m + s - MLO]);
        });
        V[m] = R.pref * w;
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
                double v = fma(R.WP[dir], V[i1 + nc(e - 1)], R.PA[dir] * V[i1]);
                if constexpr (ai > 1) {
                    constexpr int c2 = cart_dn(g1, dir) - off(e - 2);
                    constexpr int i2 = v1_off(E, e - 2) + m * nc(e - 2) + c2;
                    v = fma((double)(ai - 1) * R.o2g, fma(R.mrg, V[i2 + nc(e - 2)], V[i2]), v);
                }
                V[v1_off(E, e) + m * nc(e) + ci] = v;
            });
        });
    });
    static_for<0, NG>([&](auto ig) {
        constexpr int g = decltype(ig)::value, e = cart_shell(g);
        constexpr double inv = 1.0 / (double)cart_fact(g);
        u[g] = V[v1_off(E, e) + (g - off(e))] * inv;
    });
}

// deferred scalar of level p: (1/(2(γ+ζc)))^{LX−2p} (1/(2ζc))^p
template <int K_, int P_>
__device__ __forceinline__ double level_scale(const PrimRec &R) {
    double ck = 1.0;
#pragma unroll
    for (int i = 0; i < K_; ++i) ck *= R.cs;
#pragma unroll
    for (int i = 0; i < P_; ++i) ck *= R.o2z;
    return ck;
}

// Chain of target (TX, TY, TZ) on a register copy of the start vector u; acc += ck · (Π B^t u)[shells >= LA].
template <int LA, int E, int TX, int TY, int TZ>
__device__ __forceinline__ void chain_apply_reg(const double (&u)[off(E + 1)], const double (&r)[3], double ck,
                                                double *__restrict__ acc) {
    constexpr int NG = off(E + 1), NACC = NG - off(LA), N = TX + TY + TZ;
    if constexpr (N == 0) {
        static_for<0, NACC>([&](auto ii) { acc[decltype(ii)::value] = fma(ck, u[off(LA) + decltype(ii)::value], acc[decltype(ii)::value]); });
    } else {
        double z[NG];
        constexpr int LO0 = cmax(0, LA - N);
        static_for<off(LO0), NG>([&](auto ig) { z[decltype(ig)::value] = u[decltype(ig)::value]; });
        static_for<1, N>([&](auto ij) {
            constexpr int j = decltype(ij)::value;
            constexpr int axis = j <= TX ? 0 : (j <= TX + TY ? 1 : 2);
            constexpr int LO = cmax(0, LA - (N - j));
            chain_step<axis, LO, NG>(z, r[axis]);
        });
        constexpr int axis = N <= TX ? 0 : (N <= TX + TY ? 1 : 2);
        static_for<0, NACC>([&](auto ii) {
            constexpr int g = off(LA) + decltype(ii)::value;
            double v;
            if constexpr (cart_pow(g, axis) > 0) v = fma(r[axis], z[g], z[cart_dn(g, axis)]);
            else v = r[axis] * z[g];
            acc[g - off(LA)] = fma(ck, v, acc[g - off(LA)]);
        });
    }
}


// ---- shell-set of a lane ------------------------------------------------------------------------------------------
struct SetId { int p, a, b, x; bool live; };

// Prefix map (DF calls): the pair of a set id is the largest p with cum[p] <= sid.  A per-lane binary search over up to 3.3 M
// pairs (config 5) is a chain of 22 DEPENDENT global loads at the head of every batch — for weakly contracted classes longer
// than the arithmetic of the batch (ncu: long-scoreboard stalls 2.5–6 per issue, profiles/r02_ncu_team_df.md).  The 32 set ids
// of a warp are consecutive, so the warp searches ONCE, 32-ary (5 rounds for 3.3 M pairs: every lane probes one point, a ballot
// counts the points at or below the first id), then one coalesced load of the next 32 pair starts places every lane.
// All 32 lanes must call; lane 0 holds the smallest id and every id lies within 32 of it.
__device__ __forceinline__ void find_pair_warp(const SetMap &map, long long sid, bool live, int &p, int &xs) {
    constexpr unsigned FULL = 0xffffffffu;
    const int lane = threadIdx.x & 31;
    const long long sid0 = __shfl_sync(FULL, sid, 0);
    p = 0;
    xs = 0;
    if (sid0 >= map.nsets) return;                            // warp-uniform: no live set
    int lo = 0, hi = map.npair;                                // cum[lo] <= sid0 < cum[hi]
    while (hi - lo > 1) {
        const int step = (hi - lo + 31) >> 5;
        const long long idx = (long long)lo + (long long)(lane + 1) * step;
        const bool ok = idx < hi && map.cum[idx] <= sid0;      // cum is non-decreasing: the lanes that say yes are a prefix
        const int cnt = __popc(__ballot_sync(FULL, ok));
        lo += cnt * step;
        hi = min(hi, lo + step);
    }
    const int P0 = lo;
    const long long jn = (long long)P0 + 1 + lane;
    const long long c = jn <= map.npair ? map.cum[jn] : 0x7fffffffffffffffLL;   // start of pair P0 + 1 + lane
    long long start = map.cum[P0];
    int cnt = 0, j = 0;
#pragma unroll 1
    for (; j < 32; ++j) {
        const long long cj = __shfl_sync(FULL, c, j);
        if (cj > sid0 + 31) break;                             // warp-uniform: no id of this warp reaches pair P0 + 1 + j
        if (cj <= sid) { ++cnt; start = cj; }
    }
    int pp = P0 + cnt;
    if (cnt == 32 && live) {                                   // more than 32 pairs inside one batch (sparse survivors): finish alone
        int l2 = P0 + 32, h2 = map.npair;
        while (h2 - l2 > 1) {
            const int mid = (l2 + h2) >> 1;
            if (map.cum[mid] <= sid) l2 = mid; else h2 = mid;
        }
        pp = l2;
        start = map.cum[pp];
    }
    if (live) {
        p = pp;
        xs = (int)(sid - start);
    }
}

// With a prefix map every lane of the warp must call (find_pair_warp).
__device__ __forceinline__ SetId decode_set(const SetMap &map, long long sid, int swapped) {
    SetId s;
    s.live = sid < map.nsets;
    int p = 0, xs = 0;
    if (map.cum == nullptr) {
        if (s.live) {
            p = (int)(sid / map.nx);
            xs = (int)(sid - (long long)p * map.nx);
        }
    } else {
        find_pair_warp(map, sid, s.live, p, xs);
    }
    s.p = p;
    s.a = map.pair_list[2 * p + swapped];
    s.b = map.pair_list[2 * p + 1 - swapped];
    s.x = map.x_list[xs];
    return s;
}

// position of target (level p, component t with cumulative index g) in the target list of chain_targets(LX)
__host__ __device__ constexpr int target_index(int LX, int p, int g) {
    int o = 0;
    for (int q = 0; q < p; ++q) o += nc(LX - 2 * q);
    return o + g - off(LX - 2 * p);
}

// Partner table of the gather step, built once per block in shared memory by compile-time unrolled stores:
// for every Cartesian c the targets (level p >= 1, t = c − 2n) that contribute, with their integer weights β(c,n).
constexpr int CHAIN_MAXPART = 8;
struct PartnerTab {
    int cnt[nc(LX_MAX_L_AUX)];
    int ti[nc(LX_MAX_L_AUX)][CHAIN_MAXPART];
    int beta[nc(LX_MAX_L_AUX)][CHAIN_MAXPART];
};
template <int LX>
__device__ __forceinline__ void partner_tab_build(PartnerTab *pt) {
    static_for<0, nc(LX)>([&](auto ic) {
        constexpr int c = decltype(ic)::value, gc = off(LX) + c;
        constexpr int cx = cart_pow(gc, 0), cy = cart_pow(gc, 1), cz = cart_pow(gc, 2);
        int k = 0;
        static_for<0, cx / 2 + 1>([&](auto inx) {
            static_for<0, cy / 2 + 1>([&](auto iny) {
                static_for<0, cz / 2 + 1>([&](auto inz) {
                    constexpr int nx = decltype(inx)::value, ny = decltype(iny)::value, nz = decltype(inz)::value;
                    if constexpr (nx + ny + nz > 0) {
                        pt->ti[c][k] = target_index(LX, nx + ny + nz, cart_index(cx - 2 * nx, cy - 2 * ny, cz - 2 * nz));
                        pt->beta[c][k] = beta1(cx, nx) * beta1(cy, ny) * beta1(cz, nz);
                        ++k;
                    }
                });
            });
        });
        pt->cnt[c] = k;
    });
}

// Drop the contracted target ti (run-time, warp-uniform) of this lane's set: level 0 goes straight to its Cartesian slot
// of TC, higher levels to the staging area UB[(ti − NXC)][i][lane]; both scaled back by a! (lx_chain.cuh header).
// One copy of this code serves every target: code that runs once per batch must stay small (instruction cache).
template <int LX, int LA, int LB, int CSTR = ChainCls<LX, LA, LB>::NAB, int SLOT = ChainCls<LX, LA, LB>::SLOTN>
__device__ __forceinline__ void target_drop(int ti, const double *__restrict__ acc, double *__restrict__ TC,
                                            double *__restrict__ UB, int lane) {
    using CC = ChainCls<LX, LA, LB>;
    constexpr int NACC = CC::NACC, NXC = CC::NXC;
    // TC slot of a set: SLOT doubles, CSTR per ket component (the defaults leave room for the in-place HRR)
    double *dst = ti < NXC ? TC + (size_t)lane * SLOT + ti * CSTR : UB + (size_t)(ti - NXC) * NACC * 32 + lane;
    const int stride = ti < NXC ? 1 : 32;
    static_for<0, NACC>([&](auto ii) {
        constexpr int i = decltype(ii)::value;
        dst[i * stride] = acc[i] * (double)cart_fact(off(LA) + i);
    });
}

// a7: HRR (eq. 1) of one (set, ket component) in registers: H0 = (e0| for the shells e = LA..LA+LB in,
// (a b| out to reg[a][b] (tr: reg[b][a], the caller's order of a mirrored class).  Written for LB <= 2.
template <int LA, int LB>
__device__ __forceinline__ void hrr_store(const double (&H0)[off(LA + LB + 1) - off(LA)], const double (&AB)[3],
                                          double *__restrict__ reg, bool tr) {
    constexpr int E = LA + LB, NACC = off(E + 1) - off(LA), NA = nc(LA);
    if constexpr (LB == 0) {
        static_for<0, NACC>([&](auto ii) { reg[decltype(ii)::value] = H0[decltype(ii)::value]; });
    } else {
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
            static_for<0, NA * 3>([&](auto ii) {
                constexpr int i = decltype(ii)::value;
                reg[tr ? (i % 3) * NA + i / 3 : i] = H1[i];
            });
        } else {
            static_assert(LB <= 2, "HRR written for Lb <= 2");
            static_for<0, NA>([&](auto ial) {
                constexpr int al = decltype(ial)::value, g = off(LA) + al;
                static_for<0, 6>([&](auto ib) {
                    constexpr int bj = decltype(ib)::value, gb = off(2) + bj;
                    constexpr int d = (int)(cart_entry(gb) >> 24);
                    constexpr int b1 = cart_dn(gb, d) - off(1);
                    reg[tr ? bj * NA + al : al * 6 + bj] = fma(AB[d], H1[al * 3 + b1], H1[(cart_up(g, d) - off(LA)) * 3 + b1]);
                });
            });
        }
    }
}

// a8: a batch is one contiguous run of out[]; `nthr` threads (index tid) copy it, four independent elements in flight each.
template <int NINT, int SLOTN>
__device__ __forceinline__ void batch_copy_out(const double *__restrict__ TC, double *__restrict__ out, long long batch,
                                               long long nsets, int tid, int nthr) {
    const long long nlive = min((long long)32, nsets - batch * 32);
    const int total = (int)nlive * NINT;
    double *o = out + batch * 32 * NINT;
    for (int it0 = tid; it0 < total; it0 += nthr * 4) {
        double v[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const int it = it0 + u * nthr;
            if (it < total) {
                const int sset = it / NINT, r = it - sset * NINT;
                v[u] = TC[(size_t)sset * SLOTN + r];
            }
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const int it = it0 + u * nthr;
            if (it < total) o[it] = v[u];
        }
    }
}

// After the targets of a batch were dropped (and a block barrier): gather (e0|c) = U_{0,c} + Σ_{n>0} β(c,n) U_{|n|,c−2n},
// HRR in registers per (set = lane, c) in place in TC, then one warp per set stores / digests the finished shell-set.
template <int LX, int LA, int LB, int MODE, int NW, bool DEFER = false>
__device__ __forceinline__ void chain_epilogue(double *__restrict__ TC, const double *__restrict__ UB,
                                               const PartnerTab *__restrict__ pt, int warp, int lane,
                                               long long batch, const SetMap &map, const DevShells &aux,
                                               const DevShells &prim, double *__restrict__ out, int swapped, const DfArgs &df,
                                               const SetId &sid) {
    using CC = ChainCls<LX, LA, LB>;
    constexpr int E = CC::E, NACC = CC::NACC, NXC = CC::NXC, NA = CC::NA, NB = CC::NB, NAB = CC::NAB;
    constexpr int NINT = CC::NINT, SLOTN = CC::SLOTN;
    constexpr unsigned FULL = 0xffffffffu;
    // sid: the lane's shell-set (the caller has decoded it: a second search of the prefix map per batch is a second chain of
    // dependent global loads).  A mirrored class (caller's order [c][b][a]) gets its shell-sets transposed by the HRR stores, not by the copy-out
    const bool tr = MODE == 0 && swapped != 0;
    if constexpr (LB > 0 || LX >= 2) {
        double AB[3];
#pragma unroll
        for (int d = 0; d < 3; ++d) AB[d] = prim.center[3 * sid.a + d] - prim.center[3 * sid.b + d];
        for (int c = warp; c < NXC; c += NW) {               // run-time c: one copy of the code
            {
                double *reg = TC + (size_t)lane * SLOTN + c * NAB;
                double H0[NACC];
                static_for<0, NACC>([&](auto ii) { H0[decltype(ii)::value] = reg[decltype(ii)::value]; });
                if constexpr (LX >= 2) {
                    const int np_ = pt->cnt[c];
#pragma unroll 1
                    for (int k = 0; k < np_; ++k) {
                        const double beta = (double)pt->beta[c][k];
                        const double *ub = UB + (size_t)(pt->ti[c][k] - NXC) * NACC * 32 + lane;
                        static_for<0, NACC>([&](auto ii) {
                            constexpr int i = decltype(ii)::value;
                            H0[i] = fma(beta, ub[i * 32], H0[i]);
                        });
                    }
                }
                hrr_store<LA, LB>(H0, AB, reg, tr);
            }
        }
        __syncthreads();
    }
    // a8 (DEFER: the caller copies the batch out later, overlapped with the start of the next batch)
    if constexpr (MODE == 0 && !DEFER) batch_copy_out<NINT, SLOTN>(TC, out, batch, map.nsets, warp * 32 + lane, NW * 32);
    // a9 / a10: LANE = shell-set here too, so all 32 sets of the batch are digested at once
    if constexpr (MODE == 1) {
        // γ[bf(X)+c] += f Σ_ab (c|ab) D[bf(a)+ia, bf(b)+ib]: a lane sums its own set (the lanes of a batch mostly share the
        // pair, so the D block is a broadcast load) and adds into its own γ entries; the warps split c
        if (sid.live) {
            const double *Dab = df.D + (size_t)prim.bf_off[sid.a] * df.ld + prim.bf_off[sid.b];
            const double f = (sid.a != sid.b) ? 2.0 : 1.0;
            double *gx = df.out + aux.bf_off[sid.x];
            const double *FINl = TC + (size_t)lane * SLOTN;
            for (int c = warp; c < NXC; c += NW) {
                const double *Fc = FINl + c * NAB;
                double sum = 0.0;
                for (int ia = 0; ia < NA; ++ia)
#pragma unroll
                    for (int ib = 0; ib < NB; ++ib) sum = fma(Fc[ia * NB + ib], __ldg(Dab + (size_t)ia * df.ld + ib), sum);
                atomicAdd(gx + c, f * sum);
            }
        }
    } else if constexpr (MODE == 2) {
        // J[bf(a)+ia, bf(b)+ib] += Σ_X Σ_c (c|ab) d[bf(X)+c], mirrored: a lane contracts its own set with its d block, the
        // lanes that share a shell pair (contiguous runs of the batch) are summed by shuffles, one atomic per run and element
        const double *dx = df.D + aux.bf_off[sid.x];
        const double *FINl = TC + (size_t)lane * SLOTN;
        const unsigned livemask = __ballot_sync(FULL, sid.live);
        for (int r = warp; r < NAB; r += NW) {
            double v = 0.0;
            if (sid.live) {
#pragma unroll
                for (int c = 0; c < NXC; ++c) v = fma(FINl[c * NAB + r], __ldg(dx + c), v);
            }
            const int ia = r / NB, ib = r - ia * NB;
            unsigned rest = livemask;
            while (rest) {                                    // warp-uniform loop over the runs of equal pairs
                const int leader = __ffs(rest) - 1;
                const int pl = __shfl_sync(FULL, sid.p, leader);
                const unsigned grp = __ballot_sync(FULL, sid.live && sid.p == pl) & rest;
                double sum = (grp >> lane) & 1u ? v : 0.0;
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) sum += __shfl_xor_sync(FULL, sum, o);
                if (lane == leader) {
                    const size_t ra0 = prim.bf_off[sid.a], rb0 = prim.bf_off[sid.b];
                    atomicAdd(df.out + (ra0 + ia) * df.ld + rb0 + ib, sum);
                    if (sid.a != sid.b) atomicAdd(df.out + (rb0 + ib) * df.ld + ra0 + ia, sum);
                }
                rest &= ~grp;
            }
        }
    }
    __syncthreads();
}


// MODE 3 — solid-harmonic aux functions, fused (HGPA step 5).  For a pure ket the
// two-term relation eq. 2 is exact after projection: only the level-0 targets G_c = (Π B^c Z^{(Lx)}) are
// evaluated, and (X_m|e0) = Σ_c S_l[m][c] G_c with the real solid harmonics S_lm (lx.h, lx_cart_to_pure).  Per (set = lane,
// m): transform, HRR in registers, store into the pure region PR [set][m][a][b]; then the batch leaves coalesced.
template <int LX, int LA, int LB, int NW, int CSTR = ChainCls<LX, LA, LB>::NAB, int SLOT = ChainCls<LX, LA, LB>::SLOTN>
__device__ __forceinline__ void pure_epilogue(const double *__restrict__ TC, double *__restrict__ PR,
                                              const double *__restrict__ smat, int warp, int lane, long long batch,
                                              const SetMap &map, const DevShells &prim, double *__restrict__ out, int swapped) {
    using CC = ChainCls<LX, LA, LB>;
    constexpr int NACC = CC::NACC, NXC = CC::NXC, NAB = CC::NAB;
    constexpr int NP = 2 * LX + 1, NINTP = NP * NAB, SLOTP = NINTP | 1;
    const SetId sid = decode_set(map, batch * 32 + lane, swapped);
    double AB[3];
#pragma unroll
    for (int d = 0; d < 3; ++d) AB[d] = prim.center[3 * sid.a + d] - prim.center[3 * sid.b + d];
    const bool tr = swapped != 0;
    for (int m = warp; m < NP; m += NW) {
        double H0[NACC];
#pragma unroll
        for (int i = 0; i < NACC; ++i) H0[i] = 0.0;
        // unrolled over c: the loads of different c are independent (a rolled loop is bound by their latency); about three
        // quarters of S_l[m][·] are zeros and skipped by a warp-uniform branch
        const double *srow = smat + m * NXC;
        const double *src0 = TC + (size_t)lane * SLOT;
        static_for<0, NXC>([&](auto ic) {
            constexpr int c = decltype(ic)::value;
            const double sc = __ldg(srow + c);                    // warp-uniform
            if (sc != 0.0)
                static_for<0, NACC>([&](auto ii) { H0[decltype(ii)::value] = fma(sc, src0[c * CSTR + decltype(ii)::value], H0[decltype(ii)::value]); });
        });
        hrr_store<LA, LB>(H0, AB, PR + (size_t)lane * SLOTP + m * NAB, tr);
    }
    __syncthreads();
    batch_copy_out<NINTP, SLOTP>(PR, out, batch, map.nsets, warp * 32 + lane, NW * 32);
    __syncthreads();
}

// (e0|c)[i] = a_i! ( U_{0,c} + Σ_{n>0} β(c,n) U_{|n|,c−2n} )[i] from the accumulators of a lane that holds ALL targets of the class
// (W = 1): the gather of chain_epilogue with the partner list resolved at compile time.
template <int LX, int LA, int LB, int C_>
__device__ __forceinline__ void e0c_from_acc(const double *__restrict__ acc, double (&H0)[ChainCls<LX, LA, LB>::NACC]) {
    constexpr int NACC = ChainCls<LX, LA, LB>::NACC, gc = off(LX) + C_;
    constexpr int cx = cart_pow(gc, 0), cy = cart_pow(gc, 1), cz = cart_pow(gc, 2);
    static_for<0, NACC>([&](auto ii) { H0[decltype(ii)::value] = acc[C_ * NACC + decltype(ii)::value]; });
    static_for<0, (cx / 2 + 1) * (cy / 2 + 1) * (cz / 2 + 1)>([&](auto in) {
        constexpr int q = decltype(in)::value;
        constexpr int nz = q % (cz / 2 + 1), ny = (q / (cz / 2 + 1)) % (cy / 2 + 1), nx = q / ((cz / 2 + 1) * (cy / 2 + 1));
        if constexpr (nx + ny + nz > 0) {
            constexpr int ti = target_index(LX, nx + ny + nz, cart_index(cx - 2 * nx, cy - 2 * ny, cz - 2 * nz));
            constexpr double beta = (double)(beta1(cx, nx) * beta1(cy, ny) * beta1(cz, nz));
            static_for<0, NACC>([&](auto ii) { H0[decltype(ii)::value] = fma(beta, acc[ti * NACC + decltype(ii)::value], H0[decltype(ii)::value]); });
        }
    });
    static_for<0, NACC>([&](auto ii) { H0[decltype(ii)::value] *= (double)cart_fact(off(LA) + decltype(ii)::value); });
}

#ifndef LX_DIRECT_MAXLX
#define LX_DIRECT_MAXLX 4
#endif
// Digestion straight from the registers of a solo team (W = 1): gather and HRR (a7, eq. 1) per ket
// component on the lane's accumulators, then a9 / a10 as in chain_epilogue — without the trip of the targets and the finished
// shell-set through shared memory and without the three block barriers.  For the short batches of the low-L, weakly contracted DF
// classes that trip is a quarter of the instructions of a batch (config 5 DF-J 1.97 -> 1.87 s, config 4 9.0 -> 8.2 ms; the same
// (3|10) launch 4.47 -> 3.92 ms, profiles/r02_ncu_team_df.md).
template <int LX, int LA, int LB, int MODE>
__device__ __forceinline__ void direct_digest(const double *__restrict__ acc, const SetId &sid, int lane,
                                              const DevShells &aux, const DevShells &prim, const DfArgs &df) {
    using CC = ChainCls<LX, LA, LB>;
    constexpr int NACC = CC::NACC, NXC = CC::NXC, NA = CC::NA, NB = CC::NB, NAB = CC::NAB;
    constexpr unsigned FULL = 0xffffffffu;
    static_assert(MODE == 1 || MODE == 2, "DF modes");
    double AB[3];
#pragma unroll
    for (int d = 0; d < 3; ++d) AB[d] = prim.center[3 * sid.a + d] - prim.center[3 * sid.b + d];
    if constexpr (MODE == 1) {
        // γ[bf(X)+c] += f Σ_ab (c|ab) D[bf(a)+ia, bf(b)+ib]
        const double *Dab = df.D + (size_t)prim.bf_off[sid.a] * df.ld + prim.bf_off[sid.b];
        const double f = (sid.a != sid.b) ? 2.0 : 1.0;
        double *gx = df.out + aux.bf_off[sid.x];
        static_for<0, NXC>([&](auto ic) {
            constexpr int c = decltype(ic)::value;
            double H0[NACC], fin[NAB];
            e0c_from_acc<LX, LA, LB, c>(acc, H0);
            hrr_store<LA, LB>(H0, AB, fin, false);
            double sum = 0.0;
            static_for<0, NA>([&](auto ia) {
                static_for<0, NB>([&](auto ib) {
                    sum = fma(fin[decltype(ia)::value * NB + decltype(ib)::value], __ldg(Dab + (size_t)decltype(ia)::value * df.ld + decltype(ib)::value), sum);
                });
            });
            if (sid.live) atomicAdd(gx + c, f * sum);
        });
    } else {
        // J[bf(a)+ia, bf(b)+ib] += Σ_X Σ_c (c|ab) d[bf(X)+c], mirrored: v[r] of the lane's set in registers, the lanes that share a
        // shell pair (contiguous runs of the batch) summed by shuffles, one atomic per run and element
        const double *dx = df.D + aux.bf_off[sid.x];
        double v[NAB];
#pragma unroll
        for (int r = 0; r < NAB; ++r) v[r] = 0.0;
        static_for<0, NXC>([&](auto ic) {
            constexpr int c = decltype(ic)::value;
            double H0[NACC], fin[NAB];
            e0c_from_acc<LX, LA, LB, c>(acc, H0);
            hrr_store<LA, LB>(H0, AB, fin, false);
            const double dc = sid.live ? __ldg(dx + c) : 0.0;
            static_for<0, NAB>([&](auto ir) { v[decltype(ir)::value] = fma(fin[decltype(ir)::value], dc, v[decltype(ir)::value]); });
        });
        unsigned rest = __ballot_sync(FULL, sid.live);
        while (rest) {                                        // warp-uniform loop over the runs of equal pairs
            const int leader = __ffs(rest) - 1;
            const int pl = __shfl_sync(FULL, sid.p, leader);
            const unsigned grp = __ballot_sync(FULL, sid.live && sid.p == pl) & rest;
            const bool in = (grp >> lane) & 1u;
            const size_t ra0 = prim.bf_off[sid.a], rb0 = prim.bf_off[sid.b];
            static_for<0, NAB>([&](auto ir) {
                constexpr int r = decltype(ir)::value, ia = r / NB, ib = r - ia * NB;
                double sum = in ? v[r] : 0.0;
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) sum += __shfl_xor_sync(FULL, sum, o);
                if (lane == leader) {
                    atomicAdd(df.out + (ra0 + ia) * df.ld + rb0 + ib, sum);
                    if (sid.a != sid.b) atomicAdd(df.out + (rb0 + ib) * df.ld + ra0 + ia, sum);
                }
            });
            rest &= ~grp;
        }
    }
}

// ---- team plan: W warps, warp w owns the targets [w·NTW, (w+1)·NTW) (ordered by level) ------------------------------------
template <int LX, int LA, int LB, int W>
struct TeamCls {
    using CC = ChainCls<LX, LA, LB>;
    static constexpr int NT = CC::T.n, NTW = (NT + W - 1) / W;
    static constexpr int NUB = (NT - CC::NXC) * CC::NACC * 32;            // staging of the levels p >= 1
    static constexpr size_t smem = ((size_t)32 * CC::SLOTN + NUB + 4) * 8 + sizeof(PartnerTab);
    static constexpr int acc_doubles = NTW * CC::NACC;                   // accumulators a lane keeps
};
// smallest team whose lanes keep at most `budget` accumulator doubles (0 = none fits in 8 warps)
__host__ __device__ constexpr int team_size(int LX, int LA, int LB, int budget) {
    const int NACC = off(LA + LB + 1) - off(LA);
    int NT = 0;
    for (int p = 0; 2 * p <= LX; ++p) NT += nc(LX - 2 * p);
    for (int w = 1; w <= 8; ++w)
        if (((NT + w - 1) / w) * NACC <= budget) return w;
    return 0;
}

template <int LX, int LA, int LB, int MODE, int W, int MINB>
__global__ void __launch_bounds__(W * 32, MINB)
team_kernel(SetMap map, DevShells aux, DevShells prim, PairData pdat, const double *__restrict__ boys_tab,
            double *__restrict__ out, int swapped, DfArgs df) {
    using CC = ChainCls<LX, LA, LB>;
    using TM = TeamCls<LX, LA, LB, W>;
    // MODE 3 (pure aux functions) needs the level-0 targets only
    constexpr int E = CC::E, NG = CC::NG, NACC = CC::NACC, NT = MODE == 3 ? CC::NXC : TM::NT, NTW = (NT + W - 1) / W;
    constexpr int NUBX = MODE == 3 ? cmax(TM::NUB, 32 * (((2 * LX + 1) * CC::NAB) | 1)) : TM::NUB;   // staging / pure region
    constexpr unsigned FULL = 0xffffffffu;
    // solo teams digest from registers in the DF modes (direct_digest)
    constexpr bool DIRECT = W == 1 && LX <= LX_DIRECT_MAXLX && (MODE == 1 || MODE == 2);

    extern __shared__ double smem[];
    double *TC = smem;                                       // [set][c * NAB + ·]
    double *UB = TC + (size_t)32 * CC::SLOTN;                // [(ti − NXC)][i][set]
    PartnerTab *pt = reinterpret_cast<PartnerTab *>(UB + NUBX + 4);
    if (threadIdx.x == 0) partner_tab_build<LX>(pt);
    __syncthreads();

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const long long nbatch = (map.nsets + 31) / 32;

    for (long long batch = blockIdx.x; batch < nbatch; batch += gridDim.x) {
        const SetId sid = decode_set(map, batch * 32 + lane, swapped);
        const int Kab = min(prim.K[sid.a] * prim.K[sid.b], pdat.kstride);
        const int K = sid.live ? Kab * aux.K[sid.x] : 0;
        const int kmax = __reduce_max_sync(FULL, K);
        const double A[3] = {prim.center[3 * sid.a], prim.center[3 * sid.a + 1], prim.center[3 * sid.a + 2]};
        const double C[3] = {aux.center[3 * sid.x], aux.center[3 * sid.x + 1], aux.center[3 * sid.x + 2]};
        const long long po = pdat.pd_off ? pdat.pd_off[sid.p] : (long long)sid.p * pdat.kstride;
        const int xo0 = aux.prim_off[sid.x];

        static_for<0, W>([&](auto iw) {
            constexpr int w = decltype(iw)::value;
            constexpr int T0 = w * NTW, T1 = cmin(NT, (w + 1) * NTW);
            if constexpr (T1 > T0) {
                if (W == 1 || warp == w) {
                    constexpr int PLO = CC::T.p[T0], PHI = CC::T.p[T1 - 1];
                    constexpr int MLO = LX - 2 * PHI, MHI = LX - PLO + E;
                    double acc[(T1 - T0) * NACC];
#pragma unroll
                    for (int i = 0; i < (T1 - T0) * NACC; ++i) acc[i] = 0.0;
                    // software pipeline: the prefactors and Boys values of primitive q+1 are evaluated next to the chains
                    // of primitive q (independent instruction streams in one basic block)
                    int kx = 0, ij = 0;
                    double zc = 1.0, cxc = 0.0;
                    auto fetch = [&](int q, PrimRec &R, double (&F)[MHI - MLO + 1]) {
                        const bool on = q < K;
                        if (ij == 0) {
                            zc = aux.zeta[xo0 + (on ? kx : 0)];
                            cxc = aux.coef[xo0 + (on ? kx : 0)];
                        }
                        R = prim_rec(pdat.pd + (po + (on ? ij : 0)) * PD_STRIDE, zc, on ? cxc : 0.0, A, C);
                        if (++ij == Kab) { ij = 0; ++kx; }
                        boys_range<MLO, MHI>(boys_tab, R.T, F);
                    };
                    PrimRec R;
                    double F[MHI - MLO + 1];
                    fetch(0, R, F);
                    for (int q = 0; q < kmax; ++q) {
                        PrimRec Rn;
                        double Fn[MHI - MLO + 1];
                        fetch(q + 1, Rn, Fn);
                        static_for<PLO, PHI + 1>([&](auto ip) {
                            constexpr int p = decltype(ip)::value;
                            double u[NG];
                            vrr1_level<LX, E, p, MLO>(R, F, u);
                            const double ck = level_scale<LX - 2 * p, p>(R);
                            static_for<T0, T1>([&](auto it) {
                                constexpr int ti = decltype(it)::value;
                                if constexpr (CC::T.p[ti] == p) {
                                    constexpr int tg = CC::T.g[ti];
                                    chain_apply_reg<LA, E, cart_pow(tg, 0), cart_pow(tg, 1), cart_pow(tg, 2)>(u, R.r, ck, acc + (ti - T0) * NACC);
                                }
                            });
                        });
                        R = Rn;
#pragma unroll
                        for (int m = 0; m <= MHI - MLO; ++m) F[m] = Fn[m];
                    }
                    if constexpr (DIRECT) {
                        direct_digest<LX, LA, LB, MODE>(acc, sid, lane, aux, prim, df);
                    } else {
                        static_for<T0, T1>([&](auto it) {
                            constexpr int ti = decltype(it)::value;
                            target_drop<LX, LA, LB>(ti, acc + (ti - T0) * NACC, TC, UB, lane);
                        });
                    }
                }
            }
        });
        if constexpr (DIRECT) continue;                      // digested from registers: nothing went through shared memory
        __syncthreads();
        if constexpr (MODE == 3) pure_epilogue<LX, LA, LB, W>(TC, UB, df.D, warp, lane, batch, map, prim, out, swapped);
        else chain_epilogue<LX, LA, LB, MODE, W>(TC, UB, pt, warp, lane, batch, map, aux, prim, out, swapped, df, sid);
    }
}

template <int LX, int LA, int LB, int MODE, int W>
cudaError_t team_launch(const SetMap &map, const DevShells &aux, const DevShells &prim, const PairData &pdat,
                        const double *boys_tab, double *out, int swapped, const DfArgs &df, int num_sms,
                        cudaStream_t stream) {
    using TM = TeamCls<LX, LA, LB, W>;
    constexpr int NUBX = MODE == 3 ? cmax(TM::NUB, 32 * (((2 * LX + 1) * TM::CC::NAB) | 1)) : TM::NUB;
    constexpr size_t smem = ((size_t)32 * TM::CC::SLOTN + NUBX + 4) * 8 + sizeof(PartnerTab);
    static_assert(smem <= 227 * 1024, "team kernel: batch does not fit in shared memory");
    // registers: accumulators + start vector + chain copy (doubles), two primitive records, Boys values, scalars
    constexpr int need = 2 * (TM::acc_doubles + 2 * TM::CC::NG) + 110;
    constexpr int regs = need <= 64 ? 64 : (need <= 96 ? 96 : (need <= 128 ? 128 : (need <= 168 ? 168 : 255)));
    constexpr int by_smem = (int)((227 * 1024) / (smem + 1024));
    constexpr int by_regs = 65536 / (W * 32 * regs);
    constexpr int BPS = cmax(1, cmin(cmin(by_smem, by_regs), 32));
    auto kern = team_kernel<LX, LA, LB, MODE, W, BPS>;
    static std::atomic<unsigned long long> configured{0};
    if (cudaError_t e = ensure_dyn_smem(kern, smem, configured); e != cudaSuccess) return e;
    if (map.nsets <= 0) return cudaSuccess;
    long long blocks = (map.nsets + 31) / 32;
    const long long cap = (long long)num_sms * BPS;
    if (blocks > cap) blocks = cap;
    kern<<<(unsigned)blocks, W * 32, smem, stream>>>(map, aux, prim, pdat, boys_tab, out, swapped, df);
    return cudaGetLastError();
}

}  // namespace lx
