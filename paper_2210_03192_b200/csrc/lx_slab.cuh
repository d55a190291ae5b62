// lx_slab.cuh — "slab kernel": the owner scheme of lx_owner.cuh for La+Lb = 6, where a lane can hold the start vector (84
// doubles) but not the accumulator next to it, and where the HRR (Lb = 3, or 64 inputs for (x|42)) no longer fits registers.
//
// LANE = shell-set, one owner warp per ket component c as in lx_owner.cuh.  The bra components (all shells 0..E, E = La+Lb)
// are kept in SLAB-MAJOR order: slab s holds the components with a_x = s, a triangle of the in-slab powers (a_y, a_z),
// a_y + a_z <= E − s.
//   a3  VRR1 (eq. 3) as three nested ONE-dimensional pyramids — raising one axis needs no other axis:
//       the x line [s00]^(m), from row s the y line [s a_y 0]^(m), from each of its rows the z line [s a_y a_z]^(m) — so a
//       work item (level p, slab s) is independent of every other item and needs no shared memory but for its result;
//   a4  the chains Π B_i^{t_i} (lx_chain.cuh) run on the whole vector in the owner's registers, one read of the start vector
//       per partner; the sum over partners and primitives (a5) is kept in the owner's (e0|c) region in shared memory;
//   a7  the HRR (eq. 1) one slab of rows a_x = S at a time: the x part of b by its closed form
//       Σ_k C(b_x,k) AB_x^{b_x−k} (e0|c)[s+k] (loads of the slabs S..S+b_x), the y and z parts as up-shifting steps in registers;
//   a8  the finished rows of a shell-set leave through a small staging slot as coalesced runs (a9: contracted with D there;
//       a10: d_c is contracted BEFORE the HRR, which then runs once per batch).
// All loops over ket components, partners and steps are run-time loops around compile-time bodies: the code stays in the
// instruction cache (lx_owner.cuh explains why that matters for K = 1 classes).
// A first version cut the chains into slabs as well (x steps by the closed form (B_x^t u)[s] = Σ_j C(t,j) r_x^{t−j} u[s−j] from
// shared memory, teams of two warps per component): 15.3 ms for (6|33) against 14.4 ms now, 10.1 against 7.7 ms for (5|33);
// La+Lb = 5 moved to the owner kernel altogether (8 warps of 255 registers: 3–5× faster than either slab form).
#pragma once
#include "lx_owner.cuh"

namespace lx {

#ifndef LX_SLAB_MINW32
#define LX_SLAB_MINW32 4
#endif
#ifndef LX_SLAB_TEAM
#define LX_SLAB_TEAM 1
#endif
__host__ __device__ constexpr int tsz(int n) { return n * (n + 1) / 2; }                 // components of a triangle of size n
// slab-major component order of the bra vector (shells 0..E): slab s = a_x, inside by d = a_y + a_z, then a_z
__host__ __device__ constexpr int slab_off(int E, int s) { int o = 0; for (int q = 0; q < s; ++q) o += tsz(E - q + 1); return o; }
// the same restricted to the shells >= LA (the contracted (e0|c)): slab s keeps the degrees d >= max(0, LA − s)
__host__ __device__ constexpr int slab_dmin(int LA, int s) { return LA > s ? LA - s : 0; }
__host__ __device__ constexpr int e0_cnt(int E, int LA, int s) { return tsz(E - s + 1) - tsz(slab_dmin(LA, s)); }
__host__ __device__ constexpr int e0_off(int E, int LA, int s) { int o = 0; for (int q = 0; q < s; ++q) o += e0_cnt(E, LA, q); return o; }

template <int LX, int LA, int LB>
struct SlabCls {
    static constexpr int E = LA + LB, NG = off(E + 1), NACC = NG - off(LA);
    static constexpr int NXC = nc(LX), NA = nc(LA), NB = nc(LB), NAB = NA * NB, NINT = NXC * NAB;
    static constexpr int NLEV = LX / 2 + 1;
    // per set and start-vector buffer: u[p][slab-major g], r_x^k (k = 0..LX), r_y, r_z, ck[p]
    static constexpr int O_RXP = NLEV * NG, O_RY = O_RXP + LX + 1, O_RZ = O_RY + 1, O_CK = O_RZ + 1;
    static constexpr int UREC = O_CK + NLEV;
    // staging of one finished slab of a shell-set: the rows a (a_x = s) x all b; the largest is s = 0
    static constexpr int STG = (LA + 1) * NB;
    // A TEAM of T warps owns a ket component and shares its (e0|c) region; T = 1 (one warp per component) since the chains
    // run on the whole vector in one warp's registers; with LX_SLAB_TEAM = 2 the second warp only takes HRR rows (tuning knob).
    // Each warp has its own staging slot.  Sets per batch: 32 where that leaves room for LX_SLAB_MINW32 warps, else 16 (lanes
    // 16..31 mirror 0..15).
    static constexpr int T = LX_SLAB_TEAM;
    static constexpr int per_team32 = (NACC + T * (STG | 1)) * 32 * 8, fixed32 = UREC * 32 * 8;
    static constexpr int NS = T * ((220 * 1024 - fixed32) / per_team32) >= LX_SLAB_MINW32 ? 32 : 16;
    static constexpr int per_team = (NACC + T * (STG | 1)) * NS * 8, fixed = UREC * NS * 8;
    static constexpr int NTEAM = cmax(1, cmin(8 / T, (220 * 1024 - fixed) / per_team));
    static constexpr int NW = NTEAM * T;
    static constexpr size_t smem = (size_t)fixed + (size_t)NTEAM * per_team + 2 * sizeof(OwnHdr) + 128;
};

// One-dimensional VRR1 pyramid (eq. 3 along one axis): in[OFF + m] = f_0^(m), m = 0..K−1; out row j (offset j·K − j(j−1)/2) holds
// f_j^(m), m = 0..K−1−j, with f_{j+1}^(m) = PA f_j^(m) + WP f_j^(m+1) + j/(2γ) (f_{j−1}^(m) − (ρ/γ) f_{j−1}^(m+1)).
template <int K, int OFF, int NIN>
__device__ __forceinline__ void line_pyramid(const double (&in)[NIN], double PAi, double WPi, double o2g, double mrg,
                                             double (&out)[tsz(K)]) {
    static_for<0, K>([&](auto im) { out[decltype(im)::value] = in[OFF + decltype(im)::value]; });
    static_for<1, K>([&](auto ij) {
        constexpr int j = decltype(ij)::value, r1 = (j - 1) * K - (j - 1) * (j - 2) / 2, r0 = j * K - j * (j - 1) / 2;
        static_for<0, K - j>([&](auto im) {
            constexpr int m = decltype(im)::value;
            double v = fma(WPi, out[r1 + m + 1], PAi * out[r1 + m]);
            if constexpr (j > 1) {
                constexpr int r2 = (j - 2) * K - (j - 2) * (j - 3) / 2;
                v = fma((double)(j - 1) * o2g, fma(mrg, out[r2 + m + 1], out[r2 + m]), v);
            }
            out[r0 + m] = v;
        });
    });
}

// a3 for one work item (level p: run time, slab S: compile time) of the lane's set: u[S; a_y, a_z] = Y_p[a] / a!.
template <int LX, int E, int S, int NSs>
__device__ __noinline__ void slab_produce(int p, const PrimRec &R, const double *__restrict__ boys_tab,
                                             double *__restrict__ ub, int ls) {
    constexpr int n = E - S + 1, NG = off(E + 1);
    // W^(m) = pref Σ_s C(p,s) (−ρ/ζc)^s F_{LX−2p+m+s}(T), m = 0..E   (lx_chain.cuh header: Y_p = Δ^p Z^{(LX−2p)})
    double W[E + 1];
    static_for<0, LX / 2 + 1>([&](auto ip) {
        constexpr int P_ = decltype(ip)::value;
        if (p == P_) {
            constexpr int MLO = LX - 2 * P_, MHI = LX - P_ + E;
            double F[MHI - MLO + 1];
            boys_range<MLO, MHI>(boys_tab, R.T, F);
            static_for<0, E + 1>([&](auto im) {
                constexpr int m = decltype(im)::value;
                double w = F[m + P_];
                static_for<0, P_>([&](auto is) {
                    constexpr int s = P_ - 1 - decltype(is)::value;
                    w = fma(w, R.mrz, (double)ibinom(P_, s) * F[m + s]);
                });
                W[m] = R.pref * w;
            });
        }
    });
    // x line up to power S: only its row S is needed
    double row[n];
    if constexpr (S == 0) {
        static_for<0, n>([&](auto im) { row[decltype(im)::value] = W[decltype(im)::value]; });
    } else {
        // rows 0..S of the x pyramid; row j has E+1−j entries.  Rolling: keep two rows.
        double a[E + 1], b[E + 1];
        static_for<0, E + 1>([&](auto im) { a[decltype(im)::value] = W[decltype(im)::value]; });
        static_for<0, E>([&](auto im) {
            constexpr int m = decltype(im)::value;
            b[m] = fma(R.WP[0], a[m + 1], R.PA[0] * a[m]);
        });
        static_for<2, S + 1>([&](auto ij) {
            constexpr int j = decltype(ij)::value;               // new row j from rows j−1 (b) and j−2 (a)
            static_for<0, E + 1 - j>([&](auto im) {
                constexpr int m = decltype(im)::value;
                const double v = fma((double)(j - 1) * R.o2g, fma(R.mrg, a[m + 1], a[m]), fma(R.WP[0], b[m + 1], R.PA[0] * b[m]));
                a[m] = b[m];
                b[m] = v;
            });
            a[E + 1 - j] = b[E + 1 - j];
        });
        static_for<0, n>([&](auto im) { row[decltype(im)::value] = b[decltype(im)::value]; });
    }
    // y line inside the slab, then one z line per a_y
    double Y[tsz(n)];
    line_pyramid<n, 0, n>(row, R.PA[1], R.WP[1], R.o2g, R.mrg, Y);
    constexpr double invS = 1.0 / (double)ifact(S);
    double *us = ub + (size_t)(p * NG + slab_off(E, S)) * NSs + ls;
    static_for<0, n>([&](auto iy) {
        constexpr int ay = decltype(iy)::value, k = n - ay, ry = ay * n - ay * (ay - 1) / 2;
        double Z[tsz(k)];
        line_pyramid<k, ry, tsz(n)>(Y, R.PA[2], R.WP[2], R.o2g, R.mrg, Z);
        static_for<0, k>([&](auto iz) {
            constexpr int az = decltype(iz)::value, rz = az * k - az * (az - 1) / 2;
            constexpr double inv = invS / ((double)ifact(ay) * (double)ifact(az));
            us[(size_t)(tsz(ay + az) + az) * NSs] = Z[rz] * inv;
        });
    });
}

// ---- chains on the WHOLE bra vector in registers (La+Lb = 6: 84 doubles, 168 registers) -----------------------------------
// Where one lane can hold the whole start vector — it cannot hold the accumulator as well — the chains run as in the owner
// kernel (lx_owner.cuh: every step in registers, one read of the start vector per partner, no closed-form x part with its
// repeated loads) and only the sum over the partners goes through shared memory, into the owner's slab-major (e0|c) region.
// Measured (B200, config 3): (6|33) 15.3 -> see DESIGN.md section 10.
template <int E, int AXIS>
__device__ __forceinline__ void whole_step(double (&z)[off(E + 1)], double r) {
    // descending total degree t = s + d: the source a − 1_axis (degree t − 1) is still un-stepped when a is
    static_for<0, E + 1>([&](auto it) {
        constexpr int t = E - decltype(it)::value;
        static_for<0, t + 1>([&](auto is) {
            constexpr int sx = decltype(is)::value, d = t - sx;           // slab sx, in-slab degree d
            static_for<0, d + 1>([&](auto iq) {
                constexpr int q = decltype(iq)::value, i = slab_off(E, sx) + tsz(d) + q;
                constexpr bool has = AXIS == 0 ? sx > 0 : (AXIS == 1 ? d - q > 0 : q > 0);
                if constexpr (has) {
                    constexpr int lo = AXIS == 0 ? slab_off(E, sx - 1) + tsz(d) + q
                                                 : slab_off(E, sx) + tsz(d - 1) + (AXIS == 1 ? q : q - 1);
                    z[i] = fma(r, z[i], z[lo]);
                } else {
                    z[i] = r * z[i];
                }
            });
        });
    });
}

template <int LX, int LA, int LB>
__device__ __noinline__ void slab_chains_whole(int cx, int cy, int cz, const double *__restrict__ ub, int kprim,
                                               double *__restrict__ e0w, int ls, bool add, double scale) {
    using SC = SlabCls<LX, LA, LB>;
    constexpr int E = SC::E, NG = SC::NG, NS = SC::NS;
    auto grow = [](int ci, int ni) { return (double)((ci - 2 * ni) * (ci - 2 * ni - 1)) * (ni == 0 ? 0.5 : (ni == 1 ? 0.25 : 1.0 / 6.0)); };
    bool fresh = !add;                                           // the first partner stores, the others add
#pragma unroll 1
    for (int q = 0; q < kprim; ++q) {
        const double *uq = ub + (size_t)q * SC::UREC * NS + ls;
        const double rx = uq[(size_t)(SC::O_RXP + 1) * NS], ry = uq[SC::O_RY * NS], rz = uq[SC::O_RZ * NS];
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
                    const double *up = uq + (size_t)p * NG * NS;
                    double z[NG];
                    static_for<0, NG>([&](auto ig) { z[decltype(ig)::value] = up[(size_t)decltype(ig)::value * NS]; });
#pragma unroll 1
                    for (int k = cx - 2 * nx; k > 0; --k) whole_step<E, 0>(z, rx);
#pragma unroll 1
                    for (int k = cy - 2 * ny; k > 0; --k) whole_step<E, 1>(z, ry);
#pragma unroll 1
                    for (int k = cz - 2 * nz; k > 0; --k) whole_step<E, 2>(z, rz);
                    const double ck = beta * uq[(size_t)(SC::O_CK + p) * NS];
                    // acc (shared memory, slab-major, shells >= LA, back in the f = u a! basis) += ck z
                    static_for<0, E + 1>([&](auto is) {
                        constexpr int sx = decltype(is)::value, n = E - sx + 1, DMIN = slab_dmin(LA, sx), T0 = tsz(DMIN);
                        double *dst = e0w + (size_t)(e0_off(E, LA, sx) - T0) * NS + ls;
                        static_for<DMIN, n>([&](auto id) {
                            constexpr int d = decltype(id)::value;
                            static_for<0, d + 1>([&](auto iq) {
                                constexpr int qq = decltype(iq)::value, i = tsz(d) + qq;
                                constexpr double f = (double)ifact(sx) * (double)ifact(d - qq) * (double)ifact(qq);
                                const double v = (ck * f) * z[slab_off(E, sx) + i];
                                if (fresh) dst[(size_t)i * NS] = v;
                                else dst[(size_t)i * NS] += v;
                            });
                        });
                    });
                    fresh = false;
                    beta *= grow(cz, nz);
                }
                bxy *= grow(cy, ny);
            }
            bx *= grow(cx, nx);
        }
    }
}

// a7 + a8 for the rows a with a_x = S of one ket component: (a b| = Σ_{k <= b} Π_i C(b_i,k_i) AB_i^{b_i−k_i} (a+k 0| (eq. 1
// unrolled).  The x part of b is summed from the slabs S..S+b_x of the warp's (e0|c) region; the y and z parts are
// up-shifting steps v[a] <- AB_i v[a] + v[a+1_i] on the band of in-slab degrees d0..d0+m (d0 = LA−S, m = LB−b_x) in
// registers.  The rows (all b) of the NS sets go to the staging slot and leave as one contiguous run per set.
// MODE 1 (a9): instead of the store the lane contracts its staged rows with the D block of its pair and returns the partial
// sum Σ_{a: a_x = S} Σ_b (c|ab) D_ab.  MODE 2 (a10): e0w holds Σ_c d_c (e0|c) of the batch; the staged rows are the lane's J
// contributions, which slab_j_reduce adds to J.
struct SlabDf { const OwnHdr *hd; const int32_t *bf_off; DfArgs df; };
template <int LX, int LA, int LB, int S, int MODE>
__device__ __noinline__ double slab_hrr(const double *__restrict__ e0w, double *__restrict__ stw, const double (&AB)[3],
                                        int c, int ls, int lane, long long batch, long long nsets,
                                        double *__restrict__ out, const int *__restrict__ trs, const SlabDf &sd) {
    using SC = SlabCls<LX, LA, LB>;
    constexpr int E = SC::E, NS = SC::NS, NA = SC::NA, NB = SC::NB, NAB = SC::NAB, NXC = SC::NXC;
    constexpr int D0 = LA - S, CH = (D0 + 1) * NB, SPS = SC::STG | 1;
    double abx[LB + 1];
    abx[0] = 1.0;
#pragma unroll
    for (int k = 1; k <= LB; ++k) abx[k] = abx[k - 1] * AB[0];
    double *strow = stw + (size_t)ls * SPS;
    const bool tr = trs[ls] != 0;                               // this lane's set is stored as [c][b][a]
    static_for<0, LB + 1>([&](auto ibx) {
        constexpr int BX = decltype(ibx)::value, M = LB - BX;
        constexpr int B0 = tsz(D0), NBAND = tsz(D0 + M + 1) - B0;          // band: degrees D0..D0+M
        double W[NBAND];
        static_for<0, BX + 1>([&](auto ik) {
            constexpr int k = decltype(ik)::value;
            constexpr int base = e0_off(E, LA, S + k) - tsz(slab_dmin(LA, S + k)) + B0;   // element (d, q) of the band in slab S+k
            const double w = (double)ibinom(BX, k) * abx[BX - k];
            const double *src = e0w + (size_t)base * NS + ls;
            static_for<0, NBAND>([&](auto ii) {
                constexpr int i = decltype(ii)::value;
                if constexpr (k == 0) W[i] = w * src[(size_t)i * NS];
                else W[i] = fma(w, src[(size_t)i * NS], W[i]);
            });
        });
        static_for<0, M + 1>([&](auto iby) {
            constexpr int BY = decltype(iby)::value, BZ = M - BY;
            double v[NBAND];
            static_for<0, NBAND>([&](auto ii) { v[decltype(ii)::value] = W[decltype(ii)::value]; });
            static_for<0, M>([&](auto ist) {
                constexpr int st = decltype(ist)::value;                  // step st lowers the top degree to D0+M−st−1
                constexpr int axis = st < BY ? 1 : 2;
                static_for<D0, D0 + M - st>([&](auto id) {
                    constexpr int d = decltype(id)::value;
                    static_for<0, d + 1>([&](auto iq) {
                        constexpr int q = decltype(iq)::value;
                        constexpr int i = tsz(d) + q - B0, up = tsz(d + 1) + (axis == 1 ? q : q + 1) - B0;
                        v[i] = fma(AB[axis], v[i], v[up]);
                    });
                });
            });
            constexpr int ib = tsz(M) + BZ;
            static_for<0, D0 + 1>([&](auto iq) {
                constexpr int q = decltype(iq)::value;                    // a = (S, D0−q, q): row tsz(D0)+q of shell LA
                if (tr) strow[ib * (D0 + 1) + q] = v[q];
                else strow[q * NB + ib] = v[q];
            });
        });
    });
    __syncwarp();
    if constexpr (MODE == 0) {
        // the staged rows of a set are one run of CH doubles in out[] (mirrored classes: NB runs of D0+1).  Lanes over the
        // elements of a run; short runs (CH <= 16) take 32/CH sets per trip.  No division inside the loops.
        const int nlive = (int)min((long long)NS, nsets - batch * NS);
        double *o = out + (batch * NS * NXC + c) * NAB;
        constexpr int SPT = CH <= 16 ? 32 / CH : 1;              // sets per trip
        constexpr int NIT = (CH + 31) / 32;                      // trips per set (SPT == 1)
        const int ds = SPT > 1 ? lane / CH : 0, i0 = SPT > 1 ? lane - ds * CH : lane;
        int doff_n[NIT], doff_t[NIT];                            // offset of element i0 + 32 k within the set's shell-set
#pragma unroll
        for (int k = 0; k < NIT; ++k) {
            const int i = i0 + 32 * k;
            doff_n[k] = tsz(D0) * NB + i;
            doff_t[k] = tsz(D0) + (i / (D0 + 1)) * NA + i % (D0 + 1);
        }
        const bool lane_on = SPT > 1 ? ds < SPT : true;
        const double *src = stw + (size_t)ds * SPS + i0;
        double *dst = o + (size_t)ds * (NXC * NAB);
#pragma unroll 1
        for (int s = ds; s < nlive; s += SPT) {
            if (lane_on) {
                const bool ts = trs[s] != 0;
#pragma unroll
                for (int k = 0; k < NIT; ++k)
                    if (i0 + 32 * k < CH) dst[ts ? doff_t[k] : doff_n[k]] = src[32 * k];
            }
            src += SPT * SPS;
            dst += (size_t)SPT * (NXC * NAB);
        }
    }
    double ret = 0.0;
    if constexpr (MODE == 1) {
        const OwnHdr *hd = sd.hd;
        if (hd->p[ls] >= 0) {
            const double *Dab = sd.df.D + (size_t)(sd.bf_off[hd->a[ls]] + tsz(D0)) * sd.df.ld + sd.bf_off[hd->b[ls]];
#pragma unroll 1
            for (int q = 0; q <= D0; ++q)
#pragma unroll
                for (int ib = 0; ib < NB; ++ib) ret = fma(strow[q * NB + ib], __ldg(Dab + (size_t)q * sd.df.ld + ib), ret);
        }
    }
    __syncwarp();
    return ret;
}

// a10, last step: the rows a_x = S staged by slab_hrr<.., 2> are the sets' J contributions; warp `w` of `nw` takes the elements
// i = w, w + nw, ..: the lanes that share a shell pair (contiguous runs of the batch) are summed by shuffles, one atomic per
// run and element (mirrored for a != b).
template <int LX, int LA, int LB, int S>
__device__ __forceinline__ void slab_j_reduce(const double *__restrict__ strow, int w, int nw, int ls, int lane, const SlabDf &sd) {
    using SC = SlabCls<LX, LA, LB>;
    constexpr int NS = SC::NS, NB = SC::NB, D0 = LA - S, CH = (D0 + 1) * NB;
    constexpr unsigned FULL = 0xffffffffu;
    const OwnHdr *hd = sd.hd;
    const int pl_own = lane < NS ? hd->p[ls] : -1;
    const bool live = pl_own >= 0;
    const unsigned livemask = __ballot_sync(FULL, live);
    const int sa = hd->a[ls], sb = hd->b[ls];
    const size_t ra0 = sd.bf_off[sa] + tsz(D0), rb0 = sd.bf_off[sb];
#pragma unroll 1
    for (int i = w; i < CH; i += nw) {
        const double v = live ? strow[i] : 0.0;
        const int q = i / NB, ib = i - q * NB;
        unsigned rest = livemask;
        while (rest) {                                          // warp-uniform loop over the runs of equal pairs
            const int leader = __ffs(rest) - 1;
            const int pl = __shfl_sync(FULL, pl_own, leader);
            const unsigned grp = __ballot_sync(FULL, live && pl_own == pl) & rest;
            double sum = (grp >> lane) & 1u ? v : 0.0;
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) sum += __shfl_xor_sync(FULL, sum, o);
            if (lane == leader) {
                atomicAdd(sd.df.out + (ra0 + q) * sd.df.ld + rb0 + ib, sum);
                if (sa != sb) atomicAdd(sd.df.out + (rb0 + ib) * sd.df.ld + ra0 + q, sum);
            }
            rest &= ~grp;
        }
    }
}

// Per-primitive scalars of the lane's set (as owner_produce) for primitive q of the batch in header h.
__device__ __forceinline__ PrimRec slab_prim(const OwnHdr *h, int q, int ls, const DevShells &aux, const PairData &pdat) {
    const double A[3] = {h->A[0][ls], h->A[1][ls], h->A[2][ls]};
    const double C[3] = {h->C[0][ls], h->C[1][ls], h->C[2][ls]};
    const int Kab = h->Kab[ls], K = h->K[ls], xo0 = h->xo0[ls];
    const bool on = q < K;
    const int qq = on ? q : 0;
    const int kx = qq / Kab, ij = qq - kx * Kab;
    const double zc = aux.zeta[xo0 + kx], cxc = on ? aux.coef[xo0 + kx] : 0.0;
    return prim_rec(pdat.pd + (h->po[ls] + ij) * PD_STRIDE, zc, cxc, A, C);
}

// producer work item `item` = (slab s, level p) of primitive q into buffer ub; item 0 also writes the scalars of the primitive
template <int LX, int LA, int LB>
__device__ __forceinline__ void slab_item(int item, int q, const OwnHdr *h, double *__restrict__ ub, int ls,
                                          const DevShells &aux, const PairData &pdat, const double *__restrict__ boys_tab) {
    using SC = SlabCls<LX, LA, LB>;
    constexpr int E = SC::E, NS = SC::NS, NLEV = SC::NLEV;
    const int s = item / NLEV, p = item - s * NLEV;
    const PrimRec R = slab_prim(h, q, ls, aux, pdat);
    static_for<0, E + 1>([&](auto is) {
        constexpr int S = decltype(is)::value;
        if (s == S) slab_produce<LX, E, S, NS>(p, R, boys_tab, ub, ls);
    });
    if (item == 0) {
        double pw = 1.0;
#pragma unroll
        for (int k = 0; k <= LX; ++k) {
            ub[(size_t)(SC::O_RXP + k) * NS + ls] = pw;
            pw *= R.r[0];
        }
        ub[(size_t)SC::O_RY * NS + ls] = R.r[1];
        ub[(size_t)SC::O_RZ * NS + ls] = R.r[2];
        static_for<0, NLEV>([&](auto ip) {
            constexpr int P_ = decltype(ip)::value;
            ub[(size_t)(SC::O_CK + P_) * NS + ls] = level_scale<LX - 2 * P_, P_>(R);
        });
    }
}

// member of a team of T that takes item k of a list ordered by decreasing size ("snake": 0 1 .. T−1 T−1 .. 1 0)
__host__ __device__ constexpr int snake(int k, int T) { return (k % (2 * T)) < T ? k % T : 2 * T - 1 - k % (2 * T); }

// the chains of ket component c (member 0 of the team)
template <int LX, int LA, int LB>
__device__ __forceinline__ void slab_component_chains(int c, int wt, const double *__restrict__ ub, int kprim,
                                                      double *__restrict__ e0t, int ls, bool add, double scale) {
    int s = 0;
    while ((s + 1) * (s + 2) / 2 <= c) ++s;
    const int cz = c - s * (s + 1) / 2, cy = s - cz, cx = LX - s;
    if (wt == 0) slab_chains_whole<LX, LA, LB>(cx, cy, cz, ub, kprim, e0t, ls, add, scale);
}
// the rows (a_x = S) team member wt transfers and stores (MODE 0) or contracts with D into γ (MODE 1, a9: PAPER.md:283, :365)
template <int LX, int LA, int LB, int MODE>
__device__ __forceinline__ void slab_component_finish(int c, int wt, const OwnHdr *hd, const double *__restrict__ e0t,
                                                      double *__restrict__ stw, int ls, int lane, long long batch,
                                                      long long nsets, double *__restrict__ out, const SlabDf &sd,
                                                      const int32_t *__restrict__ aux_bf) {
    constexpr int T = SlabCls<LX, LA, LB>::T, NS = SlabCls<LX, LA, LB>::NS;
    const double AB[3] = {hd->AB[0][ls], hd->AB[1][ls], hd->AB[2][ls]};
    double part = 0.0;
    static_for<0, LA + 1>([&](auto is) {
        constexpr int S = decltype(is)::value;
        if (wt == snake(S, T)) part += slab_hrr<LX, LA, LB, S, MODE>(e0t, stw, AB, c, ls, lane, batch, nsets, out, hd->tr, sd);
    });
    if constexpr (MODE == 1) {
        // γ[bf(X)+c] += f Σ_ab (c|ab) D_ab: every team member adds the rows it transferred
        if (lane < NS && hd->p[ls] >= 0 && part != 0.0)
            atomicAdd(sd.df.out + aux_bf[hd->x[ls]] + c, (hd->a[ls] != hd->b[ls] ? 2.0 : 1.0) * part);
    }
}

template <int LX, int LA, int LB, int MODE>
__global__ void __launch_bounds__(SlabCls<LX, LA, LB>::NW * 32, 1)
slab_kernel(SetMap map, DevShells aux, DevShells prim, PairData pdat, const double *__restrict__ boys_tab,
            double *__restrict__ out, int swapped, DfArgs df) {
    using SC = SlabCls<LX, LA, LB>;
    constexpr int E = SC::E, NS = SC::NS, NW = SC::NW, NXC = SC::NXC, NLEV = SC::NLEV, NACC = SC::NACC;
    constexpr int SPS = SC::STG | 1, NITEM = (E + 1) * NLEV, T = SC::T, NTEAM = SC::NTEAM;
    constexpr unsigned FULL = 0xffffffffu;

    extern __shared__ double smem[];
    double *U = smem;                                            // [UREC][NS]
    double *E0 = U + (size_t)SC::UREC * NS;                      // [NTEAM][NACC][NS]: (e0|c) of the component a team owns
    double *ST = E0 + (size_t)NTEAM * NACC * NS;                 // [NW][NS][SPS]: staging of finished rows
    OwnHdr *hd2 = reinterpret_cast<OwnHdr *>(ST + (size_t)NW * NS * SPS);
    int *team_c = reinterpret_cast<int *>(hd2 + 2);              // ket component a team works on

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31, ls = lane & (NS - 1);
    const long long nbatch = (map.nsets + NS - 1) / NS;
    const bool tr = MODE == 0 && swapped != 0;
    const int team = warp / T, wt = warp - team * T;
    double *e0t = E0 + (size_t)team * NACC * NS, *stw = ST + (size_t)warp * NS * SPS;

    auto decode = [&](long long bb, OwnHdr *h) {
        SetId sid = decode_set(map, bb * NS + ls, swapped);
        int trs = tr ? 1 : 0;
        if constexpr (LA == LB && LB > 0) {
            // the VRR runs on the shell with the larger exponents (lx_common.cuh, shell_min_zeta): exchange the roles per set
            if (sid.live && shell_min_zeta(prim, sid.b) > shell_min_zeta(prim, sid.a)) {
                const int t = sid.a; sid.a = sid.b; sid.b = t;
                if (MODE == 0) trs ^= 1;                         // the DF modes index D and J by the exchanged roles instead
            }
        }
        h->tr[ls] = trs;
        const int Kab = min(prim.K[sid.a] * prim.K[sid.b], pdat.kstride);
        const int K = sid.live ? Kab * aux.K[sid.x] : 0;
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            const double Ad = prim.center[3 * sid.a + d];
            h->A[d][ls] = Ad;
            h->C[d][ls] = aux.center[3 * sid.x + d];
            h->AB[d][ls] = Ad - prim.center[3 * sid.b + d];
        }
        h->po[ls] = pdat.pd_off ? pdat.pd_off[sid.p] : (long long)sid.p * pdat.kstride;
        h->xo0[ls] = aux.prim_off[sid.x];
        h->Kab[ls] = Kab;
        h->K[ls] = K;
        h->a[ls] = sid.a;
        h->b[ls] = sid.b;
        h->x[ls] = sid.x;
        h->p[ls] = sid.live ? sid.p : -1;
        const int km = __reduce_max_sync(FULL, K);
        if (lane == 0) { h->kmax = km; h->ready = 0; h->next_c = 0; h->next_p = 0; }
    };
    if (warp == 0) decode(blockIdx.x, hd2);

    int it = 0;
    for (long long batch = blockIdx.x; batch < nbatch; batch += gridDim.x, ++it) {
        __syncthreads();                                         // the previous batch is finished; this batch's header is there
        OwnHdr *hd = hd2 + (it & 1), *hn = hd2 + ((it + 1) & 1);
        const int kmax = hd->kmax;
        if (warp == 0) decode(batch + gridDim.x, hn);
        const SlabDf sd{hd, prim.bf_off, df};
        // J digestion (MODE 2): the team's region sums G = Σ_c d_c (e0|c) over every component it takes; the HRR is linear and
        // does not depend on c, so it runs once per batch on Σ_teams G (the step before the HRR is where the paper's J-engine
        // contracts too)
        const double dscale_on = (MODE == 2 && lane < NS && hd->p[ls] >= 0) ? 1.0 : 0.0;
        const double *dvec = MODE == 2 ? df.D + aux.bf_off[hd->x[ls]] : nullptr;
        if constexpr (MODE == 2) {
            for (int i = wt * 32 + lane; i < NACC * NS; i += T * 32) e0t[i] = 0.0;
            named_sync(1 + team, T * 32);
        }
        if (kmax <= 1) {
            // ============ K = 1 batch: start vectors once (work items taken dynamically), then ket components dynamically ======
            while (true) {
                int item = 0;
                if (lane == 0) item = atomicAdd(&hd->next_p, 1);
                item = __shfl_sync(FULL, item, 0);
                if (item >= NITEM) break;
                slab_item<LX, LA, LB>(item, 0, hd, U, ls, aux, pdat, boys_tab);
            }
            __syncthreads();
            while (true) {
                if (wt == 0 && lane == 0) team_c[team] = atomicAdd(&hd->next_c, 1);
                named_sync(1 + team, T * 32);
                const int c = team_c[team];
                if (c >= NXC) break;
                if constexpr (MODE == 2) {
                    const double dc = dscale_on != 0.0 ? __ldg(dvec + c) : 0.0;
                    slab_component_chains<LX, LA, LB>(c, wt, U, 1, e0t, ls, true, dc);
                    named_sync(1 + team, T * 32);                // before the leader takes the next component
                } else {
                    slab_component_chains<LX, LA, LB>(c, wt, U, 1, e0t, ls, false, 1.0);
                    named_sync(1 + team, T * 32);                // (e0|c) of the team is complete
                    slab_component_finish<LX, LA, LB, MODE>(c, wt, hd, e0t, stw, ls, lane, batch, map.nsets, out, sd, aux.bf_off);
                    named_sync(1 + team, T * 32);                // ... and read
                }
            }
        } else {
            // ============ contracted batch: passes of NTEAM ket components; per pass one round per primitive ===================
#pragma unroll 1
            for (int c0 = 0; c0 < NXC; c0 += NTEAM) {
                const int c = c0 + team;
                double dc = 1.0;
                if constexpr (MODE == 2) dc = (dscale_on != 0.0 && c < NXC) ? __ldg(dvec + c) : 0.0;
#pragma unroll 1
                for (int q = 0; q < kmax; ++q) {
                    __syncthreads();                             // the start vectors of the previous round are consumed
#pragma unroll 1
                    for (int item = warp; item < NITEM; item += NW) slab_item<LX, LA, LB>(item, q, hd, U, ls, aux, pdat, boys_tab);
                    __syncthreads();
                    if (c < NXC) slab_component_chains<LX, LA, LB>(c, wt, U, 1, e0t, ls, MODE == 2 || q > 0, dc);
                }
                if constexpr (MODE != 2) {
                    __syncthreads();                             // (e0|c) of every team is complete
                    if (c < NXC) slab_component_finish<LX, LA, LB, MODE>(c, wt, hd, e0t, stw, ls, lane, batch, map.nsets, out, sd, aux.bf_off);
                }
            }
        }
        if constexpr (MODE == 2) {
            // a10: Σ over the teams, one HRR per set, then the lanes that share a shell pair are summed and added to J
            __syncthreads();
            for (int i = tid; i < NACC * NS; i += NW * 32) {
                double g = E0[i];
#pragma unroll
                for (int t = 1; t < NTEAM; ++t) g += E0[(size_t)t * NACC * NS + i];
                E0[i] = g;
            }
            __syncthreads();
            const double AB[3] = {hd->AB[0][ls], hd->AB[1][ls], hd->AB[2][ls]};
            static_for<0, (LA + NW) / NW>([&](auto ir) {           // rounds of NW row blocks: one staging slot per warp
                constexpr int S0 = decltype(ir)::value * NW;
                if constexpr (S0 > 0) __syncthreads();
                static_for<S0, cmin(S0 + NW, LA + 1)>([&](auto is) {
                    constexpr int S = decltype(is)::value;
                    if (warp == S - S0) slab_hrr<LX, LA, LB, S, 2>(E0, stw, AB, 0, ls, lane, batch, map.nsets, out, hd->tr, sd);
                });
                __syncthreads();
                static_for<S0, cmin(S0 + NW, LA + 1)>([&](auto is) {
                    constexpr int S = decltype(is)::value;
                    slab_j_reduce<LX, LA, LB, S>(ST + (size_t)(S - S0) * NS * SPS + (size_t)ls * SPS, warp, NW, ls, lane, sd);
                });
            });
        }
    }
}

// does the class (La >= Lb) run on the slab kernel?  Measured (B200, config 3, K = 1): (6|33) 32.5 -> 14.7 ms, (5|33) 15.6 ->
// 9.3 ms against the group kernel; for La+Lb >= 7 the slabs (45 + 35 doubles for (4|44)) exceed the register file together
// with the call frames and the group kernel is still faster (23.6 ms against 75 ms), so those classes stay there.  For
// Lx <= 2 a batch has too few ket components to keep the teams busy (config 5 digestion: (0|32) 21 -> 29 ms): group kernel.
__host__ __device__ constexpr bool slab_fits(int LX, int LA, int LB) {
    return LX >= 3 && LA + LB >= 5 && LA + LB <= 6 && LA >= LB && LA <= LX_MAX_L_PRIM && LX <= LX_MAX_L_AUX;   // + (1,2|33) in the γ mode, lx_inst.cu
}

template <int LX, int LA, int LB, int MODE>
cudaError_t slab_launch(const SetMap &map, const DevShells &aux, const DevShells &prim, const PairData &pdat,
                        const double *boys_tab, double *out, int swapped, const DfArgs &df, int num_sms,
                        cudaStream_t stream) {
    using SC = SlabCls<LX, LA, LB>;
    static_assert(SC::smem <= 227 * 1024, "slab kernel: batch does not fit in shared memory");
    auto kern = slab_kernel<LX, LA, LB, MODE>;
    static std::atomic<unsigned long long> configured{0};
    if (cudaError_t e = ensure_dyn_smem(kern, SC::smem, configured); e != cudaSuccess) return e;
    if (map.nsets <= 0) return cudaSuccess;
    long long blocks = (map.nsets + SC::NS - 1) / SC::NS;
    if (blocks > (long long)num_sms) blocks = num_sms;
    kern<<<(unsigned)blocks, SC::NW * 32, SC::smem, stream>>>(map, aux, prim, pdat, boys_tab, out, swapped, df);
    return cudaGetLastError();
}

}  // namespace lx
