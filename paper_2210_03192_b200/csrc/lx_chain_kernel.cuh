// lx_chain_kernel.cuh — the warp-specialised chain kernel (design and algebra: lx_chain.cuh; shared per-primitive
// arithmetic, target drop and epilogue: lx_team.cuh).
#pragma once
#include "lx_team.cuh"

// 1: classes with three or more passes re-align producers and consumers at every pass boundary (tuning aid; measured
// within 1 % of the free-running ring, which is the default)
#ifndef LX_CHAIN_REALIGN
#define LX_CHAIN_REALIGN 0
#endif

namespace lx {

template <int LX, int LA, int LB, int MODE, int NW, int MINB>
__global__ void __launch_bounds__(NW * 32, MINB)
chain_kernel(SetMap map, DevShells aux, DevShells prim, PairData pdat, const double *__restrict__ boys_tab,
             double *__restrict__ out, int swapped, DfArgs df) {
    using CC = ChainCls<LX, LA, LB>;
    constexpr int E = CC::E, NG = CC::NG, NACC = CC::NACC, NXC = CC::NXC, NA = CC::NA, NB = CC::NB, NAB = CC::NAB;
    // MODE 3 (solid-harmonic aux functions, lx_team.cuh "MODE 3"): only the passes of the level-0 targets run, the (e0|c)
    // slots are packed (NACC per ket component: the HRR writes to the pure region, which aliases the ring), one VRR1 level
    constexpr bool PURE = MODE == 3;
    constexpr int CSTR = PURE ? NACC : NAB;
    constexpr int SLOTN = PURE ? ((NXC * NACC) | 1) : CC::SLOTN;
    constexpr int ZBD = PURE ? cmax(CC::ZBD, 32 * (((2 * LX + 1) * NAB) | 1)) : CC::ZBD;
    constexpr int NPE = PURE ? (NXC + CC::P.t1[0] - 1) / CC::P.t1[0] : CC::P.npass;   // passes that hold level-0 targets
    constexpr ChainTargets T = CC::T;
    constexpr ChainPlan P = CC::P;
    constexpr unsigned FULL = 0xffffffffu;

    extern __shared__ double smem[];
    double *TC = smem;                                       // [set][c * NAB + ·]: (e0|c), then the finished shell-set
    double *ZB = TC + (size_t)32 * SLOTN;                    // ring of start-vector buffers
    double *hd0 = ZB + (size_t)ZBD;                     // two header buffers: [9][32] doubles A, C, AB; po; 6 ints; kmax
    PartnerTab *pt = reinterpret_cast<PartnerTab *>(hd0 + CC::HDRD + 4);
    if (threadIdx.x == 0) partner_tab_build<LX>(pt);

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const long long nbatch = (map.nsets + 31) / 32;

    // header of batch bb into buffer hb (warp 0, lane = set); batches past the end decode as empty sets
    auto decode_header = [&](long long bb, int hb) {
        double *hd = hd0 + (size_t)hb * CC::HDR1;
        long long *hpo = reinterpret_cast<long long *>(hd + 9 * 32);
        int *hi = reinterpret_cast<int *>(hpo + 32);
        int *s_kmax = hi + 7 * 32;
        const long long sid = bb * 32 + lane;
        const bool live = sid < map.nsets;
        int p = 0, xs = 0;
        if (map.cum == nullptr) {
            if (live) {
                p = (int)(sid / map.nx);
                xs = (int)(sid - (long long)p * map.nx);
            }
        } else {
            find_pair_warp(map, sid, live, p, xs);               // the whole warp 0 is here (lane = set)
        }
        const int a = map.pair_list[2 * p + swapped], b = map.pair_list[2 * p + 1 - swapped];
        const int x = map.x_list[xs];
        const int Kab = min(prim.K[a] * prim.K[b], pdat.kstride);
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
        hi[6 * 32 + lane] = p;
        const int km = __reduce_max_sync(FULL, K);
        if (lane == 0) *s_kmax = km;
    };
    if (warp == 0) decode_header(blockIdx.x, 0);
    int hbuf = 0;
    for (long long batch = blockIdx.x; batch < nbatch; batch += gridDim.x, hbuf ^= 1) {
        const double *hd = hd0 + (size_t)hbuf * CC::HDR1;    // this batch's header (decoded during the previous batch)
        const long long *hpo = reinterpret_cast<const long long *>(hd + 9 * 32);
        const int *hi = reinterpret_cast<const int *>(hpo + 32);
        const int *s_kmax = hi + 7 * 32;
        __syncthreads();
        const int kmax = *s_kmax;
        // the finished shell-sets of the previous batch are still in TC (nothing writes TC before the end of the first
        // pass): the consumer warps, idle while the producers fill the ring, copy them out now
        // warp 0 decodes the next batch while the producers fill the ring (it is a consumer and would idle)
        if (warp == 0) decode_header(batch + gridDim.x, hbuf ^ 1);
        if constexpr (MODE == 0) {
            if (warp < P.ncx && batch != (long long)blockIdx.x)
                batch_copy_out<CC::NINT, SLOTN>(TC, out, batch - gridDim.x, map.nsets, warp * 32 + lane, P.ncx * 32);
        }

        // ---- passes over the primitive loop: ONE ring runs through all passes (slot g = pass * kmax + q), so the producers
        // of pass i+1 fill it while the consumers of pass i finish; roles are fixed for the batch: warps [0, NCX) consume
        // (warp w holds target T0 + w of the current pass, or idles through the barriers), warps [NCX, NCX + NPX) produce.
        constexpr int NCX = P.ncx, NPX = P.npx, NBUF = NPX + 1, ZREC = P.zrec;
        constexpr int BCOUNT = (NCX + 1) * 32;               // threads on a full[] / empty[] barrier
        const int gtot = NPE * kmax;                         // ring slots of the batch
        if (warp >= NCX) {
            // ================= producers: ring slots g = j, j + NPX, ... ======================================================
            const int j = warp - NCX;
            const double Ax = hd[0 * 32 + lane], Ay = hd[1 * 32 + lane], Az = hd[2 * 32 + lane];
            const double Cx = hd[3 * 32 + lane], Cy = hd[4 * 32 + lane], Cz = hd[5 * 32 + lane];
            const long long po = hpo[lane];
            const int xo0 = hi[0 * 32 + lane], Kab = hi[1 * 32 + lane], K = hi[2 * 32 + lane];
            static_for<0, NPE>([&](auto ipass) {
                constexpr int ip = decltype(ipass)::value;
                constexpr int PLO = PURE ? 0 : P.plo[ip], NLV = PURE ? 1 : P.phi[ip] - P.plo[ip] + 1;
                const int g0 = ip * kmax;
                for (int q = ((j - g0) % NPX + NPX) % NPX; q < kmax; q += NPX) {
                    const int g = g0 + q, bsel = g % NBUF;
                    if (g >= NBUF) named_sync(1 + NBUF + bsel, BCOUNT);      // consumers are done with this buffer
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
                if constexpr (LX_CHAIN_REALIGN && CC::P.npass > 2 && ip + 1 < CC::P.npass) named_sync(15, NW * 32);
            });
            named_sync(15, NW * 32);                         // all ring traffic of the batch is done
        } else {
            // ================= consumers ===========================================================================================
            double acc[NACC];                                // lives in the consumer branch only: producers keep their registers
            static_for<0, NPE>([&](auto ipass) {
                constexpr int ip = decltype(ipass)::value;
                constexpr int T0 = P.t0[ip], NC = (PURE ? cmin(P.t1[ip], NXC) : P.t1[ip]) - P.t0[ip];
                constexpr int PLO = PURE ? 0 : P.plo[ip], NLV = PURE ? 1 : P.phi[ip] - P.plo[ip] + 1;
                static_assert(PURE || T0 + NC <= NXC || ip == P.npass - 1, "levels p >= 1 must sit in the last pass");
#pragma unroll
                for (int i = 0; i < NACC; ++i) acc[i] = 0.0;
                const int g0 = ip * kmax;
                for (int q = 0; q < kmax; ++q) {
                    const int g = g0 + q, bsel = g % NBUF;
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
                    if (g + NBUF < gtot) named_arrive(1 + NBUF + bsel, BCOUNT);   // empty[bsel]
                }
                // level-0 targets go straight to their private Cartesian slot of TC
                if (warp < NC && T0 + warp < NXC) target_drop<LX, LA, LB, CSTR, SLOTN>(T0 + warp, acc, TC, ZB, lane);
                if constexpr (LX_CHAIN_REALIGN && CC::P.npass > 2 && ip + 1 < CC::P.npass) named_sync(15, NW * 32);
            });
            named_sync(15, NW * 32);                         // all ring traffic of the batch is done
            // the targets of the levels p >= 1 (all in the last pass) go to the staging area, which aliases the idle ring
            if constexpr (!PURE && CC::T.n > NXC) {
                constexpr int T0L = P.t0[P.npass - 1], NCL = P.t1[P.npass - 1] - T0L;
                if (warp < NCL && T0L + warp >= NXC) target_drop<LX, LA, LB>(T0L + warp, acc, TC, ZB, lane);
            }
        }
        __syncthreads();
        if constexpr (PURE) pure_epilogue<LX, LA, LB, NW, CSTR, SLOTN>(TC, ZB, df.D, warp, lane, batch, map, prim, out, swapped);
        else {
            // the lane's shell-set, from the batch header in shared memory (decoded one batch ahead by warp 0)
            SetId sid;
            sid.a = hi[3 * 32 + lane];
            sid.b = hi[4 * 32 + lane];
            sid.x = hi[5 * 32 + lane];
            sid.p = hi[6 * 32 + lane];
            sid.live = batch * 32 + lane < map.nsets;
            chain_epilogue<LX, LA, LB, MODE, NW, true>(TC, ZB, pt, warp, lane, batch, map, aux, prim, out, swapped, df, sid);
        }
    }
    // the last batch of this block (the epilogue ended with a block barrier)
    if constexpr (MODE == 0) {
        if ((long long)blockIdx.x < nbatch) {
            const long long last = blockIdx.x + ((nbatch - 1 - blockIdx.x) / gridDim.x) * gridDim.x;
            batch_copy_out<CC::NINT, SLOTN>(TC, out, last, map.nsets, tid, NW * 32);
        }
    }
}

template <int LX, int LA, int LB, int MODE>
cudaError_t chain_launch(const SetMap &map, const DevShells &aux, const DevShells &prim, const PairData &pdat,
                         const double *boys_tab, double *out, int swapped, const DfArgs &df, int num_sms,
                         cudaStream_t stream) {
    using CC = ChainCls<LX, LA, LB>;
    constexpr int NW = CC::NW;
    // MODE 3: packed (e0|c) slots, the pure region aliases the ring (see the kernel)
    constexpr int SLOT3 = (CC::NXC * CC::NACC) | 1, ZBD3 = cmax(CC::ZBD, 32 * (((2 * LX + 1) * CC::NAB) | 1));
    constexpr size_t smem = MODE == 3 ? ((size_t)32 * SLOT3 + (size_t)ZBD3 + CC::HDRD + 4) * 8 + 2048 : CC::smem;
    if constexpr (smem > 227 * 1024) return cudaErrorNotSupported;   // MODE 3 only: the caller falls back
    else {
    // resident blocks per SM: shared memory, and registers (a consumer keeps NG + NACC doubles live)
    constexpr int by_smem = (int)((227 * 1024) / (smem + 1024));
    constexpr int regs = CC::E <= 2 ? 80 : (CC::E == 3 ? 128 : 168);
    constexpr int by_regs = 65536 / (NW * 32 * regs);
    constexpr int BPS = cmax(1, cmin(cmin(by_smem, by_regs), 8));
    auto kern = chain_kernel<LX, LA, LB, MODE, NW, BPS>;
    static std::atomic<unsigned long long> configured{0};
    if (cudaError_t e = ensure_dyn_smem(kern, smem, configured); e != cudaSuccess) return e;
    if (map.nsets <= 0) return cudaSuccess;
    long long blocks = (map.nsets + 31) / 32;
    const long long cap = (long long)num_sms * BPS;
    if (blocks > cap) blocks = cap;
    kern<<<(unsigned)blocks, NW * 32, smem, stream>>>(map, aux, prim, pdat, boys_tab, out, swapped, df);
    return cudaGetLastError();
    }
}

}  // namespace lx
