// lx_inst.cu — instantiates the class kernels for one aux angular momentum (INST_LX) and one digestion mode
// (INST_MODE: 0 store, 1 γ, 2 J).  Compiled once per (INST_LX, INST_MODE); no code generator: every class is a
// template instantiation.
#include <cstdlib>
#include <cstring>

#include "lx_chain_kernel.cuh"
#include "lx_dispatch.h"

#ifndef INST_LX
#error "compile with -DINST_LX=<0..6> -DINST_MODE=<0..3>"
#endif

namespace lx {

// kernel family per class: team kernel where the chain targets of a warp fit its registers,
// warp-specialised chain kernel for the other classes with La+Lb <= 4 and Lx <= 4, lane / group kernels beyond.
// LX_FAMILY=team|chain|lane in the environment overrides the choice where the named family exists (tuning aid).
#ifndef LX_TEAM_WMAX
#define LX_TEAM_WMAX 2
#endif
#ifndef LX_TEAM_BUDGET
#define LX_TEAM_BUDGET 72
#endif
static int family_override() {
    static int v = -1;
    if (v < 0) {
        const char *e = std::getenv("LX_FAMILY");
        v = !e ? 0 : (!std::strcmp(e, "team") ? 1 : (!std::strcmp(e, "chain") ? 2 : (!std::strcmp(e, "lane") ? 3 : 0)));
    }
    return v;
}

template <int LX, int LA, int LB, int MODE>
static cudaError_t class_launch(const SetMap &map, const DevShells &aux, const DevShells &prim, const PairData &pdat,
                                const double *boys_tab, double *out, int swapped, const DfArgs &df, int num_sms,
                                cudaStream_t stream) {
    constexpr bool small = LA + LB <= 4 && LX <= LX_MAX_L_AUX;   // team: any Lx; the chain kernel has its own bound (Lx <= 4)
    // (3|21) keeps all 13 targets in three warps with 80 accumulator doubles per lane: measured faster than the chain kernel
    constexpr bool wide = LX == 3 && LA == 2 && LB == 1;
    constexpr int TW = small ? team_size(LX, LA, LB, wide ? 80 : LX_TEAM_BUDGET) : 0;
    // measured (B200): for Lx <= 4 the team kernel wins for La+Lb <= 2 and wherever one or two warps hold all targets;
    // for Lx = 5, 6 it beats the lane kernel while at most three warps hold the targets
    constexpr bool has_team = TW > 0 && (LX <= 4 ? (LA + LB <= 2 || TW <= (wide ? 3 : LX_TEAM_WMAX)) : (LA + LB >= 1 && TW <= 3)), has_chain = ChainCls<LX, LA, LB>::fits, has_lane = LaneCls<LX, LA, LB>::fits;
    if constexpr (MODE == 3) {
        // fused solid-harmonic aux functions: team kernel only; the caller falls back to Cartesian + lx_cart_to_pure
        if constexpr (has_team && LX >= 2)
            return team_launch<LX, LA, LB, MODE, (TW > 0 ? TW : 1)>(map, aux, prim, pdat, boys_tab, out, swapped, df, num_sms, stream);
        else if constexpr (has_chain && LX >= 2)
            return chain_launch<LX, LA, LB, MODE>(map, aux, prim, pdat, boys_tab, out, swapped, df, num_sms, stream);
        else
            return cudaErrorNotSupported;
    } else {
    const int ov = family_override();
    if constexpr (has_team) {
        if (ov == 0 || ov == 1 || (ov == 2 && !has_chain) || (ov == 3 && !has_lane))
            return team_launch<LX, LA, LB, MODE, (TW > 0 ? TW : 1)>(map, aux, prim, pdat, boys_tab, out, swapped, df, num_sms, stream);
    }
    if constexpr (has_chain) {
        if (ov != 3 || !has_lane)
            return chain_launch<LX, LA, LB, MODE>(map, aux, prim, pdat, boys_tab, out, swapped, df, num_sms, stream);
    }
    if constexpr (has_lane)
        return lane_launch<LX, LA, LB, MODE>(map, aux, prim, pdat, boys_tab, out, swapped, df, num_sms, stream);
    else
        return group_launch<LX, LA, LB, MODE>(map, aux, prim, pdat, boys_tab, out, swapped, df, num_sms, stream);
    }
}

#define LX_CASE(LA_, LB_)                                                                                        \
    case LA_ * 8 + LB_:                                                                                           \
        return class_launch<INST_LX, LA_, LB_, INST_MODE>(map, aux, prim, pdat, boys_tab, out, swapped, df, num_sms, stream);

#define LX_CAT_(a, b, c, d) a##b##c##d
#define LX_CAT(a, b, c, d) LX_CAT_(a, b, c, d)

cudaError_t LX_CAT(launch_lx, INST_LX, _mode, INST_MODE)(int la, int lb, const SetMap &map, const DevShells &aux,
                                                           const DevShells &prim, const PairData &pdat,
                                                           const double *boys_tab, double *out, int swapped,
                                                           const DfArgs &df, int num_sms, cudaStream_t stream) {
    switch (la * 8 + lb) {
        LX_CASE(0, 0)
        LX_CASE(1, 0) LX_CASE(1, 1)
        LX_CASE(2, 0) LX_CASE(2, 1) LX_CASE(2, 2)
        LX_CASE(3, 0) LX_CASE(3, 1) LX_CASE(3, 2) LX_CASE(3, 3)
        LX_CASE(4, 0) LX_CASE(4, 1) LX_CASE(4, 2) LX_CASE(4, 3) LX_CASE(4, 4)
        default: return cudaErrorInvalidValue;
    }
}

}  // namespace lx
