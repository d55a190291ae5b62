// lx_inst.cu — instantiates the class kernels for one aux angular momentum (INST_LX) and one digestion mode
// (INST_MODE: 0 store, 1 γ, 2 J).  Compiled once per (INST_LX, INST_MODE); no code generator: every class is a
// template instantiation.
#include <cstdlib>
#include <cstring>

#include "lx_chain_kernel.cuh"
#include "lx_slab.cuh"
#include "lx_dispatch.h"

#ifndef INST_LX
#error "compile with -DINST_LX=<0..6> -DINST_MODE=<0..3>"
#endif

namespace lx {

// kernel family per class: team kernel where the chain targets of a warp fit its registers,
// warp-specialised chain kernel for the other classes with La+Lb <= 4 and Lx <= 4, lane / group kernels beyond.
// In builds with -DLX_TUNING (LX_EXTRA_NVCC=-DLX_TUNING) LX_FAMILY=team|chain|lane|owner in the environment overrides the
// choice where the named family exists; regular builds compile one family per class.
#ifdef LX_TUNING
static int family_override() {
    static int v = -1;
    if (v < 0) {
        const char *e = std::getenv("LX_FAMILY");
        v = !e ? 0 : (!std::strcmp(e, "team") ? 1 : (!std::strcmp(e, "chain") ? 2 : (!std::strcmp(e, "lane") ? 3 : (!std::strcmp(e, "owner") ? 4 : 0))));
    }
    return v;
}
#endif

template <int LX, int LA, int LB, int MODE>
static cudaError_t class_launch(const SetMap &map, const DevShells &aux, const DevShells &prim, const PairData &pdat,
                                const double *boys_tab, double *out, int swapped, const DfArgs &df, int num_sms,
                                cudaStream_t stream) {
    constexpr int TW = team_width(LX, LA, LB);
    constexpr bool has_team = TW > 0, has_chain = ChainCls<LX, LA, LB>::fits, has_lane = LaneCls<LX, LA, LB>::fits;
    if constexpr (MODE == 3) {
        // fused solid-harmonic aux functions: team kernel only; the caller falls back to Cartesian + lx_cart_to_pure
        if constexpr (has_team && LX >= 2)
            return team_launch<LX, LA, LB, MODE, (TW > 0 ? TW : 1)>(map, aux, prim, pdat, boys_tab, out, swapped, df, num_sms, stream);
        else if constexpr (has_chain && LX >= 2)
            return chain_launch<LX, LA, LB, MODE>(map, aux, prim, pdat, boys_tab, out, swapped, df, num_sms, stream);
        else
            return cudaErrorNotSupported;
    } else {
    // Lx = 5, 6 at La+Lb <= 4: one owner warp per ket component (lx_owner.cuh) where the team kernel does not apply
    constexpr bool has_owner = owner_fits(LX, LA, LB) && (LX >= 5 || owner_over_team(LX, LA, LB) || !has_team);
#ifdef LX_TUNING
    // tuning builds compile every family for every class; LX_FAMILY picks one at run time where it exists
    const int ov = family_override();
    if constexpr (has_owner) {
        if (ov == 4 || (ov == 0 && !has_team))
            return owner_launch<LX, LA, LB, MODE>(map, aux, prim, pdat, boys_tab, out, swapped, df, num_sms, stream);
    }
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
#else
    if constexpr (has_owner) {
        // weakly contracted launches (and every launch of the Lx = 5, 6 classes with La+Lb >= 3): the team / chain / lane kernels win
        // at high K, where their per-primitive work (one chain per distinct target, the owner's: one per partner) decides
        if (owner_kmax(LX, LA, LB) == (1 << 30) || (map.khint > 0 && map.khint <= owner_kmax(LX, LA, LB)))
            return owner_launch<LX, LA, LB, MODE>(map, aux, prim, pdat, boys_tab, out, swapped, df, num_sms, stream);
    }
    constexpr bool owner_only = has_owner && owner_kmax(LX, LA, LB) == (1 << 30);
    if constexpr (owner_only)
        return cudaErrorUnknown;   // not reached
    else if constexpr (has_team)
        return team_launch<LX, LA, LB, MODE, (TW > 0 ? TW : 1)>(map, aux, prim, pdat, boys_tab, out, swapped, df, num_sms, stream);
    else if constexpr (has_chain)
        return chain_launch<LX, LA, LB, MODE>(map, aux, prim, pdat, boys_tab, out, swapped, df, num_sms, stream);
    else if constexpr (has_lane)
        return lane_launch<LX, LA, LB, MODE>(map, aux, prim, pdat, boys_tab, out, swapped, df, num_sms, stream);
    else if constexpr (slab_fits(LX, LA, LB) || (MODE == 1 && LA == 3 && LB == 3 && LX >= 1))   // (1|33), (2|33) γ: 20 -> 6, 27 -> 11 ms (config 5)
        return slab_launch<LX, LA, LB, MODE>(map, aux, prim, pdat, boys_tab, out, swapped, df, num_sms, stream);
    else
        return group_launch<LX, LA, LB, MODE>(map, aux, prim, pdat, boys_tab, out, swapped, df, num_sms, stream);
#endif
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
