// lx_inst.cu — instantiates the class kernels for one aux angular momentum (INST_LX) and one digestion mode
// (INST_MODE: 0 store, 1 γ, 2 J).  Compiled once per (INST_LX, INST_MODE); no code generator: every class is a
// template instantiation.
#include "lx_chain.cuh"
#include "lx_dispatch.h"

#ifndef INST_LX
#error "compile with -DINST_LX=<0..6> -DINST_MODE=<0..2>"
#endif

namespace lx {

// kernel family per class: register-resident lane kernel where the bra components of a set fit one warp
// (La+Lb <= 3), shared-memory group kernel otherwise
template <int LX, int LA, int LB, int MODE>
static cudaError_t class_launch(const SetMap &map, const DevShells &aux, const DevShells &prim, const PairData &pdat,
                                const double *boys_tab, double *out, int swapped, const DfArgs &df, int num_sms,
                                cudaStream_t stream) {
    if constexpr (ChainCls<LX, LA, LB>::fits)
        return chain_launch<LX, LA, LB, MODE>(map, aux, prim, pdat, boys_tab, out, swapped, df, num_sms, stream);
    else if constexpr (LaneCls<LX, LA, LB>::fits)
        return lane_launch<LX, LA, LB, MODE>(map, aux, prim, pdat, boys_tab, out, swapped, df, num_sms, stream);
    else
        return group_launch<LX, LA, LB, MODE>(map, aux, prim, pdat, boys_tab, out, swapped, df, num_sms, stream);
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
