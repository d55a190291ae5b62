// lx_dispatch.h — launcher symbols defined by the lx_inst.cu translation units.
#pragma once
#include "lx_common.cuh"

namespace lx {

#define LX_DECL(LXV, MODEV)                                                                                      \
    cudaError_t launch_lx##LXV##_mode##MODEV(int la, int lb, const SetMap &map, const DevShells &aux,             \
                                             const DevShells &prim, const PairData &pdat, const double *boys_tab, \
                                             double *out, int swapped, const DfArgs &df, int num_sms,             \
                                             cudaStream_t stream);
#define LX_DECL3(LXV) LX_DECL(LXV, 0) LX_DECL(LXV, 1) LX_DECL(LXV, 2) LX_DECL(LXV, 3)
LX_DECL3(0) LX_DECL3(1) LX_DECL3(2) LX_DECL3(3) LX_DECL3(4) LX_DECL3(5) LX_DECL3(6)
#undef LX_DECL3
#undef LX_DECL

using launch_fn = cudaError_t (*)(int, int, const SetMap &, const DevShells &, const DevShells &, const PairData &,
                                  const double *, double *, int, const DfArgs &, int, cudaStream_t);

}  // namespace lx
