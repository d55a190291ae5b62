// lx_tune.h — measured per-class group sizes (threads that cooperate on one shell-set); everything else is automatic.
#pragma once
namespace lx {
#define LX_TUNE(LXV, LAV, LBV, GV) \
    template <> struct GrpTune<LXV, LAV, LBV> { static constexpr int G = GV; };
LX_TUNE(4, 2, 2, 32)
LX_TUNE(4, 2, 1, 32)
LX_TUNE(3, 2, 2, 32)
#undef LX_TUNE
}  // namespace lx
