// inst_hh.cu -- Henon-Heiles: plain fixed-step integration, Lagrangian descriptor, fixed-step SALI.
#include "launch.h"
namespace chs {
int try_launch_hh(const LaunchReq& rq) {
    if (CHS_MATCH(0, WHAT_INTEGRATE, 0, 0)) return run_col<HenonHeiles, 0, 1, MODE_NONE, IND_NONE, false, 128, 4>(rq);
    if (CHS_MATCH(0, WHAT_LD, 0, 0)) return run_ld<HenonHeiles, 128, 7>(rq);
    if (CHS_MATCH(0, WHAT_SALI, 2, 0)) return run_col<HenonHeiles, 2, 1, MODE_NORM, IND_SALI, false, 128, 1>(rq);
    return -1;
}
}  // namespace chs
