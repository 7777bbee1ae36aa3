// inst_c3.cu -- 3-DoF coupled oscillators: integration (fixed/adaptive), LD, SALI, mLE.
#include "launch.h"
namespace chs {
int try_launch_c3(const LaunchReq& rq) {
    if (CHS_MATCH(1, WHAT_INTEGRATE, 0, 0)) return run_col<Coupled3, 0, 1, MODE_NONE, IND_NONE, false, 128, 4>(rq);
    if (CHS_MATCH(1, WHAT_INTEGRATE, 0, 1)) return run_col<Coupled3, 0, 1, MODE_NONE, IND_NONE, true, 128, 3>(rq);
    if (CHS_MATCH(1, WHAT_LD, 0, 0)) return run_ld<Coupled3, 128, 3>(rq);
    if (CHS_MATCH(1, WHAT_LD, 0, 1)) return run_col_ld_adapt<Coupled3, 128, 2>(rq);
    if (CHS_MATCH(1, WHAT_SALI, 2, 0)) return run_col<Coupled3, 2, 4, MODE_NORM, IND_SALI, false, 128, 4>(rq);
    if (CHS_MATCH(1, WHAT_SALI, 2, 1)) return run_col<Coupled3, 2, 4, MODE_NORM, IND_SALI, true, 128, 3, false>(rq);
    if (CHS_MATCH(1, WHAT_LYAP, 1, 0)) return run_col<Coupled3, 1, 2, MODE_MGS, IND_NONE, false, 128, 4>(rq);
    return -1;
}
}  // namespace chs
