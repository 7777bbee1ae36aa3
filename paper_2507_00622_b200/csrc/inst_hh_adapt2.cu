// inst_hh_adapt2.cu -- Henon-Heiles, adaptive DOP8(5): GALI_3, GALI_4, Lyapunov k = 3, 4.
#include "launch.h"
namespace chs {
int try_launch_hh_adapt2(const LaunchReq& rq) {
    if (CHS_MATCH(0, WHAT_GALI, 3, 1)) return run_col<HenonHeiles, 3, 2, MODE_NORM, IND_GALI, true, 128, 2>(rq);
    if (CHS_MATCH(0, WHAT_GALI, 4, 1)) return run_col<HenonHeiles, 4, 2, MODE_NORM, IND_GALI, true, 128, 1>(rq);
    if (CHS_MATCH(0, WHAT_LYAP, 3, 1)) return run_col<HenonHeiles, 3, 2, MODE_MGS, IND_NONE, true, 128, 2>(rq);
    if (CHS_MATCH(0, WHAT_LYAP, 4, 1)) return run_col<HenonHeiles, 4, 4, MODE_MGS, IND_NONE, true, 128, 2>(rq);
    return -1;
}
}  // namespace chs
