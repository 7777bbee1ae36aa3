// inst_hh_ind.cu -- Henon-Heiles, fixed step: GALI_k (k = 2..4) and Lyapunov spectrum (k = 1..4).
#include "launch.h"
namespace chs {
int try_launch_hh_ind(const LaunchReq& rq) {
    if (CHS_MATCH(0, WHAT_GALI, 2, 0)) return run_col<HenonHeiles, 2, 1, MODE_NORM, IND_GALI, false, 128, 1>(rq);
    if (CHS_MATCH(0, WHAT_GALI, 3, 0)) return run_col<HenonHeiles, 3, 1, MODE_NORM, IND_GALI, false, 128, 1>(rq);
    if (CHS_MATCH(0, WHAT_GALI, 4, 0)) return run_col<HenonHeiles, 4, 2, MODE_NORM, IND_GALI, false, 128, 1>(rq);
    if (CHS_MATCH(0, WHAT_LYAP, 1, 0)) return run_col<HenonHeiles, 1, 1, MODE_MGS, IND_NONE, false, 128, 2>(rq);
    if (CHS_MATCH(0, WHAT_LYAP, 2, 0)) return run_col<HenonHeiles, 2, 1, MODE_MGS, IND_NONE, false, 128, 1>(rq);
    if (CHS_MATCH(0, WHAT_LYAP, 3, 0)) return run_col<HenonHeiles, 3, 1, MODE_MGS, IND_NONE, false, 128, 1, false>(rq);
    if (CHS_MATCH(0, WHAT_LYAP, 4, 0)) return run_col<HenonHeiles, 4, 2, MODE_MGS, IND_NONE, false, 128, 1>(rq);
    return -1;
}
}  // namespace chs
