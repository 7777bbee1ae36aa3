// inst_c3_more.cu -- 3-DoF coupled oscillators: the remaining k (Lyapunov k = 2..5, GALI k = 4..6,
// adaptive mLE / SALI-like GALI_2).
#include "launch.h"
namespace chs {
int try_launch_c3_more(const LaunchReq& rq) {
    if (CHS_MATCH(1, WHAT_LYAP, 2, 0)) return run_col<Coupled3, 2, 4, MODE_MGS, IND_NONE, false, 128, 4>(rq);
    if (CHS_MATCH(1, WHAT_LYAP, 3, 0)) return run_col<Coupled3, 3, 4, MODE_MGS, IND_NONE, false, 128, 4>(rq);
    if (CHS_MATCH(1, WHAT_LYAP, 4, 0)) return run_col<Coupled3, 4, 8, MODE_MGS, IND_NONE, false, 128, 3>(rq);
    if (CHS_MATCH(1, WHAT_LYAP, 5, 0)) return run_col<Coupled3, 5, 8, MODE_MGS, IND_NONE, false, 128, 3>(rq);
    if (CHS_MATCH(1, WHAT_LYAP, 1, 1)) return run_col<Coupled3, 1, 2, MODE_MGS, IND_NONE, true, 128, 2>(rq);
    if (CHS_MATCH(1, WHAT_GALI, 4, 0)) return run_col<Coupled3, 4, 8, MODE_NORM, IND_GALI, false, 128, 3>(rq);
    if (CHS_MATCH(1, WHAT_GALI, 5, 0)) return run_col<Coupled3, 5, 8, MODE_NORM, IND_GALI, false, 128, 3>(rq);
    if (CHS_MATCH(1, WHAT_GALI, 6, 0)) return run_col<Coupled3, 6, 8, MODE_NORM, IND_GALI, false, 128, 3>(rq);
    if (CHS_MATCH(1, WHAT_GALI, 2, 1)) return run_col<Coupled3, 2, 4, MODE_NORM, IND_GALI, true, 128, 3>(rq);
    return -1;
}
}  // namespace chs
