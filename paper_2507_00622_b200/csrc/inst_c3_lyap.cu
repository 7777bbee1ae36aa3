// inst_c3_lyap.cu -- 3-DoF coupled oscillators: full Lyapunov spectrum (BASELINE configs[3]).
// Fixed step: 4-lane tile per trajectory, two columns per lane (orbit + empty slot | w1, w2 | w3, w4 | w5, w6),
// blocks of 256 threads, one per SM (measured: 1150 ms against 1160 ms with two blocks of 128).
// Adaptive: 8-lane tile, one column per lane (lane 7 idle).  Also GALI_2, GALI_3.
#include "launch.h"
namespace chs {
int try_launch_c3_lyap(const LaunchReq& rq) {
    if (CHS_MATCH(1, WHAT_LYAP, 6, 0)) return run_col<Coupled3, 6, 4, MODE_MGS, IND_NONE, false, 256, 1>(rq);
    if (CHS_MATCH(1, WHAT_LYAP, 6, 1)) return run_col<Coupled3, 6, 8, MODE_MGS, IND_NONE, true, 128, 2>(rq);
    if (CHS_MATCH(1, WHAT_GALI, 2, 0)) return run_col<Coupled3, 2, 4, MODE_NORM, IND_GALI, false, 128, 4>(rq);
    if (CHS_MATCH(1, WHAT_GALI, 3, 0)) return run_col<Coupled3, 3, 4, MODE_NORM, IND_GALI, false, 128, 4>(rq);
    return -1;
}
}  // namespace chs
