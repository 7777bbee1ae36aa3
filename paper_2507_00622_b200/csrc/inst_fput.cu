// inst_fput.cu -- FPUT chain, N = 8 (BASELINE configs[4]), fixed step: the kernels beyond the basic set
// (inst_fput_n8.cu): GALI_2, GALI_3, Lyapunov k = 1, 2.  4 lanes x 2 particles per lane.
#include "fput_launch.h"
namespace chs {
int try_launch_fput8_more(const LaunchReq& rq) {
    if (rq.adaptive) return -1;
    if (rq.what == WHAT_GALI && rq.k == 2) return run_chain_t<4, 2, false, 2, MODE_NORM, IND_GALI, false, 128, 2>(rq);
    if (rq.what == WHAT_GALI && rq.k == 3) return run_chain_t<4, 2, false, 3, MODE_NORM, IND_GALI, false, 128, 2, true>(rq);
    if (rq.what == WHAT_LYAP && rq.k == 1) return run_chain_t<4, 2, false, 1, MODE_MGS, IND_NONE, false, 128, 3>(rq);
    if (rq.what == WHAT_LYAP && rq.k == 2) return run_chain_t<4, 2, false, 2, MODE_MGS, IND_NONE, false, 128, 2>(rq);
    return -1;
}
}  // namespace chs
