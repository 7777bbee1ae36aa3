// inst_fput_adapt.cu -- FPUT chain, N = 8, adaptive DOP8(5) beyond the basic set:
// SALI, GALI_2, GALI_3, Lyapunov k = 1, 4.  8 lanes x 1 particle per lane.
#include "fput_launch.h"
namespace chs {
int try_launch_fput8_adapt(const LaunchReq& rq) {
    if (!rq.adaptive) return -1;
    if (rq.what == WHAT_SALI && rq.k == 2) return run_chain_t<8, 1, false, 2, MODE_NORM, IND_SALI, true, 128, 2>(rq);
    if (rq.what == WHAT_GALI && rq.k == 2) return run_chain_t<8, 1, false, 2, MODE_NORM, IND_GALI, true, 128, 3>(rq);
    if (rq.what == WHAT_GALI && rq.k == 3) return run_chain_t<8, 1, false, 3, MODE_NORM, IND_GALI, true, 128, 2>(rq);
    if (rq.what == WHAT_LYAP && rq.k == 1) return run_chain_t<8, 1, false, 1, MODE_MGS, IND_NONE, true, 128, 3>(rq);
    if (rq.what == WHAT_LYAP && rq.k == 4) return run_chain_t<8, 1, false, 4, MODE_MGS, IND_NONE, true, 128, 2>(rq);
    return -1;
}
}  // namespace chs
