// inst_fput_adapt.cu -- FPUT chain, N = 8, adaptive DOP8(5) (Fig. 3 used the
// adaptive solver with GALI_4).
#include "fput_launch.h"
namespace chs {
int try_launch_fput_adapt(const LaunchReq& rq) {
    if (FPUT_MATCH(8, WHAT_INTEGRATE, 0, 1)) return run_chain<8, 0, MODE_NONE, IND_NONE, true, 128, 4>(rq);
    if (FPUT_MATCH(8, WHAT_SALI, 2, 1)) return run_chain<8, 2, MODE_NORM, IND_SALI, true, 128, 2>(rq);
    if (FPUT_MATCH(8, WHAT_GALI, 2, 1)) return run_chain<8, 2, MODE_NORM, IND_GALI, true, 128, 3>(rq);
    if (FPUT_MATCH(8, WHAT_GALI, 3, 1)) return run_chain<8, 3, MODE_NORM, IND_GALI, true, 128, 2>(rq);
    if (FPUT_MATCH(8, WHAT_GALI, 4, 1)) return run_chain<8, 4, MODE_NORM, IND_GALI, true, 128, 2>(rq);
    if (FPUT_MATCH(8, WHAT_LYAP, 1, 1)) return run_chain<8, 1, MODE_MGS, IND_NONE, true, 128, 4>(rq);
    if (FPUT_MATCH(8, WHAT_LYAP, 4, 1)) return run_chain<8, 4, MODE_MGS, IND_NONE, true, 128, 2>(rq);
    return -1;
}
}  // namespace chs
