// inst_fput.cu -- FPUT chain, N = 8 (BASELINE configs[4]), fixed step: integration, LD, SALI,
// GALI_k, Lyapunov.
#include "fput_launch.h"
namespace chs {
int try_launch_fput(const LaunchReq& rq) {
    if (FPUT_MATCH(8, WHAT_INTEGRATE, 0, 0)) return run_chain<8, 0, MODE_NONE, IND_NONE, false, 128, 4>(rq);
    if (FPUT_MATCH(8, WHAT_LD, 0, 0)) return run_chain_ld<8, 128, 4>(rq);
    if (FPUT_MATCH(8, WHAT_GALI, 4, 0)) return run_chain<8, 4, MODE_NORM, IND_GALI, false, 128, 3>(rq);
    if (FPUT_MATCH(8, WHAT_GALI, 2, 0)) return run_chain<8, 2, MODE_NORM, IND_GALI, false, 128, 4>(rq);
    if (FPUT_MATCH(8, WHAT_GALI, 3, 0)) return run_chain<8, 3, MODE_NORM, IND_GALI, false, 128, 4>(rq);
    if (FPUT_MATCH(8, WHAT_SALI, 2, 0)) return run_chain<8, 2, MODE_NORM, IND_SALI, false, 128, 4>(rq);
    if (FPUT_MATCH(8, WHAT_LYAP, 1, 0)) return run_chain<8, 1, MODE_MGS, IND_NONE, false, 128, 4>(rq);
    if (FPUT_MATCH(8, WHAT_LYAP, 2, 0)) return run_chain<8, 2, MODE_MGS, IND_NONE, false, 128, 4>(rq);
    if (FPUT_MATCH(8, WHAT_LYAP, 4, 0)) return run_chain<8, 4, MODE_MGS, IND_NONE, false, 128, 3>(rq);
    return -1;
}
}  // namespace chs
