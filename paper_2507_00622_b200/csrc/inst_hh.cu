// inst_hh.cu -- Henon-Heiles: plain fixed-step integration, Lagrangian descriptor, fixed-step SALI.
#include "launch.h"
namespace chs {
int try_launch_hh(const LaunchReq& rq) {
    if (CHS_MATCH(0, WHAT_INTEGRATE, 0, 0)) return run_col<HenonHeiles, 0, 1, MODE_NONE, IND_NONE, false, 128, 4>(rq);
    if (CHS_MATCH(0, WHAT_LD, 0, 0)) return run_ld<HenonHeiles, 128, 7>(rq);
    if (CHS_MATCH(0, WHAT_SALI, 2, 0)) {
        // small ensembles cannot fill the GPU with one thread per trajectory: up to 4096
        // trajectories a 4-lane tile per trajectory (orbit, w1, w2, idle) shortens each lane's dependent
        // chain: 6.4 ms against 8.7 ms for configs[0] (1024 ICs x 10^4 steps); beyond ~6000 trajectories
        // the thread-per-trajectory kernel (no idle lane) is the faster one
        if (rq.args.n_ic <= 4096) return run_col<HenonHeiles, 2, 4, MODE_NORM, IND_SALI, false, 128, 4>(rq);
        return run_col<HenonHeiles, 2, 1, MODE_NORM, IND_SALI, false, 128, 1>(rq);
    }
    return -1;
}
}  // namespace chs
