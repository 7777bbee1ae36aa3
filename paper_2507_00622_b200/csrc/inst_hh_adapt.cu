// inst_hh_adapt.cu -- Henon-Heiles, adaptive DOP8(5): plain integration, Lagrangian descriptor, SALI, GALI_k,
// Lyapunov.
#include "launch.h"
namespace chs {
int try_launch_hh_adapt(const LaunchReq& rq) {
    if (CHS_MATCH(0, WHAT_INTEGRATE, 0, 1)) return run_col<HenonHeiles, 0, 1, MODE_NONE, IND_NONE, true, 128, 4>(rq);
    if (CHS_MATCH(0, WHAT_LD, 0, 1)) return run_col_ld_adapt<HenonHeiles, 128, 3>(rq);
    if (CHS_MATCH(0, WHAT_SALI, 2, 1)) {
        // small ensembles: 4-lane tile per trajectory, as for the fixed-step kernel (inst_hh.cu)
        if (rq.args.n_ic <= 4096) return run_col<HenonHeiles, 2, 4, MODE_NORM, IND_SALI, true, 128, 3>(rq);
        return run_col<HenonHeiles, 2, 1, MODE_NORM, IND_SALI, true, 128, 1>(rq);
    }
    if (CHS_MATCH(0, WHAT_GALI, 2, 1)) return run_col<HenonHeiles, 2, 4, MODE_NORM, IND_GALI, true, 128, 3>(rq);  // (one thread per trajectory would spill)
    if (CHS_MATCH(0, WHAT_LYAP, 1, 1)) return run_col<HenonHeiles, 1, 1, MODE_MGS, IND_NONE, true, 128, 2>(rq);
    if (CHS_MATCH(0, WHAT_LYAP, 2, 1)) return run_col<HenonHeiles, 2, 1, MODE_MGS, IND_NONE, true, 128, 1>(rq);
    return -1;
}
}  // namespace chs
