// inst_fput_wide64.cu -- FPUT chain, any N <= 64 on a wide tile: one particle per thread, one trajectory
// per block of 64 threads (chain_kernels.cuh): the basic kernel set.
#include "fput_launch.h"
namespace chs {
int try_launch_fput_wide64(const LaunchReq& rq) { return fput_wide_set<64, 4>(rq); }
}  // namespace chs
