// inst_fput_wide256.cu -- FPUT chain, any N <= 256 on a wide tile: one particle per thread, one trajectory
// per block of 256 threads (chain_kernels.cuh): the basic kernel set.
#include "fput_launch.h"
namespace chs {
int try_launch_fput_wide256(const LaunchReq& rq) { return fput_wide_set<256, 1>(rq); }
}  // namespace chs
