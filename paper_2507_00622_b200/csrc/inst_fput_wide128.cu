// inst_fput_wide128.cu -- FPUT chain, any N <= 128 on a wide tile: one particle per thread, one trajectory
// per block of 128 threads (chain_kernels.cuh): the basic kernel set.
#include "fput_launch.h"
namespace chs {
int try_launch_fput_wide128(const LaunchReq& rq) { return fput_wide_set<128, 2>(rq); }
}  // namespace chs
