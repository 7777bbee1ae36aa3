// inst_fput.cu -- FPUT chain kernels (chain layout).
#include "launch.h"
namespace chs {
int try_launch_fput(const LaunchReq& rq) { (void)rq; return -1; }
}  // namespace chs
