// inst_fput_n32.cu -- FPUT chain, N = 32 (tile of 32 lanes per trajectory): the basic kernel set.
#include "fput_launch.h"
namespace chs {
int try_launch_fput_n32(const LaunchReq& rq) {
    FPUT_BASIC_SET(32)
    return -1;
}
}  // namespace chs
