// inst_fput_n4.cu -- FPUT chain, N = 4 (tile of 4 lanes per trajectory): the basic kernel set.
#include "fput_launch.h"
namespace chs {
int try_launch_fput_n4(const LaunchReq& rq) {
    FPUT_BASIC_SET(4)
    return -1;
}
}  // namespace chs
