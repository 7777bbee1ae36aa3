// inst_fput_n16.cu -- FPUT chain, N = 16 (tile of 16 lanes per trajectory): the basic kernel set.
#include "fput_launch.h"
namespace chs {
int try_launch_fput_n16(const LaunchReq& rq) {
    FPUT_BASIC_SET(16)
    return -1;
}
}  // namespace chs
