// inst_fput_pad32.cu -- FPUT chain, any N <= 32 on the padded 32-slot tile: the basic kernel set.
#include "fput_launch.h"
namespace chs {
int try_launch_fput_pad32(const LaunchReq& rq) { return fput_basic_set<32, true>(rq); }
}  // namespace chs
