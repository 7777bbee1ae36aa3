// inst_fput_pad4.cu -- FPUT chain, any N <= 4 on the padded 4-slot tile: the basic kernel set.
#include "fput_launch.h"
namespace chs {
int try_launch_fput_pad4(const LaunchReq& rq) { return fput_basic_set<4, true>(rq); }
}  // namespace chs
