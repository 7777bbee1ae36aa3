// inst_fput_pad64.cu -- FPUT chain, any N <= 64 on the padded 64-slot tile: the basic kernel set.
#include "fput_launch.h"
namespace chs {
int try_launch_fput_pad64(const LaunchReq& rq) { return fput_basic_set<64, true>(rq); }
}  // namespace chs
