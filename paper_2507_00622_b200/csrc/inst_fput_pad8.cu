// inst_fput_pad8.cu -- FPUT chain, any N <= 8 on the padded 8-slot tile: the basic kernel set.
#include "fput_launch.h"
namespace chs {
int try_launch_fput_pad8(const LaunchReq& rq) { return fput_basic_set<8, true>(rq); }
}  // namespace chs
