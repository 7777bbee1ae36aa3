// inst_fput_pad16.cu -- FPUT chain, any N <= 16 on the padded 16-slot tile: the basic kernel set.
#include "fput_launch.h"
namespace chs {
int try_launch_fput_pad16(const LaunchReq& rq) { return fput_basic_set<16, true>(rq); }
}  // namespace chs
