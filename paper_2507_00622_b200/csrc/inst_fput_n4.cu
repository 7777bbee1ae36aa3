// inst_fput_n4.cu -- FPUT chain, N = 4 exactly: the basic kernel set (fput_launch.h).
#include "fput_launch.h"
namespace chs {
int try_launch_fput_n4(const LaunchReq& rq) { return fput_basic_set<4, false>(rq); }
}  // namespace chs
