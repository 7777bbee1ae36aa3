// inst_fput_n16.cu -- FPUT chain, N = 16 exactly: the basic kernel set (fput_launch.h).
#include "fput_launch.h"
namespace chs {
int try_launch_fput_n16(const LaunchReq& rq) { return fput_basic_set<16, false>(rq); }
}  // namespace chs
