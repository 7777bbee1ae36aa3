// inst_fput_n32.cu -- FPUT chain, N = 32 exactly: the basic kernel set (fput_launch.h).
#include "fput_launch.h"
namespace chs {
int try_launch_fput_n32(const LaunchReq& rq) { return fput_basic_set<32, false>(rq); }
}  // namespace chs
