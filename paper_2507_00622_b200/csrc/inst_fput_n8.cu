// inst_fput_n8.cu -- FPUT chain, N = 8 exactly: the basic kernel set (fput_launch.h).
#include "fput_launch.h"
namespace chs {
int try_launch_fput_n8(const LaunchReq& rq) { return fput_basic_set<8, false>(rq); }
}  // namespace chs
