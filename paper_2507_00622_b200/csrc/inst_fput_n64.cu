// inst_fput_n64.cu -- FPUT chain, N = 64 exactly: the basic kernel set (fput_launch.h).
#include "fput_launch.h"
namespace chs {
int try_launch_fput_n64(const LaunchReq& rq) { return fput_basic_set<64, false>(rq); }
}  // namespace chs
