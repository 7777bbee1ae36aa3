// inst_fput_spec.cu -- FPUT chain, Lyapunov spectra with more vectors than one lane holds (PAPER.md:113:
// the spectrum "following a very similar approach to the GALI_k computation ... using QR factorization"):
// column blocks of 4 vectors on adjacent sub-tiles (chain_kernels.cuh).  Full spectra k = 2N for N = 4, 8;
// k = 8 for N = 8, 16.  Fixed step.
#include "fput_launch.h"
namespace chs {
int try_launch_fput_spec(const LaunchReq& rq) {
    if (rq.what != WHAT_LYAP || rq.adaptive) return -1;
    const int N = rq.fput_n, k = rq.k;
    if (N == 4 && k == 8) return run_chain_blocks<4, 1, false, 4, 2, 128, 2>(rq);    //  8 lanes per trajectory
    if (N == 8 && k == 8) return run_chain_blocks<8, 1, false, 4, 2, 128, 2>(rq);    // 16 lanes
    if (N == 8 && k == 16) return run_chain_blocks<8, 1, false, 4, 4, 128, 2>(rq);   // a full warp
    if (N == 16 && k == 8) return run_chain_blocks<16, 1, false, 4, 2, 128, 2>(rq);  // a full warp
    return -1;
}
}  // namespace chs
