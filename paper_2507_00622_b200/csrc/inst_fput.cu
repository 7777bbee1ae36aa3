// inst_fput.cu -- FPUT chain, N = 8 (BASELINE configs[4]): integration, GALI_k, SALI, Lyapunov.
#include "launch.h"
#include "chain_kernels.cuh"
namespace chs {
namespace {
template <int NP, int K, int MODE, int IND, bool ADAPT, int TPB, int MINB>
int run_chain(const LaunchReq& rq) {
    if (rq.n_params < 4) return (int)cudaErrorInvalidValue;
    FputParams prm{rq.params[1], rq.params[2], rq.params[3], 2.0 * rq.params[2], 3.0 * rq.params[3]};
    auto kern = run_kernel<Chain<NP, K>, MODE, IND, ADAPT, TPB, MINB>;
    const long long n_threads = rq.args.n_ic * NP;
    int r = finish_launch(rq, kern, TPB, NP, n_threads);
    if (r != -2) return r;
    const long long blocks = (n_threads + TPB - 1) / TPB;
    if (blocks == 0) return 0;
    kern<<<(unsigned)blocks, TPB, 0, rq.stream>>>(rq.tab, prm, rq.args);
    return (int)cudaGetLastError();
}
}  // namespace
#define FPUT_MATCH(NP, WHAT, KK, AD) (rq.system == 2 && rq.fput_n == (NP) && rq.what == (WHAT) && rq.k == (KK) && rq.adaptive == (AD))
int try_launch_fput(const LaunchReq& rq) {
    if (FPUT_MATCH(8, WHAT_INTEGRATE, 0, 0)) return run_chain<8, 0, MODE_NONE, IND_NONE, false, 128, 4>(rq);
    if (FPUT_MATCH(8, WHAT_INTEGRATE, 0, 1)) return run_chain<8, 0, MODE_NONE, IND_NONE, true, 128, 4>(rq);
    if (FPUT_MATCH(8, WHAT_GALI, 4, 0)) return run_chain<8, 4, MODE_NORM, IND_GALI, false, 128, 3>(rq);
    if (FPUT_MATCH(8, WHAT_GALI, 4, 1)) return run_chain<8, 4, MODE_NORM, IND_GALI, true, 128, 2>(rq);
    if (FPUT_MATCH(8, WHAT_GALI, 2, 0)) return run_chain<8, 2, MODE_NORM, IND_GALI, false, 128, 4>(rq);
    if (FPUT_MATCH(8, WHAT_GALI, 3, 0)) return run_chain<8, 3, MODE_NORM, IND_GALI, false, 128, 4>(rq);
    if (FPUT_MATCH(8, WHAT_SALI, 2, 0)) return run_chain<8, 2, MODE_NORM, IND_SALI, false, 128, 4>(rq);
    if (FPUT_MATCH(8, WHAT_LYAP, 1, 0)) return run_chain<8, 1, MODE_MGS, IND_NONE, false, 128, 4>(rq);
    if (FPUT_MATCH(8, WHAT_LYAP, 4, 0)) return run_chain<8, 4, MODE_MGS, IND_NONE, false, 128, 3>(rq);
    return -1;
}
}  // namespace chs
