// fput_launch.h -- launchers of the chain-layout kernels (FPUT), shared by inst_fput*.cu.
#pragma once
#include "launch.h"
#include "chain_kernels.cuh"
namespace chs {
inline bool fput_params(const LaunchReq& rq, FputParams& prm) {
    if (rq.n_params < 4) return false;
    prm = FputParams{rq.params[1], rq.params[2], rq.params[3], 2.0 * rq.params[2], 3.0 * rq.params[3]};
    return true;
}
template <int NP, int K, int MODE, int IND, bool ADAPT, int TPB, int MINB>
int run_chain(const LaunchReq& rq) {
    FputParams prm;
    if (!fput_params(rq, prm)) return (int)cudaErrorInvalidValue;
    auto kern = run_kernel<Chain<NP, K>, MODE, IND, ADAPT, TPB, MINB>;
    const long long n_threads = rq.args.n_ic * NP;
    int r = finish_launch(rq, kern, TPB, NP, n_threads);
    if (r != -2) return r;
    const long long blocks = run_grid(rq, kern, TPB, n_threads);
    if (blocks == 0) return 0;
    kern<<<(unsigned)blocks, TPB, 0, rq.stream>>>(rq.tab, prm, rq.args);
    return (int)cudaGetLastError();
}
template <int NP, int TPB, int MINB>
int run_chain_ld(const LaunchReq& rq) {
    FputParams prm;
    if (!fput_params(rq, prm)) return (int)cudaErrorInvalidValue;
    auto kern = ld_kernel<Chain<NP, 0>, TPB, MINB>;
    const long long n_threads = rq.args.n_ic * rq.n_dirs * NP;
    int r = finish_launch(rq, kern, TPB, NP, n_threads);
    if (r != -2) return r;
    const long long blocks = (n_threads + TPB - 1) / TPB;
    if (blocks == 0) return 0;
    kern<<<(unsigned)blocks, TPB, 0, rq.stream>>>(rq.tab, prm, rq.args, rq.dir_first, rq.n_dirs);
    return (int)cudaGetLastError();
}
#define FPUT_MATCH(NP, WHAT, KK, AD) \
    (rq.system == 2 && rq.fput_n == (NP) && rq.what == (WHAT) && rq.k == (KK) && rq.adaptive == (AD))
// the kernel set compiled for the other chain lengths (N = 4, 16, 32)
#define FPUT_BASIC_SET(NP)                                                                                          \
    if (FPUT_MATCH(NP, WHAT_INTEGRATE, 0, 0)) return run_chain<NP, 0, MODE_NONE, IND_NONE, false, 128, 4>(rq);      \
    if (FPUT_MATCH(NP, WHAT_INTEGRATE, 0, 1)) return run_chain<NP, 0, MODE_NONE, IND_NONE, true, 128, 4>(rq);       \
    if (FPUT_MATCH(NP, WHAT_LD, 0, 0)) return run_chain_ld<NP, 128, 4>(rq);                                         \
    if (FPUT_MATCH(NP, WHAT_SALI, 2, 0)) return run_chain<NP, 2, MODE_NORM, IND_SALI, false, 128, 4>(rq);           \
    if (FPUT_MATCH(NP, WHAT_GALI, 4, 0)) return run_chain<NP, 4, MODE_NORM, IND_GALI, false, 128, 3>(rq);           \
    if (FPUT_MATCH(NP, WHAT_GALI, 4, 1)) return run_chain<NP, 4, MODE_NORM, IND_GALI, true, 128, 2>(rq);            \
    if (FPUT_MATCH(NP, WHAT_LYAP, 4, 0)) return run_chain<NP, 4, MODE_MGS, IND_NONE, false, 128, 3>(rq);
}  // namespace chs
