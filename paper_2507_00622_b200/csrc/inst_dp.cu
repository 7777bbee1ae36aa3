// inst_dp.cu -- dimensionless double pendulum: generic first-order kernels: fixed-step
// and adaptive integration (the workload of the paper's Fig. 1), the Lagrangian
// descriptor, and -- one column per lane -- SALI, GALI_k and the Lyapunov spectrum.
#include "launch.h"
#include "gen_kernels.cuh"
namespace chs {
namespace {
template <class Sys, bool ADAPT, int TPB, int MINB>
int run_gen(const LaunchReq& rq) {
    typename Sys::Params prm;
    if (!Sys::make_params(rq.params, rq.n_params, prm)) return (int)cudaErrorInvalidValue;
    auto kern = gen_run_kernel<Sys, ADAPT, TPB, MINB>;
    int r = finish_launch(rq, kern, TPB, 1, rq.args.n_ic);
    if (r != -2) return r;
    const long long blocks = (rq.args.n_ic + TPB - 1) / TPB;
    if (blocks == 0) return 0;
    kern<<<(unsigned)blocks, TPB, 0, rq.stream>>>(rq.tab, prm, rq.args);
    return (int)cudaGetLastError();
}
template <class Sys, int TPB, int MINB>
int run_gen_ld_adapt(const LaunchReq& rq) {
    typename Sys::Params prm;
    if (!Sys::make_params(rq.params, rq.n_params, prm)) return (int)cudaErrorInvalidValue;
    auto kern = gen_run_kernel<Sys, true, TPB, MINB, true>;
    const long long n_threads = rq.args.n_ic * rq.args.n_dirs;
    int r = finish_launch(rq, kern, TPB, 1, n_threads);
    if (r != -2) return r;
    const long long blocks = (n_threads + TPB - 1) / TPB;
    if (blocks == 0) return 0;
    kern<<<(unsigned)blocks, TPB, 0, rq.stream>>>(rq.tab, prm, rq.args);
    return (int)cudaGetLastError();
}
template <class Sys, int TPB, int MINB>
int run_gen_ld(const LaunchReq& rq) {
    typename Sys::Params prm;
    if (!Sys::make_params(rq.params, rq.n_params, prm)) return (int)cudaErrorInvalidValue;
    auto kern = gen_ld_kernel<Sys, TPB, MINB>;
    const long long n_threads = rq.args.n_ic * rq.args.n_members * rq.n_dirs;
    int r = finish_launch(rq, kern, TPB, 1, n_threads);
    if (r != -2) return r;
    const long long blocks = (n_threads + TPB - 1) / TPB;
    if (blocks == 0) return 0;
    kern<<<(unsigned)blocks, TPB, 0, rq.stream>>>(rq.tab, prm, rq.args, rq.dir_first, rq.n_dirs);
    return (int)cudaGetLastError();
}
// orbit + K deviation vectors, one column per lane of an L-lane tile (gen_kernels.cuh gen_col_kernel)
template <class Sys, int K, int L, int MODE, int IND, bool ADAPT, int TPB, int MINB>
int run_gen_col(const LaunchReq& rq) {
    typename Sys::Params prm;
    if (!Sys::make_params(rq.params, rq.n_params, prm)) return (int)cudaErrorInvalidValue;
    auto kern = gen_col_kernel<Sys, K, L, MODE, IND, ADAPT, TPB, MINB>;
    const long long n_threads = rq.args.n_ic * L;
    int r = finish_launch(rq, kern, TPB, L, n_threads);
    if (r != -2) return r;
    const long long blocks = (n_threads + TPB - 1) / TPB;
    if (blocks == 0) return 0;
    kern<<<(unsigned)blocks, TPB, 0, rq.stream>>>(rq.tab, prm, rq.args);
    return (int)cudaGetLastError();
}
}  // namespace
int try_launch_dp(const LaunchReq& rq) {
    if (CHS_MATCH(3, WHAT_INTEGRATE, 0, 0)) return run_gen<DoublePendulum, false, 128, 3>(rq);
    if (CHS_MATCH(3, WHAT_INTEGRATE, 0, 1)) return run_gen<DoublePendulum, true, 128, 3>(rq);
    if (CHS_MATCH(3, WHAT_LD, 0, 0)) return run_gen_ld<DoublePendulum, 128, 3>(rq);
    if (CHS_MATCH(3, WHAT_LD, 0, 1)) return run_gen_ld_adapt<DoublePendulum, 128, 2>(rq);
    // solvers 3-6 of PAPER.md:49-52 for the paper's first example system
    if (CHS_MATCH(3, WHAT_SALI, 2, 0)) return run_gen_col<DoublePendulum, 2, 4, MODE_NORM, IND_SALI, false, 128, 2>(rq);
    if (CHS_MATCH(3, WHAT_SALI, 2, 1)) return run_gen_col<DoublePendulum, 2, 4, MODE_NORM, IND_SALI, true, 128, 2>(rq);
    if (CHS_MATCH(3, WHAT_GALI, 2, 0)) return run_gen_col<DoublePendulum, 2, 4, MODE_NORM, IND_GALI, false, 128, 3>(rq);
    if (CHS_MATCH(3, WHAT_GALI, 3, 0)) return run_gen_col<DoublePendulum, 3, 4, MODE_NORM, IND_GALI, false, 128, 3>(rq);
    if (CHS_MATCH(3, WHAT_GALI, 4, 0)) return run_gen_col<DoublePendulum, 4, 8, MODE_NORM, IND_GALI, false, 128, 3>(rq);
    if (CHS_MATCH(3, WHAT_LYAP, 1, 0)) return run_gen_col<DoublePendulum, 1, 2, MODE_MGS, IND_NONE, false, 128, 3>(rq);
    if (CHS_MATCH(3, WHAT_LYAP, 1, 1)) return run_gen_col<DoublePendulum, 1, 2, MODE_MGS, IND_NONE, true, 128, 2>(rq);
    if (CHS_MATCH(3, WHAT_LYAP, 2, 0)) return run_gen_col<DoublePendulum, 2, 4, MODE_MGS, IND_NONE, false, 128, 3>(rq);
    if (CHS_MATCH(3, WHAT_LYAP, 4, 0)) return run_gen_col<DoublePendulum, 4, 8, MODE_MGS, IND_NONE, false, 128, 3>(rq);
    if (CHS_MATCH(3, WHAT_LYAP, 4, 1)) return run_gen_col<DoublePendulum, 4, 8, MODE_MGS, IND_NONE, true, 128, 2>(rq);
    return -1;
}
}  // namespace chs
