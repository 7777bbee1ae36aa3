// inst_dp.cu -- dimensionless double pendulum: generic first-order kernel,
// fixed-step and adaptive integration (the workload of the paper's Fig. 1) and the
// Lagrangian descriptor (the indicator that needs no variational equations).
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
}  // namespace
int try_launch_dp(const LaunchReq& rq) {
    if (CHS_MATCH(3, WHAT_INTEGRATE, 0, 0)) return run_gen<DoublePendulum, false, 128, 3>(rq);
    if (CHS_MATCH(3, WHAT_INTEGRATE, 0, 1)) return run_gen<DoublePendulum, true, 128, 3>(rq);
    if (CHS_MATCH(3, WHAT_LD, 0, 0)) return run_gen_ld<DoublePendulum, 128, 3>(rq);
    return -1;
}
}  // namespace chs
