// launch.h -- host-side launch request shared by the C-ABI front end (chaoticus.cu) and the
// translation units that instantiate the kernels (inst_*.cu).  CUDA path only.
#pragma once
#include <cuda_runtime.h>
#include "col_kernels.cuh"

namespace chs {

enum : int { WHAT_INTEGRATE = 0, WHAT_SALI = 1, WHAT_GALI = 2, WHAT_LD = 3, WHAT_LYAP = 4 };

struct KernelInfo {
    int tpb, blocks, lanes, regs, spill_bytes;
};

struct LaunchReq {
    int system, what, k, adaptive;
    int fput_n;            // FPUT only: particles
    const double* params;  // host
    int n_params;
    Tab tab;
    RunArgs args;
    cudaStream_t stream;
    KernelInfo* info;  // non-null: report the launch shape, launch nothing
    // LD: which directions
    int dir_first, n_dirs;
};

// each returns -1 if it has no kernel for the request, else a cudaError_t (0 = success)
int try_launch_hh(const LaunchReq& rq);
int try_launch_hh_ind(const LaunchReq& rq);
int try_launch_hh_adapt(const LaunchReq& rq);
int try_launch_hh_adapt2(const LaunchReq& rq);
int try_launch_c3(const LaunchReq& rq);
int try_launch_c3_lyap(const LaunchReq& rq);
int try_launch_c3_more(const LaunchReq& rq);
int try_launch_dp(const LaunchReq& rq);
// FPUT: by chain length (fput_launch.h "tile classes")
int try_launch_fput8_more(const LaunchReq& rq);
int try_launch_fput8_adapt(const LaunchReq& rq);
int try_launch_fput_spec(const LaunchReq& rq);
int try_launch_fput_n4(const LaunchReq& rq);
int try_launch_fput_n8(const LaunchReq& rq);
int try_launch_fput_n16(const LaunchReq& rq);
int try_launch_fput_n32(const LaunchReq& rq);
int try_launch_fput_n64(const LaunchReq& rq);
int try_launch_fput_pad4(const LaunchReq& rq);
int try_launch_fput_pad8(const LaunchReq& rq);
int try_launch_fput_pad16(const LaunchReq& rq);
int try_launch_fput_pad32(const LaunchReq& rq);
int try_launch_fput_pad64(const LaunchReq& rq);
int try_launch_fput_wide64(const LaunchReq& rq);
int try_launch_fput_wide128(const LaunchReq& rq);
int try_launch_fput_wide256(const LaunchReq& rq);

// Common front part of every launcher: when rq.info is set, report the launch shape of `kern` and
// return 0 (or a CUDA error); otherwise return -2, meaning "go ahead and launch".
template <class Kern>
inline int finish_launch(const LaunchReq& rq, Kern kern, int tpb, int lanes, long long n_threads) {
    long long blocks = (n_threads + tpb - 1) / tpb;
    if (blocks > 2147483647LL) return (int)cudaErrorInvalidConfiguration;  // gridDim.x limit
    if (rq.info) {
        cudaFuncAttributes at;
        cudaError_t e = cudaFuncGetAttributes(&at, kern);
        if (e != cudaSuccess) return (int)e;
        *rq.info = KernelInfo{tpb, (int)blocks, lanes, at.numRegs, (int)at.localSizeBytes};
        return 0;
    }
    return -2;  // caller launches
}

// blocks of one resident wave of `kern` (lane-refill launches are persistent: DESIGN.md "Adaptive")
template <class Kern>
inline long long resident_blocks(Kern kern, int tpb) {
    int dev = 0, sms = 0, nb = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, kern, tpb, 0);
    return (long long)sms * (nb > 0 ? nb : 1);
}
// grid of a run_kernel launch: the whole ensemble, or one resident wave when a work queue is attached
template <class Kern>
inline long long run_grid(const LaunchReq& rq, Kern kern, int tpb, long long n_threads) {
    long long blocks = (n_threads + tpb - 1) / tpb;
    if (rq.adaptive && rq.args.queue != nullptr) {
        const long long res = resident_blocks(kern, tpb);
        if (res < blocks) blocks = res;
    }
    return blocks;
}

template <class Sys, int K, int L, int MODE, int IND, bool ADAPT, int TPB, int MINB, bool PAIR = true>
inline int run_col(const LaunchReq& rq) {
    typename Sys::Params prm;
    if (!Sys::make_params(rq.params, rq.n_params, prm)) return (int)cudaErrorInvalidValue;
    auto kern = run_kernel<Col<Sys, K, L>, MODE, IND, ADAPT, TPB, MINB, PAIR>;
    const long long n_threads = rq.args.n_ic * L;
    int r = finish_launch(rq, kern, TPB, L, n_threads);
    if (r != -2) return r;
    const long long blocks = run_grid(rq, kern, TPB, n_threads);
    if (blocks == 0) return 0;
    kern<<<(unsigned)blocks, TPB, 0, rq.stream>>>(rq.tab, prm, rq.args);
    return (int)cudaGetLastError();
}

template <class Sys, int TPB, int MINB>
inline int run_ld(const LaunchReq& rq) {
    typename Sys::Params prm;
    if (!Sys::make_params(rq.params, rq.n_params, prm)) return (int)cudaErrorInvalidValue;
    auto kern = ld_kernel<Col<Sys, 0, 1>, TPB, MINB>;
    const long long n_threads = rq.args.n_ic * rq.args.n_members * rq.n_dirs;
    int r = finish_launch(rq, kern, TPB, 1, n_threads);
    if (r != -2) return r;
    const long long blocks = (n_threads + TPB - 1) / TPB;
    if (blocks == 0) return 0;
    kern<<<(unsigned)blocks, TPB, 0, rq.stream>>>(rq.tab, prm, rq.args, rq.dir_first, rq.n_dirs);
    return (int)cudaGetLastError();
}

// adaptive Lagrangian descriptor (run_kernel<..., LD = true>): tasks = (direction, IC) pairs
template <class C, class Params, int TPB, int MINB>
inline int launch_ld_adapt(const LaunchReq& rq, const Params& prm) {
    auto kern = run_kernel<C, MODE_NONE, IND_NONE, true, TPB, MINB, true, true>;
    const long long n_threads = rq.args.n_ic * rq.args.n_dirs * C::L;
    int r = finish_launch(rq, kern, TPB, C::L, n_threads);
    if (r != -2) return r;
    const long long blocks = run_grid(rq, kern, TPB, n_threads);
    if (blocks == 0) return 0;
    kern<<<(unsigned)blocks, TPB, 0, rq.stream>>>(rq.tab, prm, rq.args);
    return (int)cudaGetLastError();
}
template <class Sys, int TPB, int MINB>
inline int run_col_ld_adapt(const LaunchReq& rq) {
    typename Sys::Params prm;
    if (!Sys::make_params(rq.params, rq.n_params, prm)) return (int)cudaErrorInvalidValue;
    return launch_ld_adapt<Col<Sys, 0, 1>, typename Sys::Params, TPB, MINB>(rq, prm);
}

#define CHS_MATCH(SYSID, WHAT, KK, AD) (rq.system == (SYSID) && rq.what == (WHAT) && rq.k == (KK) && rq.adaptive == (AD))

}  // namespace chs
