// fput_launch.h -- launchers of the chain-layout kernels (FPUT), shared by inst_fput*.cu.
//
// Tile classes: a chain of N particles runs on the smallest class that holds it.
//   in-warp  NS = 4, 8, 16, 32, 64 slots: fixed-step kernels on NS/2 lanes x 2 particles per lane; the
//            Lyapunov k = 4 and adaptive GALI_4 kernels (more registers per pair) on NS lanes x 1, NS <= 32;
//   wide     64, 128, 256 slots: one particle per thread, the tile is a thread block of that many threads
//            (chain_kernels.cuh "wide tiles").
// PAD = false: N == NS exactly; PAD = true: any N <= NS, padded with particles pinned at zero.
#pragma once
#include "launch.h"
#include "chain_kernels.cuh"
namespace chs {
inline bool fput_params(const LaunchReq& rq, FputParams& prm) {
    if (rq.n_params < 4) return false;
    prm = FputParams{rq.params[1], rq.params[2], rq.params[3], 2.0 * rq.params[2], 3.0 * rq.params[3], rq.fput_n};
    return true;
}
template <int LT, int PPL, bool PAD, int K, int MODE, int IND, bool ADAPT, int TPB, int MINB, bool COLD = false>
int run_chain_t(const LaunchReq& rq) {
    static_assert(LT <= 32 || LT == TPB, "a wide tile is the whole thread block");
    FputParams prm;
    if (!fput_params(rq, prm)) return (int)cudaErrorInvalidValue;
    if (rq.fput_n > LT * PPL || (!PAD && rq.fput_n != LT * PPL)) return (int)cudaErrorInvalidValue;
    auto kern = run_kernel<Chain<LT, PPL, K, PAD, COLD>, MODE, IND, ADAPT, TPB, MINB>;
    const long long n_threads = rq.args.n_ic * LT;
    int r = finish_launch(rq, kern, TPB, LT, n_threads);
    if (r != -2) return r;
    const long long blocks = run_grid(rq, kern, TPB, n_threads);
    if (blocks == 0) return 0;
    kern<<<(unsigned)blocks, TPB, 0, rq.stream>>>(rq.tab, prm, rq.args);
    return (int)cudaGetLastError();
}
template <int LT, int PPL, bool PAD, int TPB, int MINB>
int run_chain_ld_t(const LaunchReq& rq) {
    static_assert(LT <= 32 || LT == TPB, "a wide tile is the whole thread block");
    FputParams prm;
    if (!fput_params(rq, prm)) return (int)cudaErrorInvalidValue;
    if (rq.fput_n > LT * PPL || (!PAD && rq.fput_n != LT * PPL)) return (int)cudaErrorInvalidValue;
    auto kern = ld_kernel<Chain<LT, PPL, 0, PAD>, TPB, MINB>;
    const long long n_threads = rq.args.n_ic * rq.args.n_members * rq.n_dirs * LT;
    int r = finish_launch(rq, kern, TPB, LT, n_threads);
    if (r != -2) return r;
    const long long blocks = (n_threads + TPB - 1) / TPB;
    if (blocks == 0) return 0;
    kern<<<(unsigned)blocks, TPB, 0, rq.stream>>>(rq.tab, prm, rq.args, rq.dir_first, rq.n_dirs);
    return (int)cudaGetLastError();
}

template <int LT, int PPL, bool PAD, int TPB, int MINB>
int run_chain_ld_adapt_t(const LaunchReq& rq) {
    static_assert(LT <= 32 || LT == TPB, "a wide tile is the whole thread block");
    FputParams prm;
    if (!fput_params(rq, prm)) return (int)cudaErrorInvalidValue;
    if (rq.fput_n > LT * PPL || (!PAD && rq.fput_n != LT * PPL)) return (int)cudaErrorInvalidValue;
    return launch_ld_adapt<Chain<LT, PPL, 0, PAD>, FputParams, TPB, MINB>(rq, prm);
}

// Lyapunov spectrum with NB K vectors on NB column blocks (chain_kernels.cuh): fixed step, Gram-Schmidt
template <int LT, int PPL, bool PAD, int KB, int NB, int TPB, int MINB, bool COLD = false>
int run_chain_blocks(const LaunchReq& rq) {
    FputParams prm;
    if (!fput_params(rq, prm)) return (int)cudaErrorInvalidValue;
    if (rq.fput_n > LT * PPL || (!PAD && rq.fput_n != LT * PPL)) return (int)cudaErrorInvalidValue;
    using C = Chain<LT, PPL, KB, PAD, COLD, NB>;
    auto kern = run_kernel<C, MODE_MGS, IND_NONE, false, TPB, MINB>;
    const long long n_threads = rq.args.n_ic * C::L;
    int r = finish_launch(rq, kern, TPB, C::L, n_threads);
    if (r != -2) return r;
    const long long blocks = (n_threads + TPB - 1) / TPB;
    if (blocks == 0) return 0;
    kern<<<(unsigned)blocks, TPB, 0, rq.stream>>>(rq.tab, prm, rq.args);
    return (int)cudaGetLastError();
}

// the kernel set every tile class has: integration (fixed, adaptive), LD, SALI, GALI_4 (fixed, adaptive),
// Lyapunov k = 4.  Returns -1 for anything else.
template <int NS, bool PAD>
int fput_basic_set(const LaunchReq& rq) {
    constexpr int H = NS / 2;
    const int w = rq.what, k = rq.k;
    const bool ad = rq.adaptive != 0;
    if (w == WHAT_INTEGRATE && k == 0 && !ad) return run_chain_t<H, 2, PAD, 0, MODE_NONE, IND_NONE, false, 128, 4>(rq);
    if (w == WHAT_INTEGRATE && k == 0 && ad) return run_chain_t<H, 2, PAD, 0, MODE_NONE, IND_NONE, true, 128, 2>(rq);
    if (w == WHAT_LD && k == 0 && !ad) return run_chain_ld_t<H, 2, PAD, 128, 4>(rq);
    if (w == WHAT_LD && k == 0 && ad) return run_chain_ld_adapt_t<H, 2, PAD, 128, 2>(rq);
    if (w == WHAT_SALI && k == 2 && !ad) return run_chain_t<H, 2, PAD, 2, MODE_NORM, IND_SALI, false, 128, 2>(rq);
    // (blocks of 256, one per SM: 440 ms against 445 ms with two blocks of 128 for BASELINE configs[4])
    if (w == WHAT_GALI && k == 4 && !ad) return run_chain_t<H, 2, PAD, 4, MODE_NORM, IND_GALI, false, 256, 1, true>(rq);
    if constexpr (NS <= 32) {  // one particle per lane: these need more registers per pair
        if (w == WHAT_LYAP && k == 4 && !ad) return run_chain_t<NS, 1, PAD, 4, MODE_MGS, IND_NONE, false, 128, 2>(rq);
        if (w == WHAT_GALI && k == 4 && ad) return run_chain_t<NS, 1, PAD, 4, MODE_NORM, IND_GALI, true, 128, 2>(rq);
    }
    return -1;
}
// the same set on a wide tile of TPB threads (any N <= TPB)
template <int TPB, int MINB>
int fput_wide_set(const LaunchReq& rq) {
    const int w = rq.what, k = rq.k;
    const bool ad = rq.adaptive != 0;
    if (w == WHAT_INTEGRATE && k == 0 && !ad) return run_chain_t<TPB, 1, true, 0, MODE_NONE, IND_NONE, false, TPB, MINB>(rq);
    if (w == WHAT_INTEGRATE && k == 0 && ad) return run_chain_t<TPB, 1, true, 0, MODE_NONE, IND_NONE, true, TPB, MINB>(rq);
    if (w == WHAT_LD && k == 0 && !ad) return run_chain_ld_t<TPB, 1, true, TPB, MINB>(rq);
    if (w == WHAT_LD && k == 0 && ad) return run_chain_ld_adapt_t<TPB, 1, true, TPB, MINB>(rq);
    if (w == WHAT_SALI && k == 2 && !ad) return run_chain_t<TPB, 1, true, 2, MODE_NORM, IND_SALI, false, TPB, MINB>(rq);
    if (w == WHAT_GALI && k == 4 && !ad) return run_chain_t<TPB, 1, true, 4, MODE_NORM, IND_GALI, false, TPB, MINB>(rq);
    if (w == WHAT_GALI && k == 4 && ad) return run_chain_t<TPB, 1, true, 4, MODE_NORM, IND_GALI, true, TPB, 1>(rq);
    if (w == WHAT_LYAP && k == 4 && !ad) return run_chain_t<TPB, 1, true, 4, MODE_MGS, IND_NONE, false, TPB, MINB>(rq);
    return -1;
}
}  // namespace chs
