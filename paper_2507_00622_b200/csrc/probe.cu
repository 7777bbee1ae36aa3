// probe.cu -- FP64 FMA peak microbenchmark: 16 independent register-only
// DFMA chains per thread.  MEASUREMENT AID, not part of the product: built into its own library
// (libchaoticus_probe.so, paper_2507_00622_b200/probe.py), used by bench.py only.
// mode 0: x = fma(x, a, b), a and b fixed registers (operand-reuse friendly: the pipe's ceiling)
// mode 1: x = fma(C[i], x, b): multiplier from the constant bank (a kernel parameter), as the
//         step kernels read the tableau
// mode 2: x_i = fma(x_i, y_i, z_i) with three distinct register operands per DFMA (register-file
//         bandwidth / bank conflicts included)
#include <cuda_runtime.h>
#include "gen_kernels.cuh"  // fast_sincos; brings dop8_core.cuh: fast_sqrt, fast_rsqrt, fast_rcp
namespace {
struct PC { double c[16]; };
template <int MODE>
__global__ void __launch_bounds__(256, 2) dfma_probe_kernel(long long iters, double* out, const __grid_constant__ PC pc) {
    double x[16], y[16], z[16];
    const double a = 1.0 - 1e-9, b = 1e-9 * (double)(threadIdx.x & 7);
#pragma unroll
    for (int i = 0; i < 16; i++) {
        x[i] = (double)(i + 1) + (double)threadIdx.x * 1e-3;
        y[i] = 1.0 - 1e-9 * (double)(i + (threadIdx.x & 3));
        z[i] = 1e-9 * (double)(i + (threadIdx.x & 7));
    }
    for (long long it = 0; it < iters; it++) {
#pragma unroll
        for (int i = 0; i < 16; i++) {
            if (MODE == 0) x[i] = fma(x[i], a, b);
            if (MODE == 1) x[i] = fma(pc.c[i], x[i], b);
            if (MODE == 2) x[i] = fma(x[i], y[i], z[(i + 5) & 15]);
        }
    }
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < 16; i++) s += x[i] + (MODE == 2 ? y[i] + z[i] : 0.0);
    out[(long long)blockIdx.x * blockDim.x + threadIdx.x] = s;
}
}  // namespace
// n_blocks x n_threads threads x iters x 16 DFMA each; out DEVICE [n_blocks*n_threads] keeps the work
// alive.  Returns 0, 1 (bad argument) or 3 (CUDA error).
extern "C" int chs_probe_dfma(int mode, long long iters, int n_blocks, int n_threads, double* out, void* stream) {
    if (iters < 0 || n_blocks < 1 || n_threads < 1 || n_threads > 256 || !out || mode < 0 || mode > 2) return 1;
    PC pc;
    for (int i = 0; i < 16; i++) pc.c[i] = 1.0 - 1e-9 * (i + 1);
    cudaStream_t st = (cudaStream_t)stream;
    if (mode == 0) dfma_probe_kernel<0><<<n_blocks, n_threads, 0, st>>>(iters, out, pc);
    if (mode == 1) dfma_probe_kernel<1><<<n_blocks, n_threads, 0, st>>>(iters, out, pc);
    if (mode == 2) dfma_probe_kernel<2><<<n_blocks, n_threads, 0, st>>>(iters, out, pc);
    return cudaGetLastError() == cudaSuccess ? 0 : 3;
}

// ---- the device math helpers, one value per thread (TEST AID: tests/test_gpu_math_helpers.py measures their
// error against the host's long double; the step kernels inline the same functions) -------------------------
namespace {
__global__ void math_probe_kernel(int which, long long n, const double* __restrict__ x, double* __restrict__ o1,
                                  double* __restrict__ o2) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const double v = x[i];
    if (which == 0) o1[i] = chs::fast_sqrt(v);
    else if (which == 1) o1[i] = chs::fast_rsqrt(v);
    else if (which == 2) o1[i] = chs::fast_rcp(v);
    else {
        double sn, cs;
        chs::fast_sincos(v, &sn, &cs);
        o1[i] = sn;
        o2[i] = cs;
    }
}
}  // namespace
// which: 0 fast_sqrt, 1 fast_rsqrt, 2 fast_rcp, 3 fast_sincos (out2 = cos; otherwise out2 is not used).
// x, out1, out2 DEVICE [n].  Returns 0, 1 (bad argument) or 3 (CUDA error).
extern "C" int chs_probe_math(int which, long long n, const double* x, double* out1, double* out2, void* stream) {
    if (which < 0 || which > 3 || n < 0 || (n > 0 && (!x || !out1 || (which == 3 && !out2)))) return 1;
    if (n == 0) return 0;
    const long long blocks = (n + 255) / 256;
    if (blocks > 2147483647LL) return 1;
    math_probe_kernel<<<(unsigned)blocks, 256, 0, (cudaStream_t)stream>>>(which, n, x, out1, out2);
    return cudaGetLastError() == cudaSuccess ? 0 : 3;
}
