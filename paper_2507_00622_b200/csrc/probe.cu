// probe.cu -- FP64 FMA peak microbenchmark (include/chaoticus.h chaoticus_dfma_probe;
// DESIGN.md "Roofline"): 16 independent register-only DFMA chains per thread.
#include <cuda_runtime.h>
#include "../../include/chaoticus.h"
namespace {
__global__ void __launch_bounds__(256, 2) dfma_probe_kernel(long long iters, double* out) {
    double x[16];
    const double a = 1.0 - 1e-9, b = 1e-9 * (double)(threadIdx.x & 7);
#pragma unroll
    for (int i = 0; i < 16; i++) x[i] = (double)(i + 1) + (double)threadIdx.x * 1e-3;
    for (long long it = 0; it < iters; it++) {
#pragma unroll
        for (int i = 0; i < 16; i++) x[i] = fma(x[i], a, b);
    }
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < 16; i++) s += x[i];
    out[(long long)blockIdx.x * blockDim.x + threadIdx.x] = s;
}
}  // namespace
extern "C" int chaoticus_dfma_probe(long long iters, int n_blocks, int n_threads, double* out, void* stream) {
    if (iters < 0 || n_blocks < 1 || n_threads < 1 || n_threads > 256 || !out) return CHS_EINVAL;
    dfma_probe_kernel<<<n_blocks, n_threads, 0, (cudaStream_t)stream>>>(iters, out);
    return cudaGetLastError() == cudaSuccess ? CHS_OK : CHS_ECUDA;
}
