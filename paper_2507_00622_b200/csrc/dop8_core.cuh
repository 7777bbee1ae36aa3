// dop8_core.cuh -- the DOP8 step in separable form, layout-agnostic (CUDA path, sm_100a).
//
// PAPER.md:43 ("the 8th order ODE solver given in [51]"), PAPER.md:47-53 (fixed "DOP 8",
// adaptive "DOP 8(5)", per-step error).  DESIGN.md "Separable form":
// every system on the path has H = |p|^2/2 + V(q), so the q-half of every stage derivative is
// the p-stage value and is never stored.  A lane holds NI independent (q, p) component pairs
// ("items": orbit coordinates and/or deviation-vector coordinates); the only coupling between
// items is inside the force functor.  With F_l = force(Q_l):
//     Q_i = q + cs_i h p + h^2 sum_l A2_il F_l,   q+ = q + h p + h^2 sum_l BQ_l F_l,
//     p+ = p + h sum_l B_l F_l.
// All stage loops are compile-time (static_for over integral constants) so that state and
// stage forces live in registers and structural zeros of the tableau cost nothing.
#pragma once
#include <cuda_runtime.h>
#include <type_traits>
#include "dop8_coeffs.h"

namespace chs {

template <int I> using Int = std::integral_constant<int, I>;

template <int B, int E, class F>
__device__ __forceinline__ void static_for(F&& f) {
    if constexpr (B < E) {
        f(Int<B>{});
        static_for<B + 1, E>(f);
    }
}

// Coefficients as the kernels read them (a __grid_constant__ kernel parameter, i.e. constant
// bank operands of the DFMAs).  Fixed step: premultiplied by powers of h on the host.
// Adaptive: raw (h = 1) and the per-trajectory h is applied in registers.
struct Tab {
    double a2[12][12];  // h^2 A2
    double ap[12][12];  // h A           (P stages; Lagrangian descriptor only)
    double cs[12];      // h rowsum(A)
    double bq[12];      // h^2 b^T A
    double bp[12];      // h b
    double bl[12];      // |h| b         (LD quadrature weights)
    double e5q[12], e3q[12];  // (adaptive, raw) E5^T A, E3^T A
    double e5p[12], e3p[12];  // (adaptive, raw) E5, E3
    double d3[12];            // (adaptive, raw) b - E3: non-zero at stages 1, 9 and 12 only
    double h;                 // signed step (fixed) or 1
};

// ---- tile helpers: a trajectory is owned by a tile of L consecutive threads -------------------------
// L = 1, 2, 4, 8, 16, 32: lanes of one warp, shuffles.  L > 32 (wide chains): the tile is the WHOLE thread
// block (L == blockDim.x, one trajectory per block); the same operations go through shared memory and
// __syncthreads, and every thread of the block must reach them (run_kernel's control flow is uniform per
// trajectory, hence per block).  All results are bit-identical on every thread of the tile.
template <int L>
__device__ __forceinline__ double tile_bcast(double x, int src_lane_in_tile) {
    if constexpr (L == 1) return x;
    else if constexpr (L <= 32) return __shfl_sync(0xffffffffu, x, src_lane_in_tile, L);
    else {
        __shared__ double box;
        if ((int)threadIdx.x == src_lane_in_tile) box = x;
        __syncthreads();
        const double r = box;
        __syncthreads();
        return r;
    }
}
template <int L>
__device__ __forceinline__ long long tile_bcast_ll(long long x, int src_lane_in_tile) {
    if constexpr (L == 1) return x;
    else if constexpr (L <= 32) return __shfl_sync(0xffffffffu, x, src_lane_in_tile, L);
    else {
        __shared__ long long box;
        if ((int)threadIdx.x == src_lane_in_tile) box = x;
        __syncthreads();
        const long long r = box;
        __syncthreads();
        return r;
    }
}
template <int L>
__device__ __forceinline__ double tile_sum(double x) {  // butterfly: identical on all lanes
    if constexpr (L > 1 && L <= 32) {
#pragma unroll
        for (int d = L / 2; d >= 1; d >>= 1) x += __shfl_xor_sync(0xffffffffu, x, d, L);
    } else if constexpr (L > 32) {
        __shared__ double part[L / 32];
#pragma unroll
        for (int d = 16; d >= 1; d >>= 1) x += __shfl_xor_sync(0xffffffffu, x, d, 32);
        part[threadIdx.x >> 5] = x;  // every lane of a warp holds the same sum: no lane is special, no branch
        __syncthreads();
        x = part[0];
#pragma unroll
        for (int w = 1; w < L / 32; w++) x += part[w];  // same order on every thread
        __syncthreads();
    }
    return x;
}
// NV sums at once (renormalisation: the K squared norms; adaptive step: S5 and S3): the wide tile pays its
// two barriers once instead of NV times; in-warp tiles: NV independent butterflies
template <int L, int NV>
__device__ __forceinline__ void tile_sum_vec(double (&x)[NV]) {
    if constexpr (L <= 32) {
#pragma unroll
        for (int v = 0; v < NV; v++) x[v] = tile_sum<L>(x[v]);
    } else {
        __shared__ double part[NV][L / 32];
#pragma unroll
        for (int v = 0; v < NV; v++) {
#pragma unroll
            for (int d = 16; d >= 1; d >>= 1) x[v] += __shfl_xor_sync(0xffffffffu, x[v], d, 32);
            part[v][threadIdx.x >> 5] = x[v];
        }
        __syncthreads();
#pragma unroll
        for (int v = 0; v < NV; v++) {
            double t = part[v][0];
#pragma unroll
            for (int w = 1; w < L / 32; w++) t += part[v][w];
            x[v] = t;
        }
        __syncthreads();
    }
}
template <int L>
__device__ __forceinline__ bool tile_any(bool b) {
    if constexpr (L == 1) return b;
    else if constexpr (L <= 32) {
        unsigned m = __ballot_sync(0xffffffffu, b);
        unsigned lane = threadIdx.x & 31u;
        unsigned tmask = (L == 32) ? 0xffffffffu : (((1u << L) - 1u) << (lane & ~(unsigned)(L - 1)));
        return (m & tmask) != 0u;
    } else {
        return __syncthreads_or(b ? 1 : 0) != 0;
    }
}
// "does any thread that shares my control flow want this?": a warp for in-warp tiles, the block for wide ones
template <int L>
__device__ __forceinline__ bool group_any(bool b) {
    if constexpr (L <= 32) return __any_sync(0xffffffffu, b);
    else return __syncthreads_or(b ? 1 : 0) != 0;
}

// ---- where a fixed-step trajectory died (oracle: run_traj tests the state after every step and stops at the
// first non-finite one; n_accepted and t_final of a dead trajectory are those of that step) ----------------
// The test runs on the integer pipe (the FP64 pipe is the bound of every kernel here): Inf / NaN <=> the
// exponent field of the high word is all ones.  A lane looks at the part of the state it holds; the
// step index of the first hit is latched per lane and the tile takes the minimum once, after the loop.
// The test is made after every kDeathCheckEvery-th step and after the last one (non-finite never heals, so
// nothing is missed): a dead trajectory reports the first CHECKED step at which it was found dead, at most
// kDeathCheckEvery - 1 steps after the step the oracle stops at.  (Every step costs 1.5 - 3 % of the SALI,
// spectrum and GALI kernels and 10 % of the latency-bound configs[0]; every 8th is not measurable.)
constexpr int kDeathCheckEvery = 8;
static_assert((kDeathCheckEvery & (kDeathCheckEvery - 1)) == 0, "a power of two: the test is a mask");
__device__ __forceinline__ int exponent_field(double x) { return __double2hiint(x) & 0x7ff00000; }
template <int NI>
__device__ __forceinline__ bool lane_nonfinite(const double (&q)[NI], const double (&p)[NI]) {
    int m = 0;
#pragma unroll
    for (int c = 0; c < NI; c++) m = max(m, max(exponent_field(q[c]), exponent_field(p[c])));
    return m == 0x7ff00000;
}
// minimum over the tile of the lanes' latched steps, 0 meaning "never" on a lane and in the result
template <int L>
__device__ __forceinline__ long long tile_first_step(long long first) {
    unsigned long long x = first > 0 ? (unsigned long long)first : ~0ULL;
    if constexpr (L > 1 && L <= 32) {
#pragma unroll
        for (int d = L / 2; d >= 1; d >>= 1) {
            const unsigned long long o = __shfl_xor_sync(0xffffffffu, x, d, L);
            x = o < x ? o : x;
        }
    } else if constexpr (L > 32) {
        __shared__ unsigned long long box;
        if (threadIdx.x == 0) box = ~0ULL;
        __syncthreads();
        atomicMin(&box, x);
        __syncthreads();
        x = box;
        __syncthreads();
    }
    return x == ~0ULL ? 0 : (long long)x;
}

// ---- square roots off the slow path ----------------------------------------------------------
// MUFU.RSQ64H seed y0 (|1 - x y0^2| = |e| <= 2^-19, measured) and the quadratic Taylor polynomial of
// (1-e)^(-1/2) = 1 + e/2 + 3e^2/8 + (5/16 e^3 <= 2^-59: below half an ulp, dropped): 5 FP64 instructions none of
// which reads three distinct registers (those run at 2/3 rate), 4 dependent levels after
// the seed, no branch.  The library sqrt()/1.0/sqrt() cost 8 + ~10 instructions and a slow-path branch.
// Arguments are sums of squares: x >= 0.
__device__ __forceinline__ double rsqrt_seed(double x) {
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    return y;
}
// 1/sqrt(x); a denormal x gives inf (the seed flushes it to zero), x = 0 itself gives NaN (0 * inf in the
// correction) where 1.0/sqrt(0.0) is inf -- either way the renormalisation of a null vector is not finite.
// Measured against the host's long double over 10^7 arguments of the whole exponent range
// (tests/test_gpu_math_helpers.py): fast_sqrt <= 1 ulp, fast_rsqrt and fast_rcp <= 1.5 ulp.
__device__ __forceinline__ double fast_rsqrt(double x) {
    const double y0 = rsqrt_seed(x);
    const double e = fma(-(x * y0), y0, 1.0);
    return fma(y0 * e, fma(e, 0.375, 0.5), y0);
}
// sqrt(x); x = 0 (or denormal) gives 0
__device__ __forceinline__ double fast_sqrt(double x) {
    const double y0 = rsqrt_seed(x);
    const double g0 = x * y0;
    const double e = fma(-g0, y0, 1.0);
    const double r = fma(g0 * e, fma(e, 0.375, 0.5), g0);
    return (__double2hiint(x) < 0x00100000) ? 0.0 : r;  // integer test: stays off the FP64 pipe
}

// 1/x for x > 0 (error-norm scales): MUFU.RCP64H seed r0, e = 1 - x r0, r = r0 (1 + e + e^2 + e^3...)
// truncated after e^3 (|e| <= 2^-19: error 2^-76): 3 FP64 instructions, no slow-path branch.
__device__ __forceinline__ double fast_rcp(double x) {
    double r0;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r0) : "d"(x));
    const double e = fma(-x, r0, 1.0);
    return fma(r0, fma(e, fma(e, e, e), e), r0);
}
// ---- deferred logarithm ----------------------------------------------------------------------
// sum_k ln(r_k) of the renormalisation factors is kept as a running PRODUCT in
// (mantissa in [1,2), integer exponent) form: one DMUL and a few integer instructions per factor
// instead of a ~45-instruction log() with a slow-path branch; the logarithm is taken once, when the
// accumulator is written out.  (Also more accurate than summing rounded logarithms.)
struct LogAcc {
    double m;
    int e;
};
__device__ __forceinline__ void logacc_init(LogAcc& a) {
    a.m = 1.0;
    a.e = 0;
}
__device__ __forceinline__ void logacc_mul(LogAcc& a, double r) {  // r > 0, finite, normal
    const double t = a.m * r;
    const int hi = __double2hiint(t);
    a.e += ((hi >> 20) & 0x7ff) - 1023;
    a.m = __hiloint2double((hi & 0x800fffff) | 0x3ff00000, __double2loint(t));
}
__device__ __forceinline__ double logacc_value(const LogAcc& a) {
    return fma((double)a.e, 0.693147180559945309417232, log(a.m));
}

// Threads per block never exceed this (every launcher uses 64, 128 or 256): size of the per-thread
// "cold state" arrays in shared memory.
constexpr int kMaxTpb = 256;

// NV deferred-log accumulators per thread.  COLD = false: in registers.  COLD = true: in shared memory
// ([accumulator][thread]: conflict-free), for kernels whose step needs every register -- the accumulators
// are touched once per renormalisation, not once per stage.
template <int NV, bool COLD>
struct LogBank;
template <int NV>
struct LogBank<NV, false> {
    LogAcc a[NV > 0 ? NV : 1];
    __device__ __forceinline__ void init() {
#pragma unroll
        for (int v = 0; v < NV; v++) logacc_init(a[v]);
    }
    __device__ __forceinline__ void mul(int v, double r) { logacc_mul(a[v], r); }
    __device__ __forceinline__ double value(int v) const { return logacc_value(a[v]); }
};
template <int NV>
struct LogBank<NV, true> {
    __device__ __forceinline__ static double* m_base() {
        __shared__ double m[(NV > 0 ? NV : 1) * kMaxTpb];
        return m;
    }
    __device__ __forceinline__ static int* e_base() {
        __shared__ int e[(NV > 0 ? NV : 1) * kMaxTpb];
        return e;
    }
    __device__ __forceinline__ void init() {
#pragma unroll
        for (int v = 0; v < NV; v++) {
            m_base()[v * kMaxTpb + threadIdx.x] = 1.0;
            e_base()[v * kMaxTpb + threadIdx.x] = 0;
        }
    }
    __device__ __forceinline__ void mul(int v, double r) {
        LogAcc t{m_base()[v * kMaxTpb + threadIdx.x], e_base()[v * kMaxTpb + threadIdx.x]};
        logacc_mul(t, r);
        m_base()[v * kMaxTpb + threadIdx.x] = t.m;
        e_base()[v * kMaxTpb + threadIdx.x] = t.e;
    }
    __device__ __forceinline__ double value(int v) const {
        return logacc_value(LogAcc{m_base()[v * kMaxTpb + threadIdx.x], e_base()[v * kMaxTpb + threadIdx.x]});
    }
};

// ---- stages -------------------------------------------------------------------------------
// force(Q, Fout): evaluates the NI force components at the stage coordinates Q.
// hook(Int<i>, F): called after stage i's force is available (used by the LD quadrature).
//
// Stage coordinates of stage i (0-based) from the forces of the earlier stages.  A.A has an EMPTY first
// subdiagonal ((A.A)_{i,i-1} = 0, pinned by tests/test_library_abi.py): Q_i needs F_0 .. F_{i-2} only.
// One code path serves both steppers.  Fixed step: `tab` is premultiplied by powers of h (a2 = h^2 A.A,
// cs = h rowsum(A)), `p` is the momentum, F the forces.  Adaptive step: `tab` is raw, and the caller hands in
// u = h p in place of p and works with SCALED forces G_l = h^2 F_l (the force functor multiplies by h^2 where
// that is free): then Q_i = q + cs_i u + sum_l (A.A)_il G_l needs no further
// multiplication by the trajectory's h, and every fused multiply-add below has a constant-bank coefficient,
// i.e. at most two register sources (three-register DFMAs run at 2/3 rate).
template <int I, int NI>
__device__ __forceinline__ void dop8_stage_coords(const Tab& tab, const double (&q)[NI], const double (&p)[NI],
                                                  const double (&F)[12][NI], double (&Q)[NI]) {
    static_assert(I >= 1 && I < 12, "stage index");
#pragma unroll
    for (int c = 0; c < NI; c++) {
        double acc = fma(tab.cs[I], p[c], q[c]);
        static_for<0, I>([&](auto lc) {
            constexpr int l = decltype(lc)::value;
            if constexpr (coef::A2[I][l] != 0.0) acc = fma(tab.a2[I][l], F[l][c], acc);
        });
        Q[c] = acc;
    }
}

// The 12 stages.  PAIR = true evaluates them two at a time, (0,1), (2,3), ..., (10,11): stage 2k+1 does
// not depend on stage 2k (see above), so both stage coordinates are formed first and the two force
// evaluations -- their neighbour shuffles included -- are independent instruction streams that the
// scheduler interleaves: twice the instruction-level parallelism exactly where a lane waits on a shuffle
// and on the short dependent chain of the force.  Same operations in the same order per value: results
// are bit-identical with PAIR = false.
template <int NI, bool PAIR = true, class Force, class Hook>
__device__ __forceinline__ void dop8_stages(const Tab& tab, const double (&q)[NI], const double (&p)[NI],
                                            double (&F)[12][NI], Force&& force, Hook&& hook) {
    if constexpr (PAIR) {
        static_for<0, 6>([&](auto kc) {
            constexpr int i0 = 2 * decltype(kc)::value, i1 = i0 + 1;
            double Qb[NI];
            dop8_stage_coords<i1, NI>(tab, q, p, F, Qb);
            if constexpr (i0 == 0) {
                force.pair(q, F[0], Qb, F[i1]);
            } else {
                double Qa[NI];
                dop8_stage_coords<i0, NI>(tab, q, p, F, Qa);
                force.pair(Qa, F[i0], Qb, F[i1]);
            }
            hook(Int<i0>{}, F);
            hook(Int<i1>{}, F);
        });
    } else {
        force(q, F[0]);
        hook(Int<0>{}, F);
        static_for<1, 12>([&](auto ic) {
            constexpr int i = decltype(ic)::value;
            double Q[NI];
            dop8_stage_coords<i, NI>(tab, q, p, F, Q);
            force(Q, F[i]);
            hook(ic, F);
        });
    }
}

// 8th-order solution from the stage forces.  The first NCOMP items (the orbit's) are advanced
// with a compensated sum: y+ = y + (dy + c) by Fast2Sum, the rounding
// error of that one addition -- which is ~1/h times larger than every other rounding error of a
// step -- is carried in c to the next step.  qc/pc: carried words in, qcn/pcn: out.
// PREMUL (fixed step): premultiplied table, F = forces.  Otherwise (adaptive): raw table, u = h p,
// F = the scaled forces h^2 F_l, hinv = 1/h:  q+ = q + u + sum bq_l G_l,  p+ = p + hinv sum b_l G_l.
template <int NI, int NCOMP, bool PREMUL>
__device__ __forceinline__ void dop8_solution(const Tab& tab, double hinv, const double (&q)[NI],
                                              const double (&p)[NI], const double (&u)[NI],
                                              const double (&F)[12][NI], double (&qn)[NI], double (&pn)[NI],
                                              const double (&qc)[NCOMP > 0 ? NCOMP : 1],
                                              const double (&pc)[NCOMP > 0 ? NCOMP : 1],
                                              double (&qcn)[NCOMP > 0 ? NCOMP : 1],
                                              double (&pcn)[NCOMP > 0 ? NCOMP : 1], double (&spo)[NI]) {
    // spo (adaptive): sum_l b_l G_l per item, which the third-order error estimate reuses (dop8_error_sums)
#pragma unroll
    for (int c = 0; c < NI; c++) {
        const bool comp = c < NCOMP;
        double aq, ap;
        if constexpr (PREMUL) {
            aq = comp ? fma(tab.h, p[c], qc[comp ? c : 0]) : fma(tab.h, p[c], q[c]);
            ap = comp ? pc[comp ? c : 0] : p[c];
            static_for<0, 12>([&](auto lc) {
                constexpr int l = decltype(lc)::value;
                if constexpr (coef::BQ[l] != 0.0) aq = fma(tab.bq[l], F[l][c], aq);
                if constexpr (coef::B[l] != 0.0) ap = fma(tab.bp[l], F[l][c], ap);
            });
        } else {
            aq = comp ? u[c] + qc[comp ? c : 0] : u[c] + q[c];
            double sp = tab.bp[0] * F[0][c];
            static_for<0, 12>([&](auto lc) {
                constexpr int l = decltype(lc)::value;
                if constexpr (coef::BQ[l] != 0.0) aq = fma(tab.bq[l], F[l][c], aq);
                if constexpr (l > 0 && coef::B[l] != 0.0) sp = fma(tab.bp[l], F[l][c], sp);
            });
            ap = comp ? fma(hinv, sp, pc[comp ? c : 0]) : fma(hinv, sp, p[c]);
            spo[c] = sp;
        }
        if (comp) {  // aq, ap are increments (+ carried error): Fast2Sum
            const double tq = q[c] + aq, tp = p[c] + ap;
            qcn[comp ? c : 0] = aq - (tq - q[c]);
            pcn[comp ? c : 0] = ap - (tp - p[c]);
            qn[c] = tq;
            pn[c] = tp;
        } else {
            qn[c] = aq;
            pn[c] = ap;
        }
    }
}

// Embedded error sums of one attempted step:
// this lane's contribution to S5 = sum_c (e5_c/scale_c)^2 and S3 likewise, over its 2 NI
// components, scale_c = atol + rtol max(|y_c|, |y+_c|).  Raw tableau, F = the SCALED forces h^2 F_l:
// the sums are of (e_c / h) / scale_c (the controller multiplies the norm by |h| afterwards), i.e.
// e_q / h = hinv sum (E^T A)_l G_l,  e_p / h = hinv^2 sum E_l G_l.  `on[c]` masks padding items.
template <int NI>
__device__ __forceinline__ void dop8_error_sums(const Tab& tab, double hinv, const double (&q)[NI],
                                                const double (&p)[NI], const double (&qn)[NI],
                                                const double (&pn)[NI], const double (&F)[12][NI],
                                                const double (&sp)[NI], double rtol, double atol,
                                                const bool (&on)[NI], double& S5, double& S3) {
    const double hinv2 = hinv * hinv;
    // NACC interleaved partial sums (items c, c + NACC, ... go to sum c % NACC): the dependent chain is
    // 2 NI / NACC fused multiply-adds deep instead of 2 NI (the error norm is on the serial tail of an attempt)
    constexpr int NACC = NI < 3 ? NI : 3;
    double a5[NACC], a3[NACC];
#pragma unroll
    for (int c = 0; c < NI; c++) {
        double s5q = tab.e5q[0] * F[0][c], s3q = tab.e3q[0] * F[0][c];
        double s5p = tab.e5p[0] * F[0][c];
        // E3 is b with three entries changed (the third-order weights differ from b at stages 1, 9, 12 only):
        // sum E3_l G_l = sum b_l G_l - sum (b - E3)_l G_l, the first sum being the solution's (3 FMAs, not 8)
        double s3p = sp[c];
        static_for<0, 12>([&](auto lc) {
            constexpr int l = decltype(lc)::value;
            if constexpr (coef::B[l] != coef::E3[l]) s3p = fma(-tab.d3[l], F[l][c], s3p);
        });
        static_for<1, 12>([&](auto lc) {
            constexpr int l = decltype(lc)::value;
            if constexpr (coef::E5Q[l] != 0.0) s5q = fma(tab.e5q[l], F[l][c], s5q);
            if constexpr (coef::E3Q[l] != 0.0) s3q = fma(tab.e3q[l], F[l][c], s3q);
            if constexpr (coef::E5[l] != 0.0) s5p = fma(tab.e5p[l], F[l][c], s5p);
        });
        const double iq = hinv * fast_rcp(fma(rtol, fmax(fabs(q[c]), fabs(qn[c])), atol));
        const double ip = hinv2 * fast_rcp(fma(rtol, fmax(fabs(p[c]), fabs(pn[c])), atol));
        const double a = s5q * iq, b = s5p * ip, c3 = s3q * iq, d3 = s3p * ip;
        if (c < NACC) {
            a5[c % NACC] = on[c] ? fma(a, a, b * b) : 0.0;
            a3[c % NACC] = on[c] ? fma(c3, c3, d3 * d3) : 0.0;
        } else if (on[c]) {
            a5[c % NACC] = fma(a, a, fma(b, b, a5[c % NACC]));
            a3[c % NACC] = fma(c3, c3, fma(d3, d3, a3[c % NACC]));
        }
    }
    S5 = a5[0];
    S3 = a3[0];
#pragma unroll
    for (int k = 1; k < NACC; k++) {
        S5 += a5[k];
        S3 += a3[k];
    }
}

// per-trajectory status words (include/chaoticus.h CHS_ST_*)
enum : int { ST_OK = 0, ST_NONFINITE = 1, ST_UNDERFLOW = 2, ST_MAXSTEPS = 3 };

// x^(1/8) by three square roots (the starting step's exponent)
__device__ __forceinline__ double root8(double x) { return sqrt(sqrt(sqrt(x))); }

// ---- the step-size controller off the FP64 critical path ("Serial tail") ----
// With num = |h| S5 and den = D (S5 + 0.01 S3) the error norm is err = num / sqrt(den), so
//   accept  <=>  err < 1  <=>  num^2 < den            (no square root, no division), and
//   0.9 err^(-1/8) = 0.9 (den / num^2)^(1/16)         (the factor the NEXT step size is multiplied by).
// The factor only steers the step size (the accept test above is exact), so it is evaluated to single
// precision: log2 of a double = its exponent (integer instructions) + MUFU.LG2 of its mantissa, one MUFU.EX2;
// relative error ~3e-7.  This replaces 25 dependent FP64 instructions (one rsqrt for err, three for the
// eighth root) by ~10 short-latency ones that do not touch the FP64 pipe.  Zero / subnormal / huge arguments
// saturate into the clipping range [0.2, 10] on the correct side.
__device__ __forceinline__ float log2_coarse(double x) {  // x >= 0
    const int hi = __double2hiint(x);
    const unsigned lo = (unsigned)__double2loint(x);
    const float m = __int_as_float(0x3f800000 | ((hi & 0xfffff) << 3) | (int)(lo >> 29));  // mantissa in [1, 2)
    float l;
    asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(l) : "f"(m));
    return (float)(((hi >> 20) & 0x7ff) - 1023) + l;
}
__device__ __forceinline__ float step_factor(double num2, double den) {  // 0.9 (den/num2)^(1/16)
    const float e = fmaf(log2_coarse(den) - log2_coarse(num2), 0.0625f, -0.15200309344504997f);  // + log2(0.9)
    float f;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(f) : "f"(e));
    return f;
}

// The decision of one attempt (items 3-4), shared by every adaptive kernel.
// S5, S3: the error sums over all D components; h_try = |h|; rejected: the previous attempt of this step was
// rejected.  acc / rej: accepted / rejected (neither: S5 or S3 is NaN -- a non-finite y+); factor: what the
// next |h| is h_try times (accept: min(10, 0.9 err^(-1/8)), at most 1 right after a rejection, 10 when
// err = 0; reject: max(0.2, 0.9 err^(-1/8))).  Selects only, no branch.
struct StepDecision {
    bool acc, rej;
    double factor;
};
__device__ __forceinline__ StepDecision step_decision(double h_try, double S5, double S3, double D, bool rejected) {
    const double num = h_try * S5, den = fma(0.01, S3, S5) * D, num2 = num * num;
    const bool zero = (S5 == 0.0) && (S3 == 0.0);  // err = 0
    StepDecision d;
    d.acc = zero || num2 < den;
    d.rej = !zero && num2 >= den;
    const float ff = step_factor(num2, den);
    const double fd = (double)ff;
    const float cap = rejected ? 1.0f : 10.0f;
    const double f_acc = (zero || !(ff < cap)) ? (double)cap : fd;
    const double f_rej = (ff > 0.2f) ? fd : 0.2;
    d.factor = d.acc ? f_acc : f_rej;
    return d;
}

// 10 |nextafter(t, dir inf) - t|: the smallest step the controller allows at time t (DESIGN.md "Adaptive
// step", item 5), assembled from integer instructions: exact, branch-free, nothing on the FP64 pipe.  The
// spacing of the doubles at t is 2^(e - 1075) (e: biased exponent of t, at least 1), half of that when t is a
// power of two and the step points towards zero.  Where 10 x spacing is a normal number (e >= 50) it is
// 1.25 x 2^(k+3) -- exponent field k + 1026, mantissa 0x4000000000000; below that it is subnormal, i.e. the
// integer 10 << (e - 1) in units of 2^-1074 (t = 0: 10 x 4.9e-324, as nextafter gives).
__device__ __forceinline__ double ten_ulp(double t, double dir) {
    const int hi = __double2hiint(t), lo = __double2loint(t);
    const int e = (hi >> 20) & 0x7ff;
    const bool pow2 = ((hi & 0xfffff) | lo) == 0;
    const bool to_zero = (hi < 0) == (dir > 0.0);  // sign(t) opposite to the direction of integration
    const int adj = (pow2 && to_zero && e > 1) ? 1 : 0;
    const double normal = __hiloint2double(((e - 49 - adj) << 20) | 0x40000, 0);
    const int sh = (e > 0 ? e - 1 : 0) - adj;
    const double tiny = __longlong_as_double(10LL << (sh & 63));
    return (e - adj) >= 50 ? normal : tiny;
}

}  // namespace chs
