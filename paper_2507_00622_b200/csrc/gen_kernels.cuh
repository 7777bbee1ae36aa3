// gen_kernels.cuh -- generic first-order DOP8 kernel for NON-separable Hamiltonians (CUDA path).
//
// The dimensionless double pendulum (Eq.(1)-(3)) has a kinetic energy that depends
// on the angles, so the separable rearrangement of dop8_core.cuh does not apply: here the method
// runs in its textbook form, y' = f(y), 12 full stage derivative vectors K_i (n = 4 components:
// 9 live stage vectors = 36 doubles, fits registers), one trajectory per thread for the orbit alone
// (gen_run_kernel, gen_ld_kernel) and a tile of lanes, one column per lane, when deviation vectors ride
// along (gen_col_kernel).  Fixed step: tableau premultiplied
// by h in the constant bank; adaptive: raw tableau, per-trajectory h, the same controller as
// run_kernel.
#pragma once
#include "col_kernels.cuh"

namespace chs {

// sin and cos of one angle without the CUDA library routine's slow path (its huge-argument reduction keeps a
// 40-byte stack array -- the only local memory the library had -- behind a branch).  k = rint(x 2/pi);
// r = x - k pi/2 with pi/2 split into three doubles and three fused multiply-adds.  The first constant is the
// full 53-bit double nearest pi/2, so k * c1 is NOT a double; what saves the step is the fused multiply-add,
// which forms x - k c1 from the exact product with ONE rounding (error <= half an ulp of r, about 2^-54 for
// |r| <= pi/4), and the two corrections add pi/2's next 106 bits times k.  sin r and cos r on [-pi/4, pi/4] by
// their Taylor polynomials to r^15 / r^16 (remainders 5e-17 r and 2e-18: below half an ulp; the coefficients
// are (-1)^m / n! rounded to double); the quadrant k mod 4 swaps and negates by selects.  24 FP64
// instructions, branch-free.  Measured against the host's long double sine and cosine of the same double x
// over 10^7 arguments, |x| up to 1e8, multiples of pi/2 included (tests/test_gpu_math_helpers.py): <= 2 ulp
// of the true value everywhere (1.56 seen at |x| = 9.9e6 and 1.54 at |x| <= 10: it is the polynomial's rounding, not
// the reduction's, that sets it).
__device__ __forceinline__ void fast_sincos(double x, double* sn, double* cs) {
    const double k = rint(x * 0.6366197723675814);
    double r = fma(-k, 1.5707963267948966, x);
    r = fma(-k, 6.123233995736766e-17, r);
    r = fma(-k, -1.4973849048591698e-33, r);
    const double z = r * r;
    double ps = -7.647163731819816e-13;
    ps = fma(ps, z, 1.6059043836821613e-10);
    ps = fma(ps, z, -2.505210838544172e-08);
    ps = fma(ps, z, 2.7557319223985893e-06);
    ps = fma(ps, z, -0.0001984126984126984);
    ps = fma(ps, z, 0.008333333333333333);
    ps = fma(ps, z, -0.16666666666666666);
    const double s = fma(r * z, ps, r);
    double pc = 4.779477332387385e-14;
    pc = fma(pc, z, -1.1470745597729725e-11);
    pc = fma(pc, z, 2.08767569878681e-09);
    pc = fma(pc, z, -2.755731922398589e-07);
    pc = fma(pc, z, 2.48015873015873e-05);
    pc = fma(pc, z, -0.001388888888888889);
    pc = fma(pc, z, 0.041666666666666664);
    const double c = fma(z * z, pc, fma(-0.5, z, 1.0));
    const int q = (int)((long long)k & 3LL);
    const double a = (q & 1) ? c : s, b = (q & 1) ? s : c;  // q: 0 (s, c)  1 (c, -s)  2 (-s, -c)  3 (-c, s)
    *sn = (q & 2) ? -a : a;
    *cs = ((q + 1) & 2) ? -b : b;
}

// Dimensionless double pendulum, Eq.(1): H = p^T B^-1(cos Dtheta) p / 2
// - alpha (1+sigma) cos theta1 - cos theta2, B^-1 of PAPER.md:72 Eq.(2).  y = (theta1, theta2, p1, p2).
// Hamilton's equations (Eq.(3)) with C(x) = d(B^-1)/dx written out analytically:
//   B^-1 = M(x)/D,  D = 1 + sigma - x^2,  M = [[1/alpha^2, -x/alpha], [-x/alpha, 1+sigma]]
//   C    = 2x M/D^2 + M'/D,  M' = [[0, -1/alpha], [-1/alpha, 0]]
struct DoublePendulum {
    static constexpr int N = 4;
    struct Params { double sg1, ia, ia2, asg; };  // 1+sigma, 1/alpha, 1/alpha^2, alpha (1+sigma)
    __device__ static __forceinline__ void rhs(const Params& P, const double (&y)[4], double (&f)[4]) {
        double s1, c1, s2, c2;
        fast_sincos(y[0], &s1, &c1);
        fast_sincos(y[1], &s2, &c2);
        const double x = fma(c1, c2, s1 * s2);   // cos(theta1 - theta2)
        const double sd = fma(s1, c2, -c1 * s2); // sin(theta1 - theta2)
        const double p1 = y[2], p2 = y[3];
        const double id = fast_rcp(fma(-x, x, P.sg1));  // 1/D, D = 1 + sigma - x^2 > 0; <= 2 ulp, no slow path
        const double m01 = -x * P.ia;
        f[0] = id * fma(P.ia2, p1, m01 * p2);
        f[1] = id * fma(m01, p1, P.sg1 * p2);
        const double pMp = fma(P.ia2 * p1, p1, fma(2.0 * m01 * p1, p2, P.sg1 * p2 * p2));
        const double pCp = 2.0 * id * fma(x * id, pMp, -P.ia * p1 * p2);
        const double t = 0.5 * sd * pCp;
        f[2] = fma(-P.asg, s1, t);
        f[3] = -t - s2;
    }
    // ---- variational equations: the derivative of Eq.(3) along w = (dth1, dth2, dp1, dp2).
    // Everything that depends on the orbit's stage state only is formed once per stage (Lin), then a
    // deviation column costs ~25 FP64 instructions.  With id = 1/D, M' = dM/dx = [[0, -1/alpha], [-1/alpha, 0]]:
    //   B^-1 = M id,  C = 2x M id^2 + M' id,  C' = dC/dx = (2M + 4x M') id^2 + 8 x^2 M id^3
    //   d(theta') = B^-1 dp + dx C p,  dx = -sin(Dtheta) (dth1 - dth2)
    //   dS = (x/2) dD p^T C p + (s/2) [2 (C p)^T dp + dx p^T C' p]
    //   d(p1') = dS - alpha (1+sigma) cos(theta1) dth1,   d(p2') = -dS - cos(theta2) dth2
    // (the oracle forms C and C' by matrix products of B^-1 and dB/dx instead).
    static constexpr int NDOF = 2;
    struct Hess {};  // Col<DoublePendulum, K, L> only stores the state; its separable force() is never used
    struct Pre {};
    struct Lin {
        double b00, b01, b11, u0, u1, hx_pCp, hs, hs_pCpp, sn, a1c1, c2;
        double f[4];  // the orbit's own right-hand side at the same state
    };
    __device__ static __forceinline__ Lin lin(const Params& P, const double (&y)[4]) {
        double s1, c1, s2, c2;
        fast_sincos(y[0], &s1, &c1);
        fast_sincos(y[1], &s2, &c2);
        const double x = fma(c1, c2, s1 * s2), sd = fma(s1, c2, -c1 * s2);
        const double p1 = y[2], p2 = y[3];
        const double id = fast_rcp(fma(-x, x, P.sg1)), id2 = id * id;
        const double m01 = -x * P.ia;
        const double Mp0 = fma(P.ia2, p1, m01 * p2), Mp1 = fma(m01, p1, P.sg1 * p2);  // M p
        const double pMp = fma(p1, Mp0, p2 * Mp1), pM1p = -2.0 * P.ia * p1 * p2;           // p^T M p, p^T M' p
        const double pCp = fma(2.0 * x * id2, pMp, id * pM1p);
        const double pCpp = fma(id2, fma(4.0 * x, pM1p, 2.0 * pMp), 8.0 * x * x * id2 * id * pMp);
        Lin L;
        L.b00 = P.ia2 * id;
        L.b01 = m01 * id;
        L.b11 = P.sg1 * id;
        L.u0 = fma(2.0 * x * id2, Mp0, -P.ia * id * p2);  // C p
        L.u1 = fma(2.0 * x * id2, Mp1, -P.ia * id * p1);
        L.hx_pCp = 0.5 * x * pCp;
        L.hs = 0.5 * sd;
        L.hs_pCpp = 0.5 * sd * pCpp;
        L.sn = sd;
        L.a1c1 = P.asg * c1;
        L.c2 = c2;
        const double t = 0.5 * sd * pCp;
        L.f[0] = id * Mp0;
        L.f[1] = id * Mp1;
        L.f[2] = fma(-P.asg, s1, t);
        L.f[3] = -t - s2;
        return L;
    }
    __device__ static __forceinline__ void apply_lin(const Lin& L, const double (&w)[4], double (&g)[4]) {
        const double dD = w[0] - w[1], dx = -L.sn * dD;
        g[0] = fma(L.b00, w[2], fma(L.b01, w[3], dx * L.u0));
        g[1] = fma(L.b01, w[2], fma(L.b11, w[3], dx * L.u1));
        const double dS = fma(L.hx_pCp, dD, fma(2.0 * L.hs, fma(L.u0, w[2], L.u1 * w[3]), dx * L.hs_pCpp));
        g[2] = fma(-L.a1c1, w[0], dS);
        g[3] = fma(-L.c2, w[1], -dS);
    }
    __host__ static bool make_params(const double* p, int n, Params& out) {
        if (n < 2 || !(p[1] > 0.0) || !(p[0] > -1.0)) return false;
        out = Params{1.0 + p[0], 1.0 / p[1], 1.0 / (p[1] * p[1]), p[1] * (1.0 + p[0])};
        return true;
    }
};

// stage derivatives K_1..K_12 of one step of size h from y
template <class Sys, bool PREMUL>
__device__ __forceinline__ void dop8_generic_stages(const Tab& tab, const typename Sys::Params& prm, double h,
                                                    const double (&y)[Sys::N], double (&K)[12][Sys::N]) {
    constexpr int N = Sys::N;
    Sys::rhs(prm, y, K[0]);
    static_for<1, 12>([&](auto ic) {
        constexpr int i = decltype(ic)::value;
        double Y[N];
#pragma unroll
        for (int c = 0; c < N; c++) {
            if constexpr (PREMUL) {
                double acc = y[c];
                static_for<0, i>([&](auto jc) {
                    constexpr int j = decltype(jc)::value;
                    if constexpr (coef::A[i][j] != 0.0) acc = fma(tab.ap[i][j], K[j][c], acc);
                });
                Y[c] = acc;
            } else {
                double s = tab.ap[i][0] * K[0][c];
                static_for<1, i>([&](auto jc) {
                    constexpr int j = decltype(jc)::value;
                    if constexpr (coef::A[i][j] != 0.0) s = fma(tab.ap[i][j], K[j][c], s);
                });
                Y[c] = fma(h, s, y[c]);
            }
        }
        Sys::rhs(prm, Y, K[i]);
    });
}

// LD (adaptive only): the arc-length Lagrangian descriptor as one more component of the state (R21,
// as run_kernel's LD): threads are (direction, IC) tasks, the backward pass is the forward pass of (theta, -p);
// only M and the report ([2][n_ic]) are written.
template <class Sys, bool ADAPT, int TPB, int MINB, bool LD = false>
__global__ void __launch_bounds__(TPB, MINB)
gen_run_kernel(const __grid_constant__ Tab tab, const typename Sys::Params prm, const RunArgs a) {
    static_assert(!LD || ADAPT, "LD rides on the adaptive run");
    constexpr int N = Sys::N;
    const long long task = (long long)blockIdx.x * TPB + threadIdx.x;
    if (task >= (LD ? a.n_ic * a.n_dirs : a.n_ic)) return;
    const long long ic = LD ? task % a.n_ic : task;
    const int dsel = LD ? a.dir_first + (int)(task / a.n_ic) : 0;
    const long long out_slot = (long long)dsel * a.n_ic + ic;
    double M = 0.0;
    double y[N], yc[N];  // state and the carried rounding word of its compensated update
#pragma unroll
    for (int c = 0; c < N; c++) {
        if constexpr (LD) {
            y[c] = a.y0[(long long)c * a.n_ic + ic] * ((c >= N / 2 && dsel == 1) ? -1.0 : 1.0);
            yc[c] = 0.0;
        } else {
            y[c] = a.y[(long long)c * a.n_ic + ic];
            yc[c] = (a.resume && a.carry) ? a.carry[(long long)c * a.n_ic + ic] : 0.0;
        }
    }
    long long n_acc = 0, n_rej = 0;
    int status = ST_OK;
    double t = a.t0;

// y+ = y + (inc + carried word), Fast2Sum
#define CHS_GEN_ADVANCE()                                    \
    _Pragma("unroll") for (int c = 0; c < N; c++) {          \
        const double u_ = inc[c] + yc[c];                    \
        const double s_ = y[c] + u_;                         \
        ycn[c] = u_ - (s_ - y[c]);                           \
        yn[c] = s_;                                          \
    }

    long long first_bad = 0;  // fixed step: the first step after which the state was not finite (dop8_core.cuh)
    if constexpr (!ADAPT) {
        for (long long st = 0; st < a.n_steps; ++st) {
            double K[12][N];
            dop8_generic_stages<Sys, true>(tab, prm, 0.0, y, K);
            double inc[N], yn[N], ycn[N];
#pragma unroll
            for (int c = 0; c < N; c++) {
                double s = tab.bp[0] * K[0][c];
                static_for<1, 12>([&](auto lc) {
                    constexpr int l = decltype(lc)::value;
                    if constexpr (coef::B[l] != 0.0) s = fma(tab.bp[l], K[l][c], s);
                });
                inc[c] = s;
            }
            CHS_GEN_ADVANCE()
#pragma unroll
            for (int c = 0; c < N; c++) {
                y[c] = yn[c];
                yc[c] = ycn[c];
            }
            if ((((st + 1) & (kDeathCheckEvery - 1)) == 0 || st + 1 == a.n_steps) && first_bad == 0 && lane_nonfinite<N>(y, y))
                first_bad = st + 1;
        }
        n_acc = first_bad > 0 ? first_bad : a.n_steps;  // a dead trajectory reports the step at which it died
        t = a.t0 + (double)n_acc * a.h;
    } else {
        const double dir = (a.t_end >= a.t0) ? 1.0 : -1.0;
        const double interval = fabs(a.t_end - a.t0);
        double h_abs = a.h0;
        if (!(h_abs > 0.0)) {  // starting step (item 6)
            h_abs = 0.0;
            if (interval > 0.0) {
                double f0[N], f1[N], y1[N];
                Sys::rhs(prm, y, f0);
                double s0 = 0.0, s1 = 0.0, s2 = 0.0;
#pragma unroll
                for (int c = 0; c < N; c++) {
                    const double is = 1.0 / fma(fabs(y[c]), a.rtol, a.atol);
                    s0 += (y[c] * is) * (y[c] * is);
                    s1 += (f0[c] * is) * (f0[c] * is);
                }
                constexpr double DD = N + (LD ? 1 : 0);  // LD: one more component M (M = 0, M' = |f|, scale atol)
                double nf0 = 0.0;
                if constexpr (LD) {
#pragma unroll
                    for (int c = 0; c < N; c++) nf0 = fma(f0[c], f0[c], nf0);
                    nf0 = sqrt(nf0);
                    s1 += (nf0 / a.atol) * (nf0 / a.atol);
                }
                const double d0 = sqrt(s0 / DD), d1 = sqrt(s1 / DD);
                double ha = (d0 < 1e-5 || d1 < 1e-5) ? 1e-6 : 0.01 * d0 / d1;
                ha = fmin(ha, interval);
#pragma unroll
                for (int c = 0; c < N; c++) y1[c] = fma(ha * dir, f0[c], y[c]);
                Sys::rhs(prm, y1, f1);
                if constexpr (LD) {
                    double nf1 = 0.0;
#pragma unroll
                    for (int c = 0; c < N; c++) nf1 = fma(f1[c], f1[c], nf1);
                    const double dn = (sqrt(nf1) - nf0) / a.atol;
                    s2 += dn * dn;
                }
#pragma unroll
                for (int c = 0; c < N; c++) {
                    const double is = 1.0 / fma(fabs(y[c]), a.rtol, a.atol);
                    const double d = (f1[c] - f0[c]) * is;
                    s2 += d * d;
                }
                const double d2 = sqrt(s2 / DD) / ha;
                const double hb = (d1 <= 1e-15 && d2 <= 1e-15) ? fmax(1e-6, 1e-3 * ha) : root8(0.01 / fmax(d1, d2));
                h_abs = fmin(fmin(100.0 * ha, hb), interval);
            }
        }
        long long attempts = 0;
        bool rejected = false;
        double min_step = 0.0;
        while (status == ST_OK && dir * (a.t_end - t) > 0.0) {
            if (!rejected) {
                min_step = ten_ulp(t, dir);  // 10 |nextafter(t, dir inf) - t|
                h_abs = fmax(h_abs, min_step);
            }
            if (h_abs < min_step) { status = ST_UNDERFLOW; break; }
            if (a.max_steps > 0 && attempts >= a.max_steps) { status = ST_MAXSTEPS; break; }
            attempts++;
            double t_new = t + h_abs * dir;
            if (dir * (t_new - a.t_end) > 0.0) t_new = a.t_end;
            const double h = t_new - t, h_try = fabs(h);
            double K[12][N];
            dop8_generic_stages<Sys, false>(tab, prm, h, y, K);
            double inc[N], yn[N], ycn[N];
            double S5 = 0.0, S3 = 0.0;
            double Mn = 0.0;
            if constexpr (LD) {  // M+ = M + |h| sum b_i |K_i|_2 and the embedded errors of M (divided by h)
                double sb = 0.0, s5 = 0.0, s3 = 0.0;
                static_for<0, 12>([&](auto lc) {
                    constexpr int l = decltype(lc)::value;
                    if constexpr (coef::B[l] != 0.0) {
                        double n2 = 0.0;
#pragma unroll
                        for (int c = 0; c < N; c++) n2 = fma(K[l][c], K[l][c], n2);
                        const double nr = fast_sqrt(n2);
                        sb = fma(tab.bl[l], nr, sb);
                        s5 = fma(tab.e5p[l], nr, s5);
                        s3 = fma(tab.e3p[l], nr, s3);
                    }
                });
                Mn = fma(h_try, sb, M);
                const double isc = fast_rcp(fma(a.rtol, fmax(fabs(M), fabs(Mn)), a.atol));
                s5 *= isc;
                s3 *= isc;
                S5 = s5 * s5;
                S3 = s3 * s3;
            }
#pragma unroll
            for (int c = 0; c < N; c++) {
                double s = tab.bp[0] * K[0][c], e5 = tab.e5p[0] * K[0][c], e3 = tab.e3p[0] * K[0][c];
                static_for<1, 12>([&](auto lc) {
                    constexpr int l = decltype(lc)::value;
                    if constexpr (coef::B[l] != 0.0) s = fma(tab.bp[l], K[l][c], s);
                    if constexpr (coef::E5[l] != 0.0) e5 = fma(tab.e5p[l], K[l][c], e5);
                    if constexpr (coef::E3[l] != 0.0) e3 = fma(tab.e3p[l], K[l][c], e3);
                });
                inc[c] = h * s;
                K[0][c] = e5;  // K[0] and K[1] are dead here: reuse as scratch
                K[1][c] = e3;
            }
            CHS_GEN_ADVANCE()
#pragma unroll
            for (int c = 0; c < N; c++) {
                const double is = fast_rcp(fma(a.rtol, fmax(fabs(y[c]), fabs(yn[c])), a.atol));
                const double u = K[0][c] * is, v = K[1][c] * is;
                S5 = fma(u, u, S5);
                S3 = fma(v, v, S3);
            }
            const StepDecision dec = step_decision(h_try, S5, S3, (double)(N + (LD ? 1 : 0)), rejected);
            if (dec.acc) {
                h_abs = h_try * dec.factor;
                t = t_new;
                if constexpr (LD) M = Mn;
                bool fin = true;
#pragma unroll
                for (int c = 0; c < N; c++) {
                    y[c] = yn[c];
                    yc[c] = ycn[c];
                    fin = fin && isfinite(yn[c]);
                }
                n_acc++;
                rejected = false;
                if (!fin) status = ST_NONFINITE;
            } else if (dec.rej) {
                h_abs = h_try * dec.factor;
                rejected = true;
                n_rej++;
            } else {
                status = ST_NONFINITE;
            }
        }
    }
    bool bad = status != ST_OK;
#pragma unroll
    for (int c = 0; c < N; c++) bad = bad || !isfinite(y[c]);
    if constexpr (LD) bad = bad || !isfinite(M);
    if (bad && status == ST_OK) status = ST_NONFINITE;
    if constexpr (LD) {
        double* out = dsel == 0 ? a.ld_fwd : a.ld_bwd;
        out[ic] = bad ? nan("") : M;
        if (a.n_acc) a.n_acc[out_slot] = n_acc;
        if (a.n_rej) a.n_rej[out_slot] = n_rej;
        if (a.status) a.status[out_slot] = status;
        if (a.t_final) a.t_final[out_slot] = t;
        return;
    }
#pragma unroll
    for (int c = 0; c < N; c++) a.y[(long long)c * a.n_ic + ic] = bad ? nan("") : y[c];
    if (a.carry) {
#pragma unroll
        for (int c = 0; c < N; c++) a.carry[(long long)c * a.n_ic + ic] = bad ? 0.0 : yc[c];
    }
    if (a.n_acc) a.n_acc[ic] = n_acc;
    if (a.n_rej) a.n_rej[ic] = n_rej;
    if (a.status) a.status[ic] = status;
    if (a.t_final) a.t_final[ic] = t;
}

#undef CHS_GEN_ADVANCE

// Lagrangian descriptor with the generic form: M += |h| sum_i b_i |K_i|_2,
// K_i the full stage derivative.  One thread per (direction, IC); the backward pass is the forward
// pass of (theta, -p): the kinetic energy is a quadratic form in p, so H is even in p.
template <class Sys, int TPB, int MINB>
__global__ void __launch_bounds__(TPB, MINB)
gen_ld_kernel(const __grid_constant__ Tab tab, const typename Sys::Params prm, const RunArgs a, int dir_first,
              int n_dirs) {
    constexpr int N = Sys::N;
    const long long gt = (long long)blockIdx.x * TPB + threadIdx.x;
    const long long per_dir = a.n_ic * a.n_members;  // tasks are ordered [direction][member][ic]
    if (gt >= per_dir * n_dirs) return;
    const int dsel = dir_first + (int)(gt / per_dir);
    const long long slot = gt % per_dir;
    const int member = (int)(slot / a.n_ic);
    const long long ic = slot % a.n_ic;
    const double psign = dsel == 0 ? 1.0 : -1.0;
    double y[N];
#pragma unroll
    for (int c = 0; c < N; c++) {
        double v = a.y0[(long long)c * a.n_ic + ic];
        if (member > 0 && c == ((member - 1) >> 1)) v += ((member - 1) & 1) ? -a.sigma : a.sigma;  // neighbour
        y[c] = v * (c >= N / 2 ? psign : 1.0);
    }
    double M = 0.0;
    for (long long st = 0; st < a.n_steps; ++st) {
        double K[12][N];
        dop8_generic_stages<Sys, true>(tab, prm, 0.0, y, K);
        static_for<0, 12>([&](auto lc) {
            constexpr int l = decltype(lc)::value;
            if constexpr (coef::B[l] != 0.0) {
                double n2 = 0.0;
#pragma unroll
                for (int c = 0; c < N; c++) n2 = fma(K[l][c], K[l][c], n2);
                M = fma(tab.bl[l], fast_sqrt(n2), M);
            }
        });
#pragma unroll
        for (int c = 0; c < N; c++) {
            double s = y[c];
            static_for<0, 12>([&](auto lc) {
                constexpr int l = decltype(lc)::value;
                if constexpr (coef::B[l] != 0.0) s = fma(tab.bp[l], K[l][c], s);
            });
            y[c] = s;
        }
    }
    bool ok = true;
#pragma unroll
    for (int c = 0; c < N; c++) ok = ok && isfinite(y[c]);
    double* out = dsel == 0 ? a.ld_fwd : a.ld_bwd;
    out[slot] = ok ? M : nan("");
}

// ---- generic form WITH deviation vectors: one column per lane ------------------------------------
// PAPER.md:49-52 (solvers 3-6) for a non-separable system.  A trajectory is a tile of L >= 1 + K lanes:
// lane 0 the orbit, lane v deviation vector v, each lane its 4 components and 12 full stage derivatives in
// registers (the whole augmented state on one thread would need > 255 registers at K = 2).  Per stage the
// orbit's stage state is broadcast from lane 0 (4 shuffles), every lane forms the orbit-only terms (the two
// sincos, B^-1, C p, p^T C p, p^T C' p) and then takes f(Y) (lane 0) or Df(Y) w (the others).  State,
// renormalisation, Gram-Schmidt, SALI / GALI and the stores are the column layout's (Col<Sys, K, L>).
template <class Sys, int K, int L, int MODE, int IND, bool ADAPT, int TPB, int MINB>
__global__ void __launch_bounds__(TPB, MINB)
gen_col_kernel(const __grid_constant__ Tab tab, const typename Sys::Params prm, const RunArgs a) {
    using C = Col<Sys, K, L>;
    static_assert(C::CPL == 1 && C::ND == 2 && Sys::N == 4, "one column of 4 components per lane");
    constexpr int N = 4;
    const long long gt = (long long)blockIdx.x * TPB + threadIdx.x;
    const long long traj = gt / L;
    const bool valid = traj < a.n_ic;
    const long long ic = valid ? traj : a.n_ic - 1;  // padding tiles shadow the last trajectory
    const bool want_log = (a.logacc != nullptr) || (a.lambda != nullptr);
    C s;
    s.init(prm);
    s.load(a.y, a.w, a.n_ic, ic, 1.0);
    double qc[2] = {0.0, 0.0}, pc[2] = {0.0, 0.0};  // carried rounding words (orbit lane), as run_kernel
    if (a.resume) {
        if (a.carry && !ADAPT) s.load_carry(a.carry, a.n_ic, ic, qc, pc);
    } else {
        s.template do_renorm<MODE>(false, true);
    }
    long long n_acc = 0, n_rej = 0;
    int status = ST_OK;
    double t = a.t0;
    const bool orbit = (s.lt == 0);

    // stage derivatives of one step of size h from (s.q, s.p); PREMUL as dop8_generic_stages
    auto stages = [&](auto premul, double h, double (&Kd)[12][N]) {
        constexpr bool PREMUL = decltype(premul)::value;
        const double y[N] = {s.q[0], s.q[1], s.p[0], s.p[1]};
        static_for<0, 12>([&](auto icn) {
            constexpr int i = decltype(icn)::value;
            double Y[N];
#pragma unroll
            for (int c = 0; c < N; c++) {
                if constexpr (i == 0) {
                    Y[c] = y[c];
                } else if constexpr (PREMUL) {
                    double acc = y[c];
                    static_for<0, i>([&](auto jc) {
                        constexpr int j = decltype(jc)::value;
                        if constexpr (coef::A[i][j] != 0.0) acc = fma(tab.ap[i][j], Kd[j][c], acc);
                    });
                    Y[c] = acc;
                } else {
                    double sm = tab.ap[i][0] * Kd[0][c];
                    static_for<1, i>([&](auto jc) {
                        constexpr int j = decltype(jc)::value;
                        if constexpr (coef::A[i][j] != 0.0) sm = fma(tab.ap[i][j], Kd[j][c], sm);
                    });
                    Y[c] = fma(h, sm, y[c]);
                }
            }
            double Yo[N];
#pragma unroll
            for (int c = 0; c < N; c++) Yo[c] = tile_bcast<L>(Y[c], 0);
            const typename Sys::Lin ln = Sys::lin(prm, Yo);
            double g[N];
            Sys::apply_lin(ln, Y, g);
#pragma unroll
            for (int c = 0; c < N; c++) Kd[i][c] = orbit ? ln.f[c] : g[c];
        });
    };
    // y+ = y + (inc + carried word), Fast2Sum; returns the new carried words
    auto advance = [&](const double (&inc)[N], double (&yn)[N], double (&ycn)[N]) {
        const double y[N] = {s.q[0], s.q[1], s.p[0], s.p[1]};
        const double yc[N] = {qc[0], qc[1], pc[0], pc[1]};
#pragma unroll
        for (int c = 0; c < N; c++) {
            const double u = inc[c] + yc[c];
            const double sm = y[c] + u;
            ycn[c] = u - (sm - y[c]);
            yn[c] = sm;
        }
    };
    auto commit = [&](const double (&yn)[N], const double (&ycn)[N]) {
        s.q[0] = yn[0]; s.q[1] = yn[1]; s.p[0] = yn[2]; s.p[1] = yn[3];
        qc[0] = ycn[0]; qc[1] = ycn[1]; pc[0] = ycn[2]; pc[1] = ycn[3];
    };

    long long slot = 0;
    if constexpr (!ADAPT) {
        int cd = a.m, sd = a.sample_every;
        long long first_bad = 0;  // first step after which this lane's column was not finite (dop8_core.cuh)
        for (long long st = 1; st <= a.n_steps; ++st) {
            double Kd[12][N];
            stages(std::true_type{}, 0.0, Kd);
            double inc[N], yn[N], ycn[N];
#pragma unroll
            for (int c = 0; c < N; c++) {
                double sm = tab.bp[0] * Kd[0][c];
                static_for<1, 12>([&](auto lc) {
                    constexpr int l = decltype(lc)::value;
                    if constexpr (coef::B[l] != 0.0) sm = fma(tab.bp[l], Kd[l][c], sm);
                });
                inc[c] = sm;
            }
            advance(inc, yn, ycn);
            commit(yn, ycn);
            if (((st & (kDeathCheckEvery - 1)) == 0 || st == a.n_steps) && first_bad == 0 && lane_nonfinite<2>(s.q, s.p))
                first_bad = st;
            if constexpr (MODE != MODE_NONE) {
                if (--cd == 0 || st == a.n_steps) {
                    cd = a.m;
                    s.template do_renorm<MODE>(want_log, true);
                    s.scrub_carry(qc, pc);
                    if constexpr (IND != IND_NONE) {
                        if (a.sample_every > 0 && --sd == 0) {
                            sd = a.sample_every;
                            if (slot < a.n_samples - 1) {
                                const double v = s.template indicator<IND>();
                                if (valid && s.lt == 0) a.series[slot * a.n_ic + ic] = v;
                                slot++;
                            }
                        }
                    }
                }
            }
        }
        const long long died = tile_first_step<L>(first_bad);  // a dead trajectory reports where it died
        n_acc = died > 0 ? died : a.n_steps;
        t = a.t0 + (double)n_acc * a.h;
    } else {
        // adaptive: the tile's decisions come from tile-wide sums, identical on
        // all its lanes; tiles of one warp differ, so the loop is warp-uniform and commits are predicated
        const double dir = (a.t_end >= a.t0) ? 1.0 : -1.0;
        const double interval = fabs(a.t_end - a.t0);
        constexpr double D = (double)(N * (1 + K));
        const bool on = s.lt <= K;
        double h_abs = a.h0;
        if (!(h_abs > 0.0)) {  // starting step, item 6
            h_abs = 0.0;
            if (interval > 0.0) {
                const double y[N] = {s.q[0], s.q[1], s.p[0], s.p[1]};
                double Yo[N], f0[N], f1[N], y1[N], g[N];
#pragma unroll
                for (int c = 0; c < N; c++) Yo[c] = tile_bcast<L>(y[c], 0);
                typename Sys::Lin ln = Sys::lin(prm, Yo);
                Sys::apply_lin(ln, y, g);
                double s0 = 0.0, s1 = 0.0, s2 = 0.0;
#pragma unroll
                for (int c = 0; c < N; c++) {
                    f0[c] = orbit ? ln.f[c] : g[c];
                    const double is = 1.0 / fma(fabs(y[c]), a.rtol, a.atol);
                    if (on) {
                        s0 += (y[c] * is) * (y[c] * is);
                        s1 += (f0[c] * is) * (f0[c] * is);
                    }
                }
                const double d0 = sqrt(tile_sum<L>(s0) / D), d1 = sqrt(tile_sum<L>(s1) / D);
                double ha = (d0 < 1e-5 || d1 < 1e-5) ? 1e-6 : 0.01 * d0 / d1;
                ha = fmin(ha, interval);
#pragma unroll
                for (int c = 0; c < N; c++) y1[c] = fma(ha * dir, f0[c], y[c]);
#pragma unroll
                for (int c = 0; c < N; c++) Yo[c] = tile_bcast<L>(y1[c], 0);
                ln = Sys::lin(prm, Yo);
                Sys::apply_lin(ln, y1, g);
#pragma unroll
                for (int c = 0; c < N; c++) {
                    f1[c] = orbit ? ln.f[c] : g[c];
                    const double is = 1.0 / fma(fabs(y[c]), a.rtol, a.atol);
                    const double d = (f1[c] - f0[c]) * is;
                    if (on) s2 += d * d;
                }
                const double d2 = sqrt(tile_sum<L>(s2) / D) / ha;
                const double hb = (d1 <= 1e-15 && d2 <= 1e-15) ? fmax(1e-6, 1e-3 * ha) : root8(0.01 / fmax(d1, d2));
                h_abs = fmin(fmin(100.0 * ha, hb), interval);
            }
        }
        long long attempts = 0;
        bool rejected = false;
        double min_step = 0.0;
        int cd = a.m;
        while (true) {
            bool active = status == ST_OK && dir * (a.t_end - t) > 0.0;
            if (!__any_sync(0xffffffffu, active)) break;
            if (!rejected) {
                min_step = ten_ulp(t, dir);  // 10 |nextafter(t, dir inf) - t|
                h_abs = fmax(h_abs, min_step);
            }
            if (active && h_abs < min_step) { status = ST_UNDERFLOW; active = false; }
            if (active && a.max_steps > 0 && attempts >= a.max_steps) { status = ST_MAXSTEPS; active = false; }
            attempts += active ? 1 : 0;
            double t_new = t + h_abs * dir;
            if (dir * (t_new - a.t_end) > 0.0) t_new = a.t_end;
            const double h = t_new - t, h_try = fabs(h);
            double Kd[12][N];
            stages(std::false_type{}, h, Kd);
            double inc[N], yn[N], ycn[N], e5[N], e3[N];
#pragma unroll
            for (int c = 0; c < N; c++) {
                double sm = tab.bp[0] * Kd[0][c], a5 = tab.e5p[0] * Kd[0][c], a3 = tab.e3p[0] * Kd[0][c];
                static_for<1, 12>([&](auto lc) {
                    constexpr int l = decltype(lc)::value;
                    if constexpr (coef::B[l] != 0.0) sm = fma(tab.bp[l], Kd[l][c], sm);
                    if constexpr (coef::E5[l] != 0.0) a5 = fma(tab.e5p[l], Kd[l][c], a5);
                    if constexpr (coef::E3[l] != 0.0) a3 = fma(tab.e3p[l], Kd[l][c], a3);
                });
                inc[c] = h * sm;
                e5[c] = a5;
                e3[c] = a3;
            }
            advance(inc, yn, ycn);
            double S5 = 0.0, S3 = 0.0;
            {
                const double y[N] = {s.q[0], s.q[1], s.p[0], s.p[1]};
#pragma unroll
                for (int c = 0; c < N; c++) {
                    const double is = fast_rcp(fma(a.rtol, fmax(fabs(y[c]), fabs(yn[c])), a.atol));
                    const double u = e5[c] * is, v = e3[c] * is;
                    if (on) {
                        S5 = fma(u, u, S5);
                        S3 = fma(v, v, S3);
                    }
                }
            }
            S5 = tile_sum<L>(S5);
            S3 = tile_sum<L>(S3);
            const StepDecision dec = step_decision(h_try, S5, S3, D, rejected);
            bool ren = false;
            if (active) {
                if (dec.acc) {
                    h_abs = h_try * dec.factor;
                    t = t_new;
                    commit(yn, ycn);
                    n_acc++;
                    rejected = false;
                    const bool at_end = !(dir * (a.t_end - t) > 0.0);
                    if (MODE != MODE_NONE && (--cd == 0 || at_end)) {
                        cd = a.m;
                        ren = true;
                    }
                } else if (dec.rej) {
                    h_abs = h_try * dec.factor;
                    rejected = true;
                    n_rej++;
                } else {
                    status = ST_NONFINITE;
                }
            }
            if constexpr (MODE != MODE_NONE) {
                if (__any_sync(0xffffffffu, ren)) {
                    s.template do_renorm<MODE>(want_log, ren);
                    if (ren) s.scrub_carry(qc, pc);
                }
            }
        }
    }
    bool bad = !s.finite_all();
    bad = tile_any<L>(status != ST_OK) || bad;
    if (bad && status == ST_OK) status = ST_NONFINITE;
    double ind = 0.0;
    if constexpr (IND != IND_NONE) ind = s.template indicator<IND>();
    if (!valid) return;
    s.store(a.y, a.w, a.n_ic, ic, bad);
    if (a.carry && !ADAPT) s.store_carry(a.carry, a.n_ic, ic, qc, pc, bad);
    if constexpr (K > 0) s.store_logs(a, ic, bad, t - a.t0);
    if (s.lt == 0) {
        if constexpr (IND != IND_NONE) {
            if (a.series) {
                a.series[(a.n_samples - 1) * a.n_ic + ic] = bad ? nan("") : ind;
                if (bad)
                    for (long long r = slot; r < a.n_samples - 1; r++) a.series[r * a.n_ic + ic] = nan("");
            }
        }
        if (a.n_acc) a.n_acc[ic] = n_acc;
        if (a.n_rej) a.n_rej[ic] = n_rej;
        if (a.status) a.status[ic] = status;
        if (a.t_final) a.t_final[ic] = t;
    }
}

}  // namespace chs
