// gen_kernels.cuh -- generic first-order DOP8 kernel for NON-separable Hamiltonians (CUDA path).
//
// The dimensionless double pendulum (Eq.(1)-(3)) has a kinetic energy that depends
// on the angles, so the separable rearrangement of dop8_core.cuh does not apply: here the method
// runs in its textbook form, y' = f(y), 12 full stage derivative vectors K_i (n = 4 components:
// 9 live stage vectors = 36 doubles, fits registers), one trajectory per thread.  Orbit only
// (the paper prints no variational equations for this system).  Fixed step: tableau premultiplied
// by h in the constant bank; adaptive: raw tableau, per-trajectory h, the same controller as
// run_kernel.
#pragma once
#include "col_kernels.cuh"

namespace chs {

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
        sincos(y[0], &s1, &c1);
        sincos(y[1], &s2, &c2);
        const double x = fma(c1, c2, s1 * s2);   // cos(theta1 - theta2)
        const double sd = fma(s1, c2, -c1 * s2); // sin(theta1 - theta2)
        const double p1 = y[2], p2 = y[3];
        const double id = 1.0 / fma(-x, x, P.sg1);
        const double m01 = -x * P.ia;
        f[0] = id * fma(P.ia2, p1, m01 * p2);
        f[1] = id * fma(m01, p1, P.sg1 * p2);
        const double pMp = fma(P.ia2 * p1, p1, fma(2.0 * m01 * p1, p2, P.sg1 * p2 * p2));
        const double pCp = 2.0 * id * fma(x * id, pMp, -P.ia * p1 * p2);
        const double t = 0.5 * sd * pCp;
        f[2] = fma(-P.asg, s1, t);
        f[3] = -t - s2;
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

template <class Sys, bool ADAPT, int TPB, int MINB>
__global__ void __launch_bounds__(TPB, MINB)
gen_run_kernel(const __grid_constant__ Tab tab, const typename Sys::Params prm, const RunArgs a) {
    constexpr int N = Sys::N;
    const long long ic = (long long)blockIdx.x * TPB + threadIdx.x;
    if (ic >= a.n_ic) return;
    double y[N], yc[N];  // state and the carried rounding word of its compensated update
#pragma unroll
    for (int c = 0; c < N; c++) {
        y[c] = a.y[(long long)c * a.n_ic + ic];
        yc[c] = (a.resume && a.carry) ? a.carry[(long long)c * a.n_ic + ic] : 0.0;
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
        }
        n_acc = a.n_steps;
        t = a.t0 + (double)a.n_steps * a.h;
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
                const double d0 = sqrt(s0 / N), d1 = sqrt(s1 / N);
                double ha = (d0 < 1e-5 || d1 < 1e-5) ? 1e-6 : 0.01 * d0 / d1;
                ha = fmin(ha, interval);
#pragma unroll
                for (int c = 0; c < N; c++) y1[c] = fma(ha * dir, f0[c], y[c]);
                Sys::rhs(prm, y1, f1);
#pragma unroll
                for (int c = 0; c < N; c++) {
                    const double is = 1.0 / fma(fabs(y[c]), a.rtol, a.atol);
                    const double d = (f1[c] - f0[c]) * is;
                    s2 += d * d;
                }
                const double d2 = sqrt(s2 / N) / ha;
                const double hb = (d1 <= 1e-15 && d2 <= 1e-15) ? fmax(1e-6, 1e-3 * ha) : root8(0.01 / fmax(d1, d2));
                h_abs = fmin(fmin(100.0 * ha, hb), interval);
            }
        }
        long long attempts = 0;
        bool rejected = false;
        double min_step = 0.0;
        while (status == ST_OK && dir * (a.t_end - t) > 0.0) {
            if (!rejected) {
                min_step = 10.0 * fabs(nextafter(t, dir * INFINITY) - t);
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
            const double err = (S5 == 0.0 && S3 == 0.0) ? 0.0 : h_try * S5 * fast_rsqrt((S5 + 0.01 * S3) * (double)N);
            if (err < 1.0) {
                double factor = (err == 0.0) ? 10.0 : fmin(10.0, 0.9 * inv_root8(err));
                if (rejected) factor = fmin(factor, 1.0);
                h_abs = h_try * factor;
                t = t_new;
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
            } else if (err >= 1.0) {
                h_abs = h_try * fmax(0.2, 0.9 * inv_root8(err));
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
    if (bad && status == ST_OK) status = ST_NONFINITE;
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

}  // namespace chs
