// systems.cuh -- compiled force / Hessian functors of the named systems (CUDA path).
//
// Every system is H = |p|^2/2 + V(q): force F = -grad V(q); variational equations
// (ref [59]) d(dq)/dt = dp, d(dp)/dt = -V_qq(q) dq with V_qq at the stage orbit.
//
// Interface used by the column layout (col_kernels.cuh), NDOF coordinates per column:
//   force(prm, Q, F)          F = -grad V(Q)                        (orbit column)
//   hess(prm, Q, s, g)        the entries of  g M(s),  M(s) = V2'' + s V3''(Q)   (g = 1, or h^2 where the
//                             adaptive kernels want scaled forces: dop8_core.cuh dop8_stage_coords)
//   apply(H, x, G)            G = -H x
//   force_hess(prm, H, Q, g, F)  F = -g grad V(Q) for the orbit, reusing H = g M(1) (the same row products)
// For these cubic potentials  grad V(Q) = (V2'' + 1/2 V3''(Q)) Q  (Euler's relation for the
// homogeneous cubic part), so an orbit column can also be advanced branch-free as
// apply(hess(Q, 1/2), Q): that is what a lane does when orbit and deviation columns sit on
// different lanes of one tile.
#pragma once
#include "dop8_core.cuh"

namespace chs {

// Henon-Heiles, Eq.(4), Eq.(5): V = (x^2+y^2)/2 + x^2 y - y^3/3.
struct HenonHeiles {
    static constexpr int NDOF = 2;
    struct Params {};
    struct Hess { double xx, xy, yy; };
    __device__ static __forceinline__ void force(const Params&, const double* Q, double* F) {
        const double x = Q[0], y = Q[1];
        F[0] = -x * fma(2.0, y, 1.0);     // px' = -x - 2xy = -x (1 + 2y)   (no 3-register DFMA)
        F[1] = fma(y, y, -y) - x * x;     // py' = -y - x^2 + y^2
    }
    // V_qq = [[1+2y, 2x],[2x, 1-2y]]
    __device__ static __forceinline__ Hess hess(const Params&, const double* Q, double s, double g = 1.0) {
        const double t = 2.0 * s * g;
        return Hess{fma(t, Q[1], g), t * Q[0], fma(-t, Q[1], g)};
    }
    // -g grad V = -g (x (1 + 2y), y - y^2 + x^2) with H = g M(1): the first row is H.xx x
    __device__ static __forceinline__ void force_hess(const Params&, const Hess& H, const double* Q, double g, double* F) {
        const double x = Q[0], y = Q[1];
        F[0] = -(H.xx * x);
        F[1] = g * fma(-x, x, fma(y, y, -y));
    }
    __device__ static __forceinline__ void apply(const Hess& H, const double* x, double* G) {
        G[0] = -fma(H.xx, x[0], H.xy * x[1]);
        G[1] = -fma(H.xy, x[0], H.yy * x[1]);
    }
    // G = -(V2'' + s V3''(Q)) x with the products of x formed BEFORE Q is needed: on a multi-lane tile Q
    // (the orbit's stage coordinates) arrives by shuffle while x is the lane's own column, so only two
    // dependent FMAs per component follow the shuffle (hess + apply: four levels).
    //   G0 = -(x0 + Qy (2s x0) + Qx (2s x1)),  G1 = -(x1 + Qx (2s x0) - Qy (2s x1))
    struct Pre { double u0, u1, x0, x1; };
    __device__ static __forceinline__ Pre pre(const Params&, const double* x, double s) {
        const double s2 = 2.0 * s;
        return Pre{s2 * x[0], s2 * x[1], x[0], x[1]};
    }
    __device__ static __forceinline__ void apply_pre(const Params&, const Pre& P, const double* Q, double* G) {
        G[0] = -fma(Q[1], P.u0, fma(Q[0], P.u1, P.x0));
        G[1] = -fma(Q[0], P.u0, fma(-Q[1], P.u1, P.x1));
    }
    __host__ static bool make_params(const double*, int, Params&) { return true; }
};

// 3-DoF coupled oscillators (BASELINE.json configs[3]):
// V = sum w_i^2 q_i^2/2 + eps q1^2 q2 + eps q2^2 q3; params (w1, w2, w3, eps).
struct Coupled3 {
    static constexpr int NDOF = 3;
    struct Params { double w1s, w2s, w3s, e; };
    struct Hess { double h11, h12, h22, h23, h33; };
    __device__ static __forceinline__ void force(const Params& P, const double* Q, double* F) {
        const double q1 = Q[0], q2 = Q[1], q3 = Q[2];
        F[0] = -P.w1s * q1 - 2.0 * P.e * q1 * q2;
        F[1] = -P.w2s * q2 - P.e * q1 * q1 - 2.0 * P.e * q2 * q3;
        F[2] = -P.w3s * q3 - P.e * q2 * q2;
    }
    // V_qq = [[w1^2+2e q2, 2e q1, 0],[2e q1, w2^2+2e q3, 2e q2],[0, 2e q2, w3^2]]
    __device__ static __forceinline__ Hess hess(const Params& P, const double* Q, double s, double g = 1.0) {
        const double te = 2.0 * P.e * s * g;
        return Hess{fma(te, Q[1], g * P.w1s), te * Q[0], fma(te, Q[2], g * P.w2s), te * Q[1], g * P.w3s};
    }
    // -g grad V with H = g M(1): h12 = 2 g e q1 and h23 = 2 g e q2 carry the quadratic terms, halved
    __device__ static __forceinline__ void force_hess(const Params&, const Hess& H, const double* Q, double, double* F) {
        F[0] = -(H.h11 * Q[0]);
        F[1] = -fma(H.h22, Q[1], 0.5 * H.h12 * Q[0]);
        F[2] = -fma(H.h33, Q[2], 0.5 * H.h23 * Q[1]);
    }
    __device__ static __forceinline__ void apply(const Hess& H, const double* x, double* G) {
        G[0] = -fma(H.h11, x[0], H.h12 * x[1]);
        G[1] = -fma(H.h12, x[0], fma(H.h22, x[1], H.h23 * x[2]));
        G[2] = -fma(H.h23, x[1], H.h33 * x[2]);
    }
    // as HenonHeiles::pre / apply_pre: with t_j = 2 e s x_j and v_j = w_j^2 x_j formed ahead of Q,
    //   G0 = -(v0 + Q1 t0 + Q0 t1),  G1 = -(v1 + Q0 t0 + Q2 t1 + Q1 t2),  G2 = -(v2 + Q1 t1)
    struct Pre { double t0, t1, t2, v0, v1, v2; };
    __device__ static __forceinline__ Pre pre(const Params& P, const double* x, double s) {
        const double te = 2.0 * P.e * s;
        return Pre{te * x[0], te * x[1], te * x[2], P.w1s * x[0], P.w2s * x[1], P.w3s * x[2]};
    }
    __device__ static __forceinline__ void apply_pre(const Params&, const Pre& R, const double* Q, double* G) {
        G[0] = -fma(Q[1], R.t0, fma(Q[0], R.t1, R.v0));
        G[1] = -fma(Q[0], R.t0, fma(Q[2], R.t1, fma(Q[1], R.t2, R.v1)));
        G[2] = -fma(Q[1], R.t1, R.v2);
    }
    __host__ static bool make_params(const double* p, int n, Params& out) {
        if (n < 4) return false;
        out = Params{p[0] * p[0], p[1] * p[1], p[2] * p[2], p[3]};
        return true;
    }
};

// FPUT chain with fixed ends, Eq.(6), Eq.(7), Eq.(8);
// N+1 springs (reading R4).  Spring force phi(d) = k d + alpha d^2 + beta d^3,
// stiffness g(d) = k + 2 alpha d + 3 beta d^2.  Used by the chain layout (lane = particle).
struct FputParams {
    double k, al, be, al2, be3;  // al2 = 2 alpha, be3 = 3 beta
    int np;                      // chain length N (padded tiles: the real length)
};
__device__ __forceinline__ double fput_phi(const FputParams& P, double d) {
    return d * fma(d, fma(P.be, d, P.al), P.k);
}
__device__ __forceinline__ double fput_g(const FputParams& P, double d) {
    return fma(d, fma(P.be3, d, P.al2), P.k);
}

}  // namespace chs
