/* oracle/chaos_oracle.c
 *
 * TEST INFRASTRUCTURE -- NOT PART OF THE PRODUCT PATH.
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
 * leg may build, load or call this file.  It shares no code, header, table or helper
 * with the CUDA path under paper_2507_00622_b200/csrc/.
 *
 * A plain, slow, obviously-correct CPU statement of the hot path of
 * arxiv 2507.00622 ("Chaoticus"): ensembles of independent initial conditions of a
 * Hamiltonian ODE integrated with the 12-stage Dormand-Prince 8(5,3) method
 * (PAPER.md:43), each trajectory carrying its variational
 * equations and a chaos indicator: SALI, GALI_k via SVD
 * (PAPER.md:55), the arc-length Lagrangian descriptor or
 * the Lyapunov spectrum via QR/Gram-Schmidt.
 *
 * Form: the GENERIC first-order Runge-Kutta form.  The whole augmented state
 * (orbit + k deviation vectors, D = n(1+k) components) is one ODE y' = f(y); all 12
 * stage derivative vectors k_i are formed and stored in full, in the order and with
 * the sums exactly as the tableau states them.  No blocking, no fusion, no
 * rearrangement for separable Hamiltonians.  Loops are  for ic { for step { ... } }.
 *
 * Precision: compiled twice, -DORC_REAL=double (timed CPU baseline) and
 * -DORC_REAL_IS_LONG_DOUBLE (x86 80-bit; the parity "truth").  Interfaces are double.
 *
 * Pins (tests/, -m "not gpu"): tableau order conditions; exp(At) of uncoupled
 * oscillators; order-8 slope; energy drift; SciPy rk_step / solve_ivp(DOP853) as
 * library routines; finite-difference deviation vectors; SALI==GALI_2 identity,
 * sum(lambda)=0 and pairing; LD closed form and mirror symmetry; LAPACK SVD.
 * Nothing here is "parity unpinned" (see DESIGN.md section "Oracle pins").
 *
 * Array layout at the interface (same as the library, so the seeded generators
 * serve both): structure of arrays, component-major / IC-minor:
 *   y[c*n_ic + ic], c < n ;  w[(v*n + c)*n_ic + ic], v < k.
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#include <float.h>
#include "dop853_tableau.h"

#ifdef ORC_REAL_IS_LONG_DOUBLE
typedef long double real;
#define R_SQRT sqrtl
#define R_FABS fabsl
#define R_LOG logl
#define R_POW powl
#define R_NEXTAFTER nextafterl
#else
typedef double real;
#define R_SQRT sqrt
#define R_FABS fabs
#define R_LOG log
#define R_POW pow
#define R_NEXTAFTER nextafter
#endif

#define ORC_OK 0
#define ORC_EINVAL 1

/* system ids: same numbering as the problem statement */
#define SYS_HENON_HEILES 0
#define SYS_COUPLED3 1
#define SYS_FPUT 2
#define SYS_DOUBLE_PENDULUM 3 /* PAPER.md:66-81, not separable */

/* per-trajectory status words */
#define ST_OK 0
#define ST_NONFINITE 1
#define ST_UNDERFLOW 2
#define ST_MAXSTEPS 3

typedef struct {
    int sys;
    const double *params;
    int n; /* phase-space dimension 2N, ordering y = (q_1..q_N, p_1..p_N) */
    int k; /* number of deviation vectors */
    int ld; /* 1: the state carries one more component M with M' = |f(y)|_2 (adaptive Lagrangian descriptor) */
} prob_t;

int orc_real_bytes(void) { return (int)sizeof(real); }

/* phase-space dimension of a system; <0 if unknown */
int orc_dim(int sys, const double *params)
{
    switch (sys) {
    case SYS_HENON_HEILES: return 4;
    case SYS_COUPLED3: return 6;
    case SYS_FPUT: {
        int N = (int)params[0];
        return N >= 1 ? 2 * N : -1;
    }
    case SYS_DOUBLE_PENDULUM: return 4;
    }
    return -1;
}

/* ------------------------------------------------------------------------------------
 * Right-hand sides.  y = (q, p);  qdot = p, pdot = -grad V(q).
 * Deviation vector w = (dq, dp): dqdot = dp, dpdot = -V_qq(q) dq  (variational
 * equations, ref [59]); V_qq is evaluated at the orbit value passed in.
 * ---------------------------------------------------------------------------------- */

/* Henon-Heiles, Eq.(4), Eq.(5).  q=(x,y), p=(px,py). */
static void hh_orbit(const real *y, real *f)
{
    real x = y[0], yy = y[1], px = y[2], py = y[3];
    f[0] = px;
    f[1] = py;
    f[2] = -x - 2 * x * yy;
    f[3] = -yy - x * x + yy * yy;
}
/* V_qq = [[1+2y, 2x],[2x, 1-2y]]  (second derivatives of Eq.(4)) */
static void hh_dev(const real *y, const real *w, real *g)
{
    real x = y[0], yy = y[1];
    real dx = w[0], dy = w[1], dpx = w[2], dpy = w[3];
    g[0] = dpx;
    g[1] = dpy;
    g[2] = -((1 + 2 * yy) * dx + 2 * x * dy);
    g[3] = -(2 * x * dx + (1 - 2 * yy) * dy);
}
static real hh_energy(const real *y)
{
    real x = y[0], yy = y[1], px = y[2], py = y[3];
    return (px * px + py * py) / 2 + (x * x + yy * yy) / 2 + x * x * yy - yy * yy * yy / 3;
}

/* 3-DoF coupled oscillators (BASELINE.json configs[3]):
 * H = 1/2 sum p_i^2 + 1/2 sum w_i^2 q_i^2 + eps q1^2 q2 + eps q2^2 q3; params = (w1,w2,w3,eps) */
static void c3_orbit(const double *P, const real *y, real *f)
{
    real w1 = P[0], w2 = P[1], w3 = P[2], e = P[3];
    real q1 = y[0], q2 = y[1], q3 = y[2];
    f[0] = y[3];
    f[1] = y[4];
    f[2] = y[5];
    f[3] = -w1 * w1 * q1 - 2 * e * q1 * q2;
    f[4] = -w2 * w2 * q2 - e * q1 * q1 - 2 * e * q2 * q3;
    f[5] = -w3 * w3 * q3 - e * q2 * q2;
}
static void c3_dev(const double *P, const real *y, const real *w, real *g)
{
    real w1 = P[0], w2 = P[1], w3 = P[2], e = P[3];
    real q1 = y[0], q2 = y[1], q3 = y[2];
    real h11 = w1 * w1 + 2 * e * q2, h12 = 2 * e * q1;
    real h22 = w2 * w2 + 2 * e * q3, h23 = 2 * e * q2;
    real h33 = w3 * w3;
    g[0] = w[3];
    g[1] = w[4];
    g[2] = w[5];
    g[3] = -(h11 * w[0] + h12 * w[1]);
    g[4] = -(h12 * w[0] + h22 * w[1] + h23 * w[2]);
    g[5] = -(h23 * w[1] + h33 * w[2]);
}
static real c3_energy(const double *P, const real *y)
{
    real w1 = P[0], w2 = P[1], w3 = P[2], e = P[3];
    real q1 = y[0], q2 = y[1], q3 = y[2];
    return (y[3] * y[3] + y[4] * y[4] + y[5] * y[5]) / 2 +
           (w1 * w1 * q1 * q1 + w2 * w2 * q2 * q2 + w3 * w3 * q3 * q3) / 2 + e * q1 * q1 * q2 +
           e * q2 * q2 * q3;
}

/* FPUT chain with fixed ends, Eq.(6), Eq.(7)
 * Eq.(8): q_0 = q_{N+1} = 0.  params = (N, k, alpha, beta).
 * With Dq_i = q_i - q_{i-1}, i = 1..N+1:
 *   pdot_i = -k[Dq_i - Dq_{i+1}] - alpha[Dq_i^2 - Dq_{i+1}^2] - beta[Dq_i^3 - Dq_{i+1}^3].
 * Reading (R4): the potential has N+1 springs (i = 0..N), which is what Eq.(7)
 * with Eq.(8) differentiates; Eq.(6)'s printed upper limit N would drop the wall spring. */
static real fput_q(const real *y, int N, int i) /* q_i with walls, i = 0..N+1 */
{
    return (i <= 0 || i >= N + 1) ? (real)0 : y[i - 1];
}
static void fput_orbit(const double *P, const real *y, real *f)
{
    int N = (int)P[0];
    real kk = P[1], al = P[2], be = P[3];
    for (int i = 1; i <= N; i++) {
        real di = fput_q(y, N, i) - fput_q(y, N, i - 1);      /* Dq_i     */
        real dn = fput_q(y, N, i + 1) - fput_q(y, N, i);      /* Dq_{i+1} */
        f[i - 1] = y[N + i - 1];
        f[N + i - 1] = -kk * (di - dn) - al * (di * di - dn * dn) - be * (di * di * di - dn * dn * dn);
    }
}
/* derivative of the spring force phi(d) = k d + alpha d^2 + beta d^3 */
static real fput_g(real kk, real al, real be, real d) { return kk + 2 * al * d + 3 * be * d * d; }
static void fput_dev(const double *P, const real *y, const real *w, real *g)
{
    int N = (int)P[0];
    real kk = P[1], al = P[2], be = P[3];
    for (int i = 1; i <= N; i++) {
        real di = fput_q(y, N, i) - fput_q(y, N, i - 1);
        real dn = fput_q(y, N, i + 1) - fput_q(y, N, i);
        real ddi = fput_q(w, N, i) - fput_q(w, N, i - 1);     /* d(Dq_i)     */
        real ddn = fput_q(w, N, i + 1) - fput_q(w, N, i);     /* d(Dq_{i+1}) */
        g[i - 1] = w[N + i - 1];
        g[N + i - 1] = -(fput_g(kk, al, be, di) * ddi - fput_g(kk, al, be, dn) * ddn);
    }
}
static real fput_energy(const double *P, const real *y)
{
    int N = (int)P[0];
    real kk = P[1], al = P[2], be = P[3];
    real H = 0;
    for (int i = 1; i <= N; i++) H += y[N + i - 1] * y[N + i - 1] / 2;
    for (int i = 1; i <= N + 1; i++) { /* N+1 springs */
        real d = fput_q(y, N, i) - fput_q(y, N, i - 1);
        H += kk * d * d / 2 + al * d * d * d / 3 + be * d * d * d * d / 4;
    }
    return H;
}

/* Dimensionless double pendulum, Eq.(1), Eq.(2), Eq.(3).
 * y = (theta1, theta2, p1, p2); params = (sigma, alpha) (mass ratio, length ratio).  NOT
 * separable: the kinetic energy depends on the angles.  Written exactly as printed:
 *   theta' = B^-1(x) p,  x = cos(theta1 - theta2)
 *   p'     = sin(Dtheta)/2 * (p^T C(x) p) * (1, -1)^T - (alpha (1+sigma) sin theta1, sin theta2)^T
 *   C(x)   = -B^-1 (dB/dx) B^-1, formed here by the two matrix products,
 * with B the inverse of Eq.(2): B = [[alpha^2 (1+sigma), alpha x],[alpha x, 1]], dB/dx = [[0,alpha],[alpha,0]]. */
static void dp_binv(real sg, real al, real x, real Bi[2][2])
{
    real den = 1 + sg - x * x;
    Bi[0][0] = 1 / (al * al) / den;
    Bi[0][1] = Bi[1][0] = -x / al / den;
    Bi[1][1] = (1 + sg) / den;
}
static void dp_orbit(const double *P, const real *y, real *f)
{
    real sg = P[0], al = P[1];
    real th1 = y[0], th2 = y[1], p1 = y[2], p2 = y[3];
    real dth = th1 - th2;
#ifdef ORC_REAL_IS_LONG_DOUBLE
    real x = cosl(dth), sd = sinl(dth), s1 = sinl(th1), s2 = sinl(th2);
#else
    real x = cos(dth), sd = sin(dth), s1 = sin(th1), s2 = sin(th2);
#endif
    real Bi[2][2], dB[2][2] = {{0, al}, {al, 0}}, T[2][2], C[2][2];
    dp_binv(sg, al, x, Bi);
    for (int i = 0; i < 2; i++)
        for (int j = 0; j < 2; j++) T[i][j] = Bi[i][0] * dB[0][j] + Bi[i][1] * dB[1][j];
    for (int i = 0; i < 2; i++)
        for (int j = 0; j < 2; j++) C[i][j] = -(T[i][0] * Bi[0][j] + T[i][1] * Bi[1][j]);
    real pCp = p1 * (C[0][0] * p1 + C[0][1] * p2) + p2 * (C[1][0] * p1 + C[1][1] * p2);
    f[0] = Bi[0][0] * p1 + Bi[0][1] * p2;
    f[1] = Bi[1][0] * p1 + Bi[1][1] * p2;
    f[2] = sd / 2 * pCp - al * (1 + sg) * s1;
    f[3] = -(sd / 2 * pCp) - s2;
}
/* Variational equations of Eq.(3) (deviation vectors "satisfy the variational equations of
 * the system"; the paper does not print them for this system): the derivative of the right-hand side above
 * along w = (dth1, dth2, dp1, dp2), term by term, with x = cos(Dtheta), s = sin(Dtheta), dD = dth1 - dth2,
 * dx = -s dD:
 *   d(theta')  = B^-1 dp + dx C p
 *   d(p'_1)    = dS - alpha (1+sigma) cos(theta1) dth1,   d(p'_2) = -dS - cos(theta2) dth2,
 *   S = (s/2) p^T C p,   dS = (x/2) dD p^T C p + (s/2) [2 p^T C dp + dx p^T C' p],
 *   C' = dC/dx = -(C B' B^-1 + B^-1 B' C)    (from C = -B^-1 B' B^-1 with B' = dB/dx constant),
 * every matrix formed by the products as written. */
static void mat2_mul(const real A[2][2], const real Bm[2][2], real Cm[2][2])
{
    for (int i = 0; i < 2; i++)
        for (int j = 0; j < 2; j++) Cm[i][j] = A[i][0] * Bm[0][j] + A[i][1] * Bm[1][j];
}
static real quad2(const real A[2][2], const real *u, const real *v) /* u^T A v */
{
    return u[0] * (A[0][0] * v[0] + A[0][1] * v[1]) + u[1] * (A[1][0] * v[0] + A[1][1] * v[1]);
}
static void dp_dev(const double *P, const real *y, const real *w, real *g)
{
    real sg = P[0], al = P[1];
    real th1 = y[0], th2 = y[1];
    const real *p = y + 2, *dth = w, *dpv = w + 2;
    real dth12 = th1 - th2;
#ifdef ORC_REAL_IS_LONG_DOUBLE
    real x = cosl(dth12), sn = sinl(dth12), c1 = cosl(th1), c2 = cosl(th2);
#else
    real x = cos(dth12), sn = sin(dth12), c1 = cos(th1), c2 = cos(th2);
#endif
    real Bi[2][2], dB[2][2] = {{0, al}, {al, 0}}, T[2][2], C[2][2], U[2][2], V[2][2], Cp[2][2];
    dp_binv(sg, al, x, Bi);
    mat2_mul(Bi, dB, T);
    mat2_mul(T, Bi, C);
    for (int i = 0; i < 2; i++)
        for (int j = 0; j < 2; j++) C[i][j] = -C[i][j];          /* C  = -B^-1 B' B^-1 */
    mat2_mul(C, dB, T);
    mat2_mul(T, Bi, U);                                          /* C B' B^-1 */
    mat2_mul(Bi, dB, T);
    mat2_mul(T, C, V);                                           /* B^-1 B' C */
    for (int i = 0; i < 2; i++)
        for (int j = 0; j < 2; j++) Cp[i][j] = -(U[i][j] + V[i][j]); /* C' */
    real dD = dth[0] - dth[1], dx = -sn * dD;
    real pCp = quad2(C, p, p);
    real dS = x / 2 * dD * pCp + sn / 2 * (2 * quad2(C, p, dpv) + dx * quad2(Cp, p, p));
    g[0] = Bi[0][0] * dpv[0] + Bi[0][1] * dpv[1] + dx * (C[0][0] * p[0] + C[0][1] * p[1]);
    g[1] = Bi[1][0] * dpv[0] + Bi[1][1] * dpv[1] + dx * (C[1][0] * p[0] + C[1][1] * p[1]);
    g[2] = dS - al * (1 + sg) * c1 * dth[0];
    g[3] = -dS - c2 * dth[1];
}
static real dp_energy(const double *P, const real *y)
{
    real sg = P[0], al = P[1];
    real th1 = y[0], th2 = y[1], p1 = y[2], p2 = y[3];
#ifdef ORC_REAL_IS_LONG_DOUBLE
    real x = cosl(th1 - th2), c1 = cosl(th1), c2 = cosl(th2);
#else
    real x = cos(th1 - th2), c1 = cos(th1), c2 = cos(th2);
#endif
    real Bi[2][2];
    dp_binv(sg, al, x, Bi);
    real T = (p1 * (Bi[0][0] * p1 + Bi[0][1] * p2) + p2 * (Bi[1][0] * p1 + Bi[1][1] * p2)) / 2;
    return T - al * (1 + sg) * c1 - c2;
}

/* f(y) for the augmented state  Y = (y, w_1, ..., w_k), each block of n components */
static void rhs_aug(const prob_t *pb, const real *Y, real *F)
{
    int n = pb->n;
    switch (pb->sys) {
    case SYS_HENON_HEILES:
        hh_orbit(Y, F);
        for (int v = 1; v <= pb->k; v++) hh_dev(Y, Y + v * n, F + v * n);
        break;
    case SYS_COUPLED3:
        c3_orbit(pb->params, Y, F);
        for (int v = 1; v <= pb->k; v++) c3_dev(pb->params, Y, Y + v * n, F + v * n);
        break;
    case SYS_FPUT:
        fput_orbit(pb->params, Y, F);
        for (int v = 1; v <= pb->k; v++) fput_dev(pb->params, Y, Y + v * n, F + v * n);
        break;
    case SYS_DOUBLE_PENDULUM:
        dp_orbit(pb->params, Y, F);
        for (int v = 1; v <= pb->k; v++) dp_dev(pb->params, Y, Y + v * n, F + v * n);
        break;
    }
    /* PAPER.md:39 "the Lagrangian Descriptor must be calculated alongside the trajectory's evolution":
     * the arc-length descriptor as one more component of the ODE, M' = |f(y)|_2 (R12, R21) */
    if (pb->ld) {
        real s2 = 0;
        for (int c = 0; c < n; c++) s2 += F[c] * F[c];
        F[n * (1 + pb->k)] = R_SQRT(s2);
    }
}

static real energy(const prob_t *pb, const real *y)
{
    switch (pb->sys) {
    case SYS_HENON_HEILES: return hh_energy(y);
    case SYS_COUPLED3: return c3_energy(pb->params, y);
    case SYS_FPUT: return fput_energy(pb->params, y);
    case SYS_DOUBLE_PENDULUM: return dp_energy(pb->params, y);
    }
    return 0;
}

/* ------------------------------------------------------------------------------------
 * One DOP853 step in the generic form:
 *   k_1 = f(y);  k_i = f(y + h sum_{j<i} a_ij k_j), i = 2..12;  y+ = y + h sum_i b_i k_i.
 * K holds the 12 stage derivative vectors (12 x D), Ys is scratch (D).
 * ---------------------------------------------------------------------------------- */
static void dop853_stages(const prob_t *pb, int D, const real *y, real h, real *K, real *Ys)
{
    for (int i = 0; i < ORC_S; i++) {
        for (int c = 0; c < D; c++) {
            real s = 0;
            for (int j = 0; j < i; j++) s += (real)ORC_A[i][j] * K[j * D + c];
            Ys[c] = y[c] + h * s;
        }
        rhs_aug(pb, Ys, K + i * D);
    }
}
static void dop853_solution(int D, const real *y, real h, const real *K, real *ynew)
{
    for (int c = 0; c < D; c++) {
        real s = 0;
        for (int i = 0; i < ORC_S; i++) s += (real)ORC_B[i] * K[i * D + c];
        ynew[c] = y[c] + h * s;
    }
}

/* Error estimate of an attempted step (R2, R3: textbook DOP853
 * combination of the 5th- and 3rd-order embedded differences, RMS over ALL D components,
 * scale_c = atol + rtol max(|y_c|, |y+_c|)). */
static real dop853_error_norm(int D, const real *y, const real *ynew, real h, const real *K,
                              real rtol, real atol)
{
    real S5 = 0, S3 = 0;
    for (int c = 0; c < D; c++) {
        real a = R_FABS(y[c]), b = R_FABS(ynew[c]);
        real scale = atol + rtol * (a > b ? a : b);
        real e5 = 0, e3 = 0;
        for (int i = 0; i < ORC_S; i++) {
            e5 += (real)ORC_E5[i] * K[i * D + c];
            e3 += (real)ORC_E3[i] * K[i * D + c];
        }
        e5 /= scale;
        e3 /= scale;
        S5 += e5 * e5;
        S3 += e3 * e3;
    }
    if (S5 == 0 && S3 == 0) return 0;
    real denom = S5 + (real)0.01 * S3;
    return R_FABS(h) * S5 / R_SQRT(denom * D);
}

static real rms_scaled(int D, const real *v, const real *scale)
{
    real s = 0;
    for (int c = 0; c < D; c++) {
        real x = v[c] / scale[c];
        s += x * x;
    }
    return R_SQRT(s / D);
}

/* Starting step size when h0 <= 0 (R2; textbook heuristic, HNW II.4, with
 * exponent 1/8).  Y: augmented state, scratch arrays of D. */
static real initial_step(const prob_t *pb, int D, const real *Y, real interval, real dir, real rtol,
                         real atol, real *f0, real *y1, real *f1, real *scale)
{
    if (interval == 0) return 0;
    rhs_aug(pb, Y, f0);
    for (int c = 0; c < D; c++) scale[c] = atol + R_FABS(Y[c]) * rtol;
    real d0 = rms_scaled(D, Y, scale), d1 = rms_scaled(D, f0, scale);
    real ha = (d0 < (real)1e-5 || d1 < (real)1e-5) ? (real)1e-6 : (real)0.01 * d0 / d1;
    if (ha > interval) ha = interval;
    for (int c = 0; c < D; c++) y1[c] = Y[c] + ha * dir * f0[c];
    rhs_aug(pb, y1, f1);
    for (int c = 0; c < D; c++) f1[c] -= f0[c];
    real d2 = rms_scaled(D, f1, scale) / ha;
    real hb;
    if (d1 <= (real)1e-15 && d2 <= (real)1e-15) {
        hb = (real)1e-3 * ha;
        if (hb < (real)1e-6) hb = (real)1e-6;
    } else {
        hb = R_POW((real)0.01 / (d1 > d2 ? d1 : d2), (real)1 / 8);
    }
    real h = 100 * ha;
    if (hb < h) h = hb;
    if (interval < h) h = interval;
    return h;
}

/* ------------------------------------------------------------------------------------
 * Indicator arithmetic on the k deviation vectors W (k blocks of n, inside the augmented
 * state).
 * ---------------------------------------------------------------------------------- */
static real vnorm(int n, const real *w)
{
    real s = 0;
    for (int c = 0; c < n; c++) s += w[c] * w[c];
    return R_SQRT(s);
}

/* Renormalisation: alpha_v = ||w_v||,
 * w_v <- w_v / alpha_v, L_v += ln alpha_v (if L != NULL).  No orthogonalisation. */
static void renormalise(int n, int k, real *W, real *L)
{
    for (int v = 0; v < k; v++) {
        real a = vnorm(n, W + v * n);
        for (int c = 0; c < n; c++) W[v * n + c] /= a;
        if (L) L[v] += R_LOG(a);
    }
}

/* Modified Gram-Schmidt ("QR factorization"; BASELINE configs[3];
 * DESIGN.md "Lyapunov spectrum"): for v = 1..k: for j < v: w_v -= (q_j . w_v) q_j using
 * the UPDATED w_v; r_vv = ||w_v||; q_v = w_v / r_vv; S_v += ln r_vv. */
static void mgs(int n, int k, real *W, real *S)
{
    for (int v = 0; v < k; v++) {
        for (int j = 0; j < v; j++) {
            real d = 0;
            for (int c = 0; c < n; c++) d += W[j * n + c] * W[v * n + c];
            for (int c = 0; c < n; c++) W[v * n + c] -= d * W[j * n + c];
        }
        real r = vnorm(n, W + v * n);
        for (int c = 0; c < n; c++) W[v * n + c] /= r;
        if (S) S[v] += R_LOG(r);
    }
}

/* SALI (refs [54,56,57]): min(||w1+w2||, ||w1-w2||) of the UNIT vectors. */
static real sali_of(int n, const real *W)
{
    real sp = 0, sm = 0;
    for (int c = 0; c < n; c++) {
        real a = W[c] + W[n + c], b = W[c] - W[n + c];
        sp += a * a;
        sm += b * b;
    }
    sp = R_SQRT(sp);
    sm = R_SQRT(sm);
    return sp < sm ? sp : sm;
}

/* GALI_k ("using Singular Value Decomposition", ref [58]): product of the k
 * singular values of the n x k matrix whose columns are the unit deviation vectors.
 * SVD by one-sided (Hestenes) Jacobi: rotate column pairs until mutually orthogonal;
 * the singular values are then the column norms.  Works on a copy. */
static real gali_of(int n, int k, const real *W, real *tmp /* k*n */)
{
    memcpy(tmp, W, sizeof(real) * (size_t)n * k);
    real eps = (sizeof(real) > 8) ? (real)1e-19 : (real)1e-16;
    for (int sweep = 0; sweep < 60; sweep++) {
        int rotated = 0;
        for (int p = 0; p < k - 1; p++)
            for (int q = p + 1; q < k; q++) {
                real app = 0, aqq = 0, apq = 0;
                for (int c = 0; c < n; c++) {
                    app += tmp[p * n + c] * tmp[p * n + c];
                    aqq += tmp[q * n + c] * tmp[q * n + c];
                    apq += tmp[p * n + c] * tmp[q * n + c];
                }
                if (R_FABS(apq) <= eps * R_SQRT(app * aqq)) continue;
                rotated = 1;
                real zeta = (aqq - app) / (2 * apq);
                real t = (zeta >= 0 ? 1 : -1) / (R_FABS(zeta) + R_SQRT(1 + zeta * zeta));
                real cs = 1 / R_SQRT(1 + t * t), sn = cs * t;
                for (int c = 0; c < n; c++) {
                    real xp = tmp[p * n + c], xq = tmp[q * n + c];
                    tmp[p * n + c] = cs * xp - sn * xq;
                    tmp[q * n + c] = sn * xp + cs * xq;
                }
            }
        if (!rotated) break;
    }
    real g = 1;
    for (int v = 0; v < k; v++) g *= vnorm(n, tmp + v * n);
    return g;
}

/* ------------------------------------------------------------------------------------
 * One trajectory, start to end.  Y = augmented state (D = n(1+k)), advanced in place.
 * ---------------------------------------------------------------------------------- */
#define MODE_NONE 0   /* deviation vectors (if any) integrated, never touched           */
#define MODE_NORM 1   /* renormalise every m accepted steps (SALI, GALI, mLE)           */
#define MODE_MGS 2    /* modified Gram-Schmidt every m accepted steps (Lyapunov)        */
#define IND_NONE 0
#define IND_SALI 1
#define IND_GALI 2

typedef struct {
    int adaptive;
    real t0, h;           /* fixed: signed step */
    long long n_steps;    /* fixed */
    real t_end, rtol, atol, h0; /* adaptive; h0 <= 0: automatic */
    long long max_steps;  /* adaptive: bound on attempted steps; <= 0: none */
} stepper_t;

typedef struct {
    long long n_acc, n_rej;
    int status;
    real t_final;
    double *t_rec;      /* optional: accepted step times are recorded here (pins only) */
    long long max_rec;
} report_t;

typedef struct { /* scratch for one trajectory */
    real *K, *Ys, *Ynew, *tmp, *f0, *f1, *scale;
} work_t;

static int work_alloc(work_t *w, int D)
{
    w->K = malloc(sizeof(real) * ORC_S * (size_t)D);
    w->Ys = malloc(sizeof(real) * (size_t)D);
    w->Ynew = malloc(sizeof(real) * (size_t)D);
    w->tmp = malloc(sizeof(real) * (size_t)D);
    w->f0 = malloc(sizeof(real) * (size_t)D);
    w->f1 = malloc(sizeof(real) * (size_t)D);
    w->scale = malloc(sizeof(real) * (size_t)D);
    return w->K && w->Ys && w->Ynew && w->tmp && w->f0 && w->f1 && w->scale;
}
static void work_free(work_t *w)
{
    free(w->K); free(w->Ys); free(w->Ynew); free(w->tmp); free(w->f0); free(w->f1); free(w->scale);
}

static int all_finite(int D, const real *Y)
{
    for (int c = 0; c < D; c++)
        if (!isfinite((double)Y[c])) return 0;
    return 1;
}

static real indicator_value(const prob_t *pb, int indicator, const real *Y, real *tmp)
{
    const real *W = Y + pb->n;
    if (indicator == IND_SALI) return sali_of(pb->n, W);
    if (indicator == IND_GALI) return gali_of(pb->n, pb->k, W, tmp);
    return 0;
}

/* does the renormalisation of `mode`; accumulates logs into L (k values) */
static void do_renorm(const prob_t *pb, int mode, real *Y, real *L)
{
    if (mode == MODE_NORM) renormalise(pb->n, pb->k, Y + pb->n, L);
    else if (mode == MODE_MGS) mgs(pb->n, pb->k, Y + pb->n, L);
}

/* series: n_samples values for this trajectory written at series[s*series_stride] */
static void run_traj(const prob_t *pb, real *Y, const stepper_t *st, int mode, int indicator, int m,
                     int sample_every, long long n_samples, double *series, long long series_stride,
                     real *L, report_t *rep, work_t *wk)
{
    int D = pb->n * (1 + pb->k) + pb->ld;
    long long n_renorm = 0, slot = 0;
    rep->n_acc = rep->n_rej = 0;
    rep->status = ST_OK;
    rep->t_final = st->t0;

    /* on entry: normalise / orthonormalise once, no log accumulated (R6) */
    do_renorm(pb, mode, Y, NULL);

    if (!st->adaptive) {
        /* fixed step */
        for (long long s = 1; s <= st->n_steps; s++) {
            dop853_stages(pb, D, Y, st->h, wk->K, wk->Ys);
            dop853_solution(D, Y, st->h, wk->K, wk->Ynew);
            memcpy(Y, wk->Ynew, sizeof(real) * (size_t)D);
            rep->n_acc++;
            rep->t_final = st->t0 + (real)s * st->h;
            if (!all_finite(D, Y)) { rep->status = ST_NONFINITE; break; }
            if (mode != MODE_NONE && (s % m == 0 || s == st->n_steps)) {
                do_renorm(pb, mode, Y, L);
                n_renorm++;
                if (series && sample_every > 0 && n_renorm % sample_every == 0 && slot < n_samples - 1)
                    series[(slot++) * series_stride] = (double)indicator_value(pb, indicator, Y, wk->tmp);
            }
        }
    } else {
        /* adaptive step (R2: SciPy-style controller) */
        const real SAFETY = (real)0.9, MIN_FACTOR = (real)0.2, MAX_FACTOR = 10;
        const real EXPO = -(real)1 / 8;
        real t = st->t0;
        real dir = (st->t_end >= st->t0) ? 1 : -1;
        real h_abs = st->h0 > 0 ? st->h0
                                : initial_step(pb, D, Y, R_FABS(st->t_end - st->t0), dir, st->rtol,
                                               st->atol, wk->f0, wk->Ynew, wk->f1, wk->scale);
        long long attempts = 0;
        while (dir * (st->t_end - t) > 0 && rep->status == ST_OK) {
            real min_step = 10 * R_FABS(R_NEXTAFTER(t, dir * (real)INFINITY) - t);
            if (h_abs < min_step) h_abs = min_step;
            int accepted = 0, rejected = 0;
            while (!accepted) {
                if (h_abs < min_step) { rep->status = ST_UNDERFLOW; break; }
                if (st->max_steps > 0 && attempts >= st->max_steps) { rep->status = ST_MAXSTEPS; break; }
                attempts++;
                real h = h_abs * dir, t_new = t + h;
                if (dir * (t_new - st->t_end) > 0) t_new = st->t_end; /* land exactly on t_end */
                h = t_new - t;
                h_abs = R_FABS(h);
                dop853_stages(pb, D, Y, h, wk->K, wk->Ys);
                dop853_solution(D, Y, h, wk->K, wk->Ynew);
                real err = dop853_error_norm(D, Y, wk->Ynew, h, wk->K, st->rtol, st->atol);
                if (err < 1) {
                    real factor = (err == 0) ? MAX_FACTOR : SAFETY * R_POW(err, EXPO);
                    if (factor > MAX_FACTOR) factor = MAX_FACTOR;
                    if (rejected && factor > 1) factor = 1;
                    h_abs *= factor;
                    accepted = 1;
                    t = t_new;
                    memcpy(Y, wk->Ynew, sizeof(real) * (size_t)D);
                    if (rep->t_rec && rep->n_acc < rep->max_rec) rep->t_rec[rep->n_acc] = (double)t;
                    rep->n_acc++;
                } else if (err >= 1) {
                    real factor = SAFETY * R_POW(err, EXPO);
                    if (factor < MIN_FACTOR) factor = MIN_FACTOR;
                    h_abs *= factor;
                    rejected = 1;
                    rep->n_rej++;
                } else { /* NaN */
                    rep->status = ST_NONFINITE;
                    break;
                }
            }
            if (rep->status != ST_OK) break;
            rep->t_final = t;
            if (!all_finite(D, Y)) { rep->status = ST_NONFINITE; break; }
            if (mode != MODE_NONE && (rep->n_acc % m == 0 || !(dir * (st->t_end - t) > 0))) {
                do_renorm(pb, mode, Y, L);
                n_renorm++;
            }
        }
    }
    /* final value: indicator at the end time, from the unit vectors of the last
     * renormalisation (or of the entry normalisation when no step was taken) */
    if (series) {
        double v = (double)indicator_value(pb, indicator, Y, wk->tmp);
        if (rep->status != ST_OK) v = NAN;
        series[(n_samples - 1) * series_stride] = v;
        if (rep->status != ST_OK)
            for (long long s2 = slot; s2 < n_samples - 1; s2++) series[s2 * series_stride] = NAN;
    }
}

/* number of series slots for a fixed-step run */
long long orc_n_samples(long long n_steps, int renorm_every, int sample_every)
{
    if (sample_every <= 0) return 1;
    long long n_renorm = (n_steps + renorm_every - 1) / renorm_every;
    return n_renorm / sample_every + 1;
}

/* ------------------------------------------------------------------------------------
 * Exported ensemble entry points.  for ic { for step { ... } }, ICs spread over
 * n_threads host threads (OpenMP; trajectories are independent).
 * ---------------------------------------------------------------------------------- */
static void gather(long long n_ic, long long ic, int n, int k, const double *y, const double *w, real *Y)
{
    for (int c = 0; c < n; c++) Y[c] = y[(long long)c * n_ic + ic];
    for (int v = 0; v < k; v++)
        for (int c = 0; c < n; c++) Y[(v + 1) * n + c] = w[((long long)v * n + c) * n_ic + ic];
}
static void scatter(long long n_ic, long long ic, int n, int k, const real *Y, double *y, double *w, int bad)
{
    for (int c = 0; c < n; c++) y[(long long)c * n_ic + ic] = bad ? NAN : (double)Y[c];
    for (int v = 0; v < k; v++)
        for (int c = 0; c < n; c++)
            w[((long long)v * n + c) * n_ic + ic] = bad ? NAN : (double)Y[(v + 1) * n + c];
}

/* General run.  y [n][n_ic] in/out; w [k][n][n_ic] in/out (k may be 0, w NULL).
 * series [n_samples][n_ic] or NULL; logacc [k][n_ic] in/out accumulators or NULL (the run
 * ADDS its sum of ln(alpha_v) resp. ln(r_vv)); lambda [k][n_ic] or NULL = this run's sums
 * divided by the LENGTH |t_final - t0| of this run's time interval (R18: an exponent
 * is a growth rate per unit of elapsed |t|, also for backward-time runs).  Report arrays may be NULL. */
int orc_run(int sys, const double *params, long long n_ic, double *y, double *w, int k, int adaptive,
            double t0, double h, long long n_steps, double t_end, double rtol, double atol, double h0,
            long long max_steps, int mode, int indicator, int renorm_every, int sample_every,
            double *series, double *logacc, double *lambda, long long *n_acc, long long *n_rej,
            int *status, double *t_final, int n_threads)
{
    int n = orc_dim(sys, params);
    if (n < 0 || n_ic < 0 || k < 0 || (k > 0 && !w) || !y) return ORC_EINVAL;
    if (mode != MODE_NONE && (k < 1 || renorm_every < 1)) return ORC_EINVAL;
    if (indicator == IND_SALI && k != 2) return ORC_EINVAL;
    if (indicator == IND_GALI && (k < 2 || k > n)) return ORC_EINVAL;
    if (mode == MODE_MGS && k > n) return ORC_EINVAL;
    if (!adaptive && (h == 0 || n_steps < 0)) return ORC_EINVAL;
    if (adaptive && (!(rtol > 0) || !(atol > 0) || sample_every > 0)) return ORC_EINVAL;
    prob_t pb = {sys, params, n, k};
    stepper_t st = {adaptive, t0, h, n_steps, t_end, rtol, atol, h0, max_steps};
    int D = n * (1 + k);
    long long n_samples = adaptive ? 1 : orc_n_samples(n_steps, renorm_every < 1 ? 1 : renorm_every, sample_every);
    int m = renorm_every < 1 ? 1 : renorm_every;
    int fail = 0;
    if (n_threads < 1) n_threads = 1;
#pragma omp parallel num_threads(n_threads)
    {
        work_t wk;
        real *Y = malloc(sizeof(real) * (size_t)D);
        real *L = malloc(sizeof(real) * (size_t)(k > 0 ? k : 1));
        int ok = work_alloc(&wk, D) && Y && L;
        if (!ok) {
#pragma omp atomic write
            fail = 1;
        }
#pragma omp for schedule(dynamic, 16)
        for (long long ic = 0; ic < n_ic; ic++) {
            if (!ok) continue;
            report_t rep;
            memset(&rep, 0, sizeof rep);
            gather(n_ic, ic, n, k, y, w, Y);
            for (int v = 0; v < k; v++) L[v] = 0;
            run_traj(&pb, Y, &st, mode, indicator, m, sample_every, n_samples, series ? series + ic : NULL,
                     n_ic, L, &rep, &wk);
            int bad = rep.status != ST_OK;
            scatter(n_ic, ic, n, k, Y, y, w, bad);
            real elapsed = rep.t_final - st.t0;
            for (int v = 0; v < k; v++) {
                if (logacc) logacc[(long long)v * n_ic + ic] = bad ? NAN : logacc[(long long)v * n_ic + ic] + (double)L[v];
                if (lambda) lambda[(long long)v * n_ic + ic] = (bad || elapsed == 0) ? NAN : (double)(L[v] / R_FABS(elapsed));
            }
            if (n_acc) n_acc[ic] = rep.n_acc;
            if (n_rej) n_rej[ic] = rep.n_rej;
            if (status) status[ic] = rep.status;
            if (t_final) t_final[ic] = (double)rep.t_final;
        }
        if (ok) work_free(&wk);
        free(Y);
        free(L);
    }
    return fail ? ORC_EINVAL : ORC_OK;
}

/* Lagrangian descriptor, arc-length integrand (BASELINE
 * configs[1]): M' = ||f(x)||_2 appended to the ODE and
 * integrated with the same tableau; because M' does not depend on M this is exactly
 *   M+ = M + |h| sum_i b_i ||k_i||_2   with k_i the orbit stage derivatives.
 * Forward: step +h from y0; backward: step -h from the same y0.  y0 is not modified. */
int orc_ld(int sys, const double *params, long long n_ic, const double *y0, double t0, double h,
           long long n_steps, double *ld_fwd, double *ld_bwd, int n_threads)
{
    int n = orc_dim(sys, params);
    (void)t0; /* autonomous systems: time is bookkeeping only */
    if (n < 0 || n_ic < 0 || !y0 || !(h > 0) || n_steps < 0) return ORC_EINVAL;
    prob_t pb = {sys, params, n, 0};
    if (n_threads < 1) n_threads = 1;
#pragma omp parallel num_threads(n_threads)
    {
        work_t wk;
        real *Y = malloc(sizeof(real) * (size_t)n);
        int ok = work_alloc(&wk, n) && Y;
#pragma omp for schedule(dynamic, 16)
        for (long long ic = 0; ic < n_ic; ic++) {
            if (!ok) continue;
            for (int pass = 0; pass < 2; pass++) {
                double *out = pass == 0 ? ld_fwd : ld_bwd;
                if (!out) continue;
                real hs = pass == 0 ? (real)h : -(real)h;
                real M = 0;
                gather(n_ic, ic, n, 0, y0, NULL, Y);
                for (long long s = 0; s < n_steps; s++) {
                    dop853_stages(&pb, n, Y, hs, wk.K, wk.Ys);
                    real acc = 0;
                    for (int i = 0; i < ORC_S; i++) acc += (real)ORC_B[i] * vnorm(n, wk.K + i * n);
                    M += R_FABS(hs) * acc;
                    dop853_solution(n, Y, hs, wk.K, wk.Ynew);
                    memcpy(Y, wk.Ynew, sizeof(real) * (size_t)n);
                }
                out[ic] = all_finite(n, Y) ? (double)M : NAN;
            }
        }
        if (ok) work_free(&wk);
        free(Y);
    }
    return ORC_OK;
}

/* Lagrangian descriptors of an initial condition AND of its 2n axis neighbours (PAPER.md:57-58:
 * "Generation of neighbouring trajectories for the calculation of the chaos indicators based on
 * Lagrangian Descriptors").  For every IC x0 the members are
 *   m = 0: x0;   m = 1 + 2i: x0 + sigma e_i;   m = 2 + 2i: x0 - sigma e_i,   i = 0..n-1,
 * e_i the unit vector of phase-space component i in the library's ordering (q_1..q_N, p_1..p_N).
 * Each member's forward / backward LD is orc_ld of the displaced initial condition -- a plain loop.
 * ld_fwd, ld_bwd: [1+2n][n_ic] (row = member), either may be NULL.
 * diff_fwd, diff_bwd: [2n][n_ic] or NULL, the raw differences |M(x0 +- sigma e_i) - M(x0)|
 * (row 2i: +, row 2i+1: -).  The LD-based chaos indicators of refs [11,26,68,10,31] are built from
 * these differences; their final scalar formulas are only CITED by the paper, not printed,
 * and are therefore not restated here (R19): this function stops at what the paper defines. */
int orc_ld_neighbours(int sys, const double *params, long long n_ic, const double *y0, double sigma,
                      double t0, double h, long long n_steps, double *ld_fwd, double *ld_bwd,
                      double *diff_fwd, double *diff_bwd, int n_threads)
{
    int n = orc_dim(sys, params);
    if (n < 0 || n_ic < 0 || !y0 || !(h > 0) || n_steps < 0 || !(sigma >= 0)) return ORC_EINVAL;
    if ((diff_fwd && !ld_fwd) || (diff_bwd && !ld_bwd)) return ORC_EINVAL;
    double *yd = malloc(sizeof(double) * (size_t)n * (size_t)(n_ic > 0 ? n_ic : 1));
    if (!yd) return ORC_EINVAL;
    int rc = ORC_OK;
    for (int m = 0; m < 1 + 2 * n && rc == ORC_OK; m++) {
        memcpy(yd, y0, sizeof(double) * (size_t)n * (size_t)n_ic);
        if (m > 0) {
            int i = (m - 1) / 2;
            double delta = ((m - 1) % 2 == 0) ? sigma : -sigma;
            for (long long ic = 0; ic < n_ic; ic++) yd[(long long)i * n_ic + ic] = y0[(long long)i * n_ic + ic] + delta;
        }
        rc = orc_ld(sys, params, n_ic, yd, t0, h, n_steps, ld_fwd ? ld_fwd + (long long)m * n_ic : NULL,
                    ld_bwd ? ld_bwd + (long long)m * n_ic : NULL, n_threads);
    }
    free(yd);
    if (rc != ORC_OK) return rc;
    for (int pass = 0; pass < 2; pass++) {
        const double *M = pass == 0 ? ld_fwd : ld_bwd;
        double *D = pass == 0 ? diff_fwd : diff_bwd;
        if (!D) continue;
        for (int r = 0; r < 2 * n; r++)
            for (long long ic = 0; ic < n_ic; ic++) D[(long long)r * n_ic + ic] = fabs(M[(long long)(r + 1) * n_ic + ic] - M[ic]);
    }
    return ORC_OK;
}

/* ------------------------------------------------------------------------------------
 * Small single-trajectory entry points used only by the pins.
 * ---------------------------------------------------------------------------------- */

/* Lagrangian descriptor with the ADAPTIVE solver ("DOP 8(5) ODE solver with adaptive step size",
 * PAPER.md:39 the descriptor "calculated alongside the trajectory's evolution"; R21): the
 * augmented ODE (y, M), M' = |f(y)|_2, M(t0) = 0, through the same adaptive stepper as every other run --
 * M is one more component of the state, so it takes part in the error norm (D = n + 1) like any other.
 * Forward: t0 -> t0 + tau, ld_fwd = M.  Backward: t0 -> t0 - tau, where M decreases: ld_bwd = -M.
 * n_acc, n_rej, status: [2][n_ic] (row 0 forward, row 1 backward) or NULL.  A trajectory whose run does not
 * end with status 0 gets NaN. */
int orc_ld_adaptive(int sys, const double *params, long long n_ic, const double *y0, double t0, double tau,
                    double rtol, double atol, double h0, long long max_steps, double *ld_fwd, double *ld_bwd,
                    long long *n_acc, long long *n_rej, int *status, int n_threads)
{
    int n = orc_dim(sys, params);
    if (n < 0 || n_ic < 0 || !y0 || !(tau >= 0) || !(rtol > 0) || !(atol > 0)) return ORC_EINVAL;
    prob_t pb = {sys, params, n, 0, 1};
    int D = n + 1;
    if (n_threads < 1) n_threads = 1;
#pragma omp parallel num_threads(n_threads)
    {
        work_t wk;
        real *Y = malloc(sizeof(real) * (size_t)D);
        int ok = work_alloc(&wk, D) && Y;
#pragma omp for schedule(dynamic, 16)
        for (long long ic = 0; ic < n_ic; ic++) {
            if (!ok) continue;
            for (int pass = 0; pass < 2; pass++) {
                double *out = pass == 0 ? ld_fwd : ld_bwd;
                if (!out) continue;
                gather(n_ic, ic, n, 0, y0, NULL, Y);
                Y[n] = 0;
                stepper_t st = {1, (real)t0, 0, 0, pass == 0 ? (real)t0 + (real)tau : (real)t0 - (real)tau,
                                (real)rtol, (real)atol, (real)h0, max_steps};
                report_t rep = {0, 0, 0, 0, NULL, 0};
                run_traj(&pb, Y, &st, MODE_NONE, IND_NONE, 1, 0, 1, NULL, 0, NULL, &rep, &wk);
                int good = rep.status == ST_OK && all_finite(D, Y);
                out[ic] = good ? (double)(pass == 0 ? Y[n] : -Y[n]) : NAN;
                if (n_acc) n_acc[(long long)pass * n_ic + ic] = rep.n_acc;
                if (n_rej) n_rej[(long long)pass * n_ic + ic] = rep.n_rej;
                if (status) status[(long long)pass * n_ic + ic] = rep.status;
            }
        }
        if (ok) work_free(&wk);
        free(Y);
    }
    return ORC_OK;
}

/* f(Y) for one augmented state (AoS: y then w_1..w_k) */
int orc_rhs(int sys, const double *params, int k, const double *Y, double *F)
{
    int n = orc_dim(sys, params);
    if (n < 0) return ORC_EINVAL;
    int D = n * (1 + k);
    prob_t pb = {sys, params, n, k};
    real *a = malloc(sizeof(real) * D), *b = malloc(sizeof(real) * D);
    for (int c = 0; c < D; c++) a[c] = Y[c];
    rhs_aug(&pb, a, b);
    for (int c = 0; c < D; c++) F[c] = (double)b[c];
    free(a); free(b);
    return ORC_OK;
}
int orc_energy(int sys, const double *params, long long n_ic, const double *y, double *H)
{
    int n = orc_dim(sys, params);
    if (n < 0) return ORC_EINVAL;
    prob_t pb = {sys, params, n, 0};
    real *a = malloc(sizeof(real) * n);
    for (long long ic = 0; ic < n_ic; ic++) {
        for (int c = 0; c < n; c++) a[c] = y[(long long)c * n_ic + ic];
        H[ic] = (double)energy(&pb, a);
    }
    free(a);
    return ORC_OK;
}
/* one step on one augmented state; Kout (12*D) and err (given rtol, atol) optional */
int orc_step(int sys, const double *params, int k, double *Y, double h, double *Kout, double rtol,
             double atol, double *err)
{
    int n = orc_dim(sys, params);
    if (n < 0) return ORC_EINVAL;
    int D = n * (1 + k);
    prob_t pb = {sys, params, n, k};
    work_t wk;
    if (!work_alloc(&wk, D)) return ORC_EINVAL;
    real *a = malloc(sizeof(real) * D);
    for (int c = 0; c < D; c++) a[c] = Y[c];
    dop853_stages(&pb, D, a, (real)h, wk.K, wk.Ys);
    dop853_solution(D, a, (real)h, wk.K, wk.Ynew);
    if (err) *err = (double)dop853_error_norm(D, a, wk.Ynew, (real)h, wk.K, (real)rtol, (real)atol);
    if (Kout) for (int i = 0; i < ORC_S * D; i++) Kout[i] = (double)wk.K[i];
    for (int c = 0; c < D; c++) Y[c] = (double)wk.Ynew[c];
    free(a);
    work_free(&wk);
    return ORC_OK;
}
/* adaptive run of ONE augmented state without renormalisation, recording the accepted
 * step times (for the pin against scipy.integrate.solve_ivp(method="DOP853")).  Runs the
 * same run_traj as the ensemble entry point. */
int orc_trace_adaptive(int sys, const double *params, int k, double *Y, double t0, double t_end,
                       double rtol, double atol, double h0, long long max_rec, double *t_rec,
                       long long *n_acc, long long *n_rej)
{
    int n = orc_dim(sys, params);
    if (n < 0) return ORC_EINVAL;
    int D = n * (1 + k);
    prob_t pb = {sys, params, n, k};
    work_t wk;
    if (!work_alloc(&wk, D)) return ORC_EINVAL;
    real *a = malloc(sizeof(real) * D);
    for (int c = 0; c < D; c++) a[c] = Y[c];
    stepper_t st = {1, (real)t0, 0, 0, (real)t_end, (real)rtol, (real)atol, (real)h0, 0};
    report_t rep;
    memset(&rep, 0, sizeof rep);
    rep.t_rec = t_rec;
    rep.max_rec = max_rec;
    run_traj(&pb, a, &st, MODE_NONE, IND_NONE, 1, 0, 1, NULL, 0, NULL, &rep, &wk);
    for (int c = 0; c < D; c++) Y[c] = (double)a[c];
    *n_acc = rep.n_acc;
    *n_rej = rep.n_rej;
    free(a);
    work_free(&wk);
    return rep.status == ST_OK ? ORC_OK : ORC_EINVAL;
}
/* indicator arithmetic on k vectors given AoS (k blocks of n): mode 0: SALI (k = 2),
 * 1: GALI_k, 2: renormalise (logs out), 3: MGS (logs out).  W is modified for 2, 3. */
int orc_indicator(int what, int n, int k, double *W, double *out)
{
    real *a = malloc(sizeof(real) * (size_t)n * k), *tmp = malloc(sizeof(real) * (size_t)n * k);
    real *L = calloc((size_t)k, sizeof(real));
    for (int c = 0; c < n * k; c++) a[c] = W[c];
    if (what == 0) out[0] = (double)sali_of(n, a);
    else if (what == 1) out[0] = (double)gali_of(n, k, a, tmp);
    else if (what == 2) renormalise(n, k, a, L);
    else if (what == 3) mgs(n, k, a, L);
    if (what >= 2) {
        for (int v = 0; v < k; v++) out[v] = (double)L[v];
        for (int c = 0; c < n * k; c++) W[c] = (double)a[c];
    }
    free(a); free(tmp); free(L);
    return ORC_OK;
}
