// col_kernels.cuh -- "column layout" step kernels and the layout-generic run / LD kernels
// (CUDA path, sm_100a).
//
// A trajectory's augmented state is 1 + K columns of n = 2 NDOF components: column 0 the orbit,
// columns 1..K the deviation vectors.  The columns are dealt to a tile of L
// consecutive lanes, CPL = ceil((1+K)/L) columns per lane:
//   L = 1  : one trajectory per thread, everything in registers (Henon-Heiles, K <= 3);
//   L > 1  : CPL columns per lane for mid-size states and for small ensembles (3-DoF Lyapunov
//            spectrum: L = 4, CPL = 2; Henon-Heiles SALI up to 4096 trajectories: L = 4, CPL = 1);
//            the orbit's stage coordinates are broadcast from lane 0 by shuffle each stage,
//            Gram-Schmidt broadcasts one column at a time.
// HBM layout is structure-of-arrays (include/chaoticus.h); it is touched once at the start
// and once at the end of a call, everything in between runs out of registers.
//
// run_kernel<C, MODE, IND, ADAPT> and ld_kernel<C> are written against the per-lane state class C
// of a layout (Col<Sys,K,L> here, Chain<NP,K> in chain_kernels.cuh): C::NI (q, p) pairs per lane,
// C::L lanes per trajectory, load/store, force, do_renorm, indicator, finite_all, on_mask,
// store_logs.
#pragma once
#include <cmath>
#include "dop8_core.cuh"
#include "systems.cuh"

namespace chs {

enum : int { MODE_NONE = 0, MODE_NORM = 1, MODE_MGS = 2 };
enum : int { IND_NONE = 0, IND_SALI = 1, IND_GALI = 2 };

struct RunArgs {
    long long n_ic;
    double* y;   // [n][n_ic]
    double* w;   // [K][n][n_ic]
    // fixed
    double h;
    long long n_steps;
    // adaptive
    double t0, t_end, rtol, atol, h0;
    long long max_steps;
    // renormalisation / sampling
    int m;
    int sample_every;
    long long n_samples;
    // outputs (may be null)
    double* series;  // [n_samples][n_ic]
    double* logacc;  // [K][n_ic]  +=
    double* lambda;  // [K][n_ic]
    long long* n_acc;
    long long* n_rej;
    int* status;
    double* t_final;
    // continuation (include/chaoticus.h chs_report): carried rounding words of the orbit, [n][n_ic]
    double* carry;
    int resume;
    // Lagrangian descriptor
    const double* y0;
    double* ld_fwd;
    double* ld_bwd;
    // LD of neighbouring initial conditions: members per IC (1 = the IC itself only;
    // 1 + 2n = centre and x0 +- sigma e_i), outputs are [member][ic]
    int n_members;
    double sigma;
    // adaptive LD (run_kernel<..., LD = true>): which directions the tasks cover (0 forward, 1 backward)
    int dir_first, n_dirs;
    // adaptive runs: work queue for lane refill (device counter, zeroed before the launch), or null
    unsigned long long* queue;
};

// one-sided (Hestenes) Jacobi on k columns of n components held by ONE thread; returns the
// product of the singular values = GALI_k.  W is destroyed.
template <int N, int KK>
__device__ __forceinline__ double gali_thread(double (&W)[KK][N]) {
    const double eps = 8.9e-16;  // 4 ulp: |a_p . a_q| <= eps |a_p| |a_q|  => orthogonal
    for (int sweep = 0; sweep < 30; sweep++) {
        bool rotated = false;
#pragma unroll
        for (int p = 0; p < KK - 1; p++)
#pragma unroll
            for (int q2 = p + 1; q2 < KK; q2++) {
                double app = 0, aqq = 0, apq = 0;
#pragma unroll
                for (int c = 0; c < N; c++) {
                    app = fma(W[p][c], W[p][c], app);
                    aqq = fma(W[q2][c], W[q2][c], aqq);
                    apq = fma(W[p][c], W[q2][c], apq);
                }
                if (fabs(apq) > eps * sqrt(app * aqq)) {
                    rotated = true;
                    double zeta = (aqq - app) / (2.0 * apq);
                    double t = copysign(1.0, zeta) / (fabs(zeta) + sqrt(fma(zeta, zeta, 1.0)));
                    double cs = rsqrt(fma(t, t, 1.0)), sn = cs * t;
#pragma unroll
                    for (int c = 0; c < N; c++) {
                        double xp = W[p][c], xq = W[q2][c];
                        W[p][c] = cs * xp - sn * xq;
                        W[q2][c] = fma(sn, xp, cs * xq);
                    }
                }
            }
        if (!rotated) break;
    }
    double g = 1.0;
#pragma unroll
    for (int v = 0; v < KK; v++) {
        double s = 0;
#pragma unroll
        for (int c = 0; c < N; c++) s = fma(W[v][c], W[v][c], s);
        g *= sqrt(s);
    }
    return g;
}

// ---- per-lane view of one trajectory in the column layout -----------------------------------
template <class Sys, int K_, int L_>
struct Col {
    static constexpr int K = K_, L = L_;
    static constexpr int ND = Sys::NDOF;
    static constexpr int N = 2 * ND;
    static constexpr int NCOL = 1 + K;
    static constexpr int CPL = (NCOL + L - 1) / L;
    static constexpr int NI = CPL * ND;
    static constexpr int D = N * NCOL;
    static constexpr int NCOMP = ND;  // item j = 0: the orbit (lane 0) -- compensated update
    using Params = typename Sys::Params;

    Params prm;
    int lt;          // lane in tile
    double s_lane;   // 1/2 on the orbit lane of a multi-lane tile, else 1
    double q[NI], p[NI];
    static constexpr bool COLD = false;
    LogBank<CPL, false> lg;  // deferred-log accumulators of this lane's columns

    __device__ __forceinline__ double dcount() const { return (double)D; }
    // Which column sits in slot j of lane l.  Column 0 (the orbit) is slot 0 of lane 0.  When the other
    // lanes can hold all K deviation columns (ALONE), lane 0 holds nothing else: its remaining slots are
    // the tile's idle slots, and every lane needs ONE Hessian per force evaluation (lane 0: V2'' + V3''/2
    // for the orbit, the others: V2'' + V3'' for both of their columns).  Otherwise columns are dealt in
    // order, lane 0 mixes the orbit with deviation columns, and two Hessians are formed per lane.
    static constexpr bool ALONE = (L > 1) && ((L - 1) * CPL >= K);
    __host__ __device__ static constexpr int col_at(int lane, int j) {
        if (!ALONE) return lane * CPL + j;
        if (lane == 0) return j == 0 ? 0 : NCOL;               // NCOL and above: idle slot
        return 1 + (lane - 1) * CPL + j;
    }
    __host__ __device__ static constexpr int owner_of(int c) { return !ALONE ? c / CPL : (c == 0 ? 0 : 1 + (c - 1) / CPL); }
    __host__ __device__ static constexpr int slot_of(int c) { return !ALONE ? c % CPL : (c == 0 ? 0 : (c - 1) % CPL); }
    __device__ __forceinline__ int col_of(int j) const { return col_at(lt, j); }
    __device__ __forceinline__ bool is_dev(int j) const {
        int c = col_of(j);
        return c >= 1 && c < NCOL;
    }

    __device__ __forceinline__ void init(const typename Sys::Params& P) {
        prm = P;
        lt = (L == 1) ? 0 : (int)(threadIdx.x % L);
        s_lane = (L > 1 && lt == 0) ? 0.5 : 1.0;
        lg.init();
    }

    __device__ __forceinline__ void reset_logs() { lg.init(); }

    __device__ __forceinline__ void load(const double* y, const double* w, long long n_ic, long long ic,
                                         double psign) {
#pragma unroll
        for (int j = 0; j < CPL; j++) {
            const int c = col_of(j);
#pragma unroll
            for (int d = 0; d < ND; d++) {
                double qq = 0.0, pp = 0.0;
                if (c == 0) {
                    qq = y[(long long)d * n_ic + ic];
                    pp = psign * y[(long long)(ND + d) * n_ic + ic];
                } else if (c < NCOL) {
                    qq = w[((long long)(c - 1) * N + d) * n_ic + ic];
                    pp = w[((long long)(c - 1) * N + ND + d) * n_ic + ic];
                }
                q[j * ND + d] = qq;
                p[j * ND + d] = pp;
            }
        }
    }
    // x0 -> x0 + delta e_comp for the orbit (neighbouring initial conditions); comp in the
    // ordering of y.  psign is the momentum sign load() applied: the displacement is of the ORIGINAL IC.
    __device__ __forceinline__ void displace(int comp, double delta, double psign) {
        if (lt != 0) return;
#pragma unroll
        for (int d = 0; d < ND; d++) {
            if (comp == d) q[d] += delta;
            if (comp == ND + d) p[d] += psign * delta;
        }
    }
    __device__ __forceinline__ void store(double* y, double* w, long long n_ic, long long ic, bool bad) const {
#pragma unroll
        for (int j = 0; j < CPL; j++) {
            const int c = col_of(j);
#pragma unroll
            for (int d = 0; d < ND; d++) {
                double qq = bad ? nan("") : q[j * ND + d], pp = bad ? nan("") : p[j * ND + d];
                if (c == 0) {
                    y[(long long)d * n_ic + ic] = qq;
                    y[(long long)(ND + d) * n_ic + ic] = pp;
                } else if (c < NCOL) {
                    w[((long long)(c - 1) * N + d) * n_ic + ic] = qq;
                    w[((long long)(c - 1) * N + ND + d) * n_ic + ic] = pp;
                }
            }
        }
    }

    // carried rounding words of the orbit's compensated update (items 0..ND-1 of the orbit lane)
    // across a call boundary: carry[c][ic] in the layout of y
    __device__ __forceinline__ void load_carry(const double* cw, long long n_ic, long long ic, double (&qc)[ND],
                                               double (&pc)[ND]) const {
        if (lt == 0) {
#pragma unroll
            for (int d = 0; d < ND; d++) {
                qc[d] = cw[(long long)d * n_ic + ic];
                pc[d] = cw[(long long)(ND + d) * n_ic + ic];
            }
        }
    }
    __device__ __forceinline__ void store_carry(double* cw, long long n_ic, long long ic, const double (&qc)[ND],
                                                const double (&pc)[ND], bool bad) const {
        if (lt == 0) {
#pragma unroll
            for (int d = 0; d < ND; d++) {
                cw[(long long)d * n_ic + ic] = bad ? 0.0 : qc[d];
                cw[(long long)(ND + d) * n_ic + ic] = bad ? 0.0 : pc[d];
            }
        }
    }
    // On the other lanes of a multi-lane tile item 0 is a deviation column; the step code is the
    // same for every lane, so that column carries a rounding word too.  It is dropped at every
    // renormalisation (the vector is rescaled there anyway), so that no deviation word ever has
    // to cross a call boundary.
    __device__ __forceinline__ void scrub_carry(double (&qc)[ND], double (&pc)[ND]) const {
        if constexpr (L > 1) {
            if (lt != 0) {
#pragma unroll
                for (int d = 0; d < ND; d++) qc[d] = pc[d] = 0.0;
            }
        }
    }

    // force on all items at stage coordinates Q (Eq.(5) etc. + variational part).
    // L == 1: the orbit's force directly, one Hessian for the deviation columns.  L > 1: every column,
    // the orbit's included (s_lane = 1/2, Euler's relation), is G = -(V2'' + s V3''(Qo)) x; with one
    // column per lane the products of the lane's own x are formed while the orbit's coordinates Qo are
    // still in flight (Sys::pre / apply_pre): two or three dependent FMAs after the shuffle instead of four
    // levels (configs[0], 1024 ICs: 5.3 ms against 5.9 ms).
    // g: the factor the forces come out multiplied by (1, or h^2 in the adaptive kernels: dop8_core.cuh
    // dop8_stage_coords); where a Hessian is formed it absorbs g, so scaling costs nothing there.
    __device__ __forceinline__ void force(const double (&Q)[NI], double (&F)[NI], double g = 1.0) const {
        if constexpr (L == 1) {
            if constexpr (CPL > 1) {
                const typename Sys::Hess H = Sys::hess(prm, &Q[0], 1.0, g);
                Sys::force_hess(prm, H, &Q[0], g, &F[0]);
#pragma unroll
                for (int j = 1; j < CPL; j++) Sys::apply(H, &Q[j * ND], &F[j * ND]);
            } else {
                Sys::force(prm, &Q[0], &F[0]);
#pragma unroll
                for (int d = 0; d < ND; d++) F[d] *= g;
            }
        } else if constexpr (CPL == 1) {
            const typename Sys::Pre P = Sys::pre(prm, &Q[0], s_lane);
            double Qo[ND];
#pragma unroll
            for (int d = 0; d < ND; d++) Qo[d] = tile_bcast<L>(Q[d], 0);
            Sys::apply_pre(prm, P, Qo, &F[0]);
#pragma unroll
            for (int d = 0; d < ND; d++) F[d] *= g;
        } else {  // several columns per lane: a Hessian serves them (fewer instructions; measured faster)
            double Qo[ND];
#pragma unroll
            for (int d = 0; d < ND; d++) Qo[d] = tile_bcast<L>(Q[d], 0);
            const typename Sys::Hess H0 = Sys::hess(prm, Qo, s_lane, g);
            Sys::apply(H0, &Q[0], &F[0]);
            if constexpr (ALONE) {  // lane 0's other slots are idle: the same Hessian for every slot of a lane
#pragma unroll
                for (int j = 1; j < CPL; j++) Sys::apply(H0, &Q[j * ND], &F[j * ND]);
            } else {
                const typename Sys::Hess H1 = Sys::hess(prm, Qo, 1.0, g);
#pragma unroll
                for (int j = 1; j < CPL; j++) Sys::apply(H1, &Q[j * ND], &F[j * ND]);
            }
        }
    }
    // two independent force evaluations (dop8_stages PAIR)
    __device__ __forceinline__ void force2(const double (&Qa)[NI], double (&Fa)[NI], const double (&Qb)[NI],
                                           double (&Fb)[NI], double g = 1.0) const {
        force(Qa, Fa, g);
        force(Qb, Fb, g);
    }

    // value of component cc (0..N-1) of column `col` (compile-time), on every lane of the tile
    template <int COL>
    __device__ __forceinline__ double gather(int cc) const {
        constexpr int owner = owner_of(COL), j = slot_of(COL);
        const double v = (cc < ND) ? q[j * ND + cc] : p[j * ND + (cc - ND)];
        return tile_bcast<L>(v, owner);
    }

    // Renormalisation: w_v <- w_v/|w_v|, lg += ln|w_v|.  Lane-local.
    __device__ __forceinline__ void renorm(bool want_log, bool apply) {
#pragma unroll
        for (int j = 0; j < CPL; j++) {
            if (L == 1 && j == 0) continue;  // the orbit
            double sd[ND];  // per-coordinate q^2 + p^2, then a short sum: 2 + log2(ND) levels deep, not 2 ND
#pragma unroll
            for (int d = 0; d < ND; d++) sd[d] = fma(q[j * ND + d], q[j * ND + d], p[j * ND + d] * p[j * ND + d]);
            double s = sd[0];
#pragma unroll
            for (int d = 1; d < ND; d++) s += sd[d];
            const bool dev = is_dev(j) && apply;
            const double ri = fast_rsqrt(s);
            const double inv = dev ? ri : 1.0;
#pragma unroll
            for (int d = 0; d < ND; d++) {
                q[j * ND + d] *= inv;
                p[j * ND + d] *= inv;
            }
            if (want_log && dev) lg.mul(j, s * ri);
        }
    }

    // Modified Gram-Schmidt ("QR factorization"; BASELINE configs[3]):
    // for v = 1..K: r_vv = |w_v|, q_v = w_v/r_vv, lg_v += ln r_vv, then every later column
    // w_u -= (q_v . w_u) q_v  (right-looking order: the same operations on each column, in the
    // same order, as the textbook left-looking loop).  Warp-convergent; `apply` predicates.
    __device__ __forceinline__ void mgs(bool want_log, bool apply) {
        static_for<1, NCOL>([&](auto vc) {
            constexpr int v = decltype(vc)::value;
            constexpr int owner = owner_of(v), jv = slot_of(v);
            double wq[ND], wp[ND];
            double s = 0.0;
#pragma unroll
            for (int d = 0; d < ND; d++) {
                wq[d] = tile_bcast<L>(q[jv * ND + d], owner);
                wp[d] = tile_bcast<L>(p[jv * ND + d], owner);
            }
#pragma unroll
            for (int d = 0; d < ND; d++) s = fma(wq[d], wq[d], s);
#pragma unroll
            for (int d = 0; d < ND; d++) s = fma(wp[d], wp[d], s);
            const double inv = fast_rsqrt(s), r = s * inv;
#pragma unroll
            for (int d = 0; d < ND; d++) {
                wq[d] *= inv;
                wp[d] *= inv;
            }
            const bool mine = apply && (lt == owner);
            if (mine) {
#pragma unroll
                for (int d = 0; d < ND; d++) {
                    q[jv * ND + d] = wq[d];
                    p[jv * ND + d] = wp[d];
                }
                if (want_log) lg.mul(jv, r);
            }
#pragma unroll
            for (int j = 0; j < CPL; j++) {
                const int c = col_of(j);
                if ((L == 1) ? (j > v && apply) : (c > v && c < NCOL && apply)) {
                    double dot = 0.0;
#pragma unroll
                    for (int d = 0; d < ND; d++) dot = fma(wq[d], q[j * ND + d], dot);
#pragma unroll
                    for (int d = 0; d < ND; d++) dot = fma(wp[d], p[j * ND + d], dot);
#pragma unroll
                    for (int d = 0; d < ND; d++) {
                        q[j * ND + d] = fma(-dot, wq[d], q[j * ND + d]);
                        p[j * ND + d] = fma(-dot, wp[d], p[j * ND + d]);
                    }
                }
            }
        });
    }

    template <int MODE>
    __device__ __forceinline__ void do_renorm(bool want_log, bool apply) {
        if constexpr (MODE == MODE_NORM) renorm(want_log, apply);
        if constexpr (MODE == MODE_MGS) mgs(want_log, apply);
    }

    // SALI / GALI_k of the current unit vectors; same on all lanes
    template <int IND>
    __device__ __forceinline__ double indicator() const {
        if constexpr (IND == IND_SALI) {
            double sp = 0.0, sm = 0.0;
#pragma unroll
            for (int cc = 0; cc < N; cc++) {
                const double a = gather<1>(cc), b = gather<(K >= 2 ? 2 : 1)>(cc);
                const double u = a + b, d = a - b;
                sp = fma(u, u, sp);
                sm = fma(d, d, sm);
            }
            sp = sqrt(sp);
            sm = sqrt(sm);
            return sp < sm ? sp : sm;
        } else if constexpr (IND == IND_GALI) {
            double W[K][N];
            static_for<0, K>([&](auto vc) {
                constexpr int v = decltype(vc)::value;
#pragma unroll
                for (int cc = 0; cc < N; cc++) W[v][cc] = gather<v + 1>(cc);
            });
            return gali_thread<N, K>(W);
        } else {
            return 0.0;
        }
    }

    __device__ __forceinline__ bool finite_all() const {
        bool ok = true;
#pragma unroll
        for (int c = 0; c < NI; c++) ok = ok && isfinite(q[c]) && isfinite(p[c]);
        return !tile_any<L>(!ok);
    }

    __device__ __forceinline__ void on_mask(bool (&on)[NI]) const {
#pragma unroll
        for (int j = 0; j < CPL; j++)
#pragma unroll
            for (int d = 0; d < ND; d++) on[j * ND + d] = col_of(j) < NCOL;
    }

    // accumulated logs -> logacc (+=) and lambda (= sum / elapsed); each lane writes its own columns
    __device__ __forceinline__ void store_logs(const RunArgs& a, long long ic, bool bad, double elapsed) const {
        if constexpr (K > 0) {
#pragma unroll
            for (int j = 0; j < CPL; j++) {
                if (is_dev(j)) {
                    const long long o = (long long)(col_of(j) - 1) * a.n_ic + ic;
                    const double lv = lg.value(j);
                    if (a.logacc) a.logacc[o] = bad ? nan("") : a.logacc[o] + lv;
                    if (a.lambda) a.lambda[o] = (bad || elapsed == 0.0) ? nan("") : lv / fabs(elapsed);
                }
            }
        }
    }
};

// Starting step of the adaptive solver (item 6), any layout S
// LD: the state carries one more component M (M = 0, M' = |f|_2, scale = atol): run_kernel's LD runs
template <class S, bool LD = false>
__device__ __forceinline__ double initial_step(const S& s, double interval, double dir, double rtol, double atol) {
    constexpr int NI = S::NI, L = S::L;
    const double D = s.dcount() + (LD ? 1.0 : 0.0);
    if (interval == 0.0) return 0.0;
    bool on[NI];
    s.on_mask(on);
    double F0[NI], F1[NI], q1[NI], p1[NI];
    s.force(s.q, F0);
    double s0 = 0.0, s1 = 0.0;
#pragma unroll
    for (int c = 0; c < NI; c++) {
        const double iq = 1.0 / fma(fabs(s.q[c]), rtol, atol), ip = 1.0 / fma(fabs(s.p[c]), rtol, atol);
        if (on[c]) {
            s0 += (s.q[c] * iq) * (s.q[c] * iq) + (s.p[c] * ip) * (s.p[c] * ip);
            s1 += (s.p[c] * iq) * (s.p[c] * iq) + (F0[c] * ip) * (F0[c] * ip);
        }
    }
    double nf0 = 0.0;  // LD: |f(y)|_2 = |(p, F0)|_2
    if constexpr (LD) {
        double n2 = 0.0;
#pragma unroll
        for (int c = 0; c < NI; c++)
            if (on[c]) n2 = fma(s.p[c], s.p[c], fma(F0[c], F0[c], n2));
        nf0 = sqrt(tile_sum<L>(n2));
    }
    s0 = tile_sum<L>(s0);
    s1 = tile_sum<L>(s1);
    if constexpr (LD) s1 += (nf0 / atol) * (nf0 / atol);
    const double d0 = sqrt(s0 / D), d1 = sqrt(s1 / D);
    double ha = (d0 < 1e-5 || d1 < 1e-5) ? 1e-6 : 0.01 * d0 / d1;
    ha = fmin(ha, interval);
#pragma unroll
    for (int c = 0; c < NI; c++) {
        q1[c] = fma(ha * dir, s.p[c], s.q[c]);
        p1[c] = fma(ha * dir, F0[c], s.p[c]);
    }
    s.force(q1, F1);
    double s2 = 0.0;
#pragma unroll
    for (int c = 0; c < NI; c++) {
        const double iq = 1.0 / fma(fabs(s.q[c]), rtol, atol), ip = 1.0 / fma(fabs(s.p[c]), rtol, atol);
        const double dq = (p1[c] - s.p[c]) * iq, dp = (F1[c] - F0[c]) * ip;
        if (on[c]) s2 += dq * dq + dp * dp;
    }
    s2 = tile_sum<L>(s2);
    if constexpr (LD) {
        double n2 = 0.0;
#pragma unroll
        for (int c = 0; c < NI; c++)
            if (on[c]) n2 = fma(p1[c], p1[c], fma(F1[c], F1[c], n2));
        const double dn = (sqrt(tile_sum<L>(n2)) - nf0) / atol;
        s2 += dn * dn;
    }
    const double d2 = sqrt(s2 / D) / ha;
    double hb;
    if (d1 <= 1e-15 && d2 <= 1e-15) hb = fmax(1e-6, 1e-3 * ha);
    else hb = root8(0.01 / fmax(d1, d2));
    return fmin(fmin(100.0 * ha, hb), interval);
}

// functors handed to dop8_stages (plain structs: generic lambdas with array-reference
// parameters of dependent extent crash cudafe++ 12.9)
// SCALED: the forces come out multiplied by g (= h^2 of the attempt; adaptive kernels)
template <class C, bool SCALED = false>
struct ForceFn {
    const C& s;
    double g;
    __device__ __forceinline__ void operator()(const double (&Q)[C::NI], double (&F)[C::NI]) const {
        if constexpr (SCALED) s.force(Q, F, g);
        else s.force(Q, F);
    }
    __device__ __forceinline__ void pair(const double (&Qa)[C::NI], double (&Fa)[C::NI], const double (&Qb)[C::NI],
                                         double (&Fb)[C::NI]) const {
        if constexpr (SCALED) s.force2(Qa, Fa, Qb, Fb, g);
        else s.force2(Qa, Fa, Qb, Fb);
    }
};
struct NoHook {
    template <class I, class FF>
    __device__ __forceinline__ void operator()(I, const FF&) const {}
};
// LD quadrature: after stage i, M += |h| b_i |(P_i, F_i)|_2
template <class C>
struct LdHook {
    const Tab& tab;
    const C& s;
    double& M;
    template <int i>
    __device__ __forceinline__ void operator()(Int<i>, const double (&F)[12][C::NI]) const {
        if constexpr (coef::B[i] != 0.0) {
            double n2 = 0.0;
#pragma unroll
            for (int c = 0; c < C::NI; c++) {
                double P = s.p[c];
                static_for<0, i>([&](auto jc) {
                    constexpr int j = decltype(jc)::value;
                    if constexpr (coef::A[i][j] != 0.0) P = fma(tab.ap[i][j], F[j][c], P);
                });
                n2 = fma(P, P, fma(F[i][c], F[i][c], n2));
            }
            M = fma(tab.bl[i], fast_sqrt(tile_sum<C::L>(n2)), M);
        }
    }
};

// The same norms inside an ADAPTIVE attempt (scaled forces G = h^2 F, raw table): after stage i with b_i != 0
// keep |k_i|_2 = |(P_i, F_i)|_2, P_i = p + (1/h) sum_j a_ij G_j, F_i = G_i / h^2; the attempt then forms
// M+ = M + |h| sum b_i |k_i| and the embedded errors of M from the same eight numbers (b, E5 and E3 share
// their support).
template <class C>
struct LdNormHook {
    const Tab& tab;
    const C& s;
    double hinv, hinv2;
    double (&nrm)[12];
    template <int i>
    __device__ __forceinline__ void operator()(Int<i>, const double (&F)[12][C::NI]) const {
        if constexpr (coef::B[i] != 0.0) {
            double n2 = 0.0;
#pragma unroll
            for (int c = 0; c < C::NI; c++) {
                double P = s.p[c];
                if constexpr (i > 0) {
                    double sum = 0.0;
                    bool first = true;
                    static_for<0, i>([&](auto jc) {
                        constexpr int j = decltype(jc)::value;
                        if constexpr (coef::A[i][j] != 0.0) {
                            sum = first ? tab.ap[i][j] * F[j][c] : fma(tab.ap[i][j], F[j][c], sum);
                            first = false;
                        }
                    });
                    P = fma(hinv, sum, P);
                }
                const double f = F[i][c] * hinv2;
                n2 = fma(P, P, fma(f, f, n2));
            }
            nrm[i] = fast_sqrt(tile_sum<C::L>(n2));
        }
    }
};

// scratch word of a fixed-step trajectory's death step: its n_accepted entry, else its t_final entry (both
// are 8 bytes and are rewritten with their real content at the end of the run), else none -- then nobody
// asked where the trajectory died
__device__ __forceinline__ unsigned long long* death_word(const RunArgs& a, long long ic) {
    if (a.n_acc) return reinterpret_cast<unsigned long long*>(a.n_acc + ic);
    if (a.t_final) return reinterpret_cast<unsigned long long*>(a.t_final + ic);
    return nullptr;
}
// non-finite never heals, so the minimum over all notes of a trajectory is the first one
template <int NI>
__device__ __forceinline__ void note_death(const RunArgs& a, const double (&q)[NI], const double (&p)[NI], bool valid,
                                           long long ic, long long st) {
    if (lane_nonfinite<NI>(q, p)) {  // off the hot path
        unsigned long long* dw = death_word(a, ic);
        if (valid && dw) atomicMin(dw, (unsigned long long)st);
    }
}
template <int L>
__device__ __forceinline__ void tile_sync() {
    if constexpr (L > 32) __syncthreads();
    else if constexpr (L > 1) __syncwarp();
}

// ---- the run kernel: fixed or adaptive, with renormalisation / indicator ----------------------
// S = the per-lane state class of a layout (Col<Sys,K,L> here, Chain<NP,K> in chain_kernels.cuh)
// PAIR: evaluate the stages two at a time (dop8_core.cuh dop8_stages); off only where the extra live
// stage vector does not fit the register file.
// LD (adaptive only, K = 0): the arc-length Lagrangian descriptor rides along as one more component of the state
// (R21): tasks are (direction, IC) pairs, nothing is written back but M and the report.
template <class C, int MODE, int IND, bool ADAPT, int TPB, int MINB, bool PAIR = true, bool LD = false>
__global__ void __launch_bounds__(TPB, MINB)
run_kernel(const __grid_constant__ Tab tab, const typename C::Params prm, const RunArgs a) {
    constexpr int NI = C::NI, L = C::L, K = C::K;
    static_assert(!LD || (ADAPT && K == 0 && MODE == MODE_NONE && IND == IND_NONE), "LD rides on the plain adaptive run");
    const long long gt = (long long)blockIdx.x * TPB + threadIdx.x;
    const long long traj = gt / L;
    const bool want_log = (a.logacc != nullptr) || (a.lambda != nullptr);

    C s;
    s.init(prm);
    const ForceFn<C> force{s, 1.0};
    const NoHook nohook{};

    long long n_acc = 0, n_rej = 0;
    int status = ST_OK;
    double t = a.t0;
    constexpr int NC = C::NCOMP > 0 ? C::NCOMP : 1;
    double qc[NC], pc[NC], qcn[NC], pcn[NC];  // carried rounding errors of the orbit update
#pragma unroll
    for (int c = 0; c < NC; c++) qc[c] = pc[c] = 0.0;
    // "cold" layouts keep the carried words in shared memory between steps ([word][thread]): they are
    // read and written once per step, and the step itself needs every register
    constexpr bool COLD = C::COLD && !ADAPT;
    __shared__ double cold_carry[COLD ? 2 * NC * kMaxTpb : 1];
    static_assert(!COLD || TPB <= kMaxTpb, "TPB exceeds the cold-state arrays");

    if constexpr (!ADAPT) {
        // ---- fixed step: one trajectory per tile, every tile runs the same number of steps -------
        const bool valid = traj < a.n_ic;
        const long long ic = valid ? traj : a.n_ic - 1;  // padding tiles shadow the last trajectory
        s.load(a.y, a.w, a.n_ic, ic, 1.0);
        if (a.resume) {
            if (a.carry) s.load_carry(a.carry, a.n_ic, ic, qc, pc);
        } else {
            s.template do_renorm<MODE>(false, true);  // on entry: no log accumulated
        }
        long long slot = 0;
        int cd = a.m, sd = a.sample_every;
        if constexpr (COLD) {
#pragma unroll
            for (int c = 0; c < NC; c++) {
                cold_carry[c * kMaxTpb + threadIdx.x] = qc[c];
                cold_carry[(NC + c) * kMaxTpb + threadIdx.x] = pc[c];
            }
        }
        // The step after which the state was first not finite (the oracle tests after every step and stops
        // there) is latched in GLOBAL memory, in the trajectory's own report word (death_word): the step
        // kernels have no register to spare for it, and only lanes that are already dead ever touch it.
        for (long long st = 1; st <= a.n_steps; ++st) {
            // the oracle's test after a step, made on entry to the next one: after every kDeathCheckEvery-th
            // step here, and after the last one below
            if (((st - 1) & (kDeathCheckEvery - 1)) == 0 && st > 1) note_death<NI>(a, s.q, s.p, valid, ic, st - 1);
            double F[12][NI];
            dop8_stages<NI, PAIR>(tab, s.q, s.p, F, force, nohook);
            double qn[NI], pn[NI];
            if constexpr (COLD) {
#pragma unroll
                for (int c = 0; c < NC; c++) {
                    qc[c] = cold_carry[c * kMaxTpb + threadIdx.x];
                    pc[c] = cold_carry[(NC + c) * kMaxTpb + threadIdx.x];
                }
            }
            double spo[NI];  // (adaptive kernels only)
            dop8_solution<NI, C::NCOMP, true>(tab, 0.0, s.q, s.p, s.p, F, qn, pn, qc, pc, qcn, pcn, spo);
#pragma unroll
            for (int c = 0; c < NI; c++) {
                s.q[c] = qn[c];
                s.p[c] = pn[c];
            }
#pragma unroll
            for (int c = 0; c < NC; c++) {
                if constexpr (COLD) {
                    cold_carry[c * kMaxTpb + threadIdx.x] = qcn[c];
                    cold_carry[(NC + c) * kMaxTpb + threadIdx.x] = pcn[c];
                } else {
                    qc[c] = qcn[c];
                    pc[c] = pcn[c];
                }
            }
            if constexpr (MODE != MODE_NONE) {
                if (--cd == 0 || st == a.n_steps) {
                    cd = a.m;
                    s.template do_renorm<MODE>(want_log, true);
                    if constexpr (!COLD) s.scrub_carry(qc, pc);  // (cold layouts carry orbit words only)
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
        if (a.n_steps > 0) note_death<NI>(a, s.q, s.p, valid, ic, a.n_steps);
        n_acc = a.n_steps;
        t = a.t0 + (double)a.n_steps * a.h;
        bool bad = !s.finite_all();
        double ind = 0.0;
        if constexpr (IND != IND_NONE) ind = s.template indicator<IND>();
        if (bad) status = ST_NONFINITE;
        tile_sync<L>();  // the dead lanes' atomics are ordered before the orbit lane reads the word back
        if (!valid) return;
        s.store(a.y, a.w, a.n_ic, ic, bad);
        if constexpr (COLD) {
#pragma unroll
            for (int c = 0; c < NC; c++) {
                qc[c] = cold_carry[c * kMaxTpb + threadIdx.x];
                pc[c] = cold_carry[(NC + c) * kMaxTpb + threadIdx.x];
            }
        }
        if (a.carry) s.store_carry(a.carry, a.n_ic, ic, qc, pc, bad);
        if constexpr (K > 0) s.store_logs(a, ic, bad, t - a.t0);
        if (s.lt == 0) {
            if constexpr (IND != IND_NONE) {
                if (a.series) {
                    a.series[(a.n_samples - 1) * a.n_ic + ic] = bad ? nan("") : ind;
                    if (bad)
                        for (long long r = slot; r < a.n_samples - 1; r++) a.series[r * a.n_ic + ic] = nan("");
                }
            }
            if (unsigned long long* dw = death_word(a, ic)) {
                const unsigned long long died = *(volatile unsigned long long*)dw;
                if (died != ~0ULL) {  // a dead trajectory reports the step at which it died (where the oracle stops)
                    n_acc = (long long)died;
                    t = a.t0 + (double)n_acc * a.h;
                    status = ST_NONFINITE;
                }
            }
            if (a.n_acc) a.n_acc[ic] = n_acc;
            if (a.n_rej) a.n_rej[ic] = n_rej;
            if (a.status) a.status[ic] = status;
            if (a.t_final) a.t_final[ic] = t;
        }
    } else {
        // ---- adaptive step: every trajectory owns t, h, counters, status.
        // A tile keeps taking trajectories until none is left: with a.queue set, from a global work
        // queue (lane refill: a tile whose trajectory has ended fetches the next one instead of idling
        // until the slowest lane of its warp and block ends; the grid is then one resident wave);
        // without it, exactly one trajectory per tile.  The warp-wide loop and every section that
        // shuffles stay convergent; per-tile decisions are predicates.
        const double dir = (a.t_end >= a.t0) ? 1.0 : -1.0;
        const bool fwd = dir > 0.0;
        const double interval = fabs(a.t_end - a.t0);
        bool on[NI];
        s.on_mask(on);
        double h_abs = 0.0, min_step = 0.0;
        long long attempts = 0, ic = 0;
        bool rejected = false, need = true, fin = false, done = false, first_fetch = true;
        bool more = false;  // t has not reached t_end yet
        int cd = a.m;
        const long long n_items = LD ? a.n_ic * a.n_dirs : a.n_ic;  // LD: tasks ordered [direction][ic]
        double M = 0.0;                                              // LD: the descriptor of this task
        long long out_slot = 0;                                      // LD: row (0 fwd, 1 bwd) * n_ic + ic
        // One vote per iteration: the block below (write out the trajectories that ended in the previous
        // attempt, fetch new ones, leave when nothing is left) is entered only when some tile asks for it.
        while (true) {
            if (group_any<L>(fin || need)) {
                if (group_any<L>(fin)) {
                    bool bad = !s.finite_all();
                    bad = tile_any<L>(status != ST_OK) || bad;
                    double ind = 0.0;
                    if constexpr (IND != IND_NONE) ind = s.template indicator<IND>();
                    if (fin) {
                        const int st_out = (bad && status == ST_OK) ? (int)ST_NONFINITE : status;
                        if constexpr (LD) {
                            bad = bad || !isfinite(M);
                            if (s.lt == 0) {
                                double* out = out_slot < a.n_ic ? a.ld_fwd : a.ld_bwd;
                                out[ic] = bad ? nan("") : M;
                                if (a.n_acc) a.n_acc[out_slot] = n_acc;
                                if (a.n_rej) a.n_rej[out_slot] = n_rej;
                                if (a.status) a.status[out_slot] = (bad && st_out == ST_OK) ? (int)ST_NONFINITE : st_out;
                                if (a.t_final) a.t_final[out_slot] = t;
                            }
                        } else {
                            s.store(a.y, a.w, a.n_ic, ic, bad);
                            if constexpr (K > 0) s.store_logs(a, ic, bad, t - a.t0);
                            if (s.lt == 0) {
                                if constexpr (IND != IND_NONE) {
                                    if (a.series) a.series[ic] = bad ? nan("") : ind;  // adaptive: n_samples = 1
                                }
                                if (a.n_acc) a.n_acc[ic] = n_acc;
                                if (a.n_rej) a.n_rej[ic] = n_rej;
                                if (a.status) a.status[ic] = st_out;
                                if (a.t_final) a.t_final[ic] = t;
                            }
                        }
                        need = true;
                        fin = false;
                    }
                }
                long long nxt = n_items;  // "nothing left"
                if (a.queue != nullptr) {
                    if (need && s.lt == 0) nxt = (long long)atomicAdd(a.queue, 1ULL);
                    nxt = tile_bcast_ll<L>(nxt, 0);
                } else if (first_fetch) {
                    nxt = traj;
                }
                first_fetch = false;
                const bool got = need && nxt < n_items;
                if (need && !got) done = true;
                if (got) {
                    if constexpr (LD) {  // backward = forward of the momentum-reversed IC (ld_kernel)
                        const int dsel = a.dir_first + (int)(nxt / a.n_ic);
                        ic = nxt % a.n_ic;
                        out_slot = (long long)dsel * a.n_ic + ic;
                        s.load(a.y0, nullptr, a.n_ic, ic, dsel == 0 ? 1.0 : -1.0);
                        M = 0.0;
                    } else {
                        ic = nxt;
                        s.load(a.y, a.w, a.n_ic, ic, 1.0);
                    }
                    s.reset_logs();
                    t = a.t0;
                    more = interval > 0.0;
                    n_acc = n_rej = attempts = 0;
                    status = ST_OK;
                    rejected = false;
                    cd = a.m;
#pragma unroll
                    for (int c = 0; c < NC; c++) qc[c] = pc[c] = 0.0;
                }
                s.template do_renorm<MODE>(false, got && !a.resume);  // on entry: no log accumulated
                const double h_init = a.h0 > 0.0 ? a.h0 : initial_step<C, LD>(s, interval, dir, a.rtol, a.atol);
                if (got) h_abs = h_init;
                need = false;
                if (!group_any<L>(!done)) break;
            }

            // ---- one attempt; everything below is selects, no branch (one basic block for the scheduler) ----
            bool active = !done && status == ST_OK && more;
            {
                const double ms = ten_ulp(t, dir);  // 10 |nextafter(t, dir inf) - t|
                min_step = rejected ? min_step : ms;
                h_abs = rejected ? h_abs : fmax(h_abs, ms);
            }
            const bool under = active && h_abs < min_step;
            status = under ? (int)ST_UNDERFLOW : status;
            active = active && !under;
            const bool maxed = active && a.max_steps > 0 && attempts >= a.max_steps;
            status = maxed ? (int)ST_MAXSTEPS : status;
            active = active && !maxed;
            attempts += active ? 1 : 0;
            double t_new = t + h_abs * dir;
            if (fwd ? (t_new > a.t_end) : (t_new < a.t_end)) t_new = a.t_end;  // land exactly on t_end
            const double h = t_new - t;
            const double h_try = fabs(h);

            // scaled forces G_l = h^2 F_l and u = h p (dop8_core.cuh dop8_stage_coords): no multiplication by
            // the trajectory's own h inside the stages
            const ForceFn<C, true> force_h2{s, h * h};
            double u[NI];
#pragma unroll
            for (int c = 0; c < NI; c++) u[c] = h * s.p[c];
            double F[12][NI];
            double hinv, nrm[LD ? 12 : 1];
            if constexpr (LD) {
                hinv = fwd ? fast_rcp(h_try) : -fast_rcp(h_try);
                const LdNormHook<C> ldhook{tab, s, hinv, hinv * hinv, nrm};
                dop8_stages<NI, PAIR>(tab, s.q, u, F, force_h2, ldhook);
            } else {
                dop8_stages<NI, PAIR>(tab, s.q, u, F, force_h2, nohook);
                hinv = fwd ? fast_rcp(h_try) : -fast_rcp(h_try);  // (h = 0: inf; nothing is committed)
            }
            double qn[NI], pn[NI];
            double spo[NI];
            dop8_solution<NI, C::NCOMP, false>(tab, hinv, s.q, s.p, u, F, qn, pn, qc, pc, qcn, pcn, spo);
            double S5, S3;
            dop8_error_sums<NI>(tab, hinv, s.q, s.p, qn, pn, F, spo, a.rtol, a.atol, on, S5, S3);
            {
                double S[2] = {S5, S3};
                tile_sum_vec<L, 2>(S);
                S5 = S[0];
                S3 = S[1];
            }
            // err = |h| S5 / sqrt(D (S5 + 0.01 S3)) against 1, and the step-size factor 0.9 err^(-1/8), without
            // forming err (dop8_core.cuh "step-size controller"): accept <=> num^2 < den
            double Mn = 0.0;
            if constexpr (LD) {  // M+ and its embedded errors (divided by h, like the sums above)
                double sb = 0.0, s5 = 0.0, s3 = 0.0;
                static_for<0, 12>([&](auto ic2) {
                    constexpr int i = decltype(ic2)::value;
                    if constexpr (coef::B[i] != 0.0) {
                        sb = fma(tab.bl[i], nrm[i], sb);
                        s5 = fma(tab.e5p[i], nrm[i], s5);
                        s3 = fma(tab.e3p[i], nrm[i], s3);
                    }
                });
                Mn = fma(h_try, sb, M);
                const double isc = fast_rcp(fma(a.rtol, fmax(fabs(M), fabs(Mn)), a.atol));
                s5 *= isc;
                s3 *= isc;
                S5 = fma(s5, s5, S5);
                S3 = fma(s3, s3, S3);
            }
            const StepDecision dec = step_decision(h_try, S5, S3, s.dcount() + (LD ? 1.0 : 0.0), rejected);
            const bool acc = active && dec.acc, rej = active && dec.rej;
            if (active && !acc && !rej) status = ST_NONFINITE;  // NaN: inf or NaN in y+ (fast_rcp(inf) is NaN)
            if (acc || rej) h_abs = h_try * dec.factor;
            rejected = rej ? true : (acc ? false : rejected);
            n_acc += acc ? 1 : 0;
            n_rej += rej ? 1 : 0;
            t = acc ? t_new : t;
            if constexpr (LD) M = acc ? Mn : M;
            more = fwd ? (t < a.t_end) : (t > a.t_end);
#pragma unroll
            for (int c = 0; c < NI; c++) {
                s.q[c] = acc ? qn[c] : s.q[c];
                s.p[c] = acc ? pn[c] : s.p[c];
            }
#pragma unroll
            for (int c = 0; c < NC; c++) {
                qc[c] = acc ? qcn[c] : qc[c];
                pc[c] = acc ? pcn[c] : pc[c];
            }
            if constexpr (MODE != MODE_NONE) {
                bool ren = false;
                if (acc && (--cd == 0 || !more)) {
                    cd = a.m;
                    ren = true;
                }
                // thread layout: renormalising is lane-local and cheap, so it runs every attempt under the
                // predicate (no branch between it and the controller); tiles shuffle: only when some tile wants it
                constexpr bool ALWAYS = (L == 1) && (MODE == MODE_NORM);
                if (ALWAYS || group_any<L>(ren)) {
                    s.template do_renorm<MODE>(want_log, ren);
                    if (ren) s.scrub_carry(qc, pc);
                }
            }
            // trajectories that ended in this attempt: written out at the top of the next iteration
            fin = !done && !(status == ST_OK && more);
        }
    }
}

// ---- Lagrangian descriptor kernel (BASELINE configs[1]) ------------
// One thread per (direction, IC).  The backward pass is the forward pass of the momentum-
// reversed initial condition: H is even in p, so stepping (q, p) with -h and stepping (q, -p)
// with +h give mirror-image states bit for bit and the same |f|.
// M += |h| sum_i b_i |k_i|_2 with k_i = (P_i, F_i) the stage derivative; P_i is formed only at
// the 8 stages with b_i != 0.
// C = a layout with K = 0 (Col<Sys,0,1>: one thread per (direction, IC); Chain<N,0>: one tile).
template <class C, int TPB, int MINB>
__global__ void __launch_bounds__(TPB, MINB)
ld_kernel(const __grid_constant__ Tab tab, const typename C::Params prm, const RunArgs a, int dir_first,
          int n_dirs) {
    constexpr int NI = C::NI, L = C::L;
    const long long gt = (long long)blockIdx.x * TPB + threadIdx.x;
    const long long per_dir = a.n_ic * a.n_members;  // tasks are ordered [direction][member][ic]
    const long long task = gt / L, n_task = per_dir * n_dirs;
    const bool valid = task < n_task;
    if (L == 1 && !valid) return;
    const long long tk = valid ? task : n_task - 1;  // padding tiles shadow the last task (shuffles stay convergent)
    const int dsel = dir_first + (int)(tk / per_dir);  // 0 forward, 1 backward
    const long long slot = tk % per_dir;                // = member * n_ic + ic: the output index
    const int member = (int)(slot / a.n_ic);
    const long long ic = slot % a.n_ic;
    const double psign = dsel == 0 ? 1.0 : -1.0;
    C s;
    s.init(prm);
    s.load(a.y0, nullptr, a.n_ic, ic, psign);
    if (member > 0) s.displace((member - 1) >> 1, ((member - 1) & 1) ? -a.sigma : a.sigma, psign);
    double M = 0.0;
    const ForceFn<C> force{s, 1.0};
    LdHook<C> hook{tab, s, M};
    for (long long st = 0; st < a.n_steps; ++st) {
        double F[12][NI];
        dop8_stages<NI, false>(tab, s.q, s.p, F, force, hook);
        double qn[NI], pn[NI];
        double z[1] = {0.0}, zn[1];
        double spo[NI];
        dop8_solution<NI, 0, true>(tab, 0.0, s.q, s.p, s.p, F, qn, pn, z, z, zn, zn, spo);
#pragma unroll
        for (int c = 0; c < NI; c++) {
            s.q[c] = qn[c];
            s.p[c] = pn[c];
        }
    }
    const bool ok = s.finite_all();
    double* out = dsel == 0 ? a.ld_fwd : a.ld_bwd;
    if (valid && s.lt == 0) out[slot] = ok ? M : nan("");
}

}  // namespace chs
