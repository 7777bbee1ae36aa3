// chain_kernels.cuh -- "chain layout" for the FPUT chain (CUDA path, sm_100a).
//
// PAPER.md:98-111 Eq.(6)-(8): N particles, fixed ends, nearest-neighbour springs.  A trajectory
// is owned by a tile of L = N lanes (N = 2, 4, 8, 16, 32; one full warp per trajectory at
// N = 32), lane i <-> particle i+1.  A lane holds, for its particle, the orbit coordinate and
// the K deviation-vector coordinates: 1 + K (q, p) pairs and their stage forces, all in
// registers.  Neighbour coupling goes through warp shuffles: per column one shuffle up (the left
// neighbour's stage coordinate) and one shuffle down (the right spring's force, computed by the
// right neighbour), so every spring is evaluated once.  Norms, dot products, Gram-Schmidt and
// the Jacobi rotations of GALI_k's SVD are butterfly shuffle reductions over the tile
// (BASELINE.json north_star, configs[4]).
#pragma once
#include "col_kernels.cuh"

namespace chs {

template <int NP, int K_>
struct Chain {
    static constexpr int K = K_, L = NP;
    static constexpr int NCOL = 1 + K;
    static constexpr int NI = NCOL;
    static constexpr int N = 2 * NP;
    static constexpr int D = N * NCOL;
    static constexpr int NCOMP = 1;  // item 0: the orbit coordinate -- compensated update
    using Params = FputParams;

    Params prm;
    int lt;
    double q[NI], p[NI];
    LogAcc lg[NCOL];  // deferred-log accumulators, lg[v], v >= 1: identical on all lanes of the tile

    __device__ __forceinline__ void init(const Params& P) {
        prm = P;
        lt = (int)(threadIdx.x % L);
#pragma unroll
        for (int j = 0; j < NCOL; j++) logacc_init(lg[j]);
    }
    __device__ __forceinline__ void reset_logs() {
#pragma unroll
        for (int j = 0; j < NCOL; j++) logacc_init(lg[j]);
    }
    __device__ __forceinline__ void load(const double* y, const double* w, long long n_ic, long long ic,
                                         double psign) {
        q[0] = y[(long long)lt * n_ic + ic];
        p[0] = psign * y[(long long)(NP + lt) * n_ic + ic];
#pragma unroll
        for (int v = 1; v < NCOL; v++) {
            q[v] = w[((long long)(v - 1) * N + lt) * n_ic + ic];
            p[v] = w[((long long)(v - 1) * N + NP + lt) * n_ic + ic];
        }
    }
    __device__ __forceinline__ void store(double* y, double* w, long long n_ic, long long ic, bool bad) const {
        y[(long long)lt * n_ic + ic] = bad ? nan("") : q[0];
        y[(long long)(NP + lt) * n_ic + ic] = bad ? nan("") : p[0];
#pragma unroll
        for (int v = 1; v < NCOL; v++) {
            w[((long long)(v - 1) * N + lt) * n_ic + ic] = bad ? nan("") : q[v];
            w[((long long)(v - 1) * N + NP + lt) * n_ic + ic] = bad ? nan("") : p[v];
        }
    }
    __device__ __forceinline__ void store_logs(const RunArgs& a, long long ic, bool bad, double elapsed) const {
        if (lt != 0) return;
#pragma unroll
        for (int v = 1; v < NCOL; v++) {
            const long long o = (long long)(v - 1) * a.n_ic + ic;
            const double lv = logacc_value(lg[v]);
            if (a.logacc) a.logacc[o] = bad ? nan("") : a.logacc[o] + lv;
            if (a.lambda) a.lambda[o] = (bad || elapsed == 0.0) ? nan("") : lv / fabs(elapsed);
        }
    }
    // carried rounding word of this particle's orbit coordinate across a call boundary
    __device__ __forceinline__ void load_carry(const double* cw, long long n_ic, long long ic, double (&qc)[1],
                                               double (&pc)[1]) const {
        qc[0] = cw[(long long)lt * n_ic + ic];
        pc[0] = cw[(long long)(NP + lt) * n_ic + ic];
    }
    __device__ __forceinline__ void store_carry(double* cw, long long n_ic, long long ic, const double (&qc)[1],
                                                const double (&pc)[1], bool bad) const {
        cw[(long long)lt * n_ic + ic] = bad ? 0.0 : qc[0];
        cw[(long long)(NP + lt) * n_ic + ic] = bad ? 0.0 : pc[0];
    }
    __device__ __forceinline__ void scrub_carry(double (&)[1], double (&)[1]) const {}
    __device__ __forceinline__ void on_mask(bool (&on)[NI]) const {
#pragma unroll
        for (int c = 0; c < NI; c++) on[c] = true;
    }

    // Eq.(7) with Eq.(8): p_i' = phi(Dq_{i+1}) - phi(Dq_i), Dq_i = q_i - q_{i-1}; variational:
    // dp_i' = g(Dq_{i+1}) dDq_{i+1} - g(Dq_i) dDq_i.  Lane i evaluates its LEFT spring; the
    // right spring's value comes from lane i+1; the last lane also evaluates the wall spring.
    __device__ __forceinline__ void force(const double (&Q)[NI], double (&F)[NI]) const {
        const bool first = (lt == 0), last = (lt == L - 1);
        double qL = __shfl_up_sync(0xffffffffu, Q[0], 1, L);
        if (first) qL = 0.0;
        const double d = Q[0] - qL;
        const double phi = fput_phi(prm, d);
        const double g = fput_g(prm, d);
        const double dW = -Q[0];  // wall spring of the last particle: q_{N+1} - q_N
        double phiR = __shfl_down_sync(0xffffffffu, phi, 1, L);
        double gW = 0.0;
        if (last) {
            phiR = fput_phi(prm, dW);
            gW = fput_g(prm, dW);
        }
        F[0] = phiR - phi;
#pragma unroll
        for (int v = 1; v < NCOL; v++) {
            double xL = __shfl_up_sync(0xffffffffu, Q[v], 1, L);
            if (first) xL = 0.0;
            const double T = g * (Q[v] - xL);
            double TR = __shfl_down_sync(0xffffffffu, T, 1, L);
            if (last) TR = gW * (-Q[v]);
            F[v] = TR - T;
        }
    }

    __device__ __forceinline__ double dot(int u, int v) const {
        return tile_sum<L>(fma(q[u], q[v], p[u] * p[v]));
    }

    // w_v <- w_v/|w_v|, lg_v += ln|w_v|
    __device__ __forceinline__ void renorm(bool want_log, bool apply) {
#pragma unroll
        for (int v = 1; v < NCOL; v++) {
            const double s = dot(v, v), ri = fast_rsqrt(s);
            const double inv = apply ? ri : 1.0;
            q[v] *= inv;
            p[v] *= inv;
            if (want_log && apply) logacc_mul(lg[v], s * ri);
        }
    }
    // modified Gram-Schmidt, right-looking order (see col_kernels.cuh)
    __device__ __forceinline__ void mgs(bool want_log, bool apply) {
#pragma unroll
        for (int v = 1; v < NCOL; v++) {
            const double s = dot(v, v), ri = fast_rsqrt(s);
            const double inv = apply ? ri : 1.0;
            q[v] *= inv;
            p[v] *= inv;
            if (want_log && apply) logacc_mul(lg[v], s * ri);
#pragma unroll
            for (int u = v + 1; u < NCOL; u++) {
                double dt = dot(v, u);
                if (!apply) dt = 0.0;
                q[u] = fma(-dt, q[v], q[u]);
                p[u] = fma(-dt, p[v], p[u]);
            }
        }
    }
    template <int MODE>
    __device__ __forceinline__ void do_renorm(bool want_log, bool apply) {
        if constexpr (MODE == MODE_NORM) renorm(want_log, apply);
        if constexpr (MODE == MODE_MGS) mgs(want_log, apply);
    }

    // SALI and GALI_k (product of singular values; one-sided Jacobi,
    // the three inner products of each column pair reduced over the tile by shuffles; every lane
    // of a tile sees bit-identical sums, so the rotation decisions are tile-uniform; the sweep
    // loop is made warp-uniform with a vote).
    template <int IND>
    __device__ __forceinline__ double indicator() const {
        if constexpr (IND == IND_SALI) {
            const double uq = q[1] + q[K >= 2 ? 2 : 1], up = p[1] + p[K >= 2 ? 2 : 1];
            const double dq = q[1] - q[K >= 2 ? 2 : 1], dp = p[1] - p[K >= 2 ? 2 : 1];
            const double sp = sqrt(tile_sum<L>(fma(uq, uq, up * up)));
            const double sm = sqrt(tile_sum<L>(fma(dq, dq, dp * dp)));
            return sp < sm ? sp : sm;
        } else if constexpr (IND == IND_GALI) {
            double Wq[K], Wp[K];
#pragma unroll
            for (int v = 0; v < K; v++) {
                Wq[v] = q[v + 1];
                Wp[v] = p[v + 1];
            }
            const double eps = 8.9e-16;
            for (int sweep = 0; sweep < 30; sweep++) {
                bool rotated = false;
#pragma unroll
                for (int a = 0; a < K - 1; a++)
#pragma unroll
                    for (int b = a + 1; b < K; b++) {
                        const double app = tile_sum<L>(fma(Wq[a], Wq[a], Wp[a] * Wp[a]));
                        const double aqq = tile_sum<L>(fma(Wq[b], Wq[b], Wp[b] * Wp[b]));
                        const double apq = tile_sum<L>(fma(Wq[a], Wq[b], Wp[a] * Wp[b]));
                        const bool rot = fabs(apq) > eps * sqrt(app * aqq);
                        rotated = rotated || rot;
                        const double zeta = (aqq - app) / (2.0 * apq);
                        const double t = copysign(1.0, zeta) / (fabs(zeta) + sqrt(fma(zeta, zeta, 1.0)));
                        const double cs = rot ? rsqrt(fma(t, t, 1.0)) : 1.0, sn = rot ? cs * t : 0.0;
                        const double xq = Wq[a], yq = Wq[b], xp = Wp[a], yp = Wp[b];
                        Wq[a] = cs * xq - sn * yq;
                        Wq[b] = fma(sn, xq, cs * yq);
                        Wp[a] = cs * xp - sn * yp;
                        Wp[b] = fma(sn, xp, cs * yp);
                    }
                if (!__any_sync(0xffffffffu, rotated)) break;
            }
            double gl = 1.0;
#pragma unroll
            for (int v = 0; v < K; v++) gl *= sqrt(tile_sum<L>(fma(Wq[v], Wq[v], Wp[v] * Wp[v])));
            return gl;
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
};

}  // namespace chs
