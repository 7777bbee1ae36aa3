// chain_kernels.cuh -- "chain layout" for the FPUT chain (CUDA path, sm_100a).
//
// PAPER.md:98-111 Eq.(6)-(8): N particles, fixed ends, nearest-neighbour springs.  A trajectory
// is owned by a tile of LT consecutive lanes (LT = 2..32, a power of two), each lane holding PPL
// consecutive particles: lane l <-> particles l PPL + 1 .. (l + 1) PPL.  For each of its particles a
// lane holds the orbit coordinate and the K deviation-vector coordinates: PPL (1 + K) (q, p) pairs
// and their stage forces, all in registers.
//   * Neighbour coupling goes through warp shuffles of the STAGE COORDINATES only: per column one
//     shuffle up (the left neighbour's last particle) and one shuffle down (the right neighbour's
//     first particle), both issued before any arithmetic; springs between two particles of the same
//     lane need none.  A lane evaluates the PPL + 1 springs that touch its particles (the spring it
//     shares with its right neighbour is evaluated by both: one redundant spring per lane instead of
//     a second, dependent shuffle).  The walls q_0 = q_{N+1} = 0 (Eq.(8)) are the zeros the first /
//     last lane substitutes for the missing neighbour (a factor 0 inside the difference: no branch, no select).
//   * PPL = 2 halves the shuffles per particle and removes a third of the spring arithmetic
//     (BASELINE.json configs[4] runs as LT = 4, PPL = 2: DESIGN.md "Layouts").
//   * PAD: chains whose length is not LT PPL are padded with particles pinned at zero (coordinates
//     start at 0 and their force is masked to 0), which act as the right wall; np is the real length.
//   * Norms, dot products, Gram-Schmidt and the Jacobi rotations of GALI_k's SVD are lane-local sums
//     followed by butterfly shuffle reductions over the tile (bit-identical on all lanes).
#pragma once
#include "col_kernels.cuh"

namespace chs {

template <int LT, int PPL_, int K_, bool PAD_ = false, bool COLD_ = false, int NB_ = 1>
struct Chain {
    // NB > 1 ("column blocks", for spectra with more vectors than one lane's registers hold): the trajectory
    // is owned by NB adjacent sub-tiles of LT lanes; each sub-tile integrates its own replica of the orbit
    // (bit-identical: same operations on the same numbers) and K of the NB K deviation vectors; only the
    // Gram-Schmidt step couples the sub-tiles, through shuffles over the whole group.
    static constexpr int K = K_, PPL = PPL_, NB = NB_;
    static constexpr int L = LT * NB;  // lanes per trajectory
    static constexpr int KTOT = K * NB;
    static constexpr bool PAD = PAD_;
    static constexpr bool COLD = COLD_;  // carry words and log accumulators in shared memory
    static constexpr int NCOL = 1 + K;
    static constexpr int NI = NCOL * PPL;  // item v * PPL + j: column v (0 = orbit), local particle j
    static constexpr int NSLOT = LT * PPL;
    static constexpr int NCOMP = PPL;      // items 0..PPL-1: the orbit coordinates -- compensated update
    static_assert(NB == 1 || L <= 32, "column blocks live in one warp");
    // How the first / last lane of an in-warp tile gets the wall's zero in place of the missing neighbour: the
    // shuffled value enters the difference multiplied by the lane constant wl / wr (0 on the wall lane, 1
    // elsewhere), d = Q - wl xl as ONE fused multiply-add in place of the subtraction -- instead of selects after
    // the shuffles (2 FSEL per value: 20 per force evaluation and column pair, 12 % of the instructions of the
    // adaptive GALI_4 kernel).  With wl in {0, 1} the result is the subtraction's, bit for bit.  Measured
    // (DESIGN.md section 6): adaptive GALI_4 N = 8 20.6 -> 18.9 ms, Lyapunov k = 4 58.4 -> 55.3 ms, C5 440 -> 434 ms.
    static constexpr bool WALL_FMA = (LT <= 32);
    using Params = FputParams;

    Params prm;
    int lt;   // lane in the trajectory's group (0 .. L-1)
    int lp;   // lane in the sub-tile = which particles (0 .. LT-1)
    int blk;  // column block (0 .. NB-1)
    int np;   // real chain length (== NSLOT unless PAD)
    mutable int par;  // wide tiles: which half of the edge buffer the next exchange uses
    double wl, wr;    // 0 on the first / last lane of the tile (the wall), 1 elsewhere (WALL_FMA)
    double q[NI], p[NI];
    LogBank<NCOL, COLD> lg;  // deferred-log accumulators, v >= 1: identical on all lanes of the sub-tile

    __device__ __forceinline__ void init(const Params& P) {
        prm = P;
        lt = (int)(threadIdx.x % L);
        lp = lt % LT;
        blk = lt / LT;
        np = PAD ? P.np : NSLOT;
        par = 0;
        wl = (lp == 0) ? 0.0 : 1.0;
        wr = (lp == LT - 1) ? 0.0 : 1.0;
        lg.init();
        init_walls();
    }
    // global index (0-based) of this block's deviation column v >= 1
    __device__ __forceinline__ int gcol(int v) const { return blk * K + (v - 1); }
    __device__ __forceinline__ double dcount() const { return (double)(2 * np * (1 + KTOT)); }
    __device__ __forceinline__ bool real(int j) const { return !PAD || lp * PPL + j < np; }
    __device__ __forceinline__ void reset_logs() { lg.init(); }
    __device__ __forceinline__ void load(const double* y, const double* w, long long n_ic, long long ic,
                                         double psign) {
        const int n = 2 * np;
#pragma unroll
        for (int j = 0; j < PPL; j++) {
            const int pi = lp * PPL + j;
            const bool on = real(j);
            q[j] = on ? y[(long long)pi * n_ic + ic] : 0.0;
            p[j] = on ? psign * y[(long long)(np + pi) * n_ic + ic] : 0.0;
#pragma unroll
            for (int v = 1; v < NCOL; v++) {
                q[v * PPL + j] = on ? w[((long long)gcol(v) * n + pi) * n_ic + ic] : 0.0;
                p[v * PPL + j] = on ? w[((long long)gcol(v) * n + np + pi) * n_ic + ic] : 0.0;
            }
        }
    }
    __device__ __forceinline__ void displace(int comp, double delta, double psign) {
#pragma unroll
        for (int j = 0; j < PPL; j++) {
            const int pi = lp * PPL + j;
            if (!real(j)) continue;  // (a padded slot's index collides with a momentum component)
            if (comp == pi) q[j] += delta;
            if (comp == np + pi) p[j] += psign * delta;
        }
    }
    __device__ __forceinline__ void store(double* y, double* w, long long n_ic, long long ic, bool bad) const {
        const int n = 2 * np;
#pragma unroll
        for (int j = 0; j < PPL; j++) {
            const int pi = lp * PPL + j;
            if (!real(j)) continue;
            if (blk == 0) {  // every block holds the same orbit
                y[(long long)pi * n_ic + ic] = bad ? nan("") : q[j];
                y[(long long)(np + pi) * n_ic + ic] = bad ? nan("") : p[j];
            }
#pragma unroll
            for (int v = 1; v < NCOL; v++) {
                w[((long long)gcol(v) * n + pi) * n_ic + ic] = bad ? nan("") : q[v * PPL + j];
                w[((long long)gcol(v) * n + np + pi) * n_ic + ic] = bad ? nan("") : p[v * PPL + j];
            }
        }
    }
    __device__ __forceinline__ void store_logs(const RunArgs& a, long long ic, bool bad, double elapsed) const {
        if (lp != 0) return;
#pragma unroll
        for (int v = 1; v < NCOL; v++) {
            const long long o = (long long)gcol(v) * a.n_ic + ic;
            const double lv = lg.value(v);
            if (a.logacc) a.logacc[o] = bad ? nan("") : a.logacc[o] + lv;
            if (a.lambda) a.lambda[o] = (bad || elapsed == 0.0) ? nan("") : lv / fabs(elapsed);
        }
    }
    // carried rounding words of this lane's orbit coordinates across a call boundary
    __device__ __forceinline__ void load_carry(const double* cw, long long n_ic, long long ic, double (&qc)[PPL],
                                               double (&pc)[PPL]) const {
#pragma unroll
        for (int j = 0; j < PPL; j++) {
            const int pi = lp * PPL + j;
            qc[j] = real(j) ? cw[(long long)pi * n_ic + ic] : 0.0;
            pc[j] = real(j) ? cw[(long long)(np + pi) * n_ic + ic] : 0.0;
        }
    }
    __device__ __forceinline__ void store_carry(double* cw, long long n_ic, long long ic, const double (&qc)[PPL],
                                                const double (&pc)[PPL], bool bad) const {
#pragma unroll
        for (int j = 0; j < PPL; j++) {
            const int pi = lp * PPL + j;
            if (!real(j) || blk != 0) continue;
            cw[(long long)pi * n_ic + ic] = bad ? 0.0 : qc[j];
            cw[(long long)(np + pi) * n_ic + ic] = bad ? 0.0 : pc[j];
        }
    }
    __device__ __forceinline__ void scrub_carry(double (&)[PPL], double (&)[PPL]) const {}
    __device__ __forceinline__ void on_mask(bool (&on)[NI]) const {
#pragma unroll
        for (int v = 0; v < NCOL; v++)
#pragma unroll
            for (int j = 0; j < PPL; j++) on[v * PPL + j] = real(j);
    }

    // xl[v] = the left neighbour's last particle of column v (0 at the left wall), xr[v] = the right
    // neighbour's first particle (0 at the right wall).  In-warp tiles: shuffles.  Wide tiles (LT > 32, the
    // tile is the thread block): through shared memory.
    __device__ __forceinline__ void exchange(const double (&Q)[NI], double (&xl)[NCOL], double (&xr)[NCOL]) const {
        if constexpr (LT <= 32) {
            const bool first = (lp == 0), last = (lp == LT - 1);
#pragma unroll
            for (int v = 0; v < NCOL; v++) {
                xl[v] = __shfl_up_sync(0xffffffffu, Q[v * PPL + PPL - 1], 1, LT);
                xr[v] = __shfl_down_sync(0xffffffffu, Q[v * PPL], 1, LT);
                if constexpr (!WALL_FMA) {
                    if (first) xl[v] = 0.0;
                    if (last) xr[v] = 0.0;
                }
            }
        } else {
            // wide tile: every thread posts its first and last particle of each column in shared memory
            // ([half][column][slot], slot = lp + 1; slots 0 and LT + 1 are the walls and stay zero), one
            // __syncthreads, then reads its two neighbours' -- no branch, no lane is special
            double* bf = edge_first();
            double* bl = (PPL == 1) ? bf : edge_last();
#pragma unroll
            for (int v = 0; v < NCOL; v++) {
                bf[(par * NCOL + v) * (LT + 2) + lp + 1] = Q[v * PPL];
                if constexpr (PPL > 1) bl[(par * NCOL + v) * (LT + 2) + lp + 1] = Q[v * PPL + PPL - 1];
            }
            __syncthreads();
#pragma unroll
            for (int v = 0; v < NCOL; v++) {
                xl[v] = bl[(par * NCOL + v) * (LT + 2) + lp];
                xr[v] = bf[(par * NCOL + v) * (LT + 2) + lp + 2];
            }
            par ^= 1;
        }
    }
    // the wide tile's exchange buffers (two halves: the buffer alternates between calls, so one barrier
    // per call is enough) and their wall slots
    __device__ __forceinline__ static double* edge_first() {
        __shared__ double b[2 * NCOL * (LT + 2)];
        return b;
    }
    __device__ __forceinline__ static double* edge_last() {
        __shared__ double b[(PPL > 1 ? 2 * NCOL * (LT + 2) : 1)];
        return b;
    }
    __device__ __forceinline__ void init_walls() const {
        if constexpr (LT > 32) {
            if (lp < 2 * NCOL) {  // slots 0 and LT + 1 of every (half, column)
                edge_first()[lp * (LT + 2)] = 0.0;
                edge_first()[lp * (LT + 2) + LT + 1] = 0.0;
                if constexpr (PPL > 1) {
                    edge_last()[lp * (LT + 2)] = 0.0;
                    edge_last()[lp * (LT + 2) + LT + 1] = 0.0;
                }
            }
            __syncthreads();
        }
    }

    // Eq.(7) with Eq.(8): p_i' = phi(Dq_{i+1}) - phi(Dq_i), Dq_i = q_i - q_{i-1}; variational:
    // dp_i' = g(Dq_{i+1}) dDq_{i+1} - g(Dq_i) dDq_i.  Springs s = 0..PPL of this lane: s = 0 to the left
    // neighbour (or the left wall), s = PPL to the right neighbour (or the right wall).
    // sc: the factor the forces come out multiplied by (1, or h^2 in the adaptive kernels): it scales the
    // spring constants once per attempt (the same products for all 12 stages), nothing per spring.
    __device__ __forceinline__ void force(const double (&Q)[NI], double (&F)[NI], double sc = 1.0) const {
        FputParams prm = this->prm;
        prm.k *= sc;
        prm.al *= sc;
        prm.be *= sc;
        prm.al2 *= sc;
        prm.be3 *= sc;
        // all neighbour values first: 2 shuffles per column, none depends on arithmetic
        double xl[NCOL], xr[NCOL];
        exchange(Q, xl, xr);
        double g[PPL + 1], ph[PPL + 1];
#pragma unroll
        for (int s = 0; s <= PPL; s++) {
            double d;
            if constexpr (WALL_FMA) d = (s == 0) ? fma(-wl, xl[0], Q[0]) : (s == PPL) ? fma(wr, xr[0], -Q[PPL - 1]) : Q[s] - Q[s - 1];
            else d = (s == 0) ? Q[0] - xl[0] : (s == PPL) ? xr[0] - Q[PPL - 1] : Q[s] - Q[s - 1];
            ph[s] = fput_phi(prm, d);
            g[s] = fput_g(prm, d);
        }
#pragma unroll
        for (int j = 0; j < PPL; j++) F[j] = real(j) ? ph[j + 1] - ph[j] : 0.0;
#pragma unroll
        for (int v = 1; v < NCOL; v++) {
            const double* X = &Q[v * PPL];
            double T[PPL + 1];  // T[s] = g_s e_s for the inner springs s = 1..PPL-1
#pragma unroll
            for (int s = 1; s < PPL; s++) T[s] = g[s] * (X[s] - X[s - 1]);
            const double e0 = WALL_FMA ? fma(-wl, xl[v], X[0]) : X[0] - xl[v];
            const double eP = WALL_FMA ? fma(wr, xr[v], -X[PPL - 1]) : xr[v] - X[PPL - 1];
#pragma unroll
            for (int j = 0; j < PPL; j++) {
                double f;
                if constexpr (PPL == 1) {
                    f = fma(g[1], eP, -(g[0] * e0));
                } else {
                    if (j == 0) f = fma(-g[0], e0, T[1]);
                    else if (j == PPL - 1) f = fma(g[PPL], eP, -T[PPL - 1]);
                    else f = T[j + 1] - T[j];
                }
                F[v * PPL + j] = real(j) ? f : 0.0;
            }
        }
    }

    __device__ __forceinline__ void force2(const double (&Qa)[NI], double (&Fa)[NI], const double (&Qb)[NI],
                                           double (&Fb)[NI], double sc = 1.0) const {
        force(Qa, Fa, sc);
        force(Qb, Fb, sc);
    }

    __device__ __forceinline__ double dot(int u, int v) const {
        double s = 0.0;
#pragma unroll
        for (int j = 0; j < PPL; j++) s = fma(q[u * PPL + j], q[v * PPL + j], fma(p[u * PPL + j], p[v * PPL + j], s));
        return tile_sum<LT>(s);
    }
    __device__ __forceinline__ void scale(int v, double f) {
#pragma unroll
        for (int j = 0; j < PPL; j++) {
            q[v * PPL + j] *= f;
            p[v * PPL + j] *= f;
        }
    }

    // w_v <- w_v/|w_v|, lg_v += ln|w_v|
    __device__ __forceinline__ void renorm(bool want_log, bool apply) {
        if constexpr (K > 0) {
            double s2[K];
#pragma unroll
            for (int v = 1; v < NCOL; v++) {
                double s = 0.0;
#pragma unroll
                for (int j = 0; j < PPL; j++) s = fma(q[v * PPL + j], q[v * PPL + j], fma(p[v * PPL + j], p[v * PPL + j], s));
                s2[v - 1] = s;
            }
            tile_sum_vec<LT, K>(s2);  // all K squared norms in one reduction
#pragma unroll
            for (int v = 1; v < NCOL; v++) {
                const double s = s2[v - 1], ri = fast_rsqrt(s);
                scale(v, apply ? ri : 1.0);
                if (want_log && apply) lg.mul(v, s * ri);
            }
        }
    }
    // modified Gram-Schmidt, right-looking order (see col_kernels.cuh)
    __device__ __forceinline__ void mgs(bool want_log, bool apply) {
        if constexpr (NB == 1) {
#pragma unroll
            for (int v = 1; v < NCOL; v++) {
                const double s = dot(v, v), ri = fast_rsqrt(s);
                scale(v, apply ? ri : 1.0);
                if (want_log && apply) lg.mul(v, s * ri);
#pragma unroll
                for (int u = v + 1; u < NCOL; u++) {
                    double dt = dot(v, u);
                    if (!apply) dt = 0.0;
#pragma unroll
                    for (int j = 0; j < PPL; j++) {
                        q[u * PPL + j] = fma(-dt, q[v * PPL + j], q[u * PPL + j]);
                        p[u * PPL + j] = fma(-dt, p[v * PPL + j], p[u * PPL + j]);
                    }
                }
            }
        } else {
            // column blocks: global column g lives in block g / K as local column 1 + g % K.  It is broadcast
            // to every block (lane (b, lp) reads lane (owner, lp)), normalised there redundantly (same numbers,
            // same order: bit-identical), written back by its owner, and projected out of every later column.
            static_for<0, KTOT>([&](auto gc) {
                constexpr int g = decltype(gc)::value, owner = g / K, v = 1 + g % K;
                double wq[PPL], wp[PPL];
                double s = 0.0;
#pragma unroll
                for (int j = 0; j < PPL; j++) {
                    wq[j] = __shfl_sync(0xffffffffu, q[v * PPL + j], owner * LT + lp, L);
                    wp[j] = __shfl_sync(0xffffffffu, p[v * PPL + j], owner * LT + lp, L);
                    s = fma(wq[j], wq[j], fma(wp[j], wp[j], s));
                }
                s = tile_sum<LT>(s);
                const double ri = fast_rsqrt(s);
#pragma unroll
                for (int j = 0; j < PPL; j++) {
                    wq[j] *= ri;
                    wp[j] *= ri;
                }
                if (apply && blk == owner) {
#pragma unroll
                    for (int j = 0; j < PPL; j++) {
                        q[v * PPL + j] = wq[j];
                        p[v * PPL + j] = wp[j];
                    }
                    if (want_log) lg.mul(v, s * ri);
                }
#pragma unroll
                for (int u = 1; u < NCOL; u++) {
                    double d = 0.0;
#pragma unroll
                    for (int j = 0; j < PPL; j++) d = fma(wq[j], q[u * PPL + j], fma(wp[j], p[u * PPL + j], d));
                    d = tile_sum<LT>(d);
                    if (!(apply && gcol(u) > g)) d = 0.0;
#pragma unroll
                    for (int j = 0; j < PPL; j++) {
                        q[u * PPL + j] = fma(-d, wq[j], q[u * PPL + j]);
                        p[u * PPL + j] = fma(-d, wp[j], p[u * PPL + j]);
                    }
                }
            });
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
        static_assert(IND == IND_NONE || NB == 1, "SALI / GALI are evaluated inside one sub-tile");
        if constexpr (IND == IND_SALI) {
            constexpr int b = (K >= 2 ? 2 : 1);
            double sp = 0.0, sm = 0.0;
#pragma unroll
            for (int j = 0; j < PPL; j++) {
                const double uq = q[PPL + j] + q[b * PPL + j], up = p[PPL + j] + p[b * PPL + j];
                const double dq = q[PPL + j] - q[b * PPL + j], dp = p[PPL + j] - p[b * PPL + j];
                sp = fma(uq, uq, fma(up, up, sp));
                sm = fma(dq, dq, fma(dp, dp, sm));
            }
            sp = sqrt(tile_sum<L>(sp));
            sm = sqrt(tile_sum<L>(sm));
            return sp < sm ? sp : sm;
        } else if constexpr (IND == IND_GALI) {
            constexpr int M = 2 * PPL;  // this lane's components of a column: (q_j, p_j)
            double W[K][M];
#pragma unroll
            for (int v = 0; v < K; v++)
#pragma unroll
                for (int j = 0; j < PPL; j++) {
                    W[v][2 * j] = q[(v + 1) * PPL + j];
                    W[v][2 * j + 1] = p[(v + 1) * PPL + j];
                }
            const double eps = 8.9e-16;
            for (int sweep = 0; sweep < 30; sweep++) {
                bool rotated = false;
#pragma unroll
                for (int a = 0; a < K - 1; a++)
#pragma unroll
                    for (int b = a + 1; b < K; b++) {
                        double saa = 0.0, sbb = 0.0, sab = 0.0;
#pragma unroll
                        for (int c = 0; c < M; c++) {
                            saa = fma(W[a][c], W[a][c], saa);
                            sbb = fma(W[b][c], W[b][c], sbb);
                            sab = fma(W[a][c], W[b][c], sab);
                        }
                        const double app = tile_sum<L>(saa), aqq = tile_sum<L>(sbb), apq = tile_sum<L>(sab);
                        const bool rot = fabs(apq) > eps * sqrt(app * aqq);
                        rotated = rotated || rot;
                        const double zeta = (aqq - app) / (2.0 * apq);
                        const double t = copysign(1.0, zeta) / (fabs(zeta) + sqrt(fma(zeta, zeta, 1.0)));
                        const double cs = rot ? rsqrt(fma(t, t, 1.0)) : 1.0, sn = rot ? cs * t : 0.0;
#pragma unroll
                        for (int c = 0; c < M; c++) {
                            const double x = W[a][c], y = W[b][c];
                            W[a][c] = cs * x - sn * y;
                            W[b][c] = fma(sn, x, cs * y);
                        }
                    }
                if (!group_any<L>(rotated)) break;
            }
            double gl = 1.0;
#pragma unroll
            for (int v = 0; v < K; v++) {
                double s = 0.0;
#pragma unroll
                for (int c = 0; c < M; c++) s = fma(W[v][c], W[v][c], s);
                gl *= sqrt(tile_sum<L>(s));
            }
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
