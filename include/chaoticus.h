/* chaoticus.h -- C ABI of the B200-native (sm_100a, FP64) ensemble integrator.
 *
 * The hot path of arXiv 2507.00622 ("Chaoticus", /root/reference/PAPER.md): huge ensembles of
 * independent initial conditions of a Hamiltonian system integrated with the
 * 8th-order Dormand-Prince method, fixed step "DOP 8" or adaptive "DOP 8(5)" (PAPER.md:43,
 * PAPER.md:47-53), each trajectory carrying its variational equations and
 * accumulating a chaos indicator as it goes: SALI, GALI_k from singular values
 * (PAPER.md:55), the arc-length Lagrangian descriptor, or the
 * Lyapunov spectrum via QR / Gram-Schmidt.
 *
 * CONVENTIONS (every entry point)
 *  - Pointers marked DEVICE are CUDA device pointers to FP64 (or the stated integer type) in
 *    the current device's memory; pointers marked HOST are ordinary host pointers.
 *  - Layout is structure-of-arrays, component-major / IC-minor:
 *        y[c * n_ic + ic],            c < n            (n = phase-space dimension 2N,
 *        w[(v * n + c) * n_ic + ic],  v < k                 ordering (q_1..q_N, p_1..p_N))
 *        out[s * n_ic + ic]           for per-sample / per-vector outputs.
 *  - Ownership: the caller owns every buffer.  Device-pointer entry points allocate nothing,
 *    free nothing, and only ENQUEUE work on `stream` (a cudaStream_t passed as void*; NULL =
 *    the legacy default stream); they do not synchronise.  The *_host entry points allocate
 *    their own device scratch, copy in, run, copy out, synchronise and free before returning.
 *  - y and w are advanced IN PLACE to the final time, w is returned normalised
 *    (orthonormalised by chaoticus_lyap), so a second call continues the run.
 *  - Errors: argument errors return CHS_EINVAL (nothing is launched); a system / k / size
 *    with no compiled kernel returns CHS_EUNSUPPORTED; a CUDA failure returns CHS_ECUDA.
 *    chaoticus_last_error() gives a message.  Trouble of ONE trajectory is not a call error:
 *    it sets status[ic] (CHS_ST_*) and that trajectory's y, w and outputs are NaN.
 *  - n_ic = 0 is a valid no-op.  There is no CPU fallback: without a CUDA device every
 *    compute entry point returns CHS_ECUDA.
 */
#ifndef CHAOTICUS_H
#define CHAOTICUS_H

#ifdef __cplusplus
extern "C" {
#endif

#define CHAOTICUS_VERSION 220 /* 0.2.2: + chaoticus_ld_neighbour_diffs_noalloc */

typedef enum { CHS_OK = 0, CHS_EINVAL = 1, CHS_EUNSUPPORTED = 2, CHS_ECUDA = 3 } chs_rc;

/* Systems (the first three separable, H = |p|^2/2 + V(q)):
 *  CHS_SYS_HENON_HEILES  n = 4, no params.  PAPER.md:87 Eq.(4), Eq.(5).
 *  CHS_SYS_COUPLED3      n = 6, params (omega1, omega2, omega3, eps):
 *                        V = sum omega_i^2 q_i^2 / 2 + eps q1^2 q2 + eps q2^2 q3
 *                        (BASELINE.json configs[3]; eps = 0: uncoupled oscillators).
 *  CHS_SYS_FPUT          n = 2N, params (N, k, alpha, beta), N given as a double, fixed ends
 *                        q_0 = q_{N+1} = 0, N+1 springs.  PAPER.md:98 Eq.(6),
 *                        PAPER.md:103-106 Eq.(7), Eq.(8).  Compiled: every N from 1 to 256
 *                        (integration, LD, SALI, GALI_4, Lyapunov k = 4; N = 8 also GALI_2,3 and k = 1,2);
 *                        Lyapunov spectra on column blocks: k = 2N for N = 4, 8; k = 8 for N = 8, 16.
 *  CHS_SYS_DOUBLE_PENDULUM  n = 4, params (sigma, alpha) = (mass ratio, length ratio); state
 *                        (theta1, theta2, p1, p2).  NOT separable: Eq.(1)
 *                        Eq.(2), Eq.(3); generic first-order kernels.  Integration (fixed,
 *                        adaptive), LD, SALI (fixed, adaptive), GALI_2..4, Lyapunov k = 1, 2, 4 (k = 1, 4
 *                        also adaptive); variational equations = the derivative of Eq.(3). */
typedef enum { CHS_SYS_HENON_HEILES = 0, CHS_SYS_COUPLED3 = 1, CHS_SYS_FPUT = 2, CHS_SYS_DOUBLE_PENDULUM = 3 } chs_system;

typedef struct {
    int system;           /* chs_system */
    int n_params;         /* number of doubles at params */
    const double* params; /* HOST; read during the call only */
} chs_problem;

/* Stepper.  adaptive = 0: n_steps steps of signed size h from t0 ("DOP 8").
 * adaptive = 1: from t0 to t_end with per-trajectory step control ("DOP 8(5)", PAPER.md:48,
 * error estimate PAPER.md:53): err = |h| S5 / sqrt(D (S5 + 0.01 S3)) over all D components of
 * the augmented state, scale = atol + rtol max(|y|,|y+|); accept iff err < 1; step factor
 * 0.9 err^(-1/8) clipped to [0.2, 10] (<= 1 after a rejection); last step lands on t_end;
 * h0 <= 0 selects the automatic starting step; max_steps <= 0 = unbounded attempts. */
typedef struct {
    int adaptive;
    double t0;
    double h;            /* fixed */
    long long n_steps;   /* fixed */
    double t_end, rtol, atol, h0; /* adaptive */
    long long max_steps;          /* adaptive */
} chs_stepper;

/* Per-trajectory report and continuation state; the array members are DEVICE or NULL.
 * Checkpoint / resume: y and w are advanced in place, so a second call
 * continues the run.  The orbit is advanced with a compensated sum whose carried rounding word
 * lives in registers; `carry` takes it across a call boundary.  A
 * continuation call (resume = 1) reads `carry` on entry and does NOT normalise / orthonormalise
 * w on entry (w is the unit / orthonormal set the previous call returned).  With carry and
 * resume = 1, a fixed-step run split at a multiple of renorm_every steps gives y, w and the
 * indicator BIT-IDENTICAL to the one-call run (lognorm / logsum / lambda agree to rounding only:
 * the logarithm of a product is taken once per call).  Adaptive runs of the separable systems
 * honour resume (no entry normalisation) but neither read nor write carry: their last step is
 * clipped to t_end, so a split adaptive run is a different step sequence anyway. */
#define CHS_ST_OK 0
#define CHS_ST_NONFINITE 1
#define CHS_ST_UNDERFLOW 2
#define CHS_ST_MAXSTEPS 3
typedef struct {
    long long* n_accepted; /* [n_ic] accepted steps.  Fixed step: n_steps -- or, for a trajectory whose state
                              stopped being finite (status CHS_ST_NONFINITE), the step at which it was found
                              dead: the state is tested after every 8th step and after the last, so this is
                              at most 7 steps past the step of death; t_final = t0 + n_accepted h */
    long long* n_rejected; /* [n_ic] rejected attempts (fixed: 0) */
    int* status;           /* [n_ic] CHS_ST_* */
    double* t_final;       /* [n_ic] time reached */
    double* carry;         /* [n][n_ic] (layout of y) in/out: carried rounding words of the orbit
                              update; read on entry iff resume; written at the end of every FIXED-step
                              run (and of the double pendulum's adaptive integration); the other
                              adaptive runs carry no words and leave the array as it is (the *_host
                              forms hand back zeros after such a run with resume = 0) */
    int resume;            /* 0: fresh run (carry starts at 0, w normalised on entry);
                              1: continuation of a previous call (see above) */
} chs_report;

/* phase-space dimension n of a problem, or -1 */
int chaoticus_dim(const chs_problem* pb);
/* rows of the sali / gali output of a FIXED-step run: 1 if sample_every <= 0, else
 * ceil(n_steps / renorm_every) / sample_every + 1 (the last row is the final value) */
long long chaoticus_n_samples(long long n_steps, int renorm_every, int sample_every);

/* PAPER.md:47 (solver 1).  y DEVICE [n][n_ic] in/out. */
int chaoticus_integrate_fixed(const chs_problem* pb, long long n_ic, double* y, double t0, double h,
                              long long n_steps, const chs_report* rep, void* stream);

/* PAPER.md:48, 53 (solver 2 + error computation).  st->adaptive must be 1. */
int chaoticus_integrate_adaptive(const chs_problem* pb, long long n_ic, double* y, const chs_stepper* st,
                                 const chs_report* rep, void* stream);

/* PAPER.md:49-50 (solvers 3, 4) + PAPER.md:56: orbit + 2 deviation vectors, renormalised (not
 * orthogonalised) after every renorm_every-th accepted step and at the end;
 * SALI = min(|w1+w2|, |w1-w2|) of the unit vectors.
 *  w        DEVICE [2][n][n_ic] in/out; normalised once on entry
 *  sali     DEVICE [n_samples][n_ic]; row s < n_samples-1 = value after the
 *           (s+1)*sample_every-th renormalisation, last row = value at the end.
 *           sample_every must be 0 for adaptive runs (n_samples = 1): their accepted times differ per
 *           trajectory.  A time series of an adaptive run is taken by continuation -- consecutive calls
 *           t_j -> t_{j+1} with rep->resume = 1 (each lands on its checkpoint exactly).
 *  lognorm  DEVICE [2][n_ic] or NULL; the run ADDS sum ln|w_v| of its renormalisations. */
int chaoticus_sali(const chs_problem* pb, long long n_ic, double* y, double* w, const chs_stepper* st,
                   int renorm_every, int sample_every, double* sali, double* lognorm,
                   const chs_report* rep, void* stream);

/* As chaoticus_sali with 2 <= k <= n vectors; GALI_k = product of the k singular values of the
 * n x k matrix of unit deviation vectors. */
int chaoticus_gali(const chs_problem* pb, long long n_ic, double* y, double* w, int k, const chs_stepper* st,
                   int renorm_every, int sample_every, double* gali, double* lognorm,
                   const chs_report* rep, void* stream);

/* Arc-length Lagrangian descriptor (BASELINE.json configs[1]):
 * M_+- = integral of |f(x(t))|_2 over [t0, t0 +- n_steps h], accumulated with the tableau's own
 * quadrature, M += |h| sum_i b_i |k_i|.  y0 DEVICE [n][n_ic], NOT modified; h > 0;
 * ld_fwd, ld_bwd DEVICE [n_ic], either may be NULL.  No variational equations. */
int chaoticus_ld(const chs_problem* pb, long long n_ic, const double* y0, double t0, double h,
                 long long n_steps, double* ld_fwd, double* ld_bwd, void* stream);

/* The same descriptor with the ADAPTIVE solver (PAPER.md:48 solver 2; PAPER.md:39 the descriptor "calculated
 * alongside the trajectory's evolution"; R21): the augmented ODE (y, M), M' = |f(y)|_2, M(t0) = 0;
 * M is one more component of the state and takes part in the error norm (D = n + 1).  st->adaptive must be 1
 * and st->t_end >= st->t0: tau = t_end - t0; ld_fwd = M over [t0, t0 + tau], ld_bwd over [t0 - tau, t0].
 *  y0            DEVICE [n][n_ic], NOT modified;  ld_fwd, ld_bwd DEVICE [n_ic], either may be NULL
 *  rep           optional; its arrays are [2][n_ic] here (row 0 forward, row 1 backward; the row of a direction
 *                that was not asked for is left untouched); carry / resume are ignored.
 * A trajectory that does not end with status 0 gets NaN. */
int chaoticus_ld_adaptive(const chs_problem* pb, long long n_ic, const double* y0, const chs_stepper* st,
                          double* ld_fwd, double* ld_bwd, const chs_report* rep, void* stream);

/* Neighbouring trajectories for the LD-based chaos indicators: for every
 * IC x0 the 1 + 2n members  m = 0: x0;  m = 1 + 2i: x0 + sigma e_i;  m = 2 + 2i: x0 - sigma e_i
 * (e_i: unit vector of phase-space component i in the ordering of y) are generated ON THE DEVICE and
 * integrated in ONE launch together with the centres, forward and backward, as chaoticus_ld does.
 *  y0                DEVICE [n][n_ic], not modified;  sigma >= 0
 *  ld_fwd, ld_bwd    DEVICE [1+2n][n_ic] (row = member), either may be NULL
 *  diff_fwd/_bwd     DEVICE [2n][n_ic] or NULL: the raw differences |M(x0 +- sigma e_i) - M(x0)|
 *                    (row 2i: +, row 2i+1: -), formed on the same stream right after the LD launch;
 *                    a difference array needs the LD array of its direction.
 * The final scalar indicators of refs [11,26,68,10,31] are only cited by the paper, not printed; this call
 * returns what the paper defines -- the members' LDs and their differences (R19). */
int chaoticus_ld_neighbours(const chs_problem* pb, long long n_ic, const double* y0, double sigma, double t0,
                            double h, long long n_steps, double* ld_fwd, double* ld_bwd, double* diff_fwd,
                            double* diff_bwd, void* stream);

/* The differences of chaoticus_ld_neighbours for callers that CANNOT ALLOCATE device memory.
 * Some programs may launch work but never call cudaMalloc: a code embedded in an application that handed the
 * whole HBM to its own pool at start-up (an allocation then fails or breaks a memory budget), or a loop with
 * a latency bound, where the device-wide synchronisation hidden in cudaMalloc / cudaFree stalls all streams.
 * chaoticus_ld_neighbours makes such a caller own (1 + 2n) n_ic doubles per direction for the members'
 * descriptors although it may only want the 2n differences; this call keeps the members' descriptors in a
 * fixed array inside the library instead and hands back the differences alone.
 *  y0, sigma, t0, h, n_steps   as chaoticus_ld_neighbours (y0 DEVICE [n][n_ic], not modified)
 *  diff_fwd, diff_bwd          DEVICE [2n][n_ic], either may be NULL (both NULL: no-op): the same values,
 *                              bit for bit, as chaoticus_ld_neighbours writes to its diff arrays
 * Limit: the scratch is CHS_NOALLOC_MAX_DOUBLES doubles (8 MiB, resident on every GPU that loads the library
 * until the process ends).  A call needs round_up((1 + 2n) n_ic, 32) doubles per requested direction --
 * Henon-Heiles with both directions: n_ic <= 58 254.  A larger request returns CHS_EINVAL with the numbers in
 * chaoticus_last_error() and launches nothing; split the ensemble into slices (ICs are independent).
 * The call allocates and frees nothing: no cudaMalloc / cudaFree / cudaMallocAsync, no event or stream is
 * created.  It only enqueues on `stream`, like the other device-pointer entry points.
 * First call on a device: the library looks up the array's device address (cudaGetSymbolAddress, which also
 * makes the driver load the module there).  Make that first call during set-up, outside any stream capture.
 * Sharing: all calls on a device use the SAME array, and it keeps the previous call's contents.  Nothing in
 * it needs clearing (a call overwrites every element it later reads), but two calls whose GPU work overlaps --
 * different streams, or different host threads without ordering between their streams -- race on it and
 * give garbage.  Order them (one stream, or events) or use chaoticus_ld_neighbours with your own arrays. */
#define CHS_NOALLOC_MAX_DOUBLES (1 << 20)
int chaoticus_ld_neighbour_diffs_noalloc(const chs_problem* pb, long long n_ic, const double* y0, double sigma,
                                         double t0, double h, long long n_steps, double* diff_fwd,
                                         double* diff_bwd, void* stream);

/* PAPER.md:51-52 (solvers 5, 6): 1 <= k <= n vectors, modified Gram-Schmidt every
 * renorm_every accepted steps and at the end (orthonormalised once on entry),
 * S_v += ln r_vv.  lambda DEVICE [k][n_ic] = this run's sums / |elapsed time| (growth rates per
 * unit of |t|, also for backward-time runs: DESIGN.md R18; may be NULL);
 * logsum DEVICE [k][n_ic] or NULL: the run ADDS its sums. */
int chaoticus_lyap(const chs_problem* pb, long long n_ic, double* y, double* w, int k, const chs_stepper* st,
                   int renorm_every, double* lambda, double* logsum, const chs_report* rep, void* stream);

/* HOST-buffer forms (same meaning; all array arguments HOST, report members HOST or NULL).
 * They allocate device scratch, copy in, run on an internal stream, copy out and synchronise.
 * The scratch comes from a memory pool of the library's own (one per device, stream-ordered allocator);
 * the device's default pool and its settings are not touched.  The pool keeps what a call frees, so that
 * the next call does not go to the driver again: chaoticus_set_option("host_pool_trim", bytes_to_keep)
 * returns the rest.  rep->carry after a fresh (resume = 0) adaptive run is all zeros. */
int chaoticus_ld_host(const chs_problem* pb, long long n_ic, const double* y0, double t0, double h,
                      long long n_steps, double* ld_fwd, double* ld_bwd);
int chaoticus_ld_adaptive_host(const chs_problem* pb, long long n_ic, const double* y0, const chs_stepper* st,
                               double* ld_fwd, double* ld_bwd, const chs_report* rep);
int chaoticus_ld_neighbours_host(const chs_problem* pb, long long n_ic, const double* y0, double sigma, double t0,
                                 double h, long long n_steps, double* ld_fwd, double* ld_bwd, double* diff_fwd,
                                 double* diff_bwd);
int chaoticus_sali_host(const chs_problem* pb, long long n_ic, double* y, double* w, const chs_stepper* st,
                        int renorm_every, int sample_every, double* sali, double* lognorm,
                        const chs_report* rep);
int chaoticus_gali_host(const chs_problem* pb, long long n_ic, double* y, double* w, int k,
                        const chs_stepper* st, int renorm_every, int sample_every, double* gali,
                        double* lognorm, const chs_report* rep);
int chaoticus_lyap_host(const chs_problem* pb, long long n_ic, double* y, double* w, int k,
                        const chs_stepper* st, int renorm_every, double* lambda, double* logsum,
                        const chs_report* rep);
int chaoticus_integrate_host(const chs_problem* pb, long long n_ic, double* y, const chs_stepper* st,
                             const chs_report* rep);

/* Kernel launch shape the library would use for a call (for reporting): writes threads per
 * block, blocks, lanes per trajectory, registers per thread, spill bytes.  what: 0 integrate,
 * 1 sali, 2 gali, 3 ld, 4 lyap.  Returns CHS_EUNSUPPORTED if no kernel is compiled. */
int chaoticus_kernel_info(const chs_problem* pb, int what, int k, int adaptive, long long n_ic, int* info5);

/* Process-wide options.  "adaptive_refill" (1 = on, default; 0 = off): adaptive runs are launched as
 * one resident wave of persistent tiles that take trajectories from a device work queue, so a lane
 * (tile) whose trajectory has ended fetches the next one instead of idling until the slowest lane of
 * its warp ends.  Same results per trajectory (each trajectory's arithmetic does not depend on which
 * lane runs it: bit-identical outputs on and off).  Neutral on uniform ensembles, faster on ensembles
 * with unequal step counts.  Each call in flight owns one of 64 device work counters per
 * device (tracked by an event recorded after its launch); when all 64 are busy the call is launched
 * without refill instead (same results).  Off: one trajectory per tile, the grid covers the ensemble.
 * "host_pool_trim" (value = bytes to keep, >= 0): not a setting but an action -- the memory pool of the
 * *_host entry points on the current device gives what it holds beyond `value` bytes back to the driver
 * (it refills on the next *_host call).  Returns CHS_EINVAL for an unknown name. */
int chaoticus_set_option(const char* name, int value);

const char* chaoticus_last_error(void); /* thread-local, static storage */
int chaoticus_version(void);

#ifdef __cplusplus
}
#endif
#endif /* CHAOTICUS_H */
