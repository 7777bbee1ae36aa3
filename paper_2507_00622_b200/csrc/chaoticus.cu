// chaoticus.cu -- C-ABI front end (include/chaoticus.h): argument checks, coefficient table,
// dispatch to the compiled kernels.  No compute happens on the host; there is no CPU fallback.
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>

#include "../../include/chaoticus.h"
#include "launch.h"

#include <atomic>
#include <initializer_list>
#include <mutex>

namespace {

thread_local char g_err[512] = "";

// lane refill of the adaptive kernels: option + a pool of device work counters
// per device.  A call in flight OWNS its counter: the slot keeps an event recorded on the call's stream
// right after the kernel launch and is handed out again only once that event has completed.  When every
// slot is busy the call runs without refill (one trajectory per tile: same results, bit for bit).
std::atomic<int> g_adaptive_refill{1};
constexpr int kQueueSlots = 64, kMaxDevices = 64;
struct QueuePool {
    unsigned long long* base = nullptr;  // kQueueSlots device counters (cudaMalloc, never freed)
    cudaEvent_t done[kQueueSlots] = {};
    bool used[kQueueSlots] = {};
    bool pending[kQueueSlots] = {};  // leased, kernel not launched yet: the event does not cover it
};
QueuePool g_pools[kMaxDevices];
std::mutex g_pool_mutex;

struct QueueLease {
    unsigned long long* counter = nullptr;
    int dev = -1, slot = -1;
};

// a free counter of the current device, zeroed on `stream`; counter == nullptr: none free (or no device)
QueueLease acquire_queue(cudaStream_t stream) {
    QueueLease l;
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kMaxDevices) return l;
    std::lock_guard<std::mutex> lock(g_pool_mutex);
    QueuePool& P = g_pools[dev];
    if (!P.base && cudaMalloc((void**)&P.base, sizeof(unsigned long long) * kQueueSlots) != cudaSuccess) {
        P.base = nullptr;
        cudaGetLastError();
        return l;
    }
    for (int s = 0; s < kQueueSlots; s++) {
        if (P.used[s]) {
            if (P.pending[s] || cudaEventQuery(P.done[s]) != cudaSuccess) {
                cudaGetLastError();  // cudaErrorNotReady is not sticky, clear it
                continue;
            }
            P.used[s] = false;
        }
        if (!P.done[s] && cudaEventCreateWithFlags(&P.done[s], cudaEventDisableTiming) != cudaSuccess) {
            P.done[s] = nullptr;
            cudaGetLastError();
            return l;
        }
        if (cudaMemsetAsync(P.base + s, 0, sizeof(unsigned long long), stream) != cudaSuccess) return l;
        P.used[s] = P.pending[s] = true;  // the event is recorded by release_after_launch
        l.counter = P.base + s;
        l.dev = dev;
        l.slot = s;
        return l;
    }
    return l;
}
// the slot becomes free when everything enqueued on `stream` so far (the kernel) has completed
void release_after_launch(const QueueLease& l, cudaStream_t stream) {
    if (l.slot < 0) return;
    std::lock_guard<std::mutex> lock(g_pool_mutex);
    QueuePool& P = g_pools[l.dev];
    if (cudaEventRecord(P.done[l.slot], stream) != cudaSuccess) {
        cudaGetLastError();
        cudaStreamSynchronize(stream);  // cannot track it: wait, then the slot is free
        P.used[l.slot] = false;
    }
    P.pending[l.slot] = false;
}

// raw differences |M(x0 +- sigma e_i) - M(x0)| of the members' LDs: ld [1+2n][n_ic] ->
// diff [2n][n_ic].  A stencil over values the LD launch has just written (same stream).
__global__ void ld_diff_kernel(const double* __restrict__ ld, double* __restrict__ diff, long long n_ic, int n_rows) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_ic * n_rows) return;
    diff[i] = fabs(ld[i + n_ic] - ld[i % n_ic]);
}

int fail(int rc, const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof g_err, fmt, ap);
    va_end(ap);
    return rc;
}

// Scratch of the host-buffer entry points: one internal stream per host thread, created on first use
// and destroyed when the thread ends; device buffers come from the stream-ordered allocator, out of a
// memory pool that belongs to this library (one per device, created on first use, kept for the life of
// the process).  The pool keeps freed memory (ITS release threshold is unlimited), so after the first call an
// allocation is a pool look-up, not a cudaMalloc; the device's default pool, which other libraries in the
// process use, is left as it is.  chaoticus_set_option("host_pool_trim", 0) hands the kept memory back.
struct HostCtx {
    cudaStream_t stream = nullptr;
    int dev = -1;
    ~HostCtx() {
        if (stream) cudaStreamDestroy(stream);  // (an error during process teardown is of no consequence)
    }
};
thread_local HostCtx g_host;
cudaMemPool_t g_host_pool[kMaxDevices] = {};
std::mutex g_host_pool_mutex;

cudaError_t host_pool(int dev, cudaMemPool_t* out) {
    if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_host_pool_mutex);
    if (!g_host_pool[dev]) {
        cudaMemPoolProps props;
        std::memset(&props, 0, sizeof props);
        props.allocType = cudaMemAllocationTypePinned;
        props.handleTypes = cudaMemHandleTypeNone;
        props.location.type = cudaMemLocationTypeDevice;
        props.location.id = dev;
        cudaMemPool_t pool = nullptr;
        cudaError_t e = cudaMemPoolCreate(&pool, &props);
        if (e != cudaSuccess) return e;
        unsigned long long keep = ~0ULL;
        e = cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &keep);
        if (e != cudaSuccess) {
            cudaMemPoolDestroy(pool);
            return e;
        }
        g_host_pool[dev] = pool;
    }
    *out = g_host_pool[dev];
    return cudaSuccess;
}

// give the memory the current device's pool holds beyond keep_bytes back to the driver
int trim_host_pool(size_t keep_bytes) {
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return fail(CHS_ECUDA, "CUDA error %d: %s", (int)e, cudaGetErrorString(e));
    if (dev < 0 || dev >= kMaxDevices) return fail(CHS_ECUDA, "device %d out of range", dev);
    if (g_host.stream && g_host.dev == dev) cudaStreamSynchronize(g_host.stream);  // the frees of this thread's calls
    std::lock_guard<std::mutex> lock(g_host_pool_mutex);
    if (!g_host_pool[dev]) return CHS_OK;  // no host-buffer call was made on this device: nothing is held
    e = cudaMemPoolTrimTo(g_host_pool[dev], keep_bytes);
    if (e != cudaSuccess) return fail(CHS_ECUDA, "CUDA error %d: %s", (int)e, cudaGetErrorString(e));
    return CHS_OK;
}

// coefficients premultiplied by powers of h (fixed step), or raw with h = 1 (adaptive)
chs::Tab make_tab(double h) {
    using namespace chs;
    Tab t;
    std::memset(&t, 0, sizeof t);
    const double h2 = h * h;
    for (int i = 0; i < 12; i++) {
        for (int j = 0; j < 12; j++) {
            t.a2[i][j] = coef::A2[i][j] * h2;
            t.ap[i][j] = coef::A[i][j] * h;
        }
        t.cs[i] = coef::CS[i] * h;
        t.bq[i] = coef::BQ[i] * h2;
        t.bp[i] = coef::B[i] * h;
        t.bl[i] = coef::B[i] * std::fabs(h);
        t.e5q[i] = coef::E5Q[i];
        t.e3q[i] = coef::E3Q[i];
        t.e5p[i] = coef::E5[i];
        t.e3p[i] = coef::E3[i];
        t.d3[i] = coef::B[i] - coef::E3[i];
    }
    t.h = h;
    return t;
}

int dim_of(const chs_problem* pb, int* fput_n) {
    if (fput_n) *fput_n = 0;
    if (!pb) return -1;
    switch (pb->system) {
        case CHS_SYS_HENON_HEILES: return 4;
        case CHS_SYS_COUPLED3: return (pb->params && pb->n_params >= 4) ? 6 : -1;
        case CHS_SYS_DOUBLE_PENDULUM:
            return (pb->params && pb->n_params >= 2 && pb->params[1] > 0.0 && pb->params[0] > -1.0) ? 4 : -1;
        case CHS_SYS_FPUT: {
            if (!pb->params || pb->n_params < 4) return -1;
            const double Nd = pb->params[0];
            if (!(Nd >= 1.0) || Nd > 4096.0 || Nd != std::floor(Nd)) return -1;
            if (fput_n) *fput_n = (int)Nd;
            return 2 * (int)Nd;
        }
    }
    return -1;
}

// one table per system; FPUT picks the tile class from the chain length (fput_launch.h)
typedef int (*Launcher)(const chs::LaunchReq&);
int first_of(const chs::LaunchReq& rq, std::initializer_list<Launcher> ls) {
    for (Launcher l : ls) {
        const int r = l(rq);
        if (r != -1) return r;
    }
    return -1;
}
int dispatch_fput(const chs::LaunchReq& rq) {
    using namespace chs;
    const int N = rq.fput_n;
    int r = try_launch_fput_spec(rq);  // spectra on column blocks
    if (r != -1) return r;
    switch (N) {  // exact tiles
        case 4: r = try_launch_fput_n4(rq); break;
        case 8: r = first_of(rq, {try_launch_fput_n8, try_launch_fput8_more, try_launch_fput8_adapt}); break;
        case 16: r = try_launch_fput_n16(rq); break;
        case 32: r = try_launch_fput_n32(rq); break;
        case 64: r = try_launch_fput_n64(rq); break;
        default: break;
    }
    if (r != -1) return r;
    if (N < 4) r = try_launch_fput_pad4(rq);
    else if (N > 4 && N < 8) r = try_launch_fput_pad8(rq);
    else if (N > 8 && N < 16) r = try_launch_fput_pad16(rq);
    else if (N > 16 && N < 32) r = try_launch_fput_pad32(rq);
    else if (N > 32 && N < 64) r = try_launch_fput_pad64(rq);
    if (r != -1) return r;
    // wide tiles: longer chains, and what the in-warp classes lack above 32 particles (Lyapunov, adaptive GALI_4)
    if (N > 32 && N <= 64) return try_launch_fput_wide64(rq);
    if (N > 64 && N <= 128) return try_launch_fput_wide128(rq);
    if (N > 128 && N <= 256) return try_launch_fput_wide256(rq);
    return -1;
}
int dispatch(const chs::LaunchReq& rq) {
    using namespace chs;
    switch (rq.system) {
        case CHS_SYS_HENON_HEILES:
            return first_of(rq, {try_launch_hh, try_launch_hh_ind, try_launch_hh_adapt, try_launch_hh_adapt2});
        case CHS_SYS_COUPLED3: return first_of(rq, {try_launch_c3, try_launch_c3_lyap, try_launch_c3_more});
        case CHS_SYS_FPUT: return dispatch_fput(rq);
        case CHS_SYS_DOUBLE_PENDULUM: return try_launch_dp(rq);
        default: return -1;
    }
}

int finish(int r, const chs::LaunchReq& rq) {
    if (r == -1)
        return fail(CHS_EUNSUPPORTED, "no compiled kernel for system=%d what=%d k=%d adaptive=%d", rq.system,
                    rq.what, rq.k, rq.adaptive);
    if (r != 0) return fail(CHS_ECUDA, "CUDA error %d: %s", r, cudaGetErrorString((cudaError_t)r));
    return CHS_OK;
}

int check_stepper(const chs_stepper* st, int want_adaptive /* -1 any */) {
    if (!st) return fail(CHS_EINVAL, "stepper is NULL");
    if (want_adaptive >= 0 && (st->adaptive != 0) != (want_adaptive != 0))
        return fail(CHS_EINVAL, "stepper.adaptive = %d not valid for this entry point", st->adaptive);
    if (!st->adaptive) {
        if (!(st->h != 0.0) || !std::isfinite(st->h)) return fail(CHS_EINVAL, "fixed step: h must be finite and != 0");
        if (st->n_steps < 0) return fail(CHS_EINVAL, "fixed step: n_steps < 0");
    } else {
        if (!(st->rtol > 0.0) || !(st->atol > 0.0)) return fail(CHS_EINVAL, "adaptive: rtol and atol must be > 0");
        if (!std::isfinite(st->t_end) || !std::isfinite(st->t0)) return fail(CHS_EINVAL, "adaptive: t0/t_end not finite");
    }
    return CHS_OK;
}

// common body of integrate / sali / gali / lyap
int run_common(int what, const chs_problem* pb, long long n_ic, double* y, double* w, int k,
               const chs_stepper* st, int renorm_every, int sample_every, double* series, double* logacc,
               double* lambda, const chs_report* rep, void* stream, chs::KernelInfo* info) {
    int fput_n = 0;
    const int n = dim_of(pb, &fput_n);
    if (n < 0) return fail(CHS_EINVAL, "unknown system or bad params");
    if (n_ic < 0) return fail(CHS_EINVAL, "n_ic < 0");
    int rc = check_stepper(st, -1);
    if (rc) return rc;
    if (!info) {
        if (n_ic > 0 && !y) return fail(CHS_EINVAL, "y is NULL");
        if (n_ic > 0 && k > 0 && !w) return fail(CHS_EINVAL, "w is NULL");
    }
    if (what == chs::WHAT_INTEGRATE && k != 0) return fail(CHS_EINVAL, "integrate: k must be 0");
    if (what == chs::WHAT_SALI && k != 2) return fail(CHS_EINVAL, "sali: k must be 2");
    if (what == chs::WHAT_GALI && (k < 2 || k > n)) return fail(CHS_EINVAL, "gali: need 2 <= k <= n");
    if (what == chs::WHAT_LYAP && (k < 1 || k > n)) return fail(CHS_EINVAL, "lyap: need 1 <= k <= n");
    if (what != chs::WHAT_INTEGRATE && renorm_every < 1) return fail(CHS_EINVAL, "renorm_every < 1");
    if (sample_every < 0) return fail(CHS_EINVAL, "sample_every < 0");
    if (st->adaptive && sample_every > 0) return fail(CHS_EINVAL, "adaptive runs: sample_every must be 0");
    if ((what == chs::WHAT_SALI || what == chs::WHAT_GALI) && n_ic > 0 && !series && !info)
        return fail(CHS_EINVAL, "indicator output is NULL");

    chs::LaunchReq rq;
    std::memset(&rq, 0, sizeof rq);
    rq.system = pb->system;
    rq.what = what;
    rq.k = k;
    rq.adaptive = st->adaptive ? 1 : 0;
    rq.fput_n = fput_n;
    rq.params = pb->params;
    rq.n_params = pb->n_params;
    rq.tab = make_tab(st->adaptive ? 1.0 : st->h);
    rq.stream = (cudaStream_t)stream;
    rq.info = info;
    chs::RunArgs& a = rq.args;
    a.n_ic = n_ic;
    a.y = y;
    a.w = w;
    a.h = st->h;
    a.n_steps = st->adaptive ? 0 : st->n_steps;
    a.t0 = st->t0;
    a.t_end = st->t_end;
    a.rtol = st->rtol;
    a.atol = st->atol;
    a.h0 = st->h0;
    a.max_steps = st->max_steps;
    a.m = renorm_every < 1 ? 1 : renorm_every;
    a.sample_every = sample_every;
    a.n_samples = st->adaptive ? 1 : chaoticus_n_samples(st->n_steps, a.m, sample_every);
    a.series = series;
    a.logacc = logacc;
    a.lambda = lambda;
    if (rep) {
        a.n_acc = rep->n_accepted;
        a.n_rej = rep->n_rejected;
        a.status = rep->status;
        a.t_final = rep->t_final;
        a.carry = rep->carry;
        a.resume = rep->resume ? 1 : 0;
    }
    if (n_ic == 0 && !info) return CHS_OK;
    // Fixed step: the kernels latch the step at which a trajectory's state first stops being finite in that
    // trajectory's own report word (n_accepted, else t_final: col_kernels.cuh death_word) by atomicMin, and
    // rewrite the word with its real content at the end; it starts at all ones = "alive".
    if (!st->adaptive && !info && (a.n_acc || a.t_final)) {
        void* word = a.n_acc ? (void*)a.n_acc : (void*)a.t_final;
        const cudaError_t e = cudaMemsetAsync(word, 0xff, sizeof(long long) * (size_t)n_ic, rq.stream);
        if (e != cudaSuccess) return fail(CHS_ECUDA, "CUDA error %d: %s", (int)e, cudaGetErrorString(e));
    }
    QueueLease lease;
    if (st->adaptive && !info && g_adaptive_refill.load() != 0 && pb->system != CHS_SYS_DOUBLE_PENDULUM) {
        lease = acquire_queue(rq.stream);
        a.queue = lease.counter;  // nullptr (every counter busy): launch without refill, same results
    }
    const int r = dispatch(rq);
    release_after_launch(lease, rq.stream);
    return finish(r, rq);
}

}  // namespace

extern "C" {

int chaoticus_version(void) { return CHAOTICUS_VERSION; }

int chaoticus_set_option(const char* name, int value) {
    if (name && std::strcmp(name, "adaptive_refill") == 0) {
        g_adaptive_refill.store(value != 0 ? 1 : 0);
        return CHS_OK;
    }
    if (name && std::strcmp(name, "host_pool_trim") == 0) {
        if (value < 0) return fail(CHS_EINVAL, "host_pool_trim: bytes to keep must be >= 0");
        return trim_host_pool((size_t)value);
    }
    return fail(CHS_EINVAL, "unknown option '%s'", name ? name : "(null)");
}
const char* chaoticus_last_error(void) { return g_err; }

int chaoticus_dim(const chs_problem* pb) { return dim_of(pb, nullptr); }

long long chaoticus_n_samples(long long n_steps, int renorm_every, int sample_every) {
    if (sample_every <= 0) return 1;
    if (renorm_every < 1) renorm_every = 1;
    const long long n_renorm = (n_steps + renorm_every - 1) / renorm_every;
    return n_renorm / sample_every + 1;
}

int chaoticus_integrate_fixed(const chs_problem* pb, long long n_ic, double* y, double t0, double h,
                              long long n_steps, const chs_report* rep, void* stream) {
    chs_stepper st;
    std::memset(&st, 0, sizeof st);
    st.adaptive = 0;
    st.t0 = t0;
    st.h = h;
    st.n_steps = n_steps;
    return run_common(chs::WHAT_INTEGRATE, pb, n_ic, y, nullptr, 0, &st, 1, 0, nullptr, nullptr, nullptr, rep,
                      stream, nullptr);
}

int chaoticus_integrate_adaptive(const chs_problem* pb, long long n_ic, double* y, const chs_stepper* st,
                                 const chs_report* rep, void* stream) {
    int rc = check_stepper(st, 1);
    if (rc) return rc;
    return run_common(chs::WHAT_INTEGRATE, pb, n_ic, y, nullptr, 0, st, 1, 0, nullptr, nullptr, nullptr, rep,
                      stream, nullptr);
}

int chaoticus_sali(const chs_problem* pb, long long n_ic, double* y, double* w, const chs_stepper* st,
                   int renorm_every, int sample_every, double* sali, double* lognorm, const chs_report* rep,
                   void* stream) {
    return run_common(chs::WHAT_SALI, pb, n_ic, y, w, 2, st, renorm_every, sample_every, sali, lognorm, nullptr,
                      rep, stream, nullptr);
}

int chaoticus_gali(const chs_problem* pb, long long n_ic, double* y, double* w, int k, const chs_stepper* st,
                   int renorm_every, int sample_every, double* gali, double* lognorm, const chs_report* rep,
                   void* stream) {
    return run_common(chs::WHAT_GALI, pb, n_ic, y, w, k, st, renorm_every, sample_every, gali, lognorm, nullptr,
                      rep, stream, nullptr);
}

int chaoticus_lyap(const chs_problem* pb, long long n_ic, double* y, double* w, int k, const chs_stepper* st,
                   int renorm_every, double* lambda, double* logsum, const chs_report* rep, void* stream) {
    return run_common(chs::WHAT_LYAP, pb, n_ic, y, w, k, st, renorm_every, 0, nullptr, logsum, lambda, rep,
                      stream, nullptr);
}

static int ld_common(const chs_problem* pb, long long n_ic, const double* y0, double t0, double h,
                     long long n_steps, double* ld_fwd, double* ld_bwd, void* stream, chs::KernelInfo* info,
                     int n_members = 1, double sigma = 0.0) {
    (void)t0;  // autonomous systems: time is bookkeeping only
    int fput_n = 0;
    const int n = dim_of(pb, &fput_n);
    if (n < 0) return fail(CHS_EINVAL, "unknown system or bad params");
    if (n_ic < 0) return fail(CHS_EINVAL, "n_ic < 0");
    if (!(h > 0.0) || !std::isfinite(h)) return fail(CHS_EINVAL, "ld: h must be > 0");
    if (n_steps < 0) return fail(CHS_EINVAL, "ld: n_steps < 0");
    if (!info && n_ic > 0 && !y0) return fail(CHS_EINVAL, "y0 is NULL");
    if (!info && !ld_fwd && !ld_bwd) return CHS_OK;
    chs::LaunchReq rq;
    std::memset(&rq, 0, sizeof rq);
    rq.system = pb->system;
    rq.what = chs::WHAT_LD;
    rq.k = 0;
    rq.adaptive = 0;
    rq.fput_n = fput_n;
    rq.params = pb->params;
    rq.n_params = pb->n_params;
    rq.tab = make_tab(h);
    rq.stream = (cudaStream_t)stream;
    rq.info = info;
    rq.args.n_ic = n_ic;
    rq.args.y0 = y0;
    rq.args.h = h;
    rq.args.n_steps = n_steps;
    rq.args.ld_fwd = ld_fwd;
    rq.args.ld_bwd = ld_bwd;
    rq.args.n_members = n_members;
    rq.args.sigma = sigma;
    rq.dir_first = ld_fwd ? 0 : 1;
    rq.n_dirs = (info || (ld_fwd && ld_bwd)) ? 2 : 1;
    if (info) rq.dir_first = 0;
    if (n_ic == 0 && !info) return CHS_OK;
    return finish(dispatch(rq), rq);
}

int chaoticus_ld(const chs_problem* pb, long long n_ic, const double* y0, double t0, double h, long long n_steps,
                 double* ld_fwd, double* ld_bwd, void* stream) {
    return ld_common(pb, n_ic, y0, t0, h, n_steps, ld_fwd, ld_bwd, stream, nullptr);
}

static int ld_adaptive_common(const chs_problem* pb, long long n_ic, const double* y0, const chs_stepper* st,
                              double* ld_fwd, double* ld_bwd, const chs_report* rep, void* stream,
                              chs::KernelInfo* info) {
    int fput_n = 0;
    const int n = dim_of(pb, &fput_n);
    if (n < 0) return fail(CHS_EINVAL, "unknown system or bad params");
    if (n_ic < 0) return fail(CHS_EINVAL, "n_ic < 0");
    int rc = check_stepper(st, 1);
    if (rc) return rc;
    if (!(st->t_end >= st->t0)) return fail(CHS_EINVAL, "ld_adaptive: t_end must be >= t0 (tau = t_end - t0)");
    if (!info && n_ic > 0 && !y0) return fail(CHS_EINVAL, "y0 is NULL");
    if (!info && !ld_fwd && !ld_bwd) return CHS_OK;
    chs::LaunchReq rq;
    std::memset(&rq, 0, sizeof rq);
    rq.system = pb->system;
    rq.what = chs::WHAT_LD;
    rq.k = 0;
    rq.adaptive = 1;
    rq.fput_n = fput_n;
    rq.params = pb->params;
    rq.n_params = pb->n_params;
    rq.tab = make_tab(1.0);
    rq.stream = (cudaStream_t)stream;
    rq.info = info;
    chs::RunArgs& a = rq.args;
    a.n_ic = n_ic;
    a.y0 = y0;
    a.t0 = st->t0;
    a.t_end = st->t_end;
    a.rtol = st->rtol;
    a.atol = st->atol;
    a.h0 = st->h0;
    a.max_steps = st->max_steps;
    a.m = 1;
    a.n_samples = 1;
    a.ld_fwd = ld_fwd;
    a.ld_bwd = ld_bwd;
    a.dir_first = (info || ld_fwd) ? 0 : 1;
    a.n_dirs = (info || (ld_fwd && ld_bwd)) ? 2 : 1;
    if (rep) {
        a.n_acc = rep->n_accepted;
        a.n_rej = rep->n_rejected;
        a.status = rep->status;
        a.t_final = rep->t_final;
    }
    if (n_ic == 0 && !info) return CHS_OK;
    QueueLease lease;
    if (!info && g_adaptive_refill.load() != 0 && pb->system != CHS_SYS_DOUBLE_PENDULUM) {
        lease = acquire_queue(rq.stream);
        a.queue = lease.counter;
    }
    const int r = dispatch(rq);
    release_after_launch(lease, rq.stream);
    return finish(r, rq);
}

int chaoticus_ld_adaptive(const chs_problem* pb, long long n_ic, const double* y0, const chs_stepper* st,
                          double* ld_fwd, double* ld_bwd, const chs_report* rep, void* stream) {
    return ld_adaptive_common(pb, n_ic, y0, st, ld_fwd, ld_bwd, rep, stream, nullptr);
}

int chaoticus_ld_neighbours(const chs_problem* pb, long long n_ic, const double* y0, double sigma, double t0,
                            double h, long long n_steps, double* ld_fwd, double* ld_bwd, double* diff_fwd,
                            double* diff_bwd, void* stream) {
    const int n = dim_of(pb, nullptr);
    if (n < 0) return fail(CHS_EINVAL, "unknown system or bad params");
    if (!(sigma >= 0.0) || !std::isfinite(sigma)) return fail(CHS_EINVAL, "ld_neighbours: sigma must be finite and >= 0");
    if ((diff_fwd && !ld_fwd) || (diff_bwd && !ld_bwd))
        return fail(CHS_EINVAL, "ld_neighbours: differences need the LD array of the same direction");
    const int rc = ld_common(pb, n_ic, y0, t0, h, n_steps, ld_fwd, ld_bwd, stream, nullptr, 1 + 2 * n, sigma);
    if (rc != CHS_OK || n_ic == 0) return rc;
    const long long total = n_ic * 2LL * n;
    const unsigned blocks = (unsigned)((total + 255) / 256);
    if (diff_fwd) ld_diff_kernel<<<blocks, 256, 0, (cudaStream_t)stream>>>(ld_fwd, diff_fwd, n_ic, 2 * n);
    if (diff_bwd) ld_diff_kernel<<<blocks, 256, 0, (cudaStream_t)stream>>>(ld_bwd, diff_bwd, n_ic, 2 * n);
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(CHS_ECUDA, "CUDA error %d: %s", (int)e, cudaGetErrorString(e));
    return CHS_OK;
}

int chaoticus_kernel_info(const chs_problem* pb, int what, int k, int adaptive, long long n_ic, int* info5) {
    if (!info5) return fail(CHS_EINVAL, "info5 is NULL");
    chs::KernelInfo ki{0, 0, 0, 0, 0};
    int rc;
    if (what == chs::WHAT_LD && adaptive) {
        chs_stepper st;
        std::memset(&st, 0, sizeof st);
        st.adaptive = 1;
        st.t_end = 1.0;
        st.rtol = st.atol = 1e-6;
        rc = ld_adaptive_common(pb, n_ic, nullptr, &st, nullptr, nullptr, nullptr, nullptr, &ki);
    } else if (what == chs::WHAT_LD) {
        rc = ld_common(pb, n_ic, nullptr, 0.0, 1.0, 1, nullptr, nullptr, nullptr, &ki);
    } else {
        chs_stepper st;
        std::memset(&st, 0, sizeof st);
        st.adaptive = adaptive ? 1 : 0;
        st.h = 1.0;
        st.n_steps = 1;
        st.t_end = 1.0;
        st.rtol = st.atol = 1e-6;
        rc = run_common(what, pb, n_ic, nullptr, nullptr, k, &st, 1, 0, nullptr, nullptr, nullptr, nullptr,
                        nullptr, &ki);
    }
    if (rc) return rc;
    info5[0] = ki.tpb;
    info5[1] = ki.blocks;
    info5[2] = ki.lanes;
    info5[3] = ki.regs;
    info5[4] = ki.spill_bytes;
    return CHS_OK;
}

// ---- host-buffer forms ---------------------------------------------------------------------
namespace {
cudaError_t host_stream(cudaStream_t* out) {
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (!g_host.stream || g_host.dev != dev) {
        if (g_host.stream) cudaStreamDestroy(g_host.stream);
        g_host.stream = nullptr;
        e = cudaStreamCreateWithFlags(&g_host.stream, cudaStreamNonBlocking);
        if (e != cudaSuccess) return e;
        g_host.dev = dev;
    }
    *out = g_host.stream;
    return cudaSuccess;
}

struct DevBuf {
    void* p = nullptr;
    size_t bytes = 0;
    cudaStream_t st = nullptr;
    ~DevBuf() {
        if (p) cudaFreeAsync(p, st);
    }
    cudaError_t alloc(size_t b, cudaStream_t stream) {
        bytes = b;
        st = stream;
        if (!b) return cudaSuccess;
        int dev = 0;
        cudaError_t e = cudaGetDevice(&dev);
        if (e != cudaSuccess) return e;
        cudaMemPool_t pool = nullptr;
        e = host_pool(dev, &pool);
        if (e != cudaSuccess) return e;
        return cudaMallocFromPoolAsync(&p, b, pool, stream);
    }
};
#define CK(x)                                                                                  \
    do {                                                                                       \
        cudaError_t e_ = (x);                                                                  \
        if (e_ != cudaSuccess) {                                                               \
            if (stream) cudaStreamSynchronize(stream);                                         \
            return fail(CHS_ECUDA, "CUDA error %d: %s", (int)e_, cudaGetErrorString(e_));      \
        }                                                                                      \
    } while (0)

int run_host(int what, const chs_problem* pb, long long n_ic, double* y, double* w, int k, const chs_stepper* st,
             int renorm_every, int sample_every, double* series, double* logacc, double* lambda,
             const chs_report* rep) {
    cudaStream_t stream = nullptr;
    const int n = dim_of(pb, nullptr);
    if (n < 0) return fail(CHS_EINVAL, "unknown system or bad params");
    if (n_ic < 0) return fail(CHS_EINVAL, "n_ic < 0");
    int rc = check_stepper(st, -1);
    if (rc) return rc;
    if (n_ic == 0) return CHS_OK;
    if (!y || (k > 0 && !w)) return fail(CHS_EINVAL, "y or w is NULL");
    const long long ns = st->adaptive ? 1 : chaoticus_n_samples(st->n_steps, renorm_every, sample_every);
    const size_t by = sizeof(double) * (size_t)n * n_ic, bw = by * (size_t)k, bs = sizeof(double) * (size_t)ns * n_ic,
                 bk = sizeof(double) * (size_t)k * n_ic;
    DevBuf dy, dw, ds, dl, dlam, dacc, drej, dstat, dtf, dcar;
    CK(host_stream(&stream));
    CK(dy.alloc(by, stream));
    CK(dw.alloc(bw, stream));
    if (series) CK(ds.alloc(bs, stream));
    if (logacc) CK(dl.alloc(bk, stream));
    if (lambda) CK(dlam.alloc(bk, stream));
    chs_report drep{nullptr, nullptr, nullptr, nullptr, nullptr, 0};
    if (rep) {
        drep.resume = rep->resume;
        if (rep->carry) {
            CK(dcar.alloc(by, stream));
            drep.carry = (double*)dcar.p;
            // a fresh run starts from zero words; the kernels that carry none (adaptive runs) leave them so
            if (!drep.resume) CK(cudaMemsetAsync(dcar.p, 0, by, stream));
        }
        if (rep->n_accepted) { CK(dacc.alloc(sizeof(long long) * n_ic, stream)); drep.n_accepted = (long long*)dacc.p; }
        if (rep->n_rejected) { CK(drej.alloc(sizeof(long long) * n_ic, stream)); drep.n_rejected = (long long*)drej.p; }
        if (rep->status) { CK(dstat.alloc(sizeof(int) * n_ic, stream)); drep.status = (int*)dstat.p; }
        if (rep->t_final) { CK(dtf.alloc(sizeof(double) * n_ic, stream)); drep.t_final = (double*)dtf.p; }
    }
    CK(cudaMemcpyAsync(dy.p, y, by, cudaMemcpyHostToDevice, stream));
    if (k > 0) CK(cudaMemcpyAsync(dw.p, w, bw, cudaMemcpyHostToDevice, stream));
    if (logacc) CK(cudaMemcpyAsync(dl.p, logacc, bk, cudaMemcpyHostToDevice, stream));
    if (drep.carry && drep.resume) CK(cudaMemcpyAsync(dcar.p, rep->carry, by, cudaMemcpyHostToDevice, stream));
    rc = run_common(what, pb, n_ic, (double*)dy.p, (double*)dw.p, k, st, renorm_every, sample_every, (double*)ds.p,
                    (double*)dl.p, (double*)dlam.p, &drep, stream, nullptr);
    if (rc) {
        cudaStreamSynchronize(stream);
        return rc;
    }
    CK(cudaMemcpyAsync(y, dy.p, by, cudaMemcpyDeviceToHost, stream));
    if (k > 0) CK(cudaMemcpyAsync(w, dw.p, bw, cudaMemcpyDeviceToHost, stream));
    if (series) CK(cudaMemcpyAsync(series, ds.p, bs, cudaMemcpyDeviceToHost, stream));
    if (logacc) CK(cudaMemcpyAsync(logacc, dl.p, bk, cudaMemcpyDeviceToHost, stream));
    if (lambda) CK(cudaMemcpyAsync(lambda, dlam.p, bk, cudaMemcpyDeviceToHost, stream));
    if (rep) {
        if (rep->n_accepted) CK(cudaMemcpyAsync(rep->n_accepted, dacc.p, sizeof(long long) * n_ic, cudaMemcpyDeviceToHost, stream));
        if (rep->n_rejected) CK(cudaMemcpyAsync(rep->n_rejected, drej.p, sizeof(long long) * n_ic, cudaMemcpyDeviceToHost, stream));
        if (rep->status) CK(cudaMemcpyAsync(rep->status, dstat.p, sizeof(int) * n_ic, cudaMemcpyDeviceToHost, stream));
        if (rep->t_final) CK(cudaMemcpyAsync(rep->t_final, dtf.p, sizeof(double) * n_ic, cudaMemcpyDeviceToHost, stream));
        if (rep->carry) CK(cudaMemcpyAsync(rep->carry, dcar.p, by, cudaMemcpyDeviceToHost, stream));
    }
    CK(cudaStreamSynchronize(stream));
    return CHS_OK;
}
}  // namespace

int chaoticus_ld_host(const chs_problem* pb, long long n_ic, const double* y0, double t0, double h,
                      long long n_steps, double* ld_fwd, double* ld_bwd) {
    cudaStream_t stream = nullptr;
    const int n = dim_of(pb, nullptr);
    if (n < 0) return fail(CHS_EINVAL, "unknown system or bad params");
    if (n_ic < 0) return fail(CHS_EINVAL, "n_ic < 0");
    if (n_ic == 0 || (!ld_fwd && !ld_bwd)) return CHS_OK;
    if (!y0) return fail(CHS_EINVAL, "y0 is NULL");
    DevBuf dy, df, db;
    const size_t by = sizeof(double) * (size_t)n * n_ic, bo = sizeof(double) * (size_t)n_ic;
    CK(host_stream(&stream));
    CK(dy.alloc(by, stream));
    if (ld_fwd) CK(df.alloc(bo, stream));
    if (ld_bwd) CK(db.alloc(bo, stream));
    CK(cudaMemcpyAsync(dy.p, y0, by, cudaMemcpyHostToDevice, stream));
    int rc = chaoticus_ld(pb, n_ic, (const double*)dy.p, t0, h, n_steps, (double*)df.p, (double*)db.p, stream);
    if (rc) {
        cudaStreamSynchronize(stream);
        return rc;
    }
    if (ld_fwd) CK(cudaMemcpyAsync(ld_fwd, df.p, bo, cudaMemcpyDeviceToHost, stream));
    if (ld_bwd) CK(cudaMemcpyAsync(ld_bwd, db.p, bo, cudaMemcpyDeviceToHost, stream));
    CK(cudaStreamSynchronize(stream));
    return CHS_OK;
}

int chaoticus_ld_adaptive_host(const chs_problem* pb, long long n_ic, const double* y0, const chs_stepper* st,
                               double* ld_fwd, double* ld_bwd, const chs_report* rep) {
    cudaStream_t stream = nullptr;
    const int n = dim_of(pb, nullptr);
    if (n < 0) return fail(CHS_EINVAL, "unknown system or bad params");
    if (n_ic < 0) return fail(CHS_EINVAL, "n_ic < 0");
    int rc = check_stepper(st, 1);
    if (rc) return rc;
    if (n_ic == 0 || (!ld_fwd && !ld_bwd)) return CHS_OK;
    if (!y0) return fail(CHS_EINVAL, "y0 is NULL");
    DevBuf dy, df, db, dacc, drej, dstat, dtf;
    const size_t by = sizeof(double) * (size_t)n * n_ic, bo = sizeof(double) * (size_t)n_ic;
    CK(host_stream(&stream));
    CK(dy.alloc(by, stream));
    if (ld_fwd) CK(df.alloc(bo, stream));
    if (ld_bwd) CK(db.alloc(bo, stream));
    chs_report drep{nullptr, nullptr, nullptr, nullptr, nullptr, 0};
    if (rep) {  // report arrays are [2][n_ic]
        if (rep->n_accepted) { CK(dacc.alloc(2 * sizeof(long long) * n_ic, stream)); drep.n_accepted = (long long*)dacc.p; }
        if (rep->n_rejected) { CK(drej.alloc(2 * sizeof(long long) * n_ic, stream)); drep.n_rejected = (long long*)drej.p; }
        if (rep->status) { CK(dstat.alloc(2 * sizeof(int) * n_ic, stream)); drep.status = (int*)dstat.p; }
        if (rep->t_final) { CK(dtf.alloc(2 * sizeof(double) * n_ic, stream)); drep.t_final = (double*)dtf.p; }
        if (dacc.p) CK(cudaMemsetAsync(dacc.p, 0, dacc.bytes, stream));
        if (drej.p) CK(cudaMemsetAsync(drej.p, 0, drej.bytes, stream));
        if (dstat.p) CK(cudaMemsetAsync(dstat.p, 0, dstat.bytes, stream));
        if (dtf.p) CK(cudaMemsetAsync(dtf.p, 0, dtf.bytes, stream));
    }
    CK(cudaMemcpyAsync(dy.p, y0, by, cudaMemcpyHostToDevice, stream));
    rc = chaoticus_ld_adaptive(pb, n_ic, (const double*)dy.p, st, (double*)df.p, (double*)db.p, &drep, stream);
    if (rc) {
        cudaStreamSynchronize(stream);
        return rc;
    }
    if (ld_fwd) CK(cudaMemcpyAsync(ld_fwd, df.p, bo, cudaMemcpyDeviceToHost, stream));
    if (ld_bwd) CK(cudaMemcpyAsync(ld_bwd, db.p, bo, cudaMemcpyDeviceToHost, stream));
    if (rep) {
        if (rep->n_accepted) CK(cudaMemcpyAsync(rep->n_accepted, dacc.p, dacc.bytes, cudaMemcpyDeviceToHost, stream));
        if (rep->n_rejected) CK(cudaMemcpyAsync(rep->n_rejected, drej.p, drej.bytes, cudaMemcpyDeviceToHost, stream));
        if (rep->status) CK(cudaMemcpyAsync(rep->status, dstat.p, dstat.bytes, cudaMemcpyDeviceToHost, stream));
        if (rep->t_final) CK(cudaMemcpyAsync(rep->t_final, dtf.p, dtf.bytes, cudaMemcpyDeviceToHost, stream));
    }
    CK(cudaStreamSynchronize(stream));
    return CHS_OK;
}

int chaoticus_ld_neighbours_host(const chs_problem* pb, long long n_ic, const double* y0, double sigma, double t0,
                                 double h, long long n_steps, double* ld_fwd, double* ld_bwd, double* diff_fwd,
                                 double* diff_bwd) {
    cudaStream_t stream = nullptr;
    const int n = dim_of(pb, nullptr);
    if (n < 0) return fail(CHS_EINVAL, "unknown system or bad params");
    if (n_ic < 0) return fail(CHS_EINVAL, "n_ic < 0");
    if ((diff_fwd && !ld_fwd) || (diff_bwd && !ld_bwd))
        return fail(CHS_EINVAL, "ld_neighbours: differences need the LD array of the same direction");
    if (n_ic == 0 || (!ld_fwd && !ld_bwd)) return CHS_OK;
    if (!y0) return fail(CHS_EINVAL, "y0 is NULL");
    DevBuf dy, df, db, ddf, ddb;
    const size_t by = sizeof(double) * (size_t)n * n_ic, bo = sizeof(double) * (size_t)(1 + 2 * n) * n_ic,
                 bd = sizeof(double) * (size_t)(2 * n) * n_ic;
    CK(host_stream(&stream));
    CK(dy.alloc(by, stream));
    if (ld_fwd) CK(df.alloc(bo, stream));
    if (ld_bwd) CK(db.alloc(bo, stream));
    if (diff_fwd) CK(ddf.alloc(bd, stream));
    if (diff_bwd) CK(ddb.alloc(bd, stream));
    CK(cudaMemcpyAsync(dy.p, y0, by, cudaMemcpyHostToDevice, stream));
    int rc = chaoticus_ld_neighbours(pb, n_ic, (const double*)dy.p, sigma, t0, h, n_steps, (double*)df.p, (double*)db.p,
                                     (double*)ddf.p, (double*)ddb.p, stream);
    if (rc) {
        cudaStreamSynchronize(stream);
        return rc;
    }
    if (ld_fwd) CK(cudaMemcpyAsync(ld_fwd, df.p, bo, cudaMemcpyDeviceToHost, stream));
    if (ld_bwd) CK(cudaMemcpyAsync(ld_bwd, db.p, bo, cudaMemcpyDeviceToHost, stream));
    if (diff_fwd) CK(cudaMemcpyAsync(diff_fwd, ddf.p, bd, cudaMemcpyDeviceToHost, stream));
    if (diff_bwd) CK(cudaMemcpyAsync(diff_bwd, ddb.p, bd, cudaMemcpyDeviceToHost, stream));
    CK(cudaStreamSynchronize(stream));
    return CHS_OK;
}

int chaoticus_sali_host(const chs_problem* pb, long long n_ic, double* y, double* w, const chs_stepper* st,
                        int renorm_every, int sample_every, double* sali, double* lognorm, const chs_report* rep) {
    return run_host(chs::WHAT_SALI, pb, n_ic, y, w, 2, st, renorm_every, sample_every, sali, lognorm, nullptr, rep);
}
int chaoticus_gali_host(const chs_problem* pb, long long n_ic, double* y, double* w, int k, const chs_stepper* st,
                        int renorm_every, int sample_every, double* gali, double* lognorm, const chs_report* rep) {
    return run_host(chs::WHAT_GALI, pb, n_ic, y, w, k, st, renorm_every, sample_every, gali, lognorm, nullptr, rep);
}
int chaoticus_lyap_host(const chs_problem* pb, long long n_ic, double* y, double* w, int k, const chs_stepper* st,
                        int renorm_every, double* lambda, double* logsum, const chs_report* rep) {
    return run_host(chs::WHAT_LYAP, pb, n_ic, y, w, k, st, renorm_every, 0, nullptr, logsum, lambda, rep);
}
int chaoticus_integrate_host(const chs_problem* pb, long long n_ic, double* y, const chs_stepper* st,
                             const chs_report* rep) {
    return run_host(chs::WHAT_INTEGRATE, pb, n_ic, y, nullptr, 0, st, 1, 0, nullptr, nullptr, nullptr, rep);
}

// ---- the entry point that allocates nothing ----------------------------------------------------------
// chaoticus_ld_neighbour_diffs_noalloc (include/chaoticus.h).  Who needs it: code that may launch kernels
// but must not touch the allocator -- a solver running inside a host application that reserved all of
// the HBM for its own pool at start-up (cudaMalloc there fails, or steals from a budget someone else
// audits), or a time-critical loop where the implicit device-wide synchronisation of cudaMalloc / cudaFree
// would stall every other stream.  Such a caller can own the small outputs (2n differences per IC) but
// not the (1 + 2n) member descriptors per IC and direction that chaoticus_ld_neighbours wants as arrays;
// here those intermediate values live in the fixed array below, which belongs to the library image.
namespace {

// Scratch of the no-alloc entry point: CHS_NOALLOC_MAX_DOUBLES doubles = 8 MiB.  It is part of the
// loaded module, so every GPU on which this library's kernels are loaded holds these 8 MiB until the
// process exits.  One array per device, shared by ALL calls; it keeps whatever the last call left.
static __device__ __align__(256) double g_noalloc_scratch[CHS_NOALLOC_MAX_DOUBLES];

// In HOST code the identifier g_noalloc_scratch is only a handle for the runtime, NOT a device address
// (handing it to a kernel would fault, or quietly hit host memory on systems where the GPU can reach
// it).  The usable address is asked for once per device, with that device current, and kept here.
double* g_noalloc_ptr[kMaxDevices] = {};
std::mutex g_noalloc_mutex;

cudaError_t noalloc_scratch(double** out) {
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_noalloc_mutex);
    if (!g_noalloc_ptr[dev]) {
        double* p = nullptr;
        e = cudaGetSymbolAddress((void**)&p, g_noalloc_scratch);  // loads the module on `dev` if need be
        if (e != cudaSuccess) return e;
        g_noalloc_ptr[dev] = p;
    }
    *out = g_noalloc_ptr[dev];
    return cudaSuccess;
}

// The difference stencil of ld_diff_kernel, reading the member descriptors straight from the static
// array (device code of this file may name it; only the host needs the looked-up address):
// scratch[off + m * n_ic + ic], m < 1 + n_rows  ->  diff[r * n_ic + ic] = |M_{r+1} - M_0|, r < n_rows.
__global__ void ld_diff_noalloc_kernel(long long off, double* __restrict__ diff, long long n_ic, int n_rows) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_ic * n_rows) return;
    const double* ld = g_noalloc_scratch + off;
    diff[i] = fabs(ld[i + n_ic] - ld[i % n_ic]);
}

}  // namespace

int chaoticus_ld_neighbour_diffs_noalloc(const chs_problem* pb, long long n_ic, const double* y0, double sigma,
                                         double t0, double h, long long n_steps, double* diff_fwd,
                                         double* diff_bwd, void* stream) {
    const int n = dim_of(pb, nullptr);
    if (n < 0) return fail(CHS_EINVAL, "unknown system or bad params");
    if (n_ic < 0) return fail(CHS_EINVAL, "n_ic < 0");
    if (!(sigma >= 0.0) || !std::isfinite(sigma))
        return fail(CHS_EINVAL, "ld_neighbour_diffs_noalloc: sigma must be finite and >= 0");
    if (!diff_fwd && !diff_bwd) return CHS_OK;
    if (n_ic > 0 && !y0) return fail(CHS_EINVAL, "y0 is NULL");
    // one block of (1 + 2n) n_ic member descriptors per requested direction, each starting on a 256-byte line
    const long long members = 1 + 2LL * n;
    const int n_dirs = (diff_fwd ? 1 : 0) + (diff_bwd ? 1 : 0);
    if (n_ic > (long long)CHS_NOALLOC_MAX_DOUBLES)  // also keeps members * n_ic far from overflow
        return fail(CHS_EINVAL, "ld_neighbour_diffs_noalloc: n_ic = %lld is beyond the fixed scratch (%lld doubles)", n_ic,
                    (long long)CHS_NOALLOC_MAX_DOUBLES);
    const long long block = (members * n_ic + 31) / 32 * 32;
    if (block * n_dirs > (long long)CHS_NOALLOC_MAX_DOUBLES)
        return fail(CHS_EINVAL,
                    "ld_neighbour_diffs_noalloc: %d direction(s) x (1 + 2n = %lld) members x n_ic = %lld needs %lld doubles "
                    "of scratch, the fixed array holds %lld: split the ensemble or use chaoticus_ld_neighbours",
                    n_dirs, members, n_ic, block * n_dirs, (long long)CHS_NOALLOC_MAX_DOUBLES);
    if (n_ic == 0) return CHS_OK;
    double* scratch = nullptr;
    const cudaError_t es = noalloc_scratch(&scratch);
    if (es != cudaSuccess) return fail(CHS_ECUDA, "CUDA error %d: %s", (int)es, cudaGetErrorString(es));
    const long long off_fwd = 0, off_bwd = diff_fwd ? block : 0;
    // Nothing in the scratch has to be zero on entry: the LD launch writes every member descriptor of this
    // call (NaN for a trajectory that blew up) before the stencil, later on the same stream, reads it.
    const int rc = ld_common(pb, n_ic, y0, t0, h, n_steps, diff_fwd ? scratch + off_fwd : nullptr,
                             diff_bwd ? scratch + off_bwd : nullptr, stream, nullptr, (int)members, sigma);
    if (rc != CHS_OK) return rc;
    const long long total = n_ic * 2LL * n;
    const unsigned blocks = (unsigned)((total + 255) / 256);
    if (diff_fwd) ld_diff_noalloc_kernel<<<blocks, 256, 0, (cudaStream_t)stream>>>(off_fwd, diff_fwd, n_ic, 2 * n);
    if (diff_bwd) ld_diff_noalloc_kernel<<<blocks, 256, 0, (cudaStream_t)stream>>>(off_bwd, diff_bwd, n_ic, 2 * n);
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(CHS_ECUDA, "CUDA error %d: %s", (int)e, cudaGetErrorString(e));
    return CHS_OK;
}

}  // extern "C"
