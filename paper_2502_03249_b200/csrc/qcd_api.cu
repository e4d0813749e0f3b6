// C-ABI implementation (include/qcd.h): context, field descriptors, layout upload/download,
// operator launches and the CG solver loop with device-resident scalars.
//
// No torch types, no CPU fallback: every entry point either enqueues our kernels on the
// caller's stream or returns an error status.
#include "../../include/qcd.h"

#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <new>
#include <string>

#include "cg_kernels.cuh"
#include "cg_persistent.cuh"
#include "dslash_launch.h"
#include "gauge_kernels.cuh"
#include "lattice.cuh"
#include "layout_kernels.cuh"
#include "measure_kernels.cuh"
#include "mixed_kernels.cuh"
#include "reduce.cuh"

using namespace qcd;

// ------------------------------------------------------------------------------------------
// context
// ------------------------------------------------------------------------------------------
enum { PROF_MAX = 4096, STAGE_BYTES = 32 << 20, POLL_SLOTS = 2, HIST_CAP = 16384 };

struct qcd_field {
    qcd_ctx *ctx;
    int kind;
    void *ptr;
    size_t nbytes;
    int tg;                   // gauge fields: time links with x3 != 0 are the identity (temporal gauge)
};

struct CgState {
    bool active;
    int n;                    // right-hand sides solved in lock step
    const qcd_field *U;
    const void *b[MAXRHS];
    void *x[MAXRHS];
    double m, tol;
    int maxiter;
    cudaEvent_t ev_begin, ev_end;
    cudaGraphExec_t graph;    // replayed by cg_run on small lattices; destroyed by qcd_cg_finish after its sync
};

struct qcd_ctx {
    Lattice L;
    int prec;                 // 64 or 32
    size_t rsize;             // sizeof(real)
    cudaStream_t stream;
    CgScalars *d_scal;        // CG recurrence state, MAXRHS entries
    CgScalars *d_aux;         // scratch state for qcd_apply_M / qcd_re_dot / the mixed solver
    double *d_partials;       // stage-1 partial sums
    unsigned *d_tickets;      // first-level tickets of the two-level last-block election (reduce.cuh)
    double *d_hist;           // residual history, MAXRHS x HIST_CAP (qcd_cg_history)
    unsigned long long *d_timeline; // phase stamps of the persistent loop, 2 x TIMELINE_ITERS x TIMELINE_STAMPS (qcd_cg_timeline_*)
    bool timeline_on;
    int partials_cap;
    CgScalars *h_scal;        // pinned, POLL_SLOTS x MAXRHS entries
    cudaEvent_t poll_ev[POLL_SLOTS];
    void *d_stage;
    void *ws;
    size_t ws_bytes;
    CgState cg;
    int variant;
    int chunk;                // Dslash traversal chunk width in x2: 0 = automatic, else a divisor of N2
    int loop;                 // solver loop: 0 automatic, 1 kernel-by-kernel, 2 graph replay, 3 persistent kernel
    int persist_cluster;      // CTAs of the cluster the most recent persistent solve ran as, 0 = cooperative grid (qcd_last_cg_cluster)
    bool loop_cluster_ok;     // the one-cluster form of the persistent loop may be used (qcd_set_cg_cluster; default on)
    int loop_used;            // loop the most recent qcd_cg_solve* actually ran (qcd_last_cg_loop); 0 = none yet
    int last_n;               // right-hand sides of the most recent finished solve (qcd_cg_history)
    int dev;                  // CUDA device the context was created on; every entry point checks it is current
    long long launches;
    // profiling
    bool prof_on;
    int prof_n, prof_dropped;
    int prof_class[PROF_MAX];
    cudaEvent_t prof_ev[2 * PROF_MAX];
    bool prof_created;
    std::string err;
};

static thread_local std::string g_init_err;

static qcd_status fail(qcd_ctx *ctx, qcd_status s, const char *fmt, const char *a = "", const char *b = "")
{
    char buf[512];
    snprintf(buf, sizeof buf, fmt, a, b);
    if (ctx) ctx->err = buf; else g_init_err = buf;
    return s;
}

#define CU(ctx, call)                                                                      \
    do {                                                                                   \
        cudaError_t e_ = (call);                                                           \
        if (e_ != cudaSuccess) return fail((ctx), QCD_ECUDA, "%s: %s", #call, cudaGetErrorString(e_)); \
    } while (0)

// The context's allocations, its stream and the occupancy / cooperative-launch queries belong to the device
// that was current at qcd_init; a call made with another device current would fail late with an opaque CUDA
// error (or size a cooperative grid from the wrong SM count), so it is rejected here.
static qcd_status check_device(qcd_ctx *ctx, const char *who)
{
    int d = -1;
    if (cudaGetDevice(&d) != cudaSuccess || d != ctx->dev) {
        cudaGetLastError();
        return fail(ctx, QCD_EINVAL, "%s: the current CUDA device is not the one this context was created on (cudaSetDevice first)", who);
    }
    return QCD_OK;
}
#define DEV(ctx, who) do { const qcd_status ds_ = check_device((ctx), (who)); if (ds_) return ds_; } while (0)

// [a, a + na) and [b, b + nb) share a byte
static bool overlaps(const void *a, size_t na, const void *b, size_t nb)
{
    const uintptr_t a0 = (uintptr_t)a, b0 = (uintptr_t)b;
    return a0 < b0 + nb && b0 < a0 + na;
}

extern "C" const char *qcd_strerror(qcd_status s)
{
    switch (s) {
    case QCD_OK: return "ok";
    case QCD_EINVAL: return "invalid argument";
    case QCD_ENOMEM: return "out of memory";
    case QCD_ECUDA: return "CUDA error";
    case QCD_ENOTCONVERGED: return "CG did not converge within maxiter";
    case QCD_EBREAKDOWN: return "CG breakdown (<p,Mp> <= 0 or NaN)";
    default: return "unknown status";
    }
}

extern "C" const char *qcd_last_error(const qcd_ctx *ctx) { return ctx ? ctx->err.c_str() : g_init_err.c_str(); }

static size_t half_spinor_bytes(const qcd_ctx *c) { return (size_t)c->L.Vh * 3 * 2 * c->rsize; }

extern "C" size_t qcd_field_bytes(const qcd_ctx *ctx, int kind)
{
    if (!ctx) return 0;
    switch (kind) {
    case QCD_SPINOR_EVEN:
    case QCD_SPINOR_ODD: return half_spinor_bytes(ctx);
    case QCD_SPINOR_FULL: return 2 * half_spinor_bytes(ctx);
    case QCD_GAUGE: return (size_t)ctx->L.Vh * 72 * 2 * ctx->rsize;
    case QCD_GAUGE_2ROW: return (size_t)ctx->L.Vh * 48 * 2 * ctx->rsize;
    case QCD_COLOUR_MATRIX: return (size_t)ctx->L.Vh * 18 * 2 * ctx->rsize;
    default: return 0;
    }
}

// r, p, Ap (even), t (odd), and a second direction buffer for the persistent kernel
extern "C" size_t qcd_workspace_bytes(const qcd_ctx *ctx) { return ctx ? 5 * half_spinor_bytes(ctx) : 0; }

extern "C" size_t qcd_workspace_bytes_multi(const qcd_ctx *ctx, int n)
{
    if (!ctx || n < 1 || n > MAXRHS) return 0;
    return n == 1 ? qcd_workspace_bytes(ctx) : (size_t)n * 4 * half_spinor_bytes(ctx);
}

// target grid of the reducing vector kernel (8 waves of 148 SMs x 8 resident blocks of 256 threads)
enum { BLAS_REDUCE_GRID = 148 * 8 * 8 };
static int blas_n16(const qcd_ctx *c) { return (int)(half_spinor_bytes(c) / 16); }
static int blas_grid(const qcd_ctx *c) { const int per = BLAS_BLOCK * BLAS_ITEMS; return (blas_n16(c) + per - 1) / per; }
static int dslash_grid_max(const qcd_ctx *c) { return (c->L.Vh + 63) / 64; }   // smallest Dslash block is 64

extern "C" qcd_status qcd_init(qcd_ctx **out, const int dims[4], int precision, void *cuda_stream)
{
    if (!out || !dims) return fail(nullptr, QCD_EINVAL, "qcd_init: NULL argument");
    *out = nullptr;
    if (precision != 64 && precision != 32) return fail(nullptr, QCD_EINVAL, "qcd_init: precision must be 64 or 32");
    long long V = 1;
    for (int i = 0; i < 4; ++i) {
        if (dims[i] < 2 || (dims[i] & 1)) return fail(nullptr, QCD_EINVAL, "qcd_init: extents must be even and >= 2");
        V *= dims[i];
    }
    if (dims[0] % 4) return fail(nullptr, QCD_EINVAL, "qcd_init: N0 must be a multiple of 4");
    if (V >= (1LL << 31)) return fail(nullptr, QCD_EINVAL, "qcd_init: volume must be < 2^31 sites");

    int ndev = 0;
    cudaError_t e = cudaGetDeviceCount(&ndev);
    if (e != cudaSuccess || ndev == 0) {
        cudaGetLastError();
        return fail(nullptr, QCD_ECUDA, "qcd_init: no CUDA device (%s); there is no CPU fallback",
                    e != cudaSuccess ? cudaGetErrorString(e) : "device count 0");
    }
    int dev = 0, major = 0;
    CU(nullptr, cudaGetDevice(&dev));
    CU(nullptr, cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev));
    if (major != 10) return fail(nullptr, QCD_ECUDA, "qcd_init: kernels are built for sm_100a only");

    qcd_ctx *c = new (std::nothrow) qcd_ctx();
    if (!c) return fail(nullptr, QCD_ENOMEM, "qcd_init: host allocation failed");
    c->L.N0 = dims[0]; c->L.N1 = dims[1]; c->L.N2 = dims[2]; c->L.N3 = dims[3];
    c->L.h = dims[0] / 2; c->L.Vh = (int)(V / 2);
    c->L.s1 = c->L.h; c->L.s2 = c->L.h * dims[1]; c->L.s3 = c->L.h * dims[1] * dims[2];
    c->prec = precision; c->rsize = precision == 64 ? 8 : 4;
    c->stream = (cudaStream_t)cuda_stream;
    c->variant = 0; c->launches = 0; c->chunk = 0; c->loop = 0; c->loop_used = 0; c->last_n = 0; c->dev = dev; c->persist_cluster = 0; c->loop_cluster_ok = true;
    c->L.W = dims[2];
    c->prof_on = false; c->prof_created = false; c->prof_n = c->prof_dropped = 0;
    c->ws = nullptr; c->ws_bytes = 0;
    memset(&c->cg, 0, sizeof c->cg);
    c->d_scal = c->d_aux = nullptr; c->d_partials = nullptr; c->d_tickets = nullptr; c->h_scal = nullptr; c->d_stage = nullptr;
    c->d_hist = nullptr; c->d_timeline = nullptr; c->timeline_on = false;
    for (int i = 0; i < POLL_SLOTS; ++i) c->poll_ev[i] = nullptr;

    c->partials_cap = MAXRHS * (dslash_grid_max(c) > blas_grid(c) ? dslash_grid_max(c) : blas_grid(c));
    cudaError_t err = cudaSuccess;
    if (err == cudaSuccess) err = cudaMalloc(&c->d_scal, (MAXRHS + 1) * sizeof(CgScalars));
    if (err == cudaSuccess) err = cudaMemset(c->d_scal, 0, (MAXRHS + 1) * sizeof(CgScalars));
    if (err == cudaSuccess) err = cudaMalloc(&c->d_partials, (size_t)c->partials_cap * sizeof(double));
    const size_t groups = (size_t)(c->partials_cap / MAXRHS) / TICKET_GROUP + 1;      // per CgScalars entry
    if (err == cudaSuccess) err = cudaMalloc(&c->d_tickets, (MAXRHS + 1) * groups * sizeof(unsigned));
    if (err == cudaSuccess) err = cudaMemset(c->d_tickets, 0, (MAXRHS + 1) * groups * sizeof(unsigned));
    for (int i = 0; i <= MAXRHS && err == cudaSuccess; ++i) {
        unsigned *l1 = c->d_tickets + (size_t)i * groups;
        err = cudaMemcpy(&c->d_scal[i].l1, &l1, sizeof l1, cudaMemcpyHostToDevice);
    }
    if (err == cudaSuccess) err = cudaMalloc(&c->d_hist, (size_t)MAXRHS * HIST_CAP * sizeof(double));
    for (int i = 0; i < MAXRHS && err == cudaSuccess; ++i) {          // d_aux (entry MAXRHS) keeps hist = NULL
        double *h = c->d_hist + (size_t)i * HIST_CAP;
        const int cap = HIST_CAP;
        err = cudaMemcpy(&c->d_scal[i].hist, &h, sizeof h, cudaMemcpyHostToDevice);
        if (err == cudaSuccess) err = cudaMemcpy(&c->d_scal[i].hist_cap, &cap, sizeof cap, cudaMemcpyHostToDevice);
    }
    const size_t tl_bytes = 2 * TIMELINE_ITERS * TIMELINE_STAMPS * sizeof(unsigned long long);
    if (err == cudaSuccess) err = cudaMalloc(&c->d_timeline, tl_bytes);
    if (err == cudaSuccess) err = cudaMemset(c->d_timeline, 0, tl_bytes);
    if (err == cudaSuccess) err = cudaMalloc(&c->d_stage, STAGE_BYTES);
    if (err == cudaSuccess) err = cudaMallocHost(&c->h_scal, POLL_SLOTS * MAXRHS * sizeof(CgScalars));
    for (int i = 0; i < POLL_SLOTS && err == cudaSuccess; ++i) err = cudaEventCreateWithFlags(&c->poll_ev[i], cudaEventDisableTiming);
    if (err == cudaSuccess) err = cudaEventCreate(&c->cg.ev_begin);
    if (err == cudaSuccess) err = cudaEventCreate(&c->cg.ev_end);
    if (err != cudaSuccess) {
        fail(nullptr, err == cudaErrorMemoryAllocation ? QCD_ENOMEM : QCD_ECUDA, "qcd_init: %s", cudaGetErrorString(err));
        qcd_finalize(c);
        return err == cudaErrorMemoryAllocation ? QCD_ENOMEM : QCD_ECUDA;
    }
    c->d_aux = c->d_scal + MAXRHS;
    *out = c;
    return QCD_OK;
}

extern "C" qcd_status qcd_finalize(qcd_ctx *c)
{
    if (!c) return QCD_OK;
    cudaStreamSynchronize(c->stream);
    if (c->prof_created) for (int i = 0; i < 2 * PROF_MAX; ++i) cudaEventDestroy(c->prof_ev[i]);
    for (int i = 0; i < POLL_SLOTS; ++i) if (c->poll_ev[i]) cudaEventDestroy(c->poll_ev[i]);
    if (c->cg.ev_begin) cudaEventDestroy(c->cg.ev_begin);
    if (c->cg.ev_end) cudaEventDestroy(c->cg.ev_end);
    if (c->d_scal) cudaFree(c->d_scal);
    if (c->d_partials) cudaFree(c->d_partials);
    if (c->d_tickets) cudaFree(c->d_tickets);
    if (c->d_hist) cudaFree(c->d_hist);
    if (c->d_timeline) cudaFree(c->d_timeline);
    if (c->d_stage) cudaFree(c->d_stage);
    if (c->h_scal) cudaFreeHost(c->h_scal);
    delete c;
    return QCD_OK;
}

// ------------------------------------------------------------------------------------------
// fields
// ------------------------------------------------------------------------------------------
extern "C" qcd_status qcd_field_alloc(qcd_ctx *ctx, int kind, void *device_ptr, size_t nbytes, qcd_field **out)
{
    if (!ctx) return QCD_EINVAL;
    if (!out) return fail(ctx, QCD_EINVAL, "qcd_field_alloc: NULL out");
    *out = nullptr;
    const size_t need = qcd_field_bytes(ctx, kind);
    if (need == 0) return fail(ctx, QCD_EINVAL, "qcd_field_alloc: bad kind");
    if (!device_ptr) return fail(ctx, QCD_EINVAL, "qcd_field_alloc: NULL device pointer");
    if (((uintptr_t)device_ptr) & 255) return fail(ctx, QCD_EINVAL, "qcd_field_alloc: device pointer must be 256-byte aligned");
    if (nbytes < need) return fail(ctx, QCD_EINVAL, "qcd_field_alloc: buffer smaller than qcd_field_bytes");
    qcd_field *f = new (std::nothrow) qcd_field();
    if (!f) return fail(ctx, QCD_ENOMEM, "qcd_field_alloc: host allocation failed");
    f->ctx = ctx; f->kind = kind; f->ptr = device_ptr; f->nbytes = nbytes; f->tg = 0;
    *out = f;
    return QCD_OK;
}

extern "C" qcd_status qcd_field_free(qcd_field *f)
{
    delete f;
    return QCD_OK;
}

extern "C" qcd_status qcd_set_workspace(qcd_ctx *ctx, void *device_ptr, size_t nbytes)
{
    if (!ctx) return QCD_EINVAL;
    if (!device_ptr || (((uintptr_t)device_ptr) & 255) || nbytes < qcd_workspace_bytes(ctx))
        return fail(ctx, QCD_EINVAL, "qcd_set_workspace: need a 256-byte aligned device buffer of qcd_workspace_bytes");
    if (ctx->cg.active) return fail(ctx, QCD_EINVAL, "qcd_set_workspace: a CG solve is in progress");
    ctx->ws = device_ptr; ctx->ws_bytes = nbytes;
    return QCD_OK;
}

// half-field pointer of the requested parity inside a spinor field, or NULL
static void *half_ptr(const qcd_field *f, int parity)
{
    if (!f) return nullptr;
    if (f->kind == QCD_SPINOR_FULL) return (char *)f->ptr + (parity ? half_spinor_bytes(f->ctx) : 0);
    if (f->kind == (parity ? QCD_SPINOR_ODD : QCD_SPINOR_EVEN)) return f->ptr;
    return nullptr;
}

// ------------------------------------------------------------------------------------------
// launch bookkeeping (profiling events, launch count)
// ------------------------------------------------------------------------------------------
struct LaunchScope {
    qcd_ctx *c; int slot;
    LaunchScope(qcd_ctx *ctx, int klass) : c(ctx), slot(-1)
    {
        c->launches++;
        if (c->prof_on) {
            if (c->prof_n < PROF_MAX) {
                slot = c->prof_n++;
                c->prof_class[slot] = klass;
                cudaEventRecord(c->prof_ev[2 * slot], c->stream);
            } else c->prof_dropped++;
        }
    }
    ~LaunchScope() { if (slot >= 0) cudaEventRecord(c->prof_ev[2 * slot + 1], c->stream); }
};

extern "C" qcd_status qcd_profile_enable(qcd_ctx *ctx, int on)
{
    if (!ctx) return QCD_EINVAL;
    if (on && !ctx->prof_created) {
        for (int i = 0; i < 2 * PROF_MAX; ++i) CU(ctx, cudaEventCreate(&ctx->prof_ev[i]));
        ctx->prof_created = true;
    }
    if (on) { ctx->prof_n = 0; ctx->prof_dropped = 0; }
    ctx->prof_on = on != 0;
    return QCD_OK;
}

extern "C" qcd_status qcd_profile_read(qcd_ctx *ctx, int which, int *launches, double *total_ms)
{
    if (!ctx || which < 0 || which >= QCD_K_COUNT) return QCD_EINVAL;
    CU(ctx, cudaStreamSynchronize(ctx->stream));
    int n = 0; double tot = 0.0;
    for (int i = 0; i < ctx->prof_n; ++i) {
        if (ctx->prof_class[i] != which) continue;
        float ms = 0.f;
        CU(ctx, cudaEventElapsedTime(&ms, ctx->prof_ev[2 * i], ctx->prof_ev[2 * i + 1]));
        tot += ms; ++n;
    }
    if (launches) *launches = n;
    if (total_ms) *total_ms = tot;
    return QCD_OK;
}

extern "C" long long qcd_launch_count(const qcd_ctx *ctx) { return ctx ? ctx->launches : 0; }

extern "C" qcd_status qcd_set_traversal_chunk(qcd_ctx *ctx, int width)
{
    if (!ctx) return QCD_EINVAL;
    if (width < 0 || (width > 0 && ctx->L.N2 % width)) return fail(ctx, QCD_EINVAL, "qcd_set_traversal_chunk: width must be 0 (automatic) or a divisor of N2");
    ctx->chunk = width;
    return QCD_OK;
}

extern "C" qcd_status qcd_set_cg_loop(qcd_ctx *ctx, int mode)
{
    if (!ctx) return QCD_EINVAL;
    if (mode < 0 || mode > 3) return fail(ctx, QCD_EINVAL, "qcd_set_cg_loop: mode must be 0 .. 3");
    ctx->loop = mode;
    return QCD_OK;
}

extern "C" int qcd_last_cg_loop(const qcd_ctx *ctx) { return ctx ? ctx->loop_used : 0; }

extern "C" int qcd_last_cg_cluster(const qcd_ctx *ctx) { return (ctx && ctx->loop_used == 3) ? ctx->persist_cluster : 0; }

extern "C" qcd_status qcd_set_cg_cluster(qcd_ctx *ctx, int on)
{
    if (!ctx) return QCD_EINVAL;
    ctx->loop_cluster_ok = on != 0;
    return QCD_OK;
}

extern "C" qcd_status qcd_cg_timeline_enable(qcd_ctx *ctx, int on)
{
    if (!ctx) return QCD_EINVAL;
    if (ctx->cg.active) return fail(ctx, QCD_EINVAL, "qcd_cg_timeline_enable: a solve is in progress");
    ctx->timeline_on = on != 0;
    return QCD_OK;
}

extern "C" qcd_status qcd_cg_timeline_read(qcd_ctx *ctx, unsigned long long *host_out, int cap_iters, int *n_iters)
{
    if (!ctx) return QCD_EINVAL;
    if (!host_out || cap_iters < 0 || !n_iters) return fail(ctx, QCD_EINVAL, "qcd_cg_timeline_read: bad argument");
    if (ctx->cg.active) return fail(ctx, QCD_EINVAL, "qcd_cg_timeline_read: a solve is in progress");
    DEV(ctx, "qcd_cg_timeline_read");
    int n = cap_iters < (int)TIMELINE_ITERS ? cap_iters : (int)TIMELINE_ITERS;
    for (int blk = 0; blk < 2; ++blk)
        CU(ctx, cudaMemcpyAsync(host_out + (size_t)blk * n * TIMELINE_STAMPS, ctx->d_timeline + (size_t)blk * TIMELINE_ITERS * TIMELINE_STAMPS,
                                (size_t)n * TIMELINE_STAMPS * sizeof(unsigned long long), cudaMemcpyDeviceToHost, ctx->stream));
    CU(ctx, cudaStreamSynchronize(ctx->stream));
    // iterations that ran: the last stamp of an iteration is non-zero
    int ran = 0;
    while (ran < n && host_out[(size_t)ran * TIMELINE_STAMPS + TIMELINE_STAMPS - 1] != 0ULL) ++ran;
    *n_iters = ran;
    return QCD_OK;
}

extern "C" qcd_status qcd_set_dslash_variant(qcd_ctx *ctx, int variant)
{
    if (!ctx) return QCD_EINVAL;
    if (variant < 0 || variant > 10) return fail(ctx, QCD_EINVAL, "qcd_set_dslash_variant: unknown variant");
    ctx->variant = variant;
    return QCD_OK;
}

// ------------------------------------------------------------------------------------------
// upload / download
// ------------------------------------------------------------------------------------------
static bool is_gauge_kind(int kind) { return kind == QCD_GAUGE || kind == QCD_GAUGE_2ROW; }
static bool is_spinor_kind(int kind) { return kind == QCD_SPINOR_EVEN || kind == QCD_SPINOR_ODD || kind == QCD_SPINOR_FULL; }
static int gauge_nrow(const qcd_field *U) { return U->kind == QCD_GAUGE_2ROW ? 2 : 3; }

template <typename T>
static qcd_status transfer_t(qcd_ctx *c, const qcd_field *f, const void *host_in, void *host_out)
{
    typedef typename Cplx<T>::type C;
    const bool up = host_in != nullptr;
    const bool matrix = !is_spinor_kind(f->kind);
    const int nmu = f->kind == QCD_COLOUR_MATRIX ? 1 : 4;
    const int nrow = f->kind == QCD_GAUGE_2ROW ? 2 : 3;
    const unsigned per = matrix ? (unsigned)nmu * 9u : 3u;       // complex numbers per site in the host layout
    const size_t per_site = per * sizeof(C);
    const unsigned V = 2u * (unsigned)c->L.Vh;
    unsigned chunk = (unsigned)(STAGE_BYTES / per_site);
    C *even = nullptr, *odd = nullptr;
    if (!matrix) { even = (C *)half_ptr(f, 0); odd = (C *)half_ptr(f, 1); }
    for (unsigned i0 = 0; i0 < V; i0 += chunk) {
        const unsigned n = (V - i0 < chunk) ? V - i0 : chunk;
        const unsigned nthreads = n * per;
        const unsigned grid = (nthreads + 255) / 256;
        if (up) {
            CU(c, cudaMemcpyAsync(c->d_stage, (const char *)host_in + (size_t)i0 * per_site, (size_t)n * per_site,
                                  cudaMemcpyHostToDevice, c->stream));
            LaunchScope ls(c, QCD_K_MISC);
            if (matrix) matrix_scatter_kernel<C><<<grid, 256, 0, c->stream>>>(c->L, (const C *)c->d_stage, i0, n, (C *)f->ptr, nmu, nrow);
            else spinor_scatter_kernel<C><<<grid, 256, 0, c->stream>>>(c->L, (const C *)c->d_stage, i0, n, even, odd);
        } else {
            {
                LaunchScope ls(c, QCD_K_MISC);
                if (matrix) matrix_gather_kernel<C><<<grid, 256, 0, c->stream>>>(c->L, (C *)c->d_stage, i0, n, (const C *)f->ptr, nmu, nrow);
                else spinor_gather_kernel<C><<<grid, 256, 0, c->stream>>>(c->L, (C *)c->d_stage, i0, n, even, odd);
            }
            CU(c, cudaMemcpyAsync((char *)host_out + (size_t)i0 * per_site, c->d_stage, (size_t)n * per_site,
                                  cudaMemcpyDeviceToHost, c->stream));
        }
        CU(c, cudaGetLastError());
    }
    CU(c, cudaStreamSynchronize(c->stream));
    return QCD_OK;
}

extern "C" qcd_status qcd_field_upload(qcd_field *f, const void *host)
{
    if (!f) return QCD_EINVAL;
    if (!host) return fail(f->ctx, QCD_EINVAL, "qcd_field_upload: NULL host pointer");
    DEV(f->ctx, "qcd_field_upload");
    f->tg = 0;
    return f->ctx->prec == 64 ? transfer_t<double>(f->ctx, f, host, nullptr) : transfer_t<float>(f->ctx, f, host, nullptr);
}

extern "C" qcd_status qcd_field_download(const qcd_field *f, void *host)
{
    if (!f) return QCD_EINVAL;
    if (!host) return fail(f->ctx, QCD_EINVAL, "qcd_field_download: NULL host pointer");
    DEV(f->ctx, "qcd_field_download");
    return f->ctx->prec == 64 ? transfer_t<double>(f->ctx, f, nullptr, host) : transfer_t<float>(f->ctx, f, nullptr, host);
}

// ------------------------------------------------------------------------------------------
// Dslash launches
// ------------------------------------------------------------------------------------------
// Chunk width of the traversal (lattice.cuh traversal_site): the largest divisor W of N2 for which
// four slabs (three time slices of inputs in flight plus the outputs being written) of W rows of n
// vectors fit a fixed share of the L2.  One vector at 64^4 gives W = N2 (plain order).
enum { CHUNK_BUDGET_BYTES = 32 << 20 };
static int traversal_chunk(const qcd_ctx *c, int n)
{
    const int N2 = c->L.N2;
    if (c->chunk > 0) return c->chunk;
    const double row_bytes = (double)c->L.s2 * 6.0 * c->rsize * n;
    int W = N2;
    while (W > 1 && 4.0 * row_bytes * W > (double)CHUNK_BUDGET_BYTES) {
        int next = W - 1;
        while (next > 1 && N2 % next) --next;
        W = next;
    }
    return W;
}

// out[r](parity) = D in[r](1-parity), r < n; mode >= 1 adds the M epilogue with v[r] (parity of out)
static qcd_status dslash_launch(qcd_ctx *c, int mode, const qcd_field *U, int n, void *const *out, const void *const *in,
                                int parity, const void *const *v, double m, CgScalars *scal, int check_flag)
{
    DslashLaunch d;
    d.mode = mode; d.tg = U->tg; d.nrhs = n; d.variant = c->variant;
    d.L = c->L; d.L.W = traversal_chunk(c, n); d.parity = parity; d.U = U->ptr;
    for (int r = 0; r < MAXRHS; ++r) {
        d.in[r] = r < n ? in[r] : nullptr;
        d.out[r] = r < n ? out[r] : nullptr;
        d.v[r] = (r < n && v) ? v[r] : nullptr;
    }
    d.m2 = m * m; d.partials = c->d_partials; d.scal = scal; d.check_flag = check_flag; d.stream = c->stream;
    LaunchScope ls(c, mode == 0 ? QCD_K_DSLASH : QCD_K_DSLASH_EPI);
    cudaError_t e;
    if (c->prec == 64) e = gauge_nrow(U) == 3 ? launch_dslash_f64_r3(d) : launch_dslash_f64_r2(d);
    else e = gauge_nrow(U) == 3 ? launch_dslash_f32_r3(d) : launch_dslash_f32_r2(d);
    if (e != cudaSuccess) return fail(c, QCD_ECUDA, "dslash launch: %s", cudaGetErrorString(e));
    return QCD_OK;
}

static qcd_status dslash_one(qcd_ctx *c, int mode, const qcd_field *U, void *out, const void *in, int parity,
                             const void *v, double m, CgScalars *scal, int check_flag)
{
    return dslash_launch(c, mode, U, 1, &out, &in, parity, v ? &v : nullptr, m, scal, check_flag);
}

static qcd_status check_gauge(qcd_ctx *ctx, const qcd_field *U, const char *who)
{
    if (!U || U->ctx != ctx || !is_gauge_kind(U->kind))
        return fail(ctx, QCD_EINVAL, "%s: U must be a QCD_GAUGE or QCD_GAUGE_2ROW field of this context", who);
    return QCD_OK;
}

static qcd_status dslash_public(qcd_ctx *ctx, const qcd_field *U, int n, qcd_field *const *out, const qcd_field *const *in,
                                int out_parity, const char *who)
{
    if (!ctx) return QCD_EINVAL;
    DEV(ctx, who);
    qcd_status s = check_gauge(ctx, U, who);
    if (s) return s;
    if (n < 1 || n > MAXRHS) return fail(ctx, QCD_EINVAL, "%s: n must be 1 .. QCD_MAX_RHS", who);
    if (!out || !in) return fail(ctx, QCD_EINVAL, "%s: NULL field array", who);
    void *o[MAXRHS]; const void *i[MAXRHS];
    for (int r = 0; r < n; ++r) {
        if (!out[r] || !in[r] || out[r]->ctx != ctx || in[r]->ctx != ctx) return fail(ctx, QCD_EINVAL, "%s: fields must belong to this context", who);
        o[r] = half_ptr(out[r], out_parity);
        i[r] = half_ptr(in[r], 1 - out_parity);
        if (!o[r] || !i[r]) return fail(ctx, QCD_EINVAL, "%s: spinor parity / kind mismatch", who);
    }
    const size_t hb = half_spinor_bytes(ctx);
    for (int r = 0; r < n; ++r) {
        for (int q = 0; q < n; ++q) if (overlaps(o[r], hb, i[q], hb)) return fail(ctx, QCD_EINVAL, "%s: out must not alias in", who);
        for (int q = 0; q < r; ++q) if (overlaps(o[q], hb, o[r], hb)) return fail(ctx, QCD_EINVAL, "%s: two outputs alias", who);
    }
    return dslash_launch(ctx, 0, U, n, o, i, out_parity, nullptr, 0.0, ctx->d_aux, 0);
}

extern "C" qcd_status qcd_dslash_eo(qcd_ctx *ctx, const qcd_field *U, qcd_field *out_even, const qcd_field *in_odd)
{
    return dslash_public(ctx, U, 1, &out_even, &in_odd, 0, "qcd_dslash_eo");
}

extern "C" qcd_status qcd_dslash_oe(qcd_ctx *ctx, const qcd_field *U, qcd_field *out_odd, const qcd_field *in_even)
{
    return dslash_public(ctx, U, 1, &out_odd, &in_even, 1, "qcd_dslash_oe");
}

extern "C" qcd_status qcd_dslash_eo_multi(qcd_ctx *ctx, const qcd_field *U, int n, qcd_field *const *out_even, const qcd_field *const *in_odd)
{
    return dslash_public(ctx, U, n, out_even, in_odd, 0, "qcd_dslash_eo_multi");
}

extern "C" qcd_status qcd_dslash_oe_multi(qcd_ctx *ctx, const qcd_field *U, int n, qcd_field *const *out_odd, const qcd_field *const *in_even)
{
    return dslash_public(ctx, U, n, out_odd, in_even, 1, "qcd_dslash_oe_multi");
}

// workspace carving for n right-hand sides: r[n], p[n], Ap[n] (even half-fields) then t[n] (odd)
static void *ws_at(qcd_ctx *c, int block, int n, int rhs) { return (char *)c->ws + ((size_t)block * n + rhs) * half_spinor_bytes(c); }
static void *ws_r(qcd_ctx *c, int n = 1, int rhs = 0) { return ws_at(c, 0, n, rhs); }
static void *ws_p(qcd_ctx *c, int n = 1, int rhs = 0) { return ws_at(c, 1, n, rhs); }
static void *ws_Ap(qcd_ctx *c, int n = 1, int rhs = 0) { return ws_at(c, 2, n, rhs); }
static void *ws_t(qcd_ctx *c, int n = 1, int rhs = 0) { return ws_at(c, 3, n, rhs); }

// out = m^2 in - D_eo D_oe in on raw even half-field pointers (workspace t is the intermediate)
static qcd_status apply_M_raw(qcd_ctx *ctx, const qcd_field *U, void *out, const void *in, double m)
{
    qcd_status s = dslash_one(ctx, 0, U, ws_t(ctx), in, 1, nullptr, 0.0, ctx->d_aux, 0);      // t = D_oe in
    if (s) return s;
    return dslash_one(ctx, 1, U, out, ws_t(ctx), 0, in, m, ctx->d_aux, 0);                    // out = m^2 in - D_eo t
}

extern "C" qcd_status qcd_apply_M(qcd_ctx *ctx, const qcd_field *U, qcd_field *out_even, const qcd_field *in_even, double m)
{
    if (!ctx) return QCD_EINVAL;
    DEV(ctx, "qcd_apply_M");
    qcd_status s = check_gauge(ctx, U, "qcd_apply_M");
    if (s) return s;
    if (!(m >= 0.0)) return fail(ctx, QCD_EINVAL, "qcd_apply_M: m must be >= 0");
    if (!ctx->ws) return fail(ctx, QCD_EINVAL, "qcd_apply_M: no workspace bound (qcd_set_workspace)");
    if (ctx->cg.active) return fail(ctx, QCD_EINVAL, "qcd_apply_M: a CG solve is using the workspace");
    if (!out_even || !in_even || out_even->ctx != ctx || in_even->ctx != ctx) return fail(ctx, QCD_EINVAL, "qcd_apply_M: bad fields");
    void *o = half_ptr(out_even, 0);
    const void *i = half_ptr(in_even, 0);
    if (!o || !i) return fail(ctx, QCD_EINVAL, "qcd_apply_M: both spinors must hold even sites");
    const size_t hb = half_spinor_bytes(ctx);
    if (overlaps(o, hb, i, hb)) return fail(ctx, QCD_EINVAL, "qcd_apply_M: out must not alias in");
    if (overlaps(o, hb, ctx->ws, ctx->ws_bytes) || overlaps(i, hb, ctx->ws, ctx->ws_bytes))
        return fail(ctx, QCD_EINVAL, "qcd_apply_M: out and in must not lie inside the bound workspace");
    return apply_M_raw(ctx, U, o, i, m);
}

// ------------------------------------------------------------------------------------------
// reductions
// ------------------------------------------------------------------------------------------
extern "C" qcd_status qcd_re_dot(qcd_ctx *ctx, const qcd_field *a, const qcd_field *b, double *result)
{
    if (!ctx) return QCD_EINVAL;
    if (!a || !b || !result || a->ctx != ctx || b->ctx != ctx || a->kind != b->kind ||
        (a->kind != QCD_SPINOR_EVEN && a->kind != QCD_SPINOR_ODD))
        return fail(ctx, QCD_EINVAL, "qcd_re_dot: need two half-fields of the same kind");
    DEV(ctx, "qcd_re_dot");
    {
        LaunchScope ls(ctx, QCD_K_MISC);
        if (ctx->prec == 64)
            re_dot_kernel<double><<<blas_grid(ctx), BLAS_BLOCK, 0, ctx->stream>>>(blas_n16(ctx), (const double2 *)a->ptr, (const double2 *)b->ptr, ctx->d_partials, ctx->d_aux);
        else
            re_dot_kernel<float><<<blas_grid(ctx), BLAS_BLOCK, 0, ctx->stream>>>(blas_n16(ctx), (const float4 *)a->ptr, (const float4 *)b->ptr, ctx->d_partials, ctx->d_aux);
    }
    CU(ctx, cudaGetLastError());
    CU(ctx, cudaMemcpyAsync(&ctx->h_scal[0], ctx->d_aux, sizeof(CgScalars), cudaMemcpyDeviceToHost, ctx->stream));
    CU(ctx, cudaStreamSynchronize(ctx->stream));
    *result = ctx->h_scal[0].dot;
    return QCD_OK;
}

// Read-only streaming ceiling over a field's own bytes (measure_kernels.cuh): the denominator of
// the Dslash roofline beside the copy peak and the theoretical peak.
extern "C" qcd_status qcd_stream_read(qcd_ctx *ctx, const qcd_field *f, int reps, double *ms_per_pass)
{
    if (!ctx) return QCD_EINVAL;
    if (!f || f->ctx != ctx || reps < 1 || !ms_per_pass) return fail(ctx, QCD_EINVAL, "qcd_stream_read: need a field of this context, reps >= 1 and a result pointer");
    DEV(ctx, "qcd_stream_read");
    const size_t n16 = qcd_field_bytes(ctx, f->kind) / 16;
    const size_t per = (size_t)STREAM_BLOCK * STREAM_LOADS;
    const size_t grid = (n16 + per - 1) / per;
    if (grid > 0x7fffffffULL) return fail(ctx, QCD_EINVAL, "qcd_stream_read: field too large for one launch");
    cudaEvent_t e0, e1;
    CU(ctx, cudaEventCreate(&e0));
    CU(ctx, cudaEventCreate(&e1));
    cudaError_t err = cudaEventRecord(e0, ctx->stream);
    for (int r = 0; r < reps && err == cudaSuccess; ++r) {
        LaunchScope ls(ctx, QCD_K_MISC);
        stream_read_kernel<<<(unsigned)grid, STREAM_BLOCK, 0, ctx->stream>>>((const double2 *)f->ptr, n16, (double2 *)ctx->d_stage);
        err = cudaGetLastError();
    }
    if (err == cudaSuccess) err = cudaEventRecord(e1, ctx->stream);
    if (err == cudaSuccess) err = cudaEventSynchronize(e1);
    float ms = 0.f;
    if (err == cudaSuccess) err = cudaEventElapsedTime(&ms, e0, e1);
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    if (err != cudaSuccess) return fail(ctx, QCD_ECUDA, "qcd_stream_read: %s", cudaGetErrorString(err));
    *ms_per_pass = (double)ms / reps;
    return QCD_OK;
}

// L2-resident variant: `passes` passes over the field inside ONE launch (measure_kernels.cuh).
extern "C" qcd_status qcd_stream_read_resident(qcd_ctx *ctx, const qcd_field *f, int passes, double *ms_per_pass)
{
    if (!ctx) return QCD_EINVAL;
    if (!f || f->ctx != ctx || passes < 1 || !ms_per_pass) return fail(ctx, QCD_EINVAL, "qcd_stream_read_resident: need a field of this context, passes >= 1 and a result pointer");
    DEV(ctx, "qcd_stream_read_resident");
    const size_t n16 = qcd_field_bytes(ctx, f->kind) / 16;
    const size_t per = (size_t)STREAM_BLOCK * STREAM_LOADS;
    int sms = 0;
    CU(ctx, cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, ctx->dev));
    size_t grid = (n16 + per - 1) / per;
    if (grid > (size_t)sms * 8) grid = (size_t)sms * 8;          // 8 resident blocks of 256 threads per SM
    cudaEvent_t e0, e1;
    CU(ctx, cudaEventCreate(&e0));
    CU(ctx, cudaEventCreate(&e1));
    cudaError_t err = cudaSuccess;
    {
        LaunchScope ls(ctx, QCD_K_MISC);                          // warm-up: brings the field into the L2
        stream_read_resident_kernel<<<(unsigned)grid, STREAM_BLOCK, 0, ctx->stream>>>((const double2 *)f->ptr, n16, 2, (double2 *)ctx->d_stage);
    }
    err = cudaEventRecord(e0, ctx->stream);
    {
        LaunchScope ls(ctx, QCD_K_MISC);
        stream_read_resident_kernel<<<(unsigned)grid, STREAM_BLOCK, 0, ctx->stream>>>((const double2 *)f->ptr, n16, passes, (double2 *)ctx->d_stage);
    }
    if (err == cudaSuccess) err = cudaGetLastError();
    if (err == cudaSuccess) err = cudaEventRecord(e1, ctx->stream);
    if (err == cudaSuccess) err = cudaEventSynchronize(e1);
    float ms = 0.f;
    if (err == cudaSuccess) err = cudaEventElapsedTime(&ms, e0, e1);
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    if (err != cudaSuccess) return fail(ctx, QCD_ECUDA, "qcd_stream_read_resident: %s", cudaGetErrorString(err));
    *ms_per_pass = (double)ms / passes;
    return QCD_OK;
}

// Streaming ceiling of a mix of read and write streams (measure_kernels.cuh).
extern "C" qcd_status qcd_stream_mix(qcd_ctx *ctx, const qcd_field *src, qcd_field *dst, int read_planes, int write_planes,
                                     int reps, double *ms_per_pass)
{
    if (!ctx) return QCD_EINVAL;
    if (!src || !dst || src->ctx != ctx || dst->ctx != ctx || reps < 1 || !ms_per_pass || read_planes < 0 || write_planes < 0 ||
        read_planes + write_planes == 0)
        return fail(ctx, QCD_EINVAL, "qcd_stream_mix: need two fields of this context, reps >= 1, plane counts >= 0 and a result pointer");
    DEV(ctx, "qcd_stream_mix");
    const size_t plane = (size_t)ctx->L.Vh * 2 * ctx->rsize / 16;            // 16-byte elements per plane of Vh complex numbers
    if ((size_t)read_planes * plane * 16 > qcd_field_bytes(ctx, src->kind) || (size_t)write_planes * plane * 16 > qcd_field_bytes(ctx, dst->kind))
        return fail(ctx, QCD_EINVAL, "qcd_stream_mix: more planes than the field holds");
    if (overlaps(src->ptr, qcd_field_bytes(ctx, src->kind), dst->ptr, qcd_field_bytes(ctx, dst->kind)))
        return fail(ctx, QCD_EINVAL, "qcd_stream_mix: src and dst overlap");
    if (plane == 0) return fail(ctx, QCD_EINVAL, "qcd_stream_mix: lattice too small");
    const size_t grid = (plane + MIX_BLOCK - 1) / MIX_BLOCK;
    cudaEvent_t e0, e1;
    CU(ctx, cudaEventCreate(&e0));
    CU(ctx, cudaEventCreate(&e1));
    cudaError_t err = cudaEventRecord(e0, ctx->stream);
    for (int r = 0; r < reps && err == cudaSuccess; ++r) {
        LaunchScope ls(ctx, QCD_K_MISC);
        stream_mix_kernel<<<(unsigned)grid, MIX_BLOCK, 0, ctx->stream>>>((const double2 *)src->ptr, (double2 *)dst->ptr, plane, read_planes, write_planes);
        err = cudaGetLastError();
    }
    if (err == cudaSuccess) err = cudaEventRecord(e1, ctx->stream);
    if (err == cudaSuccess) err = cudaEventSynchronize(e1);
    float ms = 0.f;
    if (err == cudaSuccess) err = cudaEventElapsedTime(&ms, e0, e1);
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    if (err != cudaSuccess) return fail(ctx, QCD_ECUDA, "qcd_stream_mix: %s", cudaGetErrorString(err));
    *ms_per_pass = (double)ms / reps;
    return QCD_OK;
}

// Streaming ceiling of the bulk-copy (TMA) path (measure_kernels.cuh).
extern "C" qcd_status qcd_stream_bulk(qcd_ctx *ctx, const qcd_field *src, int rows, int copies, int hops, int stages, int producers,
                                      int reps, double *ms_per_pass)
{
    if (!ctx) return QCD_EINVAL;
    if (!src || src->ctx != ctx || !ms_per_pass || reps < 1 || rows < 1 || rows > 256 || copies < 1 || hops < 1 || stages < 2 || stages > BULK_MAX_STAGES ||
        producers < 1 || producers > BULK_MAX_PRODUCERS)
        return fail(ctx, QCD_EINVAL, "qcd_stream_bulk: need a field of this context, 1 <= rows <= 256, copies >= 1, hops >= 1, 2 <= stages <= 12, 1 <= producers <= 4, "
                                     "reps >= 1 and a result pointer");
    if (ctx->prec != 64) return fail(ctx, QCD_EINVAL, "qcd_stream_bulk: the hook reads 16-byte elements of a precision-64 context");
    DEV(ctx, "qcd_stream_bulk");
    const size_t plane = (size_t)ctx->L.Vh;                                  // complex doubles per plane
    const int nplanes = (int)(qcd_field_bytes(ctx, src->kind) / (plane * 16));
    if (plane % BULK_RUN || rows > nplanes) return fail(ctx, QCD_EINVAL, "qcd_stream_bulk: a plane must be a multiple of 128 sites and hold `rows` planes");
    const size_t smem = (size_t)stages * rows * copies * BULK_RUN * 16;
    int max_smem = 0, sms = 0;
    CU(ctx, cudaDeviceGetAttribute(&max_smem, cudaDevAttrMaxSharedMemoryPerBlockOptin, ctx->dev));
    CU(ctx, cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, ctx->dev));
    if (smem > (size_t)max_smem) return fail(ctx, QCD_EINVAL, "qcd_stream_bulk: stages x rows x copies x 2 KB exceeds the shared memory of a block");
    CUtensorMap map;
    CU(ctx, encode_plane_map(&map, true, src->ptr, plane * 2, nplanes, plane * 16, BULK_RUN * 2, rows));
    CU(ctx, cudaFuncSetAttribute(stream_bulk_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    const size_t ngroups = plane / BULK_RUN;
    const unsigned grid = (unsigned)(ngroups < (size_t)sms ? ngroups : (size_t)sms);
    cudaEvent_t e0, e1;
    CU(ctx, cudaEventCreate(&e0));
    CU(ctx, cudaEventCreate(&e1));
    cudaError_t err = cudaEventRecord(e0, ctx->stream);
    for (int r = 0; r < reps && err == cudaSuccess; ++r) {
        LaunchScope ls(ctx, QCD_K_MISC);
        stream_bulk_kernel<<<grid, BULK_CONSUMERS + 32 * producers, smem, ctx->stream>>>(map, nplanes, rows, copies, hops, stages, ngroups, (double2 *)ctx->d_stage);
        err = cudaGetLastError();
    }
    if (err == cudaSuccess) err = cudaEventRecord(e1, ctx->stream);
    if (err == cudaSuccess) err = cudaEventSynchronize(e1);
    float ms = 0.f;
    if (err == cudaSuccess) err = cudaEventElapsedTime(&ms, e0, e1);
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    if (err != cudaSuccess) return fail(ctx, QCD_ECUDA, "qcd_stream_bulk: %s", cudaGetErrorString(err));
    *ms_per_pass = (double)ms / reps;
    return QCD_OK;
}

// ------------------------------------------------------------------------------------------
// CG (n right-hand sides in lock step; qcd_cg_solve is n = 1)
// ------------------------------------------------------------------------------------------
template <typename T>
static RhsPtrs<typename Vec16<T>::type> rhs_ptrs(const qcd_ctx *c)
{
    typedef typename Vec16<T>::type V;
    RhsPtrs<V> p;
    for (int r = 0; r < MAXRHS; ++r) {
        p.x[r] = r < c->cg.n ? (V *)c->cg.x[r] : nullptr;
        p.b[r] = r < c->cg.n ? (const V *)c->cg.b[r] : nullptr;
    }
    return p;
}

template <typename T>
static qcd_status cg_begin_t(qcd_ctx *c)
{
    typedef typename Vec16<T>::type V;
    const int n = c->cg.n;
    LaunchScope ls(c, QCD_K_MISC);
    cg_init_kernel<T><<<dim3(blas_grid(c), n), BLAS_BLOCK, 0, c->stream>>>(
        blas_n16(c), rhs_ptrs<T>(c), (V *)ws_r(c, n), (V *)ws_p(c, n),
        c->cg.tol, c->cg.maxiter, c->d_partials, c->d_scal);
    CU(c, cudaGetLastError());
    return QCD_OK;
}

// One CG iteration:  t = D_oe p;  Ap = m^2 p - D_eo t, pAp, alpha;
// x += alpha p, r -= alpha Ap, rr', beta, stop test;  p = r + beta p.
template <typename T>
static qcd_status cg_iteration_t(qcd_ctx *c)
{
    typedef typename Vec16<T>::type V;
    const int n = c->cg.n;
    void *t[MAXRHS], *Ap[MAXRHS];
    const void *p[MAXRHS], *tc[MAXRHS];
    for (int r = 0; r < n; ++r) { t[r] = ws_t(c, n, r); Ap[r] = ws_Ap(c, n, r); p[r] = ws_p(c, n, r); tc[r] = t[r]; }
    qcd_status s = dslash_launch(c, 0, c->cg.U, n, t, p, 1, nullptr, 0.0, c->d_scal, 1);
    if (s) return s;
    s = dslash_launch(c, 2, c->cg.U, n, Ap, tc, 0, p, c->cg.m, c->d_scal, 1);
    if (s) return s;
    {
        LaunchScope ls(c, QCD_K_UPDATE_XR);
        const int chunks = (blas_grid(c) + BLAS_REDUCE_GRID - 1) / BLAS_REDUCE_GRID;          // >= 1
        cg_update_xr_kernel<T><<<dim3((blas_grid(c) + chunks - 1) / chunks, n), BLAS_BLOCK, 0, c->stream>>>(
            blas_n16(c), rhs_ptrs<T>(c), (V *)ws_r(c, n), (const V *)ws_p(c, n), (const V *)ws_Ap(c, n), c->d_partials, c->d_scal, chunks);
    }
    {
        LaunchScope ls(c, QCD_K_UPDATE_P);
        cg_update_p_kernel<T><<<dim3(blas_grid(c), n), BLAS_BLOCK, 0, c->stream>>>(blas_n16(c), (V *)ws_p(c, n), (const V *)ws_r(c, n), c->d_scal);
    }
    CU(c, cudaGetLastError());
    return QCD_OK;
}

extern "C" qcd_status qcd_cg_begin_multi(qcd_ctx *ctx, const qcd_field *U, int n, const qcd_field *const *b, qcd_field *const *x,
                                         double m, double tol, int maxiter)
{
    if (!ctx) return QCD_EINVAL;
    DEV(ctx, "qcd_cg_begin");
    qcd_status s = check_gauge(ctx, U, "qcd_cg_begin");
    if (s) return s;
    if (n < 1 || n > MAXRHS) return fail(ctx, QCD_EINVAL, "qcd_cg: n must be 1 .. QCD_MAX_RHS");
    if (!(m >= 0.0)) return fail(ctx, QCD_EINVAL, "qcd_cg: m must be >= 0");
    if (!(tol > 0.0)) return fail(ctx, QCD_EINVAL, "qcd_cg: tol must be > 0");
    if (maxiter < 0) return fail(ctx, QCD_EINVAL, "qcd_cg: maxiter must be >= 0");
    if (!b || !x) return fail(ctx, QCD_EINVAL, "qcd_cg: NULL field array");
    for (int r = 0; r < n; ++r) {
        if (!b[r] || !x[r] || b[r]->ctx != ctx || x[r]->ctx != ctx || b[r]->kind != QCD_SPINOR_EVEN || x[r]->kind != QCD_SPINOR_EVEN)
            return fail(ctx, QCD_EINVAL, "qcd_cg: b and x must be QCD_SPINOR_EVEN fields of this context");
    }
    if (!ctx->ws || ctx->ws_bytes < qcd_workspace_bytes_multi(ctx, n))
        return fail(ctx, QCD_EINVAL, "qcd_cg: workspace missing or smaller than qcd_workspace_bytes_multi (qcd_set_workspace)");
    // every x against every b (cg_init zeroes x[q] in one blockIdx.y slice while another reads b[r]), x against x,
    // and both against the workspace the solver writes
    const size_t hb = half_spinor_bytes(ctx);
    for (int r = 0; r < n; ++r) {
        for (int q = 0; q < n; ++q) if (overlaps(x[r]->ptr, hb, b[q]->ptr, hb)) return fail(ctx, QCD_EINVAL, "qcd_cg: x must not alias b");
        for (int q = 0; q < r; ++q) if (overlaps(x[q]->ptr, hb, x[r]->ptr, hb)) return fail(ctx, QCD_EINVAL, "qcd_cg: two solutions alias");
        if (overlaps(x[r]->ptr, hb, ctx->ws, ctx->ws_bytes) || overlaps(b[r]->ptr, hb, ctx->ws, ctx->ws_bytes))
            return fail(ctx, QCD_EINVAL, "qcd_cg: b and x must not lie inside the bound workspace");
    }
    if (ctx->cg.active) return fail(ctx, QCD_EINVAL, "qcd_cg_begin: a solve is already in progress");
    ctx->cg.U = U; ctx->cg.n = n; ctx->cg.m = m; ctx->cg.tol = tol; ctx->cg.maxiter = maxiter;
    for (int r = 0; r < n; ++r) { ctx->cg.b[r] = b[r]->ptr; ctx->cg.x[r] = x[r]->ptr; }
    CU(ctx, cudaEventRecord(ctx->cg.ev_begin, ctx->stream));
    s = ctx->prec == 64 ? cg_begin_t<double>(ctx) : cg_begin_t<float>(ctx);
    if (s) return s;
    ctx->cg.active = true;
    ctx->loop_used = 1;            // qcd_cg_iterate enqueues kernel by kernel; cg_run overrides it
    return QCD_OK;
}

extern "C" qcd_status qcd_cg_begin(qcd_ctx *ctx, const qcd_field *U, const qcd_field *b, qcd_field *x,
                                   double m, double tol, int maxiter)
{
    return qcd_cg_begin_multi(ctx, U, 1, &b, &x, m, tol, maxiter);
}

extern "C" qcd_status qcd_cg_iterate(qcd_ctx *ctx, int n)
{
    if (!ctx) return QCD_EINVAL;
    if (!ctx->cg.active) return fail(ctx, QCD_EINVAL, "qcd_cg_iterate: no solve in progress");
    DEV(ctx, "qcd_cg_iterate");
    if (n < 0) return fail(ctx, QCD_EINVAL, "qcd_cg_iterate: n must be >= 0");
    for (int i = 0; i < n; ++i) {
        qcd_status s = ctx->prec == 64 ? cg_iteration_t<double>(ctx) : cg_iteration_t<float>(ctx);
        if (s) return s;
    }
    return QCD_OK;
}

// copies the cg.n recurrence states to pinned slot 0 and returns a pointer to them
static qcd_status read_scalars(qcd_ctx *ctx, const CgScalars **out)
{
    CU(ctx, cudaMemcpyAsync(&ctx->h_scal[0], ctx->d_scal, ctx->cg.n * sizeof(CgScalars), cudaMemcpyDeviceToHost, ctx->stream));
    CU(ctx, cudaStreamSynchronize(ctx->stream));
    *out = &ctx->h_scal[0];
    return QCD_OK;
}

static double rel_resid_of(const CgScalars &s) { return s.bb > 0.0 ? sqrt(s.rr / s.bb) : 0.0; }

// state of a lock-step solve: running while any right-hand side runs, else the worst outcome
static int joint_state(const CgScalars *s, int n)
{
    int st = 1;
    for (int r = 0; r < n; ++r) {
        if (s[r].flag == 0) return 0;
        if (s[r].flag > st) st = s[r].flag;
    }
    return st;
}

extern "C" qcd_status qcd_cg_poll(qcd_ctx *ctx, int *state, int *iters, double *rel_resid)
{
    if (!ctx) return QCD_EINVAL;
    if (!ctx->cg.active) return fail(ctx, QCD_EINVAL, "qcd_cg_poll: no solve in progress");
    const CgScalars *s;
    qcd_status st = read_scalars(ctx, &s);
    if (st) return st;
    int k = 0; double rel = 0.0;
    for (int r = 0; r < ctx->cg.n; ++r) { if (s[r].k > k) k = s[r].k; if (rel_resid_of(s[r]) > rel) rel = rel_resid_of(s[r]); }
    if (state) *state = joint_state(s, ctx->cg.n);
    if (iters) *iters = k;
    if (rel_resid) *rel_resid = rel;
    return QCD_OK;
}

extern "C" qcd_status qcd_cg_finish_multi(qcd_ctx *ctx, qcd_cg_info *info)
{
    if (!ctx) return QCD_EINVAL;
    if (!ctx->cg.active) return fail(ctx, QCD_EINVAL, "qcd_cg_finish: no solve in progress");
    ctx->cg.active = false;
    ctx->last_n = ctx->cg.n;
    CU(ctx, cudaEventRecord(ctx->cg.ev_end, ctx->stream));
    const CgScalars *s;
    qcd_status st = read_scalars(ctx, &s);
    if (ctx->cg.graph) { cudaGraphExecDestroy(ctx->cg.graph); ctx->cg.graph = nullptr; }
    if (st) return st;
    float ms = 0.f;
    CU(ctx, cudaEventElapsedTime(&ms, ctx->cg.ev_begin, ctx->cg.ev_end));
    qcd_status res = QCD_OK;
    for (int r = 0; r < ctx->cg.n; ++r) {
        if (info) {
            info[r].iters = s[r].k; info[r].converged = s[r].flag == 1; info[r].rel_resid = rel_resid_of(s[r]);
            info[r].bnorm2 = s[r].bb; info[r].seconds = ms * 1e-3;
        }
        if (res == QCD_OK && s[r].flag != 1) res = s[r].flag == 3 ? QCD_EBREAKDOWN : QCD_ENOTCONVERGED;
    }
    if (res == QCD_EBREAKDOWN) return fail(ctx, res, "qcd_cg: breakdown (<p,Mp> <= 0 or NaN)");
    if (res == QCD_ENOTCONVERGED) return fail(ctx, res, "qcd_cg: not converged");
    return QCD_OK;
}

// Residual history of the most recent solve (recorded on the device by the kernel that advances the
// recurrence; no extra launch, no host round trip during the solve).
extern "C" qcd_status qcd_cg_history(qcd_ctx *ctx, int rhs, double *host_out, int cap, int *n)
{
    if (!ctx) return QCD_EINVAL;
    if (rhs < 0 || cap < 0 || (cap > 0 && !host_out) || !n) return fail(ctx, QCD_EINVAL, "qcd_cg_history: bad argument");
    if (rhs >= ctx->last_n) return fail(ctx, QCD_EINVAL, "qcd_cg_history: rhs must be below the number of right-hand sides of the most recent solve");
    DEV(ctx, "qcd_cg_history");
    if (ctx->cg.active) return fail(ctx, QCD_EINVAL, "qcd_cg_history: a solve is in progress (qcd_cg_finish first)");
    CgScalars s;
    CU(ctx, cudaMemcpyAsync(&ctx->h_scal[0], ctx->d_scal + rhs, sizeof(CgScalars), cudaMemcpyDeviceToHost, ctx->stream));
    CU(ctx, cudaStreamSynchronize(ctx->stream));
    s = ctx->h_scal[0];
    int m = s.k < HIST_CAP ? s.k : HIST_CAP;
    if (m > cap) m = cap;
    if (m > 0) {
        CU(ctx, cudaMemcpyAsync(host_out, ctx->d_hist + (size_t)rhs * HIST_CAP, (size_t)m * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
        CU(ctx, cudaStreamSynchronize(ctx->stream));
        for (int j = 0; j < m; ++j) host_out[j] /= s.bb;
    }
    *n = m;
    return QCD_OK;
}

extern "C" qcd_status qcd_cg_finish(qcd_ctx *ctx, qcd_cg_info *info)
{
    if (ctx && ctx->cg.active && ctx->cg.n != 1) return fail(ctx, QCD_EINVAL, "qcd_cg_finish: a multi solve is in progress (qcd_cg_finish_multi)");
    return qcd_cg_finish_multi(ctx, info);
}

// Lattices that fit the L2: the whole solve in ONE cooperative kernel (cg_persistent.cuh).
enum { PERSIST_MAX_BYTES = 96 << 20, CLUSTER_MAX_SITES = 2048 };

template <typename T, int NROW, int TG>
static qcd_status cg_persistent_launch(qcd_ctx *c, bool probe_only, bool *ok)
{
    typedef typename Cplx<T>::type C;
    PersistArgs<T> a;
    a.L = c->L; a.U = (const C *)c->cg.U->ptr;
    a.x = (C *)c->cg.x[0]; a.r = (C *)ws_r(c); a.p = (C *)ws_p(c); a.Ap = (C *)ws_Ap(c); a.t = (C *)ws_t(c);
    a.p2 = (C *)ws_at(c, 4, 1, 0);
    a.m2 = (T)(c->cg.m * c->cg.m); a.partials = c->d_partials; a.scal = c->d_scal;
    a.timeline = c->timeline_on ? c->d_timeline : nullptr;
    const int wanted_threads = c->L.Vh;                         // one thread per site (cg_persistent.cuh)

    // up to 2048 sites per parity: ONE thread-block cluster (hardware barrier, partial sums through DSMEM)
    enum { CLUSTER_BLOCK = ClusterBlock<T>::value };
    if (c->L.Vh <= CLUSTER_MAX_SITES && c->loop_cluster_ok) {
        auto kernel = cg_cluster_kernel<T, NROW, TG>;
        int ncta = 1;
        // sites per CTA: as many as the block has threads, but in fp64 at most 64 while CTAs are to be had -- the links of 64 sites for both
        // phases (147 KB) fit the L1 next to the vectors' shared memory, those of 128 (295 KB) do not and come from the L2 every iteration
        const int per_cta = sizeof(T) == 8 ? CLUSTER_BLOCK / 2 : CLUSTER_BLOCK;
        while (ncta * per_cta < wanted_threads && ncta < CLUSTER_MAX_CTAS) ncta *= 2;
        cudaLaunchConfig_t cfg;
        memset(&cfg, 0, sizeof cfg);
        cfg.gridDim = dim3(ncta); cfg.blockDim = dim3(CLUSTER_BLOCK); cfg.dynamicSmemBytes = 0; cfg.stream = c->stream;
        cudaLaunchAttribute attr[1];
        attr[0].id = cudaLaunchAttributeClusterDimension;
        attr[0].val.clusterDim.x = ncta; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
        cfg.attrs = attr; cfg.numAttrs = 1;
        cudaError_t e = cudaSuccess;
        if (ncta > 8) e = cudaFuncSetAttribute(kernel, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
        int nclusters = 0;
        if (e == cudaSuccess) e = cudaOccupancyMaxActiveClusters(&nclusters, kernel, &cfg);
        if (e == cudaSuccess && nclusters >= 1) {
            *ok = true;
            if (probe_only) return QCD_OK;
            if (c->timeline_on) CU(c, cudaMemsetAsync(c->d_timeline, 0, 2 * TIMELINE_ITERS * TIMELINE_STAMPS * sizeof(unsigned long long), c->stream));
            LaunchScope ls(c, QCD_K_MISC);
            CU(c, cudaLaunchKernelEx(&cfg, kernel, a));
            c->persist_cluster = ncta;
            return QCD_OK;
        }
        cudaGetLastError();                                     // no cluster of that size on this device: the grid version below
    }

    auto kernel = cg_persistent_kernel<T, NROW, TG>;
    enum { PERSIST_BLOCK = PersistBlock<T>::value };
    int per_sm = 0, sms = 0, coop = 0;
    CU(c, cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, c->dev));
    CU(c, cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, c->dev));
    CU(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kernel, PERSIST_BLOCK, 0));
    *ok = coop && per_sm > 0;
    if (probe_only || !*ok) return QCD_OK;
    // Every block owns an equally long range of sites (cg_persistent.cuh): launch k blocks on EVERY SM, k the smallest number
    // of co-resident blocks that covers the sites in one pass (16^4 fp64: 148 blocks of 256 threads, 222 sites each), capped by what is
    // co-resident (then a block walks its range in several trips); tiny lattices get one block per warp of work.
    int max_grid = per_sm * sms;
    if (max_grid * 2 > c->partials_cap) max_grid = c->partials_cap / 2;       // two buffers of per-block partials (solve_barrier)
    int k = (wanted_threads + sms * PERSIST_BLOCK - 1) / (sms * PERSIST_BLOCK);
    if (k > per_sm) k = per_sm;
    int grid = sms * k;
    const int by_work = (wanted_threads + 31) / 32;
    if (grid > by_work) grid = by_work;
    if (grid > max_grid) grid = max_grid;
    if (grid < 1) grid = 1;
    if (c->timeline_on) CU(c, cudaMemsetAsync(c->d_timeline, 0, 2 * TIMELINE_ITERS * TIMELINE_STAMPS * sizeof(unsigned long long), c->stream));
    void *params[] = { &a };
    LaunchScope ls(c, QCD_K_MISC);
    CU(c, cudaLaunchCooperativeKernel((const void *)kernel, dim3(grid), dim3(PERSIST_BLOCK), params, 0, c->stream));
    c->persist_cluster = 0;
    return QCD_OK;
}

static qcd_status cg_persistent(qcd_ctx *c, bool probe_only, bool *ok)
{
    const int nrow = gauge_nrow(c->cg.U), tg = c->cg.U->tg;
#define QCD_PERSIST(T)                                                                                  \
    (nrow == 3 ? (tg ? cg_persistent_launch<T, 3, 1>(c, probe_only, ok) : cg_persistent_launch<T, 3, 0>(c, probe_only, ok)) \
               : (tg ? cg_persistent_launch<T, 2, 1>(c, probe_only, ok) : cg_persistent_launch<T, 2, 0>(c, probe_only, ok)))
    return c->prec == 64 ? QCD_PERSIST(double) : QCD_PERSIST(float);
#undef QCD_PERSIST
}

// the persistent kernel serves one right-hand side whose links and work vectors fit the L2
static bool persistent_wanted(const qcd_ctx *c)
{
    if (c->cg.n != 1 || c->prof_on || c->loop == 1 || c->loop == 2) return false;
    if (c->loop == 3) return true;
    const size_t bytes = qcd_field_bytes(c, c->cg.U->kind) + 6 * half_spinor_bytes(c);
    return bytes <= (size_t)PERSIST_MAX_BYTES;
}

// Small lattices: an iteration is 4 kernels of a few microseconds each, so the host's launch rate,
// not the device, bounds the solve ("global reductions which have higher latencies ... more
// pronounced for smaller lattice sizes").  There the loop replays a CUDA graph of
// GRAPH_ITERS iterations (one launch per 4 * GRAPH_ITERS kernels).  The pointers of a solve are
// fixed and alpha, beta, the flags live on the device, so one capture serves the whole solve.
// Capture needs a non-default stream; on the legacy default stream, or while per-launch
// profiling is on, the plain loop below is used.
enum { GRAPH_ITERS = 16, GRAPH_MAX_VH = 1 << 21 };

static cudaGraphExec_t cg_capture_graph(qcd_ctx *ctx)
{
    if (ctx->loop == 1 || ctx->loop == 3) return nullptr;
    if ((ctx->L.Vh > GRAPH_MAX_VH && ctx->loop != 2) || ctx->prof_on || ctx->stream == nullptr || ctx->cg.maxiter < GRAPH_ITERS) return nullptr;
    if (cudaStreamBeginCapture(ctx->stream, cudaStreamCaptureModeThreadLocal) != cudaSuccess) { cudaGetLastError(); return nullptr; }
    const long long l0 = ctx->launches;
    const qcd_status s = qcd_cg_iterate(ctx, GRAPH_ITERS);
    ctx->launches = l0;
    cudaGraph_t graph = nullptr;
    cudaGraphExec_t exec = nullptr;
    const cudaError_t e = cudaStreamEndCapture(ctx->stream, &graph);
    if (s == QCD_OK && e == cudaSuccess && graph) {
        if (cudaGraphInstantiate(&exec, graph, 0) != cudaSuccess) exec = nullptr;
    }
    if (graph) cudaGraphDestroy(graph);
    cudaGetLastError();
    return exec;
}

// Host loop: keep two chunks of iterations in flight; after each chunk the scalars are copied
// to pinned memory and an event is recorded, and the host waits on the OLDER chunk's event
// only, so the device never idles while the host decides.  Iterations enqueued after the
// stop flag was set exit at their first instruction, so x is frozen at the exact iteration.
static qcd_status cg_run(qcd_ctx *ctx)
{
    const int maxiter = ctx->cg.maxiter, n = ctx->cg.n;
    // a FORCED loop that cannot run is an error, not a silent fall-back (the caller could not tell which loop a
    // test or a bench row exercised); what the automatic choice picked is reported by qcd_last_cg_loop
    if (ctx->loop == 2 && ctx->stream == nullptr)
        return fail(ctx, QCD_EINVAL, "qcd_cg: loop 2 (graph replay) needs a context stream other than the legacy default stream");
    if (ctx->loop == 3 && n != 1)
        return fail(ctx, QCD_EINVAL, "qcd_cg: loop 3 (persistent kernel) serves one right-hand side");
    if (persistent_wanted(ctx)) {
        bool ok = false;
        const qcd_status s = cg_persistent(ctx, false, &ok);
        if (!s && ok) ctx->loop_used = 3;
        if (s || ok) return s;              // launched (qcd_cg_finish synchronises and reads the scalars), or failed
        if (ctx->loop == 3) return fail(ctx, QCD_EINVAL, "qcd_cg: loop 3 (persistent kernel) cannot be launched cooperatively on this device");
    }
    int enq = 0, head = 0, tail = 0, pending = 0, chunk = 8;
    bool first = true;
    cudaGraphExec_t graph = cg_capture_graph(ctx);
    ctx->cg.graph = graph;
    ctx->loop_used = graph ? 2 : 1;
    if (graph) chunk = GRAPH_ITERS;
    qcd_status result = QCD_OK;
    for (;;) {
        while (pending < POLL_SLOTS && (enq < maxiter || first)) {
            int it = maxiter - enq < chunk ? maxiter - enq : chunk;
            if (graph) {
                // whole graphs only: iterations past maxiter are no-ops (flag 2 is set at k = maxiter)
                const int reps = (it + GRAPH_ITERS - 1) / GRAPH_ITERS;
                for (int g = 0; g < reps && result == QCD_OK; ++g) {
                    if (cudaGraphLaunch(graph, ctx->stream) != cudaSuccess) result = fail(ctx, QCD_ECUDA, "cudaGraphLaunch: %s", cudaGetErrorString(cudaGetLastError()));
                    ctx->launches += 4 * GRAPH_ITERS;
                }
                it = reps * GRAPH_ITERS;
            } else {
                result = qcd_cg_iterate(ctx, it);
            }
            if (result) break;
            enq += it;
            if (cudaMemcpyAsync(&ctx->h_scal[head * MAXRHS], ctx->d_scal, n * sizeof(CgScalars), cudaMemcpyDeviceToHost, ctx->stream) != cudaSuccess ||
                cudaEventRecord(ctx->poll_ev[head], ctx->stream) != cudaSuccess) {
                result = fail(ctx, QCD_ECUDA, "qcd_cg: poll copy: %s", cudaGetErrorString(cudaGetLastError()));
                break;
            }
            head = (head + 1) % POLL_SLOTS; ++pending; first = false;
            if (chunk < 64) chunk *= 2;
        }
        if (result) break;
        if (cudaEventSynchronize(ctx->poll_ev[tail]) != cudaSuccess) { result = fail(ctx, QCD_ECUDA, "qcd_cg: %s", cudaGetErrorString(cudaGetLastError())); break; }
        const int state = joint_state(&ctx->h_scal[tail * MAXRHS], n);
        tail = (tail + 1) % POLL_SLOTS; --pending;
        if (state != 0) break;
        if (pending == 0 && enq >= maxiter) break;   // defensive: flag 2 is set when k reaches maxiter
    }
    return result;
}

extern "C" qcd_status qcd_cg_solve_multi(qcd_ctx *ctx, const qcd_field *U, int n, const qcd_field *const *b, qcd_field *const *x,
                                         double m, double tol, int maxiter, qcd_cg_info *info)
{
    qcd_status s = qcd_cg_begin_multi(ctx, U, n, b, x, m, tol, maxiter);
    if (s) return s;
    s = cg_run(ctx);
    if (s) { const std::string keep = ctx->err; qcd_cg_finish_multi(ctx, nullptr); ctx->err = keep; return s; }
    return qcd_cg_finish_multi(ctx, info);
}

extern "C" qcd_status qcd_cg_solve(qcd_ctx *ctx, const qcd_field *U, const qcd_field *b, qcd_field *x,
                                   double m, double tol, int maxiter, qcd_cg_info *info)
{
    return qcd_cg_solve_multi(ctx, U, 1, &b, &x, m, tol, maxiter, info);
}

extern "C" qcd_status qcd_cg_solve_host(qcd_ctx *ctx, const qcd_field *U, qcd_field *b_dev, qcd_field *x_dev,
                                        const void *b_host, void *x_host,
                                        double m, double tol, int maxiter, qcd_cg_info *info)
{
    if (!ctx) return QCD_EINVAL;
    if (!b_host || !x_host || !b_dev || !x_dev) return fail(ctx, QCD_EINVAL, "qcd_cg_solve_host: NULL argument");
    cudaEvent_t e0, e1;
    CU(ctx, cudaEventCreate(&e0));
    CU(ctx, cudaEventCreate(&e1));
    cudaEventRecord(e0, ctx->stream);
    qcd_status s = qcd_field_upload(b_dev, b_host);
    qcd_status solve = QCD_OK;
    if (!s) {
        solve = qcd_cg_solve(ctx, U, b_dev, x_dev, m, tol, maxiter, info);
        if (solve == QCD_OK || solve == QCD_ENOTCONVERGED || solve == QCD_EBREAKDOWN) s = qcd_field_download(x_dev, x_host);
        else s = solve;
    }
    cudaEventRecord(e1, ctx->stream);
    cudaEventSynchronize(e1);
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    if (info) info->seconds = ms * 1e-3;
    return s ? s : solve;
}

// ------------------------------------------------------------------------------------------
// Variants: two-row links, temporal gauge, precision conversion
// ------------------------------------------------------------------------------------------
extern "C" qcd_status qcd_gauge_compress(qcd_ctx *ctx, const qcd_field *U, qcd_field *U12)
{
    if (!ctx) return QCD_EINVAL;
    if (!U || !U12 || U->ctx != ctx || U12->ctx != ctx || U->kind != QCD_GAUGE || U12->kind != QCD_GAUGE_2ROW)
        return fail(ctx, QCD_EINVAL, "qcd_gauge_compress: need a QCD_GAUGE source and a QCD_GAUGE_2ROW destination of this context");
    DEV(ctx, "qcd_gauge_compress");
    const size_t plane = (size_t)ctx->L.Vh * 2 * ctx->rsize;
    // rows 0 and 1 of link (parity, mu) are its first 6 planes: 8 contiguous 6-plane copies
    for (int pm = 0; pm < 8; ++pm)
        CU(ctx, cudaMemcpyAsync((char *)U12->ptr + (size_t)pm * 6 * plane, (const char *)U->ptr + (size_t)pm * 9 * plane,
                                6 * plane, cudaMemcpyDeviceToDevice, ctx->stream));
    U12->tg = U->tg;
    return QCD_OK;
}

extern "C" qcd_status qcd_gauge_set_temporal_unit(qcd_field *U, int on)
{
    if (!U) return QCD_EINVAL;
    if (!is_gauge_kind(U->kind)) return fail(U->ctx, QCD_EINVAL, "qcd_gauge_set_temporal_unit: not a gauge field");
    U->tg = on != 0;
    return QCD_OK;
}

template <typename T>
static void gauge_fix_t(qcd_ctx *c, const qcd_field *U, qcd_field *Uf, qcd_field *g)
{
    typedef typename Cplx<T>::type C;
    const int vs = c->L.N0 * c->L.N1 * c->L.N2;
    {
        LaunchScope ls(c, QCD_K_MISC);
        temporal_gauge_g_kernel<C><<<(vs + 127) / 128, 128, 0, c->stream>>>(c->L, (const C *)U->ptr, (C *)g->ptr);
    }
    for (int par = 0; par < 2; ++par) {
        LaunchScope ls(c, QCD_K_MISC);
        gauge_transform_kernel<C><<<(c->L.Vh + 127) / 128, 128, 0, c->stream>>>(c->L, par, (const C *)U->ptr, (const C *)g->ptr, (C *)Uf->ptr, 1);
    }
}

extern "C" qcd_status qcd_gauge_fix_temporal(qcd_ctx *ctx, const qcd_field *U, qcd_field *U_fixed, qcd_field *g)
{
    if (!ctx) return QCD_EINVAL;
    if (!U || !U_fixed || !g || U->ctx != ctx || U_fixed->ctx != ctx || g->ctx != ctx ||
        U->kind != QCD_GAUGE || U_fixed->kind != QCD_GAUGE || g->kind != QCD_COLOUR_MATRIX)
        return fail(ctx, QCD_EINVAL, "qcd_gauge_fix_temporal: need QCD_GAUGE U, QCD_GAUGE U_fixed and QCD_COLOUR_MATRIX g of this context");
    if (U->ptr == U_fixed->ptr) return fail(ctx, QCD_EINVAL, "qcd_gauge_fix_temporal: U_fixed must not alias U");
    DEV(ctx, "qcd_gauge_fix_temporal");
    if (ctx->prec == 64) gauge_fix_t<double>(ctx, U, U_fixed, g); else gauge_fix_t<float>(ctx, U, U_fixed, g);
    CU(ctx, cudaGetLastError());
    U_fixed->tg = 1;
    return QCD_OK;
}

extern "C" qcd_status qcd_spinor_rotate(qcd_ctx *ctx, const qcd_field *g, qcd_field *out, const qcd_field *in, int dagger)
{
    if (!ctx) return QCD_EINVAL;
    if (!g || !out || !in || g->ctx != ctx || out->ctx != ctx || in->ctx != ctx || g->kind != QCD_COLOUR_MATRIX ||
        !is_spinor_kind(in->kind) || out->kind != in->kind)
        return fail(ctx, QCD_EINVAL, "qcd_spinor_rotate: need a QCD_COLOUR_MATRIX g and two spinor fields of the same kind");
    DEV(ctx, "qcd_spinor_rotate");
    const int grid = (ctx->L.Vh + 127) / 128;
    for (int par = 0; par < 2; ++par) {
        void *o = half_ptr(out, par);
        const void *i = half_ptr(in, par);
        if (!o || !i) continue;
        LaunchScope ls(ctx, QCD_K_MISC);
        if (ctx->prec == 64)
            spinor_rotate_kernel<double2><<<grid, 128, 0, ctx->stream>>>(ctx->L, par, (const double2 *)g->ptr, (const double2 *)i, (double2 *)o, dagger != 0);
        else
            spinor_rotate_kernel<float2><<<grid, 128, 0, ctx->stream>>>(ctx->L, par, (const float2 *)g->ptr, (const float2 *)i, (float2 *)o, dagger != 0);
    }
    CU(ctx, cudaGetLastError());
    return QCD_OK;
}

extern "C" qcd_status qcd_field_convert(qcd_field *dst, const qcd_field *src)
{
    if (!dst || !src) return QCD_EINVAL;
    qcd_ctx *cd = dst->ctx, *cs = src->ctx;
    if (dst->kind != src->kind || cd->prec == cs->prec || memcmp(&cd->L, &cs->L, sizeof(Lattice)) != 0 || cd->stream != cs->stream)
        return fail(cd, QCD_EINVAL, "qcd_field_convert: need the same kind and lattice, different precisions, one stream");
    DEV(cd, "qcd_field_convert");
    const size_t n = qcd_field_bytes(cs, src->kind) / cs->rsize;
    const int grid = (int)((n + 255) / 256 < 148 * 16 ? (n + 255) / 256 : 148 * 16);
    {
        LaunchScope ls(cd, QCD_K_MISC);
        if (cs->prec == 64) convert_kernel<double, float><<<grid, 256, 0, cd->stream>>>(n, (const double *)src->ptr, (float *)dst->ptr);
        else convert_kernel<float, double><<<grid, 256, 0, cd->stream>>>(n, (const float *)src->ptr, (double *)dst->ptr);
    }
    CU(cd, cudaGetLastError());
    dst->tg = src->tg;
    return QCD_OK;
}

// ------------------------------------------------------------------------------------------
// Mixed-precision defect-correction CG (reading R21)
// ------------------------------------------------------------------------------------------
// r = b - Mx (Mx may be NULL: r = b), <r,r> -> host
static qcd_status mixed_residual(qcd_ctx *c, const void *b, const void *Mx, void *r, double *rr)
{
    {
        LaunchScope ls(c, QCD_K_MISC);
        mixed_residual_kernel<<<blas_grid(c), BLAS_BLOCK, 0, c->stream>>>(blas_n16(c), (const double2 *)b, (const double2 *)Mx, (double2 *)r, c->d_partials, c->d_aux);
    }
    CU(c, cudaGetLastError());
    CU(c, cudaMemcpyAsync(&c->h_scal[0], c->d_aux, sizeof(CgScalars), cudaMemcpyDeviceToHost, c->stream));
    CU(c, cudaStreamSynchronize(c->stream));
    *rr = c->h_scal[0].dot;
    return QCD_OK;
}

extern "C" qcd_status qcd_cg_solve_mixed(qcd_ctx *c64, qcd_ctx *c32, const qcd_field *U64, const qcd_field *U32,
                                         const qcd_field *b, qcd_field *x, qcd_field *rhs32, qcd_field *e32,
                                         double m, double tol, double inner_tol, int maxiter, int max_outer,
                                         qcd_mixed_info *info)
{
    if (!c64) return QCD_EINVAL;
    if (!c32 || c64->prec != 64 || c32->prec != 32 || memcmp(&c64->L, &c32->L, sizeof(Lattice)) != 0 || c64->stream != c32->stream)
        return fail(c64, QCD_EINVAL, "qcd_cg_solve_mixed: need a precision-64 and a precision-32 context on the same lattice and stream");
    qcd_status s = check_gauge(c64, U64, "qcd_cg_solve_mixed");
    if (s) return s;
    if (check_gauge(c32, U32, "qcd_cg_solve_mixed")) return fail(c64, QCD_EINVAL, "qcd_cg_solve_mixed: U32 must be a gauge field of ctx32");
    if (!b || !x || b->ctx != c64 || x->ctx != c64 || b->kind != QCD_SPINOR_EVEN || x->kind != QCD_SPINOR_EVEN || b->ptr == x->ptr)
        return fail(c64, QCD_EINVAL, "qcd_cg_solve_mixed: b and x must be distinct QCD_SPINOR_EVEN fields of ctx64");
    if (!rhs32 || !e32 || rhs32->ctx != c32 || e32->ctx != c32 || rhs32->kind != QCD_SPINOR_EVEN || e32->kind != QCD_SPINOR_EVEN || rhs32->ptr == e32->ptr)
        return fail(c64, QCD_EINVAL, "qcd_cg_solve_mixed: rhs32 and e32 must be distinct QCD_SPINOR_EVEN fields of ctx32");
    if (!(m >= 0.0) || !(tol > 0.0) || !(inner_tol > 0.0) || maxiter < 0 || max_outer < 0)
        return fail(c64, QCD_EINVAL, "qcd_cg_solve_mixed: need m >= 0, tol > 0, inner_tol > 0, maxiter >= 0, max_outer >= 0");
    if (!c64->ws || !c32->ws) return fail(c64, QCD_EINVAL, "qcd_cg_solve_mixed: both contexts need a workspace (qcd_set_workspace)");
    if (c64->cg.active || c32->cg.active) return fail(c64, QCD_EINVAL, "qcd_cg_solve_mixed: a CG solve is in progress");
    DEV(c64, "qcd_cg_solve_mixed");
    if (c32->dev != c64->dev) return fail(c64, QCD_EINVAL, "qcd_cg_solve_mixed: the two contexts live on different devices");

    cudaEvent_t e0, e1;
    CU(c64, cudaEventCreate(&e0));
    CU(c64, cudaEventCreate(&e1));
    cudaEventRecord(e0, c64->stream);

    qcd_mixed_info mi;
    memset(&mi, 0, sizeof mi);
    mi.true_resid = 1.0;
    qcd_status result = QCD_ENOTCONVERGED;
    const int ncplx = c64->L.Vh * 3;
    void *r = ws_r(c64), *Mx = ws_Ap(c64);
    double bb = 0.0, rr = 0.0;
    int budget = maxiter;

    CU(c64, cudaMemsetAsync(x->ptr, 0, half_spinor_bytes(c64), c64->stream));
    s = mixed_residual(c64, b->ptr, nullptr, r, &bb);                       // r = b, bb = <b,b>
    rr = bb;
    if (!s && bb == 0.0) { mi.converged = 1; mi.true_resid = 0.0; result = QCD_OK; }
    else if (!s && bb != bb) result = QCD_EBREAKDOWN;
    else while (!s) {
        const double rel = sqrt(rr / bb);
        mi.true_resid = rel;
        if (rel <= tol) { mi.converged = 1; result = QCD_OK; break; }
        if (rel != rel) { result = QCD_EBREAKDOWN; break; }
        if (mi.outer >= max_outer || budget <= 0) break;
        const double tol_in = inner_tol > 0.5 * tol / rel ? inner_tol : 0.5 * tol / rel;
        {
            LaunchScope ls(c64, QCD_K_MISC);                                  // rhs32 = fp32(r / |r|); d_aux->dot holds <r,r>
            mixed_restrict_kernel<<<(ncplx + 255) / 256, 256, 0, c64->stream>>>(ncplx, (const double2 *)r, (float2 *)rhs32->ptr, c64->d_aux);
        }
        qcd_cg_info ii;
        const qcd_status is = qcd_cg_solve(c32, U32, rhs32, e32, m, tol_in, budget, &ii);
        if (is != QCD_OK && is != QCD_ENOTCONVERGED) { s = is; if (is == QCD_EBREAKDOWN) { result = is; s = QCD_OK; } break; }
        budget -= ii.iters; mi.inner_iters += ii.iters; mi.outer += 1;
        {
            LaunchScope ls(c64, QCD_K_MISC);                                  // x += |r| fp64(e32)
            mixed_prolong_kernel<<<(ncplx + 255) / 256, 256, 0, c64->stream>>>(ncplx, (double2 *)x->ptr, (const float2 *)e32->ptr, c64->d_aux);
        }
        s = apply_M_raw(c64, U64, Mx, x->ptr, m);                           // r = b - M x in fp64
        if (s) break;
        mi.m_applications_fp64 += 1;
        s = mixed_residual(c64, b->ptr, Mx, r, &rr);
    }
    cudaEventRecord(e1, c64->stream);
    cudaEventSynchronize(e1);
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    mi.seconds = ms * 1e-3;
    if (info) *info = mi;
    if (s) { if (s != QCD_ECUDA || c64->err.empty()) fail(c64, s, "qcd_cg_solve_mixed: inner solve failed: %s", qcd_last_error(c32)); return s; }
    if (result == QCD_ENOTCONVERGED) return fail(c64, result, "qcd_cg_solve_mixed: not converged");
    if (result == QCD_EBREAKDOWN) return fail(c64, result, "qcd_cg_solve_mixed: breakdown");
    return QCD_OK;
}
