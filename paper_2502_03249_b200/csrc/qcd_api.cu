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
#include <string.h>

#include <new>
#include <string>

#include "cg_kernels.cuh"
#include "dslash.cuh"
#include "lattice.cuh"
#include "layout_kernels.cuh"
#include "reduce.cuh"

using namespace qcd;

// ------------------------------------------------------------------------------------------
// context
// ------------------------------------------------------------------------------------------
enum { PROF_MAX = 4096, STAGE_BYTES = 32 << 20, POLL_SLOTS = 2 };

struct qcd_field {
    qcd_ctx *ctx;
    int kind;
    void *ptr;
    size_t nbytes;
};

struct CgState {
    bool active;
    const qcd_field *U, *b;
    qcd_field *x;
    double m, tol;
    int maxiter;
    cudaEvent_t ev_begin, ev_end;
};

struct qcd_ctx {
    Lattice L;
    int prec;                 // 64 or 32
    size_t rsize;             // sizeof(real)
    cudaStream_t stream;
    CgScalars *d_scal;        // CG recurrence state
    CgScalars *d_aux;         // scratch state for qcd_apply_M / qcd_re_dot
    double *d_partials;       // stage-1 partial sums
    int partials_cap;
    CgScalars *h_scal;        // pinned, POLL_SLOTS entries
    cudaEvent_t poll_ev[POLL_SLOTS];
    void *d_stage;
    void *ws;
    size_t ws_bytes;
    CgState cg;
    int variant;
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
    default: return 0;
    }
}

extern "C" size_t qcd_workspace_bytes(const qcd_ctx *ctx) { return ctx ? 4 * half_spinor_bytes(ctx) : 0; }

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
    c->variant = 0; c->launches = 0;
    c->prof_on = false; c->prof_created = false; c->prof_n = c->prof_dropped = 0;
    c->ws = nullptr; c->ws_bytes = 0;
    memset(&c->cg, 0, sizeof c->cg);
    c->d_scal = c->d_aux = nullptr; c->d_partials = nullptr; c->h_scal = nullptr; c->d_stage = nullptr;
    for (int i = 0; i < POLL_SLOTS; ++i) c->poll_ev[i] = nullptr;

    c->partials_cap = dslash_grid_max(c) > blas_grid(c) ? dslash_grid_max(c) : blas_grid(c);
    cudaError_t err = cudaSuccess;
    if (err == cudaSuccess) err = cudaMalloc(&c->d_scal, 2 * sizeof(CgScalars));
    if (err == cudaSuccess) err = cudaMemset(c->d_scal, 0, 2 * sizeof(CgScalars));
    if (err == cudaSuccess) err = cudaMalloc(&c->d_partials, (size_t)c->partials_cap * sizeof(double));
    if (err == cudaSuccess) err = cudaMalloc(&c->d_stage, STAGE_BYTES);
    if (err == cudaSuccess) err = cudaMallocHost(&c->h_scal, POLL_SLOTS * sizeof(CgScalars));
    for (int i = 0; i < POLL_SLOTS && err == cudaSuccess; ++i) err = cudaEventCreateWithFlags(&c->poll_ev[i], cudaEventDisableTiming);
    if (err == cudaSuccess) err = cudaEventCreate(&c->cg.ev_begin);
    if (err == cudaSuccess) err = cudaEventCreate(&c->cg.ev_end);
    if (err != cudaSuccess) {
        fail(nullptr, err == cudaErrorMemoryAllocation ? QCD_ENOMEM : QCD_ECUDA, "qcd_init: %s", cudaGetErrorString(err));
        qcd_finalize(c);
        return err == cudaErrorMemoryAllocation ? QCD_ENOMEM : QCD_ECUDA;
    }
    c->d_aux = c->d_scal + 1;
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
    f->ctx = ctx; f->kind = kind; f->ptr = device_ptr; f->nbytes = nbytes;
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

extern "C" qcd_status qcd_set_dslash_variant(qcd_ctx *ctx, int variant)
{
    if (!ctx) return QCD_EINVAL;
    if (variant < 0 || variant > 3) return fail(ctx, QCD_EINVAL, "qcd_set_dslash_variant: unknown variant");
    ctx->variant = variant;
    return QCD_OK;
}

// ------------------------------------------------------------------------------------------
// upload / download
// ------------------------------------------------------------------------------------------
template <typename T>
static qcd_status transfer_t(qcd_ctx *c, const qcd_field *f, const void *host_in, void *host_out)
{
    typedef typename Cplx<T>::type C;
    const bool up = host_in != nullptr;
    const bool gauge = f->kind == QCD_GAUGE;
    const size_t per_site = (gauge ? 36 : 3) * sizeof(C);
    const unsigned V = 2u * (unsigned)c->L.Vh;
    unsigned chunk = (unsigned)(STAGE_BYTES / per_site);
    C *even = nullptr, *odd = nullptr;
    if (!gauge) { even = (C *)half_ptr(f, 0); odd = (C *)half_ptr(f, 1); }
    for (unsigned i0 = 0; i0 < V; i0 += chunk) {
        const unsigned n = (V - i0 < chunk) ? V - i0 : chunk;
        const unsigned nthreads = n * (gauge ? 36u : 3u);
        const unsigned grid = (nthreads + 255) / 256;
        if (up) {
            CU(c, cudaMemcpyAsync(c->d_stage, (const char *)host_in + (size_t)i0 * per_site, (size_t)n * per_site,
                                  cudaMemcpyHostToDevice, c->stream));
            LaunchScope ls(c, QCD_K_MISC);
            if (gauge) gauge_scatter_kernel<C><<<grid, 256, 0, c->stream>>>(c->L, (const C *)c->d_stage, i0, n, (C *)f->ptr);
            else spinor_scatter_kernel<C><<<grid, 256, 0, c->stream>>>(c->L, (const C *)c->d_stage, i0, n, even, odd);
        } else {
            {
                LaunchScope ls(c, QCD_K_MISC);
                if (gauge) gauge_gather_kernel<C><<<grid, 256, 0, c->stream>>>(c->L, (C *)c->d_stage, i0, n, (const C *)f->ptr);
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
    return f->ctx->prec == 64 ? transfer_t<double>(f->ctx, f, host, nullptr) : transfer_t<float>(f->ctx, f, host, nullptr);
}

extern "C" qcd_status qcd_field_download(const qcd_field *f, void *host)
{
    if (!f) return QCD_EINVAL;
    if (!host) return fail(f->ctx, QCD_EINVAL, "qcd_field_download: NULL host pointer");
    return f->ctx->prec == 64 ? transfer_t<double>(f->ctx, f, nullptr, host) : transfer_t<float>(f->ctx, f, nullptr, host);
}

// ------------------------------------------------------------------------------------------
// Dslash launches
// ------------------------------------------------------------------------------------------
template <typename T, int MODE, int BLOCK, int MINB>
static void launch_dslash_cfg(qcd_ctx *c, const DslashArgs<T> &a)
{
    const int grid = (c->L.Vh + BLOCK - 1) / BLOCK;
    dslash_kernel<T, MODE, BLOCK, MINB><<<grid, BLOCK, 0, c->stream>>>(a);
}

template <typename T, int MODE>
static void launch_dslash(qcd_ctx *c, const DslashArgs<T> &a)
{
    LaunchScope ls(c, MODE == 0 ? QCD_K_DSLASH : QCD_K_DSLASH_EPI);
    switch (c->variant) {
    default:
    case 0: launch_dslash_cfg<T, MODE, 128, 4>(c, a); break;
    case 1: launch_dslash_cfg<T, MODE, 64, 8>(c, a); break;
    case 2: launch_dslash_cfg<T, MODE, 256, 2>(c, a); break;
    case 3: launch_dslash_cfg<T, MODE, 128, 3>(c, a); break;
    }
}

// out(parity) = D in(1-parity); MODE >= 1 adds the M epilogue with v (same parity as out)
template <typename T, int MODE>
static qcd_status dslash_t(qcd_ctx *c, const void *U, void *out, const void *in, int parity, const void *v, double m,
                           CgScalars *scal, int check_flag)
{
    typedef typename Cplx<T>::type C;
    DslashArgs<T> a;
    a.L = c->L; a.parity = parity;
    a.U = (const C *)U; a.in = (const C *)in; a.out = (C *)out; a.v = (const C *)v;
    a.m2 = (T)(m * m);
    a.partials = c->d_partials; a.scal = scal; a.check_flag = check_flag;
    launch_dslash<T, MODE>(c, a);
    CU(c, cudaGetLastError());
    return QCD_OK;
}

static qcd_status dslash_dispatch(qcd_ctx *c, int mode, const void *U, void *out, const void *in, int parity,
                                  const void *v, double m, CgScalars *scal, int check_flag)
{
    if (c->prec == 64) {
        if (mode == 0) return dslash_t<double, 0>(c, U, out, in, parity, v, m, scal, check_flag);
        if (mode == 1) return dslash_t<double, 1>(c, U, out, in, parity, v, m, scal, check_flag);
        return dslash_t<double, 2>(c, U, out, in, parity, v, m, scal, check_flag);
    }
    if (mode == 0) return dslash_t<float, 0>(c, U, out, in, parity, v, m, scal, check_flag);
    if (mode == 1) return dslash_t<float, 1>(c, U, out, in, parity, v, m, scal, check_flag);
    return dslash_t<float, 2>(c, U, out, in, parity, v, m, scal, check_flag);
}

static qcd_status check_gauge(qcd_ctx *ctx, const qcd_field *U, const char *who)
{
    if (!U || U->ctx != ctx || U->kind != QCD_GAUGE) return fail(ctx, QCD_EINVAL, "%s: U must be a QCD_GAUGE field of this context", who);
    return QCD_OK;
}

static qcd_status dslash_public(qcd_ctx *ctx, const qcd_field *U, qcd_field *out, const qcd_field *in, int out_parity, const char *who)
{
    if (!ctx) return QCD_EINVAL;
    qcd_status s = check_gauge(ctx, U, who);
    if (s) return s;
    if (!out || !in || out->ctx != ctx || in->ctx != ctx) return fail(ctx, QCD_EINVAL, "%s: fields must belong to this context", who);
    void *o = half_ptr(out, out_parity);
    const void *i = half_ptr(in, 1 - out_parity);
    if (!o || !i) return fail(ctx, QCD_EINVAL, "%s: spinor parity / kind mismatch", who);
    if (o == i || out->ptr == in->ptr) return fail(ctx, QCD_EINVAL, "%s: out must not alias in", who);
    return dslash_dispatch(ctx, 0, U->ptr, o, i, out_parity, nullptr, 0.0, ctx->d_aux, 0);
}

extern "C" qcd_status qcd_dslash_eo(qcd_ctx *ctx, const qcd_field *U, qcd_field *out_even, const qcd_field *in_odd)
{
    return dslash_public(ctx, U, out_even, in_odd, 0, "qcd_dslash_eo");
}

extern "C" qcd_status qcd_dslash_oe(qcd_ctx *ctx, const qcd_field *U, qcd_field *out_odd, const qcd_field *in_even)
{
    return dslash_public(ctx, U, out_odd, in_even, 1, "qcd_dslash_oe");
}

// workspace carving: r, p, Ap (even half-fields) then t (odd half-field)
static void *ws_r(qcd_ctx *c) { return c->ws; }
static void *ws_p(qcd_ctx *c) { return (char *)c->ws + half_spinor_bytes(c); }
static void *ws_Ap(qcd_ctx *c) { return (char *)c->ws + 2 * half_spinor_bytes(c); }
static void *ws_t(qcd_ctx *c) { return (char *)c->ws + 3 * half_spinor_bytes(c); }

extern "C" qcd_status qcd_apply_M(qcd_ctx *ctx, const qcd_field *U, qcd_field *out_even, const qcd_field *in_even, double m)
{
    if (!ctx) return QCD_EINVAL;
    qcd_status s = check_gauge(ctx, U, "qcd_apply_M");
    if (s) return s;
    if (!(m >= 0.0)) return fail(ctx, QCD_EINVAL, "qcd_apply_M: m must be >= 0");
    if (!ctx->ws) return fail(ctx, QCD_EINVAL, "qcd_apply_M: no workspace bound (qcd_set_workspace)");
    if (ctx->cg.active) return fail(ctx, QCD_EINVAL, "qcd_apply_M: a CG solve is using the workspace");
    if (!out_even || !in_even || out_even->ctx != ctx || in_even->ctx != ctx) return fail(ctx, QCD_EINVAL, "qcd_apply_M: bad fields");
    void *o = half_ptr(out_even, 0);
    const void *i = half_ptr(in_even, 0);
    if (!o || !i) return fail(ctx, QCD_EINVAL, "qcd_apply_M: both spinors must hold even sites");
    if (o == i) return fail(ctx, QCD_EINVAL, "qcd_apply_M: out must not alias in");
    s = dslash_dispatch(ctx, 0, U->ptr, ws_t(ctx), i, 1, nullptr, 0.0, ctx->d_aux, 0);      // t = D_oe in
    if (s) return s;
    return dslash_dispatch(ctx, 1, U->ptr, o, ws_t(ctx), 0, i, m, ctx->d_aux, 0);           // out = m^2 in - D_eo t
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

// ------------------------------------------------------------------------------------------
// CG
// ------------------------------------------------------------------------------------------
template <typename T>
static qcd_status cg_begin_t(qcd_ctx *c)
{
    typedef typename Vec16<T>::type V;
    LaunchScope ls(c, QCD_K_MISC);
    cg_init_kernel<T><<<blas_grid(c), BLAS_BLOCK, 0, c->stream>>>(
        blas_n16(c), (const V *)c->cg.b->ptr, (V *)c->cg.x->ptr, (V *)ws_r(c), (V *)ws_p(c),
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
    qcd_status s = dslash_t<T, 0>(c, c->cg.U->ptr, ws_t(c), ws_p(c), 1, nullptr, 0.0, c->d_scal, 1);
    if (s) return s;
    s = dslash_t<T, 2>(c, c->cg.U->ptr, ws_Ap(c), ws_t(c), 0, ws_p(c), c->cg.m, c->d_scal, 1);
    if (s) return s;
    {
        LaunchScope ls(c, QCD_K_UPDATE_XR);
        cg_update_xr_kernel<T><<<blas_grid(c), BLAS_BLOCK, 0, c->stream>>>(
            blas_n16(c), (V *)c->cg.x->ptr, (V *)ws_r(c), (const V *)ws_p(c), (const V *)ws_Ap(c), c->d_partials, c->d_scal);
    }
    {
        LaunchScope ls(c, QCD_K_UPDATE_P);
        cg_update_p_kernel<T><<<blas_grid(c), BLAS_BLOCK, 0, c->stream>>>(blas_n16(c), (V *)ws_p(c), (const V *)ws_r(c), c->d_scal);
    }
    CU(c, cudaGetLastError());
    return QCD_OK;
}

extern "C" qcd_status qcd_cg_begin(qcd_ctx *ctx, const qcd_field *U, const qcd_field *b, qcd_field *x,
                                   double m, double tol, int maxiter)
{
    if (!ctx) return QCD_EINVAL;
    qcd_status s = check_gauge(ctx, U, "qcd_cg_begin");
    if (s) return s;
    if (!(m >= 0.0)) return fail(ctx, QCD_EINVAL, "qcd_cg: m must be >= 0");
    if (!(tol > 0.0)) return fail(ctx, QCD_EINVAL, "qcd_cg: tol must be > 0");
    if (maxiter < 0) return fail(ctx, QCD_EINVAL, "qcd_cg: maxiter must be >= 0");
    if (!b || !x || b->ctx != ctx || x->ctx != ctx || b->kind != QCD_SPINOR_EVEN || x->kind != QCD_SPINOR_EVEN)
        return fail(ctx, QCD_EINVAL, "qcd_cg: b and x must be QCD_SPINOR_EVEN fields of this context");
    if (b->ptr == x->ptr) return fail(ctx, QCD_EINVAL, "qcd_cg: x must not alias b");
    if (!ctx->ws) return fail(ctx, QCD_EINVAL, "qcd_cg: no workspace bound (qcd_set_workspace)");
    if (ctx->cg.active) return fail(ctx, QCD_EINVAL, "qcd_cg_begin: a solve is already in progress");
    ctx->cg.U = U; ctx->cg.b = b; ctx->cg.x = x; ctx->cg.m = m; ctx->cg.tol = tol; ctx->cg.maxiter = maxiter;
    CU(ctx, cudaEventRecord(ctx->cg.ev_begin, ctx->stream));
    s = ctx->prec == 64 ? cg_begin_t<double>(ctx) : cg_begin_t<float>(ctx);
    if (s) return s;
    ctx->cg.active = true;
    return QCD_OK;
}

extern "C" qcd_status qcd_cg_iterate(qcd_ctx *ctx, int n)
{
    if (!ctx) return QCD_EINVAL;
    if (!ctx->cg.active) return fail(ctx, QCD_EINVAL, "qcd_cg_iterate: no solve in progress");
    if (n < 0) return fail(ctx, QCD_EINVAL, "qcd_cg_iterate: n must be >= 0");
    for (int i = 0; i < n; ++i) {
        qcd_status s = ctx->prec == 64 ? cg_iteration_t<double>(ctx) : cg_iteration_t<float>(ctx);
        if (s) return s;
    }
    return QCD_OK;
}

static qcd_status read_scalars(qcd_ctx *ctx, CgScalars *out)
{
    CU(ctx, cudaMemcpyAsync(&ctx->h_scal[0], ctx->d_scal, sizeof(CgScalars), cudaMemcpyDeviceToHost, ctx->stream));
    CU(ctx, cudaStreamSynchronize(ctx->stream));
    *out = ctx->h_scal[0];
    return QCD_OK;
}

static double rel_resid_of(const CgScalars &s) { return s.bb > 0.0 ? sqrt(s.rr / s.bb) : 0.0; }

extern "C" qcd_status qcd_cg_poll(qcd_ctx *ctx, int *state, int *iters, double *rel_resid)
{
    if (!ctx) return QCD_EINVAL;
    if (!ctx->cg.active) return fail(ctx, QCD_EINVAL, "qcd_cg_poll: no solve in progress");
    CgScalars s;
    qcd_status st = read_scalars(ctx, &s);
    if (st) return st;
    if (state) *state = s.flag;
    if (iters) *iters = s.k;
    if (rel_resid) *rel_resid = rel_resid_of(s);
    return QCD_OK;
}

extern "C" qcd_status qcd_cg_finish(qcd_ctx *ctx, qcd_cg_info *info)
{
    if (!ctx) return QCD_EINVAL;
    if (!ctx->cg.active) return fail(ctx, QCD_EINVAL, "qcd_cg_finish: no solve in progress");
    ctx->cg.active = false;
    CU(ctx, cudaEventRecord(ctx->cg.ev_end, ctx->stream));
    CgScalars s;
    qcd_status st = read_scalars(ctx, &s);
    if (st) return st;
    float ms = 0.f;
    CU(ctx, cudaEventElapsedTime(&ms, ctx->cg.ev_begin, ctx->cg.ev_end));
    if (info) {
        info->iters = s.k; info->converged = s.flag == 1; info->rel_resid = rel_resid_of(s);
        info->bnorm2 = s.bb; info->seconds = ms * 1e-3;
    }
    if (s.flag == 1) return QCD_OK;
    if (s.flag == 3) return fail(ctx, QCD_EBREAKDOWN, "qcd_cg: breakdown (<p,Mp> <= 0 or NaN)");
    return fail(ctx, QCD_ENOTCONVERGED, "qcd_cg: not converged");
}

// Host loop: keep two chunks of iterations in flight; after each chunk the scalars are copied
// to pinned memory and an event is recorded, and the host waits on the OLDER chunk's event
// only, so the device never idles while the host decides.  Iterations enqueued after the
// stop flag was set exit at their first instruction, so x is frozen at the exact iteration.
static qcd_status cg_run(qcd_ctx *ctx)
{
    const int maxiter = ctx->cg.maxiter;
    int enq = 0, head = 0, tail = 0, pending = 0, chunk = 8;
    bool first = true;
    for (;;) {
        while (pending < POLL_SLOTS && (enq < maxiter || first)) {
            const int n = maxiter - enq < chunk ? maxiter - enq : chunk;
            qcd_status s = qcd_cg_iterate(ctx, n);
            if (s) return s;
            enq += n;
            CU(ctx, cudaMemcpyAsync(&ctx->h_scal[head], ctx->d_scal, sizeof(CgScalars), cudaMemcpyDeviceToHost, ctx->stream));
            CU(ctx, cudaEventRecord(ctx->poll_ev[head], ctx->stream));
            head = (head + 1) % POLL_SLOTS; ++pending; first = false;
            if (chunk < 64) chunk *= 2;
        }
        CU(ctx, cudaEventSynchronize(ctx->poll_ev[tail]));
        const int flag = ctx->h_scal[tail].flag;
        tail = (tail + 1) % POLL_SLOTS; --pending;
        if (flag != 0) break;
        if (pending == 0 && enq >= maxiter) break;   // defensive: flag 2 is set when k reaches maxiter
    }
    return QCD_OK;
}

extern "C" qcd_status qcd_cg_solve(qcd_ctx *ctx, const qcd_field *U, const qcd_field *b, qcd_field *x,
                                   double m, double tol, int maxiter, qcd_cg_info *info)
{
    qcd_status s = qcd_cg_begin(ctx, U, b, x, m, tol, maxiter);
    if (s) return s;
    s = cg_run(ctx);
    if (s) { ctx->cg.active = false; return s; }
    return qcd_cg_finish(ctx, info);
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
