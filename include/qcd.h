/*
 * qcd.h -- C ABI of the B200-native staggered Dslash / CG library (libqcd_b200.so).
 *
 * What it computes (arxiv 2502.03249, "Portable Lattice QCD implementation based on
 * OpenCL"; citations are PAPER.md line numbers of the extracted text):
 *
 *   Eq. (1), Sec. 4.2, the staggered Dirac hopping operator
 *       (D phi)(x) = sum_{mu=0..3} [ eta_mu(x) U_{x,mu} phi(x+mu)
 *                                    - eta_mu(x-mu) U^dagger_{x-mu,mu} phi(x-mu) ]
 *   restricted to its parity blocks D_eo (odd -> even) and D_oe (even -> odd), the
 *   even-odd preconditioned normal operator  M = m^2 - D_eo D_oe  on even sites
 *   (BASELINE.json north_star), and Conjugate Gradient on M x = b ("the inversion of
 *   the Dirac operator ... the most time critical part").
 *
 * Conventions: no factor 1/2; mu = 3 is time;
 * eta_mu(x) = (-1)^{x_0+...+x_{mu-1}}; periodic in mu = 0,1,2, antiperiodic in mu = 3
 * (a hop across the seam x3 = N3-1 <-> 0 carries -1); links are stored as full 3x3
 * complex matrices (18 reals), never modified by the library.
 *
 * DEVICE LAYOUT ("Structure of Arrays ... all even sites are listed
 * first, followed by all odd sites").  Lattice extents dims = (N0,N1,N2,N3), all even,
 * N0 % 4 == 0.  V = N0 N1 N2 N3, Vh = V/2.  Lexicographic index
 *       idx(x) = x0 + N0 (x1 + N1 (x2 + N2 x3)),   parity p(x) = (x0+x1+x2+x3) & 1,
 * checkerboard index cb = idx >> 1 (a bijection inside one parity).  "cplx" is
 * (re, im) of the context's real type (double for precision 64, float for 32).
 *   spinor half-field  : cplx [colour = 3][Vh]                        (3 planes)
 *   spinor full field  : even half-field followed by odd half-field   (6 planes)
 *   gauge field        : cplx [parity = 2][mu = 4][k = 3*row + col][Vh] (72 planes),
 *                        plane (p, mu, k) holds (U_{x,mu})_{row,col} of the sites x
 *                        of parity p in cb order.
 *
 * CANONICAL HOST LAYOUTS (upload / download; element type = context precision):
 *   spinor : cplx [idx][colour]            over the FULL lattice (V sites).  A half-field
 *            upload reads only the sites of its parity; a half-field download writes
 *            those sites and ZERO on the sites of the other parity.
 *   gauge  : cplx [idx][mu][row][col]      over the full lattice; [idx][mu] = U_{x,mu}.
 *
 * OWNERSHIP: every device buffer is allocated by the caller (e.g. PyTorch) and only
 * BOUND to a descriptor by qcd_field_alloc; the library never frees caller memory.
 * The context owns a few KB of device scalars / reduction partials and a 32 MiB
 * staging buffer used by upload / download.
 *
 * STREAM: all device work is enqueued on the cudaStream_t passed to qcd_init (borrowed,
 * e.g. torch.cuda.current_stream().cuda_stream; NULL = legacy default stream).
 * Operator calls are asynchronous; upload, download, qcd_cg_solve and qcd_cg_finish
 * synchronise that stream before they return.
 *
 * ERRORS: every call returns a qcd_status; nothing aborts, no exception crosses the
 * ABI.  The message of the last failure is kept per context (qcd_last_error).  There
 * is NO CPU fallback: without a CUDA device qcd_init returns QCD_ECUDA.
 */
#ifndef QCD_B200_H
#define QCD_B200_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef int qcd_status;
enum {
    QCD_OK = 0,
    QCD_EINVAL = 1,        /* bad argument (dims, kind/parity mismatch, size, alignment, aliasing) */
    QCD_ENOMEM = 2,        /* host or device allocation inside the library failed              */
    QCD_ECUDA = 3,         /* a CUDA runtime call failed; see qcd_last_error                    */
    QCD_ENOTCONVERGED = 4, /* CG stopped at maxiter; x holds the last iterate, info is filled   */
    QCD_EBREAKDOWN = 5     /* CG met <p,Mp> <= 0 or a NaN                                       */
};

/* field kinds */
enum {
    QCD_SPINOR_EVEN = 0,   /* 3 planes of Vh cplx, sites of parity 0 */
    QCD_SPINOR_ODD = 1,    /* 3 planes of Vh cplx, sites of parity 1 */
    QCD_SPINOR_FULL = 2,   /* even half-field then odd half-field    */
    QCD_GAUGE = 3          /* 72 planes of Vh cplx                   */
};

typedef struct qcd_ctx qcd_ctx;       /* opaque */
typedef struct qcd_field qcd_field;   /* opaque descriptor of a caller-owned device buffer */

typedef struct qcd_cg_info {
    int iters;             /* number of M applications performed                               */
    int converged;         /* 1 iff sqrt(rr/bb) <= tol was met                                  */
    double rel_resid;      /* sqrt(rr/bb) of the CG recurrence at exit                          */
    double bnorm2;         /* <b,b>                                                             */
    double seconds;        /* device time of the solve (CUDA events on the context stream)     */
} qcd_cg_info;

const char *qcd_strerror(qcd_status s);
/* Message of the last failing call on this context ("" if none).  ctx may be NULL: returns the
 * message of the last failing qcd_init of this thread. */
const char *qcd_last_error(const qcd_ctx *ctx);

/*
 * Create a context for a lattice (N_sigma^3 x N_tau, here general N0..N3).
 *   dims      : host pointer to 4 ints (N0,N1,N2,N3); all even, >= 2, N0 % 4 == 0, V < 2^31
 *   precision : 64 (double) or 32 (float) -- storage and field arithmetic type
 *               ("single and double precision"); reductions and CG scalars
 *               are double in both.
 *   cuda_stream : a cudaStream_t, borrowed.
 * Errors: QCD_EINVAL (dims / precision), QCD_ECUDA (no device, not compute capability 10.x,
 * or a CUDA failure), QCD_ENOMEM.
 */
qcd_status qcd_init(qcd_ctx **out, const int dims[4], int precision, void *cuda_stream);
qcd_status qcd_finalize(qcd_ctx *ctx);

/* Bytes of a field of `kind` in the device layout above (0 for a bad kind). */
size_t qcd_field_bytes(const qcd_ctx *ctx, int kind);
/* Bytes of the CG workspace: 3 even + 1 odd half-fields (r, p, Ap, t = D_oe p). */
size_t qcd_workspace_bytes(const qcd_ctx *ctx);

/*
 * Bind a caller-owned DEVICE buffer to a typed descriptor (north_star: qcd_field_alloc,
 * "SoA, even sites then odd sites"; PAPER.md:35 Latfield).
 *   device_ptr : device pointer, 256-byte aligned, at least qcd_field_bytes(ctx, kind) bytes
 *   nbytes     : size of the buffer
 * The buffer contents are not touched.  Errors: QCD_EINVAL (kind, size, alignment, NULL).
 */
qcd_status qcd_field_alloc(qcd_ctx *ctx, int kind, void *device_ptr, size_t nbytes, qcd_field **out);
qcd_status qcd_field_free(qcd_field *f);   /* frees the descriptor only */

/*
 * host <-> device with the layout permutation done on the device.
 *   host : HOST pointer to the canonical layout of the field's kind (see above), element
 *          type = context precision; pageable or pinned.
 * Both synchronise the context stream before returning.
 */
qcd_status qcd_field_upload(qcd_field *f, const void *host);
qcd_status qcd_field_download(const qcd_field *f, void *host);

/* Bind the CG workspace (device pointer, 256-byte aligned, >= qcd_workspace_bytes). */
qcd_status qcd_set_workspace(qcd_ctx *ctx, void *device_ptr, size_t nbytes);

/*
 * Parity blocks of Eq. (1).  Asynchronous on the context stream.
 *   qcd_dslash_eo : out_even = D_eo in_odd      qcd_dslash_oe : out_odd = D_oe in_even
 * U is a QCD_GAUGE field.  out must not alias in.  Kind mismatch -> QCD_EINVAL.
 * A QCD_SPINOR_FULL field may be passed for either argument: its even or odd half is used.
 */
qcd_status qcd_dslash_eo(qcd_ctx *ctx, const qcd_field *U, qcd_field *out_even, const qcd_field *in_odd);
qcd_status qcd_dslash_oe(qcd_ctx *ctx, const qcd_field *U, qcd_field *out_odd, const qcd_field *in_even);

/*
 * out_even = M in_even = m^2 in_even - D_eo D_oe in_even  (north_star).  Needs the workspace
 * (its odd half-field is the intermediate).  Asynchronous.  m < 0 -> QCD_EINVAL.
 */
qcd_status qcd_apply_M(qcd_ctx *ctx, const qcd_field *U, qcd_field *out_even, const qcd_field *in_even, double m);

/*
 * Conjugate Gradient on M x = b over even sites (algorithm = DESIGN.md
 * reading R6): x0 = 0, stop when sqrt(rr/bb) <= tol (tested before each M application) or
 * after maxiter M applications.  alpha, beta, rr, the iteration counter and the stop flag
 * live on the device; the host only polls the flag.
 *   b : QCD_SPINOR_EVEN (read only)     x : QCD_SPINOR_EVEN (output only, x0 = 0)
 *   info : host pointer, may be NULL
 * Returns QCD_OK (converged), QCD_ENOTCONVERGED, QCD_EBREAKDOWN, QCD_EINVAL (m < 0,
 * tol <= 0, maxiter < 0, kinds, missing workspace, x aliases b), QCD_ECUDA.
 * b = 0 gives x = 0, iters = 0, QCD_OK.  Synchronises the stream.
 */
qcd_status qcd_cg_solve(qcd_ctx *ctx, const qcd_field *U, const qcd_field *b, qcd_field *x,
                        double m, double tol, int maxiter, qcd_cg_info *info);

/*
 * The same solve in three pieces, for callers that interleave other work or want to time
 * a fixed number of iterations:
 *   qcd_cg_begin  : x = 0, r = p = b, rr = bb = <b,b>, k = 0             (asynchronous)
 *   qcd_cg_iterate: enqueue n more iterations; iterations after the stop   (asynchronous)
 *                   flag is set are no-ops on the device
 *   qcd_cg_finish : synchronise, read back the scalars, fill info; returns as qcd_cg_solve.
 *                   If the solve is still running (not converged, k < maxiter) it returns
 *                   QCD_ENOTCONVERGED with info describing the current state.
 *   qcd_cg_poll   : synchronise and read the device state without ending the solve:
 *                   *state = 0 running, 1 converged, 2 maxiter reached, 3 breakdown;
 *                   *iters, *rel_resid as in qcd_cg_info (any pointer may be NULL).
 */
qcd_status qcd_cg_begin(qcd_ctx *ctx, const qcd_field *U, const qcd_field *b, qcd_field *x,
                        double m, double tol, int maxiter);
qcd_status qcd_cg_iterate(qcd_ctx *ctx, int n);
qcd_status qcd_cg_poll(qcd_ctx *ctx, int *state, int *iters, double *rel_resid);
qcd_status qcd_cg_finish(qcd_ctx *ctx, qcd_cg_info *info);

/*
 * qcd_cg_solve with HOST source and solution in the canonical spinor layout (full-lattice
 * arrays, even sites used): upload b, solve, download x.  b_dev / x_dev are the device
 * fields used for staging.  info->seconds covers copies and solve.
 */
qcd_status qcd_cg_solve_host(qcd_ctx *ctx, const qcd_field *U, qcd_field *b_dev, qcd_field *x_dev,
                             const void *b_host, void *x_host,
                             double m, double tol, int maxiter, qcd_cg_info *info);

/*
 * Device-time accounting per kernel class (CUDA events recorded on the context stream
 * around each launch while enabled; used by bench.py for the roofline line).
 *   qcd_profile_enable(ctx, 1/0) : start (and reset) / stop recording
 *   qcd_profile_read : synchronises; for kernel class `which` returns the number of launches
 *                      recorded and their summed device milliseconds.
 * Classes: 0 = Dslash (D_oe / plain D_eo), 1 = D_eo + M epilogue + <p,Mp> partials,
 *          2 = fused x/r update + |r|^2, 3 = p update, 4 = init / misc.
 * At most 4096 launches are recorded per enable; later ones are counted as dropped.
 */
enum { QCD_K_DSLASH = 0, QCD_K_DSLASH_EPI = 1, QCD_K_UPDATE_XR = 2, QCD_K_UPDATE_P = 3, QCD_K_MISC = 4, QCD_K_COUNT = 5 };
qcd_status qcd_profile_enable(qcd_ctx *ctx, int on);
qcd_status qcd_profile_read(qcd_ctx *ctx, int which, int *launches, double *total_ms);
/* Total kernel launches enqueued by this context since qcd_init (for gpu_launches). */
long long qcd_launch_count(const qcd_ctx *ctx);

/*
 * Tuning knob for the Dslash kernels (bench sweeps):
 *   variant 0 = default.  Unknown variants -> QCD_EINVAL.
 */
qcd_status qcd_set_dslash_variant(qcd_ctx *ctx, int variant);

/* Re<a,b> over a half-field pair of the same kind (deterministic two-stage reduction,
 * double accumulation); synchronises.  Used by tests and by callers that need norms. */
qcd_status qcd_re_dot(qcd_ctx *ctx, const qcd_field *a, const qcd_field *b, double *result);

#ifdef __cplusplus
}
#endif
#endif /* QCD_B200_H */
