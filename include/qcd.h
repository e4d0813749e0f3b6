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
 * complex matrices (18 reals) in the headline path, never modified by the library.  The
 * paper's own traffic reductions (two-row links, temporal gauge, several
 * vectors per link load) and the mixed-precision solver are the calls of the second half
 * of this header ("Variants"); they are reported separately from the headline.
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
 *            The same full 3x3 host layout serves QCD_GAUGE_2ROW (upload keeps rows 0 and 1,
 *            download reconstructs row 2 = conj(row 0 x row 1)).
 *   colour matrix : cplx [idx][row][col]   over the full lattice.
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
    QCD_GAUGE = 3,         /* 72 planes of Vh cplx                   */
    QCD_GAUGE_2ROW = 4,    /* 48 planes: cplx [parity][mu][k = 3*row + col, row < 2][Vh] */
    QCD_COLOUR_MATRIX = 5  /* 18 planes: cplx [parity][k = 3*row + col][Vh], one 3x3 matrix per site  */
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
/* Bytes of the CG workspace: 4 even + 1 odd half-fields (r, p, Ap, t = D_oe p, and a second
 * direction buffer used by the persistent solver loop, qcd_set_cg_loop). */
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
 * A QCD_SPINOR_FULL field may be passed for either argument: its even or odd half is used (the two halves of
 * ONE full field are distinct memory, so the same full field may serve as out and in).  Aliasing is checked on
 * byte ranges of the half-fields, not on base pointers.
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
 * b and x must not overlap each other nor the bound workspace (byte ranges; QCD_EINVAL).
 * Every entry point that enqueues work returns QCD_EINVAL when the current CUDA device is not the one the context
 * was created on (qcd_init records cudaGetDevice()).
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
 * Residual history of the most recent solve of this context (SURVEY.md Sec. 5 "metrics"):
 * host_out[j] = <r,r> / <b,b> after j + 1 M applications, j = 0 .. iters-1 -- the squared relative
 * recurrence residual CG tests against tol^2 (reading R6).  Recorded on the device by the kernel
 * that advances the recurrence (no extra launch or host round trip during the solve), for the
 * first 16384 iterations of every right-hand side; all three solver loops record it.
 *   rhs      : 0 for qcd_cg_solve; 0 .. n-1 after a multi solve of n right-hand sides (rhs >= n: QCD_EINVAL)
 *   host_out : HOST array of `cap` doubles (may be NULL when cap = 0)
 *   n        : receives min(iters, cap, 16384)
 * Valid from qcd_cg_finish / the return of qcd_cg_solve until the next solve begins on the context
 * (the inner solves of qcd_cg_solve_mixed overwrite the fp32 context's history).  Synchronises.
 * Errors: QCD_EINVAL (bad argument, solve in progress), QCD_ECUDA.
 */
qcd_status qcd_cg_history(qcd_ctx *ctx, int rhs, double *host_out, int cap, int *n);

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
 * Read-only streaming ceiling (measurement hook; a half-Dslash is 96 % reads,
 * so its roofline is quoted against a read stream as well as against the copy peak and the
 * theoretical peak).  Runs `reps` passes of a kernel that does nothing but load every 16 bytes of
 * field f (any kind) once, with the Dslash's own link-load instruction (read-only path, no L1
 * allocation, L2 evict_first), times them with CUDA events on the context stream, synchronises,
 * and returns the average milliseconds per pass in *ms_per_pass (host pointer).
 * GB/s = qcd_field_bytes(ctx, kind of f) / ms.  Use a field much larger than the 126 MB L2.
 * Errors: QCD_EINVAL (NULL, foreign field, reps < 1), QCD_ECUDA.
 */
qcd_status qcd_stream_read(qcd_ctx *ctx, const qcd_field *f, int reps, double *ms_per_pass);
/*
 * The same for a field that FITS the L2 (the small-lattice regime: 16^4 links = 37.7 MB): `passes` passes over
 * the field inside ONE launch after a warm-up launch, so that the L2 -> SM rate is timed and not the kernel launch.
 * *ms_per_pass = launch time / passes.  L1 is bypassed, every pass is L2 traffic.  Errors as qcd_stream_read.
 */
qcd_status qcd_stream_read_resident(qcd_ctx *ctx, const qcd_field *f, int passes, double *ms_per_pass);
/*
 * Streaming ceiling of a MIX of read and write streams (measurement hook, the NMULTI kernels): one pass reads 16
 * bytes per thread from each of the first `read_planes` planes (of Vh complex numbers of the context's precision) of src and writes
 * 16 bytes to each of the first `write_planes` planes of dst, every thread at its own index -- the DRAM access pattern of a
 * multi-vector half-Dslash (links + n vectors read once, n vectors written) without stencil, neighbour reads or arithmetic.
 * `reps` passes, CUDA events on the context stream, synchronises; *ms_per_pass is the average.  GB/s = (read_planes +
 * write_planes) * Vh * 2 * sizeof(real) / ms.  dst is OVERWRITTEN.  Errors: QCD_EINVAL (NULL, foreign or overlapping fields, more
 * planes than a field holds, reps < 1), QCD_ECUDA.
 */
qcd_status qcd_stream_mix(qcd_ctx *ctx, const qcd_field *src, qcd_field *dst, int read_planes, int write_planes, int reps, double *ms_per_pass);
/*
 * Streaming ceiling of the BULK-COPY (TMA) path (measurement hook; precision-64 contexts, the NMULTI kernels): one block
 * per SM walks the planes of src (Vh complex numbers each) in groups of 128 consecutive sites; for each group, `hops` times, `producers`
 * warps (1 .. 4) issue `copies` tensor-map copies of `rows` planes x 128 sites (2 KB per plane) into a ring of `stages` shared-memory
 * stages (stages x copies x rows x 2 KB must fit a block's shared memory), and four consumer warps read every byte back from shared
 * memory.  Plane rows wrap around inside the field, so once hops x copies x rows exceeds the field's planes the re-reads are L2 hits,
 * like the neighbour gathers of a Dslash.  `reps` passes, CUDA events on the context stream, synchronises; *ms_per_pass is the average;
 * requested bytes per pass = (Vh / 128) * hops * copies * rows * 2048.  What it measures: the rate at which a SM takes in requested bytes
 * through the copy engine (about 15 TB/s on the chip), against the 9 - 11 TB/s of every LSU-fed Dslash kernel.
 * Errors: QCD_EINVAL (NULL, foreign field, precision 32, a range above, Vh not a multiple of 128), QCD_ECUDA.
 */
qcd_status qcd_stream_bulk(qcd_ctx *ctx, const qcd_field *src, int rows, int copies, int hops, int stages, int producers, int reps,
                           double *ms_per_pass);

/*
 * Tuning knob for the Dslash kernels (bench sweeps and A/B tests, Sec. 10):
 *   0 : the library's choice (one vector: 128-thread blocks, 3 resident per SM for the plain Dslash on full links, 4 for the
 *       kernels with the M epilogue and on two-row links; for several vectors the register kernel or the cp.async-staged
 *       kernel, whichever measured faster for that (precision, number of vectors, link storage))
 *   1, 2, 3 : one-vector kernel with 64 x 8, 256 x 2 threads x resident blocks, and 128 threads with the OTHER of 3 / 4 resident
 *       blocks than the library's choice for that kernel
 *   4 : force the staged kernel (links prefetched through shared memory by cp.async)
 *   5 : force the register kernel
 *   6, 7 : force the pair kernel (two adjacent lanes per site, half of the vectors each, the link shared through the
 *       cp.async ring) under a 168- / 128-register cap; applies to an even number of vectors >= 4 on a volume of whole
 *       64-site blocks, otherwise the library's choice runs
 *   8 : force the register kernel with the x0 / x1 neighbour rows of a block staged in shared memory; applies to 4 or 8
 *       vectors on lattices where 128 consecutive sites are whole x0-rows of one (x2, x3) plane, otherwise the library's choice
 *   9 : force the kernel whose loop over the four directions is not unrolled (3 .. 8 vectors)
 *  10 : force the bulk-copy kernel (warp-specialised: producer warps feed a shared-memory ring with tensor-map copies, consumer
 *       warps compute; plain Dslash of 2 .. 8 vectors on lattices where 128 consecutive sites are whole x0-rows of one (x2, x3)
 *       plane, otherwise the library's choice)
 * 6 .. 10 are the round-2 experiments (profiles/README.md); none measured faster than the library's choice (10 is on a
 * par with it for 6 and 8 vectors on full fp64 links and slower elsewhere).
 * Every variant computes the same result (bitwise).  Unknown variants -> QCD_EINVAL.
 */
qcd_status qcd_set_dslash_variant(qcd_ctx *ctx, int variant);
/*
 * Solver loop of qcd_cg_solve / qcd_cg_solve_multi: all three run the same
 * algorithm with the same per-site arithmetic; they differ in how the iterations reach the device.
 *   0 : chosen by the library -- the persistent kernel when one right-hand side, its links and the
 *       work vectors fit the L2 (<= 96 MB); else graph replay on small lattices when the context
 *       stream is not the legacy default stream; else kernel-by-kernel
 *   1 : kernel-by-kernel enqueue, the host polling the device-resident stop flag
 *   2 : replay of a captured CUDA graph of 16 iterations (needs a non-default stream)
 *   3 : ONE cooperative kernel runs the whole solve with grid-wide barriers between the phases
 * Else QCD_EINVAL.
 */
qcd_status qcd_set_cg_loop(qcd_ctx *ctx, int mode);
/*
 * The loop the most recent qcd_cg_solve / qcd_cg_solve_multi / inner solve of qcd_cg_solve_mixed of this context
 * actually ran: 1, 2 or 3 as above (1 also for a solve driven by qcd_cg_begin / qcd_cg_iterate); 0 before the first
 * solve or for a NULL context.  With mode 0 this is the library's choice; a FORCED mode that cannot run (2 on the
 * legacy default stream, 3 with several right-hand sides or without cooperative launch) makes the solve return
 * QCD_EINVAL instead of falling back, and forced mode 2 still runs kernel by kernel -- reported here as 1 -- while
 * per-launch profiling is on or when maxiter < 16.
 */
int qcd_last_cg_loop(const qcd_ctx *ctx);
/*
 * Loop 3 has two launch shapes: lattices of up to 2048 sites per parity (8^4) run as ONE
 * thread-block cluster of 1 .. 16 CTAs of 512 threads (barrier.cluster and distributed shared memory instead of a
 * grid-wide barrier through the L2); larger ones as a cooperative grid.  Same arithmetic, same summation orders up to
 * the shape of the final sum over blocks.
 *   qcd_last_cg_cluster : CTAs of the cluster the most recent solve ran as; 0 if it ran as a cooperative grid or did not
 *                         run loop 3.
 *   qcd_set_cg_cluster  : 0 forbids the cluster shape (A/B measurements and tests), 1 (default) allows it.
 */
int qcd_last_cg_cluster(const qcd_ctx *ctx);
qcd_status qcd_set_cg_cluster(qcd_ctx *ctx, int on);
/*
 * Traversal order of the Dslash threads: the sites are walked in
 * chunks of `width` rows of x2 ((x0,x1) fastest, x2 inside the chunk, then x3, then the chunk),
 * which keeps the time-neighbour spinors of several vectors inside the L2.  A pure permutation of
 * the work: results are independent of it.  width = 0: chosen by the library from the lattice,
 * the precision and the number of vectors (N2, i.e. the plain order, for one vector up to 64^4);
 * otherwise a divisor of N2.  Else QCD_EINVAL.
 */
qcd_status qcd_set_traversal_chunk(qcd_ctx *ctx, int width);

/*
 * Phase timeline of the persistent solver loop (measurement hook; "global
 * reductions which have higher latencies ... more pronounced for smaller lattice sizes").
 *   qcd_cg_timeline_enable(ctx, 1) : solves that run the persistent kernel (qcd_last_cg_loop() == 3) afterwards record, for their
 *       first 64 iterations, nine %globaltimer stamps (nanoseconds) per iteration in thread 0 of block 0 and of the last block:
 *       0 phase 1 (p update + D_oe) starts, 1 its work is done, 2 past grid barrier 1, 3 phase 2 (D_eo + M epilogue + block
 *       partial of <p,Mp>) done, 4 past barrier 2, 5 partials summed / alpha known, 6 phase 3 (x, r update + block partial of
 *       <r,r>) done, 7 past barrier 3, 8 partials summed / beta known.  0 switches it off (the default; no stamp is taken then).
 *   qcd_cg_timeline_read : host_out receives [2][n][9] stamps (block 0 first, then the last block), n = min(cap_iters, 64);
 *       *n_iters = how many of those iterations actually ran.  Synchronises.
 * Errors: QCD_EINVAL (NULL, solve in progress), QCD_ECUDA.
 */
qcd_status qcd_cg_timeline_enable(qcd_ctx *ctx, int on);
qcd_status qcd_cg_timeline_read(qcd_ctx *ctx, unsigned long long *host_out, int cap_iters, int *n_iters);

/* Re<a,b> over a half-field pair of the same kind (deterministic two-stage reduction,
 * double accumulation); synchronises.  Used by tests and by callers that need norms. */
qcd_status qcd_re_dot(qcd_ctx *ctx, const qcd_field *a, const qcd_field *b, double *result);

/*
 * The same dot product for callers that cannot allocate (code under CUDA graph capture, tight serving
 * loops, harnesses that forbid cudaMalloc): no qcd_ctx (qcd_init allocates), no cudaMalloc / cudaFree and no
 * allocating library routine, at set-up or later.  The reduction scratch (stage-1 partial sums + last-block
 * tickets, "dot product involving global reductions") is a file-scope __device__ array of
 * QCD_RE_DOT_STATIC_SCRATCH_BYTES (198 400 bytes) that every GPU loading the library holds until the
 * process exits; it bounds the size of one call:
 *       n_reals <= QCD_RE_DOT_STATIC_MAX_REALS = 50 331 648  (one 64^4 half-field: 3 colours x 2 reals x 64^4 / 2)
 * in both precisions.  A larger n_reals is rejected with QCD_EINVAL; use qcd_re_dot on a context there.
 *   a_dev, b_dev : DEVICE pointers (of the current device) to n_reals reals of `precision` (64: double,
 *                  32: float), e.g. two half-fields in the device layout; 16-byte aligned, n_reals * size a
 *                  multiple of 16 bytes; read only, may alias each other
 *   cuda_stream  : a cudaStream_t of the current device, borrowed (NULL = legacy default stream)
 *   result_dev   : DEVICE pointer to one double, 8-byte aligned, caller-owned: receives
 *                  sum_i a[i] b[i] (products and sums in double, the summation order of qcd_re_dot: the
 *                  two calls return the same value on the same data); 0.0 for n_reals = 0
 *   errbuf       : HOST buffer of errbuf_bytes for the message of a failure ("" on success); may be NULL
 * Asynchronous: enqueues one 1.5 KB memset of the tickets and one kernel on cuda_stream and returns; the
 * result is valid once that work has completed.  The first call on each device also resolves the array's
 * device address (cudaGetSymbolAddress, which may load the module): make it before capturing a graph.
 * SHARED SCRATCH: every call, from every thread and stream, uses the same array, which keeps the last call's
 * contents (the tickets are cleared by every call).  Calls that may overlap on the GPU -- different streams
 * without an ordering between them -- RACE on it and return garbage: order them.  Calls on one stream are safe.
 * Errors: QCD_EINVAL (NULL, precision, alignment, n_reals beyond the maximum, a pointer that is not memory of
 * the current device), QCD_ECUDA (no device -- there is no CPU fallback -- or a CUDA failure).
 */
#define QCD_RE_DOT_STATIC_MAX_REALS 50331648
#define QCD_RE_DOT_STATIC_SCRATCH_BYTES 198400
qcd_status qcd_re_dot_static(const void *a_dev, const void *b_dev, size_t n_reals, int precision,
                             void *cuda_stream, double *result_dev, char *errbuf, size_t errbuf_bytes);

/* =========================================================================================
 * Variants: the paper's Dslash optimisations (Sec. 4.3) and mixed precision.
 * ========================================================================================= */

/* Largest number of vectors one multi-vector call accepts. */
enum { QCD_MAX_RHS = 8 };

/*
 * Two-row link storage ("For each link variable, we store only the first two rows,
 * i.e. 12 floats.  The third row is reconstructed on-the-fly when needed, using the properties
 * of SU(3) matrices": row2 = conj(row0 x row1)).
 *   qcd_gauge_compress : U12 (QCD_GAUGE_2ROW) = rows 0, 1 of U (QCD_GAUGE); device to device,
 *                        asynchronous; carries U's temporal-gauge mark over.
 * Every operator and solver call of this header accepts a QCD_GAUGE_2ROW field wherever it
 * accepts a QCD_GAUGE field.  The links must be in SU(3): the reconstruction is exact only then.
 */
qcd_status qcd_gauge_compress(qcd_ctx *ctx, const qcd_field *U, qcd_field *U12);

/*
 * Temporal gauge ("We use gauge fixing to transform the temporal link variables to
 * 1_{3x3} for all the sites with the temporal coordinate t != 0"; reading R20):
 *     g(xs,0) = 1,  g(xs,t) = g(xs,t+1) U_{(xs,t),3}^dagger  (t = N3-1 .. 1),
 *     U'_{x,mu} = g(x) U_{x,mu} g(x+mu)^dagger  =>  U'_{x,3} = 1 for x3 != 0.
 *   qcd_gauge_fix_temporal : U (QCD_GAUGE) -> U_fixed (QCD_GAUGE, may not alias U) and
 *                        g (QCD_COLOUR_MATRIX).  U_fixed is MARKED temporal-gauge: kernels
 *                        applied to it (or to its qcd_gauge_compress copy) do not read the time
 *                        links of sites with x3 != 0 and use the identity instead.  Asynchronous.
 *   qcd_gauge_set_temporal_unit : set / clear that mark by hand (for links fixed elsewhere and
 *                        uploaded; qcd_field_upload clears it).
 *   qcd_spinor_rotate  : out(x) = g(x) in(x) (dagger = 0) or g(x)^dagger in(x) (dagger = 1) on
 *                        spinor fields of the same kind; out may alias in.  D[U'] (g phi) =
 *                        g D[U] phi, so M[U'] x' = g b is solved by x' = g x.
 */
qcd_status qcd_gauge_fix_temporal(qcd_ctx *ctx, const qcd_field *U, qcd_field *U_fixed, qcd_field *g);
qcd_status qcd_gauge_set_temporal_unit(qcd_field *U, int on);
qcd_status qcd_spinor_rotate(qcd_ctx *ctx, const qcd_field *g, qcd_field *out, const qcd_field *in, int dagger);

/*
 * Several vectors per link load ("applying D on multiple vectors at once.  This
 * allows each link variable to be read once and then reused for multiple vectors", NMULTI).
 *   n    : 1 .. QCD_MAX_RHS
 *   out, in, b, x, info : HOST arrays of n field pointers / n structs
 * qcd_dslash_*_multi computes out[i] = D in[i]; qcd_cg_solve_multi runs n INDEPENDENT CG solves
 * M x[i] = b[i] in lock step (each right-hand side has its own alpha, beta, iteration count and
 * stop flag on the device and is frozen at its own stopping iteration; result identical to n
 * calls of qcd_cg_solve).  The workspace must hold qcd_workspace_bytes_multi(ctx, n) bytes.
 * Returns QCD_OK if every solve converged, else the first non-OK per-solve status
 * (QCD_ENOTCONVERGED / QCD_EBREAKDOWN); info[i] describes solve i.
 */
size_t qcd_workspace_bytes_multi(const qcd_ctx *ctx, int n);
qcd_status qcd_dslash_eo_multi(qcd_ctx *ctx, const qcd_field *U, int n, qcd_field *const *out_even, const qcd_field *const *in_odd);
qcd_status qcd_dslash_oe_multi(qcd_ctx *ctx, const qcd_field *U, int n, qcd_field *const *out_odd, const qcd_field *const *in_even);
qcd_status qcd_cg_solve_multi(qcd_ctx *ctx, const qcd_field *U, int n, const qcd_field *const *b, qcd_field *const *x,
                              double m, double tol, int maxiter, qcd_cg_info *info);
/* The multi solve in pieces, as qcd_cg_begin / qcd_cg_iterate / qcd_cg_finish (bench timing). */
qcd_status qcd_cg_begin_multi(qcd_ctx *ctx, const qcd_field *U, int n, const qcd_field *const *b, qcd_field *const *x,
                              double m, double tol, int maxiter);
qcd_status qcd_cg_finish_multi(qcd_ctx *ctx, qcd_cg_info *info);

/*
 * Precision conversion on the device: dst (a field of a precision-32 context) = round to
 * nearest of src (same kind, same lattice, precision-64 context), or the widening the other
 * way.  Both contexts must use the same stream.  Asynchronous.  Carries the temporal-gauge mark.
 */
qcd_status qcd_field_convert(qcd_field *dst, const qcd_field *src);

/*
 * Mixed-precision defect-correction CG (PAPER.md:66 benchmarks CG "in single and double
 * precision"; reading R21).  Solves M x = b to a TRUE fp64 relative residual <= tol:
 *     x = 0; r = b
 *     repeat: rel = |r|/|b|; stop if rel <= tol, or after max_outer corrections, or when the
 *             inner-iteration budget maxiter is spent
 *             tol_in = max(inner_tol, 0.5 tol / rel)
 *             rhs32 = fp32(r / |r|);  e32 = CG_fp32(M[U32], rhs32, tol_in);  x += |r| fp64(e32)
 *             r = b - M[U64] x                                   (fp64)
 *   ctx64, ctx32 : contexts of precision 64 and 32 on the same lattice and stream, each with
 *                  its workspace bound
 *   U64, U32     : gauge fields of ctx64 / ctx32 (any link storage)
 *   b, x         : QCD_SPINOR_EVEN fields of ctx64;  x is output only
 *   rhs32, e32   : QCD_SPINOR_EVEN scratch fields of ctx32
 *   info         : host pointer, may be NULL
 * Returns QCD_OK / QCD_ENOTCONVERGED / QCD_EBREAKDOWN / QCD_EINVAL / QCD_ECUDA.  Synchronises.
 */
typedef struct qcd_mixed_info {
    int converged;         /* 1 iff the fp64 residual met tol                                   */
    int outer;             /* defect-correction steps = inner solves                            */
    int inner_iters;       /* fp32 CG iterations summed over the inner solves                   */
    int m_applications_fp64; /* fp64 M applications (one per correction)                        */
    double true_resid;     /* |b - M x| / |b| in fp64 at exit (computed on the device)          */
    double seconds;        /* device time of the whole solve                                    */
} qcd_mixed_info;
qcd_status qcd_cg_solve_mixed(qcd_ctx *ctx64, qcd_ctx *ctx32, const qcd_field *U64, const qcd_field *U32,
                              const qcd_field *b, qcd_field *x, qcd_field *rhs32, qcd_field *e32,
                              double m, double tol, double inner_tol, int maxiter, int max_outer,
                              qcd_mixed_info *info);

#ifdef __cplusplus
}
#endif
#endif /* QCD_B200_H */
