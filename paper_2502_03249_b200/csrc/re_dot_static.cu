// qcd_re_dot_static (include/qcd.h): the deterministic two-stage dot product of qcd_re_dot (reduce.cuh;
// PAPER.md:54 "dot product involving global reductions") for callers that cannot allocate.
//
// Every other entry point works on a qcd_ctx, and qcd_init allocates the context's reduction scratch with
// cudaMalloc.  This one takes plain device pointers and keeps its scratch -- the stage-1 partial sums and the
// last-block tickets -- in a file-scope __device__ array of fixed size, so it calls no cudaMalloc / cudaFree and
// no allocating library routine, at set-up or later.  The kernel is re_dot_kernel (cg_kernels.cuh) with the scratch
// pointers passed in: same block shape, same summation order, hence the same result as qcd_re_dot on the same data.
//
// The array's name is a HOST-SIDE STAND-IN in host code, not a device address: the address is taken once per
// device with cudaGetSymbolAddress (that device current) and handed to the kernel as an ordinary pointer.
#include "../../include/qcd.h"

#include <cuda_runtime.h>
#include <stdarg.h>
#include <stdint.h>
#include <stdio.h>

#include <mutex>

#include "cg_kernels.cuh"
#include "reduce.cuh"

namespace {

using namespace qcd;

enum {
    ITEMS_PER_BLOCK = BLAS_BLOCK * BLAS_ITEMS,                                   // 16-byte vectors per block
    MAX_BLOCKS = (int)(QCD_RE_DOT_STATIC_MAX_REALS * sizeof(double) / 16 / ITEMS_PER_BLOCK),   // 24 576 (fp64, the larger grid)
    MAX_GROUPS = (MAX_BLOCKS + TICKET_GROUP - 1) / TICKET_GROUP,                 // 384 first-level tickets
    TICKET_WORDS = MAX_GROUPS + 1,                                               // + the top-level ticket
    TICKET_DOUBLES = (TICKET_WORDS * (int)sizeof(unsigned) + 255) / 256 * 32,    // rounded up to 256 bytes
    SCRATCH_DOUBLES = MAX_BLOCKS + TICKET_DOUBLES,                               // 24 800 doubles = 198 400 bytes
    MAX_DEVICES = 64
};
static_assert(QCD_RE_DOT_STATIC_MAX_REALS * sizeof(double) % (16 * ITEMS_PER_BLOCK) == 0, "limit must be a whole number of blocks");
static_assert(SCRATCH_DOUBLES * sizeof(double) == QCD_RE_DOT_STATIC_SCRATCH_BYTES, "include/qcd.h states the scratch size");

// [0, MAX_BLOCKS) stage-1 partial sums; then TICKET_WORDS unsigned tickets (l1[MAX_GROUPS], top).
// Held by every GPU that loads the library until the process exits.  Shared by every call.
static __device__ __align__(256) double re_dot_static_scratch[SCRATCH_DOUBLES];

template <typename T>
__global__ void __launch_bounds__(BLAS_BLOCK) re_dot_static_kernel(
    int n16, const typename Vec16<T>::type *__restrict__ a, const typename Vec16<T>::type *__restrict__ b,
    double *partials, unsigned *l1, unsigned *top, double *result)
{
    double s = 0.0;
    const int base = blockIdx.x * ITEMS_PER_BLOCK + threadIdx.x;
#pragma unroll
    for (int j = 0; j < BLAS_ITEMS; ++j) {
        const int i = base + j * BLAS_BLOCK;
        if (i < n16) s += vdot(a[i], b[i]);
    }
    __shared__ double smem[BLAS_BLOCK / 32];
    __shared__ int last;
    const double bs = block_sum<BLAS_BLOCK>(s, smem);
    if (threadIdx.x == 0) {
        partials[blockIdx.x] = bs;
        last = take_ticket(top, l1);
    }
    __syncthreads();
    if (last) {
        const double d = final_sum<BLAS_BLOCK>(partials, (int)gridDim.x, smem);
        if (threadIdx.x == 0) *result = d;
    }
}

std::mutex g_mu;
double *g_scratch[MAX_DEVICES];          // device address of re_dot_static_scratch on device i, NULL until resolved

qcd_status fail(char *errbuf, size_t cap, qcd_status s, const char *fmt, ...) __attribute__((format(printf, 4, 5)));
qcd_status fail(char *errbuf, size_t cap, qcd_status s, const char *fmt, ...)
{
    if (errbuf && cap) {
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(errbuf, cap, fmt, ap);
        va_end(ap);
    }
    return s;
}

// Set-up, once per device, with that device current: resolve the device address of the scratch array.
cudaError_t scratch_of(int dev, double **out)
{
    std::lock_guard<std::mutex> lock(g_mu);
    if (!g_scratch[dev]) {
        double *p = nullptr;
        const cudaError_t err = cudaGetSymbolAddress((void **)&p, re_dot_static_scratch);
        if (err != cudaSuccess) return err;
        g_scratch[dev] = p;
    }
    *out = g_scratch[dev];
    return cudaSuccess;
}

// true iff p is device (or managed) memory of device `dev`
bool on_device(const void *p, int dev, cudaError_t *err)
{
    cudaPointerAttributes at;
    *err = cudaPointerGetAttributes(&at, p);
    if (*err != cudaSuccess) return false;
    return (at.type == cudaMemoryTypeDevice || at.type == cudaMemoryTypeManaged) && (at.type == cudaMemoryTypeManaged || at.device == dev);
}

} // namespace

extern "C" qcd_status qcd_re_dot_static(const void *a_dev, const void *b_dev, size_t n_reals, int precision,
                                        void *cuda_stream, double *result_dev, char *errbuf, size_t errbuf_bytes)
{
    if (errbuf && errbuf_bytes) errbuf[0] = 0;
    if (!a_dev || !b_dev || !result_dev) return fail(errbuf, errbuf_bytes, QCD_EINVAL, "qcd_re_dot_static: a_dev, b_dev and result_dev must not be NULL");
    if (precision != 64 && precision != 32) return fail(errbuf, errbuf_bytes, QCD_EINVAL, "qcd_re_dot_static: precision must be 64 or 32, got %d", precision);
    if (n_reals > (size_t)QCD_RE_DOT_STATIC_MAX_REALS)
        return fail(errbuf, errbuf_bytes, QCD_EINVAL,
                    "qcd_re_dot_static: n_reals = %zu exceeds QCD_RE_DOT_STATIC_MAX_REALS = %zu (the static scratch holds the partial sums of "
                    "no more; use qcd_re_dot on a context for larger fields)", n_reals, (size_t)QCD_RE_DOT_STATIC_MAX_REALS);
    const size_t rsize = precision == 64 ? sizeof(double) : sizeof(float);
    if ((n_reals * rsize) % 16 || ((uintptr_t)a_dev % 16) || ((uintptr_t)b_dev % 16) || ((uintptr_t)result_dev % 8))
        return fail(errbuf, errbuf_bytes, QCD_EINVAL, "qcd_re_dot_static: a_dev and b_dev must be 16-byte aligned and hold a multiple of 16 bytes, result_dev 8-byte aligned");
    int dev = -1;
    cudaError_t err = cudaGetDevice(&dev);
    if (err != cudaSuccess) return fail(errbuf, errbuf_bytes, QCD_ECUDA, "qcd_re_dot_static: cudaGetDevice: %s (there is no CPU fallback)", cudaGetErrorString(err));
    if (dev < 0 || dev >= MAX_DEVICES) return fail(errbuf, errbuf_bytes, QCD_EINVAL, "qcd_re_dot_static: device index %d not supported", dev);
    const void *ptrs[3] = {a_dev, b_dev, result_dev};
    const char *names[3] = {"a_dev", "b_dev", "result_dev"};
    for (int i = 0; i < 3; ++i) {
        if (!on_device(ptrs[i], dev, &err)) {
            if (err != cudaSuccess) { cudaGetLastError(); return fail(errbuf, errbuf_bytes, QCD_ECUDA, "qcd_re_dot_static: cudaPointerGetAttributes(%s): %s", names[i], cudaGetErrorString(err)); }
            return fail(errbuf, errbuf_bytes, QCD_EINVAL, "qcd_re_dot_static: %s is not device memory of the current device %d", names[i], dev);
        }
    }
    cudaStream_t stream = (cudaStream_t)cuda_stream;
    if (n_reals == 0) {                                                     // empty sum: 0.0 is all-zero bytes
        err = cudaMemsetAsync(result_dev, 0, sizeof(double), stream);
        if (err != cudaSuccess) return fail(errbuf, errbuf_bytes, QCD_ECUDA, "qcd_re_dot_static: cudaMemsetAsync: %s", cudaGetErrorString(err));
        return QCD_OK;
    }
    double *scratch = nullptr;
    err = scratch_of(dev, &scratch);
    if (err != cudaSuccess) return fail(errbuf, errbuf_bytes, QCD_ECUDA, "qcd_re_dot_static: cudaGetSymbolAddress: %s", cudaGetErrorString(err));
    double *partials = scratch;
    unsigned *l1 = (unsigned *)(scratch + MAX_BLOCKS);
    unsigned *top = l1 + MAX_GROUPS;
    const int n16 = (int)(n_reals * rsize / 16);
    const int grid = (n16 + ITEMS_PER_BLOCK - 1) / ITEMS_PER_BLOCK;        // <= MAX_BLOCKS by the size check above
    // The tickets must start at zero.  A completed call leaves them at zero (atomicInc wraps), but the array is
    // shared and keeps whatever the last call left: clear them every time, on the caller's stream.
    err = cudaMemsetAsync(l1, 0, TICKET_WORDS * sizeof(unsigned), stream);
    if (err != cudaSuccess) return fail(errbuf, errbuf_bytes, QCD_ECUDA, "qcd_re_dot_static: cudaMemsetAsync: %s", cudaGetErrorString(err));
    if (precision == 64)
        re_dot_static_kernel<double><<<grid, BLAS_BLOCK, 0, stream>>>(n16, (const double2 *)a_dev, (const double2 *)b_dev, partials, l1, top, result_dev);
    else
        re_dot_static_kernel<float><<<grid, BLAS_BLOCK, 0, stream>>>(n16, (const float4 *)a_dev, (const float4 *)b_dev, partials, l1, top, result_dev);
    err = cudaGetLastError();
    if (err != cudaSuccess) return fail(errbuf, errbuf_bytes, QCD_ECUDA, "qcd_re_dot_static: kernel launch: %s", cudaGetErrorString(err));
    return QCD_OK;
}
