// Conjugate-Gradient vector kernels ("CG update
// routine", Table 1): pure streaming over even half-fields viewed as flat
// arrays of 16-byte vectors (double2 = one complex, float4 = two complex), ITEMS vectors per
// thread issued back to back for memory-level parallelism.  alpha and beta are read from the
// device-resident CgScalars, so the host never sees them (north_star (d)).
//
//   cg_init      : x = 0, r = p = b, bb = <b,b>; last block: rr = bb, k = 0, flag
//   cg_update_xr : x += alpha p, r -= alpha Ap, partial |r|^2; last block: beta, rr, k, flag
//   cg_update_p  : p = r + beta p
//   re_dot       : Re<a,b>
//
// Several right-hand sides (NMULTI) are independent solves: blockIdx.y is the
// right-hand side, each with its own CgScalars entry, partials row and ticket; r, p, Ap are
// [nrhs][half-field] in the workspace, x and b are the caller's fields (RhsPtrs).
//
// Field arithmetic is in T; products for the reductions are formed and summed in double
// (reading R9); alpha, beta are rounded to T before they multiply a field.
#pragma once
#include "lattice.cuh"
#include "reduce.cuh"

namespace qcd {

template <typename T> struct Vec16;
template <> struct Vec16<double> { typedef double2 type; enum { N = 2 }; };
template <> struct Vec16<float>  { typedef float4 type;  enum { N = 4 }; };

__device__ __forceinline__ void vzero(double2 &a) { a.x = a.y = 0.0; }
__device__ __forceinline__ void vzero(float4 &a) { a.x = a.y = a.z = a.w = 0.f; }
__device__ __forceinline__ double vdot(const double2 &a, const double2 &b) { return a.x * b.x + a.y * b.y; }
__device__ __forceinline__ double vdot(const float4 &a, const float4 &b)
{
    return (double)a.x * (double)b.x + (double)a.y * (double)b.y + (double)a.z * (double)b.z + (double)a.w * (double)b.w;
}
// a += s * b
__device__ __forceinline__ void vaxpy(double2 &a, double s, const double2 &b) { a.x = fma(s, b.x, a.x); a.y = fma(s, b.y, a.y); }
__device__ __forceinline__ void vaxpy(float4 &a, float s, const float4 &b)
{
    a.x = fmaf(s, b.x, a.x); a.y = fmaf(s, b.y, a.y); a.z = fmaf(s, b.z, a.z); a.w = fmaf(s, b.w, a.w);
}
// a = b + s * a
__device__ __forceinline__ void vxpay(double2 &a, double s, const double2 &b) { a.x = fma(s, a.x, b.x); a.y = fma(s, a.y, b.y); }
__device__ __forceinline__ void vxpay(float4 &a, float s, const float4 &b)
{
    a.x = fmaf(s, a.x, b.x); a.y = fmaf(s, a.y, b.y); a.z = fmaf(s, a.z, b.z); a.w = fmaf(s, a.w, b.w);
}

enum { BLAS_BLOCK = 256, BLAS_ITEMS = 4 };

template <typename V>
struct RhsPtrs {
    V *x[MAXRHS];
    const V *b[MAXRHS];
};

template <typename T>
__global__ void __launch_bounds__(BLAS_BLOCK) cg_init_kernel(
    int n16, const __grid_constant__ RhsPtrs<typename Vec16<T>::type> ptrs,
    typename Vec16<T>::type *__restrict__ r, typename Vec16<T>::type *__restrict__ p,
    double tol, int maxiter, double *partials, CgScalars *scal)
{
    typedef typename Vec16<T>::type V;
    const int rhs = blockIdx.y;
    const V *__restrict__ b = ptrs.b[rhs];
    V *__restrict__ x = ptrs.x[rhs];
    r += (size_t)rhs * n16; p += (size_t)rhs * n16;
    partials += (size_t)rhs * gridDim.x; scal += rhs;
    double s = 0.0;
    const int base = blockIdx.x * (BLAS_BLOCK * BLAS_ITEMS) + threadIdx.x;
    V vb[BLAS_ITEMS];
#pragma unroll
    for (int j = 0; j < BLAS_ITEMS; ++j) {
        const int i = base + j * BLAS_BLOCK;
        if (i < n16) vb[j] = b[i];
    }
#pragma unroll
    for (int j = 0; j < BLAS_ITEMS; ++j) {
        const int i = base + j * BLAS_BLOCK;
        if (i < n16) {
            V z; vzero(z);
            x[i] = z; r[i] = vb[j]; p[i] = vb[j];
            s += vdot(vb[j], vb[j]);
        }
    }
    __shared__ double smem[BLAS_BLOCK / 32];
    __shared__ int last;
    if (publish_partial<BLAS_BLOCK>(s, partials, scal, smem, &last)) {
        const double bb = final_sum<BLAS_BLOCK>(partials, (int)gridDim.x, smem);
        if (threadIdx.x == 0) {
            scal->bb = bb; scal->rr = bb; scal->tol2bb = tol * tol * bb;
            scal->pAp = 0.0; scal->alpha = 0.0; scal->beta = 0.0;
            scal->k = 0; scal->maxiter = maxiter;
            int flag = 0;
            if (bb != bb) flag = 3;                               // NaN source
            else if (bb == 0.0 || bb <= tol * tol * bb) flag = 1; // test before the first M application
            else if (maxiter == 0) flag = 2;
            scal->flag = flag;
        }
    }
}

template <typename T>
__global__ void __launch_bounds__(BLAS_BLOCK) cg_update_xr_kernel(
    int n16, const __grid_constant__ RhsPtrs<typename Vec16<T>::type> ptrs, typename Vec16<T>::type *__restrict__ r,
    const typename Vec16<T>::type *__restrict__ p, const typename Vec16<T>::type *__restrict__ Ap,
    double *partials, CgScalars *scal, int chunks)
{
    typedef typename Vec16<T>::type V;
    const int rhs = blockIdx.y;
    scal += rhs;
    if (scal->flag != 0) return;
    V *__restrict__ x = ptrs.x[rhs];
    r += (size_t)rhs * n16; p += (size_t)rhs * n16; Ap += (size_t)rhs * n16;
    partials += (size_t)rhs * gridDim.x;
    const T alpha = (T)scal->alpha;
    double s = 0.0;
    // a block walks `chunks` segments and reduces once (the reduction tail, ~2 us, is then paid
    // by a few thousand blocks instead of every 1024 vectors)
#pragma unroll 1
    for (int ch = 0; ch < chunks; ++ch) {
    const int base = (blockIdx.x * chunks + ch) * (BLAS_BLOCK * BLAS_ITEMS) + threadIdx.x;
    V vx[BLAS_ITEMS], vr[BLAS_ITEMS], vp[BLAS_ITEMS], va[BLAS_ITEMS];
#pragma unroll
    for (int j = 0; j < BLAS_ITEMS; ++j) {
        const int i = base + j * BLAS_BLOCK;
        if (i < n16) { vx[j] = x[i]; vp[j] = p[i]; vr[j] = r[i]; va[j] = Ap[i]; }
    }
#pragma unroll
    for (int j = 0; j < BLAS_ITEMS; ++j) {
        const int i = base + j * BLAS_BLOCK;
        if (i < n16) {
            vaxpy(vx[j], alpha, vp[j]);
            vaxpy(vr[j], -alpha, va[j]);
            x[i] = vx[j]; r[i] = vr[j];
            s += vdot(vr[j], vr[j]);
        }
    }
    }
    __shared__ double smem[BLAS_BLOCK / 32];
    __shared__ int last;
    if (publish_partial<BLAS_BLOCK>(s, partials, scal, smem, &last)) {
        const double rr_new = final_sum<BLAS_BLOCK>(partials, (int)gridDim.x, smem);
        if (threadIdx.x == 0) {
            scal->beta = rr_new / scal->rr;
            scal->rr = rr_new;
            const int k = scal->k + 1;
            scal->k = k;
            if (scal->hist && k <= scal->hist_cap) scal->hist[k - 1] = rr_new;
            if (rr_new != rr_new) scal->flag = 3;
            else if (rr_new <= scal->tol2bb) scal->flag = 1;
            else if (k >= scal->maxiter) scal->flag = 2;
        }
    }
}

template <typename T>
__global__ void __launch_bounds__(BLAS_BLOCK) cg_update_p_kernel(
    int n16, typename Vec16<T>::type *__restrict__ p, const typename Vec16<T>::type *__restrict__ r,
    const CgScalars *scal)
{
    typedef typename Vec16<T>::type V;
    const int rhs = blockIdx.y;
    scal += rhs;
    if (scal->flag != 0) return;
    p += (size_t)rhs * n16; r += (size_t)rhs * n16;
    const T beta = (T)scal->beta;
    const int base = blockIdx.x * (BLAS_BLOCK * BLAS_ITEMS) + threadIdx.x;
    V vp[BLAS_ITEMS], vr[BLAS_ITEMS];
#pragma unroll
    for (int j = 0; j < BLAS_ITEMS; ++j) {
        const int i = base + j * BLAS_BLOCK;
        if (i < n16) { vp[j] = p[i]; vr[j] = r[i]; }
    }
#pragma unroll
    for (int j = 0; j < BLAS_ITEMS; ++j) {
        const int i = base + j * BLAS_BLOCK;
        if (i < n16) { vxpay(vp[j], beta, vr[j]); p[i] = vp[j]; }
    }
}

template <typename T>
__global__ void __launch_bounds__(BLAS_BLOCK) re_dot_kernel(
    int n16, const typename Vec16<T>::type *__restrict__ a, const typename Vec16<T>::type *__restrict__ b,
    double *partials, CgScalars *scal)
{
    double s = 0.0;
    const int base = blockIdx.x * (BLAS_BLOCK * BLAS_ITEMS) + threadIdx.x;
#pragma unroll
    for (int j = 0; j < BLAS_ITEMS; ++j) {
        const int i = base + j * BLAS_BLOCK;
        if (i < n16) s += vdot(a[i], b[i]);
    }
    __shared__ double smem[BLAS_BLOCK / 32];
    __shared__ int last;
    if (publish_partial<BLAS_BLOCK>(s, partials, scal, smem, &last)) {
        const double d = final_sum<BLAS_BLOCK>(partials, (int)gridDim.x, smem);
        if (threadIdx.x == 0) scal->dot = d;
    }
}

} // namespace qcd
