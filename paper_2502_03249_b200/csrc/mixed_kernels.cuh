// Vector kernels of the mixed-precision defect-correction CG (reading R21; PAPER.md:66
// "D and its inversion via CG in single and double precision"):
//
//     x = 0; r = b                                   (fp64)
//     repeat: stop when |r| / |b| <= tol
//             rhs32 = fp32(r / |r|);  e32 = CG_fp32(M32, rhs32, tol_in);  x += |r| fp64(e32)
//             r = b - M x                            (fp64, the TRUE residual)
//
//   mixed_residual : r = b - Mx (or r = b), rr = <r,r> -> scal->dot, deterministic
//   mixed_restrict : rhs32 = (float)(r / sqrt(scal->dot))
//   mixed_prolong  : x += sqrt(scal->dot) * (double) e32
#pragma once
#include "cg_kernels.cuh"

namespace qcd {

__global__ void __launch_bounds__(BLAS_BLOCK) mixed_residual_kernel(
    int n16, const double2 *__restrict__ b, const double2 *__restrict__ Mx /* may be NULL: r = b */,
    double2 *__restrict__ r, double *partials, CgScalars *scal)
{
    double s = 0.0;
    const int base = blockIdx.x * (BLAS_BLOCK * BLAS_ITEMS) + threadIdx.x;
#pragma unroll
    for (int j = 0; j < BLAS_ITEMS; ++j) {
        const int i = base + j * BLAS_BLOCK;
        if (i < n16) {
            double2 v = b[i];
            if (Mx) { const double2 m = Mx[i]; v.x -= m.x; v.y -= m.y; }
            r[i] = v;
            s += vdot(v, v);
        }
    }
    __shared__ double smem[BLAS_BLOCK / 32];
    __shared__ int last;
    if (publish_partial<BLAS_BLOCK>(s, partials, scal, smem, &last)) {
        const double d = final_sum<BLAS_BLOCK>(partials, (int)gridDim.x, smem);
        if (threadIdx.x == 0) scal->dot = d;
    }
}

// one thread per complex number
__global__ void mixed_restrict_kernel(int n, const double2 *__restrict__ r, float2 *__restrict__ rhs32, const CgScalars *scal)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const double s = sqrt(scal->dot);
    const double2 v = r[i];
    float2 o; o.x = (float)(v.x / s); o.y = (float)(v.y / s);
    rhs32[i] = o;
}

__global__ void mixed_prolong_kernel(int n, double2 *__restrict__ x, const float2 *__restrict__ e32, const CgScalars *scal)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const double s = sqrt(scal->dot);
    double2 v = x[i];
    const float2 e = e32[i];
    v.x = __dadd_rn(v.x, __dmul_rn(s, (double)e.x));    // no fma contraction: s * e is rounded first,
    v.y = __dadd_rn(v.y, __dmul_rn(s, (double)e.y));    // as in x += s * e written out
    x[i] = v;
}

} // namespace qcd
