// Input transforms of the paper's Dslash variants and precision conversion.
//
//   temporal gauge : "We use gauge fixing to transform the temporal link variables to 1_{3x3} for
//                    all the sites with the temporal coordinate t != 0."  (reading R20)
//                      g(xs, 0) = 1,   g(xs, t) = g(xs, t+1) U_{(xs,t),3}^dagger   t = N3-1 .. 1
//                      U'_{x,mu} = g(x) U_{x,mu} g(x+mu)^dagger,   phi'(x) = g(x) phi(x)
//   colour-matrix field g : cplx [parity 2][k = 3 row + col, 9][Vh]  (QCD_COLOUR_MATRIX)
#pragma once
#include "lattice.cuh"

namespace qcd {

template <typename C>
__device__ __forceinline__ C cmul(const C &a, const C &b)
{
    C r; r.x = a.x * b.x - a.y * b.y; r.y = a.x * b.y + a.y * b.x; return r;
}
template <typename C>
__device__ __forceinline__ C cmul_conj(const C &a, const C &b)      // a * conj(b)
{
    C r; r.x = a.x * b.x + a.y * b.y; r.y = a.y * b.x - a.x * b.y; return r;
}
template <typename C>
__device__ __forceinline__ void cadd(C &a, const C &b) { a.x += b.x; a.y += b.y; }

// r = a * b^dagger
template <typename C>
__device__ __forceinline__ void mat_mul_dag(C r[9], const C a[9], const C b[9])
{
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
        for (int j = 0; j < 3; ++j) {
            C s = cmul_conj(a[3 * i + 0], b[3 * j + 0]);
            cadd(s, cmul_conj(a[3 * i + 1], b[3 * j + 1]));
            cadd(s, cmul_conj(a[3 * i + 2], b[3 * j + 2]));
            r[3 * i + j] = s;
        }
}
// r = a * b
template <typename C>
__device__ __forceinline__ void mat_mul(C r[9], const C a[9], const C b[9])
{
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
        for (int j = 0; j < 3; ++j) {
            C s = cmul(a[3 * i + 0], b[0 + j]);
            cadd(s, cmul(a[3 * i + 1], b[3 + j]));
            cadd(s, cmul(a[3 * i + 2], b[6 + j]));
            r[3 * i + j] = s;
        }
}

// One thread per spatial site xs = (x0, x1, x2): walks the time line downwards from t = N3-1.
// U: full 18-real links (72 planes).  G: colour-matrix field.
template <typename C>
__global__ void temporal_gauge_g_kernel(Lattice L, const C *__restrict__ U, C *__restrict__ G)
{
    const unsigned vs = (unsigned)(L.N0 * L.N1 * L.N2);
    const unsigned xs = blockIdx.x * blockDim.x + threadIdx.x;
    if (xs >= vs) return;
    const unsigned x0 = xs % (unsigned)L.N0, x1 = (xs / (unsigned)L.N0) % (unsigned)L.N1, x2 = xs / (unsigned)(L.N0 * L.N1);
    const size_t Vh = (size_t)L.Vh;
    C g[9];
#pragma unroll
    for (int k = 0; k < 9; ++k) { g[k].x = (k % 4 == 0) ? 1 : 0; g[k].y = 0; }
    {
        const int par = (int)((x0 + x1 + x2) & 1u);
        const size_t cb = xs >> 1;
#pragma unroll
        for (int k = 0; k < 9; ++k) G[(size_t)(par * 9 + k) * Vh + cb] = g[k];
    }
    for (int t = L.N3 - 1; t >= 1; --t) {
        const unsigned idx = xs + vs * (unsigned)t;
        const int par = (int)((x0 + x1 + x2 + (unsigned)t) & 1u);
        const size_t cb = idx >> 1;
        C u[9], n[9];
#pragma unroll
        for (int k = 0; k < 9; ++k) u[k] = U[(size_t)(par * 36 + 27 + k) * Vh + cb];      // mu = 3
        mat_mul_dag(n, g, u);
#pragma unroll
        for (int k = 0; k < 9; ++k) { g[k] = n[k]; G[(size_t)(par * 9 + k) * Vh + cb] = n[k]; }
    }
}

// One thread per site of one parity: U'_{x,mu} = g(x) U_{x,mu} g(x+mu)^dagger for mu = 0..3.
// fix_time != 0: the time links with x3 != 0 are written as the exact identity (they are the
// identity up to rounding by construction of g).
template <typename C>
__global__ void gauge_transform_kernel(Lattice L, int parity, const C *__restrict__ U, const C *__restrict__ G,
                                       C *__restrict__ Uout, int fix_time)
{
    const int cb = blockIdx.x * blockDim.x + threadIdx.x;
    if (cb >= L.Vh) return;
    const size_t Vh = (size_t)L.Vh;
    const SiteGeom sg = site_geometry(L, parity, cb);
    C g[9];
#pragma unroll
    for (int k = 0; k < 9; ++k) g[k] = G[(size_t)(parity * 9 + k) * Vh + cb];
#pragma unroll
    for (int mu = 0; mu < 4; ++mu) {
        C u[9], gn[9], t[9], r[9];
#pragma unroll
        for (int k = 0; k < 9; ++k) u[k] = U[(size_t)(parity * 36 + mu * 9 + k) * Vh + cb];
#pragma unroll
        for (int k = 0; k < 9; ++k) gn[k] = G[(size_t)((1 - parity) * 9 + k) * Vh + sg.nf[mu]];
        mat_mul(t, g, u);
        mat_mul_dag(r, t, gn);
        if (mu == 3 && fix_time && sg.x3 != 0) {
#pragma unroll
            for (int k = 0; k < 9; ++k) { r[k].x = (k % 4 == 0) ? 1 : 0; r[k].y = 0; }
        }
#pragma unroll
        for (int k = 0; k < 9; ++k) Uout[(size_t)(parity * 36 + mu * 9 + k) * Vh + cb] = r[k];
    }
}

// out(x) = g(x) in(x)  (dagger: g(x)^dagger in(x)) on the sites of one parity.
template <typename C>
__global__ void spinor_rotate_kernel(Lattice L, int parity, const C *__restrict__ G, const C *__restrict__ in,
                                     C *__restrict__ out, int dagger)
{
    const int cb = blockIdx.x * blockDim.x + threadIdx.x;
    if (cb >= L.Vh) return;
    const size_t Vh = (size_t)L.Vh;
    C g[9], p[3];
#pragma unroll
    for (int k = 0; k < 9; ++k) g[k] = G[(size_t)(parity * 9 + k) * Vh + cb];
#pragma unroll
    for (int c = 0; c < 3; ++c) p[c] = in[(size_t)c * Vh + cb];
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        C s; s.x = 0; s.y = 0;
#pragma unroll
        for (int b = 0; b < 3; ++b) cadd(s, dagger ? cmul_conj(p[b], g[3 * b + a]) : cmul(g[3 * a + b], p[b]));
        out[(size_t)a * Vh + cb] = s;
    }
}

// dst[i] = (D) src[i] over n reals (round to nearest): fp64 -> fp32 copies of links and sources
// (reading R9: "fp32 inputs are the round-to-nearest of the fp64 arrays").
template <typename S, typename D>
__global__ void convert_kernel(size_t n, const S *__restrict__ src, D *__restrict__ dst)
{
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) dst[i] = (D)src[i];
}

} // namespace qcd
