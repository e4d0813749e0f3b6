// Host canonical layout <-> device SoA even/odd layout (include/qcd.h).
// Pure permutations, run on the device on a staged chunk of consecutive lexicographic sites.
#pragma once
#include "lattice.cuh"

namespace qcd {

__device__ __forceinline__ int lex_parity(const Lattice &L, unsigned idx)
{
    const unsigned x0 = idx % (unsigned)L.N0; idx /= (unsigned)L.N0;
    const unsigned x1 = idx % (unsigned)L.N1; idx /= (unsigned)L.N1;
    const unsigned x2 = idx % (unsigned)L.N2;
    const unsigned x3 = idx / (unsigned)L.N2;
    return (int)((x0 + x1 + x2 + x3) & 1u);
}

// stage: C [nsites][3] for sites i0 .. i0+nsites.  dst_even / dst_odd: 3 planes of Vh, or NULL.
template <typename C>
__global__ void spinor_scatter_kernel(Lattice L, const C *__restrict__ stage, unsigned i0, unsigned nsites,
                                      C *__restrict__ dst_even, C *__restrict__ dst_odd)
{
    const unsigned t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= nsites * 3u) return;
    const unsigned s = t / 3u, c = t % 3u;
    const unsigned idx = i0 + s;
    C *dst = lex_parity(L, idx) ? dst_odd : dst_even;
    if (dst) dst[(size_t)c * L.Vh + (idx >> 1)] = stage[t];
}

// inverse; sites whose parity has no source (NULL) are written as zero.
template <typename C>
__global__ void spinor_gather_kernel(Lattice L, C *__restrict__ stage, unsigned i0, unsigned nsites,
                                     const C *__restrict__ src_even, const C *__restrict__ src_odd)
{
    const unsigned t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= nsites * 3u) return;
    const unsigned s = t / 3u, c = t % 3u;
    const unsigned idx = i0 + s;
    const C *src = lex_parity(L, idx) ? src_odd : src_even;
    C v; v.x = 0; v.y = 0;
    if (src) v = src[(size_t)c * L.Vh + (idx >> 1)];
    stage[t] = v;
}

// Matrix fields.  stage: C [nsites][nmu][9] (row-major 3x3 per site and direction).
// Device: planes [parity][mu < nmu][k = 3 row + col < 3 nrow] of Vh.
//   gauge, full links    : nmu = 4, nrow = 3 (72 planes)
//   gauge, two-row links : nmu = 4, nrow = 2 (48 planes; "we store only the first two rows")
//   colour-matrix field  : nmu = 1, nrow = 3 (18 planes)
template <typename C>
__global__ void matrix_scatter_kernel(Lattice L, const C *__restrict__ stage, unsigned i0, unsigned nsites,
                                      C *__restrict__ dst, int nmu, int nrow)
{
    const unsigned per = (unsigned)nmu * 9u;
    const unsigned t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= nsites * per) return;
    const unsigned s = t / per, mk = t % per;
    const int mu = (int)(mk / 9u), k = (int)(mk % 9u);
    if (k >= 3 * nrow) return;                      // third row of a two-row field is not stored
    const unsigned idx = i0 + s;
    const int par = lex_parity(L, idx);
    dst[(size_t)((par * nmu + mu) * 3 * nrow + k) * L.Vh + (idx >> 1)] = stage[t];
}

// inverse; the third row of a two-row field is reconstructed: row2 = conj(row0 x row1).
template <typename C>
__global__ void matrix_gather_kernel(Lattice L, C *__restrict__ stage, unsigned i0, unsigned nsites,
                                     const C *__restrict__ src, int nmu, int nrow)
{
    const unsigned per = (unsigned)nmu * 9u;
    const unsigned t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= nsites * per) return;
    const unsigned s = t / per, mk = t % per;
    const int mu = (int)(mk / 9u), k = (int)(mk % 9u);
    const unsigned idx = i0 + s;
    const int par = lex_parity(L, idx);
    const C *base = src + (size_t)((par * nmu + mu) * 3 * nrow) * L.Vh + (idx >> 1);
    C v;
    if (k < 3 * nrow) {
        v = base[(size_t)k * L.Vh];
    } else {
        const int j = k - 6, j1 = (j + 1) % 3, j2 = (j + 2) % 3;      // c_j = conj(a_j1 b_j2 - a_j2 b_j1)
        const C a1 = base[(size_t)j1 * L.Vh], a2 = base[(size_t)j2 * L.Vh];
        const C b1 = base[(size_t)(3 + j1) * L.Vh], b2 = base[(size_t)(3 + j2) * L.Vh];
        v.x = a1.x * b2.x - a1.y * b2.y - a2.x * b1.x + a2.y * b1.y;
        v.y = -(a1.x * b2.y + a1.y * b2.x - a2.x * b1.y - a2.y * b1.x);
    }
    stage[t] = v;
}

} // namespace qcd
