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

// stage: C [nsites][4][9].  dst: 72 planes [parity][mu][k] of Vh.
template <typename C>
__global__ void gauge_scatter_kernel(Lattice L, const C *__restrict__ stage, unsigned i0, unsigned nsites,
                                     C *__restrict__ dst)
{
    const unsigned t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= nsites * 36u) return;
    const unsigned s = t / 36u, mk = t % 36u;       // mk = mu*9 + k
    const unsigned idx = i0 + s;
    const int par = lex_parity(L, idx);
    dst[(size_t)(par * 36 + (int)mk) * L.Vh + (idx >> 1)] = stage[t];
}

template <typename C>
__global__ void gauge_gather_kernel(Lattice L, C *__restrict__ stage, unsigned i0, unsigned nsites,
                                    const C *__restrict__ src)
{
    const unsigned t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= nsites * 36u) return;
    const unsigned s = t / 36u, mk = t % 36u;
    const unsigned idx = i0 + s;
    const int par = lex_parity(L, idx);
    stage[t] = src[(size_t)(par * 36 + (int)mk) * L.Vh + (idx >> 1)];
}

} // namespace qcd
