// Read-only streaming ceiling (SURVEY.md Sec. 7 "hard parts": a half-Dslash is 96 % reads, so
// the denominator that says how close it is to what the memory system can deliver is a
// kernel made of nothing but the Dslash's own link loads -- 16-byte, fully coalesced,
// read-only path, no L1 allocation, L2 evict_first -- not a copy).  Measurement hook only:
// it computes nothing the method needs.
#pragma once
#include "lattice.cuh"

namespace qcd {

enum { STREAM_BLOCK = 256, STREAM_LOADS = 8 };   // 8 independent 16-byte loads in flight per thread

__global__ void __launch_bounds__(STREAM_BLOCK) stream_read_kernel(const double2 *__restrict__ p, size_t n16, double2 *sink)
{
    const uint64_t pol = l2_policy_evict_first();
    const size_t base = (size_t)blockIdx.x * (STREAM_BLOCK * STREAM_LOADS) + threadIdx.x;
    double2 v[STREAM_LOADS];
#pragma unroll
    for (int k = 0; k < STREAM_LOADS; ++k) {
        const size_t i = base + (size_t)k * STREAM_BLOCK;
        v[k] = i < n16 ? ld_stream(p + i, pol) : make_double2(0.0, 0.0);
    }
    unsigned long long x = 0;
#pragma unroll
    for (int k = 0; k < STREAM_LOADS; ++k)
        x ^= (unsigned long long)__double_as_longlong(v[k].x) ^ (unsigned long long)__double_as_longlong(v[k].y);
    // a NaN pattern no finite field carries in every word: keeps the loads alive, never stores
    if (x == 0xfff7a5a5deadbeefULL) *sink = v[0];
}

// The same loads over a field that FITS the L2, `passes` times inside ONE launch (grid-stride; a launch per pass
// would time the launch, not the L2, at 16^4): the denominator of the small-lattice kernels, whose operands are
// served by the L2 and not by HBM.  L1 is bypassed (no_allocate), so every pass is L2 -> SM traffic.
__global__ void __launch_bounds__(STREAM_BLOCK) stream_read_resident_kernel(const double2 *__restrict__ p, size_t n16, int passes, double2 *sink)
{
    const uint64_t pol = l2_policy_evict_last();
    const size_t stride = (size_t)gridDim.x * (STREAM_BLOCK * STREAM_LOADS);
    unsigned long long x = 0;
    for (int pass = 0; pass < passes; ++pass) {
        for (size_t base = (size_t)blockIdx.x * (STREAM_BLOCK * STREAM_LOADS) + threadIdx.x; base < n16; base += stride) {
            double2 v[STREAM_LOADS];
#pragma unroll
            for (int k = 0; k < STREAM_LOADS; ++k) {
                const size_t i = base + (size_t)k * STREAM_BLOCK;
                v[k] = i < n16 ? ld_stream(p + i, pol) : make_double2(0.0, 0.0);
            }
#pragma unroll
            for (int k = 0; k < STREAM_LOADS; ++k)
                x ^= (unsigned long long)__double_as_longlong(v[k].x) ^ (unsigned long long)__double_as_longlong(v[k].y);
        }
    }
    if (x == 0xfff7a5a5deadbeefULL) *sink = make_double2(0.0, 0.0);
}

// Streaming ceiling for a MIX of read and write streams (measurement hook): every thread reads 16 bytes from each of
// `nread` planes of Vh elements and writes 16 bytes to each of `nwrite` planes, all at its own index -- the DRAM access
// pattern of a multi-vector half-Dslash (links + n input vectors read once, n output vectors written) with the stencil,
// the neighbour reads and the arithmetic taken out.  What it answers: is the 4.6 TB/s that the n = 8 kernels move the
// memory system's rate for 26 % writes over ~100 concurrent streams, or the kernels' own limit?
enum { MIX_BLOCK = 128, MIX_BATCH = 8 };
__global__ void __launch_bounds__(MIX_BLOCK) stream_mix_kernel(const double2 *__restrict__ src, double2 *__restrict__ dst,
                                                               size_t plane, int nread, int nwrite)
{
    const size_t i = (size_t)blockIdx.x * MIX_BLOCK + threadIdx.x;
    if (i >= plane) return;
    const uint64_t pol = l2_policy_evict_first();
    double2 acc = make_double2(0.0, 0.0);
    for (int k0 = 0; k0 < nread; k0 += MIX_BATCH) {
        double2 v[MIX_BATCH];
#pragma unroll
        for (int j = 0; j < MIX_BATCH; ++j) v[j] = k0 + j < nread ? ld_stream(src + (size_t)(k0 + j) * plane + i, pol) : make_double2(0.0, 0.0);
#pragma unroll
        for (int j = 0; j < MIX_BATCH; ++j) { acc.x += v[j].x; acc.y += v[j].y; }
    }
    for (int k = 0; k < nwrite; ++k) dst[(size_t)k * plane + i] = acc;
}

} // namespace qcd
