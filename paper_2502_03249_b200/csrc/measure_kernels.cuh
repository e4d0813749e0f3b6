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

// Streaming ceiling of the BULK-COPY (TMA) path (measurement hook): `producers` warps per block move `copies` tensor-map boxes of
// `rows` planes x 128 consecutive elements (2 KB per plane: a block's sites in one SoA plane, the access pattern of the multi-vector
// Dslash) per stage into a ring of S shared-memory stages; four consumer warps read every byte back from shared memory.
// What it answers: how many requested bytes per second can a SM take in through the copy engine, which holds neither registers nor
// LSU miss entries for the data in flight -- against the 9-11 TB/s at which every LSU-fed Dslash kernel saturates.
enum { BULK_CONSUMERS = 128, BULK_MAX_STAGES = 12, BULK_RUN = 128, BULK_MAX_PRODUCERS = 4 };
__global__ void __launch_bounds__(BULK_CONSUMERS + 32 * BULK_MAX_PRODUCERS) stream_bulk_kernel(const __grid_constant__ CUtensorMap tmap, int nplanes, int rows, int copies,
                                                                                                 int hops, int S, size_t ngroups, double2 *sink)
{
    extern __shared__ __align__(128) unsigned char bulk_smem[];
    __shared__ __align__(8) unsigned long long full[BULK_MAX_STAGES], empty[BULK_MAX_STAGES];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const unsigned box_bytes = (unsigned)rows * BULK_RUN * 16u, stage_bytes = box_bytes * (unsigned)copies;
    const int npw = blockDim.x / 32 - BULK_CONSUMERS / 32;
    if (threadIdx.x == 0) {
        for (int s = 0; s < S; ++s) { mbar_init(&full[s], npw); mbar_init(&empty[s], BULK_CONSUMERS / 32); }
        mbar_init_fence();
    }
    __syncthreads();
    if (warp >= BULK_CONSUMERS / 32) {
        const uint64_t pol = l2_policy_evict_first();
        const int pw = warp - BULK_CONSUMERS / 32;
        const int j_lo = copies * pw / npw, j_hi = copies * (pw + 1) / npw;
        unsigned it = 0;
        for (size_t g = blockIdx.x; g < ngroups; g += gridDim.x) {
            for (int k = 0; k < hops; ++k, ++it) {
                const unsigned s = it % (unsigned)S, use = it / (unsigned)S;
                if (use > 0) mbar_wait(&empty[s], (use & 1u) ^ 1u);
                if (lane == 0) {
                    mbar_arrive_expect_tx(&full[s], (unsigned)(j_hi - j_lo) * box_bytes);
                    for (int j = j_lo; j < j_hi; ++j) {
                        const int row0 = ((k * copies + j) * rows) % (nplanes - rows + 1);
                        tensor_copy_g2s(bulk_smem + (size_t)s * stage_bytes + (size_t)j * box_bytes, &tmap, (int)(g * BULK_RUN * 2), row0, &full[s], pol);
                    }
                }
                __syncwarp();
            }
        }
    } else {
        unsigned it = 0;
        unsigned long long x = 0;
        const int pps = rows * copies;
        for (size_t g = blockIdx.x; g < ngroups; g += gridDim.x) {
            for (int k = 0; k < hops; ++k, ++it) {
                const unsigned s = it % (unsigned)S, use = it / (unsigned)S;
                mbar_wait(&full[s], use & 1u);
                const double2 *st = reinterpret_cast<const double2 *>(bulk_smem + (size_t)s * stage_bytes);
                for (int j0 = 0; j0 < pps; j0 += 8) {
                    double2 v[8];
#pragma unroll
                    for (int j = 0; j < 8; ++j) v[j] = st[(size_t)(j0 + j < pps ? j0 + j : 0) * BULK_RUN + threadIdx.x];
#pragma unroll
                    for (int j = 0; j < 8; ++j) x ^= (unsigned long long)__double_as_longlong(v[j].x) ^ (unsigned long long)__double_as_longlong(v[j].y);
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(&empty[s]);
            }
        }
        if (x == 0xfff7a5a5deadbeefULL) *sink = make_double2(0.0, 0.0);
    }
}

} // namespace qcd
