// Deterministic two-stage reduction (north_star (c): "a deterministic two-stage warp-shuffle
// reduction for dot products"; "dot product involving global reductions").
//
// Stage 1: every block reduces its threads' double partial sums in a fixed order
//          (warp shuffle tree, then the warp sums through shared memory in warp order) and
//          writes ONE double to partials[blockIdx.x].
// Stage 2: the block that takes the last ticket (an integer atomic, the only atomic used)
//          re-reads all partials from L2 and sums them in an order that depends only on the
//          grid size, never on which block arrived last.  No floating-point atomics, so
//          results are bitwise reproducible run to run.
#pragma once
#include <cuda_runtime.h>

namespace qcd {

// Largest number of right-hand sides handled by one launch (NMULTI).
enum { MAXRHS = 8 };

// CG recurrence state, resident on the device (north_star (d)); one per right-hand side.
struct CgScalars {
    double rr;        // <r,r> of the current residual
    double bb;        // <b,b>
    double pAp;       // <p, M p>
    double alpha;     // rr / pAp
    double beta;      // rr_new / rr
    double tol2bb;    // tol^2 * bb  (stop when rr <= tol2bb)
    double dot;       // result slot of qcd_re_dot
    int k;            // M applications done
    int maxiter;
    int flag;         // 0 running, 1 converged, 2 maxiter reached, 3 breakdown
    unsigned ticket;  // top-level last-block ticket, wraps to 0 by itself (atomicInc)
    unsigned *l1;     // first-level tickets, one per group of TICKET_GROUP blocks (set once by qcd_init)
    double *hist;     // residual history: hist[j] = <r,r> after j + 1 M applications, j < hist_cap (set once by qcd_init; may be NULL)
    int hist_cap;
};

__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    return v;
}

// Sum over the block; the result is valid in thread 0.  All threads must call it.
template <int BLOCK>
__device__ __forceinline__ double block_sum(double v, double *smem /* BLOCK/32 doubles */)
{
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    v = warp_sum(v);
    if (lane == 0) smem[w] = v;
    __syncthreads();
    double s = 0.0;
    if (threadIdx.x == 0) {
#pragma unroll
        for (int i = 0; i < BLOCK / 32; ++i) s += smem[i];
    }
    return s;
}

// Two-level ticket.  65 536 blocks taking ONE ticket serialise on one L2 atomic unit (~2.3 ns each:
// 0.15 ms per reduction kernel at 64^4, measured as the difference between the epilogue kernels
// with and without the reduction).  Blocks therefore take a ticket of their group of TICKET_GROUP
// blocks (distinct addresses, spread over the L2 slices), and only the last block of a group takes
// the top-level one.  Both wrap to 0 by themselves.  Called by ONE thread after it has written its
// partial; returns true in the last block of the grid.  Which block that is does not affect the
// result: the last block re-reads all partials in index order.
enum { TICKET_GROUP = 64 };
__device__ __forceinline__ bool take_ticket(unsigned *top, unsigned *l1)
{
    __threadfence();
    const unsigned nb = gridDim.x, g = blockIdx.x / TICKET_GROUP;
    const unsigned ngroups = (nb + TICKET_GROUP - 1) / TICKET_GROUP;
    const unsigned gsize = (g == ngroups - 1) ? nb - g * TICKET_GROUP : (unsigned)TICKET_GROUP;
    if (atomicInc(l1 + g, gsize - 1) != gsize - 1) return false;
    __threadfence();
    return atomicInc(top, ngroups - 1) == ngroups - 1;
}

// Stage 1 + ticket.  Returns true (in every thread of exactly one block) when this block is
// the last to finish; that block must then call final_sum.
template <int BLOCK>
__device__ __forceinline__ bool publish_partial(double v, double *partials, CgScalars *scal, double *smem, int *smem_flag)
{
    const double s = block_sum<BLOCK>(v, smem);
    if (threadIdx.x == 0) {
        partials[blockIdx.x] = s;
        *smem_flag = take_ticket(&scal->ticket, scal->l1);
    }
    __syncthreads();
    return *smem_flag != 0;
}

// Stage 1 + ticket for N sums at once (multiple right-hand sides): sum r of
// this block goes to partials[r * stride + blockIdx.x]; ONE ticket serves all N.  For N = 1
// the summation order is that of publish_partial.  smem holds N * BLOCK/32 doubles.
template <int BLOCK, int N>
__device__ __forceinline__ bool publish_partials(const double (&v)[N], double *partials, size_t stride,
                                                 CgScalars *scal, double *smem, int *smem_flag)
{
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
#pragma unroll
    for (int r = 0; r < N; ++r) {
        const double s = warp_sum(v[r]);
        if (lane == 0) smem[r * (BLOCK / 32) + w] = s;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
#pragma unroll
        for (int r = 0; r < N; ++r) {
            double s = 0.0;
#pragma unroll
            for (int i = 0; i < BLOCK / 32; ++i) s += smem[r * (BLOCK / 32) + i];
            partials[(size_t)r * stride + blockIdx.x] = s;
        }
        *smem_flag = take_ticket(&scal->ticket, scal->l1);
    }
    __syncthreads();
    return *smem_flag != 0;
}

// Stage 2: fixed-order sum of partials[0 .. n).  Result valid in thread 0.
template <int BLOCK>
__device__ __forceinline__ double final_sum(const double *partials, int n, double *smem)
{
    __threadfence();
    double s = 0.0;
    for (int i = threadIdx.x; i < n; i += BLOCK) s += __ldcg(partials + i);
    __syncthreads();                       // smem is reused
    return block_sum<BLOCK>(s, smem);
}

} // namespace qcd
