// Persistent CG for lattices that live in the L2 ("global
// reductions which have higher latencies ... more pronounced for smaller lattice sizes").
//
// At 16^4 one CG iteration of the multi-kernel path is four kernels of 4-14 us, of which ~4 us
// each are the tail of a reduction (ticket, last block re-reads the partials) and ~1.5 us each a
// launch gap.  Here ONE cooperative kernel runs the whole solve: every block is resident, the
// phases of an iteration are separated by grid-wide barriers, and after the barrier EVERY block
// sums the per-block partials itself in index order -- no last-block serialisation, no host
// round trip, and alpha, beta, rr, k and the stop decision are bitwise identical in all blocks,
// so the control flow stays uniform across the grid.
//
//   phase 1  p' = r + beta p  (each thread for its own even site, into the OTHER p buffer) and
//            t  = D_oe p'  with p' formed on the fly at the eight neighbours from r and p: the
//            direction update needs no pass and no barrier of its own        | grid barrier
//   phase 2  Ap = m^2 p' - D_eo t;  partial Re<p',Ap> per block               | grid barrier
//            alpha = rr / sum(partials)           (every block, same order)
//   phase 3  x += alpha p';  r -= alpha Ap;  partial <r,r>                    | grid barrier
//            beta = rr' / rr;  k += 1;  stop test (every block)
//
// (p' = fma(beta, p, r) gives the same bits wherever it is evaluated; beta = 0 in the first
// iteration, where p = r = b.)
//
// Fields written inside the kernel (p, t, Ap, r, x) are read with L2-coherent loads (ld.global.cg),
// never through the read-only path; links are read-only and keep it.  The arithmetic per site is
// that of dslash_kernel (same helpers, same order).
#pragma once
#include <cooperative_groups.h>

#include "cg_kernels.cuh"
#include "dslash.cuh"

namespace qcd {

template <typename T>
struct PersistArgs {
    typedef typename Cplx<T>::type C;
    Lattice L;
    const C *U;
    C *x, *r, *p, *p2, *Ap, *t; // even half-fields (p and p2 alternate as direction vector), t odd
    T m2;
    double *partials;          // 2 x gridDim.x doubles: [0] Re<p,Ap>, [1] <r,r>
    CgScalars *scal;           // initialised by cg_init_kernel (rr, bb, tol2bb, k, maxiter, flag)
    unsigned long long *timeline;   // measurement hook (qcd_cg_timeline), NULL in normal solves: %globaltimer stamps of the
                                    // first TIMELINE_ITERS iterations, [block 0 | last block][iteration][TIMELINE_STAMPS]
};

// Stamps per iteration: 0 phase 1 starts, 1 phase 1 done, 2 past barrier 1, 3 phase 2 + block partial done, 4 past
// barrier 2, 5 <p,Ap> summed (alpha known), 6 phase 3 + block partial done, 7 past barrier 3, 8 <r,r> summed (beta known).
enum { TIMELINE_ITERS = 64, TIMELINE_STAMPS = 9 };

__device__ __forceinline__ unsigned long long global_ns()
{
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    return t;
}

__device__ __forceinline__ double2 ld_coherent(const double2 *p) { return __ldcg(p); }
__device__ __forceinline__ float2 ld_coherent(const float2 *p) { return __ldcg(p); }

// acc = (D in)(cb) for the site cb of `parity`; `in` may have been written earlier in this kernel
// FUSE: the input vector is r + beta * in, formed at every neighbour on the fly
template <typename T, int NROW, int TG, bool FUSE>
__device__ __forceinline__ void persistent_site(typename Cplx<T>::type acc[3], const Lattice &L, int parity, int cb,
                                                const typename Cplx<T>::type *U, const typename Cplx<T>::type *in,
                                                const typename Cplx<T>::type *r = nullptr, T beta = (T)0)
{
    typedef typename Cplx<T>::type C;
    const size_t Vh = (size_t)L.Vh;
    const SiteGeom g = site_geometry(L, parity, cb);
    const uint64_t pol = l2_policy_evict_last();             // everything is meant to stay in the L2 here
    const C *Uf = U + (size_t)(parity * 12 * NROW) * Vh + cb;
    const C *Ub = U + (size_t)((1 - parity) * 12 * NROW) * Vh;
    acc[0].x = acc[0].y = acc[1].x = acc[1].y = acc[2].x = acc[2].y = (T)0;
#pragma unroll
    for (int mu = 0; mu < 4; ++mu) {
        const bool unit_f = TG && mu == 3 && g.x3 != 0;
        const bool unit_b = TG && mu == 3 && g.x3 != 1;
        C uf[9], ub[9], pf[3], pb[3];
        if (!unit_f) load_link<NROW, C>(uf, Uf + (size_t)(mu * 3 * NROW) * Vh, Vh, pol);
        if (!unit_b) load_link<NROW, C>(ub, Ub + (size_t)(mu * 3 * NROW) * Vh + g.nb[mu], Vh, pol);
        const unsigned nf = g.sf[mu] < 0.f ? 1u : 0u, nb = g.sb[mu] < 0.f ? 1u : 0u;
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            pf[c] = ld_coherent(in + (size_t)c * Vh + g.nf[mu]);
            pb[c] = ld_coherent(in + (size_t)c * Vh + g.nb[mu]);
            if (FUSE) {
                const C rf = ld_coherent(r + (size_t)c * Vh + g.nf[mu]), rb = ld_coherent(r + (size_t)c * Vh + g.nb[mu]);
                pf[c].x = fma(beta, pf[c].x, rf.x); pf[c].y = fma(beta, pf[c].y, rf.y);
                pb[c].x = fma(beta, pb[c].x, rb.x); pb[c].y = fma(beta, pb[c].y, rb.y);
            }
        }
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            pf[c].x = flip_sign(pf[c].x, nf); pf[c].y = flip_sign(pf[c].y, nf);
            pb[c].x = flip_sign(pb[c].x, nb); pb[c].y = flip_sign(pb[c].y, nb);
        }
        if (!unit_f) { if (NROW == 2) reconstruct_third_row<C>(uf); mat_vec_acc<T, C>(acc, uf, pf); } else vec_acc<C>(acc, pf);
        if (!unit_b) { if (NROW == 2) reconstruct_third_row<C>(ub); matdag_vec_acc<T, C>(acc, ub, pb); } else vec_acc<C>(acc, pb);
    }
}

enum { PERSIST_BLOCK = 128 };

// sum of partials[0 .. n) in an order that depends only on n and the block size; the result is
// returned in EVERY thread of the block (identical in every block of the grid)
__device__ __forceinline__ double persistent_total(const double *partials, int n, double *smem /* PERSIST_BLOCK/32 + 1 */)
{
    double s = 0.0;
    for (int i = threadIdx.x; i < n; i += PERSIST_BLOCK) s += __ldcg(partials + i);
    __syncthreads();
    const double tot = block_sum<PERSIST_BLOCK>(s, smem);
    if (threadIdx.x == 0) smem[PERSIST_BLOCK / 32] = tot;
    __syncthreads();
    return smem[PERSIST_BLOCK / 32];
}

template <typename T, int NROW, int TG>
__global__ void __launch_bounds__(PERSIST_BLOCK, 3) cg_persistent_kernel(const PersistArgs<T> a)
{
    typedef typename Cplx<T>::type C;
    namespace cg = cooperative_groups;
    cg::grid_group grid = cg::this_grid();
    __shared__ double smem[PERSIST_BLOCK / 32 + 1];
    const int Vh = a.L.Vh;
    const size_t sVh = (size_t)Vh;
    const int gthreads = gridDim.x * PERSIST_BLOCK;
    const int gtid = blockIdx.x * PERSIST_BLOCK + threadIdx.x;
    const int nblocks = (int)gridDim.x;
    double *part_pAp = a.partials, *part_rr = a.partials + nblocks;

    // the recurrence state, replicated: every thread of every block holds the same values
    double rr = a.scal->rr;
    const double tol2bb = a.scal->tol2bb;
    const int maxiter = a.scal->maxiter;
    int k = a.scal->k, flag = a.scal->flag;
    double alpha = 0.0, beta = 0.0, pAp = 0.0;

    // timeline: thread 0 of block 0 and of the last block stamp the phase boundaries of the first iterations
    unsigned long long *tl = nullptr;
    if (a.timeline && threadIdx.x == 0 && (blockIdx.x == 0 || blockIdx.x == gridDim.x - 1))
        tl = a.timeline + (blockIdx.x == 0 ? 0 : TIMELINE_ITERS * TIMELINE_STAMPS);
    int it = 0;
#define QCD_STAMP(i) do { if (tl && it < TIMELINE_ITERS) tl[it * TIMELINE_STAMPS + (i)] = global_ns(); } while (0)

    C *p_old = a.p, *p_cur = a.p2;
    while (flag == 0) {
        QCD_STAMP(0);
        // phase 1: p_cur = r + beta p_old (own even site), t = D_oe p_cur (formed on the fly at the neighbours)
        const T be = (T)beta;
        for (int cb = gtid; cb < Vh; cb += gthreads) {
            C acc[3];
            persistent_site<T, NROW, TG, true>(acc, a.L, 1, cb, a.U, p_old, a.r, be);
            // all six loads before the first store: one L2 round trip instead of three (a load issued after a
            // store that may alias it waits for that store)
            C vp[3], vr[3];
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                vp[c] = ld_coherent(p_old + (size_t)c * sVh + cb);
                vr[c] = ld_coherent(a.r + (size_t)c * sVh + cb);
            }
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                a.t[(size_t)c * sVh + cb] = acc[c];
                vp[c].x = fma(be, vp[c].x, vr[c].x); vp[c].y = fma(be, vp[c].y, vr[c].y);
                p_cur[(size_t)c * sVh + cb] = vp[c];
            }
        }
        QCD_STAMP(1);
        grid.sync();
        QCD_STAMP(2);
        // phase 2: Ap = m^2 p - D_eo t, partial Re<p,Ap>
        double dot = 0.0;
        for (int cb = gtid; cb < Vh; cb += gthreads) {
            C acc[3];
            persistent_site<T, NROW, TG, false>(acc, a.L, 0, cb, a.U, a.t);
            C vv[3];
#pragma unroll
            for (int c = 0; c < 3; ++c) vv[c] = ld_coherent(p_cur + (size_t)c * sVh + cb);
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                C o;
                o.x = fma(a.m2, vv[c].x, -acc[c].x);
                o.y = fma(a.m2, vv[c].y, -acc[c].y);
                a.Ap[(size_t)c * sVh + cb] = o;
                dot += (double)vv[c].x * (double)o.x + (double)vv[c].y * (double)o.y;
            }
        }
        {
            const double s = block_sum<PERSIST_BLOCK>(dot, smem);
            if (threadIdx.x == 0) part_pAp[blockIdx.x] = s;
        }
        QCD_STAMP(3);
        grid.sync();
        QCD_STAMP(4);
        pAp = persistent_total(part_pAp, nblocks, smem);
        QCD_STAMP(5);
        if (!(pAp > 0.0)) { flag = 3; break; }                     // breakdown: uniform across the grid
        alpha = rr / pAp;
        // phase 3: x += alpha p, r -= alpha Ap, partial <r,r>   (elementwise over 3 Vh complex numbers)
        const T al = (T)alpha;
        double nrm = 0.0;
        for (int i = gtid; i < 3 * Vh; i += gthreads) {
            C vx = ld_coherent(a.x + i), vr = ld_coherent(a.r + i);
            const C vp = ld_coherent(p_cur + i), va = ld_coherent(a.Ap + i);
            vx.x = fma(al, vp.x, vx.x); vx.y = fma(al, vp.y, vx.y);
            vr.x = fma(-al, va.x, vr.x); vr.y = fma(-al, va.y, vr.y);
            a.x[i] = vx; a.r[i] = vr;
            nrm += (double)vr.x * (double)vr.x + (double)vr.y * (double)vr.y;
        }
        {
            __syncthreads();
            const double s = block_sum<PERSIST_BLOCK>(nrm, smem);
            if (threadIdx.x == 0) part_rr[blockIdx.x] = s;
        }
        QCD_STAMP(6);
        grid.sync();
        QCD_STAMP(7);
        const double rr_new = persistent_total(part_rr, nblocks, smem);
        QCD_STAMP(8);
        ++it;
        beta = rr_new / rr;
        rr = rr_new;
        k += 1;
        if (gtid == 0) {                                           // residual history (qcd_cg_history)
            double *const hist = a.scal->hist;
            if (hist && k <= a.scal->hist_cap) hist[k - 1] = rr_new;
        }
        if (rr_new != rr_new) flag = 3;
        else if (rr_new <= tol2bb) flag = 1;
        else if (k >= maxiter) flag = 2;
        if (flag != 0) break;
        { C *tmp = p_old; p_old = p_cur; p_cur = tmp; }            // the direction just used becomes "p" of the next update
    }
#undef QCD_STAMP
    if (gtid == 0) {
        CgScalars *s = a.scal;
        s->rr = rr; s->pAp = pAp; s->alpha = alpha; s->beta = beta; s->k = k; s->flag = flag;
    }
}

} // namespace qcd
