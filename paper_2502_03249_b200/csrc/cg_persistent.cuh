// Persistent CG for lattices that live in the L2 ("global
// reductions which have higher latencies ... more pronounced for smaller lattice sizes").
//
// At 16^4 one CG iteration of the multi-kernel path is four kernels of 4-14 us, of which ~4 us
// each are the tail of a reduction (ticket, last block re-reads the partials) and ~1.5 us each a
// launch gap.  Here ONE cooperative kernel runs the whole solve: every block is resident, the
// phases of an iteration are separated by grid-wide barriers that carry the reduction, and EVERY
// block ends a barrier with the same sum -- no last-block serialisation, no host round trip, and
// alpha, beta, rr, k and the stop decision are bitwise identical in all blocks, so the control
// flow stays uniform across the grid.
//
//   phase 1  p' = r + beta p  (for the own even site, into the OTHER p buffer) and
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
// What the phase timeline showed (qcd_cg_timeline_*, profiles/r02_small_lattice_timeline.md) and what this
// file does about it:
//   * up to 12^4 a phase is a chain of L2 round trips (~0.3 us each), not bandwidth: under a 168-register cap ptxas walks
//     the four directions one after the other (2.2 us per Dslash phase at 4^4 ... 12^4 alike).  A thread therefore gets the
//     whole register file's share of ONE 256-thread block per SM (255 registers: all loads of a site in flight at once); an
//     earlier version split a site over a quad of lanes instead, which the wider cap made unnecessary (see PersistBlock);
//   * a cooperative-groups grid.sync() costs 1.2-1.8 us and the re-read of the per-block partials after it
//     another 0.4-0.9 us: 6 of the 15.8 us of a 16^4 iteration and of the 11 us of an 8^4 one.  Two hand-written
//     replacements (every block polling every block's tagged slot, by all threads and by one warp with a 128-byte
//     line per slot) were SLOWER from 4 blocks on (2.7 us at 4 blocks, 4-5 us at 64, 7-10 us at 340: the polls
//     of an all-gather grow with the square of the grid) and grid.sync() stays for grids of several clusters.
//     Lattices of up to 2048 sites per parity (8^4) run as ONE thread-block cluster of up to 16 CTAs x 128
//     threads instead: the barrier is the hardware barrier.cluster (release / acquire at cluster scope), and the
//     partial sums are exchanged through distributed shared memory -- every CTA stores its partial into every
//     peer's slot before it arrives and sums the 16 local slots in rank order after the wait.  In that shape the
//     vectors the neighbours read (r, both direction buffers, t) live in the CTAs' shared memory as well and are
//     gathered with ld.shared::cluster, x and Ap stay in registers for the whole solve (cg_cluster_body below).
//
// Fields written inside the kernel (p, t, Ap, r, x) are read with L2-coherent loads (ld.global.cg),
// never through the read-only path; links are read-only and keep it.
#pragma once

#include <cooperative_groups.h>

#include "cg_kernels.cuh"
#include "dslash.cuh"

namespace qcd {

// ------------------------------------------------------------------------------------------
// cluster primitives (PTX ISA: barrier.cluster, mapa, st.shared::cluster)
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ unsigned cluster_ctarank() { unsigned r; asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r)); return r; }
__device__ __forceinline__ unsigned cluster_nctarank() { unsigned r; asm volatile("mov.u32 %0, %%cluster_nctarank;" : "=r"(r)); return r; }
// arrive with release, wait with acquire, both at cluster scope: the writes (global and shared) of every thread of the
// cluster before its arrive are visible to every thread of the cluster after its wait
__device__ __forceinline__ void cluster_barrier()
{
    asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");
    asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");
}
// store a double into the shared memory of CTA `rank` of the cluster, at the address that `local` has in this CTA
__device__ __forceinline__ void st_shared_cluster(double *local, unsigned rank, double v)
{
    const unsigned la = (unsigned)__cvta_generic_to_shared(local);
    unsigned ra;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(ra) : "r"(la), "r"(rank));
    asm volatile("st.shared::cluster.f64 [%0], %1;" :: "r"(ra), "d"(v) : "memory");
}

// the address, in the cluster's shared window, that the shared-memory address `local` of this CTA has in CTA `rank`
__device__ __forceinline__ unsigned cluster_map(unsigned local, unsigned rank)
{
    unsigned ra;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(ra) : "r"(local), "r"(rank));
    return ra;
}
// a complex number at cluster-window address `addr` + OFF bytes (OFF a compile-time constant: an immediate of the load)
template <int OFF>
__device__ __forceinline__ double2 ld_cluster_at(unsigned addr, double2)
{
    double2 v;
    asm volatile("ld.shared::cluster.v2.f64 {%0, %1}, [%2 + %3];" : "=d"(v.x), "=d"(v.y) : "r"(addr), "n"(OFF) : "memory");
    return v;
}
template <int OFF>
__device__ __forceinline__ float2 ld_cluster_at(unsigned addr, float2)
{
    float2 v;
    asm volatile("ld.shared::cluster.v2.f32 {%0, %1}, [%2 + %3];" : "=f"(v.x), "=f"(v.y) : "r"(addr), "n"(OFF) : "memory");
    return v;
}

template <typename T>
struct PersistArgs {
    typedef typename Cplx<T>::type C;
    Lattice L;
    const C *U;
    C *x, *r, *p, *p2, *Ap, *t; // even half-fields (p and p2 alternate as direction vector), t odd
    T m2;
    double *partials;          // grid version: gridDim.x doubles, the per-block partial sums of the current barrier
    CgScalars *scal;           // initialised by cg_init_kernel (rr, bb, tol2bb, k, maxiter, flag)
    unsigned long long *timeline;   // measurement hook (qcd_cg_timeline_*), NULL in normal solves: %globaltimer stamps of the
                                    // first TIMELINE_ITERS iterations, [block 0 | last block][iteration][TIMELINE_STAMPS]
};

// Stamps per iteration: 0 phase 1 starts, 1 phase 1 done, 2 past barrier 1, 3 phase 2 + block partial done, 4 past
// barrier 2 with <p,Ap> summed, 5 alpha known, 6 phase 3 + block partial done, 7 past barrier 3 with <r,r> summed,
// 8 beta known.
enum { TIMELINE_ITERS = 64, TIMELINE_STAMPS = 9 };

__device__ __forceinline__ unsigned long long global_ns()
{
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    return t;
}

__device__ __forceinline__ double2 ld_coherent(const double2 *p) { return __ldcg(p); }
__device__ __forceinline__ float2 ld_coherent(const float2 *p) { return __ldcg(p); }

enum { CLUSTER_MAX_CTAS = 16 };
// One thread per site, in both precisions.  A thread keeps two links and up to four neighbour vectors in flight: 34 sixteen-byte loads
// = 136 registers in fp64.  Under a 168-register cap ptxas interleaves those loads with the FMAs that consume them (four dependent round
// trips per phase instead of one), so the kernels run with a 255-register cap: ONE resident 256-thread block per SM in the grid
// version, 128-thread CTAs in the cluster version.
// Block shape of the grid version, measured per iteration (16^4 fp64 / fp32; 12^4; 16^3 x 32): 128 threads x 3 / x 4 resident
// blocks 15.7 / 16.5, 11.0 / 12.3, 29.7 / 24.4 us; 256 x 1 / x 2: 14.5 / 15.3, 10.5 / 10.6, 24.6 / 25.3; 512 x 1: 14.9 / 16.4, -, 22.6 / 23.0.
// Half as many blocks arrive at every grid barrier and half as many partial sums are re-read after it, and a thread gets its 255
// registers; 256 is best at 16^4, the BASELINE.json config.
// History (profiles/r02_small_lattice_timeline.md): under the earlier 128-register cap the fp32 kernel split a site over a QUAD of
// lanes, one direction each (phases 3-5 us -> 1-2.6 us).  With one 256-thread block per SM and 255 registers the plain form is the
// faster one in fp32 as well -- 16^4 15.1 -> 11.3 us per iteration, 16^3 x 32 25.4 -> 17.1, 8^4 8.5 -> 7.1, 4^4 7.6 -> 6.9 -- and the quad
// path is gone (in fp64 it had been slower at every size).
template <typename T> struct PersistBlock { enum { value = 256 }; };
template <typename T> struct PersistMinB { enum { value = 1 }; };
template <typename T> struct ClusterBlock { enum { value = 128 }; };   // 16 CTAs hold 2048 sites

// Barrier of the whole solve's thread set carrying this block's partial sum `block_val` (valid in thread 0; every
// thread of the block has passed a __syncthreads() after its last global store of the phase -- block_sum provides
// one).  Returns, in EVERY thread of every block, the sum of all blocks' partials in an order that depends only on
// the launch shape.
//   CLUSTER: the solve is one thread-block cluster.  Thread 0 stores the partial into slot [epoch parity][own rank] of
//            every CTA's shared memory, everybody meets at barrier.cluster, everybody adds the local slots in rank
//            order.  The parity double-buffers the slots: a CTA cannot write epoch e + 2 before all have read e.
//   grid   : cooperative launch; partials[epoch parity][block] then cooperative-groups grid.sync(), then every block re-reads
//            all partials from the L2 and sums them thread-strided and through the block tree.  (A hand-written barrier on one
//            monotonic arrival counter -- red.release + ld.acquire polling, no wait for the atomic's old value -- measured the
//            same 1.8-2.6 us per barrier at 148 blocks: the cost is the drain of the block's stores, not the barrier's protocol.)
template <int BLOCK, bool CLUSTER>
__device__ __forceinline__ double solve_barrier(double block_val, unsigned epoch, double *partials, double *smem /* BLOCK/32 + 1 */,
                                                double *cl_slots /* 2 x CLUSTER_MAX_CTAS, shared */)
{
    if (CLUSTER) {
        const unsigned n = cluster_nctarank();
        double *mine = cl_slots + (epoch & 1u) * CLUSTER_MAX_CTAS;
        if (threadIdx.x == 0) {
            const unsigned me = cluster_ctarank();
            for (unsigned r = 0; r < n; ++r) st_shared_cluster(mine + me, r, block_val);
        }
        cluster_barrier();
        double s = 0.0;
        for (unsigned r = 0; r < n; ++r) s += mine[r];
        return s;
    } else {
        namespace cg = cooperative_groups;
        partials += (size_t)(epoch & 1u) * gridDim.x;         // double-buffered like the cluster slots: a fast block may write its partial of
                                                              // barrier e + 1 (phase 3 has no data barrier in front) while a slow one still sums barrier e
        if (threadIdx.x == 0) partials[blockIdx.x] = block_val;
        cg::this_grid().sync();
        double s = 0.0;
        for (int i = threadIdx.x; i < (int)gridDim.x; i += BLOCK) s += __ldcg(partials + i);
        __syncthreads();                                      // smem is reused
        const double tot = block_sum<BLOCK>(s, smem);
        if (threadIdx.x == 0) smem[BLOCK / 32] = tot;
        __syncthreads();
        return smem[BLOCK / 32];
    }
}

// acc = (D in)(cb) for the site cb of `parity`; `in` may have been written earlier in this kernel
// FUSE: the input vector is r + beta * in, formed at every neighbour on the fly
template <typename T, int NROW, int TG, bool FUSE, bool KEEP_L1>
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
    // links requested one direction ahead, two sets of link registers used in turn (see cluster_site)
    auto load_links = [&](int mu, C (&uf)[9], C (&ub)[9]) {
        const bool unit_f = TG && mu == 3 && g.x3 != 0;
        const bool unit_b = TG && mu == 3 && g.x3 != 1;
        if (!unit_f) {
#pragma unroll
            for (int k = 0; k < 3 * NROW; ++k) uf[k] = KEEP_L1 ? ld_keep(Uf + (size_t)(mu * 3 * NROW + k) * Vh, pol) : ld_stream(Uf + (size_t)(mu * 3 * NROW + k) * Vh, pol);
        }
        if (!unit_b) {
#pragma unroll
            for (int k = 0; k < 3 * NROW; ++k) ub[k] = KEEP_L1 ? ld_keep(Ub + (size_t)(mu * 3 * NROW + k) * Vh + g.nb[mu], pol) : ld_stream(Ub + (size_t)(mu * 3 * NROW + k) * Vh + g.nb[mu], pol);
        }
    };
    auto hops = [&](int mu, C (&uf)[9], C (&ub)[9]) {
        const bool unit_f = TG && mu == 3 && g.x3 != 0;
        const bool unit_b = TG && mu == 3 && g.x3 != 1;
        C pf[3], pb[3];
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
    };
    C ufA[9], ubA[9], ufB[9], ubB[9];
    load_links(0, ufA, ubA);
    load_links(1, ufB, ubB);
    hops(0, ufA, ubA);
    load_links(2, ufA, ubA);
    hops(1, ufB, ubB);
    load_links(3, ufB, ubB);
    hops(2, ufA, ubA);
    hops(3, ufB, ubB);
}

// The grid version (cooperative launch): vectors in global memory, read through the L2.
template <typename T, int NROW, int TG, int BLOCK>
__device__ __forceinline__ void cg_persistent_body(const PersistArgs<T> &a)
{
    typedef typename Cplx<T>::type C;
    __shared__ double smem[BLOCK / 32 + 1];
    double *const cl_slots = nullptr;                           // (cluster version only)
    const int Vh = a.L.Vh;
    const size_t sVh = (size_t)Vh;
    const int gtid = blockIdx.x * BLOCK + threadIdx.x;
    // Every block owns one contiguous range of sites (the same in every phase and iteration, so phase 3 updates what the
    // same SM wrote in phase 2), all ranges equally long; the host launches a multiple of the SM count (16^4 fp64: 148
    // blocks of 222 sites instead of 256 blocks of 128 sites on 148 SMs); the range length is even so that a block starts
    // on a 32-byte sector.  Measured: no change at 16^4 (15.9 us either way -- the phases run at 80 % of the aggregate
    // L2 stream, not at a per-SM limit), kept because every SM now carries the same load at every lattice size.
    int spb = (Vh + (int)gridDim.x - 1) / (int)gridDim.x;
    spb += spb & 1;
    const int site0 = (int)blockIdx.x * spb;
    const int my_sites = Vh - site0 < spb ? (Vh - site0 > 0 ? Vh - site0 : 0) : spb;
    const int qpb = BLOCK, ql = (int)threadIdx.x;               // one thread per site: sites per trip of a block, this thread's site in the trip
    // one trip: every thread has ONE site, the same in every phase -- then what phase 3 needs (p and Ap of the site from
    // phase 2, x and r requested BEFORE the barrier that delivers alpha) is in registers when alpha arrives, Ap never goes to memory
    const bool one_trip = spb <= qpb;
    unsigned epoch = 0;

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
        for (int o = 0; o < spb; o += qpb) {                     // the same trip count in every thread
            const int cb = site0 + o + ql;
            const bool active = o + ql < my_sites;
            {
                if (active) {
                    C acc[3];
                    persistent_site<T, NROW, TG, true, false>(acc, a.L, 1, cb, a.U, p_old, a.r, be);
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
            }
        }
        QCD_STAMP(1);
        cooperative_groups::this_grid().sync();                  // data barrier: t and p_cur are complete everywhere
        QCD_STAMP(2);
        // phase 2: Ap = m^2 p - D_eo t, partial Re<p,Ap>
        double dot = 0.0;
        C kp[3], ka[3], kx[3], kr[3];                             // one trip: p, Ap, x, r of this thread's site
        for (int o = 0; o < spb; o += qpb) {
            const int cb = site0 + o + ql;
            const bool active = o + ql < my_sites;
            {
                if (active) {
                    C acc[3], vv[3];
                    persistent_site<T, NROW, TG, false, false>(acc, a.L, 0, cb, a.U, a.t);
#pragma unroll
                    for (int c = 0; c < 3; ++c) vv[c] = ld_coherent(p_cur + (size_t)c * sVh + cb);
#pragma unroll
                    for (int c = 0; c < 3; ++c) {
                        C o;
                        o.x = fma(a.m2, vv[c].x, -acc[c].x);
                        o.y = fma(a.m2, vv[c].y, -acc[c].y);
                        if (one_trip) { kp[c] = vv[c]; ka[c] = o; }
                        else a.Ap[(size_t)c * sVh + cb] = o;
                        dot += (double)vv[c].x * (double)o.x + (double)vv[c].y * (double)o.y;
                    }
                    if (one_trip) {
#pragma unroll
                        for (int c = 0; c < 3; ++c) { kx[c] = ld_coherent(a.x + (size_t)c * sVh + cb); kr[c] = ld_coherent(a.r + (size_t)c * sVh + cb); }
                    }
                }
            }
        }
        const double dot_block = block_sum<BLOCK>(dot, smem);
        QCD_STAMP(3);
        pAp = solve_barrier<BLOCK, false>(dot_block, ++epoch, a.partials, smem, cl_slots);
        QCD_STAMP(4);
        if (!(pAp > 0.0)) { flag = 3; break; }                     // breakdown: uniform across the grid
        alpha = rr / pAp;
        QCD_STAMP(5);
        // phase 3: x += alpha p, r -= alpha Ap, partial <r,r> on the block's OWN sites (Ap was written by this SM a barrier
        // ago); all loads of a thread before its first store: a load behind a store that may alias it waits for it
        const T al = (T)alpha;
        double nrm = 0.0;
        for (int o = 0; o < spb; o += qpb) {
            const int cb = site0 + o + ql;
            if (o + ql < my_sites) {
                {
                    C vx[3], vr[3], vp[3], va[3];
#pragma unroll
                    for (int c = 0; c < 3; ++c) {
                        const size_t i = (size_t)c * sVh + cb;
                        if (one_trip) { vx[c] = kx[c]; vr[c] = kr[c]; vp[c] = kp[c]; va[c] = ka[c]; }
                        else { vx[c] = ld_coherent(a.x + i); vr[c] = ld_coherent(a.r + i); vp[c] = ld_coherent(p_cur + i); va[c] = ld_coherent(a.Ap + i); }
                    }
#pragma unroll
                    for (int c = 0; c < 3; ++c) {
                        const size_t i = (size_t)c * sVh + cb;
                        vx[c].x = fma(al, vp[c].x, vx[c].x); vx[c].y = fma(al, vp[c].y, vx[c].y);
                        vr[c].x = fma(-al, va[c].x, vr[c].x); vr[c].y = fma(-al, va[c].y, vr[c].y);
                        a.x[i] = vx[c]; a.r[i] = vr[c];
                        nrm += (double)vr[c].x * (double)vr[c].x + (double)vr[c].y * (double)vr[c].y;
                    }
                }
            }
        }
        __syncthreads();                                           // smem of the previous barrier has been read by everyone
        const double nrm_block = block_sum<BLOCK>(nrm, smem);
        QCD_STAMP(6);
        const double rr_new = solve_barrier<BLOCK, false>(nrm_block, ++epoch, a.partials, smem, cl_slots);
        QCD_STAMP(7);
        beta = rr_new / rr;
        rr = rr_new;
        k += 1;
        if (gtid == 0) {                                           // residual history (qcd_cg_history)
            double *const hist = a.scal->hist;
            if (hist && k <= a.scal->hist_cap) hist[k - 1] = rr_new;
        }
        QCD_STAMP(8);
        ++it;
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

// ------------------------------------------------------------------------------------------
// The one-cluster solve with the vectors in DISTRIBUTED SHARED MEMORY.
//
// Up to 2048 sites per parity the solve is one cluster of <= 16 CTAs x 128 threads, one site per thread, the same in every
// phase and iteration.  Every vector a neighbour reads -- r, the two direction buffers, t -- then fits the CTAs' shared memory
// (4 vectors x 3 colours x 128 sites: 24 KB in fp64), each CTA holding the elements of its own sites: a neighbour element is
// read from the owner's shared memory (one mapa per hop + ld.shared::cluster with the colour as an immediate: ~215 cycles across CTAs, 38 inside the CTA, against a
// 600-700-cycle L2 round trip for ld.global.cg), x and Ap never leave registers, and the site geometry (the sixteen neighbour
// indices of the site as an odd and as an even site, their owners, the phases) is computed once, outside the iteration loop.
// Most neighbours are in the CTA itself (x0, x1 and half of the x2 neighbours of 128 consecutive sites at 8^4; all of them at
// 4^4, which is one CTA).  Links stay in global memory, L1-allocating: a CTA reads the same links in every iteration.
// Same arithmetic in the same order as cg_persistent_body (and, per site, as dslash_kernel): same iterates.
// ------------------------------------------------------------------------------------------
template <typename T>
struct ClusterHop {              // one neighbour of this thread's site: owner CTA and element inside the owner's arrays
    unsigned short rank[8], off[8];        // hop = 2 mu + (0: forward, 1: backward)
    unsigned neg;                          // bit hop: the hop's term enters with a minus sign (phase x seam)
    int nb_global[4];                      // backward neighbour index (the backward link is stored there)
    int x3;
};

template <typename T>
__device__ __forceinline__ ClusterHop<T> cluster_hops(const Lattice &L, int parity, int cb, int spb)
{
    const SiteGeom g = site_geometry(L, parity, cb);
    ClusterHop<T> h;
    h.neg = 0u;
#pragma unroll
    for (int mu = 0; mu < 4; ++mu) {
        h.rank[2 * mu] = (unsigned short)(g.nf[mu] / spb);     h.off[2 * mu] = (unsigned short)(g.nf[mu] % spb);
        h.rank[2 * mu + 1] = (unsigned short)(g.nb[mu] / spb); h.off[2 * mu + 1] = (unsigned short)(g.nb[mu] % spb);
        h.neg |= (g.sf[mu] < 0.f ? 1u : 0u) << (2 * mu);
        h.neg |= (g.sb[mu] < 0.f ? 1u : 0u) << (2 * mu + 1);
        h.nb_global[mu] = g.nb[mu];
    }
    h.x3 = g.x3;
    return h;
}

// acc = (D in)(cb) with `in` in distributed shared memory ([3][BLOCK] per CTA); FUSE: the input is r + beta * in
template <typename T, int NROW, int TG, bool FUSE, bool KEEP_L1, int BLOCK>
__device__ __forceinline__ void cluster_site(typename Cplx<T>::type acc[3], const Lattice &L, int parity, int cb, const ClusterHop<T> &h,
                                             const typename Cplx<T>::type *U, unsigned in_saddr, unsigned r_saddr, T beta)
{
    // in_saddr / r_saddr: shared-window addresses, in THIS CTA, of element [0][0] of the [3][BLOCK] arrays `in` and `r`; the same arrays of
    // the owner CTA are reached with ONE mapa per hop, the three colours are immediates of the loads
    typedef typename Cplx<T>::type C;
    const size_t Vh = (size_t)L.Vh;
    const uint64_t pol = l2_policy_evict_last();
    const C *Uf = U + (size_t)(parity * 12 * NROW) * Vh + cb;
    const C *Ub = U + (size_t)((1 - parity) * 12 * NROW) * Vh;
    acc[0].x = acc[0].y = acc[1].x = acc[1].y = acc[2].x = acc[2].y = (T)0;
    // The links of direction mu + 1 are requested BEFORE the hops of direction mu are computed (two sets of link registers, used in
    // turn): in source order ptxas keeps a direction's loads next to the FMAs that consume them, and the source-level profile of that
    // form had 44 % of all stall samples on DFMAs waiting for the link loads of their own direction (long scoreboard).
    auto load_links = [&](int mu, C (&uf)[9], C (&ub)[9]) {
        const bool unit_f = TG && mu == 3 && h.x3 != 0;
        const bool unit_b = TG && mu == 3 && h.x3 != 1;
        if (!unit_f) {
#pragma unroll
            for (int k = 0; k < 3 * NROW; ++k) uf[k] = KEEP_L1 ? ld_keep(Uf + (size_t)(mu * 3 * NROW + k) * Vh, pol) : ld_stream(Uf + (size_t)(mu * 3 * NROW + k) * Vh, pol);
        }
        if (!unit_b) {
#pragma unroll
            for (int k = 0; k < 3 * NROW; ++k) ub[k] = KEEP_L1 ? ld_keep(Ub + (size_t)(mu * 3 * NROW + k) * Vh + h.nb_global[mu], pol) : ld_stream(Ub + (size_t)(mu * 3 * NROW + k) * Vh + h.nb_global[mu], pol);
        }
    };
    auto hops = [&](int mu, C (&uf)[9], C (&ub)[9]) {
        const bool unit_f = TG && mu == 3 && h.x3 != 0;
        const bool unit_b = TG && mu == 3 && h.x3 != 1;
        C pf[3], pb[3];
        const unsigned rf = h.rank[2 * mu], of = h.off[2 * mu], rb = h.rank[2 * mu + 1], ob = h.off[2 * mu + 1];
        constexpr int COL = BLOCK * (int)sizeof(C);             // bytes between colours
        const unsigned af = cluster_map(in_saddr, rf) + of * (unsigned)sizeof(C), ab = cluster_map(in_saddr, rb) + ob * (unsigned)sizeof(C);
        pf[0] = ld_cluster_at<0>(af, C()); pf[1] = ld_cluster_at<COL>(af, C()); pf[2] = ld_cluster_at<2 * COL>(af, C());
        pb[0] = ld_cluster_at<0>(ab, C()); pb[1] = ld_cluster_at<COL>(ab, C()); pb[2] = ld_cluster_at<2 * COL>(ab, C());
        if (FUSE) {
            const unsigned d = r_saddr - in_saddr;              // the same displacement in every CTA
            C vf[3], vb[3];
            vf[0] = ld_cluster_at<0>(af + d, C()); vf[1] = ld_cluster_at<COL>(af + d, C()); vf[2] = ld_cluster_at<2 * COL>(af + d, C());
            vb[0] = ld_cluster_at<0>(ab + d, C()); vb[1] = ld_cluster_at<COL>(ab + d, C()); vb[2] = ld_cluster_at<2 * COL>(ab + d, C());
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                pf[c].x = fma(beta, pf[c].x, vf[c].x); pf[c].y = fma(beta, pf[c].y, vf[c].y);
                pb[c].x = fma(beta, pb[c].x, vb[c].x); pb[c].y = fma(beta, pb[c].y, vb[c].y);
            }
        }
        const unsigned nf = (h.neg >> (2 * mu)) & 1u, nb = (h.neg >> (2 * mu + 1)) & 1u;
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            pf[c].x = flip_sign(pf[c].x, nf); pf[c].y = flip_sign(pf[c].y, nf);
            pb[c].x = flip_sign(pb[c].x, nb); pb[c].y = flip_sign(pb[c].y, nb);
        }
        if (!unit_f) { if (NROW == 2) reconstruct_third_row<C>(uf); mat_vec_acc<T, C>(acc, uf, pf); } else vec_acc<C>(acc, pf);
        if (!unit_b) { if (NROW == 2) reconstruct_third_row<C>(ub); matdag_vec_acc<T, C>(acc, ub, pb); } else vec_acc<C>(acc, pb);
    };
    C ufA[9], ubA[9], ufB[9], ubB[9];
    load_links(0, ufA, ubA);
    load_links(1, ufB, ubB);
    hops(0, ufA, ubA);
    load_links(2, ufA, ubA);
    hops(1, ufB, ubB);
    load_links(3, ufB, ubB);
    hops(2, ufA, ubA);
    hops(3, ufB, ubB);
}

template <typename T, int NROW, int TG, int BLOCK>
__device__ __forceinline__ void cg_cluster_body(const PersistArgs<T> &a)
{
    typedef typename Cplx<T>::type C;
    // the links of a CTA's sites for BOTH phases (2 x 1152 B per site in fp64) stay in its L1 only if they fit: at 128 sites per CTA
    // they do in fp32 (147 KB) and not in fp64 (295 KB), where the second phase streams its links past the L1 instead of evicting the first's
    constexpr bool KEEP2 = sizeof(T) == 4;
    __shared__ double smem[BLOCK / 32 + 1];
    __shared__ double cl_slots[2 * CLUSTER_MAX_CTAS];
    __shared__ __align__(16) C s_r[3][BLOCK], s_p[2][3][BLOCK], s_t[3][BLOCK];
    const int Vh = a.L.Vh;
    const size_t sVh = (size_t)Vh;
    int spb = (Vh + (int)gridDim.x - 1) / (int)gridDim.x;      // sites per CTA, as in cg_persistent_body; <= BLOCK (host: ncta x BLOCK >= Vh)
    spb += spb & 1;
    const int site0 = (int)blockIdx.x * spb;
    const int my_sites = Vh - site0 < spb ? (Vh - site0 > 0 ? Vh - site0 : 0) : spb;
    const int tid = (int)threadIdx.x, cb = site0 + tid;
    const bool active = tid < my_sites;
    const int gtid = blockIdx.x * BLOCK + threadIdx.x;
    unsigned epoch = 0;

    // the thread's site: its vectors into shared memory / registers, its geometry as an odd (phase 1) and as an even site (phase 2)
    C vx[3];
    ClusterHop<T> h_odd, h_even;
    if (active) {
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            s_r[c][tid] = a.r[(size_t)c * sVh + cb];
            s_p[0][c][tid] = a.p[(size_t)c * sVh + cb];
            vx[c] = a.x[(size_t)c * sVh + cb];
        }
        h_odd = cluster_hops<T>(a.L, 1, cb, spb);
        h_even = cluster_hops<T>(a.L, 0, cb, spb);
    }
    cluster_barrier();          // every CTA runs and has filled its arrays before anyone reads them or stores into its slots

    double rr = a.scal->rr;
    const double tol2bb = a.scal->tol2bb;
    const int maxiter = a.scal->maxiter;
    int k = a.scal->k, flag = a.scal->flag;
    double alpha = 0.0, beta = 0.0, pAp = 0.0;

    unsigned long long *tl = nullptr;
    if (a.timeline && threadIdx.x == 0 && (blockIdx.x == 0 || blockIdx.x == gridDim.x - 1))
        tl = a.timeline + (blockIdx.x == 0 ? 0 : TIMELINE_ITERS * TIMELINE_STAMPS);
    int it = 0;
#define QCD_STAMP(i) do { if (tl && it < TIMELINE_ITERS) tl[it * TIMELINE_STAMPS + (i)] = global_ns(); } while (0)

    const unsigned sa_r = (unsigned)__cvta_generic_to_shared(&s_r[0][0]), sa_p = (unsigned)__cvta_generic_to_shared(&s_p[0][0][0]),
                   sa_t = (unsigned)__cvta_generic_to_shared(&s_t[0][0]);
    int old = 0;                                               // s_p[old] is p of the previous iteration, s_p[old ^ 1] receives the new one
    while (flag == 0) {
        QCD_STAMP(0);
        // phase 1: p' = r + beta p (own site, into the other buffer), t = D_oe p' with p' formed on the fly at the neighbours
        const T be = (T)beta;
        const int cur = old ^ 1;
        C vp[3];                                               // p' of the own site: phases 2 and 3 use it from registers
        if (active) {
            C acc[3];
            cluster_site<T, NROW, TG, true, true, BLOCK>(acc, a.L, 1, cb, h_odd, a.U, sa_p + (unsigned)old * (unsigned)sizeof(s_p[0]), sa_r, be);
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                const C po = s_p[old][c][tid], ro = s_r[c][tid];
                vp[c].x = fma(be, po.x, ro.x); vp[c].y = fma(be, po.y, ro.y);
                s_p[cur][c][tid] = vp[c];
                s_t[c][tid] = acc[c];
            }
        }
        QCD_STAMP(1);
        cluster_barrier();                                     // t and p' are complete everywhere
        QCD_STAMP(2);
        // phase 2: Ap = m^2 p' - D_eo t (registers), partial Re<p',Ap>
        double dot = 0.0;
        C va[3];
        if (active) {
            C acc[3];
            cluster_site<T, NROW, TG, false, KEEP2, BLOCK>(acc, a.L, 0, cb, h_even, a.U, sa_t, sa_t, (T)0);
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                va[c].x = fma(a.m2, vp[c].x, -acc[c].x);
                va[c].y = fma(a.m2, vp[c].y, -acc[c].y);
                dot += (double)vp[c].x * (double)va[c].x + (double)vp[c].y * (double)va[c].y;
            }
        }
        const double dot_block = block_sum<BLOCK>(dot, smem);
        QCD_STAMP(3);
        pAp = solve_barrier<BLOCK, true>(dot_block, ++epoch, a.partials, smem, cl_slots);
        QCD_STAMP(4);
        if (!(pAp > 0.0)) { flag = 3; break; }                     // breakdown: uniform across the cluster
        alpha = rr / pAp;
        QCD_STAMP(5);
        // phase 3: x += alpha p' (registers), r -= alpha Ap (own shared memory), partial <r,r>
        const T al = (T)alpha;
        double nrm = 0.0;
        if (active) {
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                C vr = s_r[c][tid];
                vx[c].x = fma(al, vp[c].x, vx[c].x); vx[c].y = fma(al, vp[c].y, vx[c].y);
                vr.x = fma(-al, va[c].x, vr.x); vr.y = fma(-al, va[c].y, vr.y);
                s_r[c][tid] = vr;
                nrm += (double)vr.x * (double)vr.x + (double)vr.y * (double)vr.y;
            }
        }
        __syncthreads();                                           // smem of the previous barrier has been read by everyone
        const double nrm_block = block_sum<BLOCK>(nrm, smem);
        QCD_STAMP(6);
        const double rr_new = solve_barrier<BLOCK, true>(nrm_block, ++epoch, a.partials, smem, cl_slots);
        QCD_STAMP(7);
        beta = rr_new / rr;
        rr = rr_new;
        k += 1;
        if (gtid == 0) {                                           // residual history (qcd_cg_history)
            double *const hist = a.scal->hist;
            if (hist && k <= a.scal->hist_cap) hist[k - 1] = rr_new;
        }
        QCD_STAMP(8);
        ++it;
        if (rr_new != rr_new) flag = 3;
        else if (rr_new <= tol2bb) flag = 1;
        else if (k >= maxiter) flag = 2;
        if (flag != 0) break;
        old = cur;
    }
#undef QCD_STAMP
    if (active) {
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            a.x[(size_t)c * sVh + cb] = vx[c];
            a.r[(size_t)c * sVh + cb] = s_r[c][tid];               // the workspace keeps the last residual, as the other loops leave it
        }
    }
    if (gtid == 0) {
        CgScalars *s = a.scal;
        s->rr = rr; s->pAp = pAp; s->alpha = alpha; s->beta = beta; s->k = k; s->flag = flag;
    }
    cluster_barrier();                              // no CTA exits while a peer may still read or store into its shared memory
}

// cooperative launch, any number of co-resident blocks
template <typename T, int NROW, int TG>
__global__ void __launch_bounds__(PersistBlock<T>::value, PersistMinB<T>::value) cg_persistent_kernel(const PersistArgs<T> a)
{
    cg_persistent_body<T, NROW, TG, PersistBlock<T>::value>(a);
}

// ONE cluster of 1 .. 16 CTAs (cluster dimension = grid dimension, set at launch)
template <typename T, int NROW, int TG>
__global__ void __launch_bounds__(ClusterBlock<T>::value, 1) cg_cluster_kernel(const PersistArgs<T> a)
{
    cg_cluster_body<T, NROW, TG, ClusterBlock<T>::value>(a);
}

} // namespace qcd
