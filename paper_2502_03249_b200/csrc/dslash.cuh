// Staggered hopping-term kernels: the parity blocks of Eq. (1), PAPER.md:49-54 (Sec. 4.2)
//
//   out(x) = sum_mu [ eta_mu(x) s+ U_{x,mu} phi(x+mu) - eta_mu(x-mu) s- U^dagger_{x-mu,mu} phi(x-mu) ]
//
// for the sites x of one parity; phi lives on the other parity.  s+- are the antiperiodic
// time-seam signs.  8 SU(3) x colour-vector products and 7 vector additions per site =
// 570 flop; "performance is bounded by the device bandwidth", so
// the design is about bytes in flight, not arithmetic: one thread per output site, every
// load a fully coalesced 16-byte (fp64) or 8-byte (fp32) access into an SoA plane, links
// streamed through L2 with evict_first and never allocated in L1, neighbour spinors kept
// (evict_last, L1-allocating).
//
// MODE 0: out = D phi                                   (qcd_dslash_eo / qcd_dslash_oe)
// MODE 1: out = m^2 v - D phi                           (qcd_apply_M, second half)
// MODE 2: MODE 1 + block partial of Re<v,out> and the CG alpha step in the last block
//         ("epilogue fused into the D_eo kernel")
#pragma once
#include "lattice.cuh"
#include "reduce.cuh"

namespace qcd {

template <typename T>
struct DslashArgs {
    typedef typename Cplx<T>::type C;
    Lattice L;
    int parity;            // parity of the OUTPUT sites (0: D_eo, 1: D_oe)
    const C *U;            // gauge field, 72 planes
    const C *in;           // half-field of parity 1-parity, 3 planes
    C *out;                // half-field of parity `parity`, 3 planes
    const C *v;            // MODE >= 1: half-field of parity `parity`
    T m2;                  // MODE >= 1
    double *partials;      // MODE 2
    CgScalars *scal;       // MODE 2 (and flag source when check_flag)
    int check_flag;        // return immediately when scal->flag != 0 (CG no-op iterations)
};

// acc += U * p
template <typename T, typename C>
__device__ __forceinline__ void mat_vec_acc(C acc[3], const C u[9], const C p[3])
{
#pragma unroll
    for (int a = 0; a < 3; ++a) {
#pragma unroll
        for (int b = 0; b < 3; ++b) {
            acc[a].x = fma(u[3 * a + b].x, p[b].x, acc[a].x);
            acc[a].x = fma(-u[3 * a + b].y, p[b].y, acc[a].x);
            acc[a].y = fma(u[3 * a + b].x, p[b].y, acc[a].y);
            acc[a].y = fma(u[3 * a + b].y, p[b].x, acc[a].y);
        }
    }
}

// acc += U^dagger * p
template <typename T, typename C>
__device__ __forceinline__ void matdag_vec_acc(C acc[3], const C u[9], const C p[3])
{
#pragma unroll
    for (int a = 0; a < 3; ++a) {
#pragma unroll
        for (int b = 0; b < 3; ++b) {
            // conj(u[b][a]) * p[b]
            acc[a].x = fma(u[3 * b + a].x, p[b].x, acc[a].x);
            acc[a].x = fma(u[3 * b + a].y, p[b].y, acc[a].x);
            acc[a].y = fma(u[3 * b + a].x, p[b].y, acc[a].y);
            acc[a].y = fma(-u[3 * b + a].y, p[b].x, acc[a].y);
        }
    }
}

template <typename T, int MODE, int BLOCK, int MINB>
__global__ void __launch_bounds__(BLOCK, MINB) dslash_kernel(const DslashArgs<T> a)
{
    typedef typename Cplx<T>::type C;
    if (a.check_flag && a.scal->flag != 0) return;

    const int cb = blockIdx.x * BLOCK + threadIdx.x;
    const bool active = cb < a.L.Vh;
    const size_t Vh = (size_t)a.L.Vh;
    double dot = 0.0;

    if (active) {
        const SiteGeom g = site_geometry(a.L, a.parity, cb);
        const uint64_t pol_stream = l2_policy_evict_first();
        const uint64_t pol_keep = l2_policy_evict_last();
        const C *Uf = a.U + (size_t)(a.parity * 36) * Vh + cb;          // U_{x,mu}: own parity block
        const C *Ub = a.U + (size_t)((1 - a.parity) * 36) * Vh;         // U_{x-mu,mu}: other parity block

        C acc[3];
        acc[0].x = acc[0].y = acc[1].x = acc[1].y = acc[2].x = acc[2].y = (T)0;

#pragma unroll
        for (int mu = 0; mu < 4; ++mu) {
            C uf[9], ub[9], pf[3], pb[3];
            const C *ufp = Uf + (size_t)(mu * 9) * Vh;
            const C *ubp = Ub + (size_t)(mu * 9) * Vh + g.nb[mu];
#pragma unroll
            for (int k = 0; k < 9; ++k) uf[k] = ld_stream(ufp + (size_t)k * Vh, pol_stream);
#pragma unroll
            for (int k = 0; k < 9; ++k) ub[k] = ld_stream(ubp + (size_t)k * Vh, pol_stream);
#pragma unroll
            for (int c = 0; c < 3; ++c) pf[c] = ld_keep(a.in + (size_t)c * Vh + g.nf[mu], pol_keep);
#pragma unroll
            for (int c = 0; c < 3; ++c) pb[c] = ld_keep(a.in + (size_t)c * Vh + g.nb[mu], pol_keep);
            const T sf = (T)g.sf[mu], sb = (T)g.sb[mu];
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                pf[c].x *= sf; pf[c].y *= sf;     // exact: sf, sb are +-1
                pb[c].x *= sb; pb[c].y *= sb;
            }
            mat_vec_acc<T, C>(acc, uf, pf);
            matdag_vec_acc<T, C>(acc, ub, pb);
        }

        if (MODE >= 1) {
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                const C vv = a.v[(size_t)c * Vh + cb];
                C o;
                o.x = fma(a.m2, vv.x, -acc[c].x);
                o.y = fma(a.m2, vv.y, -acc[c].y);
                a.out[(size_t)c * Vh + cb] = o;
                if (MODE == 2) dot += (double)vv.x * (double)o.x + (double)vv.y * (double)o.y;
            }
        } else {
#pragma unroll
            for (int c = 0; c < 3; ++c) a.out[(size_t)c * Vh + cb] = acc[c];
        }
    }

    if (MODE == 2) {
        __shared__ double smem[BLOCK / 32];
        __shared__ int last;
        if (publish_partial<BLOCK>(dot, a.partials, &a.scal->ticket, smem, &last)) {
            const double pAp = final_sum<BLOCK>(a.partials, (int)gridDim.x, smem);
            if (threadIdx.x == 0) {
                CgScalars *s = a.scal;
                s->pAp = pAp;
                if (!(pAp > 0.0)) s->flag = 3;          // breakdown: <p,Mp> <= 0 or NaN
                else s->alpha = s->rr / pAp;
            }
        }
    }
}

} // namespace qcd
