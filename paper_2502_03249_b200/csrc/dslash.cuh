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
//
// The paper's own traffic reductions are template parameters of the same kernel:
// NROW = 2 : "we store only the first two rows, i.e. 12 floats.  The third row is reconstructed
//            on-the-fly ... using the properties of SU(3) matrices": row2 = conj(row0 x row1)
// TG = 1   : "gauge fixing to transform the temporal link variables to 1 for all the sites with
//            the temporal coordinate t != 0": time links with t != 0 are not loaded at all
// NRHS = n : "applying D on multiple vectors at once ... each link variable to be read once and
//            then reused for multiple vectors" (NMULTI)
#pragma once
#include "lattice.cuh"
#include "reduce.cuh"

namespace qcd {

template <typename T, int NRHS>
struct DslashArgs {
    typedef typename Cplx<T>::type C;
    Lattice L;
    int parity;            // parity of the OUTPUT sites (0: D_eo, 1: D_oe)
    const C *U;            // gauge field, 2 x 4 x (3 NROW) planes
    const C *in[NRHS];     // half-fields of parity 1-parity, 3 planes each
    C *out[NRHS];          // half-fields of parity `parity`, 3 planes each
    const C *v[NRHS];      // MODE >= 1: half-fields of parity `parity`
    T m2;                  // MODE >= 1
    double *partials;      // MODE 2: [NRHS][gridDim.x]
    CgScalars *scal;       // MODE 2: NRHS entries (and flag source when check_flag)
    int check_flag;        // return immediately when every scal[r].flag != 0 (CG no-op iterations)
    int chunks;            // chunks of BLOCK sites one block walks (1 unless MODE 2, see dslash_kernel)
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

// conj(a * b - c * d)
template <typename C>
__device__ __forceinline__ C conj_cross(const C &a, const C &b, const C &c, const C &d)
{
    C r;
    r.x = a.x * b.x - a.y * b.y - c.x * d.x + c.y * d.y;
    r.y = -(a.x * b.y + a.y * b.x - c.x * d.y - c.y * d.x);
    return r;
}

// Third row of an SU(3) matrix from its first two: rows are orthonormal and
// det = 1, hence row2 = conj(row0 x row1).
template <typename C>
__device__ __forceinline__ void reconstruct_third_row(C u[9])
{
    u[6] = conj_cross(u[1], u[5], u[2], u[4]);
    u[7] = conj_cross(u[2], u[3], u[0], u[5]);
    u[8] = conj_cross(u[0], u[4], u[1], u[3]);
}

// One link = 3 NROW planes, Vh apart.
template <int NROW, typename C>
__device__ __forceinline__ void load_link(C u[9], const C *p, size_t Vh, uint64_t pol)
{
#pragma unroll
    for (int k = 0; k < 3 * NROW; ++k) u[k] = ld_stream(p + (size_t)k * Vh, pol);
}

// x -> sign * x for sign = +-1, as a flip of the IEEE sign bit: exact, and an integer-pipe
// operation (the fp64 pipe is the scarce one once several vectors share a link).
__device__ __forceinline__ double flip_sign(double x, unsigned neg)
{
    return __hiloint2double(__double2hiint(x) ^ (int)(neg << 31), __double2loint(x));
}
__device__ __forceinline__ float flip_sign(float x, unsigned neg)
{
    return __int_as_float(__float_as_int(x) ^ (int)(neg << 31));
}

template <typename T, typename C>
__device__ __forceinline__ void load_spinor(C p[3], const C *f, size_t Vh, int site, T sign, uint64_t pol)
{
#pragma unroll
    for (int c = 0; c < 3; ++c) p[c] = ld_keep(f + (size_t)c * Vh + site, pol);
    const unsigned neg = sign < (T)0 ? 1u : 0u;
#pragma unroll
    for (int c = 0; c < 3; ++c) { p[c].x = flip_sign(p[c].x, neg); p[c].y = flip_sign(p[c].y, neg); }
}

// the same from the shared-memory tile of a block (dslash_kernel, TILE): colour planes `stride` elements apart
template <typename T, typename C>
__device__ __forceinline__ void load_spinor_tile(C p[3], const C *t, int stride, T sign)
{
#pragma unroll
    for (int c = 0; c < 3; ++c) p[c] = t[(size_t)c * stride];
    const unsigned neg = sign < (T)0 ? 1u : 0u;
#pragma unroll
    for (int c = 0; c < 3; ++c) { p[c].x = flip_sign(p[c].x, neg); p[c].y = flip_sign(p[c].y, neg); }
}

template <typename C>
__device__ __forceinline__ void vec_acc(C acc[3], const C p[3])
{
#pragma unroll
    for (int c = 0; c < 3; ++c) { acc[c].x += p[c].x; acc[c].y += p[c].y; }
}

// out = acc (MODE 0) or m^2 v - acc (MODE >= 1); MODE 2 also accumulates Re<v,out> per vector.
// The 3 NRHS loads of v(x) are all issued before the first store: written as load / FMA / store per
// component, every load after the first has to wait behind the preceding store (the compiler cannot
// prove that out does not alias v), which exposes 3 NRHS memory round trips at the end of every thread
// -- measured as +1.0 ms on the four-vector kernel (3.2 instead of 2.2 ms without the loads).  v(x) is
// read once, so it is streamed like a link (read-only path, no L1 allocation, evict_first).
template <typename T, int MODE, int NRHS>
__device__ __forceinline__ void dslash_epilogue(const DslashArgs<T, NRHS> &a, int cb, typename Cplx<T>::type (&acc)[NRHS][3],
                                                double (&dot)[NRHS], uint64_t pol_stream)
{
    typedef typename Cplx<T>::type C;
    const size_t Vh = (size_t)a.L.Vh;
    if (MODE >= 1) {
        C vv[NRHS][3];
#pragma unroll
        for (int r = 0; r < NRHS; ++r)
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                // one vector: the plain load (the L2 prefetch issued before the first hop has brought the line in;
                // A/B at 64^4 is a wash in fp64 and the streamed form loses 8 % on the fp32 two-row temporal-gauge kernel)
                if (NRHS == 1) vv[r][c] = a.v[r][(size_t)c * Vh + cb];
                else vv[r][c] = ld_stream(a.v[r] + (size_t)c * Vh + cb, pol_stream);
            }
#pragma unroll
        for (int r = 0; r < NRHS; ++r) {
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                C o;
                o.x = fma(a.m2, vv[r][c].x, -acc[r][c].x);
                o.y = fma(a.m2, vv[r][c].y, -acc[r][c].y);
                a.out[r][(size_t)c * Vh + cb] = o;
                if (MODE == 2) dot[r] += (double)vv[r][c].x * (double)o.x + (double)vv[r][c].y * (double)o.y;
            }
        }
    } else {
#pragma unroll
        for (int r = 0; r < NRHS; ++r)
#pragma unroll
            for (int c = 0; c < 3; ++c) a.out[r][(size_t)c * Vh + cb] = acc[r][c];
    }
}

// MODE 2: two-stage reduction of the per-vector Re<p,Mp> and the CG alpha step in the last block.
template <typename T, int MODE, int NRHS, int BLOCK>
__device__ __forceinline__ void dslash_reduce(const DslashArgs<T, NRHS> &a, double (&dot)[NRHS])
{
    if (MODE == 2) {
        __shared__ double smem[NRHS * (BLOCK / 32)];
        __shared__ int last;
        if (publish_partials<BLOCK, NRHS>(dot, a.partials, (size_t)gridDim.x, a.scal, smem, &last)) {
            for (int r = 0; r < NRHS; ++r) {
                const double pAp = final_sum<BLOCK>(a.partials + (size_t)r * gridDim.x, (int)gridDim.x, smem);
                if (threadIdx.x == 0) {
                    CgScalars *s = a.scal + r;
                    if (s->flag == 0) {
                        s->pAp = pAp;
                        if (!(pAp > 0.0)) s->flag = 3;          // breakdown: <p,Mp> <= 0 or NaN
                        else s->alpha = s->rr / pAp;
                    }
                }
                __syncthreads();
            }
        }
    }
}

// TILE (several vectors; the host checks that a block's BLOCK sites are R = BLOCK / h whole x0-rows of one (x2, x3) plane):
// the x0 and x1 neighbours of a block's sites lie in the R + 2 rows x1 - 1 ... x1 + R of that plane -- 6 rows for the 16 row
// loads of the four hops at 64^4.  They are copied once into shared memory (cp.async, all vectors, then one barrier) and
// the hops mu = 0, 1 read them from there: 22 instead of 32 row fetches per vector go through the L2 -> SM path, the one that
// saturates (~10 TB/s under the power cap) once several vectors share a link.  Same values, same FMA
// order: bitwise identical results.
template <typename T, int MODE, int NROW, int TG, int NRHS, int BLOCK, int MINB, bool TILE = false>
__global__ void __launch_bounds__(BLOCK, MINB) dslash_kernel(const DslashArgs<T, NRHS> a)
{
    typedef typename Cplx<T>::type C;
    extern __shared__ __align__(16) unsigned char tile_smem[];
    if (a.check_flag) {
        bool all_done = true;
#pragma unroll
        for (int r = 0; r < NRHS; ++r) all_done = all_done && (a.scal[r].flag != 0);
        if (all_done) return;
    }

    const size_t Vh = (size_t)a.L.Vh;
    double dot[NRHS];
#pragma unroll
    for (int r = 0; r < NRHS; ++r) dot[r] = 0.0;

    // MODE 2 ends every block with a reduction (two block barriers, a fence, a ticket): ~2 us during
    // which the block's registers sit idle -- 25 % of a block that handles one site per thread in
    // fp32.  A block therefore walks a.chunks chunks of BLOCK sites and reduces once; the host sizes
    // the grid to a few thousand blocks (dslash_inst.cuh).
#pragma unroll 1
    for (int chunk = 0; chunk < (MODE == 2 ? a.chunks : 1); ++chunk) {
    const int tid = (blockIdx.x * (MODE == 2 ? a.chunks : 1) + chunk) * BLOCK + threadIdx.x;
    const bool active = tid < a.L.Vh;
    const int cb = active ? traversal_site(a.L, tid) : tid;
    const int tile_w = BLOCK + 2 * a.L.h;                         // elements per (vector, colour) row set: R + 2 rows of h sites
    C *tile = reinterpret_cast<C *>(tile_smem);                   // [NRHS * 3][tile_w]
    if (TILE) {
        // every thread of the block is active (Vh % BLOCK == 0) and cb = cb0 + threadIdx.x
        if (chunk > 0) __syncthreads();                           // the previous chunk's tile has been read by everyone
        const int cb0 = cb - (int)threadIdx.x;
        const int x1_0 = (int)(((unsigned)cb0 / (unsigned)a.L.h) % (unsigned)a.L.N1);
        const int plane0 = cb0 - x1_0 * a.L.h;
        for (int e = threadIdx.x; e < tile_w; e += BLOCK) {
            const int row = e / a.L.h, xh = e - row * a.L.h;
            int x1s = x1_0 - 1 + row;
            x1s += x1s < 0 ? a.L.N1 : (x1s >= a.L.N1 ? -a.L.N1 : 0);
            const size_t src = (size_t)(plane0 + x1s * a.L.h + xh);
#pragma unroll
            for (int r = 0; r < NRHS; ++r)
#pragma unroll
                for (int c = 0; c < 3; ++c) cp_async_plain(&tile[(size_t)(r * 3 + c) * tile_w + e], a.in[r] + (size_t)c * Vh + src);
        }
        cp_async_commit();
    }
    if (active) {
        const SiteGeom g = site_geometry(a.L, a.parity, cb);
        const uint64_t pol_stream = l2_policy_evict_first();
        const uint64_t pol_keep = l2_policy_evict_last();
        const C *Uf = a.U + (size_t)(a.parity * 12 * NROW) * Vh + cb;          // U_{x,mu}: own parity block
        const C *Ub = a.U + (size_t)((1 - a.parity) * 12 * NROW) * Vh;         // U_{x-mu,mu}: other parity block

        C acc[NRHS][3];
#pragma unroll
        for (int r = 0; r < NRHS; ++r)
            acc[r][0].x = acc[r][0].y = acc[r][1].x = acc[r][1].y = acc[r][2].x = acc[r][2].y = (T)0;
        if (MODE >= 1) {
            // the epilogue reads v(x) after the last hop, when nothing is left to hide a DRAM round
            // trip behind: ask the L2 for it now (no register is held)
#pragma unroll
            for (int r = 0; r < NRHS; ++r)
#pragma unroll
                for (int c = 0; c < 3; ++c) prefetch_l2(a.v[r] + (size_t)c * Vh + cb);
        }

        if (TILE) { cp_async_wait(0); __syncthreads(); }
        // element of the tile that holds site cb itself (row rho + 1 of the R + 2 rows): the x0 neighbours sit in the same row,
        // the x1 neighbours one row up / down
        const int tile_c = a.L.h + (int)threadIdx.x;

#pragma unroll
        for (int mu = 0; mu < 4; ++mu) {
            const C *ufp = Uf + (size_t)(mu * 3 * NROW) * Vh;
            const C *ubp = Ub + (size_t)(mu * 3 * NROW) * Vh + g.nb[mu];
            const T sf = (T)g.sf[mu], sb = (T)g.sb[mu];
            // temporal gauge: U_{x,3} = 1 unless x3 == 0; U_{x-3,3} = 1 unless x3 - 1 == 0
            const bool unit_f = TG && mu == 3 && g.x3 != 0;
            const bool unit_b = TG && mu == 3 && g.x3 != 1;

            if (NRHS <= 2 && !(TG && mu == 3)) {
                // every load of this direction is issued before its first use
                C uf[9], ub[9], pf[NRHS][3], pb[NRHS][3];
                load_link<NROW, C>(uf, ufp, Vh, pol_stream);
                load_link<NROW, C>(ub, ubp, Vh, pol_stream);
#pragma unroll
                for (int r = 0; r < NRHS; ++r) load_spinor<T, C>(pf[r], a.in[r], Vh, g.nf[mu], sf, pol_keep);
#pragma unroll
                for (int r = 0; r < NRHS; ++r) load_spinor<T, C>(pb[r], a.in[r], Vh, g.nb[mu], sb, pol_keep);
                if (NROW == 2) { reconstruct_third_row<C>(uf); reconstruct_third_row<C>(ub); }
#pragma unroll
                for (int r = 0; r < NRHS; ++r) {
                    mat_vec_acc<T, C>(acc[r], uf, pf[r]);
                    matdag_vec_acc<T, C>(acc[r], ub, pb[r]);
                }
            } else if (NRHS <= 2 && sizeof(T) == 4) {
                // temporal gauge, mu = 3, fp32: both neighbour vectors are requested before anything is
                // consumed; the two links are needed on one time slice each only (warp-uniform branches).
                // Measured at 64^4 (burst timings): fp32 two-row D_oe 0.45 -> 0.427 ms, D_eo + epilogue + dot 0.605 -> 0.565;
                // in fp64 the same code is slower at the 128-register cap (0.85 -> 0.92 ms), so fp64 keeps
                // the hop-by-hop form below.
                C pf[NRHS][3], pb[NRHS][3], uf[9], ub[9];
#pragma unroll
                for (int r = 0; r < NRHS; ++r) load_spinor<T, C>(pf[r], a.in[r], Vh, g.nf[mu], sf, pol_keep);
#pragma unroll
                for (int r = 0; r < NRHS; ++r) load_spinor<T, C>(pb[r], a.in[r], Vh, g.nb[mu], sb, pol_keep);
                if (!unit_f) load_link<NROW, C>(uf, ufp, Vh, pol_stream);
                if (!unit_b) load_link<NROW, C>(ub, ubp, Vh, pol_stream);
                if (!unit_f) {
                    if (NROW == 2) reconstruct_third_row<C>(uf);
#pragma unroll
                    for (int r = 0; r < NRHS; ++r) mat_vec_acc<T, C>(acc[r], uf, pf[r]);
                } else {
#pragma unroll
                    for (int r = 0; r < NRHS; ++r) vec_acc<C>(acc[r], pf[r]);
                }
                if (!unit_b) {
                    if (NROW == 2) reconstruct_third_row<C>(ub);
#pragma unroll
                    for (int r = 0; r < NRHS; ++r) matdag_vec_acc<T, C>(acc[r], ub, pb[r]);
                } else {
#pragma unroll
                    for (int r = 0; r < NRHS; ++r) vec_acc<C>(acc[r], pb[r]);
                }
            } else {
                // forward hop then backward hop: one link in registers, reused by every vector
                {
                    C u[9], p[NRHS][3];
                    if (!unit_f) load_link<NROW, C>(u, ufp, Vh, pol_stream);
                    if (TILE && mu < 2) {
                        const int e = mu == 0 ? tile_c + (g.nf[0] - cb) : tile_c + a.L.h;
#pragma unroll
                        for (int r = 0; r < NRHS; ++r) load_spinor_tile<T, C>(p[r], tile + (size_t)(r * 3) * tile_w + e, tile_w, sf);
                    } else {
#pragma unroll
                        for (int r = 0; r < NRHS; ++r) load_spinor<T, C>(p[r], a.in[r], Vh, g.nf[mu], sf, pol_keep);
                    }
                    if (!unit_f) {
                        if (NROW == 2) reconstruct_third_row<C>(u);
#pragma unroll
                        for (int r = 0; r < NRHS; ++r) mat_vec_acc<T, C>(acc[r], u, p[r]);
                    } else {
#pragma unroll
                        for (int r = 0; r < NRHS; ++r) vec_acc<C>(acc[r], p[r]);
                    }
                }
                {
                    C u[9], p[NRHS][3];
                    if (!unit_b) load_link<NROW, C>(u, ubp, Vh, pol_stream);
                    if (TILE && mu < 2) {
                        const int e = mu == 0 ? tile_c + (g.nb[0] - cb) : tile_c - a.L.h;
#pragma unroll
                        for (int r = 0; r < NRHS; ++r) load_spinor_tile<T, C>(p[r], tile + (size_t)(r * 3) * tile_w + e, tile_w, sb);
                    } else {
#pragma unroll
                        for (int r = 0; r < NRHS; ++r) load_spinor<T, C>(p[r], a.in[r], Vh, g.nb[mu], sb, pol_keep);
                    }
                    if (!unit_b) {
                        if (NROW == 2) reconstruct_third_row<C>(u);
#pragma unroll
                        for (int r = 0; r < NRHS; ++r) matdag_vec_acc<T, C>(acc[r], u, p[r]);
                    } else {
#pragma unroll
                        for (int r = 0; r < NRHS; ++r) vec_acc<C>(acc[r], p[r]);
                    }
                }
            }
        }

        dslash_epilogue<T, MODE, NRHS>(a, cb, acc, dot, pol_stream);
    }
    }
    dslash_reduce<T, MODE, NRHS, BLOCK>(a, dot);
}

// ------------------------------------------------------------------------------------------
// Staged variant for several vectors (NRHS >= 3).  With 6 NRHS accumulators per thread the
// register file allows only 8 warps per SM, and a warp that waits for a link from DRAM has
// nothing else to issue: the kernel above is latency-bound there (ncu: 70 % long-scoreboard
// stalls, no memory unit above 45 %).  Here every thread copies its own links with cp.async
// into its own column of shared memory -- DEPTH hops ahead, without holding registers -- and
// reads a link back (conflict-free LDS.128) only when the hop is computed.  No thread reads
// another thread's column, so no block-level barrier is needed: cp.async.wait_group orders a
// thread's copies with its own reads.  Hop h = 2 mu + (0: forward, 1: backward); ring of DEPTH
// hops: after hop h is consumed its column is refilled with hop h + DEPTH.
// ------------------------------------------------------------------------------------------
template <typename T, int MODE, int NROW, int TG, int NRHS, int BLOCK, int MINB, int DEPTH>
__global__ void __launch_bounds__(BLOCK, MINB) dslash_staged_kernel(const DslashArgs<T, NRHS> a)
{
    typedef typename Cplx<T>::type C;
    extern __shared__ __align__(16) unsigned char staged_smem[];
    C (*ring)[BLOCK] = reinterpret_cast<C (*)[BLOCK]>(staged_smem);       // [DEPTH * 3 NROW][BLOCK]
    if (a.check_flag) {
        bool all_done = true;
#pragma unroll
        for (int r = 0; r < NRHS; ++r) all_done = all_done && (a.scal[r].flag != 0);
        if (all_done) return;
    }

    const size_t Vh = (size_t)a.L.Vh;
    double dot[NRHS];
#pragma unroll
    for (int r = 0; r < NRHS; ++r) dot[r] = 0.0;

#pragma unroll 1
    for (int chunk = 0; chunk < (MODE == 2 ? a.chunks : 1); ++chunk) {
    const int tid = (blockIdx.x * (MODE == 2 ? a.chunks : 1) + chunk) * BLOCK + threadIdx.x;
    const bool active = tid < a.L.Vh;
    const int cb = active ? traversal_site(a.L, tid) : tid;
    if (active) {
        const SiteGeom g = site_geometry(a.L, a.parity, cb);
        const uint64_t pol_stream = l2_policy_evict_first();
        const uint64_t pol_keep = l2_policy_evict_last();
        const C *Uf = a.U + (size_t)(a.parity * 12 * NROW) * Vh + cb;
        const C *Ub = a.U + (size_t)((1 - a.parity) * 12 * NROW) * Vh;

        // issue the copies of hop h into ring column h % DEPTH (an empty group for a unit link)
        auto issue = [&](int h) {
            const int mu = h >> 1;
            const bool fwd = (h & 1) == 0;
            const bool unit = TG && mu == 3 && (fwd ? g.x3 != 0 : g.x3 != 1);
            const C *src = fwd ? Uf + (size_t)(mu * 3 * NROW) * Vh : Ub + (size_t)(mu * 3 * NROW) * Vh + g.nb[mu];
            if (!unit) {
#pragma unroll
                for (int k = 0; k < 3 * NROW; ++k)
                    cp_async_stream(&ring[(h % DEPTH) * 3 * NROW + k][threadIdx.x], src + (size_t)k * Vh, pol_stream);
            }
            cp_async_commit();
        };
#pragma unroll
        for (int h = 0; h < DEPTH; ++h) issue(h);

        C acc[NRHS][3];
#pragma unroll
        for (int r = 0; r < NRHS; ++r)
            acc[r][0].x = acc[r][0].y = acc[r][1].x = acc[r][1].y = acc[r][2].x = acc[r][2].y = (T)0;

        // the neighbour vectors of hop h + 1 are requested before hop h is computed when the
        // registers allow a second set (PIPE), so an L2 round trip hides behind 36 NRHS FMAs
        constexpr bool PIPE = (sizeof(T) == 8 ? NRHS <= 4 : NRHS <= 8);
        auto hop_site = [&](int h) { return (h & 1) == 0 ? g.nf[h >> 1] : g.nb[h >> 1]; };
        auto hop_sign = [&](int h) { return (T)((h & 1) == 0 ? g.sf[h >> 1] : g.sb[h >> 1]); };
        C pbuf[PIPE ? 2 : 1][NRHS][3];
        if (PIPE) {
#pragma unroll
            for (int r = 0; r < NRHS; ++r) load_spinor<T, C>(pbuf[0][r], a.in[r], Vh, hop_site(0), hop_sign(0), pol_keep);
        }
#pragma unroll
        for (int h = 0; h < 8; ++h) {
            const int mu = h >> 1;
            const bool fwd = (h & 1) == 0;
            const bool unit = TG && mu == 3 && (fwd ? g.x3 != 0 : g.x3 != 1);
            C (&p)[NRHS][3] = pbuf[PIPE ? (h & 1) : 0];
            if (PIPE) {
                if (h + 1 < 8) {
#pragma unroll
                    for (int r = 0; r < NRHS; ++r)
                        load_spinor<T, C>(pbuf[(h + 1) & 1][r], a.in[r], Vh, hop_site(h + 1), hop_sign(h + 1), pol_keep);
                }
            } else {
#pragma unroll
                for (int r = 0; r < NRHS; ++r) load_spinor<T, C>(p[r], a.in[r], Vh, hop_site(h), hop_sign(h), pol_keep);
            }
            // groups committed so far: min(8, h + DEPTH); hop h needs groups 0 .. h complete
            cp_async_wait((h + DEPTH < 8 ? h + DEPTH : 8) - h - 1);
            if (!unit) {
                C u[9];
#pragma unroll
                for (int k = 0; k < 3 * NROW; ++k) u[k] = ring[(h % DEPTH) * 3 * NROW + k][threadIdx.x];
                if (NROW == 2) reconstruct_third_row<C>(u);
#pragma unroll
                for (int r = 0; r < NRHS; ++r) {
                    if (fwd) mat_vec_acc<T, C>(acc[r], u, p[r]); else matdag_vec_acc<T, C>(acc[r], u, p[r]);
                }
            } else {
#pragma unroll
                for (int r = 0; r < NRHS; ++r) vec_acc<C>(acc[r], p[r]);
            }
            if (h + DEPTH < 8) issue(h + DEPTH);
        }
        dslash_epilogue<T, MODE, NRHS>(a, cb, acc, dot, pol_stream);
    }
    }
    dslash_reduce<T, MODE, NRHS, BLOCK>(a, dot);
}

// ------------------------------------------------------------------------------------------
// Pair variant for an even number of vectors (NRHS = 4, 6, 8): a site is handled by TWO adjacent lanes,
// each with NRHS / 2 of the vectors.  What it is for (profiles/README.md "n >= 3"): with all
// NRHS accumulator sets in one thread the register file allows 8 warps per SM and no second set of neighbour
// vectors, so every hop exposes the L2 latency of its vector loads (one-thread staged kernel: PIPE only up to
// n = 4 in fp64).  Halving the vectors per thread halves accumulators AND vector registers: the next hop's vectors
// are requested before the current hop is computed at every n, under a 168-register cap (12 warps).
// The link is shared through the cp.async ring of the staged kernel: the two lanes copy alternate planes of
// the link into the pair's column, meet at a __syncwarp() after their own cp.async.wait_group, and both read all
// planes (same address: a shared-memory broadcast).  A second __syncwarp() before a column is refilled keeps the
// partner's reads ahead of the overwrite.  No block barrier.  Per vector the FMAs and their order are those of the
// other kernels: results are bitwise identical.  Needs Vh % (BLOCK / 2) == 0 (the host checks).
// ------------------------------------------------------------------------------------------
template <typename T, int MODE, int NROW, int TG, int NRHS, int BLOCK, int MINB, int DEPTH>
__global__ void __launch_bounds__(BLOCK, MINB) dslash_pair_kernel(const DslashArgs<T, NRHS> a)
{
    typedef typename Cplx<T>::type C;
    static_assert(NRHS % 2 == 0, "the pair kernel splits an even number of vectors");
    constexpr int NV = NRHS / 2;                     // vectors per lane: r = half + 2 j
    constexpr int SITES = BLOCK / 2;
    extern __shared__ __align__(16) unsigned char staged_smem[];
    C (*ring)[SITES] = reinterpret_cast<C (*)[SITES]>(staged_smem);        // [DEPTH * 3 NROW][SITES]
    if (a.check_flag) {
        bool all_done = true;
#pragma unroll
        for (int r = 0; r < NRHS; ++r) all_done = all_done && (a.scal[r].flag != 0);
        if (all_done) return;
    }
    const size_t Vh = (size_t)a.L.Vh;
    const int sl = threadIdx.x >> 1, half = threadIdx.x & 1;
    // this lane's vectors, picked with static indices (a runtime index into the parameter arrays would spill them)
    const C *in_[NV], *v_[NV];
    C *out_[NV];
#pragma unroll
    for (int j = 0; j < NV; ++j) {
        in_[j] = half ? a.in[2 * j + 1] : a.in[2 * j];
        out_[j] = half ? a.out[2 * j + 1] : a.out[2 * j];
        v_[j] = half ? a.v[2 * j + 1] : a.v[2 * j];
    }
    double dot[NRHS];
#pragma unroll
    for (int r = 0; r < NRHS; ++r) dot[r] = 0.0;

#pragma unroll 1
    for (int chunk = 0; chunk < (MODE == 2 ? a.chunks : 1); ++chunk) {
        const int tid = (blockIdx.x * (MODE == 2 ? a.chunks : 1) + chunk) * SITES + sl;      // < Vh: Vh % SITES == 0
        const int cb = traversal_site(a.L, tid);
        const SiteGeom g = site_geometry(a.L, a.parity, cb);
        const uint64_t pol_stream = l2_policy_evict_first();
        const uint64_t pol_keep = l2_policy_evict_last();
        const C *Uf = a.U + (size_t)(a.parity * 12 * NROW) * Vh + cb;
        const C *Ub = a.U + (size_t)((1 - a.parity) * 12 * NROW) * Vh;

        // this lane's share of the copies of hop h (an empty group for a unit link)
        auto issue = [&](int h) {
            const int mu = h >> 1;
            const bool fwd = (h & 1) == 0;
            const bool unit = TG && mu == 3 && (fwd ? g.x3 != 0 : g.x3 != 1);
            const C *src = fwd ? Uf + (size_t)(mu * 3 * NROW) * Vh : Ub + (size_t)(mu * 3 * NROW) * Vh + g.nb[mu];
            if (!unit) {
                // planes 2 i + half, no predicate; with nine planes the last one is split into its real and imaginary half
#pragma unroll
                for (int i = 0; i < (3 * NROW) / 2; ++i) {
                    const int k = 2 * i + half;
                    cp_async_stream(&ring[(h % DEPTH) * 3 * NROW + k][sl], src + (size_t)k * Vh, pol_stream);
                }
                if ((3 * NROW) & 1)
                    cp_async_stream_half(&ring[(h % DEPTH) * 3 * NROW + 3 * NROW - 1][sl], src + (size_t)(3 * NROW - 1) * Vh, half, pol_stream);
            }
            cp_async_commit();
        };
#pragma unroll
        for (int h = 0; h < DEPTH; ++h) issue(h);

        C acc[NV][3];
#pragma unroll
        for (int j = 0; j < NV; ++j)
            acc[j][0].x = acc[j][0].y = acc[j][1].x = acc[j][1].y = acc[j][2].x = acc[j][2].y = (T)0;
        if (MODE >= 1) {
#pragma unroll
            for (int j = 0; j < NV; ++j)
#pragma unroll
                for (int c = 0; c < 3; ++c) prefetch_l2(v_[j] + (size_t)c * Vh + cb);
        }

        auto hop_site = [&](int h) { return (h & 1) == 0 ? g.nf[h >> 1] : g.nb[h >> 1]; };
        auto hop_sign = [&](int h) { return (T)((h & 1) == 0 ? g.sf[h >> 1] : g.sb[h >> 1]); };
        C pbuf[2][NV][3];
#pragma unroll
        for (int j = 0; j < NV; ++j) load_spinor<T, C>(pbuf[0][j], in_[j], Vh, hop_site(0), hop_sign(0), pol_keep);
#pragma unroll
        for (int h = 0; h < 8; ++h) {
            const int mu = h >> 1;
            const bool fwd = (h & 1) == 0;
            const bool unit = TG && mu == 3 && (fwd ? g.x3 != 0 : g.x3 != 1);
            C (&p)[NV][3] = pbuf[h & 1];
            if (h + 1 < 8) {
#pragma unroll
                for (int j = 0; j < NV; ++j)
                    load_spinor<T, C>(pbuf[(h + 1) & 1][j], in_[j], Vh, hop_site(h + 1), hop_sign(h + 1), pol_keep);
            }
            cp_async_wait((h + DEPTH < 8 ? h + DEPTH : 8) - h - 1);     // this lane's planes of hop h have landed
            __syncwarp();                                               // ... and so have the partner's
            if (!unit) {
                C u[9];
#pragma unroll
                for (int k = 0; k < 3 * NROW; ++k) u[k] = ring[(h % DEPTH) * 3 * NROW + k][sl];
                if (NROW == 2) reconstruct_third_row<C>(u);
#pragma unroll
                for (int j = 0; j < NV; ++j) {
                    if (fwd) mat_vec_acc<T, C>(acc[j], u, p[j]); else matdag_vec_acc<T, C>(acc[j], u, p[j]);
                }
            } else {
#pragma unroll
                for (int j = 0; j < NV; ++j) vec_acc<C>(acc[j], p[j]);
            }
            __syncwarp();                                               // both lanes have read the column before it is refilled
            if (h + DEPTH < 8) issue(h + DEPTH);
        }

        // epilogue for this lane's vectors (dslash_epilogue, with r = half + 2 j)
        if (MODE >= 1) {
            C vv[NV][3];
#pragma unroll
            for (int j = 0; j < NV; ++j)
#pragma unroll
                for (int c = 0; c < 3; ++c) vv[j][c] = ld_stream(v_[j] + (size_t)c * Vh + cb, pol_stream);
#pragma unroll
            for (int j = 0; j < NV; ++j) {
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    C o;
                    o.x = fma(a.m2, vv[j][c].x, -acc[j][c].x);
                    o.y = fma(a.m2, vv[j][c].y, -acc[j][c].y);
                    out_[j][(size_t)c * Vh + cb] = o;
                    // dot[] is indexed statically: lane `half` owns the even or the odd vectors
                    const double d = (double)vv[j][c].x * (double)o.x + (double)vv[j][c].y * (double)o.y;
                    if (MODE == 2) { if (half == 0) dot[2 * j] += d; else dot[2 * j + 1] += d; }
                }
            }
        } else {
#pragma unroll
            for (int j = 0; j < NV; ++j)
#pragma unroll
                for (int c = 0; c < 3; ++c) out_[j][(size_t)c * Vh + cb] = acc[j][c];
        }
    }
    dslash_reduce<T, MODE, NRHS, BLOCK>(a, dot);
}

// ------------------------------------------------------------------------------------------
// Rolled variant for many vectors (NRHS >= 5).  ncu on the fully unrolled kernels at n = 8 (profiles/README.md, r02):
// 4200 SASS instructions = 68 KB of straight-line code per thread, `gcc__cache_requests_type_instruction` at 78-87 % of
// its peak, every memory unit below 65 %, fp64 pipe at 33-40 % -- and four structurally different kernels (register,
// staged, pair, shared-memory tile) within 3 % of one another.  Eight warps per SM walking 68 KB of code at different
// places miss the 32 KB instruction cache on every line: the kernels are bound by INSTRUCTION FETCH.  Here the loop over
// the four directions is NOT unrolled (the body -- a forward and a backward hop for all vectors -- is a quarter of the
// code, and the neighbour index, phase and seam sign of direction mu are computed arithmetically from mu instead of being
// read from eight-entry arrays).  Per vector the FMAs and their order are those of the other kernels: bitwise identical.
// ------------------------------------------------------------------------------------------
template <typename T, typename C>
__device__ __forceinline__ void load_spinor_neg(C p[3], const C *f, size_t Vh, int site, unsigned neg, uint64_t pol)
{
#pragma unroll
    for (int c = 0; c < 3; ++c) p[c] = ld_keep(f + (size_t)c * Vh + site, pol);
#pragma unroll
    for (int c = 0; c < 3; ++c) { p[c].x = flip_sign(p[c].x, neg); p[c].y = flip_sign(p[c].y, neg); }
}

template <typename T, int MODE, int NROW, int TG, int NRHS, int BLOCK, int MINB>
__global__ void __launch_bounds__(BLOCK, MINB) dslash_rolled_kernel(const DslashArgs<T, NRHS> a)
{
    typedef typename Cplx<T>::type C;
    if (a.check_flag) {
        bool all_done = true;
#pragma unroll
        for (int r = 0; r < NRHS; ++r) all_done = all_done && (a.scal[r].flag != 0);
        if (all_done) return;
    }
    const size_t Vh = (size_t)a.L.Vh;
    double dot[NRHS];
#pragma unroll
    for (int r = 0; r < NRHS; ++r) dot[r] = 0.0;

#pragma unroll 1
    for (int chunk = 0; chunk < (MODE == 2 ? a.chunks : 1); ++chunk) {
    const int tid = (blockIdx.x * (MODE == 2 ? a.chunks : 1) + chunk) * BLOCK + threadIdx.x;
    const bool active = tid < a.L.Vh;
    const int cb = active ? traversal_site(a.L, tid) : tid;
    if (active) {
        // coordinates of the site (lattice.cuh site_geometry, here kept as coordinates: the per-direction quantities are
        // formed inside the rolled loop)
        const unsigned ucb = (unsigned)cb;
        const int xh = (int)(ucb % (unsigned)a.L.h);
        unsigned q = ucb / (unsigned)a.L.h;
        const int x1 = (int)(q % (unsigned)a.L.N1);
        q /= (unsigned)a.L.N1;
        const int x2 = (int)(q % (unsigned)a.L.N2);
        const int x3 = (int)(q / (unsigned)a.L.N2);
        const int rp = (x1 + x2 + x3 + a.parity) & 1;
        const uint64_t pol_stream = l2_policy_evict_first();
        const uint64_t pol_keep = l2_policy_evict_last();
        const C *uf = a.U + (size_t)(a.parity * 12 * NROW) * Vh + cb;          // U_{x,mu}, advanced by one link per direction
        const C *ub = a.U + (size_t)((1 - a.parity) * 12 * NROW) * Vh;         // U_{x-mu,mu}

        C acc[NRHS][3];
#pragma unroll
        for (int r = 0; r < NRHS; ++r)
            acc[r][0].x = acc[r][0].y = acc[r][1].x = acc[r][1].y = acc[r][2].x = acc[r][2].y = (T)0;
        if (MODE >= 1) {
#pragma unroll
            for (int r = 0; r < NRHS; ++r)
#pragma unroll
                for (int c = 0; c < 3; ++c) prefetch_l2(a.v[r] + (size_t)c * Vh + cb);
        }

        int xm = 0, Nm = 0, sm = 1;           // coordinate, extent and cb stride of direction mu (mu = 0 is special-cased)
        unsigned e = 0;                       // eta_mu(x) = (-1)^e,  e = x0 + ... + x_{mu-1} mod 2
#pragma unroll 1
        for (int mu = 0; mu < 4; ++mu) {
            int nf, nb;
            if (mu == 0) {
                nf = rp ? ((xh + 1 == a.L.h) ? cb - (a.L.h - 1) : cb + 1) : cb;
                nb = rp ? cb : ((xh == 0) ? cb + (a.L.h - 1) : cb - 1);
            } else {
                xm = mu == 1 ? x1 : (mu == 2 ? x2 : x3);
                Nm = mu == 1 ? a.L.N1 : (mu == 2 ? a.L.N2 : a.L.N3);
                sm = mu == 1 ? a.L.s1 : (mu == 2 ? a.L.s2 : a.L.s3);
                nf = (xm + 1 == Nm) ? cb - (Nm - 1) * sm : cb + sm;
                nb = (xm == 0) ? cb + (Nm - 1) * sm : cb - sm;
                e = (unsigned)(rp + (mu >= 2 ? x1 : 0) + (mu >= 3 ? x2 : 0)) & 1u;
            }
            const unsigned negf = e ^ ((mu == 3 && x3 + 1 == a.L.N3) ? 1u : 0u);      // eta, times -1 across the time seam
            const unsigned negb = (e ^ 1u) ^ ((mu == 3 && x3 == 0) ? 1u : 0u);        // MINUS eta, times -1 across the seam
            const bool unit_f = TG && mu == 3 && x3 != 0;
            const bool unit_b = TG && mu == 3 && x3 != 1;
            {
                C u[9], p[NRHS][3];
                if (!unit_f) load_link<NROW, C>(u, uf, Vh, pol_stream);
#pragma unroll
                for (int r = 0; r < NRHS; ++r) load_spinor_neg<T, C>(p[r], a.in[r], Vh, nf, negf, pol_keep);
                if (!unit_f) {
                    if (NROW == 2) reconstruct_third_row<C>(u);
#pragma unroll
                    for (int r = 0; r < NRHS; ++r) mat_vec_acc<T, C>(acc[r], u, p[r]);
                } else {
#pragma unroll
                    for (int r = 0; r < NRHS; ++r) vec_acc<C>(acc[r], p[r]);
                }
            }
            {
                C u[9], p[NRHS][3];
                if (!unit_b) load_link<NROW, C>(u, ub + nb, Vh, pol_stream);
#pragma unroll
                for (int r = 0; r < NRHS; ++r) load_spinor_neg<T, C>(p[r], a.in[r], Vh, nb, negb, pol_keep);
                if (!unit_b) {
                    if (NROW == 2) reconstruct_third_row<C>(u);
#pragma unroll
                    for (int r = 0; r < NRHS; ++r) matdag_vec_acc<T, C>(acc[r], u, p[r]);
                } else {
#pragma unroll
                    for (int r = 0; r < NRHS; ++r) vec_acc<C>(acc[r], p[r]);
                }
            }
            uf += (size_t)(3 * NROW) * Vh;
            ub += (size_t)(3 * NROW) * Vh;
        }
        dslash_epilogue<T, MODE, NRHS>(a, cb, acc, dot, pol_stream);
    }
    }
    dslash_reduce<T, MODE, NRHS, BLOCK>(a, dot);
}

} // namespace qcd
