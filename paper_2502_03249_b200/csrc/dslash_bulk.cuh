// Multi-vector Dslash fed by the bulk-copy (TMA) engine: warp-specialised producers and consumers.
//
// Why: every LSU-fed Dslash kernel of this library (register, staged, pair, tile, rolled; any precision, link storage
// and NMULTI) moves 9-11 TB/s of REQUESTED load bytes and no more, while no unit is saturated: the
// loads a SM's few fat warps can keep in flight, about 80 KB, divided by the loaded memory latency.  With one vector
// that is above the HBM rate; with several vectors per link load the neighbour gathers, served by the
// L2, push the requested bytes per site up and the kernel falls off the HBM roofline.  cp.async.bulk moves a whole
// contiguous run with ONE instruction and holds neither registers nor LSU miss entries for it: a ring of shared-memory
// stages keeps 130-200 KB per SM in flight and was measured at 14 TB/s of requested bytes (qcd_stream_bulk).
//
// Shape: a block owns BULK_SITES = 128 consecutive sites of one (x2, x3) plane (R = 128 / h whole x0-rows, h = N0 / 2) at
// a time and walks the lattice with stride gridDim.x.  In the SoA layout everything a HOP of those sites
// needs is a few contiguous runs per plane: the link planes at the sites themselves (forward) or at the neighbour sites
// (backward), and the 3 NRHS vector planes at the neighbour sites -- the same x0-rows for mu = 0 (the +-1 shift inside a
// row is applied when the row is read back), the rows one up / down for mu = 1 (two runs when the (x2, x3) plane wraps),
// all rows displaced by one x2- or x3-plane for mu = 2, 3.
//   producers (BULK_PRODUCERS warps): per hop, wait until the stage is free, announce the bytes, issue the copies -- one
//       tensor-map box per field (the 3 NROW planes of the link, the 3 planes of each vector; 1 + NRHS instructions per
//       hop), or plane by plane with 1-d bulk copies on the few blocks where a run is split;
//   consumers (BULK_SPLIT threads per site, each with its share of the vectors: 8 warps, two per scheduler): per hop,
//       wait until the stage is full, read the link and their vectors from shared memory, release the stage,
//       accumulate -- with the arithmetic of dslash_kernel, hop by hop in the same order, so the results are bitwise
//       those of the other kernels.
// What it reaches and what bounds it (profiles/r02_bulk_copy_kernel.md): fp64 full links at 64^4, n = 8: 3.41 - 3.67 ms against 3.55 - 3.57
// of the register kernel, n = 6: 2.67 - 2.70 against 2.75 - 2.89; DRAM throughput 66 % against 63 % under ncu.  Every operand crosses shared
// memory twice (written by the copy engine, read by the consumers: 152 KB per hop and block at n = 8, 1190 cycles of the 128 B/cycle
// crossbar), which together with the fp64 issue of eight consumer warps is where it stops: on a par, not ahead.  Slower for n <= 5,
// for odd n (the two halves are unequal), on two-row links and in fp32.  Kept as variant 10 (qcd_set_dslash_variant), not dispatched.
#pragma once
#include "dslash.cuh"

namespace qcd {

enum { BULK_SITES = 128, BULK_SPLIT = 2, BULK_CONSUMER_THREADS = BULK_SITES * BULK_SPLIT, BULK_PRODUCERS = 4,
       BULK_BLOCK = BULK_CONSUMER_THREADS + 32 * BULK_PRODUCERS, BULK_RING_MAX = 8 };

template <typename T, int NROW, int NRHS>
struct BulkStage {
    typedef typename Cplx<T>::type C;
    enum { LINK_PLANES = 3 * NROW, PLANES = 3 * NROW + 3 * NRHS, BYTES = PLANES * BULK_SITES * (int)sizeof(C) };
};

// Tensor maps of the fields (lattice.cuh encode_plane_map): rows = planes, inner dimension = the 2 Vh reals of a plane, box = all the
// planes a hop needs of that field (3 NROW of the gauge field, 3 of a vector) x the 128 sites of a block: ONE copy instruction per field and hop.
template <int NRHS>
struct BulkMaps {
    CUtensorMap U;
    CUtensorMap in[NRHS];
};

template <typename T, int MODE, int NROW, int TG, int NRHS>
__global__ void __launch_bounds__(BULK_BLOCK, 1) dslash_bulk_kernel(const DslashArgs<T, NRHS> a, const __grid_constant__ BulkMaps<NRHS> maps,
                                                                    int stages, int ngroups)
{
    typedef typename Cplx<T>::type C;
    typedef BulkStage<T, NROW, NRHS> St;
    constexpr int LP = St::LINK_PLANES, PLANES = St::PLANES;
    extern __shared__ __align__(128) unsigned char bulk_ring[];
    __shared__ __align__(8) unsigned long long full[BULK_RING_MAX], empty[BULK_RING_MAX];
    if (a.check_flag) {
        bool all_done = true;
#pragma unroll
        for (int r = 0; r < NRHS; ++r) all_done = all_done && (a.scal[r].flag != 0);
        if (all_done) return;
    }
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (threadIdx.x == 0) {
        for (int s = 0; s < stages; ++s) { mbar_init(&full[s], BULK_PRODUCERS); mbar_init(&empty[s], BULK_CONSUMER_THREADS / 32); }
        mbar_init_fence();
    }
    __syncthreads();

    const size_t Vh = (size_t)a.L.Vh;
    const int h = a.L.h, R = BULK_SITES / h;
    const C *Uf = a.U + (size_t)(a.parity * 12 * NROW) * Vh;               // U_{x,mu}: own parity block
    const C *Ub = a.U + (size_t)((1 - a.parity) * 12 * NROW) * Vh;         // U_{x-mu,mu}: other parity block

    if (warp >= BULK_CONSUMER_THREADS / 32) {
        // ------------------------------ producers ------------------------------
        const int pw = warp - BULK_CONSUMER_THREADS / 32;
        const uint64_t pol_stream = l2_policy_evict_first();
        const uint64_t pol_keep = l2_policy_evict_last();
        static_assert(St::PLANES <= 64 && NRHS + 1 <= 32 * BULK_PRODUCERS, "copy items of a hop");
        unsigned it = 0;
        for (int gi = blockIdx.x; gi < ngroups; gi += gridDim.x) {
            const int cb0 = traversal_site(a.L, gi * BULK_SITES);
            unsigned q = (unsigned)cb0 / (unsigned)h;
            const int x1_0 = (int)(q % (unsigned)a.L.N1);
            q /= (unsigned)a.L.N1;
            const int x2 = (int)(q % (unsigned)a.L.N2);
            const int x3 = (int)(q / (unsigned)a.L.N2);
#pragma unroll 1
            for (int hop = 0; hop < 8; ++hop, ++it) {
                const int mu = hop >> 1, back = hop & 1;
                const unsigned s = it % (unsigned)stages, use = it / (unsigned)stages;
                // source of the NEIGHBOUR rows.  contiguous: the 128 neighbour sites are one run from site src0 (one box per field);
                // otherwise (mu = 1 where the (x2, x3) plane wraps inside the block) two runs per plane, copied plane by plane
                int src0 = cb0, dst0 = 0, len0 = BULK_SITES, src1 = 0, dst1 = 0, len1 = 0;
                bool contiguous = true;
                if (mu == 1) {
                    const bool wrap = !back ? (x1_0 + R == a.L.N1) : (x1_0 == 0);
                    if (!wrap) src0 = !back ? cb0 + h : cb0 - h;
                    else if (R == 1) src0 = !back ? cb0 - x1_0 * h : cb0 + (a.L.N1 - 1) * h;
                    else {
                        contiguous = false;
                        if (!back) { len0 = (R - 1) * h; src0 = cb0 + h; dst0 = 0; len1 = h; dst1 = (R - 1) * h; src1 = cb0 - x1_0 * h; }
                        else { len0 = (R - 1) * h; src0 = cb0; dst0 = h; len1 = h; dst1 = 0; src1 = cb0 + (a.L.N1 - 1) * h; }
                    }
                } else if (mu == 2) {
                    src0 = !back ? ((x2 + 1 == a.L.N2) ? cb0 - (a.L.N2 - 1) * a.L.s2 : cb0 + a.L.s2)
                                 : ((x2 == 0) ? cb0 + (a.L.N2 - 1) * a.L.s2 : cb0 - a.L.s2);
                } else if (mu == 3) {
                    src0 = !back ? ((x3 + 1 == a.L.N3) ? cb0 - (a.L.N3 - 1) * a.L.s3 : cb0 + a.L.s3)
                                 : ((x3 == 0) ? cb0 + (a.L.N3 - 1) * a.L.s3 : cb0 - a.L.s3);
                }
                const bool unit = TG && mu == 3 && (!back ? x3 != 0 : x3 != 1);   // temporal gauge: this hop's link is the identity
                unsigned char *stage = bulk_ring + (size_t)s * St::BYTES;
                if (contiguous) {
                    // field f = 0: the link (forward: at the sites themselves), f = 1 .. NRHS: vector f - 1; field f belongs to
                    // producer warp f % BULK_PRODUCERS, lane f / BULK_PRODUCERS
                    const int f = lane * BULK_PRODUCERS + pw;
                    const bool mine = f <= NRHS && !(f == 0 && unit);
                    const unsigned bytes = !mine ? 0u : (unsigned)((f == 0 ? LP : 3) * BULK_SITES * sizeof(C));
                    const unsigned warp_bytes = __reduce_add_sync(0xffffffffu, bytes);
                    if (use > 0) mbar_wait(&empty[s], (use & 1u) ^ 1u);
                    if (lane == 0) mbar_arrive_expect_tx(&full[s], warp_bytes);
                    __syncwarp();
                    if (mine) {
                        if (f == 0) {
                            tensor_copy_g2s(stage, &maps.U, 2 * (back ? src0 : cb0), ((back ? 1 - a.parity : a.parity) * 4 + mu) * LP, &full[s], pol_stream);
                        } else {
                            const CUtensorMap *m = &maps.in[0];
#pragma unroll
                            for (int r = 1; r < NRHS; ++r) m = (f - 1 == r) ? &maps.in[r] : m;
                            tensor_copy_g2s(stage + (size_t)(LP + 3 * (f - 1)) * BULK_SITES * sizeof(C), m, 2 * src0, 0, &full[s], pol_keep);
                        }
                    }
                } else {
                    // items (plane, run): item i belongs to producer warp i % BULK_PRODUCERS; a lane walks its items twice, once to add up the
                    // bytes it will announce, once to issue the copies
                    auto item_copy = [&](int item, const C *&src, int &len, int &dst, uint64_t &pol) {
                        const int plane = item & 63, run = item >> 6;
                        src = nullptr; len = 0; dst = 0; pol = pol_keep;
                        if (plane >= PLANES) return plane;
                        if (plane < LP) {
                            if (unit) return plane;
                            pol = pol_stream;
                            if (!back) {    // forward link: at the sites themselves, one run
                                if (run == 0) { src = Uf + (size_t)(mu * LP + plane) * Vh + cb0; len = BULK_SITES; dst = 0; }
                            } else {
                                const C *base = Ub + (size_t)(mu * LP + plane) * Vh;
                                if (run == 0) { src = base + src0; len = len0; dst = dst0; }
                                else { src = base + src1; len = len1; dst = dst1; }
                            }
                        } else {
                            const int v = plane - LP;                       // vector v / 3, colour v % 3
                            const C *base = a.in[0];
#pragma unroll
                            for (int r = 1; r < NRHS; ++r) base = (v / 3 == r) ? a.in[r] : base;   // static indices: no local-memory copy of the argument array
                            base += (size_t)(v % 3) * Vh;
                            if (run == 0) { src = base + src0; len = len0; dst = dst0; }
                            else { src = base + src1; len = len1; dst = dst1; }
                        }
                        return plane;
                    };
                    unsigned bytes = 0;
                    for (int item = lane * BULK_PRODUCERS + pw; item < 128; item += 32 * BULK_PRODUCERS) {
                        const C *src; int len, dst; uint64_t pol;
                        item_copy(item, src, len, dst, pol);
                        bytes += (unsigned)len * (unsigned)sizeof(C);
                    }
                    const unsigned warp_bytes = __reduce_add_sync(0xffffffffu, bytes);
                    if (use > 0) mbar_wait(&empty[s], (use & 1u) ^ 1u);
                    if (lane == 0) mbar_arrive_expect_tx(&full[s], warp_bytes);
                    __syncwarp();
                    for (int item = lane * BULK_PRODUCERS + pw; item < 128; item += 32 * BULK_PRODUCERS) {
                        const C *src; int len, dst; uint64_t pol;
                        const int plane = item_copy(item, src, len, dst, pol);
                        if (len) bulk_copy_g2s(stage + ((size_t)plane * BULK_SITES + dst) * sizeof(C), src, (unsigned)len * (unsigned)sizeof(C), &full[s], pol);
                    }
                }
            }
        }
    } else {
        // ------------------------------ consumers: BULK_SPLIT threads per site, each with its share of the vectors ------------------------------
        // (two warps per scheduler: one warp alone cannot keep the fp64 pipe busy across its own shared-memory reads)
        const int t = (int)threadIdx.x & (BULK_SITES - 1), part = (int)threadIdx.x / BULK_SITES;
        constexpr int NV = (NRHS + BULK_SPLIT - 1) / BULK_SPLIT;           // vectors per thread: r = part * NV + j
        const int r0 = part * NV;
        C *out_[NV];
#pragma unroll
        for (int j = 0; j < NV; ++j) {
            out_[j] = a.out[j];
#pragma unroll
            for (int q = 1; q < BULK_SPLIT; ++q) out_[j] = (part == q) ? (q * NV + j < NRHS ? a.out[q * NV + j < NRHS ? q * NV + j : 0] : nullptr) : out_[j];
        }
        unsigned it = 0;
        for (int gi = blockIdx.x; gi < ngroups; gi += gridDim.x) {
            const int cb0 = traversal_site(a.L, gi * BULK_SITES);
            const int cb = cb0 + t;
            const SiteGeom g = site_geometry(a.L, a.parity, cb);
            C acc[NV][3];
#pragma unroll
            for (int j = 0; j < NV; ++j)
                acc[j][0].x = acc[j][0].y = acc[j][1].x = acc[j][1].y = acc[j][2].x = acc[j][2].y = (T)0;
#pragma unroll
            for (int mu = 0; mu < 4; ++mu) {
#pragma unroll
                for (int back = 0; back < 2; ++back, ++it) {
                    const unsigned s = it % (unsigned)stages, use = it / (unsigned)stages;
                    const C *st = reinterpret_cast<const C *>(bulk_ring + (size_t)s * St::BYTES);
                    const T sign = (T)(back ? g.sb[mu] : g.sf[mu]);
                    const bool unit = TG && mu == 3 && (!back ? g.x3 != 0 : g.x3 != 1);
                    // element of the stage that holds this site's neighbour: rows were placed by the producers, the x0 shift is applied here
                    const int e = mu == 0 ? (back ? g.nb[0] : g.nf[0]) - cb0 : t;
                    mbar_wait(&full[s], use & 1u);
                    C u[9], p[NV][3];
                    if (!unit) {
#pragma unroll
                        for (int k = 0; k < LP; ++k) u[k] = st[k * BULK_SITES + (back ? e : t)];
                    }
#pragma unroll
                    for (int j = 0; j < NV; ++j) {
                        const int r = r0 + j < NRHS ? r0 + j : NRHS - 1;      // a thread without a j-th vector re-reads the last one and drops the result
                        load_spinor_tile<T, C>(p[j], st + (size_t)(LP + 3 * r) * BULK_SITES + e, BULK_SITES, sign);
                    }
                    __syncwarp();
                    if (lane == 0) mbar_arrive(&empty[s]);
                    if (!unit) {
                        if (NROW == 2) reconstruct_third_row<C>(u);
#pragma unroll
                        for (int j = 0; j < NV; ++j) {
                            if (!back) mat_vec_acc<T, C>(acc[j], u, p[j]);
                            else matdag_vec_acc<T, C>(acc[j], u, p[j]);
                        }
                    } else {
#pragma unroll
                        for (int j = 0; j < NV; ++j) vec_acc<C>(acc[j], p[j]);
                    }
                }
            }
#pragma unroll
            for (int j = 0; j < NV; ++j)
                if (out_[j]) {
#pragma unroll
                    for (int c = 0; c < 3; ++c) out_[j][(size_t)c * Vh + cb] = acc[j][c];
                }
        }
    }
}

} // namespace qcd
