// Dispatch from a runtime DslashLaunch to one instantiation of dslash_kernel.  Included by the
// four dslash_*.cu translation units, each of which instantiates launch_dslash_impl once.
#pragma once
#include "dslash.cuh"
#include "dslash_bulk.cuh"
#include "dslash_launch.h"

namespace qcd {

// Block shape per (precision, NRHS): 128 threads; the minimum resident blocks per SM fixes the
// register cap (65536 / (128 * MINB)): accumulators grow by 6 reals per extra vector.
template <typename T, int NRHS> struct DslashCfg;
template <> struct DslashCfg<double, 1> { enum { BLOCK = 128, MINB = 4 }; };
template <> struct DslashCfg<double, 2> { enum { BLOCK = 128, MINB = 3 }; };
template <> struct DslashCfg<double, 3> { enum { BLOCK = 128, MINB = 2 }; };
template <> struct DslashCfg<double, 4> { enum { BLOCK = 128, MINB = 2 }; };
template <> struct DslashCfg<double, 5> { enum { BLOCK = 128, MINB = 2 }; };
template <> struct DslashCfg<double, 6> { enum { BLOCK = 128, MINB = 2 }; };
template <> struct DslashCfg<double, 7> { enum { BLOCK = 128, MINB = 2 }; };
template <> struct DslashCfg<double, 8> { enum { BLOCK = 128, MINB = 2 }; };
template <> struct DslashCfg<float, 1> { enum { BLOCK = 128, MINB = 4 }; };
template <> struct DslashCfg<float, 2> { enum { BLOCK = 128, MINB = 4 }; };
template <> struct DslashCfg<float, 3> { enum { BLOCK = 128, MINB = 4 }; };
template <> struct DslashCfg<float, 4> { enum { BLOCK = 128, MINB = 3 }; };
template <> struct DslashCfg<float, 5> { enum { BLOCK = 128, MINB = 3 }; };
template <> struct DslashCfg<float, 6> { enum { BLOCK = 128, MINB = 3 }; };
template <> struct DslashCfg<float, 7> { enum { BLOCK = 128, MINB = 2 }; };
template <> struct DslashCfg<float, 8> { enum { BLOCK = 128, MINB = 2 }; };

// Temporal-gauge kernels for one vector (TG = 1, NRHS = 1) move 27-55 % fewer bytes per site with the
// same index arithmetic, run below the DRAM limit and are sensitive to how many warps are resident
// and to how far ptxas hoists loads under the register cap.  Occupancy sweep at 64^4 fp64 (MINB = 2 ... 8,
// DESIGN.md Sec. 10 "Occupancy of the temporal-gauge kernels"):
//   * MODE 2 (D_eo + epilogue + dot) wants 6 blocks (80 registers, 24 warps; the chunk loop makes ptxas
//     fill a 128-register cap without putting more loads in flight): two-row 1.11 -> 0.96 ms, full 1.58 -> 1.34;
//   * MODE 0 / 1 on full links want 3 blocks (168-register cap: the loads of the next direction are
//     hoisted over the current one's FMAs): 1.44 -> 1.17-1.20 ms; on two-row links 4 blocks stay best.
// fp32 kernels keep 4 blocks everywhere (their registers hold twice the loads already).
// The plain one-vector Dslash on full links (MODE 0: D_oe, D_eo; the headline kernel) runs with THREE resident blocks (168-register
// cap: ptxas hoists the next direction's loads over the current FMAs).  A/B in alternating runs of 40 launches (round 2, variant knob):
// fp32 24^4 18.7 -> 16.6 us, 32^4 51.5 -> 47.4, 48^3 x 12 65.4 -> 60.7, 64^4 756.7 -> 739.3 (-2.3 %); fp64 24^4 31.0 -> 30.0, 32^4
// 95.1 -> 94.1, 48^3 x 12 and 64^4 -0.1 ... -0.2 %.  The reducing kernel (MODE 2) is slower that way (fp32 CG iteration 1.850 -> 1.858 ms
// with both kernels at 3 blocks although D_oe alone gains 0.022 ms) and keeps 4.
template <typename T, int MODE, int NROW, int TG, int NRHS>
struct DslashTune {
    enum { BLOCK = DslashCfg<T, NRHS>::BLOCK,
           MINB = (sizeof(T) == 8 && TG == 1 && NRHS == 1) ? (MODE == 2 ? 6 : (NROW == 3 ? 3 : DslashCfg<T, NRHS>::MINB))
                : (NRHS == 1 && TG == 0 && MODE == 0 && NROW == 3) ? 3
                                                            : DslashCfg<T, NRHS>::MINB };
};

// Kernels that end with a block reduction (MODE 2) walk several chunks of BLOCK sites per block so
// that the ~2 us reduction tail is paid once per several hundred sites, not by every 128: the grid
// is sized to about REDUCE_GRID blocks (32 waves of 148 SMs x 4 resident blocks; 4 chunks per block
// at 64^4).  Measured at 64^4: fewer, longer blocks (14 chunks) lose more in the last wave than they
// save (fp64 epilogue kernel 1.58 -> 1.68 ms), and a grid-stride order of the chunks is slower still.
enum { REDUCE_GRID = 148 * 4 * 32 };
static inline int reduce_chunks(int Vh, int block)
{
    const int blocks = (Vh + block - 1) / block;
    const int c = (blocks + REDUCE_GRID - 1) / REDUCE_GRID;
    return c < 1 ? 1 : c;
}

template <typename T, int MODE, int NROW, int TG, int NRHS, int BLOCK, int MINB>
static cudaError_t launch_cfg(const DslashLaunch &d)
{
    typedef typename Cplx<T>::type C;
    DslashArgs<T, NRHS> a;
    a.L = d.L; a.parity = d.parity; a.U = (const C *)d.U;
    for (int r = 0; r < NRHS; ++r) { a.in[r] = (const C *)d.in[r]; a.out[r] = (C *)d.out[r]; a.v[r] = (const C *)d.v[r]; }
    a.m2 = (T)d.m2; a.partials = d.partials; a.scal = d.scal; a.check_flag = d.check_flag;
    a.chunks = MODE == 2 ? reduce_chunks(d.L.Vh, BLOCK) : 1;
    const int per_block = BLOCK * a.chunks;
    const int grid = (d.L.Vh + per_block - 1) / per_block;
    dslash_kernel<T, MODE, NROW, TG, NRHS, BLOCK, MINB><<<grid, BLOCK, 0, d.stream>>>(a);
    return cudaGetLastError();
}

// Register kernel with the x0 / x1 neighbour rows of a block in shared memory (dslash.cuh, TILE).  Needs a block to be whole
// x0-rows of one (x2, x3) plane: BLOCK % h == 0, N1 % (BLOCK / h) == 0 (then Vh % BLOCK == 0 and the traversal chunks, whole
// x2-rows, keep a block's sites consecutive).
static inline bool tile_eligible(const Lattice &L, int block)
{
    return L.h <= block && block % L.h == 0 && L.N1 % (block / L.h) == 0;
}
template <typename T, int MODE, int NROW, int TG, int NRHS>
static cudaError_t launch_tile(const DslashLaunch &d)
{
    typedef typename Cplx<T>::type C;
    enum { BLOCK = DslashCfg<T, NRHS>::BLOCK, MINB = DslashCfg<T, NRHS>::MINB };
    const size_t smem = (size_t)NRHS * 3 * (BLOCK + 2 * d.L.h) * sizeof(C);
    auto kernel = dslash_kernel<T, MODE, NROW, TG, NRHS, BLOCK, MINB, true>;
    {
        const cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
    }
    DslashArgs<T, NRHS> a;
    a.L = d.L; a.parity = d.parity; a.U = (const C *)d.U;
    for (int r = 0; r < NRHS; ++r) { a.in[r] = (const C *)d.in[r]; a.out[r] = (C *)d.out[r]; a.v[r] = (const C *)d.v[r]; }
    a.m2 = (T)d.m2; a.partials = d.partials; a.scal = d.scal; a.check_flag = d.check_flag;
    a.chunks = MODE == 2 ? reduce_chunks(d.L.Vh, BLOCK) : 1;
    while (a.chunks > 1 && (d.L.Vh / BLOCK) % a.chunks) --a.chunks;
    const int grid = d.L.Vh / (BLOCK * a.chunks);
    kernel<<<grid, BLOCK, smem, d.stream>>>(a);
    return cudaGetLastError();
}

template <typename T, int MODE, int NROW, int TG, int NRHS>
static cudaError_t launch_rolled(const DslashLaunch &d)
{
    typedef typename Cplx<T>::type C;
    enum { BLOCK = DslashCfg<T, NRHS>::BLOCK, MINB = DslashCfg<T, NRHS>::MINB };
    DslashArgs<T, NRHS> a;
    a.L = d.L; a.parity = d.parity; a.U = (const C *)d.U;
    for (int r = 0; r < NRHS; ++r) { a.in[r] = (const C *)d.in[r]; a.out[r] = (C *)d.out[r]; a.v[r] = (const C *)d.v[r]; }
    a.m2 = (T)d.m2; a.partials = d.partials; a.scal = d.scal; a.check_flag = d.check_flag;
    a.chunks = MODE == 2 ? reduce_chunks(d.L.Vh, BLOCK) : 1;
    const int per_block = BLOCK * a.chunks;
    const int grid = (d.L.Vh + per_block - 1) / per_block;
    dslash_rolled_kernel<T, MODE, NROW, TG, NRHS, BLOCK, MINB><<<grid, BLOCK, 0, d.stream>>>(a);
    return cudaGetLastError();
}

// Staged kernel (links through shared memory by cp.async, dslash.cuh): ring of STAGE_DEPTH hops.
enum { STAGE_DEPTH = 4 };
template <typename T, int NRHS> struct StagedCfg { enum { BLOCK = 128, MINB = sizeof(T) == 8 ? (NRHS <= 4 ? 3 : 2) : (NRHS <= 4 ? 4 : 3) }; };

// Kernel and register cap of the PLAIN multi-vector Dslash (MODE 0) per (precision, link storage, temporal gauge, n), where a sweep of
// one resident block more / less for both kernels beat the general rule below by >= 4 % (round 2; 64^4, best of two runs of 10
// launches per choice, all choices in one process sequence; profiles/README.md "register caps"): mostly the REGISTER kernel with one
// block more than DslashCfg gives it -- more warps at a tighter cap beat the cp.async ring where both fit.
//   kernel: 0 = the general rule, 1 = register kernel, 2 = staged kernel;  minb = resident blocks of 128 threads
struct Mode0Choice { int kernel, minb; };
template <typename T>
constexpr Mode0Choice mode0_choice(int nrow, int tg, int n)
{
    if (sizeof(T) == 8) {
        if (nrow == 3 && !tg && n >= 3 && n <= 6) return {1, 3};      // 1.84 -> 1.74 (n = 3), 2.14 -> 1.97 (4), 2.85 -> 2.70 ms (6)
        if (nrow == 2 && !tg && n == 6) return {2, 3};                  // 2.50 -> 2.31 ms
        if (nrow == 2 && n == 5) return {2, 2};                         // staged instead of register: 2.29 -> 2.01, in temporal gauge 2.24 -> 1.97 ms
        if (!tg && n == 8) return {2, 2};                               // staged instead of register: full links 3.53 -> 3.32, two-row 3.31 -> 3.05 ms
    } else {
        if (nrow == 3 && !tg && n == 3) return {1, 5};                  // 0.982 -> 0.870 ms
        if (nrow == 3 && !tg && n >= 4 && n <= 6) return {1, 4};        // 1.095 -> 1.009 (4), 1.487 -> 1.341 ms (6)
        if (nrow == 2 && !tg && (n == 2 || n == 3)) return {1, 5};      // 0.612 -> 0.587, 0.777 -> 0.740 ms
        if (nrow == 2 && !tg && n == 6) return {1, 4};                  // 1.293 -> 1.207 ms
        if (nrow == 2 && !tg && n == 8) return {2, 4};                  // 1.670 -> 1.594 ms
        if (nrow == 2 && tg && n == 2) return {2, 5};                   // 0.622 -> 0.561 ms
        if (nrow == 2 && tg && n == 6) return {1, 4};                   // 1.206 -> 1.139 ms
    }
    return {0, 0};
}
// The same sweep for the REDUCING kernel (MODE 2), timed inside the lock-step CG iteration (CUDA events per launch): the round-1
// choices are within 3 % of the best everywhere except here.  (The MODE 0 choices do not carry over: applied to MODE 2 they cost up
// to 48 %.)
template <typename T>
constexpr Mode0Choice mode2_choice(int nrow, int tg, int n)
{
    if (sizeof(T) == 8) {
        if (nrow == 2 && tg && n == 2) return {1, 4};                   // 1.513 -> 1.421 ms
        if (nrow == 3 && !tg && n == 3) return {1, 3};                  // 2.378 -> 2.264 ms
        if (nrow == 2 && tg && n == 4) return {1, 3};                   // 2.148 -> 2.062 ms
    } else {
        if (nrow == 2 && tg && n == 2) return {2, 5};                   // 0.767 -> 0.685 ms
        if (nrow == 2 && !tg && n == 8) return {1, 3};                  // 2.684 -> 2.386 ms
    }
    return {0, 0};
}

template <typename T, int MODE, int NROW, int TG, int NRHS, int MINB_OVERRIDE = 0>
static cudaError_t launch_staged(const DslashLaunch &d)
{
    typedef typename Cplx<T>::type C;
    enum { BLOCK = StagedCfg<T, NRHS>::BLOCK, MINB = MINB_OVERRIDE > 0 ? MINB_OVERRIDE : (int)StagedCfg<T, NRHS>::MINB };
    const size_t smem = (size_t)STAGE_DEPTH * 3 * NROW * BLOCK * sizeof(C);
    auto kernel = dslash_staged_kernel<T, MODE, NROW, TG, NRHS, BLOCK, MINB, STAGE_DEPTH>;
    // the attribute belongs to the (function, device) pair: set on every launch (a host-side table update, no device
    // work) rather than cached per process, which a second device or a second thread would get wrong
    {
        const cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
    }
    DslashArgs<T, NRHS> a;
    a.L = d.L; a.parity = d.parity; a.U = (const C *)d.U;
    for (int r = 0; r < NRHS; ++r) { a.in[r] = (const C *)d.in[r]; a.out[r] = (C *)d.out[r]; a.v[r] = (const C *)d.v[r]; }
    a.m2 = (T)d.m2; a.partials = d.partials; a.scal = d.scal; a.check_flag = d.check_flag;
    a.chunks = MODE == 2 ? reduce_chunks(d.L.Vh, BLOCK) : 1;
    const int per_block = BLOCK * a.chunks;
    const int grid = (d.L.Vh + per_block - 1) / per_block;
    kernel<<<grid, BLOCK, smem, d.stream>>>(a);
    return cudaGetLastError();
}

// Pair kernel (two lanes per site, NRHS / 2 vectors each; dslash.cuh): 128 threads = 64 sites per block.
enum { PAIR_BLOCK = 128, PAIR_DEPTH = 4 };
template <typename T, int MODE, int NROW, int TG, int NRHS, int MINB>
static cudaError_t launch_pair(const DslashLaunch &d)
{
    typedef typename Cplx<T>::type C;
    const size_t smem = (size_t)PAIR_DEPTH * 3 * NROW * (PAIR_BLOCK / 2) * sizeof(C);
    auto kernel = dslash_pair_kernel<T, MODE, NROW, TG, NRHS, PAIR_BLOCK, MINB, PAIR_DEPTH>;
    {
        const cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
    }
    DslashArgs<T, NRHS> a;
    a.L = d.L; a.parity = d.parity; a.U = (const C *)d.U;
    for (int r = 0; r < NRHS; ++r) { a.in[r] = (const C *)d.in[r]; a.out[r] = (C *)d.out[r]; a.v[r] = (const C *)d.v[r]; }
    a.m2 = (T)d.m2; a.partials = d.partials; a.scal = d.scal; a.check_flag = d.check_flag;
    const int sites = PAIR_BLOCK / 2;
    a.chunks = MODE == 2 ? reduce_chunks(d.L.Vh, sites) : 1;
    while (a.chunks > 1 && (d.L.Vh / sites) % a.chunks) --a.chunks;       // whole chunks only: every lane of the block is active
    const int grid = d.L.Vh / (sites * a.chunks);
    kernel<<<grid, PAIR_BLOCK, smem, d.stream>>>(a);
    return cudaGetLastError();
}

// Bulk-copy kernel (dslash_bulk.cuh): needs a block's 128 sites to be whole x0-rows of one (x2, x3) plane.
static inline bool bulk_eligible(const Lattice &L) { return tile_eligible(L, BULK_SITES) && L.Vh % BULK_SITES == 0; }
template <typename T, int MODE, int NROW, int TG, int NRHS>
static cudaError_t launch_bulk(const DslashLaunch &d)
{
    typedef typename Cplx<T>::type C;
    typedef BulkStage<T, NROW, NRHS> St;
    int dev = 0, sms = 0, max_smem = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&max_smem, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
    if (e != cudaSuccess) return e;
    int stages = (max_smem - 1024) / (int)St::BYTES;
    if (stages > BULK_RING_MAX) stages = BULK_RING_MAX;
    if (stages < 2) return cudaErrorInvalidValue;
    const size_t smem = (size_t)stages * St::BYTES;
    auto kernel = dslash_bulk_kernel<T, MODE, NROW, TG, NRHS>;
    e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    DslashArgs<T, NRHS> a;
    a.L = d.L; a.parity = d.parity; a.U = (const C *)d.U;
    for (int r = 0; r < NRHS; ++r) { a.in[r] = (const C *)d.in[r]; a.out[r] = (C *)d.out[r]; a.v[r] = (const C *)d.v[r]; }
    a.m2 = (T)d.m2; a.partials = d.partials; a.scal = d.scal; a.check_flag = d.check_flag; a.chunks = 1;
    BulkMaps<NRHS> maps;
    const bool f64 = sizeof(T) == 8;
    e = encode_plane_map(&maps.U, f64, d.U, 2ull * d.L.Vh, 24ull * NROW, (unsigned long long)d.L.Vh * sizeof(C), 2 * BULK_SITES, 3 * NROW);
    for (int r = 0; r < NRHS && e == cudaSuccess; ++r)
        e = encode_plane_map(&maps.in[r], f64, d.in[r], 2ull * d.L.Vh, 3, (unsigned long long)d.L.Vh * sizeof(C), 2 * BULK_SITES, 3);
    if (e != cudaSuccess) return e;
    const int ngroups = d.L.Vh / BULK_SITES;
    const int grid = ngroups < sms ? ngroups : sms;
    kernel<<<grid, BULK_BLOCK, smem, d.stream>>>(a, maps, stages, ngroups);
    return cudaGetLastError();
}

template <typename T, int MODE, int NROW, int TG, int NRHS>
static cudaError_t launch_nrhs(const DslashLaunch &d)
{
    // variant 10 forces the bulk-copy (TMA) kernel where the lattice allows it.  Not dispatched: at 64^4 on full fp64 links it is on a par
    // with the register kernel for 6 and 8 vectors (2.67 - 2.70 / 3.41 - 3.67 ms against 2.75 - 2.89 / 3.55 - 3.57 from run to run), 11 % slower for 7
    // (the two consumer halves hold 4 and 3 vectors) and slower everywhere else (profiles/r02_bulk_copy_kernel.md)
    if constexpr (MODE == 0 && NRHS >= 2) {
        if (d.variant == 10 && bulk_eligible(d.L)) return launch_bulk<T, MODE, NROW, TG, NRHS>(d);
    }
    // variants 6 / 7 force the pair kernel at a 168- / 128-register cap (A/B sweeps); it needs an even number of vectors
    // and a volume of whole 64-site blocks
    // variant 9 forces the rolled kernel (direction loop not unrolled: a quarter of the code; dslash.cuh)
    if constexpr (MODE != 1 && NRHS >= 3) {
        if (d.variant == 9) return launch_rolled<T, MODE, NROW, TG, NRHS>(d);
    }
    // variant 8 forces the register kernel with the shared-memory tile of the x0 / x1 neighbour rows
    if constexpr (MODE != 1 && (NRHS == 4 || NRHS == 8)) {
        if (d.variant == 8 && tile_eligible(d.L, DslashCfg<T, NRHS>::BLOCK) &&
            (size_t)NRHS * 3 * (DslashCfg<T, NRHS>::BLOCK + 2 * d.L.h) * sizeof(typename Cplx<T>::type) <= 200 * 1024)
            return launch_tile<T, MODE, NROW, TG, NRHS>(d);
    }
    if constexpr (MODE != 1 && NRHS >= 4 && NRHS % 2 == 0) {
        if ((d.variant == 6 || d.variant == 7) && d.L.Vh % (PAIR_BLOCK / 2) == 0)
            return d.variant == 6 ? launch_pair<T, MODE, NROW, TG, NRHS, 3>(d) : launch_pair<T, MODE, NROW, TG, NRHS, 4>(d);
    }
    // variant 4 forces the staged kernel, variant 5 the register kernel (A/B sweeps); otherwise the
    // staged kernel serves the (precision, NRHS, link rows) where it measured faster at 64^4
    // (profiles/README.md "staged vs register kernel"): fp64 n = 3, 4; fp32 n = 8, and n >= 4 on two-row links
    if constexpr (MODE != 1 && NRHS >= 2) {
        constexpr Mode0Choice c = MODE == 0 ? mode0_choice<T>(NROW, TG, NRHS) : mode2_choice<T>(NROW, TG, NRHS);
        if (d.variant == 0) {
            if constexpr (c.kernel == 1) return launch_cfg<T, MODE, NROW, TG, NRHS, 128, c.minb>(d);
            if constexpr (c.kernel == 2) return launch_staged<T, MODE, NROW, TG, NRHS, c.minb>(d);
        }
    }
    if constexpr (MODE != 1) {
        // (the reducing kernel, MODE 2, on full links is 3-5 % faster as the register kernel at n = 3, 4: 2.35 / 2.71 ms
        // against 2.42 / 2.86 -- ncu shows the staged MODE 2 kernel requesting every link sector from the L2 twice)
        constexpr bool staged_wins = sizeof(T) == 8 ? ((NRHS == 3 || NRHS == 4) && !(MODE == 2 && NROW == 3))
                                                    : (NRHS == 8 || (NROW == 2 && NRHS >= 4));
        if (d.variant == 4 || (d.variant != 5 && staged_wins)) return launch_staged<T, MODE, NROW, TG, NRHS>(d);
    }
    if constexpr (NRHS == 1 && TG == 0) {
        switch (d.variant) {       // block-shape sweep of the headline kernel
        case 1: return launch_cfg<T, MODE, NROW, TG, 1, 64, 8>(d);
        case 2: return launch_cfg<T, MODE, NROW, TG, 1, 256, 2>(d);
        case 3: return launch_cfg<T, MODE, NROW, TG, 1, 128, (DslashTune<T, MODE, NROW, TG, 1>::MINB == 3 ? 4 : 3)>(d);   // the OTHER of 3 / 4
        default: break;
        }
    }
    return launch_cfg<T, MODE, NROW, TG, NRHS, DslashTune<T, MODE, NROW, TG, NRHS>::BLOCK, DslashTune<T, MODE, NROW, TG, NRHS>::MINB>(d);
}

template <typename T, int MODE, int NROW, int TG>
static cudaError_t launch_tg(const DslashLaunch &d)
{
    if constexpr (MODE == 1) return d.nrhs == 1 ? launch_nrhs<T, MODE, NROW, TG, 1>(d) : cudaErrorInvalidValue;
    else switch (d.nrhs) {
    case 1: return launch_nrhs<T, MODE, NROW, TG, 1>(d);
    case 2: return launch_nrhs<T, MODE, NROW, TG, 2>(d);
    case 3: return launch_nrhs<T, MODE, NROW, TG, 3>(d);
    case 4: return launch_nrhs<T, MODE, NROW, TG, 4>(d);
    case 5: return launch_nrhs<T, MODE, NROW, TG, 5>(d);
    case 6: return launch_nrhs<T, MODE, NROW, TG, 6>(d);
    case 7: return launch_nrhs<T, MODE, NROW, TG, 7>(d);
    case 8: return launch_nrhs<T, MODE, NROW, TG, 8>(d);
    default: return cudaErrorInvalidValue;
    }
}

template <typename T, int NROW>
static cudaError_t launch_dslash_impl(const DslashLaunch &d)
{
    switch (d.mode * 2 + (d.tg ? 1 : 0)) {
    case 0: return launch_tg<T, 0, NROW, 0>(d);
    case 1: return launch_tg<T, 0, NROW, 1>(d);
    case 2: return launch_tg<T, 1, NROW, 0>(d);
    case 3: return launch_tg<T, 1, NROW, 1>(d);
    case 4: return launch_tg<T, 2, NROW, 0>(d);
    case 5: return launch_tg<T, 2, NROW, 1>(d);
    default: return cudaErrorInvalidValue;
    }
}

} // namespace qcd
