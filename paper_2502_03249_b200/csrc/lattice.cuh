// Lattice geometry, device field layout and memory-access helpers shared by the kernels.
//
// Layout (include/qcd.h; "Structure of Arrays ... all even sites are listed first,
// followed by all odd sites"): idx = x0 + N0 (x1 + N1 (x2 + N2 x3)), cb = idx >> 1, every
// complex component of a field is one plane of Vh contiguous (re, im) pairs.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace qcd {

struct Lattice {
    int N0, N1, N2, N3;
    int h;        // N0 / 2 : checkerboard sites per x0-row
    int Vh;       // sites per parity
    int s1;       // cb stride of x1 (= h)
    int s2;       // cb stride of x2 (= h N1)
    int s3;       // cb stride of x3 (= h N1 N2)
    int W;        // traversal chunk width in x2 (divides N2; N2 = plain cb order), see traversal_site
};

template <typename T> struct Cplx;
template <> struct Cplx<double> { typedef double2 type; };
template <> struct Cplx<float>  { typedef float2 type; };

// L2 eviction policies (createpolicy, PTX ISA): links are read exactly once per half-Dslash
// (evict_first), neighbour spinors are read by 8 output sites (evict_last).
__device__ __forceinline__ uint64_t l2_policy_evict_first()
{
    uint64_t p;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
    return p;
}
__device__ __forceinline__ uint64_t l2_policy_evict_last()
{
    uint64_t p;
    asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(p));
    return p;
}

// streaming load: read-only path, no L1 allocation, L2 policy operand
__device__ __forceinline__ double2 ld_stream(const double2 *p, uint64_t pol)
{
    double2 r;
    asm volatile("ld.global.nc.L1::no_allocate.L2::cache_hint.v2.f64 {%0,%1}, [%2], %3;"
                 : "=d"(r.x), "=d"(r.y) : "l"(p), "l"(pol));
    return r;
}
__device__ __forceinline__ float2 ld_stream(const float2 *p, uint64_t pol)
{
    float2 r;
    asm volatile("ld.global.nc.L1::no_allocate.L2::cache_hint.v2.f32 {%0,%1}, [%2], %3;"
                 : "=f"(r.x), "=f"(r.y) : "l"(p), "l"(pol));
    return r;
}
__device__ __forceinline__ float4 ld_stream(const float4 *p, uint64_t pol)
{
    float4 r;
    asm volatile("ld.global.nc.L1::no_allocate.L2::cache_hint.v4.f32 {%0,%1,%2,%3}, [%4], %5;"
                 : "=f"(r.x), "=f"(r.y), "=f"(r.z), "=f"(r.w) : "l"(p), "l"(pol));
    return r;
}
// reused load: read-only path, L1 allocation allowed, L2 policy operand
__device__ __forceinline__ double2 ld_keep(const double2 *p, uint64_t pol)
{
    double2 r;
    asm volatile("ld.global.nc.L2::cache_hint.v2.f64 {%0,%1}, [%2], %3;"
                 : "=d"(r.x), "=d"(r.y) : "l"(p), "l"(pol));
    return r;
}
__device__ __forceinline__ float2 ld_keep(const float2 *p, uint64_t pol)
{
    float2 r;
    asm volatile("ld.global.nc.L2::cache_hint.v2.f32 {%0,%1}, [%2], %3;"
                 : "=f"(r.x), "=f"(r.y) : "l"(p), "l"(pol));
    return r;
}
__device__ __forceinline__ float4 ld_keep(const float4 *p, uint64_t pol)
{
    float4 r;
    asm volatile("ld.global.nc.L2::cache_hint.v4.f32 {%0,%1,%2,%3}, [%4], %5;"
                 : "=f"(r.x), "=f"(r.y), "=f"(r.z), "=f"(r.w) : "l"(p), "l"(pol));
    return r;
}

__device__ __forceinline__ void prefetch_l2(const void *p) { asm volatile("prefetch.global.L2 [%0];" :: "l"(p)); }

// Asynchronous global -> shared copies (LDGSTS): the data never passes through registers, so a
// thread can keep many link loads in flight without holding registers for them.  16-byte copies
// bypass L1 (.cg); 8-byte copies exist only as .ca.  L2 policy operand as for ld_stream.
__device__ __forceinline__ void cp_async_stream(double2 *smem_dst, const double2 *src, uint64_t pol)
{
    const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.cg.shared.global.L2::cache_hint [%0], [%1], 16, %2;" :: "r"(d), "l"(src), "l"(pol) : "memory");
}
__device__ __forceinline__ void cp_async_stream(float2 *smem_dst, const float2 *src, uint64_t pol)
{
    const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.ca.shared.global.L2::cache_hint [%0], [%1], 8, %2;" :: "r"(d), "l"(src), "l"(pol) : "memory");
}
// one HALF of a complex number (lane `half` of a pair copies the real or the imaginary part): lets two lanes split an
// odd number of planes without a predicated copy (a predicated cp.async with an L2 policy operand is what ptxas 12.9
// turns into an instruction sm_100a rejects)
__device__ __forceinline__ void cp_async_stream_half(double2 *smem_dst, const double2 *src, int half, uint64_t pol)
{
    const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst) + 8u * (unsigned)half;
    const char *s = reinterpret_cast<const char *>(src) + 8 * half;
    asm volatile("cp.async.ca.shared.global.L2::cache_hint [%0], [%1], 8, %2;" :: "r"(d), "l"(s), "l"(pol) : "memory");
}
__device__ __forceinline__ void cp_async_stream_half(float2 *smem_dst, const float2 *src, int half, uint64_t pol)
{
    const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst) + 4u * (unsigned)half;
    const char *s = reinterpret_cast<const char *>(src) + 4 * half;
    asm volatile("cp.async.ca.shared.global.L2::cache_hint [%0], [%1], 4, %2;" :: "r"(d), "l"(s), "l"(pol) : "memory");
}
// the same copies without an L2 policy operand (used where the copy is predicated, see cp_async_stream_half)
__device__ __forceinline__ void cp_async_plain(double2 *smem_dst, const double2 *src)
{
    const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" :: "r"(d), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_plain(float2 *smem_dst, const float2 *src)
{
    const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" :: "r"(d), "l"(src) : "memory");
}
// ---- mbarrier + bulk asynchronous copies (cp.async.bulk: the TMA engine moves a contiguous run global -> shared and
// signals an mbarrier with the bytes it wrote; no thread holds a register or an LSU miss entry for the data in flight) ----
__device__ __forceinline__ unsigned smem_addr(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long *bar, unsigned count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" :: "r"(smem_addr(bar)), "r"(count) : "memory");
}
// after the inits, before any other thread or the async proxy touches the barriers
__device__ __forceinline__ void mbar_init_fence()
{
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}
__device__ __forceinline__ void mbar_arrive(unsigned long long *bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" :: "r"(smem_addr(bar)) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(unsigned long long *bar, unsigned bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" :: "r"(smem_addr(bar)), "r"(bytes) : "memory");
}
// wait until the phase of parity `parity` has completed; a wait that never completes (a byte-count bug) traps instead of hanging the GPU
__device__ __forceinline__ void mbar_wait(unsigned long long *bar, unsigned parity)
{
    const unsigned a = smem_addr(bar);
    unsigned ok = 0;
    for (unsigned spins = 0; !ok; ++spins) {
        asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                     : "=r"(ok) : "r"(a), "r"(parity) : "memory");
        if (spins > (1u << 26)) __trap();
    }
}
// `bytes` (a multiple of 16) from 16-byte aligned global memory to 16-byte aligned shared memory; completion is counted on `bar`
__device__ __forceinline__ void bulk_copy_g2s(void *smem_dst, const void *src, unsigned bytes, unsigned long long *bar, uint64_t pol)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;"
                 :: "r"(smem_addr(smem_dst)), "l"(src), "r"(bytes), "r"(smem_addr(bar)), "l"(pol) : "memory");
}

// one BOX of a 2-d tensor map (inner coordinate c0, outer c1) -> shared memory; the box shape is fixed by the map
__device__ __forceinline__ void tensor_copy_g2s(void *smem_dst, const void *tmap, int c0, int c1, unsigned long long *bar, uint64_t pol)
{
    asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1, {%2, %3}], [%4], %5;"
                 :: "r"(smem_addr(smem_dst)), "l"(tmap), "r"(c0), "r"(c1), "r"(smem_addr(bar)), "l"(pol) : "memory");
}

__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
// wait until at most `pending` of this thread's most recent groups are still in flight
// (the operand must be an immediate: the switch folds once the caller's loop is unrolled)
__device__ __forceinline__ void cp_async_wait(int pending)
{
    switch (pending) {
    case 0: asm volatile("cp.async.wait_group 0;" ::: "memory"); break;
    case 1: asm volatile("cp.async.wait_group 1;" ::: "memory"); break;
    case 2: asm volatile("cp.async.wait_group 2;" ::: "memory"); break;
    case 3: asm volatile("cp.async.wait_group 3;" ::: "memory"); break;
    case 4: asm volatile("cp.async.wait_group 4;" ::: "memory"); break;
    case 5: asm volatile("cp.async.wait_group 5;" ::: "memory"); break;
    case 6: asm volatile("cp.async.wait_group 6;" ::: "memory"); break;
    default: asm volatile("cp.async.wait_group 7;" ::: "memory"); break;
    }
}

// Traversal order of the Dslash threads.  Thread t of the grid handles site cb = t in the plain
// order.  With several vectors per link load the spinor working set between the two uses of a
// time-neighbour (two full time slices) outgrows the L2, and every spinor is fetched from DRAM
// more than once.  The chunked order walks x2 in chunks of W rows: (x0, x1) fastest, then x2
// inside the chunk, then x3, then the chunk -- the x3 reuse distance shrinks from 2 N2 to 2 W
// rows of h N1 sites, at the price of re-reading 2 of every W rows at the chunk edges.
// A pure permutation of which thread handles which site: results do not depend on it.
__device__ __forceinline__ int traversal_site(const Lattice &L, int t)
{
    if (L.W == L.N2) return t;
    const unsigned R = (unsigned)L.s2;                     // sites per x2-row
    const unsigned rowp = (unsigned)t / R, off = (unsigned)t - rowp * R;
    const unsigned per = (unsigned)(L.W * L.N3);           // rows per chunk
    const unsigned chunk = rowp / per, rem = rowp - chunk * per;
    const unsigned x3 = rem / (unsigned)L.W, x2lo = rem - x3 * (unsigned)L.W;
    const unsigned row = chunk * (unsigned)L.W + x2lo + (unsigned)L.N2 * x3;
    return (int)(row * R + off);
}

// Site geometry of one checkerboard index: coordinates, the 8
// neighbour checkerboard indices (all in the OTHER parity), Kogut-Susskind phases and the
// antiperiodic-time seam signs, all from integer arithmetic on (parity, cb).
struct SiteGeom {
    int nf[4], nb[4];   // cb of x+mu, x-mu
    float sf[4], sb[4]; // eta_mu(x) * seam sign of the forward hop ; MINUS eta_mu(x-mu) * seam sign of the backward hop
    int x3;             // time coordinate (temporal-gauge kernels: which time links are the identity)
};

__device__ __forceinline__ SiteGeom site_geometry(const Lattice &L, int parity, int cb)
{
    SiteGeom g;
    const unsigned ucb = (unsigned)cb;
    const int xh = (int)(ucb % (unsigned)L.h);
    unsigned r = ucb / (unsigned)L.h;
    const int x1 = (int)(r % (unsigned)L.N1);
    r /= (unsigned)L.N1;
    const int x2 = (int)(r % (unsigned)L.N2);
    const int x3 = (int)(r / (unsigned)L.N2);
    const int rp = (x1 + x2 + x3 + parity) & 1;      // x0 = 2 xh + rp, so x0 & 1 == rp

    // mu = 0: the neighbour sits in the same x0-row of the other parity
    g.nf[0] = rp ? ((xh + 1 == L.h) ? cb - (L.h - 1) : cb + 1) : cb;
    g.nb[0] = rp ? cb : ((xh == 0) ? cb + (L.h - 1) : cb - 1);
    g.nf[1] = (x1 + 1 == L.N1) ? cb - (L.N1 - 1) * L.s1 : cb + L.s1;
    g.nb[1] = (x1 == 0) ? cb + (L.N1 - 1) * L.s1 : cb - L.s1;
    g.nf[2] = (x2 + 1 == L.N2) ? cb - (L.N2 - 1) * L.s2 : cb + L.s2;
    g.nb[2] = (x2 == 0) ? cb + (L.N2 - 1) * L.s2 : cb - L.s2;
    g.nf[3] = (x3 + 1 == L.N3) ? cb - (L.N3 - 1) * L.s3 : cb + L.s3;
    g.nb[3] = (x3 == 0) ? cb + (L.N3 - 1) * L.s3 : cb - L.s3;

    // eta_0 = 1, eta_1 = (-1)^{x0}, eta_2 = (-1)^{x0+x1}, eta_3 = (-1)^{x0+x1+x2};
    // eta_mu does not depend on x_mu, so eta_mu(x-mu) = eta_mu(x) (extents are even).
    const float e1 = rp ? -1.f : 1.f;
    const float e2 = ((rp + x1) & 1) ? -1.f : 1.f;
    const float e3 = ((rp + x1 + x2) & 1) ? -1.f : 1.f;
    g.sf[0] = 1.f;  g.sb[0] = -1.f;
    g.sf[1] = e1;   g.sb[1] = -e1;
    g.sf[2] = e2;   g.sb[2] = -e2;
    g.sf[3] = (x3 + 1 == L.N3) ? -e3 : e3;           // forward hop across the time seam
    g.sb[3] = (x3 == 0) ? e3 : -e3;                  // backward hop across the time seam
    g.x3 = x3;
    return g;
}

// Host: tensor map of `planes` rows of `row_elems` elements (8-byte doubles or 4-byte floats), rows `row_stride_bytes` apart,
// with a box of box_rows x box_elems.  cuTensorMapEncodeTiled is taken from the driver through the runtime (no libcuda link).
static inline cudaError_t encode_plane_map(CUtensorMap *map, bool f64, const void *base, unsigned long long row_elems, unsigned long long planes,
                                           unsigned long long row_stride_bytes, unsigned box_elems, unsigned box_rows)
{
    typedef CUresult (*encode_fn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *, const cuuint32_t *,
                                  const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
    static encode_fn fn = nullptr;
    if (!fn) {
        void *p = nullptr;
        cudaDriverEntryPointQueryResult qr;
        const cudaError_t e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qr);
        if (e != cudaSuccess) return e;
        if (qr != cudaDriverEntryPointSuccess || !p) return cudaErrorNotSupported;
        fn = (encode_fn)p;
    }
    const cuuint64_t gdim[2] = {row_elems, planes};
    const cuuint64_t gstride[1] = {row_stride_bytes};
    const cuuint32_t box[2] = {box_elems, box_rows};
    const cuuint32_t estr[2] = {1, 1};
    const CUresult r = fn(map, f64 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT64 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, const_cast<void *>(base), gdim, gstride, box, estr,
                          CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS ? cudaSuccess : cudaErrorInvalidValue;
}

} // namespace qcd
