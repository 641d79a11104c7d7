// common.cuh -- shared device helpers and workspace types of libncclx_b200 (sm_100a only).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#if defined(__CUDA_ARCH__) && (__CUDA_ARCH__ < 1000)
#error "libncclx_b200 is written for sm_100a (B200) only"
#endif

namespace xdev {

// One (source s, destination d) segment of the AllToAllv, in destination-major order
// q = d*R + s -- the order in which the packed receive buffers are laid out,
// so consecutive work items write consecutive HBM addresses.
struct __align__(32) SegDesc {
    unsigned long long src;   // absolute address of send[s][soff[s][d]]
    unsigned long long dst;   // absolute address of recv[d][roff[d][s]]
    long long bytes;          // C[s][d] * elem_size
    int pfx[2];               // inclusive tile-count prefix WITHIN column d: [0] bulk list, [1] vector list
};
static_assert(sizeof(SegDesc) == 32, "SegDesc must be 32 bytes");

enum { LIST_BULK = 0, LIST_VEC = 1 };

// Device-resident control block.  The claim counters are zero between kernels: the copy kernel's last
// CTA resets them on its way out (workctl_checkout); ncclx_init zeroes them once.
struct WorkCtl {
    unsigned int next[2];     // dynamic tile-claim counters, one per work list
    unsigned int status;      // sticky: bit 0 = negative count seen
    unsigned int done;        // CTAs of the running copy kernel that have drained their engines
    unsigned int pad_probe;   // sink of the streaming micro-probe (never read)
    unsigned int barArrive;   // counts_kernel's grid barrier: CTAs that have published their block sums ...
    unsigned int barDepart;   // ... and CTAs that have passed it (the last one zeroes both)
};

struct Workspace {
    long long* soff;          // R*R, soff[s*R+d]
    long long* roff;          // R*R, roff[d*R+s]
    SegDesc* desc;            // R*R, desc[d*R+s]
    int* colTiles[2];         // R each: tiles of list L in column d
    int* colKiB;              // R: KiB of column d's bulk-list segments (-> average tile size -> bulk engines per CTA)
    int* coarse[2];           // R*ceil(colLen/32) each: tiles of list L in column d before its descriptor 32*j
    WorkCtl* ctl;
    long long* blockSum;      // COUNTS_MAX_CTAS * R: blockSum[j*R+s] = sum of row s of C over CTA j's columns (counts_kernel)
};
constexpr int COUNTS_MAX_CTAS = 128;

__device__ __forceinline__ int lane_id() { return threadIdx.x & 31; }

// Classification shared by the counts kernel (which builds the per-list tile prefixes) and the copy
// kernel (which re-derives a segment's tile count from its descriptor): number of tiles the segment
// contributes to work list L.  A segment is on exactly one list: BULK iff source and destination are
// 16-byte aligned and it has at least bulkMinBytes bytes.
struct ClassParams {
    long long bulkMinBytes;
    int tileShift[2];
};
__device__ __forceinline__ int seg_tiles(int L, unsigned long long src, unsigned long long dst, long long bytes,
                                         const ClassParams& cp) {
    if (bytes <= 0) return 0;
    const bool bulk = (((src | dst) & 15ull) == 0) && bytes >= cp.bulkMinBytes;
    if (bulk != (L == 0)) return 0;
    return (int)((bytes + (1ll << cp.tileShift[L]) - 1) >> cp.tileShift[L]);
}

__device__ __forceinline__ long long warp_incl_scan(long long v) {
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        long long n = __shfl_up_sync(0xffffffffu, v, o);
        if (lane_id() >= o) v += n;
    }
    return v;
}
__device__ __forceinline__ int warp_incl_scan(int v) {
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        int n = __shfl_up_sync(0xffffffffu, v, o);
        if (lane_id() >= o) v += n;
    }
    return v;
}
__device__ __forceinline__ long long warp_sum(long long v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// ---- programmatic dependent launch (PDL) ------------------------------------------------------
// The copy kernel is launched with programmatic stream serialization: its CTAs may become resident and
// run their prologue while the counts kernel drains; griddep_wait() blocks until the counts grid has
// completed and its writes are visible.  Both are no-ops when the launch carries no such attribute.
__device__ __forceinline__ void griddep_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
__device__ __forceinline__ void griddep_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

// L2 prefetch: a hint with no correctness implication (L2 is the GPU's point of coherence, so a line prefetched before
// griddepcontrol.wait cannot go stale) -- used to pull cold metadata into L2 in ONE DRAM round trip.
__device__ __forceinline__ void prefetch_l2(const void* p) { asm volatile("prefetch.global.L2 [%0];" :: "l"(p)); }

// ---- L2 eviction priorities -------------------------------------------------------------------
// A call's METADATA (count matrix, pointer tables, split lengths, index lists: a few hundred KB) is read again by the
// next call, but the payload streamed in between is many times the 126 MB L2, so by then every metadata line has gone
// back to DRAM and the metadata kernel pays cold-DRAM round trips (measured with per-CTA %globaltimer stamps: 1-2.5 us
// each, worse from the die the line does not live on).  Metadata loads therefore carry an evict_last policy, payload
// bulk copies an evict_first one: the stream passes through L2 without displacing what will be read again.
__device__ __forceinline__ unsigned long long l2_policy_keep() {
    unsigned long long p;
    asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(p));
    return p;
}
__device__ __forceinline__ unsigned long long l2_policy_stream() {
    unsigned long long p;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
    return p;
}
__device__ __forceinline__ long long ld_keep(const long long* a, unsigned long long pol) {
    long long v;
    asm volatile("ld.global.L2::cache_hint.b64 %0, [%1], %2;" : "=l"(v) : "l"(a), "l"(pol) : "memory");
    return v;
}
__device__ __forceinline__ unsigned long long ld_keep_ptr(const void* const* a, unsigned long long pol) {
    unsigned long long v;
    asm volatile("ld.global.L2::cache_hint.b64 %0, [%1], %2;" : "=l"(v) : "l"(a), "l"(pol) : "memory");
    return v;
}

// ---- streaming global accesses --------------------------------------------------------------
// (No ld.global.nc anywhere: with programmatic dependent launch a kernel's CTAs are resident while the kernel before
// it in the stream still writes the very bytes they will read after griddepcontrol.wait, and the non-coherent path
// formally needs data that is read-only for the kernel's whole lifetime.)
__device__ __forceinline__ uint4 ld_stream(const uint4* p) {      // coherent; may alias an output (in-place)
    uint4 r;
    asm volatile("ld.global.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p) : "memory");
    return r;
}
__device__ __forceinline__ void st_stream(uint4* p, const uint4& v) {
    asm volatile("st.global.L1::no_allocate.v4.u32 [%0], {%1,%2,%3,%4};"
                 :: "l"(p), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
}

// 256-bit global accesses (sm_100: LDG.E.256 / STG.E.256): half the load instructions of the 128-bit
// form and 32 B per lane per request; measured +10 % on the 16-stream reduction.
struct u32x8 { uint4 lo, hi; };
__device__ __forceinline__ u32x8 ld_stream256(const void* p) {     // may alias an output (in-place)
    u32x8 r;
    asm volatile("ld.global.L1::no_allocate.v8.u32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                 : "=r"(r.lo.x), "=r"(r.lo.y), "=r"(r.lo.z), "=r"(r.lo.w), "=r"(r.hi.x), "=r"(r.hi.y), "=r"(r.hi.z), "=r"(r.hi.w)
                 : "l"(p) : "memory");
    return r;
}
__device__ __forceinline__ void st_stream256(void* p, const u32x8& v) {
    asm volatile("st.global.L1::no_allocate.v8.u32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};"
                 :: "l"(p), "r"(v.lo.x), "r"(v.lo.y), "r"(v.lo.z), "r"(v.lo.w), "r"(v.hi.x), "r"(v.hi.y), "r"(v.hi.z), "r"(v.hi.w)
                 : "memory");
}

// ---- mbarrier + cp.async.bulk (descriptor-less 1-D TMA) --------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" :: "r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void fence_mbar_init() {
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
// orders this thread's generic-proxy accesses to shared memory before later async-proxy (TMA) accesses
__device__ __forceinline__ void fence_proxy_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" :: "r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" :: "r"(bar) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint32_t bar, uint32_t parity) {
    uint32_t ok;
    asm volatile("{\n\t.reg .pred p;\n\t"
                 "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
                 "selp.u32 %0, 1, 0, p;\n\t}"
                 : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
    return ok != 0;
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    while (!mbar_try_wait(bar, parity)) { }
}
// global -> shared, completion counted in bytes on `bar`
__device__ __forceinline__ void bulk_g2s(uint32_t dst_smem, const void* src, uint32_t bytes, uint32_t bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 :: "r"(dst_smem), "l"(src), "r"(bytes), "r"(bar) : "memory");
}
// the same two with an L2 eviction policy (payload: l2_policy_stream())
__device__ __forceinline__ void bulk_g2s(uint32_t dst_smem, const void* src, uint32_t bytes, uint32_t bar, unsigned long long pol) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;"
                 :: "r"(dst_smem), "l"(src), "r"(bytes), "r"(bar), "l"(pol) : "memory");
}
__device__ __forceinline__ void bulk_s2g(void* dst, uint32_t src_smem, uint32_t bytes, unsigned long long pol) {
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group.L2::cache_hint [%0], [%1], %2, %3;"
                 :: "l"(dst), "r"(src_smem), "r"(bytes), "l"(pol) : "memory");
}
// shared -> global, tracked by the issuing thread's bulk async-group
__device__ __forceinline__ void bulk_s2g(void* dst, uint32_t src_smem, uint32_t bytes) {
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;"
                 :: "l"(dst), "r"(src_smem), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void bulk_wait_read() {
    asm volatile("cp.async.bulk.wait_group.read %0;" :: "n"(N) : "memory");
}
template <int N> __device__ __forceinline__ void bulk_wait_all() {
    asm volatile("cp.async.bulk.wait_group %0;" :: "n"(N) : "memory");
}

}  // namespace xdev
