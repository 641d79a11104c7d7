// topk_kernel.cuh -- SURVEY.md section 8(f) NEXT-3: top-k MoE dispatch / combine (the router
// sends each token to k experts; Table 3 L493-516 runs k = 1 and k = 4).  Joins the two halves of this build:
//   dispatch  = the AllToAllv of the (virtual) expert-sorted send buffer, with the k-fold token duplication
//               done on the way: a token row is READ ONCE and written to its k destinations, the sorted
//               k*T-row buffer is never materialised (saves its write and re-read);
//   combine   = the inverse AllToAllv FUSED with the fixed-order fp32 sum of reduce_kernel: the k expert
//               outputs of a token are gathered from the packed receive buffers, accumulated in router order
//               j = 0..k-1, rounded once, and written to the token's row.
// Metadata (device-resident, read at execution): pos[s][t][j] = row of copy j of token t in rank s's virtual
// sorted buffer; C[s][d] rows per destination.  counts_kernel has already turned C into soff / roff (in rows).
//
// One warp per token, tokens taken in order by the whole grid (moving window of HBM, as in segment_copy_kernel);
// lanes 0..k-1 resolve the k copies in parallel (binary search of p in row s of soff), then all lanes stream
// the row with 256-bit (or 128-bit) accesses, TOPK_UNROLL vectors per lane in flight per copy.
#pragma once
#include "common.cuh"
#include "reduce_kernel.cuh"

namespace xdev {

constexpr int TOPK_THREADS = 128;               // 4 warps per CTA, up to 16 CTAs per SM: measured 1.6 % faster on the dispatch than 256 x 8 (512 x 4: 6 % slower)
constexpr int TOPK_UNROLL = 2;             // dispatch: vectors per lane in flight per copy (4 measured 8 % slower)
constexpr int TOPK_COMBINE_UNROLL = 4;     // combine: 4 measured 1 % faster than 2

struct TopkArgs {
    const void* const* tokens;    // dispatch: R token matrices (T x width)      combine: unused
    void* const* packed;          // dispatch: recv[d] (out)                     combine: Y[d] (in)
    void* const* out;             // combine: Z_s (T x width)
    const int* pos;               // R*T*k
    const long long* C;           // user's count matrix in rows (for the range check)
    const long long* soff;        // ws, rows
    const long long* roff;        // ws, rows
    WorkCtl* ctl;
    int R, T, k;
    long long rowBytes;
};

// lane j < k: address of row (copy j of token t of rank s) inside packed[d]; 0 if the position is invalid
__device__ __forceinline__ unsigned long long topk_resolve(const TopkArgs& a, int s, int t, int j, bool& bad) {
    const long long p = a.pos[((size_t)s * a.T + t) * a.k + j];
    const long long* so = a.soff + (size_t)s * a.R;
    int lo = 0, hi = a.R;                                   // largest d with so[d] <= p
    if (p < 0) { bad = true; return 0ull; }
    while (hi - lo > 1) {
        const int mid = (lo + hi) >> 1;
        if (so[mid] <= p) lo = mid; else hi = mid;
    }
    const int d = lo;
    long long c = a.C[(size_t)s * a.R + d];
    c = c > 0 ? c : 0;
    if (p >= so[d] + c) { bad = true; return 0ull; }
    const long long row = a.roff[(size_t)d * a.R + s] + (p - so[d]);
    return (unsigned long long)a.packed[d] + (unsigned long long)(row * a.rowBytes);
}

// One token row through the LSU: read once (256-bit loads, TOPK_UNROLL vectors per lane in flight), written to its k
// destinations; any alignment (byte copy when a pointer or the row size is not a multiple of 32).  `mine`: lane j < k
// holds the address of copy j (0: invalid position, skipped).
__device__ __forceinline__ void topk_dispatch_row_lsu(const TopkArgs& a, const unsigned char* src, unsigned long long mine, int lane) {
    unsigned long long al = (unsigned long long)src | (unsigned long long)a.rowBytes | mine;
    al = __reduce_or_sync(0xffffffffu, (unsigned int)(al & 31ull));
    if ((al & 31ull) == 0) {
        const long long nv = a.rowBytes >> 5;
        for (long long c0 = 0; c0 < nv; c0 += 32 * TOPK_UNROLL) {      // warp-uniform trip count (shuffles inside)
            const long long c = c0 + lane;
            u32x8 x[TOPK_UNROLL];
#pragma unroll
            for (int u = 0; u < TOPK_UNROLL; ++u)
                if (c + 32 * u < nv) x[u] = ld_stream256(src + (c + 32 * u) * 32);
            for (int j = 0; j < a.k; ++j) {
                const unsigned long long dlo = __shfl_sync(0xffffffffu, (unsigned int)mine, j);
                const unsigned long long dhi = __shfl_sync(0xffffffffu, (unsigned int)(mine >> 32), j);
                unsigned char* dst = reinterpret_cast<unsigned char*>((dhi << 32) | dlo);
                if (dst) {
#pragma unroll
                    for (int u = 0; u < TOPK_UNROLL; ++u)
                        if (c + 32 * u < nv) st_stream256(dst + (c + 32 * u) * 32, x[u]);
                }
            }
        }
    } else {                                            // any alignment: byte copy, same mapping
        for (int j = 0; j < a.k; ++j) {
            const unsigned long long dlo = __shfl_sync(0xffffffffu, (unsigned int)mine, j);
            const unsigned long long dhi = __shfl_sync(0xffffffffu, (unsigned int)(mine >> 32), j);
            unsigned char* dst = reinterpret_cast<unsigned char*>((dhi << 32) | dlo);
            if (dst)
                for (long long b = lane; b < a.rowBytes; b += 32) dst[b] = src[b];
        }
    }
}

__global__ void __launch_bounds__(TOPK_THREADS) topk_dispatch_kernel(const TopkArgs a) {
    const int lane = lane_id();
    const long long nTok = (long long)a.R * a.T;
    const long long wStride = (long long)gridDim.x * (TOPK_THREADS / 32);
    griddep_wait();                                         // soff / roff come from counts_kernel
    for (long long tok = (long long)blockIdx.x * (TOPK_THREADS / 32) + (threadIdx.x >> 5); tok < nTok; tok += wStride) {
        const int s = (int)(tok / a.T), t = (int)(tok - (long long)s * a.T);
        bool bad = false;
        const unsigned long long mine = lane < a.k ? topk_resolve(a, s, t, lane, bad) : 0ull;
        if (__any_sync(0xffffffffu, bad) && lane == 0) atomicOr(&a.ctl->status, 2u);
        const unsigned char* src = reinterpret_cast<const unsigned char*>(a.tokens[s]) + (size_t)t * a.rowBytes;
        topk_dispatch_row_lsu(a, src, mine, lane);
    }
}


template <int DT>
__global__ void __launch_bounds__(TOPK_THREADS) topk_combine_kernel(const TopkArgs a) {
    constexpr int ES = DT == RED_F32 ? 4 : 2;
    const int lane = lane_id();
    const long long nTok = (long long)a.R * a.T;
    const long long wStride = (long long)gridDim.x * (TOPK_THREADS / 32);
    griddep_wait();
    for (long long tok = (long long)blockIdx.x * (TOPK_THREADS / 32) + (threadIdx.x >> 5); tok < nTok; tok += wStride) {
        const int s = (int)(tok / a.T), t = (int)(tok - (long long)s * a.T);
        bool bad = false;
        const unsigned long long mine = lane < a.k ? topk_resolve(a, s, t, lane, bad) : 0ull;
        if (__any_sync(0xffffffffu, bad) && lane == 0) atomicOr(&a.ctl->status, 2u);
        unsigned char* dst = reinterpret_cast<unsigned char*>(a.out[s]) + (size_t)t * a.rowBytes;
        unsigned long long al = (unsigned long long)dst | (unsigned long long)a.rowBytes | mine;
        al = __reduce_or_sync(0xffffffffu, (unsigned int)(al & 31ull));
        if ((al & 31ull) == 0) {
            const long long nv = a.rowBytes >> 5;
            for (long long c0 = 0; c0 < nv; c0 += 32 * TOPK_COMBINE_UNROLL) {      // warp-uniform trip count (shuffles inside)
                const long long c = c0 + lane;
                Acc<DT> lo[TOPK_COMBINE_UNROLL], hi[TOPK_COMBINE_UNROLL];
                bool have = false;
                for (int j = 0; j < a.k; ++j) {
                    const unsigned long long slo = __shfl_sync(0xffffffffu, (unsigned int)mine, j);
                    const unsigned long long shi = __shfl_sync(0xffffffffu, (unsigned int)(mine >> 32), j);
                    const unsigned char* src = reinterpret_cast<const unsigned char*>((shi << 32) | slo);
                    if (!src) continue;
                    u32x8 x[TOPK_COMBINE_UNROLL];
#pragma unroll
                    for (int u = 0; u < TOPK_COMBINE_UNROLL; ++u)
                        if (c + 32 * u < nv) x[u] = ld_stream256(src + (c + 32 * u) * 32);
#pragma unroll
                    for (int u = 0; u < TOPK_COMBINE_UNROLL; ++u)
                        if (c + 32 * u < nv) {
                            if (!have) { lo[u].set(x[u].lo); hi[u].set(x[u].hi); }
                            else { lo[u].add(x[u].lo); hi[u].add(x[u].hi); }
                        }
                    have = true;
                }
#pragma unroll
                for (int u = 0; u < TOPK_COMBINE_UNROLL; ++u)
                    if (c + 32 * u < nv) {
                        u32x8 o;
                        if (have) { o.lo = lo[u].pack(); o.hi = hi[u].pack(); }
                        else { o.lo = make_uint4(0, 0, 0, 0); o.hi = make_uint4(0, 0, 0, 0); }
                        st_stream256(dst + (c + 32 * u) * 32, o);
                    }
            }
        } else {                                            // scalar path, same arithmetic
            const long long ne = a.rowBytes / ES;
            for (long long e0 = 0; e0 < ne; e0 += 32) {
                const long long e = e0 + lane;
                float acc = 0.0f;
                bool have = false;
                for (int j = 0; j < a.k; ++j) {
                    const unsigned long long slo = __shfl_sync(0xffffffffu, (unsigned int)mine, j);
                    const unsigned long long shi = __shfl_sync(0xffffffffu, (unsigned int)(mine >> 32), j);
                    const void* src = reinterpret_cast<const void*>((shi << 32) | slo);
                    if (!src) continue;
                    const float y = e < ne ? load_elem<DT>(src, (unsigned long long)e) : 0.0f;
                    acc = have ? __fadd_rn(acc, y) : y;
                    have = true;
                }
                if (e < ne) store_elem<DT>(dst, (unsigned long long)e, acc);
            }
        }
    }
}

}  // namespace xdev
