// dynamic_kernel.cuh -- work-list builders for the paper's full AllToAllvDynamic metadata interface
// (section 6.1.2): sendSplitLengths + sendIndices +
// sendIndicesBlockLens on the send side, per-source recvbuffs with the sender's padding preserved and
// recvAllSplitLengths on the receive side.  It reuses steps a3/a4 (descriptor table + segment_copy_kernel)
// with one more indirection: a segment is one (source s, destination d, list position j) triple, i.e. one
// whole split, copied to the SAME offset in recvbuffs[d][s] that it has in send[s] (L439 "paddings are
// reserved", Fig. 17).
//
//   dyn_prep_kernel   grid R: CTA s scans rank s's split lengths into offsets O_s (exclusive), scans its
//                     block lengths into list offsets ioff[s][.], and broadcasts L_s to every receiver's
//                     recvAllSplitLengths[d][s][.] (L439: every rank receives all split lengths).
//   dyn_desc_kernel   grid R: CTA d walks column d's slots (s, j), j < maxBlockLen, in s-major order (one warp
//                     per 32-slot block) and writes descriptors, per-column tile prefixes and the coarse index
//                     exactly like counts_kernel's phase 2.
#pragma once
#include "common.cuh"

namespace ncclx {

constexpr int DYN_PREP_THREADS = 256;

struct DynArgs {
    const void* const* send;          // R
    void* const* recvbuffs;           // R*R, [d*R+s]
    const long long* L;               // R*n split lengths
    const long long* indices;         // R*maxIndices
    const long long* blockLens;       // R*R
    long long* recvAll;               // R*R*n out
    long long* O;                     // ws: R*n exclusive offsets
    long long* ioff;                  // ws: R*R exclusive list offsets
    Workspace ws;
    int R, n, maxIndices, maxBlockLen, elemSize;
    ClassParams cls;
};

__global__ void __launch_bounds__(DYN_PREP_THREADS) dyn_prep_kernel(const DynArgs a) {
    const int s = blockIdx.x, lane = lane_id(), warp = threadIdx.x >> 5;
    const int R = a.R, n = a.n;
    griddep_launch_dependents();
    const long long* Ls = a.L + (size_t)s * n;
    constexpr int U = 4;                                   // loads issued per round trip
    if (warp == 0) {                                       // exclusive scan of the split lengths
        long long run = 0;
        bool neg = false;
        for (int i0 = 0; i0 < n; i0 += 32 * U) {
            long long v[U];
#pragma unroll
            for (int u = 0; u < U; ++u) { const int i = i0 + u * 32 + lane; v[u] = i < n ? Ls[i] : 0; }
#pragma unroll
            for (int u = 0; u < U; ++u) {
                const int i = i0 + u * 32 + lane;
                if (v[u] < 0) { neg = true; v[u] = 0; }
                const long long incl = warp_incl_scan(v[u]);
                if (i < n) a.O[(size_t)s * n + i] = run + incl - v[u];
                run += __shfl_sync(0xffffffffu, incl, 31);
            }
        }
        if (__any_sync(0xffffffffu, neg) && lane == 0) atomicOr(&a.ws.ctl->status, 1u);
    } else if (warp == 1) {                                // exclusive scan of the block lengths
        long long run = 0;
        bool bad = false;
        for (int d0 = 0; d0 < R; d0 += 32 * U) {
            long long v[U];
#pragma unroll
            for (int u = 0; u < U; ++u) { const int dd = d0 + u * 32 + lane; v[u] = dd < R ? a.blockLens[(size_t)s * R + dd] : 0; }
#pragma unroll
            for (int u = 0; u < U; ++u) {
                const int dd = d0 + u * 32 + lane;
                if (v[u] < 0) { bad = true; v[u] = 0; }
                if (v[u] > a.maxBlockLen) { bad = true; v[u] = a.maxBlockLen; }
                const long long incl = warp_incl_scan(v[u]);
                if (dd < R) a.ioff[(size_t)s * R + dd] = run + incl - v[u];
                run += __shfl_sync(0xffffffffu, incl, 31);
            }
        }
        if (__any_sync(0xffffffffu, bad) && lane == 0) atomicOr(&a.ws.ctl->status, 4u);
    }
    // every receiver gets all of rank s's split lengths: a thread keeps its values in registers and writes
    // them to the R receivers back to back (coalesced across the CTA, no index arithmetic per store)
    for (int i = threadIdx.x; i < n; i += DYN_PREP_THREADS) {
        long long v = Ls[i];
        v = v > 0 ? v : 0;
        long long* out = a.recvAll + (size_t)s * n + i;
        for (int d = 0; d < R; ++d) out[(size_t)d * R * n] = v;
    }
}

// CTA per destination column d, one warp per 32-slot block of the column (rounds of DYN_DESC_WARPS blocks):
// the blocks' dependent load chains (block length / list offset -> index -> split length / offset) run
// concurrently, three L2 round trips per round instead of five per block in sequence; the tile prefixes of
// the blocks are then chained through shared memory.
constexpr int DYN_DESC_WARPS = 8;

__global__ void __launch_bounds__(DYN_DESC_WARPS * 32) dyn_desc_kernel(const DynArgs a) {
    __shared__ int sTot[2][DYN_DESC_WARPS];
    __shared__ unsigned int sStatus;
    const int d = blockIdx.x, lane = lane_id(), warp = threadIdx.x >> 5;
    const int R = a.R, n = a.n, J = a.maxBlockLen;
    const int colLen = R * J;
    const int nb = (colLen + 31) >> 5;
    griddep_launch_dependents();
    if (threadIdx.x == 0) sStatus = 0u;
    griddep_wait();                                        // O / ioff come from dyn_prep_kernel
    int base[2] = {0, 0};                                  // tiles of the column before this round (CTA-uniform)
    unsigned int st = 0;
    for (int b0 = 0; b0 < nb; b0 += DYN_DESC_WARPS) {
        const int b = b0 + warp;
        const int k = b * 32 + lane;
        unsigned long long src = 0, dst = 0;
        long long bytes = 0;
        if (b < nb && k < colLen) {
            const int s = k / J, j = k - s * J;
            long long bl = a.blockLens[(size_t)s * R + d];                     // round trip 1: four independent loads
            const long long pos = a.ioff[(size_t)s * R + d] + j;
            const unsigned long long sp = (unsigned long long)a.send[s];
            const unsigned long long rp = (unsigned long long)a.recvbuffs[(size_t)d * R + s];
            bl = bl < 0 ? 0 : (bl > J ? J : bl);
            if (j < bl) {
                if (pos >= a.maxIndices) st |= 4u;
                else {
                    const long long idx = a.indices[(size_t)s * a.maxIndices + pos];   // round trip 2
                    if (idx < 0 || idx >= n) st |= 2u;
                    else {
                        const long long len = a.L[(size_t)s * n + idx];                 // round trip 3: two independent loads
                        const long long off = a.O[(size_t)s * n + idx];
                        bytes = (len > 0 ? len : 0) * a.elemSize;
                        src = sp + (unsigned long long)(off * a.elemSize);
                        dst = rp + (unsigned long long)(off * a.elemSize);
                    }
                }
            }
        }
        const int tb = seg_tiles(LIST_BULK, src, dst, bytes, a.cls);
        const int tv = seg_tiles(LIST_VEC, src, dst, bytes, a.cls);
        const long long it = warp_incl_scan(((long long)tb << 32) | (long long)(unsigned int)tv);
        const long long last = __shfl_sync(0xffffffffu, it, 31);
        if (lane == 0) { sTot[0][warp] = (int)(last >> 32); sTot[1][warp] = (int)(unsigned int)last; }
        __syncthreads();
        int pre[2] = {base[0], base[1]};                   // tiles before this warp's block
        int all[2] = {0, 0};
#pragma unroll
        for (int w = 0; w < DYN_DESC_WARPS; ++w) {
            const int t0 = sTot[0][w], t1 = sTot[1][w];
            if (w < warp) { pre[0] += t0; pre[1] += t1; }
            all[0] += t0; all[1] += t1;
        }
        if (b < nb) {
            if (lane < 2) a.ws.coarse[lane][(size_t)d * nb + b] = lane ? pre[1] : pre[0];
            if (k < colLen) {
                uint4* out = reinterpret_cast<uint4*>(a.ws.desc + (size_t)d * colLen + k);
                out[0] = make_uint4((unsigned int)src, (unsigned int)(src >> 32), (unsigned int)dst, (unsigned int)(dst >> 32));
                out[1] = make_uint4((unsigned int)bytes, (unsigned int)((unsigned long long)bytes >> 32),
                                    (unsigned int)(pre[0] + (int)(it >> 32)), (unsigned int)(pre[1] + (int)(unsigned int)it));
            }
        }
        base[0] += all[0]; base[1] += all[1];
        __syncthreads();                                   // sTot is rewritten in the next round
    }
    st = __reduce_or_sync(0xffffffffu, st);
    if (lane == 0 && st) atomicOr(&sStatus, st);
    __syncthreads();
    if (threadIdx.x == 0) {
        a.ws.colTiles[LIST_BULK][d] = base[0];
        a.ws.colTiles[LIST_VEC][d] = base[1];
        if (sStatus) atomicOr(&a.ws.ctl->status, sStatus);
    }
}

}  // namespace ncclx
