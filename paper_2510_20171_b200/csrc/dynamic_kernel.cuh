// dynamic_kernel.cuh -- work-list builder for the paper's full AllToAllvDynamic metadata interface
// (section 6.1.2): sendSplitLengths + sendIndices +
// sendIndicesBlockLens on the send side, per-source recvbuffs with the sender's padding preserved and
// recvAllSplitLengths on the receive side.  It reuses steps a3/a4 (descriptor table + segment_copy_kernel)
// with one more indirection: a segment is one (source s, destination d, list position j) triple, i.e. one
// whole split, copied to the SAME offset in recvbuffs[d][s] that it has in send[s] (L439 "paddings are
// reserved", Fig. 17).
//
// ONE metadata kernel (round 1 had two, 12 us in front of a 70 us copy):
//   dyn_build_kernel  grid R x 512 threads: CTA d builds column d of the table, slots k = s*J + j, j < J =
//                     maxBlockLen, in s-major order.
//     phase A  warp per source s (32 sources in flight per CTA): the warp re-derives what it needs of rank s's
//              metadata instead of reading it from a preceding kernel -- list offset ioff[s][d] = sum of row s of
//              the block lengths before d; then, for its <= J list entries at once (lane j <-> entry j), the split
//              index, and the split's offset O_s[idx] and length from ONE warp scan per 32 split lengths with a
//              per-lane shuffle pick.  All of a source's loads except the index load are independent (two L2
//              round trips per source).  Results go to a slot array in shared memory (in the table itself when the
//              column has more than DYN_SMEM_SLOTS slots).
//     phase B  all threads, slots in order: tiles per slot, block-wide scan -> per-list inclusive tile prefixes,
//              descriptors, the coarse index (prefix before every 32nd slot) and the column totals, exactly like
//              counts_kernel's phase 2.
//   recvAllSplitLengths (L439: every rank receives all split lengths; R copies of the R x nsplits matrix) is NOT
//   written here: the descriptor builder does not need it, so it rides along with the payload as the copy kernel's
//   side job (copy_kernel.cuh, SideJob) instead of sitting on the critical path.
#pragma once
#include "common.cuh"

namespace xdev {

constexpr int DYN_THREADS = 512;
constexpr int DYN_WARPS = DYN_THREADS / 32;
constexpr int DYN_SMEM_SLOTS = 4096;      // columns up to this many slots are staged in shared memory (32 B per slot)
constexpr int DYN_SU = 4;                 // sources a warp works on at once (their dependent loads overlap)
constexpr int DYN_PL = 5;                 // split lengths per lane and scan step
constexpr int DYN_CHUNK = 32 * DYN_PL;    // split lengths scanned per step: 160 covers 128 experts + redundant ones in ONE step

struct DynArgs {
    const void* const* send;          // R
    void* const* recvbuffs;           // R*R, [d*R+s]
    const long long* L;               // R*n split lengths
    const long long* indices;         // R*maxIndices
    const long long* blockLens;       // R*R
    Workspace ws;                     // desc / coarse / colTiles / ctl of the plan slot
    int R, n, maxIndices, maxBlockLen, elemSize;
    ClassParams cls;
};


struct __align__(32) DynSlot {        // same 32-byte stride as SegDesc, so the table itself can serve as the slot array
    unsigned long long src, dst;
    long long bytes;
    long long pad;
};

__host__ __device__ inline size_t dyn_smem_bytes(int colLen) {
    return colLen <= DYN_SMEM_SLOTS ? (size_t)colLen * sizeof(DynSlot) : 32;
}

// dynamic smem: DynSlot[colLen] if colLen <= DYN_SMEM_SLOTS
__global__ void __launch_bounds__(DYN_THREADS, 1) dyn_build_kernel(const DynArgs a) {
    extern __shared__ __align__(32) unsigned char dyn_smem[];
    __shared__ long long sWarpTot[DYN_WARPS];
    __shared__ unsigned int sStatus;
    const int d = blockIdx.x, lane = lane_id(), warp = threadIdx.x >> 5;
    const int R = a.R, n = a.n, J = a.maxBlockLen;
    const int colLen = R * J;
    const int nb = (colLen + 31) >> 5;
    DynSlot* slots = colLen <= DYN_SMEM_SLOTS ? reinterpret_cast<DynSlot*>(dyn_smem)
                                              : reinterpret_cast<DynSlot*>(a.ws.desc + (size_t)d * colLen);
    griddep_launch_dependents();
    if (threadIdx.x == 0) sStatus = 0u;
    // (before the dependency wait: a hint, and L2 is the point of coherence, so a line fetched early cannot go stale)
    // pull the (cold) metadata into L2 with ONE DRAM round trip: the R CTAs prefetch disjoint slices of the three arrays,
    // so the dependent loads below (block lengths -> list offset -> split index -> split offset) are L2 hits for all
    {
        const size_t gtid = (size_t)blockIdx.x * DYN_THREADS + threadIdx.x, gn = (size_t)gridDim.x * DYN_THREADS;
        const size_t lL = ((size_t)R * n * 8 + 127) >> 7, lB = ((size_t)R * R * 8 + 127) >> 7, lI = ((size_t)R * a.maxIndices * 8 + 127) >> 7;
        for (size_t i = gtid; i < lL + lB + lI; i += gn) {
            const char* p = i < lL ? reinterpret_cast<const char*>(a.L) + (i << 7)
                          : i < lL + lB ? reinterpret_cast<const char*>(a.blockLens) + ((i - lL) << 7)
                                        : reinterpret_cast<const char*>(a.indices) + ((i - lL - lB) << 7);
            prefetch_l2(p);
        }
    }
    griddep_wait();                                        // the metadata may have been written by the stream's previous kernel
    unsigned int st = 0;
    const unsigned long long keep = l2_policy_keep();      // metadata inputs stay in L2 across the payload stream (common.cuh)

    // ---- phase A: DYN_SU sources per warp at a time ------------------------------------------------------------
    for (int sBase = warp; sBase < R; sBase += DYN_WARPS * DYN_SU) {
        int src[DYN_SU];
        long long lv[DYN_SU][DYN_PL];                      // the first DYN_CHUNK split lengths: lane l holds PL*l .. PL*l + PL-1
        long long bv[DYN_SU][4];                           // the first 128 block lengths of row s: lane l holds l, l+32, ..
        unsigned long long sp[DYN_SU], rp[DYN_SU];
        // round trip 1: everything that does not depend on anything
#pragma unroll
        for (int u = 0; u < DYN_SU; ++u) {
            const int s = sBase + u * DYN_WARPS;
            src[u] = s;
            const bool on = s < R;
            const long long* Ls = a.L + (size_t)(on ? s : 0) * n;
            const long long* bls = a.blockLens + (size_t)(on ? s : 0) * R;
#pragma unroll
            for (int q = 0; q < DYN_PL; ++q) {
                const int i = DYN_PL * lane + q;
                lv[u][q] = (on && i < n) ? ld_keep(Ls + i, keep) : 0;
            }
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                const int dd = q * 32 + lane;
                bv[u][q] = (on && dd < R) ? ld_keep(bls + dd, keep) : 0;
            }
            sp[u] = on ? ld_keep_ptr(a.send + s, keep) : 0ull;
            rp[u] = on ? ld_keep_ptr(a.recvbuffs + (size_t)d * R + s, keep) : 0ull;
        }
        long long ioff[DYN_SU];
        int bl[DYN_SU];
#pragma unroll
        for (int u = 0; u < DYN_SU; ++u) {
            long long before = 0, mine = 0;
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                const int dd = q * 32 + lane;
                long long v = bv[u][q];
                if (v < 0) { st |= 4u; v = 0; }
                if (v > J) { st |= 4u; v = J; }
                if (dd < d) before += v;
                if (dd == d) mine = v;
            }
            if (src[u] < R) {
                const long long* bls = a.blockLens + (size_t)src[u] * R;
                for (int dd = 128 + lane; dd < R; dd += 32) {      // R > 128: the rest of the row
                    long long v = ld_keep(bls + dd, keep);
                    if (v < 0) { st |= 4u; v = 0; }
                    if (v > J) { st |= 4u; v = J; }
                    if (dd < d) before += v;
                    if (dd == d) mine = v;
                }
            }
            ioff[u] = warp_sum(before);
            bl[u] = (int)warp_sum(mine);
        }
        for (int j0 = 0; j0 < J; j0 += 32) {               // one pass per 32 list entries (J <= 32: one pass)
            const int j = j0 + lane;
            // round trip 2: this lane's split index, for all DYN_SU sources at once
            long long idx[DYN_SU];
            bool live[DYN_SU];
#pragma unroll
            for (int u = 0; u < DYN_SU; ++u) {
                idx[u] = -1; live[u] = false;
                if (src[u] < R && j < bl[u]) {
                    const long long pos = ioff[u] + j;
                    if (pos >= a.maxIndices) st |= 4u;
                    else idx[u] = ld_keep(a.indices + (size_t)src[u] * a.maxIndices + pos, keep);
                }
            }
#pragma unroll
            for (int u = 0; u < DYN_SU; ++u) {
                if (src[u] < R && j < bl[u] && ioff[u] + j < a.maxIndices) {
                    if (idx[u] < 0 || idx[u] >= n) { st |= 2u; idx[u] = -1; }
                    else live[u] = true;
                }
            }
            // offsets: exclusive prefix sums of the split lengths, DYN_CHUNK at a time, for all DYN_SU sources together (their
            // shuffle chains interleave): lane l holds lengths 4l .. 4l+3 of the chunk, one 64-bit warp scan of the lane totals,
            // then every lane PICKS offset and length of its own split from the owning lane's registers by shuffle -- no
            // shared-memory strip, no warp barriers (round 2a: 8 serialised scan + strip rounds, ~5 us of the kernel's 7 us phase A)
            long long base[DYN_SU], off[DYN_SU], len[DYN_SU];
#pragma unroll
            for (int u = 0; u < DYN_SU; ++u) { base[u] = 0; off[u] = 0; len[u] = 0; }
            for (int c0 = 0; c0 < n; c0 += DYN_CHUNK) {
                long long x[DYN_SU][DYN_PL];
#pragma unroll
                for (int u = 0; u < DYN_SU; ++u) {
                    const long long* Ls = a.L + (size_t)(src[u] < R ? src[u] : 0) * n;
#pragma unroll
                    for (int q = 0; q < DYN_PL; ++q) {
                        const int i = c0 + DYN_PL * lane + q;
                        x[u][q] = c0 == 0 ? lv[u][q] : ((src[u] < R && i < n) ? ld_keep(Ls + i, keep) : 0);
                    }
                }
#pragma unroll
                for (int u = 0; u < DYN_SU; ++u) {
#pragma unroll
                    for (int q = 0; q < DYN_PL; ++q) {
                        if (x[u][q] < 0) { if (j0 == 0) st |= 1u; x[u][q] = 0; }
                    }
                    long long tot = 0;
#pragma unroll
                    for (int q = 0; q < DYN_PL; ++q) tot += x[u][q];
                    const long long incl = warp_incl_scan(tot);
                    const long long excl = base[u] + incl - tot;
                    const bool mineHere = live[u] && idx[u] >= c0 && idx[u] < c0 + DYN_CHUNK;
                    const int rel = mineHere ? (int)(idx[u] - c0) : 0;
                    const int from = rel / DYN_PL, r = rel - from * DYN_PL;
                    long long o = __shfl_sync(0xffffffffu, excl, from), l = 0;
#pragma unroll
                    for (int q = 0; q < DYN_PL; ++q) {
                        const long long y = __shfl_sync(0xffffffffu, x[u][q], from);
                        if (q < r) o += y;
                        if (q == r) l = y;
                    }
                    if (mineHere) { off[u] = o; len[u] = l; }
                    base[u] += __shfl_sync(0xffffffffu, incl, 31);
                }
            }
#pragma unroll
            for (int u = 0; u < DYN_SU; ++u) {
                if (src[u] < R && j < J) {
                    DynSlot o;
                    o.bytes = live[u] ? len[u] * a.elemSize : 0;
                    o.src = live[u] ? sp[u] + (unsigned long long)(off[u] * a.elemSize) : 0ull;
                    o.dst = live[u] ? rp[u] + (unsigned long long)(off[u] * a.elemSize) : 0ull;
                    o.pad = 0;
                    slots[(size_t)src[u] * J + j] = o;
                }
            }
        }
    }
    st = __reduce_or_sync(0xffffffffu, st);
    if (lane == 0 && st) atomicOr(&sStatus, st);
    __syncthreads();

    // ---- phase B: tile prefixes in slot order, descriptors, coarse index ------------------------------------------
    long long run = 0;                                     // tiles of the column before this round: bulk << 32 | vector
    long long myBulkBytes = 0;
    for (int k0 = 0; k0 < colLen; k0 += DYN_THREADS) {
        const int k = k0 + threadIdx.x;
        DynSlot sl;
        sl.src = sl.dst = 0ull; sl.bytes = 0; sl.pad = 0;
        if (k < colLen) sl = slots[k];
        const int tb = seg_tiles(LIST_BULK, sl.src, sl.dst, sl.bytes, a.cls);
        const int tv = seg_tiles(LIST_VEC, sl.src, sl.dst, sl.bytes, a.cls);
        if (tb > 0) myBulkBytes += sl.bytes;
        const long long it = warp_incl_scan(((long long)tb << 32) | (long long)(unsigned int)tv);
        if (lane == 31) sWarpTot[warp] = it;
        __syncthreads();
        long long pre = run, all = 0;
#pragma unroll 8
        for (int w = 0; w < DYN_WARPS; ++w) {
            const long long t = sWarpTot[w];
            if (w < warp) pre += t;
            all += t;
        }
        if (k0 + warp * 32 < colLen && lane < 2)
            a.ws.coarse[lane][(size_t)d * nb + ((k0 >> 5) + warp)] = lane ? (int)(unsigned int)pre : (int)(pre >> 32);
        if (k < colLen) {
            const long long p = pre + it;
            uint4* out = reinterpret_cast<uint4*>(a.ws.desc + (size_t)d * colLen + k);
            out[0] = make_uint4((unsigned int)sl.src, (unsigned int)(sl.src >> 32), (unsigned int)sl.dst, (unsigned int)(sl.dst >> 32));
            out[1] = make_uint4((unsigned int)sl.bytes, (unsigned int)((unsigned long long)sl.bytes >> 32),
                                (unsigned int)(p >> 32), (unsigned int)p);
        }
        run += all;
        __syncthreads();                                   // sWarpTot is rewritten in the next round
    }
    myBulkBytes = warp_sum(myBulkBytes);
    if (lane == 0) sWarpTot[warp] = myBulkBytes;           // (the last round's barrier has passed: sWarpTot is free)
    __syncthreads();
    if (threadIdx.x == 0) {
        long long bb = 0;
        for (int w = 0; w < DYN_WARPS; ++w) bb += sWarpTot[w];
        a.ws.colTiles[LIST_BULK][d] = (int)(run >> 32);
        a.ws.colTiles[LIST_VEC][d] = (int)(unsigned int)run;
        a.ws.colKiB[d] = (int)(bb >> 10);
        if (sStatus) atomicOr(&a.ws.ctl->status, sStatus);
    }
}

}  // namespace xdev
