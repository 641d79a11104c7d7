// dynamic_kernel.cuh -- work-list builder for the paper's full AllToAllvDynamic metadata interface
// (section 6.1.2): sendSplitLengths + sendIndices +
// sendIndicesBlockLens on the send side, per-source recvbuffs with the sender's padding preserved and
// recvAllSplitLengths on the receive side.  It reuses steps a3/a4 (descriptor table + segment_copy_kernel)
// with one more indirection: a segment is one (source s, destination d, list position j) triple, i.e. one
// whole split, copied to the SAME offset in recvbuffs[d][s] that it has in send[s] (L439 "paddings are
// reserved", Fig. 17).
//
// ONE metadata kernel (round 1 had two, 12 us in front of a 70 us copy):
//   dyn_build_kernel  grid R x 1024 threads: CTA d builds column d of the table, slots k = s*J + j, j < J =
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

constexpr int DYN_THREADS = 1024;
constexpr int DYN_WARPS = DYN_THREADS / 32;
constexpr int DYN_SMEM_SLOTS = 4096;      // columns up to this many slots are staged in shared memory (32 B per slot)

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

// dynamic smem: DynSlot[min(colLen, DYN_SMEM_SLOTS)] (none when the column is longer)
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
    griddep_wait();                                        // the metadata may have been written by the stream's previous kernel
    unsigned int st = 0;

    // ---- phase A: warp per source ----------------------------------------------------------------------------
    for (int s = warp; s < R; s += DYN_WARPS) {
        const long long* Ls = a.L + (size_t)s * n;
        const long long* bls = a.blockLens + (size_t)s * R;
        // round trip 1: row s of the block lengths, the first 128 split lengths, both base pointers
        constexpr int PRE = 4;
        long long lpre[PRE];
#pragma unroll
        for (int u = 0; u < PRE; ++u) { const int i = u * 32 + lane; lpre[u] = i < n ? Ls[i] : 0; }
        const unsigned long long sp = (unsigned long long)a.send[s];
        const unsigned long long rp = (unsigned long long)a.recvbuffs[(size_t)d * R + s];
        long long before = 0, mine = 0;
        for (int d0 = 0; d0 < R; d0 += 32 * 4) {
            long long v[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) { const int dd = d0 + u * 32 + lane; v[u] = dd < R ? bls[dd] : 0; }
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const int dd = d0 + u * 32 + lane;
                if (v[u] < 0) { st |= 4u; v[u] = 0; }
                if (v[u] > J) { st |= 4u; v[u] = J; }
                if (dd < d) before += v[u];
                if (dd == d) mine = v[u];
            }
        }
        const long long ioff = warp_sum(before);
        const int bl = (int)warp_sum(mine);
        for (int j0 = 0; j0 < J; j0 += 32) {               // one pass per 32 list entries (J <= 32: one pass)
            const int j = j0 + lane;
            // round trip 2: this lane's split index
            long long idx = -1;
            bool live = false;
            if (j < bl) {
                const long long pos = ioff + j;
                if (pos >= a.maxIndices) st |= 4u;
                else {
                    idx = a.indices[(size_t)s * a.maxIndices + pos];
                    if (idx < 0 || idx >= n) { st |= 2u; idx = -1; }
                    else live = true;
                }
            }
            // one scan per 32 split lengths; every lane picks offset and length of ITS split from the lane that holds it
            long long base = 0, off = 0, len = 0;
            for (int i0 = 0; i0 < n; i0 += 32) {
                long long v;
                if (i0 < PRE * 32) {
                    v = lpre[0];
#pragma unroll
                    for (int u = 1; u < PRE; ++u) if ((i0 >> 5) == u) v = lpre[u];
                } else {
                    v = i0 + lane < n ? Ls[i0 + lane] : 0;
                }
                if (v < 0) { if (j0 == 0) st |= 1u; v = 0; }
                const long long incl = warp_incl_scan(v);
                const int from = (int)(idx - i0) & 31;
                const long long po = __shfl_sync(0xffffffffu, base + incl - v, from);
                const long long pl = __shfl_sync(0xffffffffu, v, from);
                if (live && idx >= i0 && idx < i0 + 32) { off = po; len = pl; }
                base += __shfl_sync(0xffffffffu, incl, 31);
            }
            if (j < J) {
                DynSlot o;
                o.bytes = live ? len * a.elemSize : 0;
                o.src = live ? sp + (unsigned long long)(off * a.elemSize) : 0ull;
                o.dst = live ? rp + (unsigned long long)(off * a.elemSize) : 0ull;
                o.pad = 0;
                slots[(size_t)s * J + j] = o;
            }
        }
    }
    st = __reduce_or_sync(0xffffffffu, st);
    if (lane == 0 && st) atomicOr(&sStatus, st);
    __syncthreads();

    // ---- phase B: tile prefixes in slot order, descriptors, coarse index ------------------------------------------
    long long run = 0;                                     // tiles of the column before this round: bulk << 32 | vector
    for (int k0 = 0; k0 < colLen; k0 += DYN_THREADS) {
        const int k = k0 + threadIdx.x;
        DynSlot sl;
        sl.src = sl.dst = 0ull; sl.bytes = 0; sl.pad = 0;
        if (k < colLen) sl = slots[k];
        const int tb = seg_tiles(LIST_BULK, sl.src, sl.dst, sl.bytes, a.cls);
        const int tv = seg_tiles(LIST_VEC, sl.src, sl.dst, sl.bytes, a.cls);
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
    if (threadIdx.x == 0) {
        a.ws.colTiles[LIST_BULK][d] = (int)(run >> 32);
        a.ws.colTiles[LIST_VEC][d] = (int)(unsigned int)run;
        if (sStatus) atomicOr(&a.ws.ctl->status, sStatus);
    }
}

}  // namespace xdev
