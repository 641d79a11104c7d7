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
//   dyn_desc_kernel   grid R: warp d walks column d's slots (s, j), j < maxBlockLen, in s-major order and
//                     writes descriptors + per-column tile prefixes exactly like counts_kernel's phase 2.
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
    if (warp == 0) {                                       // exclusive scan of the split lengths
        long long run = 0;
        bool neg = false;
        for (int i0 = 0; i0 < n; i0 += 32) {
            long long v = i0 + lane < n ? Ls[i0 + lane] : 0;
            if (v < 0) { neg = true; v = 0; }
            const long long incl = warp_incl_scan(v);
            if (i0 + lane < n) a.O[(size_t)s * n + i0 + lane] = run + incl - v;
            run += __shfl_sync(0xffffffffu, incl, 31);
        }
        if (neg) atomicOr(&a.ws.ctl->status, 1u);
    } else if (warp == 1) {                                // exclusive scan of the block lengths
        long long run = 0;
        bool bad = false;
        for (int d0 = 0; d0 < R; d0 += 32) {
            long long v = d0 + lane < R ? a.blockLens[(size_t)s * R + d0 + lane] : 0;
            if (v < 0) { bad = true; v = 0; }
            if (v > a.maxBlockLen) { bad = true; v = a.maxBlockLen; }
            const long long incl = warp_incl_scan(v);
            if (d0 + lane < R) a.ioff[(size_t)s * R + d0 + lane] = run + incl - v;
            run += __shfl_sync(0xffffffffu, incl, 31);
        }
        if (bad) atomicOr(&a.ws.ctl->status, 4u);
    }
    // every receiver gets all of rank s's split lengths
    for (int k = threadIdx.x; k < R * n; k += DYN_PREP_THREADS) {
        const int d = k / n, i = k - d * n;
        const long long v = Ls[i];
        a.recvAll[((size_t)d * R + s) * n + i] = v > 0 ? v : 0;
    }
}

// one warp per CTA: column d
__global__ void __launch_bounds__(32) dyn_desc_kernel(const DynArgs a) {
    const int d = blockIdx.x, lane = lane_id();
    const int R = a.R, n = a.n, J = a.maxBlockLen;
    const int colLen = R * J;
    griddep_launch_dependents();
    griddep_wait();                                        // O / ioff come from dyn_prep_kernel
    int runT[2] = {0, 0};
    unsigned int st = 0;
    const int nb = (colLen + 31) >> 5;
    for (int k0 = 0; k0 < colLen; k0 += 32) {
        if (lane < 2) a.ws.coarse[lane][(size_t)d * nb + (k0 >> 5)] = lane ? runT[1] : runT[0];
        const int k = k0 + lane;
        unsigned long long src = 0, dst = 0;
        long long bytes = 0;
        if (k < colLen) {
            const int s = k / J, j = k - s * J;
            long long bl = a.blockLens[(size_t)s * R + d];
            bl = bl < 0 ? 0 : (bl > J ? J : bl);
            const long long pos = a.ioff[(size_t)s * R + d] + j;
            if (j < bl) {
                if (pos >= a.maxIndices) st |= 4u;
                else {
                    const long long idx = a.indices[(size_t)s * a.maxIndices + pos];
                    if (idx < 0 || idx >= n) st |= 2u;
                    else {
                        const long long len = a.L[(size_t)s * n + idx];
                        const long long off = a.O[(size_t)s * n + idx];
                        bytes = (len > 0 ? len : 0) * a.elemSize;
                        src = (unsigned long long)a.send[s] + (unsigned long long)(off * a.elemSize);
                        dst = (unsigned long long)a.recvbuffs[(size_t)d * R + s] + (unsigned long long)(off * a.elemSize);
                    }
                }
            }
        }
        const int tb = seg_tiles(LIST_BULK, src, dst, bytes, a.cls);
        const int tv = seg_tiles(LIST_VEC, src, dst, bytes, a.cls);
        const long long it = warp_incl_scan(((long long)tb << 32) | (long long)(unsigned int)tv);
        if (k < colLen) {
            uint4* out = reinterpret_cast<uint4*>(a.ws.desc + (size_t)d * colLen + k);
            out[0] = make_uint4((unsigned int)src, (unsigned int)(src >> 32), (unsigned int)dst, (unsigned int)(dst >> 32));
            out[1] = make_uint4((unsigned int)bytes, (unsigned int)((unsigned long long)bytes >> 32),
                                (unsigned int)(runT[0] + (int)(it >> 32)), (unsigned int)(runT[1] + (int)(unsigned int)it));
        }
        const long long last = __shfl_sync(0xffffffffu, it, 31);
        runT[0] += (int)(last >> 32);
        runT[1] += (int)(unsigned int)last;
    }
    st = __reduce_or_sync(0xffffffffu, st);
    if (lane == 0) {
        a.ws.colTiles[LIST_BULK][d] = runT[0];
        a.ws.colTiles[LIST_VEC][d] = runT[1];
        if (st) atomicOr(&a.ws.ctl->status, st);
    }
}

}  // namespace ncclx
