// fused_kernel.cuh -- the single-launch small-message path of ncclx_alltoallv_dev (SURVEY.md section 8(f)
// NEXT-4: "single fused scan+copy kernel"; section 6.2: at small sizes the latency is
// the preparation overhead T_c*(N-1), half of it the control exchange, and the paper's answer is a
// "small-message fast path to bypass the default bookkeeping and load balancing logic").
//
// For R <= FUSED_MAX_R the whole call -- a1 transpose, a2 offset scans, a3 work list, a4 copy -- is ONE
// kernel: the R x R count matrix is at most 8 KB, so EVERY CTA reads it (one L2 round trip), rebuilds
// all offsets and the complete descriptor table in its own shared memory with warp scans, and goes
// straight to copying; nothing is handed from one kernel (or CTA) to another.  CTA 0 alone writes the
// user-visible results of the metadata steps (RC, soff, roff, status).  Differences from the two-kernel
// path, all possible because every CTA knows the byte total:
//   * the TILE SIZE is chosen on the device from the total (about two tiles per engine, between 4 KiB
//     and the configured maximum), so a 1 MB call spreads over all SMs instead of 32 of them;
//   * the first tile of every engine is assigned statically (tile e to engine e): a call of up to one
//     tile per engine issues no atomic at all; larger calls continue with the in-order dynamic claims
//     of the big path, on counters that reset themselves (workctl_checkout);
//   * descriptor look-ups (window loads, searches) hit shared memory, not L2.
// The result is bit-identical to the two-kernel path (pure data movement; same offsets).
#pragma once
#include "copy_kernel.cuh"

namespace xdev {

constexpr int FUSED_MAX_R = 32;            // R*R <= 1024 descriptors = 32 KB of shared memory

struct FusedArgs {
    const void* const* send;               // device table
    void* const* recv;                     // device table
    const long long* C;                    // R*R, by reference
    long long* RC;                         // R*R out
    long long* soff;                       // workspace copies for ncclx_alltoallv_last_offsets
    long long* roff;
    WorkCtl* ctl;                          // this path's own self-resetting claim counters
    unsigned int* status;                  // the library's status word
    int R;
    long long elemSize;
    unsigned int ringBytes;                // multiple of 128, >= 32 KB (the prologue's scratch aliases the ring)
    int kmax;                              // as CopyArgs::kmax
    int minTileShift[2];
    int bulkEngines;                       // as CopyArgs::bulkEngines
    ClassParams cls;                       // tileShift[] = upper bounds; the kernel picks the actual shifts
};

__host__ __device__ inline size_t fused_desc_offset(int R) {     // from the end of the ring; keeps SegDesc 32 B-aligned
    return (COPY_MBAR_BYTES + 2 * (size_t)(R + 1) * 4 + 31) & ~(size_t)31;
}
__host__ __device__ inline size_t fused_aux_bytes(int R) { return fused_desc_offset(R) + (size_t)R * R * sizeof(SegDesc); }

__device__ __forceinline__ int floor_log2_ll(long long v) { return v <= 0 ? 0 : 63 - __clzll(v); }

// dynamic smem: [ring: ringBytes][mbar: COPY_MBAR_COUNT x u64][colBase bulk: R+1][colBase vec: R+1][pad][SegDesc R*R]
__global__ void __launch_bounds__(COPY_THREADS, 1) alltoallv_fused_kernel(const FusedArgs a) {
    extern __shared__ __align__(128) unsigned char smem[];
    const int lane = lane_id();
    const int warp = threadIdx.x >> 5;
    constexpr int NW = COPY_THREADS / 32;
    const int R = a.R, RR = R * R;
    unsigned long long* mbar = reinterpret_cast<unsigned long long*>(smem + a.ringBytes);
    int* colBase[2];
    colBase[0] = reinterpret_cast<int*>(mbar + COPY_MBAR_COUNT);
    colBase[1] = colBase[0] + (R + 1);
    SegDesc* sdesc = reinterpret_cast<SegDesc*>(smem + a.ringBytes + fused_desc_offset(R));
    // prologue scratch, dead before the first TMA load lands in the ring (<= 17.3 KB at R = 32)
    long long* cnt = reinterpret_cast<long long*>(smem);
    long long* sof = cnt + RR;
    unsigned long long* sendPtr = reinterpret_cast<unsigned long long*>(sof + RR);
    unsigned long long* recvPtr = sendPtr + R;
    long long* rowTot = reinterpret_cast<long long*>(recvPtr + R);
    int* colT[2];
    colT[0] = reinterpret_cast<int*>(rowTot + R);
    colT[1] = colT[0] + R;
    const bool writer = blockIdx.x == 0;
    int* const nullptrs[2] = {nullptr, nullptr};

    griddep_launch_dependents();           // a following call of this library may start its prologue
    for (int i = threadIdx.x; i < COPY_MBAR_COUNT; i += COPY_THREADS) mbar_init(smem_u32(&mbar[i]), 1);
    fence_mbar_init();
    griddep_wait();                        // everything below reads what the stream's previous kernel wrote

    // ---- step 0: the whole count matrix and both pointer tables -> shared memory (one round trip) -----
    bool sawNeg = false;
    for (int i = threadIdx.x; i < RR; i += COPY_THREADS) {
        long long c = a.C[i];
        if (c < 0) { sawNeg = true; c = 0; }
        cnt[i] = c;
    }
    if (threadIdx.x < R) sendPtr[threadIdx.x] = (unsigned long long)a.send[threadIdx.x];
    else if (threadIdx.x >= 32 && threadIdx.x < 32 + R) recvPtr[threadIdx.x - 32] = (unsigned long long)a.recv[threadIdx.x - 32];
    if (sawNeg && writer) atomicOr(a.status, 1u);
    __syncthreads();

    // ---- step 1 (a2): warp per source row: soff = exclusive scan along the row; row totals -----------
    for (int s = warp; s < R; s += NW) {
        const long long c = lane < R ? cnt[s * R + lane] : 0;
        const long long incl = warp_incl_scan(c);
        if (lane < R) {
            sof[s * R + lane] = incl - c;
            if (writer) a.soff[s * R + lane] = incl - c;
        }
        if (lane == 31) rowTot[s] = incl;
    }
    __syncthreads();

    // ---- step 2: tile sizes from the byte total (every thread computes the same values) --------------
    long long totalElems = 0;
    for (int s = 0; s < R; ++s) totalElems += rowTot[s];
    const long long totalBytes = totalElems * a.elemSize;
    // about two tiles per engine, assuming the engine split of a call that is all on one list (E bulk engines by the
    // regimes of plan_ring: up to 48 / 96 maximum-size tiles per CTA; 16 vector engines)
    int E0 = a.bulkEngines;
    if (E0 == 0) {
        const long long maxTiles = totalBytes >> a.cls.tileShift[LIST_BULK];
        E0 = maxTiles <= 48ll * gridDim.x ? 4 : (maxTiles <= 96ll * gridDim.x ? 2 : 1);
    }
    ClassParams cls = a.cls;
    cls.tileShift[LIST_BULK] = max(a.minTileShift[LIST_BULK], min(a.cls.tileShift[LIST_BULK], floor_log2_ll(totalBytes / (2ll * gridDim.x * E0))));
    cls.tileShift[LIST_VEC] = max(a.minTileShift[LIST_VEC], min(a.cls.tileShift[LIST_VEC], floor_log2_ll(totalBytes / (2ll * gridDim.x * COPY_WARPS))));

    // ---- step 3 (a1, a2, a3): warp per destination column: RC, roff, descriptors, tile prefixes ------
    for (int d = warp; d < R; d += NW) {
        const bool valid = lane < R;
        const long long c = valid ? cnt[lane * R + d] : 0;
        const long long incl = warp_incl_scan(c);
        const long long ro = incl - c;
        const long long bytes = c * a.elemSize;
        unsigned long long src = 0, dst = 0;
        int tb = 0, tv = 0;
        if (valid) {
            src = sendPtr[lane] + (unsigned long long)(sof[lane * R + d] * a.elemSize);
            dst = recvPtr[d] + (unsigned long long)(ro * a.elemSize);
            tb = seg_tiles(LIST_BULK, src, dst, bytes, cls);
            tv = seg_tiles(LIST_VEC, src, dst, bytes, cls);
        }
        const long long it = warp_incl_scan(((long long)tb << 32) | (long long)(unsigned int)tv);
        const int ib = (int)(it >> 32);
        const int iv = (int)(unsigned int)it;
        if (valid) {
            const int q = d * R + lane;
            uint4* out = reinterpret_cast<uint4*>(sdesc + q);
            out[0] = make_uint4((unsigned int)src, (unsigned int)(src >> 32), (unsigned int)dst, (unsigned int)(dst >> 32));
            out[1] = make_uint4((unsigned int)bytes, (unsigned int)((unsigned long long)bytes >> 32), (unsigned int)ib, (unsigned int)iv);
            if (writer) { a.RC[q] = c; a.roff[q] = ro; }
        }
        if (lane == 31) { colT[LIST_BULK][d] = ib; colT[LIST_VEC][d] = iv; }
    }
    __syncthreads();
    if (warp < 2) {                        // cross-column tile bases (R <= 32: one warp scan per list)
        const int* ct = warp ? colT[1] : colT[0];
        int* cb = warp ? colBase[1] : colBase[0];
        const int v = lane < R ? ct[lane] : 0;
        const int incl = warp_incl_scan(v);
        if (lane == 0) cb[0] = 0;
        if (lane < R) cb[lane + 1] = incl;
    }
    fence_proxy_async_smem();              // scratch reads/writes (generic proxy) before TMA writes to the same bytes
    __syncthreads();                       // the scratch is dead from here on; the ring may be filled

    // ---- a4: the copy engines of the big path, fed from shared memory; the first tile of every engine is static ----
    const bool usedCounters = run_copy_engines<true>(sdesc, colBase, nullptrs, a.ctl, cls, R, R, a.bulkEngines, a.kmax, 1, -1, 2, smem, mbar,
                                                     a.ringBytes);
    workctl_checkout(a.ctl, usedCounters);
}

}  // namespace xdev
