// counts_kernel.cuh -- steps a1-a3 of the hot path:
//   a1  RC[d][s] = C[s][d]                     the paper's "metadata exchange"
//   a2  soff (row-wise) / roff (column-wise) exclusive scans of the R x R count matrix (L381, L429)
//   a3  byte-balanced work list: per-segment descriptors + tile-count prefixes (L425 "multi-blocks
//       copy in parallel"; replaces the serial T_c*(N-1) issue loop of L447)
// all on the device, from the counts as they are in memory when the kernel RUNS (L401, L409).
//
// Parallel decomposition with no inter-CTA communication: CTA j owns the W destination
// columns [j*W, j*W+W).  Everything indexed by destination (RC row d, roff row d, descriptor row
// d, per-column tile totals) is produced by the owner; the only cross-column quantity, the
// row-wise send offset soff[s][d], is rebuilt by the owner from row s's prefix C[s][0..d0) (an
// L2-resident re-read of at most R*R*8 bytes per CTA).  The cross-column tile base is left to
// the copy kernel, which scans the R per-column totals itself.
//
// This kernel sits on the small-message latency path (config 5: ~5 % of the call), so all global
// loads are issued up front with high memory-level parallelism: each warp sums ROWS_PER_PASS rows
// at once (ROWS_PER_PASS independent loads per lane per step) and the pointer tables are staged
// in shared memory while those loads fly; phase 2 then only reads shared memory and streams out
// its results.
#pragma once
#include "common.cuh"

namespace xdev {

constexpr int COUNTS_THREADS = 512;
constexpr int COUNTS_ROWS_PER_PASS = 8;
constexpr int COUNTS_COLS_UNROLL = 4;     // x32 lanes = 128 prefix columns per pass

struct CountsArgs {
    const void* const* send;      // device table (null: no descriptors wanted, offsets and RC only)
    void* const* recv;            // device table (null likewise)
    const long long* C;           // R*R, by reference
    long long* RC;                // R*R out
    Workspace ws;
    int R;
    int W;                        // columns per CTA (<= 32)
    long long elemSize;               // bytes per count unit (an element, or a whole row for the top-k calls)
    ClassParams cls;
};

// dynamic smem: long long cval[R][W+1], sofs[R][W+1] (+1: conflict-free column reads), u64 sendPtr[R], recvPtr[W]
__global__ void __launch_bounds__(COUNTS_THREADS) counts_kernel(const CountsArgs a) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int R = a.R, W = a.W, P = W + 1;
    long long* cval = reinterpret_cast<long long*>(smem_raw);
    long long* sofs = cval + (size_t)R * P;
    unsigned long long* sendPtr = reinterpret_cast<unsigned long long*>(sofs + (size_t)R * P);
    unsigned long long* recvPtr = sendPtr + R;

    const int lane = lane_id();
    const int warp = threadIdx.x >> 5;
    constexpr int nwarps = COUNTS_THREADS / 32;
    constexpr int RB = COUNTS_ROWS_PER_PASS;
    constexpr int DU = COUNTS_COLS_UNROLL;
    const int d0 = blockIdx.x * W;
    const int Wc = min(W, R - d0);

    griddep_launch_dependents();                 // let the copy kernel's CTAs start their prologue
    griddep_wait();                              // (launched with PDL itself: the stream's previous kernel must be complete)
    // pointer tables: issue the loads now, park them in shared memory only after phase 1's loads are
    // in flight too (one DRAM round trip instead of two on a cold start)
    constexpr int PT = 2;                        // covers R <= 1024 with 512 threads
    unsigned long long sp[PT];
#pragma unroll
    for (int i = 0; i < PT; ++i) {
        const int s = threadIdx.x + i * COUNTS_THREADS;
        sp[i] = (s < R && a.send) ? (unsigned long long)a.send[s] : 0ull;        // null tables: offsets only (top-k calls)
    }
    const unsigned long long rp = (threadIdx.x < Wc && a.recv) ? (unsigned long long)a.recv[d0 + threadIdx.x] : 0ull;
    bool parked = false;

    // ---- phase 1: warp per group of RB source rows: soff for the owned columns ---------------
    bool sawNeg = false;
    for (int sb = warp * RB; sb < R; sb += nwarps * RB) {
        long long part[RB], c[RB];
#pragma unroll
        for (int r = 0; r < RB; ++r) {
            part[r] = 0;
            c[r] = (sb + r < R && lane < Wc) ? a.C[(size_t)(sb + r) * R + d0 + lane] : 0;
        }
        // prefix columns [0, d0): RB x DU independent loads are issued before any of them is consumed
        for (int db = 0; db < d0; db += 32 * DU) {
            long long v[RB][DU];
#pragma unroll
            for (int r = 0; r < RB; ++r) {
#pragma unroll
                for (int u = 0; u < DU; ++u) {
                    const int d = db + u * 32 + lane;
                    v[r][u] = (sb + r < R && d < d0) ? a.C[(size_t)(sb + r) * R + d] : 0;
                }
            }
#pragma unroll
            for (int r = 0; r < RB; ++r) {
#pragma unroll
                for (int u = 0; u < DU; ++u) part[r] += v[r][u] > 0 ? v[r][u] : 0;
            }
        }
        if (!parked) {                                            // every thread passes here at most once
            parked = true;
#pragma unroll
            for (int i = 0; i < PT; ++i) {
                const int s = threadIdx.x + i * COUNTS_THREADS;
                if (s < R) sendPtr[s] = sp[i];
            }
            if (threadIdx.x < Wc) recvPtr[threadIdx.x] = rp;
        }
#pragma unroll
        for (int r = 0; r < RB; ++r) {
            const int s = sb + r;
            if (s >= R) break;                                    // warp-uniform
            const long long base = warp_sum(part[r]);
            long long cc = c[r];
            if (cc < 0) { sawNeg = true; cc = 0; }
            const long long incl = warp_incl_scan(cc);
            if (lane < Wc) {
                const long long so = base + incl - cc;
                cval[(size_t)s * P + lane] = cc;
                sofs[(size_t)s * P + lane] = so;
                a.ws.soff[(size_t)s * R + d0 + lane] = so;
            }
        }
    }
    if (!parked) {                                                // warps that owned no row group
#pragma unroll
        for (int i = 0; i < PT; ++i) {
            const int s = threadIdx.x + i * COUNTS_THREADS;
            if (s < R) sendPtr[s] = sp[i];
        }
        if (threadIdx.x < Wc) recvPtr[threadIdx.x] = rp;
    }
    if (sawNeg) atomicOr(&a.ws.ctl->status, 1u);
    __syncthreads();

    // ---- phase 2: warp per owned destination column d: RC, roff, descriptors, tile prefixes --
    for (int j = warp; j < Wc; j += nwarps) {
        const int d = d0 + j;
        const unsigned long long dstBase = recvPtr[j];
        long long run = 0;
        int runT[2] = {0, 0};
        const int nb = (R + 31) >> 5;
        for (int s0 = 0; s0 < R; s0 += 32) {
            if (lane < 2) a.ws.coarse[lane][(size_t)d * nb + (s0 >> 5)] = lane ? runT[1] : runT[0];     // coarse index for the copy kernel's search
            const int s = s0 + lane;
            const bool valid = s < R;
            const long long c = valid ? cval[(size_t)s * P + j] : 0;
            const long long incl = warp_incl_scan(c);
            const long long ro = run + incl - c;
            const long long bytes = c * a.elemSize;
            unsigned long long src = 0, dst = 0;
            int tb = 0, tv = 0;
            if (valid) {
                src = sendPtr[s] + (unsigned long long)(sofs[(size_t)s * P + j] * a.elemSize);
                dst = dstBase + (unsigned long long)(ro * a.elemSize);
                tb = seg_tiles(LIST_BULK, src, dst, bytes, a.cls);
                tv = seg_tiles(LIST_VEC, src, dst, bytes, a.cls);
            }
            const long long it = warp_incl_scan(((long long)tb << 32) | (long long)(unsigned int)tv);   // both lists at once
            const int ib = (int)(it >> 32);
            const int iv = (int)(unsigned int)it;
            if (valid) {
                const size_t q = (size_t)d * R + s;
                a.RC[q] = c;
                a.ws.roff[q] = ro;
                uint4* out = reinterpret_cast<uint4*>(a.ws.desc + q);
                out[0] = make_uint4((unsigned int)src, (unsigned int)(src >> 32), (unsigned int)dst, (unsigned int)(dst >> 32));
                out[1] = make_uint4((unsigned int)bytes, (unsigned int)((unsigned long long)bytes >> 32),
                                    (unsigned int)(runT[0] + ib), (unsigned int)(runT[1] + iv));
            }
            run += __shfl_sync(0xffffffffu, incl, 31);
            runT[0] += __shfl_sync(0xffffffffu, ib, 31);
            runT[1] += __shfl_sync(0xffffffffu, iv, 31);
        }
        if (lane == 0) {
            a.ws.colTiles[LIST_BULK][d] = runT[0];
            a.ws.colTiles[LIST_VEC][d] = runT[1];
        }
    }
}

}  // namespace xdev
