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
#pragma once
#include "common.cuh"

namespace ncclx {

constexpr int COUNTS_THREADS = 512;

struct CountsArgs {
    const void* const* send;      // device table
    void* const* recv;            // device table
    const long long* C;           // R*R, by reference
    long long* RC;                // R*R out
    Workspace ws;
    int R;
    int W;                        // columns per CTA (<= 32)
    int elemSize;
    int tileShift[2];             // log2 tile bytes: bulk, vector
    long long bulkMinBytes;       // >= 16; segments below it (or unaligned) go to the vector list
    int forceVector;
};

// dynamic smem: long long cval[R][W+1], sofs[R][W+1]   (+1: conflict-free column reads)
__global__ void __launch_bounds__(COUNTS_THREADS) counts_kernel(const CountsArgs a) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int R = a.R, W = a.W, P = W + 1;
    long long* cval = reinterpret_cast<long long*>(smem_raw);
    long long* sofs = cval + (size_t)R * P;

    const int lane = lane_id();
    const int warp = threadIdx.x >> 5;
    const int nwarps = COUNTS_THREADS / 32;
    const int d0 = blockIdx.x * W;
    const int Wc = min(W, R - d0);

    if (blockIdx.x == 0 && threadIdx.x == 0) {   // the copy kernel follows on the same stream
        a.ws.ctl->next[0] = 0u;
        a.ws.ctl->next[1] = 0u;
    }

    // ---- phase 1: warp per source row s: soff for the owned columns -------------------------
    bool sawNeg = false;
    for (int s = warp; s < R; s += nwarps) {
        const long long* row = a.C + (size_t)s * R;
        long long part = 0;
        for (int d = lane; d < d0; d += 32) {
            long long c = row[d];
            part += c > 0 ? c : 0;
        }
        const long long base = warp_sum(part);
        long long c = 0;
        if (lane < Wc) {
            c = row[d0 + lane];
            if (c < 0) { sawNeg = true; c = 0; }
        }
        const long long incl = warp_incl_scan(c);
        if (lane < Wc) {
            const long long so = base + incl - c;
            cval[(size_t)s * P + lane] = c;
            sofs[(size_t)s * P + lane] = so;
            a.ws.soff[(size_t)s * R + d0 + lane] = so;
        }
    }
    if (sawNeg) atomicOr(&a.ws.ctl->status, 1u);
    __syncthreads();

    // ---- phase 2: warp per owned destination column d: RC, roff, descriptors, tile prefixes --
    const long long tileB = 1ll << a.tileShift[LIST_BULK];
    const long long tileV = 1ll << a.tileShift[LIST_VEC];
    for (int j = warp; j < Wc; j += nwarps) {
        const int d = d0 + j;
        const unsigned long long dstBase = (unsigned long long)a.recv[d];
        long long run = 0;
        int runT[2] = {0, 0};
        for (int s0 = 0; s0 < R; s0 += 32) {
            const int s = s0 + lane;
            const bool valid = s < R;
            const long long c = valid ? cval[(size_t)s * P + j] : 0;
            const long long incl = warp_incl_scan(c);
            const long long ro = run + incl - c;
            const long long bytes = c * a.elemSize;
            unsigned long long src = 0, dst = 0;
            int tb = 0, tv = 0;
            if (valid) {
                src = (unsigned long long)a.send[s] + (unsigned long long)(sofs[(size_t)s * P + j] * a.elemSize);
                dst = dstBase + (unsigned long long)(ro * a.elemSize);
                if (bytes > 0) {
                    const bool bulk = !a.forceVector && (((src | dst) & 15ull) == 0) && bytes >= a.bulkMinBytes;
                    if (bulk) tb = (int)((bytes + tileB - 1) >> a.tileShift[LIST_BULK]);
                    else      tv = (int)((bytes + tileV - 1) >> a.tileShift[LIST_VEC]);
                }
            }
            const int ib = warp_incl_scan(tb);
            const int iv = warp_incl_scan(tv);
            if (valid) {
                const size_t q = (size_t)d * R + s;
                a.RC[q] = c;
                a.ws.roff[q] = ro;
                SegDesc sd;
                sd.src = src; sd.dst = dst; sd.bytes = bytes;
                sd.pfx[LIST_BULK] = runT[0] + ib;
                sd.pfx[LIST_VEC] = runT[1] + iv;
                uint4* out = reinterpret_cast<uint4*>(a.ws.desc + q);
                const uint4* in = reinterpret_cast<const uint4*>(&sd);
                out[0] = in[0];
                out[1] = in[1];
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

}  // namespace ncclx
