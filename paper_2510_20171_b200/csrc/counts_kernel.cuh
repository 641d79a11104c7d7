// counts_kernel.cuh -- steps a1-a3 of the hot path:
//   a1  RC[d][s] = C[s][d]                     the paper's "metadata exchange"
//   a2  soff (row-wise) / roff (column-wise) exclusive scans of the R x R count matrix (L381, L429)
//   a3  byte-balanced work list: per-segment descriptors + tile-count prefixes (L425 "multi-blocks
//       copy in parallel"; replaces the serial T_c*(N-1) issue loop of L447)
// all on the device, from the counts as they are in memory when the kernel RUNS (L401, L409).
//
// Parallel decomposition: CTA j owns the W destination columns [j*W, j*W+W).  Everything indexed by destination (RC
// row d, roff row d, descriptor row d, per-column tile totals) is produced by the owner; the only cross-column
// quantity is the row-wise send offset soff[s][d] = (row s's prefix over the columns before d0) + a running sum:
//   R <= 128  the owner rebuilds that prefix from C[s][0..d0) itself (an L2-resident re-read of at most 128 KB per CTA,
//             no inter-CTA communication: cheaper than any barrier at this size);
//   R  > 128  every CTA reads only its own R x W block, publishes one block sum per row, and after ONE grid barrier adds
//             up the block sums of the CTAs before it (R*j values instead of R*d0: the re-read grows as R^3 / W over the
//             grid and was 23 / 81 / 181 us of the kernel at R = 256 / 512 / 1024; now 112 / 411 / 1480 us per call
//             instead of 116 / 437 / 1571).
// The cross-column tile base is left to the copy kernel, which scans the R per-column totals itself.
//
// This kernel sits on the small-message latency path (config 5: ~5 % of the call; a per-CTA %globaltimer timeline
// of it is in profiles/r2_cfg5_timeline.md), so both phases are laid out for latency: phase 1 issues all global
// loads up front (a few lanes per row, no warp scans), the pointer tables are staged in shared memory while
// those loads fly, and phase 2 spreads the (column, row block) items over all warps and only reads shared memory.
#pragma once
#include "common.cuh"

namespace xdev {

constexpr int COUNTS_THREADS = 512;
constexpr int COUNTS_BARRIER_POLLS = 8192;   // ~2-4 ms of polling before a CTA falls back to the barrier-free prefix (see phase 1)

struct CountsArgs {
    const void* const* send;      // device table (null: no descriptors wanted, offsets and RC only)
    void* const* recv;            // device table (null likewise)
    const long long* C;           // R*R, by reference
    long long* RC;                // R*R out
    Workspace ws;
    int R;
    int W;                        // columns per CTA (<= 32)
    int blockSums;                // 1: phase 1 through per-CTA block sums and a grid barrier (R > 128); 0: row prefixes re-read from C
    long long elemSize;               // bytes per count unit (an element, or a whole row for the top-k calls)
    ClassParams cls;
};


// dynamic smem: long long cval[R][W+1], sofs[R][W+1] (+1: conflict-free column reads), u64 sendPtr[R], recvPtr[W],
//               long long tileTot[W*nb], rowsBefore[W*nb], byteTot[W*nb]   (nb = ceil(R/32))
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
    const int d0 = blockIdx.x * W;
    const int Wc = min(W, R - d0);

    griddep_launch_dependents();                 // let the copy kernel's CTAs start their prologue
    // the count matrix is usually cold (the previous call streamed far more than L2 holds): the grid prefetches all of
    // it into L2 with one DRAM round trip, before and after the dependency wait (before: while the stream's previous
    // kernel drains; after: in case that took long enough for the lines to be evicted again)
    const size_t cLines = ((size_t)R * R * 8 + 127) >> 7;
    const size_t gtid = (size_t)blockIdx.x * COUNTS_THREADS + threadIdx.x, gthreads = (size_t)gridDim.x * COUNTS_THREADS;
    for (size_t i = gtid; i < cLines; i += gthreads) prefetch_l2(reinterpret_cast<const char*>(a.C) + (i << 7));
    griddep_wait();                              // (launched with PDL itself: the stream's previous kernel must be complete)
    for (size_t i = gtid; i < cLines; i += gthreads) prefetch_l2(reinterpret_cast<const char*>(a.C) + (i << 7));
    // pointer tables: issue the loads now, park them in shared memory after phase 1's loads are in flight too (one
    // DRAM round trip instead of two on a cold start)
    constexpr int PT = 2;                        // covers R <= 1024 with 512 threads
    const unsigned long long keep = l2_policy_keep();    // metadata inputs stay in L2 across the payload stream (common.cuh)
    unsigned long long sp[PT];
#pragma unroll
    for (int i = 0; i < PT; ++i) {
        const int s = threadIdx.x + i * COUNTS_THREADS;
        sp[i] = (s < R && a.send) ? ld_keep_ptr(a.send + s, keep) : 0ull;        // null tables: offsets only (top-k calls)
    }
    const unsigned long long rp = (threadIdx.x < Wc && a.recv) ? ld_keep_ptr(a.recv + d0 + threadIdx.x, keep) : 0ull;

    bool sawNeg = false;
    if (!a.blockSums) {
        // (R <= 128) the row prefix straight from the count matrix: at most 128 KB of L2-resident re-reads per CTA cost
        // less than a grid barrier (measured, graph replay p50: config 5 155.0 vs 157.0 us, R = 64 x 10 KB 26.0 vs 28.1 us)
        // ---- phase 1: soff for the owned columns = row prefix C[s][0..d0) + running sum over the owned columns ------
        // LPR lanes share a row (LPR = 512 / R rounded down to a power of two, 8..32): lane q sums the prefix columns
        // q, q + LPR, ..., all loads independent (a handful per lane at R <= 128), then log2(LPR) shuffle steps combine
        // the row.  (Round 1 gave a warp 8 rows and ran a 64-bit warp reduction AND a warp scan per row: ~5 us of
        // dependent shuffles at R = 128; this is one round trip plus a few adds.)
        int LPR = 32;
        while (LPR > 8 && LPR * R > COUNTS_THREADS) LPR >>= 1;    // >= 8 lanes (64 contiguous bytes) per row: coalescing at large R
        const int rowsPerPass = COUNTS_THREADS / LPR;
        const int q = threadIdx.x & (LPR - 1);
        for (int row0 = 0; row0 < R; row0 += rowsPerPass) {
            const int s = row0 + threadIdx.x / LPR;
            const bool valid = s < R;
            const long long* row = a.C + (size_t)(valid ? s : 0) * R;
            constexpr int OW = 4;                                          // owned columns kept in registers (W <= 4: R <= 128)
            long long own[OW];
    #pragma unroll
            for (int j = 0; j < OW; ++j) own[j] = (valid && q == 0 && j < Wc) ? ld_keep(row + d0 + j, keep) : 0;
            long long part = 0;
            constexpr int LU = 16;                                         // independent loads per trip
            for (int dd = q; dd < d0; dd += LPR * LU) {
                long long v[LU];
    #pragma unroll
                for (int u = 0; u < LU; ++u) { const int x = dd + u * LPR; v[u] = (valid && x < d0) ? ld_keep(row + x, keep) : 0; }
    #pragma unroll
                for (int u = 0; u < LU; ++u) part += v[u] > 0 ? v[u] : 0;
            }
            if (row0 == 0) {                                               // every thread passes here exactly once
    #pragma unroll
                for (int i = 0; i < PT; ++i) {
                    const int t = threadIdx.x + i * COUNTS_THREADS;
                    if (t < R) sendPtr[t] = sp[i];
                }
                if (threadIdx.x < Wc) recvPtr[threadIdx.x] = rp;
            }
            for (int o = LPR >> 1; o > 0; o >>= 1) part += __shfl_xor_sync(0xffffffffu, part, o);
            if (valid && q == 0) {
                long long run = part;
    #pragma unroll
                for (int j = 0; j < OW; ++j) {
                    if (j < Wc) {
                        long long cc = own[j];
                        if (cc < 0) { sawNeg = true; cc = 0; }
                        cval[(size_t)s * P + j] = cc;
                        sofs[(size_t)s * P + j] = run;
                        a.ws.soff[(size_t)s * R + d0 + j] = run;
                        run += cc;
                    }
                }
                for (int j = OW; j < Wc; ++j) {
                    long long cc = ld_keep(row + d0 + j, keep);
                    if (cc < 0) { sawNeg = true; cc = 0; }
                    cval[(size_t)s * P + j] = cc;
                    sofs[(size_t)s * P + j] = run;
                    a.ws.soff[(size_t)s * R + d0 + j] = run;
                    run += cc;
                }
            }
        }
    } else {
        // ---- phase 1: soff for the owned columns = (row prefix over the columns of CTAs 0..j-1) + running sum over the owned ones ----
        // Round 1 / 2a rebuilt the row prefix C[s][0..d0) in every CTA from the count matrix itself: R*d0 loads per CTA, all
        // CTAs pulling the same lines through L2 -- 2 to 6.5 us per CTA at R = 128 (per-CTA stamps), and 23 / 81 / 181 us for
        // the whole kernel at R = 256 / 512 / 1024.  Now every CTA reads ONLY its own R x W block (coalesced), publishes one
        // block sum per row, and after one grid barrier adds up the block sums of the CTAs before it (R*j values instead of
        // R*d0).  The barrier is safe: the grid has at most COUNTS_MAX_CTAS small CTAs, all of which are resident before any
        // dependent kernel may start (griddepcontrol.launch_dependents fires only once every CTA has issued it), and no kernel
        // that could hold SMs depends on this one.
        for (int i = threadIdx.x; i < R * Wc; i += COUNTS_THREADS) {            // own block -> shared memory, clamped
            const int s = i / Wc, j = i - s * Wc;
            long long cc = ld_keep(a.C + (size_t)s * R + d0 + j, keep);
            if (cc < 0) { sawNeg = true; cc = 0; }
            cval[(size_t)s * P + j] = cc;
        }
    #pragma unroll
        for (int i = 0; i < PT; ++i) {
            const int t = threadIdx.x + i * COUNTS_THREADS;
            if (t < R) sendPtr[t] = sp[i];
        }
        if (threadIdx.x < Wc) recvPtr[threadIdx.x] = rp;
        __syncthreads();
        const int G = (int)gridDim.x;
        for (int s = threadIdx.x; s < R; s += COUNTS_THREADS) {                 // running sums inside the block, block sum out
            long long run = 0;
            for (int j = 0; j < Wc; ++j) { sofs[(size_t)s * P + j] = run; run += cval[(size_t)s * P + j]; }
            if (G > 1) a.ws.blockSum[(size_t)blockIdx.x * R + s] = run;
        }
        __shared__ int sTimedOut;
        if (G > 1) {
            __syncthreads();
            if (threadIdx.x == 0) {
                __threadfence();
                atomicAdd(&a.ws.ctl->barArrive, 1u);
                // bounded wait: should the grid ever NOT be resident as a whole (two such metadata kernels of > 700 ranks
                // dispatched interleaved on two streams would each hold part of the device), a CTA gives up after a few
                // milliseconds, rebuilds its row prefixes from the count matrix like the R <= 128 path, and leaves --
                // freeing its SM, so the barrier can never deadlock; results are the same either way
                unsigned int seen = 0;
                for (int it = 0; it < COUNTS_BARRIER_POLLS; ++it) {
                    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(seen) : "l"(&a.ws.ctl->barArrive) : "memory");
                    if (seen >= (unsigned int)G) break;
                    if (it > 64) __nanosleep(256);
                }
                sTimedOut = seen < (unsigned int)G ? 1 : 0;
#ifdef XDEV_TEST_FORCE_BARRIER_TIMEOUT
                if (blockIdx.x & 1) sTimedOut = 1;                 // test builds: odd CTAs take the fallback although everyone arrived
#endif
            }
            __syncthreads();
        } else if (threadIdx.x == 0) {
            sTimedOut = 0;
        }
        if (G <= 1) __syncthreads();
        const bool timedOut = sTimedOut != 0;
        for (int s = threadIdx.x; s < R; s += COUNTS_THREADS) {                 // + the block sums of the CTAs before this one
            long long pre = 0;
            constexpr int BU = 8;
            if (!timedOut) {
                for (int jb = 0; jb < (int)blockIdx.x; jb += BU) {
                    long long v[BU];
    #pragma unroll
                    for (int u = 0; u < BU; ++u) v[u] = jb + u < (int)blockIdx.x ? __ldcg(a.ws.blockSum + (size_t)(jb + u) * R + s) : 0;   // L2: written by other CTAs of this grid
    #pragma unroll
                    for (int u = 0; u < BU; ++u) pre += v[u];
                }
            } else {
                const long long* row = a.C + (size_t)s * R;
                for (int x = 0; x < d0; ++x) { const long long v = ld_keep(row + x, keep); pre += v > 0 ? v : 0; }
            }
            for (int j = 0; j < Wc; ++j) {
                const long long o = sofs[(size_t)s * P + j] + pre;
                sofs[(size_t)s * P + j] = o;
                a.ws.soff[(size_t)s * R + d0 + j] = o;
            }
        }
        if (G > 1 && threadIdx.x == 0) {                                        // last CTA past the barrier re-arms it
            if (atomicAdd(&a.ws.ctl->barDepart, 1u) == (unsigned int)G - 1u) {
                a.ws.ctl->barArrive = 0u; a.ws.ctl->barDepart = 0u;
                __threadfence();
            }
        }
    }
    if (sawNeg) atomicOr(&a.ws.ctl->status, 1u);
    __syncthreads();

    // ---- phase 2: one work item per (owned column j, block b of 32 source rows), items round-robin over the warps ----
    // (round 1 ran one warp per COLUMN, serially over the row blocks: with few columns per CTA most warps idled through
    //  the longest dependent chain of the kernel.)  An item needs two column-wise prefixes: the elements before the block
    //  (-> roff, destination addresses) and the tiles before it (-> work-list prefixes).  The first is a masked sum over
    //  shared memory; the second depends on the first (tile counts depend on the addresses), so: the front half computes
    //  every item's tile totals, the back half (after one barrier) adds the tile base and writes everything out.
    const int nb = (R + 31) >> 5;
    const int nItems = Wc * nb;
    long long* tileTot = reinterpret_cast<long long*>(recvPtr + W);      // [W*nb] tiles of the item: bulk << 32 | vector
    long long* rowsBefore = tileTot + (size_t)W * nb;                    // [W*nb] elements of the column before the block
    long long* byteTot = rowsBefore + (size_t)W * nb;                    // [W*nb] bytes of the item's bulk-list segments
    struct Item { int j, b, s; bool valid; long long c, ro, bytes, it; unsigned long long src, dst; int tb; };
    // front half: everything that does not need the other items' tile totals
    auto front = [&](int item, bool first) {
        Item x;
        x.j = item / nb; x.b = item - x.j * nb;
        long long run;
        if (first) {
            long long part = 0;
            for (int sp2 = lane; sp2 < x.b * 32; sp2 += 32) part += cval[(size_t)sp2 * P + x.j];
            run = warp_sum(part);
            if (lane == 0) rowsBefore[item] = run;
        } else {
            run = rowsBefore[item];
        }
        x.s = x.b * 32 + lane;
        x.valid = x.s < R;
        x.c = x.valid ? cval[(size_t)x.s * P + x.j] : 0;
        const long long incl = warp_incl_scan(x.c);
        x.ro = run + incl - x.c;
        x.bytes = x.c * a.elemSize;
        x.src = 0; x.dst = 0; x.tb = 0;
        int tv = 0;
        if (x.valid) {
            x.src = sendPtr[x.s] + (unsigned long long)(sofs[(size_t)x.s * P + x.j] * a.elemSize);
            x.dst = recvPtr[x.j] + (unsigned long long)(x.ro * a.elemSize);
            x.tb = seg_tiles(LIST_BULK, x.src, x.dst, x.bytes, a.cls);
            tv = seg_tiles(LIST_VEC, x.src, x.dst, x.bytes, a.cls);
        }
        x.it = warp_incl_scan(((long long)x.tb << 32) | (long long)(unsigned int)tv);   // both lists at once
        if (first) {
            const long long bb = warp_sum(x.tb > 0 ? x.bytes : 0);
            if (lane == 31) tileTot[item] = x.it;
            if (lane == 0) byteTot[item] = bb;
        }
        return x;
    };
    // back half (after the barrier): tile base of the item inside its column, then everything is written out
    auto back = [&](const Item& x) {
        const int d = d0 + x.j;
        long long base = 0, allT = 0, allB = 0;                        // tiles of the column before this block / in total
        for (int bp = lane; bp < nb; bp += 32) {
            const long long t = tileTot[(size_t)x.j * nb + bp];
            if (bp < x.b) base += t;
            allT += t;
            allB += byteTot[(size_t)x.j * nb + bp];
        }
        base = warp_sum(base);
        if (lane < 2) a.ws.coarse[lane][(size_t)d * nb + x.b] = lane ? (int)(unsigned int)base : (int)(base >> 32);   // coarse index for the copy kernel's search
        if (x.valid) {
            const size_t q = (size_t)d * R + x.s;
            const long long pf = base + x.it;
            a.RC[q] = x.c;
            a.ws.roff[q] = x.ro;
            uint4* out = reinterpret_cast<uint4*>(a.ws.desc + q);
            out[0] = make_uint4((unsigned int)x.src, (unsigned int)(x.src >> 32), (unsigned int)x.dst, (unsigned int)(x.dst >> 32));
            out[1] = make_uint4((unsigned int)x.bytes, (unsigned int)((unsigned long long)x.bytes >> 32),
                                (unsigned int)(pf >> 32), (unsigned int)pf);
        }
        if (x.b == 0) {                                                // column totals, once per column
            allT = warp_sum(allT);
            allB = warp_sum(allB);
            if (lane == 0) {
                a.ws.colTiles[LIST_BULK][d] = (int)(allT >> 32);
                a.ws.colTiles[LIST_VEC][d] = (int)(unsigned int)allT;
                a.ws.colKiB[d] = (int)(allB >> 10);
            }
        }
    };
    if (nItems <= nwarps) {
        // at most one item per warp (R <= 128 with 32 CTAs): its state stays in registers across the barrier, nothing is
        // computed twice
        Item x{};
        if (warp < nItems) x = front(warp, true);
        __syncthreads();
        if (warp < nItems) back(x);
    } else {
        for (int item = warp; item < nItems; item += nwarps) (void)front(item, true);
        __syncthreads();
        for (int item = warp; item < nItems; item += nwarps) back(front(item, false));
    }
}

}  // namespace xdev
