// copy_kernel.cuh -- step a4 of the hot path: the byte-balanced variable-segment copy
// ("GPU side launches multi-blocks to copy data in parallel"; Fig. 3 L156 in-kernel
// D2D / P2P copy).  Every peer is local HBM here, so this kernel IS the AllToAllv payload term
// S/BW of L447.
//
// B200 design (not the paper's H100 kernel):
//   * persistent grid, one CTA per SM, work discovered on the device from the descriptor table the
//     metadata kernel wrote -- the host knows neither sizes nor tile counts, so the launch is
//     graph-capturable with a fixed grid (L387, L401);
//   * work unit = a tile of at most 2^tileShift bytes of ONE segment; after one static first chunk per
//     engine, tiles are claimed dynamically, in order, in guided chunks from a global counter that
//     resets itself => balance by BYTES (and by time), not by segment or by rank (config 3 skew is
//     250x across segments, 150x across ranks);
//   * EVERY payload byte is loaded by the TMA (descriptor-less 1-D cp.async.bulk global->shared, completion on
//     an mbarrier) into a byte-granular ring in shared memory, so ~200 KB of loads are in flight per SM without
//     register staging, whatever the alignment:
//       - "bulk" list (source, destination 16-byte aligned, >= bulkMinBytes): tiles of 32 KiB, stored with
//         cp.async.bulk shared->global; one elected lane of warp 0 (or of warps 0..E-1) issues everything;
//       - "vector" list (short segments and ANY other alignment -- counts are element-granular):
//         each engine warp owns a share of the ring and loads the 16-byte-aligned SPAN that covers a 4 KiB piece
//         of its tile; when source and destination are misaligned differently the warp realigns the piece IN PLACE
//         in shared memory (funnel shifts), and the body goes out as one cp.async.bulk shared->global as well
//         (head / tail bytes, < 16 at the ends of a tile, by lanes).  (Round 1 copied these global->registers->
//         global with ~61 KB in flight per SM: 3.7 TB/s; warp stores from shared memory: 6.09-6.14 TB/s on 1.4-1.7 GB
//         calls; TMA stores: 6.21-6.23 TB/s; the aligned bulk list on the same bytes: 6.72 TB/s.)
//   * the ring is split between the two lists on the device, grid-uniformly, from their tile totals.
#pragma once
#include "common.cuh"

namespace xdev {

constexpr int COPY_THREADS = 512;          // 16 warps: bulk engines first, then vector engines (split chosen on the device)
constexpr int COPY_WARPS = COPY_THREADS / 32;
constexpr int COPY_SLOTS = 32;             // outstanding bulk tiles per engine (mbarriers; slot j lives in lane j): <= 32
constexpr int COPY_MAX_ENGINES = 4;        // bulk engines (warps 0..E-1) per CTA, each with its own share of the ring
constexpr int VEC_SLOTS = 16;              // outstanding staged pieces per vector engine
constexpr int VEC_SUB_BYTES = 4096;        // bytes of a vector tile staged per TMA load (multiple of 16, <= 4096: slot word)
constexpr int VEC_DIRECT_MAX = 48;         // pieces shorter than this are copied by lanes, global -> global
constexpr int VEC_MAX_IN_BULK_MIX = 13;    // vector engines when both lists have work: the bulk engines keep >= 3/16 of the ring (>= 1 tile)
constexpr int COPY_MBAR_COUNT = COPY_MAX_ENGINES * COPY_SLOTS + COPY_WARPS * VEC_SLOTS;
constexpr int COPY_MBAR_BYTES = COPY_MBAR_COUNT * 8;
constexpr int COPY_KMAX_LONG = 2;          // max tiles per dynamic claim when segments average >= 8 tiles (measured: config 3)
constexpr int COPY_KMAX_LONG_VEC = 2;   // the same for the vector list (16 engines per CTA, 16 KiB tiles)
constexpr int COPY_KMAX_VEC = 8;           // max tiles per dynamic claim on the vector list
#define PAYLOAD_POL(p) , p
constexpr int COPY_CLAIM_DIV = 8;          // guided claims: K = remaining / (COPY_CLAIM_DIV * engines), clamped to [1, kmax]: an engine holds up to three
                                           // chunks (current, staged, claimed), so chunks shrink early (config 5: 2 -> 4: 163 -> 157 us with two engines)

// Optional side job for the warps that are not engines at the start of the kernel: `copies` copies of the int64
// array src[0..n) (negative values written as 0) to dst + c*n.  AllToAllvDynamic's recvAllSplitLengths (PAPER.md
// L439: every rank receives all split lengths) rides along with the payload instead of sitting in front of it.
struct SideJob {
    const long long* src;
    long long* dst;                        // null: no side job
    long long n;
    int copies;
};

struct CopyArgs {
    const SegDesc* desc;
    const int* colTiles[2];
    const int* colKiB;                     // per column: KiB of its bulk-list segments (metadata kernel)
    const int* coarse[2];                  // per list: tiles of column d before its descriptor 32*j, [d*nb + j] (metadata kernel)
    WorkCtl* ctl;
    int ncols;                             // destination columns of the descriptor table (= R)
    int colLen;                            // descriptor slots per column (R for the plain call, R*maxBlockLen for the dynamic one)
    int useCoarse;                         // 1: stage both coarse indexes in shared memory (2*ncols*nb ints)
    unsigned int ringBytes;                // shared-memory ring size, multiple of 128
    int kmax;                              // max tiles per dynamic claim on the bulk list (short-segment regime)
    int bulkEngines;                       // E = 1, 2 or 4 bulk engine warps per CTA; 0 = chosen on the device from the tile count
    ClassParams cls;
    SideJob side;
};

__host__ __device__ inline int coarse_blocks(int colLen) { return (colLen + 31) >> 5; }

// Warp-uniform cursor over one work list.  All lanes hold identical state except the descriptor
// WINDOWS: lane i caches descriptor q = qw + i of the destination-major table, and the next 32 are
// prefetched into a second register set, so stepping from one segment to the next non-empty one of
// this list is a ballot over registers instead of a chain of dependent L2 reads (config 5 has a new
// segment every ~2 tiles).
// Finding the segment that owns a freshly claimed tile index: binary search over the column bases,
// then over the column's COARSE index (tiles before every 32nd descriptor) -- both in shared memory --
// which names the one 32-descriptor block to load; the final position is a ballot over that window.
// Short-segment regime (config 5: a claim of 6 tiles is ~150 KB, the next one lies ~2000 descriptors
// ahead): the search and the window load of the NEXT chunk are issued while the current chunk is being
// copied (claims run two chunks ahead, windows one), so the engine never waits for metadata after
// start-up.  Long-segment regime (config 3): small in-order claims resolve inside the cached windows.
// Without a coarse index (table too large for shared memory) the block is found by a 128-ary search in L2.
// SM = true: the descriptor table lives in SHARED memory (single-launch path, fused_kernel.cuh).
// What all engines of one work list share, in shared memory (one copy per list and CTA): keeps ~25 registers per
// thread out of the cursor, whose cold fields were being spilled in the engines' hot loops.
struct CursorEnv {
    const SegDesc* desc;
    const int* colBase;                    // smem, ncols+1 entries, colBase[ncols] = total tiles
    const int* coarse;                     // smem, ncols*nb entries, or null
    unsigned int* counter;
    ClassParams cls;
    int ncols, colLen, nb, RR, total, nEngines, kmax, kmin, claimDiv;
    int staticK;                           // first chunk is assigned statically: [engineId*staticK, +staticK)
    int dynBase;                           // tiles >= dynBase are claimed dynamically
    bool longSegs, indexed, pipelined;
    bool rr;                               // chunks are dealt round-robin (engine e takes chunks e, e + nEngines, ...): no claim counter
};
__device__ __forceinline__ void cursor_env_init(CursorEnv* e, int L, const SegDesc* desc, const int* colBase, const int* coarse,
                                                unsigned int* counter, const ClassParams& cls, int ncols, int colLen, int nEngines,
                                                int kmax, int kmaxLong, int staticK, int claimDiv, bool rr) {
    e->desc = desc; e->colBase = colBase; e->coarse = coarse; e->counter = counter; e->cls = cls;
    e->ncols = ncols; e->colLen = colLen; e->nb = coarse_blocks(colLen); e->RR = ncols * colLen;
    e->total = colBase[ncols];
    e->nEngines = nEngines > 0 ? nEngines : 1;
    // long segments (>= 8 tiles each on average): claims resolve inside the cached window, so take
    // small chunks and keep all SMs in a tight moving window of HBM; short segments: amortise the
    // per-claim work over a few tiles and hide it behind the previous chunk.
    e->longSegs = (long long)e->total >= 8ll * e->RR;
    e->indexed = coarse != nullptr || e->nb == 1;
    e->pipelined = e->indexed && !e->longSegs;
    e->kmax = e->longSegs ? kmaxLong : kmax;
    e->staticK = staticK;
    e->rr = rr;
    e->claimDiv = claimDiv;
    // a short list (few tiles per engine) pays per claim, a long one for the imbalance of its last chunks
    e->kmin = e->total >= 32 * e->nEngines ? 1 : 2;          // (always 1: R = 64 x 10 KB +2 us, NEXT-1 +2 us)
    e->dynBase = staticK * e->nEngines;
    (void)L;
}

// Number of entries of the non-decreasing shared-memory array arr[0..n) that are <= key, found by the whole warp: 32-ary
// rounds (every lane probes the last entry of one block, one ballot per round) instead of a binary search's chain of
// dependent shared-memory loads -- 2 rounds for n <= 1024 where the binary search needed 10.  Warp-uniform result.
__device__ __forceinline__ int warp_count_le(const int* arr, int n, int key) {
    const int lane = lane_id();
    int base = 0, span = n;
    while (span > 32) {
        const int step = (span + 31) >> 5;
        const int i = (lane + 1) * step - 1;               // last entry of block `lane` (blocks that stick out do not count)
        const bool le = i < span && arr[base + i] <= key;
        const int m = __popc(__ballot_sync(0xffffffffu, le));
        base += m * step;
        span = min(step, n - base);
    }
    const bool le = lane < span && arr[base + lane] <= key;
    return base + __popc(__ballot_sync(0xffffffffu, le));
}

// K = clamp(avail / unit, lo, hi) without a division (hi is small: a handful of multiply-compares)
__device__ __forceinline__ int clamped_quotient(int avail, int unit, int lo, int hi) {
    if (hi > 8) return max(lo, min(hi, avail / unit));
    int k = lo;
    while (k < hi && (k + 1) * unit <= avail) ++k;
    return k;
}

template <int L, bool SM = false>
struct Cursor {
    const CursorEnv* env;                  // everything that is the same for all engines of the list (shared memory)
    int tileShift, engineId;
    int pendCur, pendK;                    // lane 0: a chunk claimed ahead of need (atomic in flight)
    int rrNext;                            // round-robin mode: this engine's next chunk
    int t, tEnd;                           // current tile, end of the claimed chunk
    int q, kInSeg, segTiles;               // current segment, tile within it, its tile count
    unsigned long long src, dst;
    long long bytes;
    int qw, qn;                            // bases of the current / prefetched window
    uint4 w0, w1, n0, n1;                  // this lane's descriptor in each window
    int cCur, cK, cQw, cEnd, cPrev, cTl;   // pipelined mode: the staged NEXT chunk and where it starts
    uint4 c0, c1;                          // its window (load in flight until adopt())
    bool first, exhausted, haveWindow, cHave, needPrefetch;

    __device__ __forceinline__ void load_desc(int qq, uint4& a, uint4& b) const {
        if (qq < env->RR) {
            const uint4* p = reinterpret_cast<const uint4*>(env->desc + qq);
            if constexpr (SM) { a = p[0]; b = p[1]; } else { a = ld_stream(p); b = ld_stream(p + 1); }   // coherent: the kernel before us wrote them (PDL)
        } else {
            a = make_uint4(0, 0, 0, 0); b = make_uint4(0, 0, 0, 0);
        }
    }
    __device__ __forceinline__ int my_tiles() const {
        return seg_tiles(L, ((unsigned long long)w0.y << 32) | w0.x, ((unsigned long long)w0.w << 32) | w0.z,
                         (long long)(((unsigned long long)w1.y << 32) | w1.x), env->cls);
    }
    __device__ __forceinline__ void take(int fromLane) {    // adopt the descriptor held by lane `fromLane`
        const unsigned int sx = __shfl_sync(0xffffffffu, w0.x, fromLane), sy = __shfl_sync(0xffffffffu, w0.y, fromLane);
        const unsigned int dx = __shfl_sync(0xffffffffu, w0.z, fromLane), dy = __shfl_sync(0xffffffffu, w0.w, fromLane);
        const unsigned int bx = __shfl_sync(0xffffffffu, w1.x, fromLane), by = __shfl_sync(0xffffffffu, w1.y, fromLane);
        src = ((unsigned long long)sy << 32) | sx;
        dst = ((unsigned long long)dy << 32) | dx;
        bytes = (long long)(((unsigned long long)by << 32) | bx);
        segTiles = __shfl_sync(0xffffffffu, my_tiles(), fromLane);
        q = qw + fromLane;
    }

    // env->staticK tiles per engine are assigned statically ([engineId*env->staticK, +env->staticK): no atomic on the
    // start-up path); tiles >= env->staticK*env->nEngines are claimed dynamically, IN ORDER, in guided chunks.
    // Measured on B200: the in-order dynamic claim keeps all SMs inside one moving window of HBM and is
    // ~7 % faster than contiguous static ranges (148 far-apart streams), so only the FIRST chunk of each
    // engine is static (chunk e to engine e, which is also what in-order claims would hand out).
    __device__ __forceinline__ void init(const CursorEnv* env_, int engineId_) {
        env = env_;
        engineId = engineId_;
        tileShift = env_->cls.tileShift[L];
        pendCur = env->total; pendK = 0;        // reads as "drained" unless a claim is issued
        rrNext = env->dynBase + engineId * env->staticK;
        t = tEnd = 0; q = 0; kInSeg = segTiles = 0; src = dst = 0; bytes = 0;
        qw = qn = 0; w0 = w1 = n0 = n1 = c0 = c1 = make_uint4(0, 0, 0, 0);
        cCur = cK = cQw = cEnd = cPrev = cTl = 0;
        first = true;
        haveWindow = false;
        cHave = needPrefetch = false;
        exhausted = (env->total == 0);
        if (exhausted) return;
        if (!env->pipelined) {
            if (env->total > env->dynBase) claim_issue(env->dynBase);
        } else if (env->staticK > 0) {
            const int c = engineId * env->staticK;
            if (c < env->total) stage_next(c, env->staticK);             // else: nothing for this engine (then env->total <= env->dynBase)
            if (env->total > env->dynBase) claim_issue(env->dynBase);
        } else {
            claim_issue(env->dynBase);
            prefetch_next();                                   // waits for the atomic once, at start-up
        }
    }

    // Lane 0 issues the atomic for a later dynamic chunk; the result is consumed one chunk (env->pipelined:
    // two chunks) later, so its L2 round trip overlaps the copying.
    __device__ __forceinline__ void claim_issue(int counterHint) {
        if (env->rr) {                          // all lanes alike; no atomic
            pendK = env->staticK; pendCur = rrNext; rrNext += env->staticK * env->nEngines;
            return;
        }
        if (lane_id() == 0) {
            const int rem = env->total - min(env->total, counterHint);
            pendK = clamped_quotient(rem, env->claimDiv * env->nEngines, env->kmin, env->kmax);
            pendCur = env->dynBase + (int)atomicAdd(env->counter, (unsigned int)pendK);
        }
    }

    // Shared-memory search: column d that owns global tile tt, tile index tl inside the column, the
    // 32-descriptor block j of the column that holds it and the tiles of the column before that block.
    __device__ __forceinline__ void find_block(int tt, int& d, int& tl, int& j, int& prev) const {
        const int* cb = env->colBase;
        d = warp_count_le(cb + 1, env->ncols, tt);          // cb[d] <= tt < cb[d+1]  (cb[ncols] = total > tt)
        tl = tt - cb[d];
        j = 0; prev = 0;
        const int nb = env->nb;
        if (nb > 1) {
            const int* cr = env->coarse + d * nb;            // cr[0] = 0, non-decreasing
            j = warp_count_le(cr + 1, nb - 1, tl);           // cr[j] <= tl < cr[j+1]  (cr[nb] = +inf)
            prev = cr[j];
        }
    }
    // The current window holds the segment that owns tile tl of its column (prev tiles lie before the
    // window, colEnd = first descriptor index of the next column): select it.
    __device__ __forceinline__ void position(int tl, int prev, int colEnd) {
        const int pf = L == LIST_BULK ? (int)w1.z : (int)w1.w;
        const int m = __popc(__ballot_sync(0xffffffffu, qw + lane_id() < colEnd && pf <= tl));
        const int before = __shfl_sync(0xffffffffu, pf, m > 0 ? m - 1 : 0);
        take(m);
        kInSeg = tl - (m > 0 ? before : prev);
    }

    // Find the segment that owns global tile index tt (0 <= tt < env->total) and (re)load the windows there.
    __device__ __forceinline__ void locate(int tt) {
        const int lane = lane_id();
        if (env->indexed) {
            int d, tl, j, prev;
            find_block(tt, d, tl, j, prev);
            qw = d * env->colLen + 32 * j;
            load_desc(qw + lane, w0, w1);
            qn = qw + 32;
            load_desc(qn + lane, n0, n1);
            position(tl, prev, (d + 1) * env->colLen);
            return;
        }
        const int d = warp_count_le(env->colBase + 1, env->ncols, tt);
        const int tl = tt - env->colBase[d];
        const SegDesc* col = env->desc + (size_t)d * env->colLen;
        int s0 = 0, n = env->colLen;                 // smallest s with col[s].pfx[L] > tl lies in [s0, s0+n)
        while (n >= 32) {                  // 128-ary rounds: every lane probes 4 block ends per L2 round trip; ends with at most
                                           // 31 candidates, so that they AND the predecessor slot fit in one 32-descriptor window
            const int step = (n + 127) >> 7;
            int cnt = 0;
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const int b = lane * 4 + u;
                const int idx = s0 + min((b + 1) * step, n) - 1;
                const int pv = col[idx].pfx[L];
                cnt += (pv <= tl) ? 1 : 0;
            }
            int m = cnt;                   // blocks entirely <= tl (monotone, so a plain count)
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) m += __shfl_xor_sync(0xffffffffu, m, o);
            s0 += m * step;
            n = min(step, n - m * step);
        }
        // last round doubles as the window load; the window starts one descriptor early so that the
        // predecessor's prefix (needed for the tile index inside the segment) comes with it
        const int sb = s0 > 0 ? s0 - 1 : 0;
        qw = d * env->colLen + sb;
        load_desc(qw + lane, w0, w1);
        qn = qw + 32;
        load_desc(qn + lane, n0, n1);
        position(tl, 0, (d + 1) * env->colLen);
    }

    // ---- env->pipelined mode ------------------------------------------------------------------------
    __device__ __forceinline__ void stage_next(int cur, int k) {   // chunk [cur, cur+k): find its block, start the window load
        int d, j;
        find_block(cur, d, cTl, j, cPrev);
        cCur = cur; cK = k;
        cQw = d * env->colLen + 32 * j;
        cEnd = (d + 1) * env->colLen;
        load_desc(cQw + lane_id(), c0, c1);
        cHave = true;
    }
    __device__ __forceinline__ void prefetch_next() {      // consume the pending claim, stage it, claim one more
        needPrefetch = false;
        const int pc = __shfl_sync(0xffffffffu, pendCur, 0);
        const int pk = __shfl_sync(0xffffffffu, pendK, 0);
        if (pc >= env->total || pc < 0) { cHave = false; return; }
        stage_next(pc, pk);
        claim_issue(pc + pk);
    }
    __device__ __forceinline__ void adopt() {              // the staged chunk becomes the current one
        t = cCur;
        tEnd = min(cCur + cK, env->total);
        qw = cQw; w0 = c0; w1 = c1;
        qn = qw + 32;
        load_desc(qn + lane_id(), n0, n1);
        position(cTl, cPrev, cEnd);
        haveWindow = true;
        cHave = false;
        needPrefetch = true;
    }

    // Step to the next segment of this list (t stays inside the claimed chunk, so one exists).
    __device__ __forceinline__ void advance_segment() {
        int cl = q - qw;                   // lane that holds the current segment
        while (true) {
            const unsigned int later = cl >= 31 ? 0u : (0xffffffffu << (cl + 1));
            const unsigned int mask = __ballot_sync(0xffffffffu, my_tiles() > 0) & later;
            if (mask) { take(__ffs(mask) - 1); break; }
            qw = qn; w0 = n0; w1 = n1;     // slide: prefetched window becomes current, prefetch the next
            qn = qw + 32;
            load_desc(qn + lane_id(), n0, n1);
            cl = -1;
            if (qw >= env->RR) { exhausted = true; break; }      // cannot happen while t < env->total
        }
        kInSeg = 0;
    }

    // Jump forward by `delta` tiles of this list using only the cached windows (current + prefetched):
    // no memory round trip when the target lies within ~64 descriptors, which is the common case for
    // in-order claims over long segments.  Returns false if the target is farther (caller searches).
    __device__ __forceinline__ bool advance_by(int delta) {
        const int rem = segTiles - kInSeg;
        if (delta < rem) { kInSeg += delta; return true; }
        delta -= rem;
        int cl = q - qw;
        for (int pass = 0; pass < 2; ++pass) {     // current window, then the already-prefetched one
            const int mt = (lane_id() > cl) ? my_tiles() : 0;
            const int incl = warp_incl_scan(mt);
            const int tot = __shfl_sync(0xffffffffu, incl, 31);
            if (delta < tot) {
                const int l = __ffs(__ballot_sync(0xffffffffu, incl > delta)) - 1;
                const int before = __shfl_sync(0xffffffffu, incl - mt, l);
                take(l);
                kInSeg = delta - before;
                return true;
            }
            delta -= tot;
            qw = qn; w0 = n0; w1 = n1;     // slide to the prefetched window, prefetch the next
            qn = qw + 32;
            load_desc(qn + lane_id(), n0, n1);
            cl = -1;
            if (qw >= env->RR) return false;
        }
        return false;
    }

    // Make (t, segment) valid; false when the list is drained.
    __device__ __forceinline__ bool ensure() {
        if (exhausted) return false;
        if (t < tEnd) {
            if (needPrefetch) prefetch_next();     // (env->pipelined) after the chunk's first tile is on its way
            if (kInSeg >= segTiles) advance_segment();
            return !exhausted;
        }
        if (env->pipelined) {
            if (needPrefetch) prefetch_next();
            if (!cHave) { exhausted = true; return false; }
            adopt();
            return true;
        }
        int cur, k;
        if (first && env->staticK > 0) {        // static share: no atomic on the start-up path
            first = false;
            cur = engineId * env->staticK;
            k = env->staticK;
            if (cur >= env->total) { exhausted = true; return false; }
        } else {
            first = false;
            cur = __shfl_sync(0xffffffffu, pendCur, 0);
            k = __shfl_sync(0xffffffffu, pendK, 0);
            if (cur >= env->total || cur < 0) { exhausted = true; return false; }
            claim_issue(cur + k);
        }
        const bool near = env->longSegs && haveWindow && cur >= t && advance_by(cur - t);
        t = cur;
        tEnd = min(cur + k, env->total);
        if (!near) locate(t);
        haveWindow = true;
        return true;
    }

    __device__ __forceinline__ long long tile_off() const { return (long long)kInSeg << tileShift; }
    __device__ __forceinline__ void next() { ++t; ++kInSeg; }
};

// ---- vector list: shared memory -> global with any alignment --------------------------------------------------
// Destination vector j (16-byte aligned) = bytes [sh + 16 j, sh + 16 j + 16) of the aligned shared-memory image:
// the two aligned 16-byte words that straddle it, joined with funnel shifts (sh = 4*WSEL + bsh/8).  WSEL is a template
// parameter so that the word selection is static; the (warp-uniform) dispatch happens once per piece.
template <int WSEL>
__device__ __forceinline__ uint4 shift_join(const uint4& a, const uint4& b, const int bsh) {
    const unsigned int w[8] = {a.x, a.y, a.z, a.w, b.x, b.y, b.z, b.w};
    return make_uint4(__funnelshift_r(w[WSEL], w[WSEL + 1], bsh), __funnelshift_r(w[WSEL + 1], w[WSEL + 2], bsh),
                      __funnelshift_r(w[WSEL + 2], w[WSEL + 3], bsh), __funnelshift_r(w[WSEL + 3], w[WSEL + 4], bsh));
}
// The drain: one warp writes a landed piece to global memory at any alignment.  The body is realigned IN PLACE in shared memory (vector i of the destination-aligned
// image overwrites slot i of the source-aligned one: every batch reads its 32 or 64 slots + the one after them into
// registers before any lane writes), so that one cp.async.bulk shared -> global can store it; returns the shared-memory
// address and the byte count of the body for the elected lane to issue.  Head / tail bytes (< 16 each, only at the ends
// of a tile) are stored by lanes first: the head shares a 16-byte word with body slot 0.
template <int WSEL>
__device__ __forceinline__ void realign_body(uint4* sv, const unsigned int nvec, const int bsh, const unsigned int lane) {
    unsigned int i0 = 0;
    for (; i0 + 64 <= nvec; i0 += 64) {
        const unsigned int i = i0 + lane;
        const uint4 a0 = sv[i], b0 = sv[i + 1], a1 = sv[i + 32], b1 = sv[i + 33];
        __syncwarp();
        sv[i] = shift_join<WSEL>(a0, b0, bsh);
        sv[i + 32] = shift_join<WSEL>(a1, b1, bsh);
        __syncwarp();
    }
    for (; i0 < nvec; i0 += 32) {
        const unsigned int i = i0 + lane;
        uint4 a = make_uint4(0, 0, 0, 0), b = a;
        if (i < nvec) { a = sv[i]; b = sv[i + 1]; }
        __syncwarp();
        if (i < nvec) sv[i] = shift_join<WSEL>(a, b, bsh);
        __syncwarp();
    }
}
__device__ __forceinline__ void warp_drain_realign(unsigned char* dst, unsigned char* sm, const unsigned int ms, const unsigned int len,
                                                   unsigned char*& bodyDst, uint32_t& bodySmem, unsigned int& bodyBytes) {
    const unsigned int lane = (unsigned int)lane_id();
    unsigned int hb = (16u - (unsigned int)((unsigned long long)dst & 15ull)) & 15u;
    if (hb > len) hb = len;
    const unsigned int pos = ms + hb;                      // shared-memory offset of the first body byte
    const unsigned int nvec = (len - hb) >> 4;
    const unsigned int done = hb + (nvec << 4);
    if (lane < hb) dst[lane] = sm[ms + lane];
    if (lane < len - done) dst[done + lane] = sm[ms + done + lane];
    const unsigned int sh = pos & 15u;
    uint4* sv = reinterpret_cast<uint4*>(sm) + (pos >> 4);
    if (sh != 0 && nvec) {
        __syncwarp();                                      // the head bytes have been read
        const int bsh = (int)(sh & 3u) * 8;
        switch (sh >> 2) {                                 // warp-uniform, once per piece
        case 0:  realign_body<0>(sv, nvec, bsh, lane); break;
        case 1:  realign_body<1>(sv, nvec, bsh, lane); break;
        case 2:  realign_body<2>(sv, nvec, bsh, lane); break;
        default: realign_body<3>(sv, nvec, bsh, lane); break;
        }
        fence_proxy_async_smem();                          // this lane's generic writes -> visible to the TMA store
    }
    __syncwarp();
    bodyDst = dst + hb;
    bodySmem = smem_u32(sv);
    bodyBytes = nvec << 4;
}

// ================= bulk engine: byte-granular TMA ring driven by one elected lane (one warp) ========
// The ring is a circular BYTE buffer (not fixed-size stages): every tile takes exactly
// align128(len) bytes, so short tiles (config 5: 10-28 KiB) keep as many bytes in flight as
// long ones.  Up to COPY_SLOTS tiles are outstanding; slot j's bookkeeping (destination,
// length, smem offset, virtual start) lives in the registers of lane j.
// A store's ring bytes are reclaimed with cp.async.bulk.wait_group.read as soon as the NEXT store has been issued
// (keeping up to 8 stores unreclaimed was measured 10 % slower on config 5: the ring is for LOADS in flight).
template <bool SM>
__device__ __forceinline__ void bulk_engine(Cursor<LIST_BULK, SM>& cur, unsigned char* ring, unsigned long long* mbar,
                                            const unsigned int ringBytes) {
    const int lane = lane_id();
    const unsigned int tileBytes = 1u << cur.tileShift;
    const uint32_t ring0 = smem_u32(ring);
    const unsigned long long pol = l2_policy_stream(); (void)pol;
    unsigned long long mDst = 0;          // slot registers (lane j <-> slot j)
    unsigned int mLen = 0, mOff = 0, mV = 0;
    unsigned int vHead = 0, phys = 0;     // virtual (mod 2^32) and physical allocation offsets
    int iLoad = 0, iStore = 0, freed = 0;  // stores [0, freed) have finished reading their smem; freed <= iStore <= iLoad
    bool more = cur.ensure();
    while (true) {
        // fill: issue loads while a slot and enough ring bytes are free
        while (more) {
            const long long off = cur.tile_off();
            const long long rest = cur.bytes - off;
            const unsigned int len = rest < (long long)tileBytes ? (unsigned int)rest : tileBytes;
            const unsigned int len16 = len & ~15u;
            const unsigned char* srcp = reinterpret_cast<const unsigned char*>(cur.src + off);
            unsigned char* dstp = reinterpret_cast<unsigned char*>(cur.dst + off);
            if (len16) {
                const unsigned int pad = phys + len16 > ringBytes ? ringBytes - phys : 0u;   // wrap
                const unsigned int vTail = freed < iLoad ? __shfl_sync(0xffffffffu, mV, freed % COPY_SLOTS) : vHead;
                if (iLoad - freed >= COPY_SLOTS || vHead + pad + len16 - vTail > ringBytes) break;   // store a landed tile first
                const unsigned int vStart = vHead + pad;
                const unsigned int po = pad ? 0u : phys;
                const int slot = iLoad % COPY_SLOTS;
                if (lane == slot) { mDst = (unsigned long long)dstp; mLen = len16; mOff = po; mV = vStart; }
                if (lane == 0) {
                    const uint32_t bar = smem_u32(&mbar[slot]);
                    mbar_expect_tx(bar, len16);
                    bulk_g2s(ring0 + po, srcp, len16, bar PAYLOAD_POL(pol));
                }
                const unsigned int adv = (len16 + 127u) & ~127u;
                vHead = vStart + adv;
                phys = po + adv;
                if (phys >= ringBytes) phys = 0;
                ++iLoad;
            }
            const int tail = (int)(len & 15u);        // only the last tile of a ragged segment
            if (lane < tail) dstp[len16 + lane] = srcp[len16 + lane];
            cur.next();
            more = cur.ensure();
        }
        if (iStore == iLoad) {
            if (!more) break;
            // nothing in flight and nothing left to reclaim, yet the next tile does not fit behind the
            // allocation point: restart the ring at offset 0
            if (lane == 0) bulk_wait_read<0>();
            freed = iStore;
            phys = 0;
            continue;
        }
        const int slot = iStore % COPY_SLOTS;
        mbar_wait(smem_u32(&mbar[slot]), (uint32_t)((iStore / COPY_SLOTS) & 1));
        const unsigned int dlo = __shfl_sync(0xffffffffu, (unsigned int)mDst, slot);
        const unsigned int dhi = __shfl_sync(0xffffffffu, (unsigned int)(mDst >> 32), slot);
        const unsigned int slen = __shfl_sync(0xffffffffu, mLen, slot);
        const unsigned int soff = __shfl_sync(0xffffffffu, mOff, slot);
        if (lane == 0) {
            bulk_s2g(reinterpret_cast<void*>(((unsigned long long)dhi << 32) | dlo), ring0 + soff, slen PAYLOAD_POL(pol));
            bulk_commit();
        }
        ++iStore;
        if (iStore - freed > 1) {                                 // at most ONE store keeps its ring bytes: reclaim the older one
            if (lane == 0) bulk_wait_read<1>();
            ++freed;
        }
        __syncwarp();
    }
    if (lane == 0) bulk_wait_all<0>();
}

// ================= vector engine: one warp, its own share of the ring, TMA loads + warp stores ================
// The engine walks its tiles in pieces of at most VEC_SUB_BYTES; the first piece of a tile ends where the
// DESTINATION reaches a 16-byte boundary, so every later piece of the tile starts destination-aligned and only the
// tile's ends need byte stores.  For a piece [s, s+len) of the source, the TMA loads the aligned span
// [s & ~15, align16(s + len)) -- cp.async.bulk needs 16-byte aligned addresses and sizes, not aligned SEGMENTS;
// the up-to-15 bytes read on either side share a 16-byte word with valid data, so they lie inside the caller's
// allocation.  Up to VEC_SLOTS pieces are in flight per engine (bookkeeping in lanes 0..15, as in the bulk engine),
// also across tile and segment boundaries.  A landed piece is realigned by the whole warp and stored by the TMA
// (warp_drain_realign); its ring bytes are released once that store has read them (one store may be outstanding), as in
// the bulk engine.
// The engine runs on either work list (L): when the bulk list holds only a small part of a mostly unaligned call,
// the vector engines sweep it up as well (plan_ring: bulkByVec) instead of idling warps as bulk engines.
// Measured (R = 16, 360 MB each way, odd bf16 counts): the loop is instruction-issue bound, so per-piece work is kept
// minimal -- tile state in registers, one packed slot word, word selection of the funnel shift resolved per piece.
template <int L, bool SM>
__device__ __forceinline__ void vector_engine(Cursor<L, SM>& cur, unsigned char* ring, unsigned long long* mbar,
                                              const unsigned int ringBytes, int& pieceSeq) {
    const int lane = lane_id();
    const unsigned int tileBytes = 1u << cur.tileShift;
    const uint32_t ring0 = smem_u32(ring);
    const unsigned long long pol = l2_policy_stream(); (void)pol;
    unsigned long long mDst = 0;          // slot registers (lane j <-> slot j, j < VEC_SLOTS)
    unsigned int mPack = 0, mAlloc = 0;   // ring offset >> 7 | len << 11 | source misalignment << 24;  ring bytes to release
    unsigned int used = 0, phys = 0;      // ring bytes held by pieces in flight (incl. wrap padding); allocation offset
    int freed = pieceSeq; (void)freed;    // (TMA-store drain) pieces [.., freed) have released their ring bytes: freed <= iStore <= iLoad
    int iLoad = pieceSeq, iStore = pieceSeq;   // piece numbers continue across the engine's runs: slot = number mod VEC_SLOTS, and the
                                               // slot's mbarrier has completed number / VEC_SLOTS phases before this piece
    unsigned long long tS = 0, tD = 0;    // the rest of the current tile
    unsigned int tRem = 0;
    bool more = cur.ensure();
    while (true) {
        while (more) {
            if (tRem == 0) {
                const long long toff = cur.tile_off();
                const long long rest = cur.bytes - toff;
                tRem = rest < (long long)tileBytes ? (unsigned int)rest : tileBytes;
                tS = cur.src + (unsigned long long)toff;
                tD = cur.dst + (unsigned long long)toff;
            }
            unsigned int len = VEC_SUB_BYTES - ((unsigned int)tD & 15u);
            if (len > tRem) len = tRem;
            if (len < VEC_DIRECT_MAX) {                            // tiny piece: lanes copy it directly
                const unsigned char* sp = reinterpret_cast<const unsigned char*>(tS);
                unsigned char* dp = reinterpret_cast<unsigned char*>(tD);
                for (unsigned int b = lane; b < len; b += 32) dp[b] = sp[b];
            } else {
                const unsigned int ms = (unsigned int)tS & 15u;
                const unsigned int ld = (ms + len + 15u) & ~15u;
                const unsigned int adv = (ld + 127u) & ~127u;
                const unsigned int pad = phys + ld > ringBytes ? ringBytes - phys : 0u;   // wrap
                if (iLoad - freed >= VEC_SLOTS || used + pad + adv > ringBytes) break;    // drain a landed piece first
                const unsigned int po = pad ? 0u : phys;
                const int slot = iLoad & (VEC_SLOTS - 1);
                if (lane == slot) { mDst = tD; mPack = (po >> 7) | (len << 11) | (ms << 24); mAlloc = pad + adv; }
                if (lane == 0) {
                    const uint32_t bar = smem_u32(&mbar[slot]);
                    mbar_expect_tx(bar, ld);
                    bulk_g2s(ring0 + po, reinterpret_cast<const void*>(tS - ms), ld, bar PAYLOAD_POL(pol));
                }
                used += pad + adv;
                phys = po + adv;
                if (phys >= ringBytes) phys = 0;
                ++iLoad;
            }
            tS += len; tD += len; tRem -= len;
            if (tRem == 0) {
                cur.next();
                more = cur.ensure();
            }
        }
        if (iStore == iLoad) {
            if (!more) break;
            if (lane == 0) { bulk_wait_read<0>(); fence_proxy_async_smem(); }   // the stores still reading their ring bytes
            __syncwarp();
            freed = iStore; used = 0;
            phys = 0;                      // nothing in flight: restart the ring at offset 0 (the piece did not fit behind phys)
            continue;
        }
        const int slot = iStore & (VEC_SLOTS - 1);
        mbar_wait(smem_u32(&mbar[slot]), (uint32_t)((iStore / VEC_SLOTS) & 1));
        const unsigned int dlo = __shfl_sync(0xffffffffu, (unsigned int)mDst, slot);
        const unsigned int dhi = __shfl_sync(0xffffffffu, (unsigned int)(mDst >> 32), slot);
        const unsigned int pk = __shfl_sync(0xffffffffu, mPack, slot);
        {
            unsigned char* bDst; uint32_t bSm; unsigned int bBytes;
            warp_drain_realign(reinterpret_cast<unsigned char*>(((unsigned long long)dhi << 32) | dlo), ring + ((pk & 0x7ffu) << 7),
                               pk >> 24, (pk >> 11) & 0x1fffu, bDst, bSm, bBytes);
            if (lane == 0) {
                if (bBytes) bulk_s2g(bDst, bSm, bBytes PAYLOAD_POL(pol));
                bulk_commit();                             // one group per piece (possibly empty), so that groups count pieces
            }
            ++iStore;
            if (iStore - freed > 1) {                      // at most ONE store keeps its ring bytes: release the older piece
                if (lane == 0) { bulk_wait_read<1>(); fence_proxy_async_smem(); }   // (lanes' head / tail byte reads precede the syncwarp of the drain)
                __syncwarp();
                used -= __shfl_sync(0xffffffffu, mAlloc, freed & (VEC_SLOTS - 1));
                ++freed;
            }
        }
    }
    if (lane == 0) bulk_wait_all<0>();     // shared memory stays valid until every store has read it (and the run's writes are done)
    __syncwarp();
    pieceSeq = iLoad;
}

// The claim counters reset themselves: every CTA checks out once all its engines are drained (each
// engine has consumed every atomic it issued by then), and the last one out zeroes the counters, so the
// same work list can be executed again (ncclx_alltoallv_execute_dev) and the single-launch path needs
// no preceding kernel to clear them.  `used` must be grid-uniform.
__device__ __forceinline__ void workctl_checkout(WorkCtl* ctl, bool used) {
    __syncthreads();
    if (threadIdx.x == 0 && used) {
        __threadfence();
        if (atomicAdd(&ctl->done, 1u) == gridDim.x - 1) {
            ctl->next[0] = 0u; ctl->next[1] = 0u; ctl->done = 0u;
            __threadfence();
        }
    }
}

// How a CTA's 16 warps and its ring are divided between the two work lists -- grid-uniform: depends only on the
// lists' tile totals.
//   * no vector tiles: E bulk engines share the whole ring.  E = 4 for a call of few tiles per SM (bound by the
//     per-tile latency of one elected lane -- measured: R = 64 with one 10 KB row per pair takes 40 us with one
//     engine and 27 us with four), 2 up to 96 tiles per SM, else 1 (HBM-bound: one deep ring is slightly better,
//     config 3: -0.7 % with two engines) -- but never fewer than the average tile size asks for (short tiles);
//   * no bulk tiles, or the bulk list holds less than ~1/9 of the bytes: all 16 warps are vector engines with 1/16 of
//     the ring each; they take the vector list first and then sweep up the bulk list (bulkByVec);
//   * otherwise: the vector engines get one 1/16 unit each, as many as their share of the bytes (1..13), the bulk
//     engines the rest (>= 3/16 of the ring; the host sized the bulk tile to fit that).
struct RingPlan {
    int E, NV;                             // bulk engines = warps [0, E), vector engines = warps [E, E + NV)
    bool bulkByVec;                        // the vector engines also process the bulk list (E == 0 although it has tiles)
    unsigned int bulkShare, vecShare;      // ring bytes per bulk / per vector engine (multiples of 128)
    unsigned int vecBase;                  // ring offset of vector engine 0's share
};
__device__ __forceinline__ RingPlan plan_ring(int requestedE, int bulkTiles, int vecTiles, int grid, unsigned int ringBytes,
                                              int bulkShift, int vecShift, long long bulkKiB) {
    RingPlan p;
    const unsigned int unit = (ringBytes / COPY_WARPS) & ~127u;
    unsigned int bulkBytes = ringBytes;
    p.NV = 0;
    p.bulkByVec = false;
    if (vecTiles > 0) {
        const long long wb = (long long)bulkTiles << bulkShift, wv = (long long)vecTiles << vecShift;
        if (wb * 8 <= wv) { p.NV = COPY_WARPS; bulkBytes = 0; p.bulkByVec = bulkTiles > 0; }
        else {
            p.NV = (int)((wv * COPY_WARPS + (wb + wv) / 2) / (wb + wv));
            p.NV = max(1, min(VEC_MAX_IN_BULK_MIX, p.NV));
            bulkBytes = ringBytes - (unsigned int)p.NV * unit;
        }
    }
    int E = 0;
    if (bulkTiles > 0 && !p.bulkByVec) {
        E = requestedE;
        if (E == 0) {
            E = bulkTiles <= 48 * grid ? 4 : (bulkTiles <= 96 * grid ? 2 : 1);
            // one engine turns a tile around in ~1.2 us (measured: R = 256 / 512 with one 14 KB row per pair, 1 vs 4
            // engines: 173 -> 114 us, 587 -> 393 us), an SM's share of HBM is ~23 GB/s each way: E x average tile >= ~30 KB
            if (bulkKiB >= 0) {                            // average tile = bulkKiB KiB / bulkTiles, compared without dividing
                const int need = bulkKiB >= 30ll * bulkTiles ? 1 : (bulkKiB >= 15ll * bulkTiles ? 2 : 4);
                E = max(E, need);
            }
        }
        while (E > 1 && (unsigned long long)E * (((1u << bulkShift) + 127u) & ~127u) > bulkBytes) E >>= 1;    // a tile must fit in one share
        if (E + p.NV > COPY_WARPS) E = COPY_WARPS - p.NV;
    }
    p.E = E;
    p.bulkShare = (E == 0 ? 0u : E == 1 ? bulkBytes : E == 2 ? bulkBytes >> 1 : E == 4 ? bulkBytes >> 2 : bulkBytes / (unsigned int)E) & ~127u;
    p.vecShare = unit;
    p.vecBase = bulkBytes & ~127u;
    return p;
}

// First chunk of every engine is static (chunk e to engine e; see Cursor::init).
__device__ __forceinline__ int static_first_chunk(int total, int nEngines, int kmax, int kmaxLong, int RR) {
    if (nEngines <= 0) return 0;
    const int km = (long long)total >= 8ll * RR ? kmaxLong : kmax;
    return clamped_quotient(total, 4 * nEngines, 1, km);
}

// A vector engine warp's whole job, as ONE out-of-line function: the vector path is ~200 KB of SASS (two lists x four
// word selections of the funnel shift, fully inlined cursors) that an aligned call never executes.  Kept out of line, the
// prologue -> plan -> bulk engine path is one compact ~80 KB stretch of code; with everything inlined, builds differed by
// 1.7-2 us per call on the small-message shapes depending on where the compiler happened to place that path (measured:
// identical sources +- the vector code, config 5 155.1 vs 156.9 us, R = 64 x 10 KB 26.0 vs 27.4 us).  The cursors are
// constructed in here so that they live in registers.
template <bool SM>
__device__ __noinline__ void vector_role(const CursorEnv* envs, int engineId, unsigned char* myRing, unsigned long long* myBar,
                                         unsigned int share, bool bulkToo) {
    int pieceSeq = 0;
    {
        Cursor<LIST_VEC, SM> cur;
        cur.init(&envs[LIST_VEC], engineId);
        vector_engine<LIST_VEC, SM>(cur, myRing, myBar, share, pieceSeq);
    }
    if (bulkToo) {
        Cursor<LIST_BULK, SM> cur;
        cur.init(&envs[LIST_BULK], engineId);
        vector_engine<LIST_BULK, SM>(cur, myRing, myBar, share, pieceSeq);
    }
}

// Step a4 for one CTA: split warps and ring (plan_ring), run the engines.  Returns whether any dynamic claim counter
// may have been used (grid-uniform; for workctl_checkout).  fusedStatic > 0: the single-launch path's static share.
template <bool SM>
__device__ __forceinline__ bool run_copy_engines(const SegDesc* desc, int* const colBase[2], int* const coarse[2], WorkCtl* ctl,
                                                 const ClassParams& cls, int ncols, int colLen, int requestedE, int kmax,
                                                 int fusedStatic, long long bulkKiB, int claimDiv, unsigned char* smem, unsigned long long* mbar,
                                                 unsigned int ringBytes) {
    __shared__ CursorEnv envs[2];
    const int warp = threadIdx.x >> 5;
    const int totB = colBase[LIST_BULK][ncols], totV = colBase[LIST_VEC][ncols];
    const RingPlan rp = plan_ring(requestedE, totB, totV, (int)gridDim.x, ringBytes, cls.tileShift[LIST_BULK], cls.tileShift[LIST_VEC], bulkKiB);
    const int nV = (int)gridDim.x * rp.NV;
    const int nB = rp.bulkByVec ? nV : (int)gridDim.x * rp.E;
    const int RR = ncols * colLen;
    // Short lists (at most RR_TILES_PER_ENGINE tiles per engine: the small-message regime, a call of ~10 us) are dealt ROUND-ROBIN,
    // chunk c to engine c mod nEngines: same HBM order as in-order claims, but no atomic round trip sits between an
    // engine and its next tile.  Measured (graph replay p50): R = 64 x one 10 KB row per pair 28.1 -> 26.0 us, R = 128 x
    // 14 KB for 28 % of pairs 31.6 -> 30.1 us, and no longer build-dependent (with claims the same sources landed on
    // either value depending on instruction scheduling).  Longer lists need the claims' balance by TIME: round-robin
    // there costs config 5 +17 us, config 3 +14 % (measured with 64 / unlimited).
    constexpr int RR_TILES_PER_ENGINE = 16;
    const bool rrB = fusedStatic == 0 && nB > 0 && (long long)totB <= (long long)RR_TILES_PER_ENGINE * nB;
    const bool rrV = fusedStatic == 0 && nV > 0 && (long long)totV <= (long long)RR_TILES_PER_ENGINE * nV;
    const int stB = fusedStatic > 0 ? fusedStatic : rrB ? clamped_quotient(totB, 32 * nB, 1, (long long)totB >= 8ll * RR ? COPY_KMAX_LONG : min(kmax, 8))
                                                        : static_first_chunk(totB, nB, kmax, COPY_KMAX_LONG, RR);
    const int stV = fusedStatic > 0 ? fusedStatic : rrV ? clamped_quotient(totV, 32 * nV, 1, (long long)totV >= 8ll * RR ? COPY_KMAX_LONG_VEC : COPY_KMAX_VEC)
                                                        : static_first_chunk(totV, nV, COPY_KMAX_VEC, COPY_KMAX_LONG_VEC, RR);
    if (threadIdx.x == 0)
        cursor_env_init(&envs[LIST_BULK], LIST_BULK, desc, colBase[LIST_BULK], coarse[LIST_BULK], &ctl->next[LIST_BULK], cls, ncols, colLen,
                        nB, kmax, COPY_KMAX_LONG, stB, claimDiv, rrB);
    if (threadIdx.x == 32)
        cursor_env_init(&envs[LIST_VEC], LIST_VEC, desc, colBase[LIST_VEC], coarse[LIST_VEC], &ctl->next[LIST_VEC], cls, ncols, colLen,
                        nV, COPY_KMAX_VEC, COPY_KMAX_LONG_VEC, stV, claimDiv, rrV);
    __syncthreads();
    if (warp < rp.E) {
        Cursor<LIST_BULK, SM> cur;
        cur.init(&envs[LIST_BULK], (int)blockIdx.x * rp.E + warp);
        bulk_engine<SM>(cur, smem + (size_t)warp * rp.bulkShare, mbar + warp * COPY_SLOTS, rp.bulkShare);
    } else if (warp < rp.E + rp.NV) {
        const int v = warp - rp.E;
        vector_role<SM>(envs, (int)blockIdx.x * rp.NV + v, smem + rp.vecBase + (size_t)v * rp.vecShare,
                        mbar + COPY_MAX_ENGINES * COPY_SLOTS + v * VEC_SLOTS, rp.vecShare, rp.bulkByVec);
    }
    return (nB > 0 && totB > stB * nB && !rrB) || (nV > 0 && totV > stV * nV && !rrV);
}

// Side job (see SideJob): warps [firstWarp, 16) of every CTA, before their engine role.
__device__ __forceinline__ void run_side_job(const SideJob& j, int firstWarp) {
    const int warp = threadIdx.x >> 5;
    if (!j.dst || warp < firstWarp) return;
    const long long nthreads = (long long)gridDim.x * (COPY_WARPS - firstWarp) * 32;
    const long long tid = ((long long)blockIdx.x * (COPY_WARPS - firstWarp) + (warp - firstWarp)) * 32 + lane_id();
    for (long long i = tid; i < j.n; i += nthreads) {
        long long v = j.src[i];
        v = v > 0 ? v : 0;
        long long* out = j.dst + i;
        for (int c = 0; c < j.copies; ++c) out[(long long)c * j.n] = v;
    }
}

// dynamic smem layout: [ring: ringBytes][mbar: COPY_MBAR_COUNT x u64][bulk KiB: i64][colBase bulk: R+1 ints][colBase vec: R+1 ints]
//                      [coarse bulk: R*nb ints][coarse vec: R*nb ints]   (the last two only if useCoarse)
__global__ void __launch_bounds__(COPY_THREADS, 1) segment_copy_kernel(const CopyArgs a) {
    extern __shared__ __align__(128) unsigned char smem[];
    const int lane = lane_id();
    const int warp = threadIdx.x >> 5;
    const int R = a.ncols;
    unsigned long long* mbar = reinterpret_cast<unsigned long long*>(smem + a.ringBytes);
    int* colBase[2];
    long long* totKiB = reinterpret_cast<long long*>(mbar + COPY_MBAR_COUNT);
    colBase[0] = reinterpret_cast<int*>(totKiB + 1);
    colBase[1] = colBase[0] + (R + 1);
    const int nbR = R * coarse_blocks(a.colLen);
    int* coarse[2] = {nullptr, nullptr};
    if (a.useCoarse) { coarse[0] = colBase[1] + (R + 1); coarse[1] = coarse[0] + nbR; }

    // ---- prologue: mbarrier init (overlaps the metadata kernel under PDL), then cross-column tile
    //      bases = scan of the R per-column totals the metadata kernel wrote, and the coarse indexes ----
    griddep_launch_dependents();           // the next call's metadata kernel may become resident (it waits for us)
    for (int i = threadIdx.x; i < COPY_MBAR_COUNT; i += COPY_THREADS) mbar_init(smem_u32(&mbar[i]), 1);
    fence_mbar_init();
    griddep_wait();
    // every global load of the prologue is issued before the first one is consumed (one L2 round trip for the CTA, not one
    // per 32 columns): warps 0 / 1 scan the two lists' column totals, warp 2 sums the bulk bytes, warps 3.. stage the indexes
    if (a.useCoarse && warp >= 3) {
        for (int i = threadIdx.x - 96; i < 2 * nbR; i += COPY_THREADS - 96)
            coarse[0][i] = i < nbR ? a.coarse[0][i] : a.coarse[1][i - nbR];
    }
    if (warp < 2) {
        const int* ct = warp ? a.colTiles[1] : a.colTiles[0];
        int* cb = warp ? colBase[1] : colBase[0];
        int run = 0;
        if (lane == 0) cb[0] = 0;
        constexpr int PU = 4;                  // 128 columns per trip
        for (int c0 = 0; c0 < R; c0 += 32 * PU) {
            int v[PU];
#pragma unroll
            for (int u = 0; u < PU; ++u) { const int c = c0 + u * 32 + lane; v[u] = c < R ? ct[c] : 0; }
#pragma unroll
            for (int u = 0; u < PU; ++u) {
                const int c = c0 + u * 32 + lane;
                const int incl = warp_incl_scan(v[u]);
                if (c < R) cb[c + 1] = run + incl;
                run += __shfl_sync(0xffffffffu, incl, 31);
            }
        }
    } else if (warp == 2) {                    // bytes of the bulk list (-> average tile size, plan_ring)
        long long k = 0;
        for (int c = lane; c < R; c += 32) k += a.colKiB[c];
        k = warp_sum(k);
        if (lane == 0) *totKiB = k;
    }
    __syncthreads();

    run_side_job(a.side, COPY_WARPS / 2);
    const bool usedCounters = run_copy_engines<false>(a.desc, colBase, coarse, a.ctl, a.cls, a.ncols, a.colLen, a.bulkEngines, a.kmax, 0,
                                                      *totKiB, COPY_CLAIM_DIV, smem, mbar, a.ringBytes);
    workctl_checkout(a.ctl, usedCounters);
}

}  // namespace xdev
