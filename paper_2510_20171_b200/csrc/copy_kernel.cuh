// copy_kernel.cuh -- step a4 of the hot path: the byte-balanced variable-segment copy
// ("GPU side launches multi-blocks to copy data in parallel"; Fig. 3 L156 in-kernel
// D2D / P2P copy).  Every peer is local HBM here, so this kernel IS the AllToAllv payload term
// S/BW of L447.
//
// B200 design (not the paper's H100 kernel):
//   * persistent grid, one CTA per SM (x ctasPerSM), work discovered on the device from the
//     descriptor table the counts kernel wrote -- the host knows neither sizes nor tile counts,
//     so the launch is graph-capturable with a fixed grid (L387, L401);
//   * work unit = a tile of at most 2^tileShift bytes of ONE segment; tiles are claimed
//     dynamically in guided chunks from a global counter => balance by BYTES (and by time), not
//     by segment or by rank (config 3 skew is 250x across segments, 150x across ranks);
//   * LONG / aligned segments ("bulk" list): warp 0 drives a ring of shared-memory stages with
//     descriptor-less 1-D TMA: cp.async.bulk global->shared (mbarrier complete_tx) and
//     cp.async.bulk shared->global (bulk async-groups).  One elected lane issues everything;
//     S-1 tile loads (tens of KB) stay in flight per SM with no register staging;
//   * SHORT or unaligned segments ("vector" list): warps 1..N-1 copy with 16-byte vectorised,
//     fully coalesced ld/st (falling back to 8/4/2/1-byte units when source and destination
//     misalignment differ), head/tail bytes handled per tile.
#pragma once
#include "common.cuh"

namespace ncclx {

constexpr int COPY_THREADS = 512;          // warp 0: bulk engine; warps 1..15: vector engines
constexpr int COPY_SLOTS = 16;             // outstanding bulk tiles per engine (mbarriers); <= 32

struct CopyArgs {
    const SegDesc* desc;
    const int* colTiles[2];
    WorkCtl* ctl;
    int ncols;                             // destination columns of the descriptor table (= R)
    int colLen;                            // descriptor slots per column (R for the plain call, R*maxBlockLen for the dynamic one)
    unsigned int ringBytes;                // shared-memory ring size, multiple of 128, >= 3 tiles
    int staticEighths;                     // 0..8: share of the tiles assigned statically (contiguous per engine)
    int kmax[2];                           // max tiles per dynamic claim, per list (short-segment regime)
    int kmaxLong;                          // same, when segments average >= 8 tiles
    ClassParams cls;
};

// Warp-uniform cursor over one work list.  All lanes hold identical state except the descriptor
// WINDOW: lane i caches descriptor q = qw + i of the destination-major table, and the next 32 are
// prefetched into a second register set, so stepping from one segment to the next non-empty one of
// this list is a ballot over registers instead of a chain of dependent L2 reads (config 5 has a new
// segment every ~2 tiles).  Only a fresh claim pays the search: smem binary search over columns,
// then a warp-wide 32-ary search over the column's tile prefixes.
template <int L>
struct Cursor {
    const SegDesc* desc;
    const int* colBase;                    // smem, ncols+1 entries, colBase[ncols] = total tiles
    unsigned int* counter;
    ClassParams cls;
    int ncols, colLen, RR, tileShift, total, nEngines, kmax, kmin;
    int staticK, engineId;                 // first chunk is assigned statically: [engineId*staticK, +staticK)
    int dynBase;                           // tiles >= dynBase are claimed dynamically
    int pendCur, pendK;                    // lane 0: the NEXT chunk, claimed ahead of need (atomic in flight)
    int t, tEnd;                           // current tile, end of the claimed chunk
    int q, kInSeg, segTiles;               // current segment, tile within it, its tile count
    unsigned long long src, dst;
    long long bytes;
    int qw, qn;                            // bases of the current / prefetched window
    uint4 w0, w1, n0, n1;                  // this lane's descriptor in each window
    bool first, exhausted, haveWindow, longSegs;

    __device__ __forceinline__ void load_desc(int qq, uint4& a, uint4& b) const {
        if (qq < RR) {
            const uint4* p = reinterpret_cast<const uint4*>(desc + qq);
            a = __ldg(p); b = __ldg(p + 1);
        } else {
            a = make_uint4(0, 0, 0, 0); b = make_uint4(0, 0, 0, 0);
        }
    }
    __device__ __forceinline__ int my_tiles() const {
        return seg_tiles(L, ((unsigned long long)w0.y << 32) | w0.x, ((unsigned long long)w0.w << 32) | w0.z,
                         (long long)(((unsigned long long)w1.y << 32) | w1.x), cls);
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

    __device__ __forceinline__ void init(const CopyArgs& a, const int* colBase_, int nEngines_, int engineId_, int kmax_) {
        desc = a.desc; colBase = colBase_; counter = &a.ctl->next[L]; cls = a.cls;
        ncols = a.ncols; colLen = a.colLen; RR = a.ncols * a.colLen; tileShift = a.cls.tileShift[L]; total = colBase_[a.ncols];
        nEngines = nEngines_; engineId = engineId_;
        // long segments (>= 8 tiles each on average): claims resolve inside the cached window, so take
        // small chunks and keep all SMs in a tight moving window of HBM; short segments: every claim
        // pays a search, amortise it over more tiles.
        longSegs = total >= 8 * RR;
        kmax = longSegs ? a.kmaxLong : kmax_;
        // staticEighths/8 of the tiles can be split evenly and statically (contiguous range per engine);
        // the rest is claimed dynamically, IN ORDER, in guided chunks.  Measured on B200: the in-order
        // dynamic claim keeps all SMs inside one moving window of HBM and is ~7 % faster than contiguous
        // static ranges (148 far-apart streams), so the default is fully dynamic (staticEighths = 0).
        staticK = (int)(((long long)total * a.staticEighths / 8) / nEngines);
        kmin = total >= 8 * nEngines ? 2 : 1;
        dynBase = staticK * nEngines;
        pendCur = pendK = 0;
        t = tEnd = 0; q = 0; kInSeg = segTiles = 0; src = dst = 0; bytes = 0;
        qw = qn = 0; w0 = w1 = n0 = n1 = make_uint4(0, 0, 0, 0);
        first = true;
        haveWindow = false;
        exhausted = (total == 0);
        if (!exhausted) claim_issue(dynBase);
    }

    // Lane 0 issues the atomic for the next dynamic chunk; the result is only consumed by claim_take(),
    // so its L2 round trip overlaps the tiles of the current chunk.
    __device__ __forceinline__ void claim_issue(int counterHint) {
        if (lane_id() == 0) {
            const int rem = total - min(total, counterHint);
            pendK = max(kmin, min(kmax, rem / (2 * nEngines)));
            pendCur = dynBase + (int)atomicAdd(counter, (unsigned int)pendK);
        }
    }

    // Find the segment that owns global tile index tt (0 <= tt < total) and (re)load the windows there.
    __device__ __forceinline__ void locate(int tt) {
        const int lane = lane_id();
        int lo = 0, hi = ncols;            // colBase[lo] <= tt < colBase[hi]
        while (hi - lo > 1) {
            const int mid = (lo + hi) >> 1;
            if (colBase[mid] <= tt) lo = mid; else hi = mid;
        }
        const int d = lo;
        const int tl = tt - colBase[d];
        const SegDesc* col = desc + (size_t)d * colLen;
        int s0 = 0, n = colLen;                 // smallest s with col[s].pfx[L] > tl lies in [s0, s0+n)
        while (n > 32) {                   // 128-ary rounds: every lane probes 4 block ends per L2 round trip
            const int step = (n + 127) >> 7;
            int cnt = 0;
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const int b = lane * 4 + u;
                const int idx = s0 + min((b + 1) * step, n) - 1;
                cnt += (__ldg(&col[idx].pfx[L]) <= tl) ? 1 : 0;
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
        const int nn = n + (s0 - sb);
        qw = d * colLen + sb;
        load_desc(qw + lane, w0, w1);
        qn = qw + 32;
        load_desc(qn + lane, n0, n1);
        const int pf = L == LIST_BULK ? (int)w1.z : (int)w1.w;
        const int m = __popc(__ballot_sync(0xffffffffu, lane < nn && pf <= tl));
        const int prevInWin = __shfl_sync(0xffffffffu, pf, m > 0 ? m - 1 : 0);
        const int prev = m > 0 ? prevInWin : 0;
        take(m);
        kInSeg = tl - prev;
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
            if (qw >= RR) { exhausted = true; break; }      // cannot happen while t < total
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
            if (qw >= RR) return false;
        }
        return false;
    }

    // Make (t, segment) valid; false when the list is drained.
    __device__ __forceinline__ bool ensure() {
        if (exhausted) return false;
        if (t < tEnd) {
            if (kInSeg >= segTiles) advance_segment();
            return !exhausted;
        }
        int cur, k;
        if (first && staticK > 0) {        // static share: no atomic on the start-up path
            first = false;
            cur = engineId * staticK;
            k = staticK;
        } else {
            first = false;
            cur = __shfl_sync(0xffffffffu, pendCur, 0);
            k = __shfl_sync(0xffffffffu, pendK, 0);
            if (cur >= total || cur < 0) { exhausted = true; return false; }
            claim_issue(cur + k);
        }
        const bool near = longSegs && haveWindow && cur >= t && advance_by(cur - t);
        t = cur;
        tEnd = min(cur + k, total);
        if (!near) locate(t);
        haveWindow = true;
        return true;
    }

    __device__ __forceinline__ long long tile_off() const { return (long long)kInSeg << tileShift; }
    __device__ __forceinline__ void next() { ++t; ++kInSeg; }
};

// ---- vector path -------------------------------------------------------------------------------
template <typename T> __device__ __forceinline__ T ld_unit(const T* p) { return __ldg(p); }
template <> __device__ __forceinline__ uint4 ld_unit<uint4>(const uint4* p) { return ld_stream_nc(p); }
template <typename T> __device__ __forceinline__ void st_unit(T* p, const T& v) { *p = v; }
template <> __device__ __forceinline__ void st_unit<uint4>(uint4* p, const uint4& v) { st_stream(p, v); }

template <typename T, int U>
__device__ __forceinline__ void warp_copy_units(const unsigned char* src, unsigned char* dst, long long n) {
    const T* s = reinterpret_cast<const T*>(src);
    T* d = reinterpret_cast<T*>(dst);
    long long i = lane_id();
    for (; i + (U - 1) * 32 < n; i += U * 32) {
        T v[U];
#pragma unroll
        for (int j = 0; j < U; ++j) v[j] = ld_unit(s + i + j * 32);
#pragma unroll
        for (int j = 0; j < U; ++j) st_unit(d + i + j * 32, v[j]);
    }
    for (; i < n; i += 32) st_unit(d + i, ld_unit(s + i));
}

// Copy len bytes src -> dst with one warp; any alignment.
__device__ __forceinline__ void warp_copy_bytes(const unsigned char* src, unsigned char* dst, long long len) {
    const unsigned int diff = (unsigned int)(((unsigned long long)src ^ (unsigned long long)dst) & 15ull);
    const int g = diff == 0 ? 16 : (int)(diff & (0u - diff));          // common alignment granule
    long long head = (long long)((g - (int)((unsigned long long)dst & (unsigned long long)(g - 1))) & (g - 1));
    if (head > len) head = len;
    if (lane_id() < head) dst[lane_id()] = __ldg(src + lane_id());    // head < 16 <= 32 lanes
    src += head; dst += head; len -= head;
    const long long units = len / g;
    switch (g) {
    case 16: warp_copy_units<uint4, 8>(src, dst, units); break;
    case 8:  warp_copy_units<uint2, 8>(src, dst, units); break;
    case 4:  warp_copy_units<unsigned int, 8>(src, dst, units); break;
    case 2:  warp_copy_units<unsigned short, 8>(src, dst, units); break;
    default: warp_copy_units<unsigned char, 8>(src, dst, units); break;
    }
    const long long done = units * g;
    const int tail = (int)(len - done);                                // < 16
    if (lane_id() < tail) dst[done + lane_id()] = __ldg(src + done + lane_id());
}

// dynamic smem layout: [ring: ringBytes][mbar: COPY_SLOTS x u64][colBase bulk: R+1 ints][colBase vec: R+1 ints]
__global__ void __launch_bounds__(COPY_THREADS, 1) segment_copy_kernel(const CopyArgs a) {
    extern __shared__ __align__(128) unsigned char smem[];
    const int lane = lane_id();
    const int warp = threadIdx.x >> 5;
    const int R = a.ncols;
    unsigned long long* mbar = reinterpret_cast<unsigned long long*>(smem + a.ringBytes);
    int* colBase[2];
    colBase[0] = reinterpret_cast<int*>(mbar + COPY_SLOTS);
    colBase[1] = colBase[0] + (R + 1);

    // ---- prologue: mbarrier init (overlaps the counts kernel under PDL), then cross-column tile
    //      bases = scan of the R per-column totals the counts kernel wrote -------------------------
    if (warp == 2 && lane == 0) {
        for (int i = 0; i < COPY_SLOTS; ++i) mbar_init(smem_u32(&mbar[i]), 1);
        fence_mbar_init();
    }
    griddep_wait();
    if (warp < 2) {
        const int* ct = a.colTiles[warp];
        int* cb = colBase[warp];
        int run = 0;
        if (lane == 0) cb[0] = 0;
        for (int c0 = 0; c0 < R; c0 += 32) {
            const int v = c0 + lane < R ? ct[c0 + lane] : 0;
            const int incl = warp_incl_scan(v);
            if (c0 + lane < R) cb[c0 + lane + 1] = run + incl;
            run += __shfl_sync(0xffffffffu, incl, 31);
        }
    }
    __syncthreads();

    if (warp == 0) {
        // ================= bulk engine: byte-granular TMA ring driven by one elected lane ========
        // The ring is a circular BYTE buffer (not fixed-size stages): every tile takes exactly
        // align128(len) bytes, so short tiles (config 5: 10-28 KiB) keep as many bytes in flight as
        // long ones.  Up to COPY_SLOTS tiles are outstanding; slot j's bookkeeping (destination,
        // length, smem offset, virtual start) lives in the registers of lane j.
        Cursor<LIST_BULK> cur;
        cur.init(a, colBase[LIST_BULK], (int)gridDim.x, (int)blockIdx.x, a.kmax[LIST_BULK]);
        const unsigned int tileBytes = 1u << a.cls.tileShift[LIST_BULK];
        const unsigned int ringBytes = a.ringBytes;
        const uint32_t ring0 = smem_u32(smem);
        unsigned long long mDst = 0;          // slot registers (lane j <-> slot j)
        unsigned int mLen = 0, mOff = 0, mV = 0;
        unsigned int vHead = 0, phys = 0;     // virtual (mod 2^32) and physical allocation offsets
        int iLoad = 0, iStore = 0, freed = 0;  // stores [0, freed) have finished reading their smem
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
                    if (iLoad - freed >= COPY_SLOTS) break;
                    const unsigned int pad = phys + len16 > ringBytes ? ringBytes - phys : 0u;   // wrap
                    const unsigned int vTail = freed < iLoad ? __shfl_sync(0xffffffffu, mV, freed % COPY_SLOTS) : vHead;
                    if (vHead + pad + len16 - vTail > ringBytes) break;
                    const unsigned int vStart = vHead + pad;
                    const unsigned int po = pad ? 0u : phys;
                    const int slot = iLoad % COPY_SLOTS;
                    if (lane == slot) { mDst = (unsigned long long)dstp; mLen = len16; mOff = po; mV = vStart; }
                    if (lane == 0) {
                        const uint32_t bar = smem_u32(&mbar[slot]);
                        mbar_expect_tx(bar, len16);
                        bulk_g2s(ring0 + po, srcp, len16, bar);
                    }
                    const unsigned int adv = (len16 + 127u) & ~127u;
                    vHead = vStart + adv;
                    phys = po + adv;
                    if (phys >= ringBytes) phys = 0;
                    ++iLoad;
                }
                const int tail = (int)(len & 15u);        // only the last tile of a ragged segment
                if (lane < tail) dstp[len16 + lane] = __ldg(srcp + len16 + lane);
                cur.next();
                more = cur.ensure();
            }
            if (iStore == iLoad) {
                if (!more) break;
                // every issued tile is stored but the next one does not fit behind the last store's
                // not-yet-released bytes: release everything and restart the ring at offset 0
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
                bulk_s2g(reinterpret_cast<void*>(((unsigned long long)dhi << 32) | dlo), ring0 + soff, slen);
                bulk_commit();
                if (more) bulk_wait_read<1>();            // releases the smem of every store but this one
            }
            freed = max(freed, iStore);                   // (only consulted while `more`)
            ++iStore;
            __syncwarp();
        }
        if (lane == 0) bulk_wait_all<0>();
    } else {
        // ================= vector engines: one warp per tile ===================================
        Cursor<LIST_VEC> cur;
        cur.init(a, colBase[LIST_VEC], (int)gridDim.x * (COPY_THREADS / 32 - 1),
                 (int)blockIdx.x * (COPY_THREADS / 32 - 1) + warp - 1, a.kmax[LIST_VEC]);
        const long long tileBytes = 1ll << a.cls.tileShift[LIST_VEC];
        while (cur.ensure()) {
            const long long off = cur.tile_off();
            const long long rest = cur.bytes - off;
            const long long len = rest < tileBytes ? rest : tileBytes;
            warp_copy_bytes(reinterpret_cast<const unsigned char*>(cur.src + off),
                            reinterpret_cast<unsigned char*>(cur.dst + off), len);
            cur.next();
        }
    }
}

}  // namespace ncclx
