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
constexpr int COPY_MAX_STAGES = 8;
constexpr int COPY_KMAX_BULK = 16;         // max tiles per claim
constexpr int COPY_KMAX_VEC = 8;

struct CopyArgs {
    const SegDesc* desc;
    const int* colTiles[2];
    WorkCtl* ctl;
    int R;
    int tileShift[2];
    int stages;                            // ring stages of 2^tileShift[BULK] bytes
};

// Warp-uniform cursor over one work list.  All lanes hold identical state.
template <int L>
struct Cursor {
    const SegDesc* desc;
    const int* colBase;                    // smem, R+1 entries, colBase[R] = total tiles
    unsigned int* counter;
    int R, tileShift, total, nEngines, kmax;
    int t, tEnd;                           // current tile, end of the claimed chunk
    int segFirst, segEnd;                  // tile range of the current segment
    unsigned long long src, dst;
    long long bytes;
    bool exhausted;

    __device__ __forceinline__ void init(const CopyArgs& a, const int* colBase_, int nEngines_, int kmax_) {
        desc = a.desc; colBase = colBase_; counter = &a.ctl->next[L];
        R = a.R; tileShift = a.tileShift[L]; total = colBase_[a.R];
        nEngines = nEngines_; kmax = kmax_;
        t = tEnd = 0; segFirst = segEnd = 0; src = dst = 0; bytes = 0;
        exhausted = (total == 0);
    }

    // Find the segment that owns global tile index tt (0 <= tt < total).
    __device__ __forceinline__ void locate(int tt) {
        const int lane = lane_id();
        int lo = 0, hi = R;                // colBase[lo] <= tt < colBase[hi]
        while (hi - lo > 1) {
            const int mid = (lo + hi) >> 1;
            if (colBase[mid] <= tt) lo = mid; else hi = mid;
        }
        const int d = lo;
        const int base = colBase[d];
        const int tl = tt - base;
        const SegDesc* col = desc + (size_t)d * R;
        int s0 = 0, n = R;                 // smallest s with col[s].pfx[L] > tl lies in [s0, s0+n)
        while (n > 32) {
            const int step = (n + 31) >> 5;
            const int idx = s0 + min((lane + 1) * step, n) - 1;
            const int v = __ldg(&col[idx].pfx[L]);
            const int m = __popc(__ballot_sync(0xffffffffu, v <= tl));
            s0 += m * step;
            n = min(step, n - m * step);
        }
        const int v = lane < n ? __ldg(&col[s0 + lane].pfx[L]) : 0x7fffffff;
        const int m = __popc(__ballot_sync(0xffffffffu, v <= tl));
        const int s = s0 + m;
        const uint4* p = reinterpret_cast<const uint4*>(col + s);
        const uint4 w0 = __ldg(p), w1 = __ldg(p + 1);
        const int prev = s > 0 ? __ldg(&col[s - 1].pfx[L]) : 0;
        src = ((unsigned long long)w0.y << 32) | w0.x;
        dst = ((unsigned long long)w0.w << 32) | w0.z;
        bytes = (long long)(((unsigned long long)w1.y << 32) | w1.x);
        const int pf = L == LIST_BULK ? (int)w1.z : (int)w1.w;
        segFirst = base + prev;
        segEnd = base + pf;
    }

    // Make (t, segment) valid; false when the list is drained.
    __device__ __forceinline__ bool ensure() {
        if (exhausted) return false;
        if (t < tEnd) {
            if (t >= segEnd) locate(t);
            return true;
        }
        int cur = 0, k = 0;
        if (lane_id() == 0) {
            const unsigned int seen = *reinterpret_cast<volatile unsigned int*>(counter);
            const int rem = total - (int)min(seen, (unsigned int)total);
            k = max(1, min(kmax, rem / (2 * nEngines)));
            cur = (int)atomicAdd(counter, (unsigned int)k);
        }
        cur = __shfl_sync(0xffffffffu, cur, 0);
        k = __shfl_sync(0xffffffffu, k, 0);
        if (cur >= total) { exhausted = true; return false; }
        t = cur;
        tEnd = min(cur + k, total);
        locate(t);
        return true;
    }

    __device__ __forceinline__ long long tile_off() const { return (long long)(t - segFirst) << tileShift; }
    __device__ __forceinline__ void next() { ++t; }
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

// dynamic smem layout: [ring: stages << tileShiftB][mbar: 8 x u64][stDst: 8 x u64][stLen: 8 x u32]
//                      [colBase bulk: R+1 ints][colBase vec: R+1 ints]
__global__ void __launch_bounds__(COPY_THREADS, 1) segment_copy_kernel(const CopyArgs a) {
    extern __shared__ __align__(128) unsigned char smem[];
    const int lane = lane_id();
    const int warp = threadIdx.x >> 5;
    const int R = a.R;
    const size_t ringBytes = (size_t)a.stages << a.tileShift[LIST_BULK];
    unsigned long long* mbar = reinterpret_cast<unsigned long long*>(smem + ringBytes);
    unsigned long long* stDst = mbar + COPY_MAX_STAGES;
    unsigned int* stLen = reinterpret_cast<unsigned int*>(stDst + COPY_MAX_STAGES);
    int* colBase[2];
    colBase[0] = reinterpret_cast<int*>(stLen + COPY_MAX_STAGES);
    colBase[1] = colBase[0] + (R + 1);

    // ---- prologue: cross-column tile bases (scan of R per-column totals), mbarrier init ------
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
    } else if (warp == 2 && lane == 0) {
        for (int i = 0; i < a.stages; ++i) mbar_init(smem_u32(&mbar[i]), 1);
        fence_mbar_init();
    }
    __syncthreads();

    if (warp == 0) {
        // ================= bulk engine: TMA ring driven by one elected lane ====================
        Cursor<LIST_BULK> cur;
        cur.init(a, colBase[LIST_BULK], (int)gridDim.x, COPY_KMAX_BULK);
        const int S = a.stages;
        const unsigned int tileBytes = 1u << a.tileShift[LIST_BULK];
        const uint32_t ring0 = smem_u32(smem);
        int iLoad = 0, iStore = 0;
        bool more = cur.ensure();
        while (true) {
            // fill: issue loads while a stage is free (its previous store has finished READING smem)
            while (more && iLoad < max(iStore - 1, 0) + S) {
                const long long off = cur.tile_off();
                const long long rest = cur.bytes - off;
                const unsigned int len = rest < (long long)tileBytes ? (unsigned int)rest : tileBytes;
                const unsigned int len16 = len & ~15u;
                const unsigned char* srcp = reinterpret_cast<const unsigned char*>(cur.src + off);
                unsigned char* dstp = reinterpret_cast<unsigned char*>(cur.dst + off);
                if (len16) {
                    const int st = iLoad % S;
                    if (lane == 0) {
                        stDst[st] = (unsigned long long)dstp;
                        stLen[st] = len16;
                        const uint32_t bar = smem_u32(&mbar[st]);
                        mbar_expect_tx(bar, len16);
                        bulk_g2s(ring0 + ((uint32_t)st << a.tileShift[LIST_BULK]), srcp, len16, bar);
                    }
                    ++iLoad;
                }
                const int tail = (int)(len & 15u);        // only the last tile of a ragged segment
                if (lane < tail) dstp[len16 + lane] = __ldg(srcp + len16 + lane);
                cur.next();
                more = cur.ensure();
            }
            if (iStore == iLoad) {
                if (!more) break;
                continue;
            }
            const int st = iStore % S;
            mbar_wait(smem_u32(&mbar[st]), (uint32_t)((iStore / S) & 1));
            if (lane == 0) {
                bulk_s2g(reinterpret_cast<void*>(stDst[st]), ring0 + ((uint32_t)st << a.tileShift[LIST_BULK]), stLen[st]);
                bulk_commit();
                if (more) bulk_wait_read<1>();            // frees the stage of store iStore-1
            }
            ++iStore;
            __syncwarp();
        }
        if (lane == 0) bulk_wait_all<0>();
    } else {
        // ================= vector engines: one warp per tile ===================================
        Cursor<LIST_VEC> cur;
        cur.init(a, colBase[LIST_VEC], (int)gridDim.x * (COPY_THREADS / 32 - 1), COPY_KMAX_VEC);
        const long long tileBytes = 1ll << a.tileShift[LIST_VEC];
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
