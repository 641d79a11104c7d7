// reduce_kernel.cuh -- steps r1 / r2 of the hot path: the in-kernel sum behind AllReduce and
// ReduceScatter (the Reduce / ReduceCopy step of the paper's FTAR ring, section 5.3
// L335-337, Fig. 9: "combine the reduction and forwarding copy ... avoids redundant HBM
// load ... avoid unnecessary HBM stores ... enhance instruction level parallelism").
//
// Numeric contract (BASELINE.json north_star): acc = (float)x_0;
// acc = acc + (float)x_k for k = 1..R-1 in binary32 round-to-nearest-even, no FTZ, no
// reassociation; ONE rounding to the output type; NaN results canonical.
//
// B200 design: HBM-bound streaming kernel.  Each thread owns one 32-byte vector position
// (bf16x16 / f16x16 / fp32x8; 16-byte vectors when only 16 B alignment holds) per tile and issues the
// 256-bit loads (LDG.E.256) of CH ranks back to back (CH independent 32 B loads in flight per thread,
// L1 no-allocate) before the ordered fp32 adds;
// inputs are read exactly once and the result is written straight to the R outputs
// (AllReduce) or to the owning rank's block (ReduceScatter): no intermediate HBM round trip.
// The device pointer tables are staged once per CTA into shared memory.
#pragma once
#include <cuda_bf16.h>
#include <cuda_fp16.h>
#include "common.cuh"

namespace xdev {

constexpr int REDUCE_THREADS = 128;        // CTA size of long reductions
constexpr int REDUCE_THREADS_SHORT = 64;                   // ... and of short ones (below kReduceShortBytes of input: twice as many, smaller
                                                           // CTAs for the hardware scheduler to deal out; config 2 23.1 -> 22.8 us per call,
                                                           // while config 4 prefers 128: +0.3 % with 64)
enum { RED_BF16 = 0, RED_F32 = 1, RED_F16 = 2 };

struct ReduceArgs {
    const void* const* send;     // device table, R pointers
    void* const* recv;           // device table, R pointers
    unsigned long long blockElems; // AllReduce: count; ReduceScatter: recvcount
    int R;
    int scatter;                 // 0: AllReduce (1 block, R outputs), 1: ReduceScatter (R blocks)
    int prefetchTiles;           // > 0: CTAs b < prefetchCtas pull tiles b, b + prefetchCtas, ... (this many) into L2 BEFORE the
    int prefetchCtas;            //      dependency wait (short calls under PDL)
};

template <int DT> struct Acc;    // accumulators for one 16-byte vector

template <> struct Acc<RED_BF16> {
    float v[8];
    __device__ __forceinline__ void set(const uint4& u) {
        const unsigned int w[4] = {u.x, u.y, u.z, u.w};
#pragma unroll
        for (int i = 0; i < 4; ++i) { v[2 * i] = __uint_as_float(w[i] << 16); v[2 * i + 1] = __uint_as_float(w[i] & 0xffff0000u); }
    }
    __device__ __forceinline__ void add(const uint4& u) {
        const unsigned int w[4] = {u.x, u.y, u.z, u.w};
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            v[2 * i] = __fadd_rn(v[2 * i], __uint_as_float(w[i] << 16));
            v[2 * i + 1] = __fadd_rn(v[2 * i + 1], __uint_as_float(w[i] & 0xffff0000u));
        }
    }
    __device__ __forceinline__ uint4 pack() const {
        unsigned int w[4];
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            __nv_bfloat162 h = __floats2bfloat162_rn(v[2 * i], v[2 * i + 1]);   // cvt.rn.bf16x2.f32, NaN -> 0x7FFF
            w[i] = *reinterpret_cast<unsigned int*>(&h);
        }
        return make_uint4(w[0], w[1], w[2], w[3]);
    }
};

template <> struct Acc<RED_F16> {
    float v[8];
    __device__ __forceinline__ static float2 up(unsigned int w) {
        return __half22float2(*reinterpret_cast<const __half2*>(&w));
    }
    __device__ __forceinline__ void set(const uint4& u) {
        const unsigned int w[4] = {u.x, u.y, u.z, u.w};
#pragma unroll
        for (int i = 0; i < 4; ++i) { float2 f = up(w[i]); v[2 * i] = f.x; v[2 * i + 1] = f.y; }
    }
    __device__ __forceinline__ void add(const uint4& u) {
        const unsigned int w[4] = {u.x, u.y, u.z, u.w};
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            float2 f = up(w[i]);
            v[2 * i] = __fadd_rn(v[2 * i], f.x);
            v[2 * i + 1] = __fadd_rn(v[2 * i + 1], f.y);
        }
    }
    __device__ __forceinline__ uint4 pack() const {
        unsigned int w[4];
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            __half2 h = __floats2half2_rn(v[2 * i], v[2 * i + 1]);              // NaN -> 0x7FFF
            w[i] = *reinterpret_cast<unsigned int*>(&h);
        }
        return make_uint4(w[0], w[1], w[2], w[3]);
    }
};

__device__ __forceinline__ unsigned int canon_f32(float f) {
    return (f != f) ? 0x7fffffffu : __float_as_uint(f);
}

template <> struct Acc<RED_F32> {
    float v[4];
    __device__ __forceinline__ void set(const uint4& u) {
        v[0] = __uint_as_float(u.x); v[1] = __uint_as_float(u.y); v[2] = __uint_as_float(u.z); v[3] = __uint_as_float(u.w);
    }
    __device__ __forceinline__ void add(const uint4& u) {
        v[0] = __fadd_rn(v[0], __uint_as_float(u.x)); v[1] = __fadd_rn(v[1], __uint_as_float(u.y));
        v[2] = __fadd_rn(v[2], __uint_as_float(u.z)); v[3] = __fadd_rn(v[3], __uint_as_float(u.w));
    }
    __device__ __forceinline__ uint4 pack() const {
        return make_uint4(canon_f32(v[0]), canon_f32(v[1]), canon_f32(v[2]), canon_f32(v[3]));
    }
};

// scalar helpers (unaligned / ragged path), same arithmetic
template <int DT> __device__ __forceinline__ float load_elem(const void* p, unsigned long long i);
template <> __device__ __forceinline__ float load_elem<RED_BF16>(const void* p, unsigned long long i) {
    return __uint_as_float((unsigned int)reinterpret_cast<const volatile unsigned short*>(p)[i] << 16);
}
template <> __device__ __forceinline__ float load_elem<RED_F16>(const void* p, unsigned long long i) {
    unsigned short b = reinterpret_cast<const volatile unsigned short*>(p)[i];
    return __half2float(*reinterpret_cast<const __half*>(&b));
}
template <> __device__ __forceinline__ float load_elem<RED_F32>(const void* p, unsigned long long i) {
    return reinterpret_cast<const volatile float*>(p)[i];
}
template <int DT> __device__ __forceinline__ void store_elem(void* p, unsigned long long i, float acc);
template <> __device__ __forceinline__ void store_elem<RED_BF16>(void* p, unsigned long long i, float acc) {
    __nv_bfloat16 h = __float2bfloat16_rn(acc);
    reinterpret_cast<unsigned short*>(p)[i] = *reinterpret_cast<unsigned short*>(&h);
}
template <> __device__ __forceinline__ void store_elem<RED_F16>(void* p, unsigned long long i, float acc) {
    __half h = __float2half_rn(acc);
    unsigned short b = *reinterpret_cast<unsigned short*>(&h);
    if (acc != acc) b = 0x7fff;
    reinterpret_cast<unsigned short*>(p)[i] = b;
}
template <> __device__ __forceinline__ void store_elem<RED_F32>(void* p, unsigned long long i, float acc) {
    reinterpret_cast<unsigned int*>(p)[i] = canon_f32(acc);
}

// One tile of THREADS vector positions: every thread reduces one VB-byte vector (VB = 32: one 256-bit
// load per rank; VB = 16: one 128-bit load per rank) over all R ranks and writes the result.
template <int DT, int CH, int VB>
__device__ __forceinline__ void reduce_vectors(const ReduceArgs& a, const unsigned char* const* sp, unsigned char* const* rp,
                                               unsigned long long n, int nblocks) {
    constexpr int ES = DT == RED_F32 ? 4 : 2;
    constexpr int EPV = VB / ES;
    const int R = a.R;
    const unsigned long long nvec = n / EPV;                       // full vectors per block
    const unsigned int tpb = (unsigned int)((nvec + blockDim.x - 1) / blockDim.x);
    const unsigned long long ntiles = (unsigned long long)tpb * nblocks;
    for (unsigned long long t = blockIdx.x; t < ntiles; t += gridDim.x) {
        const unsigned int blk = a.scatter ? (unsigned int)(t / tpb) : 0u;
        const unsigned int tb = (unsigned int)(t - (unsigned long long)blk * tpb);
        const unsigned long long v = (unsigned long long)tb * blockDim.x + threadIdx.x;
        if (v < nvec) {
            const unsigned long long inOff = ((unsigned long long)blk * nvec + v) * VB;   // n*ES % VB == 0 when scatter
            Acc<DT> acc0, acc1;
            for (int k0 = 0; k0 < R; k0 += CH) {
                if constexpr (VB == 32) {
                    u32x8 x[CH];
#pragma unroll
                    for (int j = 0; j < CH; ++j)
                        if (k0 + j < R) x[j] = ld_stream256(sp[k0 + j] + inOff);
#pragma unroll
                    for (int j = 0; j < CH; ++j)
                        if (k0 + j < R) {
                            if (k0 + j == 0) { acc0.set(x[j].lo); acc1.set(x[j].hi); }
                            else { acc0.add(x[j].lo); acc1.add(x[j].hi); }
                        }
                } else {
                    uint4 x[CH];
#pragma unroll
                    for (int j = 0; j < CH; ++j)
                        if (k0 + j < R) x[j] = ld_stream(reinterpret_cast<const uint4*>(sp[k0 + j] + inOff));
#pragma unroll
                    for (int j = 0; j < CH; ++j)
                        if (k0 + j < R) { if (k0 + j == 0) acc0.set(x[j]); else acc0.add(x[j]); }
                }
            }
            if constexpr (VB == 32) {
                u32x8 o;
                o.lo = acc0.pack(); o.hi = acc1.pack();
                if (a.scatter) st_stream256(rp[blk] + v * VB, o);
                else for (int r = 0; r < R; ++r) st_stream256(rp[r] + v * VB, o);
            } else {
                const uint4 o = acc0.pack();
                if (a.scatter) st_stream(reinterpret_cast<uint4*>(rp[blk] + v * VB), o);
                else for (int r = 0; r < R; ++r) st_stream(reinterpret_cast<uint4*>(rp[r] + v * VB), o);
            }
        }
    }
    // ragged tail of an AllReduce (count % EPV elements), scalar
    if (!a.scatter && blockIdx.x == 0) {
        const unsigned long long i = nvec * EPV + threadIdx.x;
        if (i < n) {
            float acc = load_elem<DT>(sp[0], i);
            for (int k = 1; k < R; ++k) acc = __fadd_rn(acc, load_elem<DT>(sp[k], i));
            for (int r = 0; r < R; ++r) store_elem<DT>(rp[r], i, acc);
        }
    }
}

// dynamic smem: const void* sp[R]; void* rp[R]
template <int DT, int CH, int TH>
__global__ void __launch_bounds__(TH) reduce_kernel(const ReduceArgs a) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const unsigned char** sp = reinterpret_cast<const unsigned char**>(smem_raw);
    unsigned char** rp = reinterpret_cast<unsigned char**>(smem_raw) + a.R;
    __shared__ int sMis;
    const int R = a.R;
    constexpr int ES = DT == RED_F32 ? 4 : 2;

    griddep_launch_dependents();           // no-ops unless launched with programmatic stream serialisation (short calls)
    // Short calls under PDL: the first wave of CTAs is resident while the stream's previous kernel drains, so it pulls
    // INPUT tiles into L2 now (prefetch.global.L2: a hint, and L2 is the point of coherence, so a line fetched early
    // cannot go stale even if that kernel still writes it) -- for an input that fits L2, all of it: the DRAM reads then
    // run at full memory-level parallelism from before the wait on, decoupled from the SMs' load/store issue, and overlap
    // the predecessor's tail (config 2 in a graph of back-to-back calls).
    if (a.prefetchTiles > 0 && R <= 32 && (int)blockIdx.x < a.prefetchCtas) {
        const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
        const unsigned long long mine = lane < R ? (unsigned long long)a.send[lane] : 0ull;
        const unsigned long long n0 = a.blockElems;
        const unsigned long long nvec = n0 * ES / 32;
        const unsigned int tpb = (unsigned int)((nvec + TH - 1) / TH);
        const unsigned long long ntiles = (unsigned long long)tpb * (a.scatter ? R : 1);
        unsigned long long t = blockIdx.x;
        for (int i = 0; i < a.prefetchTiles && t < ntiles; ++i, t += (unsigned long long)a.prefetchCtas) {
            const unsigned int blk = a.scatter ? (unsigned int)(t / tpb) : 0u;
            const unsigned long long v0 = (t - (unsigned long long)blk * tpb) * TH;     // first vector of the tile
            for (int k = warp; k < R; k += TH / 32) {
                const unsigned long long base = __shfl_sync(0xffffffffu, mine, k);
                for (int ln = lane; ln < TH / 4; ln += 32) {                             // the tile's 128-byte lines
                    const unsigned long long o = v0 * 32 + (unsigned long long)ln * 128;
                    if (base && o < nvec * 32) prefetch_l2(reinterpret_cast<const void*>(base + blk * nvec * 32 + o));
                }
            }
        }
    }
    griddep_wait();
    if (threadIdx.x == 0) sMis = 0;
    __syncthreads();
    int mis = 0;
    for (int k = threadIdx.x; k < R; k += TH) {
        const unsigned char* s = reinterpret_cast<const unsigned char*>(a.send[k]);
        unsigned char* r = reinterpret_cast<unsigned char*>(a.recv[k]);
        sp[k] = s; rp[k] = r;
        mis |= (int)(((unsigned long long)s | (unsigned long long)r) & 31ull);
    }
    if (mis) atomicOr(&sMis, mis);
    __syncthreads();
    const unsigned long long n = a.blockElems;
    const int nblocks = a.scatter ? R : 1;
    const int misAll = sMis | (a.scatter ? (int)((n * ES) & 31ull) : 0);   // block stride must keep the alignment

    if ((misAll & 31) == 0) {
        reduce_vectors<DT, CH, 32>(a, sp, rp, n, nblocks);
    } else if ((misAll & 15) == 0) {
        reduce_vectors<DT, CH, 16>(a, sp, rp, n, nblocks);
    } else {
        // scalar path: any alignment, same arithmetic, one element per thread
        const unsigned long long total = n * nblocks;
        for (unsigned long long i = (unsigned long long)blockIdx.x * TH + threadIdx.x; i < total;
             i += (unsigned long long)gridDim.x * TH) {
            float acc = load_elem<DT>(sp[0], i);
            for (int k = 1; k < R; ++k) acc = __fadd_rn(acc, load_elem<DT>(sp[k], i));
            if (a.scatter) {
                const unsigned long long blk = i / n;
                store_elem<DT>(rp[blk], i - blk * n, acc);
            } else {
                for (int r = 0; r < R; ++r) store_elem<DT>(rp[r], i, acc);
            }
        }
    }
}

// ---- FTAR-style ReduceCopy step (section 5.3, Fig. 9) ---------
// One pipeline step of the paper's ring: an incoming chunk `a` (what the previous peer sent) is summed
// with the local chunk `b`; the result goes to the local output `out` (Reduce), to the forward buffer
// `fwd` that the next peer will receive (ReduceCopy: "combine the reduction and forwarding copy ... avoids
// redundant HBM load"; `out` may be NULL in the intermediate steps: "avoid unnecessary HBM stores"), or
// both.  The message is processed in fixed chunks of S bytes (paper: 8 MB) by a FIXED, small number of
// CTAs (paper: 2 CTAs x 512 threads suffice against the network): throughput per CTA comes from
// instruction-level parallelism (L335 "enhance instruction level parallelism to saturate GPU resources").
// Two variants (NCCLX_PARAM_REDUCECOPY_TMA):
//   reducecopy_kernel      512 threads, software-pipelined: the 2 x RC_UNROLL 256-bit loads of tile i+1 are issued
//                          before the adds and stores of tile i (also across chunk boundaries), so the CTA never
//                          alternates between a load phase and a store phase (round 1 did: 96 GB/s per CTA);
//   reducecopy_tma_kernel  a producer warp streams `a` and `b` through a 6-stage shared-memory ring with
//                          cp.async.bulk (192 KB in flight per CTA, no registers); 512 consumer threads add from
//                          shared memory and store.
constexpr int RC_THREADS = 512;
constexpr int RC_UNROLL = 2;

struct ReduceCopyArgs {
    const unsigned char* a;
    const unsigned char* b;
    unsigned char* out;          // may be null
    unsigned char* fwd;          // may be null
    unsigned long long count;    // elements
    unsigned long long chunkElems;
};

// Walks the message chunk by chunk (in order), and inside a chunk in tiles of `tileVecs` 32-byte vectors, tile index
// blockIdx.x, += gridDim.x.  Vector path only (chunk bytes % 32 == 0).
template <int ES>
struct RcTileIt {
    unsigned long long count, chunkElems, c0, t, nvec, tileVecs;
    __device__ __forceinline__ void chunk_begin() {
        const unsigned long long cn = min(chunkElems, count - c0);
        nvec = cn / (32 / ES);
        t = (unsigned long long)blockIdx.x * tileVecs;
    }
    __device__ __forceinline__ void init(const ReduceCopyArgs& p, unsigned long long tileVecs_) {
        count = p.count; chunkElems = p.chunkElems; tileVecs = tileVecs_; c0 = 0;
        chunk_begin();
        settle();
    }
    __device__ __forceinline__ void settle() {             // skip chunks in which this CTA has no tile (left)
        while (t >= nvec) {
            c0 += chunkElems;
            if (c0 >= count) return;
            chunk_begin();
        }
    }
    __device__ __forceinline__ bool valid() const { return c0 < count; }
    __device__ __forceinline__ void advance() { t += (unsigned long long)gridDim.x * tileVecs; settle(); }
    __device__ __forceinline__ unsigned long long byte_off() const { return c0 * ES + t * 32; }   // of the tile's first vector
    __device__ __forceinline__ unsigned long long vecs() const { return min(tileVecs, nvec - t); }
};

template <int DT>
__device__ __forceinline__ u32x8 rc_add(const u32x8& xa, const u32x8& xb) {
    Acc<DT> lo, hi;
    lo.set(xa.lo); hi.set(xa.hi);
    lo.add(xb.lo); hi.add(xb.hi);
    u32x8 o;
    o.lo = lo.pack(); o.hi = hi.pack();
    return o;
}

// elements after the last full 32-byte vector (only the last chunk can have any), scalar
template <int DT>
__device__ __forceinline__ void rc_ragged_tail(const ReduceCopyArgs& p, int tid) {
    constexpr int ES = DT == RED_F32 ? 4 : 2;
    constexpr int EPV = 32 / ES;
    if (blockIdx.x != 0) return;
    const unsigned long long lastC0 = ((p.count - 1) / p.chunkElems) * p.chunkElems;
    const unsigned long long i = lastC0 + ((p.count - lastC0) / EPV) * EPV + tid;
    if (i < p.count) {
        const float acc = __fadd_rn(load_elem<DT>(p.a, i), load_elem<DT>(p.b, i));
        if (p.out) store_elem<DT>(p.out, i, acc);
        if (p.fwd) store_elem<DT>(p.fwd, i, acc);
    }
}

template <int DT>
__global__ void __launch_bounds__(RC_THREADS) reducecopy_kernel(const ReduceCopyArgs p) {
    constexpr int ES = DT == RED_F32 ? 4 : 2;
    const bool vec = ((((unsigned long long)p.a | (unsigned long long)p.b | (unsigned long long)p.out |
                        (unsigned long long)p.fwd) & 31ull) == 0) && ((p.chunkElems * ES) & 31ull) == 0;
    if (vec) {
        // a CTA's tile = RC_UNROLL x 512 vectors, interleaved so that every load instruction is coalesced
        RcTileIt<ES> it;
        it.init(p, (unsigned long long)RC_THREADS * RC_UNROLL);
        u32x8 xa[RC_UNROLL], xb[RC_UNROLL];
        unsigned long long off = 0, nv = 0;
        if (it.valid()) {
            off = it.byte_off(); nv = it.vecs();
#pragma unroll
            for (int u = 0; u < RC_UNROLL; ++u) {
                const unsigned long long v = (unsigned long long)u * RC_THREADS + threadIdx.x;
                if (v < nv) { xa[u] = ld_stream256(p.a + off + v * 32); xb[u] = ld_stream256(p.b + off + v * 32); }
            }
        }
        while (it.valid()) {
            it.advance();
            u32x8 na[RC_UNROLL], nb[RC_UNROLL];
            unsigned long long noff = 0, nnv = 0;
            if (it.valid()) {                              // tile i+1's loads go out before tile i's adds and stores
                noff = it.byte_off(); nnv = it.vecs();
#pragma unroll
                for (int u = 0; u < RC_UNROLL; ++u) {
                    const unsigned long long v = (unsigned long long)u * RC_THREADS + threadIdx.x;
                    if (v < nnv) { na[u] = ld_stream256(p.a + noff + v * 32); nb[u] = ld_stream256(p.b + noff + v * 32); }
                }
            }
#pragma unroll
            for (int u = 0; u < RC_UNROLL; ++u) {
                const unsigned long long v = (unsigned long long)u * RC_THREADS + threadIdx.x;
                if (v < nv) {
                    const u32x8 o = rc_add<DT>(xa[u], xb[u]);
                    if (p.out) st_stream256(p.out + off + v * 32, o);
                    if (p.fwd) st_stream256(p.fwd + off + v * 32, o);
                }
            }
#pragma unroll
            for (int u = 0; u < RC_UNROLL; ++u) { xa[u] = na[u]; xb[u] = nb[u]; }
            off = noff; nv = nnv;
        }
        rc_ragged_tail<DT>(p, threadIdx.x);
    } else {
        for (unsigned long long c0 = 0; c0 < p.count; c0 += p.chunkElems) {        // chunk by chunk, in order
            const unsigned long long cn = min(p.chunkElems, p.count - c0);
            for (unsigned long long i = c0 + (unsigned long long)blockIdx.x * RC_THREADS + threadIdx.x; i < c0 + cn;
                 i += (unsigned long long)gridDim.x * RC_THREADS) {
                const float acc = __fadd_rn(load_elem<DT>(p.a, i), load_elem<DT>(p.b, i));
                if (p.out) store_elem<DT>(p.out, i, acc);
                if (p.fwd) store_elem<DT>(p.fwd, i, acc);
            }
        }
    }
}

// ---- TMA-fed variant ------------------------------------------------------------------------------------------
constexpr int RCT_CONSUMERS = 512;
constexpr int RCT_THREADS = RCT_CONSUMERS + 32;            // + one producer warp
constexpr int RCT_STAGES = 6;
constexpr int RCT_TILE_BYTES = RCT_CONSUMERS * 32;         // per input: one 32-byte vector per consumer thread
constexpr int RCT_SMEM_BYTES = RCT_STAGES * 2 * RCT_TILE_BYTES + 2 * RCT_STAGES * 8 + 128;

// dynamic smem: [stage][a tile | b tile] ... [full mbarriers][empty mbarriers]; requires the vector-path alignment
// (checked by the host)
template <int DT>
__global__ void __launch_bounds__(RCT_THREADS, 1) reducecopy_tma_kernel(const ReduceCopyArgs p) {
    constexpr int ES = DT == RED_F32 ? 4 : 2;
    extern __shared__ __align__(128) unsigned char rct_smem[];
    unsigned long long* full = reinterpret_cast<unsigned long long*>(rct_smem + RCT_STAGES * 2 * RCT_TILE_BYTES);
    unsigned long long* empty = full + RCT_STAGES;
    const int warp = threadIdx.x >> 5, lane = lane_id();
    if (threadIdx.x < RCT_STAGES) {
        mbar_init(smem_u32(&full[threadIdx.x]), 1);
        mbar_init(smem_u32(&empty[threadIdx.x]), RCT_CONSUMERS / 32);
    }
    fence_mbar_init();
    __syncthreads();
    RcTileIt<ES> it;
    it.init(p, RCT_CONSUMERS);
    if (warp == RCT_CONSUMERS / 32) {                      // producer warp: one elected lane issues the bulk loads
        if (lane == 0) {
            for (unsigned int i = 0; it.valid(); ++i, it.advance()) {
                const unsigned int st = i % RCT_STAGES;
                if (i >= RCT_STAGES) mbar_wait(smem_u32(&empty[st]), ((i / RCT_STAGES) - 1) & 1);
                const unsigned int bytes = (unsigned int)it.vecs() * 32u;
                const uint32_t bar = smem_u32(&full[st]);
                const uint32_t dst = smem_u32(rct_smem + (size_t)st * 2 * RCT_TILE_BYTES);
                mbar_expect_tx(bar, 2 * bytes);
                bulk_g2s(dst, p.a + it.byte_off(), bytes, bar);
                bulk_g2s(dst + RCT_TILE_BYTES, p.b + it.byte_off(), bytes, bar);
            }
        }
    } else {
        for (unsigned int i = 0; it.valid(); ++i, it.advance()) {
            const unsigned int st = i % RCT_STAGES;
            mbar_wait(smem_u32(&full[st]), (i / RCT_STAGES) & 1);
            const unsigned long long off = it.byte_off();
            if (threadIdx.x < it.vecs()) {
                const unsigned char* sa = rct_smem + (size_t)st * 2 * RCT_TILE_BYTES + threadIdx.x * 32;
                u32x8 xa, xb;
                xa.lo = *reinterpret_cast<const uint4*>(sa); xa.hi = *reinterpret_cast<const uint4*>(sa + 16);
                xb.lo = *reinterpret_cast<const uint4*>(sa + RCT_TILE_BYTES); xb.hi = *reinterpret_cast<const uint4*>(sa + RCT_TILE_BYTES + 16);
                const u32x8 o = rc_add<DT>(xa, xb);
                if (p.out) st_stream256(p.out + off + threadIdx.x * 32, o);
                if (p.fwd) st_stream256(p.fwd + off + threadIdx.x * 32, o);
            }
            __syncwarp();                                  // the warp's reads of the stage are done
            if (lane == 0) mbar_arrive(smem_u32(&empty[st]));
        }
        rc_ragged_tail<DT>(p, threadIdx.x);
    }
}

}  // namespace xdev
