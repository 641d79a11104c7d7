// ncclx_b200.cu -- host launch layer + C ABI of libncclx_b200.so (see include/ncclx_b200.h).
// Host code only validates arguments and enqueues fixed-grid kernels: no allocation, no
// synchronisation and no host<->device copy on the device entry points, so they are
// CUDA-graph capturable.  There is no CPU fallback.
#include <cuda_runtime.h>

#include <atomic>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <vector>

#include "../../include/ncclx_b200.h"
#include "common.cuh"
#include "copy_kernel.cuh"
#include "counts_kernel.cuh"
#include "dynamic_kernel.cuh"
#include "fused_kernel.cuh"
#include "probe_kernel.cuh"
#include "reduce_kernel.cuh"
#include "topk_kernel.cuh"

using namespace xdev;

namespace {

struct EventPair { cudaEvent_t a, b; };

enum { PLAN_NONE = 0, PLAN_A2A = 1, PLAN_DYN = 2, PLAN_TOPK = 3 };

// Everything a payload launch needs, fixed when the work list is built (prepare): a later ncclx_set_param cannot
// make an existing plan inconsistent.
struct CopyLaunch {
    int ncols = 0, colLen = 0;
    ClassParams cls{};
    unsigned int ringBytes = 0;
    size_t smem = 0;
    int kmax = 0, bulkEngines = 0, pdl = 0, useCoarse = 0;
    const SegDesc* desc = nullptr;
    const int* coarse[2] = {nullptr, nullptr};
    SideJob side{};
};

struct Context {
    bool ready = false;
    int device = -1;
    int maxRanks = 0;
    int smCount = 0;
    int maxSmemOptin = 0;
    Workspace wsPlan[NCCLX_NUM_PLANS]{};  // one workspace per plan slot; slot 0 also serves the one-call entry points
    struct PlanState { int kind = PLAN_NONE; int R = 0; CopyLaunch cl{}; const long long* topkC = nullptr; } plan[NCCLX_NUM_PLANS];
    WorkCtl* fusedCtl = nullptr;          // claim counters of the single-launch path (self-resetting)
    long long* fusedSoff = nullptr;       // the single-launch path's own offset matrices: it leaves every plan slot alone
    long long* fusedRoff = nullptr;
    bool lastOffsetsFused = false;        // which of the two ncclx_alltoallv_last_offsets reads
    void* wsBase = nullptr;
    // tunables (ncclx_param_t order)
    int64_t params[NCCLX_PARAM_COUNT_] = {1024, 16, 0, 15, 1, 6, 32, 0, 1, 0};
    // profiling
    std::vector<EventPair> events[NCCLX_KERNEL_COUNT_];
    std::atomic<int64_t> launches{0};
    long long* rcScratch = nullptr;   // R*R, RC sink for calls that do not return it
    // AllToAllvDynamic workspace (ncclx_init_dynamic): one descriptor table + coarse indexes per plan slot
    void* dynBase = nullptr;
    SegDesc* dynDesc[NCCLX_NUM_PLANS] = {};
    int* dynCoarse[NCCLX_NUM_PLANS][2] = {};
    int dynMaxSplits = 0;
    int64_t dynMaxSegments = 0;
    // host-path staging (device memory, grown on demand)
    void* stage[4] = {nullptr, nullptr, nullptr, nullptr};   // 0 send data, 1 recv data, 2 meta, 3 spare
    size_t stageCap[4] = {0, 0, 0, 0};
    int lastCuda = 0;
    std::mutex mu;                        // every entry point that reads params / plans or launches takes it
};

Context g;
using Lock = std::lock_guard<std::mutex>;

constexpr size_t kMaxProfiledLaunches = 8192;

int cudaFail(cudaError_t e) {
    g.lastCuda = (int)e;
    cudaGetLastError();
    return NCCLX_ERR_CUDA;
}
#define CK(x) do { cudaError_t e_ = (x); if (e_ != cudaSuccess) return cudaFail(e_); } while (0)

int elemSizeOf(int dtype) {
    switch (dtype) {
    case NCCLX_BF16: return 2;
    case NCCLX_F32: return 4;
    case NCCLX_F16: return 2;
    case NCCLX_U8: return 1;
    default: return 0;
    }
}

size_t alignUp(size_t v, size_t a) { return (v + a - 1) / a * a; }

bool isCapturing(cudaStream_t s) {
    cudaStreamCaptureStatus st = cudaStreamCaptureStatusNone;
    if (cudaStreamIsCapturing(s, &st) != cudaSuccess) { cudaGetLastError(); return false; }
    return st != cudaStreamCaptureStatusNone;
}

// Brackets a launch with events when profiling is on and the stream is not capturing; a launch is counted only once
// it has succeeded (ok()).
struct LaunchScope {
    int kernel;
    cudaStream_t stream;
    bool timed = false, good = false;
    EventPair ev{};
    LaunchScope(int k, cudaStream_t s) : kernel(k), stream(s) {
        if (g.params[NCCLX_PARAM_PROFILE] && g.events[k].size() < kMaxProfiledLaunches && !isCapturing(s)) {
            if (cudaEventCreate(&ev.a) == cudaSuccess && cudaEventCreate(&ev.b) == cudaSuccess) {
                timed = true;
                cudaEventRecord(ev.a, s);
            }
        }
    }
    void ok() { good = true; g.launches.fetch_add(1, std::memory_order_relaxed); }
    ~LaunchScope() {
        if (!timed) return;
        if (good) { cudaEventRecord(ev.b, stream); g.events[kernel].push_back(ev); }
        else { cudaEventDestroy(ev.a); cudaEventDestroy(ev.b); }
    }
};

constexpr size_t kMaxCoarseBytes = 16 * 1024;     // both coarse indexes; larger tables fall back to the L2 search
constexpr int kVecTileShift = 14;                 // vector-list work unit: 16 KiB (staged in 2 KiB pieces)
constexpr int kCountsBlockSumMinRanks = 128;      // above this many ranks the counts kernel's phase 1 goes through block sums + a grid barrier
constexpr int kScanCtas = 32;                     // upper bound on CTAs of the counts kernel
constexpr int kFusedMinTileShift = 12;            // smallest bulk tile the single-launch path may choose

size_t coarseBytes(int ncols, int colLen) {        // 0: not staged (trivial for colLen <= 32, or too large)
    const int nb = coarse_blocks(colLen);
    const size_t b = 2 * (size_t)ncols * nb * 4;
    return (nb > 1 && b <= kMaxCoarseBytes) ? b : 0;
}
size_t copyAuxBytes(int ncols, int colLen) { return COPY_MBAR_BYTES + 2 * (size_t)(ncols + 1) * 4 + coarseBytes(ncols, colLen) + 16; }

// shared memory of one copy CTA: all the SM has, minus room for a co-resident metadata CTA (PDL overlap)
size_t copyBudget() { return (size_t)g.maxSmemOptin - 20 * 1024; }

// Ring size: the budget minus bookkeeping, rounded down to 128 B.
unsigned int chooseRingBytes(int ncols, int colLen) {
    const size_t budget = copyBudget(), aux = copyAuxBytes(ncols, colLen);
    return (unsigned int)(budget > aux ? (budget - aux) & ~(size_t)127 : 0);
}

// What a bulk tile has to fit into (plan_ring in copy_kernel.cuh): ONCE into the smallest share the bulk engines can
// be left with when the vector list has most of the bytes (the vector engines take at most VEC_MAX_IN_BULK_MIX
// sixteenths of the ring; the device then runs one bulk engine), and ~2.5 times into an engine's share of the whole
// ring when the call is all bulk.
bool bulkTileFits(int tileShift, size_t ring, int engines) {
    const size_t unit = (ring / COPY_WARPS) & ~(size_t)127;
    const size_t tile = (size_t)1 << tileShift;
    return tile <= ring - VEC_MAX_IN_BULK_MIX * unit && 5 * tile / 2 <= ring / (size_t)(engines > 0 ? engines : 1);
}

size_t countsSmemBytes(int R, int W) { return 2 * (size_t)R * (W + 1) * 8 + (size_t)(R + W) * 8 + 3 * (size_t)W * ((R + 31) / 32) * 8; }

int countsW(int R) {
    // columns per CTA: spread over at most kScanCtas CTAs (CTA j re-reads the row prefixes C[s][0..d0) from L2: more CTAs
    // = more redundant reads -- one column per CTA at R = 128 was measured 2 us slower), at most 32 columns, and
    // 2*R*(W+1)*8 <= smem
    int W = (R + kScanCtas - 1) / kScanCtas;
    if (W < 1) W = 1;
    if (W > 32) W = 32;
    const size_t budget = (size_t)g.maxSmemOptin - 1024;
    while (W > 1 && countsSmemBytes(R, W) > budget) --W;
    return W;
}

// Tile sizes shared by the metadata kernel (tile prefixes) and the copy kernel: the bulk tile must fit the SMALLEST
// ring any launch can get (max_ranks columns, a full coarse index); see bulkTileFits.
ClassParams classParams() {
    ClassParams c{};
    const size_t worstAux = COPY_MBAR_BYTES + 2 * (size_t)(g.maxRanks + 1) * 4 + kMaxCoarseBytes + 16 + 128;
    const size_t budget = copyBudget();
    const size_t ring = budget > worstAux ? budget - worstAux : 0;
    c.tileShift[0] = (int)g.params[NCCLX_PARAM_BULK_TILE_SHIFT];
    while (c.tileShift[0] > 10 && !bulkTileFits(c.tileShift[0], ring, (int)g.params[NCCLX_PARAM_COPY_BULK_ENGINES])) --c.tileShift[0];
    c.tileShift[1] = kVecTileShift;
    c.bulkMinBytes = g.params[NCCLX_PARAM_BULK_MIN_BYTES] < 16 ? 16 : g.params[NCCLX_PARAM_BULK_MIN_BYTES];
    return c;
}

void setPdl(cudaLaunchConfig_t& cfg, cudaLaunchAttribute* attr, bool on) {
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = on ? 1 : 0;
}

// Host-computable part of a payload launch, checked BEFORE the call's first kernel is enqueued ("nothing is enqueued
// on error"): ring size against the work list's bulk tile.
int planCopy(CopyLaunch& cl, const Workspace& ws, const SegDesc* desc, const int* const coarse[2], int ncols, int colLen,
             const ClassParams& cls) {
    (void)ws;
    cl = CopyLaunch{};
    cl.ncols = ncols; cl.colLen = colLen; cl.cls = cls;
    cl.desc = desc; cl.coarse[0] = coarse[0]; cl.coarse[1] = coarse[1];
    cl.useCoarse = coarseBytes(ncols, colLen) > 0 ? 1 : 0;
    cl.bulkEngines = (int)g.params[NCCLX_PARAM_COPY_BULK_ENGINES];
    cl.kmax = (int)g.params[NCCLX_PARAM_COPY_KMAX];
    cl.pdl = g.params[NCCLX_PARAM_PDL] ? 1 : 0;
    cl.ringBytes = chooseRingBytes(ncols, colLen);
    // the work list's bulk tile must fit this launch's ring (a larger tile could never be staged)
    if (!bulkTileFits(cls.tileShift[0], cl.ringBytes, cl.bulkEngines)) return NCCLX_ERR_ARG;
    if ((size_t)VEC_SUB_BYTES + 256 > ((cl.ringBytes / COPY_WARPS) & ~127u)) return NCCLX_ERR_ARG;
    cl.smem = (size_t)cl.ringBytes + copyAuxBytes(ncols, colLen);
    return NCCLX_OK;
}

int launchCopy(const Workspace& ws, const CopyLaunch& cl, cudaStream_t stream) {
    CopyArgs cp{};
    cp.desc = cl.desc; cp.colTiles[0] = ws.colTiles[0]; cp.colTiles[1] = ws.colTiles[1]; cp.colKiB = ws.colKiB;
    cp.coarse[0] = cl.coarse[0]; cp.coarse[1] = cl.coarse[1];
    cp.useCoarse = cl.useCoarse;
    cp.ctl = ws.ctl; cp.ncols = cl.ncols; cp.colLen = cl.colLen;
    cp.cls = cl.cls;
    cp.bulkEngines = cl.bulkEngines;
    cp.ringBytes = cl.ringBytes;
    cp.kmax = cl.kmax;
    cp.side = cl.side;
    LaunchScope ls(NCCLX_KERNEL_COPY, stream);
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3((unsigned)g.smCount);
    cfg.blockDim = dim3(COPY_THREADS);
    cfg.dynamicSmemBytes = cl.smem;
    cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    setPdl(cfg, attr, cl.pdl != 0);
    CK(cudaLaunchKernelEx(&cfg, segment_copy_kernel, cp));
    ls.ok();
    return NCCLX_OK;
}

int launchCounts(const Workspace& ws, const void* const* send, const int64_t* C, void* const* recv, int64_t* RC, int R,
                 long long es, const ClassParams& cls, cudaStream_t stream) {
    CountsArgs ca{};
    ca.send = send; ca.recv = recv;
    ca.C = reinterpret_cast<const long long*>(C);
    ca.RC = reinterpret_cast<long long*>(RC);
    ca.ws = ws; ca.R = R; ca.W = countsW(R); ca.elemSize = es;
    ca.blockSums = R > kCountsBlockSumMinRanks ? 1 : 0;
    ca.cls = cls;
    const int G = (R + ca.W - 1) / ca.W;
    if (G > COUNTS_MAX_CTAS) return NCCLX_ERR_ARG;        // (cannot happen for R <= NCCLX_MAX_RANKS: W >= 12 there)
    const size_t csm = countsSmemBytes(R, ca.W);
    LaunchScope ls(NCCLX_KERNEL_COUNTS, stream);
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3((unsigned)G);
    cfg.blockDim = dim3(COUNTS_THREADS);
    cfg.dynamicSmemBytes = csm;
    cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    setPdl(cfg, attr, g.params[NCCLX_PARAM_PDL] != 0);   // back-to-back calls: becomes resident while the previous copy kernel drains
    CK(cudaLaunchKernelEx(&cfg, counts_kernel, ca));
    ls.ok();
    return NCCLX_OK;
}

// Single-launch path (fused_kernel.cuh): ring = what is left of the SM's shared memory after the R*R
// descriptors; the maximum bulk tile still has to fit 2.5 times into the smallest bulk share.
int planFused(FusedArgs& fa, int R) {
    fa = FusedArgs{};
    fa.cls = classParams();
    const size_t budget = (size_t)g.maxSmemOptin - 1024;
    const size_t aux = fused_aux_bytes(R);
    if (budget < aux + 64 * 1024) return NCCLX_ERR_ARG;
    fa.ringBytes = (unsigned int)((budget - aux) & ~(size_t)127);
    if ((size_t)VEC_SUB_BYTES + 256 > ((fa.ringBytes / COPY_WARPS) & ~127u)) return NCCLX_ERR_ARG;   // as planCopy: a vector engine's share must hold one staged piece
    fa.bulkEngines = (int)g.params[NCCLX_PARAM_COPY_BULK_ENGINES];
    while (fa.cls.tileShift[0] > 10 && !bulkTileFits(fa.cls.tileShift[0], fa.ringBytes, fa.bulkEngines)) --fa.cls.tileShift[0];
    fa.kmax = (int)g.params[NCCLX_PARAM_COPY_KMAX];
    fa.minTileShift[0] = kFusedMinTileShift < fa.cls.tileShift[0] ? kFusedMinTileShift : fa.cls.tileShift[0];
    fa.minTileShift[1] = 10 < fa.cls.tileShift[1] ? 10 : fa.cls.tileShift[1];
    return NCCLX_OK;
}

int launchFused(FusedArgs& fa, const void* const* send, const int64_t* C, void* const* recv, int64_t* RC, int R, int es,
                cudaStream_t stream) {
    fa.send = send; fa.recv = recv;
    fa.C = reinterpret_cast<const long long*>(C);
    fa.RC = reinterpret_cast<long long*>(RC);
    fa.soff = g.fusedSoff; fa.roff = g.fusedRoff;
    fa.ctl = g.fusedCtl; fa.status = &g.wsPlan[0].ctl->status;
    fa.R = R; fa.elemSize = es;
    LaunchScope ls(NCCLX_KERNEL_FUSED, stream);
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3((unsigned)g.smCount);
    cfg.blockDim = dim3(COPY_THREADS);
    cfg.dynamicSmemBytes = (size_t)fa.ringBytes + fused_aux_bytes(R);
    cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    setPdl(cfg, attr, g.params[NCCLX_PARAM_PDL] != 0);
    CK(cudaLaunchKernelEx(&cfg, alltoallv_fused_kernel, fa));
    ls.ok();
    g.lastOffsetsFused = true;
    return NCCLX_OK;
}

// a1-a3 into plan slot `p` (validated first), optionally followed by a4.
int prepareA2A(int p, const void* const* send, const int64_t* C, void* const* recv, int64_t* RC, int R, int es,
               cudaStream_t stream) {
    Context::PlanState& ps = g.plan[p];
    const Workspace& ws = g.wsPlan[p];
    CopyLaunch cl;
    int rc = planCopy(cl, ws, ws.desc, ws.coarse, R, R, classParams());
    if (rc) return rc;
    ps.kind = PLAN_NONE;
    rc = launchCounts(ws, send, C, recv, RC, R, es, cl.cls, stream);
    if (rc) return rc;
    ps.kind = PLAN_A2A; ps.R = R; ps.cl = cl;
    if (p == 0) g.lastOffsetsFused = false;
    return NCCLX_OK;
}

int launchAllToAllv(const void* const* send, const int64_t* C, void* const* recv, int64_t* RC, int R, int es,
                    cudaStream_t stream) {
    if (R <= FUSED_MAX_R && R <= (int)g.params[NCCLX_PARAM_FUSED_MAX_RANKS]) {
        FusedArgs fa;
        int rc = planFused(fa, R);
        if (rc) return rc;
        return launchFused(fa, send, C, recv, RC, R, es, stream);
    }
    int rc = prepareA2A(0, send, C, recv, RC, R, es, stream);
    if (rc) return rc;
    return launchCopy(g.wsPlan[0], g.plan[0].cl, stream);
}

constexpr size_t kReducePdlMaxBytes = (size_t)1 << 30;   // reductions below this many input bytes launch with PDL
constexpr size_t kReducePrefetchAllBytes = (size_t)96 << 20;
constexpr size_t kReduceShortBytes = (size_t)256 << 20;   // reductions below this many input bytes run on 64-thread CTAs

template <int DT, int TH>
int launchReduceDT(const ReduceArgs& ra, int grid, size_t smem, bool pdl, cudaStream_t stream) {
    LaunchScope ls(NCCLX_KERNEL_REDUCE, stream);
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3((unsigned)grid);
    cfg.blockDim = dim3(TH);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    setPdl(cfg, attr, pdl);
    if (ra.R <= 4) CK(cudaLaunchKernelEx(&cfg, reduce_kernel<DT, 4, TH>, ra));
    else if (ra.R <= 8) CK(cudaLaunchKernelEx(&cfg, reduce_kernel<DT, 8, TH>, ra));
    else CK(cudaLaunchKernelEx(&cfg, reduce_kernel<DT, 16, TH>, ra));
    ls.ok();
    return NCCLX_OK;
}

int launchReduce(const void* const* send, void* const* recv, size_t blockElems, int R, int dtype, int scatter,
                 cudaStream_t stream) {
    if (blockElems == 0) return NCCLX_OK;
    ReduceArgs ra{};
    ra.send = send; ra.recv = recv; ra.blockElems = blockElems; ra.R = R; ra.scatter = scatter;
    const int es = elemSizeOf(dtype);
    const unsigned long long totalVec = ((unsigned long long)blockElems * (scatter ? R : 1) * es + 31) / 32;
    const size_t inBytes0 = (size_t)blockElems * (scatter ? R : 1) * es * (size_t)R;
    const bool shortCall = inBytes0 < kReduceShortBytes;        // short: 64-thread CTAs, twice as many
    const unsigned long long th = shortCall ? REDUCE_THREADS_SHORT : REDUCE_THREADS;
    unsigned long long tiles = (totalVec + th - 1) / th + (scatter ? R : 0);
    unsigned long long grid = (unsigned long long)g.smCount * (unsigned long long)g.params[NCCLX_PARAM_REDUCE_CTAS_PER_SM] * (shortCall ? 2 : 1);
    if (grid > tiles) grid = tiles;
    if (grid < 1) grid = 1;
    const size_t smem = 2 * (size_t)R * sizeof(void*);
    // programmatic dependent launch hides ~0.5 us of the launch gap between back-to-back SHORT reductions (config 2:
    // a 20 us kernel) but costs a long one 0.3-0.6 % (config 4: the next kernel's CTAs take SM slots early), and
    // the host knows the size: gate it
    const size_t inBytes = (size_t)blockElems * (scatter ? R : 1) * es * (size_t)R;
    const bool pdl = g.params[NCCLX_PARAM_PDL] != 0 && inBytes < kReducePdlMaxBytes;
    // under PDL the CTAs prefetch their first tiles into L2 before the dependency wait: everything when the input fits
    // L2 comfortably, else the first two tiles (the first wave)
    if (pdl) {                                             // every CTA its own first tiles (all of them when the input fits L2)
        ra.prefetchCtas = (int)grid;
        ra.prefetchTiles = inBytes <= kReducePrefetchAllBytes ? (int)((tiles + grid - 1) / grid) : 2;
    }
    switch (dtype) {
    case NCCLX_BF16: return shortCall ? launchReduceDT<RED_BF16, REDUCE_THREADS_SHORT>(ra, (int)grid, smem, pdl, stream)
                                      : launchReduceDT<RED_BF16, REDUCE_THREADS>(ra, (int)grid, smem, pdl, stream);
    case NCCLX_F32: return shortCall ? launchReduceDT<RED_F32, REDUCE_THREADS_SHORT>(ra, (int)grid, smem, pdl, stream)
                                     : launchReduceDT<RED_F32, REDUCE_THREADS>(ra, (int)grid, smem, pdl, stream);
    case NCCLX_F16: return shortCall ? launchReduceDT<RED_F16, REDUCE_THREADS_SHORT>(ra, (int)grid, smem, pdl, stream)
                                     : launchReduceDT<RED_F16, REDUCE_THREADS>(ra, (int)grid, smem, pdl, stream);
    default: return NCCLX_ERR_DTYPE;
    }
}

int ensureStage(int i, size_t bytes) {
    if (bytes <= g.stageCap[i]) return NCCLX_OK;
    if (g.stage[i]) { CK(cudaFree(g.stage[i])); g.stage[i] = nullptr; g.stageCap[i] = 0; }
    const size_t cap = alignUp(bytes, (size_t)2 << 20);
    CK(cudaMalloc(&g.stage[i], cap));
    g.stageCap[i] = cap;
    return NCCLX_OK;
}

// Device-visible address of a pinned (cudaHostAlloc / cudaHostRegister) host buffer, or nullptr when the
// memory is pageable: pinned buffers are read and written by the kernels DIRECTLY over PCIe (zero-copy: the
// H2D and D2H halves of the call overlap on the full-duplex link), pageable ones go through device staging.
void* mappedDevicePtr(const void* host) {
    cudaPointerAttributes at{};
    if (cudaPointerGetAttributes(&at, host) != cudaSuccess) { cudaGetLastError(); return nullptr; }
    if (at.type != cudaMemoryTypeHost || !at.devicePointer) return nullptr;
    return at.devicePointer;
}

int checkCommon(int R) {
    if (!g.ready) return NCCLX_ERR_NOT_INITIALIZED;
    if (R < 1) return NCCLX_ERR_ARG;
    if (R > g.maxRanks) return NCCLX_ERR_NOT_INITIALIZED;
    return NCCLX_OK;
}

void freeAll() {
    if (g.wsBase) { cudaFree(g.wsBase); g.wsBase = nullptr; }
    if (g.dynBase) { cudaFree(g.dynBase); g.dynBase = nullptr; g.dynMaxSplits = 0; g.dynMaxSegments = 0; }
    for (int i = 0; i < 4; ++i) {
        if (g.stage[i]) { cudaFree(g.stage[i]); g.stage[i] = nullptr; g.stageCap[i] = 0; }
    }
    for (auto& v : g.events) {
        for (auto& e : v) { cudaEventDestroy(e.a); cudaEventDestroy(e.b); }
        v.clear();
    }
    for (auto& ps : g.plan) ps = Context::PlanState{};
    cudaGetLastError();
    g.ready = false;
}

template <typename K>
int optInSmem(K kernel, int bytes) {
    cudaFuncAttributes fa{};
    CK(cudaFuncGetAttributes(&fa, kernel));
    const int room = g.maxSmemOptin - (int)fa.sharedSizeBytes;    // static + dynamic shared memory share the opt-in limit
    CK(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes < room ? bytes : room));
    return NCCLX_OK;
}

int topkCommon(int R, int T, int k, int width, int es) {
    int rc = checkCommon(R);
    if (rc) return rc;
    if (T < 0 || k < 1 || k > 32 || width < 1) return NCCLX_ERR_ARG;
    if (!es) return NCCLX_ERR_DTYPE;
    return NCCLX_OK;
}

constexpr int kTopkCtasPerSm = 16;

int topkGrid(long long tokens) {
    long long ctas = (tokens + TOPK_THREADS / 32 - 1) / (TOPK_THREADS / 32);
    const long long cap = (long long)g.smCount * kTopkCtasPerSm;
    return (int)(ctas < 1 ? 1 : (ctas > cap ? cap : ctas));
}

template <typename K>
int launchTopk(K kernel, const TopkArgs& ta, cudaStream_t s) {
    LaunchScope ls(NCCLX_KERNEL_TOPK, s);
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3((unsigned)topkGrid((long long)ta.R * ta.T));
    cfg.blockDim = dim3(TOPK_THREADS);
    cfg.stream = s;
    cudaLaunchAttribute attr[1];
    setPdl(cfg, attr, g.params[NCCLX_PARAM_PDL] != 0);
    CK(cudaLaunchKernelEx(&cfg, kernel, ta));
    ls.ok();
    return NCCLX_OK;
}

// a1/a2 of a top-k call into plan slot p: offsets in ROWS (count unit = one row); the descriptor table is not used.
int prepareTopk(int p, const int64_t* C, int64_t* RC, int R, cudaStream_t s) {
    Context::PlanState& ps = g.plan[p];
    ps.kind = PLAN_NONE;
    int rc = launchCounts(g.wsPlan[p], nullptr, C, nullptr, RC, R, 1, classParams(), s);
    if (rc) return rc;
    ps.kind = PLAN_TOPK; ps.R = R; ps.topkC = reinterpret_cast<const long long*>(C);
    return NCCLX_OK;
}

TopkArgs topkArgs(int p, const int32_t* pos, int R, int T, int k, long long rowBytes) {
    TopkArgs ta{};
    ta.pos = pos;
    ta.C = g.plan[p].topkC;                // the count matrix given to prepare (by reference, for the range check)
    ta.soff = g.wsPlan[p].soff; ta.roff = g.wsPlan[p].roff; ta.ctl = g.wsPlan[p].ctl;
    ta.R = R; ta.T = T; ta.k = k; ta.rowBytes = rowBytes;
    return ta;
}

int launchTopkDispatch(int p, const void* const* tokens, const int32_t* pos, void* const* recv, int R, int T, int k,
                       long long rowBytes, cudaStream_t s) {
    if (T == 0) return NCCLX_OK;
    TopkArgs ta = topkArgs(p, pos, R, T, k, rowBytes);
    ta.tokens = tokens; ta.packed = recv; ta.out = nullptr;
    return launchTopk(topk_dispatch_kernel, ta, s);
}

int launchTopkCombine(int p, const void* const* expert_out, const int32_t* pos, void* const* out, int R, int T, int k,
                      long long rowBytes, int dtype, cudaStream_t s) {
    if (T == 0) return NCCLX_OK;
    TopkArgs ta = topkArgs(p, pos, R, T, k, rowBytes);
    ta.tokens = nullptr; ta.packed = const_cast<void* const*>(expert_out); ta.out = out;
    switch (dtype) {
    case NCCLX_BF16: return launchTopk(topk_combine_kernel<RED_BF16>, ta, s);
    case NCCLX_F32: return launchTopk(topk_combine_kernel<RED_F32>, ta, s);
    default: return launchTopk(topk_combine_kernel<RED_F16>, ta, s);
    }
}

// AllToAllvDynamic metadata phase into plan slot p: ONE kernel builds the (s, d, j) descriptor table; the
// recvAllSplitLengths broadcast is attached to the payload launch as its side job.
int prepareDynamic(int p, const void* const* send, const int64_t* L, int nsplits, const int64_t* indices, int maxIndices,
                   const int64_t* blockLens, int maxBlockLen, void* const* recvbuffs, int64_t* recvAll, int R, int es,
                   cudaStream_t s) {
    Context::PlanState& ps = g.plan[p];
    Workspace ws = g.wsPlan[p];
    ws.desc = g.dynDesc[p]; ws.coarse[0] = g.dynCoarse[p][0]; ws.coarse[1] = g.dynCoarse[p][1];
    const int colLen = R * maxBlockLen;
    CopyLaunch cl;
    int rc = planCopy(cl, ws, ws.desc, ws.coarse, R, colLen, classParams());
    if (rc) return rc;
    cl.side.src = reinterpret_cast<const long long*>(L);
    cl.side.dst = reinterpret_cast<long long*>(recvAll);
    cl.side.n = (long long)R * nsplits;
    cl.side.copies = R;
    DynArgs da{};
    da.send = send; da.recvbuffs = recvbuffs;
    da.L = reinterpret_cast<const long long*>(L);
    da.indices = reinterpret_cast<const long long*>(indices);
    da.blockLens = reinterpret_cast<const long long*>(blockLens);
    da.ws = ws;
    da.R = R; da.n = nsplits; da.maxIndices = maxIndices; da.maxBlockLen = maxBlockLen; da.elemSize = es;
    da.cls = cl.cls;
    ps.kind = PLAN_NONE;
    {
        LaunchScope ls(NCCLX_KERNEL_DYN, s);
        cudaLaunchConfig_t cfg{};
        cfg.gridDim = dim3((unsigned)R);
        cfg.blockDim = dim3(DYN_THREADS);
        cfg.dynamicSmemBytes = dyn_smem_bytes(colLen);
        cfg.stream = s;
        cudaLaunchAttribute attr[1];
        setPdl(cfg, attr, g.params[NCCLX_PARAM_PDL] != 0);
        CK(cudaLaunchKernelEx(&cfg, dyn_build_kernel, da));
        ls.ok();
    }
    ps.kind = PLAN_DYN; ps.R = R; ps.cl = cl;
    return NCCLX_OK;
}

int checkDynamic(const void* const* send, const int64_t* L, int nsplits, const int64_t* indices, int maxIndices,
                 const int64_t* blockLens, int maxBlockLen, void* const* recvbuffs, int64_t* recvAll, int R, int es) {
    int rc = checkCommon(R);
    if (rc) return rc;
    if (!send || !L || !indices || !blockLens || !recvbuffs || !recvAll) return NCCLX_ERR_ARG;
    if (nsplits < 1 || maxIndices < 1 || maxBlockLen < 1) return NCCLX_ERR_ARG;
    if (!g.dynBase || nsplits > g.dynMaxSplits || (int64_t)R * R * maxBlockLen > g.dynMaxSegments)
        return NCCLX_ERR_NOT_INITIALIZED;
    if (!es) return NCCLX_ERR_DTYPE;
    return NCCLX_OK;
}

}  // namespace

extern "C" {

int ncclx_version(void) { return NCCLX_B200_VERSION; }

const char* ncclx_strerror(int code) {
    switch (code) {
    case NCCLX_OK: return "ok";
    case NCCLX_ERR_ARG: return "invalid argument";
    case NCCLX_ERR_DTYPE: return "unsupported dtype for this call";
    case NCCLX_ERR_NOT_INITIALIZED: return "not initialised, or R / work-list size exceeds what init was given";
    case NCCLX_ERR_CUDA: return "CUDA runtime error";
    case NCCLX_ERR_CAPTURE: return "host-synchronous call while the stream is capturing";
    case NCCLX_ERR_TOO_LARGE: return "R exceeds NCCLX_STATIC_MAX_RANKS (32), the fixed capacity of ncclx_alltoallv_static_dev's built-in scratch";
    default: return "unknown error code";
    }
}

int ncclx_last_cuda_error(void) { return g.lastCuda; }
const char* ncclx_last_cuda_error_string(void) { return cudaGetErrorString((cudaError_t)g.lastCuda); }

static int initLocked(int max_ranks, int device) {
    CK(cudaSetDevice(device));
    cudaDeviceProp prop{};
    CK(cudaGetDeviceProperties(&prop, device));
    if (prop.major < 10) { g.lastCuda = (int)cudaErrorNoKernelImageForDevice; return NCCLX_ERR_CUDA; }
    g.device = device;
    g.smCount = prop.multiProcessorCount;
    g.maxSmemOptin = (int)prop.sharedMemPerBlockOptin;
    g.maxRanks = max_ranks;

    const size_t rr = (size_t)max_ranks * max_ranks;
    size_t off = 0;
    size_t oSoff[NCCLX_NUM_PLANS], oRoff[NCCLX_NUM_PLANS], oDesc[NCCLX_NUM_PLANS], oCt0[NCCLX_NUM_PLANS],
        oCt1[NCCLX_NUM_PLANS], oCtl[NCCLX_NUM_PLANS], oCo0[NCCLX_NUM_PLANS], oCo1[NCCLX_NUM_PLANS], oKib[NCCLX_NUM_PLANS], oBs[NCCLX_NUM_PLANS];
    const size_t coarseInts = (size_t)max_ranks * coarse_blocks(max_ranks);
    for (int p = 0; p < NCCLX_NUM_PLANS; ++p) {
        oSoff[p] = off; off = alignUp(off + rr * 8, 256);
        oRoff[p] = off; off = alignUp(off + rr * 8, 256);
        oDesc[p] = off; off = alignUp(off + rr * sizeof(SegDesc), 256);
        oCt0[p] = off; off = alignUp(off + (size_t)max_ranks * 4, 256);
        oCt1[p] = off; off = alignUp(off + (size_t)max_ranks * 4, 256);
        oKib[p] = off; off = alignUp(off + (size_t)max_ranks * 4, 256);
        oCtl[p] = off; off = alignUp(off + sizeof(WorkCtl), 256);
        oCo0[p] = off; off = alignUp(off + coarseInts * 4, 256);
        oCo1[p] = off; off = alignUp(off + coarseInts * 4, 256);
        oBs[p] = off; off = alignUp(off + (size_t)COUNTS_MAX_CTAS * max_ranks * 8, 256);
    }
    const size_t oFctl = off; off = alignUp(off + sizeof(WorkCtl), 256);
    const size_t oRcs = off; off = alignUp(off + rr * 8, 256);
    const size_t fusedRR = (size_t)FUSED_MAX_R * FUSED_MAX_R * 8;
    const size_t oFso = off; off = alignUp(off + fusedRR, 256);
    const size_t oFro = off; off = alignUp(off + fusedRR, 256);
    CK(cudaMalloc(&g.wsBase, off));
    CK(cudaMemset(g.wsBase, 0, off));
    char* b = static_cast<char*>(g.wsBase);
    for (int p = 0; p < NCCLX_NUM_PLANS; ++p) {
        Workspace& w = g.wsPlan[p];
        w.soff = reinterpret_cast<long long*>(b + oSoff[p]);
        w.roff = reinterpret_cast<long long*>(b + oRoff[p]);
        w.desc = reinterpret_cast<SegDesc*>(b + oDesc[p]);
        w.colTiles[0] = reinterpret_cast<int*>(b + oCt0[p]);
        w.colTiles[1] = reinterpret_cast<int*>(b + oCt1[p]);
        w.colKiB = reinterpret_cast<int*>(b + oKib[p]);
        w.ctl = reinterpret_cast<WorkCtl*>(b + oCtl[p]);
        w.coarse[0] = reinterpret_cast<int*>(b + oCo0[p]);
        w.coarse[1] = reinterpret_cast<int*>(b + oCo1[p]);
        w.blockSum = reinterpret_cast<long long*>(b + oBs[p]);
        g.plan[p] = Context::PlanState{};
    }
    g.fusedCtl = reinterpret_cast<WorkCtl*>(b + oFctl);
    g.rcScratch = reinterpret_cast<long long*>(b + oRcs);
    g.fusedSoff = reinterpret_cast<long long*>(b + oFso);
    g.fusedRoff = reinterpret_cast<long long*>(b + oFro);
    g.lastOffsetsFused = false;

    int rc;
    if ((rc = optInSmem(segment_copy_kernel, g.maxSmemOptin))) return rc;
    if ((rc = optInSmem(counts_kernel, g.maxSmemOptin))) return rc;
    if ((rc = optInSmem(alltoallv_fused_kernel, g.maxSmemOptin))) return rc;
    if ((rc = optInSmem(dyn_build_kernel, (int)dyn_smem_bytes(DYN_SMEM_SLOTS)))) return rc;
    if ((rc = optInSmem(reducecopy_tma_kernel<RED_BF16>, RCT_SMEM_BYTES))) return rc;
    if ((rc = optInSmem(reducecopy_tma_kernel<RED_F32>, RCT_SMEM_BYTES))) return rc;
    if ((rc = optInSmem(reducecopy_tma_kernel<RED_F16>, RCT_SMEM_BYTES))) return rc;
    CK(cudaDeviceSynchronize());
    g.launches = 0;
    return NCCLX_OK;
}

int ncclx_init(int max_ranks, int device) {
    Lock lk(g.mu);
    if (max_ranks < 1 || max_ranks > NCCLX_MAX_RANKS) return NCCLX_ERR_ARG;
    if (g.ready || g.wsBase) freeAll();
    const int rc = initLocked(max_ranks, device);
    if (rc) { freeAll(); return rc; }                      // no workspace is left behind by a failed init
    g.ready = true;
    return NCCLX_OK;
}

int ncclx_finalize(void) {
    Lock lk(g.mu);
    if (!g.ready) return NCCLX_ERR_NOT_INITIALIZED;
    cudaDeviceSynchronize();
    freeAll();
    return NCCLX_OK;
}

int ncclx_sm_count(void) { return g.ready ? g.smCount : 0; }

int ncclx_alltoallv_dev(const void* const* send, const int64_t* sendcounts_dev, void* const* recv,
                        int64_t* recvcounts_dev, int R, ncclx_dtype_t dtype, ncclx_stream_t stream) {
    Lock lk(g.mu);
    int rc = checkCommon(R);
    if (rc) return rc;
    if (!send || !sendcounts_dev || !recv || !recvcounts_dev) return NCCLX_ERR_ARG;
    if (sendcounts_dev == recvcounts_dev) return NCCLX_ERR_ARG;
    const int es = elemSizeOf((int)dtype);
    if (!es) return NCCLX_ERR_DTYPE;
    return launchAllToAllv(send, sendcounts_dev, recv, recvcounts_dev, R, es, static_cast<cudaStream_t>(stream));
}

int ncclx_alltoallv_prepare_dev(int plan, const void* const* send, const int64_t* sendcounts_dev, void* const* recv,
                                int64_t* recvcounts_dev, int R, ncclx_dtype_t dtype, ncclx_stream_t stream) {
    Lock lk(g.mu);
    int rc = checkCommon(R);
    if (rc) return rc;
    if (plan < 0 || plan >= NCCLX_NUM_PLANS) return NCCLX_ERR_ARG;
    if (!send || !sendcounts_dev || !recv || !recvcounts_dev) return NCCLX_ERR_ARG;
    if (sendcounts_dev == recvcounts_dev) return NCCLX_ERR_ARG;
    const int es = elemSizeOf((int)dtype);
    if (!es) return NCCLX_ERR_DTYPE;
    return prepareA2A(plan, send, sendcounts_dev, recv, recvcounts_dev, R, es, static_cast<cudaStream_t>(stream));
}

int ncclx_alltoallv_execute_dev(int plan, ncclx_stream_t stream) {
    Lock lk(g.mu);
    if (!g.ready) return NCCLX_ERR_NOT_INITIALIZED;
    if (plan < 0 || plan >= NCCLX_NUM_PLANS) return NCCLX_ERR_ARG;
    const Context::PlanState& ps = g.plan[plan];
    if (ps.kind != PLAN_A2A && ps.kind != PLAN_DYN) return NCCLX_ERR_ARG;
    return launchCopy(g.wsPlan[plan], ps.cl, static_cast<cudaStream_t>(stream));
}

int ncclx_alltoallv_last_offsets(int64_t* soff_host, int64_t* roff_host, int R, ncclx_stream_t stream) {
    Lock lk(g.mu);
    int rc = checkCommon(R);
    if (rc) return rc;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    if (isCapturing(s)) return NCCLX_ERR_CAPTURE;
    CK(cudaStreamSynchronize(s));
    const size_t bytes = (size_t)R * R * 8;
    if (g.lastOffsetsFused && R > FUSED_MAX_R) return NCCLX_ERR_ARG;       // the last call had at most 32 ranks
    if (soff_host) CK(cudaMemcpy(soff_host, g.lastOffsetsFused ? g.fusedSoff : g.wsPlan[0].soff, bytes, cudaMemcpyDeviceToHost));
    if (roff_host) CK(cudaMemcpy(roff_host, g.lastOffsetsFused ? g.fusedRoff : g.wsPlan[0].roff, bytes, cudaMemcpyDeviceToHost));
    return NCCLX_OK;
}

int ncclx_device_status(uint32_t* status_host, ncclx_stream_t stream) {
    Lock lk(g.mu);
    if (!g.ready) return NCCLX_ERR_NOT_INITIALIZED;
    if (!status_host) return NCCLX_ERR_ARG;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    if (isCapturing(s)) return NCCLX_ERR_CAPTURE;
    CK(cudaStreamSynchronize(s));
    uint32_t all = 0;
    for (int p = 0; p < NCCLX_NUM_PLANS; ++p) {
        uint32_t v = 0;
        CK(cudaMemcpy(&v, &g.wsPlan[p].ctl->status, 4, cudaMemcpyDeviceToHost));
        if (v) CK(cudaMemset(&g.wsPlan[p].ctl->status, 0, 4));
        all |= v;
    }
    *status_host = all;
    return NCCLX_OK;
}

int ncclx_init_dynamic(int max_splits, int64_t max_segments) {
    Lock lk(g.mu);
    if (!g.ready) return NCCLX_ERR_NOT_INITIALIZED;
    if (max_splits < 1 || max_segments < 1 || max_segments > ((int64_t)1 << 28)) return NCCLX_ERR_ARG;
    if (g.dynBase) { CK(cudaFree(g.dynBase)); g.dynBase = nullptr; g.dynMaxSplits = 0; g.dynMaxSegments = 0; }
    for (auto& ps : g.plan) if (ps.kind == PLAN_DYN) ps.kind = PLAN_NONE;
    size_t off = 0, oD[NCCLX_NUM_PLANS], oC0[NCCLX_NUM_PLANS], oC1[NCCLX_NUM_PLANS];
    const size_t dynCoarseInts = (size_t)max_segments / 32 + g.maxRanks + 32;   // ncols * ceil(colLen/32) <= segments/32 + ncols
    for (int p = 0; p < NCCLX_NUM_PLANS; ++p) {
        oD[p] = off; off = alignUp(off + (size_t)max_segments * sizeof(SegDesc), 256);
        oC0[p] = off; off = alignUp(off + dynCoarseInts * 4, 256);
        oC1[p] = off; off = alignUp(off + dynCoarseInts * 4, 256);
    }
    CK(cudaMalloc(&g.dynBase, off));
    if (cudaMemset(g.dynBase, 0, off) != cudaSuccess) {
        const cudaError_t e = cudaGetLastError();
        cudaFree(g.dynBase); g.dynBase = nullptr;
        return cudaFail(e);
    }
    char* b = static_cast<char*>(g.dynBase);
    for (int p = 0; p < NCCLX_NUM_PLANS; ++p) {
        g.dynDesc[p] = reinterpret_cast<SegDesc*>(b + oD[p]);
        g.dynCoarse[p][0] = reinterpret_cast<int*>(b + oC0[p]);
        g.dynCoarse[p][1] = reinterpret_cast<int*>(b + oC1[p]);
    }
    g.dynMaxSplits = max_splits;
    g.dynMaxSegments = max_segments;
    return NCCLX_OK;
}

int ncclx_alltoallv_dynamic_prepare_dev(int plan, const void* const* send, const int64_t* sendSplitLengths_dev, int nsplits,
                                        const int64_t* sendIndices_dev, int maxIndices,
                                        const int64_t* sendIndicesBlockLens_dev, int maxBlockLen, void* const* recvbuffs,
                                        int64_t* recvAllSplitLengths_dev, int R, ncclx_dtype_t dtype, ncclx_stream_t stream) {
    Lock lk(g.mu);
    const int es = elemSizeOf((int)dtype);
    int rc = checkDynamic(send, sendSplitLengths_dev, nsplits, sendIndices_dev, maxIndices, sendIndicesBlockLens_dev, maxBlockLen,
                          recvbuffs, recvAllSplitLengths_dev, R, es);
    if (rc) return rc;
    if (plan < 0 || plan >= NCCLX_NUM_PLANS) return NCCLX_ERR_ARG;
    return prepareDynamic(plan, send, sendSplitLengths_dev, nsplits, sendIndices_dev, maxIndices, sendIndicesBlockLens_dev,
                          maxBlockLen, recvbuffs, recvAllSplitLengths_dev, R, es, static_cast<cudaStream_t>(stream));
}

int ncclx_alltoallv_dynamic_dev(const void* const* send, const int64_t* sendSplitLengths_dev, int nsplits,
                                const int64_t* sendIndices_dev, int maxIndices,
                                const int64_t* sendIndicesBlockLens_dev, int maxBlockLen, void* const* recvbuffs,
                                int64_t* recvAllSplitLengths_dev, int R, ncclx_dtype_t dtype, ncclx_stream_t stream) {
    Lock lk(g.mu);
    const int es = elemSizeOf((int)dtype);
    int rc = checkDynamic(send, sendSplitLengths_dev, nsplits, sendIndices_dev, maxIndices, sendIndicesBlockLens_dev, maxBlockLen,
                          recvbuffs, recvAllSplitLengths_dev, R, es);
    if (rc) return rc;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    rc = prepareDynamic(0, send, sendSplitLengths_dev, nsplits, sendIndices_dev, maxIndices, sendIndicesBlockLens_dev,
                        maxBlockLen, recvbuffs, recvAllSplitLengths_dev, R, es, s);
    if (rc) return rc;
    return launchCopy(g.wsPlan[0], g.plan[0].cl, s);
}

int ncclx_allreduce_sum(const void* const* send, void* const* recv, size_t count, int R, ncclx_dtype_t dtype,
                        ncclx_stream_t stream) {
    Lock lk(g.mu);
    int rc = checkCommon(R);
    if (rc) return rc;
    if (!send || !recv) return NCCLX_ERR_ARG;
    if (!(dtype == NCCLX_BF16 || dtype == NCCLX_F32 || dtype == NCCLX_F16)) return NCCLX_ERR_DTYPE;
    return launchReduce(send, recv, count, R, (int)dtype, 0, static_cast<cudaStream_t>(stream));
}

int ncclx_reducescatter_sum(const void* const* send, void* const* recv, size_t recvcount, int R,
                            ncclx_dtype_t dtype, ncclx_stream_t stream) {
    Lock lk(g.mu);
    int rc = checkCommon(R);
    if (rc) return rc;
    if (!send || !recv) return NCCLX_ERR_ARG;
    if (!(dtype == NCCLX_BF16 || dtype == NCCLX_F32 || dtype == NCCLX_F16)) return NCCLX_ERR_DTYPE;
    return launchReduce(send, recv, recvcount, R, (int)dtype, 1, static_cast<cudaStream_t>(stream));
}

int ncclx_moe_dispatch_topk_dev(const void* const* tokens, const int32_t* pos_dev, const int64_t* sendcounts_rows_dev,
                                void* const* recv, int64_t* recvcounts_rows_dev, int R, int T, int k, int width,
                                ncclx_dtype_t dtype, ncclx_stream_t stream) {
    Lock lk(g.mu);
    const int es = elemSizeOf((int)dtype);
    int rc = topkCommon(R, T, k, width, es);
    if (rc) return rc;
    if (!tokens || !pos_dev || !sendcounts_rows_dev || !recv || !recvcounts_rows_dev) return NCCLX_ERR_ARG;
    if (sendcounts_rows_dev == recvcounts_rows_dev) return NCCLX_ERR_ARG;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    rc = prepareTopk(0, sendcounts_rows_dev, recvcounts_rows_dev, R, s);
    if (rc) return rc;
    return launchTopkDispatch(0, tokens, pos_dev, recv, R, T, k, (long long)width * es, s);
}

int ncclx_moe_combine_topk_sum_dev(const void* const* expert_out, const int32_t* pos_dev,
                                   const int64_t* sendcounts_rows_dev, void* const* out, int R, int T, int k,
                                   int width, ncclx_dtype_t dtype, ncclx_stream_t stream) {
    Lock lk(g.mu);
    const int es = elemSizeOf((int)dtype);
    int rc = topkCommon(R, T, k, width, es);
    if (rc) return rc;
    if (!(dtype == NCCLX_BF16 || dtype == NCCLX_F32 || dtype == NCCLX_F16)) return NCCLX_ERR_DTYPE;
    if (!expert_out || !pos_dev || !sendcounts_rows_dev || !out) return NCCLX_ERR_ARG;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    // offsets of the DISPATCH's count matrix; its transpose goes to a scratch sink
    rc = prepareTopk(0, sendcounts_rows_dev, reinterpret_cast<int64_t*>(g.rcScratch), R, s);
    if (rc) return rc;
    return launchTopkCombine(0, expert_out, pos_dev, out, R, T, k, (long long)width * es, (int)dtype, s);
}

int ncclx_moe_topk_prepare_dev(int plan, const int64_t* sendcounts_rows_dev, int64_t* recvcounts_rows_dev, int R,
                               ncclx_stream_t stream) {
    Lock lk(g.mu);
    int rc = checkCommon(R);
    if (rc) return rc;
    if (plan < 0 || plan >= NCCLX_NUM_PLANS) return NCCLX_ERR_ARG;
    if (!sendcounts_rows_dev || !recvcounts_rows_dev || sendcounts_rows_dev == recvcounts_rows_dev) return NCCLX_ERR_ARG;
    return prepareTopk(plan, sendcounts_rows_dev, recvcounts_rows_dev, R, static_cast<cudaStream_t>(stream));
}

int ncclx_moe_dispatch_topk_execute_dev(int plan, const void* const* tokens, const int32_t* pos_dev, void* const* recv,
                                        int T, int k, int width, ncclx_dtype_t dtype, ncclx_stream_t stream) {
    Lock lk(g.mu);
    if (!g.ready) return NCCLX_ERR_NOT_INITIALIZED;
    if (plan < 0 || plan >= NCCLX_NUM_PLANS || g.plan[plan].kind != PLAN_TOPK) return NCCLX_ERR_ARG;
    const int es = elemSizeOf((int)dtype);
    const int R = g.plan[plan].R;
    int rc = topkCommon(R, T, k, width, es);
    if (rc) return rc;
    if (!tokens || !pos_dev || !recv) return NCCLX_ERR_ARG;
    return launchTopkDispatch(plan, tokens, pos_dev, recv, R, T, k, (long long)width * es, static_cast<cudaStream_t>(stream));
}

int ncclx_moe_combine_topk_sum_execute_dev(int plan, const void* const* expert_out, const int32_t* pos_dev, void* const* out,
                                           int T, int k, int width, ncclx_dtype_t dtype, ncclx_stream_t stream) {
    Lock lk(g.mu);
    if (!g.ready) return NCCLX_ERR_NOT_INITIALIZED;
    if (plan < 0 || plan >= NCCLX_NUM_PLANS || g.plan[plan].kind != PLAN_TOPK) return NCCLX_ERR_ARG;
    const int es = elemSizeOf((int)dtype);
    const int R = g.plan[plan].R;
    int rc = topkCommon(R, T, k, width, es);
    if (rc) return rc;
    if (!(dtype == NCCLX_BF16 || dtype == NCCLX_F32 || dtype == NCCLX_F16)) return NCCLX_ERR_DTYPE;
    if (!expert_out || !pos_dev || !out) return NCCLX_ERR_ARG;
    return launchTopkCombine(plan, expert_out, pos_dev, out, R, T, k, (long long)width * es, (int)dtype,
                             static_cast<cudaStream_t>(stream));
}

int ncclx_reducecopy_sum(const void* a, const void* b, void* out, void* fwd, size_t count, ncclx_dtype_t dtype,
                         size_t chunk_bytes, int num_ctas, ncclx_stream_t stream) {
    Lock lk(g.mu);
    if (!g.ready) return NCCLX_ERR_NOT_INITIALIZED;
    if (!a || !b || (!out && !fwd) || num_ctas < 0 || num_ctas > 65535) return NCCLX_ERR_ARG;
    if (!(dtype == NCCLX_BF16 || dtype == NCCLX_F32 || dtype == NCCLX_F16)) return NCCLX_ERR_DTYPE;
    if (count == 0) return NCCLX_OK;
    const int es = elemSizeOf((int)dtype);
    if (chunk_bytes == 0) chunk_bytes = (size_t)8 << 20;
    if (chunk_bytes % es) return NCCLX_ERR_ARG;
    if (num_ctas == 0) num_ctas = 2;
    ReduceCopyArgs ra{};
    ra.a = static_cast<const unsigned char*>(a); ra.b = static_cast<const unsigned char*>(b);
    ra.out = static_cast<unsigned char*>(out); ra.fwd = static_cast<unsigned char*>(fwd);
    ra.count = count; ra.chunkElems = chunk_bytes / es;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    const bool aligned = ((((uintptr_t)a | (uintptr_t)b | (uintptr_t)out | (uintptr_t)fwd) & 31u) == 0) && (chunk_bytes & 31u) == 0;
    LaunchScope ls(NCCLX_KERNEL_REDUCE, s);
    if (g.params[NCCLX_PARAM_REDUCECOPY_TMA] && aligned) {
        switch (dtype) {
        case NCCLX_BF16: reducecopy_tma_kernel<RED_BF16><<<num_ctas, RCT_THREADS, RCT_SMEM_BYTES, s>>>(ra); break;
        case NCCLX_F32: reducecopy_tma_kernel<RED_F32><<<num_ctas, RCT_THREADS, RCT_SMEM_BYTES, s>>>(ra); break;
        default: reducecopy_tma_kernel<RED_F16><<<num_ctas, RCT_THREADS, RCT_SMEM_BYTES, s>>>(ra); break;
        }
    } else {
        switch (dtype) {
        case NCCLX_BF16: reducecopy_kernel<RED_BF16><<<num_ctas, RC_THREADS, 0, s>>>(ra); break;
        case NCCLX_F32: reducecopy_kernel<RED_F32><<<num_ctas, RC_THREADS, 0, s>>>(ra); break;
        default: reducecopy_kernel<RED_F16><<<num_ctas, RC_THREADS, 0, s>>>(ra); break;
        }
    }
    CK(cudaGetLastError());
    ls.ok();
    return NCCLX_OK;
}

// ---- host-buffer forms -----------------------------------------------------------------------

int ncclx_alltoallv_host(const void* const* send, const int64_t* sendcounts_host, void* const* recv,
                         int64_t* recvcounts_host, int R, ncclx_dtype_t dtype, ncclx_stream_t stream) {
    Lock lk(g.mu);
    int rc = checkCommon(R);
    if (rc) return rc;
    if (!send || !sendcounts_host || !recv || !recvcounts_host) return NCCLX_ERR_ARG;
    const int es = elemSizeOf((int)dtype);
    if (!es) return NCCLX_ERR_DTYPE;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    if (isCapturing(s)) return NCCLX_ERR_CAPTURE;

    std::vector<size_t> sBytes(R, 0), rBytes(R, 0), sOff(R), rOff(R);
    for (int i = 0; i < R; ++i)
        for (int j = 0; j < R; ++j) {
            const int64_t c = sendcounts_host[(size_t)i * R + j];
            if (c > 0) { sBytes[i] += (size_t)c * es; rBytes[j] += (size_t)c * es; }
        }
    for (int i = 0; i < R; ++i)
        if ((sBytes[i] && !send[i]) || (rBytes[i] && !recv[i])) return NCCLX_ERR_ARG;
    const size_t rr = (size_t)R * R * 8;
    const size_t metaBytes = 2 * rr + 2 * (size_t)R * 8;
    if ((rc = ensureStage(2, metaBytes))) return rc;
    char* meta = static_cast<char*>(g.stage[2]);
    int64_t* dC = reinterpret_cast<int64_t*>(meta);
    int64_t* dRC = reinterpret_cast<int64_t*>(meta + rr);
    void** dSend = reinterpret_cast<void**>(meta + 2 * rr);
    void** dRecv = dSend + R;
    std::vector<void*> tab(2 * (size_t)R, nullptr);

    // zero-copy when every buffer in use is pinned: the kernels read send[] and write recv[] in host memory
    bool zeroCopy = g.params[NCCLX_PARAM_HOST_ZERO_COPY] != 0;
    for (int i = 0; i < R && zeroCopy; ++i) {
        if (sBytes[i] && !(tab[i] = mappedDevicePtr(send[i]))) zeroCopy = false;
        if (rBytes[i] && !(tab[R + i] = mappedDevicePtr(recv[i]))) zeroCopy = false;
    }
    if (zeroCopy) {
        for (int i = 0; i < R; ++i) {              // unused slots still need a valid, aligned address
            if (!tab[i]) tab[i] = g.stage[2];
            if (!tab[R + i]) tab[R + i] = g.stage[2];
        }
        CK(cudaMemcpyAsync(dC, sendcounts_host, rr, cudaMemcpyHostToDevice, s));
        CK(cudaMemcpyAsync(dSend, tab.data(), 2 * (size_t)R * 8, cudaMemcpyHostToDevice, s));
        rc = launchAllToAllv(reinterpret_cast<const void* const*>(dSend), dC, dRecv, dRC, R, es, s);
        if (rc) return rc;
        CK(cudaMemcpyAsync(recvcounts_host, dRC, rr, cudaMemcpyDeviceToHost, s));
        CK(cudaStreamSynchronize(s));
        return NCCLX_OK;
    }

    size_t sTot = 0, rTot = 0;
    for (int i = 0; i < R; ++i) { sOff[i] = sTot; sTot += alignUp(sBytes[i], 256); rOff[i] = rTot; rTot += alignUp(rBytes[i], 256); }
    if ((rc = ensureStage(0, sTot + 256))) return rc;
    if ((rc = ensureStage(1, rTot + 256))) return rc;
    for (int i = 0; i < R; ++i) {
        tab[i] = static_cast<char*>(g.stage[0]) + sOff[i];
        tab[R + i] = static_cast<char*>(g.stage[1]) + rOff[i];
    }
    CK(cudaMemcpyAsync(dC, sendcounts_host, rr, cudaMemcpyHostToDevice, s));
    CK(cudaMemcpyAsync(dSend, tab.data(), 2 * (size_t)R * 8, cudaMemcpyHostToDevice, s));
    for (int i = 0; i < R; ++i)
        if (sBytes[i]) CK(cudaMemcpyAsync(tab[i], send[i], sBytes[i], cudaMemcpyHostToDevice, s));
    rc = launchAllToAllv(reinterpret_cast<const void* const*>(dSend), dC, dRecv, dRC, R, es, s);
    if (rc) return rc;
    for (int i = 0; i < R; ++i)
        if (rBytes[i]) CK(cudaMemcpyAsync(recv[i], tab[R + i], rBytes[i], cudaMemcpyDeviceToHost, s));
    CK(cudaMemcpyAsync(recvcounts_host, dRC, rr, cudaMemcpyDeviceToHost, s));
    CK(cudaStreamSynchronize(s));
    return NCCLX_OK;
}

static int reduceHost(const void* const* send, void* const* recv, size_t blockElems, int R, int dtype, int scatter,
                      cudaStream_t s) {
    int rc = checkCommon(R);
    if (rc) return rc;
    if (!send || !recv) return NCCLX_ERR_ARG;
    if (!(dtype == NCCLX_BF16 || dtype == NCCLX_F32 || dtype == NCCLX_F16)) return NCCLX_ERR_DTYPE;
    if (isCapturing(s)) return NCCLX_ERR_CAPTURE;
    if (blockElems == 0) return NCCLX_OK;
    const int es = elemSizeOf(dtype);
    const size_t inBytes = blockElems * (scatter ? (size_t)R : 1) * es;
    const size_t outBytes = blockElems * es;
    for (int i = 0; i < R; ++i)
        if (!send[i] || !recv[i]) return NCCLX_ERR_ARG;
    if ((rc = ensureStage(2, 2 * (size_t)R * 8))) return rc;
    void** dSend = static_cast<void**>(g.stage[2]);
    std::vector<void*> tab(2 * (size_t)R, nullptr);

    // zero-copy pays when the outbound bytes are comparable to the inbound ones (AllReduce: equal), because the
    // two directions then share the link; a ReduceScatter's output is 1/R of its input and the staged copies
    // are as fast (measured: R = 16, 2 GiB in: 41.5 ms staged, 42.0 ms zero-copy)
    bool zeroCopy = g.params[NCCLX_PARAM_HOST_ZERO_COPY] != 0 && outBytes * 4 >= inBytes;
    for (int i = 0; i < R && zeroCopy; ++i)
        if (!(tab[i] = mappedDevicePtr(send[i])) || !(tab[R + i] = mappedDevicePtr(recv[i]))) zeroCopy = false;
    if (zeroCopy) {                                // inputs streamed from, results written to, pinned host memory
        CK(cudaMemcpyAsync(dSend, tab.data(), 2 * (size_t)R * 8, cudaMemcpyHostToDevice, s));
        rc = launchReduce(reinterpret_cast<const void* const*>(dSend), dSend + R, blockElems, R, dtype, scatter, s);
        if (rc) return rc;
        CK(cudaStreamSynchronize(s));
        return NCCLX_OK;
    }

    const size_t inPitch = alignUp(inBytes, 256), outPitch = alignUp(outBytes, 256);
    if ((rc = ensureStage(0, inPitch * R))) return rc;
    if ((rc = ensureStage(1, outPitch * R))) return rc;
    for (int i = 0; i < R; ++i) {
        tab[i] = static_cast<char*>(g.stage[0]) + inPitch * i;
        tab[R + i] = static_cast<char*>(g.stage[1]) + outPitch * i;
    }
    CK(cudaMemcpyAsync(dSend, tab.data(), 2 * (size_t)R * 8, cudaMemcpyHostToDevice, s));
    for (int i = 0; i < R; ++i) CK(cudaMemcpyAsync(tab[i], send[i], inBytes, cudaMemcpyHostToDevice, s));
    rc = launchReduce(reinterpret_cast<const void* const*>(dSend), dSend + R, blockElems, R, dtype, scatter, s);
    if (rc) return rc;
    for (int i = 0; i < R; ++i) CK(cudaMemcpyAsync(recv[i], tab[R + i], outBytes, cudaMemcpyDeviceToHost, s));
    CK(cudaStreamSynchronize(s));
    return NCCLX_OK;
}

int ncclx_allreduce_sum_host(const void* const* send, void* const* recv, size_t count, int R, ncclx_dtype_t dtype,
                             ncclx_stream_t stream) {
    Lock lk(g.mu);
    return reduceHost(send, recv, count, R, (int)dtype, 0, static_cast<cudaStream_t>(stream));
}

int ncclx_reducescatter_sum_host(const void* const* send, void* const* recv, size_t recvcount, int R,
                                 ncclx_dtype_t dtype, ncclx_stream_t stream) {
    Lock lk(g.mu);
    return reduceHost(send, recv, recvcount, R, (int)dtype, 1, static_cast<cudaStream_t>(stream));
}

// ---- tuning / measurement --------------------------------------------------------------------

static int streamProbe(int mode, const void* src, void* dst, size_t bytes, int num_ctas, cudaStream_t s) {
    if (!g.ready) return NCCLX_ERR_NOT_INITIALIZED;
    if (mode < 0 || mode > 3 || ((mode == 0 || mode == 2) && !src) || (mode != 0 && !dst) || bytes % 32) return NCCLX_ERR_ARG;
    if ((((uintptr_t)src | (uintptr_t)dst) & 31u) != 0 || num_ctas < 0 || num_ctas > 65535) return NCCLX_ERR_ARG;
    if (bytes == 0) return NCCLX_OK;
    if (mode == 3) {
        if (bytes % PROBE_BULK_BYTES) return NCCLX_ERR_ARG;
        stream_probe_bulk_store_kernel<<<num_ctas ? num_ctas : g.smCount * 4, 128, 0, s>>>(static_cast<unsigned char*>(dst), bytes / PROBE_BULK_BYTES);
    } else if (num_ctas == 0) {
        stream_probe_kernel<PROBE_THREADS><<<g.smCount * 8, PROBE_THREADS, 0, s>>>(
            mode, static_cast<const unsigned char*>(src), static_cast<unsigned char*>(dst), bytes / 32, &g.wsPlan[0].ctl->pad_probe);
    } else {                                       // few-CTA form: 1024 threads x 4 x 32 B = 128 KB in flight per CTA
        stream_probe_kernel<PROBE_THREADS_FEW><<<num_ctas, PROBE_THREADS_FEW, 0, s>>>(
            mode, static_cast<const unsigned char*>(src), static_cast<unsigned char*>(dst), bytes / 32, &g.wsPlan[0].ctl->pad_probe);
    }
    CK(cudaGetLastError());
    return NCCLX_OK;
}

int ncclx_stream_probe(int mode, const void* src, void* dst, size_t bytes, ncclx_stream_t stream) {
    Lock lk(g.mu);
    return streamProbe(mode, src, dst, bytes, 0, static_cast<cudaStream_t>(stream));
}

int ncclx_stream_probe_ctas(int mode, const void* src, void* dst, size_t bytes, int num_ctas, ncclx_stream_t stream) {
    Lock lk(g.mu);
    if (num_ctas < 1) return NCCLX_ERR_ARG;
    return streamProbe(mode, src, dst, bytes, num_ctas, static_cast<cudaStream_t>(stream));
}

int ncclx_set_param(int param, int64_t value) {
    Lock lk(g.mu);
    if (param < 0 || param >= NCCLX_PARAM_COUNT_) return NCCLX_ERR_ARG;
    switch (param) {
    case NCCLX_PARAM_BULK_MIN_BYTES: if (value < 16) return NCCLX_ERR_ARG; break;
    case NCCLX_PARAM_REDUCE_CTAS_PER_SM: if (value < 1 || value > 64) return NCCLX_ERR_ARG; break;
    case NCCLX_PARAM_BULK_TILE_SHIFT: if (value < 12 || value > 16) return NCCLX_ERR_ARG; break;
    case NCCLX_PARAM_COPY_KMAX: if (value < 1 || value > 64) return NCCLX_ERR_ARG; break;
    case NCCLX_PARAM_FUSED_MAX_RANKS: if (value < 0 || value > FUSED_MAX_R) return NCCLX_ERR_ARG; break;
    case NCCLX_PARAM_COPY_BULK_ENGINES: if (value != 0 && value != 1 && value != 2 && value != 4) return NCCLX_ERR_ARG; break;
    default: if (value < 0 || value > 1) return NCCLX_ERR_ARG; break;       // PROFILE, PDL, HOST_ZERO_COPY, REDUCECOPY_TMA
    }
    g.params[param] = value;
    return NCCLX_OK;
}

int ncclx_get_param(int param, int64_t* value) {
    Lock lk(g.mu);
    if (param < 0 || param >= NCCLX_PARAM_COUNT_ || !value) return NCCLX_ERR_ARG;
    *value = g.params[param];
    return NCCLX_OK;
}

int ncclx_profile_read(int kernel, double* total_ms, int64_t* launches) {
    Lock lk(g.mu);
    if (kernel < 0 || kernel >= NCCLX_KERNEL_COUNT_ || !total_ms || !launches) return NCCLX_ERR_ARG;
    double tot = 0;
    for (auto& e : g.events[kernel]) {
        CK(cudaEventSynchronize(e.b));
        float ms = 0;
        CK(cudaEventElapsedTime(&ms, e.a, e.b));
        tot += ms;
    }
    *total_ms = tot;
    *launches = (int64_t)g.events[kernel].size();
    return NCCLX_OK;
}

int ncclx_profile_reset(void) {
    Lock lk(g.mu);
    for (auto& v : g.events) {
        for (auto& e : v) { cudaEventDestroy(e.a); cudaEventDestroy(e.b); }
        v.clear();
    }
    g.launches = 0;
    return NCCLX_OK;
}

int64_t ncclx_launch_count(void) { return g.launches.load(); }

}  // extern "C"

// ---- AllToAllv without any allocation: ncclx_alltoallv_static_dev ------------------------------------------
//
// For callers that must not (or cannot) call cudaMalloc -- see the header for who they are.  The single-launch
// kernel (alltoallv_fused_kernel) is launched with its scratch pointers aimed at the file-scope device array
// below instead of at the ncclx_init workspace.  Nothing here reads or writes the Context `g` apart from the
// last-CUDA-error slot that the CK macro fills.
//
// The array is part of the library's device image: each GPU that loads the image holds these 16.5 KiB until the
// process ends.  Layout: [0,256) WorkCtl claim counters | [256,512) fallback status word | soff R*R i64 | roff R*R i64.
// IMPORTANT for anyone editing this: in HOST code the identifier `ncclx_static_scratch` is only a handle for the
// runtime, not an address a kernel can use.  The device address is fetched once per device with
// cudaGetSymbolAddress (staticSetup) and only that pointer is handed to the kernel.
static_assert(sizeof(xdev::WorkCtl) <= 256, "control block must fit its 256-byte slot");
static_assert(NCCLX_STATIC_MAX_RANKS <= xdev::FUSED_MAX_R, "the static entry point rides on the single-launch kernel");
static __device__ __align__(256) unsigned char ncclx_static_scratch[NCCLX_STATIC_SCRATCH_BYTES];

namespace {

constexpr int kStaticMaxDevices = 64;
constexpr size_t kStaticClearBytes = 512;          // counters + status: what has to be zero when the kernel starts

struct StaticDev {
    bool ready = false;
    unsigned char* scratch = nullptr;              // DEVICE address of ncclx_static_scratch on this device
    int smCount = 0;
    int smemOptin = 0;
    int smemDynamicMax = 0;                        // what the kernel was opted in to
};
StaticDev gStatic[kStaticMaxDevices];
std::mutex gStaticMu;

// Once per device, with that device current.  Not done under stream capture (symbol look-up may load the module).
int staticSetup(int dev, StaticDev& sd, cudaStream_t s) {
    if (isCapturing(s)) return NCCLX_ERR_CAPTURE;
    int major = 0;
    CK(cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev));
    if (major < 10) { g.lastCuda = (int)cudaErrorNoKernelImageForDevice; return NCCLX_ERR_CUDA; }
    CK(cudaDeviceGetAttribute(&sd.smCount, cudaDevAttrMultiProcessorCount, dev));
    CK(cudaDeviceGetAttribute(&sd.smemOptin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev));
    void* p = nullptr;
    CK(cudaGetSymbolAddress(&p, ncclx_static_scratch));
    if (!p) { g.lastCuda = (int)cudaErrorInvalidSymbol; return NCCLX_ERR_CUDA; }
    cudaFuncAttributes fa{};
    CK(cudaFuncGetAttributes(&fa, alltoallv_fused_kernel));
    sd.smemDynamicMax = sd.smemOptin - (int)fa.sharedSizeBytes;
    CK(cudaFuncSetAttribute(alltoallv_fused_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, sd.smemDynamicMax));
    sd.scratch = static_cast<unsigned char*>(p);
    sd.ready = true;
    return NCCLX_OK;
}

}  // namespace

extern "C" int ncclx_alltoallv_static_dev(const void* const* send, const int64_t* sendcounts_dev, void* const* recv,
                                          int64_t* recvcounts_dev, uint32_t* status_dev, int R, ncclx_dtype_t dtype,
                                          ncclx_stream_t stream) {
    // size and argument checks first: they need no device
    if (R < 1) return NCCLX_ERR_ARG;
    if (R > NCCLX_STATIC_MAX_RANKS) return NCCLX_ERR_TOO_LARGE;
    if (!send || !sendcounts_dev || !recv || !recvcounts_dev) return NCCLX_ERR_ARG;
    if (sendcounts_dev == recvcounts_dev) return NCCLX_ERR_ARG;
    const int es = elemSizeOf((int)dtype);
    if (!es) return NCCLX_ERR_DTYPE;

    std::lock_guard<std::mutex> lk(gStaticMu);
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    int dev = -1;
    CK(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kStaticMaxDevices) return NCCLX_ERR_ARG;
    StaticDev& sd = gStatic[dev];
    if (!sd.ready) {
        const int rc = staticSetup(dev, sd, s);
        if (rc) return rc;
    }

    // launch geometry with the library's default tunables (the result does not depend on them)
    FusedArgs fa{};
    fa.cls.bulkMinBytes = 1024;
    fa.cls.tileShift[LIST_BULK] = 15;
    fa.cls.tileShift[LIST_VEC] = kVecTileShift;
    fa.bulkEngines = 0;
    fa.kmax = 6;
    const int room = sd.smemOptin - 1024 < sd.smemDynamicMax ? sd.smemOptin - 1024 : sd.smemDynamicMax;   // as planFused: 1 KB kept for static shared memory
    const size_t budget = room > 0 ? (size_t)room : 0;
    const size_t aux = fused_aux_bytes(R);
    if (budget < aux + 64 * 1024) { g.lastCuda = (int)cudaErrorInvalidConfiguration; return NCCLX_ERR_CUDA; }
    fa.ringBytes = (unsigned int)((budget - aux) & ~(size_t)127);
    if ((size_t)VEC_SUB_BYTES + 256 > ((fa.ringBytes / COPY_WARPS) & ~127u)) { g.lastCuda = (int)cudaErrorInvalidConfiguration; return NCCLX_ERR_CUDA; }
    while (fa.cls.tileShift[LIST_BULK] > 10 && !bulkTileFits(fa.cls.tileShift[LIST_BULK], fa.ringBytes, fa.bulkEngines)) --fa.cls.tileShift[LIST_BULK];
    fa.minTileShift[LIST_BULK] = kFusedMinTileShift < fa.cls.tileShift[LIST_BULK] ? kFusedMinTileShift : fa.cls.tileShift[LIST_BULK];
    fa.minTileShift[LIST_VEC] = 10 < fa.cls.tileShift[LIST_VEC] ? 10 : fa.cls.tileShift[LIST_VEC];

    fa.send = send; fa.recv = recv;
    fa.C = reinterpret_cast<const long long*>(sendcounts_dev);
    fa.RC = reinterpret_cast<long long*>(recvcounts_dev);
    fa.ctl = reinterpret_cast<WorkCtl*>(sd.scratch);
    fa.status = status_dev ? status_dev : reinterpret_cast<unsigned int*>(sd.scratch + 256);
    fa.soff = reinterpret_cast<long long*>(sd.scratch + kStaticClearBytes);
    fa.roff = fa.soff + (size_t)NCCLX_STATIC_MAX_RANKS * NCCLX_STATIC_MAX_RANKS;
    fa.R = R; fa.elemSize = es;

    // The array still holds the previous call's state.  The counters normally return to zero by themselves, but a
    // kernel that was aborted half-way would leave them dirty, so they are cleared in stream order every time.
    CK(cudaMemsetAsync(sd.scratch, 0, kStaticClearBytes, s));
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3((unsigned)sd.smCount);
    cfg.blockDim = dim3(COPY_THREADS);
    cfg.dynamicSmemBytes = (size_t)fa.ringBytes + aux;
    cfg.stream = s;
    cfg.attrs = nullptr; cfg.numAttrs = 0;          // plain stream order: the memset above has to be complete first
    CK(cudaLaunchKernelEx(&cfg, alltoallv_fused_kernel, fa));
    return NCCLX_OK;
}
