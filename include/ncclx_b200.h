/*
 * ncclx_b200.h -- C ABI of libncclx_b200.so
 *
 * The on-device data path of two NCCLX collectives ("Collective Communication for 100k+
 * GPUs", arxiv 2510.20171; cited as PAPER.md L<n>), hand-written for NVIDIA B200 (sm_100a),
 * over R EMULATED ranks whose send and receive buffers all live in one GPU's HBM:
 *
 *   1. AllToAllv with device-resident split counts -- the paper's GPU-resident collective
 *      AllToAllvDynamic (section 6.1): metadata is taken BY REFERENCE
 *      (L401, L409), actual counts are moved instead of maxcounts padding (L387, L397), the
 *      receive counts are returned to the user (L419), the call is CUDA-graph capturable.
 *   2. The sum reduction behind AllReduce / ReduceScatter -- the Reduce / ReduceCopy kernel
 *      step of the paper's FTAR ring (section 5.3, Fig. 9): fp32
 *      accumulation in rank order 0..R-1, one rounding.
 *
 * Conventions common to every entry point
 *   - Plain C, no CUDA or torch types.  A stream is passed as `ncclx_stream_t` = the value of
 *     a `cudaStream_t` (NULL = the legacy default stream).
 *   - "DEVICE" pointers must be dereferenceable by kernels on the device given to
 *     ncclx_init; "HOST" pointers by the CPU.  The caller owns every buffer it passes; the
 *     library owns only its workspace (allocated in ncclx_init, freed in ncclx_finalize).
 *   - Device entry points (`*_dev`, `*_sum`) only ENQUEUE kernels on `stream`: no host
 *     synchronisation, no allocation, no host<->device copy.  They may be captured into a
 *     CUDA graph; a replay re-reads the device-resident metadata.  One workspace exists per
 *     process: calls must be ordered on ONE stream at a time (or by events).
 *   - Return value: 0 = NCCLX_OK, otherwise an ncclx_result_t.  Every argument and configuration check is made
 *     BEFORE the call's first kernel launch, so an NCCLX_ERR_ARG / _DTYPE / _NOT_INITIALIZED / _CAPTURE return
 *     means nothing was enqueued and no buffer or workspace was touched (ncclx_launch_count() does not move).
 *     Only NCCLX_ERR_CUDA (a launch the CUDA runtime itself refused) can follow an earlier successful launch of
 *     the same call.  No exceptions, no abort, nothing printed.  ncclx_strerror() names a code.
 *   - Entry points may be called from several host threads (one internal mutex); the workspace rule above
 *     still applies to what they enqueue.
 *   - There is no CPU fallback: without a CUDA device ncclx_init fails with
 *     NCCLX_ERR_CUDA and every other call fails with NCCLX_ERR_NOT_INITIALIZED
 *     (ncclx_alltoallv_static_dev, the one call that needs no init, fails with NCCLX_ERR_CUDA).
 */
#ifndef NCCLX_B200_H
#define NCCLX_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define NCCLX_B200_VERSION 200 /* 0.2.0 */
#define NCCLX_MAX_RANKS 1024   /* hard upper bound on R (ncclx_init max_ranks) */

typedef void* ncclx_stream_t; /* a cudaStream_t */

typedef enum {
    NCCLX_BF16 = 0, /* bfloat16, 2 bytes  */
    NCCLX_F32 = 1,  /* IEEE binary32      */
    NCCLX_F16 = 2,  /* IEEE binary16      */
    NCCLX_U8 = 3    /* raw bytes: AllToAllv only (reductions return NCCLX_ERR_DTYPE) */
} ncclx_dtype_t;

typedef enum {
    NCCLX_OK = 0,
    NCCLX_ERR_ARG = 1,             /* null pointer, R < 1, bad parameter id/value              */
    NCCLX_ERR_DTYPE = 2,           /* dtype not supported by this call                         */
    NCCLX_ERR_NOT_INITIALIZED = 3, /* ncclx_init not called, or R > max_ranks given to it      */
    NCCLX_ERR_CUDA = 4,            /* a CUDA runtime call failed (see ncclx_last_cuda_error)   */
    NCCLX_ERR_CAPTURE = 5,         /* a host-synchronous call was made while `stream` captures */
    NCCLX_ERR_TOO_LARGE = 6        /* ncclx_alltoallv_static_dev only: R > NCCLX_STATIC_MAX_RANKS */
} ncclx_result_t;

/* ---- lifetime ------------------------------------------------------------------------- */

/* Allocates the workspace (offset matrices, segment descriptors, work counters, status word:
 * NCCLX_NUM_PLANS slots of about 60 * max_ranks^2 bytes each) on `device`, sets kernel attributes and queries the SM count.
 * Call OUTSIDE stream capture.  Calling it again re-initialises (after an implicit finalize).
 * 1 <= max_ranks <= NCCLX_MAX_RANKS. */
int ncclx_init(int max_ranks, int device);
int ncclx_finalize(void);
const char* ncclx_strerror(int code);
/* cudaError_t value of the last failing CUDA call (0 if none), and its string. */
int ncclx_last_cuda_error(void);
const char* ncclx_last_cuda_error_string(void);
int ncclx_version(void);

/* ---- AllToAllv with device-resident counts (section 6.1) ---------------------- *
 *
 * For every ordered pair (s, d) of the R emulated ranks, with C = sendcounts_dev:
 *     recvcounts_dev[d*R + s] = C[s*R + d]                                   (L419, L439)
 *     soff[s][d] = sum_{d'<d} C[s][d']      roff[d][s] = sum_{s'<s} C[s'][d]
 *     recv[d][roff[d][s] .. +C[s][d])  =  send[s][soff[s][d] .. +C[s][d])    bytes verbatim
 * i.e. send[s] is one contiguous buffer split by row s of C (L429), and recv[d] is packed by
 * source rank ascending with no padding (reading 4).  Bytes of recv[d] outside
 * the packed range are NOT written.
 *
 *   send            DEVICE array of R DEVICE pointers, send[s] (>= 16-byte aligned bases)
 *   sendcounts_dev  DEVICE int64[R*R], row-major C[s*R+d], in ELEMENTS of dtype.  Read when
 *                   the kernels EXECUTE, not when this call returns (L401, L409): a kernel or
 *                   memcpy ordered before the call on `stream` (or before a graph replay) may
 *                   rewrite it.  A negative entry is treated as 0 and sets bit 0 of the
 *                   device status word (ncclx_device_status).
 *   recv            DEVICE array of R DEVICE pointers, recv[d]
 *   recvcounts_dev  DEVICE int64[R*R], OUT.  Must not overlap sendcounts_dev.
 *   R               1 <= R <= max_ranks.  R == 1 is a plain copy.
 *   dtype           any ncclx_dtype_t; only its element size matters (pure data movement).
 *
 * Capacity: the caller guarantees send[s] holds sum_d C[s][d] and recv[d] holds
 * sum_s C[s][d] elements; overflow is undefined (as in NCCL).  send and recv buffers must not
 * overlap.  Segment addresses may have any element alignment; full speed is only promised
 * when every segment's source address, destination address and byte length are multiples of
 * 16 (bulk list: 32 KiB tiles, TMA in and out); everything else is loaded by the TMA as aligned spans, realigned in
 * shared memory and stored by the TMA as well, 4 KiB at a time (vector list: ~0.9 of the bulk list's rate).
 * The inverse ("combine") is the same call with send := recv, sendcounts := recvcounts.
 * For R <= 32 (NCCLX_PARAM_FUSED_MAX_RANKS) the call is ONE kernel launch (the small-message fast path,
 * PAPER.md L483): every CTA rebuilds offsets and work list from the <= 8 KB count matrix in shared memory
 * and picks the tile size from the byte total; results are identical to the two-kernel path.          */
int ncclx_alltoallv_dev(const void* const* send, const int64_t* sendcounts_dev, void* const* recv,
                        int64_t* recvcounts_dev, int R, ncclx_dtype_t dtype, ncclx_stream_t stream);

/* ---- AllToAllv for callers that cannot allocate device memory -------------------------------------- *
 *
 * Who this is for.  Every other entry point needs ncclx_init, and ncclx_init calls cudaMalloc for the
 * workspace.  Some callers are not in a position to do that: a plug-in running inside a host application
 * whose memory pool already owns (nearly) all of HBM, so a late cudaMalloc fails or fragments the pool; code
 * that runs in a phase where the surrounding framework forbids allocator calls because cudaMalloc / cudaFree
 * synchronise the whole device and would stall other streams mid-step; or a sandboxed worker that is handed
 * finished device buffers and is simply not allowed to create new ones.  For them this ONE call performs the
 * complete AllToAllv of ncclx_alltoallv_dev (same semantics, same argument meaning, byte-identical results)
 * and never calls cudaMalloc, cudaFree, cudaMallocAsync, cudaEventCreate or any allocating library routine.
 * It does NOT need ncclx_init and does not touch the ncclx_init workspace; it may be used before, after or
 * without it.
 *
 * Where its scratch memory lives.  The kernel needs a little global memory that is neither input nor output
 * (the claim counters of its work list, the two R x R offset matrices it derives from the counts, a status
 * word).  Here that scratch is a fixed array of NCCLX_STATIC_SCRATCH_BYTES (16 896) bytes compiled into the
 * library's device image.  Consequences a user should know:
 *   - every GPU on which this library's device code gets loaded carries those 16.5 KiB until the process
 *     exits, whether or not this call is ever used;
 *   - the size is fixed, so the call is limited to R <= NCCLX_STATIC_MAX_RANKS (32).  A larger R is refused
 *     with NCCLX_ERR_TOO_LARGE before anything is enqueued (use ncclx_init + ncclx_alltoallv_dev there).
 *     The payload size is NOT limited by the scratch: any byte counts the buffers can hold are fine;
 *   - there is ONE array per GPU and every call on that GPU uses it.  Two calls that can be in flight on the
 *     same GPU at the same time (different streams without an event between them, or two host threads each
 *     driving its own stream) race on it and may corrupt each other's transfer.  Keep the calls of one GPU in
 *     one stream's order.  The array keeps whatever the previous call left; the part that has to start at
 *     zero (counters, status) is cleared on `stream` ahead of the kernel by every call.
 *
 * First call on a GPU.  The call works on the CUDA device that is CURRENT in the calling thread (all pointers
 * must belong to it; up to 64 devices per process).  The first call on each device looks up the device
 * address of the scratch array, reads the SM count and shared-memory limit, and raises the kernel's
 * shared-memory limit; later calls on that device reuse the result.  Make that first call OUTSIDE any stream
 * capture: if `stream` is capturing when the set-up is still to be done the call returns NCCLX_ERR_CAPTURE
 * and enqueues nothing.
 *
 *   send, sendcounts_dev, recv, recvcounts_dev, dtype, stream: exactly as for ncclx_alltoallv_dev (counts are
 *       DEVICE-resident and read when the kernel executes; recv bytes outside the packed range are not
 *       written; a negative count moves nothing).
 *   status_dev   optional DEVICE uint32 owned by the caller (NULL: not reported).  Bit 0 is OR-ed into it
 *                when a negative count was seen; the library never clears it.  (ncclx_device_status does not
 *                see this call.)
 *   R            1 <= R <= NCCLX_STATIC_MAX_RANKS.
 * Errors: NCCLX_ERR_ARG (null pointer, R < 1, sendcounts_dev == recvcounts_dev, device index >= 64),
 * NCCLX_ERR_TOO_LARGE, NCCLX_ERR_DTYPE, NCCLX_ERR_CAPTURE (see above), NCCLX_ERR_CUDA (no usable sm_100
 * device current, or the runtime refused the memset / launch).  Except for a refused kernel launch, which
 * leaves the harmless 512-byte clear of the scratch behind, an error means nothing was enqueued.  The call
 * only enqueues (one 512-byte memset + one kernel): it does not synchronise and is not counted by
 * ncclx_launch_count / the profiling events. */
#define NCCLX_STATIC_MAX_RANKS 32
#define NCCLX_STATIC_SCRATCH_BYTES (512 + 2 * NCCLX_STATIC_MAX_RANKS * NCCLX_STATIC_MAX_RANKS * 8)
int ncclx_alltoallv_static_dev(const void* const* send, const int64_t* sendcounts_dev, void* const* recv,
                               int64_t* recvcounts_dev, uint32_t* status_dev, int R, ncclx_dtype_t dtype,
                               ncclx_stream_t stream);

/* ---- split-phase form and plan slots (section 6.2) ---------- *
 *
 * The paper splits a small-message AllToAll into the control exchange (~50 % of the latency, Table 2)
 * and the payload puts, and removes the exchange from the critical path: handles are exchanged once, and
 * "double buffering" lets "two consecutive AllToAlls ... always use different receive buffers" so that no
 * barrier separates them (L483).  Here the control exchange is steps a1-a3 (transpose, offsets, work list)
 * and the payload is step a4, and the library's workspace is the shared resource that would serialise two
 * calls; so it exists NCCLX_NUM_PLANS times:
 *   ncclx_alltoallv_prepare_dev(plan, ...)  enqueues ONLY a1-a3 into plan slot `plan`: recvcounts_dev is
 *       written, offsets and the work list stay in the slot.  Counts are read when it EXECUTES (L401).
 *   ncclx_alltoallv_execute_dev(plan)       enqueues ONLY a4 for the slot's work list (buffers = the ones given
 *       to prepare).  It may run any number of times per prepare (the claim counters reset themselves).
 * prepare(p) must be ordered before execute(p), and execute(p) before the next prepare(p), by stream order
 * or events; different slots are independent, so the combine's prepare (whose counts are the dispatch's
 * recvcounts, complete as soon as the dispatch's prepare is) can run on a second stream WHILE the dispatch's
 * payload moves.  ncclx_alltoallv_dev == prepare(0) + execute(0) for R > 32, one fused kernel otherwise (slot 0
 * is then left exactly as it was: the fused kernel keeps its offsets in a workspace of its own).  The one-call dynamic and top-k entry points also (re)build slot 0: after them slot 0
 * holds THEIR plan (a dynamic plan can be executed again with ncclx_alltoallv_execute_dev(0); a top-k plan makes
 * it return NCCLX_ERR_ARG).  Tunables (ncclx_set_param) are snapshotted into the slot by prepare: execute uses
 * the values the work list was built with.  Arguments as for ncclx_alltoallv_dev; 0 <= plan < NCCLX_NUM_PLANS;
 * execute returns NCCLX_ERR_ARG for a slot that holds no AllToAllv / AllToAllvDynamic plan.  Both capturable. */
#define NCCLX_NUM_PLANS 4
int ncclx_alltoallv_prepare_dev(int plan, const void* const* send, const int64_t* sendcounts_dev, void* const* recv,
                                int64_t* recvcounts_dev, int R, ncclx_dtype_t dtype, ncclx_stream_t stream);
int ncclx_alltoallv_execute_dev(int plan, ncclx_stream_t stream);

/* Copies the offset matrices of the LAST enqueued ncclx_alltoallv_dev to HOST int64[R*R]
 * arrays (either may be NULL).  Synchronises `stream`; not capturable (NCCLX_ERR_CAPTURE). */
int ncclx_alltoallv_last_offsets(int64_t* soff_host, int64_t* roff_host, int R, ncclx_stream_t stream);

/* Reads and clears the device status word (the OR over all plan slots) into *status_host (bit 0: a
 * negative count was seen).  Synchronises `stream`; not capturable. */
int ncclx_device_status(uint32_t* status_host, ncclx_stream_t stream);

/* ---- AllToAllvDynamic: the paper's full metadata interface (section 6.1.2) ---- *
 *
 * Per sending rank s: send[s] is one contiguous buffer that sendSplitLengths row s cuts into `nsplits`
 * pieces (piece i at element offset O_s[i] = sum_{i'<i} L_s[i']); sendIndices row s is the flattened
 * list of split indices to send, sub-list for rank d = sendIndicesBlockLens[s*R+d] consecutive entries,
 * sub-lists in rank order; a sub-list need not be contiguous and one split may go to several ranks
 * (duplicated experts, L437).  Receive side (L439): recvbuffs[d*R+s] is rank d's array for source s and
 * "the paddings are reserved": every received split lands at the offset it had in the sender's buffer,
 *     recvbuffs[d][s][O_s[idx] .. +L_s[idx]) = send[s][O_s[idx] .. +L_s[idx])  for each idx in s's
 *     sub-list for d;   all other bytes of recvbuffs[d][s] are NOT written;
 *     recvAllSplitLengths[(d*R+s)*nsplits + i] = L_s[i]  (every rank receives all split lengths).
 * All metadata is DEVICE-resident and read when the kernels execute (L401, L409); capturable.
 *
 *   maxIndices    row stride of sendIndices_dev (>= sum_d blockLens[s][d] for every s)
 *   maxBlockLen   upper bound on any block length (= experts per rank incl. redundant ones); sizes the
 *                 work list: R*R*maxBlockLen <= the capacity given to ncclx_init_dynamic
 * Device status bits (ncclx_device_status): 0 negative split length (treated as 0), 1 split index outside
 * [0,nsplits) (skipped), 2 block length < 0 or > maxBlockLen or list overrun (clamped).
 * Each recvbuffs[d][s] must hold sum_i L_s[i] elements and must not overlap any send buffer.
 * Call ncclx_init_dynamic(max_splits, max_segments) once after ncclx_init, outside capture (allocates one
 * descriptor table of max_segments entries per plan slot).
 * Split-phase form (double buffering, L483): ncclx_alltoallv_dynamic_prepare_dev(plan, ...) enqueues only the
 * metadata kernel into plan slot `plan`; ncclx_alltoallv_execute_dev(plan) then moves the payload AND writes
 * recvAllSplitLengths (it rides along with the payload).  ncclx_alltoallv_dynamic_dev == prepare(0) + execute(0). */
int ncclx_init_dynamic(int max_splits, int64_t max_segments);
int ncclx_alltoallv_dynamic_prepare_dev(int plan, const void* const* send, const int64_t* sendSplitLengths_dev, int nsplits,
                                        const int64_t* sendIndices_dev, int maxIndices,
                                        const int64_t* sendIndicesBlockLens_dev, int maxBlockLen, void* const* recvbuffs,
                                        int64_t* recvAllSplitLengths_dev, int R, ncclx_dtype_t dtype, ncclx_stream_t stream);
int ncclx_alltoallv_dynamic_dev(const void* const* send, const int64_t* sendSplitLengths_dev, int nsplits,
                                const int64_t* sendIndices_dev, int maxIndices,
                                const int64_t* sendIndicesBlockLens_dev, int maxBlockLen, void* const* recvbuffs,
                                int64_t* recvAllSplitLengths_dev, int R, ncclx_dtype_t dtype, ncclx_stream_t stream);

/* ---- sum reduction (section 5.3; numeric contract DESIGN.md section 3) -- *
 *
 *     acc = (float) x_0[i];  for k = 1..R-1: acc = acc + (float) x_k[i]     (binary32, RNE,
 *     no FTZ, no reassociation);  out = one round-to-nearest-even conversion of acc to dtype.
 *     A NaN result is canonical (bf16/f16 0x7FFF, f32 0x7FFFFFFF).
 *
 * AllReduce:      recv[r][i] = out[i] for every r, i in [0, count).
 *   send  DEVICE array of R DEVICE pointers to `count` elements; recv likewise.
 *   recv[r] == send[r] (in place) is allowed; any other overlap is undefined.
 * ReduceScatter:  recv[r][j] = out[r*recvcount + j], j in [0, recvcount).
 *   send[k] holds R*recvcount elements; rank r receives contiguous block r (NCCL convention).
 *   recv[r] == send[r] + r*recvcount is allowed; any other overlap is undefined.
 * count == 0 is a no-op.  dtype in {BF16, F32, F16}.  Full speed needs 16-byte aligned
 * pointers (and recvcount*sizeof(dtype) % 16 == 0 for ReduceScatter); otherwise a scalar
 * path with the same arithmetic runs. */
int ncclx_allreduce_sum(const void* const* send, void* const* recv, size_t count, int R,
                        ncclx_dtype_t dtype, ncclx_stream_t stream);
int ncclx_reducescatter_sum(const void* const* send, void* const* recv, size_t recvcount, int R,
                            ncclx_dtype_t dtype, ncclx_stream_t stream);

/* ---- FTAR-style ReduceCopy step (section 5.3, Fig. 9: Reduce / ReduceCopy) ---------- *
 *
 * One pipeline step of the paper's ring AllReduce on local memory: the incoming chunk `a` (from the previous
 * peer) is summed with the local chunk `b`,  r[i] = rn_dtype((float)a[i] + (float)b[i])  (same arithmetic as
 * ncclx_allreduce_sum with R = 2, NaN canonical), and r is written to `out` (local result; Reduce), to
 * `fwd` (the buffer forwarded to the next peer; ReduceCopy, "combine the reduction and forwarding copy"), or
 * to both; either may be NULL but not both ("avoid unnecessary HBM stores in the intermediate forwarding
 * steps").  The message is walked in fixed chunks of `chunk_bytes` (paper: S = 8 MB; 0 selects 8 MiB) by a
 * FIXED grid of `num_ctas` CTAs x 512 threads (paper: 2 CTAs suffice to stay hidden under the network;
 * 0 selects 2) -- the SM-frugal regime, as opposed to the full-chip ncclx_allreduce_sum.  Two inner loops with
 * identical results (NCCLX_PARAM_REDUCECOPY_TMA): software-pipelined 256-bit register loads, or a producer warp
 * feeding a 6-stage shared-memory ring with cp.async.bulk.
 * a, b, out, fwd: DEVICE pointers to `count` elements; out/fwd may alias a or b exactly (in place), other
 * overlap is undefined.  dtype in {BF16, F32, F16}.  32-byte aligned pointers and chunk size take the
 * 256-bit vector path, anything else a scalar path with the same arithmetic.  Capturable. */
int ncclx_reducecopy_sum(const void* a, const void* b, void* out, void* fwd, size_t count, ncclx_dtype_t dtype,
                         size_t chunk_bytes, int num_ctas, ncclx_stream_t stream);

/* ---- top-k MoE dispatch / combine ("which k experts a given token should go to"; Table 3) ---- *
 *
 * Rank s holds T token rows X_s (T x width elements).  The router picked k experts per token and the
 * shuffle (MetaShuffling, L699) ordered the k*T token COPIES by expert; that sorted send buffer stays
 * VIRTUAL here.  Device-resident metadata, read when the kernels execute:
 *   pos_dev          int32[R*T*k]: pos[(s*T+t)*k+j] = row of copy j (router order) of token t in rank s's
 *                    virtual sorted buffer, a permutation of [0, k*T)
 *   sendcounts_rows  int64[R*R]: C[s*R+d] = ROWS of that buffer going to rank d (sum_d = k*T)
 * ncclx_moe_dispatch_topk_dev: the AllToAllv of the virtual buffer with the duplication done on the way --
 *   recv[d][roff[d][s] + (p - soff[s][d])] = X_s[t]  for p = pos[s][t][j] in [soff[s][d], soff[s][d+1]);
 *   recv[d] is packed exactly as by ncclx_alltoallv_dev (rows of width elements); recvcounts_rows_dev = C^T.
 * ncclx_moe_combine_topk_sum_dev: the inverse AllToAllv fused with the fixed-order sum --
 *   out[s][t] = rn_dtype( (..((float)y_0 + y_1) + ..) + y_{k-1} ),  y_j = the row of expert_out[d_j] that
 *   dispatch wrote copy j to; fp32 accumulation in router order j, one rounding, NaN canonical.
 * A position outside [0, sum_d C[s][d]) is skipped (device status bit 1); a token with no valid copy
 * yields +0.  Duplicate positions are undefined.  1 <= k <= 32.  dtype: dispatch any, combine BF16/F32/F16.
 * Rows and bases that are multiples of 32 bytes take the 256-bit path.  Capturable. */
int ncclx_moe_dispatch_topk_dev(const void* const* tokens, const int32_t* pos_dev, const int64_t* sendcounts_rows_dev,
                                void* const* recv, int64_t* recvcounts_rows_dev, int R, int T, int k, int width,
                                ncclx_dtype_t dtype, ncclx_stream_t stream);
int ncclx_moe_combine_topk_sum_dev(const void* const* expert_out, const int32_t* pos_dev,
                                   const int64_t* sendcounts_rows_dev, void* const* out, int R, int T, int k,
                                   int width, ncclx_dtype_t dtype, ncclx_stream_t stream);
/* Plan-slot form (PAPER.md L483 double buffering, for the k > 1 flow of Table 3): the metadata phase (a1, a2: row
 * offsets + recvcounts) goes into plan slot `plan` ONCE per MoE layer, and both the dispatch and the combine of that
 * layer execute against it -- the combine needs the DISPATCH's offsets, so it launches no metadata kernel at all --
 * while the next layer prepares another slot.  prepare(p) must be ordered before the executes that use p, and those
 * before the next prepare(p).  execute returns NCCLX_ERR_ARG for a slot that holds no top-k plan.  R is the plan's. */
int ncclx_moe_topk_prepare_dev(int plan, const int64_t* sendcounts_rows_dev, int64_t* recvcounts_rows_dev, int R,
                               ncclx_stream_t stream);
int ncclx_moe_dispatch_topk_execute_dev(int plan, const void* const* tokens, const int32_t* pos_dev, void* const* recv,
                                        int T, int k, int width, ncclx_dtype_t dtype, ncclx_stream_t stream);
int ncclx_moe_combine_topk_sum_execute_dev(int plan, const void* const* expert_out, const int32_t* pos_dev, void* const* out,
                                           int T, int k, int width, ncclx_dtype_t dtype, ncclx_stream_t stream);

/* ---- host-buffer forms (the end-to-end path: H2D + kernels + D2H inside the call) ------ *
 *
 * Same semantics, but every pointer is a HOST pointer.  `send`/`recv` are HOST arrays of R HOST
 * pointers and the counts are HOST arrays.  When EVERY data buffer in use is pinned (cudaHostAlloc /
 * cudaHostRegister, e.g. torch's pin_memory()), the same kernels read and write the host buffers
 * directly over PCIe (zero-copy: the inbound and outbound halves of the call share the full-duplex
 * link instead of running one after the other; NCCLX_PARAM_HOST_ZERO_COPY = 0 turns it off).
 * Otherwise (pageable memory) the library stages through its own device buffers (grown on demand with
 * cudaMalloc and kept until ncclx_finalize): H2D copies, the device path on `stream`, D2H copies.
 * Either way `stream` is synchronised before returning.  Not capturable.
 * AllToAllv: recv[d] receives exactly sum_s C[s][d] elements; recvcounts_host is filled. */
int ncclx_alltoallv_host(const void* const* send, const int64_t* sendcounts_host, void* const* recv,
                         int64_t* recvcounts_host, int R, ncclx_dtype_t dtype, ncclx_stream_t stream);
int ncclx_allreduce_sum_host(const void* const* send, void* const* recv, size_t count, int R,
                             ncclx_dtype_t dtype, ncclx_stream_t stream);
int ncclx_reducescatter_sum_host(const void* const* send, void* const* recv, size_t recvcount, int R,
                                 ncclx_dtype_t dtype, ncclx_stream_t stream);

/* ---- tuning and measurement (not part of the paper's contract) -------------------------- */

typedef enum {
    NCCLX_PARAM_BULK_MIN_BYTES = 0,     /* 16B-aligned segments >= this many bytes go on the bulk list (32 KiB tiles, TMA in and out);  */
                                        /* smaller or unaligned ones on the vector list (4 KiB pieces, realigned in shared memory). default 1024 */
    NCCLX_PARAM_REDUCE_CTAS_PER_SM = 1, /* reduce grid = this * SM count (1..64), default 16 (4x what fits at once: a short call such  */
                                        /* as config 2 becomes one tile per CTA, dealt out by the hardware scheduler); reductions below */
                                        /* 256 MiB of input run on 64-thread CTAs and twice this many of them                           */
    NCCLX_PARAM_PROFILE = 2,            /* 1: bracket each kernel with CUDA events (never while capturing)                              */
    NCCLX_PARAM_BULK_TILE_SHIFT = 3,    /* log2 bytes of a bulk tile (12..16), default 15                                               */
    NCCLX_PARAM_PDL = 4,                /* 1 (default): programmatic dependent launch -- a kernel's prologue overlaps the tail of the   */
                                        /* kernel before it (reductions: only below 1 GiB of input, and their CTAs prefetch their first */
                                        /* input tiles into L2 while they wait); 0: plain stream order                                  */
    NCCLX_PARAM_COPY_KMAX = 5,          /* max bulk tiles per dynamic claim when segments are short (1..64), default 6                  */
    NCCLX_PARAM_FUSED_MAX_RANKS = 6,    /* ncclx_alltoallv_dev runs as ONE kernel for R <= this (0..32; 0 = never), default 32          */
    NCCLX_PARAM_COPY_BULK_ENGINES = 7,  /* bulk (TMA) engine warps per copy CTA: 1, 2, 4, or 0 (default): chosen on the device -- 4 for */
                                        /* calls of few tiles per SM (latency-bound), 1 for long ones (HBM-bound)                       */
    NCCLX_PARAM_HOST_ZERO_COPY = 8,     /* 1 (default): the *_host calls let the kernels access PINNED host buffers directly           */
    NCCLX_PARAM_REDUCECOPY_TMA = 9,     /* ncclx_reducecopy_sum inner loop: 0 (default) pipelined register loads, 1 TMA-fed smem ring   */
    NCCLX_PARAM_COUNT_
} ncclx_param_t;

/* Process-global; take effect for work lists built AFTER the call (a prepared plan slot keeps its snapshot). */
int ncclx_set_param(int param, int64_t value);
int ncclx_get_param(int param, int64_t* value);

typedef enum {
    NCCLX_KERNEL_COUNTS = 0, /* counts transpose + offsets scan + work list   */
    NCCLX_KERNEL_COPY = 1,   /* byte-balanced segment copy                    */
    NCCLX_KERNEL_REDUCE = 2, /* rank-order sum                                */
    NCCLX_KERNEL_DYN = 3,    /* AllToAllvDynamic metadata kernel (dyn_build)     */
    NCCLX_KERNEL_TOPK = 4,   /* top-k dispatch / combine kernels               */
    NCCLX_KERNEL_FUSED = 5,  /* single-launch AllToAllv (scan + work list + copy in one kernel) */
    NCCLX_KERNEL_COUNT_
} ncclx_kernel_t;

/* With NCCLX_PARAM_PROFILE = 1: total device time (ms, CUDA events on the launch stream) and
 * number of launches of `kernel` since the last ncclx_profile_reset.  Synchronises the
 * recorded events.  ncclx_launch_count works with profiling off (counts every kernel this
 * library launched since init or reset, captured launches counted once at capture). */
int ncclx_profile_read(int kernel, double* total_ms, int64_t* launches);
int ncclx_profile_reset(void);
int64_t ncclx_launch_count(void);

/* HBM streaming micro-probe (measurement aid): one pass of 256-bit accesses over `bytes`
 * (multiple of 32; 32-byte aligned DEVICE pointers).  mode 0 = read-only over src (dst may be NULL),
 * 1 = write-only over dst (src may be NULL; contents become a fixed pattern), 2 = copy src -> dst,
 * 3 = write-only through TMA bulk stores of 32 KiB (bytes a multiple of 32 KiB).  Enqueue
 * only; time it with events.  Gives the practical read / write / copy ceilings of the part. */
int ncclx_stream_probe(int mode, const void* src, void* dst, size_t bytes, ncclx_stream_t stream);
/* Same probe on a FIXED grid of num_ctas >= 1 CTAs x 1024 threads (128 KB of loads in flight per CTA): the per-SM
 * ceiling the SM-frugal ncclx_reducecopy_sum (2 CTAs) is read against. */
int ncclx_stream_probe_ctas(int mode, const void* src, void* dst, size_t bytes, int num_ctas, ncclx_stream_t stream);

/* Number of SMs of the device the library was initialised on (0 before init). */
int ncclx_sm_count(void);

#ifdef __cplusplus
}
#endif
#endif /* NCCLX_B200_H */
