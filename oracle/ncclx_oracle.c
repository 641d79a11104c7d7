/*
 * ncclx_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * A plain, slow, obviously-correct CPU statement of what the hot path computes,
 * written from the paper (/root/reference/PAPER.md, cited as L<n>) and from the
 * readings listed in DESIGN.md section 3.  It shares no code, header, table or helper with
 * the CUDA path under paper_2510_20171_b200/csrc/ and neither includes the other.
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
 * legs may load it.
 *
 * Both operations have exactly one correct result, so the oracle is the DEFINITION
 * written out, not an algorithm:
 *
 *   AllToAllv with by-reference split counts (section 6.1 "send counts
 *   contains how much data to be sent to each peer"; L401-409 metadata by reference;
 *   L419 "update other metadata such as receive counts and return them"; L429
 *   sendbuff is one contiguous buffer split by the counts; L439 receive side):
 *       RC[d][s]   = C[s][d]
 *       soff[s][d] = sum_{d'<d} C[s][d']          (exclusive, along row s)
 *       roff[d][s] = sum_{s'<s} C[s'][d]          (exclusive, down column d)
 *       recv[d][roff[d][s] .. +C[s][d]) = send[s][soff[s][d] .. +C[s][d])   bytes verbatim
 *     every byte of recv[d] outside those ranges keeps its pre-call value.
 *
 *   Sum reduction behind AllReduce / ReduceScatter (section 5.3 "combine the
 *   reduction and forwarding copy in the ReduceScatter phase"; the numeric contract
 *   is BASELINE.json's: fp32 accumulate in rank order 0..R-1, one rounding):
 *       acc = (float)x_0[i]; for k = 1..R-1: acc = acc + (float)x_k[i]   (binary32, RNE)
 *       out = round-to-nearest-even to the output type, NaN canonicalised
 *     AllReduce: the same value to every out[r][i].
 *     ReduceScatter: out[r][j] from element r*n + j (contiguous block r to rank r).
 *
 * Parity pins: tests/test_oracle_*.py (hand-worked example, conservation, transpose,
 * round trip, numpy block transpose, tagged payload closed form, IEEE rounding vectors,
 * order-distinguishing vector, exact small-integer sums, fp64 error bound).  Nothing in
 * this file is "parity unpinned".
 *
 * Build: gcc -O2 -fno-fast-math -ffp-contract=off -fopenmp -shared -fPIC (oracle/build.py).
 * The only parallelism is an OpenMP "for" over independent destination ranks / element
 * ranges; per element the arithmetic order is exactly the definition's.
 */
#include <stddef.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

enum { ORACLE_BF16 = 0, ORACLE_F32 = 1, ORACLE_F16 = 2, ORACLE_U8 = 3 };

static int elem_size(int dtype) {
    switch (dtype) {
    case ORACLE_BF16: return 2;
    case ORACLE_F32:  return 4;
    case ORACLE_F16:  return 2;
    case ORACLE_U8:   return 1;
    default:          return 0;
    }
}

int oracle_elem_size(int dtype) { return elem_size(dtype); }

/* ---- bit-level helpers (IEEE 754 definitions, written out) ------------------------- */

static float bits_to_f32(uint32_t u) { float f; memcpy(&f, &u, 4); return f; }
static uint32_t f32_to_bits(float f) { uint32_t u; memcpy(&u, &f, 4); return u; }

/* bf16 is the top 16 bits of binary32: widening is exact. */
static float bf16_to_f32(uint16_t h) { return bits_to_f32((uint32_t)h << 16); }

/* binary32 -> bf16, round to nearest, ties to even; NaN -> 0x7FFF (reading 13). */
uint16_t oracle_f32_to_bf16_rne(uint32_t u) {
    if ((u & 0x7F800000u) == 0x7F800000u && (u & 0x007FFFFFu) != 0) return 0x7FFF;
    return (uint16_t)((u + 0x7FFFu + ((u >> 16) & 1u)) >> 16);
}

/* binary16 -> binary32 (exact). */
static float f16_to_f32(uint16_t h) {
    uint32_t sign = (uint32_t)(h & 0x8000u) << 16;
    uint32_t exp = (h >> 10) & 0x1Fu;
    uint32_t man = h & 0x3FFu;
    if (exp == 0x1F) return bits_to_f32(sign | 0x7F800000u | (man << 13));
    if (exp == 0) {
        if (man == 0) return bits_to_f32(sign);
        /* subnormal half: value = man * 2^-24, normalise */
        int e = -1;
        do { man <<= 1; e++; } while ((man & 0x400u) == 0);
        man &= 0x3FFu;
        return bits_to_f32(sign | ((uint32_t)(127 - 15 - e) << 23) | (man << 13));
    }
    return bits_to_f32(sign | ((exp + 127 - 15) << 23) | (man << 13));
}

/* binary32 -> binary16, round to nearest even; NaN -> 0x7FFF. */
uint16_t oracle_f32_to_f16_rne(uint32_t u) {
    uint32_t sign = (u >> 16) & 0x8000u;
    uint32_t a = u & 0x7FFFFFFFu;
    if (a > 0x7F800000u) return 0x7FFF;
    if (a == 0x7F800000u) return (uint16_t)(sign | 0x7C00u);
    int32_t e = (int32_t)(a >> 23) - 127;          /* unbiased exponent (for normals) */
    uint32_t m = a & 0x007FFFFFu;
    if (a < 0x00800000u) return (uint16_t)sign;    /* fp32 subnormal: far below half's range */
    if (e > 15) return (uint16_t)(sign | 0x7C00u); /* >= 2^16: overflow to inf */
    if (e >= -14) {
        /* normal half candidate: 10-bit mantissa, drop 13 bits with RNE */
        uint32_t h = ((uint32_t)(e + 15) << 10) | (m >> 13);
        uint32_t rem = m & 0x1FFFu;
        if (rem > 0x1000u || (rem == 0x1000u && (h & 1u))) h++;   /* carry may reach inf: correct */
        return (uint16_t)(sign | h);
    }
    if (e < -25) return (uint16_t)sign;            /* below half the smallest subnormal */
    /* subnormal half: value = (1.m) * 2^e, unit = 2^-24 */
    uint32_t full = m | 0x00800000u;               /* 24-bit significand */
    int shift = -e - 14 + 13;                      /* bits to drop: 14..24 */
    uint32_t h = full >> shift;
    uint32_t rem = full & ((1u << shift) - 1u);
    uint32_t half = 1u << (shift - 1);
    if (rem > half || (rem == half && (h & 1u))) h++;
    return (uint16_t)(sign | h);
}

static uint32_t canon_nan_f32(float f) {
    uint32_t u = f32_to_bits(f);
    if ((u & 0x7FFFFFFFu) > 0x7F800000u) return 0x7FFFFFFFu;
    return u;
}

static float load_as_f32(const void* p, size_t i, int dtype);
static void store_from_f32(void* p, size_t i, int dtype, float acc);

/* ---- AllToAllv --------------------------------------------------------------------- */

/* Steps 1-3 of SURVEY section 8(c.1).  Negative counts are reported (return value = how many)
 * and treated as 0 (reading 9).  All arrays are R*R row-major int64. */
int oracle_alltoallv_offsets(const int64_t* C, int R, int64_t* RC, int64_t* soff, int64_t* roff) {
    int neg = 0;
    for (int s = 0; s < R; s++)
        for (int d = 0; d < R; d++) {
            int64_t c = C[(size_t)s * R + d];
            if (c < 0) { neg++; c = 0; }
            RC[(size_t)d * R + s] = c;
        }
    for (int s = 0; s < R; s++) {
        int64_t run = 0;
        for (int d = 0; d < R; d++) {
            soff[(size_t)s * R + d] = run;
            run += RC[(size_t)d * R + s];
        }
    }
    for (int d = 0; d < R; d++) {
        int64_t run = 0;
        for (int s = 0; s < R; s++) {
            roff[(size_t)d * R + s] = run;
            run += RC[(size_t)d * R + s];
        }
    }
    return neg;
}

/* Step 4: the copies.  send[s], recv[d] are host pointers; recv keeps its pre-call bytes
 * everywhere the definition does not write.  scratch = 3*R*R int64 supplied by the caller
 * (RC is returned through RC; soff/roff through scratch so the caller can compare them). */
int oracle_alltoallv(const void* const* send, const int64_t* C, void* const* recv, int64_t* RC,
                     int64_t* soff, int64_t* roff, int R, int dtype, int nthreads) {
    int e = elem_size(dtype);
    if (e == 0 || R < 1) return -1;
    int neg = oracle_alltoallv_offsets(C, R, RC, soff, roff);
    if (nthreads < 1) nthreads = 1;
#pragma omp parallel for schedule(dynamic, 1) num_threads(nthreads)
    for (int d = 0; d < R; d++)
        for (int s = 0; s < R; s++) {
            int64_t c = RC[(size_t)d * R + s];
            if (c > 0)
                memcpy((char*)recv[d] + roff[(size_t)d * R + s] * e,
                       (const char*)send[s] + soff[(size_t)s * R + d] * e, (size_t)c * e);
        }
    return neg;
}

/* ---- AllToAllvDynamic: the paper's full metadata interface (section 6.1.2) ----
 *
 * Per sending rank s (L429): sendbuff = one contiguous buffer; sendSplitLengths L_s[0..n) split it into
 * n pieces, piece i at element offset O_s[i] = sum_{i'<i} L_s[i']; sendIndices = the flattened 2-D list
 * "which splits go to which rank" (sub-list of rank d = blockLens[s][d] consecutive entries, sub-lists in
 * rank order; entries need not be contiguous and a split may appear in several sub-lists: duplicated
 * experts, L437).  Receive side (L439): recvbuffs[d][s] is rank d's array for source s; "the paddings
 * are reserved": a received split keeps the offset it had in the sender's buffer (Fig. 17: rank 1's data
 * from rank 0 = splits {0,2,3} "contains the padding of index 1"), so
 *     recvbuffs[d][s][O_s[idx] .. +L_s[idx]) = send[s][O_s[idx] .. +L_s[idx])   for every idx in s's
 *     sub-list for d;  everything else in recvbuffs[d][s] keeps its pre-call bytes;
 * recvAllSplitLengths[d][s][i] = L_s[i]: every rank receives ALL ranks' split lengths (L439).
 * Readings: negative lengths count as 0 (status bit 0); an index outside [0,n) is
 * skipped (bit 1); a block length < 0 or > maxBlockLen is clamped (bit 2).
 * Arrays: L = R*n, indices = R*maxIndices (row stride), blockLens = R*R, recvbuffs = R*R host pointers
 * [d*R+s], recvAll = R*R*n.  Returns the status bits. */
int oracle_alltoallv_dynamic(const void* const* send, const int64_t* L, int n, const int64_t* indices,
                             int maxIndices, const int64_t* blockLens, int maxBlockLen, void* const* recvbuffs,
                             int64_t* recvAll, int R, int dtype) {
    int e = elem_size(dtype);
    if (e == 0 || R < 1 || n < 1) return -1;
    int status = 0;
    for (int d = 0; d < R; d++)
        for (int s = 0; s < R; s++)
            for (int i = 0; i < n; i++) {
                int64_t l = L[(size_t)s * n + i];
                if (l < 0) { status |= 1; l = 0; }
                recvAll[((size_t)d * R + s) * n + i] = l;
            }
    for (int s = 0; s < R; s++) {
        int64_t pos = 0;                                   /* read position in s's index list */
        for (int d = 0; d < R; d++) {
            int64_t bl = blockLens[(size_t)s * R + d];
            if (bl < 0) { status |= 4; bl = 0; }
            if (bl > maxBlockLen) { status |= 4; bl = maxBlockLen; }
            for (int64_t j = 0; j < bl; j++) {
                if (pos + j >= maxIndices) { status |= 4; break; }
                int64_t idx = indices[(size_t)s * maxIndices + pos + j];
                if (idx < 0 || idx >= n) { status |= 2; continue; }
                int64_t off = 0;
                for (int64_t i = 0; i < idx; i++) { int64_t l = L[(size_t)s * n + i]; off += l > 0 ? l : 0; }
                int64_t len = L[(size_t)s * n + idx];
                if (len > 0)
                    memcpy((char*)recvbuffs[(size_t)d * R + s] + off * e, (const char*)send[s] + off * e, (size_t)len * e);
            }
            pos += bl;
        }
    }
    return status;
}

/* ---- top-k MoE dispatch / combine (Table 3) -----
 *
 * The router sends every token to k experts (L383); MetaShuffling then sorts the k*T token COPIES by
 * expert into the AllToAllv send buffer (L699).  Here that sorted buffer is VIRTUAL: pos[s][t*k+j] = p
 * says "the j-th copy (router order j = 0..k-1) of rank s's token t sits at row p of rank s's sorted
 * send buffer", and C[s][d] (in ROWS) splits that buffer by destination exactly as in the plain call.
 *   dispatch: recv[d][roff[d][s] + (p - soff[s][d])] = X_s[t]       for the d with soff[s][d] <= p < soff[s][d+1]
 *             (the plain AllToAllv of the virtual buffer; the token row is duplicated on the way)
 *   combine:  Z_s[t] = rn_dtype( (..((float)y_0 + y_1) + ..) + y_{k-1} ),  y_j = Y[d_j][that same row],
 *             fp32 accumulation in router order j, ONE rounding -- the inverse AllToAllv fused with the
 *             fixed-order sum of this build's reduction (no weights: scaling is the caller's, reading 11).
 * A position outside [0, sum_d C[s][d]) is skipped (status bit 1); a token with no valid copy gets +0.
 * tokens[s] / out[s]: T rows of `width` elements; recv[d] / Y[d]: packed like the plain call. */
static int locate_row(const int64_t* soff, const int64_t* roff, const int64_t* RC, int R, int s, int64_t p,
                      int* d_out, int64_t* row_out) {
    for (int d = 0; d < R; d++) {
        int64_t lo = soff[(size_t)s * R + d], c = RC[(size_t)d * R + s];
        if (p >= lo && p < lo + c) { *d_out = d; *row_out = roff[(size_t)d * R + s] + (p - lo); return 1; }
    }
    return 0;
}

int oracle_moe_dispatch_topk(const void* const* tokens, const int32_t* pos, const int64_t* Crows, void* const* recv,
                             int64_t* RC, int64_t* soff, int64_t* roff, int R, int T, int k, int width, int dtype) {
    int e = elem_size(dtype);
    if (e == 0 || R < 1 || T < 0 || k < 1 || width < 1) return -1;
    int status = oracle_alltoallv_offsets(Crows, R, RC, soff, roff) ? 1 : 0;
    size_t row = (size_t)width * e;
    for (int s = 0; s < R; s++)
        for (int t = 0; t < T; t++)
            for (int j = 0; j < k; j++) {
                int64_t p = pos[((size_t)s * T + t) * k + j];
                int d; int64_t r;
                if (p < 0 || !locate_row(soff, roff, RC, R, s, p, &d, &r)) { status |= 2; continue; }
                memcpy((char*)recv[d] + (size_t)r * row, (const char*)tokens[s] + (size_t)t * row, row);
            }
    return status;
}

int oracle_moe_combine_topk_sum(const void* const* Y, const int32_t* pos, const int64_t* Crows, void* const* out,
                                int R, int T, int k, int width, int dtype) {
    if (R < 1 || T < 0 || k < 1 || width < 1 || !(dtype == ORACLE_BF16 || dtype == ORACLE_F32 || dtype == ORACLE_F16)) return -1;
    size_t rr = (size_t)R * R;
    int64_t* RC = (int64_t*)malloc(3 * rr * sizeof(int64_t));
    int64_t* soff = RC + rr; int64_t* roff = soff + rr;
    int status = oracle_alltoallv_offsets(Crows, R, RC, soff, roff) ? 1 : 0;
    for (int s = 0; s < R; s++)
        for (int t = 0; t < T; t++)
            for (int c = 0; c < width; c++) {
                float acc = 0.0f;
                int have = 0;
                for (int j = 0; j < k; j++) {
                    int64_t p = pos[((size_t)s * T + t) * k + j];
                    int d; int64_t r;
                    if (p < 0 || !locate_row(soff, roff, RC, R, s, p, &d, &r)) { status |= 2; continue; }
                    float y = load_as_f32(Y[d], (size_t)r * width + c, dtype);
                    acc = have ? acc + y : y;
                    have = 1;
                }
                store_from_f32(out[s], (size_t)t * width + c, dtype, acc);
            }
    free(RC);
    return status;
}

/* ---- sum reduction ------------------------------------------------------------------ */

static float load_as_f32(const void* p, size_t i, int dtype) {
    switch (dtype) {
    case ORACLE_BF16: return bf16_to_f32(((const uint16_t*)p)[i]);
    case ORACLE_F16:  return f16_to_f32(((const uint16_t*)p)[i]);
    default:          return ((const float*)p)[i];
    }
}

static void store_from_f32(void* p, size_t i, int dtype, float acc) {
    switch (dtype) {
    case ORACLE_BF16: ((uint16_t*)p)[i] = oracle_f32_to_bf16_rne(f32_to_bits(acc)); break;
    case ORACLE_F16:  ((uint16_t*)p)[i] = oracle_f32_to_f16_rne(f32_to_bits(acc)); break;
    default:          ((uint32_t*)p)[i] = canon_nan_f32(acc); break;
    }
}

/* One output element: fp32 accumulate in rank order, starting from x_0 (reading 11). */
static float reduce_one(const void* const* send, size_t i, int R, int dtype) {
    float acc = load_as_f32(send[0], i, dtype);   /* built without fast-math: no reassociation; SSE: no widening */
    for (int k = 1; k < R; k++) {
        float x = load_as_f32(send[k], i, dtype);
        acc = acc + x;
    }
    return acc;
}

int oracle_allreduce_sum(const void* const* send, void* const* recv, size_t count, int R, int dtype,
                         int nthreads) {
    if (R < 1 || !(dtype == ORACLE_BF16 || dtype == ORACLE_F32 || dtype == ORACLE_F16)) return -1;
    if (nthreads < 1) nthreads = 1;
#pragma omp parallel for schedule(static) num_threads(nthreads)
    for (size_t i = 0; i < count; i++) {
        float acc = reduce_one(send, i, R, dtype);
        for (int r = 0; r < R; r++) store_from_f32(recv[r], i, dtype, acc);
    }
    return 0;
}

/* send[k] holds R*recvcount elements; recv[r] receives block r (reading 16). */
int oracle_reducescatter_sum(const void* const* send, void* const* recv, size_t recvcount, int R,
                             int dtype, int nthreads) {
    if (R < 1 || !(dtype == ORACLE_BF16 || dtype == ORACLE_F32 || dtype == ORACLE_F16)) return -1;
    if (nthreads < 1) nthreads = 1;
    for (int r = 0; r < R; r++) {
#pragma omp parallel for schedule(static) num_threads(nthreads)
        for (size_t j = 0; j < recvcount; j++) {
            float acc = reduce_one(send, (size_t)r * recvcount + j, R, dtype);
            store_from_f32(recv[r], j, dtype, acc);
        }
    }
    return 0;
}

/* Sampled form for full-size parity: out[t] = reduction of element idx[t] over the R
 * gathered inputs vals[k*T + t] (already gathered by the caller), same arithmetic. */
int oracle_reduce_samples(const void* vals, void* out, size_t T, int R, int dtype) {
    if (R < 1 || !(dtype == ORACLE_BF16 || dtype == ORACLE_F32 || dtype == ORACLE_F16)) return -1;
    int e = elem_size(dtype);
    for (size_t t = 0; t < T; t++) {
        float acc = load_as_f32(vals, t, dtype);
        for (int k = 1; k < R; k++) {
            float x = load_as_f32((const char*)vals + (size_t)k * T * e, t, dtype);
            acc = acc + x;
        }
        store_from_f32(out, t, dtype, acc);
    }
    return 0;
}
