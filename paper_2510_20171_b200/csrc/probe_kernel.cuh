// probe_kernel.cuh -- HBM streaming micro-probe (measurement aid: "run a read-only and a
// write-only streaming micro-probe once to show what a read-dominated mix can reach on this part").  Not on the
// hot path: it gives the practical ceilings the roofline fractions of the real kernels are read against.
//   mode 0  read-only : every 32-byte vector of src is loaded once (256-bit, L1 no-allocate) and folded into a
//                       checksum that is written only if it hits an impossible value (keeps the loads alive)
//   mode 1  write-only: every 32-byte vector of dst is stored once (256-bit, L1 no-allocate)
//   mode 2  copy      : dst = src with the same loads and stores
//   mode 3  write-only through the TMA: dst is filled with cp.async.bulk shared->global stores of 32 KiB
#pragma once
#include "common.cuh"

namespace xdev {

constexpr int PROBE_THREADS = 256;         // full-chip form: 8 CTAs per SM
constexpr int PROBE_THREADS_FEW = 1024;    // few-CTA form (per-SM ceiling): one CTA fills an SM, 128 KB of loads in flight
constexpr int PROBE_UNROLL = 4;

template <int NT>
__global__ void __launch_bounds__(NT) stream_probe_kernel(int mode, const unsigned char* src, unsigned char* dst,
                                                                      unsigned long long nvec, unsigned int* sink) {
    const unsigned long long stride = (unsigned long long)gridDim.x * NT * PROBE_UNROLL;
    unsigned int acc = 0;
    for (unsigned long long base = (unsigned long long)blockIdx.x * NT * PROBE_UNROLL; base < nvec; base += stride) {
        u32x8 v[PROBE_UNROLL];
#pragma unroll
        for (int u = 0; u < PROBE_UNROLL; ++u) {
            const unsigned long long i = base + (unsigned long long)u * NT + threadIdx.x;
            if (mode != 1) {
                if (i < nvec) v[u] = ld_stream256(src + i * 32);
            } else {
                v[u].lo = make_uint4((unsigned int)i, 1u, 2u, 3u);
                v[u].hi = make_uint4(4u, 5u, 6u, 7u);
            }
        }
#pragma unroll
        for (int u = 0; u < PROBE_UNROLL; ++u) {
            const unsigned long long i = base + (unsigned long long)u * NT + threadIdx.x;
            if (i < nvec) {
                if (mode == 0) acc ^= v[u].lo.x ^ v[u].lo.y ^ v[u].lo.z ^ v[u].lo.w ^ v[u].hi.x ^ v[u].hi.y ^ v[u].hi.z ^ v[u].hi.w;
                else st_stream256(dst + i * 32, v[u]);
            }
        }
    }
    if (mode == 0 && acc == 0x9e3779b9u) *sink = acc;      // practically never true: only keeps the loads observable
}

constexpr int PROBE_BULK_BYTES = 32 * 1024;

__global__ void __launch_bounds__(128) stream_probe_bulk_store_kernel(unsigned char* dst, unsigned long long nchunks) {
    __shared__ __align__(128) unsigned char buf[PROBE_BULK_BYTES];
    for (int i = threadIdx.x; i < PROBE_BULK_BYTES / 4; i += 128) reinterpret_cast<unsigned int*>(buf)[i] = (unsigned int)i;
    fence_proxy_async_smem();
    __syncthreads();
    if (threadIdx.x == 0) {
        for (unsigned long long c = blockIdx.x; c < nchunks; c += gridDim.x) {
            bulk_s2g(dst + c * PROBE_BULK_BYTES, smem_u32(buf), PROBE_BULK_BYTES);
            bulk_commit();
            bulk_wait_read<6>();           // the source never changes; only bound the queue depth
        }
        bulk_wait_all<0>();
    }
}

}  // namespace xdev
