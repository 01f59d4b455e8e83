// psl_index.cuh -- small kernels around the PSL index (paper method 3): pass B's histogram over
// the keyed records, the SoA view of the bare index, offsets[] by search over the sorted keys.  The two sort passes
// themselves are in psl_index_big.cuh.
#pragma once

#include "psl_bigtile.cuh"

namespace psl {

constexpr int kIdxMaxLo = 2048;   // most buckets of pass A
constexpr int kIdxMaxHi = 2048;   // most buckets of pass B
__device__ __forceinline__ void ring_issue_stream(uint32_t* s_dst, uint64_t* bar, const void* src, uint32_t bytes)
{
    if (bulk_ok(src, bytes)) {
        mbar_expect_tx(bar, bytes);
        tma_load_1d_stream(s_dst, src, bytes, bar);
    }
}

// INDEX pass B count: histogram of the high digits (key >> lo_bits) over the CTA's segment of the keyed
// records.  Reads the key word of every 32-byte record.
__global__ void __launch_bounds__(kThreads) k_count_keys(const uint4* __restrict__ aos, const uint32_t* __restrict__ n_ptr,
                                                        uint32_t B, uint32_t lo_bits, uint32_t* __restrict__ table,
                                                        uint32_t stride, uint32_t split)
{
    extern __shared__ __align__(128) uint8_t smem[];
    uint32_t* hist = reinterpret_cast<uint32_t*>(smem);
    const CountSmem L = count_layout(0, 0, B, 0);
    const uint32_t rmask = (1u << L.rlog) - 1u;
    const uint32_t n = *n_ptr;
    Span sp = {0u, (n + kTile - 1) / kTile, 0u, split};
    uint32_t t0, t1;
    split_segment_of(sp, t0, t1);
    for (uint32_t i = threadIdx.x; i < (B << L.rlog); i += kThreads) hist[i] = 0;
    __syncthreads();
    const uint32_t first = t0 * kTile, last = min(n, t1 * (uint32_t)kTile);
    const uint32_t* keys = reinterpret_cast<const uint32_t*>(aos);
#pragma unroll 4
    for (uint32_t i = first + threadIdx.x; i < last; i += kThreads) {
        const uint32_t hi = __ldg(keys + 8 * (size_t)i) >> lo_bits;
        atomicAdd(&hist[(hi << L.rlog) + (lane_id() & rmask)], 1u);
    }
    __syncthreads();
    for (uint32_t b = threadIdx.x; b < B; b += kThreads) {
        uint32_t c = 0;
        for (uint32_t r = 0; r <= rmask; ++r) c += hist[(b << L.rlog) + ((r + lane_id()) & rmask)];
        table[(size_t)b * stride + blockIdx.x] = c;
    }
}

// The bare index as SoA arrays (psl_build_batches with beam == NULL): a streaming transpose of the keyed records.
__global__ void __launch_bounds__(256) k_index_to_soa(const uint4* __restrict__ aos, const uint32_t* __restrict__ n_ptr, IdxOut out)
{
    const uint32_t n = *n_ptr;
    for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
        const uint4 a = __ldg(aos + 2 * (size_t)i), b = __ldg(aos + 2 * (size_t)i + 1);
        out.E[i] = __uint_as_float(a.y);
        out.x[i] = __uint_as_float(a.z);
        out.y[i] = __uint_as_float(a.w);
        out.u[i] = __uint_as_float(b.x);
        out.v[i] = __uint_as_float(b.y);
        out.wt[i] = __uint_as_float(b.z);
        out.src[i] = b.w;
    }
}

// offsets[k] = number of index slots whose key is < k (binary search over the sorted keyed records; k = 0..K)
__global__ void k_offsets_by_search_keyed(const uint4* __restrict__ aos, const uint32_t* __restrict__ n_ptr, uint32_t K,
                                          uint32_t* __restrict__ offsets)
{
    uint32_t k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k > K) return;
    const uint32_t* keys = reinterpret_cast<const uint32_t*>(aos);
    uint32_t lo = 0, hi = *n_ptr;
    while (lo < hi) {
        uint32_t mid = lo + ((hi - lo) >> 1);
        if (__ldg(keys + 8 * (size_t)mid) < k) lo = mid + 1; else hi = mid;
    }
    offsets[k] = lo;
}

}  // namespace psl
