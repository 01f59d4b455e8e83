// psl_static.cuh -- kernels of psl_count_static (include/psl.h): the key histogram counts[K] (a1-a4, a8: how many
// particles every (type, energy, position) bin holds) of DEVICE-resident records, for callers
// that cannot allocate.  k_count_static is k_count_raw<IDX = false, BEAM = 0> (psl_partition.cuh) cut down to one
// contiguous record buffer: the same TMA ring, the same privatised shared-memory histogram, the same per-CTA table
// column.  Its scratch -- the table, the per-CTA statistics and the edge table -- lives in the file-scope device array
// of psl_api.cu; the kernels get its address as an argument.
#pragma once

#include "psl_partition.cuh"

namespace psl {

constexpr uint32_t kStaticMaxKeys = kMaxBuckets;  // 2048
constexpr uint32_t kStaticMaxCols = 320;          // most CTAs of one histogram launch (two per SM)
constexpr uint32_t kStaticMaxEdges = 1025;        // n_ebins <= 1024
// byte offsets inside the scratch array
constexpr uint32_t kStaticEdgesOff = 0;
constexpr uint32_t kStaticStatsOff = 4352;                                               // 1025 floats, rounded up to 256
constexpr uint32_t kStaticTableOff = kStaticStatsOff + kStaticMaxCols * 48;              // SegStats is 48 bytes
constexpr uint32_t kStaticBytes = kStaticTableOff + kStaticMaxKeys * kStaticMaxCols * 4; // 2 641 152 bytes
static_assert(sizeof(SegStats) == 48, "scratch layout");
static_assert(kStaticStatsOff % 256 == 0 && kStaticTableOff % 256 == 0, "scratch layout");
static_assert(kStaticMaxEdges * 4 <= kStaticStatsOff, "scratch layout");

struct CountTotals {  // psl_count_totals
    unsigned long long n_in, n_invalid, n_outside_grid, n_binned;
};

// the edge table travels as a kernel argument, 512 entries at a time
struct EdgeBatch {
    float e[512];
};
__global__ void k_static_edges(float* __restrict__ dst, const __grid_constant__ EdgeBatch eb, uint32_t first, uint32_t m)
{
    for (uint32_t i = threadIdx.x; i < m; i += blockDim.x) dst[first + i] = eb.e[i];
}

// CTA s histograms tiles [n_tiles s / S, n_tiles (s + 1) / S) of the buffer and writes column s of the table
template <bool POS, bool EDGES>
__global__ void __launch_bounds__(kThreads, 2) k_count_static(const uint8_t* __restrict__ records, uint32_t n_records,
                                                             const __grid_constant__ DevGrid g, uint32_t B,
                                                             uint32_t* __restrict__ table, uint32_t stride,
                                                             SegStats* __restrict__ sstats)
{
    extern __shared__ __align__(128) uint8_t smem[];
    const CountSmem L = count_layout(kTile * kRecBytes, kStagesCount, B, g.n_ebins + 1);
    uint32_t* hist = reinterpret_cast<uint32_t*>(smem + L.hist);
    float* s_edges = reinterpret_cast<float*>(smem + L.edges);
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem + L.bars);
    const uint32_t rmask = (1u << L.rlog) - 1u;
    const uint32_t n_tiles = (n_records + kTile - 1) / kTile;
    const Span sp = {0u, n_tiles, 0u, 1u};
    uint32_t t0, t1;
    segment_of(sp, t0, t1);
    const uint32_t n = t1 - t0;
    auto tile_ptr = [&](uint32_t t) { return records + (size_t)t * kTile * kRecBytes; };
    auto tile_count = [&](uint32_t t) { return min((uint32_t)kTile, n_records - t * (uint32_t)kTile); };
    auto stage_ptr = [&](uint32_t i) { return reinterpret_cast<uint32_t*>(smem + L.ring + (i % kStagesCount) * L.stage_bytes); };

    if (threadIdx.x == 0) {
        for (int k = 0; k < kStagesCount; ++k) mbar_init(&bars[k], 1);
        mbar_fence_init();
        for (uint32_t k = 0; k < (uint32_t)kStagesCount && k < n; ++k)
            ring_issue(stage_ptr(k), &bars[k], tile_ptr(t0 + k), tile_count(t0 + k) * kRecBytes);
    }
    for (uint32_t i = threadIdx.x; i < (B << L.rlog); i += kThreads) hist[i] = 0;
    stage_edges(g, s_edges);
    __syncthreads();

    DevBeam none;  // BEAM = 0: never read
    none.has_beam = 0;
    ThreadStats st;
    uint32_t phase_bits = 0;
    for (uint32_t i = 0; i < n; ++i) {
        const uint32_t stage = i % kStagesCount;
        uint32_t* raw = stage_ptr(i);
        const uint32_t count = tile_count(t0 + i);
        ring_acquire(raw, &bars[stage], phase_bits, stage, tile_ptr(t0 + i), count * kRecBytes);
        Rec rec[kRounds];
        bool have[kRounds];
#pragma unroll
        for (int r = 0; r < kRounds; ++r) {
            const int idx = (int)(warp_id() * (uint32_t)kWarpSpan + (uint32_t)r * 32u + lane_id());
            have[r] = idx < (int)count;
            rec[r] = rec_from_smem(raw, have[r] ? idx : 0);
        }
#pragma unroll
        for (int r = 0; r < kRounds; ++r) {
            uint32_t key;
            const int cls = classify<POS, EDGES, 0>(g, none, rec[r], s_edges, key);
            st.n_inv += have[r] & (cls == C_INVALID);
            if (POS) st.n_out += have[r] & (cls == C_OUTSIDE);
            if (have[r] & (cls == C_SURVIVOR)) {
                st.n_surv += 1;
                atomicAdd(&hist[(key << L.rlog) + (lane_id() & rmask)], 1u);
            }
        }
        __syncthreads();  // every thread is done with the stage
        if (threadIdx.x == 0 && i + kStagesCount < n)
            ring_issue(raw, &bars[stage], tile_ptr(t0 + i + kStagesCount), tile_count(t0 + i + kStagesCount) * kRecBytes);
    }
    __syncthreads();
    for (uint32_t b = threadIdx.x; b < B; b += kThreads) {
        uint32_t c = 0;
        for (uint32_t r = 0; r <= rmask; ++r) c += hist[(b << L.rlog) + ((r + lane_id()) & rmask)];
        table[(size_t)b * stride + blockIdx.x] = c;
    }
    write_seg_stats(st, &sstats[blockIdx.x]);
}

// counts[b] = sum over the launch's columns (one warp per key); the last CTA adds up the statistics instead.
// n_cols = 0 (no records): zeros.
__global__ void __launch_bounds__(256) k_static_sum(const uint32_t* __restrict__ table, uint32_t stride, uint32_t n_cols,
                                                    uint32_t K, const SegStats* __restrict__ sstats,
                                                    unsigned long long n_in, uint32_t* __restrict__ counts,
                                                    CountTotals* __restrict__ totals)
{
    if (blockIdx.x == gridDim.x - 1) {
        if (totals == nullptr || warp_id() != 0) return;
        unsigned long long inv = 0, out = 0, surv = 0;
        for (uint32_t c = lane_id(); c < n_cols; c += 32) {
            inv += sstats[c].n_invalid;
            out += sstats[c].n_outside;
            surv += sstats[c].n_surv;
        }
        for (int o = 16; o > 0; o >>= 1) {
            inv += __shfl_xor_sync(0xFFFFFFFFu, inv, o);
            out += __shfl_xor_sync(0xFFFFFFFFu, out, o);
            surv += __shfl_xor_sync(0xFFFFFFFFu, surv, o);
        }
        if (lane_id() == 0) {
            totals->n_in = n_in;
            totals->n_invalid = inv;
            totals->n_outside_grid = out;
            totals->n_binned = surv;
        }
        return;
    }
    const uint32_t b = blockIdx.x * 8 + warp_id();
    if (b >= K) return;
    uint32_t acc = 0;
    for (uint32_t c = lane_id(); c < n_cols; c += 32) acc += table[(size_t)b * stride + c];
    acc = __reduce_add_sync(0xFFFFFFFFu, acc);
    if (lane_id() == 0) counts[b] = acc;
}

}  // namespace psl
