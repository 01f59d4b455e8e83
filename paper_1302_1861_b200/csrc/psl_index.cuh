// psl_index.cuh -- the one-off sort behind the PSL index (paper method 3): two stable LSD
// passes over the full key, split into two balanced digits key = hi * 2^s + lo (each <= 2048 buckets).
//
//   pass A: raw 28-byte records -> 32-byte keyed records {key, E, x, y, u, v, wt, src}, stably partitioned by lo
//   pass B: keyed records -> the index: keyed records sorted by the full key (stable partition by hi)
//
// With ~1100 buckets and 1024-record tiles a tile holds about one record per bucket, so there are no runs to
// stage: every record is written once as ONE full 32-byte sector by a pair of lanes (one request per sector;
// measured on B200: 35 G sectors/s against 17.7 G/s when a thread writes the two halves itself, DESIGN.md
// "Kernels").  Ranks: per-warp private uint16 counters + __match_any_sync, a 16-byte-vector scan over the 8
// warps, the running first free slot of every bucket kept in registers (thread t owns buckets 8t..8t+7).
#pragma once

#include "psl_bigtile.cuh"

namespace psl {

constexpr int kIdxMaxLo = 2048;   // most buckets of pass A
constexpr int kIdxMaxHi = 2048;   // most buckets of pass B
constexpr int kStagesIdxA = 2;

struct IdxASmem {
    uint32_t ring, stage_bytes, cnt, run, misc, skey, sdest, edges, desc, bars, total;
};

__host__ __device__ inline IdxASmem idx_a_layout(uint32_t B, uint32_t n_edges)
{
    IdxASmem L;
    uint32_t p = 0;
    L.stage_bytes = round_up(kTile * kRecBytes, 128);
    L.ring = p;  p += kStagesIdxA * L.stage_bytes;
    L.cnt = p;   p += round_up(kWarps * round_up(B, 8) * 2, 16);  // [kWarps][Bp] uint16 running counts
    L.run = p;   p += round_up(B * 4, 16);   // first slot of every bucket for this tile
    L.misc = p;  p += 64 * 4;
    L.skey = p;  p += kTile * 4;             // full key of every record of the tile, kNone = dropped
    L.sdest = p; p += kTile * 4;             // slot of every record
    L.edges = p; p += round_up(n_edges * 4, 16);
    L.desc = p;  p += kStagesIdxA * 16;
    L.bars = p;  p += kStagesIdxA * 8;
    L.total = p;
    return L;
}

__device__ __forceinline__ void ring_issue_stream(uint32_t* s_dst, uint64_t* bar, const void* src, uint32_t bytes)
{
    if (bulk_ok(src, bytes)) {
        mbar_expect_tx(bar, bytes);
        tma_load_1d_stream(s_dst, src, bytes, bar);
    }
}

template <bool POS, bool EDGES>
__global__ void __launch_bounds__(kThreads, 3) k_scatter_idx_a(const ChunkDesc* __restrict__ chunks, uint32_t n_chunks,
                                                              Span sp, const __grid_constant__ DevGrid g,
                                                              const __grid_constant__ DevBeam bm, uint32_t B,
                                                              uint32_t lo_bits, const uint32_t* __restrict__ table,
                                                              uint32_t stride, uint4* __restrict__ aos)
{
    extern __shared__ __align__(128) uint8_t smem[];
    __shared__ uint32_t s_grp[kWarps][32];  // warp_rank_claim's group words
    s_grp[threadIdx.x >> 5][threadIdx.x & 31] = 0u;
    const IdxASmem L = idx_a_layout(B, g.n_ebins + 1);
    uint32_t* run = reinterpret_cast<uint32_t*>(smem + L.run);
    uint32_t* skey = reinterpret_cast<uint32_t*>(smem + L.skey);
    uint32_t* sdest = reinterpret_cast<uint32_t*>(smem + L.sdest);
    float* s_edges = reinterpret_cast<float*>(smem + L.edges);
    TileDesc* s_desc = reinterpret_cast<TileDesc*>(smem + L.desc);
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem + L.bars);
    const uint32_t w = warp_id();
    const uint32_t lo_mask = (1u << lo_bits) - 1u;
    const uint32_t col = sp.col0 + blockIdx.x * sp.split;

    uint32_t t0, t1;
    segment_of(sp, t0, t1);
    const uint32_t n = t1 - t0;
    ChunkDesc ccur = {nullptr, 0u, 0u, 0u, 0u};  // thread 0: the chunk of the tile it described last
    if (threadIdx.x == 0) {
        for (int k = 0; k < kStagesIdxA; ++k) mbar_init(&bars[k], 1);
        mbar_fence_init();
        for (uint32_t k = 0; k < (uint32_t)kStagesIdxA && k < n; ++k) {
            TileDesc d = raw_tile(chunks, n_chunks, t0 + k, ccur);
            s_desc[k] = d;
            ring_issue_stream(reinterpret_cast<uint32_t*>(smem + L.ring + k * L.stage_bytes), &bars[k], d.ptr, d.count * kRecBytes);
        }
    }
    const uint32_t Bp = round_up(B, 8);
    uint16_t* cnt = reinterpret_cast<uint16_t*>(smem + L.cnt);
    uint32_t* misc = reinterpret_cast<uint32_t*>(smem + L.misc);
    {
        uint32_t* cz = reinterpret_cast<uint32_t*>(cnt);
        for (uint32_t k = threadIdx.x; k < kWarps * Bp / 2; k += kThreads) cz[k] = 0;
    }
    uint32_t grun[8];  // thread t keeps the running first free slot of buckets 8t..8t+7
#pragma unroll
    for (int k = 0; k < 8; ++k) {
        uint32_t b = threadIdx.x * 8 + k;
        grun[k] = b < B ? table[(size_t)b * stride + col] : 0u;
    }
    stage_edges(g, s_edges);
    __syncthreads();

    uint32_t phase_bits = 0;
    for (uint32_t i = 0; i < n; ++i) {
        const uint32_t stage = i % kStagesIdxA;
        uint32_t* raw = reinterpret_cast<uint32_t*>(smem + L.ring + stage * L.stage_bytes);
        const TileDesc td = s_desc[stage];
        ring_acquire(raw, &bars[stage], phase_bits, stage, td.ptr, td.count * kRecBytes);

        // keys (a1-a4) and stable ranks inside the warp's 128 consecutive records
        uint32_t packed[kRounds];  // key << 9 | rank   (key < 2^22)
        {
            Rec rec[kRounds];
#pragma unroll
            for (int r = 0; r < kRounds; ++r) {
                int idx = w * kWarpSpan + r * 32 + lane_id();
                rec[r] = rec_from_smem(raw, idx < (int)td.count ? idx : 0);
                if (g.apr) {
                    apr_apply(g.apr_seed, td.first_index + (uint32_t)idx, rec[r]);
                    if (idx < (int)td.count) {
                        uint32_t* p = raw + idx * kRecWords;
                        p[2] = __float_as_uint(rec[r].x); p[3] = __float_as_uint(rec[r].y);
                        p[4] = __float_as_uint(rec[r].u); p[5] = __float_as_uint(rec[r].v);
                    }
                }
            }
#pragma unroll
            for (int r = 0; r < kRounds; ++r) {
                int idx = w * kWarpSpan + r * 32 + lane_id();
                uint32_t key;
                int cls = classify<POS, EDGES, 0>(g, bm, rec[r], s_edges, key);
                packed[r] = (idx < (int)td.count && cls == C_SURVIVOR) ? key : kNone;
            }
            uint32_t bk[kRounds], rk[kRounds];
#pragma unroll
            for (int r = 0; r < kRounds; ++r) bk[r] = packed[r] == kNone ? kNone : (packed[r] & lo_mask);
            warp_rank_claim<kRounds>(bk, rk, cnt + w * Bp, s_grp[w]);
#pragma unroll
            for (int r = 0; r < kRounds; ++r) packed[r] = packed[r] == kNone ? kNone : ((packed[r] << 9) | rk[r]);
        }
        __syncthreads();
        finish_ranks<false>(cnt, B, Bp, run, nullptr, misc, grun);
#pragma unroll
        for (int r = 0; r < kRounds; ++r) {
            const uint32_t idx = w * kWarpSpan + r * 32 + lane_id();
            uint32_t key = kNone, dest = kNone;
            if (packed[r] != kNone) {
                key = packed[r] >> 9;
                const uint32_t bucket = key & lo_mask;
                dest = run[bucket] + cnt[w * Bp + bucket] + (packed[r] & 511u);
            }
            skey[idx] = key;
            sdest[idx] = dest;
        }
        __syncwarp();
        // one full 32-byte sector per record: lanes 2k and 2k+1 write its two halves in one instruction
        {
            const uint32_t half = lane_id() & 1u;
#pragma unroll 4
            for (int it = 0; it < kWarpSpan / 16; ++it) {
                const uint32_t idx = w * kWarpSpan + it * 16 + (lane_id() >> 1);
                const uint32_t dest = sdest[idx];
                if (dest != kNone) {
                    const uint32_t* p = raw + idx * kRecWords;
                    uint4 v;
                    if (half == 0) v = make_uint4(skey[idx], p[1], p[2], p[3]);
                    else v = make_uint4(p[4], p[5], p[6], td.first_index + idx);
                    aos[2 * (size_t)dest + half] = v;
                }
            }
        }
        __syncwarp();
        zero_row(cnt + w * Bp, Bp);
        __syncthreads();  // the stage, skey and sdest are free again
        if (threadIdx.x == 0 && i + kStagesIdxA < n) {
            TileDesc d = raw_tile(chunks, n_chunks, t0 + i + kStagesIdxA, ccur);
            s_desc[stage] = d;
            ring_issue_stream(raw, &bars[stage], d.ptr, d.count * kRecBytes);
        }
        if (kStagesIdxA == 1) __syncthreads();  // the descriptor just written is read at the top of the next tile
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

struct IdxBSmem {
    uint32_t ring, stage_bytes, cnt, run, misc, sdest, desc, bar, total;
};

__host__ __device__ inline IdxBSmem idx_b_layout(uint32_t B)
{
    IdxBSmem L;
    uint32_t p = 0;
    L.stage_bytes = kTile * 32;
    L.ring = p;  p += 2 * L.stage_bytes;     // two stages: the next tile loads while this one is ranked and written
    L.cnt = p;   p += round_up(kWarps * round_up(B, 8) * 2, 16);
    L.run = p;   p += round_up(B * 4, 16);
    L.misc = p;  p += 64 * 4;
    L.sdest = p; p += kTile * 4;
    L.desc = p;  p += 16;
    L.bar = p;   p += 16;
    L.total = p;
    return L;
}

// INDEX pass B: keyed records (sorted by low digit) -> the index: keyed records sorted by the full key.  Same
// shape as pass A: running slots per bucket in shared memory, one warp assigns slots in input order, one full
// 32-byte sector per record.  With <= 2048 buckets the lines being filled (buckets x CTAs x 128 B) stay in L2
// until they are complete, so DRAM sees whole lines.
__global__ void __launch_bounds__(kThreads, 4) k_scatter_idx_b(const uint4* __restrict__ aos_in,
                                                              const uint32_t* __restrict__ n_ptr, uint32_t B,
                                                              uint32_t lo_bits, const uint32_t* __restrict__ table,
                                                              uint32_t stride, uint4* __restrict__ aos_out)
{
    extern __shared__ __align__(128) uint8_t smem[];
    __shared__ uint32_t s_grp[kWarps][32];  // warp_rank_claim's group words
    s_grp[threadIdx.x >> 5][threadIdx.x & 31] = 0u;
    const IdxBSmem L = idx_b_layout(B);
    uint32_t* ring = reinterpret_cast<uint32_t*>(smem + L.ring);
    uint32_t* run = reinterpret_cast<uint32_t*>(smem + L.run);
    uint32_t* sdest = reinterpret_cast<uint32_t*>(smem + L.sdest);
    uint64_t* bar = reinterpret_cast<uint64_t*>(smem + L.bar);
    uint16_t* cnt = reinterpret_cast<uint16_t*>(smem + L.cnt);
    uint32_t* misc = reinterpret_cast<uint32_t*>(smem + L.misc);
    const uint32_t Bp = round_up(B, 8);
    const uint32_t w = warp_id();
    const uint32_t n_rec = *n_ptr;

    Span sp = {0u, (n_rec + kTile - 1) / kTile, 0u, 1u};
    uint32_t t0, t1;
    segment_of(sp, t0, t1);
    const uint32_t n = t1 - t0;
    auto issue = [&](uint32_t i) {  // thread 0; 32-byte records from a 256-byte aligned array: always bulk-copyable
        TileDesc d = keyed_tile(aos_in, n_rec, t0 + i);
        mbar_expect_tx(&bar[i & 1u], d.count * 32u);
        tma_load_1d_stream(ring + (i & 1u) * (kTile * 8), d.ptr, d.count * 32u, &bar[i & 1u]);
    };
    if (threadIdx.x == 0) {
        mbar_init(&bar[0], 1);
        mbar_init(&bar[1], 1);
        mbar_fence_init();
        if (n > 0) issue(0);
        if (n > 1) issue(1);
    }
    {
        uint32_t* cz = reinterpret_cast<uint32_t*>(cnt);
        for (uint32_t k = threadIdx.x; k < kWarps * Bp / 2; k += kThreads) cz[k] = 0;
    }
    uint32_t grun[8];
#pragma unroll
    for (int k = 0; k < 8; ++k) {
        uint32_t b = threadIdx.x * 8 + k;
        grun[k] = b < B ? table[(size_t)b * stride + blockIdx.x] : 0u;
    }
    __syncthreads();

    for (uint32_t i = 0; i < n; ++i) {
        const uint32_t count = keyed_tile(aos_in, n_rec, t0 + i).count;
        const uint32_t* raw = ring + (i & 1u) * (kTile * 8);
        const uint4* s_rec = reinterpret_cast<const uint4*>(raw);
        mbar_wait(&bar[i & 1u], (i >> 1) & 1u);
        uint32_t packed[kRounds];  // bucket << 9 | rank
#pragma unroll
        for (int r = 0; r < kRounds; ++r) {
            const uint32_t idx = w * kWarpSpan + r * 32 + lane_id();
            packed[r] = idx < count ? (raw[idx * 8] >> lo_bits) : kNone;
        }
        {
            uint32_t rk[kRounds];
            warp_rank_claim<kRounds>(packed, rk, cnt + w * Bp, s_grp[w]);
#pragma unroll
            for (int r = 0; r < kRounds; ++r) packed[r] = packed[r] == kNone ? kNone : ((packed[r] << 9) | rk[r]);
        }
        __syncthreads();
        finish_ranks<false>(cnt, B, Bp, run, nullptr, misc, grun);
#pragma unroll
        for (int r = 0; r < kRounds; ++r) {
            uint32_t dest = kNone;
            if (packed[r] != kNone) {
                const uint32_t bucket = packed[r] >> 9;
                dest = run[bucket] + cnt[w * Bp + bucket] + (packed[r] & 511u);
            }
            sdest[w * kWarpSpan + r * 32 + lane_id()] = dest;
        }
        __syncwarp();
        {
            const uint32_t half = lane_id() & 1u;
#pragma unroll 4
            for (int it = 0; it < kWarpSpan / 16; ++it) {
                const uint32_t idx = w * kWarpSpan + it * 16 + (lane_id() >> 1);
                const uint32_t dest = sdest[idx];
                if (dest != kNone) aos_out[2 * (size_t)dest + half] = s_rec[2 * idx + half];
            }
        }
        __syncwarp();
        zero_row(cnt + w * Bp, Bp);
        __syncthreads();
        if (threadIdx.x == 0 && i + 2 < n) issue(i + 2);
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
