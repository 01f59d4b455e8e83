// psl_index.cuh -- the one-off sort behind the PSL index (paper method 3): two stable LSD
// passes over the full key, split as key = hi * 2^s + lo with hi < 256 and lo < 8192.
//
// What shapes these kernels on B200 is the rate of distinct 128-byte lines the stores touch (about 35 G
// line-writes/s chip-wide), not bytes:
//   pass A (by lo, up to 8192 buckets = the position bins): a tile of 1024 records has about one record per
//     bucket, so no staging can make runs; every record is written once as ONE full 32-byte sector
//     {key, E, x, y, u, v, wt, src} by a pair of lanes (one request per record).  Ranks need no per-warp
//     counter matrix: the CTA keeps the running first free slot of every bucket of its segment in shared
//     memory and one warp walks the tile's keys in input order (__match_any_sync per 32 keys).
//   pass B (by hi, <= 256 buckets = type x energy): the 4096-record-tile staged scatter of psl_bigtile.cuh
//     on keyed input, SoA out -- runs of tens of records per key and tile.
#pragma once

#include "psl_bigtile.cuh"

namespace psl {

constexpr int kIdxMaxLo = 8192;   // most buckets of pass A
constexpr int kIdxMaxHi = 256;    // most buckets of pass B
constexpr int kStagesIdxA = 1;

struct IdxASmem {
    uint32_t ring, stage_bytes, run, skey, sdest, edges, desc, bars, total;
};

__host__ __device__ inline IdxASmem idx_a_layout(uint32_t B, uint32_t n_edges)
{
    IdxASmem L;
    uint32_t p = 0;
    L.stage_bytes = round_up(kTile * kRecBytes, 128);
    L.ring = p;  p += kStagesIdxA * L.stage_bytes;
    L.run = p;   p += round_up(B * 4, 16);   // first free slot of every bucket, running over the segment
    L.skey = p;  p += kTile * 4;             // full key of every record of the tile, kNone = dropped
    L.sdest = p; p += kTile * 4;             // slot of every record
    L.edges = p; p += round_up(n_edges * 4, 16);
    L.desc = p;  p += kStagesIdxA * 16;
    L.bars = p;  p += kStagesIdxA * 8;
    L.total = p;
    return L;
}

template <bool POS, bool EDGES>
__global__ void __launch_bounds__(kThreads, 3) k_scatter_idx_a(const ChunkDesc* __restrict__ chunks, uint32_t n_chunks,
                                                              Span sp, const __grid_constant__ DevGrid g,
                                                              const __grid_constant__ DevBeam bm, uint32_t B,
                                                              uint32_t lo_bits, const uint32_t* __restrict__ table,
                                                              uint32_t stride, uint4* __restrict__ aos)
{
    extern __shared__ __align__(128) uint8_t smem[];
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
    if (threadIdx.x == 0) {
        for (int k = 0; k < kStagesIdxA; ++k) mbar_init(&bars[k], 1);
        mbar_fence_init();
        for (uint32_t k = 0; k < (uint32_t)kStagesIdxA && k < n; ++k) {
            TileDesc d = raw_tile(chunks, n_chunks, t0 + k);
            s_desc[k] = d;
            ring_issue(reinterpret_cast<uint32_t*>(smem + L.ring + k * L.stage_bytes), &bars[k], d.ptr, d.count * kRecBytes);
        }
    }
    for (uint32_t b = threadIdx.x; b < B; b += kThreads) run[b] = table[(size_t)b * stride + col];
    stage_edges(g, s_edges);
    __syncthreads();

    uint32_t phase_bits = 0;
    for (uint32_t i = 0; i < n; ++i) {
        const uint32_t stage = i % kStagesIdxA;
        uint32_t* raw = reinterpret_cast<uint32_t*>(smem + L.ring + stage * L.stage_bytes);
        const TileDesc td = s_desc[stage];
        ring_acquire(raw, &bars[stage], phase_bits, stage, td.ptr, td.count * kRecBytes);

        // keys of the tile (a1-a4); thread t takes records t, t + 256, ...
        {
            Rec rec[kRounds];
#pragma unroll
            for (int r = 0; r < kRounds; ++r) {
                int idx = r * kThreads + threadIdx.x;
                rec[r] = rec_from_smem(raw, idx < (int)td.count ? idx : 0);
            }
#pragma unroll
            for (int r = 0; r < kRounds; ++r) {
                int idx = r * kThreads + threadIdx.x;
                uint32_t key;
                int cls = classify<POS, EDGES, 0>(g, bm, rec[r], s_edges, key);
                skey[idx] = (idx < (int)td.count && cls == C_SURVIVOR) ? key : kNone;
            }
        }
        __syncthreads();
        // slots, in input order: one warp walks the tile 32 keys at a time
        if (w == 0) {
#pragma unroll 4
            for (int r = 0; r < kTile / 32; ++r) {
                const uint32_t key = skey[r * 32 + lane_id()];
                const uint32_t bucket = key == kNone ? kNone : (key & lo_mask);
                const uint32_t peers = __match_any_sync(0xFFFFFFFFu, bucket);
                const int leader = __ffs(peers) - 1;
                uint32_t base = 0;
                if ((int)lane_id() == leader && bucket != kNone) {
                    base = run[bucket];
                    run[bucket] = base + __popc(peers);
                }
                base = __shfl_sync(0xFFFFFFFFu, base, leader);
                sdest[r * 32 + lane_id()] = bucket == kNone ? kNone : base + __popc(peers & lanemask_lt());
            }
        }
        __syncthreads();
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
        __syncthreads();  // the stage, skey and sdest are free again
        if (threadIdx.x == 0 && i + kStagesIdxA < n) {
            TileDesc d = raw_tile(chunks, n_chunks, t0 + i + kStagesIdxA);
            s_desc[stage] = d;
            ring_issue(raw, &bars[stage], d.ptr, d.count * kRecBytes);
        }
    }
}

// INDEX pass B count: histogram of the high digits (key >> lo_bits) over the CTA's segment of the keyed
// records.  Reads the key word of every 32-byte record.
__global__ void __launch_bounds__(kThreads) k_count_keys(const uint4* __restrict__ aos, const uint32_t* __restrict__ n_ptr,
                                                        uint32_t B, uint32_t lo_bits, uint32_t* __restrict__ table,
                                                        uint32_t stride)
{
    extern __shared__ __align__(128) uint8_t smem[];
    uint32_t* hist = reinterpret_cast<uint32_t*>(smem);
    const CountSmem L = count_layout(0, 0, B, 0);
    const uint32_t rmask = (1u << L.rlog) - 1u;
    const uint32_t n = *n_ptr;
    Span sp = {0u, (n + kTile - 1) / kTile, 0u, 1u};
    uint32_t t0, t1;
    segment_of(sp, t0, t1);
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

constexpr int kIdxBStages = 5;  // 4 being worked on + 1 in flight (32 KB each)

struct IdxBSmem {
    uint32_t ring, stage_bytes, cnt, gcur, lstart, pdest, perm, misc, desc, bars, total;
};

__host__ __device__ inline IdxBSmem idx_b_layout(uint32_t B)
{
    IdxBSmem L;
    uint32_t p = 0;
    L.stage_bytes = kTile * 32;
    L.ring = p;   p += kIdxBStages * L.stage_bytes;
    L.cnt = p;    p += round_up(kBigWarps * round_up(B, 8) * 2, 16);
    L.gcur = p;   p += round_up(B * 4, 16);
    L.lstart = p; p += round_up(B * 4, 16);
    L.pdest = p;  p += kBigTile * 4;
    L.perm = p;   p += kBigTile * 2;
    L.misc = p;   p += 64 * 4;
    L.desc = p;   p += kIdxBStages * 16;
    L.bars = p;   p += kIdxBStages * 8;
    L.total = p;
    return L;
}

// INDEX pass B scatter: keyed records (sorted by low digit) -> SoA index sorted by the full key, plus the
// full key of every slot (used once, by binary search, to build offsets[K+1]).  4096-record tiles.
__global__ void __launch_bounds__(kBigThreads, 1) k_scatter_idx_b(const uint4* __restrict__ aos,
                                                                 const uint32_t* __restrict__ n_ptr, uint32_t B,
                                                                 uint32_t lo_bits, const uint32_t* __restrict__ table,
                                                                 uint32_t stride, IdxOut out)
{
    extern __shared__ __align__(128) uint8_t smem[];
    const uint32_t Bp = round_up(B, 8);
    const IdxBSmem L = idx_b_layout(B);
    uint16_t* cnt = reinterpret_cast<uint16_t*>(smem + L.cnt);
    uint32_t* gcur = reinterpret_cast<uint32_t*>(smem + L.gcur);
    uint32_t* lstart = reinterpret_cast<uint32_t*>(smem + L.lstart);
    uint32_t* pdest = reinterpret_cast<uint32_t*>(smem + L.pdest);
    uint16_t* perm = reinterpret_cast<uint16_t*>(smem + L.perm);
    uint32_t* misc = reinterpret_cast<uint32_t*>(smem + L.misc);
    TileDesc* s_desc = reinterpret_cast<TileDesc*>(smem + L.desc);
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem + L.bars);
    const uint32_t w = warp_id();
    const uint32_t n_rec = *n_ptr;

    Span sp = {0u, (n_rec + kTile - 1) / kTile, 0u, 1u};
    uint32_t t0, t1;
    segment_of(sp, t0, t1);
    const uint32_t n = t1 - t0;

    auto stage_ptr = [&](uint32_t i) { return reinterpret_cast<uint32_t*>(smem + L.ring + (i % kIdxBStages) * L.stage_bytes); };
    auto issue = [&](uint32_t i) {  // thread 0; 32-byte records from a 256-byte aligned array: always bulk-copyable
        TileDesc d = keyed_tile(aos, n_rec, t0 + i);
        s_desc[i % kIdxBStages] = d;
        mbar_expect_tx(&bars[i % kIdxBStages], d.count * 32u);
        tma_load_1d(stage_ptr(i), d.ptr, d.count * 32u, &bars[i % kIdxBStages]);
    };
    if (threadIdx.x == 0) {
        for (int k = 0; k < kIdxBStages; ++k) mbar_init(&bars[k], 1);
        mbar_fence_init();
        for (uint32_t k = 0; k < (uint32_t)kIdxBStages && k < n; ++k) issue(k);
    }
    {
        uint32_t* cz = reinterpret_cast<uint32_t*>(cnt);
        for (uint32_t i = threadIdx.x; i < kBigWarps * Bp / 2; i += kBigThreads) cz[i] = 0;
    }
    uint32_t grun[8];
#pragma unroll
    for (int k = 0; k < 8; ++k) {
        uint32_t b = threadIdx.x * 8 + k;
        grun[k] = b < B ? table[(size_t)b * stride + blockIdx.x] : 0u;
    }
    __syncthreads();

    for (uint32_t base = 0; base < n; base += kBigQ) {
        const uint32_t nq = min((uint32_t)kBigQ, n - base);
        uint32_t packed[kBigRounds];
#pragma unroll
        for (int r = 0; r < kBigRounds; ++r) packed[r] = kNone;
        const uint32_t q = w / (kBigWarps / kBigQ);
        if (q < nq) {
            const uint32_t i = base + q;
            const TileDesc td = s_desc[i % kIdxBStages];
            mbar_wait(&bars[i % kIdxBStages], (i / kIdxBStages) & 1u);
            const uint32_t* raw = stage_ptr(i);
            const uint32_t first = (w % (kBigWarps / kBigQ)) * kBigSpan;
#pragma unroll
            for (int r = 0; r < kBigRounds; ++r) {
                const uint32_t idx = first + r * 32 + lane_id();
                packed[r] = idx < td.count ? (raw[idx * 8] >> lo_bits) : kNone;
            }
#pragma unroll
            for (int r = 0; r < kBigRounds; ++r) {
                uint32_t bucket = packed[r];
                uint32_t rank = warp_rank(bucket, cnt + w * Bp);
                packed[r] = bucket == kNone ? kNone : ((bucket << 9) | rank);
            }
        }
        __syncthreads();
        const uint32_t n_part = finish_ranks<true, kBigWarps>(cnt, B, Bp, gcur, lstart, misc, grun);

#pragma unroll
        for (int r = 0; r < kBigRounds; ++r) {
            if (packed[r] != kNone) {
                uint32_t bucket = packed[r] >> 9, rank = packed[r] & 511u;
                uint32_t rel = cnt[w * Bp + bucket] + rank;
                uint32_t p = lstart[bucket] + rel;
                perm[p] = (uint16_t)(w * kBigSpan + r * 32 + lane_id());
                pdest[p] = gcur[bucket] + rel;
            }
        }
        __syncwarp();
        zero_row(cnt + w * Bp, Bp);
        __syncthreads();

        for (uint32_t j = threadIdx.x; j < n_part; j += kBigThreads) {
            const uint32_t irec = perm[j];
            const uint32_t dest = pdest[j];
            const uint4* s_rec = reinterpret_cast<const uint4*>(stage_ptr(base + irec / kTile)) + 2 * (irec % kTile);
            const uint4 a = s_rec[0], b = s_rec[1];
            out.key[dest] = a.x;
            out.E[dest] = __uint_as_float(a.y);
            out.x[dest] = __uint_as_float(a.z);
            out.y[dest] = __uint_as_float(a.w);
            out.u[dest] = __uint_as_float(b.x);
            out.v[dest] = __uint_as_float(b.y);
            out.wt[dest] = __uint_as_float(b.z);
            out.src[dest] = b.w;
        }
        __syncthreads();
        if (threadIdx.x == 0)
            for (uint32_t k = 0; k < nq; ++k)
                if (base + kIdxBStages + k < n) issue(base + kIdxBStages + k);
        __syncthreads();  // the next tile reads descriptors just written
    }
}

}  // namespace psl
