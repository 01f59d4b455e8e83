// psl_index_big.cuh -- INDEX passes A and B (paper method 3): two stable LSD passes over the full
// key, split into two balanced digits key = hi * 2^s + lo (each <= 2048 buckets), with tile-sorted staging.
//
//   pass A: raw 28-byte records -> 32-byte keyed records {key, E, x, y, u, v, wt, src}, stably partitioned by lo
//   pass B: keyed records -> the index: keyed records sorted by the full key (stable partition by hi)
//
// A tile is two ring stages of 1024 records that stay where TMA put them.  Warp w owns records [256 w, 256 w + 256) of
// the tile (a quarter of a stage): per-warp private uint16 counters + claimed peer masks (warp_rank_claim) give stable
// ranks, finish_ranks the prefix over the 8 warps; the records are then ordered by (bucket, input order) inside the
// tile, and every record leaves as ONE 32-byte store request, so that a run of records of one bucket is one request
// per 128-byte line.
#pragma once

#include "psl_index.cuh"

namespace psl {

// Two 256-thread CTAs per SM, each on 2048-record tiles (two ring stages, no prefetch stage: while one CTA waits for its
// next tile the other one ranks or writes).  Measured at config 4 / 5 against one 512-thread CTA per SM on 4096-record
// tiles with 1-2 stages of prefetch: pass A 3.29 -> 3.07 ms / 16.4 -> 15.3 ms, pass B 3.06 -> 2.77 / 15.2 -> 13.7 ms:
// the phases of a tile use different units (ranks: counters and the claim words; write-out: the LSU), and a second,
// independent CTA fills the slots the barriers leave empty.  Runs per bucket halve (2 records), which costs less.
constexpr int kIdxBigQ = 2;                               // ring stages per tile
constexpr int kIdxBigTile = kIdxBigQ * kTile;             // 2048 records
constexpr int kIdxBigStagesRaw = 2;    // pass A (28 KB each)
constexpr int kIdxBigStagesKeyed = 2;  // pass B (32 KB each)
constexpr int kIdxBigThreads = 128 * kIdxBigQ;            // 256
constexpr int kIdxBigWarps = kIdxBigThreads / 32;         // 8
constexpr int kIdxBigSpan = kIdxBigTile / kIdxBigWarps;   // 256 records per warp
constexpr int kIdxBigRounds = kIdxBigSpan / 32;           // 8

struct IdxBigSmem {
    uint32_t ring, stage_bytes, cnt, gcur, lstart, perm, pbkt, edges, misc, grp, desc, bars, total;
};

__host__ __device__ inline IdxBigSmem idx_big_layout(bool keyed, uint32_t B, uint32_t n_edges)
{
    IdxBigSmem L;
    uint32_t p = 0;
    L.stage_bytes = round_up(kTile * (keyed ? 32 : kRecBytes), 128);
    const uint32_t stages = keyed ? kIdxBigStagesKeyed : kIdxBigStagesRaw;
    L.ring = p;   p += stages * L.stage_bytes;
    L.cnt = p;    p += round_up(kIdxBigWarps * round_up(B, 8) * 2, 16);
    L.gcur = p;   p += round_up(B, 8) * 4;                // Bp entries
    L.lstart = p; p += round_up(B, 8) * 4;
    L.perm = p;   p += kIdxBigTile * 4;                   // tile-sorted slot -> bucket << 12 | record in tile
    L.pbkt = p;
    L.edges = p;  p += round_up(n_edges * 4, 16);
    L.misc = p;   p += 64 * 4;
    L.grp = p;    p += kIdxBigWarps * 32 * 4;
    L.desc = p;   p += stages * 16;
    L.bars = p;   p += stages * 8;
    L.total = p;
    return L;
}

// one per-chunk histogram launch of pass A: its span and how many segments (scatter CTAs) it was cut into
struct SpanSeg {
    Span sp;
    uint32_t n_seg;
};

// Pass A (KEYED = false) walks ALL chunk launches in one kernel: CTA s takes segment s of every span that has one,
// with the running slots re-read from that span's table columns.  Pass B (KEYED = true) has one span, computed
// from *n_ptr.
template <bool KEYED, bool POS, bool EDGES>
__global__ void __launch_bounds__(kIdxBigThreads, 2) k_scatter_idx_big(const ChunkDesc* __restrict__ chunks, uint32_t n_chunks,
                                                                const SpanSeg* __restrict__ spans, uint32_t n_spans, Span sp,
                                                                const uint4* __restrict__ aos_in,
                                                                const uint32_t* __restrict__ n_ptr,
                                                                const __grid_constant__ DevGrid g,
                                                                const __grid_constant__ DevBeam bm, uint32_t B,
                                                                uint32_t lo_bits, const uint32_t* __restrict__ table,
                                                                uint32_t stride, uint4* __restrict__ aos_out)
{
    extern __shared__ __align__(128) uint8_t smem[];
    constexpr uint32_t kRecB = KEYED ? 32u : (uint32_t)kRecBytes;
    constexpr uint32_t kIdxBigStages = KEYED ? kIdxBigStagesKeyed : kIdxBigStagesRaw;
    const uint32_t Bp = round_up(B, 8);
    const IdxBigSmem L = idx_big_layout(KEYED, B, g.n_ebins + 1);
    uint16_t* cnt = reinterpret_cast<uint16_t*>(smem + L.cnt);
    uint32_t* gcur = reinterpret_cast<uint32_t*>(smem + L.gcur);
    uint32_t* lstart = reinterpret_cast<uint32_t*>(smem + L.lstart);
    uint32_t* slot = reinterpret_cast<uint32_t*>(smem + L.perm);  // tile-sorted slot -> bucket << 12 | record in tile
    float* s_edges = reinterpret_cast<float*>(smem + L.edges);
    uint32_t* misc = reinterpret_cast<uint32_t*>(smem + L.misc);
    uint32_t* grp = reinterpret_cast<uint32_t*>(smem + L.grp);  // warp_rank_claim's group words, 32 per warp
    TileDesc* s_desc = reinterpret_cast<TileDesc*>(smem + L.desc);
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem + L.bars);
    const uint32_t w = warp_id();
    grp[threadIdx.x] = 0u;
    const uint32_t lo_mask = (1u << lo_bits) - 1u;
    const uint32_t n_rec = KEYED ? *n_ptr : 0u;
    uint32_t goff = 0;  // ring stages this CTA has consumed in earlier spans (stage and parity bookkeeping runs on)
    uint32_t t0 = 0, n = 0;
    auto stage_ptr = [&](uint32_t i) { return reinterpret_cast<uint32_t*>(smem + L.ring + ((goff + i) % kIdxBigStages) * L.stage_bytes); };
    ChunkDesc ccur = {nullptr, 0u, 0u, 0u, 0u};  // thread 0: the chunk of the tile it described last
    auto issue = [&](uint32_t i) {  // thread 0
        TileDesc d = KEYED ? keyed_tile(aos_in, n_rec, t0 + i) : raw_tile(chunks, n_chunks, t0 + i, ccur);
        s_desc[(goff + i) % kIdxBigStages] = d;
        ring_issue_stream(stage_ptr(i), &bars[(goff + i) % kIdxBigStages], d.ptr, d.count * kRecB);
    };
    if (threadIdx.x == 0) {
        for (int k = 0; k < kIdxBigStages; ++k) mbar_init(&bars[k], 1);
        mbar_fence_init();
    }
    {
        uint32_t* cz = reinterpret_cast<uint32_t*>(cnt);
        for (uint32_t i = threadIdx.x; i < kIdxBigWarps * Bp / 2; i += kIdxBigThreads) cz[i] = 0;
    }
    if (!KEYED) stage_edges(g, s_edges);
    __syncthreads();

    const uint32_t n_iter = KEYED ? 1u : n_spans;
    uint32_t* const ring = reinterpret_cast<uint32_t*>(smem + L.ring);
    const uint32_t stage_words = L.stage_bytes / 4;
    for (uint32_t si = 0; si < n_iter; ++si) {
    uint32_t S = gridDim.x;
    if (KEYED) {
        sp.tile_begin = 0;
        sp.n_tiles = (n_rec + kTile - 1) / kTile;
        sp.col0 = 0;
    } else {
        sp = spans[si].sp;
        S = spans[si].n_seg;
        if (blockIdx.x >= S) continue;  // this span was cut into fewer segments than there are CTAs
    }
    const uint32_t col = sp.col0 + blockIdx.x * sp.split;
    {
        const unsigned long long nt = sp.n_tiles, s_ = blockIdx.x;
        t0 = sp.tile_begin + (uint32_t)(nt * s_ / S);
        n = sp.tile_begin + (uint32_t)(nt * (s_ + 1) / S) - t0;  // ring stages (1024-record tiles) in this segment
    }
    if (threadIdx.x == 0)
        for (uint32_t k = 0; k < (uint32_t)kIdxBigStages && k < n; ++k) issue(k);
    uint32_t grun[8];  // thread t keeps the running first free slot of buckets 8t..8t+7
#pragma unroll
    for (int k = 0; k < 8; ++k) {
        uint32_t b = threadIdx.x * 8 + k;
        grun[k] = b < B ? table[(size_t)b * stride + col] : 0u;
    }
    __syncthreads();

    for (uint32_t base = 0; base < n; base += kIdxBigQ) {
        const uint32_t nq = min((uint32_t)kIdxBigQ, n - base);
        // the tile's four ring stages: word offset into the ring and load-order index of the first record
        const uint32_t s0 = (goff + base) % kIdxBigStages;
        const uint32_t s1 = s0 + 1 < kIdxBigStages ? s0 + 1 : s0 + 1 - kIdxBigStages;
        const uint32_t s2 = s0 + 2 < kIdxBigStages ? s0 + 2 : s0 + 2 - kIdxBigStages;
        const uint32_t s3 = s0 + 3 < kIdxBigStages ? s0 + 3 : s0 + 3 - kIdxBigStages;
        const uint32_t o0 = s0 * stage_words, o1 = s1 * stage_words, o2 = s2 * stage_words, o3 = s3 * stage_words;
        uint32_t f0 = 0, f1 = 0, f2 = 0, f3 = 0;
        if (!KEYED) {
            f0 = s_desc[s0].first_index;
            if (nq > 1) f1 = s_desc[s1].first_index;
            if (nq > 2) f2 = s_desc[s2].first_index;
            if (nq > 3) f3 = s_desc[s3].first_index;
        }
        // stages TMA could not fill (unaligned source, ragged last tile): fetched by all threads, then the
        // stage's barrier is completed by hand so that every stage flips its phase once per use
        bool manual = false;
        for (uint32_t q = 0; q < nq; ++q) {
            const uint32_t sq = q == 0 ? s0 : (q == 1 ? s1 : (q == 2 ? s2 : s3));
            const TileDesc d = s_desc[sq];
            if (!bulk_ok(d.ptr, d.count * kRecB)) {
                const uint32_t* src = reinterpret_cast<const uint32_t*>(d.ptr);
                uint32_t* dst = ring + sq * stage_words;
                for (uint32_t k = threadIdx.x; k < d.count * (kRecB / 4); k += kIdxBigThreads) dst[k] = __ldg(src + k);
                manual = true;
            }
        }
        if (manual) {
            __syncthreads();
            if (threadIdx.x == 0)
                for (uint32_t q = 0; q < nq; ++q) {
                    const uint32_t sq = q == 0 ? s0 : (q == 1 ? s1 : (q == 2 ? s2 : s3));
                    const TileDesc d = s_desc[sq];
                    if (!bulk_ok(d.ptr, d.count * kRecB)) mbar_arrive(&bars[sq]);
                }
        }

        // buckets and stable ranks inside the warp's 256 records (a quarter of ring stage base + w / 4)
        uint32_t bkt[kIdxBigRounds], rnk[kIdxBigRounds];
#pragma unroll
        for (int r = 0; r < kIdxBigRounds; ++r) bkt[r] = kNone;
        const uint32_t q = w / (kIdxBigWarps / kIdxBigQ);
        if (q < nq) {
            const uint32_t sq = q == 0 ? s0 : (q == 1 ? s1 : (q == 2 ? s2 : s3));
            const uint32_t count = s_desc[sq].count;
            mbar_wait(&bars[sq], ((goff + base + q) / kIdxBigStages) & 1u);
            uint32_t* raw = ring + sq * stage_words;
            const uint32_t first = (w % (kIdxBigWarps / kIdxBigQ)) * kIdxBigSpan;
            if (KEYED) {
#pragma unroll
                for (int r = 0; r < kIdxBigRounds; ++r) {
                    const uint32_t idx = first + r * 32 + lane_id();
                    bkt[r] = idx < count ? (raw[idx * 8] >> lo_bits) : kNone;
                }
            } else {
#pragma unroll
                for (int h = 0; h < kIdxBigRounds; h += 4) {
                    Rec rec[4];
#pragma unroll
                    for (int r = 0; r < 4; ++r) {
                        const uint32_t idx = first + (h + r) * 32 + lane_id();
                        rec[r] = rec_from_smem(raw, idx < count ? (int)idx : 0);
                        if (g.apr) {  // the redistributed position and direction are what the index stores
                            apr_apply(g.apr_seed, s_desc[sq].first_index + idx, rec[r]);
                            if (idx < count) {
                                uint32_t* p = raw + idx * kRecWords;
                                p[2] = __float_as_uint(rec[r].x); p[3] = __float_as_uint(rec[r].y);
                                p[4] = __float_as_uint(rec[r].u); p[5] = __float_as_uint(rec[r].v);
                            }
                        }
                    }
#pragma unroll
                    for (int r = 0; r < 4; ++r) {
                        const uint32_t idx = first + (h + r) * 32 + lane_id();
                        uint32_t key;
                        const int cls = classify<POS, EDGES, 0>(g, bm, rec[r], s_edges, key);
                        const bool keep = idx < count && cls == C_SURVIVOR;
                        // the key takes the place of the type word of the staged record (the type is part of the key)
                        if (idx < count) raw[idx * kRecWords] = keep ? key : kNone;
                        bkt[h + r] = keep ? (key & lo_mask) : kNone;
                    }
                }
            }
        }
        warp_rank_claim<kIdxBigRounds>(bkt, rnk, cnt + w * Bp, grp + w * 32);
        __syncthreads();
        const uint32_t n_part = finish_ranks<true, kIdxBigWarps>(cnt, B, Bp, gcur, lstart, misc, grun);

        // tile-sorted order
#pragma unroll
        for (int r = 0; r < kIdxBigRounds; ++r) {
            if (bkt[r] != kNone) {
                const uint32_t p = lstart[bkt[r]] + cnt[w * Bp + bkt[r]] + rnk[r];
                slot[p] = (bkt[r] << 12) | (w * kIdxBigSpan + r * 32 + lane_id());  // bucket | record in tile
            }
        }
        __syncwarp();
        zero_row(cnt + w * Bp, Bp);
        __syncthreads();
        // write-out: thread j takes tile-sorted slots j, j + 512, ...: one 32-byte store request per record, so a run
        // of records of one bucket leaves as one request per 128-byte line
#pragma unroll 2
        for (uint32_t j = threadIdx.x; j < n_part; j += kIdxBigThreads) {
            const uint32_t sv = slot[j];
            const uint32_t bucket = sv >> 12, irec = sv & 4095u;
            const uint32_t dest = gcur[bucket] + (j - lstart[bucket]);
            const uint32_t qq = irec / kTile, ir = irec % kTile;
            const uint32_t off = qq == 0 ? o0 : (qq == 1 ? o1 : (qq == 2 ? o2 : o3));
            uint4 a, b;
            if (KEYED) {
                const uint4* p = reinterpret_cast<const uint4*>(ring + off) + 2 * ir;
                a = p[0];
                b = p[1];
            } else {
                const uint32_t* p = ring + off + ir * kRecWords;
                const uint32_t fi = qq == 0 ? f0 : (qq == 1 ? f1 : (qq == 2 ? f2 : f3));
                a = make_uint4(p[0], p[1], p[2], p[3]);
                b = make_uint4(p[4], p[5], p[6], fi + ir);
            }
            stg_record(aos_out + 2 * (size_t)dest, a, b);
        }
        __syncthreads();  // the tile's stages and the slot list are free again
        if (threadIdx.x == 0)
            for (uint32_t k = 0; k < nq; ++k)
                if (base + kIdxBigStages + k < n) issue(base + kIdxBigStages + k);
        __syncthreads();  // the next tile reads descriptors just written
    }
    goff += n;
    }  // spans
}

}  // namespace psl
