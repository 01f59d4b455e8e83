// psl_bigtile.cuh -- ONTHEFLY scatter with 4096-record tiles (keys <= 256), one 512-thread CTA per SM.
//
// Why a second scatter kernel: the SoA output is written as runs (one per populated key per tile per array),
// and on B200 what bounds this kernel is not bytes but the number of distinct 128-byte lines the stores
// touch -- about 35 G line-writes/s over the whole chip (measured).  Runs shorter than a
// line waste that budget, and their length is (records per tile) x (share of the key).  A tile four times
// longer makes the runs four times longer for the same number of line-writes per run.
//
// Layout: the ring has kBigStages stages of kTile records; a big tile is kBigQ consecutive ring stages of the
// CTA's segment, so the records stay where TMA put them and the remaining stages prefetch the next tile.
// Warp w owns records [w*256, (w+1)*256) of the big tile (inside one stage), so stable ranks are again
// per-warp counters + a scan over the 16 warps.
#pragma once

#include "psl_partition.cuh"

namespace psl {

constexpr int kBigThreads = 512;
constexpr int kBigWarps = kBigThreads / 32;          // 16
constexpr int kBigQ = 4;                             // ring stages per big tile
constexpr int kBigTile = kBigQ * kTile;              // 4096 records
constexpr int kBigStages = 6;                        // 4 being worked on + 2 in flight
constexpr int kBigSpan = kBigTile / kBigWarps;       // 256 consecutive records per warp
constexpr int kBigRounds = kBigSpan / 32;            // 8
constexpr int kBigMaxKeys = 256;

struct BigSmem {
    uint32_t ring, stage_bytes, cnt, gcur, lstart, pdest, perm, edges, misc, desc, bars, total;
};

__host__ __device__ inline BigSmem big_layout(uint32_t B, uint32_t n_edges)
{
    BigSmem L;
    uint32_t p = 0;
    L.stage_bytes = round_up(kTile * kRecBytes, 128);
    L.ring = p;   p += kBigStages * L.stage_bytes;
    L.cnt = p;    p += round_up(kBigWarps * round_up(B, 8) * 2, 16);
    L.gcur = p;   p += round_up(B * 4, 16);
    L.lstart = p; p += round_up(B * 4, 16);
    L.pdest = p;  p += kBigTile * 4;
    L.perm = p;   p += kBigTile * 2;
    L.edges = p;  p += round_up(n_edges * 4, 16);
    L.misc = p;   p += 64 * 4;
    L.desc = p;   p += kBigStages * 16;
    L.bars = p;   p += kBigStages * 8;
    L.total = p;
    return L;
}

__device__ __forceinline__ void mbar_arrive(uint64_t* bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}

template <bool POS, bool EDGES, int BEAM, bool PROJ>
__global__ void __launch_bounds__(kBigThreads, 1) k_scatter_otf_big(const ChunkDesc* __restrict__ chunks, uint32_t n_chunks,
                                                                   Span sp, const __grid_constant__ DevGrid g,
                                                                   const __grid_constant__ DevBeam bm, uint32_t B,
                                                                   const uint32_t* __restrict__ table, uint32_t stride,
                                                                   SoAOut out, SegStats* sstats, const FusedScan fs,
                                                                   const StatsTail st)
{
    extern __shared__ __align__(128) uint8_t smem[];
    const uint32_t Bp = round_up(B, 8);
    const BigSmem L = big_layout(B, g.n_ebins + 1);
    uint16_t* cnt = reinterpret_cast<uint16_t*>(smem + L.cnt);
    uint32_t* gcur = reinterpret_cast<uint32_t*>(smem + L.gcur);
    uint32_t* lstart = reinterpret_cast<uint32_t*>(smem + L.lstart);
    uint32_t* pdest = reinterpret_cast<uint32_t*>(smem + L.pdest);
    uint16_t* perm = reinterpret_cast<uint16_t*>(smem + L.perm);
    float* s_edges = reinterpret_cast<float*>(smem + L.edges);
    uint32_t* misc = reinterpret_cast<uint32_t*>(smem + L.misc);
    TileDesc* s_desc = reinterpret_cast<TileDesc*>(smem + L.desc);
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem + L.bars);
    const uint32_t w = warp_id();
    const uint32_t col = sp.col0 + blockIdx.x * sp.split;

    uint32_t t0, t1;
    segment_of(sp, t0, t1);
    const uint32_t n = t1 - t0;  // ring stages (tiles of kTile records) in this segment

    auto stage_ptr = [&](uint32_t i) { return reinterpret_cast<uint32_t*>(smem + L.ring + (i % kBigStages) * L.stage_bytes); };
    ChunkDesc ccur = {nullptr, 0u, 0u, 0u, 0u};  // thread 0: the chunk of the tile it described last
    auto issue = [&](uint32_t i) {  // thread 0
        TileDesc d = raw_tile(chunks, n_chunks, t0 + i, ccur);
        s_desc[i % kBigStages] = d;
        ring_issue(stage_ptr(i), &bars[i % kBigStages], d.ptr, d.count * kRecBytes);
    };
    if (threadIdx.x == 0) {
        for (int k = 0; k < kBigStages; ++k) mbar_init(&bars[k], 1);
        mbar_fence_init();
        for (uint32_t k = 0; k < (uint32_t)kBigStages && k < n; ++k) issue(k);
    }
    {
        uint32_t* cz = reinterpret_cast<uint32_t*>(cnt);
        for (uint32_t i = threadIdx.x; i < kBigWarps * Bp / 2; i += kBigThreads) cz[i] = 0;
    }
    uint32_t grun[8];
    griddep_wait();  // the histogram kernel's table and statistics from here on
    if (fs.n_cols != 0) {
        fused_first_slots<kBigWarps>(fs, table, stride, B, col, gcur, lstart, misc, grun);
    } else {
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            uint32_t b = threadIdx.x * 8 + k;
            grun[k] = b < B ? table[(size_t)b * stride + col] : 0u;
        }
    }
    stage_edges(g, s_edges);
    __syncthreads();

    double sum_out = 0.0;
    for (uint32_t base = 0; base < n; base += kBigQ) {
        const uint32_t nq = min((uint32_t)kBigQ, n - base);
        // stages TMA could not fill (unaligned source, ragged last tile): fetched by all threads, then the
        // stage's barrier is completed by hand so that every stage flips its phase once per use
        bool manual = false;
        for (uint32_t q = 0; q < nq; ++q) {
            const TileDesc d = s_desc[(base + q) % kBigStages];
            if (!bulk_ok(d.ptr, d.count * kRecBytes)) {
                const uint32_t* src = reinterpret_cast<const uint32_t*>(d.ptr);
                uint32_t* dst = stage_ptr(base + q);
                for (uint32_t k = threadIdx.x; k < d.count * kRecWords; k += kBigThreads) dst[k] = __ldg(src + k);
                manual = true;
            }
        }
        if (manual) {
            __syncthreads();
            if (threadIdx.x == 0)
                for (uint32_t q = 0; q < nq; ++q) {
                    const TileDesc d = s_desc[(base + q) % kBigStages];
                    if (!bulk_ok(d.ptr, d.count * kRecBytes)) mbar_arrive(&bars[(base + q) % kBigStages]);
                }
        }

        // bucket and stable rank inside the warp's 256 records (all inside ring stage base + w / 4)
        uint32_t packed[kBigRounds];
#pragma unroll
        for (int r = 0; r < kBigRounds; ++r) packed[r] = kNone;
        const uint32_t q = w / (kBigWarps / kBigQ);
        if (q < nq) {
            const uint32_t i = base + q;
            const TileDesc td = s_desc[i % kBigStages];
            mbar_wait(&bars[i % kBigStages], (i / kBigStages) & 1u);
            const uint32_t* raw = stage_ptr(i);
            const int first = (int)(w % (kBigWarps / kBigQ)) * kBigSpan;
#pragma unroll
            for (int h = 0; h < kBigRounds; h += 4) {
                Rec rec[4];
#pragma unroll
                for (int r = 0; r < 4; ++r) {
                    int idx = first + (h + r) * 32 + (int)lane_id();
                    rec[r] = rec_from_smem(raw, idx < (int)td.count ? idx : 0);
                }
#pragma unroll
                for (int r = 0; r < 4; ++r) {
                    int idx = first + (h + r) * 32 + (int)lane_id();
                    uint32_t key;
                    int cls = classify<POS, EDGES, BEAM>(g, bm, rec[r], s_edges, key);
                    packed[h + r] = (idx < (int)td.count && cls == C_SURVIVOR) ? key : kNone;
                }
            }
        }
        {
            uint32_t rk[kBigRounds];
            warp_rank_match<kBigRounds>(packed, rk, cnt + w * Bp);
#pragma unroll
            for (int r = 0; r < kBigRounds; ++r) packed[r] = packed[r] == kNone ? kNone : ((packed[r] << 9) | rk[r]);
        }
        __syncthreads();
        const uint32_t n_part = finish_ranks<true, kBigWarps>(cnt, B, Bp, gcur, lstart, misc, grun);

        // tile-sorted order
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

        // write-out: thread j takes tile-sorted slots j, j + 512, ...
        for (uint32_t j = threadIdx.x; j < n_part; j += kBigThreads) {
            const uint32_t irec = perm[j];
            const uint32_t dest = pdest[j];
            const uint32_t i = base + (irec / kTile);
            Rec rec = rec_from_smem(stage_ptr(i), (int)(irec % kTile));
            float qq = q_of(rec.u, rec.v), wz, xm = 0.0f, ym = 0.0f, wt;
            if (PROJ) {
                float tx, ty;
                slopes(rec.u, rec.v, qq, wz, tx, ty);
                xm = __fadd_rn(rec.x, __fmul_rn(tx, bm.dzM));
                ym = __fadd_rn(rec.y, __fmul_rn(ty, bm.dzM));
                wt = final_weight(bm, rec.wt, xm, ym);
            } else {
                wz = __fsqrt_rn(qq);
                wt = bm.has_beam ? __fmul_rn(rec.wt, bm.mu) : rec.wt;
            }
            out.E[dest] = rec.E;
            out.x[dest] = rec.x;
            out.y[dest] = rec.y;
            out.u[dest] = rec.u;
            out.v[dest] = rec.v;
            out.w[dest] = wz;
            out.wt[dest] = wt;
            out.src[dest] = s_desc[i % kBigStages].first_index + (irec % kTile);
            if (PROJ && bm.out_proj) {
                out.xp[dest] = xm;
                out.yp[dest] = ym;
            }
            sum_out += (double)wt;
        }
        __syncthreads();  // the tile's stages and perm/pdest are free again
        if (threadIdx.x == 0)
            for (uint32_t k = 0; k < nq; ++k)
                if (base + kBigStages + k < n) issue(base + kBigStages + k);
        __syncthreads();  // the next tile reads two of the descriptors just written
    }
    sum_out = warp_sum_double(sum_out);
    __shared__ double s_d[kBigWarps];
    if (lane_id() == 0) s_d[w] = sum_out;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0.0;
        for (int k = 0; k < kBigWarps; ++k) t += s_d[k];
        sstats[col].sum_out = t;
    }
    stats_tail(st, sstats);
}

}  // namespace psl
