// psl_compact.cuh -- ONTHEFLY scatter for a beam that rejects (jaws, zero-weight policy), keys <= 256.
//
// The histogram kernel of such a beam (k_count_raw with `comp`) has already classified every record; it leaves
// the survivors, in load order, as 32-byte records {key, E, x, y, u, v, wt, src_index} in its segment's own
// region of the workspace.  This kernel therefore never reads the rejected records (86 % of config 3) nor
// repeats the jaw arithmetic: it reads 32 B per SURVIVOR instead of 28 B per RECORD, ranks by the stored key
// and writes the SoA batches -- the 4096-record-tile machinery of psl_bigtile.cuh over a different source,
// where a tile now holds 4096 survivors, so the runs per key are as long as without a beam.
//
// Source of CTA s: the regions of the sp.split histogram CTAs that shared its segment, in order; region h
// starts at record (first tile of the sub-segment) * kTile of `comp` and holds sstats[col + h].n_surv records.
#pragma once

#include "psl_bigtile.cuh"

namespace psl {

constexpr int kCompWords = 8;
constexpr int kCompBytes = kCompWords * 4;
constexpr int kCompStages = 6;  // 4 being worked on + 2 in flight
constexpr int kCompMaxSplit = 4;

__host__ __device__ inline BigSmem comp_layout(uint32_t B)
{
    BigSmem L;
    uint32_t p = 0;
    L.stage_bytes = kTile * kCompBytes;
    L.ring = p;   p += kCompStages * L.stage_bytes;
    L.cnt = p;    p += round_up(kBigWarps * round_up(B, 8) * 2, 16);
    L.gcur = p;   p += round_up(B * 4, 16);
    L.lstart = p; p += round_up(B * 4, 16);
    L.pdest = p;  p += kBigTile * 4;
    L.perm = p;   p += kBigTile * 2;
    L.edges = p;
    L.misc = p;   p += 64 * 4;
    L.desc = p;   p += kCompStages * 16;
    L.bars = p;   p += kCompStages * 8;
    L.total = p;
    return L;
}

template <bool PROJ>
__global__ void __launch_bounds__(kBigThreads, 1) k_scatter_comp_big(const uint4* __restrict__ comp, Span sp,
                                                                    const __grid_constant__ DevBeam bm, uint32_t B,
                                                                    const uint32_t* __restrict__ table, uint32_t stride,
                                                                    SoAOut out, SegStats* sstats, const FusedScan fs,
                                                                    const StatsTail st)
{
    extern __shared__ __align__(128) uint8_t smem[];
    const uint32_t Bp = round_up(B, 8);
    const BigSmem L = comp_layout(B);
    uint16_t* cnt = reinterpret_cast<uint16_t*>(smem + L.cnt);
    uint32_t* gcur = reinterpret_cast<uint32_t*>(smem + L.gcur);
    uint32_t* lstart = reinterpret_cast<uint32_t*>(smem + L.lstart);
    uint32_t* pdest = reinterpret_cast<uint32_t*>(smem + L.pdest);
    uint16_t* perm = reinterpret_cast<uint16_t*>(smem + L.perm);
    uint32_t* misc = reinterpret_cast<uint32_t*>(smem + L.misc);
    TileDesc* s_desc = reinterpret_cast<TileDesc*>(smem + L.desc);
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem + L.bars);
    const uint32_t w = warp_id();
    const uint32_t col = sp.col0 + blockIdx.x * sp.split;

    if (threadIdx.x == 0) {
        for (int k = 0; k < kCompStages; ++k) mbar_init(&bars[k], 1);
        mbar_fence_init();
    }
    {
        uint32_t* cz = reinterpret_cast<uint32_t*>(cnt);
        for (uint32_t i = threadIdx.x; i < kBigWarps * Bp / 2; i += kBigThreads) cz[i] = 0;
    }
    griddep_wait();  // the histogram kernel's table, statistics and compacted survivors from here on

    // the sub-segments of this CTA's segment: first record of the region, survivors in it
    uint32_t sub_base[kCompMaxSplit], sub_n[kCompMaxSplit];
    uint32_t n = 0;  // ring stages (tiles of up to kTile survivors)
    {
        const unsigned long long nt = sp.n_tiles, S = gridDim.x, s = blockIdx.x;
        const uint32_t a = (uint32_t)(nt * s / S), b = (uint32_t)(nt * (s + 1) / S);
#pragma unroll
        for (int h = 0; h < kCompMaxSplit; ++h) {
            sub_base[h] = 0;
            sub_n[h] = 0;
            if (h < (int)sp.split) {
                sub_base[h] = (sp.tile_begin + a + (uint32_t)((unsigned long long)(b - a) * h / sp.split)) * (uint32_t)kTile;
                sub_n[h] = __ldcg(&sstats[col + h].n_surv);
                n += (sub_n[h] + kTile - 1) / kTile;
            }
        }
    }
    auto comp_tile = [&](uint32_t i) {
        TileDesc d;
        d.ptr = comp;
        d.first_index = 0;
        d.count = 0;
        bool found = false;
#pragma unroll
        for (int h = 0; h < kCompMaxSplit; ++h) {
            const uint32_t th = (sub_n[h] + kTile - 1) / kTile;
            if (!found && i < th) {
                d.ptr = comp + (size_t)(sub_base[h] + i * kTile) * 2;
                d.count = min((uint32_t)kTile, sub_n[h] - i * kTile);
                found = true;
            }
            if (!found) i -= th;
        }
        return d;
    };
    auto stage_ptr = [&](uint32_t i) { return reinterpret_cast<uint32_t*>(smem + L.ring + (i % kCompStages) * L.stage_bytes); };
    auto issue = [&](uint32_t i) {  // thread 0
        TileDesc d = comp_tile(i);
        s_desc[i % kCompStages] = d;
        mbar_expect_tx(&bars[i % kCompStages], d.count * kCompBytes);
        tma_load_1d(stage_ptr(i), d.ptr, d.count * kCompBytes, &bars[i % kCompStages]);
    };
    if (threadIdx.x == 0)
        for (uint32_t k = 0; k < (uint32_t)kCompStages && k < n; ++k) issue(k);

    uint32_t grun[8];
    if (fs.n_cols != 0) {
        fused_first_slots<kBigWarps>(fs, table, stride, B, col, gcur, lstart, misc, grun);
    } else {
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            uint32_t b = threadIdx.x * 8 + k;
            grun[k] = b < B ? table[(size_t)b * stride + col] : 0u;
        }
    }
    __syncthreads();

    double sum_out = 0.0;
    for (uint32_t base = 0; base < n; base += kBigQ) {
        const uint32_t nq = min((uint32_t)kBigQ, n - base);
        // stable rank inside the warp's 256 survivors (all inside ring stage base + w / 4), by the stored key
        uint32_t packed[kBigRounds];
#pragma unroll
        for (int r = 0; r < kBigRounds; ++r) packed[r] = kNone;
        const uint32_t q = w / (kBigWarps / kBigQ);
        if (q < nq) {
            const uint32_t i = base + q;
            const TileDesc td = s_desc[i % kCompStages];
            mbar_wait(&bars[i % kCompStages], (i / kCompStages) & 1u);
            const uint32_t* raw = stage_ptr(i);
            const int first = (int)(w % (kBigWarps / kBigQ)) * kBigSpan;
#pragma unroll
            for (int r = 0; r < kBigRounds; ++r) {
                const int idx = first + r * 32 + (int)lane_id();
                packed[r] = idx < (int)td.count ? raw[idx * kCompWords] : kNone;
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
            const uint4* p = reinterpret_cast<const uint4*>(stage_ptr(base + (irec / kTile))) + (irec % kTile) * 2;
            const uint4 lo = p[0], hi = p[1];
            Rec rec;
            rec.type = 0;
            rec.E = __uint_as_float(lo.y); rec.x = __uint_as_float(lo.z); rec.y = __uint_as_float(lo.w);
            rec.u = __uint_as_float(hi.x); rec.v = __uint_as_float(hi.y); rec.wt = __uint_as_float(hi.z);
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
            out.src[dest] = hi.w;
            if (PROJ && bm.out_proj) {
                out.xp[dest] = xm;
                out.yp[dest] = ym;
            }
            sum_out += (double)wt;
        }
        __syncthreads();  // the tile's stages and perm/pdest are free again
        if (threadIdx.x == 0)
            for (uint32_t k = 0; k < nq; ++k)
                if (base + kCompStages + k < n) issue(base + kCompStages + k);
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
