// psl_partition.cuh -- the stable partition passes (histogram -> exclusive scan -> stable scatter).
//
// One pass splits a stream of records into B <= kMaxBuckets buckets, keeping input order inside a bucket:
//   count   : each CTA histograms one tile of kTile records into table[bucket][tile]          (a8)
//   scan    : ONE exclusive scan over the table read bucket-major, tile-minor                  (a9)
//             => table[b][t] = (slots of all buckets < b) + (slots of bucket b in tiles < t)
//   scatter : each CTA re-derives the buckets of its tile, ranks every record among the records of the
//             same bucket that precede it in the tile (per-warp private counters + __match_any_sync, then
//             a scan over the 8 warps), and writes it to table[b][tile] + rank                  (a10)
// Ranks come from ordered prefix sums only -- atomics are used for counting, never for claiming slots -- so
// the output is the unique stable order, bit-identical from run to run.
//
// ONTHEFLY (paper methods 1/2): one pass, bucket = the (type, energy) key, raw 28-byte
// records in, transport-ready SoA out.  INDEX (method 3): two LSD passes over the full
// (type, energy, y, x) key split as key = hi * 2^s + lo: pass A (raw -> 32-byte keyed records, by lo), pass
// B (keyed records -> SoA index, by hi).
#pragma once

#include "psl_device.cuh"

namespace psl {

constexpr int kScanThreads = 256;
constexpr int kScanRows = 16;
constexpr int kScanBlock = kScanThreads * kScanRows;  // 4096 table entries per scan CTA

struct SoAOut {
    float *E, *x, *y, *u, *v, *w, *wt, *xp, *yp;
    uint32_t* src;
};

struct IdxOut {
    float *E, *x, *y, *u, *v, *wt;
    uint32_t* src;
    uint32_t* key;
};

// ---- shared-memory carve-up of the tile kernels (dynamic shared memory) --------------------------------
struct TileSmem {
    uint32_t* raw;     // staged input tile
    uint16_t* cnt;     // [kWarps][Bp] per-warp running counts -> exclusive over warps
    uint32_t* lstart;  // [B] first local (tile-sorted) slot of each bucket
    uint32_t* gbase;   // [B] first global slot of each bucket for this tile
    uint16_t* perm;    // [kTile] tile-sorted slot -> record in tile
    uint16_t* pbkt;    // [kTile] tile-sorted slot -> bucket
    float* edges;      // [n_ebins+1]
    uint32_t* misc;    // 64 words: scan scratch
    uint64_t* bar;     // mbarrier
};

__host__ __device__ inline uint32_t round_up(uint32_t a, uint32_t m) { return (a + m - 1) / m * m; }

__host__ __device__ inline uint32_t tile_smem_bytes(uint32_t in_bytes, uint32_t B, uint32_t n_edges, bool ranks,
                                                    bool reorder)
{
    uint32_t s = round_up(in_bytes, 128);
    if (ranks) s += round_up(kWarps * round_up(B, 8) * 2, 16);
    else s += round_up(B * 4, 16);  // plain histogram
    if (ranks) s += 2 * round_up(B * 4, 16);
    if (reorder) s += 2 * kTile * 2;
    s += round_up(n_edges * 4, 16);
    s += 64 * 4 + 16;
    return s;
}

__device__ __forceinline__ TileSmem carve(uint8_t* base, uint32_t in_bytes, uint32_t B, uint32_t n_edges, bool ranks,
                                          bool reorder)
{
    TileSmem t;
    uint8_t* p = base;
    t.raw = reinterpret_cast<uint32_t*>(p);
    p += round_up(in_bytes, 128);
    t.cnt = reinterpret_cast<uint16_t*>(p);
    if (ranks) p += round_up(kWarps * round_up(B, 8) * 2, 16);
    else p += round_up(B * 4, 16);
    t.lstart = reinterpret_cast<uint32_t*>(p);
    if (ranks) p += round_up(B * 4, 16);
    t.gbase = reinterpret_cast<uint32_t*>(p);
    if (ranks) p += round_up(B * 4, 16);
    t.perm = reinterpret_cast<uint16_t*>(p);
    if (reorder) p += kTile * 2;
    t.pbkt = reinterpret_cast<uint16_t*>(p);
    if (reorder) p += kTile * 2;
    t.edges = reinterpret_cast<float*>(p);
    p += round_up(n_edges * 4, 16);
    t.misc = reinterpret_cast<uint32_t*>(p);
    p += 64 * 4;
    t.bar = reinterpret_cast<uint64_t*>(p);
    return t;
}

__device__ __forceinline__ void stage_edges(const DevGrid& g, float* s_edges)
{
    if (g.ebin_mode != 0)
        for (int i = threadIdx.x; i <= g.n_ebins; i += blockDim.x) s_edges[i] = g.e_edges[i];
}

// After every warp has ranked its slice: turn cnt[w][b] into the exclusive prefix over warps, lstart[b]
// into the exclusive prefix over buckets of the tile totals, and fetch gbase[b] = table[b][tile].
// Returns the number of records of the tile that take part.  Contains __syncthreads.
__device__ __forceinline__ uint32_t finish_ranks(const TileSmem& s, uint32_t B, uint32_t Bp, const uint32_t* table,
                                                 uint32_t stride, uint32_t tile)
{
    __syncthreads();
    const uint32_t ipt = (B + kThreads - 1) / kThreads;  // <= 8 buckets per thread, blocked
    const uint32_t b0 = threadIdx.x * ipt;
    uint32_t tot[kMaxBuckets / kThreads];
    uint32_t mine = 0;
#pragma unroll
    for (uint32_t k = 0; k < kMaxBuckets / kThreads; ++k) {
        tot[k] = 0;
        uint32_t b = b0 + k;
        if (k < ipt && b < B) {
            uint32_t run = 0;
#pragma unroll
            for (int w = 0; w < kWarps; ++w) {
                uint32_t c = s.cnt[w * Bp + b];
                s.cnt[w * Bp + b] = (uint16_t)run;
                run += c;
            }
            tot[k] = run;
            mine += run;
        }
    }
    uint32_t total;
    uint32_t ex = block_excl_scan(mine, s.misc, &total);
#pragma unroll
    for (uint32_t k = 0; k < kMaxBuckets / kThreads; ++k) {
        uint32_t b = b0 + k;
        if (k < ipt && b < B) {
            s.lstart[b] = ex;
            ex += tot[k];
            s.gbase[b] = table[(size_t)b * stride + tile];
        }
    }
    __syncthreads();
    return total;
}

// ------------------------------------------------------------------------------------------------------
// count over raw records.  IDX = false: ONTHEFLY, bucket = key of survivors (jaws applied).
//                          IDX = true : INDEX pass A, bucket = key & lo_mask of valid in-grid records.
// Also writes the tile's statistics (every record falls in exactly one class).
// ------------------------------------------------------------------------------------------------------
template <bool IDX>
__global__ void __launch_bounds__(kThreads) k_count_raw(const TileDesc* __restrict__ tiles, uint32_t tile0,
                                                       const __grid_constant__ DevGrid g,
                                                       const __grid_constant__ DevBeam bm, uint32_t B,
                                                       uint32_t lo_mask, uint32_t* __restrict__ table,
                                                       uint32_t stride, TileStats* __restrict__ tstats)
{
    extern __shared__ __align__(128) uint8_t smem[];
    TileSmem s = carve(smem, kTile * kRecBytes, B, g.n_ebins + 1, false, false);
    uint32_t* hist = reinterpret_cast<uint32_t*>(s.cnt);
    const uint32_t tile = tile0 + blockIdx.x;
    const TileDesc td = tiles[tile];

    if (threadIdx.x == 0) {
        mbar_init(s.bar, 1);
        mbar_fence_init();
    }
    for (uint32_t b = threadIdx.x; b < B; b += kThreads) hist[b] = 0;
    stage_edges(g, s.edges);
    __syncthreads();
    load_tile_bytes(s.raw, td.ptr, td.count * kRecBytes, s.bar, 0);

    uint32_t n_inv = 0, n_out = 0, n_jaw = 0, n_zero = 0, n_surv = 0;
    double sum_in = 0.0, sum_idx = 0.0;
#pragma unroll 2
    for (int r = 0; r < kRounds; ++r) {
        int idx = r * kThreads + threadIdx.x;
        uint32_t bucket = kNone;
        if (idx < (int)td.count) {
            Rec rec = rec_from_smem(s.raw, idx);
            uint32_t key;
            int cls = classify_raw(g, bm, rec, s.edges, key);
            if (cls != C_INVALID) sum_in += (double)rec.wt;
            if (cls != C_INVALID && cls != C_OUTSIDE) sum_idx += (double)rec.wt;
            n_inv += cls == C_INVALID;
            n_out += cls == C_OUTSIDE;
            n_jaw += cls == C_JAW;
            n_zero += cls == C_ZERO;
            n_surv += cls == C_SURVIVOR;
            if (cls == C_SURVIVOR) bucket = IDX ? (key & lo_mask) : key;
        }
        // warp-aggregated shared-memory histogram: one atomic per distinct bucket per warp-round
        uint32_t active = __ballot_sync(0xFFFFFFFFu, bucket != kNone);
        if (bucket != kNone) {
            uint32_t peers = __match_any_sync(active, bucket);
            if ((int)lane_id() == __ffs(peers) - 1) atomicAdd(&hist[bucket], (uint32_t)__popc(peers));
        }
    }
    __syncthreads();
    for (uint32_t b = threadIdx.x; b < B; b += kThreads) table[(size_t)b * stride + tile] = hist[b];

    // tile statistics, reduced in a fixed order
    n_inv = __reduce_add_sync(0xFFFFFFFFu, n_inv);
    n_out = __reduce_add_sync(0xFFFFFFFFu, n_out);
    n_jaw = __reduce_add_sync(0xFFFFFFFFu, n_jaw);
    n_zero = __reduce_add_sync(0xFFFFFFFFu, n_zero);
    n_surv = __reduce_add_sync(0xFFFFFFFFu, n_surv);
    sum_in = warp_sum_double(sum_in);
    sum_idx = warp_sum_double(sum_idx);
    __shared__ uint32_t s_n[kWarps][5];
    __shared__ double s_d[kWarps][2];
    if (lane_id() == 0) {
        uint32_t w = warp_id();
        s_n[w][0] = n_inv; s_n[w][1] = n_out; s_n[w][2] = n_jaw; s_n[w][3] = n_zero; s_n[w][4] = n_surv;
        s_d[w][0] = sum_in; s_d[w][1] = sum_idx;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        TileStats ts = {0, 0, 0, 0, 0, 0, 0.0, 0.0, 0.0};
        for (int w = 0; w < kWarps; ++w) {
            ts.n_invalid += s_n[w][0]; ts.n_outside += s_n[w][1]; ts.n_jaw += s_n[w][2];
            ts.n_zero += s_n[w][3]; ts.n_surv += s_n[w][4];
            ts.sum_in += s_d[w][0]; ts.sum_idx += s_d[w][1];
        }
        tstats[tile] = ts;
    }
}

// ------------------------------------------------------------------------------------------------------
// exclusive scan of the table read bucket-major / tile-minor (virtual index v = b * n_tiles + t lives at
// table[b * stride + t]).  Three small kernels: per-CTA sums, scan of the sums, in-place scan.
// ------------------------------------------------------------------------------------------------------
__device__ __forceinline__ size_t table_phys(uint32_t v, uint32_t n_tiles, uint32_t stride)
{
    uint32_t b = v / n_tiles;
    return (size_t)b * stride + (v - b * n_tiles);
}

__global__ void __launch_bounds__(kScanThreads) k_scan_reduce(const uint32_t* __restrict__ table, uint32_t n_tiles,
                                                             uint32_t stride, uint32_t L,
                                                             uint32_t* __restrict__ block_sums)
{
    __shared__ uint32_t s_w[kScanThreads / 32];
    uint32_t base = blockIdx.x * kScanBlock;
    uint32_t acc = 0;
#pragma unroll 4
    for (int r = 0; r < kScanRows; ++r) {
        uint32_t v = base + r * kScanThreads + threadIdx.x;
        if (v < L) acc += table[table_phys(v, n_tiles, stride)];
    }
    acc = __reduce_add_sync(0xFFFFFFFFu, acc);
    if (lane_id() == 0) s_w[warp_id()] = acc;
    __syncthreads();
    if (threadIdx.x == 0) {
        uint32_t t = 0;
        for (int w = 0; w < kScanThreads / 32; ++w) t += s_w[w];
        block_sums[blockIdx.x] = t;
    }
}

// single CTA: exclusive scan of block_sums in place, grand total to *total_out
__global__ void __launch_bounds__(1024) k_scan_sums(uint32_t* __restrict__ block_sums, uint32_t n,
                                                    uint32_t* __restrict__ total_out)
{
    __shared__ uint32_t s_misc[64];
    uint32_t carry = 0;
    for (uint32_t base = 0; base < n; base += 1024) {
        uint32_t i = base + threadIdx.x;
        uint32_t v = i < n ? block_sums[i] : 0u;
        uint32_t tot;
        uint32_t ex = block_excl_scan(v, s_misc, &tot);
        if (i < n) block_sums[i] = carry + ex;
        carry += tot;
        __syncthreads();
    }
    if (threadIdx.x == 0) *total_out = carry;
}

__global__ void __launch_bounds__(kScanThreads) k_scan_apply(uint32_t* __restrict__ table, uint32_t n_tiles,
                                                            uint32_t stride, uint32_t L,
                                                            const uint32_t* __restrict__ block_sums)
{
    __shared__ uint32_t s_misc[64];
    uint32_t base = blockIdx.x * kScanBlock;
    uint32_t carry = block_sums[blockIdx.x];
    for (int r = 0; r < kScanRows; ++r) {
        uint32_t v = base + r * kScanThreads + threadIdx.x;
        size_t p = 0;
        uint32_t x = 0;
        if (v < L) {
            p = table_phys(v, n_tiles, stride);
            x = table[p];
        }
        uint32_t tot;
        uint32_t ex = block_excl_scan(x, s_misc, &tot);
        if (v < L) table[p] = carry + ex;
        carry += tot;
        __syncthreads();
    }
}

// ONTHEFLY: offsets[k] = first slot of key k = scanned table[k][0]; counts; per-(type,energy) batch offsets.
__global__ void k_offsets_from_table(const uint32_t* __restrict__ table, uint32_t stride, uint32_t K,
                                     const uint32_t* __restrict__ total, uint32_t* __restrict__ offsets,
                                     uint32_t* __restrict__ counts, uint32_t n_pos, uint32_t n_batches,
                                     uint32_t* __restrict__ batch_offsets)
{
    uint32_t k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k > K) return;
    uint32_t o = (k < K) ? table[(size_t)k * stride] : *total;
    offsets[k] = o;
    if (k < K) counts[k] = ((k + 1 < K) ? table[(size_t)(k + 1) * stride] : *total) - o;
    if (k % n_pos == 0 && k / n_pos <= n_batches) batch_offsets[k / n_pos] = o;
}

// ------------------------------------------------------------------------------------------------------
// ONTHEFLY scatter: raw records -> transport-ready SoA (a1-a4, a6, a7, a10 fused).
// The tile is staged once in shared memory; survivors are ordered inside the tile by (key, input order) so
// that consecutive threads write consecutive slots of a key (block-local staging before the global scatter).
// ------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(kThreads) k_scatter_otf(const TileDesc* __restrict__ tiles,
                                                         const __grid_constant__ DevGrid g,
                                                         const __grid_constant__ DevBeam bm, uint32_t B,
                                                         const uint32_t* __restrict__ table, uint32_t stride,
                                                         SoAOut out, TileStats* __restrict__ tstats)
{
    extern __shared__ __align__(128) uint8_t smem[];
    const uint32_t Bp = round_up(B, 8);
    TileSmem s = carve(smem, kTile * kRecBytes, B, g.n_ebins + 1, true, true);
    const uint32_t tile = blockIdx.x;
    const TileDesc td = tiles[tile];
    const uint32_t w = warp_id();

    if (threadIdx.x == 0) {
        mbar_init(s.bar, 1);
        mbar_fence_init();
    }
    for (uint32_t i = threadIdx.x; i < kWarps * Bp / 2; i += kThreads) reinterpret_cast<uint32_t*>(s.cnt)[i] = 0;
    stage_edges(g, s.edges);
    __syncthreads();
    load_tile_bytes(s.raw, td.ptr, td.count * kRecBytes, s.bar, 0);

    // pass 1 over the tile: bucket and stable rank inside the warp's slice
    uint32_t packed[kRounds];  // bucket << 9 | rank   (bucket < 2^11... stored in 22 bits, rank < 2^9)
#pragma unroll
    for (int r = 0; r < kRounds; ++r) {
        int idx = w * kWarpSpan + r * 32 + lane_id();
        uint32_t bucket = kNone;
        if (idx < (int)td.count) {
            Rec rec = rec_from_smem(s.raw, idx);
            uint32_t key;
            if (classify_raw(g, bm, rec, s.edges, key) == C_SURVIVOR) bucket = key;
        }
        uint32_t rank = warp_rank(bucket, s.cnt + w * Bp);
        packed[r] = bucket == kNone ? kNone : ((bucket << 9) | rank);
    }
    uint32_t n_part = finish_ranks(s, B, Bp, table, stride, tile);

    // tile-sorted order
#pragma unroll
    for (int r = 0; r < kRounds; ++r) {
        if (packed[r] != kNone) {
            uint32_t bucket = packed[r] >> 9, rank = packed[r] & 511u;
            uint32_t p = s.lstart[bucket] + s.cnt[w * Bp + bucket] + rank;
            s.perm[p] = (uint16_t)(w * kWarpSpan + r * 32 + lane_id());
            s.pbkt[p] = (uint16_t)bucket;
        }
    }
    __syncthreads();

    // write-out: thread j takes tile-sorted slot j
    double sum_out = 0.0;
    for (uint32_t j = threadIdx.x; j < n_part; j += kThreads) {
        uint32_t i = s.perm[j], bucket = s.pbkt[j];
        uint32_t dest = s.gbase[bucket] + (j - s.lstart[bucket]);
        Rec rec = rec_from_smem(s.raw, (int)i);
        float q = q_of(rec.u, rec.v), wz, tx, ty;
        slopes(rec.u, rec.v, q, wz, tx, ty);
        float xm = __fadd_rn(rec.x, __fmul_rn(tx, bm.dzM));
        float ym = __fadd_rn(rec.y, __fmul_rn(ty, bm.dzM));
        float wt = final_weight(bm, rec.wt, xm, ym);
        out.E[dest] = rec.E;
        out.x[dest] = rec.x;
        out.y[dest] = rec.y;
        out.u[dest] = rec.u;
        out.v[dest] = rec.v;
        out.w[dest] = wz;
        out.wt[dest] = wt;
        out.src[dest] = td.first_index + i;
        if (bm.out_proj) {
            out.xp[dest] = xm;
            out.yp[dest] = ym;
        }
        sum_out += (double)wt;
    }
    sum_out = warp_sum_double(sum_out);
    __shared__ double s_d[kWarps];
    if (lane_id() == 0) s_d[w] = sum_out;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0.0;
        for (int k = 0; k < kWarps; ++k) t += s_d[k];
        tstats[tile].sum_out = t;
    }
}

// ------------------------------------------------------------------------------------------------------
// INDEX pass A: raw records -> 32-byte keyed records {key, E, x, y, u, v, wt, src}, stably partitioned by
// the low digit of the key.  One record = one full 32-byte sector, written by its own thread.
// Also writes the high digit of every record (uint16) to hi16[] in the new order, which is all pass B's
// count needs to read.
// ------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(kThreads) k_scatter_idx_a(const TileDesc* __restrict__ tiles,
                                                           const __grid_constant__ DevGrid g,
                                                           const __grid_constant__ DevBeam bm, uint32_t B,
                                                           uint32_t lo_bits, const uint32_t* __restrict__ table,
                                                           uint32_t stride, uint4* __restrict__ aos,
                                                           uint16_t* __restrict__ hi16)
{
    extern __shared__ __align__(128) uint8_t smem[];
    const uint32_t Bp = round_up(B, 8);
    TileSmem s = carve(smem, kTile * kRecBytes, B, g.n_ebins + 1, true, false);
    const uint32_t tile = blockIdx.x;
    const TileDesc td = tiles[tile];
    const uint32_t w = warp_id();
    const uint32_t lo_mask = (1u << lo_bits) - 1u;

    if (threadIdx.x == 0) {
        mbar_init(s.bar, 1);
        mbar_fence_init();
    }
    for (uint32_t i = threadIdx.x; i < kWarps * Bp / 2; i += kThreads) reinterpret_cast<uint32_t*>(s.cnt)[i] = 0;
    stage_edges(g, s.edges);
    __syncthreads();
    load_tile_bytes(s.raw, td.ptr, td.count * kRecBytes, s.bar, 0);

    uint32_t packed[kRounds];  // key << 9 | rank   (key < 2^22)
#pragma unroll
    for (int r = 0; r < kRounds; ++r) {
        int idx = w * kWarpSpan + r * 32 + lane_id();
        uint32_t key = kNone;
        if (idx < (int)td.count) {
            Rec rec = rec_from_smem(s.raw, idx);
            if (classify_raw(g, bm, rec, s.edges, key) != C_SURVIVOR) key = kNone;
        }
        uint32_t rank = warp_rank(key == kNone ? kNone : (key & lo_mask), s.cnt + w * Bp);
        packed[r] = key == kNone ? kNone : ((key << 9) | rank);
    }
    finish_ranks(s, B, Bp, table, stride, tile);

#pragma unroll
    for (int r = 0; r < kRounds; ++r) {
        if (packed[r] != kNone) {
            uint32_t key = packed[r] >> 9, rank = packed[r] & 511u, bucket = key & lo_mask;
            uint32_t dest = s.gbase[bucket] + s.cnt[w * Bp + bucket] + rank;
            int idx = w * kWarpSpan + r * 32 + lane_id();
            const uint32_t* p = s.raw + idx * kRecWords;
            aos[2 * (size_t)dest + 0] = make_uint4(key, p[1], p[2], p[3]);
            aos[2 * (size_t)dest + 1] = make_uint4(p[4], p[5], p[6], td.first_index + idx);
            hi16[dest] = (uint16_t)(key >> lo_bits);
        }
    }
}

// INDEX pass B count: histogram of the uint16 high digits, tile by tile of the pass-A output.
__global__ void __launch_bounds__(kThreads) k_count_hi16(const uint16_t* __restrict__ hi16,
                                                        const uint32_t* __restrict__ n_ptr, uint32_t B,
                                                        uint32_t* __restrict__ table, uint32_t stride)
{
    extern __shared__ __align__(128) uint8_t smem[];
    uint32_t* hist = reinterpret_cast<uint32_t*>(smem);
    const uint32_t tile = blockIdx.x;
    const uint32_t n = *n_ptr;
    const uint32_t first = tile * kTile;
    const uint32_t count = first < n ? min((uint32_t)kTile, n - first) : 0u;
    for (uint32_t b = threadIdx.x; b < B; b += kThreads) hist[b] = 0;
    __syncthreads();
#pragma unroll
    for (int r = 0; r < kRounds; ++r) {
        uint32_t idx = r * kThreads + threadIdx.x;
        uint32_t bucket = idx < count ? (uint32_t)hi16[first + idx] : kNone;
        uint32_t active = __ballot_sync(0xFFFFFFFFu, bucket != kNone);
        if (bucket != kNone) {
            uint32_t peers = __match_any_sync(active, bucket);
            if ((int)lane_id() == __ffs(peers) - 1) atomicAdd(&hist[bucket], (uint32_t)__popc(peers));
        }
    }
    __syncthreads();
    for (uint32_t b = threadIdx.x; b < B; b += kThreads) table[(size_t)b * stride + tile] = hist[b];
}

// ------------------------------------------------------------------------------------------------------
// INDEX pass B scatter: keyed records (sorted by low digit) -> SoA index sorted by the full key, plus the
// full key of every slot (used once, by binary search, to build offsets[K+1]).
// ------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(kThreads) k_scatter_idx_b(const uint4* __restrict__ aos,
                                                           const uint16_t* __restrict__ hi16,
                                                           const uint32_t* __restrict__ n_ptr, uint32_t B,
                                                           const uint32_t* __restrict__ table, uint32_t stride,
                                                           IdxOut out)
{
    extern __shared__ __align__(128) uint8_t smem[];
    const uint32_t Bp = round_up(B, 8);
    TileSmem s = carve(smem, kTile * 32, B, 0, true, true);
    const uint32_t tile = blockIdx.x;
    const uint32_t n = *n_ptr;
    const uint32_t first = tile * kTile;
    if (first >= n) return;
    const uint32_t count = min((uint32_t)kTile, n - first);
    const uint32_t w = warp_id();

    if (threadIdx.x == 0) {
        mbar_init(s.bar, 1);
        mbar_fence_init();
    }
    for (uint32_t i = threadIdx.x; i < kWarps * Bp / 2; i += kThreads) reinterpret_cast<uint32_t*>(s.cnt)[i] = 0;
    __syncthreads();
    if (threadIdx.x == 0) {  // 32-byte records from a 256-byte-aligned array: always bulk-copyable
        mbar_expect_tx(s.bar, count * 32);
        tma_load_1d(s.raw, aos + 2 * (size_t)first, count * 32, s.bar);
    }

    uint32_t packed[kRounds];
#pragma unroll
    for (int r = 0; r < kRounds; ++r) {
        uint32_t idx = w * kWarpSpan + r * 32 + lane_id();
        uint32_t bucket = idx < count ? (uint32_t)hi16[first + idx] : kNone;
        uint32_t rank = warp_rank(bucket, s.cnt + w * Bp);
        packed[r] = bucket == kNone ? kNone : ((bucket << 9) | rank);
    }
    uint32_t n_part = finish_ranks(s, B, Bp, table, stride, tile);

#pragma unroll
    for (int r = 0; r < kRounds; ++r) {
        if (packed[r] != kNone) {
            uint32_t bucket = packed[r] >> 9, rank = packed[r] & 511u;
            uint32_t p = s.lstart[bucket] + s.cnt[w * Bp + bucket] + rank;
            s.perm[p] = (uint16_t)(w * kWarpSpan + r * 32 + lane_id());
            s.pbkt[p] = (uint16_t)bucket;
        }
    }
    mbar_wait(s.bar, 0);
    __syncthreads();

    const uint4* s_rec = reinterpret_cast<const uint4*>(s.raw);
    for (uint32_t j = threadIdx.x; j < n_part; j += kThreads) {
        uint32_t i = s.perm[j], bucket = s.pbkt[j];
        uint32_t dest = s.gbase[bucket] + (j - s.lstart[bucket]);
        uint4 a = s_rec[2 * i + 0], b = s_rec[2 * i + 1];
        out.key[dest] = a.x;
        out.E[dest] = __uint_as_float(a.y);
        out.x[dest] = __uint_as_float(a.z);
        out.y[dest] = __uint_as_float(a.w);
        out.u[dest] = __uint_as_float(b.x);
        out.v[dest] = __uint_as_float(b.y);
        out.wt[dest] = __uint_as_float(b.z);
        out.src[dest] = b.w;
    }
}

// offsets[k] = number of sorted slots whose key is < k (binary search; k = 0..K).  keys[0..n) ascending.
__global__ void k_offsets_by_search(const uint32_t* __restrict__ keys, const uint32_t* __restrict__ n_ptr, uint32_t K,
                                    uint32_t* __restrict__ offsets)
{
    uint32_t k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k > K) return;
    uint32_t lo = 0, hi = *n_ptr;
    while (lo < hi) {
        uint32_t mid = lo + ((hi - lo) >> 1);
        if (keys[mid] < k) lo = mid + 1; else hi = mid;
    }
    offsets[k] = lo;
}

__global__ void k_counts_from_offsets(const uint32_t* __restrict__ offsets, uint32_t K, uint32_t* __restrict__ counts,
                                      uint32_t n_pos, uint32_t n_batches, uint32_t* __restrict__ batch_offsets)
{
    uint32_t k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k > K) return;
    uint32_t o = offsets[k];
    if (k < K) counts[k] = offsets[k + 1] - o;
    if (k % n_pos == 0 && k / n_pos <= n_batches) batch_offsets[k / n_pos] = o;
}

// describe the tiles of one chunk: tile t covers records [t*kTile, ...) of the chunk
__global__ void k_fill_tiles(TileDesc* __restrict__ tiles, uint32_t tile0, uint32_t n_tiles, const uint8_t* base,
                             uint32_t first_index, uint32_t n_records)
{
    uint32_t t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= n_tiles) return;
    TileDesc d;
    d.ptr = base + (size_t)t * kTile * kRecBytes;
    d.first_index = first_index + t * kTile;
    d.count = min((uint32_t)kTile, n_records - t * kTile);
    tiles[tile0 + t] = d;
}

// fixed-order reduction of the per-tile statistics into one record (single CTA)
struct DevStats {
    unsigned long long n_invalid, n_outside, n_jaw, n_zero, n_surv;
    double sum_in, sum_idx, sum_out;
};

__global__ void __launch_bounds__(1024) k_reduce_stats(const TileStats* __restrict__ ts, uint32_t n_tiles,
                                                       DevStats* __restrict__ out)
{
    __shared__ unsigned long long s_n[32][5];
    __shared__ double s_d[32][3];
    unsigned long long n[5] = {0, 0, 0, 0, 0};
    double d[3] = {0.0, 0.0, 0.0};
    for (uint32_t t = threadIdx.x; t < n_tiles; t += 1024) {
        TileStats x = ts[t];
        n[0] += x.n_invalid; n[1] += x.n_outside; n[2] += x.n_jaw; n[3] += x.n_zero; n[4] += x.n_surv;
        d[0] += x.sum_in; d[1] += x.sum_idx; d[2] += x.sum_out;
    }
    for (int k = 0; k < 5; ++k)
        for (int o = 16; o > 0; o >>= 1) n[k] += __shfl_xor_sync(0xFFFFFFFFu, n[k], o);
    for (int k = 0; k < 3; ++k) d[k] = warp_sum_double(d[k]);
    if (lane_id() == 0) {
        for (int k = 0; k < 5; ++k) s_n[warp_id()][k] = n[k];
        for (int k = 0; k < 3; ++k) s_d[warp_id()][k] = d[k];
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        DevStats r = {0, 0, 0, 0, 0, 0.0, 0.0, 0.0};
        for (int w = 0; w < 32; ++w) {
            r.n_invalid += s_n[w][0]; r.n_outside += s_n[w][1]; r.n_jaw += s_n[w][2]; r.n_zero += s_n[w][3];
            r.n_surv += s_n[w][4];
            r.sum_in += s_d[w][0]; r.sum_idx += s_d[w][1]; r.sum_out += s_d[w][2];
        }
        *out = r;
    }
}

}  // namespace psl
