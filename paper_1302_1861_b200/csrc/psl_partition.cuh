// psl_partition.cuh -- the stable partition passes (histogram -> exclusive scan -> stable scatter).
//
// One pass splits a stream of records into B <= kMaxBuckets buckets, keeping input order inside a bucket.
// The stream is cut into S <= kMaxSegments contiguous SEGMENTS of whole tiles, one per persistent CTA
// (S = SMs x resident CTAs, so the grid is exactly one wave):
//   count   : CTA s streams its segment through a ring of TMA-filled shared-memory stages and histograms it
//             into a privatised shared-memory table; table[bucket][s] is written once at the end       (a8)
//   scan    : ONE exclusive scan over the table read bucket-major, segment-minor                      (a9)
//             => table[b][s] = (slots of all buckets < b) + (slots of bucket b in segments < s)
//   scatter : CTA s walks the same segment tile by tile with the same ring, keeping the running first free
//             slot of every bucket in registers.  Inside a tile every record is ranked among the records of
//             its bucket that precede it (per-warp private counters + __match_any_sync, then a scan over the
//             8 warps), staged in tile-sorted order in shared memory and written out in runs            (a10)
// Ranks come from ordered prefix sums only -- atomics are used for counting, never for claiming slots -- so
// the output is the unique stable order, bit-identical from run to run.
//
// ONTHEFLY (paper methods 1/2): one pass, bucket = the (type, energy) key, raw 28-byte
// records in, transport-ready SoA out (this file: 1024-record tiles; psl_bigtile.cuh: 4096-record tiles).
// INDEX (method 3): two LSD passes over the full (type, energy, y, x) key, psl_index.cuh;
// they share the histogram, scan and ranking code below.
#pragma once

#include "psl_device.cuh"

namespace psl {

constexpr int kScanThreads = 256;
constexpr int kScanRows = 16;
constexpr int kScanBlock = kScanThreads * kScanRows;  // 4096 table entries per scan CTA

constexpr int kStagesCount = 3;   // ring depth of the histogram kernels (28 KB stages; 2 when the histogram is large)
constexpr int kStagesRaw = 3;     // ring depth of the scatter kernels that read raw records
constexpr int kHistBytes = 16384; // privatised histogram budget of the histogram kernels

struct SoAOut {
    float *E, *x, *y, *u, *v, *w, *wt, *xp, *yp;
    uint32_t* src;
};

struct IdxOut {  // SoA view of the bare index
    float *E, *x, *y, *u, *v, *wt;
    uint32_t* src;
};

// which tiles a launch covers and which table columns its CTAs own: CTA s of the launch (gridDim.x CTAs)
// takes tiles tile_begin + [s*n_tiles/S, (s+1)*n_tiles/S) and column col0 + s.
// The histogram kernel may run `split` CTAs per segment (each on a contiguous part of it, with a table column
// of its own: gridDim.x = S * split); the scatter CTA of segment s then starts from column col0 + s * split.
struct Span {
    uint32_t tile_begin, n_tiles, col0, split;
};

__host__ __device__ inline uint32_t round_up(uint32_t a, uint32_t m) { return (a + m - 1) / m * m; }

// ---- shared-memory carve-up of the scatter kernels (dynamic shared memory, offsets in bytes) ---------
struct PartSmem {
    uint32_t ring, stage_bytes, cnt, gcur, lstart, perm, pdest, edges, misc, desc, bars, total;
};

__host__ __device__ inline PartSmem part_layout(uint32_t tile_bytes, uint32_t stages, uint32_t B, uint32_t n_edges,
                                                bool staged)
{
    PartSmem L;
    uint32_t p = 0;
    L.stage_bytes = round_up(tile_bytes, 128);
    L.ring = p;   p += stages * L.stage_bytes;
    L.cnt = p;    p += round_up(kWarps * round_up(B, 8) * 2, 16);  // [kWarps][Bp] uint16
    L.gcur = p;   p += round_up(B * 4, 16);                        // first global slot of each bucket, this tile
    L.lstart = p; if (staged) p += round_up(B * 4, 16);            // first tile-sorted slot of each bucket
    L.pdest = p;  if (staged) p += kTile * 4;                      // tile-sorted slot -> global slot
    L.perm = p;   if (staged) p += kTile * 2;                      // tile-sorted slot -> record in tile
    L.edges = p;  p += round_up(n_edges * 4, 16);
    L.misc = p;   p += 64 * 4;                                     // scan scratch
    L.desc = p;   p += stages * 16;                                // TileDesc per stage
    L.bars = p;   p += stages * 8;                                 // "full" mbarrier per stage
    L.total = p;
    return L;
}

// ---- histogram kernels --------------------------------------------------------------------------------
struct CountSmem {
    uint32_t ring, stage_bytes, hist, edges, desc, bars, total, rlog;
};

// R = 2^rlog interleaved copies of the histogram (copy = lane mod R) keep the lanes of a warp on
// different words; R is the largest power of two <= 32 with B * R * 4 <= kHistBytes.
__host__ __device__ inline CountSmem count_layout(uint32_t tile_bytes, uint32_t stages, uint32_t B, uint32_t n_edges)
{
    CountSmem L;
    uint32_t p = 0;
    L.rlog = 5;
    while (L.rlog > 0 && (B << L.rlog) * 4u > (uint32_t)kHistBytes) --L.rlog;
    L.stage_bytes = round_up(tile_bytes, 128);
    L.ring = p;  p += stages * L.stage_bytes;
    L.hist = p;  p += round_up((B << L.rlog) * 4, 16);
    L.edges = p; p += round_up(n_edges * 4, 16);
    L.desc = p;  p += stages * 16;
    L.bars = p;  p += stages * 8;
    L.total = p;
    return L;
}

__device__ __forceinline__ void stage_edges(const DevGrid& g, float* s_edges)
{
    if (g.ebin_mode != 0)
        for (int i = threadIdx.x; i <= g.n_ebins; i += blockDim.x) s_edges[i] = g.e_edges[i];
}

// one entry of the chunk table (psl_load_chunk)
__global__ void k_set_chunk(ChunkDesc* __restrict__ dst, ChunkDesc d) { *dst = d; }

// up to 128 entries at once (the descriptors travel as a kernel argument)
struct ChunkBatch {
    ChunkDesc d[128];
};
__global__ void k_set_chunks(ChunkDesc* __restrict__ dst, const __grid_constant__ ChunkBatch b, uint32_t n)
{
    griddep_launch();
    if (threadIdx.x < n) dst[threadIdx.x] = b.d[threadIdx.x];
}

// tile id -> descriptor.  Raw records: binary search over the chunk table (tiles never straddle chunks).
__device__ __forceinline__ TileDesc raw_tile(const ChunkDesc* __restrict__ chunks, uint32_t n_chunks, uint32_t t)
{
    uint32_t lo = 0, hi = n_chunks - 1;
    while (lo < hi) {
        uint32_t mid = (lo + hi + 1) >> 1;
        if (__ldg(&chunks[mid].tile0) <= t) lo = mid; else hi = mid - 1;
    }
    const ChunkDesc c = chunks[lo];
    const uint32_t local = (t - c.tile0) * (uint32_t)kTile;
    TileDesc d;
    d.ptr = c.ptr + (size_t)local * kRecBytes;
    d.first_index = c.first_index + local;
    d.count = min((uint32_t)kTile, c.n_records - local);
    return d;
}

// The same with the chunk of the caller's previous tile kept in `cur` (registers; start it zeroed): consecutive tiles
// nearly always share a chunk, and the search above is a chain of log2(n_chunks) dependent loads that thread 0 runs
// between two barriers of every tile loop (105 chunks: 7 loads + the descriptor, four times per 4096-record tile).
__device__ __forceinline__ TileDesc raw_tile(const ChunkDesc* __restrict__ chunks, uint32_t n_chunks, uint32_t t, ChunkDesc& cur)
{
    if (!(t >= cur.tile0 && (unsigned long long)(t - cur.tile0) * (unsigned long long)kTile < cur.n_records)) {
        uint32_t lo = 0, hi = n_chunks - 1;
        while (lo < hi) {
            uint32_t mid = (lo + hi + 1) >> 1;
            if (__ldg(&chunks[mid].tile0) <= t) lo = mid; else hi = mid - 1;
        }
        cur = chunks[lo];
    }
    const uint32_t local = (t - cur.tile0) * (uint32_t)kTile;
    TileDesc d;
    d.ptr = cur.ptr + (size_t)local * kRecBytes;
    d.first_index = cur.first_index + local;
    d.count = min((uint32_t)kTile, cur.n_records - local);
    return d;
}

// the segment of CTA s: tiles [t0, t1)
__device__ __forceinline__ void segment_of(const Span& sp, uint32_t& t0, uint32_t& t1)
{
    const unsigned long long n = sp.n_tiles, S = gridDim.x, s = blockIdx.x;
    t0 = sp.tile_begin + (uint32_t)(n * s / S);
    t1 = sp.tile_begin + (uint32_t)(n * (s + 1) / S);
}

// the part of its segment a histogram CTA takes when sp.split CTAs share a segment
__device__ __forceinline__ void split_segment_of(const Span& sp, uint32_t& t0, uint32_t& t1)
{
    const unsigned long long n = sp.n_tiles, S = gridDim.x / sp.split, s = blockIdx.x / sp.split, h = blockIdx.x % sp.split;
    const uint32_t a = (uint32_t)(n * s / S), b = (uint32_t)(n * (s + 1) / S);
    t0 = sp.tile_begin + a + (uint32_t)((unsigned long long)(b - a) * h / sp.split);
    t1 = sp.tile_begin + a + (uint32_t)((unsigned long long)(b - a) * (h + 1) / sp.split);
}

// ---- the ring: stage = i % STAGES, one "full" mbarrier per stage, refilled by thread 0 ------------------
__device__ __forceinline__ bool bulk_ok(const void* src, uint32_t bytes)
{
    return ((reinterpret_cast<uintptr_t>(src) & 15u) == 0) && ((bytes & 15u) == 0) && bytes > 0;
}

// thread 0: start the copy of one tile into a free stage (tiles that cannot be bulk-copied -- a source that
// is not 16-byte aligned, or the ragged last tile -- are fetched by all threads in ring_acquire instead)
__device__ __forceinline__ void ring_issue(uint32_t* s_dst, uint64_t* bar, const void* src, uint32_t bytes)
{
    if (bulk_ok(src, bytes)) {
        mbar_expect_tx(bar, bytes);
        tma_load_1d(s_dst, src, bytes, bar);
    }
}

// all threads: wait until the stage holds its tile.  `phase` is this thread's parity bit for the stage.
__device__ __forceinline__ void ring_acquire(uint32_t* s_dst, uint64_t* bar, uint32_t& phase_bits, uint32_t stage,
                                             const void* src, uint32_t bytes)
{
    if (bulk_ok(src, bytes)) {
        mbar_wait(bar, (phase_bits >> stage) & 1u);
        phase_bits ^= 1u << stage;
    } else {
        const uint32_t* g = reinterpret_cast<const uint32_t*>(src);
        for (uint32_t i = threadIdx.x; i < bytes / 4; i += blockDim.x) s_dst[i] = __ldg(g + i);
        __syncthreads();
    }
}

// After every warp has ranked its slice of the tile: thread t owns buckets 8t..8t+7 (one 16-byte row piece
// per warp).  Turns cnt[w][b] into the exclusive prefix over warps, publishes gcur[b] = first global slot
// of bucket b for this tile and advances the thread's running slots grun[8].  With STAGED also lstart[b] =
// exclusive prefix over buckets of the tile totals; returns the number of records that take part.
// Must be called by all threads after a __syncthreads; ends with a __syncthreads.
template <bool STAGED, int NW = kWarps>
__device__ __forceinline__ uint32_t finish_ranks(uint16_t* cnt, uint32_t B, uint32_t Bp, uint32_t* gcur, uint32_t* lstart,
                                                 uint32_t* misc, uint32_t (&grun)[8])
{
    const uint32_t b0 = threadIdx.x * 8;
    uint32_t t8[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    uint32_t mine = 0;
    if (b0 < Bp) {
        uint4 run = make_uint4(0, 0, 0, 0);  // 8 packed uint16 running sums (no carry: a tile has <= 1024 records)
#pragma unroll
        for (int w = 0; w < NW; ++w) {
            uint4* p = reinterpret_cast<uint4*>(cnt + w * Bp + b0);
            uint4 c = *p;
            c.x &= kRankCountMask2; c.y &= kRankCountMask2; c.z &= kRankCountMask2; c.w &= kRankCountMask2;  // warp_rank_claim's claim bits
            *p = run;
            run.x += c.x; run.y += c.y; run.z += c.z; run.w += c.w;
        }
        t8[0] = run.x & 0xFFFFu; t8[1] = run.x >> 16; t8[2] = run.y & 0xFFFFu; t8[3] = run.y >> 16;
        t8[4] = run.z & 0xFFFFu; t8[5] = run.z >> 16; t8[6] = run.w & 0xFFFFu; t8[7] = run.w >> 16;
#pragma unroll
        for (int k = 0; k < 8; ++k) mine += t8[k];
    }
    uint32_t total = 0, ex = 0;
    if (STAGED) {
        if (Bp <= 256) {  // every bucket belongs to a thread of warp 0: a warp scan, no barrier
            if (warp_id() == 0) {
                uint32_t inc = warp_incl_scan(mine);
                ex = inc - mine;
                if (lane_id() == 31) misc[32] = inc;
            }
        } else {
            ex = block_excl_scan(mine, misc, &total);
        }
    }
    if (b0 < Bp) {
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            if (b0 + k < B) {
                if (STAGED) lstart[b0 + k] = ex;
                ex += t8[k];
                gcur[b0 + k] = grun[k];
                grun[k] += t8[k];
            }
        }
    }
    __syncthreads();
    if (STAGED && Bp <= 256) total = misc[32];
    return total;
}

// a warp clears its own row of the counter matrix (only that warp ever touches it outside finish_ranks)
__device__ __forceinline__ void zero_row(uint16_t* row, uint32_t Bp)
{
    uint4* p = reinterpret_cast<uint4*>(row);
    for (uint32_t i = lane_id(); i < Bp / 8; i += 32) p[i] = make_uint4(0, 0, 0, 0);
}

// ------------------------------------------------------------------------------------------------------
// per-segment statistics: per-thread running values, reduced once per CTA in a fixed order
// ------------------------------------------------------------------------------------------------------
struct ThreadStats {
    uint32_t n_inv = 0, n_out = 0, n_jaw = 0, n_zero = 0, n_surv = 0;
    double sum_in = 0.0, sum_idx = 0.0;
};

__device__ __forceinline__ void write_seg_stats(ThreadStats t, SegStats* __restrict__ dst)
{
    __shared__ uint32_t s_n[kWarps][5];
    __shared__ double s_d[kWarps][2];
    t.n_inv = __reduce_add_sync(0xFFFFFFFFu, t.n_inv);
    t.n_out = __reduce_add_sync(0xFFFFFFFFu, t.n_out);
    t.n_jaw = __reduce_add_sync(0xFFFFFFFFu, t.n_jaw);
    t.n_zero = __reduce_add_sync(0xFFFFFFFFu, t.n_zero);
    t.n_surv = __reduce_add_sync(0xFFFFFFFFu, t.n_surv);
    t.sum_in = warp_sum_double(t.sum_in);
    t.sum_idx = warp_sum_double(t.sum_idx);
    if (lane_id() == 0) {
        uint32_t w = warp_id();
        s_n[w][0] = t.n_inv; s_n[w][1] = t.n_out; s_n[w][2] = t.n_jaw; s_n[w][3] = t.n_zero; s_n[w][4] = t.n_surv;
        s_d[w][0] = t.sum_in; s_d[w][1] = t.sum_idx;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        SegStats ts = {0, 0, 0, 0, 0, 0, 0.0, 0.0, 0.0};
        for (int w = 0; w < kWarps; ++w) {
            ts.n_invalid += s_n[w][0]; ts.n_outside += s_n[w][1]; ts.n_jaw += s_n[w][2];
            ts.n_zero += s_n[w][3]; ts.n_surv += s_n[w][4];
            ts.sum_in += s_d[w][0]; ts.sum_idx += s_d[w][1];
        }
        *dst = ts;
    }
}

// ------------------------------------------------------------------------------------------------------
// count over raw records.  IDX = false: ONTHEFLY, bucket = key of survivors (jaws applied).
//                          IDX = true : INDEX pass A, bucket = key & lo_mask of valid in-grid records.
// Also writes the segment's statistics (every record falls in exactly one class).
// ------------------------------------------------------------------------------------------------------
template <bool IDX, bool POS, bool EDGES, int BEAM>
__global__ void __launch_bounds__(kThreads, 2) k_count_raw(const ChunkDesc* __restrict__ chunks, uint32_t n_chunks,
                                                          Span sp, const __grid_constant__ DevGrid g,
                                                          const __grid_constant__ DevBeam bm, uint32_t B,
                                                          uint32_t lo_mask, uint32_t* __restrict__ table,
                                                          uint32_t stride, SegStats* __restrict__ sstats,
                                                          uint32_t n_stages, uint8_t* __restrict__ codes,
                                                          uint4* __restrict__ comp)
{
    extern __shared__ __align__(128) uint8_t smem[];
    __shared__ uint32_t s_comp[2][kWarps];  // (tile tag << 8 | survivors) per warp, by tile parity
    // a warp takes 128 consecutive records of the tile, 32 per round
    auto rec_idx = [](int r) { return warp_id() * (uint32_t)kWarpSpan + (uint32_t)r * 32u + lane_id(); };
    const CountSmem L = count_layout(kTile * kRecBytes, n_stages, B, g.n_ebins + 1);
    uint32_t* hist = reinterpret_cast<uint32_t*>(smem + L.hist);
    float* s_edges = reinterpret_cast<float*>(smem + L.edges);
    TileDesc* s_desc = reinterpret_cast<TileDesc*>(smem + L.desc);
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem + L.bars);
    const uint32_t rmask = (1u << L.rlog) - 1u;

    uint32_t t0, t1;
    split_segment_of(sp, t0, t1);
    const uint32_t n = t1 - t0;

    ChunkDesc ccur = {nullptr, 0u, 0u, 0u, 0u};  // thread 0: the chunk of the tile it described last
    griddep_launch();  // the scatter behind this kernel may set up and prefetch on SMs this grid has left
    griddep_wait();    // the chunk table (k_set_chunks) when this kernel was itself launched as a dependent
    if (threadIdx.x == 0) {
        for (uint32_t k = 0; k < n_stages; ++k) mbar_init(&bars[k], 1);
        mbar_fence_init();
        for (uint32_t k = 0; k < n_stages && k < n; ++k) {
            TileDesc d = raw_tile(chunks, n_chunks, t0 + k, ccur);
            s_desc[k] = d;
            ring_issue(reinterpret_cast<uint32_t*>(smem + L.ring + k * L.stage_bytes), &bars[k], d.ptr, d.count * kRecBytes);
        }
    }
    for (uint32_t i = threadIdx.x; i < (B << L.rlog); i += kThreads) hist[i] = 0;
    if (threadIdx.x < 2 * kWarps) (&s_comp[0][0])[threadIdx.x] = 0u;  // tag 0 = no tile: shared memory keeps the last launch's words
    stage_edges(g, s_edges);
    __syncthreads();

    ThreadStats st;
    uint32_t phase_bits = 0;
    // survivors of a rejecting beam, compacted in load order into the segment's own region of `comp` (32-byte
    // records {key, E, x, y, u, v, wt, src_index}, region = the segment's first record): what the scatter reads
    const bool compact = !IDX && BEAM != 0 && comp != nullptr;
    uint32_t comp_next = t0 * (uint32_t)kTile;
    for (uint32_t i = 0; i < n; ++i) {
        const uint32_t stage = i % n_stages;
        uint32_t* raw = reinterpret_cast<uint32_t*>(smem + L.ring + stage * L.stage_bytes);
        const TileDesc td = s_desc[stage];
        ring_acquire(raw, &bars[stage], phase_bits, stage, td.ptr, td.count * kRecBytes);
        // all of the thread's records first, then straight-line classification: independent chains interleave
        Rec rec[kRounds];
        bool have[kRounds];
        uint32_t skey[kRounds];  // compact: the key of a survivor, kNone otherwise
#pragma unroll
        for (int r = 0; r < kRounds; ++r) {
            const int idx = (int)rec_idx(r);
            have[r] = idx < (int)td.count;
            rec[r] = rec_from_smem(raw, have[r] ? idx : 0);
            if (IDX && g.apr) apr_apply(g.apr_seed, td.first_index + (uint32_t)idx, rec[r]);
        }
#pragma unroll
        for (int r = 0; r < kRounds; ++r) {
            uint32_t key;
            const int cls = classify<POS, EDGES, BEAM>(g, bm, rec[r], s_edges, key);
            const bool valid = have[r] & (cls != C_INVALID);
            st.sum_in += (double)(valid ? rec[r].wt : 0.0f);
            if (POS) st.sum_idx += (double)((valid & (cls != C_OUTSIDE)) ? rec[r].wt : 0.0f);
            st.n_inv += have[r] & (cls == C_INVALID);
            if (POS) st.n_out += have[r] & (cls == C_OUTSIDE);
            if (BEAM != 0) st.n_jaw += have[r] & (cls == C_JAW);
            if (BEAM == 2) st.n_zero += have[r] & (cls == C_ZERO);
            skey[r] = kNone;
            if (have[r] & (cls == C_SURVIVOR)) {
                st.n_surv += 1;
                const uint32_t bucket = IDX ? (key & lo_mask) : key;
                atomicAdd(&hist[(bucket << L.rlog) + (lane_id() & rmask)], 1u);
                skey[r] = key;
            }
            // one byte per record for the scatter of a rejecting beam: its key (< 255) or 255 = dropped, so that the
            // jaw / zero-weight arithmetic is not repeated there
            if (!IDX && codes != nullptr && have[r])
                codes[td.first_index + rec_idx(r)] = (uint8_t)(cls == C_SURVIVOR ? key : 255u);
        }
        if (!IDX && BEAM != 0) {
            if (compact) {
                // Stable: a warp's 128 records are consecutive, so its survivors follow those of the warps before it.
                // No barrier: every warp publishes (tile tag, survivors) in one word and spins only on the warps before
                // it; the tile's total is read one tile later from the other parity's slots, complete by then.
                volatile uint32_t* slot = s_comp[i & 1u];
                if (i != 0) {
                    const uint32_t pv = lane_id() < (uint32_t)kWarps ? (s_comp[(i & 1u) ^ 1u][lane_id()] & 0xFFu) : 0u;
                    comp_next += __reduce_add_sync(0xFFFFFFFFu, pv);
                }
                uint32_t bal[kRounds], wc = 0;
#pragma unroll
                for (int r = 0; r < kRounds; ++r) {
                    bal[r] = __ballot_sync(0xFFFFFFFFu, skey[r] != kNone);
                    wc += __popc(bal[r]);
                }
                if (lane_id() == 0) slot[warp_id()] = ((i + 1u) << 8) | wc;
                uint32_t v = 0;
                if (lane_id() < warp_id()) {
                    do { v = slot[lane_id()]; } while ((v >> 8) != i + 1u);
                    v &= 0xFFu;
                }
                // Survivors are stored one by one (two 16-byte stores each): the kernel is issue-bound with a jaw test
                // (62-67 % issue utilisation), and staging them in shared memory for whole-line stores -- per tile or
                // per warp -- cost more instructions than the stores saved (measured: 0.36 ms against 0.33 ms).
                uint32_t ex = comp_next + __reduce_add_sync(0xFFFFFFFFu, v);
#pragma unroll
                for (int r = 0; r < kRounds; ++r) {
                    if (skey[r] != kNone) {
                        uint4* dst = comp + (size_t)(ex + __popc(bal[r] & lanemask_lt())) * 2;
                        dst[0] = make_uint4(skey[r], __float_as_uint(rec[r].E), __float_as_uint(rec[r].x), __float_as_uint(rec[r].y));
                        dst[1] = make_uint4(__float_as_uint(rec[r].u), __float_as_uint(rec[r].v), __float_as_uint(rec[r].wt),
                                            td.first_index + rec_idx(r));
                    }
                    ex += __popc(bal[r]);
                }
            }
        }
        __syncthreads();  // every thread is done with the stage
        if (threadIdx.x == 0 && i + n_stages < n) {
            TileDesc d = raw_tile(chunks, n_chunks, t0 + i + n_stages, ccur);
            s_desc[stage] = d;
            ring_issue(raw, &bars[stage], d.ptr, d.count * kRecBytes);
        }
    }
    __syncthreads();
    const uint32_t col = sp.col0 + blockIdx.x;
    for (uint32_t b = threadIdx.x; b < B; b += kThreads) {
        uint32_t c = 0;
        for (uint32_t r = 0; r <= rmask; ++r) c += hist[(b << L.rlog) + ((r + lane_id()) & rmask)];
        table[(size_t)b * stride + col] = c;
    }
    if (!POS) st.sum_idx = st.sum_in;  // no grid to fall out of
    write_seg_stats(st, &sstats[col]);
}

// ------------------------------------------------------------------------------------------------------
// exclusive scan of the table read bucket-major / column-minor (virtual index v = b * n_cols + c lives at
// table[b * stride + c]).  Three small kernels: per-CTA sums, scan of the sums, in-place scan.
// ------------------------------------------------------------------------------------------------------
__device__ __forceinline__ size_t table_phys(uint32_t v, uint32_t n_cols, uint32_t stride)
{
    uint32_t b = v / n_cols;
    return (size_t)b * stride + (v - b * n_cols);
}

__global__ void __launch_bounds__(kScanThreads) k_scan_reduce(const uint32_t* __restrict__ table, uint32_t n_cols,
                                                             uint32_t stride, uint32_t L,
                                                             uint32_t* __restrict__ block_sums)
{
    __shared__ uint32_t s_w[kScanThreads / 32];
    uint32_t base = blockIdx.x * kScanBlock;
    uint32_t acc = 0;
#pragma unroll 4
    for (int r = 0; r < kScanRows; ++r) {
        uint32_t v = base + r * kScanThreads + threadIdx.x;
        if (v < L) acc += table[table_phys(v, n_cols, stride)];
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

__global__ void __launch_bounds__(kScanThreads) k_scan_apply(uint32_t* __restrict__ table, uint32_t n_cols,
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
            p = table_phys(v, n_cols, stride);
            x = table[p];
        }
        uint32_t tot;
        uint32_t ex = block_excl_scan(x, s_misc, &tot);
        if (v < L) table[p] = carry + ex;
        carry += tot;
        __syncthreads();
    }
}

// Small tables (a few keys x one wave of segments): the whole scan in ONE CTA -- a warp scans a row (bucket) at a
// time with coalesced loads, the row totals are scanned by the CTA, the row bases are added back -- followed
// (ONTHEFLY, offsets != nullptr) by what k_offsets_from_table computes.  B <= kMaxBuckets rows.
__global__ void __launch_bounds__(1024) k_scan_small(uint32_t* __restrict__ table, uint32_t n_cols, uint32_t stride,
                                                     uint32_t B, uint32_t* __restrict__ total_out, uint32_t K,
                                                     uint32_t* __restrict__ offsets, uint32_t* __restrict__ counts,
                                                     uint32_t n_pos, uint32_t n_batches,
                                                     uint32_t* __restrict__ batch_offsets)
{
    __shared__ uint32_t s_misc[64];
    __shared__ uint32_t s_row[kMaxBuckets];
    const uint32_t w = warp_id();
    for (uint32_t row = w; row < B; row += 32) {
        uint32_t* r = table + (size_t)row * stride;
        constexpr int kPieces = (kMaxSegments + 31) / 32;  // all loads of the row in flight before the first scan
        uint32_t x[kPieces];
#pragma unroll
        for (int k = 0; k < kPieces; ++k) {
            const uint32_t c = k * 32 + lane_id();
            x[k] = c < n_cols ? r[c] : 0u;
        }
        uint32_t carry = 0;
#pragma unroll
        for (int k = 0; k < kPieces; ++k) {
            const uint32_t c = k * 32 + lane_id();
            if (k * 32 < (int)n_cols) {
                const uint32_t inc = warp_incl_scan(x[k]);
                if (c < n_cols) r[c] = carry + inc - x[k];
                carry += __shfl_sync(0xFFFFFFFFu, inc, 31);
            }
        }
        if (lane_id() == 0) s_row[row] = carry;
    }
    __syncthreads();
    // exclusive scan of the row totals: thread t takes rows 2t, 2t+1
    const uint32_t r0 = 2 * threadIdx.x;
    const uint32_t a0 = r0 < B ? s_row[r0] : 0u, a1 = r0 + 1 < B ? s_row[r0 + 1] : 0u;
    uint32_t total;
    const uint32_t ex = block_excl_scan(a0 + a1, s_misc, &total);
    if (r0 < B) s_row[r0] = ex;
    if (r0 + 1 < B) s_row[r0 + 1] = ex + a0;
    __syncthreads();
    for (uint32_t row = w; row < B; row += 32) {
        uint32_t* r = table + (size_t)row * stride;
        const uint32_t base = s_row[row];
        for (uint32_t c = lane_id(); c < n_cols; c += 32) r[c] += base;
    }
    if (threadIdx.x == 0) *total_out = total;
    if (offsets == nullptr) return;
    for (uint32_t k = threadIdx.x; k <= K; k += 1024) {  // offsets[k] = scanned table[k][0] = the row base
        const uint32_t o = (k < K) ? s_row[k] : total;
        offsets[k] = o;
        if (k < K) counts[k] = ((k + 1 < K) ? s_row[k + 1] : total) - o;
        if (k % n_pos == 0 && k / n_pos <= n_batches) batch_offsets[k / n_pos] = o;
    }
}

// The same scan folded into the scatter kernel's prologue (small tables only): the table keeps the RAW counts
// and every scatter CTA derives its own first slots -- row totals (-> key offsets, scanned by warp 0) plus the
// sum of the row's columns before its own.  The table sits in L2 (the histogram kernel has just written it), the
// reads overlap the first record copies, and one kernel launch plus its serial 25 us leave the step.
// CTA 0 also writes what k_scan_small writes for the host (offsets, counts, batch offsets, total).
struct FusedScan {
    uint32_t n_cols;  // 0: the table is already scanned
    uint32_t n_pos, n_batches;
    uint32_t *total_out, *offsets, *counts, *batch_offsets;
    uint32_t* batch_offsets_host;  // mapped pinned copy of batch_offsets (may be null)
};

// On return (after a __syncthreads() by the caller before s_off / s_part are reused) grun[k] holds the first slot
// of bucket 8 * threadIdx.x + k for this CTA's column.  B <= 256; s_off, s_part: B words each; NW warps.
template <int NW>
__device__ __forceinline__ void fused_first_slots(const FusedScan& fs, const uint32_t* __restrict__ table, uint32_t stride,
                                                  uint32_t B, uint32_t col, uint32_t* s_off, uint32_t* s_part,
                                                  uint32_t* s_total, uint32_t (&grun)[8])
{
    const uint32_t w = warp_id(), lane = lane_id();
    // Four rows x 320 columns of loads in flight per warp (the loop is L2 round trips, not bytes); CTAs start at
    // different rows so that they do not all ask the same L2 slice for the same line at once.
    constexpr int kRowsInFlight = 4, kPieces = 10;
    const uint32_t rot = (blockIdx.x * 13u) % B;
    for (uint32_t j0 = w; j0 < B; j0 += kRowsInFlight * NW) {
        uint32_t tot[kRowsInFlight], part[kRowsInFlight];
#pragma unroll
        for (int a = 0; a < kRowsInFlight; ++a) tot[a] = part[a] = 0u;
        for (uint32_t c0 = 0; c0 < fs.n_cols; c0 += 32 * kPieces) {
            uint32_t v[kRowsInFlight][kPieces];
#pragma unroll
            for (int a = 0; a < kRowsInFlight; ++a) {
                const uint32_t j = j0 + a * NW;
                const uint32_t row = j + rot < B ? j + rot : j + rot - B;
                const uint32_t* r = table + (size_t)(j < B ? row : 0u) * stride;
#pragma unroll
                for (int k = 0; k < kPieces; ++k) {
                    const uint32_t c = c0 + k * 32 + lane;
                    v[a][k] = (j < B && c < fs.n_cols) ? r[c] : 0u;
                }
            }
#pragma unroll
            for (int a = 0; a < kRowsInFlight; ++a)
#pragma unroll
                for (int k = 0; k < kPieces; ++k) {
                    const uint32_t c = c0 + k * 32 + lane;
                    tot[a] += v[a][k];
                    part[a] += c < col ? v[a][k] : 0u;
                }
        }
#pragma unroll
        for (int a = 0; a < kRowsInFlight; ++a) {
            const uint32_t j = j0 + a * NW;
            const uint32_t row = j + rot < B ? j + rot : j + rot - B;
            const uint32_t t = __reduce_add_sync(0xFFFFFFFFu, tot[a]);
            const uint32_t q = __reduce_add_sync(0xFFFFFFFFu, part[a]);
            if (lane == 0 && j < B) {
                s_off[row] = t;
                s_part[row] = q;
            }
        }
    }
    __syncthreads();
    if (w == 0) {  // exclusive scan of the row totals: lane takes rows 8 * lane .. 8 * lane + 7
        uint32_t v[8], s = 0;
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            const uint32_t b = lane * 8 + k;
            v[k] = b < B ? s_off[b] : 0u;
            s += v[k];
        }
        const uint32_t inc = warp_incl_scan(s);
        uint32_t ex = inc - s;
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            const uint32_t b = lane * 8 + k;
            if (b < B) s_off[b] = ex;
            ex += v[k];
        }
        if (lane == 31) *s_total = inc;
    }
    __syncthreads();
#pragma unroll
    for (int k = 0; k < 8; ++k) {
        const uint32_t b = threadIdx.x * 8 + k;
        grun[k] = b < B ? s_off[b] + s_part[b] : 0u;
    }
    if (blockIdx.x == 0) {
        const uint32_t total = *s_total;
        if (threadIdx.x == 0) *fs.total_out = total;
        for (uint32_t k = threadIdx.x; k <= B; k += blockDim.x) {
            const uint32_t o = (k < B) ? s_off[k] : total;
            fs.offsets[k] = o;
            if (k < B) fs.counts[k] = ((k + 1 < B) ? s_off[k + 1] : total) - o;
            if (k % fs.n_pos == 0 && k / fs.n_pos <= fs.n_batches) {
                fs.batch_offsets[k / fs.n_pos] = o;
                if (fs.batch_offsets_host != nullptr) fs.batch_offsets_host[k / fs.n_pos] = o;
            }
        }
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

// fixed-order reduction of the per-segment statistics into one record (single CTA)
struct DevStats {
    unsigned long long n_invalid, n_outside, n_jaw, n_zero, n_surv;
    double sum_in, sum_idx, sum_out;
};

// the reduction proper, by one CTA of any size; out_host (may be null) is the mapped pinned copy the host reads
__device__ __forceinline__ void reduce_stats_cta(const SegStats* ts, uint32_t n_cols, DevStats* out, DevStats* out_host)
{
    __shared__ unsigned long long s_n[32][5];
    __shared__ double s_d[32][3];
    unsigned long long n[5] = {0, 0, 0, 0, 0};
    double d[3] = {0.0, 0.0, 0.0};
    for (uint32_t t = threadIdx.x; t < n_cols; t += blockDim.x) {
        // L2 loads: the records may have been written by other CTAs of the running kernel (stats_tail)
        const uint4* p = reinterpret_cast<const uint4*>(ts + t);
        const uint4 a = __ldcg(p), b = __ldcg(p + 1), c = __ldcg(p + 2);
        n[0] += a.x; n[1] += a.y; n[2] += a.z; n[3] += a.w; n[4] += b.x;
        d[0] += __hiloint2double((int)b.w, (int)b.z);
        d[1] += __hiloint2double((int)c.y, (int)c.x);
        d[2] += __hiloint2double((int)c.w, (int)c.z);
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
        for (uint32_t w = 0; w < blockDim.x / 32; ++w) {
            r.n_invalid += s_n[w][0]; r.n_outside += s_n[w][1]; r.n_jaw += s_n[w][2]; r.n_zero += s_n[w][3];
            r.n_surv += s_n[w][4];
            r.sum_in += s_d[w][0]; r.sum_idx += s_d[w][1]; r.sum_out += s_d[w][2];
        }
        *out = r;
        if (out_host != nullptr) *out_host = r;
    }
}

__global__ void __launch_bounds__(1024) k_reduce_stats(const SegStats* __restrict__ ts, uint32_t n_cols,
                                                       DevStats* __restrict__ out)
{
    reduce_stats_cta(ts, n_cols, out, nullptr);
}

// The same reduction as the tail of a scatter kernel: each CTA, having written its SegStats, takes a ticket; the
// last one reduces all n_cols records in the same fixed order and leaves the ticket at zero for the next launch.
struct StatsTail {
    uint32_t n_cols;  // 0: off (k_reduce_stats follows)
    uint32_t* ticket;
    DevStats *out, *out_host;
};

__device__ __forceinline__ void stats_tail(const StatsTail& st, const SegStats* sstats)
{
    if (st.n_cols == 0) return;
    __shared__ uint32_t s_last;
    if (threadIdx.x == 0) {
        __threadfence();  // this CTA's SegStats before its ticket
        s_last = atomicAdd(st.ticket, 1u) == gridDim.x - 1 ? 1u : 0u;
    }
    __syncthreads();
    if (s_last == 0) return;
    __threadfence();
    reduce_stats_cta(sstats, st.n_cols, st.out, st.out_host);
    if (threadIdx.x == 0) *st.ticket = 0u;
}

// prologue shared by the scatter kernels: barriers, first STAGES copies, zeroed counters, running slots
template <int STAGES, typename DescFn>
__device__ __forceinline__ void scatter_prologue(uint8_t* smem, const PartSmem& L, uint32_t B, uint32_t Bp, uint32_t n,
                                                 uint32_t t0, uint32_t rec_bytes, DescFn desc_of,
                                                 const uint32_t* __restrict__ table, uint32_t stride, uint32_t col,
                                                 uint32_t (&grun)[8])
{
    TileDesc* s_desc = reinterpret_cast<TileDesc*>(smem + L.desc);
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem + L.bars);
    if (threadIdx.x == 0) {
        for (int k = 0; k < STAGES; ++k) mbar_init(&bars[k], 1);
        mbar_fence_init();
        for (uint32_t k = 0; k < (uint32_t)STAGES && k < n; ++k) {
            TileDesc d = desc_of(t0 + k);
            s_desc[k] = d;
            ring_issue(reinterpret_cast<uint32_t*>(smem + L.ring + k * L.stage_bytes), &bars[k], d.ptr, d.count * rec_bytes);
        }
    }
    uint32_t* cz = reinterpret_cast<uint32_t*>(smem + L.cnt);
    for (uint32_t i = threadIdx.x; i < kWarps * Bp / 2; i += kThreads) cz[i] = 0;
    griddep_wait();  // the histogram kernel's table (and code bytes, statistics) from here on
#pragma unroll
    for (int k = 0; k < 8; ++k) {
        uint32_t b = threadIdx.x * 8 + k;
        grun[k] = b < B ? table[(size_t)b * stride + col] : 0u;
    }
}

// ------------------------------------------------------------------------------------------------------
// ONTHEFLY scatter: raw records -> transport-ready SoA (a1-a4, a6, a7, a10 fused).
// Survivors are ordered inside the tile by (key, input order) so that consecutive threads write consecutive
// slots of a key (block-local staging before the global scatter).
// ------------------------------------------------------------------------------------------------------
// PROJ: the ray slopes are needed at write-out (a fluence map to look up, or PSL_OUT_PROJ).
template <bool POS, bool EDGES, int BEAM, bool PROJ>
__global__ void __launch_bounds__(kThreads, 2) k_scatter_otf(const ChunkDesc* __restrict__ chunks, uint32_t n_chunks,
                                                            Span sp, const __grid_constant__ DevGrid g,
                                                            const __grid_constant__ DevBeam bm, uint32_t B,
                                                            const uint32_t* __restrict__ table, uint32_t stride,
                                                            SoAOut out, SegStats* sstats,
                                                            const uint8_t* __restrict__ codes, const FusedScan fs,
                                                            const StatsTail st)
{
    extern __shared__ __align__(128) uint8_t smem[];
    const uint32_t Bp = round_up(B, 8);
    const PartSmem L = part_layout(kTile * kRecBytes, kStagesRaw, B, g.n_ebins + 1, true);
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
    const uint32_t n = t1 - t0;
    uint32_t grun[8];
    ChunkDesc ccur = {nullptr, 0u, 0u, 0u, 0u};  // the chunk of the tile this thread described last
    auto desc_of = [&](uint32_t t) { return raw_tile(chunks, n_chunks, t, ccur); };
    scatter_prologue<kStagesRaw>(smem, L, B, Bp, n, t0, kRecBytes, desc_of, table, stride, col, grun);
    if (fs.n_cols != 0) fused_first_slots<kWarps>(fs, table, stride, B, col, gcur, lstart, misc, grun);  // raw table
    stage_edges(g, s_edges);
    __syncthreads();

    double sum_out = 0.0;
    uint32_t phase_bits = 0;
    uint32_t code_next[kRounds] = {255u, 255u, 255u, 255u};  // the histogram kernel's bytes for the NEXT tile
    if (codes != nullptr && n > 0) {
        const TileDesc nd = s_desc[0];
#pragma unroll
        for (int r = 0; r < kRounds; ++r) {
            const uint32_t idx = w * kWarpSpan + r * 32 + lane_id();
            code_next[r] = idx < nd.count ? (uint32_t)__ldg(codes + nd.first_index + idx) : 255u;
        }
    }
    for (uint32_t i = 0; i < n; ++i) {
        const uint32_t stage = i % kStagesRaw;
        uint32_t* raw = reinterpret_cast<uint32_t*>(smem + L.ring + stage * L.stage_bytes);
        const TileDesc td = s_desc[stage];
        ring_acquire(raw, &bars[stage], phase_bits, stage, td.ptr, td.count * kRecBytes);

        // bucket and stable rank inside the warp's slice of the tile
        uint32_t packed[kRounds];  // bucket << 9 | rank   (bucket < 2^11, rank < 2^7)
        if (codes != nullptr) {
            // the histogram kernel left the key of every record (255 = dropped): nothing to decode or test here; the
            // bytes of the next tile are fetched now and used one iteration later
#pragma unroll
            for (int r = 0; r < kRounds; ++r) packed[r] = code_next[r] == 255u ? kNone : code_next[r];
            if (i + 1 < n) {
                const TileDesc nd = s_desc[(i + 1) % kStagesRaw];
#pragma unroll
                for (int r = 0; r < kRounds; ++r) {
                    const uint32_t idx = w * kWarpSpan + r * 32 + lane_id();
                    code_next[r] = idx < nd.count ? (uint32_t)__ldg(codes + nd.first_index + idx) : 255u;
                }
            }
        } else {
            Rec rec[kRounds];
#pragma unroll
            for (int r = 0; r < kRounds; ++r) {
                int idx = w * kWarpSpan + r * 32 + lane_id();
                rec[r] = rec_from_smem(raw, idx < (int)td.count ? idx : 0);
            }
#pragma unroll
            for (int r = 0; r < kRounds; ++r) {  // straight-line: the four classifications interleave
                int idx = w * kWarpSpan + r * 32 + lane_id();
                uint32_t key;
                int cls = classify<POS, EDGES, BEAM>(g, bm, rec[r], s_edges, key);
                packed[r] = (idx < (int)td.count && cls == C_SURVIVOR) ? key : kNone;
            }
        }
        {
            uint32_t rk[kRounds];
            warp_rank_match<kRounds>(packed, rk, cnt + w * Bp);  // ranks: round r before round r + 1
#pragma unroll
            for (int r = 0; r < kRounds; ++r) packed[r] = packed[r] == kNone ? kNone : ((packed[r] << 9) | rk[r]);
        }
        __syncthreads();
        const uint32_t n_part = finish_ranks<true>(cnt, B, Bp, gcur, lstart, misc, grun);

        // tile-sorted order
#pragma unroll
        for (int r = 0; r < kRounds; ++r) {
            if (packed[r] != kNone) {
                uint32_t bucket = packed[r] >> 9, rank = packed[r] & 511u;
                uint32_t rel = cnt[w * Bp + bucket] + rank;  // among the tile's records of this bucket
                uint32_t p = lstart[bucket] + rel;
                perm[p] = (uint16_t)(w * kWarpSpan + r * 32 + lane_id());
                pdest[p] = gcur[bucket] + rel;
            }
        }
        __syncwarp();
        zero_row(cnt + w * Bp, Bp);
        __syncthreads();

        // write-out: thread j takes tile-sorted slot j
        for (uint32_t j = threadIdx.x; j < n_part; j += kThreads) {
            const uint32_t irec = perm[j];
            const uint32_t dest = pdest[j];
            Rec rec = rec_from_smem(raw, (int)irec);
            float q = q_of(rec.u, rec.v), wz, xm = 0.0f, ym = 0.0f, wt;
            if (PROJ) {
                float tx, ty;
                slopes(rec.u, rec.v, q, wz, tx, ty);
                xm = __fadd_rn(rec.x, __fmul_rn(tx, bm.dzM));
                ym = __fadd_rn(rec.y, __fmul_rn(ty, bm.dzM));
                wt = final_weight(bm, rec.wt, xm, ym);
            } else {  // no map, no projected outputs: the weight is wt or wt * mu
                wz = __fsqrt_rn(q);
                wt = bm.has_beam ? __fmul_rn(rec.wt, bm.mu) : rec.wt;
            }
            out.E[dest] = rec.E;
            out.x[dest] = rec.x;
            out.y[dest] = rec.y;
            out.u[dest] = rec.u;
            out.v[dest] = rec.v;
            out.w[dest] = wz;
            out.wt[dest] = wt;
            out.src[dest] = td.first_index + irec;
            if (PROJ && bm.out_proj) {
                out.xp[dest] = xm;
                out.yp[dest] = ym;
            }
            sum_out += (double)wt;
        }
        __syncthreads();  // the stage and perm/pdest are free again
        if (threadIdx.x == 0 && i + kStagesRaw < n) {
            TileDesc d = raw_tile(chunks, n_chunks, t0 + i + kStagesRaw, ccur);
            s_desc[stage] = d;
            ring_issue(raw, &bars[stage], d.ptr, d.count * kRecBytes);
        }
    }
    sum_out = warp_sum_double(sum_out);
    __shared__ double s_d[kWarps];
    if (lane_id() == 0) s_d[w] = sum_out;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0.0;
        for (int k = 0; k < kWarps; ++k) t += s_d[k];
        sstats[col].sum_out = t;
    }
    stats_tail(st, sstats);
}

// tiles of the pass-A output: n keyed records (32 bytes each), contiguous
__device__ __forceinline__ TileDesc keyed_tile(const uint4* aos, uint32_t n, uint32_t t)
{
    TileDesc d;
    d.ptr = aos + 2 * (size_t)t * kTile;
    d.first_index = t * kTile;
    d.count = min((uint32_t)kTile, n - t * (uint32_t)kTile);
    return d;
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

}  // namespace psl
