// psl_device.cuh -- device-side building blocks shared by the kernels of libpsl_b200 (sm_100a only).
//
// Holds: the kernel-parameter structs, the per-record arithmetic of the hot path (validity, energy bin,
// position bin, key, jaw projection, fluence lookup -- include/psl.h "Arithmetic contract"), the 1-D TMA
// bulk-load of a tile of packed records into shared memory, and small block-level utilities.
// This file shares nothing with oracle/ (the CPU checker).
#pragma once

#include <cuda_runtime.h>
#include <float.h>
#include <stdint.h>

namespace psl {

constexpr int kTile = 1024;              // records per tile: the unit one CTA stages, ranks and writes at a time
constexpr int kThreads = 256;            // threads per CTA in the tile kernels
constexpr int kWarps = kThreads / 32;    // 8
constexpr int kRounds = kTile / kThreads;  // 4 records per thread
constexpr int kWarpSpan = kTile / kWarps;  // 128 consecutive records owned by one warp
constexpr int kMaxSegments = 592;        // most CTAs (= table columns) one partition launch uses: 148 SMs x 4
constexpr int kRecWords = 7;             // 28-byte packed record
constexpr int kRecBytes = 28;
constexpr int kMaxBuckets = 2048;        // most buckets one partition pass handles
constexpr uint32_t kNone = 0xFFFFFFFFu;

enum : int { C_SURVIVOR = 0, C_INVALID = 1, C_OUTSIDE = 2, C_ROI = 3, C_JAW = 4, C_ZERO = 5 };

struct DevGrid {
    int32_t n_types, ebin_mode, n_ebins;
    float e_min, dE;
    const float* e_edges;  // DEVICE, n_ebins+1 (edge mode)
    int32_t has_pos, n_xbins, n_ybins, ix0, iy0;
    float inv_dx, inv_dy;
    uint32_t n_pos;
    uint32_t apr;                  // PSL_APR: azimuthal particle redistribution before binning (INDEX mode)
    unsigned long long apr_seed;
};

// counter-based generator (reading S2): the output function of splitmix64 applied to (seed, a), then to (that, b)
constexpr unsigned long long kGamma64 = 0x9E3779B97F4A7C15ull;

__host__ __device__ __forceinline__ unsigned long long mix64(unsigned long long z)
{
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
    return z ^ (z >> 31);
}
__host__ __device__ __forceinline__ uint32_t rng32(unsigned long long seed, unsigned long long a, unsigned long long b)
{
    const unsigned long long h = mix64(seed + kGamma64 * (a + 1ull));
    return (uint32_t)(mix64(h + kGamma64 * (b + 1ull)) >> 32);
}
__host__ __device__ __forceinline__ uint32_t below(uint32_t r, uint32_t n)
{
    return (uint32_t)(((unsigned long long)r * (unsigned long long)n) >> 32);
}

struct DevBeam {
    int32_t has_beam, has_jaws;
    float X1, X2, Y1, Y2;  // aperture at the jaw planes
    float dzJx, dzJy;      // z_jaw - z_plane
    int32_t has_map;
    const float* fluence;  // DEVICE
    int32_t map_nx, map_ny, px0, py0;
    float inv_mdx, inv_mdy;
    float dzM;             // z_map - z_plane
    float mu;
    uint32_t drop_zero;
    uint32_t out_proj;
};

struct ChunkDesc {  // 24 bytes, one per psl_load_chunk; tiles never straddle chunks
    const uint8_t* ptr;    // DEVICE, first record of the chunk
    uint32_t first_index;  // load-order index of that record
    uint32_t n_records;
    uint32_t tile0;        // global id of the chunk's first tile
    uint32_t pad;
};

struct TileDesc {  // 16 bytes
    const void* ptr;       // first record of the tile
    uint32_t first_index;  // load-order index of that record
    uint32_t count;        // 1..kTile
};

struct SegStats {  // 48 bytes, one per table column (= one CTA's segment), reduced in a fixed order
    uint32_t n_invalid, n_outside, n_jaw, n_zero, n_surv, pad;
    double sum_in, sum_idx, sum_out;
};

struct Rec {
    int32_t type;
    float E, x, y, u, v, wt;
};

// ------------------------------------------------------------------------------------------------
// per-record arithmetic.  Every floating-point operation is an explicit round-to-nearest intrinsic so
// that no FMA can be formed (the TU is also compiled with -fmad=false).
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ bool is_finite(float a) { return fabsf(a) <= FLT_MAX; }

// q = 1 - (u*u + v*v)   (records carry direction; the third cosine follows from the other two)
__device__ __forceinline__ float q_of(float u, float v)
{
    return __fsub_rn(1.0f, __fadd_rn(__fmul_rn(u, u), __fmul_rn(v, v)));
}

__device__ __forceinline__ bool rec_valid(const Rec& r, float q)
{
    return ((uint32_t)r.type <= 2u) && is_finite(r.E) && is_finite(r.x) && is_finite(r.y) && is_finite(r.u) &&
           is_finite(r.v) && is_finite(r.wt) && (r.E > 0.0f) && (q > 0.0f);
}

// Energy bin: linear = floor((E - e_min)/dE) clamped; edge table = number of interior edges <= E.
__device__ __forceinline__ int energy_bin(const DevGrid& g, float E, const float* s_edges)
{
    if (g.ebin_mode == 0) {
        float t = __fdiv_rn(__fsub_rn(E, g.e_min), g.dE);
        if (t < 0.0f) return 0;
        if (t >= (float)g.n_ebins) return g.n_ebins - 1;
        return (int)floorf(t);
    }
    int lo = 1, hi = g.n_ebins;  // first k in [1, n_ebins) with edges[k] > E
    while (lo < hi) {
        int mid = (lo + hi) >> 1;
        if (s_edges[mid] <= E) lo = mid + 1; else hi = mid;
    }
    return lo - 1;
}

// Bin of a coordinate on a grid whose bin k covers [k*d, (k+1)*d) in absolute coordinates and whose first
// bin is i0 ("[x_i, x_i+dx]"; also used for fluence-map pixels).
__device__ __forceinline__ bool axis_bin(float x, float inv_d, int i0, int n, int& out)
{
    float f = floorf(__fmul_rn(x, inv_d));
    bool ok = (f >= (float)i0) && (f < (float)(i0 + n));
    out = ok ? ((int)f - i0) : 0;
    return ok;
}

__device__ __forceinline__ int type_division(const DevGrid& g, int type) { return (g.n_types == 2 && type > 1) ? 1 : type; }

// Slopes dx/dz, dy/dz of the ray: t = 1/w, tx = u*t, ty = v*t with w = sqrt(q).
__device__ __forceinline__ void slopes(float u, float v, float q, float& w, float& tx, float& ty)
{
    w = __fsqrt_rn(q);
    float t = __fdiv_rn(1.0f, w);
    tx = __fmul_rn(u, t);
    ty = __fmul_rn(v, t);
}

// Jaw accept/reject: half-open aperture at one thin plane per jaw pair.
__device__ __forceinline__ bool jaw_pass(const DevBeam& b, float x, float y, float tx, float ty)
{
    float xj = __fadd_rn(x, __fmul_rn(tx, b.dzJx));
    float yj = __fadd_rn(y, __fmul_rn(ty, b.dzJy));
    return (b.X1 <= xj) && (xj < b.X2) && (b.Y1 <= yj) && (yj < b.Y2);
}

// Final weight: containing pixel of the map at z_map, 0 outside, (wt*F)*mu.
__device__ __forceinline__ float final_weight(const DevBeam& b, float wt, float xm, float ym)
{
    if (!b.has_beam) return wt;
    if (!b.has_map) return __fmul_rn(wt, b.mu);
    int px, py;
    float F = 0.0f;
    if (axis_bin(xm, b.inv_mdx, b.px0, b.map_nx, px) && axis_bin(ym, b.inv_mdy, b.py0, b.map_ny, py))
        F = __ldg(b.fluence + (size_t)py * (size_t)b.map_nx + (size_t)px);
    return __fmul_rn(__fmul_rn(wt, F), b.mu);
}

// Azimuthal particle redistribution: record `index` of the load order turns by 2 pi r / 2^32 about the
// beam axis, r = rng32(seed, index, 0) -- position and direction by the same angle.  cos and sin in fp32 by fixed
// operations (reading S7): nearest quarter turn, remainder |a| <= pi/4, Taylor polynomials in Horner form.
__device__ __forceinline__ void apr_cos_sin(uint32_t r, float& c, float& s)
{
    const uint32_t k = (uint32_t)(((unsigned long long)r + 0x20000000ull) >> 30);
    const int32_t rem = (int32_t)(r - (k << 30));
    const float a = __fmul_rn((float)rem, 1.46291807926715968e-9f);  // pi / 2^31
    const float a2 = __fmul_rn(a, a);
    float t = __fmul_rn(2.75573192239858925e-6f, a2);
    t = __fmul_rn(__fadd_rn(t, -1.98412698412698413e-4f), a2);
    t = __fmul_rn(__fadd_rn(t, 8.33333333333333322e-3f), a2);
    t = __fmul_rn(__fadd_rn(t, -1.66666666666666657e-1f), a2);
    const float sn = __fadd_rn(a, __fmul_rn(t, a));
    float q = __fmul_rn(2.48015873015873016e-5f, a2);
    q = __fmul_rn(__fadd_rn(q, -1.38888888888888894e-3f), a2);
    q = __fmul_rn(__fadd_rn(q, 4.16666666666666644e-2f), a2);
    q = __fmul_rn(__fadd_rn(q, -0.5f), a2);
    const float cs = __fadd_rn(1.0f, q);
    const uint32_t kk = k & 3u;
    c = kk == 0 ? cs : (kk == 1 ? -sn : (kk == 2 ? -cs : sn));
    s = kk == 0 ? sn : (kk == 1 ? cs : (kk == 2 ? -sn : -cs));
}

__device__ __forceinline__ void apr_apply(unsigned long long seed, uint32_t index, Rec& r)
{
    float c, s;
    apr_cos_sin(rng32(seed, index, 0), c, s);
    const float x = __fsub_rn(__fmul_rn(r.x, c), __fmul_rn(r.y, s));
    const float y = __fadd_rn(__fmul_rn(r.x, s), __fmul_rn(r.y, c));
    const float u = __fsub_rn(__fmul_rn(r.u, c), __fmul_rn(r.v, s));
    const float v = __fadd_rn(__fmul_rn(r.u, s), __fmul_rn(r.v, c));
    r.x = x; r.y = y; r.u = u; r.v = v;
}

// Steps 1-4 (+6, +8 when a beam is given) for one raw record.  Returns the class; key is valid for every
// class except C_INVALID / C_OUTSIDE.  Straight-line code (selects, no data-dependent branches) so that the
// records a thread owns are classified in an interleaved instruction stream.  Compile-time features:
//   POS   the grid has position bins (a3)            EDGES  energy bins from the edge table (a2)
//   BEAM  0: nothing rejects a valid in-grid record  1: jaws only (a6)  2: run-time jaws / PSL_DROP_ZERO_WEIGHT
template <bool POS, bool EDGES, int BEAM>
__device__ __forceinline__ int classify(const DevGrid& g, const DevBeam& b, const Rec& r, const float* s_edges, uint32_t& key)
{
    const float q = q_of(r.u, r.v);
    // q > 0 already implies finite u and v (an infinite or NaN cosine makes q -inf or NaN)
    const bool valid = ((uint32_t)r.type <= 2u) & is_finite(r.E) & is_finite(r.x) & is_finite(r.y) & is_finite(r.wt) &
                       (r.E > 0.0f) & (q > 0.0f);
    int ix = 0, iy = 0;
    bool inside = true;
    if (POS) {
        const bool okx = axis_bin(r.x, g.inv_dx, g.ix0, g.n_xbins, ix);
        const bool oky = axis_bin(r.y, g.inv_dy, g.iy0, g.n_ybins, iy);
        inside = okx & oky;
    }
    int ie;
    if (!EDGES) {
        // floor((E - e_min) / dE) clamped into [0, n_ebins - 1]; one IEEE division
        float t = floorf(__fdiv_rn(__fsub_rn(r.E, g.e_min), g.dE));
        ie = (int)fminf(fmaxf(t, 0.0f), (float)(g.n_ebins - 1));
    } else {
        int lo = 1, hi = g.n_ebins;  // first k in [1, n_ebins) with edges[k] > E
        while (lo < hi) {
            int mid = (lo + hi) >> 1;
            if (s_edges[mid] <= r.E) lo = mid + 1; else hi = mid;
        }
        ie = lo - 1;
    }
    const int td = min(r.type, g.n_types - 1);  // n_types == 2 merges electrons and positrons
    uint32_t k = (uint32_t)(td * g.n_ebins + ie);
    if (POS) k = k * g.n_pos + (uint32_t)(iy * g.n_xbins + ix);
    key = k;
    int cls = C_SURVIVOR;
    if (BEAM == 1) {
        float w, tx, ty;
        slopes(r.u, r.v, q, w, tx, ty);
        if (!jaw_pass(b, r.x, r.y, tx, ty)) cls = C_JAW;
    }
    if (BEAM == 2) {
        if (valid && inside && (b.has_jaws || b.drop_zero)) {
            float w, tx, ty;
            slopes(r.u, r.v, q, w, tx, ty);
            if (b.has_jaws && !jaw_pass(b, r.x, r.y, tx, ty)) {
                cls = C_JAW;
            } else if (b.drop_zero) {
                float xm = __fadd_rn(r.x, __fmul_rn(tx, b.dzM));
                float ym = __fadd_rn(r.y, __fmul_rn(ty, b.dzM));
                if (final_weight(b, r.wt, xm, ym) == 0.0f) cls = C_ZERO;
            }
        }
    }
    if (!inside) cls = C_OUTSIDE;
    if (!valid) cls = C_INVALID;
    return cls;
}

// which BEAM variant of classify() a beam needs
__host__ __device__ inline int beam_variant(const DevBeam& b)
{
    if (!b.has_beam || (!b.has_jaws && !b.drop_zero)) return 0;
    return b.drop_zero ? 2 : 1;
}

// ------------------------------------------------------------------------------------------------
// shared-memory tile of packed records: 1-D TMA bulk copy (cp.async.bulk, SASS UBLKCP) completing on an
// mbarrier; scalar fallback when the source is not 16-byte aligned or the byte count is not a multiple
// of 16 (only the ragged last tile of a chunk).
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
// Programmatic dependent launch: a kernel launched with programmaticStreamSerializationAllowed may start while
// the kernel before it in the stream still runs; griddep_wait() returns once that kernel has finished and its
// writes are visible (at once when the launch carried no such attribute).  griddep_launch() in the earlier kernel
// lets the later one take SMs as they free up.
__device__ __forceinline__ void griddep_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void griddep_launch() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

__device__ __forceinline__ void mbar_fence_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t phase)
{
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "WAIT_%=:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra DONE_%=;\n\t"
        "bra WAIT_%=;\n\t"
        "DONE_%=:\n\t}" ::"r"(smem_u32(bar)), "r"(phase) : "memory");
}
__device__ __forceinline__ void tma_load_1d(void* smem_dst, const void* gsrc, uint32_t bytes, uint64_t* bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     smem_u32(smem_dst)),
                 "l"(gsrc), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}

// the same copy with an L2 evict-first policy: a read-once stream must not push half-filled output lines
// out of L2 (the INDEX passes rely on L2 to merge their 32-byte sector writes into whole lines)
__device__ __forceinline__ void tma_load_1d_stream(void* smem_dst, const void* gsrc, uint32_t bytes, uint64_t* bar)
{
    uint64_t pol;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;" ::"r"(
            smem_u32(smem_dst)),
        "l"(gsrc), "r"(bytes), "r"(smem_u32(bar)), "l"(pol)
        : "memory");
}

// Bring `bytes` (a multiple of 4) from global into s_dst.  Must be called by all threads of the CTA; `bar`
// must have been initialised (count 1) and made visible with a __syncthreads.  Ends with the data visible
// to every thread.
__device__ __forceinline__ void load_tile_bytes(uint32_t* s_dst, const void* gsrc, uint32_t bytes, uint64_t* bar,
                                                uint32_t phase)
{
    bool bulk = ((reinterpret_cast<uintptr_t>(gsrc) & 15u) == 0) && ((bytes & 15u) == 0) && bytes > 0;
    if (bulk) {
        if (threadIdx.x == 0) {
            mbar_expect_tx(bar, bytes);
            tma_load_1d(s_dst, gsrc, bytes, bar);
        }
        mbar_wait(bar, phase);
    } else {
        const uint32_t* g = reinterpret_cast<const uint32_t*>(gsrc);
        for (uint32_t i = threadIdx.x; i < bytes / 4; i += blockDim.x) s_dst[i] = __ldg(g + i);
        __syncthreads();
    }
}

__device__ __forceinline__ Rec rec_from_smem(const uint32_t* s_raw, int idx)
{
    const uint32_t* p = s_raw + idx * kRecWords;  // stride 7 words across lanes: conflict-free
    Rec r;
    r.type = (int32_t)p[0];
    r.E = __uint_as_float(p[1]);
    r.x = __uint_as_float(p[2]);
    r.y = __uint_as_float(p[3]);
    r.u = __uint_as_float(p[4]);
    r.v = __uint_as_float(p[5]);
    r.wt = __uint_as_float(p[6]);
    return r;
}

// ------------------------------------------------------------------------------------------------
// block utilities (kThreads threads)
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t lane_id() { return threadIdx.x & 31u; }
__device__ __forceinline__ uint32_t warp_id() { return threadIdx.x >> 5; }
__device__ __forceinline__ uint32_t lanemask_lt() { return (1u << lane_id()) - 1u; }

__device__ __forceinline__ uint32_t warp_incl_scan(uint32_t v)
{
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        uint32_t n = __shfl_up_sync(0xFFFFFFFFu, v, o);
        if ((int)lane_id() >= o) v += n;
    }
    return v;
}

// exclusive scan of one value per thread over the CTA; s_warp holds >= kWarps+1 words; returns the
// exclusive prefix, *total receives the CTA sum.  Contains two __syncthreads.
__device__ __forceinline__ uint32_t block_excl_scan(uint32_t v, uint32_t* s_warp, uint32_t* total)
{
    uint32_t inc = warp_incl_scan(v);
    if (lane_id() == 31) s_warp[warp_id()] = inc;
    __syncthreads();
    if (warp_id() == 0) {
        uint32_t w = lane_id() < (uint32_t)(blockDim.x >> 5) ? s_warp[lane_id()] : 0u;
        uint32_t wi = warp_incl_scan(w);
        if (lane_id() < (uint32_t)(blockDim.x >> 5)) s_warp[lane_id()] = wi - w;
        if (lane_id() == 31) s_warp[32] = wi;
    }
    __syncthreads();
    uint32_t r = s_warp[warp_id()] + inc - v;
    *total = s_warp[32];
    return r;
}

__device__ __forceinline__ double warp_sum_double(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xFFFFFFFFu, v, o);
    return v;
}

// Stable rank of a record inside its warp's slice of the tile: records of one warp arrive in rounds of 32 consecutive
// records; `cnt` is the warp's private running count per bucket (uint16 per bucket, zeroed per tile).  Lanes with
// bucket == kNone take no part.  Must be called by all 32 lanes.  Ranks WITHOUT MATCH.ANY.  Measured on B200: one
// __match_any_sync costs ~2 cycles per distinct value on a unit the whole SM shares -- ~58 cycles per warp instruction
// with ~1000 buckets, 1.8 cycles per record, a third of an INDEX pass.  Here the lanes of a round CLAIM their bucket
// instead: the top 5 bits of the warp's private 16-bit counter take the lane id (the low 11 bits keep the count; a warp
// ranks at most 2047 records of a bucket per tile), one store wins, every lane reads the word back; a lane that reads
// its own id has the bucket to itself or won it.  Losers exist only when lanes of the round share a bucket: each
// loser ORs its lane bit into its winner's word of `grp` (32 words per warp, all zero between calls), and every lane
// reads its winner's word: the peer mask of all colliding buckets at once (config 4: pass B 3.40 -> 3.04 ms against
// resolving one bucket per ballot).  The counters must be read through kRankCountMask by whoever sums them.
constexpr uint32_t kRankCountBits = 11;
constexpr uint32_t kRankCountMask = (1u << kRankCountBits) - 1u;
constexpr uint32_t kRankCountMask2 = kRankCountMask | (kRankCountMask << 16);  // two packed counters

template <int R>
__device__ __forceinline__ void warp_rank_claim(const uint32_t (&bucket)[R], uint32_t (&rank)[R], uint16_t* cnt, uint32_t* grp)
{
    const uint32_t lane = lane_id(), lt = lanemask_lt();
#pragma unroll
    for (int r = 0; r < R; ++r) {
        const uint32_t b = bucket[r];
        const bool act = b != kNone;
        const uint32_t base = act ? ((uint32_t)cnt[b] & kRankCountMask) : 0u;
        __syncwarp();
        if (act) cnt[b] = (uint16_t)(base | (lane << kRankCountBits));
        __syncwarp();
        const uint32_t win = act ? ((uint32_t)cnt[b] >> kRankCountBits) : lane;
        uint32_t peers = 1u << lane;
        if (__any_sync(0xFFFFFFFFu, win != lane)) {
            if (win != lane) atomicOr(&grp[win], 1u << lane);
            __syncwarp();
            const uint32_t m = grp[win];
            if (m != 0u) peers = m | (1u << win);
            __syncwarp();
            if (win == lane && m != 0u) grp[lane] = 0u;
        }
        const uint32_t before = __popc(peers & lt);
        if (act && before == 0u) cnt[b] = (uint16_t)(base + __popc(peers));  // the lowest peer; claim bits cleared
        __syncwarp();
        rank[r] = base + before;
    }
}

// The same contract with MATCH.ANY: for the ONTHEFLY kernels.  Their <= 2048 (type, energy) keys follow the energy
// spectrum, a round of 32 records holds ~20 colliding pairs, and MATCH.ANY's cost falls with the number of distinct
// values while the claim loop's grows with the number of collisions (measured at config 2: scatter 0.203 ms with
// MATCH.ANY, 0.222 ms with claims).  Counters are plain counts here (no claim bits).
template <int R>
__device__ __forceinline__ void warp_rank_match(const uint32_t (&bucket)[R], uint32_t (&rank)[R], uint16_t* cnt)
{
    uint32_t peers[R];
#pragma unroll
    for (int r = 0; r < R; ++r) peers[r] = __match_any_sync(0xFFFFFFFFu, bucket[r]);
    const uint32_t lt = lanemask_lt();
#pragma unroll
    for (int r = 0; r < R; ++r) {
        const bool act = bucket[r] != kNone;
        const uint32_t before = __popc(peers[r] & lt);
        const uint32_t base = act ? cnt[bucket[r]] : 0u;  // every peer reads the same word
        __syncwarp();
        if (act && before == 0u) cnt[bucket[r]] = (uint16_t)(base + __popc(peers[r]));
        __syncwarp();
        rank[r] = base + before;
    }
}

// one 32-byte record in ONE store request (STG.E.256, sm_100+); dst must be 32-byte aligned
__device__ __forceinline__ void stg_record(uint4* dst, const uint4& a, const uint4& b)
{
    asm volatile("st.global.v8.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};" ::"l"(dst), "r"(a.x), "r"(a.y), "r"(a.z), "r"(a.w),
                 "r"(b.x), "r"(b.y), "r"(b.z), "r"(b.w));
}

}  // namespace psl
