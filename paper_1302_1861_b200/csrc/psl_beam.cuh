// psl_beam.cuh -- per-beam batches from the pre-sorted PSL index (paper method 3).
//
// The index stores every valid in-grid record sorted by key = ((t*N_E + ie)*N_y + iy)*N_x + ix, so the
// records of one (type, energy, row iy) and columns rx0..rx1 are ONE contiguous range.  The host turns the
// beam's ROI into that list of row segments from its copy of offsets[] (no device work, no record is read):
// position bins outside the ROI are skipped without touching their records.
// The kernel below walks the concatenated segments ("virtual" order = key order), applies the jaw test
// (PAPER.md:55), the fluence-map weight and MU weight, and compacts the survivors
// stably: virtual order IS the required output order, so the batch layout is a plain stream compaction.
// The global slot of a tile's first survivor comes from a decoupled look-back over tile aggregates -- an
// ordered prefix sum, so the result is deterministic.
#pragma once

#include "psl_device.cuh"
#include "psl_partition.cuh"

namespace psl {

struct SegTable {
    const uint32_t* vstart;   // [n_seg+1] virtual index of each segment's first record; vstart[n_seg] = M
    const uint32_t* src;      // [n_seg] slot of that record in the index
    const uint32_t* keybase;  // [n_seg] key of column 0 of the segment's row
    uint32_t n_seg;
    uint32_t M;               // records selected by the ROI
};

struct IdxIn {
    const uint4* aos;  // the index: 32-byte keyed records {key, E, x, y, u, v, wt, src} sorted by key
};

struct BeamTileStats {  // 16 bytes
    uint32_t n_zero, n_surv;
    double sum_out;
};

constexpr unsigned long long kFlagAggregate = 1ull << 62;
constexpr unsigned long long kFlagInclusive = 2ull << 62;
constexpr unsigned long long kFlagMask = 3ull << 62;

__device__ __forceinline__ unsigned long long ld_state(const unsigned long long* p)
{
    return *reinterpret_cast<const volatile unsigned long long*>(p);
}

// last s in [lo, hi] with vstart[s] <= v  (vstart[lo] <= v guaranteed)
__device__ __forceinline__ uint32_t seg_of(const uint32_t* __restrict__ vstart, uint32_t lo, uint32_t hi, uint32_t v)
{
    while (lo < hi) {
        uint32_t mid = lo + ((hi - lo + 1) >> 1);
        if (__ldg(vstart + mid) <= v) lo = mid; else hi = mid - 1;
    }
    return lo;
}

// one 32-byte keyed record in ONE request (LDG.E.256, sm_100+): the two 16-byte halves as separate loads make every
// warp touch each sector twice
__device__ __forceinline__ void ldg_record(const uint4* p, uint4& a, uint4& b)
{
    asm volatile("ld.global.nc.v8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                 : "=r"(a.x), "=r"(a.y), "=r"(a.z), "=r"(a.w), "=r"(b.x), "=r"(b.y), "=r"(b.z), "=r"(b.w)
                 : "l"(p));
}

// the same by a whole warp, 32 probes per round: 3 rounds of dependent loads instead of 13 at 4608 segments (the
// one-thread search of the tile's first and last segment was close to half of a tile's 10 us)
__device__ __forceinline__ uint32_t seg_of_warp(const uint32_t* __restrict__ vstart, uint32_t lo, uint32_t hi, uint32_t v)
{
    while (lo < hi) {
        const uint32_t step = (hi - lo) / 32u + 1u;
        const uint32_t idx = lo + (lane_id() + 1u) * step;
        const bool le = idx <= hi && __ldg(vstart + idx) <= v;
        const uint32_t c = __popc(__ballot_sync(0xFFFFFFFFu, le));  // vstart is non-decreasing: the lanes that pass are a prefix
        const uint32_t nlo = lo + c * step;
        hi = min(hi, nlo + step - 1u);
        lo = nlo;
    }
    return lo;
}

// 4 records per thread, 4 CTAs per SM (64 registers): the kernel is a chain of dependent latencies per tile (ticket ->
// segment search -> loads -> look-back -> stores), so what pays is warps in flight -- 8 records per thread at 2 CTAs per
// SM (122 registers) took 11.5 ms for config 5's nine beams, this shape 9.4 ms
constexpr int kBeamRounds = 4;                         // index records per thread
constexpr int kBeamOcc = 4;                            // CTAs per SM
constexpr int kBeamTile = kBeamRounds * kThreads;      // 1024 index records per CTA
constexpr int kBeamArrays = 12;  // E x y u v w wt xp yp src key + spare

__global__ void __launch_bounds__(kThreads, kBeamOcc) k_beam_compact(SegTable seg, IdxIn in, const __grid_constant__ DevGrid g,
                                                             const __grid_constant__ DevBeam bm, SoAOut out,
                                                             uint32_t* __restrict__ out_key,
                                                             unsigned long long* __restrict__ tile_state,
                                                             uint32_t* __restrict__ tile_counter,
                                                             BeamTileStats* __restrict__ bstats,
                                                             uint32_t* __restrict__ n_surv_out)
{
    // Two phases, no shared-memory staging: (1) every thread loads its 8 records of the tile (16 independent
    // 16-byte loads in flight), applies jaws / map / MU weight and keeps the results in registers;
    // (2) after the tile's first output slot is known (look-back), survivors are stored straight from
    // registers -- compaction is monotonic, so consecutive kept lanes write consecutive slots.
    __shared__ uint32_t s_cnt[kBeamRounds * kWarps];  // survivors per (round, warp), then their exclusive prefix
    __shared__ uint32_t s_ctl[5];                     // tile, seg_first, seg_last, first output slot, survivors
    __shared__ double s_d[kWarps];
    __shared__ uint32_t s_z[kWarps];

    const uint32_t w = warp_id();
    if (threadIdx.x == 0) s_ctl[0] = atomicAdd(tile_counter, 1u);  // tiles are handed out in order
    __syncthreads();
    const uint32_t tile = s_ctl[0];
    const uint32_t v0 = tile * kBeamTile;
    const uint32_t cnt = min((uint32_t)kBeamTile, seg.M - v0);
    if (w < 2) {  // warp 0: the segment of the tile's first record; warp 1: of its last
        const uint32_t sg = seg_of_warp(seg.vstart, 0, seg.n_seg - 1, w == 0 ? v0 : v0 + cnt - 1);
        if (lane_id() == 0) s_ctl[1 + w] = sg;
    }
    __syncthreads();
    const uint32_t s_first = s_ctl[1], s_last = s_ctl[2];

    uint4 ra[kBeamRounds], rb[kBeamRounds];
    bool have[kBeamRounds];
#pragma unroll
    for (int r = 0; r < kBeamRounds; ++r) {
        const uint32_t lv = r * kThreads + threadIdx.x;
        have[r] = lv < cnt;
        ra[r] = make_uint4(0, 0, 0, 0);
        rb[r] = make_uint4(0, 0, 0, 0);
        if (have[r]) {
            const uint32_t vv = v0 + lv;
            const uint32_t sg = s_first == s_last ? s_first : seg_of(seg.vstart, s_first, s_last, vv);
            const uint32_t p = __ldg(seg.src + sg) + (vv - __ldg(seg.vstart + sg));
            ldg_record(in.aos + 2 * (size_t)p, ra[r], rb[r]);
        }
    }
    float wz[kBeamRounds], wt[kBeamRounds], xm[kBeamRounds], ym[kBeamRounds];
    uint32_t pre[kBeamRounds];
    uint32_t keepbits = 0, n_zero = 0;
    double sum_out = 0.0;
#pragma unroll
    for (int r = 0; r < kBeamRounds; ++r) {
        const float x = __uint_as_float(ra[r].z), y = __uint_as_float(ra[r].w);
        const float u = __uint_as_float(rb[r].x), v = __uint_as_float(rb[r].y);
        const float q = q_of(u, v);
        float tx, ty;
        slopes(u, v, q, wz[r], tx, ty);
        bool keep = have[r] && (!(bm.has_jaws) || jaw_pass(bm, x, y, tx, ty));
        xm[r] = __fadd_rn(x, __fmul_rn(tx, bm.dzM));
        ym[r] = __fadd_rn(y, __fmul_rn(ty, bm.dzM));
        wt[r] = have[r] ? final_weight(bm, __uint_as_float(rb[r].z), xm[r], ym[r]) : 0.0f;
        if (keep && bm.drop_zero && wt[r] == 0.0f) {
            keep = false;
            n_zero += 1;
        }
        const uint32_t ballot = __ballot_sync(0xFFFFFFFFu, keep);
        if (lane_id() == 0) s_cnt[r * kWarps + w] = __popc(ballot);
        pre[r] = __popc(ballot & lanemask_lt());
        if (keep) {
            keepbits |= 1u << r;
            sum_out += (double)wt[r];
        }
    }
    __syncthreads();

    // warp 0: exclusive prefix of the (round, warp) counts, then the decoupled look-back over tile aggregates
    if (w == 0) {
        constexpr int kPer = kBeamRounds * kWarps / 32;  // counts per lane
        uint32_t c[kPer], sum = 0;
#pragma unroll
        for (int k = 0; k < kPer; ++k) { c[k] = s_cnt[kPer * lane_id() + k]; sum += c[k]; }
        const uint32_t inc = warp_incl_scan(sum);
        uint32_t run = inc - sum;
#pragma unroll
        for (int k = 0; k < kPer; ++k) { s_cnt[kPer * lane_id() + k] = run; run += c[k]; }
        const uint32_t total = __shfl_sync(0xFFFFFFFFu, inc, 31);
        uint32_t excl = 0;
        if (tile == 0) {
            if (lane_id() == 0) atomicExch(&tile_state[0], kFlagInclusive | (unsigned long long)total);
        } else {
            if (lane_id() == 0) atomicExch(&tile_state[tile], kFlagAggregate | (unsigned long long)total);
            int look = (int)tile - 1;
            while (true) {
                int idx = look - (int)lane_id();
                unsigned long long st;
                do {
                    st = idx >= 0 ? ld_state(&tile_state[idx]) : kFlagInclusive;
                } while (__any_sync(0xFFFFFFFFu, (st & kFlagMask) == 0ull));
                uint32_t incl = __ballot_sync(0xFFFFFFFFu, (st & kFlagMask) == kFlagInclusive);
                uint32_t val = (uint32_t)(st & 0xFFFFFFFFull);
                if (incl) {
                    int first = __ffs(incl) - 1;
                    val = ((int)lane_id() <= first) ? val : 0u;
                    excl += __reduce_add_sync(0xFFFFFFFFu, val);
                    break;
                }
                excl += __reduce_add_sync(0xFFFFFFFFu, val);
                look -= 32;
            }
            if (lane_id() == 0) atomicExch(&tile_state[tile], kFlagInclusive | (unsigned long long)(excl + total));
        }
        if (lane_id() == 0) {
            s_ctl[3] = excl;
            s_ctl[4] = total;
            if (v0 + cnt == seg.M) *n_surv_out = excl + total;  // last tile
        }
    }
    sum_out = warp_sum_double(sum_out);
    n_zero = __reduce_add_sync(0xFFFFFFFFu, n_zero);
    if (lane_id() == 0) {
        s_d[w] = sum_out;
        s_z[w] = n_zero;
    }
    __syncthreads();
    const uint32_t gbase = s_ctl[3];

#pragma unroll
    for (int r = 0; r < kBeamRounds; ++r) {
        if (keepbits & (1u << r)) {
            const size_t d = (size_t)gbase + s_cnt[r * kWarps + w] + pre[r];
            out.E[d] = __uint_as_float(ra[r].y);
            out.x[d] = __uint_as_float(ra[r].z);
            out.y[d] = __uint_as_float(ra[r].w);
            out.u[d] = __uint_as_float(rb[r].x);
            out.v[d] = __uint_as_float(rb[r].y);
            out.w[d] = wz[r];
            out.wt[d] = wt[r];
            if (bm.out_proj) {
                out.xp[d] = xm[r];
                out.yp[d] = ym[r];
            }
            out.src[d] = rb[r].w;
            out_key[d] = ra[r].x;
        }
    }
    if (threadIdx.x == 0) {
        BeamTileStats bs = {0, s_ctl[4], 0.0};
        for (int k = 0; k < kWarps; ++k) {
            bs.sum_out += s_d[k];
            bs.n_zero += s_z[k];
        }
        bstats[tile] = bs;
    }
}

struct DevBeamStats {
    unsigned long long n_zero, n_surv;
    double sum_out;
};

__global__ void __launch_bounds__(1024) k_reduce_beam_stats(const BeamTileStats* __restrict__ ts, uint32_t n_tiles,
                                                            DevBeamStats* __restrict__ out)
{
    __shared__ unsigned long long s_n[32][2];
    __shared__ double s_d[32];
    unsigned long long nz = 0, ns = 0;
    double d = 0.0;
    for (uint32_t t = threadIdx.x; t < n_tiles; t += 1024) {
        BeamTileStats x = ts[t];
        nz += x.n_zero;
        ns += x.n_surv;
        d += x.sum_out;
    }
    for (int o = 16; o > 0; o >>= 1) {
        nz += __shfl_xor_sync(0xFFFFFFFFu, nz, o);
        ns += __shfl_xor_sync(0xFFFFFFFFu, ns, o);
    }
    d = warp_sum_double(d);
    if (lane_id() == 0) {
        s_n[warp_id()][0] = nz;
        s_n[warp_id()][1] = ns;
        s_d[warp_id()] = d;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        DevBeamStats r = {0, 0, 0.0};
        for (int k = 0; k < 32; ++k) {
            r.n_zero += s_n[k][0];
            r.n_surv += s_n[k][1];
            r.sum_out += s_d[k];
        }
        *out = r;
    }
}

}  // namespace psl
