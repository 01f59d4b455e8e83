// psl_plan.cuh -- from the PSL index to transport launches (sec. 2.3.3).
//
//   budgets   P_ij = N_sim * P_j / N_total,  E_ij = N_sim * E_j / N_total from the index's counts[]
//   sampling  the launch list of one (type, energy) division: round-robin over the selected PSLs, rr_group particles
//             from each per round, random start with wrap-around, random field per particle
//   emit      gather the listed index records, each against ITS field: jaw test, fluence / MU weight (PAPER.md:55-57,
//             :99), collimator / gantry / couch rotation and projection to the phantom surface, stable
//             compaction into transport-ready SoA arrays
// The generator is counter-based (reading S2: splitmix64's output function on (seed, PSL, counter)), so the
// list is a pure function of the plan: bit-identical to the oracle's sequential reading loop.
#pragma once

#include "psl_beam.cuh"

namespace psl {

constexpr int kMaxPlanBeams = 32;
// the fields' ROI bin rectangles (inclusive; a field without ROI covers the grid) and the box around all of them
struct PlanSel {
    int32_t sel[kMaxPlanBeams][4];
    uint32_t n_beams;
    int32_t bx0, bx1, by0, by1;
};

__device__ __forceinline__ uint32_t plan_mask(const PlanSel& s, int ix, int iy)
{
    uint32_t m = 0;
    for (uint32_t i = 0; i < s.n_beams; ++i)
        if (s.sel[i][0] <= ix && ix <= s.sel[i][1] && s.sel[i][2] <= iy && iy <= s.sel[i][3]) m |= 1u << i;
    return m;
}

// N_total^psl = sum over fields and over each field's selected PSLs of the PSL's particle count
__global__ void __launch_bounds__(256) k_plan_total(const uint32_t* __restrict__ counts, uint32_t K, uint32_t n_pos,
                                                    uint32_t n_xbins, const __grid_constant__ PlanSel sel,
                                                    unsigned long long* __restrict__ total)
{
    unsigned long long acc = 0;
    for (uint32_t k = blockIdx.x * blockDim.x + threadIdx.x; k < K; k += gridDim.x * blockDim.x) {
        const uint32_t pos = k % n_pos;
        acc += (unsigned long long)__popc(plan_mask(sel, (int)(pos % n_xbins), (int)(pos / n_xbins))) * counts[k];
    }
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xFFFFFFFFu, acc, o);
    if (lane_id() == 0 && acc != 0) atomicAdd(total, acc);  // integers: the sum does not depend on the order
}

// one CTA per (type, energy) division: budget[k], mask[k] for its PSLs, the length of its launch list and the number
// of round-robin rounds it takes
__global__ void __launch_bounds__(256) k_plan_budgets(const uint32_t* __restrict__ counts, uint32_t n_pos, uint32_t n_xbins,
                                                      const __grid_constant__ PlanSel sel, unsigned long long n_simulate,
                                                      const unsigned long long* __restrict__ total_ptr, uint32_t rr_group,
                                                      uint32_t* __restrict__ budget, uint32_t* __restrict__ mask,
                                                      unsigned long long* __restrict__ list_len,
                                                      unsigned long long* __restrict__ rounds)
{
    __shared__ unsigned long long s_len[8], s_rnd[8];
    const unsigned long long total = *total_ptr;
    const uint32_t k0 = blockIdx.x * n_pos;
    unsigned long long len = 0, rnd = 0;
    for (uint32_t pos = threadIdx.x; pos < n_pos; pos += blockDim.x) {
        const uint32_t m = plan_mask(sel, (int)(pos % n_xbins), (int)(pos / n_xbins));
        uint32_t b = 0;
        if (m != 0 && total != 0) {
            const unsigned __int128 p = (unsigned __int128)n_simulate * (unsigned __int128)counts[k0 + pos];
            b = (uint32_t)(p / total);
        }
        budget[k0 + pos] = b;
        mask[k0 + pos] = m;
        const unsigned long long share = counts[k0 + pos] == 0 ? 0ull : (unsigned long long)b * __popc(m);
        len += share;
        const unsigned long long r = (share + rr_group - 1) / rr_group;
        rnd = r > rnd ? r : rnd;
    }
    for (int o = 16; o > 0; o >>= 1) {
        len += __shfl_xor_sync(0xFFFFFFFFu, len, o);
        const unsigned long long x = __shfl_xor_sync(0xFFFFFFFFu, rnd, o);
        rnd = x > rnd ? x : rnd;
    }
    if (lane_id() == 0) { s_len[warp_id()] = len; s_rnd[warp_id()] = rnd; }
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int w = 1; w < 8; ++w) { len += s_len[w]; rnd = s_rnd[w] > rnd ? s_rnd[w] : rnd; }
        list_len[blockIdx.x] = len;
        rounds[blockIdx.x] = rnd;
    }
}

// The launch list of one division.  Round rho of the reading loop takes, from every PSL that still has particles to
// give, its reads number [rho G, min((rho + 1) G, share)); rounds are independent of one another once the list position
// of a round's first entry is known: sum over PSLs of min(share, rho G).  A CTA takes rounds blockIdx.x, + gridDim.x, ...
// and walks the PSLs of the fields' bounding box in spatial order with a running block scan.
__global__ void __launch_bounds__(256) k_sample_batch(const uint32_t* __restrict__ counts, const uint32_t* __restrict__ offsets,
                                                      const uint32_t* __restrict__ budget, const uint32_t* __restrict__ mask,
                                                      uint32_t k0, uint32_t n_xbins, int32_t bx0, int32_t bx1, int32_t by0,
                                                      int32_t by1, uint32_t G, unsigned long long seed,
                                                      const unsigned long long* __restrict__ rounds_ptr,
                                                      uint32_t* __restrict__ slot_out, uint8_t* __restrict__ beam_out)
{
    __shared__ uint32_t s_scan[64];
    __shared__ unsigned long long s_red[8];
    const unsigned long long n_rounds = *rounds_ptr;
    const uint32_t bw = (uint32_t)(bx1 - bx0 + 1), n_box = bw * (uint32_t)(by1 - by0 + 1);
    for (unsigned long long rho = blockIdx.x; rho < n_rounds; rho += gridDim.x) {
        const unsigned long long before = rho * G;
        // list position of the round's first entry
        unsigned long long f = 0;
        for (uint32_t i = threadIdx.x; i < n_box; i += blockDim.x) {
            const uint32_t k = k0 + (uint32_t)(by0 + (int32_t)(i / bw)) * n_xbins + (uint32_t)(bx0 + (int32_t)(i % bw));
            const unsigned long long share = counts[k] == 0 ? 0ull : (unsigned long long)budget[k] * __popc(mask[k]);
            f += share < before ? share : before;
        }
        for (int o = 16; o > 0; o >>= 1) f += __shfl_xor_sync(0xFFFFFFFFu, f, o);
        if (lane_id() == 0) s_red[warp_id()] = f;
        __syncthreads();
        f = 0;
        for (int w = 0; w < 8; ++w) f += s_red[w];
        // the round itself
        unsigned long long base = f;
        for (uint32_t i0 = 0; i0 < n_box; i0 += blockDim.x) {
            const uint32_t i = i0 + threadIdx.x;
            uint32_t k = 0, g = 0, m = 0, c = 0;
            if (i < n_box) {
                k = k0 + (uint32_t)(by0 + (int32_t)(i / bw)) * n_xbins + (uint32_t)(bx0 + (int32_t)(i % bw));
                m = mask[k];
                c = counts[k];
                const unsigned long long share = c == 0 ? 0ull : (unsigned long long)budget[k] * __popc(m);
                g = share > before ? (uint32_t)(share - before < G ? share - before : G) : 0u;
            }
            uint32_t tot;
            const uint32_t ex = block_excl_scan(g, s_scan, &tot);
            if (g != 0) {
                const uint32_t start = below(rng32(seed, k, 0), c);
                const uint32_t nsel = __popc(m);
                for (uint32_t j = 0; j < g; ++j) {
                    const unsigned long long r = before + j;  // the PSL's read number
                    const unsigned long long e = base + ex + j;
                    slot_out[e] = offsets[k] + (uint32_t)((start + r) % c);
                    uint32_t which = below(rng32(seed, k, 1ull + r), nsel), mm = m;
                    for (uint32_t z = 0; z < which; ++z) mm &= mm - 1u;  // drop the lowest `which` set bits
                    beam_out[e] = (uint8_t)(__ffs(mm) - 1);
                }
            }
            base += tot;
            __syncthreads();
        }
    }
}

// ---- emit -------------------------------------------------------------------------------------------------------
struct PlanBeam {  // one field on the device: the hot path's DevBeam plus its patient-frame rotation
    DevBeam b;
    float M[9];
    float pad[3];
};

struct LaunchOut {
    float *E, *X, *Y, *Z, *U, *V, *W, *wt;
    uint32_t* src;
    uint8_t* beam;
};

struct LaunchStats {
    unsigned long long n_jaw, n_zero, n_missed, n_launched;
};

__device__ __forceinline__ float rot_row(const float* m, float a, float b, float c)
{
    return __fadd_rn(__fadd_rn(__fmul_rn(m[0], a), __fmul_rn(m[1], b)), __fmul_rn(m[2], c));
}

// where the ray P + t D, t >= 0, enters the box (slab test, one IEEE division per bound); false = it misses
__device__ __forceinline__ bool surface_point(const float (&P)[3], const float (&D)[3], const float* lo, const float* hi, float (&S)[3])
{
    float tnear = 0.0f, tfar = __int_as_float(0x7F800000);
    bool ok = true;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        if (D[a] == 0.0f) {
            if (P[a] < lo[a] || P[a] > hi[a]) ok = false;
        } else {
            const float t1 = __fdiv_rn(__fsub_rn(lo[a], P[a]), D[a]);
            const float t2 = __fdiv_rn(__fsub_rn(hi[a], P[a]), D[a]);
            const float tn = t1 < t2 ? t1 : t2, tf = t1 < t2 ? t2 : t1;
            if (tn > tnear) tnear = tn;
            if (tf < tfar) tfar = tf;
        }
    }
    if (!ok || !(tnear <= tfar)) return false;
#pragma unroll
    for (int a = 0; a < 3; ++a) S[a] = __fadd_rn(P[a], __fmul_rn(tnear, D[a]));
    return true;
}

struct PhantomBox {
    float lo[3], hi[3];
};

constexpr int kEmitPer = 4;                        // list entries per thread
constexpr int kEmitTile = kThreads * kEmitPer;     // 1024 per CTA

__global__ void __launch_bounds__(kThreads) k_emit(const uint4* __restrict__ index, const uint32_t* __restrict__ slot,
                                                  const uint8_t* __restrict__ beam_id, uint32_t n_list,
                                                  const PlanBeam* __restrict__ beams, uint32_t n_beams, float dz_iso,
                                                  uint32_t drop_zero, const __grid_constant__ PhantomBox box, LaunchOut out,
                                                  unsigned long long* __restrict__ tile_state,
                                                  uint32_t* __restrict__ tile_counter, LaunchStats* __restrict__ stats)
{
    __shared__ uint32_t s_warp[kWarps * kEmitPer];
    __shared__ uint32_t s_ctl[3];
    if (threadIdx.x == 0) s_ctl[0] = atomicAdd(tile_counter, 1u);  // tiles are handed out in order
    __syncthreads();
    const uint32_t tile = s_ctl[0];
    const uint32_t e0 = tile * kEmitTile;
    const uint32_t w = warp_id();

    // entries r * 256 + threadIdx.x of the tile: list order = (round, warp, lane)
    float oE[kEmitPer], oS[kEmitPer][3], oD[kEmitPer][3], owt[kEmitPer];
    uint32_t osrc[kEmitPer], obm[kEmitPer], pre[kEmitPer];
    uint32_t keepbits = 0, n_jaw = 0, n_zero = 0, n_miss = 0;
#pragma unroll
    for (int r = 0; r < kEmitPer; ++r) {
        const uint32_t e = e0 + r * kThreads + threadIdx.x;
        bool keep = false;
        obm[r] = 0;
        if (e < n_list) {
            const uint32_t bi = beam_id[e];
            obm[r] = bi;
            if (bi < n_beams) {
                uint4 ra, rb;
                ldg_record(index + 2 * (size_t)__ldg(slot + e), ra, rb);
                const PlanBeam& pb = beams[bi];
                const float x = __uint_as_float(ra.z), y = __uint_as_float(ra.w);
                const float u = __uint_as_float(rb.x), v = __uint_as_float(rb.y);
                const float q = q_of(u, v);
                float wz, tx, ty;
                slopes(u, v, q, wz, tx, ty);
                keep = !pb.b.has_jaws || jaw_pass(pb.b, x, y, tx, ty);
                if (!keep) n_jaw += 1;
                const float xm = __fadd_rn(x, __fmul_rn(tx, pb.b.dzM)), ym = __fadd_rn(y, __fmul_rn(ty, pb.b.dzM));
                const float wt = final_weight(pb.b, __uint_as_float(rb.z), xm, ym);
                if (keep && drop_zero && wt == 0.0f) { keep = false; n_zero += 1; }
                float P[3], D[3];
                const float nw = -wz;
                P[0] = rot_row(pb.M + 0, x, y, dz_iso); P[1] = rot_row(pb.M + 3, x, y, dz_iso); P[2] = rot_row(pb.M + 6, x, y, dz_iso);
                D[0] = rot_row(pb.M + 0, u, v, nw); D[1] = rot_row(pb.M + 3, u, v, nw); D[2] = rot_row(pb.M + 6, u, v, nw);
                float S[3] = {0.0f, 0.0f, 0.0f};
                if (keep && !surface_point(P, D, box.lo, box.hi, S)) { keep = false; n_miss += 1; }
                oE[r] = __uint_as_float(ra.y);
                owt[r] = wt;
                osrc[r] = rb.w;
#pragma unroll
                for (int a = 0; a < 3; ++a) { oS[r][a] = S[a]; oD[r][a] = D[a]; }
            }
        }
        const uint32_t ballot = __ballot_sync(0xFFFFFFFFu, keep);
        if (lane_id() == 0) s_warp[r * kWarps + w] = __popc(ballot);
        pre[r] = __popc(ballot & lanemask_lt());
        if (keep) keepbits |= 1u << r;
    }
    __syncthreads();
    if (w == 0) {  // exclusive prefix of the 32 (round, warp) counts, then the look-back over the tiles before this one
        const uint32_t c = s_warp[lane_id()];
        const uint32_t inc = warp_incl_scan(c);
        s_warp[lane_id()] = inc - c;
        const uint32_t total = __shfl_sync(0xFFFFFFFFu, inc, 31);
        uint32_t excl = 0;
        if (tile == 0) {
            if (lane_id() == 0) atomicExch(&tile_state[0], kFlagInclusive | (unsigned long long)total);
        } else {
            if (lane_id() == 0) atomicExch(&tile_state[tile], kFlagAggregate | (unsigned long long)total);
            int look = (int)tile - 1;
            while (true) {
                const int idx = look - (int)lane_id();
                unsigned long long st;
                do {
                    st = idx >= 0 ? ld_state(&tile_state[idx]) : kFlagInclusive;
                } while (__any_sync(0xFFFFFFFFu, (st & kFlagMask) == 0ull));
                const uint32_t incl = __ballot_sync(0xFFFFFFFFu, (st & kFlagMask) == kFlagInclusive);
                uint32_t val = (uint32_t)(st & 0xFFFFFFFFull);
                if (incl) {
                    const int first = __ffs(incl) - 1;
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
            s_ctl[1] = excl;
            if (e0 + kEmitTile >= n_list) stats->n_launched = excl + total;  // last tile
        }
    }
    n_jaw = __reduce_add_sync(0xFFFFFFFFu, n_jaw);
    n_zero = __reduce_add_sync(0xFFFFFFFFu, n_zero);
    n_miss = __reduce_add_sync(0xFFFFFFFFu, n_miss);
    if (lane_id() == 0) {
        if (n_jaw) atomicAdd(&stats->n_jaw, (unsigned long long)n_jaw);
        if (n_zero) atomicAdd(&stats->n_zero, (unsigned long long)n_zero);
        if (n_miss) atomicAdd(&stats->n_missed, (unsigned long long)n_miss);
    }
    __syncthreads();
    const uint32_t gbase = s_ctl[1];
#pragma unroll
    for (int r = 0; r < kEmitPer; ++r) {
        if (keepbits & (1u << r)) {
            const size_t d = (size_t)gbase + s_warp[r * kWarps + w] + pre[r];
            out.E[d] = oE[r];
            out.X[d] = oS[r][0]; out.Y[d] = oS[r][1]; out.Z[d] = oS[r][2];
            out.U[d] = oD[r][0]; out.V[d] = oD[r][1]; out.W[d] = oD[r][2];
            out.wt[d] = owt[r];
            out.src[d] = osrc[r];
            out.beam[d] = (uint8_t)obm[r];
        }
    }
}

// ---- capacity-N emission: when does each bin of the latest ONTHEFLY build fill up? ---------------------
// key k ships floor(c_k / N) full bins, the j-th when its (j + 1) N-th survivor arrives = load-order index
// src[off_k + (j + 1) N - 1] (the build's output is in load order inside a key); what is left goes last, in key order.
struct FlushOut {
    uint32_t *key, *first, *count;
};

// one CTA, K <= kMaxBuckets keys: full[k], exclusive prefixes of the full and of the partial events
__global__ void __launch_bounds__(1024) k_flush_plan(const uint32_t* __restrict__ counts, uint32_t K, uint32_t N,
                                                     uint32_t* __restrict__ full_start, uint32_t* __restrict__ part_start,
                                                     uint32_t* __restrict__ totals)
{
    __shared__ uint32_t s_misc[64];
    const uint32_t k0 = 2 * threadIdx.x;
    uint32_t f[2] = {0, 0}, p[2] = {0, 0};
    for (int a = 0; a < 2; ++a)
        if (k0 + a < K) {
            f[a] = counts[k0 + a] / N;
            p[a] = counts[k0 + a] % N != 0 ? 1u : 0u;
        }
    uint32_t tf, tp;
    const uint32_t ef = block_excl_scan(f[0] + f[1], s_misc, &tf);
    __syncthreads();
    const uint32_t ep = block_excl_scan(p[0] + p[1], s_misc, &tp);
    if (k0 < K) { full_start[k0] = ef; part_start[k0] = ep; }
    if (k0 + 1 < K) { full_start[k0 + 1] = ef + f[0]; part_start[k0 + 1] = ep + p[0]; }
    if (threadIdx.x == 0) { totals[0] = tf; totals[1] = tp; }
}

// unsorted full events (trigger, key, first slot) and the partial events in their final places
__global__ void __launch_bounds__(256) k_flush_events(const uint32_t* __restrict__ counts, const uint32_t* __restrict__ offsets,
                                                      const uint32_t* __restrict__ src, uint32_t K, uint32_t N,
                                                      const uint32_t* __restrict__ full_start,
                                                      const uint32_t* __restrict__ part_start,
                                                      const uint32_t* __restrict__ totals, uint32_t cap,
                                                      uint32_t* __restrict__ trig, uint32_t* __restrict__ tkey,
                                                      uint32_t* __restrict__ tfirst, FlushOut out)
{
    const uint32_t n_full = totals[0];
    if (n_full + totals[1] > cap) return;  // the host reports PSL_ERR_CAPACITY
    for (uint32_t k = blockIdx.x; k < K; k += gridDim.x) {
        const uint32_t c = counts[k], nf = c / N, o = offsets[k], fs = full_start[k];
        for (uint32_t j = threadIdx.x; j < nf; j += blockDim.x) {
            trig[fs + j] = src[o + (j + 1) * N - 1];
            tkey[fs + j] = k;
            tfirst[fs + j] = o + j * N;
        }
        if (threadIdx.x == 0 && c % N != 0) {
            const uint32_t e = n_full + part_start[k];
            out.key[e] = k;
            out.first[e] = o + nf * N;
            out.count[e] = c % N;
        }
    }
}

// rank of every full event among the triggers (all different: they are load-order indices) = its place in the schedule
__global__ void __launch_bounds__(256) k_flush_order(const uint32_t* __restrict__ trig, const uint32_t* __restrict__ tkey,
                                                     const uint32_t* __restrict__ tfirst, const uint32_t* __restrict__ totals,
                                                     uint32_t cap, uint32_t N, FlushOut out)
{
    __shared__ uint32_t s_t[1024];
    const uint32_t n = totals[0];
    if (n + totals[1] > cap) return;
    for (uint32_t e0 = blockIdx.x * blockDim.x; e0 < n; e0 += gridDim.x * blockDim.x) {
        const uint32_t e = e0 + threadIdx.x;
        const uint32_t mine = e < n ? trig[e] : 0xFFFFFFFFu;
        uint32_t rank = 0;
        for (uint32_t b = 0; b < n; b += 1024) {
            __syncthreads();
            for (uint32_t i = threadIdx.x; i < 1024; i += blockDim.x) s_t[i] = b + i < n ? trig[b + i] : 0xFFFFFFFFu;
            __syncthreads();
            const uint32_t m = n - b < 1024u ? n - b : 1024u;
            for (uint32_t i = 0; i < m; ++i) rank += s_t[i] < mine ? 1u : 0u;
        }
        if (e < n) {
            out.key[rank] = tkey[e];
            out.first[rank] = tfirst[e];
            out.count[rank] = N;
        }
    }
}

}  // namespace psl
