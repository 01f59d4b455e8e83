// psl_api.cu -- host side of libpsl_b200.so: the C-ABI of include/psl.h.
//
// Argument checking, workspace carving, stream/event plumbing and kernel launches only; every step of the
// hot path runs in the kernels of psl_partition.cuh / psl_beam.cuh.  There is no CPU fallback: without a
// CUDA device every call that needs one returns PSL_ERR_CUDA.
#include "../../include/psl.h"

#include <math.h>
#include <stdarg.h>
#include <stdlib.h>
#include <stdio.h>
#include <string.h>

#include <mutex>
#include <new>
#include <utility>
#include <vector>

#include "psl_beam.cuh"
#include "psl_compact.cuh"
#include "psl_bigtile.cuh"
#include "psl_index.cuh"
#include "psl_index_big.cuh"
#include "psl_device.cuh"
#include "psl_partition.cuh"
#include "psl_plan.cuh"
#include "psl_static.cuh"

using namespace psl;

namespace {

thread_local char g_err[256] = "";

constexpr uint64_t kAlign = 256;
constexpr uint32_t kIdxSplit = 2;  // INDEX: one scatter CTA per SM, two histogram CTAs (= table columns) per segment
constexpr uint64_t kScanSmallMax = 131072;  // table entries the single-CTA scan takes
constexpr uint64_t kStageBytes = 32ull << 20;  // pinned staging buffers for pageable sources (two of them)

struct Layout {
    uint64_t total = 0;
    uint64_t raw = 0, chunks = 0, spans = 0, sstats = 0, scan_sums = 0, scalars = 0, edges = 0, stats = 0, batch_off = 0;
    // ONTHEFLY
    uint64_t table = 0, out[10] = {0}, offsets = 0, counts = 0, codes = 0, comp = 0;
    // INDEX
    uint64_t table_a = 0, table_b = 0, aos = 0, aos_index = 0, idx[7] = {0}, idx_offsets = 0, idx_counts = 0,
             idx_batch_off = 0;
    uint64_t seg = 0, beam_out[10] = {0}, beam_keys = 0, beam_offsets = 0, beam_counts = 0, lookback = 0, bstats = 0,
             beam_stats = 0;
    // INDEX, sampling layer (max_launch_records > 0)
    uint64_t plan_budget = 0, plan_mask = 0, plan_len = 0, plan_rounds = 0, plan_total = 0, plan_beams = 0, l_slot = 0, l_beam = 0,
             l_out[8] = {0}, l_src = 0, l_beam_of = 0, l_state = 0, l_stats = 0;
    // ONTHEFLY, capacity-N emission (max_launch_records > 0)
    uint64_t f_full = 0, f_part = 0, f_totals = 0, f_trig = 0, f_tkey = 0, f_tfirst = 0, f_key = 0, f_first = 0, f_count = 0;
};

struct Derived {
    uint32_t K = 0, n_batches = 0, n_pos = 0;
    uint32_t lo_bits = 0, B_lo = 0, B_hi = 0;
    uint32_t tiles_cap = 0, cols_cap = 0, max_chunks = 0;  // cols = table columns = segments over all launches
    uint64_t max_beam = 0;
    uint32_t max_seg = 0;
    uint32_t scan_blocks_cap = 0;
};

void set_err(char* dst, const char* fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(dst, 256, fmt, ap);
    va_end(ap);
}

bool is_integer_ratio(float a, float d, int32_t* out)
{
    double r = (double)a / (double)d;
    double n = nearbyint(r);
    if (fabs(r - n) > 1e-6 * fmax(1.0, fabs(r))) return false;
    if (fabs(n) > 1e9) return false;
    *out = (int32_t)n;
    return true;
}

psl_status check_geometry(const psl_geometry& g, char* err)
{
    bool ok = isfinite(g.z_src) && isfinite(g.z_plane) && isfinite(g.z_jaw_x) && isfinite(g.z_jaw_y) && isfinite(g.z_map) &&
              isfinite(g.z_iso) && g.z_src < g.z_plane && g.z_plane <= g.z_jaw_x && g.z_plane <= g.z_jaw_y &&
              g.z_plane <= g.z_map && g.z_jaw_x <= g.z_iso && g.z_jaw_y <= g.z_iso && g.z_map <= g.z_iso;
    if (!ok) {
        set_err(err, "geometry: need z_src < z_plane <= z_jaw_x, z_jaw_y, z_map <= z_iso");
        return PSL_ERR_GEOMETRY;
    }
    return PSL_OK;
}

psl_status derive(const psl_config* c, Derived* d, char* err)
{
    if (!c) { set_err(err, "config is NULL"); return PSL_ERR_ARG; }
    if (c->struct_size != sizeof(psl_config)) { set_err(err, "config.struct_size %u != %zu", c->struct_size, sizeof(psl_config)); return PSL_ERR_ARG; }
    if (c->mode != PSL_MODE_ONTHEFLY && c->mode != PSL_MODE_INDEX) { set_err(err, "config.mode"); return PSL_ERR_ARG; }
    if (c->n_types != 2 && c->n_types != 3) { set_err(err, "config.n_types must be 2 or 3"); return PSL_ERR_ARG; }
    if (c->n_ebins < 1 || c->n_ebins > 1024) { set_err(err, "config.n_ebins must be 1..1024"); return PSL_ERR_ARG; }
    if (c->ebin_mode == PSL_EBIN_LINEAR) {
        if (!(isfinite(c->e_min) && isfinite(c->e_max) && c->e_max > c->e_min)) { set_err(err, "config: need e_max > e_min"); return PSL_ERR_ARG; }
    } else if (c->ebin_mode == PSL_EBIN_EDGES) {
        if (!c->e_edges) { set_err(err, "config.e_edges is NULL in edge mode"); return PSL_ERR_ARG; }
        for (int i = 0; i < c->n_ebins; ++i)
            if (!(c->e_edges[i] < c->e_edges[i + 1])) { set_err(err, "config.e_edges must be strictly ascending"); return PSL_ERR_ARG; }
    } else { set_err(err, "config.ebin_mode"); return PSL_ERR_ARG; }
    if (c->n_xbins < 1 || c->n_ybins < 1 || c->n_xbins > 4096 || c->n_ybins > 4096) { set_err(err, "config.n_xbins/n_ybins must be 1..4096"); return PSL_ERR_ARG; }
    uint64_t n_pos = (uint64_t)c->n_xbins * (uint64_t)c->n_ybins;
    if (n_pos > 1 || c->mode == PSL_MODE_INDEX) {
        int32_t t;
        if (!(c->dx > 0 && c->dy > 0 && isfinite(c->dx) && isfinite(c->dy))) { set_err(err, "config: dx, dy must be positive"); return PSL_ERR_ARG; }
        if (n_pos > 1 && (!is_integer_ratio(c->x_min, c->dx, &t) || !is_integer_ratio(c->y_min, c->dy, &t))) { set_err(err, "config: x_min/dx and y_min/dy must be integers"); return PSL_ERR_ARG; }
    }
    psl_status gs = check_geometry(c->geom, err);
    if (gs != PSL_OK) return gs;
    uint64_t K = (uint64_t)c->n_types * c->n_ebins * n_pos;
    if (c->max_records == 0 || c->max_records >= (1ull << 32)) { set_err(err, "config.max_records must be 1..2^32-1"); return PSL_ERR_ARG; }
    if (c->max_host_records > c->max_records) { set_err(err, "config.max_host_records > max_records"); return PSL_ERR_ARG; }
    if (c->max_launch_records >= (1ull << 32)) { set_err(err, "config.max_launch_records must be < 2^32"); return PSL_ERR_ARG; }
    if ((c->flags & PSL_APR) && c->mode != PSL_MODE_INDEX) { set_err(err, "PSL_APR needs PSL_MODE_INDEX"); return PSL_ERR_ARG; }
    d->K = (uint32_t)K;
    d->n_pos = (uint32_t)n_pos;
    d->n_batches = (uint32_t)(c->n_types * c->n_ebins);
    d->max_chunks = c->max_chunks ? c->max_chunks : 4096u;
    uint64_t tiles_cap = (c->max_records + kTile - 1) / kTile + d->max_chunks;
    // ONTHEFLY builds in one launch over all chunks; INDEX counts chunk by chunk as the chunks land
    uint64_t cols_cap = kMaxSegments;
    if (c->mode == PSL_MODE_INDEX) {
        // a chunk of nt tiles takes min(nt, segments per launch) x kIdxSplit columns: at most kIdxSplit per tile
        cols_cap = (uint64_t)d->max_chunks * kMaxSegments;
        if (cols_cap > (uint64_t)kIdxSplit * tiles_cap) cols_cap = (uint64_t)kIdxSplit * tiles_cap;
    }
    if (c->mode == PSL_MODE_ONTHEFLY) {
        if (K > kMaxBuckets) { set_err(err, "ONTHEFLY mode handles at most %d keys (got %llu); use PSL_MODE_INDEX", kMaxBuckets, (unsigned long long)K); return PSL_ERR_ARG; }
    } else {
        if (K > (uint64_t)kIdxMaxHi * kIdxMaxLo) { set_err(err, "INDEX mode handles at most %d keys", kIdxMaxHi * kIdxMaxLo); return PSL_ERR_ARG; }
        // key = hi * 2^lo_bits + lo, two balanced digits: what matters is that (buckets x CTAs x 128 B), the lines
        // being filled at any time, stays inside the 126 MB L2 in both passes
        uint32_t bits = 0;
        while ((1ull << bits) < K) ++bits;
        uint32_t lo = bits / 2;
        while ((((K - 1) >> lo) + 1) > (uint64_t)kIdxMaxHi) ++lo;
        d->lo_bits = lo;
        d->B_lo = (uint32_t)((K < (1ull << lo)) ? K : (1ull << lo));
        if (d->B_lo < 1) d->B_lo = 1;
        d->B_hi = (uint32_t)(((K - 1) >> lo) + 1);
        if ((uint64_t)d->B_lo * cols_cap >= (1ull << 32)) { set_err(err, "buckets x segments overflows 32 bits"); return PSL_ERR_CAPACITY; }
        d->max_beam = c->max_beam_records ? c->max_beam_records : c->max_records;
        if (d->max_beam > c->max_records) d->max_beam = c->max_records;
        d->max_seg = d->n_batches * (uint32_t)c->n_ybins;
    }
    d->tiles_cap = (uint32_t)tiles_cap;
    d->cols_cap = (uint32_t)cols_cap;
    uint64_t Lmax = c->mode == PSL_MODE_ONTHEFLY ? K * cols_cap
                                                  : ((uint64_t)d->B_lo * cols_cap > (uint64_t)d->B_hi * kMaxSegments
                                                         ? (uint64_t)d->B_lo * cols_cap
                                                         : (uint64_t)d->B_hi * kMaxSegments);
    d->scan_blocks_cap = (uint32_t)((Lmax + kScanBlock - 1) / kScanBlock);
    return PSL_OK;
}

uint64_t take(uint64_t* cur, uint64_t bytes)
{
    uint64_t at = *cur;
    *cur = (at + bytes + kAlign - 1) / kAlign * kAlign;
    return at;
}

void plan(const psl_config* c, const Derived& d, Layout* L)
{
    uint64_t cur = 0;
    const uint64_t N = c->max_records;
    const bool proj = (c->flags & PSL_OUT_PROJ) != 0;
    L->raw = take(&cur, c->max_host_records * kRecBytes);
    L->chunks = take(&cur, (uint64_t)d.max_chunks * sizeof(ChunkDesc));
    L->spans = take(&cur, (uint64_t)d.max_chunks * sizeof(SpanSeg));
    L->sstats = take(&cur, (uint64_t)d.cols_cap * sizeof(SegStats));
    L->scan_sums = take(&cur, (uint64_t)(d.scan_blocks_cap + 1) * 4);
    L->scalars = take(&cur, 64);
    L->edges = take(&cur, (uint64_t)(c->n_ebins + 1) * 4);
    L->stats = take(&cur, sizeof(DevStats));
    L->batch_off = take(&cur, (uint64_t)(d.n_batches + 1) * 4);
    if (c->mode == PSL_MODE_ONTHEFLY) {
        L->table = take(&cur, (uint64_t)d.K * d.cols_cap * 4);
        for (int i = 0; i < 10; ++i) L->out[i] = ((i == 7 || i == 8) && !proj) ? 0 : take(&cur, N * 4);
        L->offsets = take(&cur, (uint64_t)(d.K + 1) * 4);
        L->counts = take(&cur, (uint64_t)d.K * 4);
        if (c->max_launch_records) {
            const uint64_t E = c->max_launch_records;
            L->f_full = take(&cur, (uint64_t)d.K * 4); L->f_part = take(&cur, (uint64_t)d.K * 4); L->f_totals = take(&cur, 8);
            L->f_trig = take(&cur, E * 4); L->f_tkey = take(&cur, E * 4); L->f_tfirst = take(&cur, E * 4);
            L->f_key = take(&cur, E * 4); L->f_first = take(&cur, E * 4); L->f_count = take(&cur, E * 4);
        }
        L->codes = take(&cur, N);  // one byte per record: the histogram kernel's verdict for the scatter of a rejecting beam
        // few keys: the survivors of a rejecting beam, compacted per histogram segment (32 B each, a segment's region
        // starts at its first record, so only the survivors' share of it is ever touched)
        if (round_up(d.K, 8) <= (uint32_t)kBigMaxKeys) L->comp = take(&cur, (uint64_t)d.tiles_cap * kTile * kCompBytes);
    } else {
        L->table_a = take(&cur, (uint64_t)d.B_lo * d.cols_cap * 4);
        L->table_b = take(&cur, (uint64_t)d.B_hi * kMaxSegments * 4);
        {   // pass A output; once the index is built the SoA view of the bare index (7 arrays) lives in the same bytes
            const uint64_t view_bytes = 7 * ((N * 4 + kAlign - 1) / kAlign * kAlign);
            L->aos = take(&cur, N * 32 > view_bytes ? N * 32 : view_bytes);
            uint64_t view = L->aos;
            for (int i = 0; i < 7; ++i) L->idx[i] = take(&view, N * 4);
        }
        L->aos_index = take(&cur, N * 32);  // the index: keyed records sorted by the full key
        L->idx_offsets = take(&cur, (uint64_t)(d.K + 1) * 4);
        L->idx_counts = take(&cur, (uint64_t)d.K * 4);
        L->idx_batch_off = take(&cur, (uint64_t)(d.n_batches + 1) * 4);
        L->seg = take(&cur, (uint64_t)(3 * d.max_seg + 1) * 4);
        for (int i = 0; i < 10; ++i) L->beam_out[i] = ((i == 7 || i == 8) && !proj) ? 0 : take(&cur, d.max_beam * 4);
        L->beam_keys = take(&cur, d.max_beam * 4);
        L->beam_offsets = take(&cur, (uint64_t)(d.K + 1) * 4);
        L->beam_counts = take(&cur, (uint64_t)d.K * 4);
        uint64_t bt = (d.max_beam + kBeamTile - 1) / kBeamTile + 1;
        L->lookback = take(&cur, bt * 8);
        L->bstats = take(&cur, bt * sizeof(BeamTileStats));
        L->beam_stats = take(&cur, sizeof(DevBeamStats));
        if (c->max_launch_records) {
            const uint64_t E = c->max_launch_records;
            L->plan_budget = take(&cur, (uint64_t)d.K * 4); L->plan_mask = take(&cur, (uint64_t)d.K * 4);
            L->plan_len = take(&cur, (uint64_t)d.n_batches * 8); L->plan_rounds = take(&cur, (uint64_t)d.n_batches * 8);
            L->plan_total = take(&cur, 8);
            L->plan_beams = take(&cur, (uint64_t)kMaxPlanBeams * sizeof(PlanBeam));
            L->l_slot = take(&cur, E * 4); L->l_beam = take(&cur, E);
            for (int i = 0; i < 8; ++i) L->l_out[i] = take(&cur, E * 4);
            L->l_src = take(&cur, E * 4); L->l_beam_of = take(&cur, E);
            L->l_state = take(&cur, ((E + kEmitTile - 1) / kEmitTile + 1) * 8);
            L->l_stats = take(&cur, sizeof(LaunchStats) + 16);  // + the tile counter
        }
    }
    L->total = cur;
}

enum ResultKind { RES_NONE = 0, RES_OTF = 1, RES_INDEX = 2, RES_BEAM = 3 };

// ---- kernel variants: the features a configuration / beam does not use are compiled out ------------------
using CountFn = void (*)(const ChunkDesc*, uint32_t, Span, DevGrid, DevBeam, uint32_t, uint32_t, uint32_t*, uint32_t, SegStats*, uint32_t, uint8_t*, uint4*);
using ScatterCompFn = void (*)(const uint4*, Span, DevBeam, uint32_t, const uint32_t*, uint32_t, SoAOut, SegStats*, FusedScan, StatsTail);
using ScatterOtfFn = void (*)(const ChunkDesc*, uint32_t, Span, DevGrid, DevBeam, uint32_t, const uint32_t*, uint32_t, SoAOut, SegStats*,
                              const uint8_t*, FusedScan, StatsTail);
using ScatterBigFn = void (*)(const ChunkDesc*, uint32_t, Span, DevGrid, DevBeam, uint32_t, const uint32_t*, uint32_t, SoAOut, SegStats*, FusedScan, StatsTail);

template <bool POS, bool EDGES>
CountFn count_otf_pe(int beam)
{
    return beam == 0 ? k_count_raw<false, POS, EDGES, 0> : (beam == 1 ? k_count_raw<false, POS, EDGES, 1> : k_count_raw<false, POS, EDGES, 2>);
}
CountFn count_otf_fn(bool pos, bool edges, int beam)
{
    return pos ? (edges ? count_otf_pe<true, true>(beam) : count_otf_pe<true, false>(beam))
               : (edges ? count_otf_pe<false, true>(beam) : count_otf_pe<false, false>(beam));
}
CountFn count_idx_fn(bool pos, bool edges)
{
    return pos ? (edges ? k_count_raw<true, true, true, 0> : k_count_raw<true, true, false, 0>)
               : (edges ? k_count_raw<true, false, true, 0> : k_count_raw<true, false, false, 0>);
}
template <bool POS, bool EDGES, bool PROJ>
ScatterOtfFn scatter_otf_pep(int beam)
{
    return beam == 0 ? k_scatter_otf<POS, EDGES, 0, PROJ> : (beam == 1 ? k_scatter_otf<POS, EDGES, 1, PROJ> : k_scatter_otf<POS, EDGES, 2, PROJ>);
}
template <bool POS, bool EDGES>
ScatterOtfFn scatter_otf_pe(int beam, bool proj)
{
    return proj ? scatter_otf_pep<POS, EDGES, true>(beam) : scatter_otf_pep<POS, EDGES, false>(beam);
}
ScatterOtfFn scatter_otf_fn(bool pos, bool edges, int beam, bool proj)
{
    return pos ? (edges ? scatter_otf_pe<true, true>(beam, proj) : scatter_otf_pe<true, false>(beam, proj))
               : (edges ? scatter_otf_pe<false, true>(beam, proj) : scatter_otf_pe<false, false>(beam, proj));
}
template <bool POS, bool EDGES, bool PROJ>
ScatterBigFn scatter_big_pep(int beam)
{
    return beam == 0 ? k_scatter_otf_big<POS, EDGES, 0, PROJ> : (beam == 1 ? k_scatter_otf_big<POS, EDGES, 1, PROJ> : k_scatter_otf_big<POS, EDGES, 2, PROJ>);
}
template <bool POS, bool EDGES>
ScatterBigFn scatter_big_pe(int beam, bool proj)
{
    return proj ? scatter_big_pep<POS, EDGES, true>(beam) : scatter_big_pep<POS, EDGES, false>(beam);
}
// the 4096-record-tile scatter (keys <= kBigMaxKeys)
ScatterBigFn scatter_big_fn(bool pos, bool edges, int beam, bool proj)
{
    return pos ? (edges ? scatter_big_pe<true, true>(beam, proj) : scatter_big_pe<true, false>(beam, proj))
               : (edges ? scatter_big_pe<false, true>(beam, proj) : scatter_big_pe<false, false>(beam, proj));
}
using ScatterIdxBigFn = void (*)(const ChunkDesc*, uint32_t, const SpanSeg*, uint32_t, Span, const uint4*, const uint32_t*, DevGrid, DevBeam,
                                 uint32_t, uint32_t, const uint32_t*, uint32_t, uint4*);
// the 4096-record-tile INDEX passes: A (raw records in) per grid features, B (keyed records in)
ScatterIdxBigFn scatter_idx_big_a_fn(bool pos, bool edges)
{
    return pos ? (edges ? k_scatter_idx_big<false, true, true> : k_scatter_idx_big<false, true, false>)
               : (edges ? k_scatter_idx_big<false, false, true> : k_scatter_idx_big<false, false, false>);
}
ScatterIdxBigFn scatter_idx_big_b_fn() { return k_scatter_idx_big<true, false, false>; }
}  // namespace

struct psl_ctx {
    psl_config cfg;
    Derived d;
    Layout L;
    DevGrid grid;
    std::vector<float> edges;
    uint8_t* ws = nullptr;
    cudaStream_t stream = nullptr, copy_stream = nullptr;
    cudaEvent_t ev_chunk = nullptr, ev_main = nullptr, ev_batch = nullptr, ev_seg = nullptr, ev_stage[2] = {nullptr, nullptr};
    void* h_stage[2] = {nullptr, nullptr};
    int stage_next = 0;
    // pinned host mirrors
    uint32_t* h_batch_off = nullptr;   // n_batches+1
    uint32_t* h_idx_offsets = nullptr; // K+1 (INDEX)
    uint32_t* h_seg = nullptr;         // 3*max_seg+1
    DevStats* h_stats = nullptr;
    DevStats* d_h_stats = nullptr;      // device views of the pinned copies (null: not mapped, copies are used)
    uint32_t* d_h_batch_off = nullptr;
    DevBeamStats* h_beam_stats = nullptr;
    uint32_t* h_scalars = nullptr;
    bool seg_pending = false;
    // launch shapes: persistent CTAs per launch (= SMs x resident CTAs of the scatter kernel, one wave)
    uint32_t S_otf = 0, S_otf_small = 0, S_a = 0, S_b = 0, S_comp = 0;
    uint32_t sm_scatter_small = 0, sm_scatter_comp = 0;
    bool compact = false;  // ONTHEFLY with few keys, rejecting beam: the histogram kernel compacts the survivors
    bool big_tiles = false;  // ONTHEFLY with few keys: the 4096-record-tile scatter
    uint32_t count_stages = kStagesCount, count_split = 1;
    uint32_t sm_count_raw = 0, sm_scatter_otf = 0, sm_idx_a = 0, sm_count_b = 0, sm_idx_b = 0;  // dynamic smem bytes
    uint32_t split_a = 1, split_b = 1;  // histogram CTAs (= table columns) per scatter segment
    struct ChunkLaunch { Span span; uint32_t n_seg; };
    std::vector<ChunkDesc> pending_chunks;  // ONTHEFLY: chunk descriptors not yet on the device
    uint32_t chunks_uploaded = 0;
    std::vector<ChunkLaunch> idx_launches;
    std::vector<SpanSeg> h_spans;  // INDEX: the per-chunk count launches, replayed by pass A's scatter
    std::vector<uint32_t> h_idx_batch_off;  // INDEX: batch offsets of the bare index (n_batches+1)
    // sampling layer
    bool plan_set = false;
    psl_plan plan = {};
    PlanSel plan_sel = {};
    std::vector<PlanBeam> h_plan_beams;
    unsigned long long* h_plan = nullptr;  // pinned: [0] N_total, [1 .. n_batches] list lengths, then the rounds
    LaunchStats* h_launch_stats = nullptr;
    uint32_t* h_flush_totals = nullptr;
    // state
    uint64_t n_records = 0, n_host_records = 0;
    uint32_t n_tiles = 0, n_chunks = 0, n_cols = 0;
    uint32_t tiles_counted = 0, cols_bound = 0;  // INDEX: tiles already histogrammed; columns if every chunk were counted alone
    bool ragged = false;  // a chunk with n % 4 != 0 was loaded: no more chunks may follow
    bool indexed = false, soa_view = false;
    int result = RES_NONE;
    DevStats idx_stats = {};
    uint64_t n_idx = 0, last_M = 0;
    uint64_t launches = 0;
    // optional kernel timing (psl_profile_*)
    bool profiling = false;
    struct Bracket { int cls; cudaEvent_t a, b; };
    std::vector<Bracket> brackets;        // recorded since the last read
    std::vector<cudaEvent_t> event_pool;  // timing events ready for reuse
    char err[256] = "";
};

namespace {

#define CU(call)                                                                                           \
    do {                                                                                                   \
        cudaError_t e_ = (call);                                                                           \
        if (e_ != cudaSuccess) {                                                                           \
            set_err(ctx->err, "%s failed: %s (%s:%d)", #call, cudaGetErrorString(e_), __FILE__, __LINE__); \
            return PSL_ERR_CUDA;                                                                           \
        }                                                                                                  \
    } while (0)

#define LAUNCHED()                                    \
    do {                                              \
        ctx->launches += 1;                           \
        CU(cudaGetLastError());                       \
    } while (0)

cudaEvent_t prof_event(psl_ctx* ctx)
{
    cudaEvent_t e = nullptr;
    if (!ctx->event_pool.empty()) {
        e = ctx->event_pool.back();
        ctx->event_pool.pop_back();
    } else if (cudaEventCreate(&e) != cudaSuccess) {
        e = nullptr;
    }
    return e;
}

// RAII bracket: records a timing event on the stream before and after the launches in its scope
struct Prof {
    psl_ctx* ctx;
    int cls;
    cudaEvent_t a = nullptr;
    Prof(psl_ctx* c, int k) : ctx(c), cls(k)
    {
        if (ctx->profiling && ctx->brackets.size() < 65536) {
            a = prof_event(ctx);
            if (a) cudaEventRecord(a, ctx->stream);
        }
    }
    ~Prof()
    {
        if (!a) return;
        cudaEvent_t b = prof_event(ctx);
        if (b) {
            cudaEventRecord(b, ctx->stream);
            ctx->brackets.push_back({cls, a, b});
        } else {
            ctx->event_pool.push_back(a);
        }
    }
};

// launch with programmatic stream serialisation (psl_device.cuh, griddep_wait): the kernel may start while its
// predecessor in the stream drains.  Off while kernels are bracketed by events.
template <typename... Params, typename... Args>
cudaError_t launch_after(bool overlap, void (*fn)(Params...), uint32_t grid, uint32_t block, uint32_t smem, cudaStream_t st,
                         Args&&... args)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(grid);
    cfg.blockDim = dim3(block);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = overlap ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, fn, std::forward<Args>(args)...);
}

template <typename T>
T* at(psl_ctx* ctx, uint64_t off) { return reinterpret_cast<T*>(ctx->ws + off); }

uint32_t* scalar(psl_ctx* ctx, int i) { return at<uint32_t>(ctx, ctx->L.scalars) + i; }
enum { SC_TOTAL = 0, SC_NIDX = 1, SC_TILE_COUNTER = 2, SC_BEAM_NSURV = 3, SC_TICKET = 4 };

DevGrid make_grid(const psl_config& c, const Derived& d, const float* dev_edges)
{
    DevGrid g;
    g.n_types = c.n_types;
    g.ebin_mode = c.ebin_mode;
    g.n_ebins = c.n_ebins;
    g.e_min = c.e_min;
    g.dE = c.ebin_mode == PSL_EBIN_LINEAR ? (float)(((double)c.e_max - (double)c.e_min) / (double)c.n_ebins) : 1.0f;
    g.e_edges = dev_edges;
    g.has_pos = d.n_pos > 1;
    g.n_xbins = c.n_xbins;
    g.n_ybins = c.n_ybins;
    g.ix0 = g.iy0 = 0;
    g.inv_dx = g.inv_dy = 1.0f;
    if (g.has_pos) {
        is_integer_ratio(c.x_min, c.dx, &g.ix0);
        is_integer_ratio(c.y_min, c.dy, &g.iy0);
        g.inv_dx = (float)(1.0 / (double)c.dx);
        g.inv_dy = (float)(1.0 / (double)c.dy);
    }
    g.n_pos = d.n_pos;
    g.apr = (c.flags & PSL_APR) ? 1u : 0u;
    g.apr_seed = c.apr_seed;
    return g;
}

float edge_at_jaw_plane(float edge_iso, float z_jaw, const psl_geometry& g)
{
    return (float)((double)edge_iso * ((double)z_jaw - (double)g.z_src) / ((double)g.z_iso - (double)g.z_src));
}

psl_status make_beam(const psl_ctx* ctx, const psl_beam* b, DevBeam* out, char* err)
{
    const psl_config& c = ctx->cfg;
    DevBeam v;
    memset(&v, 0, sizeof v);
    v.dzM = c.geom.z_map - c.geom.z_plane;
    v.mu = 1.0f;
    v.out_proj = (c.flags & PSL_OUT_PROJ) ? 1u : 0u;
    if (b) {
        v.has_beam = 1;
        if (!isfinite(b->mu_weight)) { set_err(err, "beam.mu_weight is not finite"); return PSL_ERR_ARG; }
        v.mu = b->mu_weight;
        v.drop_zero = (c.flags & PSL_DROP_ZERO_WEIGHT) ? 1u : 0u;
        if (b->has_jaws) {
            if (!(b->jaw_x1 <= b->jaw_x2 && b->jaw_y1 <= b->jaw_y2)) { set_err(err, "beam: jaw edges out of order"); return PSL_ERR_ARG; }
            v.has_jaws = 1;
            v.X1 = edge_at_jaw_plane(b->jaw_x1, c.geom.z_jaw_x, c.geom);
            v.X2 = edge_at_jaw_plane(b->jaw_x2, c.geom.z_jaw_x, c.geom);
            v.Y1 = edge_at_jaw_plane(b->jaw_y1, c.geom.z_jaw_y, c.geom);
            v.Y2 = edge_at_jaw_plane(b->jaw_y2, c.geom.z_jaw_y, c.geom);
            v.dzJx = c.geom.z_jaw_x - c.geom.z_plane;
            v.dzJy = c.geom.z_jaw_y - c.geom.z_plane;
        }
        if (b->fluence) {
            if (b->map_nx < 1 || b->map_ny < 1 || !(b->map_dx > 0) || !(b->map_dy > 0)) { set_err(err, "beam: bad fluence map shape"); return PSL_ERR_ARG; }
            if (!is_integer_ratio(b->map_x0, b->map_dx, &v.px0) || !is_integer_ratio(b->map_y0, b->map_dy, &v.py0)) { set_err(err, "beam: map_x0/map_dx and map_y0/map_dy must be integers"); return PSL_ERR_ARG; }
            v.has_map = 1;
            v.fluence = b->fluence;
            v.map_nx = b->map_nx;
            v.map_ny = b->map_ny;
            v.inv_mdx = (float)(1.0 / (double)b->map_dx);
            v.inv_mdy = (float)(1.0 / (double)b->map_dy);
        }
        if (b->has_roi) {
            if (c.mode != PSL_MODE_INDEX) { set_err(err, "beam.has_roi needs PSL_MODE_INDEX"); return PSL_ERR_ARG; }
            if (!(isfinite(b->roi_x1) && isfinite(b->roi_x2) && isfinite(b->roi_y1) && isfinite(b->roi_y2))) { set_err(err, "beam: ROI is not finite"); return PSL_ERR_ARG; }
        }
    }
    *out = v;
    return PSL_OK;
}

// bins c of [origin + c d, origin + (c+1) d) with positive-length overlap with (lo, hi)
void select_axis(double origin, double d, int n, double lo, double hi, int* first, int* last)
{
    const double fg = floor((lo - origin) / d) - 1.0;  // clamped in double: the ROI may lie far outside the grid
    int f = !(fg > 0.0) ? 0 : (fg >= (double)n ? n : (int)fg);
    while (f < n && !(origin + (double)(f + 1) * d > lo)) ++f;
    double lg = floor((hi - origin) / d) + 1.0;
    int l = lg >= (double)n ? n - 1 : (lg < 0 ? -1 : (int)lg);
    while (l >= 0 && !(origin + (double)l * d < hi)) --l;
    *first = f;
    *last = l;
}

void roi_bins(const psl_config& c, const psl_beam* b, int32_t out[4])
{
    if (!b || !b->has_roi) {
        out[0] = 0; out[1] = c.n_xbins - 1; out[2] = 0; out[3] = c.n_ybins - 1;
        return;
    }
    select_axis(c.x_min, c.dx, c.n_xbins, b->roi_x1, b->roi_x2, &out[0], &out[1]);
    select_axis(c.y_min, c.dy, c.n_ybins, b->roi_y1, b->roi_y2, &out[2], &out[3]);
}

template <typename Kern>
cudaError_t allow_smem(Kern k, uint32_t bytes)
{
    return cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
}

// exclusive scan of table (virtual order bucket-major, tile-minor); grand total -> *total_dev
psl_status run_scan(psl_ctx* ctx, uint32_t* table, uint32_t B, uint32_t n_cols, uint32_t stride, uint32_t* total_dev)
{
    uint64_t L64 = (uint64_t)B * n_cols;
    uint32_t L = (uint32_t)L64;
    uint32_t nb = (uint32_t)((L64 + kScanBlock - 1) / kScanBlock);
    uint32_t* sums = at<uint32_t>(ctx, ctx->L.scan_sums);
    Prof prof(ctx, PSL_K_SCAN);
    k_scan_reduce<<<nb, kScanThreads, 0, ctx->stream>>>(table, n_cols, stride, L, sums);
    LAUNCHED();
    k_scan_sums<<<1, 1024, 0, ctx->stream>>>(sums, nb, total_dev);
    LAUNCHED();
    k_scan_apply<<<nb, kScanThreads, 0, ctx->stream>>>(table, n_cols, stride, L, sums);
    LAUNCHED();
    return PSL_OK;
}

SoAOut soa_out(psl_ctx* ctx, const uint64_t off[10])
{
    SoAOut o;
    o.E = at<float>(ctx, off[0]); o.x = at<float>(ctx, off[1]); o.y = at<float>(ctx, off[2]);
    o.u = at<float>(ctx, off[3]); o.v = at<float>(ctx, off[4]); o.w = at<float>(ctx, off[5]);
    o.wt = at<float>(ctx, off[6]);
    o.xp = at<float>(ctx, off[7]); o.yp = at<float>(ctx, off[8]);
    o.src = at<uint32_t>(ctx, off[9]);
    return o;
}

// chunk descriptors not yet on the device: uploaded 128 at a time (they travel as a kernel argument)
psl_status upload_chunks(psl_ctx* ctx)
{
    ChunkDesc* chunks = at<ChunkDesc>(ctx, ctx->L.chunks);
    for (size_t f = 0; f < ctx->pending_chunks.size(); f += 128) {
        ChunkBatch cb;
        const uint32_t m = (uint32_t)(ctx->pending_chunks.size() - f < 128 ? ctx->pending_chunks.size() - f : 128);
        memcpy(cb.d, ctx->pending_chunks.data() + f, m * sizeof(ChunkDesc));
        k_set_chunks<<<1, 128, 0, ctx->stream>>>(chunks + ctx->chunks_uploaded, cb, m);
        LAUNCHED();
        ctx->chunks_uploaded += m;
    }
    ctx->pending_chunks.clear();
    return PSL_OK;
}

// INDEX: a8 for pass A over every tile loaded since the last count, in ONE launch.  HOST chunks are counted as they
// land (the launch overlaps the transfer of the next chunk); DEVICE chunks wait here until a HOST chunk or the index
// build flushes them, so a phase-space that is already resident is counted by one launch, not one per chunk
// (105 launches of 48 us at config 5 cost 1.5 ms of tails and launch gaps).
psl_status count_pending_tiles(psl_ctx* ctx)
{
    const uint32_t nt = ctx->n_tiles - ctx->tiles_counted;
    if (nt == 0) return PSL_OK;
    psl_status s = upload_chunks(ctx);
    if (s != PSL_OK) return s;
    DevBeam none;
    memset(&none, 0, sizeof none);
    psl_ctx::ChunkLaunch cl;
    cl.span = {ctx->tiles_counted, nt, ctx->n_cols, ctx->split_a};
    cl.n_seg = nt < ctx->S_a ? nt : ctx->S_a;
    if (ctx->n_cols + cl.n_seg * ctx->split_a > ctx->d.cols_cap) { set_err(ctx->err, "out of table columns"); return PSL_ERR_CAPACITY; }
    {
        Prof prof(ctx, PSL_K_COUNT);
        count_idx_fn(ctx->grid.has_pos != 0, ctx->grid.ebin_mode != 0)<<<cl.n_seg * ctx->split_a, kThreads, ctx->sm_count_raw, ctx->stream>>>(
            at<ChunkDesc>(ctx, ctx->L.chunks), ctx->n_chunks, cl.span, ctx->grid, none, ctx->d.B_lo, (1u << ctx->d.lo_bits) - 1u,
            at<uint32_t>(ctx, ctx->L.table_a), ctx->d.cols_cap, at<SegStats>(ctx, ctx->L.sstats), ctx->count_stages, nullptr, nullptr);
        LAUNCHED();
    }
    ctx->idx_launches.push_back(cl);
    ctx->n_cols += cl.n_seg * ctx->split_a;
    ctx->tiles_counted = ctx->n_tiles;
    return PSL_OK;
}

psl_status build_onthefly(psl_ctx* ctx, const DevBeam& bm)
{
    const Derived& d = ctx->d;
    const Layout& L = ctx->L;
    uint32_t* table = at<uint32_t>(ctx, L.table);
    uint32_t* offsets = at<uint32_t>(ctx, L.offsets);
    uint32_t* counts = at<uint32_t>(ctx, L.counts);
    uint32_t* batch_off = at<uint32_t>(ctx, L.batch_off);
    DevStats* stats = at<DevStats>(ctx, L.stats);
    const uint32_t nt = ctx->n_tiles;
    StatsTail tail;
    bool to_host = false;
    if (nt == 0) {
        CU(cudaMemsetAsync(offsets, 0, (uint64_t)(d.K + 1) * 4, ctx->stream));
        CU(cudaMemsetAsync(counts, 0, (uint64_t)d.K * 4, ctx->stream));
        CU(cudaMemsetAsync(batch_off, 0, (uint64_t)(d.n_batches + 1) * 4, ctx->stream));
        CU(cudaMemsetAsync(stats, 0, sizeof(DevStats), ctx->stream));
    } else {
        ChunkDesc* chunks = at<ChunkDesc>(ctx, L.chunks);
        {
            psl_status us = upload_chunks(ctx);
            if (us != PSL_OK) return us;
        }
        SegStats* ss = at<SegStats>(ctx, L.sstats);
        const bool pos = ctx->grid.has_pos != 0, edges = ctx->grid.ebin_mode != 0, proj = bm.has_map || bm.out_proj;
        const int bv = beam_variant(bm);
        // 4096-record tiles pay when most records are written out (long runs per key); when jaws reject most of
        // them the kernel is a read stream and two 1024-record-tile CTAs per SM overlap better
        const bool big = ctx->big_tiles && bv == 0;
        // ... unless the histogram kernel compacts the survivors: then the scatter reads only those, in 4096-survivor tiles
        const bool compact = ctx->compact && bv != 0;
        const uint32_t S_max = big ? ctx->S_otf : (compact ? ctx->S_comp : ctx->S_otf_small), split = (big || compact) ? ctx->count_split : 1u;
        const uint32_t S = nt < S_max ? nt : S_max;  // one persistent CTA per segment, one wave
        const Span span = {0u, nt, 0u, split};
        const uint32_t n_cols = S * split;
        // a beam that rejects (jaws, zero-weight policy): the histogram kernel leaves one byte per record (key or
        // 255 = dropped) and the scatter ranks from those instead of repeating the projection arithmetic
        uint8_t* codes = (!big && !compact && bv != 0 && d.K <= 254) ? at<uint8_t>(ctx, L.codes) : nullptr;
        uint4* comp = compact ? at<uint4>(ctx, L.comp) : nullptr;
        {
            Prof prof(ctx, PSL_K_COUNT);
            CU(launch_after(!ctx->profiling, count_otf_fn(pos, edges, bv), n_cols, kThreads, ctx->sm_count_raw, ctx->stream, (const ChunkDesc*)chunks,
                            ctx->n_chunks, span, ctx->grid, bm, d.K, 0u, table, d.cols_cap, ss, ctx->count_stages, codes, comp));
            LAUNCHED();
        }
        // few keys: the table is small and stays raw -- the scatter CTAs scan it themselves (fused_first_slots)
        FusedScan fs;
        memset(&fs, 0, sizeof fs);
        memset(&tail, 0, sizeof tail);
        if (ctx->big_tiles) {  // K <= 256, either tile size
            // ... and the last of them to finish reduces the statistics; both results go straight to the mapped
            // pinned copies the host reads (no reduce launch, no device-to-host copies behind the scatter)
            tail.n_cols = n_cols; tail.ticket = scalar(ctx, SC_TICKET); tail.out = stats; tail.out_host = ctx->d_h_stats;
            fs.batch_offsets_host = ctx->d_h_batch_off;
            to_host = ctx->d_h_stats != nullptr && ctx->d_h_batch_off != nullptr;
            fs.n_cols = n_cols; fs.n_pos = d.n_pos; fs.n_batches = d.n_batches;
            fs.total_out = scalar(ctx, SC_TOTAL); fs.offsets = offsets; fs.counts = counts; fs.batch_offsets = batch_off;
        } else if ((uint64_t)d.K * n_cols <= kScanSmallMax) {  // one small kernel for scan + offsets
            Prof prof(ctx, PSL_K_SCAN);
            k_scan_small<<<1, 1024, 0, ctx->stream>>>(table, n_cols, d.cols_cap, d.K, scalar(ctx, SC_TOTAL), d.K, offsets,
                                                      counts, d.n_pos, d.n_batches, batch_off);
            LAUNCHED();
        } else {
            psl_status s = run_scan(ctx, table, d.K, n_cols, d.cols_cap, scalar(ctx, SC_TOTAL));
            if (s != PSL_OK) return s;
            k_offsets_from_table<<<(d.K + 1 + 255) / 256, 256, 0, ctx->stream>>>(table, d.cols_cap, d.K, scalar(ctx, SC_TOTAL),
                                                                               offsets, counts, d.n_pos, d.n_batches, batch_off);
            LAUNCHED();
        }
        {
            Prof prof(ctx, PSL_K_SCATTER);
            // directly behind the histogram kernel (fused scan, no event bracket): programmatic dependent launch
            const bool overlap = fs.n_cols != 0 && !ctx->profiling;
            const uint32_t* ctable = table;
            const uint8_t* ccodes = codes;
            if (compact)
                CU(launch_after(overlap, proj ? (ScatterCompFn)k_scatter_comp_big<true> : (ScatterCompFn)k_scatter_comp_big<false>, S, kBigThreads,
                                ctx->sm_scatter_comp, ctx->stream, (const uint4*)comp, span, bm, d.K, ctable, d.cols_cap, soa_out(ctx, L.out), ss, fs, tail));
            else if (big)
                CU(launch_after(overlap, scatter_big_fn(pos, edges, bv, proj), S, kBigThreads, ctx->sm_scatter_otf, ctx->stream, (const ChunkDesc*)chunks,
                                ctx->n_chunks, span, ctx->grid, bm, d.K, ctable, d.cols_cap, soa_out(ctx, L.out), ss, fs, tail));
            else
                CU(launch_after(overlap, scatter_otf_fn(pos, edges, bv, proj), S, kThreads, ctx->sm_scatter_small, ctx->stream, (const ChunkDesc*)chunks,
                                ctx->n_chunks, span, ctx->grid, bm, d.K, ctable, d.cols_cap, soa_out(ctx, L.out), ss, ccodes, fs, tail));
            LAUNCHED();
        }
        if (tail.n_cols == 0) {
            k_reduce_stats<<<1, 1024, 0, ctx->stream>>>(ss, n_cols, stats);
            LAUNCHED();
        }
    }
    if (!to_host) {
        CU(cudaMemcpyAsync(ctx->h_batch_off, batch_off, (uint64_t)(d.n_batches + 1) * 4, cudaMemcpyDeviceToHost, ctx->stream));
        CU(cudaMemcpyAsync(ctx->h_stats, stats, sizeof(DevStats), cudaMemcpyDeviceToHost, ctx->stream));
    }
    CU(cudaEventRecord(ctx->ev_batch, ctx->stream));
    ctx->result = RES_OTF;
    return PSL_OK;
}

IdxOut idx_out(psl_ctx* ctx)
{
    const Layout& L = ctx->L;
    IdxOut o;
    o.E = at<float>(ctx, L.idx[0]); o.x = at<float>(ctx, L.idx[1]); o.y = at<float>(ctx, L.idx[2]);
    o.u = at<float>(ctx, L.idx[3]); o.v = at<float>(ctx, L.idx[4]); o.wt = at<float>(ctx, L.idx[5]);
    o.src = at<uint32_t>(ctx, L.idx[6]);
    return o;
}

// INDEX: the one-off sort of every valid in-grid record by the full key ("only needs to be
// performed once per phase-space").  Pass-A counts were taken chunk by chunk in psl_load_chunk.
psl_status finalize_index(psl_ctx* ctx)
{
    const Derived& d = ctx->d;
    const Layout& L = ctx->L;
    uint32_t* idx_offsets = at<uint32_t>(ctx, L.idx_offsets);
    uint32_t* idx_counts = at<uint32_t>(ctx, L.idx_counts);
    uint32_t* idx_batch = at<uint32_t>(ctx, L.idx_batch_off);
    DevStats* stats = at<DevStats>(ctx, L.stats);
    const uint32_t nt = ctx->n_tiles;
    {
        psl_status cs = count_pending_tiles(ctx);  // DEVICE chunks loaded since the last HOST chunk
        if (cs != PSL_OK) return cs;
    }
    if (nt == 0) {
        CU(cudaMemsetAsync(idx_offsets, 0, (uint64_t)(d.K + 1) * 4, ctx->stream));
        CU(cudaMemsetAsync(idx_counts, 0, (uint64_t)d.K * 4, ctx->stream));
        CU(cudaMemsetAsync(idx_batch, 0, (uint64_t)(d.n_batches + 1) * 4, ctx->stream));
        CU(cudaMemsetAsync(stats, 0, sizeof(DevStats), ctx->stream));
        CU(cudaMemsetAsync(scalar(ctx, SC_NIDX), 0, 4, ctx->stream));
    } else {
        DevBeam none;
        memset(&none, 0, sizeof none);
        const ChunkDesc* chunks = at<ChunkDesc>(ctx, L.chunks);
        uint32_t* table_a = at<uint32_t>(ctx, L.table_a);
        uint32_t* table_b = at<uint32_t>(ctx, L.table_b);
        uint4* aos = at<uint4>(ctx, L.aos);
        psl_status s = run_scan(ctx, table_a, d.B_lo, ctx->n_cols, d.cols_cap, scalar(ctx, SC_NIDX));
        if (s != PSL_OK) return s;
        {
            Prof prof(ctx, PSL_K_INDEX_A);
            {
                // ONE launch walks every chunk's span with the segments the counts were taken on
                std::vector<SpanSeg>& hs = ctx->h_spans;  // lives as long as the context: the copy below is asynchronous
                hs.clear();
                uint32_t grid = 1;
                for (const psl_ctx::ChunkLaunch& cl : ctx->idx_launches) {
                    hs.push_back({cl.span, cl.n_seg});
                    if (cl.n_seg > grid) grid = cl.n_seg;
                }
                SpanSeg* d_spans = at<SpanSeg>(ctx, L.spans);
                CU(cudaMemcpyAsync(d_spans, hs.data(), hs.size() * sizeof(SpanSeg), cudaMemcpyHostToDevice, ctx->stream));
                const Span unused = {0u, 0u, 0u, 1u};
                scatter_idx_big_a_fn(ctx->grid.has_pos != 0, ctx->grid.ebin_mode != 0)<<<grid, kIdxBigThreads, ctx->sm_idx_a, ctx->stream>>>(
                    chunks, ctx->n_chunks, d_spans, (uint32_t)hs.size(), unused, nullptr, nullptr, ctx->grid, none, d.B_lo, d.lo_bits, table_a,
                    d.cols_cap, aos);
                LAUNCHED();
            }
        }
        // pass B runs over the n_idx <= n_records keyed records; the device knows n_idx, the host only the bound
        uint32_t ntb = (uint32_t)((ctx->n_records + kTile - 1) / kTile);
        const uint32_t Sb = ntb < ctx->S_b ? ntb : ctx->S_b;
        {
            Prof prof(ctx, PSL_K_COUNT_KEYS);
            k_count_keys<<<Sb * ctx->split_b, kThreads, ctx->sm_count_b, ctx->stream>>>(aos, scalar(ctx, SC_NIDX), d.B_hi, d.lo_bits, table_b,
                                                                                     kMaxSegments, ctx->split_b);
            LAUNCHED();
        }
        if ((uint64_t)d.B_hi * Sb * ctx->split_b <= kScanSmallMax) {
            Prof prof(ctx, PSL_K_SCAN);
            k_scan_small<<<1, 1024, 0, ctx->stream>>>(table_b, Sb * ctx->split_b, kMaxSegments, d.B_hi, scalar(ctx, SC_TOTAL), 0, nullptr, nullptr,
                                                      1, 0, nullptr);
            LAUNCHED();
        } else {
            s = run_scan(ctx, table_b, d.B_hi, Sb * ctx->split_b, kMaxSegments, scalar(ctx, SC_TOTAL));
            if (s != PSL_OK) return s;
        }
        {
            Prof prof(ctx, PSL_K_INDEX_B);
            const Span spb = {0u, 0u, 0u, ctx->split_b};
            scatter_idx_big_b_fn()<<<Sb, kIdxBigThreads, ctx->sm_idx_b, ctx->stream>>>(nullptr, 0, nullptr, 0, spb, aos, scalar(ctx, SC_NIDX), ctx->grid, none,
                                                                                d.B_hi, d.lo_bits, table_b, kMaxSegments,
                                                                                at<uint4>(ctx, L.aos_index));
            LAUNCHED();
        }
        k_offsets_by_search_keyed<<<(d.K + 1 + 255) / 256, 256, 0, ctx->stream>>>(at<uint4>(ctx, L.aos_index), scalar(ctx, SC_NIDX), d.K, idx_offsets);
        LAUNCHED();
        k_counts_from_offsets<<<(d.K + 1 + 255) / 256, 256, 0, ctx->stream>>>(idx_offsets, d.K, idx_counts, d.n_pos, d.n_batches, idx_batch);
        LAUNCHED();
        k_reduce_stats<<<1, 1024, 0, ctx->stream>>>(at<SegStats>(ctx, L.sstats), ctx->n_cols, stats);
        LAUNCHED();
    }
    CU(cudaMemcpyAsync(ctx->h_idx_offsets, idx_offsets, (uint64_t)(d.K + 1) * 4, cudaMemcpyDeviceToHost, ctx->stream));
    CU(cudaMemcpyAsync(ctx->h_stats, stats, sizeof(DevStats), cudaMemcpyDeviceToHost, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));
    ctx->idx_stats = *ctx->h_stats;
    ctx->n_idx = ctx->h_idx_offsets[d.K];
    // the bare index's batch offsets: a host array of their own (h_batch_off is the target of every beam build's
    // asynchronous copy)
    ctx->h_idx_batch_off.resize(d.n_batches + 1);
    for (uint32_t b = 0; b <= d.n_batches; ++b) ctx->h_idx_batch_off[b] = ctx->h_idx_offsets[(uint64_t)b * d.n_pos];
    ctx->indexed = true;
    return PSL_OK;
}

psl_status expose_index(psl_ctx* ctx)
{
    if (!ctx->soa_view && ctx->n_idx > 0) {  // the index is kept as keyed records; the SoA arrays are made on demand
        k_index_to_soa<<<1184, 256, 0, ctx->stream>>>(at<uint4>(ctx, ctx->L.aos_index), scalar(ctx, SC_NIDX), idx_out(ctx));
        LAUNCHED();
        ctx->soa_view = true;
    }
    CU(cudaEventRecord(ctx->ev_batch, ctx->stream));
    ctx->result = RES_INDEX;
    return PSL_OK;
}

psl_status build_beam_from_index(psl_ctx* ctx, const psl_beam* beam, const DevBeam& bm)
{
    const Derived& d = ctx->d;
    const Layout& L = ctx->L;
    const psl_config& c = ctx->cfg;
    int32_t sel[4];
    roi_bins(c, beam, sel);
    const bool empty = sel[0] > sel[1] || sel[2] > sel[3];
    const uint32_t n_rows = empty ? 0u : (uint32_t)(sel[3] - sel[2] + 1);
    const uint32_t n_seg = d.n_batches * n_rows;

    // row segments from the host copy of offsets[]: no device work, no record touched
    if (ctx->seg_pending) {
        CU(cudaEventSynchronize(ctx->ev_seg));
        ctx->seg_pending = false;
    }
    uint32_t* vstart = ctx->h_seg;
    uint32_t* src = ctx->h_seg + (d.max_seg + 1);
    uint32_t* keybase = src + d.max_seg;
    uint64_t M = 0;
    uint32_t sidx = 0;
    for (uint32_t b = 0; b < d.n_batches && !empty; ++b) {
        for (int32_t iy = sel[2]; iy <= sel[3]; ++iy) {
            uint32_t row = (b * (uint32_t)c.n_ybins + (uint32_t)iy) * (uint32_t)c.n_xbins;
            uint32_t lo = ctx->h_idx_offsets[row + (uint32_t)sel[0]];
            uint32_t hi = ctx->h_idx_offsets[row + (uint32_t)sel[1] + 1];
            vstart[sidx] = (uint32_t)M;
            src[sidx] = lo;
            keybase[sidx] = row;
            M += hi - lo;
            ++sidx;
        }
    }
    vstart[n_seg] = (uint32_t)M;
    if (M > d.max_beam) {
        set_err(ctx->err, "beam ROI selects %llu records, more than max_beam_records %llu", (unsigned long long)M, (unsigned long long)d.max_beam);
        return PSL_ERR_CAPACITY;
    }
    uint32_t* d_seg = at<uint32_t>(ctx, L.seg);
    uint32_t* beam_offsets = at<uint32_t>(ctx, L.beam_offsets);
    uint32_t* beam_counts = at<uint32_t>(ctx, L.beam_counts);
    uint32_t* batch_off = at<uint32_t>(ctx, L.batch_off);
    uint32_t* beam_keys = at<uint32_t>(ctx, L.beam_keys);
    DevBeamStats* bstat = at<DevBeamStats>(ctx, L.beam_stats);
    const uint32_t nt = (uint32_t)((M + kBeamTile - 1) / kBeamTile);
    CU(cudaMemsetAsync(scalar(ctx, SC_TILE_COUNTER), 0, 8, ctx->stream));  // tile counter + survivor count
    if (nt == 0) {
        CU(cudaMemsetAsync(bstat, 0, sizeof(DevBeamStats), ctx->stream));
    } else {
        CU(cudaMemcpyAsync(d_seg, ctx->h_seg, (uint64_t)(3 * d.max_seg + 1) * 4, cudaMemcpyHostToDevice, ctx->stream));
        CU(cudaEventRecord(ctx->ev_seg, ctx->stream));
        ctx->seg_pending = true;
        CU(cudaMemsetAsync(at<uint8_t>(ctx, L.lookback), 0, (uint64_t)nt * 8, ctx->stream));
        SegTable st;
        st.vstart = d_seg;
        st.src = d_seg + (d.max_seg + 1);
        st.keybase = st.src + d.max_seg;
        st.n_seg = n_seg;
        st.M = (uint32_t)M;
        IdxIn in;
        in.aos = at<uint4>(ctx, L.aos_index);
        {
            Prof prof(ctx, PSL_K_BEAM);
            k_beam_compact<<<nt, kThreads, 0, ctx->stream>>>(st, in, ctx->grid, bm, soa_out(ctx, L.beam_out), beam_keys,
                                                                         at<unsigned long long>(ctx, L.lookback),
                                                                         scalar(ctx, SC_TILE_COUNTER), at<BeamTileStats>(ctx, L.bstats),
                                                                         scalar(ctx, SC_BEAM_NSURV));
            LAUNCHED();
        }
        k_reduce_beam_stats<<<1, 1024, 0, ctx->stream>>>(at<BeamTileStats>(ctx, L.bstats), nt, bstat);
        LAUNCHED();
    }
    k_offsets_by_search<<<(d.K + 1 + 255) / 256, 256, 0, ctx->stream>>>(beam_keys, scalar(ctx, SC_BEAM_NSURV), d.K, beam_offsets);
    LAUNCHED();
    k_counts_from_offsets<<<(d.K + 1 + 255) / 256, 256, 0, ctx->stream>>>(beam_offsets, d.K, beam_counts, d.n_pos, d.n_batches, batch_off);
    LAUNCHED();
    CU(cudaMemcpyAsync(ctx->h_batch_off, batch_off, (uint64_t)(d.n_batches + 1) * 4, cudaMemcpyDeviceToHost, ctx->stream));
    CU(cudaMemcpyAsync(ctx->h_beam_stats, bstat, sizeof(DevBeamStats), cudaMemcpyDeviceToHost, ctx->stream));
    CU(cudaEventRecord(ctx->ev_batch, ctx->stream));
    ctx->last_M = M;
    ctx->result = RES_BEAM;
    return PSL_OK;
}

psl_status fill_stats(psl_ctx* ctx, psl_stats* st)
{
    if (ctx->result == RES_NONE) { set_err(ctx->err, "no build yet"); return PSL_ERR_STATE; }
    CU(cudaStreamSynchronize(ctx->stream));
    memset(st, 0, sizeof *st);
    st->n_in = ctx->n_records;
    if (ctx->result == RES_OTF) {
        const DevStats& s = *ctx->h_stats;
        st->n_invalid = s.n_invalid; st->n_outside_grid = s.n_outside; st->n_jaw_rejected = s.n_jaw;
        st->n_zero_weight = s.n_zero; st->n_survivors = s.n_surv;
        st->sum_wt_in = s.sum_in; st->sum_wt_indexed = s.sum_idx; st->sum_wt_out = s.sum_out;
    } else {
        const DevStats& s = ctx->idx_stats;
        st->n_invalid = s.n_invalid; st->n_outside_grid = s.n_outside;
        st->sum_wt_in = s.sum_in; st->sum_wt_indexed = s.sum_idx;
        if (ctx->result == RES_INDEX) {
            st->n_survivors = ctx->n_idx;
            st->sum_wt_out = s.sum_idx;
        } else {
            const DevBeamStats& b = *ctx->h_beam_stats;
            st->n_roi_skipped = ctx->n_idx - ctx->last_M;
            st->n_zero_weight = b.n_zero;
            st->n_survivors = b.n_surv;
            st->n_jaw_rejected = ctx->last_M - b.n_zero - b.n_surv;
            st->sum_wt_out = b.sum_out;
        }
    }
    return PSL_OK;
}

}  // namespace

// =================================================================================================
// C-ABI
// =================================================================================================
extern "C" {

uint64_t psl_workspace_bytes(const psl_config* cfg)
{
    Derived d;
    if (derive(cfg, &d, g_err) != PSL_OK) return 0;
    Layout L;
    plan(cfg, d, &L);
    return L.total;
}

const char* psl_last_error(const psl_ctx* ctx) { return ctx ? ctx->err : g_err; }

uint64_t psl_kernel_launches(const psl_ctx* ctx) { return ctx ? ctx->launches : 0; }

void psl_destroy(psl_ctx* ctx)
{
    if (!ctx) return;
    cudaSetDevice(ctx->cfg.device);
    if (ctx->stream) cudaStreamSynchronize(ctx->stream);
    if (ctx->copy_stream) {
        cudaStreamSynchronize(ctx->copy_stream);
        cudaStreamDestroy(ctx->copy_stream);
    }
    cudaEvent_t evs[] = {ctx->ev_chunk, ctx->ev_main, ctx->ev_batch, ctx->ev_seg, ctx->ev_stage[0], ctx->ev_stage[1]};
    for (cudaEvent_t e : evs)
        if (e) cudaEventDestroy(e);
    for (auto& br : ctx->brackets) {
        cudaEventDestroy(br.a);
        cudaEventDestroy(br.b);
    }
    for (cudaEvent_t e : ctx->event_pool) cudaEventDestroy(e);
    void* hp[] = {ctx->h_stage[0], ctx->h_stage[1], ctx->h_batch_off, ctx->h_idx_offsets, ctx->h_seg, ctx->h_stats,
                  ctx->h_beam_stats, ctx->h_scalars, ctx->h_plan, ctx->h_launch_stats, ctx->h_flush_totals};
    for (void* p : hp)
        if (p) cudaFreeHost(p);
    delete ctx;
}

psl_status psl_create(const psl_config* cfg, psl_ctx** out)
{
    if (!out) { set_err(g_err, "out is NULL"); return PSL_ERR_ARG; }
    Derived d;
    psl_status s = derive(cfg, &d, g_err);
    if (s != PSL_OK) return s;
    Layout L;
    plan(cfg, d, &L);
    if (!cfg->workspace || (reinterpret_cast<uintptr_t>(cfg->workspace) & (kAlign - 1))) { set_err(g_err, "config.workspace must be a 256-byte aligned DEVICE pointer"); return PSL_ERR_ARG; }
    if (cfg->workspace_bytes < L.total) { set_err(g_err, "workspace too small: %llu < %llu bytes", (unsigned long long)cfg->workspace_bytes, (unsigned long long)L.total); return PSL_ERR_CAPACITY; }

    psl_ctx* ctx = new (std::nothrow) psl_ctx();
    if (!ctx) { set_err(g_err, "out of host memory"); return PSL_ERR_ARG; }
    ctx->cfg = *cfg;
    ctx->d = d;
    ctx->L = L;
    ctx->ws = static_cast<uint8_t*>(cfg->workspace);
    ctx->stream = static_cast<cudaStream_t>(cfg->stream);
    if (cfg->ebin_mode == PSL_EBIN_EDGES) {
        ctx->edges.assign(cfg->e_edges, cfg->e_edges + cfg->n_ebins + 1);
        ctx->cfg.e_edges = ctx->edges.data();
    } else {
        ctx->cfg.e_edges = nullptr;
    }
    auto fail = [&](psl_status code) {
        memcpy(g_err, ctx->err, sizeof g_err);
        psl_destroy(ctx);
        return code;
    };
#define CUC(call)                                                                                   \
    do {                                                                                            \
        cudaError_t e_ = (call);                                                                    \
        if (e_ != cudaSuccess) {                                                                    \
            set_err(ctx->err, "%s failed: %s", #call, cudaGetErrorString(e_));                      \
            return fail(PSL_ERR_CUDA);                                                              \
        }                                                                                           \
    } while (0)
    CUC(cudaSetDevice(cfg->device));
    CUC(cudaStreamCreateWithFlags(&ctx->copy_stream, cudaStreamNonBlocking));
    cudaEvent_t* evs[] = {&ctx->ev_chunk, &ctx->ev_main, &ctx->ev_batch, &ctx->ev_seg, &ctx->ev_stage[0], &ctx->ev_stage[1]};
    for (cudaEvent_t* e : evs) CUC(cudaEventCreateWithFlags(e, cudaEventDisableTiming));
    CUC(cudaHostAlloc(&ctx->h_batch_off, (uint64_t)(d.n_batches + 1) * 4, cudaHostAllocMapped));
    CUC(cudaHostAlloc(&ctx->h_stats, sizeof(DevStats), cudaHostAllocMapped));
    if (cudaHostGetDevicePointer(&ctx->d_h_stats, ctx->h_stats, 0) != cudaSuccess ||
        cudaHostGetDevicePointer(&ctx->d_h_batch_off, ctx->h_batch_off, 0) != cudaSuccess) {
        (void)cudaGetLastError();
        ctx->d_h_stats = nullptr;
        ctx->d_h_batch_off = nullptr;
    }
    CUC(cudaMemsetAsync(at<uint8_t>(ctx, L.scalars), 0, 64, ctx->stream));
    CUC(cudaHostAlloc(&ctx->h_beam_stats, sizeof(DevBeamStats), cudaHostAllocDefault));
    CUC(cudaHostAlloc(&ctx->h_scalars, 64, cudaHostAllocDefault));
    if (cfg->max_launch_records) {
        CUC(cudaHostAlloc(&ctx->h_plan, (uint64_t)(2 * d.n_batches + 1) * 8, cudaHostAllocDefault));
        CUC(cudaHostAlloc(&ctx->h_launch_stats, sizeof(LaunchStats), cudaHostAllocDefault));
        CUC(cudaHostAlloc(&ctx->h_flush_totals, 8, cudaHostAllocDefault));
    }
    if (cfg->mode == PSL_MODE_INDEX) {
        CUC(cudaHostAlloc(&ctx->h_idx_offsets, (uint64_t)(d.K + 1) * 4, cudaHostAllocDefault));
        CUC(cudaHostAlloc(&ctx->h_seg, (uint64_t)(3 * d.max_seg + 1) * 4, cudaHostAllocDefault));
    }
    float* dev_edges = at<float>(ctx, L.edges);
    if (cfg->ebin_mode == PSL_EBIN_EDGES)
        CUC(cudaMemcpyAsync(dev_edges, ctx->edges.data(), (uint64_t)(cfg->n_ebins + 1) * 4, cudaMemcpyHostToDevice, ctx->stream));
    ctx->grid = make_grid(ctx->cfg, d, dev_edges);

    // dynamic shared memory opt-in, and the launch width: SMs x resident CTAs of the scatter kernel (one wave)
    const uint32_t ne = cfg->n_ebins + 1;
    int sms = 0;
    CUC(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, cfg->device));
    auto width = [&](int occ) {
        uint32_t s = (uint32_t)sms * (uint32_t)(occ > 0 ? occ : 1);
        return s > (uint32_t)kMaxSegments ? (uint32_t)kMaxSegments : s;
    };
    int occ = 0;
    if (cfg->mode == PSL_MODE_ONTHEFLY) {
        ctx->count_stages = d.K * 4 > 8192 ? 2 : kStagesCount;
        ctx->sm_count_raw = count_layout(kTile * kRecBytes, ctx->count_stages, d.K, ne).total;
        ctx->big_tiles = round_up(d.K, 8) <= (uint32_t)kBigMaxKeys;
        ctx->sm_scatter_otf = ctx->big_tiles ? big_layout(d.K, ne).total : part_layout(kTile * kRecBytes, kStagesRaw, d.K, ne, true).total;
        const bool pos = d.n_pos > 1, edges = cfg->ebin_mode == PSL_EBIN_EDGES;
        ctx->sm_scatter_small = part_layout(kTile * kRecBytes, kStagesRaw, d.K, ne, true).total;
        for (int bv = 0; bv < 3; ++bv) {
            CUC(allow_smem(count_otf_fn(pos, edges, bv), ctx->sm_count_raw));
            for (int pj = 0; pj < 2; ++pj) {
                CUC(allow_smem(scatter_otf_fn(pos, edges, bv, pj != 0), ctx->sm_scatter_small));
                if (ctx->big_tiles) CUC(allow_smem(scatter_big_fn(pos, edges, bv, pj != 0), ctx->sm_scatter_otf));
            }
        }
        CUC(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, scatter_otf_fn(pos, edges, 2, true), kThreads, ctx->sm_scatter_small));
        ctx->S_otf_small = width(occ);
        if (ctx->big_tiles) {
            CUC(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, scatter_big_fn(pos, edges, 2, true), kBigThreads, ctx->sm_scatter_otf));
            ctx->S_otf = width(occ);
        }
        ctx->count_split = ctx->big_tiles ? 2 : 1;  // one scatter CTA per SM, two histogram CTAs
        if (ctx->big_tiles && ctx->L.comp != 0 && !(cfg->flags & PSL_NO_COMPACT)) {
            int max_smem = 0;
            CUC(cudaDeviceGetAttribute(&max_smem, cudaDevAttrMaxSharedMemoryPerBlockOptin, cfg->device));
            ctx->sm_scatter_comp = comp_layout(d.K).total;
            if (ctx->sm_scatter_comp + 3072 <= (uint32_t)max_smem) {  // + the kernel's static shared memory
                CUC(allow_smem(k_scatter_comp_big<true>, ctx->sm_scatter_comp));
                CUC(allow_smem(k_scatter_comp_big<false>, ctx->sm_scatter_comp));
                ctx->S_comp = width(1);
                ctx->compact = true;
            }
        }
    } else {
        ctx->count_stages = d.B_lo * 4 > 8192 ? 2 : kStagesCount;
        ctx->sm_count_raw = count_layout(kTile * kRecBytes, ctx->count_stages, d.B_lo, ne).total;
        // the two sort passes: 2048-record tiles, two CTAs per SM when the counters leave room (they do up to ~1900 buckets)
        ctx->split_a = ctx->split_b = kIdxSplit;
        ctx->sm_idx_a = idx_big_layout(false, d.B_lo, ne).total;
        ctx->sm_count_b = count_layout(0, 0, d.B_hi, 0).total;
        ctx->sm_idx_b = idx_big_layout(true, d.B_hi, ne).total;
        const bool pos = d.n_pos > 1, edges = cfg->ebin_mode == PSL_EBIN_EDGES;
        CUC(allow_smem(count_idx_fn(pos, edges), ctx->sm_count_raw));
        CUC(allow_smem(scatter_idx_big_a_fn(pos, edges), ctx->sm_idx_a));
        CUC(allow_smem(k_count_keys, ctx->sm_count_b));
        CUC(allow_smem(scatter_idx_big_b_fn(), ctx->sm_idx_b));
        CUC(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, scatter_idx_big_a_fn(pos, edges), kIdxBigThreads, ctx->sm_idx_a));
        ctx->S_a = width(occ);
        CUC(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, scatter_idx_big_b_fn(), kIdxBigThreads, ctx->sm_idx_b));
        ctx->S_b = width(occ);
    }
    CUC(cudaStreamSynchronize(ctx->stream));
#undef CUC
    *out = ctx;
    return PSL_OK;
}

psl_status psl_reset(psl_ctx* ctx)
{
    if (!ctx) return PSL_ERR_ARG;
    CU(cudaSetDevice(ctx->cfg.device));
    // later host-chunk copies must not overtake kernels of an earlier build that still read the landing zone
    CU(cudaStreamSynchronize(ctx->copy_stream));  // every HOST source buffer has been read: the caller may reuse them
    CU(cudaEventRecord(ctx->ev_main, ctx->stream));
    CU(cudaStreamWaitEvent(ctx->copy_stream, ctx->ev_main, 0));
    ctx->n_records = ctx->n_host_records = 0;
    ctx->n_tiles = ctx->n_chunks = ctx->n_cols = 0;
    ctx->tiles_counted = ctx->cols_bound = 0;
    ctx->idx_launches.clear();
    ctx->pending_chunks.clear();
    ctx->chunks_uploaded = 0;
    ctx->ragged = false;
    ctx->indexed = false;
    ctx->soa_view = false;
    ctx->result = RES_NONE;
    ctx->n_idx = ctx->last_M = 0;
    ctx->plan_set = false;
    return PSL_OK;
}

psl_status psl_wait_loads(psl_ctx* ctx)
{
    if (!ctx) return PSL_ERR_ARG;
    CU(cudaStreamSynchronize(ctx->copy_stream));
    return PSL_OK;
}

psl_status psl_load_chunk(psl_ctx* ctx, const void* records, uint64_t n, int32_t mem_kind)
{
    if (!ctx) return PSL_ERR_ARG;
    if (mem_kind != PSL_MEM_PAGEABLE && mem_kind != PSL_MEM_PINNED && mem_kind != PSL_MEM_DEVICE) { set_err(ctx->err, "load_chunk: bad mem_kind"); return PSL_ERR_ARG; }
    if (n == 0) return PSL_OK;
    if (!records) { set_err(ctx->err, "load_chunk: records is NULL"); return PSL_ERR_ARG; }
    if (ctx->indexed) { set_err(ctx->err, "load_chunk: the index is already finalised; psl_reset first"); return PSL_ERR_STATE; }
    if (ctx->ragged) { set_err(ctx->err, "load_chunk: a chunk whose size is not a multiple of 4 must be the last one"); return PSL_ERR_ARG; }
    if (ctx->n_records + n > ctx->cfg.max_records) { set_err(ctx->err, "load_chunk: more than max_records"); return PSL_ERR_CAPACITY; }
    if (ctx->n_chunks + 1 > ctx->d.max_chunks) { set_err(ctx->err, "load_chunk: more than max_chunks"); return PSL_ERR_CAPACITY; }
    const bool host = mem_kind != PSL_MEM_DEVICE;
    if (host && ctx->n_host_records + n > ctx->cfg.max_host_records) { set_err(ctx->err, "load_chunk: more host records than max_host_records"); return PSL_ERR_CAPACITY; }
    const uint32_t nt = (uint32_t)((n + kTile - 1) / kTile);
    if (ctx->cfg.mode == PSL_MODE_INDEX) {  // checked before anything is enqueued: a failing call leaves the context as it was
        const uint32_t n_seg = nt < ctx->S_a ? nt : ctx->S_a;
        if (ctx->cols_bound + n_seg * ctx->split_a > ctx->d.cols_cap) { set_err(ctx->err, "load_chunk: out of table columns"); return PSL_ERR_CAPACITY; }
        ctx->cols_bound += n_seg * ctx->split_a;  // chunks counted together take no more columns than counted alone
    }
    CU(cudaSetDevice(ctx->cfg.device));

    const uint8_t* dev_ptr;
    if (host) {
        uint8_t* dst = at<uint8_t>(ctx, ctx->L.raw) + ctx->n_host_records * kRecBytes;
        const uint64_t bytes = n * kRecBytes;
        if (mem_kind == PSL_MEM_PINNED) {
            CU(cudaMemcpyAsync(dst, records, bytes, cudaMemcpyHostToDevice, ctx->copy_stream));
        } else {
            // pageable source: double-buffered pinned staging, the CPU copy of piece i+1 overlaps the DMA of piece i
            for (int k = 0; k < 2; ++k)
                if (!ctx->h_stage[k]) CU(cudaHostAlloc(&ctx->h_stage[k], kStageBytes, cudaHostAllocDefault));
            const uint8_t* srcp = static_cast<const uint8_t*>(records);
            for (uint64_t off = 0; off < bytes; off += kStageBytes) {
                uint64_t piece = bytes - off < kStageBytes ? bytes - off : kStageBytes;
                int k = ctx->stage_next;
                CU(cudaEventSynchronize(ctx->ev_stage[k]));
                memcpy(ctx->h_stage[k], srcp + off, piece);
                CU(cudaMemcpyAsync(dst + off, ctx->h_stage[k], piece, cudaMemcpyHostToDevice, ctx->copy_stream));
                CU(cudaEventRecord(ctx->ev_stage[k], ctx->copy_stream));
                ctx->stage_next = k ^ 1;
            }
        }
        CU(cudaEventRecord(ctx->ev_chunk, ctx->copy_stream));
        CU(cudaStreamWaitEvent(ctx->stream, ctx->ev_chunk, 0));
        dev_ptr = dst;
    } else {
        if (reinterpret_cast<uintptr_t>(records) & 3u) { set_err(ctx->err, "load_chunk: DEVICE records must be 4-byte aligned"); return PSL_ERR_ARG; }
        dev_ptr = static_cast<const uint8_t*>(records);
    }

    const uint32_t tile0 = ctx->n_tiles;
    ChunkDesc cd;
    cd.ptr = dev_ptr;
    cd.first_index = (uint32_t)ctx->n_records;
    cd.n_records = (uint32_t)n;
    cd.tile0 = tile0;
    cd.pad = 0;
    ctx->pending_chunks.push_back(cd);  // uploaded 128 at a time by the next launch that reads the chunk table
    ctx->n_records += n;
    if (host) ctx->n_host_records += n;
    ctx->n_tiles += nt;
    ctx->n_chunks += 1;
    if (n % 4) ctx->ragged = true;
    ctx->result = RES_NONE;
    if (ctx->cfg.mode == PSL_MODE_INDEX && host) return count_pending_tiles(ctx);  // overlaps the next chunk's transfer
    return PSL_OK;
}

psl_status psl_build_batches(psl_ctx* ctx, const psl_beam* beam, psl_stats* stats)
{
    if (!ctx) return PSL_ERR_ARG;
    CU(cudaSetDevice(ctx->cfg.device));
    DevBeam bm;
    psl_status s = make_beam(ctx, beam, &bm, ctx->err);
    if (s != PSL_OK) return s;
    if (ctx->cfg.mode == PSL_MODE_ONTHEFLY) {
        s = build_onthefly(ctx, bm);
    } else {
        if (!ctx->indexed) {
            s = finalize_index(ctx);
            if (s != PSL_OK) return s;
        }
        s = beam ? build_beam_from_index(ctx, beam, bm) : expose_index(ctx);
    }
    if (s != PSL_OK) return s;
    if (stats) return fill_stats(ctx, stats);
    return PSL_OK;
}

psl_status psl_get_stats(psl_ctx* ctx, psl_stats* stats)
{
    if (!ctx || !stats) return PSL_ERR_ARG;
    return fill_stats(ctx, stats);
}

psl_status psl_get_tables(psl_ctx* ctx, const uint32_t** counts, const uint32_t** offsets, uint32_t* n_keys)
{
    if (!ctx) return PSL_ERR_ARG;
    if (ctx->result == RES_NONE) { set_err(ctx->err, "get_tables: no build yet"); return PSL_ERR_STATE; }
    const Layout& L = ctx->L;
    uint64_t c = ctx->result == RES_OTF ? L.counts : (ctx->result == RES_INDEX ? L.idx_counts : L.beam_counts);
    uint64_t o = ctx->result == RES_OTF ? L.offsets : (ctx->result == RES_INDEX ? L.idx_offsets : L.beam_offsets);
    if (counts) *counts = at<uint32_t>(ctx, c);
    if (offsets) *offsets = at<uint32_t>(ctx, o);
    if (n_keys) *n_keys = ctx->d.K;
    return PSL_OK;
}

psl_status psl_get_batch(psl_ctx* ctx, int32_t t, int32_t ie, psl_batch* out)
{
    if (!ctx || !out) return PSL_ERR_ARG;
    if (ctx->result == RES_NONE) { set_err(ctx->err, "get_batch: no build yet"); return PSL_ERR_STATE; }
    const bool whole = (t == -1 && ie == -1);
    if (!whole && (t < 0 || t >= ctx->cfg.n_types || ie < 0 || ie >= ctx->cfg.n_ebins)) { set_err(ctx->err, "get_batch: (t, ie) out of range"); return PSL_ERR_ARG; }
    CU(cudaEventSynchronize(ctx->ev_batch));
    const Derived& d = ctx->d;
    const Layout& L = ctx->L;
    uint32_t b = whole ? 0u : (uint32_t)(t * ctx->cfg.n_ebins + ie);
    const uint32_t* boff = ctx->result == RES_INDEX ? ctx->h_idx_batch_off.data() : ctx->h_batch_off;
    uint32_t first = boff[b];
    uint32_t last = boff[whole ? d.n_batches : b + 1];
    memset(out, 0, sizeof *out);
    out->first = first;
    out->count = last - first;
    out->n_bins = whole ? d.K : d.n_pos;
    const bool proj = (ctx->cfg.flags & PSL_OUT_PROJ) != 0;
    if (ctx->result == RES_INDEX) {
        out->E = at<float>(ctx, L.idx[0]) + first; out->x = at<float>(ctx, L.idx[1]) + first; out->y = at<float>(ctx, L.idx[2]) + first;
        out->u = at<float>(ctx, L.idx[3]) + first; out->v = at<float>(ctx, L.idx[4]) + first; out->wt = at<float>(ctx, L.idx[5]) + first;
        out->src_index = at<uint32_t>(ctx, L.idx[6]) + first;
        out->bin_offsets = at<uint32_t>(ctx, L.idx_offsets) + (uint64_t)b * d.n_pos;
    } else {
        const uint64_t* o = ctx->result == RES_OTF ? L.out : L.beam_out;
        out->E = at<float>(ctx, o[0]) + first; out->x = at<float>(ctx, o[1]) + first; out->y = at<float>(ctx, o[2]) + first;
        out->u = at<float>(ctx, o[3]) + first; out->v = at<float>(ctx, o[4]) + first; out->w = at<float>(ctx, o[5]) + first;
        out->wt = at<float>(ctx, o[6]) + first;
        if (proj) {
            out->xp = at<float>(ctx, o[7]) + first;
            out->yp = at<float>(ctx, o[8]) + first;
        }
        out->src_index = at<uint32_t>(ctx, o[9]) + first;
        out->bin_offsets = at<uint32_t>(ctx, ctx->result == RES_OTF ? L.offsets : L.beam_offsets) + (uint64_t)b * d.n_pos;
    }
    return PSL_OK;
}

psl_status psl_profile_enable(psl_ctx* ctx, int32_t on)
{
    if (!ctx) return PSL_ERR_ARG;
    ctx->profiling = on != 0;
    return PSL_OK;
}

psl_status psl_profile_read(psl_ctx* ctx, psl_profile* out)
{
    if (!ctx || !out) return PSL_ERR_ARG;
    CU(cudaSetDevice(ctx->cfg.device));
    CU(cudaStreamSynchronize(ctx->stream));
    memset(out, 0, sizeof *out);
    for (auto& br : ctx->brackets) {
        float ms = 0.0f;
        if (cudaEventElapsedTime(&ms, br.a, br.b) == cudaSuccess) {
            out->ms[br.cls] += (double)ms;
            out->launches[br.cls] += 1;
        }
        ctx->event_pool.push_back(br.a);
        ctx->event_pool.push_back(br.b);
    }
    ctx->brackets.clear();
    return PSL_OK;
}

// patient-frame rotation of a field: Rz(-couch) Ry(gantry) Rz(collimator), formed in double, rounded once
static void field_matrix(const psl_beam& b, float M[9])
{
    const double rad = 3.14159265358979323846 / 180.0;
    const double a[3] = {(double)b.coll_deg * rad, (double)b.gantry_deg * rad, -(double)b.couch_deg * rad};
    double R[3][9];
    for (int i = 0; i < 3; ++i) {
        const double c = cos(a[i]), s_ = sin(a[i]);
        if (i == 1) { const double m[9] = {c, 0, s_, 0, 1, 0, -s_, 0, c}; memcpy(R[i], m, sizeof m); }
        else { const double m[9] = {c, -s_, 0, s_, c, 0, 0, 0, 1}; memcpy(R[i], m, sizeof m); }
    }
    double GC[9], T[9];
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j) {
            GC[3 * i + j] = 0;
            for (int k = 0; k < 3; ++k) GC[3 * i + j] += R[1][3 * i + k] * R[0][3 * k + j];
        }
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j) {
            T[3 * i + j] = 0;
            for (int k = 0; k < 3; ++k) T[3 * i + j] += R[2][3 * i + k] * GC[3 * k + j];
        }
    for (int i = 0; i < 9; ++i) M[i] = (float)T[i];
}

psl_status psl_plan_set(psl_ctx* ctx, const psl_plan* plan, uint64_t* n_total_psl, const uint64_t** list_len)
{
    if (!ctx || !plan) return PSL_ERR_ARG;
    if (plan->struct_size != sizeof(psl_plan)) { set_err(ctx->err, "plan.struct_size %u != %zu", plan->struct_size, sizeof(psl_plan)); return PSL_ERR_ARG; }
    if (ctx->cfg.mode != PSL_MODE_INDEX || ctx->cfg.max_launch_records == 0) { set_err(ctx->err, "plan_set: needs PSL_MODE_INDEX and max_launch_records > 0"); return PSL_ERR_STATE; }
    if (!ctx->indexed) { set_err(ctx->err, "plan_set: build the index first (psl_build_batches)"); return PSL_ERR_STATE; }
    if (plan->n_beams < 1 || plan->n_beams > (uint32_t)kMaxPlanBeams || !plan->beams) { set_err(ctx->err, "plan: 1..%d fields", kMaxPlanBeams); return PSL_ERR_ARG; }
    if (plan->rr_group < 1) { set_err(ctx->err, "plan.rr_group must be >= 1"); return PSL_ERR_ARG; }
    for (int a = 0; a < 3; ++a)
        if (!(isfinite(plan->phantom_lo[a]) && isfinite(plan->phantom_hi[a]) && plan->phantom_lo[a] < plan->phantom_hi[a])) { set_err(ctx->err, "plan: phantom box"); return PSL_ERR_ARG; }
    CU(cudaSetDevice(ctx->cfg.device));
    const Derived& d = ctx->d;
    const Layout& L = ctx->L;
    PlanSel sel;
    memset(&sel, 0, sizeof sel);
    sel.n_beams = plan->n_beams;
    sel.bx0 = ctx->cfg.n_xbins; sel.bx1 = -1; sel.by0 = ctx->cfg.n_ybins; sel.by1 = -1;
    std::vector<PlanBeam> pbs(plan->n_beams);
    for (uint32_t i = 0; i < plan->n_beams; ++i) {
        const psl_beam& b = plan->beams[i];
        if (!(isfinite(b.gantry_deg) && isfinite(b.coll_deg) && isfinite(b.couch_deg))) { set_err(ctx->err, "plan: field %u has a non-finite angle", i); return PSL_ERR_ARG; }
        memset(&pbs[i], 0, sizeof(PlanBeam));
        psl_status ms = make_beam(ctx, &b, &pbs[i].b, ctx->err);
        if (ms != PSL_OK) return ms;
        field_matrix(b, pbs[i].M);
        roi_bins(ctx->cfg, &b, sel.sel[i]);
        if (sel.sel[i][0] <= sel.sel[i][1] && sel.sel[i][2] <= sel.sel[i][3]) {
            sel.bx0 = sel.sel[i][0] < sel.bx0 ? sel.sel[i][0] : sel.bx0; sel.bx1 = sel.sel[i][1] > sel.bx1 ? sel.sel[i][1] : sel.bx1;
            sel.by0 = sel.sel[i][2] < sel.by0 ? sel.sel[i][2] : sel.by0; sel.by1 = sel.sel[i][3] > sel.by1 ? sel.sel[i][3] : sel.by1;
        }
    }
    ctx->h_plan_beams = pbs;  // lives as long as the context: the copy below is asynchronous
    ctx->plan = *plan;
    ctx->plan.beams = nullptr;
    ctx->plan_sel = sel;
    unsigned long long* total = at<unsigned long long>(ctx, L.plan_total);
    CU(cudaMemcpyAsync(at<PlanBeam>(ctx, L.plan_beams), ctx->h_plan_beams.data(), pbs.size() * sizeof(PlanBeam), cudaMemcpyHostToDevice, ctx->stream));
    CU(cudaMemsetAsync(total, 0, 8, ctx->stream));
    {
        Prof prof(ctx, PSL_K_SAMPLE);
        k_plan_total<<<592, 256, 0, ctx->stream>>>(at<uint32_t>(ctx, L.idx_counts), d.K, d.n_pos, (uint32_t)ctx->cfg.n_xbins, sel, total);
        LAUNCHED();
        k_plan_budgets<<<d.n_batches, 256, 0, ctx->stream>>>(at<uint32_t>(ctx, L.idx_counts), d.n_pos, (uint32_t)ctx->cfg.n_xbins, sel,
                                                            (unsigned long long)plan->n_simulate, total, plan->rr_group,
                                                            at<uint32_t>(ctx, L.plan_budget), at<uint32_t>(ctx, L.plan_mask),
                                                            at<unsigned long long>(ctx, L.plan_len), at<unsigned long long>(ctx, L.plan_rounds));
        LAUNCHED();
    }
    CU(cudaMemcpyAsync(ctx->h_plan, total, 8, cudaMemcpyDeviceToHost, ctx->stream));
    CU(cudaMemcpyAsync(ctx->h_plan + 1, at<uint8_t>(ctx, L.plan_len), (uint64_t)d.n_batches * 8, cudaMemcpyDeviceToHost, ctx->stream));
    CU(cudaMemcpyAsync(ctx->h_plan + 1 + d.n_batches, at<uint8_t>(ctx, L.plan_rounds), (uint64_t)d.n_batches * 8, cudaMemcpyDeviceToHost, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));
    ctx->plan_set = true;
    if (n_total_psl) *n_total_psl = ctx->h_plan[0];
    if (list_len) *list_len = reinterpret_cast<const uint64_t*>(ctx->h_plan + 1);
    return PSL_OK;
}

psl_status psl_plan_tables(psl_ctx* ctx, const uint32_t** budget, const uint32_t** mask)
{
    if (!ctx) return PSL_ERR_ARG;
    if (!ctx->plan_set) { set_err(ctx->err, "plan_tables: no plan"); return PSL_ERR_STATE; }
    if (budget) *budget = at<uint32_t>(ctx, ctx->L.plan_budget);
    if (mask) *mask = at<uint32_t>(ctx, ctx->L.plan_mask);
    return PSL_OK;
}

psl_status psl_sample_batch(psl_ctx* ctx, int32_t t, int32_t ie, psl_launch* out)
{
    if (!ctx || !out) return PSL_ERR_ARG;
    if (!ctx->plan_set) { set_err(ctx->err, "sample_batch: psl_plan_set first"); return PSL_ERR_STATE; }
    if (t < 0 || t >= ctx->cfg.n_types || ie < 0 || ie >= ctx->cfg.n_ebins) { set_err(ctx->err, "sample_batch: (t, ie) out of range"); return PSL_ERR_ARG; }
    CU(cudaSetDevice(ctx->cfg.device));
    const Derived& d = ctx->d;
    const Layout& L = ctx->L;
    const uint32_t b = (uint32_t)(t * ctx->cfg.n_ebins + ie);
    const unsigned long long len = ctx->h_plan[1 + b], rounds = ctx->h_plan[1 + d.n_batches + b];
    if (len > ctx->cfg.max_launch_records) {
        set_err(ctx->err, "sample_batch: the launch list has %llu entries, more than max_launch_records %llu", len, (unsigned long long)ctx->cfg.max_launch_records);
        return PSL_ERR_CAPACITY;
    }
    memset(out, 0, sizeof *out);
    LaunchStats* stats = at<LaunchStats>(ctx, L.l_stats);
    uint32_t* counter = reinterpret_cast<uint32_t*>(stats + 1);
    uint32_t* slot = at<uint32_t>(ctx, L.l_slot);
    uint8_t* beam = at<uint8_t>(ctx, L.l_beam);
    CU(cudaMemsetAsync(stats, 0, sizeof(LaunchStats) + 16, ctx->stream));
    if (len > 0) {
        const PlanSel& sel = ctx->plan_sel;
        const uint32_t nt = (uint32_t)((len + kEmitTile - 1) / kEmitTile);
        CU(cudaMemsetAsync(at<uint8_t>(ctx, L.l_state), 0, (uint64_t)nt * 8, ctx->stream));
        LaunchOut lo;
        lo.E = at<float>(ctx, L.l_out[0]); lo.X = at<float>(ctx, L.l_out[1]); lo.Y = at<float>(ctx, L.l_out[2]); lo.Z = at<float>(ctx, L.l_out[3]);
        lo.U = at<float>(ctx, L.l_out[4]); lo.V = at<float>(ctx, L.l_out[5]); lo.W = at<float>(ctx, L.l_out[6]); lo.wt = at<float>(ctx, L.l_out[7]);
        lo.src = at<uint32_t>(ctx, L.l_src); lo.beam = at<uint8_t>(ctx, L.l_beam_of);
        PhantomBox box;
        for (int a = 0; a < 3; ++a) { box.lo[a] = ctx->plan.phantom_lo[a]; box.hi[a] = ctx->plan.phantom_hi[a]; }
        Prof prof(ctx, PSL_K_SAMPLE);
        const uint32_t grid = (uint32_t)(rounds < 1184ull ? rounds : 1184ull);
        k_sample_batch<<<grid, 256, 0, ctx->stream>>>(at<uint32_t>(ctx, L.idx_counts), at<uint32_t>(ctx, L.idx_offsets),
                                                      at<uint32_t>(ctx, L.plan_budget), at<uint32_t>(ctx, L.plan_mask), b * d.n_pos,
                                                      (uint32_t)ctx->cfg.n_xbins, sel.bx0, sel.bx1, sel.by0, sel.by1, ctx->plan.rr_group,
                                                      (unsigned long long)ctx->plan.seed, at<unsigned long long>(ctx, L.plan_rounds) + b,
                                                      slot, beam);
        LAUNCHED();
        k_emit<<<nt, kThreads, 0, ctx->stream>>>(at<uint4>(ctx, L.aos_index), slot, beam, (uint32_t)len, at<PlanBeam>(ctx, L.plan_beams),
                                                 ctx->plan.n_beams, ctx->cfg.geom.z_iso - ctx->cfg.geom.z_plane,
                                                 (ctx->cfg.flags & PSL_DROP_ZERO_WEIGHT) ? 1u : 0u, box, lo,
                                                 at<unsigned long long>(ctx, L.l_state), counter, stats);
        LAUNCHED();
        out->slot = slot; out->beam = beam;
        out->E = lo.E; out->X = lo.X; out->Y = lo.Y; out->Z = lo.Z; out->U = lo.U; out->V = lo.V; out->W = lo.W; out->wt = lo.wt;
        out->src_index = lo.src; out->beam_of = lo.beam;
    }
    CU(cudaMemcpyAsync(ctx->h_launch_stats, stats, sizeof(LaunchStats), cudaMemcpyDeviceToHost, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));
    out->n_list = (uint32_t)len;
    out->n_launch = (uint32_t)ctx->h_launch_stats->n_launched;
    out->n_jaw_rejected = ctx->h_launch_stats->n_jaw;
    out->n_zero_weight = ctx->h_launch_stats->n_zero;
    out->n_missed = ctx->h_launch_stats->n_missed;
    return PSL_OK;
}

psl_status psl_flush_schedule(psl_ctx* ctx, uint32_t capacity, psl_flush* out)
{
    if (!ctx || !out) return PSL_ERR_ARG;
    if (ctx->cfg.mode != PSL_MODE_ONTHEFLY || ctx->cfg.max_launch_records == 0) { set_err(ctx->err, "flush_schedule: needs PSL_MODE_ONTHEFLY and max_launch_records > 0"); return PSL_ERR_STATE; }
    if (ctx->result != RES_OTF) { set_err(ctx->err, "flush_schedule: no build yet"); return PSL_ERR_STATE; }
    if (capacity < 1) { set_err(ctx->err, "flush_schedule: capacity must be >= 1"); return PSL_ERR_ARG; }
    CU(cudaSetDevice(ctx->cfg.device));
    const Derived& d = ctx->d;
    const Layout& L = ctx->L;
    const uint32_t cap = (uint32_t)ctx->cfg.max_launch_records;
    uint32_t* totals = at<uint32_t>(ctx, L.f_totals);
    FlushOut fo = {at<uint32_t>(ctx, L.f_key), at<uint32_t>(ctx, L.f_first), at<uint32_t>(ctx, L.f_count)};
    {
        Prof prof(ctx, PSL_K_OTHER);
        k_flush_plan<<<1, 1024, 0, ctx->stream>>>(at<uint32_t>(ctx, L.counts), d.K, capacity, at<uint32_t>(ctx, L.f_full), at<uint32_t>(ctx, L.f_part), totals);
        LAUNCHED();
        k_flush_events<<<d.K < 592u ? d.K : 592u, 256, 0, ctx->stream>>>(at<uint32_t>(ctx, L.counts), at<uint32_t>(ctx, L.offsets), at<uint32_t>(ctx, L.out[9]),
                                                                          d.K, capacity, at<uint32_t>(ctx, L.f_full), at<uint32_t>(ctx, L.f_part), totals, cap,
                                                                          at<uint32_t>(ctx, L.f_trig), at<uint32_t>(ctx, L.f_tkey), at<uint32_t>(ctx, L.f_tfirst), fo);
        LAUNCHED();
        k_flush_order<<<592, 256, 0, ctx->stream>>>(at<uint32_t>(ctx, L.f_trig), at<uint32_t>(ctx, L.f_tkey), at<uint32_t>(ctx, L.f_tfirst), totals, cap, capacity, fo);
        LAUNCHED();
    }
    CU(cudaMemcpyAsync(ctx->h_flush_totals, totals, 8, cudaMemcpyDeviceToHost, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));
    const unsigned long long ne = (unsigned long long)ctx->h_flush_totals[0] + ctx->h_flush_totals[1];
    if (ne > cap) { set_err(ctx->err, "flush_schedule: %llu shipments, more than max_launch_records %u", ne, cap); return PSL_ERR_CAPACITY; }
    out->n_events = (uint32_t)ne;
    out->key = fo.key; out->first = fo.first; out->count = fo.count;
    return PSL_OK;
}

psl_status psl_roi_bins(const psl_ctx* ctx, const psl_beam* beam, int32_t bins_out[4])
{
    if (!ctx || !bins_out) return PSL_ERR_ARG;
    roi_bins(ctx->cfg, beam, bins_out);
    return PSL_OK;
}

psl_status psl_roi_from_jaws(const psl_geometry* g, const psl_beam* beam, float margin, float roi_out[4])
{
    if (!g || !beam || !roi_out) { set_err(g_err, "roi_from_jaws: NULL argument"); return PSL_ERR_ARG; }
    psl_status s = check_geometry(*g, g_err);
    if (s != PSL_OK) return s;
    if (!(g->z_jaw_x < g->z_iso && g->z_jaw_y < g->z_iso)) { set_err(g_err, "roi_from_jaws: jaw planes must be upstream of the isocentre"); return PSL_ERR_GEOMETRY; }
    const double zj[2] = {g->z_jaw_x, g->z_jaw_y};
    const double e1[2] = {beam->jaw_x1, beam->jaw_y1}, e2[2] = {beam->jaw_x2, beam->jaw_y2};
    for (int a = 0; a < 2; ++a) {
        // the line from the field centre at z_iso through the jaw edge, extended up to z_plane
        double to_jaw = (zj[a] - (double)g->z_src) / ((double)g->z_iso - (double)g->z_src);
        double mid = 0.5 * (e1[a] + e2[a]);
        double reach = ((double)g->z_iso - (double)g->z_plane) / ((double)g->z_iso - zj[a]);
        roi_out[2 * a + 0] = (float)(mid + (e1[a] * to_jaw - mid) * reach - (double)margin);
        roi_out[2 * a + 1] = (float)(mid + (e2[a] * to_jaw - mid) * reach + (double)margin);
    }
    return PSL_OK;
}

}  // extern "C"

// ---------------------------------------------------------------------------------------------------------------------
// psl_count_static: the entry point that allocates nothing (include/psl.h).  Its scratch is this file-scope array, part
// of the library image on every GPU that loads it.  In HOST code the name below is only a stand-in for the symbol, not a
// device address: the address is looked up once per device with cudaGetSymbolAddress (that device current) and the
// kernels get it as an argument.
// ---------------------------------------------------------------------------------------------------------------------
static __device__ __align__(256) unsigned char g_static_scratch[kStaticBytes];
static_assert(kStaticBytes == PSL_STATIC_SCRATCH_BYTES && kStaticMaxKeys == PSL_STATIC_MAX_KEYS, "psl.h states the limits");

namespace {

struct StaticDev {
    bool ready = false;
    uint8_t* scratch = nullptr;  // DEVICE address of g_static_scratch on this device
    int sms = 0;
};
constexpr int kStaticMaxDevices = 64;
StaticDev g_static_dev[kStaticMaxDevices];
std::mutex g_static_mu;

using CountStaticFn = void (*)(const uint8_t*, uint32_t, DevGrid, uint32_t, uint32_t*, uint32_t, SegStats*);
CountStaticFn count_static_fn(bool pos, bool edges)
{
    return pos ? (edges ? k_count_static<true, true> : k_count_static<true, false>)
               : (edges ? k_count_static<false, true> : k_count_static<false, false>);
}

#define CUS(call)                                                                                       \
    do {                                                                                                \
        cudaError_t e_ = (call);                                                                        \
        if (e_ != cudaSuccess) {                                                                        \
            set_err(g_err, "psl_count_static: %s failed: %s", #call, cudaGetErrorString(e_));           \
            return PSL_ERR_CUDA;                                                                        \
        }                                                                                               \
    } while (0)

// once per device, with that device current
psl_status static_setup(int device, StaticDev* out)
{
    std::lock_guard<std::mutex> lock(g_static_mu);
    StaticDev& sd = g_static_dev[device];
    if (!sd.ready) {
        void* p = nullptr;
        CUS(cudaGetSymbolAddress(&p, g_static_scratch));
        if (!p || (reinterpret_cast<uintptr_t>(p) & (kAlign - 1))) { set_err(g_err, "psl_count_static: bad scratch address"); return PSL_ERR_CUDA; }
        CUS(cudaDeviceGetAttribute(&sd.sms, cudaDevAttrMultiProcessorCount, device));
        // the most dynamic shared memory any configuration takes: three stages, a 16 KB histogram, 1025 edges
        const uint32_t smem_max = count_layout(kTile * kRecBytes, kStagesCount, kStaticMaxKeys, kStaticMaxEdges).total;
        for (int v = 0; v < 4; ++v) CUS(allow_smem(count_static_fn((v & 1) != 0, (v & 2) != 0), smem_max));
        sd.scratch = static_cast<uint8_t*>(p);
        sd.ready = true;
    }
    *out = sd;
    return PSL_OK;
}

}  // namespace

extern "C" psl_status psl_count_static(const psl_config* cfg, const void* records, uint64_t n, uint32_t* counts, psl_count_totals* totals)
{
    static_assert(sizeof(psl_count_totals) == sizeof(CountTotals), "psl_count_totals layout");
    if (!cfg) { set_err(g_err, "psl_count_static: config is NULL"); return PSL_ERR_ARG; }
    if (cfg->struct_size != sizeof(psl_config)) { set_err(g_err, "config.struct_size %u != %zu", cfg->struct_size, sizeof(psl_config)); return PSL_ERR_ARG; }
    if (n >= (1ull << 32)) { set_err(g_err, "psl_count_static: %llu records; one call takes fewer than 2^32", (unsigned long long)n); return PSL_ERR_CAPACITY; }
    if (cfg->n_types >= 1 && cfg->n_ebins >= 1 && cfg->n_xbins >= 1 && cfg->n_ybins >= 1) {
        const uint64_t K64 = (uint64_t)cfg->n_types * (uint64_t)cfg->n_ebins * (uint64_t)cfg->n_xbins * (uint64_t)cfg->n_ybins;
        if (K64 > kStaticMaxKeys) {
            set_err(g_err, "psl_count_static: %llu keys; the static scratch holds at most %u (use a context in PSL_MODE_INDEX)",
                    (unsigned long long)K64, kStaticMaxKeys);
            return PSL_ERR_CAPACITY;
        }
    }
    psl_config c = *cfg;  // the grid checks of psl_create, on a configuration that asks for nothing else
    c.mode = PSL_MODE_ONTHEFLY;
    c.max_records = n ? n : 1;
    c.max_host_records = 0;
    c.max_beam_records = 0;
    c.max_chunks = 1;
    c.flags = 0;
    c.max_launch_records = 0;
    Derived d;
    psl_status s = derive(&c, &d, g_err);
    if (s != PSL_OK) return s;
    if (!counts) { set_err(g_err, "psl_count_static: counts is NULL"); return PSL_ERR_ARG; }
    if (n != 0 && (!records || (reinterpret_cast<uintptr_t>(records) & 3u))) { set_err(g_err, "psl_count_static: records must be a 4-byte aligned DEVICE pointer"); return PSL_ERR_ARG; }
    if (cfg->device < 0 || cfg->device >= kStaticMaxDevices) { set_err(g_err, "psl_count_static: config.device"); return PSL_ERR_ARG; }
    CUS(cudaSetDevice(cfg->device));
    StaticDev sd;
    s = static_setup(cfg->device, &sd);
    if (s != PSL_OK) return s;

    cudaStream_t stream = static_cast<cudaStream_t>(cfg->stream);
    float* dev_edges = reinterpret_cast<float*>(sd.scratch + kStaticEdgesOff);
    SegStats* ss = reinterpret_cast<SegStats*>(sd.scratch + kStaticStatsOff);
    uint32_t* table = reinterpret_cast<uint32_t*>(sd.scratch + kStaticTableOff);
    const bool edges = cfg->ebin_mode == PSL_EBIN_EDGES;
    const uint32_t nt = (uint32_t)((n + kTile - 1) / kTile);
    uint32_t S = 2u * (uint32_t)sd.sms;  // two resident CTAs per SM: one wave
    if (S > kStaticMaxCols) S = kStaticMaxCols;
    if (S > nt) S = nt;
    if (S != 0) {
        if (edges) {
            const uint32_t ne = (uint32_t)cfg->n_ebins + 1u;
            for (uint32_t f = 0; f < ne; f += 512) {
                EdgeBatch eb;
                const uint32_t m = ne - f < 512u ? ne - f : 512u;
                memcpy(eb.e, cfg->e_edges + f, m * sizeof(float));
                k_static_edges<<<1, 256, 0, stream>>>(dev_edges, eb, f, m);
                CUS(cudaGetLastError());
            }
        }
        const DevGrid grid = make_grid(c, d, dev_edges);
        const uint32_t smem = count_layout(kTile * kRecBytes, kStagesCount, d.K, (uint32_t)cfg->n_ebins + 1u).total;
        count_static_fn(grid.has_pos != 0, edges)<<<S, kThreads, smem, stream>>>(static_cast<const uint8_t*>(records), (uint32_t)n, grid, d.K,
                                                                                table, kStaticMaxCols, ss);
        CUS(cudaGetLastError());
    }
    k_static_sum<<<(d.K + 7) / 8 + 1, 256, 0, stream>>>(table, kStaticMaxCols, S, d.K, ss, (unsigned long long)n, counts,
                                                        reinterpret_cast<CountTotals*>(totals));
    CUS(cudaGetLastError());
    return PSL_OK;
}
