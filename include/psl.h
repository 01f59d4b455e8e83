/*
 * psl.h -- C-ABI of the B200 phase-space source library (libpsl_b200.so).
 *
 * The data-parallel hot path of Townson et al., "GPU-based Monte Carlo radiotherapy dose
 * calculation using phase-space sources" (arXiv 1302.1861; PAPER.md = /root/reference/PAPER.md):
 * packed linac phase-space records are loaded in chunks (sec. 2.3.3), decoded,
 * tested against the secondary-collimator (jaw) model (sec. 2.2), weighted by the
 * fluence map, culled by the phase-space-let (PSL) region of interest
 * and bucketed by particle type, energy bin and position bin
 * into contiguous structure-of-arrays batches, "one energy division before proceeding to the
 * next".  Every step runs in CUDA kernels for sm_100a; there is no CPU path.
 *
 * Conventions
 *   - Plain C, no torch types.  Every pointer says HOST or DEVICE.
 *   - Beam's-eye-view frame: beam axis +z through (0,0); lengths in cm, energies in MeV.
 *   - All work is enqueued on psl_config.stream (plus one internal copy stream ordered to it with
 *     events).  Calls return once the work is enqueued unless stated otherwise.
 *   - Errors are return codes; nothing aborts, nothing throws, and a call that fails leaves the
 *     context as it was before the call.  psl_last_error() gives a one-line description.
 *   - A context is not thread-safe.  Total records per context < 2^32.
 *   - Every call that touches the device makes psl_config.device the calling thread's current CUDA device and leaves
 *     it current.
 *
 * Arithmetic contract: every expression that decides a bin, a key, the jaw
 * predicate or a map pixel is evaluated in fp32, one IEEE-754 round-to-nearest operation at a
 * time, with no FMA contraction; outputs E, x, y, u, v are bit copies of the inputs.
 */
#ifndef PSL_H
#define PSL_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct psl_ctx psl_ctx; /* opaque; one per phase-space */

typedef enum {
    PSL_OK = 0,
    PSL_ERR_ARG = 1,      /* bad argument or configuration */
    PSL_ERR_STATE = 2,    /* call out of order (e.g. psl_get_batch before psl_build_batches) */
    PSL_ERR_CAPACITY = 3, /* workspace too small, or more records / chunks than configured */
    PSL_ERR_GEOMETRY = 4, /* planes out of order */
    PSL_ERR_CUDA = 5      /* a CUDA runtime call failed; see psl_last_error() */
} psl_status;

enum { PSL_MODE_ONTHEFLY = 0, /* paper methods 1 and 2: sort on the fly by (type, energy) */
       PSL_MODE_INDEX = 1 };  /* paper method 3: pre-sorted PSL index, per-beam ROI selection */
enum { PSL_EBIN_LINEAR = 0,   /* n_ebins uniform bins on [e_min, e_max] */
       PSL_EBIN_EDGES = 1 };  /* caller-supplied ascending edge table with n_ebins+1 entries */
enum { PSL_MEM_PAGEABLE = 0, PSL_MEM_PINNED = 1, PSL_MEM_DEVICE = 2 };
enum { PSL_OUT_PROJ = 1u,           /* also write xp, yp: the position at the fluence-map plane */
       PSL_DROP_ZERO_WEIGHT = 2u,   /* drop survivors whose final weight is exactly 0 (default: keep) */
       PSL_NO_COMPACT = 4u,         /* diagnostic, same results: ONTHEFLY with <= 256 keys and a rejecting beam takes the
                                       two-pass path (histogram, then scatter over all records) instead of compacting
                                       the survivors in the histogram pass; used for A/B runs and tests */
       PSL_APR = 8u };              /* INDEX mode: azimuthal particle redistribution of every record
                                       before it is binned: record i of the load order turns about the beam axis by
                                       2 pi r / 2^32, r from psl_config.apr_seed and i; position and direction together */

/* One phase-space particle: 28 bytes, packed, little-endian.  type: 0 photon, 1 electron, 2 positron.
 * (u, v) are direction cosines; the third one is w = sqrt(1 - u^2 - v^2) > 0 (always downstream). */
typedef struct {
    int32_t type;
    float E, x, y, u, v, wt;
} psl_record;

/* z of each plane along the beam axis.  Must satisfy z_src < z_plane <= z_jaw_x, z_jaw_y, z_map <= z_iso. */
typedef struct {
    float z_src, z_plane, z_jaw_x, z_jaw_y, z_map, z_iso;
} psl_geometry;

typedef struct {
    uint32_t struct_size; /* sizeof(psl_config), checked */
    int32_t mode;         /* PSL_MODE_* */
    int32_t n_types;      /* 3, or 2 = electrons and positrons share a division */
    int32_t ebin_mode;    /* PSL_EBIN_* */
    int32_t n_ebins;
    float e_min, e_max;
    const float* e_edges; /* HOST, n_ebins+1 ascending floats, copied by psl_create; NULL in linear mode */
    int32_t n_xbins, n_ybins; /* 1 x 1 = no position bins (methods 1 and 2) */
    float x_min, y_min, dx, dy; /* grid origin and bin size at z_plane; x_min/dx and y_min/dy must be integers */
    psl_geometry geom;
    uint64_t max_records;      /* capacity: total records loaded between resets */
    uint64_t max_host_records; /* of those, how many may arrive from HOST memory (device landing zone) */
    uint64_t max_beam_records; /* INDEX mode: most records one beam's ROI may select; 0 = max_records */
    uint32_t max_chunks;       /* most psl_load_chunk calls between resets; 0 = 4096 */
    uint32_t flags;            /* PSL_OUT_PROJ | PSL_DROP_ZERO_WEIGHT | PSL_NO_COMPACT | PSL_APR */
    uint64_t apr_seed;         /* PSL_APR: seed of the redistribution angles */
    uint64_t max_launch_records; /* INDEX mode: longest launch list psl_sample_batch may build (0 = sampling layer unused);
                                    ONTHEFLY mode: most bin shipments psl_flush_schedule may report (0 = unused) */
    int32_t device;            /* CUDA device ordinal */
    void* stream;              /* cudaStream_t owned by the caller (NULL = default stream) */
    void* workspace;           /* DEVICE memory owned by the caller, 256-byte aligned */
    uint64_t workspace_bytes;  /* >= psl_workspace_bytes(cfg) */
} psl_config;

/* One treatment field.  NULL beam = method 1: no jaws, no map, weight untouched. */
typedef struct {
    int32_t has_jaws;
    float jaw_x1, jaw_x2, jaw_y1, jaw_y2; /* aperture [x1,x2) x [y1,y2) as projected at z_iso */
    const float* fluence;                 /* DEVICE, map_ny x map_nx row-major fp32, or NULL = no map */
    int32_t map_nx, map_ny;
    float map_x0, map_y0, map_dx, map_dy; /* pixel grid at z_map; map_x0/map_dx, map_y0/map_dy integers */
    int32_t has_roi;                      /* INDEX mode only */
    float roi_x1, roi_x2, roi_y1, roi_y2; /* rectangle at z_plane */
    float mu_weight;                      /* MU_i / MU_total */
    float gantry_deg, coll_deg, couch_deg; /* the field's rotations: used by psl_sample_batch, ignored by
                                              psl_build_batches (whose batches stay in the beam's-eye-view frame) */
} psl_beam;

/* Every record loaded is counted in exactly one of the six n_* classes below (tested in this order). */
typedef struct {
    uint64_t n_in;
    uint64_t n_invalid;      /* type not in {0,1,2}, a non-finite field, E <= 0, or u^2+v^2 >= 1 */
    uint64_t n_outside_grid; /* valid, but outside the position grid */
    uint64_t n_roi_skipped;  /* in a position bin the ROI does not select (their records are never read) */
    uint64_t n_jaw_rejected; /* hit a jaw */
    uint64_t n_zero_weight;  /* dropped because of PSL_DROP_ZERO_WEIGHT */
    uint64_t n_survivors;
    double sum_wt_in;      /* sum of wt over valid records */
    double sum_wt_indexed; /* sum of wt over valid records inside the grid */
    double sum_wt_out;     /* sum of final weights over survivors */
} psl_stats;

/* A contiguous run of output slots.  All pointers are DEVICE, BORROWED from the workspace and valid
 * until the next psl_build_batches / psl_reset / psl_destroy on the context.  Each array pointer
 * addresses slot `first` (i.e. element 0 of the batch).  Slots are ordered by key
 * key = ((t * n_ebins + ie) * n_ybins + iy) * n_xbins + ix, input order inside a key. */
typedef struct {
    uint32_t first;  /* absolute slot of the first element */
    uint32_t count;
    const float *E, *x, *y, *u, *v; /* bit copies of the record fields */
    const float* w;                 /* sqrt(1-u^2-v^2); NULL for the bare index */
    const float* wt;                /* final weight (wt * F) * mu_weight; the record's wt for the bare index */
    const float *xp, *yp;           /* position at z_map; NULL unless PSL_OUT_PROJ */
    const uint32_t* src_index;      /* load-order index of the record */
    const uint32_t* bin_offsets;    /* n_bins+1 ABSOLUTE slot offsets of this batch's position bins */
    uint32_t n_bins;                /* n_xbins * n_ybins */
} psl_batch;

/* Limits.  K = n_types * n_ebins * n_xbins * n_ybins keys.  PSL_MODE_ONTHEFLY: K <= 2048 (one partition pass;
 * K <= 256 takes the 4096-record-tile scatter).  PSL_MODE_INDEX: K <= 2048 * 2048 (two passes over two balanced
 * digits of the key).  n_ebins <= 1024, n_xbins, n_ybins <= 4096, fewer than 2^32 records per context.  Anything
 * beyond is PSL_ERR_ARG from psl_workspace_bytes (0) / psl_create. */

/* Bytes of device workspace a configuration needs (cfg->workspace* ignored).  0 on a bad configuration. */
uint64_t psl_workspace_bytes(const psl_config* cfg);

/* Validate, copy the configuration, carve the workspace.  May allocate small pinned HOST buffers and one
 * CUDA stream + a few events.  *out is untouched on error (the reason is then readable with
 * psl_last_error(NULL)). */
psl_status psl_create(const psl_config* cfg, psl_ctx** out);

/* Append n records ("particle data are copied in chunks").  `records` is HOST pageable, HOST
 * pinned or DEVICE memory per mem_kind.  n must be a multiple of 4 except for the last chunk loaded before
 * psl_reset (PSL_ERR_ARG for any chunk after it).  HOST chunks are copied on the internal copy stream into the workspace (pageable ones through two
 * pinned staging buffers); the source must stay untouched until psl_wait_loads() or any later
 * synchronising call returns.  DEVICE chunks are BORROWED, not copied: they must stay valid and unchanged
 * until the next psl_reset/psl_destroy (ONTHEFLY) or until the index is finalised (INDEX).  In INDEX mode
 * a HOST chunk's keys are counted as soon as it lands, overlapping the next chunk's transfer; DEVICE chunks are
 * counted together by one launch when the next HOST chunk arrives or the index is finalised. */
psl_status psl_load_chunk(psl_ctx* ctx, const void* records, uint64_t n, int32_t mem_kind);

/* Block the HOST until every chunk loaded so far has left its source buffer. */
psl_status psl_wait_loads(psl_ctx* ctx);

/* ONTHEFLY: decode every loaded record, apply the beam's jaws / fluence map / MU weight, histogram,
 * scan and stably scatter the survivors by (type, energy[, position]) key.  May be called again with a
 * different beam.  INDEX: the first call finalises the index (sort of all valid in-grid records by the
 * full key; synchronises once); with beam != NULL it then builds that beam's batches from the index,
 * reading only the position bins the ROI selects.  beam == NULL exposes the index itself.
 * stats may be NULL; if not, the call synchronises the stream and fills it. */
psl_status psl_build_batches(psl_ctx* ctx, const psl_beam* beam, psl_stats* stats);

/* Synchronise and report the statistics of the latest build. */
psl_status psl_get_stats(psl_ctx* ctx, psl_stats* stats);

/* The (type division t, energy bin ie) batch of the latest build; t = ie = -1 gives the whole output as
 * one run.  Waits for the (tiny) batch-offset copy of that build, not for the whole stream. */
psl_status psl_get_batch(psl_ctx* ctx, int32_t t, int32_t ie, psl_batch* out);

/* DEVICE pointers to counts[K] and offsets[K+1] of the latest build. */
psl_status psl_get_tables(psl_ctx* ctx, const uint32_t** counts, const uint32_t** offsets, uint32_t* n_keys);

/* HOST only.  ROI rectangle {x1, x2, y1, y2} at z_plane for a beam's jaws (Fig. 1 caption
 * PAPER.md:196): per axis, the line from the field centre at z_iso through the jaw edge at the jaw plane,
 * extended to z_plane, widened by `margin`.  PSL_ERR_GEOMETRY unless z_jaw < z_iso on both axes. */
psl_status psl_roi_from_jaws(const psl_geometry* g, const psl_beam* beam, float margin, float roi_out[4]);

/* HOST only.  The inclusive rectangle {rx0, rx1, ry0, ry1} of position bins with positive-area overlap with
 * the beam's ROI ("any portion of its area"); rx0 > rx1 or ry0 > ry1 when nothing is selected. */
psl_status psl_roi_bins(const psl_ctx* ctx, const psl_beam* beam, int32_t bins_out[4]);

/* ---- From the index to transport launches (sec. 2.3.3) -------------------
 * A plan = the fields of a treatment plan + how many particles to simulate.  psl_plan_set gives every selected PSL its
 * share; psl_sample_batch then builds, for one (type, energy) division, the launch list (which index particle, for
 * which field, in the order the paper's reading loop visits them) and turns it into transport-ready particles. */
typedef struct {
    uint32_t struct_size;  /* sizeof(psl_plan), checked */
    uint32_t n_beams;      /* 1..32 */
    const psl_beam* beams; /* HOST array of n_beams fields, copied by psl_plan_set; their fluence maps are DEVICE
                              memory of the caller and must stay valid for as long as the plan is sampled from */
    uint64_t n_simulate;   /* N_total^simulated: particles to simulate over all fields */
    uint64_t seed;         /* of the random starts and field assignments; give every GPU of a job its own */
    uint32_t rr_group;     /* particles read from a PSL at a time ("a few"); >= 1 */
    uint32_t reserved;     /* 0 */
    float phantom_lo[3], phantom_hi[3]; /* the patient phantom: an axis-aligned box in the patient frame, cm, origin at
                                           the isocentre.  Patient frame: p = Rz(-couch) Ry(gantry) Rz(collimator) p_b with
                                           p_b = (x, y, z_iso - z_plane), direction (u, v, -w) (reading S5) */
} psl_plan;

/* Budgets: N_total^psl = sum over fields of the particles in the PSLs each selects; every selected PSL k
 * gives floor(n_simulate * counts[k] / N_total^psl) particles to EACH field that selects it.  Needs a finalised index
 * (psl_build_batches once).  Synchronises.  *n_total_psl and *list_len (HOST, n_types * n_ebins entries owned by the
 * context, valid until the next psl_plan_set / psl_reset: the launch-list length of every division) may be NULL. */
psl_status psl_plan_set(psl_ctx* ctx, const psl_plan* plan, uint64_t* n_total_psl, const uint64_t** list_len);

/* DEVICE pointers to budget[K] and field mask[K] (bit i: field i selects the PSL) of the current plan. */
psl_status psl_plan_tables(psl_ctx* ctx, const uint32_t** budget, const uint32_t** mask);

/* The launch of one division.  All pointers DEVICE, BORROWED, valid until the next psl_sample_batch / psl_plan_set /
 * psl_reset / psl_destroy. */
typedef struct {
    uint32_t n_list;   /* entries of the launch list */
    uint32_t n_launch; /* of those: passed their field's jaws (and PSL_DROP_ZERO_WEIGHT) and reach the phantom */
    const uint32_t* slot;  /* n_list: position of the particle in the index (psl_build_batches(NULL) order) */
    const uint8_t* beam;   /* n_list: the field it was assigned to */
    const float *E, *X, *Y, *Z, *U, *V, *W, *wt; /* n_launch, in list order: energy, entry point on the phantom surface and
                                                    direction in the patient frame, weight (wt * F) * mu of its field */
    const uint32_t* src_index; /* n_launch: load-order index of the record */
    const uint8_t* beam_of;    /* n_launch: field */
    uint64_t n_jaw_rejected, n_zero_weight, n_missed; /* list entries dropped, by reason (tested in this order) */
} psl_launch;

/* Round-robin over the division's selected PSLs in spatial order, rr_group reads from each per round until its share
 * (budget x fields that selected it) is used up; a PSL's first read starts at a random particle and wraps around; every
 * read goes to one of the PSL's fields at random.  Then per entry: jaw test of its field
 * (PAPER.md:55), fluence-map and MU weight, rotations and projection to the phantom surface
 * (PAPER.md:105).  PSL_ERR_CAPACITY if the list is longer than max_launch_records.  Synchronises. */
psl_status psl_sample_batch(psl_ctx* ctx, int32_t t, int32_t ie, psl_launch* out);

/* ---- Bins of capacity N (methods 1 and 2) ---------------------------------------------------------------
 * The shipments of the latest ONTHEFLY build had its bins been sent to the transport engine whenever one held
 * `capacity` particles: shipment e = `count[e]` particles of key `key[e]`, output slots [first[e], first[e] + count[e]),
 * in the order the bins fill up as the records arrive; the partially filled bins go last, in key order. */
typedef struct {
    uint32_t n_events;
    const uint32_t *key, *first, *count; /* DEVICE, BORROWED until the next build / psl_reset */
} psl_flush;
psl_status psl_flush_schedule(psl_ctx* ctx, uint32_t capacity, psl_flush* out);

/* Forget all chunks and results (keeps the configuration and workspace).  Blocks the HOST until every HOST chunk
 * loaded so far has left its source buffer (as psl_wait_loads); work already enqueued on the stream is not waited for. */
psl_status psl_reset(psl_ctx* ctx);

void psl_destroy(psl_ctx* ctx);

/* Last error of this context (ctx == NULL: of the last failed psl_create / context-free call on this thread). */
const char* psl_last_error(const psl_ctx* ctx);

/* Number of kernels this context has launched since creation (for bench.py's gpu_launches). */
uint64_t psl_kernel_launches(const psl_ctx* ctx);

/* Optional device-side timing of the library's own kernels, by class, with CUDA events recorded on the
 * context's stream around each launch (a few microseconds of overhead per build while enabled). */
enum { PSL_K_COUNT = 0,   /* histogram passes over raw records (a1-a4, a6, a8) */
       PSL_K_SCAN = 1,    /* exclusive scans (a9) */
       PSL_K_SCATTER = 2, /* ONTHEFLY decode + jaw + fluence + stable scatter (a1-a7, a10) */
       PSL_K_INDEX_A = 3, /* INDEX pass A scatter (a11) */
       PSL_K_INDEX_B = 4, /* INDEX pass B scatter (a11) */
       PSL_K_BEAM = 5,    /* per-beam ROI + jaw + fluence + compaction from the index (a5-a7, a10) */
       PSL_K_OTHER = 6,   /* offsets / statistics / tile descriptors */
       PSL_K_COUNT_KEYS = 7, /* INDEX pass B histogram over the keyed records (a8 of the second digit) */
       PSL_K_SAMPLE = 8,  /* sampling layer over the index: budgets, round-robin gather */
       PSL_K_CLASSES = 9 };
typedef struct {
    double ms[PSL_K_CLASSES];         /* summed device time */
    uint64_t launches[PSL_K_CLASSES]; /* timed brackets (SCAN: one bracket = its three kernels) */
} psl_profile;
psl_status psl_profile_enable(psl_ctx* ctx, int32_t on);
/* Synchronises the stream, returns the totals since the last read (or enable) and clears them. */
psl_status psl_profile_read(psl_ctx* ctx, psl_profile* out);

/* ---- The one call that allocates nothing ------------------------------------------------------------------------------
 * For callers that may not call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid
 * it): how many particles every (type, energy, position) bin holds (the P_j of the budgets,
 * PAPER.md:86-90) -- counts[key] over the valid records inside the grid, key as in psl_batch -- the same numbers
 * psl_build_batches(ctx, NULL) + psl_get_tables give, without a context and without a workspace.  The scratch of the
 * histogram kernel (one table column per CTA, the per-CTA statistics, the energy-edge table) lives in ONE array of
 * PSL_STATIC_SCRATCH_BYTES (2.52 MiB) that is part of the library image: every GPU that loads libpsl_b200.so holds it
 * until the process exits.  The call makes no cudaMalloc / cudaFree / cudaHostAlloc / stream or event creation; it
 * enqueues at most five kernels on cfg->stream and returns (it does not synchronise).
 *
 *   cfg      read: struct_size, n_types, ebin_mode, n_ebins, e_min, e_max, e_edges, n_xbins, n_ybins, x_min, y_min, dx,
 *            dy, geom (all checked as by psl_create), device, stream.  Ignored: mode, max_*, flags, apr_seed, workspace*.
 *   records  DEVICE, n packed psl_record, 4-byte aligned (16-byte aligned buffers take the bulk-copy path); read only
 *   counts   DEVICE, K = n_types * n_ebins * n_xbins * n_ybins uint32, written in full (zeros when n == 0)
 *   totals   DEVICE or NULL
 * Limits (PSL_ERR_CAPACITY beyond them, nothing enqueued): K <= PSL_STATIC_MAX_KEYS, n < 2^32.
 * Shared state: all calls on a GPU use the same array, which keeps the previous call's contents.  Nothing in it has to
 * start at zero -- every word a call reads, the same call has written before (columns [0, CTAs) of rows [0, K), the
 * statistics of those CTAs, the edges [0, n_ebins]) -- so calls one after another on ONE stream need no clearing in
 * between.  Calls that can overlap on the GPU (different streams without an event between them, or two host threads)
 * RACE on the array and give wrong counts: order them.  The first call on a device looks up the array's address and
 * opts the kernels into their shared memory (no allocation either, but make it before a graph capture starts). */
enum { PSL_STATIC_MAX_KEYS = 2048, PSL_STATIC_SCRATCH_BYTES = 2641152 };
typedef struct {
    uint64_t n_in, n_invalid, n_outside_grid, n_binned; /* n_in = n; the three classes add up to it (cf. psl_stats) */
} psl_count_totals;
psl_status psl_count_static(const psl_config* cfg, const void* records, uint64_t n, uint32_t* counts, psl_count_totals* totals);

#ifdef __cplusplus
}
#endif
#endif /* PSL_H */
