/*
 * psl_oracle.c -- CPU ORACLE for the phase-space source hot path.  TEST INFRASTRUCTURE ONLY.
 *
 * A plain, slow, single-threaded restatement of what the hot path computes, written from
 * /root/reference/PAPER.md (Townson et al., arXiv 1302.1861) and the readings listed in
 * DESIGN.md section "Readings".  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may build, load or call it.  It shares no code,
 * header, table or helper with paper_1302_1861_b200/ (the CUDA product path) and neither
 * imports the other.
 *
 * What the method reaches has a plain definition, so the oracle IS that definition:
 *     filter the records, then stably sort the survivors by key.
 *   - PAPER.md:47  (sec. 2.1)  "each particle is placed into the energy bin corresponding to the
 *                               correct particle type"                      -> key by (type, energy)
 *   - PAPER.md:55  (sec. 2.2)  "simple geometrical tests ... accept ... or reject" -> jaw predicate
 *   - PAPER.md:57  (sec. 2.2)  "projected to the MLC plane. A weighting factor determined by the
 *                               particles position in the fluence map ... the two factors are
 *                               multiplied"                                 -> fluence weight
 *   - PAPER.md:75  (sec. 2.3.2) type -> N_E energy ranges -> position bins [x_i,x_i+dx] x [y_i,y_i+dy]
 *   - PAPER.md:80  (sec. 2.3.3) ROI rectangle; "A PSL is considered ... if any portion of its area
 *                               is within the region of interest"            -> ROI bin selection
 *   - PAPER.md:99  (sec. 2.3.3) w'_p = w_p MU_i/MU_total                     -> mu_weight factor
 *   - PAPER.md:101 (sec. 2.3.3) "finish ... one energy division before proceeding to the next"
 *                                                                            -> key order (reading G5)
 * Precision: north_star fixes fp32 for every expression that decides a bin, a key or the jaw
 * predicate ("identical fp32 floor arithmetic, with FMA contraction disabled"); each such
 * expression below is one IEEE operation per line.  Compile with -O2 -ffp-contract=off
 * -fno-fast-math (oracle/psl_oracle.py does).  Sums of weights are accumulated in double.
 *
 * Pins (tests/test_oracle_pins.py, -m "not gpu"): closed forms at every bin edge, double-precision
 * interval binning, numpy's stable argsort, brute-force O(N^2) slot counting, the paper's worked
 * key-space example (400 position bins x 10 energies x 2 types = 8000 PSLs),
 * pencil-ray / point-source projection closed forms, constant and index fluence maps, ROI area
 * brute force, index-route == direct-route.  Nothing here is "parity unpinned".
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

typedef struct {
    int32_t type; /* 0 photon, 1 electron, 2 positron (reading G1) */
    float E, x, y, u, v, wt;
} orc_record; /* 28 bytes */

typedef struct {
    int32_t n_types;   /* 3, or 2 = electrons and positrons merged */
    int32_t ebin_mode; /* 0 linear on [e_min, e_max], 1 caller-supplied edge table */
    int32_t n_ebins;
    float e_min, e_max;
    const float* e_edges; /* n_ebins+1 ascending edges (edge mode) */
    int32_t n_xbins, n_ybins;
    float x_min, y_min, dx, dy;
    float z_src, z_plane, z_jaw_x, z_jaw_y, z_map, z_iso;
    uint32_t flags; /* bit 1: drop survivors whose final weight is exactly 0 */
} orc_config;

typedef struct {
    int32_t has_jaws;
    float jaw_x1, jaw_x2, jaw_y1, jaw_y2; /* aperture edges as projected at z_iso */
    const float* fluence;                 /* map_ny x map_nx, row-major, or NULL */
    int32_t map_nx, map_ny;
    float map_x0, map_y0, map_dx, map_dy; /* at the z_map plane */
    int32_t has_roi;
    float roi_x1, roi_x2, roi_y1, roi_y2; /* at the z_plane */
    float mu_weight;                      /* MU_i / MU_total */
} orc_beam;

typedef struct {
    uint64_t n_in, n_invalid, n_outside_grid, n_roi_skipped, n_jaw_rejected, n_zero_weight, n_survivors;
    double sum_wt_in;      /* sum of wt over valid records */
    double sum_wt_indexed; /* sum of wt over valid records inside the position grid */
    double sum_wt_out;     /* sum of final weights over survivors */
} orc_stats;

enum { ORC_SURVIVOR = 0, ORC_INVALID = 1, ORC_OUTSIDE_GRID = 2, ORC_ROI_SKIPPED = 3, ORC_JAW_REJECTED = 4,
       ORC_ZERO_WEIGHT = 5 };
#define ORC_FLAG_DROP_ZERO_WEIGHT 2u

/* -------------------------------------------------------------------------------------------
 * step 1: validity (reading G15).  q = 1 - (u^2 + v^2), one rounding per operation.
 * ------------------------------------------------------------------------------------------- */
float orc_q(float u, float v)
{
    float a = u * u;
    float b = v * v;
    float s = a + b;
    float q = 1.0f - s;
    return q;
}

int orc_valid(const orc_record* r)
{
    if (r->type < 0 || r->type > 2) return 0;
    if (!isfinite(r->E) || !isfinite(r->x) || !isfinite(r->y) || !isfinite(r->u) || !isfinite(r->v) ||
        !isfinite(r->wt))
        return 0;
    if (!(r->E > 0.0f)) return 0;
    if (!(orc_q(r->u, r->v) > 0.0f)) return 0;
    return 1;
}

/* direction cosine along the beam axis, always downstream (+z) (reading G1) */
float orc_w(float u, float v) { return sqrtf(orc_q(u, v)); }

/* -------------------------------------------------------------------------------------------
 * step 2: energy bin.  PAPER.md:75: "the first of these files will contain only particles with
 * energy in [0, Emax/N_E]".  Half-open bins, clamped into [0, N_E-1] (reading G4).
 * ------------------------------------------------------------------------------------------- */
float orc_bin_width(const orc_config* c)
{
    return (float)(((double)c->e_max - (double)c->e_min) / (double)c->n_ebins);
}

int32_t orc_energy_bin(const orc_config* c, float E)
{
    if (c->ebin_mode == 0) {
        float dE = orc_bin_width(c);
        float d = E - c->e_min;
        float g = d / dE;
        if (g < 0.0f) return 0;
        if (g >= (float)c->n_ebins) return c->n_ebins - 1;
        return (int32_t)floorf(g);
    }
    /* edge table: the number of interior edges at or below E */
    int32_t ie = 0;
    for (int32_t k = 1; k <= c->n_ebins - 1; ++k)
        if (c->e_edges[k] <= E) ie += 1;
    return ie;
}

/* -------------------------------------------------------------------------------------------
 * step 3: position bin.  bin k covers [k*dx, (k+1)*dx) in absolute plane
 * coordinates; the grid starts at the integer bin ix0 = x_min/dx (reading G16: no subtraction
 * of the origin in floating point).
 * ------------------------------------------------------------------------------------------- */
int32_t orc_origin_bin(float origin, float d) { return (int32_t)lround((double)origin / (double)d); }

int orc_axis_bin(float x, float origin, float d, int32_t nbins, int32_t* out)
{
    float inv = (float)(1.0 / (double)d);
    int32_t i0 = orc_origin_bin(origin, d);
    float p = x * inv;
    float f = floorf(p);
    if (!(f >= (float)i0)) return 0;
    if (!(f < (float)(i0 + nbins))) return 0;
    *out = (int32_t)f - i0;
    return 1;
}

int orc_position_bin(const orc_config* c, float x, float y, int32_t* ix, int32_t* iy)
{
    if (c->n_xbins * c->n_ybins == 1) { /* no position bins (methods 1 and 2) */
        *ix = 0;
        *iy = 0;
        return 1;
    }
    if (!orc_axis_bin(x, c->x_min, c->dx, c->n_xbins, ix)) return 0;
    if (!orc_axis_bin(y, c->y_min, c->dy, c->n_ybins, iy)) return 0;
    return 1;
}

/* step 4: key, type-major, then energy, then row iy, then column ix (reading G5) */
uint32_t orc_key(const orc_config* c, int32_t type, int32_t ie, int32_t ix, int32_t iy)
{
    int32_t t = (c->n_types == 2 && type > 1) ? 1 : type;
    uint32_t npos = (uint32_t)(c->n_xbins * c->n_ybins);
    return ((uint32_t)(t * c->n_ebins + ie)) * npos + (uint32_t)(iy * c->n_xbins + ix);
}

uint32_t orc_n_keys(const orc_config* c) { return (uint32_t)(c->n_types * c->n_ebins * c->n_xbins * c->n_ybins); }

/* -------------------------------------------------------------------------------------------
 * step 5: ROI -> selected bin rectangle ("any portion of its area is within the
 * region of interest"; reading G6: positive-area overlap).  Brute force over every bin.
 * out = {rx0, rx1, ry0, ry1} inclusive; empty selection gives rx0 > rx1 (or ry0 > ry1).
 * ------------------------------------------------------------------------------------------- */
static void orc_axis_select(float origin, float d, int32_t nbins, float lo, float hi, int32_t* first, int32_t* last)
{
    *first = nbins;
    *last = -1;
    for (int32_t c = 0; c < nbins; ++c) {
        double left = (double)origin + (double)c * (double)d;
        double right = (double)origin + (double)(c + 1) * (double)d;
        if (left < (double)hi && right > (double)lo) {
            if (c < *first) *first = c;
            if (c > *last) *last = c;
        }
    }
}

void orc_roi_bins(const orc_config* c, const orc_beam* b, int32_t out[4])
{
    orc_axis_select(c->x_min, c->dx, c->n_xbins, b->roi_x1, b->roi_x2, &out[0], &out[1]);
    orc_axis_select(c->y_min, c->dy, c->n_ybins, b->roi_y1, b->roi_y2, &out[2], &out[3]);
}

/* ROI construction (Fig. 1 caption PAPER.md:196; reading G7): per axis, the line from
 * the field centre at z_iso through the jaw edge at the jaw plane, extended up to z_plane.
 * Returns 0 on success, 1 if a jaw plane is not strictly upstream of the isocentre. */
int orc_roi_from_jaws(const orc_config* c, const orc_beam* b, float margin, float roi[4])
{
    double zs = c->z_src, zp = c->z_plane, zi = c->z_iso;
    double zj[2] = { c->z_jaw_x, c->z_jaw_y };
    double e1[2] = { b->jaw_x1, b->jaw_y1 }, e2[2] = { b->jaw_x2, b->jaw_y2 };
    for (int a = 0; a < 2; ++a) {
        if (!(zj[a] < zi)) return 1;
        double centre = 0.5 * (e1[a] + e2[a]);
        double scale = (zj[a] - zs) / (zi - zs); /* iso -> jaw plane, seen from the source */
        double j1 = e1[a] * scale, j2 = e2[a] * scale;
        double lever = (zi - zp) / (zi - zj[a]);
        roi[2 * a + 0] = (float)(centre + (j1 - centre) * lever - (double)margin);
        roi[2 * a + 1] = (float)(centre + (j2 - centre) * lever + (double)margin);
    }
    return 0;
}

/* -------------------------------------------------------------------------------------------
 * step 6: jaw accept / reject.  One thin plane per jaw pair, half-open aperture,
 * edges given at isocentre and scaled to the jaw plane from the source (reading G8).
 * ------------------------------------------------------------------------------------------- */
float orc_jaw_edge(float edge_iso, float z_jaw, float z_src, float z_iso)
{
    return (float)((double)edge_iso * ((double)z_jaw - (double)z_src) / ((double)z_iso - (double)z_src));
}

void orc_slopes(const orc_record* r, float* tx, float* ty)
{
    float w = orc_w(r->u, r->v);
    float t = 1.0f / w;
    *tx = r->u * t;
    *ty = r->v * t;
}

int orc_jaw_pass(const orc_config* c, const orc_beam* b, const orc_record* r)
{
    float tx, ty;
    orc_slopes(r, &tx, &ty);
    float dzx = c->z_jaw_x - c->z_plane;
    float dzy = c->z_jaw_y - c->z_plane;
    float sx = tx * dzx;
    float sy = ty * dzy;
    float xj = r->x + sx;
    float yj = r->y + sy;
    float X1 = orc_jaw_edge(b->jaw_x1, c->z_jaw_x, c->z_src, c->z_iso);
    float X2 = orc_jaw_edge(b->jaw_x2, c->z_jaw_x, c->z_src, c->z_iso);
    float Y1 = orc_jaw_edge(b->jaw_y1, c->z_jaw_y, c->z_src, c->z_iso);
    float Y2 = orc_jaw_edge(b->jaw_y2, c->z_jaw_y, c->z_src, c->z_iso);
    return (X1 <= xj && xj < X2 && Y1 <= yj && yj < Y2) ? 1 : 0;
}

/* -------------------------------------------------------------------------------------------
 * step 7: projection to the fluence-map plane and weight (readings G11, G12).
 * Containing pixel, no interpolation; outside the map the factor is 0; wt' = (wt*F)*mu.
 * ------------------------------------------------------------------------------------------- */
void orc_project_map(const orc_config* c, const orc_record* r, float* xm, float* ym)
{
    float tx, ty;
    orc_slopes(r, &tx, &ty);
    float dz = c->z_map - c->z_plane;
    float sx = tx * dz;
    float sy = ty * dz;
    *xm = r->x + sx;
    *ym = r->y + sy;
}

float orc_fluence_at(const orc_beam* b, float xm, float ym)
{
    int32_t px, py;
    if (!orc_axis_bin(xm, b->map_x0, b->map_dx, b->map_nx, &px)) return 0.0f;
    if (!orc_axis_bin(ym, b->map_y0, b->map_dy, b->map_ny, &py)) return 0.0f;
    return b->fluence[(size_t)py * (size_t)b->map_nx + (size_t)px];
}

float orc_final_weight(const orc_config* c, const orc_beam* b, const orc_record* r, float* xm, float* ym)
{
    orc_project_map(c, r, xm, ym);
    if (b == NULL) return r->wt;
    if (b->fluence == NULL) return r->wt * b->mu_weight;
    float F = orc_fluence_at(b, *xm, *ym);
    float a = r->wt * F;
    return a * b->mu_weight;
}

/* -------------------------------------------------------------------------------------------
 * steps 1-8 for one record: which of the six classes it falls in (tested in this order) and,
 * for records that are valid and inside the grid, its key.
 * ------------------------------------------------------------------------------------------- */
int orc_classify(const orc_config* c, const orc_beam* b, const int32_t* sel /* orc_roi_bins, if has_roi */,
                 const orc_record* r, uint32_t* key)
{
    *key = 0xFFFFFFFFu;
    if (!orc_valid(r)) return ORC_INVALID;
    int32_t ix, iy;
    if (!orc_position_bin(c, r->x, r->y, &ix, &iy)) return ORC_OUTSIDE_GRID;
    *key = orc_key(c, r->type, orc_energy_bin(c, r->E), ix, iy);
    if (b == NULL) return ORC_SURVIVOR;
    if (b->has_roi && !(sel[0] <= ix && ix <= sel[1] && sel[2] <= iy && iy <= sel[3])) return ORC_ROI_SKIPPED;
    if (b->has_jaws && !orc_jaw_pass(c, b, r)) return ORC_JAW_REJECTED;
    if (c->flags & ORC_FLAG_DROP_ZERO_WEIGHT) {
        float xm, ym;
        if (orc_final_weight(c, b, r, &xm, &ym) == 0.0f) return ORC_ZERO_WEIGHT;
    }
    return ORC_SURVIVOR;
}

/* -------------------------------------------------------------------------------------------
 * step 9: the whole result.  counts[K], offsets[K+1], and the survivors laid out by key with
 * input order inside each key (readings G13, G14): slot(i) = offsets[key(i)] + #{j in S: j < i,
 * key(j) = key(i)}.  beam == NULL gives method 1 / the PSL index itself (S = valid and in grid).
 * cls (n bytes) and keys (n words) may be NULL.  Output arrays hold at least n elements.
 * Returns the number of survivors.
 * ------------------------------------------------------------------------------------------- */
uint64_t orc_build(const orc_config* c, const orc_beam* b, const orc_record* rec, uint64_t n, uint32_t* counts,
                   uint32_t* offsets, float* oE, float* ox, float* oy, float* ou, float* ov, float* ow, float* owt,
                   float* oxm, float* oym, uint32_t* osrc, uint8_t* cls, uint32_t* keys, orc_stats* st)
{
    uint32_t K = orc_n_keys(c);
    uint8_t* my_cls = cls ? cls : (uint8_t*)malloc(n ? n : 1);
    uint32_t* my_keys = keys ? keys : (uint32_t*)malloc((n ? n : 1) * sizeof(uint32_t));
    orc_stats s;
    memset(&s, 0, sizeof s);
    memset(counts, 0, (size_t)K * sizeof(uint32_t));

    int32_t sel[4] = { 0, 0, 0, 0 };
    if (b && b->has_roi) orc_roi_bins(c, b, sel);

    s.n_in = n;
    for (uint64_t i = 0; i < n; ++i) {
        int k = orc_classify(c, b, sel, &rec[i], &my_keys[i]);
        my_cls[i] = (uint8_t)k;
        if (k != ORC_INVALID) s.sum_wt_in += (double)rec[i].wt;
        if (k != ORC_INVALID && k != ORC_OUTSIDE_GRID) s.sum_wt_indexed += (double)rec[i].wt;
        switch (k) {
        case ORC_INVALID: s.n_invalid++; break;
        case ORC_OUTSIDE_GRID: s.n_outside_grid++; break;
        case ORC_ROI_SKIPPED: s.n_roi_skipped++; break;
        case ORC_JAW_REJECTED: s.n_jaw_rejected++; break;
        case ORC_ZERO_WEIGHT: s.n_zero_weight++; break;
        default: s.n_survivors++; counts[my_keys[i]]++; break;
        }
    }

    offsets[0] = 0;
    for (uint32_t k = 0; k < K; ++k) offsets[k + 1] = offsets[k] + counts[k];

    uint32_t* cursor = (uint32_t*)malloc((size_t)(K ? K : 1) * sizeof(uint32_t));
    memcpy(cursor, offsets, (size_t)K * sizeof(uint32_t));
    for (uint64_t i = 0; i < n; ++i) {
        if (my_cls[i] != ORC_SURVIVOR) continue;
        const orc_record* r = &rec[i];
        uint32_t slot = cursor[my_keys[i]]++;
        float xm, ym;
        float wt = orc_final_weight(c, b, r, &xm, &ym);
        oE[slot] = r->E;
        ox[slot] = r->x;
        oy[slot] = r->y;
        ou[slot] = r->u;
        ov[slot] = r->v;
        ow[slot] = orc_w(r->u, r->v);
        owt[slot] = wt;
        oxm[slot] = xm;
        oym[slot] = ym;
        osrc[slot] = (uint32_t)i;
        s.sum_wt_out += (double)wt;
    }
    free(cursor);
    if (!cls) free(my_cls);
    if (!keys) free(my_keys);
    if (st) *st = s;
    return s.n_survivors;
}

/* ---- array forms of the scalar steps, for the pins ---- */
void orc_energy_bins(const orc_config* c, const float* E, uint64_t n, int32_t* out)
{
    for (uint64_t i = 0; i < n; ++i) out[i] = orc_energy_bin(c, E[i]);
}

void orc_axis_bins(const float* x, uint64_t n, float origin, float d, int32_t nbins, int32_t* out)
{
    for (uint64_t i = 0; i < n; ++i) {
        int32_t b;
        out[i] = orc_axis_bin(x[i], origin, d, nbins, &b) ? b : -1;
    }
}

void orc_classify_all(const orc_config* c, const orc_beam* b, const orc_record* rec, uint64_t n, uint8_t* cls,
                      uint32_t* keys)
{
    int32_t sel[4] = { 0, 0, 0, 0 };
    if (b && b->has_roi) orc_roi_bins(c, b, sel);
    for (uint64_t i = 0; i < n; ++i) cls[i] = (uint8_t)orc_classify(c, b, sel, &rec[i], &keys[i]);
}

void orc_jaw_points(const orc_config* c, const orc_record* rec, uint64_t n, float* xj, float* yj)
{
    for (uint64_t i = 0; i < n; ++i) {
        float tx, ty;
        orc_slopes(&rec[i], &tx, &ty);
        float dzx = c->z_jaw_x - c->z_plane;
        float dzy = c->z_jaw_y - c->z_plane;
        float sx = tx * dzx;
        float sy = ty * dzy;
        xj[i] = rec[i].x + sx;
        yj[i] = rec[i].y + sy;
    }
}

uint32_t orc_record_bytes(void) { return (uint32_t)sizeof(orc_record); }
