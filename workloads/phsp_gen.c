/*
 * phsp_gen.c -- seeded synthetic phase-space generator (INPUTS ONLY).
 *
 * This module produces the packed 28-byte records that stand in for the paper's
 * BEAMnrc phase-space of a 6 MV Varian 21EX (section 2.6), which is not
 * available here.  It holds none of the method's arithmetic: no binning, no jaw test,
 * no fluence lookup, no sorting.  Both the CPU oracle (oracle/) and the CUDA library
 * (paper_1302_1861_b200/) consume the bytes it writes; neither shares anything else.
 *
 * Recipe (BASELINE.json configs 1-5, restated in DESIGN.md "Input recipe"):
 *   type     : u < 0.98 photon(0), < 0.998 electron(1), else positron(2)
 *   energy   : photon   p(E) ~ E exp(-E/0.5 MeV) on [0.01, 6] MeV (mode 0.5 MeV, exponential tail),
 *                       drawn as Gamma(2, 0.5) = -0.5 ln(u1 u2) with rejection outside the range;
 *              e-/e+    uniform on [0.01, 6] MeV
 *   position : (x, y) uniform on [-half_x, half_x) x [-half_y, half_y) at the scoring plane
 *   direction: point source `src_dist` cm upstream on the axis; theta_x = atan(x/src_dist) + N(0, sigma),
 *              tx = tan(theta_x), same for y; (u, v) = (tx, ty)/sqrt(1 + tx^2 + ty^2)
 *   weight   : 1.0
 * All arithmetic in double, stored as fp32.
 *
 * Random numbers are counter-based: uniform(seed, record index, draw index), so any range
 * of records can be generated independently (chunked, threaded) and reproducibly.
 */
#include <math.h>
#include <stddef.h>
#include <stdint.h>

typedef struct {
    int32_t type;
    float E, x, y, u, v, wt;
} wl_record; /* 28 bytes, packed, little-endian */

typedef struct {
    uint64_t seed;
    double half_x, half_y;
    double src_dist;
    double sigma_rad;
    double frac_photon;   /* 0.98  */
    double frac_electron; /* 0.018 */
    double e_lo, e_hi;    /* 0.01, 6.0 */
    double e_scale;       /* 0.5 */
} wl_params;

static inline uint64_t wl_mix64(uint64_t z)
{
    z += 0x9E3779B97F4A7C15ull;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
    return z ^ (z >> 31);
}

/* uniform on the open interval (0, 1) */
static inline double wl_u01(uint64_t seed, uint64_t idx, uint32_t draw)
{
    uint64_t h = wl_mix64(wl_mix64(seed ^ wl_mix64(idx)) + (uint64_t)draw);
    return ((double)(h >> 11) + 0.5) * (1.0 / 9007199254740992.0);
}

static void wl_one(const wl_params* p, uint64_t idx, wl_record* r)
{
    const double two_pi = 6.283185307179586476925286766559;
    double ut = wl_u01(p->seed, idx, 0);
    int32_t type = ut < p->frac_photon ? 0 : (ut < p->frac_photon + p->frac_electron ? 1 : 2);

    double E;
    if (type == 0) {
        E = -1.0;
        for (uint32_t a = 0; a < 8; ++a) {
            double u1 = wl_u01(p->seed, idx, 5 + 2 * a);
            double u2 = wl_u01(p->seed, idx, 6 + 2 * a);
            double e = -p->e_scale * log(u1 * u2);
            if (e >= p->e_lo && e <= p->e_hi) { E = e; break; }
        }
        if (E < 0.0) E = p->e_scale; /* 8 rejections in a row: probability < 1e-28 */
    } else {
        E = p->e_lo + (p->e_hi - p->e_lo) * wl_u01(p->seed, idx, 5);
    }

    double x = p->half_x * (2.0 * wl_u01(p->seed, idx, 1) - 1.0);
    double y = p->half_y * (2.0 * wl_u01(p->seed, idx, 2) - 1.0);

    double a = wl_u01(p->seed, idx, 3), b = wl_u01(p->seed, idx, 4);
    double rad = sqrt(-2.0 * log(a));
    double n1 = rad * cos(two_pi * b), n2 = rad * sin(two_pi * b);

    double tx = tan(atan(x / p->src_dist) + p->sigma_rad * n1);
    double ty = tan(atan(y / p->src_dist) + p->sigma_rad * n2);
    double inv = 1.0 / sqrt(1.0 + tx * tx + ty * ty);

    r->type = type;
    r->E = (float)E;
    r->x = (float)x;
    r->y = (float)y;
    r->u = (float)(tx * inv);
    r->v = (float)(ty * inv);
    r->wt = 1.0f;
}

/* Fill out[0..n) with records first..first+n of the stream defined by *p. */
void wl_generate(const wl_params* p, uint64_t first, uint64_t n, wl_record* out)
{
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < (int64_t)n; ++i) wl_one(p, first + (uint64_t)i, &out[i]);
}

uint32_t wl_record_bytes(void) { return (uint32_t)sizeof(wl_record); }
