/*
 * hough_oracle.c -- CPU ORACLE.  TEST INFRASTRUCTURE ONLY.
 *
 * Plain, slow, single-threaded, obviously-correct C99 restatement of the hot path of
 * Halyo, LeGresley, Lujan, "Massively Parallel Computing and the Search for Jets and Black Holes at
 * the LHC" (arXiv:1309.6275): Hough-transform voting (section 5: "for each piece of
 * input data votes are added to the feature instances that would include that input data"), peak
 * finding ("looking for local maxima in the parameter space"), candidate -> track
 * parameters ("measure ... the transverse momentum of prompt or non-prompt tracks") and
 * the jet / displaced-jet selection (in the phi-cone form BASELINE.json:north_star
 * fixes).  The paper prints no formula; every concrete formula is north_star's, and every point the
 * paper leaves open follows the readings R1-R30 of SURVEY.md section 8(c), restated in DESIGN.md.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may call
 * this.  It shares no code, header, table or constant with the CUDA path (paper_1309_6275_b200/csrc)
 * and neither includes the other.
 *
 * Build:  gcc -O2 -std=c99 -ffp-contract=off -fno-fast-math -shared -fPIC hough_oracle.c -lm
 * (-ffp-contract=off is mandatory: the per-vote arithmetic is IEEE fp32 with one rounding per
 *  operation, no FMA.  x86-64 SSE2 scalar arithmetic evaluates float expressions in float.)
 *
 * Parity pins (tests/test_oracle_pins.py, -m "not gpu"): P1 closed-form circle geometry, P2 noiseless
 * bin-centred track peaks at its generating bin with count = layers crossed, P3 vote conservation
 * against an independent fp64 count, P4 brute-force division-free circle-fit membership, P5 additivity
 * / permutation invariants, P6-P8 peak definition brute force + special cases, P9 track closed forms,
 * P10-P11 jet brute force + special cases, P12 a hand-built end-to-end event.  Nothing in the paper
 * pins the *choice* of readings R4, R5, R12-R14, R18 (no worked example exists) -- those are pinned
 * to north_star only.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#ifndef M_PI
#define M_PI 3.14159265358979323846
#endif

typedef struct {
    uint32_t n_phi0, n_kappa, n_d0;   /* n_d0 == 1: prompt 2D mode (d0 == 0, kappa = 2 s / r) */
    float kappa_max;                  /* 1/mm; kappa axis [-kappa_max, +kappa_max) */
    float d0_min, d0_max;             /* mm; 3D mode only */
    float b_tesla;
    uint32_t n_layers;                /* 1..16 */
} oracle_grid;

typedef struct { uint32_t lin; uint16_t count; uint16_t mask; } oracle_peak;
typedef struct { float pt, phi0, d0; int32_t q; int32_t jet; } oracle_track;
typedef struct { uint32_t seed_track, n_tracks, n_displaced; float phi, sum_pt; } oracle_jet;

/* ---- O-0 tables: computed in double, each result rounded once to fp32 ------------------------- */

static double phi0_centre(const oracle_grid *g, uint32_t ip)
{
    return ((double)ip + 0.5) * (2.0 * M_PI / (double)g->n_phi0);
}

static float d0_centre(const oracle_grid *g, uint32_t id)
{
    if (g->n_d0 == 1) return 0.0f;
    return (float)((double)g->d0_min +
                   ((double)id + 0.5) * (((double)g->d0_max - (double)g->d0_min) / (double)g->n_d0));
}

static float inv_dkappa(const oracle_grid *g)
{
    return (float)((double)g->n_kappa / (2.0 * (double)g->kappa_max));
}

/* exported so tests can look at the tables */
void oracle_tables(const oracle_grid *g, float *c0, float *s0, float *d0c, float *inv_dk)
{
    for (uint32_t ip = 0; ip < g->n_phi0; ++ip) {
        c0[ip] = (float)cos(phi0_centre(g, ip));
        s0[ip] = (float)sin(phi0_centre(g, ip));
    }
    for (uint32_t id = 0; id < g->n_d0; ++id) d0c[id] = d0_centre(g, id);
    *inv_dk = inv_dkappa(g);
}

/* ---- O-1 hit preparation: sin/cos of the hit azimuth, evaluated in double and rounded once to fp32 ---- */
/* (reading R6: the correctly-rounded fp32 of the real value, obtained by fp64 evaluation + one rounding) */

static float hit_sin(float phi) { return (float)sin((double)phi); }
static float hit_cos(float phi) { return (float)cos((double)phi); }

/* exported so a test can compare the CUDA path's prepared records with these values bit for bit (R6) */
void oracle_hit_prep(uint64_t n_hits, const float *phi, float *sp, float *cp)
{
    for (uint64_t h = 0; h < n_hits; ++h) { sp[h] = hit_sin(phi[h]); cp[h] = hit_cos(phi[h]); }
}

/* ---- O-2: one candidate (hit, id, ip) -> kappa bin, or -1 if it does not vote ------------------ */
/* Every statement below is exactly one IEEE fp32 operation (compiled with -ffp-contract=off).      */

static int vote_bin(int mode3d, float r, float r2, float sp, float cp, float c0, float s0,
                    float d0c, float two_d0, float d0sq, float kmax, float inv_dk, float nk_f)
{
    float m1 = sp * c0;
    float m2 = cp * s0;
    float s = m1 - m2;                 /* sin(phi - phi0c) by the difference identity */
    float kappa;
    if (!mode3d) {
        float two_s = 2.0f * s;        /* exact */
        kappa = two_s / r;             /* kappa = 2 s / r */
    } else {
        float rs = r * s;
        float t = rs + d0c;
        float num = 2.0f * t;          /* exact */
        float a = two_d0 * rs;
        float b = r2 + a;
        float den = b + d0sq;
        kappa = num / den;             /* 2 (r s + d0) / (r^2 + 2 d0 r s + d0^2); 0/0 -> NaN, x/0 -> inf */
    }
    float v = kappa + kmax;
    float u = v * inv_dk;
    if (u >= 0.0f && u < nk_f)         /* NaN, +-inf fail; -0.0f passes -> bin 0 */
        return (int)u;                 /* truncation == floor since u >= 0 */
    return -1;
}

/*
 * O-1 + O-2 for one event, restricted to d0 bins [id_lo, id_hi) and phi0 bins [ip_lo, ip_hi).
 * count/mask are the FULL event planes [n_d0][n_phi0][n_kappa] (caller zeroes them); only columns in the
 * requested ranges are touched.  Returns the number of votes cast.
 */
int64_t oracle_vote(const oracle_grid *g, uint64_t n_hits, const float *r, const float *phi,
                    const uint8_t *layer, uint32_t id_lo, uint32_t id_hi, uint32_t ip_lo, uint32_t ip_hi,
                    uint16_t *count, uint16_t *mask)
{
    const int mode3d = g->n_d0 > 1;
    const float kmax = g->kappa_max;
    const float inv_dk = inv_dkappa(g);
    const float nk_f = (float)g->n_kappa;
    int64_t votes = 0;
    /* O-0 tables for this grid */
    float *c0 = (float *)malloc(sizeof(float) * g->n_phi0);
    float *s0 = (float *)malloc(sizeof(float) * g->n_phi0);
    float *d0c = (float *)malloc(sizeof(float) * g->n_d0);
    float inv_dk_unused;
    oracle_tables(g, c0, s0, d0c, &inv_dk_unused);
    for (uint64_t h = 0; h < n_hits; ++h) {
        if (layer[h] >= g->n_layers) continue;                 /* R9: invalid hit ignored */
        const float sp = hit_sin(phi[h]);                      /* O-1 */
        const float cp = hit_cos(phi[h]);
        const float rr = r[h];
        const float r2 = rr * rr;
        const uint16_t bit = (uint16_t)(1u << layer[h]);
        for (uint32_t ip = ip_lo; ip < ip_hi; ++ip) {
            for (uint32_t id = id_lo; id < id_hi; ++id) {
                const float two_d0 = 2.0f * d0c[id];           /* exact */
                const float d0sq = d0c[id] * d0c[id];
                int ik = vote_bin(mode3d, rr, r2, sp, cp, c0[ip], s0[ip], d0c[id], two_d0, d0sq,
                                  kmax, inv_dk, nk_f);
                if (ik >= 0) {
                    size_t b = ((size_t)id * g->n_phi0 + ip) * g->n_kappa + (size_t)ik;
                    count[b] = (uint16_t)(count[b] + 1);
                    mask[b] |= bit;
                    ++votes;
                }
            }
        }
    }
    free(c0); free(s0); free(d0c);
    return votes;
}

/* Same arithmetic, for a list of sampled columns: out planes are [n_cols][n_kappa] (caller zeroes). */
int64_t oracle_vote_columns(const oracle_grid *g, uint64_t n_hits, const float *r, const float *phi,
                            const uint8_t *layer, uint32_t n_cols, const uint32_t *col_id,
                            const uint32_t *col_ip, uint16_t *count, uint16_t *mask)
{
    const int mode3d = g->n_d0 > 1;
    const float kmax = g->kappa_max;
    const float inv_dk = inv_dkappa(g);
    const float nk_f = (float)g->n_kappa;
    int64_t votes = 0;
    for (uint64_t h = 0; h < n_hits; ++h) {
        if (layer[h] >= g->n_layers) continue;
        const float sp = hit_sin(phi[h]);
        const float cp = hit_cos(phi[h]);
        const float rr = r[h];
        const float r2 = rr * rr;
        const uint16_t bit = (uint16_t)(1u << layer[h]);
        for (uint32_t c = 0; c < n_cols; ++c) {
            const float c0 = (float)cos(phi0_centre(g, col_ip[c]));
            const float s0 = (float)sin(phi0_centre(g, col_ip[c]));
            const float d0c = d0_centre(g, col_id[c]);
            const float two_d0 = 2.0f * d0c;
            const float d0sq = d0c * d0c;
            int ik = vote_bin(mode3d, rr, r2, sp, cp, c0, s0, d0c, two_d0, d0sq, kmax, inv_dk, nk_f);
            if (ik >= 0) {
                size_t b = (size_t)c * g->n_kappa + (size_t)ik;
                count[b] = (uint16_t)(count[b] + 1);
                mask[b] |= bit;
                ++votes;
            }
        }
    }
    return votes;
}

/* ---- O-3 peaks --------------------------------------------------------------------------------- */

static int popcount16(uint16_t m)
{
    int n = 0;
    while (m) { n += m & 1u; m >>= 1; }
    return n;
}

/*
 * Scan lin ascending; bin b is a peak iff popcount(mask[b]) >= l_min and for every existing neighbour n
 * (phi0 periodic, kappa and d0 clipped): count[b] > count[n] or (count[b] == count[n] and lin(b) < lin(n)).
 * Writes the first max_peaks peaks; returns the total number found.
 */
uint64_t oracle_peaks(const oracle_grid *g, const uint16_t *count, const uint16_t *mask, uint32_t l_min,
                      uint32_t max_peaks, oracle_peak *peaks)
{
    const int64_t ND = g->n_d0, NP = g->n_phi0, NK = g->n_kappa;
    uint64_t total = 0;
    for (int64_t id = 0; id < ND; ++id)
        for (int64_t ip = 0; ip < NP; ++ip)
            for (int64_t ik = 0; ik < NK; ++ik) {
                const int64_t lin = (id * NP + ip) * NK + ik;
                if (popcount16(mask[lin]) < (int)l_min) continue;
                const uint16_t c = count[lin];
                int is_peak = 1;
                for (int dd = -1; dd <= 1 && is_peak; ++dd) {
                    const int64_t jd = id + dd;
                    if (jd < 0 || jd >= ND) continue;                  /* d0 clipped (dd == 0 only in 2D) */
                    for (int dp = -1; dp <= 1 && is_peak; ++dp) {
                        const int64_t jp = (ip + dp + NP) % NP;        /* phi0 periodic */
                        for (int dk = -1; dk <= 1; ++dk) {
                            if (dd == 0 && dp == 0 && dk == 0) continue;
                            const int64_t jk = ik + dk;
                            if (jk < 0 || jk >= NK) continue;          /* kappa clipped */
                            const int64_t nlin = (jd * NP + jp) * NK + jk;
                            if (nlin == lin) continue;                 /* n_phi0 < 3 degenerate wrap onto self */
                            const uint16_t cn = count[nlin];
                            if (!(c > cn || (c == cn && lin < nlin))) { is_peak = 0; break; }
                        }
                    }
                }
                if (is_peak) {
                    if (total < max_peaks) {
                        peaks[total].lin = (uint32_t)lin;
                        peaks[total].count = c;
                        peaks[total].mask = mask[lin];
                    }
                    ++total;
                }
            }
    return total;
}

/* ---- O-4 tracks -------------------------------------------------------------------------------- */

void oracle_tracks(const oracle_grid *g, const oracle_peak *peaks, uint32_t n_stored, oracle_track *tracks)
{
    const double kmax = (double)g->kappa_max;
    for (uint32_t j = 0; j < n_stored; ++j) {
        const uint32_t lin = peaks[j].lin;
        const uint32_t ik = lin % g->n_kappa;
        const uint32_t ip = (lin / g->n_kappa) % g->n_phi0;
        const uint32_t id = lin / g->n_kappa / g->n_phi0;
        const double kc = -kmax + ((double)ik + 0.5) * (2.0 * kmax / (double)g->n_kappa);
        tracks[j].pt = (float)(0.3e-3 * (double)g->b_tesla / fabs(kc));
        tracks[j].phi0 = (float)phi0_centre(g, ip);
        tracks[j].d0 = d0_centre(g, id);
        tracks[j].q = (kc < 0.0) ? +1 : -1;           /* R17: q = -sign(kappa) */
        tracks[j].jet = -1;
    }
}

/* ---- O-5 jets ---------------------------------------------------------------------------------- */

/*
 * Seeded fixed-cone clustering in phi0 on integer keys.  tracks[] must come from oracle_tracks (its .jet
 * fields are overwritten).  Stores the first max_jets jets, returns the total; *flag = 1 iff any jet
 * (stored or not) has n_displaced >= n_displaced_min.
 */
uint32_t oracle_jets(const oracle_grid *g, const oracle_peak *peaks, uint32_t n_stored, float cone_rad,
                     float d0_cut_mm, uint32_t n_displaced_min, uint32_t max_jets, oracle_track *tracks,
                     oracle_jet *jets, uint8_t *flag)
{
    const int NP = (int)g->n_phi0, NK = (int)g->n_kappa;
    const int cone_bins = (int)floor((double)cone_rad * (double)g->n_phi0 / (2.0 * M_PI));
    int *a = (int *)malloc(sizeof(int) * (n_stored ? n_stored : 1));
    int *ipj = (int *)malloc(sizeof(int) * (n_stored ? n_stored : 1));
    uint8_t *dsp = (uint8_t *)malloc(n_stored ? n_stored : 1);
    uint8_t *assigned = (uint8_t *)calloc(n_stored ? n_stored : 1, 1);
    for (uint32_t j = 0; j < n_stored; ++j) {
        const uint32_t lin = peaks[j].lin;
        const int ik = (int)(lin % g->n_kappa);
        const uint32_t id = lin / g->n_kappa / g->n_phi0;
        ipj[j] = (int)((lin / g->n_kappa) % g->n_phi0);
        a[j] = abs(2 * ik - (NK - 1));                      /* smaller = higher pT */
        dsp[j] = (g->n_d0 > 1) && (fabsf(d0_centre(g, id)) > d0_cut_mm);
        tracks[j].jet = -1;
    }
    uint32_t J = 0;
    *flag = 0;
    for (;;) {
        int64_t seed = -1;
        for (uint32_t j = 0; j < n_stored; ++j)             /* smallest (a_j, j) among unassigned */
            if (!assigned[j] && (seed < 0 || a[j] < a[seed])) seed = j;
        if (seed < 0) break;
        uint32_t n_tracks = 0, n_disp = 0;
        double sum_pt = 0.0;
        for (uint32_t m = 0; m < n_stored; ++m) {
            if (assigned[m]) continue;
            int d = abs(ipj[m] - ipj[seed]);
            if (NP - d < d) d = NP - d;
            if (d <= cone_bins) {
                assigned[m] = 1;
                ++n_tracks;
                n_disp += dsp[m];
                sum_pt += (double)tracks[m].pt;             /* ascending track index */
                if (J < max_jets) tracks[m].jet = (int32_t)J;
            }
        }
        if (J < max_jets) {
            jets[J].seed_track = (uint32_t)seed;
            jets[J].n_tracks = n_tracks;
            jets[J].n_displaced = n_disp;
            jets[J].phi = tracks[seed].phi0;
            jets[J].sum_pt = (float)sum_pt;
        }
        if (n_disp >= n_displaced_min) *flag = 1;
        ++J;
    }
    free(a); free(ipj); free(dsp); free(assigned);
    return J;
}

/* ================================================================================================ */
/* O-6 / O-7: the paper's SECOND Hough transform -- tracks -> displaced vertices (PAPER.md:117,       */
/* section 6: "the corresponding parameter space representation of these tracks is processed by a   */
/* second application of the Hough transform ... to identify not straight lines but sinusoids which */
/* contain a significant number of tracks, indicating that this is a location of a displaced jet";  */
/* "the same peak finding algorithm is applied to the parameter space of this second Hough          */
/* transform"; features at the interaction point are excluded "by setting a lower     */
/* bound on the radius").  The paper gives no formula; readings R34-R39 fix it:           */
/*   - vertex space = (phi_v, R_v) bins, phi_v periodic over [0, 2pi), R_v over [r_min, r_max) with  */
/*     r_min the beam-pipe radius (the paper's lower bound); lin = iv * NR + ir (R_v fastest);       */
/*   - a track (d0, phi0, kappa) (R1 convention) crosses the circle of radius r about the origin on  */
/*     its outgoing branch at azimuth phi0 + asin(s), s = (kappa (r^2 + d0^2) - 2 d0) /              */
/*     (2 r (1 - kappa d0)) (north_star's curvature formula solved for s; to first order             */
/*     d0 = -r s = R_v sin(phi0 - phi_v): the sinusoid of the paper); one vote per (track, R_v bin)  */
/*     at the bin centre radius, into the phi_v bin that holds the crossing azimuth;                 */
/*   - no transcendental per vote: (cos, sin) of the crossing azimuth by rotating the track's        */
/*     (cos phi0, sin phi0) by (sqrt(1 - s^2), s), and the phi_v bin by comparing that direction     */
/*     with the bin-edge directions (cross products, binary search inside the quadrant); every step  */
/*     below is one IEEE fp32 operation (+, -, *, /, sqrt are all correctly rounded);                */
/*   - tracks compatible with the interaction point, |d0| <= d0_cut (the displaced-track cut of R20),  */
/*     do not vote: a track through the origin crosses EVERY radius at nearly its own phi0, so prompt  */
/*     tracks that merely share a phi0 bin would pile up at all radii; this is the paper's            */
/*     interaction-point filter applied to the transform's input as well as to its radius axis;       */
/*   - peaks: rule O-3 on the (phi_v, R_v) grid with the count threshold n_min; oracle_vertices      */
/*     literally calls oracle_peaks with a "thermometer" mask of min(count, 16) bits, so that        */
/*     popcount(mask) >= n_min <=> count >= n_min for n_min <= 16.                                   */
/* Pins: tests/test_oracle_pins.py P14-P17.                                                          */
/* ================================================================================================ */

typedef struct {
    uint32_t n_phi, n_r;              /* phi_v bins (multiple of 4), R_v bins (multiple of 8: the peak finder's axis rule) */
    float r_min, r_max;               /* mm; r_min = beam pipe radius (interaction-point filter) */
} oracle_vgrid;

typedef struct { float r, phi; uint32_t n_tracks, lin; } oracle_vertex;

static float vtx_r_centre(const oracle_vgrid *v, uint32_t ir)
{
    return (float)((double)v->r_min + ((double)ir + 0.5) * (((double)v->r_max - (double)v->r_min) / (double)v->n_r));
}
static double vtx_phi_edge(const oracle_vgrid *v, uint32_t k) { return (double)k * (2.0 * M_PI / (double)v->n_phi); }

/* phi_v bin of the direction (x, y): quadrant from the signs, then the largest edge k of the quadrant with
   cross(e_k, (x, y)) >= 0, by binary search; e_k = (cos, sin)(k * 2pi/n_phi) rounded once from double. */
static uint32_t angle_bin(const oracle_vgrid *v, const float *ex, const float *ey, float x, float y)
{
    uint32_t q;                                   /* [0,pi/2): x>0,y>=0  [pi/2,pi): x<=0,y>0  [pi,3pi/2): x<0,y<=0  else */
    if (x > 0.0f && y >= 0.0f) q = 0u;
    else if (x <= 0.0f && y > 0.0f) q = 1u;
    else if (x < 0.0f && y <= 0.0f) q = 2u;
    else q = 3u;
    uint32_t lo = q * (v->n_phi / 4u), hi = lo + v->n_phi / 4u - 1u;
    while (lo < hi) {
        const uint32_t mid = (lo + hi + 1u) / 2u;
        const float a = ex[mid] * y;
        const float b = ey[mid] * x;
        const float cr = a - b;
        if (cr >= 0.0f) lo = mid; else hi = mid - 1u;
    }
    return lo;
}

/* exported for the pins */
uint32_t oracle_angle_bin(const oracle_vgrid *v, float x, float y)
{
    float *ex = (float *)malloc(sizeof(float) * v->n_phi), *ey = (float *)malloc(sizeof(float) * v->n_phi);
    for (uint32_t k = 0; k < v->n_phi; ++k) { ex[k] = (float)cos(vtx_phi_edge(v, k)); ey[k] = (float)sin(vtx_phi_edge(v, k)); }
    const uint32_t b = angle_bin(v, ex, ey, x, y);
    free(ex); free(ey);
    return b;
}

/*
 * O-6 vote: tracks given by fp32 parameters d0 [mm], (s0, c0) = (sin, cos) phi0, kappa [1/mm].
 * count is the vertex plane [n_phi][n_r] (caller zeroes).  Returns the number of votes.
 */
int64_t oracle_vertex_vote(const oracle_vgrid *v, uint32_t n_tracks, const float *d0, const float *s0, const float *c0,
                           const float *kappa, float d0_cut, uint16_t *count)
{
    float *ex = (float *)malloc(sizeof(float) * v->n_phi), *ey = (float *)malloc(sizeof(float) * v->n_phi);
    for (uint32_t k = 0; k < v->n_phi; ++k) { ex[k] = (float)cos(vtx_phi_edge(v, k)); ey[k] = (float)sin(vtx_phi_edge(v, k)); }
    int64_t votes = 0;
    for (uint32_t j = 0; j < n_tracks; ++j) {
        if (!(fabsf(d0[j]) > d0_cut)) continue;    /* prompt-compatible track: does not vote */
        const float kd = kappa[j] * d0[j];
        const float w = 1.0f - kd;                 /* 1 - kappa d0 */
        const float d2 = d0[j] * d0[j];
        const float two_d0 = 2.0f * d0[j];         /* exact */
        for (uint32_t ir = 0; ir < v->n_r; ++ir) {
            const float r = vtx_r_centre(v, ir);
            const float r2 = r * r;
            const float t1 = r2 + d2;
            const float t2 = kappa[j] * t1;
            const float num = t2 - two_d0;         /* kappa (r^2 + d0^2) - 2 d0 */
            const float two_r = 2.0f * r;          /* exact */
            const float den = two_r * w;           /* 2 r (1 - kappa d0) */
            const float s = num / den;             /* sin of the crossing azimuth relative to phi0 */
            if (!(fabsf(s) <= 1.0f)) continue;     /* the track does not reach radius r (NaN fails too) */
            const float ss = s * s;
            const float om = 1.0f - ss;
            const float cd = sqrtf(om);            /* outgoing branch: cos >= 0 */
            const float xa = c0[j] * cd;
            const float xb = s0[j] * s;
            const float x = xa - xb;               /* cos(phi0 + asin s) */
            const float ya = s0[j] * cd;
            const float yb = c0[j] * s;
            const float y = ya + yb;               /* sin(phi0 + asin s) */
            const uint32_t iv = angle_bin(v, ex, ey, x, y);
            const size_t b = (size_t)iv * v->n_r + ir;
            count[b] = (uint16_t)(count[b] + 1);
            ++votes;
        }
    }
    free(ex); free(ey);
    return votes;
}

/*
 * O-6 + O-7 for one event's stored peaks of the FIRST transform: bin-centre track parameters
 * (d0c, phi0c tables of O-0; kappa_c = (float)(-kmax + (ik + 1/2) 2 kmax / NK) from double), vote, then the SAME
 * peak finder (oracle_peaks, rule O-3: phi_v periodic, R_v clipped, ties to the lower lin) with threshold n_min
 * (1..16) on the vertex plane.  Writes the first max_vertices vertices, returns the total; *flag = total > 0.
 * count_out (may be NULL) receives the vertex plane [n_phi][n_r].
 */
uint32_t oracle_vertices(const oracle_grid *g, const oracle_vgrid *v, const oracle_peak *peaks, uint32_t n_stored,
                         float d0_cut, uint32_t n_min, uint32_t max_vertices, oracle_vertex *out, uint8_t *flag,
                         uint16_t *count_out)
{
    const size_t bins = (size_t)v->n_phi * v->n_r;
    uint16_t *count = (uint16_t *)calloc(bins, sizeof(uint16_t));
    uint16_t *mask = (uint16_t *)calloc(bins, sizeof(uint16_t));
    float *d0 = (float *)malloc(sizeof(float) * (n_stored ? n_stored : 1));
    float *s0 = (float *)malloc(sizeof(float) * (n_stored ? n_stored : 1));
    float *c0 = (float *)malloc(sizeof(float) * (n_stored ? n_stored : 1));
    float *kap = (float *)malloc(sizeof(float) * (n_stored ? n_stored : 1));
    const double kmax = (double)g->kappa_max;
    for (uint32_t j = 0; j < n_stored; ++j) {
        const uint32_t lin = peaks[j].lin;
        const uint32_t ik = lin % g->n_kappa;
        const uint32_t ip = (lin / g->n_kappa) % g->n_phi0;
        const uint32_t id = lin / g->n_kappa / g->n_phi0;
        d0[j] = d0_centre(g, id);
        s0[j] = (float)sin(phi0_centre(g, ip));
        c0[j] = (float)cos(phi0_centre(g, ip));
        kap[j] = (float)(-kmax + ((double)ik + 0.5) * (2.0 * kmax / (double)g->n_kappa));
    }
    oracle_vertex_vote(v, n_stored, d0, s0, c0, kap, d0_cut, count);
    for (size_t b = 0; b < bins; ++b) {                       /* thermometer mask: popcount = min(count, 16) */
        const uint32_t c = count[b] < 16 ? count[b] : 16;
        mask[b] = (uint16_t)((1u << c) - 1u);
    }
    /* the same peak finder, on a 2D grid whose periodic axis is phi_v and whose clipped axis is R_v */
    oracle_grid pg;
    memset(&pg, 0, sizeof(pg));
    pg.n_d0 = 1; pg.n_phi0 = v->n_phi; pg.n_kappa = v->n_r; pg.n_layers = 16;
    oracle_peak *pk = (oracle_peak *)malloc(sizeof(oracle_peak) * (max_vertices ? max_vertices : 1));
    const uint64_t total = oracle_peaks(&pg, count, mask, n_min, max_vertices, pk);
    const uint64_t n_out = total < max_vertices ? total : max_vertices;
    for (uint64_t i = 0; i < n_out; ++i) {
        const uint32_t iv = pk[i].lin / v->n_r, ir = pk[i].lin % v->n_r;
        out[i].r = vtx_r_centre(v, ir);
        out[i].phi = (float)(((double)iv + 0.5) * (2.0 * M_PI / (double)v->n_phi));
        out[i].n_tracks = pk[i].count;
        out[i].lin = pk[i].lin;
    }
    *flag = total > 0 ? 1 : 0;
    if (count_out) memcpy(count_out, count, bins * sizeof(uint16_t));
    free(count); free(mask); free(d0); free(s0); free(c0); free(kap); free(pk);
    return (uint32_t)total;
}

/* ================================================================================================ */
/* O-2h / O-2f: physics-quality voting variants (the paper's future work is       */
/* "efficiency and purity improvements").  DESIGN.md readings R40-R42.                 */
/*   ORACLE_VOTE_HEMI  forward-hemisphere cut: a (hit, column) pair votes only if                    */
/*                     ch = fl(fl(cp*c0) + fl(sp*s0)) = cos(phi - phi0c) > 0 -- removes the mirror    */
/*                     solutions (phi0 + pi, -d0, -kappa) of reading R5 and halves the votes.         */
/*   ORACLE_VOTE_FILL  kappa-range filling: instead of one vote at the column CENTRE (R4), the O-2   */
/*                     chain is evaluated at the two phi0 EDGES of the column, phi0e(j) = j 2pi/NPHI  */
/*                     (tables of NPHI edges, each (float)cos / (float)sin of the double angle; edge  */
/*                     NPHI is edge 0), giving ua, ub; the hit votes once in EVERY kappa bin between  */
/*                     floor(min) and floor(max), clipped to the axis -- the curve of a hit becomes a  */
/*                     connected band, so tracks that are not aligned with a bin centre collect all   */
/*                     their layers in one bin.  No vote if either u is NaN or both lie on the same   */
/*                     side outside the axis.  The hemisphere test (if set) stays at the centre.      */
/* ================================================================================================ */

enum { ORACLE_VOTE_HEMI = 1u, ORACLE_VOTE_FILL = 2u };

/* u of O-2 (the kappa-bin coordinate before the range test) for one (hit, d0 bin, direction (c0, s0)) */
static float vote_u(int mode3d, float r, float r2, float sp, float cp, float c0, float s0, float d0c, float two_d0,
                    float d0sq, float kmax, float inv_dk)
{
    float m1 = sp * c0;
    float m2 = cp * s0;
    float s = m1 - m2;
    float kappa;
    if (!mode3d) {
        float two_s = 2.0f * s;
        kappa = two_s / r;
    } else {
        float rs = r * s;
        float t = rs + d0c;
        float num = 2.0f * t;
        float a = two_d0 * rs;
        float b = r2 + a;
        float den = b + d0sq;
        kappa = num / den;
    }
    float v = kappa + kmax;
    float u = v * inv_dk;
    return u;
}

int64_t oracle_vote_variant(const oracle_grid *g, uint32_t flags, uint64_t n_hits, const float *r, const float *phi,
                            const uint8_t *layer, uint16_t *count, uint16_t *mask)
{
    const int mode3d = g->n_d0 > 1;
    const float kmax = g->kappa_max;
    const float inv_dk = inv_dkappa(g);
    const float nk_f = (float)g->n_kappa;
    const int NK = (int)g->n_kappa;
    int64_t votes = 0;
    float *c0 = (float *)malloc(sizeof(float) * g->n_phi0), *s0 = (float *)malloc(sizeof(float) * g->n_phi0);
    float *ce = (float *)malloc(sizeof(float) * g->n_phi0), *se = (float *)malloc(sizeof(float) * g->n_phi0);
    float *d0c = (float *)malloc(sizeof(float) * g->n_d0);
    float inv_unused;
    oracle_tables(g, c0, s0, d0c, &inv_unused);
    for (uint32_t j = 0; j < g->n_phi0; ++j) {                 /* column edges: phi0e(j) = j * 2pi / NPHI */
        const double a = (double)j * (2.0 * M_PI / (double)g->n_phi0);
        ce[j] = (float)cos(a);
        se[j] = (float)sin(a);
    }
    for (uint64_t h = 0; h < n_hits; ++h) {
        if (layer[h] >= g->n_layers) continue;
        const float sp = hit_sin(phi[h]);
        const float cp = hit_cos(phi[h]);
        const float rr = r[h];
        const float r2 = rr * rr;
        const uint16_t bit = (uint16_t)(1u << layer[h]);
        for (uint32_t ip = 0; ip < g->n_phi0; ++ip) {
            if (flags & ORACLE_VOTE_HEMI) {
                float h1 = cp * c0[ip];
                float h2 = sp * s0[ip];
                float ch = h1 + h2;                            /* cos(phi - phi0c) */
                if (!(ch > 0.0f)) continue;
            }
            const uint32_t jp = (ip + 1 == g->n_phi0) ? 0 : ip + 1;
            for (uint32_t id = 0; id < g->n_d0; ++id) {
                const float two_d0 = 2.0f * d0c[id];
                const float d0sq = d0c[id] * d0c[id];
                int klo, khi;
                if (flags & ORACLE_VOTE_FILL) {
                    const float ua = vote_u(mode3d, rr, r2, sp, cp, ce[ip], se[ip], d0c[id], two_d0, d0sq, kmax, inv_dk);
                    const float ub = vote_u(mode3d, rr, r2, sp, cp, ce[jp], se[jp], d0c[id], two_d0, d0sq, kmax, inv_dk);
                    if (!(ua == ua) || !(ub == ub)) continue;  /* NaN at an edge: no vote */
                    const float lo = (ua < ub) ? ua : ub, hi = (ua < ub) ? ub : ua;
                    if (hi < 0.0f || lo >= nk_f) continue;     /* the whole band lies outside the axis */
                    klo = (lo < 0.0f) ? 0 : (int)lo;
                    khi = (hi >= nk_f) ? NK - 1 : (int)hi;
                } else {
                    const float u = vote_u(mode3d, rr, r2, sp, cp, c0[ip], s0[ip], d0c[id], two_d0, d0sq, kmax, inv_dk);
                    if (!(u >= 0.0f && u < nk_f)) continue;
                    klo = khi = (int)u;
                }
                for (int k = klo; k <= khi; ++k) {
                    size_t b = ((size_t)id * g->n_phi0 + ip) * g->n_kappa + (size_t)k;
                    count[b] = (uint16_t)(count[b] + 1);
                    mask[b] |= bit;
                    ++votes;
                }
            }
        }
    }
    free(c0); free(s0); free(ce); free(se); free(d0c);
    return votes;
}
