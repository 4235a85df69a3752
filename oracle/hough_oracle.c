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
