/*
 * hough.h -- C-ABI boundary of the B200-native Hough trigger hot path.
 *
 * Method: Halyo, LeGresley, Lujan, "Massively Parallel Computing and the Search for Jets and Black Holes
 * at the LHC", arXiv:1309.6275 (text in PAPER.md).  The paper gives the pipeline in words only
 * (section 6: "the hit data for an event is processed using the Hough transform to compute
 * the parameter space representation.  Candidate tracks are identified by finding local maxima, or peaks,
 * in the parameter space"); the concrete formulas, bin layout and selection rules are those of
 * BASELINE.json:north_star as read in DESIGN.md ("Readings").
 *
 * Everything here is plain C: opaque context, POD structs, raw pointers.  Unless a parameter is marked
 * HOST, every pointer is a DEVICE pointer owned (allocated and freed) by the caller; `stream` is a
 * cudaStream_t passed as void*.  All work is enqueued on `stream`; only hough_create, hough_destroy,
 * hough_status, hough_trigger_host and hough_microbench synchronise.  Calls on one context must be
 * stream-ordered by the caller (the context owns a per-call workspace).  No entry point allocates or
 * frees device memory except hough_create / hough_destroy (hough_jets_static needs neither of them).
 * There is no CPU fallback anywhere: without a CUDA device hough_create fails with HOUGH_ECUDA.
 *
 * Notation: E events; ND, NPHI, NK bins in d0, phi0, kappa; bin (id, ip, ik) has linear index
 * lin = (id*NPHI + ip)*NK + ik (kappa fastest).  Units: mm, rad, 1/mm, T, GeV.
 */
#ifndef HOUGH_H_
#define HOUGH_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct hough_ctx hough_ctx;

typedef struct {
    uint32_t n_phi0;               /* phi0 bins over [0, 2pi), centres (ip + 1/2) * 2pi/NPHI; >= 4                    */
    uint32_t n_kappa;              /* kappa bins over [-kappa_max, +kappa_max), half-open; multiple of 8, >= 8        */
    uint32_t n_d0;                 /* 1 -> prompt 2D mode (d0 == 0, kappa = 2 s / r); >= 2 -> 3D mode                 */
    float    kappa_max;            /* 1/mm, > 0 (configs: 0.3e-3 * 3.8 / 1.0)                                         */
    float    d0_min, d0_max;       /* mm; d0 bins over [d0_min, d0_max), centres; ignored in 2D mode                  */
    float    b_tesla;              /* only used for pT = 0.3e-3 * B / |kappa|                                         */
    uint32_t n_layers;             /* 1..16 (layer mask is 16 bits); hits with layer >= n_layers are ignored          */
    uint32_t max_events;           /* per call, <= 1<<20                                                              */
    uint64_t max_hits;             /* per call, total over events (sizes the prepared-hit workspace), < 2^32          */
    uint32_t max_peaks_per_event;  /* capacity of the per-event peak / track lists                                    */
    uint32_t max_jets_per_event;   /* capacity of the per-event jet list                                              */
    uint32_t host_chunk_events;    /* hough_trigger_host: events per internal launch; 0 disables that entry point.
                                      If > 0 the context owns host staging buffers for max_events / max_hits, the
                                      planes of ONE event (fallback for events that overflow the candidate buffer),
                                      and hough_vote_peaks accepts at most host_chunk_events events per call        */
    uint32_t max_candidates_per_event; /* fused path: capacity of the per-event peak-candidate buffer (16 B each);
                                      0 = default max(4 * max_peaks_per_event, 4096)                                  */
    /* vertex space of the second Hough transform (hough_vertices); n_vtx_phi == 0 disables it */
    uint32_t n_vtx_phi;            /* phi_v bins over [0, 2pi), periodic; multiple of 4, >= 8                         */
    uint32_t n_vtx_r;              /* R_v bins over [vtx_r_min, vtx_r_max), half-open; multiple of 8, >= 8;
                                      n_vtx_phi * n_vtx_r * 2 bytes must fit in shared memory (<= 200 KB)            */
    float    vtx_r_min, vtx_r_max; /* mm; vtx_r_min = radius inside which vertices are dropped (beam pipe, 30 mm)     */
    uint32_t max_vertices_per_event; /* with a vertex grid, max_peaks_per_event must be <= 65535 (16-bit vertex counts)  */
    uint32_t vote_flags;           /* physics-quality voting variants (O-2h / O-2f), accumulator
                                      path only: HOUGH_VOTE_HEMI | HOUGH_VOTE_FILL; 0 = the normative one-vote-per-column-
                                      centre rule of north_star.  hough_vote_peaks / hough_trigger_host* return
                                      HOUGH_EUNSUPPORTED when it is not 0                                             */
    uint32_t max_plane_events;     /* accumulator path: events per hough_peaks call the peak finder's scratch is sized for
                                      (per event: 1 bit per bin + 2 B per 256 bins); 0 = max_events.  hough_peaks returns
                                      HOUGH_EINVAL beyond it.  A context that is only used through hough_vote_peaks /
                                      hough_trigger_host* can set 1 (the host path's overflow fallback needs one event): on
                                      C5 that is 8.4 MB instead of 34 GB for max_events = 4096                           */
    uint32_t debug_flags;          /* HOUGH_DEBUG_*: which kernel variant runs where the library would choose by itself.
                                      For tests and measurements; 0 in production.  They change speed, never results.
                                      (The library reads no environment variable and keeps no state outside a context,
                                      SURVEY.md section 5.)                                                             */
} hough_config;

enum {
    HOUGH_DEBUG_NO_MIRROR = 1u,    /* plain tiles also on grids whose tables allow mirror tiles (hence no mask tiles)   */
    HOUGH_DEBUG_TILES_COUNT = 2u,  /* hough_vote_peaks: always count + mask tiles                                       */
    HOUGH_DEBUG_TILES_MASK = 4u    /* hough_vote_peaks: mask tiles whenever the grid has them (not both TILES bits)     */
};

enum {
    HOUGH_VOTE_HEMI = 1u,   /* forward-hemisphere cut: a (hit, column) votes only if cos(phi - phi0c) > 0 (no mirror peaks) */
    HOUGH_VOTE_FILL = 2u    /* kappa-range filling: one vote in every kappa bin between the values at the two phi0 edges
                               of the column, so a hit's curve is a connected band ("efficiency ... improvements") */
};

typedef struct { uint32_t lin; uint16_t count; uint16_t mask; } hough_peak;                     /*  8 B */
typedef struct { float pt, phi0, d0; int32_t q; int32_t jet; } hough_track;                     /* 20 B */
typedef struct { uint32_t seed_track, n_tracks, n_displaced; float phi, sum_pt; } hough_jet;    /* 20 B */
typedef struct { float r, phi; uint32_t n_tracks; uint32_t lin; } hough_vertex;                 /* 16 B */

enum {
    HOUGH_OK = 0,
    HOUGH_EINVAL = -1,       /* bad config / null pointer / size over the configured maximum / bad scalar argument */
    HOUGH_ECUDA = -2,        /* CUDA runtime error (text via hough_strerror)                                        */
    HOUGH_ENOMEM = -3,       /* device allocation failed in hough_create                                            */
    HOUGH_EUNSUPPORTED = -4, /* configuration valid but outside what the kernels are built for                      */
    HOUGH_ETOOLARGE = -5     /* hough_jets_static: the call needs more scratch than the library's fixed array holds  */
};

/* sticky status bits (hough_status) for conditions only visible on the device; they never trap */
enum {
    HOUGH_ST_EVENT_TOO_LARGE = 1u,   /* an event has > 65535 hits: its counts may wrap (uint16), results undefined  */
    HOUGH_ST_BAD_OFFSETS = 2u,       /* hit_offsets not non-decreasing or beyond n_hits_total                        */
    HOUGH_ST_CANDIDATE_OVERFLOW = 8u,/* hough_vote_peaks: an event had more peak candidates than
                                        max_candidates_per_event; its n_peaks reads HOUGH_N_PEAKS_OVERFLOW           */
    HOUGH_ST_TRIG_ROUNDING = 4u      /* informational: some sin/cos(phi) lay within a few fp64 ulps of an fp32
                                        rounding boundary, so its correctly-rounded fp32 value is not certain
                                        (reading R6; probability ~1e-8 per hit)                            */
};

/*
 * Create a context.  HOST pointers.  Validates cfg, builds the constant tables in double precision
 * (cos/sin of the phi0 bin centres, d0 bin centres, 2*d0, d0^2, NK/(2*kappa_max)), rounds each once to
 * fp32, uploads them, and allocates ALL the workspaces: no other call allocates (no hidden
 * allocations).  Device footprint in bytes, with bins = ND*NPHI*NK, PE = max_plane_events (or max_events if 0),
 * FE = host_chunk_events (or max_events if 0), CC = max_candidates_per_event (or its default), CC2 = CC rounded up to
 * a power of two:
 *     36 * max_hits                                        prepared hits (sorted + unsorted record, sort key)
 *   + PE * (bins / 8 + 2 * ceil(bins / 256))               peak bitmap and group counts of hough_peaks
 *   + 8 * max_events * max_peaks_per_event                 clustering keys of hough_jets
 *   + FE * (16 * CC + 8 * CC2 + 8)                         fused path: candidates, their sort keys, counters
 *   + tables and per-event segment / bucket tables         (a few KB per event)
 * and, if host_chunk_events > 0 (hough_trigger_host*):
 *   + 9 * max_hits + 4 * bins                              staged hits; the planes of ONE event (overflow fallback)
 *   + max_events * (28 * max_peaks_per_event + 20 * max_jets_per_event + 16 * max_vertices_per_event + 18)
 *                                                          peak / track / jet / vertex lists and counters of the batch
 * Synchronous.
 */
int hough_create(const hough_config* cfg, hough_ctx** out);
int hough_destroy(hough_ctx* ctx);

/* bytes of ONE accumulator plane (count or mask) for n_events events: n_events * ND*NPHI*NK * 2 */
size_t hough_plane_bytes(const hough_ctx* ctx, uint32_t n_events);

/*
 * A0-A2  Hough vote ("for each piece of input data votes are added to the feature instances that
 * would include that input data"; "prompt or non-prompt tracks").  For every hit h of event e and
 * every (id, ip): s = sin(phi_h - phi0c(ip)) (formed as sin(phi)cos(phi0c) - cos(phi)sin(phi0c) from
 * correctly-rounded fp32 factors), kappa = 2 (r s + d0c) / (r^2 + 2 d0c r s + d0c^2)  (2D: 2 s / r), in IEEE
 * fp32 without FMA in the fixed order of DESIGN.md O-2; if floor((kappa + kappa_max) * NK/(2 kappa_max)) is in
 * [0, NK): count[e][id][ip][ik] += 1 and mask[e][id][ip][ik] |= 1 << layer_h.
 *
 *   d_hit_offsets [n_events+1] u32  CSR, non-decreasing.  off[0] is the base: hits of event e are the elements
 *                 [off[e]-off[0], off[e+1]-off[0]) of d_r / d_phi / d_layer, so a sub-batch of a larger CSR batch
 *                 is passed as (offsets + e0, r + off[e0], ...); off[n_events]-off[0] <= n_hits_total
 *   d_r, d_phi    [n_hits_total] f32, d_layer [n_hits_total] u8   (r > 0 expected; any float is handled IEEE-wise)
 *   d_count, d_mask [n_events][ND][NPHI][NK] u16 each, 16-byte aligned; FULLY overwritten (no memset needed)
 * Precondition: <= 65535 hits per event (else HOUGH_ST_EVENT_TOO_LARGE is raised).
 * Returns HOUGH_EINVAL if n_events > max_events or n_hits_total > max_hits or a pointer is null.
 */
int hough_vote(hough_ctx* ctx, uint32_t n_events, const uint32_t* d_hit_offsets, uint64_t n_hits_total,
               const float* d_r, const float* d_phi, const uint8_t* d_layer,
               uint16_t* d_count, uint16_t* d_mask, void* stream);

/*
 * A3-A4  Peak finding + ordered compaction ("looking for local maxima in the parameter space").
 * Bin b is a peak iff popcount(mask[b]) >= l_min and (count[b], -lin(b)) is strictly greatest over its 3x3
 * (2D) / 3x3x3 (3D) neighbourhood; phi0 is periodic, kappa and d0 are clipped.  Peaks of each event are
 * written in ascending lin.
 *   d_peaks   [n_events][max_peaks_per_event]; only the first min(n_peaks[e], max_peaks) records are written
 *   d_n_peaks [n_events] u32: the TRUE number of peaks found (may exceed the capacity)
 * l_min must be in [1, n_layers]; n_events <= max_plane_events (if that is not 0) and <= max_events.
 * Precondition: the planes are accumulators as hough_vote writes them, i.e.
 * count[b] >= popcount(mask[b]) for every bin (a bin with count < l_min is rejected without reading its mask).
 */
int hough_peaks(hough_ctx* ctx, uint32_t n_events, const uint16_t* d_count, const uint16_t* d_mask,
                uint32_t l_min, hough_peak* d_peaks, uint32_t* d_n_peaks, void* stream);

/*
 * A0-A4 fused  Vote -> peaks without the accumulator in HBM ("the hit data ... is
 * processed using the Hough transform to compute the parameter space representation.  Candidate tracks are
 * identified by finding local maxima", and PAPER.md:109: the transform is limited "more by memory access
 * operations rather than the computational rate").  Same result as hough_vote followed by hough_peaks -- the same
 * peaks, in ascending lin, with the same count / mask, and the true total -- but the vote kernel finds the peak
 * candidates (popcount(mask) >= l_min) while its tile is in shared memory and a second kernel recomputes, from the
 * hits, the counts it needs (O-2 verbatim, so the counts are the accumulator's).  No plane is written.  Two kinds
 * of tile: "mask tiles" accumulate only the layer masks (one shared reduction per vote, twice the
 * kappa range per tile) and have the count of every candidate and of its 26 neighbours recomputed; "count + mask
 * tiles" accumulate both, compare a candidate with its neighbours inside the tile and have only the neighbours
 * across a tile border recomputed.  A call starts with mask tiles when the grid allows them (mirror-symmetric
 * tables) and few chance candidates are expected, and votes the events whose candidates overflow the buffer again
 * with count + mask tiles, on the device; the result does not depend on the kind of tile (hough_config.debug_flags
 * HOUGH_DEBUG_TILES_MASK / HOUGH_DEBUG_TILES_COUNT force one: tests).
 *   arguments as hough_vote / hough_peaks.  Capacity: if an event has more than max_candidates_per_event
 *   candidates (count + mask tiles), HOUGH_ST_CANDIDATE_OVERFLOW is raised and d_n_peaks[e] =
 *   HOUGH_N_PEAKS_OVERFLOW (no record of that event is valid; hough_jets treats it as an event without tracks):
 *   re-run such events through hough_vote + hough_peaks (hough_trigger_host does).
 * Returns HOUGH_EINVAL as hough_vote / hough_peaks do, and if n_events exceeds the fused capacity
 * (host_chunk_events if that is > 0, else max_events).
 */
#define HOUGH_N_PEAKS_OVERFLOW 0xFFFFFFFFu
int hough_vote_peaks(hough_ctx* ctx, uint32_t n_events, const uint32_t* d_hit_offsets, uint64_t n_hits_total,
                     const float* d_r, const float* d_phi, const uint8_t* d_layer, uint32_t l_min,
                     hough_peak* d_peaks, uint32_t* d_n_peaks, void* stream);

/*
 * A5-A6  Peak -> track conversion and phi-cone track-jets ("measure ... the transverse momentum";
 * PAPER.md:113-123 jets / displaced jets, in north_star's phi-cone form).  For the T = min(n_peaks, max_peaks)
 * stored peaks of each event: track j = {pT = 0.3e-3*B/|kappa_c|, phi0_c, d0_c, q = -sign(kappa_c), jet};
 * seeded fixed-cone clustering on integer bin keys: seed = unassigned track with the smallest
 * (|2 ik - (NK-1)|, j); members = unassigned tracks within floor(cone_rad*NPHI/2pi) phi0 bins (wrapped,
 * inclusive); a track is displaced iff |d0_c| > d0_cut_mm; flag[e] = 1 iff some jet has
 * n_displaced >= n_displaced_min.
 *   d_tracks [n_events][max_peaks_per_event], d_jets [n_events][max_jets_per_event],
 *   d_n_jets [n_events] u32 TRUE number of jets, d_flag [n_events] u8.
 * Tracks of jets beyond the capacity keep jet = -1.
 */
int hough_jets(hough_ctx* ctx, uint32_t n_events, const hough_peak* d_peaks, const uint32_t* d_n_peaks,
               float cone_rad, float d0_cut_mm, uint32_t n_displaced_min,
               hough_track* d_tracks, hough_jet* d_jets, uint32_t* d_n_jets, uint8_t* d_flag, void* stream);

/*
 * hough_jets without a context and without any allocation -- for callers that are not allowed to allocate.
 *
 * Who that is: a trigger process that handed out all of its device memory at start-up and runs under a fixed
 * budget (a cudaMalloc there fails, or is forbidden by the experiment's framework); a latency-critical loop, where
 * cudaMalloc / cudaFree would stall every stream of the device; a plug-in hosted by another runtime that owns the
 * allocator and hands the plug-in nothing but its input and output buffers.  None of them can call hough_create,
 * which allocates the workspaces of the whole path.  This one call gives them A5-A6 (same definition, same kernel
 * and same results as hough_jets: PAPER.md:87): it takes the grid description from a HOST
 * hough_config, the inputs and outputs from the caller, and keeps its two pieces of scratch -- the table of d0 bin
 * centres and the clustering keys of events with more than 4096 tracks -- in an array that is part of the
 * library's device image (a file-scope `static __device__` array in csrc/jets.cu, about 4 MB, held by every GPU
 * that loads the library until the process exits).  It calls no cudaMalloc, cudaFree or allocating library routine.
 *
 *   cfg   HOST.  Read: n_phi0, n_kappa, n_d0, kappa_max, d0_min, d0_max, b_tesla, max_peaks_per_event,
 *         max_jets_per_event (checked as hough_create checks them); every other field is ignored.
 *   other arguments: DEVICE pointers, exactly as hough_jets.
 * Limits (the scratch is fixed): n_events * max_peaks_per_event <= HOUGH_JETS_STATIC_MAX_TRACKS and
 * n_d0 <= HOUGH_JETS_STATIC_MAX_D0; beyond them the call does nothing and returns HOUGH_ETOOLARGE.
 * HOUGH_EINVAL for a null pointer or a bad cfg / cone_rad / d0_cut_mm; HOUGH_ECUDA as elsewhere.
 *
 * Set-up: the first call on each device (with that device current) looks up the device address of the scratch
 * array once and checks that the device is sm_100-class; make that first call before any stream capture.
 * Sharing: every call on a device uses the same array.  Nothing in it has to start at zero -- each call writes the
 * d0 table and every key it later reads -- but it keeps the last call's contents, so two calls that overlap on the
 * GPU (different streams, no dependency between them) race: order them on one stream or with events.
 * Asynchronous on `stream` like hough_jets.
 */
#define HOUGH_JETS_STATIC_MAX_TRACKS (1u << 19)   /* 524 288 clustering keys of 8 B = 4 MiB */
#define HOUGH_JETS_STATIC_MAX_D0 4096u            /* d0 bin centres, 16 KiB                 */
int hough_jets_static(const hough_config* cfg, uint32_t n_events, const hough_peak* d_peaks, const uint32_t* d_n_peaks,
                      float cone_rad, float d0_cut_mm, uint32_t n_displaced_min,
                      hough_track* d_tracks, hough_jet* d_jets, uint32_t* d_n_jets, uint8_t* d_flag, void* stream);

/*
 * The paper's SECOND Hough transform: tracks -> displaced vertices (section 6: "the corresponding
 * parameter space representation of these tracks is processed by a second application of the Hough transform ...
 * to identify not straight lines but sinusoids which contain a significant number of tracks ... the same peak
 * finding algorithm is applied to the parameter space of this second Hough transform"; the tracks from
 * the interaction point are excluded "by setting a lower bound on the radius"; cost proportional to
 * the number of tracks).  DESIGN.md O-6 / O-7.
 * For the T = min(n_peaks, max_peaks) stored peaks of each event (bin-centre track parameters d0c, phi0c, kappa_c):
 * every track with |d0c| > d0_cut_mm votes, for each R_v bin centre r it reaches, into the phi_v bin of the azimuth
 * phi0 + asin(s), s = (kappa (r^2 + d0^2) - 2 d0) / (2 r (1 - kappa d0)), at which its outgoing branch crosses
 * radius r (to first order d0 = R_v sin(phi0 - phi_v): the sinusoid of the paper), in IEEE fp32 without a
 * transcendental per vote.  Vertices = bins of the (phi_v, R_v) plane with count >= n_min that are strict local
 * maxima of (count, -lin) over the 3x3 neighbourhood (phi_v periodic, R_v clipped), lin = iv * NR + ir, in
 * ascending lin; r / phi are bin centres, n_tracks the count.
 *   d_vertices   [n_events][max_vertices_per_event]; d_n_vertices [n_events] u32 TRUE total; d_flag [n_events] u8
 *   = 1 iff the event has a vertex;  d_vertex_plane: optional (may be null) [n_events][n_vtx_phi][n_vtx_r] u16,
 *   receives the vote counts (tests).
 * n_min in [1, HOUGH_VTX_N_MIN_MAX]: the range over which the result is checked against the oracle (its reuse of the
 * peak finder, "the same peak finding algorithm", covers thresholds up to 16); HOUGH_EINVAL outside it, and
 * if the context was created without a vertex grid.  Counts are 16-bit: a context with a vertex grid must have
 * max_peaks_per_event <= 65535 (hough_create rejects more), so no bin can receive more votes than it can hold.
 */
#define HOUGH_VTX_N_MIN_MAX 16u
int hough_vertices(hough_ctx* ctx, uint32_t n_events, const hough_peak* d_peaks, const uint32_t* d_n_peaks,
                   float d0_cut_mm, uint32_t n_min, hough_vertex* d_vertices, uint32_t* d_n_vertices, uint8_t* d_flag,
                   uint16_t* d_vertex_plane, void* stream);

/*
 * End-to-end trigger on HOST buffers (the call bench.py's e2e leg times): copies the hits to the device,
 * runs the fused vote -> peaks path and the jets in launches of cfg.host_chunk_events events, and copies
 * n_peaks / n_jets / flag (and, if non-null, peaks and jets) back.  Events that overflowed the candidate buffer
 * are re-run one by one through the accumulator path (hough_vote + hough_peaks on the context's one-event planes),
 * so the results are always those of the definition.  All h_* pointers are HOST memory (pinned memory makes the
 * copies asynchronous); synchronises `stream` before returning.
 * ms_stage (HOST, may be null) receives the device time in ms spent in {vote (incl. candidate scan), peaks
 * (recount + ordering), jets}, the fallback's launches included.  A call with ms_stage uses the context's stage
 * profile: it starts from an empty profile (intervals accumulated with hough_profile and not yet read are dropped)
 * and leaves hough_profile's on / off setting as it found it, also when it returns an error.
 * Status: the overflow is repaired inside the call, so the call clears HOUGH_ST_CANDIDATE_OVERFLOW on the device
 * after the last fallback (a bit raised by an earlier hough_vote_peaks on this context and not yet read by
 * hough_status goes with it); the other status bits are untouched.
 */
int hough_trigger_host(hough_ctx* ctx, uint32_t n_events, const uint32_t* h_hit_offsets, uint64_t n_hits_total,
                       const float* h_r, const float* h_phi, const uint8_t* h_layer,
                       uint32_t l_min, float cone_rad, float d0_cut_mm, uint32_t n_displaced_min,
                       uint32_t* h_n_peaks, uint32_t* h_n_jets, uint8_t* h_flag,
                       hough_peak* h_peaks /* [n_events][max_peaks] or null */,
                       hough_jet* h_jets /* [n_events][max_jets] or null */,
                       float* ms_stage /* [3] or null */, void* stream);

/*
 * The same with the second Hough transform run after the jets (context created with a vertex grid):
 * h_n_vertices [n_events] u32, h_vtx_flag [n_events] u8, h_vertices [n_events][max_vertices] or null.
 * vtx_n_min = 0 skips the second transform; otherwise it is hough_vertices' n_min (1..HOUGH_VTX_N_MIN_MAX).
 * ms_stage, if not null, has FOUR entries: {vote, peaks, jets, vertices}.
 */
int hough_trigger_host_vtx(hough_ctx* ctx, uint32_t n_events, const uint32_t* h_hit_offsets, uint64_t n_hits_total,
                           const float* h_r, const float* h_phi, const uint8_t* h_layer,
                           uint32_t l_min, float cone_rad, float d0_cut_mm, uint32_t n_displaced_min,
                           uint32_t vtx_n_min,
                           uint32_t* h_n_peaks, uint32_t* h_n_jets, uint8_t* h_flag,
                           hough_peak* h_peaks, hough_jet* h_jets,
                           uint32_t* h_n_vertices, uint8_t* h_vtx_flag, hough_vertex* h_vertices,
                           float* ms_stage /* [4] or null */, void* stream);

/* Synchronises the stream of the last call on ctx and returns (and keeps) the sticky status bits.  HOST out. */
int hough_status(hough_ctx* ctx, uint32_t* host_status_bits);

/*
 * Per-stage device timing with CUDA events on the caller's stream (what bench.py's roofline uses).  While enabled,
 * every call on ctx records an event before each stage and one at its end.  hough_profile_read waits for the last
 * recorded event and returns the milliseconds accumulated since the previous read in
 * h_ms[0..4] = {hit preparation, vote kernel, peak kernels (stencil + compaction, or recount + ordering), jets,
 * vertices} and the number of calls seen.  HOST out.  Costs one event record (a few microseconds) per stage while enabled.
 */
int hough_profile(hough_ctx* ctx, int enable);
int hough_profile_read(hough_ctx* ctx, float* h_ms /* [5] */, uint32_t* h_calls /* may be null */);

/*
 * Which kind of tile the last fused launch on ctx (hough_vote_peaks, or the last chunk of hough_trigger_host*) STARTED
 * with -- the library's own speed heuristic unless debug_flags forces one: 0 = no fused launch yet,
 * 1 = count + mask tiles (two shared reductions per vote), 2 = mask tiles (one shared reduction per vote; events whose
 * candidates overflowed were voted again with count + mask tiles).  The result never depends on it; bench.py uses it to
 * charge the right number of shared reductions in the roofline.  HOST out.
 */
int hough_last_tile_kind(const hough_ctx* ctx, int* host_kind);

/* Number of kernel launches this context has enqueued since creation (bench.py's gpu_launches).  HOST out. */
int hough_launch_count(const hough_ctx* ctx, uint64_t* host_count);

/*
 * Roofline micro-benchmarks: measured on the current device, synchronous.
 *   kind 0: conflict-free 32-bit shared-memory atomics (add + or, result unused)   -> atomics / s
 *   kind 1: dependent-free fp32 non-FMA arithmetic (FADD/FMUL)                      -> thread-instructions / s
 *   kind 2: HBM read  (sum-reduce a buffer of `bytes`)                              -> bytes / s
 *   kind 3: HBM write (fill a buffer of `bytes`)                                    -> bytes / s
 *   kind 4: packed fp32x2 non-FMA arithmetic (FMUL2/FADD2, register operands)       -> packed thread-instructions / s
 *   kind 5: stores of all SMs into an L2-resident buffer, fully coalesced           -> bytes / s
 *   kind 6: the same with the vote flush's pattern (64 B per lane pair, 1 KB rows)  -> bytes / s
 * `bytes` is only used by kinds 2 and 3.  HOST out.
 */
int hough_microbench(int kind, size_t bytes, double* host_rate);

/*
 * Debug exports (synchronous, HOST out; not part of the hot path).
 *
 * hough_debug_prepared_hits: the prepared records of the LAST hough_vote / hough_trigger_host call on ctx, in the
 *   caller's hit order: h_rec[4*h + 0..3] = {RN32(sin phi_h), RN32(cos phi_h), r_h, bit pattern 0x10000 << layer_h}
 *   (O-1; hits that are ignored -- layer >= n_layers or non-finite phi -- read {0, 1, r, 0}).  Lets a test compare
 *   sp / cp bit for bit with the oracle's (reading R6: the residual double-rounding risk that
 *   HOUGH_ST_TRIG_ROUNDING reports).  h_trig_risk (may be null) receives the number of hits the device flagged.
 * hough_debug_div_check: runs the vote kernel's branch-free division and packed O-2 tail next to the plain IEEE
 *   reference (__fdiv_rn, scalar tail) on n_pairs generated operand pairs (tame range, rounding midpoints, bin
 *   edges, vanishing denominators) for a kappa axis of n_kappa bins over +-kappa_max.
 *   h_out[0] = quotients that differ in any bit, h_out[1] = bin decisions that differ, h_out[2] = pairs that
 *   landed inside the axis (the test is not vacuous).  DESIGN.md readings R31-R33.
 */
int hough_debug_prepared_hits(hough_ctx* ctx, uint64_t n_hits, float* h_rec /* [n_hits][4] */, uint32_t* h_trig_risk);
int hough_debug_div_check(uint64_t n_pairs, uint64_t seed, float kappa_max, uint32_t n_kappa, uint64_t* h_out /* [3] */);

const char* hough_strerror(int code);

#ifdef __cplusplus
}
#endif
#endif /* HOUGH_H_ */
