// Internal declarations shared by the translation units of libhough_b200.so (sm_100a only).
// Nothing here is visible across the C-ABI (include/hough.h) and nothing here is shared with oracle/.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include <vector>

#include "hough.h"

#define HOUGH_MAX_LAYERS 16

// hough_vertices on at most kVtxSplitEvents events runs kVtxSplit blocks per event (single-event latency)
constexpr uint32_t kVtxSplitEvents = 8;
constexpr uint32_t kVtxSplit = 16;

// Prepared hit record (float4): {RN32(sin phi), RN32(cos phi), r, bits}, bits = (0x10000 << layer) | wild, where
// "wild" marks a hit whose r is outside [2^-20, 2^20] or not finite (no window pruning, generic IEEE division).

// Hits that can reach a tile starting at phi0 column ip0, for one (layer, d0 strip): the hit's own phi0 column
// pb lies in [ip0 + a_i, ip0 + a_i + len_i) mod NPHI for i = 0 or 1.  len <= 0: no run; len >= NPHI: every hit.
struct TileWin { int a0, len0, a1, len1; };

// per event: start of the 16 layer segments and of the wild segment in the sorted records, then the end
constexpr int kSegStride = HOUGH_MAX_LAYERS + 2;

// Fused path: one peak candidate found in a vote tile.  cm = count | mask << 16; need = neighbour columns the tile
// could not check, bit (dd+1)*3 + (dp+1), and bit 9 = "count not known yet" (mask tiles: the recount fills it in);
// state = 0 pending the recount, 1 confirmed peak, 2 rejected.
struct PeakCand { uint32_t lin, cm, need, state; };

struct VotePlan {
    int k_lane;                      // KL: rows per lane; a tile has 32 * KL rows
    int tile_w;                      // phi0 columns per tile (8 in 3D, 32 * KL in 2D)
    int ids_per_tile;                // d0 bins per tile (4 * KL in 3D, 1 in 2D)
    int sh;                          // phi bucket of the hit sort = phi0 column >> sh
    uint32_t nb;                     // phi buckets per layer
    uint32_t stage_hits;             // records per stage of the hit ring
    int nk_tile;                     // kappa bins per tile (<= NK; NK split into nk_seg segments if it does not fit)
    int nk_seg;
    int threads;
    size_t smem_bytes;
    int n_strips, n_tiles;           // ceil(ND/K), ceil(NPHI/W)  (mirror: (NPHI/2)/W)
    bool mirror;                     // mirror tiles: each (hit, row) evaluation also votes the row's mirror image
};

struct PeakPlan {
    int unit_bins;                   // bins per lane-load of the stencil: 16 (256-bit) or 8 (128-bit)
    int blocks_per_sm[2];            // resident blocks of the 128-bit / 256-bit kernel
    int threads;
};

struct hough_ctx {
    hough_config cfg;
    int device;
    int sm_count;
    // constant tables (device), fp32 rounded once from double
    float* d_c0; float* d_s0;                 // [NPHI]
    float* d_d0c; float* d_two_d0; float* d_d0sq;   // [ND]
    float kmax, inv_dk, nk_f;
    float* d_ce; float* d_se;                 // [NPHI] (cos, sin) of the phi0 column edges j * 2pi / NPHI (voting variant FILL)
    float* d_kc;                              // [NK] kappa bin centres, fp32 rounded once from double (O-6)
    float* d_vex; float* d_vey;               // [n_vtx_phi] phi_v bin-edge directions (cos, sin)(k * 2pi / n_vtx_phi)
    float* d_vrc;                             // [n_vtx_r] R_v bin centres
    uint32_t* d_vtx_gplane;                   // [kVtxSplitEvents][n_vtx_phi * n_vtx_r / 2] vertex planes of the split kernel (zero between calls)
    uint32_t* d_vtx_done;                     // [kVtxSplitEvents] finished-block counters of the split kernel (zero between calls)
    bool tame_tables;                         // d0 centres and kappa_max inside the range div_rn_tame is proven for
    // per-call workspace
    float4* d_rec_u;                          // [max_hits] prepared hits in input order (sort scratch)
    uint32_t* d_key;                          // [max_hits] sort keys (sort scratch)
    float4* d_rec;                            // [max_hits] prepared hits sorted per event by (layer, phi bucket)
    uint32_t* d_seg;                          // [max_events][kSegStride]
    uint16_t* d_btab;                         // [max_events][16][nb + 1] bucket starts relative to the layer segment
    uint32_t* d_layer_r;                      // [4*16] float bits: min r, max r per layer (live), then the last call's copy
    TileWin* d_tilewin;                       // [nk_seg][16][n_strips]
    TileWin* d_tilewin_mo;                    // the same for the mask-tile plan of the fused path (vote_mo), if any
    uint32_t* d_status;                       // [2]: sticky bits, trig-risk counter
    uint32_t* d_tilectr;                      // [2]: vote kernel tile ticket + finished-block count (zero between launches)
    uint32_t plane_events;                    // events per hough_peaks call: cfg.max_plane_events, or max_events if that is 0
    uint8_t* d_bitmap;                        // [plane_events][bins/8], a group's bytes defined where d_grpcnt > 0
    uint16_t* d_grpcnt;                       // [plane_events][ceil(bins/256)] peaks per group of 256 / 512 bins
    uint64_t* d_jetkeys;                      // [max_events][max_peaks]
    // fused vote -> peaks
    uint32_t fused_events;                    // events per fused launch the buffers below are sized for
    uint32_t cand_cap, cand_cap_pow2;         // candidates per event (cfg.max_candidates_per_event or its default)
    PeakCand* d_cand;                         // [fused_events][cand_cap]
    uint32_t* d_cand_n;                       // [fused_events], zero between calls
    unsigned long long* d_sortkeys;           // [fused_events][cand_cap_pow2] sort scratch for events beyond the SMEM sort
    // host path
    uint16_t* d_hp_count; uint16_t* d_hp_mask;     // [bins]: the planes of ONE event (fallback of hough_trigger_host)
    uint32_t* d_hp_off; float* d_hp_r; float* d_hp_phi; uint8_t* d_hp_layer;
    hough_peak* d_hp_peaks; hough_track* d_hp_tracks; hough_jet* d_hp_jets;
    uint32_t* d_hp_npeaks; uint32_t* d_hp_njets; uint8_t* d_hp_flag;
    hough_vertex* d_hp_vertices; uint32_t* d_hp_nvtx; uint8_t* d_hp_vflag;
    // per-stage CUDA-event timing (hough_profile): marks recorded on the caller's stream around the launches
    bool prof_on;
    std::vector<cudaEvent_t> ev_pool;         // created on first use, reused, freed in hough_destroy
    std::vector<int> ev_label;                // stage that STARTS at the mark (0 prep, 1 vote, 2 peaks, 3 jets, 4 vertices), -1: end of a call
    size_t ev_used;
    VotePlan vote;
    VotePlan vote_mo;                         // fused path, mask-only mirror tiles (has_mo): larger kappa range per tile
    bool has_mo;
    int fused_scheme;                         // 0: choose per call by occupancy, 1: count + mask tiles, 2: mask tiles (cfg.debug_flags)
    int last_tile_kind;                       // tiles the last fused launch started with: 0 none yet, 1 count + mask, 2 mask (hough_last_tile_kind)
    double prep_hits_per_event;               // mean hits per event of the last launch_prep (tile choice of the fused path)
    uint32_t* d_redo;                         // [1 + fused_events]: number and indices of the events whose mask-tile candidates overflowed
    PeakPlan peak;
    cudaStream_t last_stream;
    uint64_t launches;
    uint32_t status_host;
};

// launchers (each returns a cudaError_t from the launch; all asynchronous on `st`)
cudaError_t launch_prep(hough_ctx* c, uint32_t n_events, const uint32_t* d_off, uint64_t n_hits,
                        const float* d_r, const float* d_phi, const uint8_t* d_layer, cudaStream_t st);
cudaError_t launch_vote(hough_ctx* c, uint32_t first_event, uint32_t n_events, uint16_t* d_count, uint16_t* d_mask,
                        cudaStream_t st);
cudaError_t launch_peaks(hough_ctx* c, uint32_t n_events, const uint16_t* d_count, const uint16_t* d_mask,
                         uint32_t l_min, hough_peak* d_peaks, uint32_t* d_n_peaks, cudaStream_t st);
cudaError_t launch_jets(hough_ctx* c, uint32_t n_events, const hough_peak* d_peaks, const uint32_t* d_n_peaks,
                        int cone_bins, float d0_cut, uint32_t n_min, hough_track* d_tracks, hough_jet* d_jets,
                        uint32_t* d_n_jets, uint8_t* d_flag, cudaStream_t st);
// hough_jets_static: no context; scratch in the library's own static device array (jets.cu)
cudaError_t launch_jets_static(const hough_config* g, uint32_t n_events, const hough_peak* d_peaks,
                               const uint32_t* d_n_peaks, int cone_bins, float d0_cut, uint32_t n_min,
                               hough_track* d_tracks, hough_jet* d_jets, uint32_t* d_n_jets, uint8_t* d_flag,
                               cudaStream_t st);
cudaError_t launch_vote_fused(hough_ctx* c, uint32_t first_event, uint32_t n_events, uint32_t l_min, cudaStream_t st);
cudaError_t launch_recount(hough_ctx* c, uint32_t first_event, uint32_t n_events, cudaStream_t st);
cudaError_t launch_peaks_finalize(hough_ctx* c, uint32_t n_events, hough_peak* d_peaks, uint32_t* d_n_peaks,
                                  cudaStream_t st);
cudaError_t launch_vertices(hough_ctx* c, uint32_t n_events, const hough_peak* d_peaks, const uint32_t* d_n_peaks,
                            float d0_cut, uint32_t n_min, hough_vertex* d_vertices, uint32_t* d_n_vertices,
                            uint8_t* d_flag, uint16_t* d_plane, cudaStream_t st);
cudaError_t plan_vote(hough_ctx* c, bool mirror_ok);
cudaError_t plan_peaks(hough_ctx* c);
cudaError_t run_div_check(uint64_t n_pairs, uint64_t seed, float kmax, int nk, unsigned long long* host_out3);
