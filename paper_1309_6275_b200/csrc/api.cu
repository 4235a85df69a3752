// C-ABI entry points of libhough_b200.so (see include/hough.h): validation, table construction, stream-ordered
// launches.  No compute happens on the host; there is no CPU fallback.
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <new>
#include <vector>

#include "hough_internal.cuh"

namespace {

thread_local char g_errbuf[256] = "";

int cuda_fail(cudaError_t err, const char* what)
{
    snprintf(g_errbuf, sizeof(g_errbuf), "CUDA error in %s: %s", what, cudaGetErrorString(err));
    return HOUGH_ECUDA;
}

#define CK(call, what)                                            \
    do {                                                          \
        cudaError_t err__ = (call);                               \
        if (err__ != cudaSuccess) return cuda_fail(err__, what);  \
    } while (0)

template <typename T>
cudaError_t dev_alloc(T** p, size_t n)
{
    *p = nullptr;
    if (n == 0) n = 1;
    return cudaMalloc(reinterpret_cast<void**>(p), n * sizeof(T));
}

void free_all(hough_ctx* c)
{
    cudaFree(c->d_c0); cudaFree(c->d_s0); cudaFree(c->d_d0c); cudaFree(c->d_two_d0); cudaFree(c->d_d0sq);
    cudaFree(c->d_rec); cudaFree(c->d_rec_u); cudaFree(c->d_key); cudaFree(c->d_seg); cudaFree(c->d_btab);
    cudaFree(c->d_layer_r); cudaFree(c->d_tilewin); cudaFree(c->d_tilewin_mo); cudaFree(c->d_redo); cudaFree(c->d_vtx_gplane); cudaFree(c->d_vtx_done); cudaFree(c->d_status); cudaFree(c->d_tilectr);
    cudaFree(c->d_bitmap); cudaFree(c->d_grpcnt); cudaFree(c->d_jetkeys);
    cudaFree(c->d_cand); cudaFree(c->d_cand_n); cudaFree(c->d_sortkeys);
    cudaFree(c->d_ce); cudaFree(c->d_se);
    cudaFree(c->d_kc); cudaFree(c->d_vex); cudaFree(c->d_vey); cudaFree(c->d_vrc);
    cudaFree(c->d_hp_vertices); cudaFree(c->d_hp_nvtx); cudaFree(c->d_hp_vflag);
    cudaFree(c->d_hp_count); cudaFree(c->d_hp_mask); cudaFree(c->d_hp_off); cudaFree(c->d_hp_r);
    cudaFree(c->d_hp_phi); cudaFree(c->d_hp_layer); cudaFree(c->d_hp_peaks); cudaFree(c->d_hp_tracks);
    cudaFree(c->d_hp_jets); cudaFree(c->d_hp_npeaks); cudaFree(c->d_hp_njets); cudaFree(c->d_hp_flag);
    for (cudaEvent_t ev : c->ev_pool) cudaEventDestroy(ev);
    c->ev_pool.clear();
}

// hough_profile: a mark on the stream; the interval up to the next mark of the same call is charged to `label`
constexpr size_t kMaxProfMarks = 1u << 18;
void prof_mark(hough_ctx* c, int label, cudaStream_t st)
{
    if (!c->prof_on || c->ev_used >= kMaxProfMarks) return;
    if (c->ev_used == c->ev_pool.size()) {
        cudaEvent_t ev = nullptr;
        if (cudaEventCreate(&ev) != cudaSuccess) { cudaGetLastError(); return; }
        c->ev_pool.push_back(ev);
        c->ev_label.push_back(-1);
    }
    cudaEventRecord(c->ev_pool[c->ev_used], st);
    c->ev_label[c->ev_used] = label;
    ++c->ev_used;
}

bool config_ok(const hough_config* g)
{
    if (g->n_phi0 < 4 || g->n_phi0 > (1u << 20)) return false;
    if (g->n_kappa < 8 || g->n_kappa % 8 != 0 || g->n_kappa > (1u << 20)) return false;
    if (g->n_d0 < 1 || g->n_d0 > (1u << 16)) return false;
    if ((uint64_t)g->n_phi0 * g->n_kappa * g->n_d0 > 0xffffffffull) return false;      // lin is u32
    if (!(g->kappa_max > 0.f) || !isfinite(g->kappa_max)) return false;
    if (g->n_d0 > 1 && !(g->d0_max > g->d0_min && isfinite(g->d0_min) && isfinite(g->d0_max))) return false;
    if (!isfinite(g->b_tesla)) return false;
    if (g->n_layers < 1 || g->n_layers > HOUGH_MAX_LAYERS) return false;
    if (g->max_events < 1 || g->max_events > (1u << 20)) return false;
    if (g->max_hits < 1 || g->max_hits > 0xffffffffull) return false;
    if (g->max_peaks_per_event < 1 || g->max_jets_per_event < 1) return false;
    if (g->host_chunk_events > g->max_events) return false;
    if (g->max_plane_events > g->max_events) return false;
    if (g->max_candidates_per_event > (1u << 24)) return false;
    if (g->vote_flags & ~(uint32_t)(HOUGH_VOTE_HEMI | HOUGH_VOTE_FILL)) return false;
    if (g->debug_flags & ~(uint32_t)(HOUGH_DEBUG_NO_MIRROR | HOUGH_DEBUG_TILES_COUNT | HOUGH_DEBUG_TILES_MASK)) return false;
    if ((g->debug_flags & HOUGH_DEBUG_TILES_COUNT) && (g->debug_flags & HOUGH_DEBUG_TILES_MASK)) return false;
    if (g->n_vtx_phi != 0) {                                   // vertex grid of the second transform
        if (g->n_vtx_phi < 8 || g->n_vtx_phi % 4 != 0 || g->n_vtx_r < 8 || g->n_vtx_r % 8 != 0) return false;
        if ((uint64_t)g->n_vtx_phi * g->n_vtx_r * 2 > 200u * 1024u) return false;
        if ((uint64_t)g->n_vtx_phi * g->n_vtx_r * 2 + (2ull * g->n_vtx_phi + g->n_vtx_r) * 4 +
                (uint64_t)g->n_vtx_phi * g->n_vtx_r / 8 > 220u * 1024u) return false;
        if (!(g->vtx_r_min > 0.f) || !(g->vtx_r_max > g->vtx_r_min) || !isfinite(g->vtx_r_max)) return false;
        if (g->max_vertices_per_event < 1) return false;
        // every stored track votes at most once per R_v bin and the vertex plane counts in 16 bits (two counts per
        // 32-bit word, vertices.cu): more than 65535 tracks could carry from one bin into its neighbour
        if (g->max_peaks_per_event > 65535u) return false;
    }
    return true;
}

// hough_trigger_host: takes sticky status bits back once the condition they report has been repaired
__global__ void status_clear_kernel(uint32_t* status, uint32_t bits) { atomicAnd(status, ~bits); }

}  // namespace

extern "C" {

const char* hough_strerror(int code)
{
    switch (code) {
        case HOUGH_OK: return "ok";
        case HOUGH_EINVAL: return "invalid argument";
        case HOUGH_ECUDA: return g_errbuf[0] ? g_errbuf : "CUDA runtime error";
        case HOUGH_ENOMEM: return "device allocation failed";
        case HOUGH_EUNSUPPORTED: return "configuration not supported by the kernels";
        case HOUGH_ETOOLARGE:
            return "hough_jets_static: n_events * max_peaks_per_event exceeds HOUGH_JETS_STATIC_MAX_TRACKS or n_d0 exceeds "
                   "HOUGH_JETS_STATIC_MAX_D0 (the scratch array is fixed; create a context and use hough_jets instead)";
    }
    return "unknown error code";
}

int hough_create(const hough_config* cfg, hough_ctx** out)
{
    if (!cfg || !out) return HOUGH_EINVAL;
    *out = nullptr;
    if (!config_ok(cfg)) return HOUGH_EINVAL;
    int dev = 0;
    CK(cudaGetDevice(&dev), "cudaGetDevice");
    cudaDeviceProp prop;
    CK(cudaGetDeviceProperties(&prop, dev), "cudaGetDeviceProperties");
    if (prop.major < 10) {
        snprintf(g_errbuf, sizeof(g_errbuf), "device sm_%d%d is not sm_100-class", prop.major, prop.minor);
        return HOUGH_ECUDA;
    }
    hough_ctx* c = new (std::nothrow) hough_ctx();          // value-initialised: every pointer null, every counter 0
    if (!c) return HOUGH_ENOMEM;
    c->cfg = *cfg;
    c->device = dev;
    c->sm_count = prop.multiProcessorCount;

    // O-0 tables: double precision, each value rounded once to fp32
    const uint32_t NP = cfg->n_phi0, ND = cfg->n_d0, NK = cfg->n_kappa;
    std::vector<float> c0(NP), s0(NP), d0c(ND), two_d0(ND), d0sq(ND);
    const double pi = 3.14159265358979323846;
    for (uint32_t ip = 0; ip < NP; ++ip) {
        const double ph = ((double)ip + 0.5) * (2.0 * pi / (double)NP);
        c0[ip] = (float)cos(ph);
        s0[ip] = (float)sin(ph);
    }
    for (uint32_t id = 0; id < ND; ++id) {
        float d = 0.f;
        if (ND > 1)
            d = (float)((double)cfg->d0_min + ((double)id + 0.5) * (((double)cfg->d0_max - (double)cfg->d0_min) / (double)ND));
        volatile float dd = d * d;                    // one fp32 multiply, kept out of any contraction
        d0c[id] = d; two_d0[id] = 2.0f * d; d0sq[id] = dd;
    }
    // O-6 tables: kappa bin centres, phi_v edge directions, R_v bin centres (double, rounded once)
    std::vector<float> kc(NK), vex, vey, vrc;
    for (uint32_t ik = 0; ik < NK; ++ik)
        kc[ik] = (float)(-(double)cfg->kappa_max + ((double)ik + 0.5) * (2.0 * (double)cfg->kappa_max / (double)NK));
    if (cfg->n_vtx_phi) {
        vex.resize(cfg->n_vtx_phi); vey.resize(cfg->n_vtx_phi); vrc.resize(cfg->n_vtx_r);
        for (uint32_t k = 0; k < cfg->n_vtx_phi; ++k) {
            const double a = (double)k * (2.0 * pi / (double)cfg->n_vtx_phi);
            vex[k] = (float)cos(a); vey[k] = (float)sin(a);
        }
        for (uint32_t ir = 0; ir < cfg->n_vtx_r; ++ir)
            vrc[ir] = (float)((double)cfg->vtx_r_min +
                              ((double)ir + 0.5) * (((double)cfg->vtx_r_max - (double)cfg->vtx_r_min) / (double)cfg->n_vtx_r));
    }
    // mirror tiles need tables that are antisymmetric bit for bit: c0[ip + N/2] == -c0[ip], s0 likewise, d0c[ND-1-id] == -d0c[id]
    std::vector<float> ce(NP), se(NP);                         // column edges (voting variant FILL)
    for (uint32_t j = 0; j < NP; ++j) {
        const double a = (double)j * (2.0 * pi / (double)NP);
        ce[j] = (float)cos(a); se[j] = (float)sin(a);
    }
    bool mirror_ok = NP % 2 == 0 && !(cfg->debug_flags & HOUGH_DEBUG_NO_MIRROR) && cfg->vote_flags == 0;
    for (uint32_t ip = 0; mirror_ok && ip < NP / 2; ++ip)
        mirror_ok = c0[ip + NP / 2] == -c0[ip] && s0[ip + NP / 2] == -s0[ip];
    for (uint32_t id = 0; mirror_ok && id < ND; ++id) mirror_ok = d0c[ND - 1 - id] == -d0c[id];
    if (plan_vote(c, mirror_ok) != cudaSuccess || plan_peaks(c) != cudaSuccess) { delete c; return HOUGH_EUNSUPPORTED; }
    // fused path: which tiles hough_vote_peaks uses on a grid that has both kinds: cfg.debug_flags can force
    // count + mask tiles (1) or mask-only tiles (2); otherwise (0) chosen per call by occupancy
    c->fused_scheme = (cfg->debug_flags & HOUGH_DEBUG_TILES_COUNT) ? 1 : (cfg->debug_flags & HOUGH_DEBUG_TILES_MASK) ? 2 : 0;
    c->prep_hits_per_event = 0.0;
    // the branch-free exact division of the vote kernel is only used inside this range (vote.cu, div_rn_tame)
    c->tame_tables = cfg->kappa_max >= 9.094947e-13f && cfg->kappa_max <= 1.0995116e12f;      // [2^-40, 2^40]
    for (uint32_t id = 0; id < ND; ++id) {
        const float a = fabsf(d0c[id]);
        if (!(a == 0.f || (a >= 9.5367431640625e-07f && a <= 1048576.f))) c->tame_tables = false;
    }
    c->kmax = cfg->kappa_max;
    c->inv_dk = (float)((double)NK / (2.0 * (double)cfg->kappa_max));
    c->nk_f = (float)NK;

    const size_t bins = (size_t)ND * NP * NK;
    cudaError_t err = cudaSuccess;
    auto A = [&](cudaError_t e2) { if (err == cudaSuccess) err = e2; };
    A(dev_alloc(&c->d_c0, NP)); A(dev_alloc(&c->d_s0, NP));
    A(dev_alloc(&c->d_d0c, ND)); A(dev_alloc(&c->d_two_d0, ND)); A(dev_alloc(&c->d_d0sq, ND));
    A(dev_alloc(&c->d_kc, NK));
    A(dev_alloc(&c->d_ce, NP)); A(dev_alloc(&c->d_se, NP));
    A(dev_alloc(&c->d_vex, cfg->n_vtx_phi)); A(dev_alloc(&c->d_vey, cfg->n_vtx_phi)); A(dev_alloc(&c->d_vrc, cfg->n_vtx_r));
    if (cfg->n_vtx_phi) {
        A(dev_alloc(&c->d_vtx_gplane, (size_t)kVtxSplitEvents * cfg->n_vtx_phi * cfg->n_vtx_r / 2));
        A(dev_alloc(&c->d_vtx_done, kVtxSplitEvents));
    }
    A(dev_alloc(&c->d_rec, cfg->max_hits)); A(dev_alloc(&c->d_rec_u, cfg->max_hits)); A(dev_alloc(&c->d_key, cfg->max_hits));
    A(dev_alloc(&c->d_seg, (size_t)cfg->max_events * kSegStride));
    A(dev_alloc(&c->d_btab, (size_t)cfg->max_events * HOUGH_MAX_LAYERS * (c->vote.nb + 1)));
    A(dev_alloc(&c->d_layer_r, 4 * HOUGH_MAX_LAYERS));   // live min / max per layer + the copy the recount reads
    A(dev_alloc(&c->d_tilewin, (size_t)c->vote.nk_seg * HOUGH_MAX_LAYERS * c->vote.n_strips));
    if (c->has_mo) A(dev_alloc(&c->d_tilewin_mo, (size_t)c->vote_mo.nk_seg * HOUGH_MAX_LAYERS * c->vote_mo.n_strips));
    A(dev_alloc(&c->d_status, 2));
    A(dev_alloc(&c->d_tilectr, 2));
    // peak-finder scratch of the accumulator path: sized for the events ONE hough_peaks call may bring
    c->plane_events = cfg->max_plane_events ? cfg->max_plane_events : cfg->max_events;
    A(dev_alloc(&c->d_bitmap, (size_t)c->plane_events * (bins / 8)));
    A(dev_alloc(&c->d_grpcnt, (size_t)c->plane_events * ((bins + 255) / 256)));
    A(dev_alloc(&c->d_jetkeys, (size_t)cfg->max_events * cfg->max_peaks_per_event));
    // fused vote -> peaks: candidate buffers for the events of one fused launch
    c->fused_events = cfg->host_chunk_events ? cfg->host_chunk_events : cfg->max_events;
    {
        uint64_t cap = cfg->max_candidates_per_event;
        if (cap == 0) { cap = 4ull * cfg->max_peaks_per_event; if (cap < 4096) cap = 4096; if (cap > (1u << 24)) cap = 1u << 24; }
        c->cand_cap = (uint32_t)cap;
        c->cand_cap_pow2 = 1;
        while (c->cand_cap_pow2 < c->cand_cap) c->cand_cap_pow2 <<= 1;
    }
    A(dev_alloc(&c->d_cand, (size_t)c->fused_events * c->cand_cap));
    A(dev_alloc(&c->d_cand_n, c->fused_events));
    A(dev_alloc(&c->d_redo, (size_t)c->fused_events + 1));
    A(dev_alloc(&c->d_sortkeys, (size_t)c->fused_events * c->cand_cap_pow2));
    if (cfg->host_chunk_events > 0) {
        const size_t E = cfg->max_events, H = cfg->max_hits;
        A(dev_alloc(&c->d_hp_count, bins));                    // one event: the fallback of hough_trigger_host
        A(dev_alloc(&c->d_hp_mask, bins));
        A(dev_alloc(&c->d_hp_off, E + 1)); A(dev_alloc(&c->d_hp_r, H)); A(dev_alloc(&c->d_hp_phi, H));
        A(dev_alloc(&c->d_hp_layer, H));
        A(dev_alloc(&c->d_hp_peaks, E * cfg->max_peaks_per_event));
        A(dev_alloc(&c->d_hp_tracks, E * cfg->max_peaks_per_event));
        A(dev_alloc(&c->d_hp_jets, E * cfg->max_jets_per_event));
        A(dev_alloc(&c->d_hp_npeaks, E)); A(dev_alloc(&c->d_hp_njets, E)); A(dev_alloc(&c->d_hp_flag, E));
        if (cfg->n_vtx_phi) {
            A(dev_alloc(&c->d_hp_vertices, E * cfg->max_vertices_per_event));
            A(dev_alloc(&c->d_hp_nvtx, E)); A(dev_alloc(&c->d_hp_vflag, E));
        }
    }
    if (err != cudaSuccess) {
        cuda_fail(err, "hough_create allocation");
        free_all(c); delete c;
        cudaGetLastError();
        return (err == cudaErrorMemoryAllocation) ? HOUGH_ENOMEM : HOUGH_ECUDA;
    }
    uint32_t lr[4 * HOUGH_MAX_LAYERS];
    for (int i = 0; i < HOUGH_MAX_LAYERS; ++i) {
        lr[i] = lr[2 * HOUGH_MAX_LAYERS + i] = 0x7f800000u;
        lr[HOUGH_MAX_LAYERS + i] = lr[3 * HOUGH_MAX_LAYERS + i] = 0u;
    }
    A(cudaMemcpy(c->d_c0, c0.data(), NP * 4, cudaMemcpyHostToDevice));
    A(cudaMemcpy(c->d_s0, s0.data(), NP * 4, cudaMemcpyHostToDevice));
    A(cudaMemcpy(c->d_d0c, d0c.data(), ND * 4, cudaMemcpyHostToDevice));
    A(cudaMemcpy(c->d_two_d0, two_d0.data(), ND * 4, cudaMemcpyHostToDevice));
    A(cudaMemcpy(c->d_d0sq, d0sq.data(), ND * 4, cudaMemcpyHostToDevice));
    A(cudaMemcpy(c->d_layer_r, lr, sizeof(lr), cudaMemcpyHostToDevice));
    A(cudaMemcpy(c->d_kc, kc.data(), NK * 4, cudaMemcpyHostToDevice));
    A(cudaMemcpy(c->d_ce, ce.data(), NP * 4, cudaMemcpyHostToDevice));
    A(cudaMemcpy(c->d_se, se.data(), NP * 4, cudaMemcpyHostToDevice));
    if (cfg->n_vtx_phi) {
        A(cudaMemcpy(c->d_vex, vex.data(), vex.size() * 4, cudaMemcpyHostToDevice));
        A(cudaMemcpy(c->d_vey, vey.data(), vey.size() * 4, cudaMemcpyHostToDevice));
        A(cudaMemcpy(c->d_vrc, vrc.data(), vrc.size() * 4, cudaMemcpyHostToDevice));
    }
    A(cudaMemset(c->d_status, 0, 8));
    A(cudaMemset(c->d_tilectr, 0, 8));
    if (cfg->n_vtx_phi) {
        A(cudaMemset(c->d_vtx_gplane, 0, (size_t)kVtxSplitEvents * cfg->n_vtx_phi * cfg->n_vtx_r * 2));
        A(cudaMemset(c->d_vtx_done, 0, kVtxSplitEvents * 4));
    }
    // all-empty windows until the first call with hits computes them (build_windows_kernel skips unchanged r ranges)
    A(cudaMemset(c->d_tilewin, 0, (size_t)c->vote.nk_seg * HOUGH_MAX_LAYERS * c->vote.n_strips * sizeof(TileWin)));
    if (c->has_mo)
        A(cudaMemset(c->d_tilewin_mo, 0, (size_t)c->vote_mo.nk_seg * HOUGH_MAX_LAYERS * c->vote_mo.n_strips * sizeof(TileWin)));
    A(cudaMemset(c->d_cand_n, 0, (size_t)c->fused_events * 4));
    if (err != cudaSuccess) { cuda_fail(err, "hough_create upload"); free_all(c); delete c; return HOUGH_ECUDA; }
    *out = c;
    return HOUGH_OK;
}

int hough_destroy(hough_ctx* ctx)
{
    if (!ctx) return HOUGH_EINVAL;
    cudaDeviceSynchronize();
    free_all(ctx);
    delete ctx;
    return HOUGH_OK;
}

size_t hough_plane_bytes(const hough_ctx* ctx, uint32_t n_events)
{
    if (!ctx) return 0;
    return (size_t)n_events * ctx->cfg.n_d0 * ctx->cfg.n_phi0 * ctx->cfg.n_kappa * 2;
}

int hough_vote(hough_ctx* ctx, uint32_t n_events, const uint32_t* d_hit_offsets, uint64_t n_hits_total,
               const float* d_r, const float* d_phi, const uint8_t* d_layer, uint16_t* d_count, uint16_t* d_mask,
               void* stream)
{
    if (!ctx || !d_hit_offsets || !d_count || !d_mask) return HOUGH_EINVAL;
    if (n_hits_total > 0 && (!d_r || !d_phi || !d_layer)) return HOUGH_EINVAL;
    if (n_events > ctx->cfg.max_events || n_hits_total > ctx->cfg.max_hits) return HOUGH_EINVAL;
    if (((uintptr_t)d_count | (uintptr_t)d_mask) & 15u) return HOUGH_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    ctx->last_stream = st;
    if (n_events == 0) return HOUGH_OK;
    prof_mark(ctx, 0, st);
    CK(launch_prep(ctx, n_events, d_hit_offsets, n_hits_total, d_r, d_phi, d_layer, st), "hit preparation");
    prof_mark(ctx, 1, st);
    CK(launch_vote(ctx, 0, n_events, d_count, d_mask, st), "vote kernel");
    prof_mark(ctx, -1, st);
    return HOUGH_OK;
}

int hough_peaks(hough_ctx* ctx, uint32_t n_events, const uint16_t* d_count, const uint16_t* d_mask, uint32_t l_min,
                hough_peak* d_peaks, uint32_t* d_n_peaks, void* stream)
{
    if (!ctx || !d_count || !d_mask || !d_peaks || !d_n_peaks) return HOUGH_EINVAL;
    if (n_events > ctx->plane_events || l_min < 1 || l_min > ctx->cfg.n_layers) return HOUGH_EINVAL;
    if (((uintptr_t)d_count | (uintptr_t)d_mask) & 15u) return HOUGH_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    ctx->last_stream = st;
    prof_mark(ctx, 2, st);
    CK(launch_peaks(ctx, n_events, d_count, d_mask, l_min, d_peaks, d_n_peaks, st), "peak kernels");
    prof_mark(ctx, -1, st);
    return HOUGH_OK;
}

int hough_vote_peaks(hough_ctx* ctx, uint32_t n_events, const uint32_t* d_hit_offsets, uint64_t n_hits_total,
                     const float* d_r, const float* d_phi, const uint8_t* d_layer, uint32_t l_min, hough_peak* d_peaks,
                     uint32_t* d_n_peaks, void* stream)
{
    if (!ctx || !d_hit_offsets || !d_peaks || !d_n_peaks) return HOUGH_EINVAL;
    if (n_hits_total > 0 && (!d_r || !d_phi || !d_layer)) return HOUGH_EINVAL;
    if (n_events > ctx->cfg.max_events || n_events > ctx->fused_events || n_hits_total > ctx->cfg.max_hits) return HOUGH_EINVAL;
    if (l_min < 1 || l_min > ctx->cfg.n_layers) return HOUGH_EINVAL;
    if (ctx->cfg.vote_flags != 0) return HOUGH_EUNSUPPORTED;      // voting variants: accumulator path only
    cudaStream_t st = (cudaStream_t)stream;
    ctx->last_stream = st;
    if (n_events == 0) return HOUGH_OK;
    prof_mark(ctx, 0, st);
    CK(launch_prep(ctx, n_events, d_hit_offsets, n_hits_total, d_r, d_phi, d_layer, st), "hit preparation");
    prof_mark(ctx, 1, st);
    CK(launch_vote_fused(ctx, 0, n_events, l_min, st), "fused vote kernel");
    prof_mark(ctx, 2, st);
    CK(launch_recount(ctx, 0, n_events, st), "recount kernel");
    CK(launch_peaks_finalize(ctx, n_events, d_peaks, d_n_peaks, st), "peak ordering kernel");
    prof_mark(ctx, -1, st);
    return HOUGH_OK;
}

static int cone_bins_of(float cone_rad, uint32_t n_phi0)
{
    const double pi = 3.14159265358979323846;
    double b = floor((double)cone_rad * (double)n_phi0 / (2.0 * pi));
    if (b > (double)n_phi0) b = (double)n_phi0;
    return (int)b;
}

int hough_jets(hough_ctx* ctx, uint32_t n_events, const hough_peak* d_peaks, const uint32_t* d_n_peaks, float cone_rad,
               float d0_cut_mm, uint32_t n_displaced_min, hough_track* d_tracks, hough_jet* d_jets,
               uint32_t* d_n_jets, uint8_t* d_flag, void* stream)
{
    if (!ctx || !d_peaks || !d_n_peaks || !d_tracks || !d_jets || !d_n_jets || !d_flag) return HOUGH_EINVAL;
    if (n_events > ctx->cfg.max_events || !(cone_rad >= 0.f) || !isfinite(cone_rad) || isnan(d0_cut_mm)) return HOUGH_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    ctx->last_stream = st;
    prof_mark(ctx, 3, st);
    CK(launch_jets(ctx, n_events, d_peaks, d_n_peaks, cone_bins_of(cone_rad, ctx->cfg.n_phi0), d0_cut_mm,
                   n_displaced_min, d_tracks, d_jets, d_n_jets, d_flag, st), "jet kernel");
    prof_mark(ctx, -1, st);
    return HOUGH_OK;
}

// hough_jets for callers that may not allocate (no context, no cudaMalloc): see include/hough.h and jets.cu.
int hough_jets_static(const hough_config* cfg, uint32_t n_events, const hough_peak* d_peaks, const uint32_t* d_n_peaks,
                      float cone_rad, float d0_cut_mm, uint32_t n_displaced_min, hough_track* d_tracks, hough_jet* d_jets,
                      uint32_t* d_n_jets, uint8_t* d_flag, void* stream)
{
    if (!cfg || !d_peaks || !d_n_peaks || !d_tracks || !d_jets || !d_n_jets || !d_flag) return HOUGH_EINVAL;
    // the fields the jet kernel reads, with hough_create's conditions on them
    if (cfg->n_phi0 < 4 || cfg->n_phi0 > (1u << 20)) return HOUGH_EINVAL;
    if (cfg->n_kappa < 8 || cfg->n_kappa % 8 != 0 || cfg->n_kappa > (1u << 20)) return HOUGH_EINVAL;
    if (cfg->n_d0 < 1 || cfg->n_d0 > (1u << 16)) return HOUGH_EINVAL;
    if ((uint64_t)cfg->n_phi0 * cfg->n_kappa * cfg->n_d0 > 0xffffffffull) return HOUGH_EINVAL;
    if (!(cfg->kappa_max > 0.f) || !isfinite(cfg->kappa_max) || !isfinite(cfg->b_tesla)) return HOUGH_EINVAL;
    if (cfg->n_d0 > 1 && !(cfg->d0_max > cfg->d0_min && isfinite(cfg->d0_min) && isfinite(cfg->d0_max))) return HOUGH_EINVAL;
    if (cfg->max_peaks_per_event < 1 || cfg->max_jets_per_event < 1) return HOUGH_EINVAL;
    if (!(cone_rad >= 0.f) || !isfinite(cone_rad) || isnan(d0_cut_mm)) return HOUGH_EINVAL;
    // the scratch is a fixed array: refuse what does not fit instead of writing past it
    if (cfg->n_d0 > HOUGH_JETS_STATIC_MAX_D0) return HOUGH_ETOOLARGE;
    if ((uint64_t)n_events * cfg->max_peaks_per_event > (uint64_t)HOUGH_JETS_STATIC_MAX_TRACKS) return HOUGH_ETOOLARGE;
    CK(launch_jets_static(cfg, n_events, d_peaks, d_n_peaks, cone_bins_of(cone_rad, cfg->n_phi0), d0_cut_mm,
                          n_displaced_min, d_tracks, d_jets, d_n_jets, d_flag, (cudaStream_t)stream),
       "hough_jets_static (scratch address look-up or kernel launch)");
    return HOUGH_OK;
}

int hough_vertices(hough_ctx* ctx, uint32_t n_events, const hough_peak* d_peaks, const uint32_t* d_n_peaks, float d0_cut_mm,
                   uint32_t n_min, hough_vertex* d_vertices, uint32_t* d_n_vertices, uint8_t* d_flag,
                   uint16_t* d_vertex_plane, void* stream)
{
    if (!ctx || !d_peaks || !d_n_peaks || !d_vertices || !d_n_vertices || !d_flag) return HOUGH_EINVAL;
    if (ctx->cfg.n_vtx_phi == 0 || n_events > ctx->cfg.max_events || n_min < 1 || n_min > HOUGH_VTX_N_MIN_MAX || isnan(d0_cut_mm))
        return HOUGH_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    ctx->last_stream = st;
    prof_mark(ctx, 4, st);
    CK(launch_vertices(ctx, n_events, d_peaks, d_n_peaks, d0_cut_mm, n_min, d_vertices, d_n_vertices, d_flag,
                       d_vertex_plane, st), "vertex kernel");
    prof_mark(ctx, -1, st);
    return HOUGH_OK;
}

int hough_trigger_host_vtx(hough_ctx* ctx, uint32_t n_events, const uint32_t* h_hit_offsets, uint64_t n_hits_total,
                           const float* h_r, const float* h_phi, const uint8_t* h_layer, uint32_t l_min, float cone_rad,
                           float d0_cut_mm, uint32_t n_displaced_min, uint32_t vtx_n_min, uint32_t* h_n_peaks,
                           uint32_t* h_n_jets, uint8_t* h_flag, hough_peak* h_peaks, hough_jet* h_jets,
                           uint32_t* h_n_vertices, uint8_t* h_vtx_flag, hough_vertex* h_vertices, float* ms_stage,
                           void* stream)
{
    if (!ctx || !h_hit_offsets || !h_n_peaks || !h_n_jets || !h_flag) return HOUGH_EINVAL;
    if (ctx->cfg.host_chunk_events == 0) return HOUGH_EINVAL;
    if (ctx->cfg.vote_flags != 0) return HOUGH_EUNSUPPORTED;      // voting variants: accumulator path only
    if (n_hits_total > 0 && (!h_r || !h_phi || !h_layer)) return HOUGH_EINVAL;
    if (n_events > ctx->cfg.max_events || n_hits_total > ctx->cfg.max_hits) return HOUGH_EINVAL;
    if (l_min < 1 || l_min > ctx->cfg.n_layers || !(cone_rad >= 0.f) || !isfinite(cone_rad) || isnan(d0_cut_mm))
        return HOUGH_EINVAL;
    const bool vtx = vtx_n_min != 0;                            // 0: the second transform is not run
    if (vtx && (ctx->cfg.n_vtx_phi == 0 || vtx_n_min > HOUGH_VTX_N_MIN_MAX || !h_n_vertices || !h_vtx_flag)) return HOUGH_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    ctx->last_stream = st;
    const int n_stage = vtx ? 4 : 3;
    if (ms_stage) for (int i = 0; i < n_stage; ++i) ms_stage[i] = 0.f;
    if (n_events == 0) return HOUGH_OK;
    const hough_config& g = ctx->cfg;
    CK(cudaMemcpyAsync(ctx->d_hp_off, h_hit_offsets, ((size_t)n_events + 1) * 4, cudaMemcpyHostToDevice, st), "H2D offsets");
    if (n_hits_total) {
        CK(cudaMemcpyAsync(ctx->d_hp_r, h_r, n_hits_total * 4, cudaMemcpyHostToDevice, st), "H2D r");
        CK(cudaMemcpyAsync(ctx->d_hp_phi, h_phi, n_hits_total * 4, cudaMemcpyHostToDevice, st), "H2D phi");
        CK(cudaMemcpyAsync(ctx->d_hp_layer, h_layer, n_hits_total, cudaMemcpyHostToDevice, st), "H2D layer");
    }
    // ms_stage: the context's stage profile (hough_profile) is switched on for this call and read at its end
    // (documented in hough.h: a call with ms_stage starts from an empty profile, so intervals the caller had
    // accumulated with hough_profile and not yet read are dropped -- as are marks left behind by a profile that was
    // switched off without a read).  The guard puts the caller's setting back on EVERY way out, error returns included.
    struct ProfRestore {
        hough_ctx* c; bool was_on; bool armed;
        ~ProfRestore() { if (armed) c->prof_on = was_on; }
    } prof_restore{ctx, ctx->prof_on, ms_stage != nullptr};
    if (ms_stage) {
        float drop[5]; uint32_t nc = 0;
        hough_profile_read(ctx, drop, &nc);                      // empties the mark list whatever state it was in
        ctx->prof_on = true;
    }
    auto peaks_of = [&](uint32_t e) { return ctx->d_hp_peaks + (size_t)e * g.max_peaks_per_event; };
    auto tail = [&](uint32_t e0, uint32_t ne, int cone_bins) -> cudaError_t {   // jets (+ vertices) of events [e0, e0 + ne)
        prof_mark(ctx, 3, st);
        cudaError_t err = launch_jets(ctx, ne, peaks_of(e0), ctx->d_hp_npeaks + e0, cone_bins, d0_cut_mm, n_displaced_min,
                                      ctx->d_hp_tracks + (size_t)e0 * g.max_peaks_per_event,
                                      ctx->d_hp_jets + (size_t)e0 * g.max_jets_per_event, ctx->d_hp_njets + e0,
                                      ctx->d_hp_flag + e0, st);
        if (err != cudaSuccess || !vtx) return err;
        prof_mark(ctx, 4, st);
        return launch_vertices(ctx, ne, peaks_of(e0), ctx->d_hp_npeaks + e0, d0_cut_mm, vtx_n_min,
                               ctx->d_hp_vertices + (size_t)e0 * g.max_vertices_per_event, ctx->d_hp_nvtx + e0,
                               ctx->d_hp_vflag + e0, nullptr, st);
    };
    // hits are prepared once for the whole batch; the chunks then share the prepared records
    prof_mark(ctx, 0, st);
    CK(launch_prep(ctx, n_events, ctx->d_hp_off, n_hits_total, ctx->d_hp_r, ctx->d_hp_phi, ctx->d_hp_layer, st), "hit preparation");
    const int cone_bins = cone_bins_of(cone_rad, g.n_phi0);
    for (uint32_t e0 = 0; e0 < n_events; e0 += g.host_chunk_events) {
        const uint32_t ne = (n_events - e0 < g.host_chunk_events) ? n_events - e0 : g.host_chunk_events;
        prof_mark(ctx, 1, st);
        CK(launch_vote_fused(ctx, e0, ne, l_min, st), "fused vote kernel");
        prof_mark(ctx, 2, st);
        CK(launch_recount(ctx, e0, ne, st), "recount kernel");
        CK(launch_peaks_finalize(ctx, ne, peaks_of(e0), ctx->d_hp_npeaks + e0, st), "peak ordering kernel");
        CK(tail(e0, ne, cone_bins), "jet / vertex kernels");
    }
    prof_mark(ctx, -1, st);
    CK(cudaMemcpyAsync(h_n_peaks, ctx->d_hp_npeaks, (size_t)n_events * 4, cudaMemcpyDeviceToHost, st), "D2H n_peaks");
    CK(cudaStreamSynchronize(st), "hough_trigger_host synchronize");
    // events whose candidates did not fit the buffer: the accumulator path, one event at a time, on the context's
    // one-event planes (the prepared hits of the whole batch are still in the workspace)
    uint32_t n_repaired = 0;
    for (uint32_t e = 0; e < n_events; ++e) {
        if (h_n_peaks[e] != HOUGH_N_PEAKS_OVERFLOW) continue;
        prof_mark(ctx, 1, st);                                   // the fallback's time belongs to ms_stage as well
        CK(launch_vote(ctx, e, 1, ctx->d_hp_count, ctx->d_hp_mask, st), "vote kernel (fallback)");
        prof_mark(ctx, 2, st);
        CK(launch_peaks(ctx, 1, ctx->d_hp_count, ctx->d_hp_mask, l_min, peaks_of(e), ctx->d_hp_npeaks + e, st),
           "peak kernels (fallback)");
        CK(tail(e, 1, cone_bins), "jet / vertex kernels (fallback)");
        prof_mark(ctx, -1, st);
        CK(cudaMemcpyAsync(h_n_peaks + e, ctx->d_hp_npeaks + e, 4, cudaMemcpyDeviceToHost, st), "D2H n_peaks (fallback)");
        ++n_repaired;
    }
    if (n_repaired) {
        // every overflowed event now holds the accumulator path's (exact) result: the overflow bit this call raised
        // would report an error that no longer exists
        status_clear_kernel<<<1, 1, 0, st>>>(ctx->d_status, (uint32_t)HOUGH_ST_CANDIDATE_OVERFLOW);
        ++ctx->launches;
        CK(cudaGetLastError(), "status kernel");
    }
    CK(cudaMemcpyAsync(h_n_jets, ctx->d_hp_njets, (size_t)n_events * 4, cudaMemcpyDeviceToHost, st), "D2H n_jets");
    CK(cudaMemcpyAsync(h_flag, ctx->d_hp_flag, (size_t)n_events, cudaMemcpyDeviceToHost, st), "D2H flag");
    if (h_peaks)
        CK(cudaMemcpyAsync(h_peaks, ctx->d_hp_peaks, (size_t)n_events * g.max_peaks_per_event * sizeof(hough_peak),
                           cudaMemcpyDeviceToHost, st), "D2H peaks");
    if (h_jets)
        CK(cudaMemcpyAsync(h_jets, ctx->d_hp_jets, (size_t)n_events * g.max_jets_per_event * sizeof(hough_jet),
                           cudaMemcpyDeviceToHost, st), "D2H jets");
    if (vtx) {
        CK(cudaMemcpyAsync(h_n_vertices, ctx->d_hp_nvtx, (size_t)n_events * 4, cudaMemcpyDeviceToHost, st), "D2H n_vertices");
        CK(cudaMemcpyAsync(h_vtx_flag, ctx->d_hp_vflag, (size_t)n_events, cudaMemcpyDeviceToHost, st), "D2H vertex flag");
        if (h_vertices)
            CK(cudaMemcpyAsync(h_vertices, ctx->d_hp_vertices, (size_t)n_events * g.max_vertices_per_event * sizeof(hough_vertex),
                               cudaMemcpyDeviceToHost, st), "D2H vertices");
    }
    CK(cudaStreamSynchronize(st), "hough_trigger_host synchronize");
    if (ms_stage) {
        float ms[5]; uint32_t nc = 0;
        hough_profile_read(ctx, ms, &nc);
        ms_stage[0] = ms[0] + ms[1]; ms_stage[1] = ms[2]; ms_stage[2] = ms[3];
        if (vtx) ms_stage[3] = ms[4];
    }
    return HOUGH_OK;
}

int hough_trigger_host(hough_ctx* ctx, uint32_t n_events, const uint32_t* h_hit_offsets, uint64_t n_hits_total,
                       const float* h_r, const float* h_phi, const uint8_t* h_layer, uint32_t l_min, float cone_rad,
                       float d0_cut_mm, uint32_t n_displaced_min, uint32_t* h_n_peaks, uint32_t* h_n_jets,
                       uint8_t* h_flag, hough_peak* h_peaks, hough_jet* h_jets, float* ms_stage, void* stream)
{
    return hough_trigger_host_vtx(ctx, n_events, h_hit_offsets, n_hits_total, h_r, h_phi, h_layer, l_min, cone_rad,
                                  d0_cut_mm, n_displaced_min, 0u, h_n_peaks, h_n_jets, h_flag, h_peaks, h_jets, nullptr,
                                  nullptr, nullptr, ms_stage, stream);
}

int hough_status(hough_ctx* ctx, uint32_t* host_status_bits)
{
    if (!ctx || !host_status_bits) return HOUGH_EINVAL;
    CK(cudaStreamSynchronize(ctx->last_stream), "hough_status synchronize");
    uint32_t st[2] = {0, 0};
    CK(cudaMemcpy(st, ctx->d_status, 8, cudaMemcpyDeviceToHost), "hough_status copy");
    ctx->status_host |= st[0];
    *host_status_bits = ctx->status_host;
    return HOUGH_OK;
}

int hough_debug_prepared_hits(hough_ctx* ctx, uint64_t n_hits, float* h_rec, uint32_t* h_trig_risk)
{
    if (!ctx || (n_hits > 0 && !h_rec) || n_hits > ctx->cfg.max_hits) return HOUGH_EINVAL;
    CK(cudaStreamSynchronize(ctx->last_stream), "hough_debug_prepared_hits synchronize");
    if (n_hits) CK(cudaMemcpy(h_rec, ctx->d_rec_u, n_hits * sizeof(float4), cudaMemcpyDeviceToHost), "prepared-hit copy");
    if (h_trig_risk) {
        uint32_t st[2] = {0, 0};
        CK(cudaMemcpy(st, ctx->d_status, 8, cudaMemcpyDeviceToHost), "status copy");
        *h_trig_risk = st[1];
    }
    return HOUGH_OK;
}

int hough_debug_div_check(uint64_t n_pairs, uint64_t seed, float kappa_max, uint32_t n_kappa, uint64_t* h_out)
{
    if (!h_out || !(kappa_max > 0.f) || n_kappa < 8 || n_kappa > (1u << 20)) return HOUGH_EINVAL;
    unsigned long long out[3] = {0, 0, 0};
    CK(run_div_check(n_pairs, seed, kappa_max, (int)n_kappa, out), "division check kernel");
    for (int i = 0; i < 3; ++i) h_out[i] = out[i];
    return HOUGH_OK;
}

int hough_profile(hough_ctx* ctx, int enable)
{
    if (!ctx) return HOUGH_EINVAL;
    ctx->prof_on = enable != 0;
    return HOUGH_OK;
}

int hough_profile_read(hough_ctx* ctx, float* h_ms, uint32_t* h_calls)
{
    if (!ctx || !h_ms) return HOUGH_EINVAL;
    for (int i = 0; i < 5; ++i) h_ms[i] = 0.f;
    uint32_t calls = 0;
    if (ctx->ev_used) CK(cudaEventSynchronize(ctx->ev_pool[ctx->ev_used - 1]), "hough_profile_read synchronize");
    for (size_t i = 0; i + 1 < ctx->ev_used; ++i) {
        const int label = ctx->ev_label[i];
        if (label < 0) { ++calls; continue; }                  // end of a call: the gap to the next call is nobody's
        float ms = 0.f;
        if (cudaEventElapsedTime(&ms, ctx->ev_pool[i], ctx->ev_pool[i + 1]) == cudaSuccess) h_ms[label > 4 ? 4 : label] += ms;
    }
    if (ctx->ev_used) ++calls;
    ctx->ev_used = 0;
    if (h_calls) *h_calls = calls;
    return HOUGH_OK;
}

int hough_last_tile_kind(const hough_ctx* ctx, int* host_kind)
{
    if (!ctx || !host_kind) return HOUGH_EINVAL;
    *host_kind = ctx->last_tile_kind;
    return HOUGH_OK;
}

int hough_launch_count(const hough_ctx* ctx, uint64_t* host_count)
{
    if (!ctx || !host_count) return HOUGH_EINVAL;
    *host_count = ctx->launches;
    return HOUGH_OK;
}

}  // extern "C"
