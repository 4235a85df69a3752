// The paper's second Hough transform: tracks -> displaced vertices (sm_100a).
//
// PAPER.md:117 (section 6): "the corresponding parameter space representation of these tracks is processed by a
// second application of the Hough transform ... to identify not straight lines but sinusoids which contain a
// significant number of tracks, indicating that this is a location of a displaced jet or black hole ... the same
// peak finding algorithm is applied to the parameter space of this second Hough transform"; the jet of
// tracks from the interaction point is excluded "by setting a lower bound on the radius"; the cost is
// proportional to the number of tracks.  Normative arithmetic: DESIGN.md O-6 / O-7 (readings R34-R39).
//
// One block per event; the whole vertex accumulator (phi_v x R_v bins, 16-bit counts, two per 32-bit word) lives in
// shared memory, so nothing but the peak list of the first transform is read and nothing but the vertex list written.
// (Calls with at most kVtxSplitEvents events -- single-event latency -- run kVtxSplit blocks per event instead, which
// vote into the event's plane in global memory; the last block to finish takes it into shared memory for O-7.)
//   O-6  a warp takes a track (bin-centre parameters d0c, (cos, sin) phi0c, kappa_c of its peak), its lanes the R_v
//        bins: s = (kappa (r^2 + d0^2) - 2 d0) / (2 r (1 - kappa d0)) with IEEE division, the crossing direction by
//        rotating (cos phi0, sin phi0) by (sqrt(1 - s^2), s) with IEEE sqrt, the phi_v bin by a cross-product binary
//        search over the bin-edge directions of the quadrant: no transcendental per vote, every step one IEEE fp32
//        operation, so the bins are the oracle's.  One shared-memory atomic per vote.
//   O-7  rule O-3 on the (phi_v, R_v) grid with a count threshold (phi_v periodic, R_v clipped, ties to the lower
//        linear index): a ballot per chunk of 32 bins, then a block scan of the popcounts for the ordered
//        compaction; true total, capacity cut.
#include "hough_internal.cuh"

namespace {

constexpr int kVtxThreads = 1024;

struct VtxParams {
    const hough_peak* peaks; const uint32_t* n_peaks;
    hough_vertex* vertices; uint32_t* n_vertices; uint8_t* flag; uint16_t* plane;
    const float* d0c; const float* c0; const float* s0; const float* kc;      // first transform's bin centres
    const float* ex; const float* ey; const float* rc;                       // vertex grid: edge directions, R_v centres
    uint32_t n_events, max_peaks, max_vertices;
    int n_d0, n_phi0, n_kappa;
    int n_vphi, n_vr;
    float d0_cut;
    uint32_t n_min;
    double dphi_v;
    // SPLIT kernel (a handful of events: single-event latency): `split` blocks share an event's tracks and vote into the
    // event's plane in global memory; the last block to finish takes the plane into shared memory and finds the peaks
    uint32_t split;
    uint32_t* gplane;                // [kVtxSplitEvents][bins / 2], zero between calls
    uint32_t* done;                  // [kVtxSplitEvents], zero between calls
};

__device__ __forceinline__ uint32_t angle_bin(const float* ex, const float* ey, int n_vphi, float x, float y)
{
    uint32_t q;                                  // [0,pi/2): x>0,y>=0   [pi/2,pi): x<=0,y>0   [pi,3pi/2): x<0,y<=0   else
    if (x > 0.0f && y >= 0.0f) q = 0u;
    else if (x <= 0.0f && y > 0.0f) q = 1u;
    else if (x < 0.0f && y <= 0.0f) q = 2u;
    else q = 3u;
    uint32_t lo = q * ((uint32_t)n_vphi / 4u), hi = lo + (uint32_t)n_vphi / 4u - 1u;
    while (lo < hi) {
        const uint32_t mid = (lo + hi + 1u) / 2u;
        const float cr = __fsub_rn(__fmul_rn(ex[mid], y), __fmul_rn(ey[mid], x));
        if (cr >= 0.0f) lo = mid; else hi = mid - 1u;
    }
    return lo;
}

__device__ __forceinline__ uint32_t vcount(const uint32_t* acc, uint32_t b)
{
    return (acc[b >> 1] >> (16u * (b & 1u))) & 0xffffu;
}

// O-3 on the vertex plane for bin (iv, ir) with count c >= n_min
__device__ __forceinline__ bool vtx_is_peak(const uint32_t* acc, int NPV, int NR, int iv, int ir, uint32_t c)
{
    const uint32_t lin = (uint32_t)iv * (uint32_t)NR + (uint32_t)ir;
#pragma unroll
    for (int dp = -1; dp <= 1; ++dp) {
        int jv = iv + dp;
        jv = (jv < 0) ? jv + NPV : (jv >= NPV ? jv - NPV : jv);
#pragma unroll
        for (int dr = -1; dr <= 1; ++dr) {
            if (dp == 0 && dr == 0) continue;
            const int jr = ir + dr;
            if (jr < 0 || jr >= NR) continue;
            const uint32_t nl = (uint32_t)jv * (uint32_t)NR + (uint32_t)jr;
            const uint32_t cn = vcount(acc, nl);
            if (!(c > cn || (c == cn && lin < nl))) return false;
        }
    }
    return true;
}

template <bool SPLIT>
__global__ void __launch_bounds__(kVtxThreads) vertex_kernel(const VtxParams p)
{
    extern __shared__ uint32_t acc[];                            // [n_vphi * n_vr / 2]: two 16-bit counts per word, then tables
    __shared__ uint32_t s_warp[kVtxThreads / 32];
    __shared__ uint32_t s_total;
    __shared__ uint32_t s_last;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const uint32_t e = SPLIT ? blockIdx.x / p.split : blockIdx.x;
    const uint32_t sub = SPLIT ? blockIdx.x - e * p.split : 0u;
    const uint32_t n_sub = SPLIT ? p.split : 1u;
    const int NPV = p.n_vphi, NR = p.n_vr;
    const uint32_t bins = (uint32_t)NPV * (uint32_t)NR;
    // the edge directions (binary-searched per vote) and the R_v centres live in shared memory behind the accumulator
    float* s_ex = reinterpret_cast<float*>(acc + bins / 2);
    float* s_ey = s_ex + NPV;
    float* s_rc = s_ey + NPV;
    for (uint32_t i = tid; i < bins / 2; i += kVtxThreads) acc[i] = 0u;
    for (int i = tid; i < NPV; i += kVtxThreads) { s_ex[i] = p.ex[i]; s_ey[i] = p.ey[i]; }
    for (int i = tid; i < NR; i += kVtxThreads) s_rc[i] = p.rc[i];
    __syncthreads();

    const uint32_t np_e = p.n_peaks[e];
    const uint32_t T = (np_e == HOUGH_N_PEAKS_OVERFLOW) ? 0u : min(np_e, p.max_peaks);
    const hough_peak* pk = p.peaks + (size_t)e * p.max_peaks;
    // ---- O-6: one warp per track, lanes over the R_v bins ----
    uint32_t* const vote_plane = SPLIT ? p.gplane + (size_t)e * (bins / 2) : acc;
    for (uint32_t j = sub * (kVtxThreads / 32) + warp; j < T; j += n_sub * (kVtxThreads / 32)) {
        const uint32_t lin = pk[j].lin;
        const uint32_t ik = lin % (uint32_t)p.n_kappa, t = lin / (uint32_t)p.n_kappa;
        const uint32_t ip = t % (uint32_t)p.n_phi0, id = t / (uint32_t)p.n_phi0;
        const float d0 = (p.n_d0 > 1) ? __ldg(p.d0c + id) : 0.0f;
        if (!(fabsf(d0) > p.d0_cut)) continue;                   // prompt-compatible track: does not vote (warp-uniform)
        const float c0 = __ldg(p.c0 + ip), s0 = __ldg(p.s0 + ip), kap = __ldg(p.kc + ik);
        const float kd = __fmul_rn(kap, d0);
        const float w = __fsub_rn(1.0f, kd);
        const float d2 = __fmul_rn(d0, d0);
        const float two_d0 = __fadd_rn(d0, d0);
        for (int ir = lane; ir < NR; ir += 32) {
            const float r = s_rc[ir];
            const float r2 = __fmul_rn(r, r);
            const float num = __fsub_rn(__fmul_rn(kap, __fadd_rn(r2, d2)), two_d0);
            const float den = __fmul_rn(__fadd_rn(r, r), w);
            const float s = __fdiv_rn(num, den);
            if (!(fabsf(s) <= 1.0f)) continue;                   // the track does not reach this radius
            const float cd = __fsqrt_rn(__fsub_rn(1.0f, __fmul_rn(s, s)));
            const float x = __fsub_rn(__fmul_rn(c0, cd), __fmul_rn(s0, s));
            const float y = __fadd_rn(__fmul_rn(s0, cd), __fmul_rn(c0, s));
            const uint32_t b = angle_bin(s_ex, s_ey, NPV, x, y) * (uint32_t)NR + (uint32_t)ir;
            atomicAdd(&vote_plane[b >> 1], 1u << (16u * (b & 1u)));
        }
    }
    if (SPLIT) {
        // the last block of the event to get here takes the finished plane into shared memory (and leaves zeros behind)
        __threadfence();
        __syncthreads();
        if (tid == 0) s_last = (atomicAdd(p.done + e, 1u) == p.split - 1u) ? 1u : 0u;
        __syncthreads();
        if (!s_last) return;
        __threadfence();
        for (uint32_t i = tid; i < bins / 2; i += kVtxThreads) { acc[i] = __ldcg(vote_plane + i); vote_plane[i] = 0u; }
        if (tid == 0) p.done[e] = 0u;
    }
    __syncthreads();
    if (p.plane) {                                               // optional: the vertex plane itself (tests)
        uint32_t* out = reinterpret_cast<uint32_t*>(p.plane + (size_t)e * bins);
        for (uint32_t i = tid; i < bins / 2; i += kVtxThreads) out[i] = acc[i];
    }
    // ---- O-7: peaks in ascending linear index ----
    // pass 1: chunks of 32 consecutive bins, one bin per lane (conflict-free shared-memory reads), the peak predicate
    // of a chunk kept as a 32-bit ballot; pass 2: every thread owns a contiguous range of chunks, a block scan of the
    // popcounts gives the position of each peak in linear-index order.
    uint32_t* s_ballot = reinterpret_cast<uint32_t*>(s_rc + NR);     // [bins / 32]
    const uint32_t chunks = bins / 32u;                              // bins % 32 == 0 (n_vtx_phi % 4 == 0, n_vtx_r % 8 == 0)
    for (uint32_t q = warp; q < chunks; q += kVtxThreads / 32) {
        const uint32_t bb = q * 32u + (uint32_t)lane;
        const uint32_t c = vcount(acc, bb);
        const bool pk1 = c >= p.n_min && vtx_is_peak(acc, NPV, NR, (int)(bb / (uint32_t)NR), (int)(bb % (uint32_t)NR), c);
        const uint32_t bal = __ballot_sync(0xffffffffu, pk1);
        if (lane == 0) s_ballot[q] = bal;
    }
    __syncthreads();
    const uint32_t per = (chunks + kVtxThreads - 1) / kVtxThreads;
    const uint32_t q_lo = min((uint32_t)tid * per, chunks), q_hi = min(q_lo + per, chunks);
    uint32_t mine = 0;
    for (uint32_t q = q_lo; q < q_hi; ++q) mine += (uint32_t)__popc(s_ballot[q]);
    uint32_t incl = mine;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const uint32_t t = __shfl_up_sync(0xffffffffu, incl, d);
        if (lane >= d) incl += t;
    }
    if (lane == 31) s_warp[warp] = incl;
    __syncthreads();
    if (warp == 0) {
        const uint32_t wsum = (lane < kVtxThreads / 32) ? s_warp[lane] : 0u;
        uint32_t winc = wsum;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const uint32_t t = __shfl_up_sync(0xffffffffu, winc, d);
            if (lane >= d) winc += t;
        }
        if (lane < kVtxThreads / 32) s_warp[lane] = winc - wsum;
        if (lane == 31) s_total = winc;
    }
    __syncthreads();
    uint32_t pos = s_warp[warp] + incl - mine;
    hough_vertex* out = p.vertices + (size_t)e * p.max_vertices;
    for (uint32_t q = q_lo; q < q_hi && pos < p.max_vertices; ++q) {
        uint32_t word = s_ballot[q];
        while (word && pos < p.max_vertices) {
            const uint32_t bb = q * 32u + (uint32_t)(__ffs(word) - 1);
            word &= word - 1;
            const int iv = (int)(bb / (uint32_t)NR), ir = (int)(bb % (uint32_t)NR);
            hough_vertex vx;
            vx.r = s_rc[ir];
            vx.phi = (float)(((double)iv + 0.5) * p.dphi_v);
            vx.n_tracks = vcount(acc, bb); vx.lin = bb;
            out[pos++] = vx;
        }
    }
    if (tid == 0) { p.n_vertices[e] = s_total; p.flag[e] = s_total > 0u ? 1 : 0; }
}

}  // namespace

cudaError_t launch_vertices(hough_ctx* c, uint32_t n_events, const hough_peak* d_peaks, const uint32_t* d_n_peaks,
                            float d0_cut, uint32_t n_min, hough_vertex* d_vertices, uint32_t* d_n_vertices,
                            uint8_t* d_flag, uint16_t* d_plane, cudaStream_t st)
{
    if (n_events == 0) return cudaSuccess;
    VtxParams p;
    p.peaks = d_peaks; p.n_peaks = d_n_peaks; p.vertices = d_vertices; p.n_vertices = d_n_vertices; p.flag = d_flag;
    p.plane = d_plane;
    p.d0c = c->d_d0c; p.c0 = c->d_c0; p.s0 = c->d_s0; p.kc = c->d_kc;
    p.ex = c->d_vex; p.ey = c->d_vey; p.rc = c->d_vrc;
    p.n_events = n_events; p.max_peaks = c->cfg.max_peaks_per_event; p.max_vertices = c->cfg.max_vertices_per_event;
    p.n_d0 = (int)c->cfg.n_d0; p.n_phi0 = (int)c->cfg.n_phi0; p.n_kappa = (int)c->cfg.n_kappa;
    p.n_vphi = (int)c->cfg.n_vtx_phi; p.n_vr = (int)c->cfg.n_vtx_r;
    p.d0_cut = d0_cut; p.n_min = n_min;
    p.dphi_v = 6.283185307179586476925286766559 / (double)c->cfg.n_vtx_phi;
    const size_t bins = (size_t)c->cfg.n_vtx_phi * c->cfg.n_vtx_r;
    const size_t smem = bins * 2 + (2 * (size_t)c->cfg.n_vtx_phi + c->cfg.n_vtx_r) * 4 + bins / 32 * 4;
    // a handful of events (single-event latency): several blocks per event
    const bool split = n_events <= kVtxSplitEvents && c->d_vtx_gplane != nullptr;
    p.split = split ? kVtxSplit : 1u;
    p.gplane = c->d_vtx_gplane; p.done = c->d_vtx_done;
    cudaError_t err = cudaFuncSetAttribute(split ? vertex_kernel<true> : vertex_kernel<false>,
                                           cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (err != cudaSuccess) return err;
    if (split) vertex_kernel<true><<<n_events * kVtxSplit, kVtxThreads, smem, st>>>(p);
    else vertex_kernel<false><<<n_events, kVtxThreads, smem, st>>>(p);
    ++c->launches;
    return cudaGetLastError();
}
