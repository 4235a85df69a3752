// A5 peak -> track conversion and A6 seeded phi-cone track-jets, one warp per event (sm_100a); for small batches
// (single-event latency) one block of 8 warps per event.
//
// DESIGN.md O-4 / O-5 (PAPER.md:87 transverse-momentum measurement; PAPER.md:113-123 jets and the
// interaction-point remark; clustering rule from north_star as read in R17-R22).  All decisions are taken on
// integer bin keys; floats only appear in the reported fields (tolerance 1e-5).
#include <mutex>

#include "hough_internal.cuh"

namespace {

constexpr double kTwoPi = 6.283185307179586476925286766559;
constexpr uint64_t KEY_ASSIGNED = 1ull << 63;

struct JetParams {
    const hough_peak* peaks; const uint32_t* n_peaks;
    hough_track* tracks; hough_jet* jets; uint32_t* n_jets; uint8_t* flag;
    uint64_t* keys;
    const float* d0c;
    uint32_t n_events, max_peaks, max_jets;
    int n_d0, n_phi0, n_kappa;
    float kmax, b_tesla, d0_cut;
    int cone_bins;
    uint32_t n_min;
};

__device__ __forceinline__ uint64_t warp_min_u64(uint64_t v)
{
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) {
        const uint64_t o = __shfl_xor_sync(0xffffffffu, v, d);
        v = (o < v) ? o : v;
    }
    return v;
}

// one block of NW warps per event (NW = 1: large batches, many events per SM; NW = 8: a handful of events, where the
// length of the per-jet passes over the tracks is what counts); the clustering keys live in shared memory when the
// event's tracks fit (kSmemKeys of them), else in the context's global workspace
constexpr uint32_t kSmemKeys = 4096;

template <int NW>
__global__ void __launch_bounds__(32 * NW) jets_kernel(const JetParams p)
{
    __shared__ uint64_t s_keys[kSmemKeys];
    __shared__ uint64_t s_best[NW];
    __shared__ uint32_t s_cnt[NW][2];
    __shared__ double s_pt[NW];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    constexpr uint32_t NT = 32u * NW;
    const uint32_t e = blockIdx.x;
    if (e >= p.n_events) return;
    const uint32_t np_e = p.n_peaks[e];
    const uint32_t T = (np_e == HOUGH_N_PEAKS_OVERFLOW) ? 0u : min(np_e, p.max_peaks);   // overflowed fused event: no tracks
    const hough_peak* pk = p.peaks + (size_t)e * p.max_peaks;
    hough_track* trk = p.tracks + (size_t)e * p.max_peaks;
    hough_jet* jets = p.jets + (size_t)e * p.max_jets;
    uint64_t* keys = (T <= kSmemKeys) ? s_keys : p.keys + (size_t)e * p.max_peaks;
    const int NK = p.n_kappa, N = p.n_phi0;
    const double kmax = (double)p.kmax;
    auto block_sync = [&]() { if (NW == 1) __syncwarp(); else __syncthreads(); };

    // A5: tracks, and the integer keys of the clustering: [63] assigned, [32..55] a = |2 ik - (NK-1)|,
    // [1..21] ip, [0] displaced
    for (uint32_t j = tid; j < T; j += NT) {
        const uint32_t lin = pk[j].lin;
        const uint32_t ik = lin % (uint32_t)NK, t = lin / (uint32_t)NK;
        const uint32_t ip = t % (uint32_t)N, id = t / (uint32_t)N;
        const double kc = -kmax + ((double)ik + 0.5) * (2.0 * kmax / (double)NK);
        hough_track tr;
        tr.pt = (float)(0.3e-3 * (double)p.b_tesla / fabs(kc));
        tr.phi0 = (float)(((double)ip + 0.5) * (kTwoPi / (double)N));
        const float d0 = (p.n_d0 > 1) ? p.d0c[id] : 0.0f;
        tr.d0 = d0;
        tr.q = (kc < 0.0) ? +1 : -1;
        tr.jet = -1;
        trk[j] = tr;
        const uint32_t a = (uint32_t)abs(2 * (int)ik - (NK - 1));
        const uint32_t disp = (p.n_d0 > 1 && fabsf(d0) > p.d0_cut) ? 1u : 0u;
        keys[j] = ((uint64_t)a << 32) | ((uint64_t)ip << 1) | disp;
    }
    block_sync();

    // A6: repeat { seed = unassigned track with the smallest (a, j); members = unassigned within the cone }
    uint32_t J = 0;
    bool any_flag = false;
    for (;;) {
        uint64_t best = ~0ull;
        for (uint32_t j = tid; j < T; j += NT) {
            const uint64_t k = keys[j];
            if (!(k & KEY_ASSIGNED)) {
                const uint64_t cand = (k & 0x00ffffff00000000ull) | j;
                best = (cand < best) ? cand : best;
            }
        }
        best = warp_min_u64(best);
        if (NW > 1) {
            if (lane == 0) s_best[warp] = best;
            __syncthreads();
#pragma unroll
            for (int w = 0; w < NW; ++w) { const uint64_t o = s_best[w]; best = (o < best) ? o : best; }
        }
        if (best == ~0ull) break;                                // block-uniform
        const uint32_t seed = (uint32_t)(best & 0xffffffffu);
        const int ip_seed = (int)((keys[seed] >> 1) & 0xfffffu);
        block_sync();                                            // every thread has read the seed's key
        uint32_t n_tracks = 0, n_disp = 0;
        double sum_pt = 0.0;
        for (uint32_t j = tid; j < T; j += NT) {
            const uint64_t k = keys[j];
            if (k & KEY_ASSIGNED) continue;
            int d = abs((int)((k >> 1) & 0xfffffu) - ip_seed);
            d = min(d, N - d);
            if (d <= p.cone_bins) {
                keys[j] = k | KEY_ASSIGNED;
                ++n_tracks;
                n_disp += (uint32_t)(k & 1u);
                sum_pt += (double)trk[j].pt;
                if (J < p.max_jets) trk[j].jet = (int32_t)J;
            }
        }
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) {
            n_tracks += __shfl_xor_sync(0xffffffffu, n_tracks, d);
            n_disp += __shfl_xor_sync(0xffffffffu, n_disp, d);
            sum_pt += __shfl_xor_sync(0xffffffffu, sum_pt, d);
        }
        if (NW > 1) {
            if (lane == 0) { s_cnt[warp][0] = n_tracks; s_cnt[warp][1] = n_disp; s_pt[warp] = sum_pt; }
            __syncthreads();                                     // also orders the key updates before the next round
            n_tracks = 0; n_disp = 0; sum_pt = 0.0;
#pragma unroll
            for (int w = 0; w < NW; ++w) { n_tracks += s_cnt[w][0]; n_disp += s_cnt[w][1]; sum_pt += s_pt[w]; }
        } else {
            __syncwarp();
        }
        if (tid == 0 && J < p.max_jets) {
            hough_jet jt;
            jt.seed_track = seed; jt.n_tracks = n_tracks; jt.n_displaced = n_disp;
            jt.phi = trk[seed].phi0; jt.sum_pt = (float)sum_pt;
            jets[J] = jt;
        }
        any_flag = any_flag || (n_disp >= p.n_min);
        ++J;
    }
    if (tid == 0) { p.n_jets[e] = J; p.flag[e] = any_flag ? 1 : 0; }
}

}  // namespace

cudaError_t launch_jets(hough_ctx* c, uint32_t n_events, const hough_peak* d_peaks, const uint32_t* d_n_peaks,
                        int cone_bins, float d0_cut, uint32_t n_min, hough_track* d_tracks, hough_jet* d_jets,
                        uint32_t* d_n_jets, uint8_t* d_flag, cudaStream_t st)
{
    if (n_events == 0) return cudaSuccess;
    JetParams p;
    p.peaks = d_peaks; p.n_peaks = d_n_peaks; p.tracks = d_tracks; p.jets = d_jets; p.n_jets = d_n_jets;
    p.flag = d_flag; p.keys = c->d_jetkeys; p.d0c = c->d_d0c;
    p.n_events = n_events; p.max_peaks = c->cfg.max_peaks_per_event; p.max_jets = c->cfg.max_jets_per_event;
    p.n_d0 = (int)c->cfg.n_d0; p.n_phi0 = (int)c->cfg.n_phi0; p.n_kappa = (int)c->cfg.n_kappa;
    p.kmax = c->kmax; p.b_tesla = c->cfg.b_tesla; p.d0_cut = d0_cut; p.cone_bins = cone_bins; p.n_min = n_min;
    // few events (single-event latency): eight warps share an event's passes over its tracks
    if (n_events < 64) jets_kernel<8><<<n_events, 256, 0, st>>>(p);
    else jets_kernel<1><<<n_events, 32, 0, st>>>(p);
    ++c->launches;
    return cudaGetLastError();
}

// ---- hough_jets_static: the same kernel for callers that may not allocate ---------------------------------------
//
// Some users of this library cannot create a context because hough_create calls cudaMalloc: a trigger process whose
// device memory was all handed out at start-up, a real-time loop that cannot afford the device-wide stall of an
// allocation, a plug-in whose host runtime owns the allocator.  For them the two pieces of global scratch that
// jets_kernel needs live in the array below, which is part of this library's device image: it exists on every GPU
// that loads the library, from module load to process exit, and nobody has to allocate or free it.
//
// Layout: [0, kStaticD0Words) the d0 bin centres (float, written by static_d0_table_kernel at every call),
// then HOUGH_JETS_STATIC_MAX_TRACKS clustering keys (the kernel uses them for events with more than kSmemKeys tracks;
// it writes key j of an event before any thread reads it, so nothing has to be cleared between calls).
// All calls on a device share the array: calls that overlap on the GPU race.
namespace {

constexpr size_t kStaticD0Words = HOUGH_JETS_STATIC_MAX_D0 / 2;                        // uint64 words holding the floats
constexpr size_t kStaticWords = kStaticD0Words + (size_t)HOUGH_JETS_STATIC_MAX_TRACKS;
static __device__ __align__(256) unsigned long long g_jets_static_scratch[kStaticWords];

// In host code `g_jets_static_scratch` is only the host-side handle of the symbol, not a device address; the address
// a kernel can use comes from cudaGetSymbolAddress, asked once per device with that device current.
constexpr int kMaxStaticDevices = 64;
std::mutex g_static_mutex;
void* g_static_addr[kMaxStaticDevices] = {};

cudaError_t static_scratch_of_current_device(void** out)
{
    int dev = -1;
    cudaError_t err = cudaGetDevice(&dev);
    if (err != cudaSuccess) return err;
    if (dev < 0 || dev >= kMaxStaticDevices) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_static_mutex);
    if (!g_static_addr[dev]) {
        int major = 0;
        err = cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev);
        if (err != cudaSuccess) return err;
        if (major < 10) return cudaErrorNoKernelImageForDevice;      // the library holds sm_100a code only
        void* p = nullptr;
        err = cudaGetSymbolAddress(&p, g_jets_static_scratch);
        if (err != cudaSuccess) return err;
        if (!p) return cudaErrorInvalidSymbol;
        g_static_addr[dev] = p;
    }
    *out = g_static_addr[dev];
    return cudaSuccess;
}

// d0 bin centres exactly as hough_create forms them on the host (O-0: double arithmetic, one operation per step,
// rounded once to fp32); the *_rn intrinsics keep the compiler from contracting the multiply and the add
__global__ void static_d0_table_kernel(float* d0c, uint32_t nd, double d0_min, double d0_max)
{
    const uint32_t id = blockIdx.x * blockDim.x + threadIdx.x;
    if (id >= nd) return;
    const double w = __ddiv_rn(__dsub_rn(d0_max, d0_min), (double)nd);
    d0c[id] = __double2float_rn(__dadd_rn(d0_min, __dmul_rn((double)id + 0.5, w)));
}

}  // namespace

cudaError_t launch_jets_static(const hough_config* g, uint32_t n_events, const hough_peak* d_peaks,
                               const uint32_t* d_n_peaks, int cone_bins, float d0_cut, uint32_t n_min,
                               hough_track* d_tracks, hough_jet* d_jets, uint32_t* d_n_jets, uint8_t* d_flag,
                               cudaStream_t st)
{
    void* base = nullptr;
    cudaError_t err = static_scratch_of_current_device(&base);
    if (err != cudaSuccess) return err;
    if (n_events == 0) return cudaSuccess;
    float* d0c = reinterpret_cast<float*>(base);
    if (g->n_d0 > 1) {
        static_d0_table_kernel<<<(g->n_d0 + 255) / 256, 256, 0, st>>>(d0c, g->n_d0, (double)g->d0_min, (double)g->d0_max);
        err = cudaGetLastError();
        if (err != cudaSuccess) return err;
    }
    JetParams p;
    p.peaks = d_peaks; p.n_peaks = d_n_peaks; p.tracks = d_tracks; p.jets = d_jets; p.n_jets = d_n_jets;
    p.flag = d_flag;
    p.keys = reinterpret_cast<uint64_t*>(base) + kStaticD0Words;
    p.d0c = d0c;
    p.n_events = n_events; p.max_peaks = g->max_peaks_per_event; p.max_jets = g->max_jets_per_event;
    p.n_d0 = (int)g->n_d0; p.n_phi0 = (int)g->n_phi0; p.n_kappa = (int)g->n_kappa;
    p.kmax = g->kappa_max; p.b_tesla = g->b_tesla; p.d0_cut = d0_cut; p.cone_bins = cone_bins; p.n_min = n_min;
    if (n_events < 64) jets_kernel<8><<<n_events, 256, 0, st>>>(p);
    else jets_kernel<1><<<n_events, 32, 0, st>>>(p);
    return cudaGetLastError();
}
