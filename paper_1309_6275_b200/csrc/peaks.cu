// A3 peak stencil + A4 ordered compaction (sm_100a).
//
// Definition (O-3; "looking for local maxima in the parameter space"): bin b is a peak
// iff popcount(mask[b]) >= l_min and, for every existing neighbour n in the 3x3(x3) neighbourhood (phi0
// periodic, kappa and d0 clipped), count[b] > count[n] or (count[b] == count[n] and lin(b) < lin(n)).
// A peak therefore needs count[b] >= popcount(mask[b]) >= l_min >= 1.
//
// Stencil kernel = one streaming pass over the count plane.  The plane of an event is cut, in linear-index
// order, into units of UB bins (UB = 16: one 256-bit load per lane; UB = 8: one 128-bit load when the plane is
// not a whole number of 32-byte units) and groups of 32 units (one warp-wide load: 1 KB or 512 B, contiguous).
// A warp takes kUnroll consecutive groups per iteration and has the loads of its next iteration in flight while
// it examines the current one (software pipeline): the pass is bound by HBM, not by instruction issue (about 3
// thread instructions per bin).  Per unit the packed
// 16-bit maximum (VIMNMX3.U16x2) is compared with l_min; only bins with count >= l_min (rare at the trigger
// thresholds) read their mask word and, if popcount(mask) >= l_min, run the 8 / 26-neighbour test, whose reads
// go to L2 (the neighbouring rows and d0 slabs were streamed by neighbouring warps a moment earlier).
// Output: one bit per bin, written only for groups that hold a peak, and a peak count per group.
// Compaction kernel: one block per event scans the group counts in linear-index order (block prefix sum,
// 8 groups per thread) and writes the first max_peaks records; n_peaks is the true total.
#include "hough_internal.cuh"

namespace {

#ifndef STENCIL_UNROLL
#define STENCIL_UNROLL 4
#endif
#ifndef STENCIL_MINB
#define STENCIL_MINB 3
#endif
constexpr int kUnroll = STENCIL_UNROLL;           // groups per warp iteration
constexpr int kStencilThreads = 256;

struct PeakParams {
    const uint16_t* count;
    const uint16_t* mask;
    uint8_t* bitmap;             // [E][bins/8], a group's bytes are only defined where grpcnt > 0
    uint16_t* grpcnt;            // [E][groups_per_event] peaks per group of 32*UB bins
    int n_d0, n_phi0, n_kappa;
    uint32_t n_events;
    uint32_t bins;               // per event
    uint32_t units;              // per event = bins / UB
    uint32_t groups;             // per event = ceil(units / 32)
    uint32_t quads;              // per event = ceil(groups / kUnroll)
    uint32_t l_min;
};

__device__ __forceinline__ void load_unit(const uint16_t* p, uint32_t (&r)[8])
{
    asm volatile("ld.global.nc.L1::no_allocate.v8.u32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7])
                 : "l"(p));
}
__device__ __forceinline__ void load_unit(const uint16_t* p, uint32_t (&r)[4])
{
    asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]) : "l"(p));
}

__device__ __forceinline__ uint32_t packed_max(const uint32_t (&r)[8])
{
    const uint32_t a = __vimax3_u16x2(r[0], r[1], r[2]);
    const uint32_t b = __vimax3_u16x2(r[3], r[4], r[5]);
    return __vimax3_u16x2(__vimax3_u16x2(r[6], r[7], a), b, b);
}
__device__ __forceinline__ uint32_t packed_max(const uint32_t (&r)[4])
{
    return __vimax3_u16x2(__vimax3_u16x2(r[0], r[1], r[2]), r[3], r[3]);
}

__device__ __forceinline__ bool any_half_ge(uint32_t m, uint32_t l_min)
{
    return (m & 0xffffu) >= l_min || (m >> 16) >= l_min;
}

// O-3 for one bin with count c >= l_min at linear index lin of event planes cnt_e / msk_e.  Three batches of
// loads, each issued before its first comparison (after the mask test): the kappa neighbours, the two phi0 rows of the own d0 slab
// (hot in L2: streamed by the neighbouring warps), then the six rows of the slabs id-1 / id+1.  A clipped
// neighbour reads as 0, which never beats c >= 1.
__device__ __noinline__ bool is_peak(const uint16_t* __restrict__ cnt_e, const uint16_t* __restrict__ msk_e,
                                     uint32_t lin, uint32_t c, int ND, int N, int NK, uint32_t l_min)
{
    // the mask test first: one load, and on dense accumulators (C4: 0.7 % of the bins reach l_min votes, almost
    // all of them isolated spikes of same-layer hits) it rejects 99.5 % of the candidates that 26 neighbour loads
    // would let through
    if ((uint32_t)__popc((uint32_t)__ldg(msk_e + lin)) < l_min) return false;
    const uint32_t row = lin / (uint32_t)NK;
    const int k = (int)(lin - row * (uint32_t)NK);
    const int id = (int)(row / (uint32_t)N);
    const int ip = (int)(row - (uint32_t)id * (uint32_t)N);
    const bool has_l = k > 0, has_r = k + 1 < NK;
    // same row: the left neighbour has the smaller linear index (must be strictly smaller), the right one may tie
    const uint32_t vl = has_l ? (uint32_t)__ldg(cnt_e + lin - 1) : 0u;
    const uint32_t vr = has_r ? (uint32_t)__ldg(cnt_e + lin + 1) : 0u;
    if (!(vl < c && vr <= c)) return false;
    const int ipm = (ip == 0) ? N - 1 : ip - 1, ipp = (ip == N - 1) ? 0 : ip + 1;
    // max over the three kappa offsets of row nrow must be < c if that row precedes ours in linear-index
    // order, <= c otherwise (rows differ, so the order of the indices is the order of the rows)
    auto row_ok = [&](uint32_t nrow, bool ok) {
        const uint16_t* r = cnt_e + (size_t)nrow * NK + k;
        const uint32_t v0 = (ok && has_l) ? (uint32_t)__ldg(r - 1) : 0u;
        const uint32_t v1 = ok ? (uint32_t)__ldg(r) : 0u;
        const uint32_t v2 = (ok && has_r) ? (uint32_t)__ldg(r + 1) : 0u;
        return max(max(v0, v1), v2) < ((nrow < row) ? c : c + 1u);
    };
    const uint32_t base = (uint32_t)id * (uint32_t)N;
    const bool a0 = row_ok(base + (uint32_t)ipm, true), a1 = row_ok(base + (uint32_t)ipp, true);
    if (!(a0 && a1)) return false;
    const bool dn = id > 0, up = id + 1 < ND;
    const uint32_t bd = dn ? base - (uint32_t)N : base, bu = up ? base + (uint32_t)N : base;
    const bool b0 = row_ok(bd + (uint32_t)ipm, dn), b1 = row_ok(bd + (uint32_t)ip, dn), b2 = row_ok(bd + (uint32_t)ipp, dn);
    const bool c0 = row_ok(bu + (uint32_t)ipm, up), c1 = row_ok(bu + (uint32_t)ip, up), c2 = row_ok(bu + (uint32_t)ipp, up);
    return b0 && b1 && b2 && c0 && c1 && c2;
}

// Bit j set: bin j of the unit has count >= l_min (packed 16-bit compare, two bins per instruction).  On the
// accumulators of the five configs a neighbour inside the unit almost never beats such a bin (1 % at C4), so no
// in-register neighbour prefilter: the mask test that follows rejects far more (99.5 % at C4) for one load.
template <int NW>
__device__ __forceinline__ uint32_t unit_candidates(const uint32_t (&d)[NW], uint32_t lmin2)
{
    uint32_t bits = 0;
#pragma unroll
    for (int w = 0; w < NW; ++w) {
        const uint32_t t = __vcmpgeu2(d[w], lmin2) & 0x00010001u;   // bit 0: low bin, bit 16: high bin
        bits |= ((t | (t >> 15)) & 3u) << (2 * w);
    }
    return bits;
}

template <int UB>
__global__ void __launch_bounds__(kStencilThreads, STENCIL_MINB) peak_stencil_kernel(const PeakParams p)
{
    constexpr int NW = UB / 2;                                   // 32-bit words per unit
    const int lane = threadIdx.x & 31;
    const uint32_t n_warps = gridDim.x * (kStencilThreads / 32);
    const uint32_t gw = blockIdx.x * (kStencilThreads / 32) + (threadIdx.x >> 5);
    const uint64_t total_quads = (uint64_t)p.n_events * p.quads;

    // software pipeline: the loads of the next iteration are in flight while this one is examined (on dense
    // accumulators the candidates' mask loads would otherwise serialise with the stream)
    auto load_quad = [&](uint64_t q, uint32_t (&dst)[kUnroll][NW]) {
        const uint32_t e = (uint32_t)(q / p.quads);
        const uint32_t g0 = (uint32_t)(q - (uint64_t)e * p.quads) * kUnroll;
        const uint16_t* cnt_e = p.count + (size_t)e * p.bins;
#pragma unroll
        for (int u = 0; u < kUnroll; ++u) {
            const uint32_t unit = (g0 + u) * 32u + lane;
            if (unit < p.units) load_unit(cnt_e + (size_t)unit * UB, dst[u]);
            else {
#pragma unroll
                for (int w = 0; w < NW; ++w) dst[u][w] = 0;
            }
        }
    };
    uint32_t d[kUnroll][NW], dn[kUnroll][NW];
    if (gw < total_quads) load_quad(gw, dn);
    for (uint64_t q = gw; q < total_quads; q += n_warps) {
        const uint32_t e = (uint32_t)(q / p.quads);
        const uint32_t qi = (uint32_t)(q - (uint64_t)e * p.quads);
        const uint16_t* cnt_e = p.count + (size_t)e * p.bins;
        const uint32_t g0 = qi * kUnroll;
#pragma unroll
        for (int u = 0; u < kUnroll; ++u)
#pragma unroll
            for (int w = 0; w < NW; ++w) d[u][w] = dn[u][w];
        if (q + n_warps < total_quads) load_quad(q + n_warps, dn);
        uint32_t m = packed_max(d[0]);
#pragma unroll
        for (int u = 1; u < kUnroll; ++u) { const uint32_t t = packed_max(d[u]); m = __vimax3_u16x2(m, t, t); }
        const bool ge = any_half_ge(m, p.l_min);
        uint32_t bits[kUnroll];
#pragma unroll
        for (int u = 0; u < kUnroll; ++u) bits[u] = 0;
        if (ge) {                                                // some bin of this lane may be a peak
            const uint32_t lmin2 = p.l_min | (p.l_min << 16);
            const uint16_t* msk_e = p.mask + (size_t)e * p.bins;
            uint32_t cand[kUnroll], mfirst[kUnroll];
#pragma unroll
            for (int u = 0; u < kUnroll; ++u)
                cand[u] = unit_candidates<NW>(d[u], lmin2);
            // the mask words of the first candidate of every unit are fetched together (dense accumulators: most
            // units with a candidate have exactly one, and its mask rejects it), then the survivors are tested
#pragma unroll
            for (int u = 0; u < kUnroll; ++u) {
                mfirst[u] = 0xffffu;
                if (cand[u]) mfirst[u] = (uint32_t)__ldg(msk_e + ((g0 + u) * 32u + lane) * UB + (__ffs(cand[u]) - 1));
            }
#pragma unroll
            for (int u = 0; u < kUnroll; ++u)
                if (cand[u] && (uint32_t)__popc(mfirst[u]) < p.l_min) cand[u] &= cand[u] - 1;
#pragma unroll
            for (int u = 0; u < kUnroll; ++u) {
                const uint32_t lin0 = ((g0 + u) * 32u + lane) * UB;
                uint32_t cd = cand[u];
                while (cd) {
                    const int j = __ffs(cd) - 1;
                    cd &= cd - 1;
                    const uint32_t c = (uint32_t)__ldg(cnt_e + lin0 + j);       // re-read: no dynamic register indexing
                    if (is_peak(cnt_e, msk_e, lin0 + j, c, p.n_d0, p.n_phi0, p.n_kappa, p.l_min)) bits[u] |= 1u << j;
                }
            }
        }
        uint16_t* gc = p.grpcnt + (size_t)e * p.groups;
#pragma unroll
        for (int u = 0; u < kUnroll; ++u) {
            const uint32_t g = g0 + u;
            if (g >= p.groups) break;                            // warp-uniform
            const unsigned any = __ballot_sync(0xffffffffu, bits[u] != 0);
            uint32_t n = 0;
            if (any) {                                           // warp-uniform
                n = __reduce_add_sync(0xffffffffu, (uint32_t)__popc(bits[u]));
                const uint32_t unit = g * 32u + lane;
                if (unit < p.units) {
                    uint8_t* bm = p.bitmap + (size_t)e * (p.bins / 8) + (size_t)unit * (UB / 8);
                    if (UB == 16) *reinterpret_cast<uint16_t*>(bm) = (uint16_t)bits[u];
                    else *bm = (uint8_t)bits[u];
                }
            }
            if (lane == 0) gc[g] = (uint16_t)n;
        }
    }
}

// ---- A4: ordered compaction from the group counts + bitmap --------------------------------------------------

constexpr int kCompactThreads = 1024;
constexpr int kGroupsPerThread = 8;

__global__ void __launch_bounds__(kCompactThreads) peak_compact_kernel(const uint16_t* __restrict__ count,
                                                                       const uint16_t* __restrict__ mask,
                                                                       const uint8_t* __restrict__ bitmap,
                                                                       const uint16_t* __restrict__ grpcnt,
                                                                       uint32_t bins, uint32_t groups,
                                                                       uint32_t group_bins, uint32_t max_peaks,
                                                                       hough_peak* __restrict__ peaks,
                                                                       uint32_t* __restrict__ n_peaks)
{
    __shared__ uint32_t s_warp[32];
    __shared__ uint32_t s_total;
    const uint32_t e = blockIdx.x;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const uint8_t* bm = bitmap + (size_t)e * (bins / 8);
    const uint16_t* gc = grpcnt + (size_t)e * groups;
    const uint16_t* cnt_e = count + (size_t)e * bins;
    const uint16_t* msk_e = mask + (size_t)e * bins;
    hough_peak* out = peaks + (size_t)e * max_peaks;
    const uint32_t group_bytes = group_bins / 8;
    // 32-bit reads of a group's bitmap: groups are at most 64 bytes, and word aligned if the event's bitmap is
    const bool words_ok = group_bytes <= 64u && (group_bytes & 3u) == 0u && ((reinterpret_cast<uintptr_t>(bm) & 3u) == 0);
    uint32_t running = 0;
    for (uint32_t base = 0; base < groups; base += kCompactThreads * kGroupsPerThread) {
        const uint32_t g_first = base + (uint32_t)tid * kGroupsPerThread;
        uint32_t cg[kGroupsPerThread];
        uint32_t c = 0;
#pragma unroll
        for (int i = 0; i < kGroupsPerThread; ++i) {
            cg[i] = (g_first + i < groups) ? (uint32_t)gc[g_first + i] : 0u;
            c += cg[i];
        }
        // block exclusive prefix sum of c
        uint32_t incl = c;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const uint32_t t = __shfl_up_sync(0xffffffffu, incl, d);
            if (lane >= d) incl += t;
        }
        if (lane == 31) s_warp[warp] = incl;
        __syncthreads();
        if (warp == 0) {
            uint32_t wsum = s_warp[lane], winc = wsum;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                const uint32_t t = __shfl_up_sync(0xffffffffu, winc, d);
                if (lane >= d) winc += t;
            }
            s_warp[lane] = winc - wsum;
            if (lane == 31) s_total = winc;
        }
        __syncthreads();
        uint32_t pos = running + s_warp[warp] + incl - c;
        if (c > 0 && pos < max_peaks) {
            for (int i = 0; i < kGroupsPerThread && pos < max_peaks; ++i) {
                if (cg[i] == 0) continue;
                const uint32_t g = g_first + i;
                const uint8_t* gp = bm + (size_t)g * group_bytes;
                const uint32_t lin_g = g * group_bins;
                const uint32_t nbytes = min(group_bytes, bins / 8 - g * group_bytes);     // ragged last group
                if (words_ok && (nbytes & 3u) == 0u) {                  // the group's bitmap as 32-bit words, all loads first
                    const uint32_t* gw = reinterpret_cast<const uint32_t*>(gp);
                    uint32_t wv[16];
#pragma unroll
                    for (int w = 0; w < 16; ++w) wv[w] = ((uint32_t)w * 4u < nbytes) ? __ldg(gw + w) : 0u;
#pragma unroll
                    for (int w = 0; w < 16; ++w) {
                        uint32_t word = wv[w];
                        while (word && pos < max_peaks) {
                            const int qb = __ffs(word) - 1;
                            word &= word - 1;
                            const uint32_t lin = lin_g + (uint32_t)w * 32u + qb;
                            hough_peak pk;
                            pk.lin = lin; pk.count = cnt_e[lin]; pk.mask = msk_e[lin];
                            out[pos++] = pk;
                        }
                    }
                } else {
                    for (uint32_t b = 0; b < nbytes && pos < max_peaks; ++b) {
                        uint32_t byte = gp[b];
                        while (byte && pos < max_peaks) {
                            const int qb = __ffs(byte) - 1;
                            byte &= byte - 1;
                            const uint32_t lin = lin_g + b * 8 + qb;
                            hough_peak pk;
                            pk.lin = lin; pk.count = cnt_e[lin]; pk.mask = msk_e[lin];
                            out[pos++] = pk;
                        }
                    }
                }
            }
        }
        running += s_total;
        __syncthreads();
    }
    if (tid == 0) n_peaks[e] = running;
}

// ---- fused path: order the confirmed candidates of an event ------------------------------------------------
// One block per event.  The confirmed candidates (state == 1) are compacted into 64-bit keys lin << 32 | cm, sorted
// ascending with a bitonic network (in shared memory up to kSortSmemKeys keys, in the context's global scratch
// beyond), and the first max_peaks are written as hough_peak records; n_peaks is the true total.  An event whose
// candidates did not fit the candidate buffer gets n_peaks = HOUGH_N_PEAKS_OVERFLOW and raises the sticky bit.
// The event's candidate counter is reset for the next call.

constexpr int kFinalThreads = 1024;
constexpr uint32_t kSortSmemKeys = 16384;                       // 128 KB of dynamic shared memory

__global__ void __launch_bounds__(kFinalThreads) peaks_finalize_kernel(const PeakCand* __restrict__ cand,
                                                                       uint32_t* __restrict__ cand_n, uint32_t cap,
                                                                       unsigned long long* __restrict__ gkeys,
                                                                       uint32_t cap_pow2, uint32_t max_peaks,
                                                                       hough_peak* __restrict__ peaks,
                                                                       uint32_t* __restrict__ n_peaks,
                                                                       uint32_t* __restrict__ status)
{
    extern __shared__ unsigned long long skeys[];
    __shared__ uint32_t s_warp[32];
    __shared__ uint32_t s_total;
    const uint32_t e = blockIdx.x;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const uint32_t n_raw = cand_n[e];
    const uint32_t n = min(n_raw, cap);
    const PeakCand* ce = cand + (size_t)e * cap;
    unsigned long long* keys = (n <= kSortSmemKeys) ? skeys : gkeys + (size_t)e * cap_pow2;
    uint32_t running = 0;
    for (uint32_t base = 0; base < n; base += kFinalThreads) {
        const uint32_t idx = base + (uint32_t)tid;
        bool alive = false;
        unsigned long long key = 0;
        if (idx < n) {
            const PeakCand pc = ce[idx];
            alive = pc.state == 1u;
            key = ((unsigned long long)pc.lin << 32) | pc.cm;
        }
        const unsigned bal = __ballot_sync(0xffffffffu, alive);
        if (lane == 0) s_warp[warp] = (uint32_t)__popc(bal);
        __syncthreads();
        if (warp == 0) {
            const uint32_t wsum = s_warp[lane];
            uint32_t winc = wsum;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                const uint32_t t = __shfl_up_sync(0xffffffffu, winc, d);
                if (lane >= d) winc += t;
            }
            s_warp[lane] = winc - wsum;
            if (lane == 31) s_total = winc;
        }
        __syncthreads();
        if (alive) keys[running + s_warp[warp] + (uint32_t)__popc(bal & ((1u << lane) - 1u))] = key;
        running += s_total;
        __syncthreads();
    }
    uint32_t m = 1;
    while (m < running) m <<= 1;
    for (uint32_t i = running + (uint32_t)tid; i < m; i += kFinalThreads) keys[i] = ~0ull;
    __syncthreads();
    for (uint32_t k = 2; k <= m; k <<= 1)
        for (uint32_t j = k >> 1; j > 0; j >>= 1) {
            for (uint32_t i = (uint32_t)tid; i < m; i += kFinalThreads) {
                const uint32_t x = i ^ j;
                if (x > i) {
                    const unsigned long long a = keys[i], b = keys[x];
                    if ((a > b) == ((i & k) == 0u)) { keys[i] = b; keys[x] = a; }
                }
            }
            __syncthreads();
        }
    hough_peak* out = peaks + (size_t)e * max_peaks;
    const uint32_t n_out = min(running, max_peaks);
    for (uint32_t i = (uint32_t)tid; i < n_out; i += kFinalThreads) {
        const unsigned long long key = keys[i];
        hough_peak pk;
        pk.lin = (uint32_t)(key >> 32); pk.count = (uint16_t)(key & 0xffffu); pk.mask = (uint16_t)((key >> 16) & 0xffffu);
        out[i] = pk;
    }
    if (tid == 0) {
        const bool over = n_raw > cap;
        n_peaks[e] = over ? HOUGH_N_PEAKS_OVERFLOW : running;
        if (over) atomicOr(status, (uint32_t)HOUGH_ST_CANDIDATE_OVERFLOW);
        cand_n[e] = 0u;
    }
}

}  // namespace

cudaError_t plan_peaks(hough_ctx* c)
{
    PeakPlan& pp = c->peak;
    const uint64_t bins = (uint64_t)c->cfg.n_d0 * c->cfg.n_phi0 * c->cfg.n_kappa;
    pp.threads = kStencilThreads;
    pp.unit_bins = (bins % 16 == 0) ? 16 : 8;                    // n_kappa % 8 == 0 is a hough_create precondition
    cudaError_t err = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&pp.blocks_per_sm[0], peak_stencil_kernel<8>,
                                                                    kStencilThreads, 0);
    if (err != cudaSuccess) return err;
    return cudaOccupancyMaxActiveBlocksPerMultiprocessor(&pp.blocks_per_sm[1], peak_stencil_kernel<16>,
                                                         kStencilThreads, 0);
}

cudaError_t launch_peaks(hough_ctx* c, uint32_t n_events, const uint16_t* d_count, const uint16_t* d_mask,
                         uint32_t l_min, hough_peak* d_peaks, uint32_t* d_n_peaks, cudaStream_t st)
{
    if (n_events == 0) return cudaSuccess;
    const PeakPlan& pp = c->peak;
    PeakParams p;
    p.count = d_count; p.mask = d_mask; p.bitmap = c->d_bitmap; p.grpcnt = c->d_grpcnt;
    p.n_d0 = (int)c->cfg.n_d0; p.n_phi0 = (int)c->cfg.n_phi0; p.n_kappa = (int)c->cfg.n_kappa;
    p.n_events = n_events; p.l_min = l_min;
    p.bins = (uint32_t)((uint64_t)c->cfg.n_d0 * c->cfg.n_phi0 * c->cfg.n_kappa);
    // 256-bit loads need 32-byte aligned units: every event plane starts at a multiple of 32 bytes iff the
    // caller's base pointer does and bins % 16 == 0
    const int ub = (pp.unit_bins == 16 && (((uintptr_t)d_count) & 31u) == 0) ? 16 : 8;
    p.units = p.bins / (uint32_t)ub;
    p.groups = (p.units + 31u) / 32u;
    p.quads = (p.groups + kUnroll - 1) / kUnroll;
    const uint64_t total_quads = (uint64_t)n_events * p.quads;
    const uint64_t warps_wanted = total_quads;
    uint64_t nb = (warps_wanted + (kStencilThreads / 32) - 1) / (kStencilThreads / 32);
    const uint64_t cap = (uint64_t)c->sm_count * pp.blocks_per_sm[ub == 16];    // one resident wave
    if (nb > cap) nb = cap;
    if (ub == 16) peak_stencil_kernel<16><<<(unsigned)nb, kStencilThreads, 0, st>>>(p);
    else peak_stencil_kernel<8><<<(unsigned)nb, kStencilThreads, 0, st>>>(p);
    ++c->launches;
    cudaError_t err = cudaGetLastError();
    if (err != cudaSuccess) return err;
    peak_compact_kernel<<<n_events, kCompactThreads, 0, st>>>(d_count, d_mask, c->d_bitmap, c->d_grpcnt, p.bins,
                                                              p.groups, 32u * (uint32_t)ub,
                                                              c->cfg.max_peaks_per_event, d_peaks, d_n_peaks);
    ++c->launches;
    return cudaGetLastError();
}

cudaError_t launch_peaks_finalize(hough_ctx* c, uint32_t n_events, hough_peak* d_peaks, uint32_t* d_n_peaks,
                                  cudaStream_t st)
{
    if (n_events == 0) return cudaSuccess;
    const size_t smem = (size_t)kSortSmemKeys * sizeof(unsigned long long);
    cudaError_t err = cudaFuncSetAttribute(peaks_finalize_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (err != cudaSuccess) return err;
    peaks_finalize_kernel<<<n_events, kFinalThreads, smem, st>>>(c->d_cand, c->d_cand_n, c->cand_cap, c->d_sortkeys,
                                                                 c->cand_cap_pow2, c->cfg.max_peaks_per_event, d_peaks,
                                                                 d_n_peaks, c->d_status);
    ++c->launches;
    return cudaGetLastError();
}
