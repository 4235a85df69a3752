// A3 peak stencil + A4 ordered compaction (sm_100a).
//
// Definition (O-3; "looking for local maxima in the parameter space"): bin b is a peak
// iff popcount(mask[b]) >= l_min and, for every existing neighbour n in the 3x3(x3) neighbourhood (phi0
// periodic, kappa and d0 clipped), count[b] > count[n] or (count[b] == count[n] and lin(b) < lin(n)).
// Because l_min >= 1 implies count[b] >= 1, a clipped neighbour is equivalent to a neighbour with count 0.
//
// Stencil kernel.  A block owns TP phi0 rows x all kappa and marches along d0 with a ring of NSLOT count slabs
// ((TP+2) rows with the phi0 halo, dense, no padding) in shared memory.  One thread fills the ring with 1-D
// bulk async copies (cp.async.bulk ... mbarrier::complete_tx) NSLOT-3 slabs ahead, so every count byte is
// pulled from HBM once (the halo rows come from L2) with no register staging.  Each step has two dense passes:
//   pass 1  every thread reads 8 kappa bins per 128-bit shared load, rejects the vector if its packed maximum
//           is below l_min (a peak needs count >= popcount(mask) >= l_min) and otherwise appends the bins with
//           count >= l_min to a block queue;
//   pass 2  one thread per queued bin runs the 8 / 26-neighbour test (same slab first, then the previous and
//           the next slab only if some lane of the warp survived), and reads the mask plane only for bins that
//           are local maxima.
// The result is one bit per bin, written only for rows that hold a peak, plus a peak count per (d0, phi0) row.
// Compaction kernel: one block per event scans the row counts in linear-index order (block prefix sum) and
// writes the first max_peaks records; n_peaks is the true total.
#include "hough_internal.cuh"

namespace {

// ---- mbarrier / bulk-copy primitives (PTX ISA: mbarrier, cp.async.bulk) ------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar)
{
    asm volatile("{\n\t.reg .b64 st;\n\tmbarrier.arrive.shared::cta.b64 st, [%0];\n\t}" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t* bar, uint32_t bytes)
{
    asm volatile("{\n\t.reg .b64 st;\n\tmbarrier.arrive.expect_tx.shared::cta.b64 st, [%0], %1;\n\t}"
                 ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity)
{
    asm volatile(
        "{\n\t.reg .pred p;\n"
        "WAIT_%=:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra DONE_%=;\n\t"
        "bra WAIT_%=;\n"
        "DONE_%=:\n\t}"
        ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void* smem_dst, const void* gmem_src, uint32_t bytes, uint64_t* bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(smem_dst)), "l"(gmem_src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}

struct PeakParams {
    const uint16_t* count;
    const uint16_t* mask;
    uint8_t* bitmap;             // [E][ND*NPHI][NK/8], a row is only defined where rowcnt > 0
    uint16_t* rowcnt;            // [E][ND*NPHI] peaks per (d0, phi0) row (<= NK/2)
    int n_d0, n_phi0, n_kappa;
    int seg_len, n_seg, n_tiles;
    uint32_t l_min;
    int qcap;
};

// count of the bin at element offset o of a slab row, or of its left / right kappa neighbour (0 beyond the axis)
__device__ __forceinline__ uint32_t max3_row(const uint16_t* row, int k, int NK)
{
    uint32_t m = row[k];
    if (k > 0) m = max(m, (uint32_t)row[k - 1]);
    if (k < NK - 1) m = max(m, (uint32_t)row[k + 1]);
    return m;
}

template <int TP, int NSLOT, int NT>
__global__ void __launch_bounds__(NT) peak_stencil_kernel(const PeakParams p)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int NK = p.n_kappa, N = p.n_phi0, ND = p.n_d0;
    const int slab_elems = (TP + 2) * NK;
    const int row_bytes = NK / 8;                                // bitmap bytes per row
    uint16_t* slabs = reinterpret_cast<uint16_t*>(smem_raw);                                  // [NSLOT][(TP+2)*NK]
    uint32_t* queue = reinterpret_cast<uint32_t*>(smem_raw + (size_t)NSLOT * slab_elems * 2);  // [qcap]
    uint32_t* rowbits = queue + p.qcap;                                                         // [ceil(TP*NK/8 / 4)]
    const int rowbits_words = (TP * row_bytes + 7) / 8 * 2;                                     // even: keeps bars 8-aligned
    uint32_t* rowcnt_s = rowbits + rowbits_words;                                               // [TP]
    uint32_t* q_n2 = rowcnt_s + TP;                                                             // [2] alternate by step
    uint64_t* bars = reinterpret_cast<uint64_t*>(q_n2 + 2);                                     // [NSLOT]
    const int tid = threadIdx.x;

    uint32_t b = blockIdx.x;
    const int tile = b % p.n_tiles; b /= p.n_tiles;
    const int seg = b % p.n_seg;
    const uint32_t e = b / p.n_seg;
    const int ip0 = tile * TP;
    const int rows_valid = min(TP, N - ip0);                     // centre rows this block owns
    const int id_a = seg * p.seg_len, id_b = min(ND, id_a + p.seg_len);
    const int vec_per_row = NK / 8;
    const size_t ev_bins = (size_t)ND * N * NK;
    const size_t ev_rows = (size_t)ND * N;
    const uint16_t* cnt_e = p.count + (size_t)e * ev_bins;
    const uint16_t* msk_e = p.mask + (size_t)e * ev_bins;
    uint8_t* bm_e = p.bitmap + (size_t)e * ev_rows * row_bytes;
    uint16_t* rc_e = p.rowcnt + (size_t)e * ev_rows;

    if (tid == 0) {
        for (int s = 0; s < NSLOT; ++s) mbar_init(&bars[s], 1);
        q_n2[0] = 0; q_n2[1] = 0;
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    for (int i = tid; i < rowbits_words + TP; i += NT) rowbits[i] = 0;   // rowbits and rowcnt_s are contiguous
    __syncthreads();

    // slab `id` lives in slot (id - (id_a-1)) % NSLOT; its k-th use of the slot completes phase k
    auto rel_of = [&](int id) { return id - (id_a - 1); };
    auto issue_slab = [&](int id) {                              // thread 0 only
        const int rel = rel_of(id);
        uint64_t* bar = &bars[rel % NSLOT];
        if (id < 0 || id >= ND) { mbar_arrive(bar); return; }    // nothing to load: just complete the phase
        uint16_t* dst = slabs + (size_t)(rel % NSLOT) * slab_elems;
        const uint16_t* src = cnt_e + (size_t)id * N * NK;
        const int rows_needed = rows_valid + 2;                  // smem rows 0 .. rows_valid+1
        mbar_arrive_expect_tx(bar, (uint32_t)rows_needed * NK * 2);
        // smem row j holds global row (ip0 - 1 + j) mod N; merge runs of consecutive global rows
        int j = 0;
        while (j < rows_needed) {
            int gr = (ip0 - 1 + j) % N; if (gr < 0) gr += N;
            int run = min(rows_needed - j, N - gr);
            bulk_g2s(dst + (size_t)j * NK, src + (size_t)gr * NK, (uint32_t)run * NK * 2, bar);
            j += run;
        }
    };

    constexpr int AHEAD = NSLOT - 3;                             // slabs in flight beyond id+1
    if (tid == 0)
        for (int id = id_a - 1; id <= id_a + 1 + AHEAD; ++id) issue_slab(id);

    for (int id = id_a; id < id_b; ++id) {
        // slabs id-1, id, id+1 must have landed (earlier phases of these barriers completed long ago)
        if (id == id_a) {
            mbar_wait(&bars[rel_of(id - 1) % NSLOT], (rel_of(id - 1) / NSLOT) & 1);
            mbar_wait(&bars[rel_of(id) % NSLOT], (rel_of(id) / NSLOT) & 1);
        }
        mbar_wait(&bars[rel_of(id + 1) % NSLOT], (rel_of(id + 1) / NSLOT) & 1);
        const uint16_t* s_prev = slabs + (size_t)(rel_of(id - 1) % NSLOT) * slab_elems;
        const uint16_t* s_cur = slabs + (size_t)(rel_of(id) % NSLOT) * slab_elems;
        const uint16_t* s_next = slabs + (size_t)(rel_of(id + 1) % NSLOT) * slab_elems;
        const bool has_prev = id > 0, has_next = id + 1 < ND;
        uint32_t* q_n = q_n2 + (id & 1);                         // reset two steps before its next use

        // ---- pass 1: queue the bins with count >= l_min ----
        const int n_vec = rows_valid * vec_per_row;
        for (int t = tid; t < n_vec; t += NT) {
            const int o = NK + t * 8;                            // element offset in the slab (row j+1 = centre row j)
            const uint4 c8 = *reinterpret_cast<const uint4*>(s_cur + o);
            const uint32_t m2 = __vmaxu2(__vmaxu2(c8.x, c8.y), __vmaxu2(c8.z, c8.w));
            if (max(m2 & 0xffffu, m2 >> 16) >= p.l_min) {
                const uint32_t w[4] = {c8.x, c8.y, c8.z, c8.w};
#pragma unroll
                for (int q = 0; q < 8; ++q) {
                    const uint32_t c = (w[q >> 1] >> ((q & 1) * 16)) & 0xffffu;
                    if (c >= p.l_min) {
                        const uint32_t slot = atomicAdd(q_n, 1u);
                        if (slot < (uint32_t)p.qcap) queue[slot] = (uint32_t)(o + q);
                    }
                }
            }
        }
        __syncthreads();
        const uint32_t n_q = *q_n;
        const bool overflow = n_q > (uint32_t)p.qcap;            // stress case: walk every bin instead of the queue
        const uint32_t n_items = overflow ? (uint32_t)(rows_valid * NK) : n_q;

        // ---- pass 2: full neighbourhood test of the queued bins ----
        for (uint32_t base = 0; base < n_items; base += NT) {
            const uint32_t t = base + tid;
            bool ok = false;
            int o = 0, k = 0, j = 0;
            uint32_t c = 0;
            if (t < n_items) {
                o = overflow ? (int)(NK + t) : (int)queue[t];
                j = o / NK - 1; k = o - (j + 1) * NK;
                c = s_cur[o];
                ok = c >= p.l_min;
            }
            if (ok) {
                const int ip = ip0 + j;
                // neighbours with a smaller linear index must be strictly smaller, the others may tie
                const uint32_t left = (k > 0) ? (uint32_t)s_cur[o - 1] : 0u;
                const uint32_t right = (k < NK - 1) ? (uint32_t)s_cur[o + 1] : 0u;
                ok = (left < c) && (right <= c);
                if (ok) {
                    const uint32_t up = max3_row(s_cur + o - k - NK, k, NK), dn = max3_row(s_cur + o - k + NK, k, NK);
                    ok = ((ip == 0) ? (up <= c) : (up < c)) &&           // row ip-1 wraps to NPHI-1 > ip
                         ((ip == N - 1) ? (dn < c) : (dn <= c));         // row ip+1 wraps to 0 < ip
                }
            }
            if (__any_sync(0xffffffffu, ok)) {
                if (ok && has_prev) {
                    const uint16_t* r0 = s_prev + o - k;
                    const uint32_t m = max(max(max3_row(r0 - NK, k, NK), max3_row(r0, k, NK)), max3_row(r0 + NK, k, NK));
                    ok = m < c;
                }
                if (ok && has_next) {
                    const uint16_t* r0 = s_next + o - k;
                    const uint32_t m = max(max(max3_row(r0 - NK, k, NK), max3_row(r0, k, NK)), max3_row(r0 + NK, k, NK));
                    ok = m <= c;
                }
                if (ok) {
                    const size_t lin = ((size_t)id * N + (ip0 + j)) * NK + k;
                    if ((uint32_t)__popc((uint32_t)__ldg(msk_e + lin)) >= p.l_min) {
                        const int byte = j * row_bytes + (k >> 3);
                        atomicOr(&rowbits[byte >> 2], (1u << (k & 7)) << ((byte & 3) * 8));
                        atomicAdd(&rowcnt_s[j], 1u);
                    }
                }
            }
        }
        __syncthreads();                                         // slab id-1 is free; rowbits / rowcnt_s complete

        if (tid == 0) {
            issue_slab(id + 2 + AHEAD);
            *q_n = 0;
        }
        // ---- write the row counts, and the bitmap rows that hold a peak ----
        const size_t row0 = (size_t)id * N + ip0;
        if (tid < rows_valid) rc_e[row0 + tid] = (uint16_t)rowcnt_s[tid];
        bool dirty = false;
        for (int j = 0; j < rows_valid; ++j) {
            if (rowcnt_s[j] == 0) continue;                      // block-uniform
            dirty = true;
            const uint8_t* srcb = reinterpret_cast<const uint8_t*>(rowbits) + (size_t)j * row_bytes;
            uint8_t* dstb = bm_e + (row0 + j) * row_bytes;
            for (int i = tid; i < row_bytes; i += NT) dstb[i] = srcb[i];
        }
        if (dirty) {                                             // block-uniform
            __syncthreads();
            for (int i = tid; i < rowbits_words + TP; i += NT) rowbits[i] = 0;
            // ordered before the next pass 2 by the next step's barrier after pass 1
        }
    }
    // drain the copies still in flight before the block (and its shared memory) goes away
    if (tid == 0)
        for (int id = id_b + 1; id <= id_b + 1 + AHEAD; ++id) mbar_wait(&bars[rel_of(id) % NSLOT], (rel_of(id) / NSLOT) & 1);
}

// ---- A4: ordered compaction from the row counts + bitmap rows ----------------------------------------------

__global__ void __launch_bounds__(1024) peak_compact_kernel(const uint16_t* __restrict__ count,
                                                            const uint16_t* __restrict__ mask,
                                                            const uint8_t* __restrict__ bitmap,
                                                            const uint16_t* __restrict__ rowcnt, int n_rows,
                                                            int n_kappa, uint32_t max_peaks,
                                                            hough_peak* __restrict__ peaks,
                                                            uint32_t* __restrict__ n_peaks)
{
    __shared__ uint32_t s_warp[32];
    __shared__ uint32_t s_total;
    const uint32_t e = blockIdx.x;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int row_bytes = n_kappa / 8;
    const size_t ev_bins = (size_t)n_rows * n_kappa;
    const uint8_t* bm = bitmap + (size_t)e * n_rows * row_bytes;
    const uint16_t* rc = rowcnt + (size_t)e * n_rows;
    const uint16_t* cnt_e = count + (size_t)e * ev_bins;
    const uint16_t* msk_e = mask + (size_t)e * ev_bins;
    hough_peak* out = peaks + (size_t)e * max_peaks;
    uint32_t running = 0;
    for (int base = 0; base < n_rows; base += 1024) {
        const int row = base + tid;
        const uint32_t c = (row < n_rows) ? (uint32_t)rc[row] : 0u;
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
            const uint8_t* rp = bm + (size_t)row * row_bytes;
            for (int i = 0; i < row_bytes && pos < max_peaks; ++i) {
                uint32_t byte = rp[i];
                while (byte && pos < max_peaks) {
                    const int q = __ffs(byte) - 1;
                    byte &= byte - 1;
                    const size_t lin = (size_t)row * n_kappa + i * 8 + q;
                    hough_peak pk;
                    pk.lin = (uint32_t)lin; pk.count = cnt_e[lin]; pk.mask = msk_e[lin];
                    out[pos++] = pk;
                }
            }
        }
        running += s_total;
        __syncthreads();
    }
    if (tid == 0) n_peaks[e] = running;
}

constexpr int kSlots = 5;
constexpr int kStencilThreads = 256;

size_t stencil_smem_bytes(int tp, int nk, int qcap)
{
    const size_t slabs = (size_t)kSlots * (tp + 2) * nk * 2;
    const size_t rowbits_words = ((size_t)tp * (nk / 8) + 7) / 8 * 2;
    return slabs + (size_t)qcap * 4 + rowbits_words * 4 + (size_t)tp * 4 + 8 + (size_t)kSlots * 8;
}

template <int TP>
cudaError_t launch_stencil(const PeakParams& p, uint32_t nb, size_t smem, cudaStream_t st)
{
    auto kern = peak_stencil_kernel<TP, kSlots, kStencilThreads>;
    cudaError_t err = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (err != cudaSuccess) return err;
    kern<<<nb, kStencilThreads, smem, st>>>(p);
    return cudaGetLastError();
}

}  // namespace

cudaError_t plan_peaks(hough_ctx* c)
{
    PeakPlan& pp = c->peak;
    const int nk = (int)c->cfg.n_kappa;
    pp.threads = kStencilThreads;
    // largest tile height whose ring fits twice on an SM (else once)
    const int cand[4] = {16, 8, 4, 2};
    pp.tp = 0;
    for (int pass = 0; pass < 2 && pp.tp == 0; ++pass)
        for (int i = 0; i < 4; ++i) {
            const int qcap = 2 * nk > 2048 ? 2048 : 2 * nk;
            const size_t s = stencil_smem_bytes(cand[i], nk, qcap);
            if (s <= (pass == 0 ? 112u * 1024u : 226u * 1024u)) { pp.tp = cand[i]; pp.qcap = qcap; pp.smem_bytes = s; break; }
        }
    if (pp.tp == 0) return cudaErrorInvalidConfiguration;
    pp.n_tiles = (int)((c->cfg.n_phi0 + pp.tp - 1) / pp.tp);
    return cudaSuccess;
}

cudaError_t launch_peaks(hough_ctx* c, uint32_t n_events, const uint16_t* d_count, const uint16_t* d_mask,
                         uint32_t l_min, hough_peak* d_peaks, uint32_t* d_n_peaks, cudaStream_t st)
{
    if (n_events == 0) return cudaSuccess;
    const PeakPlan& pp = c->peak;
    PeakParams p;
    p.count = d_count; p.mask = d_mask; p.bitmap = c->d_bitmap; p.rowcnt = c->d_rowcnt;
    p.n_d0 = (int)c->cfg.n_d0; p.n_phi0 = (int)c->cfg.n_phi0; p.n_kappa = (int)c->cfg.n_kappa;
    p.n_tiles = pp.n_tiles; p.l_min = l_min; p.qcap = pp.qcap;
    // split d0 into segments only when there are too few blocks to fill the machine
    int n_seg = 1;
    const uint64_t base_blocks = (uint64_t)n_events * pp.n_tiles;
    const uint64_t want = (uint64_t)c->sm_count * 4;
    if (base_blocks < want && p.n_d0 >= 8) {
        n_seg = (int)((want + base_blocks - 1) / base_blocks);
        if (n_seg > p.n_d0 / 4) n_seg = p.n_d0 / 4;
        if (n_seg < 1) n_seg = 1;
    }
    p.seg_len = (p.n_d0 + n_seg - 1) / n_seg;
    p.n_seg = (p.n_d0 + p.seg_len - 1) / p.seg_len;
    const uint64_t nb = base_blocks * p.n_seg;
    if (nb > 0x7fffffffull) return cudaErrorInvalidConfiguration;
    cudaError_t err;
    switch (pp.tp) {
        case 16: err = launch_stencil<16>(p, (uint32_t)nb, pp.smem_bytes, st); break;
        case 8: err = launch_stencil<8>(p, (uint32_t)nb, pp.smem_bytes, st); break;
        case 4: err = launch_stencil<4>(p, (uint32_t)nb, pp.smem_bytes, st); break;
        default: err = launch_stencil<2>(p, (uint32_t)nb, pp.smem_bytes, st); break;
    }
    ++c->launches;
    if (err != cudaSuccess) return err;
    peak_compact_kernel<<<n_events, 1024, 0, st>>>(d_count, d_mask, c->d_bitmap, c->d_rowcnt, p.n_d0 * p.n_phi0,
                                                   p.n_kappa, c->cfg.max_peaks_per_event, d_peaks, d_n_peaks);
    ++c->launches;
    return cudaGetLastError();
}
