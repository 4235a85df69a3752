// A3 peak stencil + A4 ordered compaction (sm_100a).
//
// Definition (O-3; "looking for local maxima in the parameter space"): bin b is a peak
// iff popcount(mask[b]) >= l_min and, for every existing neighbour n in the 3x3(x3) neighbourhood (phi0
// periodic, kappa and d0 clipped), count[b] > count[n] or (count[b] == count[n] and lin(b) < lin(n)).
// Because l_min >= 1 implies count[b] >= 1, a clipped neighbour is equivalent to a neighbour with count 0,
// so halos outside the grid are zero-filled.
//
// Stencil kernel: a block owns TP phi0 rows x all kappa and marches along d0, keeping a ring of NSLOT count
// slabs ((TP+2) rows with halo) in shared memory, filled by cp.async NSLOT-3 slabs ahead; every count byte is
// read from HBM once (plus the phi0 halo rows, which the neighbouring block has just pulled into L2).  Each
// thread tests 8 kappa bins (one 128-bit shared load) with a packed-max quick reject; the mask plane is only
// touched for bins that already are local maxima.  The result is one bit per bin (a byte per 8 bins).
// Compaction kernel: one block per event scans the bitmap in linear-index order (popcount per row, block
// prefix sum) and writes the first max_peaks records; n_peaks is the true total.
#include "hough_internal.cuh"

namespace {

__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gmem_src)
{
    const unsigned s = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(s), "l"(gmem_src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N) : "memory"); }

struct PeakParams {
    const uint16_t* count;
    const uint16_t* mask;
    uint8_t* bitmap;
    int n_d0, n_phi0, n_kappa;
    int seg_len, n_seg, n_tiles;
    uint32_t l_min;
};

__device__ __forceinline__ uint32_t max3_u16(const uint16_t* p)      // max of p[-1], p[0], p[1]
{
    return max(max((uint32_t)p[-1], (uint32_t)p[0]), (uint32_t)p[1]);
}

template <int TP, int NSLOT, int NT>
__global__ void __launch_bounds__(NT) peak_stencil_kernel(const PeakParams p)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int NK = p.n_kappa, N = p.n_phi0, ND = p.n_d0;
    const int pitch = NK + 16;                                   // u16 elements; data at [8, 8+NK)
    const int slab_elems = (TP + 2) * pitch;
    uint16_t* slabs = reinterpret_cast<uint16_t*>(smem_raw);
    const int tid = threadIdx.x;

    uint32_t b = blockIdx.x;
    const int tile = b % p.n_tiles; b /= p.n_tiles;
    const int seg = b % p.n_seg;
    const uint32_t e = b / p.n_seg;
    const int ip0 = tile * TP;
    const int id_a = seg * p.seg_len, id_b = min(ND, id_a + p.seg_len);
    const int vec_per_row = NK / 8;
    const size_t ev_bins = (size_t)ND * N * NK;
    const uint16_t* cnt_e = p.count + (size_t)e * ev_bins;
    const uint16_t* msk_e = p.mask + (size_t)e * ev_bins;
    uint8_t* bm_e = p.bitmap + (size_t)e * (ev_bins / 8);

    // zero the kappa pads of every slot once (loads never touch them)
    for (int i = tid; i < NSLOT * (TP + 2) * 16; i += NT) {
        const int row = i / 16, c = i % 16;
        slabs[(size_t)row * pitch + (c < 8 ? c : NK + c)] = 0;
    }

    auto slot_of = [&](int id) { return ((id % NSLOT) + NSLOT) % NSLOT; };
    auto load_slab = [&](int id) {                               // async fill (or zero fill) of slab `id`
        uint16_t* dst = slabs + (size_t)slot_of(id) * slab_elems;
        const int nvec = (TP + 2) * vec_per_row;
        if (id < 0 || id >= ND) {
            for (int i = tid; i < nvec; i += NT) {
                const int row = i / vec_per_row, v = i % vec_per_row;
                *reinterpret_cast<uint4*>(dst + (size_t)row * pitch + 8 + v * 8) = make_uint4(0, 0, 0, 0);
            }
        } else {
            const uint16_t* src = cnt_e + (size_t)id * N * NK;
            for (int i = tid; i < nvec; i += NT) {
                const int row = i / vec_per_row, v = i % vec_per_row;
                int ip = ip0 - 1 + row;
                ip %= N; if (ip < 0) ip += N;                    // phi0 periodic
                cp_async16(dst + (size_t)row * pitch + 8 + v * 8, src + (size_t)ip * NK + v * 8);
            }
        }
    };

    constexpr int AHEAD = NSLOT - 3;                             // slabs in flight beyond id+1 (ring of AHEAD+3)
    for (int id = id_a - 1; id <= id_a + 1 + AHEAD; ++id) { load_slab(id); cp_async_commit(); }

    for (int id = id_a; id < id_b; ++id) {
        cp_async_wait<AHEAD>();                                  // slabs up to id+1 have landed
        __syncthreads();
        const uint16_t* s_prev = slabs + (size_t)slot_of(id - 1) * slab_elems;
        const uint16_t* s_cur = slabs + (size_t)slot_of(id) * slab_elems;
        const uint16_t* s_next = slabs + (size_t)slot_of(id + 1) * slab_elems;
        for (int t = tid; t < TP * vec_per_row; t += NT) {
            const int j = t / vec_per_row, v = t % vec_per_row;
            const int ip = ip0 + j;
            if (ip >= N) break;
            const size_t row_off = (size_t)(j + 1) * pitch + 8 + v * 8;
            const uint4 c8 = *reinterpret_cast<const uint4*>(s_cur + row_off);
            uint32_t bits = 0;
            // quick reject: a peak needs count >= popcount(mask) >= l_min
            const uint32_t m2 = __vmaxu2(__vmaxu2(c8.x, c8.y), __vmaxu2(c8.z, c8.w));
            if (max(m2 & 0xffffu, m2 >> 16) >= p.l_min) {
                const uint32_t w[4] = {c8.x, c8.y, c8.z, c8.w};
#pragma unroll
                for (int q = 0; q < 8; ++q) {
                    const uint32_t c = (w[q >> 1] >> ((q & 1) * 16)) & 0xffffu;
                    if (c < p.l_min) continue;
                    const size_t o = row_off + q;
                    // neighbours with a smaller linear index must be strictly smaller, the others may tie
                    const uint32_t up = max3_u16(s_cur + o - pitch), dn = max3_u16(s_cur + o + pitch);
                    uint32_t prev = max(max(max3_u16(s_prev + o - pitch), max3_u16(s_prev + o)), max3_u16(s_prev + o + pitch));
                    uint32_t next = max(max(max3_u16(s_next + o - pitch), max3_u16(s_next + o)), max3_u16(s_next + o + pitch));
                    bool ok = (prev < c) && (next <= c) && ((uint32_t)s_cur[o - 1] < c) && ((uint32_t)s_cur[o + 1] <= c);
                    ok = ok && ((ip == 0 && N > 1) ? (up <= c) : (up < c));          // row ip-1 wraps to NPHI-1 > ip
                    ok = ok && ((ip == N - 1 && N > 1) ? (dn < c) : (dn <= c));      // row ip+1 wraps to 0 < ip
                    if (ok) {
                        const size_t lin = ((size_t)id * N + ip) * NK + v * 8 + q;
                        if ((uint32_t)__popc((uint32_t)__ldg(msk_e + lin)) >= p.l_min) bits |= 1u << q;
                    }
                }
            }
            bm_e[((size_t)id * N + ip) * vec_per_row + v] = (uint8_t)bits;
        }
        __syncthreads();                                         // slot of slab id-1 is free again
        load_slab(id + 2 + AHEAD);
        cp_async_commit();
    }
    cp_async_wait<0>();
}

// ---- A4: ordered compaction from the bitmap --------------------------------------------------------

__global__ void __launch_bounds__(1024) peak_compact_kernel(const uint16_t* __restrict__ count,
                                                            const uint16_t* __restrict__ mask,
                                                            const uint8_t* __restrict__ bitmap, int n_rows, int n_kappa,
                                                            uint32_t max_peaks, hough_peak* __restrict__ peaks,
                                                            uint32_t* __restrict__ n_peaks)
{
    __shared__ uint32_t s_warp[32];
    __shared__ uint32_t s_total;
    const uint32_t e = blockIdx.x;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int row_bytes = n_kappa / 8;
    const size_t ev_bins = (size_t)n_rows * n_kappa;
    const uint8_t* bm = bitmap + (size_t)e * (ev_bins / 8);
    const uint16_t* cnt_e = count + (size_t)e * ev_bins;
    const uint16_t* msk_e = mask + (size_t)e * ev_bins;
    hough_peak* out = peaks + (size_t)e * max_peaks;
    uint32_t running = 0;
    for (int base = 0; base < n_rows; base += 1024) {
        const int row = base + tid;
        uint32_t c = 0;
        const uint8_t* rp = bm + (size_t)row * row_bytes;
        if (row < n_rows) {
            if ((row_bytes & 15) == 0) {
                for (int i = 0; i < row_bytes; i += 16) {
                    const uint4 w = __ldg(reinterpret_cast<const uint4*>(rp + i));
                    c += __popc(w.x) + __popc(w.y) + __popc(w.z) + __popc(w.w);
                }
            } else {
                for (int i = 0; i < row_bytes; ++i) c += __popc((uint32_t)rp[i]);
            }
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

template <int TP, int NSLOT>
cudaError_t launch_stencil(const PeakParams& p, uint32_t nb, size_t smem, cudaStream_t st)
{
    auto kern = peak_stencil_kernel<TP, NSLOT, 256>;
    cudaError_t err = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (err != cudaSuccess) return err;
    kern<<<nb, 256, smem, st>>>(p);
    return cudaGetLastError();
}

constexpr int kSlots = 5;

}  // namespace

cudaError_t plan_peaks(hough_ctx* c)
{
    PeakPlan& pp = c->peak;
    const size_t pitch_b = ((size_t)c->cfg.n_kappa + 16) * 2;
    pp.threads = 256;
    // largest tile height whose ring fits twice on an SM
    const int cand[3] = {16, 8, 4};
    pp.tp = 0;
    for (int i = 0; i < 3; ++i) {
        const size_t s = (size_t)kSlots * (cand[i] + 2) * pitch_b;
        if (s <= 110 * 1024 || (i == 2 && s <= 227 * 1024)) { pp.tp = cand[i]; pp.smem_bytes = s; break; }
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
    p.count = d_count; p.mask = d_mask; p.bitmap = c->d_bitmap;
    p.n_d0 = (int)c->cfg.n_d0; p.n_phi0 = (int)c->cfg.n_phi0; p.n_kappa = (int)c->cfg.n_kappa;
    p.n_tiles = pp.n_tiles; p.l_min = l_min;
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
        case 16: err = launch_stencil<16, kSlots>(p, (uint32_t)nb, pp.smem_bytes, st); break;
        case 8: err = launch_stencil<8, kSlots>(p, (uint32_t)nb, pp.smem_bytes, st); break;
        default: err = launch_stencil<4, kSlots>(p, (uint32_t)nb, pp.smem_bytes, st); break;
    }
    ++c->launches;
    if (err != cudaSuccess) return err;
    peak_compact_kernel<<<n_events, 1024, 0, st>>>(d_count, d_mask, c->d_bitmap, p.n_d0 * p.n_phi0, p.n_kappa,
                                                   c->cfg.max_peaks_per_event, d_peaks, d_n_peaks);
    ++c->launches;
    return cudaGetLastError();
}
