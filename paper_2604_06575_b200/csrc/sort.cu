// sort.cu -- step S2: stable least-significant-digit radix sort of (key, fp64 coefficient) pairs.
//
// One kernel per digit ("single pass per digit"): a block takes the next tile through an atomic ticket,
// ranks its records by digit with warp-synchronous matching (stable, insensitive to skewed digits),
// publishes the tile's per-bin counts and obtains the counts of all earlier tiles by decoupled look-back,
// then scatters keys and coefficients through shared memory so that global stores are contiguous per bin.
// The histogram of the NEXT pass's digit is accumulated on the way (keys are in registers anyway), so no
// pass ever re-reads the keys just to count.  Coefficients are opaque 64-bit payloads here.
#include "kernels.h"

namespace polylab {

template <typename K, int THREADS, int ITEMS>
struct SortSmem {
    static constexpr int TILE = THREADS * ITEMS;
    static constexpr int NW = THREADS / 32;
    static constexpr size_t stage_bytes = (size_t)TILE * sizeof(K);
    static constexpr size_t bytes = stage_bytes + (size_t)(2 * NW * kRadix + 2 * kRadix + NW + 4) * sizeof(uint32_t);
};

template <typename K, int THREADS, int ITEMS, int MINB>
__global__ void __launch_bounds__(THREADS, MINB)
sort_pass_kernel(const K* __restrict__ keys_in, const double* __restrict__ coef_in, K* __restrict__ keys_out,
                 double* __restrict__ coef_out, uint32_t n, int dpos, uint32_t dmask, int npos, uint32_t nmask,
                 int has_next, uint32_t* tile_state, uint32_t flag_partial, uint32_t flag_inclusive,
                 const uint32_t* __restrict__ hist_this, uint32_t* hist_next, uint32_t* ticket)
{
    static_assert(THREADS == kRadix, "one thread per bin");
    using S = SortSmem<K, THREADS, ITEMS>;
    constexpr int TILE = S::TILE, NW = S::NW;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    K* stage = (K*)smem_raw;
    double* stage_c = (double*)smem_raw;
    uint32_t* whist = (uint32_t*)(smem_raw + S::stage_bytes);      // [NW][256] this pass's digit, per warp
    uint32_t* whist2 = whist + NW * kRadix;                        // [NW][256] next pass's digit, per warp
    uint32_t* sm_bin_start = whist2 + NW * kRadix;                 // [256]
    uint32_t* sm_delta = sm_bin_start + kRadix;                    // [256]
    uint32_t* scratch = sm_delta + kRadix;                         // [NW + 1], then the tile id

    const unsigned tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
    if (tid == 0) scratch[NW + 2] = atomicAdd(ticket, 1u);
    for (int i = tid; i < 2 * NW * kRadix; i += THREADS) whist[i] = 0u;
    __syncthreads();
    const uint32_t tile = scratch[NW + 2];
    const uint32_t tile_base = tile * (uint32_t)TILE;
    const uint32_t tile_n = min((uint32_t)TILE, n - tile_base);

    // ---- load keys: warp w owns records [w*32*ITEMS, (w+1)*32*ITEMS) of the tile, item j of lane l is j*32+l
    const uint32_t chunk = warp * 32u * ITEMS + lane;
    K key[ITEMS];
#pragma unroll
    for (int j = 0; j < ITEMS; ++j) {
        const uint32_t li = chunk + j * 32u;
        key[j] = (li < tile_n) ? keys_in[tile_base + li] : key_max<K>();
    }

    // ---- rank within the warp, in record order (stable)
    uint32_t* my_hist = whist + warp * kRadix;
    uint32_t* my_hist2 = whist2 + warp * kRadix;
    const unsigned lt = lanemask_lt();
    uint32_t pos[ITEMS];
#pragma unroll
    for (int j = 0; j < ITEMS; ++j) {
        const bool valid = (chunk + j * 32u) < tile_n;
        const uint32_t d = key_digit(key[j], dpos, dmask);
        const unsigned m = match_digit(d, valid);
        const uint32_t prev = my_hist[d];
        uint32_t d2 = 0, prev2 = 0;
        unsigned m2 = 0;
        if (has_next) {
            d2 = key_digit(key[j], npos, nmask);
            m2 = match_digit(d2, valid);
            prev2 = my_hist2[d2];
        }
        __syncwarp();
        if (valid && (m & lt) == 0u) my_hist[d] = prev + __popc(m);
        if (has_next && valid && (m2 & lt) == 0u) my_hist2[d2] = prev2 + __popc(m2);
        __syncwarp();
        pos[j] = prev + __popc(m & lt);
    }
    __syncthreads();

    // ---- per-bin: exclusive offsets over warps, tile count, next-digit histogram, look-back publication
    const unsigned b = tid;
    uint32_t count = 0;
#pragma unroll
    for (int w = 0; w < NW; ++w) {
        const uint32_t c = whist[w * kRadix + b];
        whist[w * kRadix + b] = count;
        count += c;
    }
    uint32_t* my_state = tile_state + (size_t)tile * kRadix + b;
    st_volatile_u32(my_state, (count << 2) | (tile == 0 ? flag_inclusive : flag_partial));
    if (has_next) {
        uint32_t c2 = 0;
#pragma unroll
        for (int w = 0; w < NW; ++w) c2 += whist2[w * kRadix + b];
        if (c2) atomicAdd(&hist_next[b], c2);
    }
    uint32_t total;
    const uint32_t bin_start = block_exclusive_scan<THREADS>(count, scratch, &total);
    sm_bin_start[b] = bin_start;
    const uint32_t gbase = block_exclusive_scan<THREADS>(hist_this[b], scratch, &total);   // syncs: sm_bin_start visible

    // ---- scatter keys into shared memory at their position in the sorted tile
#pragma unroll
    for (int j = 0; j < ITEMS; ++j) {
        if ((chunk + j * 32u) < tile_n) {
            const uint32_t d = key_digit(key[j], dpos, dmask);
            pos[j] += sm_bin_start[d] + my_hist[d];
            stage[pos[j]] = key[j];
        }
    }
    // coefficients: issue the loads now, they land while the look-back runs
    double c[ITEMS];
#pragma unroll
    for (int j = 0; j < ITEMS; ++j) {
        const uint32_t li = chunk + j * 32u;
        c[j] = (li < tile_n) ? coef_in[tile_base + li] : 0.0;
    }

    // ---- decoupled look-back: number of records with digit b in all earlier tiles
    uint32_t excl = 0;
    if (tile > 0) {
        const uint32_t* p = my_state - kRadix;
        while (true) {
            const uint32_t w = ld_volatile_u32(p);
            const uint32_t f = w & 3u;
            if (f == flag_inclusive) { excl += w >> 2; break; }
            if (f == flag_partial) { excl += w >> 2; p -= kRadix; }
        }
        st_volatile_u32(my_state, ((excl + count) << 2) | flag_inclusive);
    }
    sm_delta[b] = gbase + excl - bin_start;      // destination of sorted-tile slot s with digit b: s + delta[b]
    __syncthreads();

    // ---- write keys: slot s of the sorted tile, contiguous per bin
    uint32_t dst[ITEMS];
#pragma unroll
    for (int k = 0; k < ITEMS; ++k) {
        const uint32_t s = k * THREADS + tid;
        if (s < tile_n) {
            const K kk = stage[s];
            dst[k] = s + sm_delta[key_digit(kk, dpos, dmask)];
            keys_out[dst[k]] = kk;
        }
    }
    __syncthreads();
#pragma unroll
    for (int j = 0; j < ITEMS; ++j)
        if ((chunk + j * 32u) < tile_n) stage_c[pos[j]] = c[j];
    __syncthreads();
#pragma unroll
    for (int k = 0; k < ITEMS; ++k) {
        const uint32_t s = k * THREADS + tid;
        if (s < tile_n) coef_out[dst[k]] = stage_c[s];
    }
}

template <typename K, int ITEMS, int MINB>
static int launch_sort_pass_t(const Plan& plan, int pass, int64_t n, const void* keys_in, const double* coef_in,
                              void* keys_out, double* coef_out, uint32_t* tile_state, Control* ctl, cudaStream_t stream)
{
    using S = SortSmem<K, kSortThreads, ITEMS>;
    auto kern = sort_pass_kernel<K, kSortThreads, ITEMS, MINB>;
    static bool attr_set = false;
    if (!attr_set) {
        cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)S::bytes);
        attr_set = true;
    }
    const unsigned tiles = (unsigned)((n + S::TILE - 1) / S::TILE);
    const int has_next = pass + 1 < plan.npasses;
    const int npos = has_next ? plan.digit_pos[pass + 1] : 0;
    const uint32_t nmask = has_next ? (1u << plan.digit_bits[pass + 1]) - 1u : 0u;
    const uint32_t fp = (pass & 1) ? 3u : 1u, fi = (pass & 1) ? 0u : 2u;     // flag parity: no re-zeroing between passes
    kern<<<tiles, kSortThreads, S::bytes, stream>>>((const K*)keys_in, coef_in, (K*)keys_out, coef_out, (uint32_t)n,
                                                    plan.digit_pos[pass], (1u << plan.digit_bits[pass]) - 1u, npos, nmask,
                                                    has_next, tile_state, fp, fi, ctl->hist[pass], ctl->hist[pass + 1],
                                                    &ctl->ticket[pass]);
    return 1;
}

int launch_sort_pass(const Plan& plan, int pass, int64_t n, const void* keys_in, const double* coef_in, void* keys_out,
                     double* coef_out, uint32_t* tile_state, Control* ctl, cudaStream_t stream)
{
    if (n <= 0) return 0;
    if (plan.key_bytes == 8)
        return launch_sort_pass_t<uint64_t, kSortItems64, 3>(plan, pass, n, keys_in, coef_in, keys_out, coef_out, tile_state,
                                                             ctl, stream);
    return launch_sort_pass_t<Key128, kSortItems128, 3>(plan, pass, n, keys_in, coef_in, keys_out, coef_out, tile_state, ctl,
                                                        stream);
}

}  // namespace polylab
