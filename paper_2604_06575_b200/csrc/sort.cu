// sort.cu -- step S2: stable least-significant-digit radix sort of (key, fp64 coefficient) pairs.
//
// One kernel per digit ("single pass per digit"): a block takes the next tile through an atomic ticket,
// ranks its records by digit with warp-synchronous matching (stable, insensitive to skewed digits),
// publishes the tile's per-bin counts and obtains the counts of all earlier tiles by decoupled look-back,
// then scatters keys and coefficients through shared memory so that global stores are contiguous per bin.
// The histogram of the NEXT pass's digit is accumulated on the way (keys are in registers anyway), so no
// pass ever re-reads the keys just to count.  Coefficients are opaque 64-bit payloads here.
//
// The kernel is issue-bound before it is DRAM-bound (profiles/r1a_baseline.md), so the body is written for
// few instructions per record: digits never straddle a 32-bit key word (one select, one shift, one mask),
// full tiles run a copy of the body without bounds checks, and the second warp match (for the next digit's
// histogram) is compiled out of passes that do not need it.
#include "kernels.h"

namespace polylab {

template <typename K, int THREADS, int ITEMS>
struct SortSmem {
    static constexpr int TILE = THREADS * ITEMS;
    static constexpr int NW = THREADS / 32;
    static constexpr size_t stage_bytes = (size_t)TILE * sizeof(K);
    // per-warp histograms of this digit, the block's histogram of the next digit, bin starts, deltas, scan scratch
    static constexpr size_t total_bytes = stage_bytes + (size_t)(NW * kRadix + 3 * kRadix + NW + 4) * sizeof(uint32_t);
    static constexpr size_t bytes() { return total_bytes; }
};

constexpr int kHoleyWindow = 64, kHoleyBack = 24;                      // the holey reader prefetches the descriptors of tiles blockIdx.x - 24 .. + 39
constexpr size_t kHoleyBytes = 16 + kHoleyWindow * sizeof(uint2);     // its tile descriptor + that window, in shared memory

struct PassArgs {
    const void* keys_in;
    const double* coef_in;
    void* keys_out;
    double* coef_out;
    uint32_t n;
    int dword, dshift;          // this pass's digit: 32-bit word of the key, shift inside it
    uint32_t dmask;
    int nword, nshift;          // the next pass's digit (kernels with NEXT)
    uint32_t nmask;
    uint32_t* tile_state;
    uint32_t flag_partial, flag_inclusive;
    const uint32_t* hist_this;
    uint32_t* hist_next;
    uint32_t* ticket;
    int reverse_lanes;          // POLYLAB_FLAG_DEBUG_UNSTABLE: the atomic kernel maps lane l to record 31 - l
    // Slack bins (first prefix pass without an exact histogram, api.cu): hist_this holds per-bin CAPACITIES, so the bins
    // of the output are laid out with holes.  A tile that overruns a bin raises slack_overflow (the output is void then; writes
    // are clamped to the buffer) and the last tile leaves the exact bin counts in slack_count.
    uint32_t* slack_count;      // [256] or nullptr
    uint32_t* slack_overflow;
    uint32_t last_tile;
    uint32_t slack_limit;       // last valid position of the output buffers
    // ... and the pass that READS such an output (sort_pass_holey_kernel): its tiles never cross a bin.  Tile t is the
    // slack_tiles[t].y records from physical position slack_tiles[t].x (y == 0: past the last tile), in bin order
    // (slack_tiles_kernel; at most n / TILE + 256 tiles).
    const uint2* slack_tiles;
    // S1 fused into the pass (ROWS > 0): keys are packed in registers from contiguous exponent rows of ROWS bytes
    const uint8_t* rows;
    int exp_bytes;
    int32_t* status;
    // X1 fused into the pass (ROWS == kLoadProducts): record q = i*xnb + j is the product of term i of a and term j of b
    const void* xa_keys;
    const void* xb_keys;
    const double* xa_coef;
    const double* xb_coef;
    uint32_t xnb;
};
constexpr int kLoadProducts = -1;

// Step S1 inside the radix pass: exponent row t (ROWS = 8 or 16 contiguous bytes) -> key, with the range check of
// pack.cu (an exponent above plan.bound sets `bad`).  BYTES: u8 exponents, every field 8 bits wide and unbounded, rows
// as long as the key: the key is the byte-reversed row.
template <typename K, int ROWS, bool BYTES>
__device__ __forceinline__ K pack_row_inline(const PassArgs& a, const Plan& plan, uint32_t t, bool& bad)
{
    uint32_t w[ROWS / 4];
    if (ROWS == 16) {
        const uint4 q = __ldg((const uint4*)(a.rows + (size_t)t * ROWS));
        w[0] = q.x; w[ROWS / 4 > 1 ? 1 : 0] = q.y; w[ROWS / 4 > 2 ? 2 : 0] = q.z; w[ROWS / 4 > 3 ? 3 : 0] = q.w;
    } else {
        const uint2 q = __ldg((const uint2*)(a.rows + (size_t)t * ROWS));
        w[0] = q.x; w[ROWS / 4 > 1 ? 1 : 0] = q.y;
    }
    K key;
    key_zero(key);
    if (BYTES) {
        uint64_t h[ROWS / 8];
#pragma unroll
        for (int i = 0; i < ROWS / 8; ++i)
            h[i] = ((uint64_t)__byte_perm(w[2 * i], 0u, 0x0123) << 32) | (uint64_t)__byte_perm(w[2 * i + 1], 0u, 0x0123);
        key_from_halves(key, h[0], h[ROWS / 8 - 1]);
        return key;
    }
    const int es = a.exp_bytes;
#pragma unroll
    for (int k = 0; k < ROWS; ++k) {
        if (k * es < ROWS) {
            uint32_t e;
            if (es == 4) e = w[(k < ROWS / 4) ? k : 0];
            else if (es == 2) e = (w[(k < ROWS / 2) ? (k >> 1) : 0] >> (16 * (k & 1))) & 0xffffu;
            else e = (w[k >> 2] >> (8 * (k & 3))) & 0xffu;
            // an out-of-range exponent is reported AND clamped: the digit histogram was built from the rows with the same
            // clamp (pack.cu, row_hist_kernel), and the scatter must agree with it bin for bin
            if (e > plan.bound[k]) { bad = true; e = plan.bound[k]; }
            key_or_field(key, e, plan.shift[k]);
        }
    }
    return key;
}

// RANK_ATOMIC: rank a record among the warp's records of the same digit with ONE shared-memory atomic (the old
// value of the warp's counter).  Lanes of one warp instruction that hit the same counter receive their old
// values in ascending lane order on sm_100a (measured, profiles/r1b_shared_atomics.md; not documented), which
// is what makes the pass stable; the reduce step verifies the sorted order and the call falls back to the
// ballot-matching kernel (RANK_ATOMIC = false) if it ever does not hold.
template <typename K, int THREADS, int ITEMS, bool NEXT, bool FULL, bool RANK_ATOMIC, int ROWS, bool BYTES = false, bool SLACK = false, bool HOLEY = false>
__device__ __forceinline__ void sort_tile_body(const PassArgs& a, const Plan* plan, unsigned char* smem_raw, uint32_t tile,
                                               uint32_t tile_base, uint32_t tile_n)
{
    using S = SortSmem<K, THREADS, ITEMS>;
    constexpr int NW = S::NW;
    K* stage = (K*)smem_raw;
    double* stage_c = (double*)smem_raw;
    uint32_t* whist = (uint32_t*)(smem_raw + S::stage_bytes);      // [NW][256] this pass's digit, per warp
    uint32_t* bhist2 = whist + NW * kRadix;                        // [256] next pass's digit, whole block (NEXT only)
    uint32_t* sm_bin_start = bhist2 + kRadix;                      // [256]
    uint32_t* sm_delta = sm_bin_start + kRadix;                    // [256]
    uint32_t* scratch = sm_delta + kRadix;                         // [NW + 1], then the tile id

    const K* __restrict__ keys_in = (const K*)a.keys_in;
    const double* __restrict__ coef_in = a.coef_in;
    K* __restrict__ keys_out = (K*)a.keys_out;
    double* __restrict__ coef_out = a.coef_out;
    const unsigned tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;

    // ---- load keys: warp w owns records [w*32*ITEMS, (w+1)*32*ITEMS) of the tile, item j of lane l is j*32+l
    const uint32_t chunk = warp * 32u * ITEMS + ((RANK_ATOMIC && a.reverse_lanes) ? 31u - lane : lane);
    K key[ITEMS];
    bool bad = false;
#pragma unroll
    for (int j = 0; j < ITEMS; ++j) {
        const uint32_t li = chunk + j * 32u;
        if (FULL || li < tile_n) {
            if (ROWS > 0) key[j] = pack_row_inline<K, (ROWS > 0 ? ROWS : 8), BYTES>(a, *plan, tile_base + li, bad);
            else if (ROWS == kLoadProducts) {
                // step X1 in registers: key = ka_i + kb_j (fields never carry into each other), the product is never stored
                const uint32_t q = tile_base + li, i = q / a.xnb, jj = q - i * a.xnb;
                key[j] = key_add(((const K*)a.xa_keys)[i], ((const K*)a.xb_keys)[jj]);
            } else key[j] = keys_in[tile_base + li];
        } else key[j] = key_max<K>();
    }
    if (ROWS > 0 && bad) atomicMax(a.status, (int)POLYLAB_ERR_EXPONENT_RANGE);
#define POLYLAB_DIGIT(j) ((key_word(key[j], a.dword) >> a.dshift) & a.dmask)

    // ---- rank within the warp, in record order (stable)
    uint32_t* my_hist = whist + warp * kRadix;
    uint32_t pos[ITEMS];
    if (RANK_ATOMIC) {
#pragma unroll
        for (int j = 0; j < ITEMS; ++j) {
            pos[j] = 0u;
            if (FULL || (chunk + j * 32u) < tile_n) pos[j] = atomicAdd(&my_hist[POLYLAB_DIGIT(j)], 1u);
            __syncwarp();                                   // item j's atomics are performed before item j+1's
        }
    } else {
        const unsigned lt = lanemask_lt();
#pragma unroll
        for (int j = 0; j < ITEMS; ++j) {
            const uint32_t dj = POLYLAB_DIGIT(j);
            unsigned m = match_digit_all(dj);
            bool valid = true;
            if (!FULL) {
                valid = (chunk + j * 32u) < tile_n;
                m &= __ballot_sync(kFullMask, valid);
            }
            const uint32_t prev = my_hist[dj];
            __syncwarp();
            if (valid && (m & lt) == 0u) my_hist[dj] = prev + __popc(m);
            __syncwarp();
            pos[j] = prev + __popc(m & lt);
        }
    }
    if (NEXT) {
        // histogram of the next pass's digit: plain shared-memory atomics (no order needed; Blackwell's ATOMS
        // absorbs same-address lanes, measured 2.7 SM-cycles per warp-op uniform or skewed vs 22 for a warp match)
#pragma unroll
        for (int j = 0; j < ITEMS; ++j)
            if (FULL || (chunk + j * 32u) < tile_n) atomicAdd(&bhist2[(key_word(key[j], a.nword) >> a.nshift) & a.nmask], 1u);
    }
    __syncthreads();

    // ---- per-bin: exclusive offsets over warps, tile count, next-digit histogram, look-back publication
    const unsigned b = tid;
    const bool bt = tid < (unsigned)kRadix;              // the first 256 threads own one bin each
    uint32_t count = 0;
    uint32_t* my_state = a.tile_state + (size_t)tile * kRadix + (bt ? b : 0u);
    if (bt) {
#pragma unroll
        for (int w = 0; w < NW; ++w) {
            const uint32_t c = whist[w * kRadix + b];
            whist[w * kRadix + b] = count;
            count += c;
        }
        st_volatile_u32(my_state, (count << 2) | (tile == 0 ? a.flag_inclusive : a.flag_partial));
        if (NEXT) {
            const uint32_t c2 = bhist2[b];
            if (c2) atomicAdd(&a.hist_next[b], c2);
        }
    }
    uint32_t total;
    const uint32_t bin_start = block_exclusive_scan<THREADS>(count, scratch, &total);
    if (bt) sm_bin_start[b] = bin_start;
    const uint32_t hist_b = bt ? a.hist_this[b] : 0u;
    // (slack check below: the capacity waits in shared memory, in the next-digit histogram's slot, consumed above -- a second
    // global load after the look-back would sit on every tile's critical path, a register through it spills)
    if (SLACK && bt) bhist2[b] = hist_b;
    const uint32_t gbase = block_exclusive_scan<THREADS>(hist_b, scratch, &total);   // syncs: sm_bin_start visible

    // ---- scatter keys into shared memory at their position in the sorted tile
#pragma unroll
    for (int j = 0; j < ITEMS; ++j) {
        if (FULL || (chunk + j * 32u) < tile_n) {
            const uint32_t dj = POLYLAB_DIGIT(j);
            pos[j] += sm_bin_start[dj] + my_hist[dj];
            stage[pos[j]] = key[j];
        }
    }
#undef POLYLAB_DIGIT
    // coefficients: issue the loads now, they land while the look-back runs
    double c[ITEMS];
    if constexpr (HOLEY || SLACK) {
        static_assert(ROWS != kLoadProducts, "slack bins are written by the fused-rows pass and read by the plain one");
        // HOLEY: the tile's start is re-read from the descriptor in shared memory (live through the ranking it costs 17
        // spills); the SLACK instantiation goes through the same copy because ptxas then spills 20 bytes instead of 36
        const uint32_t tb = HOLEY ? *(volatile const uint32_t*)(smem_raw + S::total_bytes) : tile_base;
#pragma unroll
        for (int j = 0; j < ITEMS; ++j) {
            const uint32_t li = chunk + j * 32u;
            c[j] = (FULL || li < tile_n) ? coef_in[tb + li] : 0.0;
        }
    } else {
#pragma unroll
        for (int j = 0; j < ITEMS; ++j) {
            const uint32_t li = chunk + j * 32u;
            if (ROWS == kLoadProducts) {
                const uint32_t q = tile_base + li, i = q / a.xnb, jj = q - i * a.xnb;
                c[j] = (FULL || li < tile_n) ? __dmul_rn(a.xa_coef[i], a.xb_coef[jj]) : 0.0;     // one IEEE multiplication, never contracted
            } else c[j] = (FULL || li < tile_n) ? coef_in[tile_base + li] : 0.0;
        }
    }

    // ---- decoupled look-back: number of records with digit b in all earlier tiles.  The walk over the predecessors
    // is the longest stall of the kernel when done one dependent load at a time (profiles/r1b), so LB states are
    // fetched per round trip and consumed in order up to the first inclusive one (or the first not yet published).
    uint32_t excl = 0;
    if (tile > 0 && bt) {
        constexpr int LB = 8;
        int64_t t = (int64_t)tile - 1;                       // nearest predecessor not consumed yet
        bool done = false;
        while (!done) {
            uint32_t w[LB];
#pragma unroll
            for (int i = 0; i < LB; ++i)
                w[i] = (t - i >= 0) ? ld_volatile_u32(a.tile_state + (size_t)(t - i) * kRadix + b) : a.flag_inclusive;
            int used = 0;
            bool open = true;                                // still consuming this window
#pragma unroll
            for (int i = 0; i < LB; ++i) {
                const uint32_t f = w[i] & 3u;
                if (open && f == a.flag_inclusive) { excl += w[i] >> 2; done = true; open = false; }
                else if (open && f == a.flag_partial) { excl += w[i] >> 2; ++used; }
                else open = false;                           // not published yet: poll again from here
            }
            t -= used;
        }
        st_volatile_u32(my_state, ((excl + count) << 2) | a.flag_inclusive);
    }
    if (bt) sm_delta[b] = gbase + excl - bin_start;      // destination of sorted-tile slot s with digit b: s + delta[b]
    if (SLACK && bt) {
        // slack bins: hist_this are capacities.  A tile that overruns one raises the flag (nothing of the call's output is
        // valid then: it re-runs with an exact histogram; the writes below stay inside the buffer by clamping); the last
        // tile's inclusive totals are the exact bin counts.
        if (excl + count > bhist2[b]) *a.slack_overflow = 1u;
        if (tile == a.last_tile) a.slack_count[b] = excl + count;
    }
    __syncthreads();

    // ---- write keys: slot s of the sorted tile, contiguous per bin
    uint32_t dst[ITEMS];
#pragma unroll
    for (int k = 0; k < ITEMS; ++k) {
        const uint32_t s = k * THREADS + tid;
        if (FULL || s < tile_n) {
            const K kk = stage[s];
            dst[k] = s + sm_delta[(key_word(kk, a.dword) >> a.dshift) & a.dmask];
            if (SLACK) dst[k] = min(dst[k], a.slack_limit);
            keys_out[dst[k]] = kk;
        }
    }
    __syncthreads();
#pragma unroll
    for (int j = 0; j < ITEMS; ++j)
        if (FULL || (chunk + j * 32u) < tile_n) stage_c[pos[j]] = c[j];
    __syncthreads();
#pragma unroll
    for (int k = 0; k < ITEMS; ++k) {
        const uint32_t s = k * THREADS + tid;
        if (FULL || s < tile_n) coef_out[dst[k]] = stage_c[s];
    }
}

template <typename K, int THREADS, int ITEMS, int MINB, bool NEXT, bool RANK_ATOMIC>
__global__ void __launch_bounds__(THREADS, MINB) sort_pass_kernel(const __grid_constant__ PassArgs a)
{
    static_assert(THREADS >= kRadix && THREADS % 32 == 0, "the first 256 threads own one bin each");
    using S = SortSmem<K, THREADS, ITEMS>;
    constexpr int TILE = S::TILE, NW = S::NW;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    uint32_t* whist = (uint32_t*)(smem_raw + S::stage_bytes);
    uint32_t* scratch = whist + NW * kRadix + 3 * kRadix;

    const unsigned tid = threadIdx.x;
    if (tid == 0) scratch[NW + 2] = atomicAdd(a.ticket, 1u);
    for (int i = tid; i < (NW + 1) * kRadix; i += THREADS) whist[i] = 0u;
    __syncthreads();
    const uint32_t tile = scratch[NW + 2];
    const uint32_t tile_base = tile * (uint32_t)TILE;
    const uint32_t tile_n = min((uint32_t)TILE, a.n - tile_base);
    if (tile_n == (uint32_t)TILE) sort_tile_body<K, THREADS, ITEMS, NEXT, true, RANK_ATOMIC, 0>(a, nullptr, smem_raw, tile, tile_base, tile_n);
    else sort_tile_body<K, THREADS, ITEMS, NEXT, false, RANK_ATOMIC, 0>(a, nullptr, smem_raw, tile, tile_base, tile_n);
}

// The same pass over an input whose bins were laid out with slack by the previous pass (see PassArgs::slack_tiles): the
// tiles are cut per bin, so a tile is one contiguous, 128-byte aligned piece of the input exactly as in sort_pass_kernel.
// Measured on 2e8 records against the plain pass (1.97 ms): compact tiling with every record mapped through the holes by a
// per-tile binary search over the bin starts 2.20 ms, by a block-wide count 2.10, with the bin tables copied to shared memory
// by every block 2.07-2.12 (a million requests for the same two dozen L2 lines); one descriptor per tile, as here: see
// profiles/r2_state.md.  The descriptors of the tiles around blockIdx.x are fetched while the ticket is in flight: tickets are
// handed out in start order, so the block's tile is nearly always among them.  The grid is sized for the worst case; blocks past the last tile leave.
template <typename K, int THREADS, int ITEMS, int MINB, bool NEXT>
__global__ void __launch_bounds__(THREADS, MINB) sort_pass_holey_kernel(const __grid_constant__ PassArgs a)
{
    using S = SortSmem<K, THREADS, ITEMS>;
    constexpr int NW = S::NW;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    uint32_t* whist = (uint32_t*)(smem_raw + S::stage_bytes);
    uint32_t* scratch = whist + NW * kRadix + 3 * kRadix;
    uint32_t* desc = (uint32_t*)(smem_raw + S::total_bytes);

    const unsigned tid = threadIdx.x;
    if (tid == 0) scratch[NW + 2] = atomicAdd(a.ticket, 1u);
    uint2* win = (uint2*)(desc + 4);
    const uint32_t w0 = max(blockIdx.x, (unsigned)kHoleyBack) - kHoleyBack;
    if (tid >= 32 && tid < 32 + kHoleyWindow) {
        const uint32_t t = w0 + (tid - 32);
        win[tid - 32] = t < gridDim.x ? __ldg(a.slack_tiles + t) : make_uint2(0u, 0u);
    }
    for (int i = tid; i < (NW + 1) * kRadix; i += THREADS) whist[i] = 0u;
    __syncthreads();
    const uint32_t tile = scratch[NW + 2];
    uint2 d;
    if (tile - w0 < (uint32_t)kHoleyWindow) {                    // (block-uniform)
        d = win[tile - w0];
        if (tid == 0) desc[0] = d.x;                             // (the body re-reads the tile's start after its first barrier)
    } else {
        if (tid == 0) {
            d = __ldg(a.slack_tiles + tile);
            desc[0] = d.x; desc[1] = d.y;
        }
        __syncthreads();
        d = make_uint2(desc[0], desc[1]);
    }
    const uint32_t tile_base = d.x, tile_n = d.y;
    if (tile_n == 0u) return;
    if (tile_n == (uint32_t)S::TILE) sort_tile_body<K, THREADS, ITEMS, NEXT, true, true, 0, false, false, true>(a, nullptr, smem_raw, tile, tile_base, tile_n);
    else sort_tile_body<K, THREADS, ITEMS, NEXT, false, true, 0, false, false, true>(a, nullptr, smem_raw, tile, tile_base, tile_n);
}

// For the holey reader: one descriptor per tile (physical start, records), the tiles cut per bin of the exact counts the
// writing pass left (bin b: ceil(count_b / tile) tiles from the exclusive prefix of the capacities); every block recomputes
// the two 256-entry prefixes.  Also sets the states of the tiles beyond the previous pass's tile count to "not published"
// (zeroed words would read as inclusive totals under the reader's flag parity).
__global__ void __launch_bounds__(kRadix) slack_tiles_kernel(const uint32_t* __restrict__ count, const uint32_t* __restrict__ cap, uint32_t tile,
                                                             uint32_t max_tiles, uint2* __restrict__ desc, uint32_t* extra_state,
                                                             uint32_t extra_words, uint32_t unpublished)
{
    __shared__ uint32_t scratch[kRadix / 32 + 2];
    __shared__ uint32_t ts[kRadix + 1], ps[kRadix], cn[kRadix];
    const unsigned b = threadIdx.x;
    uint32_t total;
    const uint32_t c = count[b];
    const uint32_t te = block_exclusive_scan<kRadix>((c + tile - 1u) / tile, scratch, &total);
    ts[b] = te; cn[b] = c;
    if (b == kRadix - 1) ts[kRadix] = total;
    __syncthreads();
    ps[b] = block_exclusive_scan<kRadix>(cap[b], scratch, &total);
    __syncthreads();
    const uint32_t t = blockIdx.x * kRadix + b;
    if (t < max_tiles) {
        uint2 d = make_uint2(0u, 0u);
        if (t < ts[kRadix]) {
            uint32_t lo = 0, hi = kRadix;                        // the LAST bin whose first tile is <= t (empty bins share their successor's)
            while (hi - lo > 1u) {
                const uint32_t mid = (lo + hi) >> 1;
                if (ts[mid] <= t) lo = mid; else hi = mid;
            }
            const uint32_t off = (t - ts[lo]) * tile;
            d.x = ps[lo] + off;
            d.y = min(tile, cn[lo] - off);
        }
        desc[t] = d;
    }
    for (uint32_t i = t; i < extra_words; i += gridDim.x * kRadix) extra_state[i] = unpublished;
}

// The same pass with S1 fused in: reads exponent rows instead of keys (first pass of the bucket path).
template <typename K, int THREADS, int ITEMS, int MINB, bool NEXT, int ROWS, bool BYTES, bool SLACK = false>
__global__ void __launch_bounds__(THREADS, MINB) sort_pass_rows_kernel(const __grid_constant__ PassArgs a, const __grid_constant__ Plan plan)
{
    using S = SortSmem<K, THREADS, ITEMS>;
    constexpr int TILE = S::TILE, NW = S::NW;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    uint32_t* whist = (uint32_t*)(smem_raw + S::stage_bytes);
    uint32_t* scratch = whist + NW * kRadix + 3 * kRadix;

    const unsigned tid = threadIdx.x;
    if (tid == 0) scratch[NW + 2] = atomicAdd(a.ticket, 1u);
    for (int i = tid; i < (NW + 1) * kRadix; i += THREADS) whist[i] = 0u;
    __syncthreads();
    const uint32_t tile = scratch[NW + 2];
    const uint32_t tile_base = tile * (uint32_t)TILE;
    const uint32_t tile_n = min((uint32_t)TILE, a.n - tile_base);
    if (tile_n == (uint32_t)TILE) sort_tile_body<K, THREADS, ITEMS, NEXT, true, true, ROWS, BYTES, SLACK>(a, &plan, smem_raw, tile, tile_base, tile_n);
    else sort_tile_body<K, THREADS, ITEMS, NEXT, false, true, ROWS, BYTES, SLACK>(a, &plan, smem_raw, tile, tile_base, tile_n);
}

template <typename K, int THREADS, int ITEMS, int MINB, bool NEXT, bool RANK_ATOMIC>
static void launch_sort_pass_k(const PassArgs& a, unsigned tiles, cudaStream_t stream)
{
    using S = SortSmem<K, THREADS, ITEMS>;
    auto kern = sort_pass_kernel<K, THREADS, ITEMS, MINB, NEXT, RANK_ATOMIC>;
    ensure_dynamic_smem(kern, (size_t)S::bytes());
    kern<<<tiles, THREADS, S::bytes(), stream>>>(a);
}

template <typename K, int THREADS, int ITEMS, int MINB>
static int launch_sort_pass_t(const Plan& plan, int pass, int next, int seq, int64_t n, const void* keys_in,
                              const double* coef_in, void* keys_out, double* coef_out, uint32_t* tile_state, Control* ctl,
                              bool safe_rank, bool debug_unstable, const ExpView* rows, const ExpandSrc* xs, cudaStream_t stream,
                              const SlackIO* slack)
{
    using S = SortSmem<K, THREADS, ITEMS>;
    const unsigned tiles = (unsigned)((n + S::TILE - 1) / S::TILE);
    const bool has_next = next >= 0;
    PassArgs a;
    a.keys_in = keys_in; a.coef_in = coef_in; a.keys_out = keys_out; a.coef_out = coef_out;
    a.n = (uint32_t)n;
    a.dword = plan.digit_pos[pass] >> 5; a.dshift = plan.digit_pos[pass] & 31; a.dmask = (1u << plan.digit_bits[pass]) - 1u;
    a.nword = has_next ? plan.digit_pos[next] >> 5 : 0;
    a.nshift = has_next ? plan.digit_pos[next] & 31 : 0;
    a.nmask = has_next ? (1u << plan.digit_bits[next]) - 1u : 0u;
    a.tile_state = tile_state;
    a.flag_partial = (seq & 1) ? 3u : 1u;                  // flag parity: no re-zeroing between passes
    a.flag_inclusive = (seq & 1) ? 0u : 2u;
    a.hist_this = ctl->hist[pass]; a.hist_next = ctl->hist[has_next ? next : kMaxPasses]; a.ticket = &ctl->ticket[seq];
    a.reverse_lanes = debug_unstable ? 1 : 0;
    a.slack_count = nullptr; a.slack_overflow = nullptr; a.last_tile = tiles - 1u; a.slack_tiles = nullptr;
    a.slack_limit = 0u;
    if (slack && slack->write) { a.slack_count = ctl->slack_count; a.slack_overflow = &ctl->slack_overflow; a.slack_limit = slack->capacity - 1u; }
    if (slack && slack->read) {
        // the previous pass left holes: prefixes of its exact counts and of its capacities, then the holey reader
        const unsigned max_tiles = tiles + kSlackExtraTiles;          // sum of ceil(count_b / TILE) <= n / TILE + 256
        slack_tiles_kernel<<<(max_tiles + kRadix - 1) / kRadix, kRadix, 0, stream>>>(ctl->slack_count, slack->cap, (uint32_t)S::TILE, max_tiles, slack->tiles,
                                                                                      tile_state + (size_t)tiles * kRadix,
                                                                                      (uint32_t)kSlackExtraTiles * kRadix, ((seq - 1) & 1) ? 3u : 1u);
        a.slack_tiles = slack->tiles;
        auto go = [&](auto kern) {
            ensure_dynamic_smem(kern, (size_t)S::bytes() + kHoleyBytes);
            kern<<<max_tiles, THREADS, S::bytes() + kHoleyBytes, stream>>>(a);
        };
        if (has_next) go(sort_pass_holey_kernel<K, THREADS, ITEMS, MINB, true>);
        else go(sort_pass_holey_kernel<K, THREADS, ITEMS, MINB, false>);
        return 2;
    }
    a.rows = nullptr; a.exp_bytes = 0; a.status = &ctl->status;
    a.xa_keys = nullptr; a.xb_keys = nullptr; a.xa_coef = nullptr; a.xb_coef = nullptr; a.xnb = 1;
    if (xs) {
        a.xa_keys = xs->ka; a.xb_keys = xs->kb; a.xa_coef = (const double*)xs->ca.p; a.xb_coef = (const double*)xs->cb.p; a.xnb = (uint32_t)xs->nb;   // fp64 here: api.cu widens fp32 operands
        auto go = [&](auto kern) {
            ensure_dynamic_smem(kern, (size_t)S::bytes());
            kern<<<tiles, THREADS, S::bytes(), stream>>>(a, plan);
        };
        if (has_next) go(sort_pass_rows_kernel<K, THREADS, ITEMS, MINB, true, kLoadProducts, false>);
        else go(sort_pass_rows_kernel<K, THREADS, ITEMS, MINB, false, kLoadProducts, false>);
        return 1;
    }
    if (rows) {
        a.rows = (const uint8_t*)rows->base; a.exp_bytes = rows->exp_bytes;
        bool fast = rows->exp_bytes == 1 && plan.nvars * rows->exp_bytes == (int)sizeof(K);
        for (int v = 0; v < plan.nvars && fast; ++v) fast = plan.width[v] == 8 && plan.bound[v] >= 255u;
        const int rb = plan.nvars * rows->exp_bytes;
        auto go = [&](auto kern) {
            ensure_dynamic_smem(kern, (size_t)S::bytes());
            kern<<<tiles, THREADS, S::bytes(), stream>>>(a, plan);
        };
        constexpr int KB = (int)sizeof(K);          // the byte-reversal path needs rows as long as the key
        if (a.slack_count && has_next) {               // slack bins: the first of two or more prefix passes (always has a next digit)
            if (fast) go(sort_pass_rows_kernel<K, THREADS, ITEMS, MINB, true, KB, true, true>);
            else if (rb == 16) go(sort_pass_rows_kernel<K, THREADS, ITEMS, MINB, true, 16, false, true>);
            else go(sort_pass_rows_kernel<K, THREADS, ITEMS, MINB, true, 8, false, true>);
            return 1;
        }
        if (fast) { if (has_next) go(sort_pass_rows_kernel<K, THREADS, ITEMS, MINB, true, KB, true>); else go(sort_pass_rows_kernel<K, THREADS, ITEMS, MINB, false, KB, true>); }
        else if (rb == 16) { if (has_next) go(sort_pass_rows_kernel<K, THREADS, ITEMS, MINB, true, 16, false>); else go(sort_pass_rows_kernel<K, THREADS, ITEMS, MINB, false, 16, false>); }
        else { if (has_next) go(sort_pass_rows_kernel<K, THREADS, ITEMS, MINB, true, 8, false>); else go(sort_pass_rows_kernel<K, THREADS, ITEMS, MINB, false, 8, false>); }
        return 1;
    }
    if (safe_rank) {
        if (has_next) launch_sort_pass_k<K, THREADS, ITEMS, MINB, true, false>(a, tiles, stream);
        else launch_sort_pass_k<K, THREADS, ITEMS, MINB, false, false>(a, tiles, stream);
    } else {
        if (has_next) launch_sort_pass_k<K, THREADS, ITEMS, MINB, true, true>(a, tiles, stream);
        else launch_sort_pass_k<K, THREADS, ITEMS, MINB, false, true>(a, tiles, stream);
    }
    return 1;
}

int launch_sort_pass(const Plan& plan, int pass, int next, int seq, int64_t n, const void* keys_in, const double* coef_in,
                     void* keys_out, double* coef_out, uint32_t* tile_state, Control* ctl, bool safe_rank,
                     bool debug_unstable, cudaStream_t stream, const ExpView* rows, const ExpandSrc* xs, const SlackIO* slack)
{
    if (n <= 0) return 0;
    if (plan.key_bytes == 8)
        return launch_sort_pass_t<uint64_t, kSortThreads64, kSortItems64, 3>(plan, pass, next, seq, n, keys_in, coef_in, keys_out, coef_out,
                                                             tile_state, ctl, safe_rank, debug_unstable, rows, xs, stream, slack);
    if (plan.key_bytes == 16)
        return launch_sort_pass_t<Key128, kSortThreads128, kSortItems128, 2>(plan, pass, next, seq, n, keys_in, coef_in, keys_out, coef_out,
                                                            tile_state, ctl, safe_rank, debug_unstable, rows, xs, stream, slack);
    return launch_sort_pass_t<Key256, kSortThreads256, kSortItems256, 2>(plan, pass, next, seq, n, keys_in, coef_in, keys_out, coef_out,
                                                        tile_state, ctl, safe_rank, debug_unstable, nullptr, xs, stream, slack);
}

}  // namespace polylab
