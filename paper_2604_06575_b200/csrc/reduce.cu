// reduce.cu -- steps S3 (segmented sum of like terms), S4 (prune) and S5 (unpack).
//
// S3: after the sort equal monomials are adjacent; "merges repeated monomials" is a
// reduce-by-key: one output (key, sum) per run of equal keys.  S4/S5: "removes coefficients below a
// user-chosen tolerance" (reading A2: keep iff |s| > tol), order-preserving compaction and
// decoding of the surviving keys back to exponent rows.
//
// Summation order (reading A6): inside a thread left to right over its consecutive records, across
// threads by a fixed shuffle tree, across tiles left to right in the fix-up kernel -- a fixed function of
// n, never of timing, so results are bit-reproducible run to run.
#include "kernels.h"

namespace polylab {

// ----------------------------------------------------------------------------------------------- S3

template <typename K, int THREADS, int ITEMS>
__global__ void __launch_bounds__(THREADS)
reduce_kernel(const K* __restrict__ keys, CoefIn coefs, uint32_t n, K* __restrict__ ukeys,
              double* __restrict__ usums, ReduceScratch sc, Control* ctl)
{
    constexpr int TILE = THREADS * ITEMS, NW = THREADS / 32;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    K* skeys = (K*)smem_raw;
    double* scoef = (double*)(smem_raw + (size_t)TILE * sizeof(K));
    __shared__ uint32_t scratch[NW + 2];
    __shared__ uint32_t sm_tile, sm_hb;
    __shared__ uint32_t wagg_f[NW];
    __shared__ double wagg_v[NW];

    const unsigned tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
    if (tid == 0) sm_tile = atomicAdd(&ctl->ticket[kTicketReduce], 1u);
    __syncthreads();
    const uint32_t tile = sm_tile;
    const uint32_t tile_base = tile * (uint32_t)TILE;
    const uint32_t tile_n = min((uint32_t)TILE, n - tile_base);

#pragma unroll
    for (int k = 0; k < ITEMS; ++k) {
        const uint32_t s = k * THREADS + tid;
        if (s < tile_n) {
            skeys[s] = keys[tile_base + s];
            scoef[s] = coefs[tile_base + s];
        }
    }
    __syncthreads();

    const uint32_t first = tid * ITEMS;
    // key of the record before this thread's first one (if any)
    K kprev0;
    key_zero(kprev0);
    bool has_prev = false;
    if (first < tile_n) {
        if (first > 0) { kprev0 = skeys[first - 1]; has_prev = true; }
        else if (tile_base > 0) { kprev0 = keys[tile_base - 1]; has_prev = true; }
    }

    // ---- phase 1: heads, sum before the first head, sum after the last head
    uint32_t nh = 0;
    double acc = 0.0;
    bool descending = false;                         // a key below its predecessor: the sort failed (see sort.cu)
    {
        K kp = kprev0;
        bool hp = has_prev;
#pragma unroll
        for (int j = 0; j < ITEMS; ++j) {
            if (first + j < tile_n) {
                const K kk = skeys[first + j];
                const bool head = !hp || !key_eq(kk, kp);
                descending |= hp && key_lt(kk, kp);
                if (head) { ++nh; acc = scoef[first + j]; }
                else acc = __dadd_rn(acc, scoef[first + j]);
                kp = kk;
                hp = true;
            }
        }
    }
    if (descending) ctl->unsorted = 1u;
    uint32_t H;
    const uint32_t hb = block_exclusive_scan<THREADS>(nh, scratch, &H);

    // ---- segmented scan of (has head, sum since last head) across the block -> carry into each thread
    SegPair incl;
    incl.f = nh > 0;
    incl.v = acc;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        SegPair l;
        l.f = __shfl_up_sync(kFullMask, incl.f, o);
        l.v = __shfl_up_sync(kFullMask, incl.v, o);
        if (lane >= (unsigned)o) incl = seg_combine(l, incl);
    }
    if (lane == 31) { wagg_f[warp] = incl.f; wagg_v[warp] = incl.v; }
    SegPair carry;                                   // exclusive within the warp
    carry.f = __shfl_up_sync(kFullMask, incl.f, 1);
    carry.v = __shfl_up_sync(kFullMask, incl.v, 1);
    if (lane == 0) { carry.f = 0; carry.v = 0.0; }
    __syncthreads();
    {
        SegPair wp;
        wp.f = 0;
        wp.v = 0.0;
        for (unsigned w = 0; w < warp; ++w) {
            SegPair a;
            a.f = wagg_f[w];
            a.v = wagg_v[w];
            wp = seg_combine(wp, a);
        }
        carry = seg_combine(wp, carry);
        incl = seg_combine(wp, incl);
    }

    // ---- look-back: heads in all earlier tiles
    if (warp == 0) {
        const uint32_t r = warp_lookback_u32(sc.tile_state, tile, H);
        if (lane == 0) sm_hb = r;
    }
    __syncthreads();
    const uint32_t HB = sm_hb;

    // ---- phase 2: write every segment that ends inside this thread
    {
        const uint32_t slot0 = HB + hb;              // output index of this thread's first head
        uint32_t nh2 = 0;
        double a2 = 0.0;
        K kp = kprev0;
        bool hp = has_prev;
#pragma unroll
        for (int j = 0; j < ITEMS; ++j) {
            if (first + j < tile_n) {
                const K kk = skeys[first + j];
                const bool head = !hp || !key_eq(kk, kp);
                if (head) {
                    if (nh2 == 0) {
                        // closes the segment carried in from earlier threads (or earlier tiles)
                        const double total = __dadd_rn(carry.v, a2);
                        if (carry.f) { usums[slot0 - 1] = total; ukeys[slot0 - 1] = kp; }
                        else if (hp) sc.tile_frag[tile] = total;          // its head lies in an earlier tile
                    } else {
                        usums[slot0 + nh2 - 1] = a2;
                        ukeys[slot0 + nh2 - 1] = kp;
                    }
                    ++nh2;
                    a2 = scoef[first + j];
                } else a2 = __dadd_rn(a2, scoef[first + j]);
                kp = kk;
                hp = true;
            }
        }
    }
    if (tid == THREADS - 1) {
        // the segment still open at the end of the tile
        if (incl.f) { usums[HB + H - 1] = incl.v; ukeys[HB + H - 1] = skeys[tile_n - 1]; }
        else sc.tile_frag[tile] = incl.v;                                 // no head in the whole tile
        sc.tile_heads[tile] = H;
        sc.tile_hb[tile] = HB;
        if (tile_base + tile_n == n) ctl->distinct = HB + H;
    }
    if (tid == 0) {
        // does the tile start in the middle of a segment?
        sc.tile_cont[tile] = (tile_base > 0 && key_eq(skeys[0], kprev0)) ? 1 : 0;
    }
}

// Adds the leading fragments of later tiles to segments that cross tile boundaries.  One warp per tile that is the FIRST
// continuation of a segment: the fragments of the following tiles are taken 32 at a time, summed by a fixed butterfly
// (every lane ends with the same value) and added chunk by chunk -- a fixed function of the layout, and the error of a run
// of n equal keys grows as (n / (32 * tile) + 5 + ...) * 2^-53 * A_m instead of n / tile (a run of 2^30 records stays far
// inside the 1e-12 * A_m bound).
__global__ void __launch_bounds__(256) reduce_fixup_kernel(uint32_t ntiles, double* __restrict__ usums, ReduceScratch sc)
{
    const uint32_t t = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const unsigned lane = lane_id();
    if (t == 0 || t >= ntiles) return;
    if (!sc.tile_cont[t] || sc.tile_heads[t - 1] == 0) return;      // not the first continuation of a segment (warp-uniform)
    const uint32_t slot = sc.tile_hb[t] - 1;
    double s = usums[slot];
    uint32_t u0 = t;
    while (true) {
        // lane l looks at tile u0 + l: it belongs to the chain iff every tile in (u0, u0 + l] continues the segment and no
        // tile in [u0, u0 + l) holds a head (a tile with a head ends the chain, its own fragment included)
        const uint32_t u = u0 + lane;
        const bool in = u < ntiles;
        const bool cont = in && (u == t || sc.tile_cont[u]);
        const bool head = in && sc.tile_heads[u] > 0;
        const unsigned stop_before = __ballot_sync(kFullMask, !cont);       // first lane that is not part of the chain
        const unsigned stop_after = __ballot_sync(kFullMask, head);         // first lane that ends it
        int last = 31;                                                       // last lane whose fragment is added
        if (stop_before) last = min(last, __ffs(stop_before) - 2);
        if (stop_after) last = min(last, __ffs(stop_after) - 1);
        double f = ((int)lane <= last) ? sc.tile_frag[u] : 0.0;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) f = __dadd_rn(f, __shfl_xor_sync(kFullMask, f, o));
        if (last >= 0) s = __dadd_rn(s, f);
        if (stop_before | stop_after) break;                                 // the chain ended in this window (maybe in its last lane)
        u0 += 32u;
    }
    if (lane == 0) usums[slot] = s;
}

template <typename K>
static int launch_reduce_t(int64_t n, const void* keys, CoefIn coefs, void* ukeys, double* usums,
                           const ReduceScratch& sc, Control* ctl, cudaStream_t stream)
{
    constexpr int TILE = kReduceTile;
    const size_t smem = (size_t)TILE * (sizeof(K) + sizeof(double));
    auto kern = reduce_kernel<K, kReduceThreads, kReduceItems>;
    ensure_dynamic_smem(kern, (size_t)smem);
    const unsigned tiles = (unsigned)((n + TILE - 1) / TILE);
    kern<<<tiles, kReduceThreads, smem, stream>>>((const K*)keys, coefs, (uint32_t)n, (K*)ukeys, usums, sc, ctl);
    if (tiles > 1) {
        reduce_fixup_kernel<<<(unsigned)(((uint64_t)tiles * 32 + 255) / 256), 256, 0, stream>>>(tiles, usums, sc);
        return 2;
    }
    return 1;
}

int launch_reduce(int key_bytes, int64_t n, const void* keys, CoefIn coefs, void* ukeys, double* usums,
                  const ReduceScratch& sc, Control* ctl, cudaStream_t stream)
{
    if (n <= 0) return 0;
    if (key_bytes == 8) return launch_reduce_t<uint64_t>(n, keys, coefs, ukeys, usums, sc, ctl, stream);
    if (key_bytes == 16) return launch_reduce_t<Key128>(n, keys, coefs, ukeys, usums, sc, ctl, stream);
    return launch_reduce_t<Key256>(n, keys, coefs, ukeys, usums, sc, ctl, stream);
}

// ------------------------------------------------------------------------------------------ S4 + S5

template <typename K, int THREADS, int ITEMS>
__global__ void __launch_bounds__(THREADS)
prune_unpack_kernel(const K* __restrict__ ukeys, const double* __restrict__ usums, double tol,
                    const __grid_constant__ Plan plan, CoefOut out_coef, void* out_exps, int exp_bytes,
                    int wpr, int64_t out_capacity, uint32_t* tile_state, Control* ctl, int64_t* out_count_device,
                    K* __restrict__ out_keys)
{
    constexpr int TILE = THREADS * ITEMS, NW = THREADS / 32;
    __shared__ uint32_t scratch[NW + 2];
    __shared__ uint16_t sel[TILE];                     // the tile's survivors, compacted: positions inside the tile
    __shared__ uint32_t sm_tile, sm_base;
    const unsigned tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
    const uint32_t U = ctl->distinct;
    while (true) {
        __syncthreads();                               // sm_tile / sm_base of the previous round are consumed
        if (tid == 0) sm_tile = atomicAdd(&ctl->ticket[kTicketPrune], 1u);
        __syncthreads();
        const uint32_t tile = sm_tile;
        const uint64_t tile_base = (uint64_t)tile * TILE;
        if (tile_base >= U) {
            if (tile == 0 && tid == 0) {               // zero polynomial (reading A3)
                ctl->survivors = 0;
                if (out_count_device) *out_count_device = 0;
            }
            break;
        }
        const uint32_t tile_n = (uint32_t)min((uint64_t)TILE, (uint64_t)U - tile_base);
        const uint32_t first = tid * ITEMS;
        double s[ITEMS];
        uint32_t keep = 0, cnt = 0;
#pragma unroll
        for (int j = 0; j < ITEMS; ++j) {
            s[j] = 0.0;
            if (first + j < tile_n) {
                s[j] = usums[tile_base + first + j];
                if (fabs(s[j]) > tol) { keep |= 1u << j; ++cnt; }      // NaN compares false: dropped (A12)
            }
        }
        uint32_t total;
        const uint32_t excl = block_exclusive_scan<THREADS>(cnt, scratch, &total);
        if (warp == 0) {
            const uint32_t r = warp_lookback_u32(tile_state, tile, total);
            if (lane == 0) sm_base = r;
        }
        __syncthreads();
        // survivors' positions, compacted in order; then the block writes them together so that consecutive threads
        // store consecutive words of the output (a thread writing its own 8 rows touched 32 sectors per store)
        {
            uint32_t q = excl;
#pragma unroll
            for (int j = 0; j < ITEMS; ++j)
                if (keep & (1u << j)) sel[q++] = (uint16_t)(first + j);
        }
        __syncthreads();
        const uint64_t obase = sm_base;
        for (uint32_t i = tid; i < total; i += THREADS)
            if ((int64_t)(obase + i) < out_capacity) out_coef.store(obase + i, usums[tile_base + sel[i]]);
        if (out_keys) {
            // packed output (the intermediate powers of polylab_pow_simplify): the survivors' keys stay keys
            for (uint32_t i = tid; i < total; i += THREADS)
                if ((int64_t)(obase + i) < out_capacity) out_keys[obase + i] = ukeys[tile_base + sel[i]];
        } else if (wpr > 0) {
            uint32_t* __restrict__ ow = (uint32_t*)out_exps;
            for (uint32_t f = tid; f < total * (uint32_t)wpr; f += THREADS) {
                const uint32_t i = f / (uint32_t)wpr, w = f - i * (uint32_t)wpr;
                if ((int64_t)(obase + i) < out_capacity)
                    ow[(obase + i) * (uint64_t)wpr + w] = unpack_row_word(plan, ukeys[tile_base + sel[i]], (int)w, exp_bytes);
            }
        } else {
            for (uint32_t i = tid; i < total; i += THREADS) {
                if ((int64_t)(obase + i) < out_capacity) {
                    const K kk = ukeys[tile_base + sel[i]];
                    for (int v = 0; v < plan.nvars; ++v)
                        store_exp(out_exps, exp_bytes, (int64_t)(obase + i) * plan.nvars + v, key_get_field(kk, plan.shift[v], plan.width[v]));
                }
            }
        }
        if (tile_base + tile_n == U && tid == 0) {
            ctl->survivors = sm_base + total;
            if (out_count_device) *out_count_device = (int64_t)(sm_base + total);
        }
    }
}

// Asynchronous calls (POLYLAB_FLAG_DEVICE_COUNT): the status the host would have read back, on the device.  A failed
// self-check (unstable ranking, a bucket too long for a tile, a slack bin too small) is POLYLAB_ERR_RETRY: nothing valid was
// emitted.
__global__ void async_status_kernel(const Control* ctl, int32_t* status_device, int64_t* out_count_device)
{
    const int32_t st = ctl->status != POLYLAB_OK ? ctl->status : (ctl->unsorted || ctl->overflow || ctl->slack_overflow) ? (int32_t)POLYLAB_ERR_RETRY : (int32_t)POLYLAB_OK;
    if (status_device) *status_device = st;
    if (st == POLYLAB_ERR_RETRY && out_count_device) *out_count_device = 0;
}

int launch_async_status(const Control* ctl, int32_t* status_device, int64_t* out_count_device, cudaStream_t stream)
{
    async_status_kernel<<<1, 1, 0, stream>>>(ctl, status_device, out_count_device);
    return 1;
}

int launch_prune_unpack(const Plan& plan, int64_t max_units, const void* ukeys, const double* usums, double tol,
                        CoefOut out_coef, void* out_exps, int exp_bytes, int64_t out_capacity, uint32_t* tile_state,
                        Control* ctl, int64_t* out_count_device, cudaStream_t stream, void* out_keys)
{
    if (max_units <= 0) return 0;
    int64_t blocks = (max_units + kPruneTile - 1) / kPruneTile;
    if (blocks > sm_count() * 8) blocks = sm_count() * 8;
    if (plan.key_bytes == 8)
        prune_unpack_kernel<uint64_t, kPruneThreads, kPruneItems><<<(unsigned)blocks, kPruneThreads, 0, stream>>>(
            (const uint64_t*)ukeys, usums, tol, plan, out_coef, out_exps, exp_bytes, row_words(plan.nvars, exp_bytes, out_exps),
            out_capacity, tile_state, ctl, out_count_device, (uint64_t*)out_keys);
    else if (plan.key_bytes == 16)
        prune_unpack_kernel<Key128, kPruneThreads, kPruneItems><<<(unsigned)blocks, kPruneThreads, 0, stream>>>(
            (const Key128*)ukeys, usums, tol, plan, out_coef, out_exps, exp_bytes, row_words(plan.nvars, exp_bytes, out_exps),
            out_capacity, tile_state, ctl, out_count_device, (Key128*)out_keys);
    else
        prune_unpack_kernel<Key256, kPruneThreads, kPruneItems><<<(unsigned)blocks, kPruneThreads, 0, stream>>>(
            (const Key256*)ukeys, usums, tol, plan, out_coef, out_exps, exp_bytes, row_words(plan.nvars, exp_bytes, out_exps),
            out_capacity, tile_state, ctl, out_count_device, (Key256*)out_keys);
    return 1;
}

}  // namespace polylab
