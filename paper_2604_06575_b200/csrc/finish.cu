// finish.cu -- the "bucket path" of step S2 and steps S3-S5 fused behind it.
//
// An LSD radix sort reads and writes every (key, coefficient) pair once per digit: 16 times for a 128-bit key.
// When the most significant digits spread the keys evenly, that is wasted traffic: k stable passes over the TOP k
// digits alone (the same sort_pass_kernel, most significant digits only) leave the array partitioned into buckets
// of keys that share their top T bits, in ascending bucket order, and a bucket that fits shared memory can be
// finished on chip.  This file is that finish:
//
//   tile_bounds_kernel   cuts the prefix-sorted array into tiles of whole buckets: tile t owns the buckets that
//                        START in positions [t*TILE, (t+1)*TILE); tile_start[t] is found by a binary search for the
//                        first change of prefix at or after t*TILE.  A bucket longer than CAP - TILE sets
//                        ctl->overflow and the call falls back to the plain LSD path.  TILE is chosen per call
//                        (api.cu): CAP minus room for the longest bucket expected from N / 2^T.
//   finish_kernel        one block per tile: loads its buckets (<= CAP records) into shared memory, sorts them
//                        there by the remaining low bits (stable LSD over a permutation of 16-bit indices, then by
//                        bucket ordinal), and -- the records of equal monomials now being adjacent and no run
//                        crossing a tile -- does the segmented sum (S3), the prune (S4, keep iff |s| > tol, reading
//                        A2), the order-preserving compaction (look-back over the tiles' survivor counts) and the
//                        unpack (S5) straight into the caller's output.  HBM traffic: N*(W+8) read, U'*(8+E) written.
//
// The local sort first tries the `nfast` most significant of the low digits only (enough to separate the distinct
// keys of a bucket unless two share all those bits) and checks the result against the full keys while it computes the
// head flags; a tile that fails the check re-sorts on every low digit (ctl->refinish counts them).
//
// Summation order (reading A6): equal keys keep their input order through every stable step; a tile sums left to
// right inside a thread and by a fixed shuffle tree across threads -- a function of the data layout only, so
// results are bit-reproducible run to run.
#include "kernels.h"

namespace polylab {

template <typename K> struct KeyWords;
template <> struct KeyWords<uint64_t> {
    static constexpr int N = 2;
    __device__ static __forceinline__ void store(uint32_t* skw, int cap, uint32_t i, uint64_t k)
    {
        skw[i] = (uint32_t)k;
        skw[cap + i] = (uint32_t)(k >> 32);
    }
    __device__ static __forceinline__ uint64_t load(const uint32_t* skw, int cap, uint32_t i)
    {
        return (uint64_t)skw[i] | ((uint64_t)skw[cap + i] << 32);
    }
};
template <> struct KeyWords<Key128> {
    static constexpr int N = 4;
    __device__ static __forceinline__ void store(uint32_t* skw, int cap, uint32_t i, const Key128& k)
    {
        skw[i] = (uint32_t)k.lo;
        skw[cap + i] = (uint32_t)(k.lo >> 32);
        skw[2 * cap + i] = (uint32_t)k.hi;
        skw[3 * cap + i] = (uint32_t)(k.hi >> 32);
    }
    __device__ static __forceinline__ Key128 load(const uint32_t* skw, int cap, uint32_t i)
    {
        Key128 k;
        k.lo = (uint64_t)skw[i] | ((uint64_t)skw[cap + i] << 32);
        k.hi = (uint64_t)skw[2 * cap + i] | ((uint64_t)skw[3 * cap + i] << 32);
        return k;
    }
};

// ------------------------------------------------------------------------------------- tile bounds

template <typename K>
__global__ void __launch_bounds__(256) tile_bounds_kernel(const K* __restrict__ keys, uint32_t n, int pfx_pos,
                                                          uint32_t fin_tile, uint32_t ntiles,
                                                          uint32_t* __restrict__ tile_start, Control* ctl)
{
    const uint32_t t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t > ntiles) return;
    if (t == 0) { tile_start[0] = 0u; return; }
    const uint64_t s64 = (uint64_t)t * fin_tile;
    if (s64 >= n) { tile_start[t] = n; return; }
    const uint32_t s = (uint32_t)s64;
    const K ref = keys[s - 1];
    uint32_t lo = s, hi = (uint32_t)min((uint64_t)n, s64 + (uint64_t)(kFinCap - fin_tile));
    if (hi < n && same_prefix(keys[hi], ref, pfx_pos)) {      // the bucket of record s-1 runs past what a tile can own
        ctl->overflow = 1u;
        tile_start[t] = s;
        return;
    }
    while (lo < hi) {                                         // smallest p in [lo, hi] whose prefix differs (p == n counts)
        const uint32_t mid = lo + (hi - lo) / 2;
        if (same_prefix(keys[mid], ref, pfx_pos)) lo = mid + 1;
        else hi = mid;
    }
    tile_start[t] = lo;
}

// --------------------------------------------------------------------------------- local radix pass

struct FinishSmem {
    static constexpr int NW = kFinThreads / 32;
    // doubles first, then 32-bit words, then 16-bit indices
    template <typename K> __host__ __device__ static constexpr size_t off_words() { return (size_t)kFinCap * sizeof(double); }
    template <typename K> __host__ __device__ static constexpr size_t off_whist() { return off_words<K>() + (size_t)KeyWords<K>::N * kFinCap * 4; }
    template <typename K> __host__ __device__ static constexpr size_t off_sbin() { return off_whist<K>() + (size_t)NW * kRadix * 4; }
    template <typename K> __host__ __device__ static constexpr size_t off_scratch() { return off_sbin<K>() + (size_t)kRadix * 4; }
    template <typename K> __host__ __device__ static constexpr size_t off_u16() { return off_scratch<K>() + 64 * 4; }
    template <typename K> __host__ __device__ static constexpr size_t bytes() { return off_u16<K>() + (size_t)3 * kFinCap * 2; }
};

// One stable counting-sort pass over the permutation: pout = pin reordered by the 8-bit (or narrower) digit
// (src[r] >> shift) & mask of record r.  Warp w ranks the contiguous chunk [w*per, (w+1)*per) of positions with one
// shared-memory atomic per record on its own histogram row (lane order inside a warp instruction, item order across
// instructions: the same measured property as sort.cu's RANK_ATOMIC, re-verified by the caller's order check).
template <typename SRC>
__device__ __forceinline__ void local_pass(const SRC* __restrict__ src, int shift, uint32_t mask, const uint16_t* pin,
                                           uint16_t* pout, uint32_t n_loc, uint32_t* whist, uint32_t* sbin, uint32_t* scratch)
{
    constexpr int NW = FinishSmem::NW;
    constexpr int R = kFinCap / kFinThreads;                  // rounds of 32 records per warp at full capacity
    static_assert(kFinCap % kFinThreads == 0, "capacity must be a whole number of rounds");
    const unsigned tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
    for (int i = tid; i < NW * kRadix; i += kFinThreads) whist[i] = 0u;
    __syncthreads();
    const uint32_t per = (((n_loc + NW - 1) / NW) + 31u) & ~31u;
    const uint32_t wbase = warp * per;
    uint32_t* my_hist = whist + warp * kRadix;
    uint32_t rd[R];                                           // record (13 bits) | digit (8) << 13 | rank in warp (9) << 21
#pragma unroll
    for (int j = 0; j < R; ++j) {
        rd[j] = 0xffffffffu;
        const uint32_t i = wbase + j * 32u + lane;
        if (j * 32u < per && i < n_loc) {
            const uint32_t r = pin[i];
            const uint32_t d = ((uint32_t)src[r] >> shift) & mask;
            const uint32_t rank = atomicAdd(&my_hist[d], 1u);
            rd[j] = r | (d << 13) | (rank << 21);
        }
        __syncwarp();
    }
    __syncthreads();
    uint32_t count = 0;
    if (tid < kRadix) {
#pragma unroll
        for (int w = 0; w < NW; ++w) {
            const uint32_t c = whist[w * kRadix + tid];
            whist[w * kRadix + tid] = count;
            count += c;
        }
    }
    uint32_t total;
    const uint32_t bin_start = block_exclusive_scan<kFinThreads>(count, scratch, &total);
    if (tid < kRadix) sbin[tid] = bin_start;
    __syncthreads();
#pragma unroll
    for (int j = 0; j < R; ++j) {
        if (rd[j] != 0xffffffffu) {
            const uint32_t r = rd[j] & 0x1fffu, d = (rd[j] >> 13) & 0xffu, rank = rd[j] >> 21;
            pout[sbin[d] + my_hist[d] + rank] = (uint16_t)r;
        }
    }
    __syncthreads();
}

struct FinishArgs {
    const void* keys;
    const double* coefs;
    uint32_t n, ntiles;
    uint32_t fin_tile;              // positions per tile; a tile owns at most kFinCap records
    const uint32_t* tile_start;     // [ntiles + 1]
    uint32_t* tile_state;           // [ntiles] look-back words, zero before the kernel
    int pfx_pos;                    // the prefix is the key bits at positions >= pfx_pos
    int nlow;                       // plan digits below the prefix: digits [0, nlow)
    int nfast;                      // how many of them (the most significant ones) the first attempt sorts on
    double tol;
    double* out_coef;
    void* out_exps;
    int exp_bytes;
    int64_t out_capacity;
    Control* ctl;
    int64_t* out_count_device;
};

template <typename K>
__device__ __forceinline__ void emit_term(const FinishArgs& a, const Plan& plan, uint64_t o, double s, const K& kk)
{
    if ((int64_t)o >= a.out_capacity) return;
    a.out_coef[o] = s;
    for (int v = 0; v < plan.nvars; ++v)
        store_exp(a.out_exps, a.exp_bytes, (int64_t)o * plan.nvars + v, key_get_field(kk, plan.shift[v], plan.width[v]));
}

// ------------------------------------------------------------------------------------ finish kernel

template <typename K>
__global__ void __launch_bounds__(kFinThreads, 1) finish_kernel(const __grid_constant__ FinishArgs a, const __grid_constant__ Plan plan)
{
    constexpr int THREADS = kFinThreads, CAP = kFinCap, NW = THREADS / 32, IT = CAP / THREADS;
    static_assert(CAP <= 8192 && CAP / NW <= 512 && IT <= 16, "index packing of local_pass / head masks");
    using KW = KeyWords<K>;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double* scoef = (double*)smem_raw;
    uint32_t* skw = (uint32_t*)(smem_raw + FinishSmem::off_words<K>());
    uint32_t* whist = (uint32_t*)(smem_raw + FinishSmem::off_whist<K>());
    uint32_t* sbin = (uint32_t*)(smem_raw + FinishSmem::off_sbin<K>());
    uint32_t* scratch = (uint32_t*)(smem_raw + FinishSmem::off_scratch<K>());     // [0..NW+1] scan, [40] tile, [41] base
    uint16_t* perm0 = (uint16_t*)(smem_raw + FinishSmem::off_u16<K>());
    uint16_t* perm1 = perm0 + CAP;
    uint16_t* ord = perm1 + CAP;
    __shared__ uint32_t wagg_f[NW];
    __shared__ double wagg_v[NW];

    const unsigned tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
    if (a.ctl->overflow) return;                              // set by tile_bounds_kernel: the call will re-run on the LSD path
    if (tid == 0) scratch[40] = atomicAdd(&a.ctl->ticket[kTicketFinish], 1u);
    __syncthreads();
    const uint32_t tile = scratch[40];
    const uint32_t lo = a.tile_start[tile], hi = a.tile_start[tile + 1];
    uint32_t n_loc = 0;
    if ((uint64_t)lo < ((uint64_t)tile + 1) * a.fin_tile && hi > lo) n_loc = min(hi - lo, (uint32_t)CAP);

    // ---- load the tile's buckets: keys as word planes (random word reads then spread over all banks), coefficients
    const K* __restrict__ gkeys = (const K*)a.keys + lo;
    const double* __restrict__ gcoef = a.coefs + lo;
    for (uint32_t i = tid; i < n_loc; i += THREADS) {
        KW::store(skw, CAP, i, gkeys[i]);
        scoef[i] = gcoef[i];
        perm0[i] = (uint16_t)i;
    }
    __syncthreads();

    // ---- bucket ordinal of every record (the input is sorted by prefix, so buckets are contiguous)
    const uint32_t first = tid * IT;
    uint32_t nbuckets;
    {
        uint32_t hm = 0, nh = 0;
        bool descending = false;
        K kp;
        key_zero(kp);
        if (first > 0 && first < n_loc) kp = KW::load(skw, CAP, first - 1);
#pragma unroll
        for (int j = 0; j < IT; ++j) {
            if (first + j < n_loc) {
                const K kk = KW::load(skw, CAP, first + j);
                const bool head = (first + j == 0) || !same_prefix(kk, kp, a.pfx_pos);
                descending |= (first + j > 0) && head && key_lt(kk, kp);
                if (head) { hm |= 1u << j; ++nh; }
                kp = kk;
            }
        }
        if (descending) a.ctl->unsorted = 1u;                 // the prefix passes were not stable (see sort.cu)
        const uint32_t excl = block_exclusive_scan<THREADS>(nh, scratch, &nbuckets);
        uint32_t o = excl;
#pragma unroll
        for (int j = 0; j < IT; ++j) {
            if (first + j < n_loc) {
                if (hm & (1u << j)) ++o;
                ord[first + j] = (uint16_t)(o - 1u);
            }
        }
    }
    __syncthreads();

    // ---- local sort + head flags; the order check decides whether the fast digit list was enough
    const uint16_t* perm = perm0;
    uint32_t hm = 0, nh = 0;
    double acc = 0.0;
    int d_lo = (a.nfast < a.nlow) ? a.nlow - a.nfast : 0;
    while (true) {
        uint16_t* pin = perm0;
        uint16_t* pout = perm1;
        for (int d = d_lo; d < a.nlow; ++d) {
            const int pos = plan.digit_pos[d];
            local_pass<uint32_t>(skw + (size_t)(pos >> 5) * CAP, pos & 31, (1u << plan.digit_bits[d]) - 1u, pin, pout, n_loc,
                                 whist, sbin, scratch);
            uint16_t* t = pin; pin = pout; pout = t;
        }
        for (int ob = 0; nbuckets > 1 && ((nbuckets - 1u) >> ob) != 0u; ob += kRadixBits) {
            local_pass<uint16_t>(ord, ob, (uint32_t)kRadix - 1u, pin, pout, n_loc, whist, sbin, scratch);
            uint16_t* t = pin; pin = pout; pout = t;
        }
        perm = pin;
        // heads of runs of equal keys, the sum since the last head, and the order check
        hm = 0; nh = 0; acc = 0.0;
        bool viol = false;
        K kp;
        key_zero(kp);
        if (first > 0 && first < n_loc) kp = KW::load(skw, CAP, perm[first - 1]);
#pragma unroll
        for (int j = 0; j < IT; ++j) {
            if (first + j < n_loc) {
                const uint32_t r = perm[first + j];
                const K kk = KW::load(skw, CAP, r);
                const bool head = (first + j == 0) || !key_eq(kk, kp);
                viol |= (first + j > 0) && key_lt(kk, kp);
                if (head) { hm |= 1u << j; ++nh; acc = scoef[r]; }
                else acc = __dadd_rn(acc, scoef[r]);
                kp = kk;
            }
        }
        if (!__syncthreads_or(viol ? 1 : 0)) break;
        if (d_lo == 0) {                                      // every digit was sorted on and the order is still wrong
            if (tid == 0) a.ctl->unsorted = 1u;
            break;
        }
        d_lo = 0;
        if (tid == 0) atomicAdd(&a.ctl->refinish, 1u);
        for (uint32_t i = tid; i < n_loc; i += THREADS) perm0[i] = (uint16_t)i;
        __syncthreads();
    }

    // ---- S3: segmented scan of (has head, sum since last head) across the block; no run crosses a tile
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
    SegPair carry;                                            // exclusive within the warp
    carry.f = __shfl_up_sync(kFullMask, incl.f, 1);
    carry.v = __shfl_up_sync(kFullMask, incl.v, 1);
    if (lane == 0) { carry.f = 0; carry.v = 0.0; }
    __syncthreads();
    {
        SegPair wp;
        wp.f = 0;
        wp.v = 0.0;
        for (unsigned w = 0; w < warp; ++w) {
            SegPair x;
            x.f = wagg_f[w];
            x.v = wagg_v[w];
            wp = seg_combine(wp, x);
        }
        carry = seg_combine(wp, carry);
        incl = seg_combine(wp, incl);
    }

    // ---- S4: which of the runs that END in this thread survive (a run ends where the next head is met; the run still
    // open at the end of the tile is closed by the last thread, whose inclusive scan value is its sum)
    uint32_t keep = 0, nkeep = 0;
    {
        uint32_t k = 0;
        double a2 = 0.0;
#pragma unroll
        for (int j = 0; j < IT; ++j) {
            if (first + j < n_loc) {
                const double c = scoef[perm[first + j]];
                if (hm & (1u << j)) {
                    if (first + j > 0) {
                        const double total = (k == 0) ? __dadd_rn(carry.v, a2) : a2;
                        if (fabs(total) > a.tol) { keep |= 1u << k; ++nkeep; }     // NaN compares false: dropped (A12)
                        ++k;
                    }
                    a2 = c;
                } else a2 = __dadd_rn(a2, c);
            }
        }
    }
    const bool last_keep = (tid == THREADS - 1) && n_loc > 0 && fabs(incl.v) > a.tol;
    uint32_t tile_keep;
    const uint32_t kexcl = block_exclusive_scan<THREADS>(nkeep + (last_keep ? 1u : 0u), scratch, &tile_keep);
    if (warp == 0) {
        const uint32_t r = warp_lookback_u32(a.tile_state, tile, tile_keep);
        if (lane == 0) scratch[41] = r;
    }
    __syncthreads();
    const uint32_t base = scratch[41];

    // ---- S5: write the survivors in order
    {
        uint64_t o = (uint64_t)base + kexcl;
        uint32_t k = 0;
        double a2 = 0.0;
        uint32_t rprev = 0;
#pragma unroll
        for (int j = 0; j < IT; ++j) {
            if (first + j < n_loc) {
                const uint32_t r = perm[first + j];
                const double c = scoef[r];
                if (hm & (1u << j)) {
                    if (first + j > 0) {
                        if (keep & (1u << k)) {
                            const double total = (k == 0) ? __dadd_rn(carry.v, a2) : a2;
                            if (j == 0) rprev = perm[first - 1];
                            emit_term<K>(a, plan, o, total, KW::load(skw, CAP, rprev));
                            ++o;
                        }
                        ++k;
                    }
                    a2 = c;
                } else a2 = __dadd_rn(a2, c);
                rprev = r;
            }
        }
        if (last_keep) emit_term<K>(a, plan, o, incl.v, KW::load(skw, CAP, perm[n_loc - 1]));
    }
    {
        uint32_t tot_heads;                                   // distinct monomials of the tile, for the statistics
        (void)block_exclusive_scan<THREADS>(nh, scratch, &tot_heads);
        if (tid == 0 && tot_heads) atomicAdd(&a.ctl->distinct, tot_heads);
    }
    if (tile == a.ntiles - 1 && tid == 0) {
        a.ctl->survivors = base + tile_keep;
        if (a.out_count_device) *a.out_count_device = (int64_t)(base + tile_keep);
    }
}

// ---------------------------------------------------------------------------------------- launchers

template <typename K>
static int launch_finish_t(const Plan& plan, int prefix_passes, int nfast, int fin_tile, int64_t n, const void* keys, const double* coefs,
                           double tol, double* out_coef, void* out_exps, int exp_bytes, int64_t out_capacity,
                           uint32_t* tile_start, uint32_t* tile_state, Control* ctl, int64_t* out_count_device,
                           cudaStream_t stream)
{
    const uint32_t ntiles = (uint32_t)((n + fin_tile - 1) / fin_tile);
    const int nlow = plan.npasses - prefix_passes;
    const int pfx_pos = plan.digit_pos[nlow];
    tile_bounds_kernel<K><<<(ntiles + 1 + 255) / 256, 256, 0, stream>>>((const K*)keys, (uint32_t)n, pfx_pos, (uint32_t)fin_tile, ntiles, tile_start, ctl);
    auto kern = finish_kernel<K>;
    constexpr size_t smem = FinishSmem::bytes<K>();
    static bool attr_set = false;
    if (!attr_set) {
        cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        attr_set = true;
    }
    FinishArgs a;
    a.keys = keys; a.coefs = coefs; a.n = (uint32_t)n; a.ntiles = ntiles; a.fin_tile = (uint32_t)fin_tile; a.tile_start = tile_start; a.tile_state = tile_state;
    a.pfx_pos = pfx_pos; a.nlow = nlow; a.nfast = nfast; a.tol = tol; a.out_coef = out_coef; a.out_exps = out_exps;
    a.exp_bytes = exp_bytes; a.out_capacity = out_capacity; a.ctl = ctl; a.out_count_device = out_count_device;
    kern<<<ntiles, kFinThreads, smem, stream>>>(a, plan);
    return 2;
}

int launch_finish(const Plan& plan, int prefix_passes, int nfast, int fin_tile, int64_t n, const void* keys, const double* coefs, double tol,
                  double* out_coef, void* out_exps, int exp_bytes, int64_t out_capacity, uint32_t* tile_start,
                  uint32_t* tile_state, Control* ctl, int64_t* out_count_device, cudaStream_t stream)
{
    if (n <= 0 || prefix_passes < 1 || prefix_passes > plan.npasses || fin_tile < kFinMinTile || fin_tile >= kFinCap) return 0;
    if (plan.key_bytes == 8)
        return launch_finish_t<uint64_t>(plan, prefix_passes, nfast, fin_tile, n, keys, coefs, tol, out_coef, out_exps, exp_bytes,
                                         out_capacity, tile_start, tile_state, ctl, out_count_device, stream);
    return launch_finish_t<Key128>(plan, prefix_passes, nfast, fin_tile, n, keys, coefs, tol, out_coef, out_exps, exp_bytes, out_capacity,
                                   tile_start, tile_state, ctl, out_count_device, stream);
}

}  // namespace polylab
