// common.cuh -- shared device/host definitions of the polylab-b200 CUDA path (sm_100a).
//
// Nothing here is shared with oracle/: the oracle never packs keys.  The key layout follows
// variable 0 occupies the most significant field, fields are right-aligned to
// bit 0, field v is w_v = bitlen(m_v) bits wide (0 bits when the variable is identically zero), so
// that unsigned order of keys = ascending lexicographic order of exponent rows (reading A1, the
// order of the paper's transcripts PAPER.md:195-201).
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/polylab.h"

namespace polylab {

constexpr int kMaxVars = POLYLAB_MAX_NVARS;
constexpr int kMaxPasses = 32;          // 256 bits / 8-bit digits
constexpr int kRadixBits = 8;           // widest digit
constexpr int kRadix = 1 << kRadixBits; // bins per pass
constexpr unsigned kFullMask = 0xffffffffu;

// ------------------------------------------------------------------------------------ keys

// 128-bit key, 16-byte aligned so that one key is one vector load/store.
struct __align__(16) Key128 {
    uint64_t hi, lo;     // memory order (hi, lo): the layout polylab_pack_keys exposes
};

// 256-bit key for wide variable sets ("multi-word for wide variable sets"; the 500-variable sparse quartics
// of PAPER.md:546 are the paper's own wide case): four 64-bit limbs, most significant first, like Key128's (hi, lo).
struct __align__(32) Key256 {
    uint64_t q[4];       // q[0] most significant
};

__host__ __device__ inline bool key_eq(uint64_t a, uint64_t b) { return a == b; }
__host__ __device__ inline bool key_eq(const Key128& a, const Key128& b) { return a.lo == b.lo && a.hi == b.hi; }
__host__ __device__ inline bool key_lt(uint64_t a, uint64_t b) { return a < b; }
__host__ __device__ inline bool key_lt(const Key128& a, const Key128& b) { return a.hi < b.hi || (a.hi == b.hi && a.lo < b.lo); }

__host__ __device__ inline bool key_eq(const Key256& a, const Key256& b) { return a.q[0] == b.q[0] && a.q[1] == b.q[1] && a.q[2] == b.q[2] && a.q[3] == b.q[3]; }
__host__ __device__ inline bool key_lt(const Key256& a, const Key256& b)
{
#pragma unroll
    for (int i = 0; i < 3; ++i)
        if (a.q[i] != b.q[i]) return a.q[i] < b.q[i];
    return a.q[3] < b.q[3];
}
__device__ __forceinline__ uint32_t key_word(const Key256& k, int wi)
{
    const int l = wi >> 1;                               // 64-bit limb, 0 = least significant
    const uint64_t h = l == 0 ? k.q[3] : l == 1 ? k.q[2] : l == 2 ? k.q[1] : k.q[0];
    return (wi & 1) ? (uint32_t)(h >> 32) : (uint32_t)h;
}
__device__ __forceinline__ Key256 key_add(const Key256& a, const Key256& b)
{
    Key256 r;
    uint64_t carry = 0;
#pragma unroll
    for (int i = 3; i >= 0; --i) {                       // fields never carry into each other, limbs may
        const uint64_t s = a.q[i] + b.q[i], t = s + carry;
        carry = (s < a.q[i]) || (t < s) ? 1ull : 0ull;
        r.q[i] = t;
    }
    return r;
}
__host__ __device__ inline bool same_prefix(const Key256& a, const Key256& b, int pos)
{
#pragma unroll
    for (int l = 3; l >= 0; --l) {                       // limb l holds bits [64 l, 64 l + 64)
        const uint64_t x = a.q[3 - l] ^ b.q[3 - l];
        if (pos >= 64 * (l + 1)) break;
        if (pos <= 64 * l) { if (x) return false; }
        else return (x >> (pos - 64 * l)) == 0;
    }
    return true;
}
__device__ __forceinline__ void key_or_field(Key256& k, uint32_t e, int shift)
{
    const int l = shift >> 6, sh = shift & 63;
    const uint64_t lo = (uint64_t)e << sh, hi = sh > 32 ? (uint64_t)e >> (64 - sh) : 0ull;
#pragma unroll
    for (int i = 0; i < 4; ++i) {                        // selects, not dynamically indexed registers
        if (3 - i == l) k.q[i] |= lo;
        if (3 - i == l + 1) k.q[i] |= hi;
    }
}
__device__ __forceinline__ uint32_t key_get_field(const Key256& k, int shift, int width)
{
    if (width == 0) return 0u;
    const int l = shift >> 6, sh = shift & 63;
    uint64_t a = 0, b = 0;                               // limb l and the one above it
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        if (3 - i == l) a = k.q[i];
        if (3 - i == l + 1) b = k.q[i];
    }
    const uint64_t w = sh == 0 ? a : ((a >> sh) | (b << (64 - sh)));
    return (uint32_t)(w & ((width == 32) ? 0xffffffffull : ((1ull << width) - 1)));
}

// 32-bit word `wi` of a key (0 = least significant).  wi is uniform across a kernel: the selects cost 1-3 instructions.
__device__ __forceinline__ uint32_t key_word(uint64_t k, int wi) { return wi ? (uint32_t)(k >> 32) : (uint32_t)k; }
__device__ __forceinline__ uint32_t key_word(const Key128& k, int wi)
{
    const uint64_t h = (wi & 2) ? k.hi : k.lo;
    return (wi & 1) ? (uint32_t)(h >> 32) : (uint32_t)h;
}
// byte offset of word `wi` inside the key as stored in memory (Key128 is stored (hi, lo))
template <typename K> __host__ __device__ inline int key_word_byte_offset(int wi);
template <> __host__ __device__ inline int key_word_byte_offset<uint64_t>(int wi) { return wi * 4; }
template <> __host__ __device__ inline int key_word_byte_offset<Key128>(int wi) { return (wi ^ 2) * 4; }
template <> __host__ __device__ inline int key_word_byte_offset<Key256>(int wi) { return (wi ^ 6) * 4; }

// The digit of `mask`'s width at bit `pos` (0 = least significant).  The plan never lets a digit straddle a
// 32-bit word (make_plan), so a digit is one shift and one mask of one word.
template <typename K>
__device__ __forceinline__ uint32_t key_digit(const K& k, int pos, uint32_t mask) { return (key_word(k, pos >> 5) >> (pos & 31)) & mask; }

__device__ __forceinline__ uint64_t key_add(uint64_t a, uint64_t b) { return a + b; }
__device__ __forceinline__ Key128 key_add(const Key128& a, const Key128& b)
{
    Key128 r;
    r.lo = a.lo + b.lo;
    r.hi = a.hi + b.hi + (r.lo < a.lo ? 1ull : 0ull);   // fields never carry into each other, words may
    return r;
}

// do a and b agree on all bits at positions >= pos?  (the "prefix" of the bucket path, finish.cu)
__host__ __device__ inline bool same_prefix(uint64_t a, uint64_t b, int pos) { return ((a ^ b) >> pos) == 0; }
__host__ __device__ inline bool same_prefix(const Key128& a, const Key128& b, int pos)
{
    if (pos >= 64) return ((a.hi ^ b.hi) >> (pos - 64)) == 0;
    return a.hi == b.hi && ((a.lo ^ b.lo) >> pos) == 0;
}

template <typename K> __device__ __forceinline__ K key_max();
template <> __device__ __forceinline__ uint64_t key_max<uint64_t>() { return ~0ull; }
template <> __device__ __forceinline__ Key128 key_max<Key128>() { Key128 k; k.lo = ~0ull; k.hi = ~0ull; return k; }
template <> __device__ __forceinline__ Key256 key_max<Key256>() { Key256 k; k.q[0] = k.q[1] = k.q[2] = k.q[3] = ~0ull; return k; }

// OR `e << shift` into a key (shift + width <= key bits by construction of the plan)
__device__ __forceinline__ void key_or_field(uint64_t& k, uint32_t e, int shift) { k |= (uint64_t)e << shift; }
__device__ __forceinline__ void key_or_field(Key128& k, uint32_t e, int shift)
{
    if (shift >= 64) k.hi |= (uint64_t)e << (shift - 64);
    else {
        k.lo |= (uint64_t)e << shift;
        if (shift > 32) k.hi |= (uint64_t)e >> (64 - shift);   // e has 32 bits: spills iff shift > 32
    }
}
__device__ __forceinline__ uint32_t key_get_field(uint64_t k, int shift, int width)
{
    return width == 0 ? 0u : (uint32_t)((k >> shift) & ((width == 32) ? 0xffffffffull : ((1ull << width) - 1)));
}
__device__ __forceinline__ uint32_t key_get_field(const Key128& k, int shift, int width)
{
    if (width == 0) return 0u;
    uint64_t w;
    if (shift >= 64) w = k.hi >> (shift - 64);
    else if (shift == 0) w = k.lo;
    else w = (k.lo >> shift) | (k.hi << (64 - shift));
    return (uint32_t)(w & ((width == 32) ? 0xffffffffull : ((1ull << width) - 1)));
}
// key from its most / least significant 64-bit halves (for a 64-bit key both arguments are the key)
__device__ __forceinline__ void key_from_halves(uint64_t& k, uint64_t hi, uint64_t lo) { (void)hi; k = lo; }
__device__ __forceinline__ void key_from_halves(Key128& k, uint64_t hi, uint64_t lo) { k.hi = hi; k.lo = lo; }
__device__ __forceinline__ uint64_t key_top64(uint64_t k) { return k; }          // most significant 64 bits of a key
__device__ __forceinline__ uint64_t key_top64(const Key128& k) { return k.hi; }
__device__ __forceinline__ void key_zero(uint64_t& k) { k = 0; }
__device__ __forceinline__ void key_zero(Key128& k) { k.lo = 0; k.hi = 0; }
__device__ __forceinline__ void key_zero(Key256& k) { k.q[0] = k.q[1] = k.q[2] = k.q[3] = 0; }
__device__ __forceinline__ void key_from_halves(Key256& k, uint64_t hi, uint64_t lo) { k.q[0] = hi; k.q[1] = 0; k.q[2] = 0; k.q[3] = lo; }   // (never used: no fused pack for 256-bit keys)
__device__ __forceinline__ uint64_t key_top64(const Key256& k) { return k.q[0]; }

// --------------------------------------------------------------------------------- coefficients

// Coefficient arrays at the ABI are fp64, or fp32 with opts->coef_type = POLYLAB_COEF_F32 (the paper's
// polylab_precision('set','single')): single-precision STORAGE.  Every fp32 value is widened on its first
// load, all arithmetic of the path (products, sums, the prune comparison) stays fp64, and a result is rounded to fp32 once,
// when it is stored.  Workspace intermediates are always fp64.  CoefIn / CoefOut carry the pointer with its type so that
// kernels index them like plain arrays.
struct CoefIn {
    const void* p;
    int f32;
    CoefIn() : p(nullptr), f32(0) {}
    CoefIn(const double* d) : p(d), f32(0) {}
    CoefIn(const void* q, int is_f32) : p(q), f32(is_f32) {}
    __device__ __forceinline__ double operator[](size_t i) const
    {
        return f32 ? (double)__ldg((const float*)p + i) : __ldg((const double*)p + i);
    }
    __host__ __device__ CoefIn operator+(size_t off) const { return CoefIn((const char*)p + off * (f32 ? 4 : 8), f32); }
};
struct CoefOut {
    void* p;
    int f32;
    CoefOut() : p(nullptr), f32(0) {}
    CoefOut(double* d) : p(d), f32(0) {}
    CoefOut(void* q, int is_f32) : p(q), f32(is_f32) {}
    __device__ __forceinline__ void store(size_t i, double v) const
    {
        if (f32) ((float*)p)[i] = __double2float_rn(v);
        else ((double*)p)[i] = v;
    }
};

// ------------------------------------------------------------------------------------ plan

// Key layout and pass table, computed on the host from the per-variable maxima (step S0) and passed
// to kernels by value.
struct Plan {
    int32_t nvars;
    int32_t key_bits;                  // B
    int32_t key_bytes;                 // W: 8, 16 or 32
    int32_t npasses;                   // P
    uint8_t shift[kMaxVars];           // bit position of field v
    uint8_t width[kMaxVars];           // w_v
    uint32_t bound[kMaxVars];          // largest exponent an INPUT row may hold in variable v
    uint8_t digit_pos[kMaxPasses];     // bit position of pass p's digit
    uint8_t digit_bits[kMaxPasses];    // its width (<= kRadixBits)
};

// How an exponent matrix is addressed: element (t,v) at base[t*term_stride + v*var_stride].
struct ExpView {
    const void* base;
    int64_t term_stride;
    int64_t var_stride;
    int32_t exp_bytes;                 // 1, 2 or 4
    int32_t row_major_contiguous;      // term_stride == nvars && var_stride == 1 && base 16-byte aligned
};

__device__ __forceinline__ uint32_t load_exp(const void* base, int exp_bytes, int64_t idx)
{
    if (exp_bytes == 1) return ((const uint8_t*)base)[idx];
    if (exp_bytes == 2) return ((const uint16_t*)base)[idx];
    return ((const uint32_t*)base)[idx];
}
__device__ __forceinline__ void store_exp(void* base, int exp_bytes, int64_t idx, uint32_t e)
{
    if (exp_bytes == 1) ((uint8_t*)base)[idx] = (uint8_t)e;
    else if (exp_bytes == 2) ((uint16_t*)base)[idx] = (uint16_t)e;
    else ((uint32_t*)base)[idx] = e;
}

// 32-bit word `w` of the unpacked exponent row of key kk (S5) when rows are written as words: exp_bytes 1 -> variables
// 4w..4w+3, 2 -> 2w, 2w+1, 4 -> w.  Usable when nvars * exp_bytes is a multiple of 4 and the output base is 4-byte aligned.
template <typename K>
__device__ __forceinline__ uint32_t unpack_row_word(const Plan& plan, const K& kk, int w, int exp_bytes)
{
    if (exp_bytes == 4) return key_get_field(kk, plan.shift[w], plan.width[w]);
    if (exp_bytes == 2)
        return key_get_field(kk, plan.shift[2 * w], plan.width[2 * w]) |
               (key_get_field(kk, plan.shift[2 * w + 1], plan.width[2 * w + 1]) << 16);
    return key_get_field(kk, plan.shift[4 * w], plan.width[4 * w]) |
           (key_get_field(kk, plan.shift[4 * w + 1], plan.width[4 * w + 1]) << 8) |
           (key_get_field(kk, plan.shift[4 * w + 2], plan.width[4 * w + 2]) << 16) |
           (key_get_field(kk, plan.shift[4 * w + 3], plan.width[4 * w + 3]) << 24);
}
__host__ inline int row_words(int nvars, int exp_bytes, const void* out_exps)
{
    const int rb = nvars * exp_bytes;
    return (rb % 4 == 0 && ((uintptr_t)out_exps & 3) == 0) ? rb / 4 : 0;      // 0: rows cannot be written as words
}

// S1 for one variable: range check against the plan's bound, field into the key (pack.cu, table.cu)
template <typename K>
__device__ __forceinline__ void pack_field(K& key, uint32_t e, int v, const Plan& plan, bool& bad)
{
    bad |= e > plan.bound[v];
    key_or_field(key, e, plan.shift[v]);     // width 0 => bound 0 => e must be 0: nothing is OR-ed
}

// 16-byte asynchronous copy global -> shared (both 16-byte aligned); completion through cp.async.commit_group / wait_group
__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gmem_src)
{
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"((uint32_t)__cvta_generic_to_shared(smem_dst)), "l"(gmem_src) : "memory");
}

// --------------------------------------------------------------------------- control block

// Small device-side state at the head of the workspace, zeroed at the start of every call.
struct Control {
    uint32_t hist[kMaxPasses + 1][kRadix];   // digit histograms, one per pass (filled one pass ahead)
    uint32_t ticket[kMaxPasses + 4];         // dynamic tile ids: sort passes, then reduce, then prune
    uint32_t max_exp[2][kMaxVars];           // S0 results (operand a, operand b)
    int32_t status;                          // polylab_status of data-dependent checks
    uint32_t distinct;                       // U
    uint32_t survivors;                      // U'
    uint32_t unsorted;                       // S3 saw a key smaller than its predecessor (the sort was not stable)
    uint32_t overflow;                       // bucket path: a bucket does not fit a finish tile (skewed prefix digits)
    uint32_t refinish;                       // bucket path: finish tiles that needed the full local digit list
    uint32_t fin_count;                      // bucket path: tiles that own records (length of the work list)
    uint32_t tab_count;                      // table path: distinct keys inserted so far (= U after the insert pass)
    uint32_t tab_overflow;                   // table path: more distinct keys than the table was sized for -> sort path
    uint32_t slack_overflow;                 // slack bins (sort.cu): a bin's capacity, estimated from a sample, was too small
    uint32_t fin2_count;                     // bucket path: tiles the sorting finish kernel did behind the group kernel (one add per block)
    uint32_t grp_fail;                       // bucket path: tiles the group kernel tried and gave back
    uint32_t grp_off;                        // bucket path: sticky, set once most tiles were given back: the group kernel stops trying
    uint32_t grp_left;                       // bucket path: tiles the group kernel did not finish (one add per block)
    uint32_t fin_ticket;                     // bucket path: next work-list entry the sorting kernel behind the group kernel hands out
    uint32_t slack_count[kRadix];            // exact bin counts of the pass that wrote with slack
    uint32_t slack_cap[kRadix];              // the capacities (kept for the reading pass)
    uint32_t est[kRadix];                    // histogram of the first prefix digit over a SAMPLE of the rows
};

constexpr int kTicketReduce = kMaxPasses;
constexpr int kTicketPrune = kMaxPasses + 1;

// ------------------------------------------------------------------------- warp/block helpers

__device__ __forceinline__ unsigned lane_id() { return threadIdx.x & 31u; }
__device__ __forceinline__ unsigned lanemask_lt() { return (1u << (threadIdx.x & 31u)) - 1u; }

// lanes of the warp that are `valid` and hold the same digit d (< 256) as the calling lane
__device__ __forceinline__ unsigned match_digit(uint32_t d, bool valid)
{
    unsigned mask = __ballot_sync(kFullMask, valid);
#pragma unroll
    for (int b = 0; b < kRadixBits; ++b) {
        const bool bit = (d >> b) & 1u;
        const unsigned m = __ballot_sync(kFullMask, bit);
        mask &= bit ? m : ~m;
    }
    return mask;
}

// lanes of the warp holding the same digit d (< 256) as the calling lane; all 32 lanes participate
__device__ __forceinline__ unsigned match_digit_all(uint32_t d)
{
    unsigned mask = kFullMask;
#pragma unroll
    for (int b = 0; b < kRadixBits; ++b) {
        const unsigned x = 0u - ((d >> b) & 1u);            // all ones iff bit b of d is set
        const unsigned m = __ballot_sync(kFullMask, x != 0u);
        mask &= ~(m ^ x);                                   // keep the lanes whose bit b equals ours
    }
    return mask;
}

// volatile accesses for the decoupled look-back words (value and flag share one 32-bit word)
__device__ __forceinline__ uint32_t ld_volatile_u32(const uint32_t* p)
{
    uint32_t v;
    asm volatile("ld.volatile.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_volatile_u32(uint32_t* p, uint32_t v)
{
    asm volatile("st.volatile.global.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}

// Exclusive scan of one uint32 per thread over a block of THREADS (multiple of 32, <= 1024).
// `warp_scratch` holds THREADS/32 + 1 words of shared memory; returns the exclusive prefix and
// stores the block total in *total.  Contains two __syncthreads().
template <int THREADS>
__device__ __forceinline__ uint32_t block_exclusive_scan(uint32_t x, uint32_t* warp_scratch, uint32_t* total)
{
    constexpr int NW = THREADS / 32;
    const unsigned lane = lane_id(), warp = threadIdx.x >> 5;
    uint32_t incl = x;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const uint32_t y = __shfl_up_sync(kFullMask, incl, o);
        if (lane >= (unsigned)o) incl += y;
    }
    if (lane == 31) warp_scratch[warp] = incl;
    __syncthreads();
    if (warp == 0) {
        uint32_t w = lane < NW ? warp_scratch[lane] : 0u;
        uint32_t wi = w;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t y = __shfl_up_sync(kFullMask, wi, o);
            if (lane >= (unsigned)o) wi += y;
        }
        if (lane < NW) warp_scratch[lane] = wi - w;      // exclusive warp offsets
        if (lane == NW - 1) warp_scratch[NW] = wi;       // block total
    }
    __syncthreads();
    *total = warp_scratch[NW];
    return warp_scratch[warp] + incl - x;
}

// Segmented-sum scan element: (any head seen, sum since the last head); used by S3 (reduce.cu, finish.cu).
struct SegPair {
    uint32_t f;
    double v;
};
__device__ __forceinline__ SegPair seg_combine(const SegPair& l, const SegPair& r)
{
    SegPair o;
    o.f = l.f | r.f;
    o.v = r.f ? r.v : __dadd_rn(l.v, r.v);
    return o;
}

// Decoupled look-back over single-word tile states: word = (value << 2) | flag.
constexpr uint32_t kFlagInvalid = 0, kFlagPartial = 1, kFlagInclusive = 2;

// Called by ONE warp of the block.  Publishes `count` for tile `tile`, walks back over the
// predecessors (32 at a time) and returns the sum of the counts of tiles < tile (valid in all lanes).
// state[] must be zero before the kernel; tiles are handed out by an atomic ticket so every
// predecessor is resident and makes progress.
__device__ __forceinline__ uint32_t warp_lookback_u32(uint32_t* state, uint32_t tile, uint32_t count)
{
    const unsigned lane = lane_id();
    if (tile == 0) {
        if (lane == 0) st_volatile_u32(&state[0], (count << 2) | kFlagInclusive);
        return 0u;
    }
    if (lane == 0) st_volatile_u32(&state[tile], (count << 2) | kFlagPartial);
    uint32_t excl = 0;
    int64_t base = (int64_t)tile - 1;                  // lane l looks at tile base - l
    while (true) {
        const int64_t t = base - lane;
        uint32_t w = kFlagInclusive;                   // tiles before 0: inclusive, value 0
        if (t >= 0) {
            do { w = ld_volatile_u32(&state[t]); } while ((w & 3u) == kFlagInvalid);
        }
        const unsigned incl_mask = __ballot_sync(kFullMask, (w & 3u) == kFlagInclusive);
        // lanes up to and including the nearest inclusive one contribute
        const int stop = incl_mask ? (__ffs(incl_mask) - 1) : 31;
        uint32_t v = (lane <= (unsigned)stop) ? (w >> 2) : 0u;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(kFullMask, v, o);
        excl += v;
        if (incl_mask) break;
        base -= 32;
    }
    if (lane == 0) st_volatile_u32(&state[tile], ((excl + count) << 2) | kFlagInclusive);
    return excl;
}

}  // namespace polylab
