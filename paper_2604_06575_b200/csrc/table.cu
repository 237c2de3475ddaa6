// table.cu -- the low-cardinality fast path: when far fewer distinct monomials than terms are
// expected, the like terms are merged in a table BEFORE any sort, and only the U distinct monomials are sorted.
//
// This is the paper's own regime -- "coefficient aggregation, repeated-term merging" after "large intermediate symbolic
// expansions" (section 6.3): simplify(p_4^3) takes 2,000,376 raw product terms to 6188.
//
//   table_insert_kernel   every record finds its slot -- the packed key itself when 2^B slots are affordable (DENSE), else
//                         an open-addressing hash table on the 64-bit key (linear probing, atomicCAS) -- and raises the
//                         slot's MAXIMUM COEFFICIENT EXPONENT (atomicMax, almost always skipped after a plain read).  New
//                         keys receive dense ordinals 0..U-1; more than `limit` of them (collapse below 4x) sets
//                         `overflow` and the call continues on the sort path.
//   table_accum_kernel    every record is added to its monomial's accumulator as a FIXED-POINT integer relative to that
//                         maximum exponent: two signed 64-bit limbs of p bits each (p = 62 - ceil(log2 N) >= 36), integer
//                         atomics.  Integer addition is associative and commutative, so the sum does not depend on the
//                         order in which the hardware performs the atomics: results are bit-reproducible and invariant
//                         under permutations of the input.  A term within 2^-(2p-53) of its monomial's largest term is
//                         represented exactly; smaller ones are truncated at 2^-(2p-1) of the largest, so
//                         |s - exact| <= n_m * 2^-(2p-1) * A_m + 3 * 2^-53 |s|  <=  2^-45 * A_m for N <= 2^26 (the path's
//                         limit), inside north_star's 1e-12 * A_m.  The first 8192 ordinals are accumulated in shared
//                         memory (a 64-bit add is two native 32-bit atomics chained by the carry the first one returns),
//                         the rest by red.global.add.u64.
//   table_finalize_kernel (hash) turns every slot into (key, fp64 sum) at its ordinal; the U pairs then go through the
//                         ordinary radix sort / prune / unpack of sort.cu and reduce.cu -- a sort of U, not of N.
//   table_dense_emit_kernel (dense) walks the 2^B slots in index order -- which IS the canonical monomial order -- with
//                         the prune (S4), an order-preserving compaction (decoupled look-back) and the unpack (S5).
//
// Non-finite coefficients (reading A12): a slot whose maximum exponent is 2047 only records which of +inf, -inf, NaN it
// saw; its sum is +-inf, or NaN (dropped by the prune) for NaN or inf - inf, as an IEEE sum in any order would give.
#include "kernels.h"

namespace polylab {

constexpr uint32_t kMetaNonFinite = 2048u;             // meta = biased exponent + 1; 2047 + 1 marks inf / NaN

__device__ __forceinline__ uint32_t hash_key(uint64_t k)
{
    k ^= k >> 33; k *= 0xff51afd7ed558ccdull; k ^= k >> 33; k *= 0xc4ceb9fe1a85ec53ull; k ^= k >> 33;
    return (uint32_t)k;
}

__device__ __forceinline__ uint32_t coef_meta(double c) { return (uint32_t)((__double_as_longlong(c) >> 52) & 0x7ff) + 1u; }

// record q of the source: (key, coefficient).  PRODUCTS: term-product expansion X1 on packed operands, in registers.
template <bool PRODUCTS>
__device__ __forceinline__ void load_record(const TableSrc& s, uint32_t q, uint64_t& key, double& c)
{
    if (PRODUCTS) {
        const uint32_t i = q / s.nb, j = q - i * s.nb;
        key = ((const uint64_t*)s.ka)[i] + ((const uint64_t*)s.kb)[j];      // fields never carry into each other (plan)
        c = __dmul_rn(s.ca[i], s.cb[j]);                                    // one IEEE multiplication, never contracted
    } else {
        key = s.keys[q];
        c = s.coef[q];
    }
}

// slot of `key`: DENSE -> the key; hash -> linear probing, one 16-byte load per probe (key, ordinal, meta together).
// INSERT claims an empty slot (stored key + 1, 0 = empty).  The loads of the insert pass may be served by L1: a stored key
// never changes, so a cached non-zero key is right for ever and a stale zero only sends the lane to the atomicCAS, which
// returns the truth; a stale meta is only ever too LOW and costs a redundant atomicMax.  The accumulate pass reads a
// table that no longer changes (ld.global.nc).  Returns false when the probe limit is hit (the caller raises `overflow`).
template <bool DENSE, bool INSERT>
__device__ __forceinline__ bool find_slot(const TableArgs& t, uint64_t key, uint32_t& slot, bool& inserted, uint32_t& ord, uint32_t& meta)
{
    inserted = false;
    if (DENSE) {
        slot = ord = (uint32_t)key;
        if (INSERT) asm volatile("ld.global.ca.u32 %0, [%1];" : "=r"(meta) : "l"(t.meta + slot));
        else meta = __ldg(t.meta + slot);
        return true;
    }
    const uint64_t want = key + 1ull;
    uint32_t h = hash_key(key) & t.cmask;
    for (int probe = 0; probe < 256; ++probe) {
        uint4 q;
        if (INSERT) asm volatile("ld.global.ca.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(q.x), "=r"(q.y), "=r"(q.z), "=r"(q.w) : "l"(t.slots + h));
        else q = __ldg((const uint4*)(t.slots + h));
        uint64_t cur = ((uint64_t)q.y << 32) | q.x;
        if (INSERT && cur == 0ull) {
            cur = atomicCAS((unsigned long long*)&t.slots[h].key1, 0ull, (unsigned long long)want);
            if (cur == 0ull) { inserted = true; cur = want; }
            q.w = 0u;                                       // (a meta read beside an empty key says nothing)
        }
        if (cur == want) { slot = h; ord = q.z; meta = q.w; return true; }
        if (!INSERT && cur == 0ull) return false;           // cannot happen after a complete insert pass
        h = (h + 1u) & t.cmask;
    }
    return false;
}

constexpr int kTabThreads = 256;
constexpr int kTabItems = 8;
constexpr int kTabTile = kTabThreads * kTabItems;

// One record of the insert pass; called by all 32 lanes of a warp together (`valid` masks the tail).
template <bool DENSE>
__device__ __forceinline__ void insert_record(const TableArgs& t, bool valid, uint64_t key, double c, unsigned lane)
{
    uint32_t slot = 0, ord_unused, meta = 0;
    bool ins = false, ok = true;
    if (valid) ok = find_slot<DENSE, true>(t, key, slot, ins, ord_unused, meta);
    if (!DENSE) {
        // dense ordinals for the new keys: one atomicAdd per warp instruction
        const unsigned m = __ballot_sync(kFullMask, ins);
        if (m) {
            uint32_t b = 0;
            if (lane == (unsigned)(__ffs(m) - 1)) b = atomicAdd(&t.ctl->tab_count, (uint32_t)__popc(m));
            b = __shfl_sync(kFullMask, b, __ffs(m) - 1);
            if (ins) t.slots[slot].ord = b + __popc(m & lanemask_lt());
            if (b + __popc(m) > t.limit) t.ctl->tab_overflow = 1u;
        }
        if (!ok) t.ctl->tab_overflow = 1u;
    }
    if (valid && ok) {
        const uint32_t e = coef_meta(c);
        if (meta < e) atomicMax(DENSE ? &t.meta[slot] : &t.slots[slot].meta, e);
    }
}

template <bool PRODUCTS, bool DENSE>
__global__ void __launch_bounds__(kTabThreads) table_insert_kernel(const __grid_constant__ TableSrc src, const __grid_constant__ TableArgs t)
{
    const unsigned lane = lane_id();
    const uint32_t ntiles = (src.n + kTabTile - 1) / kTabTile;
    for (uint32_t tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
        if (!DENSE) {                                       // abandoned by another block: stop (warp-uniform decision)
            const uint32_t ov = __shfl_sync(kFullMask, lane == 0 ? *(volatile uint32_t*)&t.ctl->tab_overflow : 0u, 0);
            if (ov) return;
        }
        const uint32_t base = tile * kTabTile + threadIdx.x;
#pragma unroll 2
        for (int k = 0; k < kTabItems; ++k) {
            const uint32_t q = base + k * kTabThreads;
            const bool valid = q < src.n;
            uint64_t key = 0;
            double c = 0.0;
            if (valid) load_record<PRODUCTS>(src, q, key, c);
            insert_record<DENSE>(t, valid, key, c, lane);
        }
    }
}

// S1 fused into the insert pass (simplify with contiguous row-major exponent rows): a tile of rows comes into shared memory
// by double-buffered 16-byte cp.async copies exactly as in pack_rows_staged_kernel (pack.cu); each thread packs its row,
// stores the key -- the accumulate pass and, should the table be abandoned, the sort path read it -- and inserts it.  Saves
// the pack kernel's launch and one read of the keys.  Blocks never stop early here (every key must be written); once the
// table is abandoned they stop inserting.
template <int ES, bool DENSE>
__global__ void __launch_bounds__(kTabThreads) table_insert_rows_kernel(const uint8_t* __restrict__ base, int64_t nterms, int tile_rows,
                                                                        const __grid_constant__ Plan plan, uint64_t* __restrict__ keys,
                                                                        CoefIn coef, const __grid_constant__ TableArgs t, int hd)
{
    extern __shared__ __align__(16) unsigned char stage[];          // two buffers of tile_rows * row bytes + 16
    __shared__ uint32_t sh[kRadix];
    const unsigned lane = lane_id();
    for (int b = threadIdx.x; b < kRadix; b += kTabThreads) sh[b] = 0u;
    const int rb = plan.nvars * ES;
    const int dpos = plan.digit_pos[hd >= 0 ? hd : 0];
    const uint32_t dmask = (1u << plan.digit_bits[hd >= 0 ? hd : 0]) - 1u;
    const int64_t nbytes = nterms * rb;
    const int bufsz = (tile_rows * rb + 16 + 15) & ~15;
    const int64_t step = (int64_t)gridDim.x * tile_rows;
    auto issue = [&](int buf, int64_t t0) {
        if (t0 < nterms) {
            const int nr = (int)min((int64_t)tile_rows, nterms - t0);
            const int64_t b0 = t0 * rb, b1 = b0 + (int64_t)nr * rb, a0 = b0 & ~(int64_t)15;
            unsigned char* dst = stage + (size_t)buf * bufsz;
            for (int64_t off = a0 + 16 * (int64_t)threadIdx.x; off < b1; off += 16 * kTabThreads) {
                if (off + 16 <= nbytes) cp_async16(dst + (off - a0), base + off);
                else for (int64_t b = off; b < nbytes; ++b) dst[b - a0] = base[b];
            }
        }
        asm volatile("cp.async.commit_group;" ::: "memory");
    };
    bool bad = false;
    int64_t t0 = (int64_t)blockIdx.x * tile_rows;
    issue(0, t0);
    for (int it = 0; t0 < nterms; ++it, t0 += step) {
        const int cur = it & 1;
        issue(cur ^ 1, t0 + step);
        asm volatile("cp.async.wait_group 1;" ::: "memory");
        __syncthreads();
        const int nr = (int)min((int64_t)tile_rows, nterms - t0);
        const int64_t b0 = t0 * rb, a0 = b0 & ~(int64_t)15;
        const unsigned char* src = stage + (size_t)cur * bufsz + (b0 - a0);
        // once the table is abandoned the block only packs (a full table would cost 256 probes per record); warp-uniform
        const bool live = DENSE || __shfl_sync(kFullMask, lane == 0 ? *(volatile uint32_t*)&t.ctl->tab_overflow : 0u, 0) == 0u;
        for (int r0 = 0; r0 < nr; r0 += kTabThreads) {               // every lane of a warp takes part in insert_record
            const int r = r0 + (int)threadIdx.x;
            const bool valid = r < nr;
            uint64_t key = 0;
            double c = 0.0;
            if (valid) {
                const unsigned char* row = src + (int64_t)r * rb;
                for (int v = 0; v < plan.nvars; ++v) {
                    const uint32_t e = ES == 1 ? row[v] : ES == 2 ? ((const uint16_t*)row)[v] : ((const uint32_t*)row)[v];
                    pack_field(key, e, v, plan, bad);
                }
                keys[t0 + r] = key;
                c = coef[(size_t)(t0 + r)];
                if (hd >= 0) atomicAdd(&sh[key_digit(key, dpos, dmask)], 1u);
            }
            if (live) insert_record<DENSE>(t, valid, key, c, lane);
        }
        __syncthreads();
    }
    asm volatile("cp.async.wait_group 0;" ::: "memory");
    if (bad) atomicMax(&t.ctl->status, (int)POLYLAB_ERR_EXPONENT_RANGE);
    if (hd >= 0) {
        __syncthreads();
        for (int b = threadIdx.x; b < kRadix; b += kTabThreads)
            if (sh[b]) atomicAdd(&t.ctl->hist[hd][b], sh[b]);
    }
}

// c as two signed p-bit limbs relative to the slot's maximum exponent E (biased, 1..2046; zero / denormal slots use 1):
// x = c * 2^(1022 - E) has |x| < 1;  hi = trunc(x * 2^p),  lo = trunc((x * 2^p - hi) * 2^p).  Every step is an exact scaling
// or an exact subtraction; only the final truncation drops bits (below 2^-2p of the scale).
__device__ __forceinline__ void to_fixed(double c, uint32_t meta, int p, long long& hi, long long& lo)
{
    const int E = max((int)meta - 1, 1);
    const int k = 1022 - E + p, k1 = k >> 1, k2 = k - k1;                           // 2^k in two normal factors
    const double f1 = __longlong_as_double((long long)(k1 + 1023) << 52), f2 = __longlong_as_double((long long)(k2 + 1023) << 52);
    const double y = __dmul_rn(__dmul_rn(c, f1), f2);   // |y| < 2^p, exact
    hi = (long long)y;                                  // truncation (cvt.rzi)
    const double r = __dsub_rn(y, (double)hi);          // exact, |r| < 1
    lo = (long long)__dmul_rn(r, __longlong_as_double((long long)(p + 1023) << 52));
}

__device__ __forceinline__ double from_fixed(long long hi, long long lo, uint32_t meta, int p)
{
    if (meta >= kMetaNonFinite) {                       // hi holds the flags: 1 = +inf seen, 2 = -inf seen, 4 = NaN seen
        const unsigned f = (unsigned)hi & 7u;
        if ((f & 4u) || (f & 3u) == 3u) return __longlong_as_double(0x7ff8000000000000ll);
        return (f & 1u) ? __longlong_as_double(0x7ff0000000000000ll) : __longlong_as_double((long long)0xfff0000000000000ull);
    }
    const int E = max((int)meta - 1, 1);
    const __int128 v = ((__int128)hi << p) + (__int128)lo;
    const long long top = (long long)(v >> 64);
    const unsigned long long bot = (unsigned long long)v;
    const double d = __dadd_rn(__dmul_rn((double)top, 18446744073709551616.0), (double)bot);
    return scalbn(d, E - 1022 - 2 * p);
}

__device__ __forceinline__ void red_add_u64(unsigned long long* p, long long v)
{
    asm volatile("red.global.add.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}
__device__ __forceinline__ void red_or_u64(unsigned long long* p, unsigned long long v)
{
    asm volatile("red.global.or.b64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}

// 64-bit add into shared memory with two native 32-bit atomics: the low word's old value tells whether this very
// addition carried (the low-word atomics are totally ordered, so the carries add up to the carries of the exact sum)
__device__ __forceinline__ void smem_add64(uint32_t* w, long long v)
{
    const uint32_t vl = (uint32_t)v, vh = (uint32_t)((unsigned long long)v >> 32);
    const uint32_t old = atomicAdd(&w[0], vl);
    const uint32_t carry = (old + vl < old) ? 1u : 0u;
    if (vh + carry) atomicAdd(&w[1], vh + carry);
}

constexpr int kAccThreads = 1024;
constexpr int kAccSlots = 8192;                         // ordinals accumulated in shared memory: 8192 * 16 bytes

template <bool PRODUCTS, bool DENSE>
__global__ void __launch_bounds__(kAccThreads, 1) table_accum_kernel(const __grid_constant__ TableSrc src, const __grid_constant__ TableArgs t)
{
    extern __shared__ __align__(16) uint32_t sm[];      // [kAccSlots][4]: hi.lo32, hi.hi32, lo.lo32, lo.hi32
    const uint32_t nsm = t.nsm;                        // ordinals accumulated in shared memory (0: none, the launch has no shared memory)
    for (uint32_t i = threadIdx.x; i < nsm * 4u; i += blockDim.x) sm[i] = 0u;
    __syncthreads();
    const uint32_t stride = gridDim.x * blockDim.x;
    for (uint32_t q0 = blockIdx.x * blockDim.x + threadIdx.x; q0 < src.n; q0 += 4 * stride) {
        uint64_t key[4];
        double c[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            key[u] = 0; c[u] = 0.0;
            if (q0 + u * stride < src.n) load_record<PRODUCTS>(src, q0 + u * stride, key[u], c[u]);
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const uint32_t q = q0 + u * stride;
            if (q >= src.n) continue;
            uint32_t slot = 0, ord = 0, meta = 0;
            bool ins;
            if (!find_slot<DENSE, false>(t, key[u], slot, ins, ord, meta)) { t.ctl->unsorted = 1u; continue; }     // a key the insert pass did not see
            if (meta >= kMetaNonFinite) {
                const long long bits = __double_as_longlong(c[u]);
                if (coef_meta(c[u]) >= kMetaNonFinite)
                    red_or_u64(&t.acc_hi[ord], (bits & 0x000fffffffffffffll) ? 4ull : (bits < 0 ? 2ull : 1ull));
                continue;
            }
            long long hi, lo;
            to_fixed(c[u], meta, t.p, hi, lo);
            if (ord < nsm) {
                if (hi) smem_add64(&sm[ord * 4u], hi);
                if (lo) smem_add64(&sm[ord * 4u + 2u], lo);
            } else {
                if (hi) red_add_u64(&t.acc_hi[ord], hi);
                if (lo) red_add_u64(&t.acc_lo[ord], lo);
            }
        }
    }
    __syncthreads();
    for (uint32_t i = threadIdx.x; i < nsm; i += blockDim.x) {
        const uint4 w = *(const uint4*)&sm[i * 4u];
        const long long hi = (long long)(((unsigned long long)w.y << 32) | w.x), lo = (long long)(((unsigned long long)w.w << 32) | w.z);
        if (hi) red_add_u64(&t.acc_hi[i], hi);
        if (lo) red_add_u64(&t.acc_lo[i], lo);
    }
}

// hash table -> (key, sum)[U] at the slots' ordinals
__global__ void __launch_bounds__(256) table_finalize_kernel(const __grid_constant__ TableArgs t, uint64_t* __restrict__ ukeys,
                                                             double* __restrict__ usums)
{
    const uint32_t cap = t.cmask + 1u;
    for (uint32_t h = blockIdx.x * blockDim.x + threadIdx.x; h < cap; h += gridDim.x * blockDim.x) {
        const TableSlot s = t.slots[h];
        if (s.key1 == 0ull) continue;
        ukeys[s.ord] = s.key1 - 1ull;
        usums[s.ord] = from_fixed((long long)t.acc_hi[s.ord], (long long)t.acc_lo[s.ord], s.meta, t.p);
    }
}

// dense table -> output: slots in index order are the monomials in canonical order
constexpr int kDenseThreads = 256;
constexpr int kDenseItems = 8;
constexpr int kDenseTile = kDenseThreads * kDenseItems;

__global__ void __launch_bounds__(kDenseThreads) table_dense_emit_kernel(const __grid_constant__ TableArgs t, const __grid_constant__ Plan plan,
                                                                         double tol, CoefOut out_coef, void* out_exps,
                                                                         int exp_bytes, int wpr, int64_t out_capacity, uint32_t* tile_state,
                                                                         int64_t* out_count_device)
{
    constexpr int NW = kDenseThreads / 32;
    __shared__ uint32_t scratch[NW + 2];
    __shared__ uint32_t sm_tile, sm_base;
    const unsigned tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
    const uint32_t nslots = t.nord;
    const uint32_t ntiles = (nslots + kDenseTile - 1) / kDenseTile;
    while (true) {
        __syncthreads();
        if (tid == 0) sm_tile = atomicAdd(&t.ctl->ticket[kTicketPrune], 1u);
        __syncthreads();
        const uint32_t tile = sm_tile;
        if (tile >= ntiles) break;
        const uint32_t first = tile * kDenseTile + tid * kDenseItems;
        double s[kDenseItems];
        uint32_t keep = 0, cnt = 0, present = 0;
#pragma unroll
        for (int j = 0; j < kDenseItems; ++j) {
            const uint32_t k = first + j;
            s[j] = 0.0;
            if (k < nslots) {
                const uint32_t meta = t.meta[k];
                if (meta) {
                    ++present;
                    s[j] = from_fixed((long long)t.acc_hi[k], (long long)t.acc_lo[k], meta, t.p);
                    if (fabs(s[j]) > tol) { keep |= 1u << j; ++cnt; }                  // NaN compares false: dropped (A12)
                }
            }
        }
        uint32_t total;
        const uint32_t excl = block_exclusive_scan<kDenseThreads>(cnt | (present << 16), scratch, &total);
        if (warp == 0) {
            const uint32_t r = warp_lookback_u32(tile_state, tile, total & 0xffffu);
            if (lane == 0) sm_base = r;
        }
        __syncthreads();
        uint64_t o = (uint64_t)sm_base + (excl & 0xffffu);
#pragma unroll
        for (int j = 0; j < kDenseItems; ++j) {
            if (keep & (1u << j)) {
                if ((int64_t)o < out_capacity) {
                    out_coef.store(o, s[j]);
                    const uint64_t kk = first + j;
                    if (wpr > 0) {
                        uint32_t* row = (uint32_t*)out_exps + o * (uint64_t)wpr;
                        for (int w = 0; w < wpr; ++w) row[w] = unpack_row_word(plan, kk, w, exp_bytes);
                    } else {
                        for (int v = 0; v < plan.nvars; ++v)
                            store_exp(out_exps, exp_bytes, (int64_t)o * plan.nvars + v, key_get_field(kk, plan.shift[v], plan.width[v]));
                    }
                }
                ++o;
            }
        }
        if (tid == 0) {
            if (total >> 16) atomicAdd(&t.ctl->distinct, total >> 16);
            if (tile == ntiles - 1) {
                t.ctl->survivors = sm_base + (total & 0xffffu);
                if (out_count_device) *out_count_device = (int64_t)(sm_base + (total & 0xffffu));
            }
        }
    }
}

// ---------------------------------------------------------------------------------------- launchers

int launch_table_insert(const TableSrc& src, const TableArgs& t, bool dense, cudaStream_t stream)
{
    if (src.n == 0) return 0;
    int64_t blocks = ((int64_t)src.n + kTabTile - 1) / kTabTile;
    if (blocks > sm_count() * 8) blocks = sm_count() * 8;
    const bool prod = src.keys == nullptr;
    if (prod) { if (dense) table_insert_kernel<true, true><<<(unsigned)blocks, kTabThreads, 0, stream>>>(src, t); else table_insert_kernel<true, false><<<(unsigned)blocks, kTabThreads, 0, stream>>>(src, t); }
    else { if (dense) table_insert_kernel<false, true><<<(unsigned)blocks, kTabThreads, 0, stream>>>(src, t); else table_insert_kernel<false, false><<<(unsigned)blocks, kTabThreads, 0, stream>>>(src, t); }
    return 1;
}

int launch_table_insert_rows(const ExpView& ev, int64_t nterms, const Plan& plan, uint64_t* keys, CoefIn coef, const TableArgs& t,
                             bool dense, int hd, cudaStream_t stream)
{
    if (nterms <= 0) return 0;
    const int rb = plan.nvars * ev.exp_bytes;
    int tile_rows = 16384 / rb;                              // at most 16 KB of rows per tile, two tiles in shared memory
    tile_rows = tile_rows > 1024 ? 1024 : tile_rows < 32 ? 32 : tile_rows / 32 * 32;
    int64_t blocks = (nterms + tile_rows - 1) / tile_rows;
    if (blocks > sm_count() * 6) blocks = sm_count() * 6;
    const size_t smem = 2 * (((size_t)tile_rows * rb + 16 + 15) & ~(size_t)15);
    const uint8_t* base = (const uint8_t*)ev.base;
#define POLYLAB_TIR(ES, D) table_insert_rows_kernel<ES, D><<<(unsigned)blocks, kTabThreads, smem, stream>>>(base, nterms, tile_rows, plan, keys, coef, t, hd)
    if (ev.exp_bytes == 1) { if (dense) POLYLAB_TIR(1, true); else POLYLAB_TIR(1, false); }
    else if (ev.exp_bytes == 2) { if (dense) POLYLAB_TIR(2, true); else POLYLAB_TIR(2, false); }
    else { if (dense) POLYLAB_TIR(4, true); else POLYLAB_TIR(4, false); }
#undef POLYLAB_TIR
    return 1;
}

int launch_table_accum(const TableSrc& src, const TableArgs& t_in, bool dense, cudaStream_t stream)
{
    if (src.n == 0) return 0;
    // Hash table: ordinals are handed out in order of first appearance, so the monomials that occur most often get the
    // lowest ones with high probability -- the first 8192 are accumulated in shared memory by one block of 1024 threads per SM
    // (same-address global atomics serialise at ~35 cycles each: config 4's constant term alone is hit 3e5 times).  Dense
    // table: a slot index says nothing about frequency, so beyond 8192 slots everything goes to global memory, from eight
    // blocks of 256 threads per SM.
    TableArgs t = t_in;
    t.nsm = (!dense || t.nord <= (uint32_t)kAccSlots) ? (t.nord < (uint32_t)kAccSlots ? t.nord : (uint32_t)kAccSlots) : 0u;
    const int threads = t.nsm ? kAccThreads : 256;
    int64_t blocks = ((int64_t)src.n + threads * 4 - 1) / (threads * 4);
    const int64_t maxb = t.nsm ? sm_count() : sm_count() * 8;
    if (blocks > maxb) blocks = maxb;
    const size_t smem = (size_t)t.nsm * 16;
    const bool prod = src.keys == nullptr;
    auto go = [&](auto kern) {
        ensure_dynamic_smem(kern, (size_t)((size_t)kAccSlots * 16));
        kern<<<(unsigned)blocks, threads, smem, stream>>>(src, t);
    };
    if (prod) { if (dense) go(table_accum_kernel<true, true>); else go(table_accum_kernel<true, false>); }
    else { if (dense) go(table_accum_kernel<false, true>); else go(table_accum_kernel<false, false>); }
    return 1;
}

int launch_table_finalize(const TableArgs& t, uint64_t* ukeys, double* usums, cudaStream_t stream)
{
    int64_t blocks = ((int64_t)t.cmask + 1 + 255) / 256;
    if (blocks > sm_count() * 16) blocks = sm_count() * 16;
    table_finalize_kernel<<<(unsigned)blocks, 256, 0, stream>>>(t, ukeys, usums);
    return 1;
}

int launch_table_dense_emit(const TableArgs& t, const Plan& plan, double tol, CoefOut out_coef, void* out_exps, int exp_bytes,
                            int64_t out_capacity, uint32_t* tile_state, int64_t* out_count_device, cudaStream_t stream)
{
    int64_t blocks = ((int64_t)t.nord + kDenseTile - 1) / kDenseTile;
    if (blocks > sm_count() * 8) blocks = sm_count() * 8;
    if (blocks < 1) blocks = 1;
    table_dense_emit_kernel<<<(unsigned)blocks, kDenseThreads, 0, stream>>>(t, plan, tol, out_coef, out_exps, exp_bytes,
                                                                          row_words(plan.nvars, exp_bytes, out_exps), out_capacity, tile_state,
                                                                          out_count_device);
    return 1;
}

}  // namespace polylab
