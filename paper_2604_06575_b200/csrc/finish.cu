// finish.cu -- the "bucket path" of step S2 and steps S3-S5 fused behind it.
//
// An LSD radix sort reads and writes every (key, coefficient) pair once per digit: 16 times for a 128-bit key.
// When the most significant digits spread the keys evenly, that is wasted traffic: k stable passes over the TOP k
// digits alone (the same sort_pass_kernel, most significant digits only) leave the array partitioned into buckets
// of keys that share their top T bits, in ascending bucket order, and a bucket that fits shared memory can be
// finished on chip.  This file is that finish:
//
//   tile_bounds_kernel   cuts the prefix-sorted array into tiles of whole buckets: tile t owns the buckets that
//                        START in positions [t*TILE, (t+1)*TILE); a tile's start is found by a binary search for the
//                        first change of prefix at or after t*TILE.  A bucket longer than CAP - TILE sets
//                        ctl->overflow and the call falls back to the plain LSD path.  TILE is chosen per call
//                        (api.cu): CAP minus room for the longest bucket expected from N / 2^T.  Tiles that own
//                        records go on a work list; every tile start is checked to be a strict prefix increase.
//   finish_group_kernel  (round 2) tried first on every work-list tile: like terms are grouped through a shared-memory hash
//                        table, only the tile's distinct keys are put in order, one stable counting pass places the
//                        records; the tiles it finishes are marked in the work list, finish_kernel does the rest (see the
//                        comment above the kernel; bit-identical results).
//   finish_kernel        one block per work-list tile (<= CAP = 4608 records, 256 threads, four blocks per SM).
//                        Shared memory holds 10 bytes per record, not the record: two 32-bit ping-pong buffers of sort
//                        elements (record index in the low 13 bits, the not yet consumed sort bits above) and one
//                        16-bit array (head flags -> bucket ordinals -> ranks -> final permutation).  The block
//                        streams its keys once (bucket heads, the key bits below the prefix), builds the composite
//                        sort word "bucket ordinal above the top key bits" (<= 27 bits), sorts it with stable
//                        counting-sort passes on 9-bit digits, brings the coefficients into sorted order through the
//                        inverse permutation (coalesced read), gathers the keys through the permutation (L2 hits),
//                        and -- records of equal monomials now being adjacent and no run crossing a tile -- does the
//                        segmented sum (S3) and the prune (S4, keep iff |s| > tol, reading A2) and leaves the tile's
//                        survivors compacted in order at the tile's own position.  Tiles are independent (no
//                        look-back: a tile only knows its count at the very end, and waiting in order for slow
//                        predecessors left SMs idle).
//   tile_sum_kernel, tile_scan_kernel   exclusive scan of the tiles' survivor counts (chunk sums, then the scan).
//   emit_kernel          S5: one warp per work-list tile copies the tile's survivors to the tile's scanned offset and
//                        unpacks the keys into the caller's output -- order-preserving compaction across tiles.
//                        HBM traffic of all of them: N*(W+8) read, U'*(W+8) written and read, U'*(8+E) written.
//
// The local sort first uses only as many key bits below the prefix as fit the composite sort word (enough to separate
// the distinct keys of a bucket unless two of them share all those bits) and checks the order against the full keys
// while it computes the head flags; a tile that fails the check re-sorts on every bit below the prefix, 18 at a time,
// cutting them out of the keys through the current permutation (ctl->refinish counts such tiles).
//
// Summation order (reading A6): equal keys keep their input order through every stable step; a tile sums left to
// right inside a thread and by a fixed shuffle tree across threads -- a function of the data layout only, so
// results are bit-reproducible run to run (the work list's order varies, the tiles' results do not).
#include "kernels.h"

namespace polylab {

// ------------------------------------------------------------------------------------- tile bounds

// start of tile t: the first position >= t*fin_tile where the prefix changes (0 for t = 0, n past the end)
template <typename K>
__device__ __forceinline__ uint32_t tile_first_change(const K* __restrict__ keys, uint32_t n, int pfx_pos, uint32_t fin_tile,
                                                      uint32_t t, bool* overflow)
{
    if (t == 0) return 0u;
    const uint64_t s64 = (uint64_t)t * fin_tile;
    if (s64 >= n) return n;
    const uint32_t s = (uint32_t)s64;
    const K ref = keys[s - 1];
    uint32_t lo = s, hi = (uint32_t)min((uint64_t)n, s64 + (uint64_t)(kFinCap - fin_tile));
    if (hi < n && same_prefix(keys[hi], ref, pfx_pos)) {      // the bucket of record s-1 runs past what a tile can own
        *overflow = true;
        return s;
    }
    while (lo < hi) {                                         // smallest p in [lo, hi] whose prefix differs (p == n counts)
        const uint32_t mid = lo + (hi - lo) / 2;
        if (same_prefix(keys[mid], ref, pfx_pos)) lo = mid + 1;
        else hi = mid;
    }
    return lo;
}

template <typename K>
__global__ void __launch_bounds__(256) tile_bounds_kernel(const K* __restrict__ keys, uint32_t n, int pfx_pos,
                                                          uint32_t fin_tile, uint32_t ntiles,
                                                          uint32_t* __restrict__ tile_start, uint4* __restrict__ worklist,
                                                          Control* ctl)
{
    const uint32_t t = blockIdx.x * blockDim.x + threadIdx.x;
    bool overflow = false, owns = false;
    uint32_t lo = 0, hi = 0;
    if (t <= ntiles) {
        lo = tile_first_change(keys, n, pfx_pos, fin_tile, t, &overflow);
        tile_start[t] = lo;
        if (t < ntiles) {
            hi = tile_first_change(keys, n, pfx_pos, fin_tile, t + 1, &overflow);
            owns = (uint64_t)lo < ((uint64_t)t + 1) * fin_tile && hi > lo;        // a bucket starts inside the tile
            // in a prefix-sorted array a tile without a bucket start has lo == hi (both searches find the same change);
            // anything else would leave the records of [lo, hi) to nobody
            if (hi != lo && !owns && !overflow) ctl->unsorted = 1u;
        }
        // a tile starts a new bucket: its first prefix must be above the record before it (finish_kernel checks the
        // order inside a tile; together they prove that every bucket is contiguous, i.e. that the prefix passes were stable)
        if (t > 0 && lo < n && !overflow) {
            const K kb = keys[lo - 1], kf = keys[lo];
            if (!key_lt(kb, kf) || same_prefix(kb, kf, pfx_pos)) ctl->unsorted = 1u;
        }
        if (overflow) ctl->overflow = 1u;
    }
    // work list of the tiles that own records (any order: tiles are independent), one atomic per warp
    const unsigned m = __ballot_sync(kFullMask, owns);
    if (m) {
        const unsigned lane = lane_id();
        uint32_t base = 0;
        if (lane == (unsigned)(__ffs(m) - 1)) base = atomicAdd(&ctl->fin_count, (uint32_t)__popc(m));
        base = __shfl_sync(kFullMask, base, __ffs(m) - 1);
        // tile, first record, end, and whether its first and last record share their prefix (then, if the array is sorted
        // by prefix, the tile holds a single bucket)
        if (owns) worklist[base + __popc(m & lanemask_lt())] = make_uint4(t, lo, hi, same_prefix(keys[lo], keys[hi - 1], pfx_pos) ? 1u : 0u);
    }
}

// --------------------------------------------------------------------------------- local radix pass

struct FinishSmem {
    static constexpr int NW = kFinThreads / 32;
    // [X u32][Y u32]: ping-pong buffers of sort elements, reused for the gathered coefficients (8 bytes per record) once
    // the sort is done; [P u16]: head flags, then bucket ordinals, then the final permutation; per-warp histograms; scratch
    static constexpr size_t off_x = 0;
    static constexpr size_t off_y = (size_t)kFinCap * 4;
    static constexpr size_t off_p = off_y + (size_t)kFinCap * 4;
    static constexpr size_t off_whist = off_p + (size_t)kFinCap * 2;
    // the histogram rows double as the inverse permutation (16 bits per record) between the sort and the sums
    static constexpr size_t whist_bytes = (size_t)NW * kFinBins * 2 > (size_t)kFinCap * 2 ? (size_t)NW * kFinBins * 2 : (size_t)kFinCap * 2;
    static constexpr size_t off_scratch = off_whist + whist_bytes;
    static constexpr size_t bytes = off_scratch + 64 * 4;
};

// One stable counting-sort pass on a digit of `dbits` <= 9 bits.  A sort element is one 32-bit word: the record's index
// in the tile in its low 13 bits, the not yet consumed sort bits above (least significant digit first), so a pass
// reads its input sequentially and never dereferences an index.  FIRST: the input is the composite sort word itself
// (up to 27 bits), position = record index.  Warp w owns the contiguous chunk [w*per, (w+1)*per) of positions and row w of
// the histogram: 512 16-bit counters, two per word, bumped with one shared-memory atomic per record and sweep.
// Sweep 1 counts; the bins are then turned into the first output slot of every (warp, digit) pair; sweep 2 takes slots
// with the same atomic in the same order.  Stability rests on the order in which one warp's shared-memory atomics to
// one word return (lane order within an instruction, program order across instructions: measured on sm_100a,
// profiles/r1b_shared_atomics.md) and is re-verified by the caller's order check.
template <bool FIRST, bool RANKS>
__device__ __forceinline__ void local_pass(const uint32_t* __restrict__ in, uint32_t* __restrict__ out, int dbits, uint32_t n_loc,
                                           uint32_t* whist, uint32_t* scratch, uint16_t* ranks, int pre = 0)
{
    // pre (FIRST only): the input words are shifted right by this before use (a one-bucket tile sorts on the raw key bits
    // as they were cut, without a pass that rewrites them)
    constexpr int NW = FinishSmem::NW, ROW = kFinBins / 2;    // words per histogram row
    constexpr int BPT = kFinBins / kFinThreads;               // bins per thread in the scan step
    static_assert(BPT >= 1 && BPT * kFinThreads == kFinBins, "whole bins per thread in the scan step");
    const unsigned tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
    const uint32_t mask = (1u << dbits) - 1u;
    uint32_t* my_hist = whist + warp * ROW;
    uint16_t* h16 = (uint16_t*)whist;                          // [NW][kFinBins], bin b of warp w at w*kFinBins + b
#pragma unroll
    for (int b = 0; b < ROW / 32; ++b) my_hist[b * 32 + lane] = 0u;
    __syncwarp();
    const uint32_t per = (((n_loc + NW - 1) / NW) + 31u) & ~31u;
    const uint32_t wbeg = min(warp * per, n_loc), wend = min(wbeg + per, n_loc);
    if (RANKS) {
        // sweep 1 counts AND ranks: the atomic's old value is the record's rank among its warp's records of the digit
        for (uint32_t base = wbeg; base < wend; base += 64u) {      // two rounds per iteration: both loads first
            const uint32_t i0 = base + lane, i1 = i0 + 32u;
            const uint32_t e0 = (i0 < wend) ? (FIRST ? in[i0] >> pre : in[i0]) : 0u, e1 = (i1 < wend) ? (FIRST ? in[i1] >> pre : in[i1]) : 0u;
            if (i0 < wend) {
                const uint32_t d = (FIRST ? e0 : (e0 >> 13)) & mask;
                const uint32_t sh = (d & 1u) * 16u;
                ranks[i0] = (uint16_t)(atomicAdd(&my_hist[d >> 1], 1u << sh) >> sh);
            }
            __syncwarp();
            if (i1 < wend) {
                const uint32_t d = (FIRST ? e1 : (e1 >> 13)) & mask;
                const uint32_t sh = (d & 1u) * 16u;
                ranks[i1] = (uint16_t)(atomicAdd(&my_hist[d >> 1], 1u << sh) >> sh);
            }
            __syncwarp();
        }
    } else {
        for (uint32_t i = wbeg + lane; i < wend; i += 32u) {
            const uint32_t d = (FIRST ? (in[i] >> pre) : (in[i] >> 13)) & mask;
            atomicAdd(&my_hist[d >> 1], 1u << ((d & 1u) * 16u));
        }
    }
    __syncthreads();
    {
        uint32_t c[BPT][NW];
        uint32_t count = 0;
#pragma unroll
        for (int q = 0; q < BPT; ++q)
#pragma unroll
            for (int w = 0; w < NW; ++w) c[q][w] = h16[w * kFinBins + tid * BPT + q];
#pragma unroll
        for (int q = 0; q < BPT; ++q)
#pragma unroll
            for (int w = 0; w < NW; ++w) { const uint32_t x = c[q][w]; c[q][w] = count; count += x; }
        uint32_t total;
        const uint32_t bin_start = block_exclusive_scan<kFinThreads>(count, scratch, &total);
#pragma unroll
        for (int q = 0; q < BPT; ++q)
#pragma unroll
            for (int w = 0; w < NW; ++w) h16[w * kFinBins + tid * BPT + q] = (uint16_t)(bin_start + c[q][w]);
    }
    __syncthreads();
    if (RANKS) {
        // sweep 2 needs no atomics and no order: slot = first slot of (warp, digit) + rank
        const uint16_t* my16 = h16 + warp * kFinBins;
#pragma unroll 4
        for (uint32_t i = wbeg + lane; i < wend; i += 32u) {
            const uint32_t e = FIRST ? (in[i] >> pre) : in[i];
            const uint32_t d = (FIRST ? e : (e >> 13)) & mask;
            const uint32_t slot = (uint32_t)my16[d] + ranks[i];
            out[slot] = FIRST ? (i | ((e >> dbits) << 13)) : ((e & 0x1fffu) | ((e >> (13 + dbits)) << 13));
        }
    } else {
        for (uint32_t base = wbeg; base < wend; base += 32u) {
            const uint32_t i = base + lane;
            if (i < wend) {
                const uint32_t e = FIRST ? (in[i] >> pre) : in[i];
                const uint32_t d = (FIRST ? e : (e >> 13)) & mask;
                const uint32_t sh = (d & 1u) * 16u;
                const uint32_t slot = (atomicAdd(&my_hist[d >> 1], 1u << sh) >> sh) & 0xffffu;
                out[slot] = FIRST ? (i | ((e >> dbits) << 13)) : ((e & 0x1fffu) | ((e >> (13 + dbits)) << 13));
            }
            __syncwarp();
        }
    }
    __syncthreads();
}

// all passes over `nbits` sort bits (9 per pass); returns with the result in *cur (swaps *cur / *oth as it goes)
// RANKS: a free 16-bit-per-record array is available for the ranks (fast attempt: the ordinal array is dead once the
// composite sort word exists), which halves the atomics
template <bool FIRST0, bool RANKS>
__device__ __forceinline__ void local_sort_bits(uint32_t** cur, uint32_t** oth, int nbits, uint32_t n_loc, uint32_t* whist,
                                                uint32_t* scratch, uint16_t* ranks, int pre = 0)
{
    bool first = FIRST0;
    for (int done = 0; done < nbits; done += kFinDigit) {
        const int dbits = min(kFinDigit, nbits - done);
        if (first) local_pass<true, RANKS>(*cur, *oth, dbits, n_loc, whist, scratch, ranks, pre);
        else local_pass<false, RANKS>(*cur, *oth, dbits, n_loc, whist, scratch, ranks);
        first = false;
        uint32_t* t = *cur; *cur = *oth; *oth = t;
    }
}

struct FinishArgs {
    const void* keys;
    const double* coefs;
    uint32_t n, ntiles;
    uint32_t fin_tile;              // positions per tile; a tile owns at most kFinCap records
    const uint32_t* tile_start;     // [ntiles + 1]
    uint4* worklist;                // the ctl->fin_count tiles that own records: (tile, first record, end, flags); flag bit 0: first and
                                    // last record share the prefix; bit 1: set by the group kernel when it has finished the tile
    uint32_t max_list;              // group kernel: most tiles that can own records (one per bucket)
    int behind_group;               // finish_kernel: the group kernel ran first -- a smaller grid walks the list in chunks and skips the done tiles
    int no_group;                   // group kernel, test hook: hand every tile on
    uint32_t* tile_state;           // [ntiles + 1] survivors per tile, zero before the kernel
    int pfx_pos;                    // the prefix is the key bits at positions >= pfx_pos
    int fast_bits;                  // most key bits below the prefix the first attempt sorts on (test hook; 32 = no limit)
    double tol;
    void* ukeys;                    // survivors of tile t, compacted in order: (ukeys, usums)[tile_start[t] + q], q < tile_state[t]
    double* usums;
    Control* ctl;
};

struct EmitArgs {
    const void* ukeys;
    const double* usums;
    uint32_t ntiles;
    const uint32_t* tile_start;     // [ntiles + 1]
    const uint32_t* tile_off;       // [ntiles + 1] exclusive scan of the tiles' survivor counts; [ntiles] = U'
    CoefOut out_coef;
    void* out_exps;
    int exp_bytes;
    int wpr;                        // > 0: rows are written as this many 32-bit words (common.cuh, row_words)
    int64_t out_capacity;
    const uint4* worklist;          // the tiles that own records (ctl->fin_count of them, at most max_list processed by finish_kernel)
    uint32_t max_list;
    const Control* ctl;
};

template <typename K>
__device__ __forceinline__ void emit_term(const EmitArgs& a, const Plan& plan, uint64_t o, double s, const K& kk)
{
    a.out_coef.store(o, s);
    if (a.wpr > 0) {
        uint32_t* row = (uint32_t*)a.out_exps + o * (uint64_t)a.wpr;
        for (int w = 0; w < a.wpr; ++w) row[w] = unpack_row_word(plan, kk, w, a.exp_bytes);
        return;
    }
    for (int v = 0; v < plan.nvars; ++v)
        store_exp(a.out_exps, a.exp_bytes, (int64_t)o * plan.nvars + v, key_get_field(kk, plan.shift[v], plan.width[v]));
}

// ------------------------------------------------------------------- S3 + S4 of a tile (shared tail)

// A thread walks `itn` consecutive sorted positions [first, first + itn) of its tile: heads of runs of equal keys, the sum
// since the last head, and S4 for the runs that END inside its stretch.
struct RunState {
    uint32_t hm = 0, nh = 0;            // head mask of the thread's positions, number of heads
    uint32_t keep = 0, nkeep = 0;       // bit k: the k-th run that ends in this thread survives the prune
    uint32_t nclosed = 0;               // runs that end in this thread
    double acc = 0.0, part0 = 0.0;      // sum since the last head; this thread's part of the first run that ends here
};

__device__ __forceinline__ void run_step(RunState& r, bool head, double c, uint32_t j, uint32_t pos, double tol, double* scs)
{
    if (head) {
        // S4 for the run that ENDS here (a run ends where the next head is met): a run that also began in this thread has
        // its whole sum in acc; the first one needs the other threads' part (finish_tail)
        if (pos > 0) {
            if (r.nclosed == 0) r.part0 = r.acc;
            else if (fabs(r.acc) > tol) {                  // NaN compares false: dropped (A12)
                r.keep |= 1u << r.nclosed;
                ++r.nkeep;
                scs[pos - 1] = r.acc;                      // the run's sum, parked on its last record (own position)
            }
            ++r.nclosed;
        }
        r.hm |= 1u << j; ++r.nh; r.acc = c;
    } else r.acc = __dadd_rn(r.acc, c);
}

// Segmented scan across the block, prune, and the tile's survivors compacted in order at the tile's own place.
// key_of(pos, q): the key of the run that ends at sorted position pos, q = the run's ordinal in the tile.
template <typename K, typename KeyOf>
__device__ __forceinline__ void finish_tail(const FinishArgs& a, const RunState& r, double* scs, uint32_t* scratch, uint32_t first,
                                            uint32_t n_loc, uint32_t lo, uint32_t tile, KeyOf key_of)
{
    constexpr int THREADS = kFinThreads, NW = THREADS / 32;
    __shared__ uint32_t wagg_f[NW];
    __shared__ double wagg_v[NW];
    const unsigned tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
    uint32_t keep = r.keep, nkeep = r.nkeep;

    // ---- S3: segmented scan of (has head, sum since last head) across the block; no run crosses a tile
    SegPair incl;
    incl.f = r.nh > 0;
    incl.v = r.acc;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        SegPair l;
        l.f = __shfl_up_sync(kFullMask, incl.f, o);
        l.v = __shfl_up_sync(kFullMask, incl.v, o);
        if (lane >= (unsigned)o) incl = seg_combine(l, incl);
    }
    if (lane == 31) { wagg_f[warp] = incl.f; wagg_v[warp] = incl.v; }
    SegPair carry;                                 // exclusive within the warp
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

    // ---- S4 for the first run that ends in this thread (its head lies in an earlier thread); the run still open at the
    // end of the tile is closed by the last thread, whose inclusive scan value is its sum
    const uint32_t chm = (first == 0) ? (r.hm & ~1u) : r.hm;    // the heads that close a run (every head but the tile's first record)
    if (r.nclosed > 0) {
        const double total0 = __dadd_rn(carry.v, r.part0);
        if (fabs(total0) > a.tol) {
            keep |= 1u;
            ++nkeep;
            scs[first + (__ffs(chm) - 1) - 1] = total0;             // its last record is the one before that head (maybe the previous thread's: nobody else touches it)
        }
    }
    const bool last_keep = (tid == THREADS - 1) && n_loc > 0 && fabs(incl.v) > a.tol;
    // one scan for two counts (each at most CAP < 2^16): survivors in the low half, heads (distinct monomials) in the high half
    uint32_t tile_keep, tot_heads;
    uint32_t kexcl = block_exclusive_scan<THREADS>((nkeep + (last_keep ? 1u : 0u)) | (r.nh << 16), scratch, &tile_keep);
    const uint32_t hexcl = kexcl >> 16;            // heads in the threads before this one
    kexcl &= 0xffffu;
    tot_heads = tile_keep >> 16;
    tile_keep &= 0xffffu;

    // ---- the tile's survivors, compacted in order at the tile's own place; S5 (emit_kernel) puts the tiles together
    {
        K* __restrict__ uk = (K*)a.ukeys + lo;
        double* __restrict__ us = a.usums + lo;
        uint32_t o = kexcl;
        uint32_t k = 0;
        // head number hexcl + k (+ 1 in the thread that holds the tile's first record, whose own head closes nothing)
        // closes run number hexcl + k (- 1 elsewhere)
        uint32_t q = hexcl - (first == 0 ? 0u : 1u);
        for (uint32_t m = chm; m != 0u; m &= m - 1u, ++k, ++q) {    // the runs that end in this thread, in order
            if (keep & (1u << k)) {
                const uint32_t pos = first + (__ffs(m) - 1) - 1;    // the run's last record, where its sum was parked
                us[o] = scs[pos];
                uk[o] = key_of(pos, q);
                ++o;
            }
        }
        if (last_keep) { us[o] = incl.v; uk[o] = key_of(n_loc - 1, tot_heads - 1u); }
    }
    if (tid == 0) {
        if (tot_heads) atomicAdd(&a.ctl->distinct, tot_heads);      // distinct monomials, for the statistics
        a.tile_state[tile] = tile_keep;
    }
}

// ------------------------------------------------------------------------------------ finish kernel

// One work-list tile through the sorting finish: local sort, S3, S4 (the body of finish_kernel).
template <typename K>
__device__ __forceinline__ void finish_tile(const FinishArgs& a, unsigned char* smem_raw, const uint4 wl)
{
    constexpr int THREADS = kFinThreads, CAP = kFinCap;
    static_assert(CAP <= 8192 && CAP / THREADS <= 32, "13-bit record indices in the sort elements, 32-bit head masks");
    uint32_t* bx = (uint32_t*)(smem_raw + FinishSmem::off_x);
    uint32_t* by = (uint32_t*)(smem_raw + FinishSmem::off_y);
    uint16_t* py = (uint16_t*)(smem_raw + FinishSmem::off_p);              // head flags -> ordinals -> final permutation
    uint32_t* whist = (uint32_t*)(smem_raw + FinishSmem::off_whist);
    uint32_t* scratch = (uint32_t*)(smem_raw + FinishSmem::off_scratch);   // [0..NW+1] scans
    double* scs = (double*)smem_raw;               // coefficients in sorted order, over X / Y once the sort is done
    static_assert(FinishSmem::whist_bytes >= (size_t)kFinCap * 2, "the inverse permutation borrows the histogram rows");

    const unsigned tid = threadIdx.x;
    const uint32_t tile = wl.x, lo = wl.y, hi = wl.z;
    const uint32_t n_loc = hi > lo ? min(hi - lo, (uint32_t)CAP) : 0u;
    const K* __restrict__ gkeys = (const K*)a.keys + lo;
    const double* __restrict__ gcoef = a.coefs + lo;
    // sorted positions per thread in the blocked phases; odd, so that the threads' strided shared-memory accesses
    // (stride itn elements) spread over all banks
    const uint32_t itn = ((n_loc + THREADS - 1) / THREADS) | 1u;
    const uint32_t first = tid * itn;
    // pull the tile's keys and coefficients towards L2 now: the key stream below is read in batches and the coefficients
    // only after the sort, and both would otherwise wait out a full DRAM round trip when their turn comes
    for (uint32_t i = tid * 8u; i < n_loc; i += THREADS * 8u)                 // one 128-byte line of keys (64-bit keys: half a line)
        asm volatile("prefetch.global.L2 [%0];" ::"l"(gkeys + i));
    for (uint32_t i = tid * 16u; i < n_loc; i += THREADS * 16u)               // one 128-byte line of coefficients
        asm volatile("prefetch.global.L2 [%0];" ::"l"(gcoef + i));

    // raw sort bits of the fast attempt: the (up to 32) key bits just below the prefix
    const int rbits = min(32, a.pfx_pos);
    bool full = (rbits == 0);                      // nothing below the prefix: only the ordinal is sorted on
    RunState r;
    bool try_single = wl.w != 0u && !full;        // first and last record share the prefix: probably one bucket
    while (true) {
        // ---- stream the keys once: bucket heads and the raw sort bits
        bool descending = false, later_head = false;
        if (try_single) {
            // one-bucket candidate: no neighbour is needed, every prefix must equal the first record's (four records per
            // thread in flight); a record that differs sends the tile through the general stream below
            const K k0 = gkeys[0];
            for (uint32_t i0 = tid; i0 < n_loc; i0 += 4 * THREADS) {
                K k[4];
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    const uint32_t i = i0 + u * THREADS;
                    k[u] = k0;
                    if (i < n_loc) k[u] = gkeys[i];
                }
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    const uint32_t i = i0 + u * THREADS;
                    if (i < n_loc) {
                        later_head |= !same_prefix(k[u], k0, a.pfx_pos);
                        bx[i] = key_get_field(k[u], a.pfx_pos - rbits, rbits);
                    }
                }
            }
            if (__syncthreads_or(later_head ? 1 : 0)) {   // not a single bucket after all (or not sorted): general path
                try_single = false;
                continue;
            }
        } else if (a.pfx_pos >= 8 * (int)sizeof(K) - 64) {
            // the prefix lies in the key's most significant 64 bits: only those are fetched from the left neighbour, and
            // four records per thread are in flight (all loads issued before the first use)
            for (uint32_t i0 = tid; i0 < n_loc; i0 += 4 * THREADS) {
                K k[4];
                uint64_t ph[4];
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    const uint32_t i = i0 + u * THREADS;
                    key_zero(k[u]);
                    ph[u] = 0;
                    if (i < n_loc) {
                        k[u] = gkeys[i];
                        if (i > 0) ph[u] = *(const uint64_t*)(gkeys + (i - 1));     // Key128 is stored (hi, lo)
                    }
                }
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    const uint32_t i = i0 + u * THREADS;
                    if (i < n_loc) {
                        const int hs = a.pfx_pos - (8 * (int)sizeof(K) - 64);              // prefix position inside the top half
                        const uint64_t pk = key_top64(k[u]) >> hs, pp = ph[u] >> hs;
                        const bool head = (i == 0) || pk != pp;
                        descending |= (i > 0) && pk < pp;
                        later_head |= head && i > 0;
                        bx[i] = full ? i : key_get_field(k[u], a.pfx_pos - rbits, rbits);
                        py[i] = head ? 1 : 0;
                    }
                }
            }
        } else {
            for (uint32_t i = tid; i < n_loc; i += THREADS) {
                const K k = gkeys[i];
                bool head = true;
                if (i > 0) {
                    const K kp = gkeys[i - 1];
                    head = !same_prefix(k, kp, a.pfx_pos);
                    descending |= head && key_lt(k, kp);
                    later_head |= head;
                }
                bx[i] = full ? i : key_get_field(k, a.pfx_pos - rbits, rbits);
                py[i] = head ? 1 : 0;
            }
        }
        if (descending) a.ctl->unsorted = 1u;      // the prefix passes were not stable (see sort.cu)
        const bool one_bucket = try_single || (!__syncthreads_or(later_head ? 1 : 0) && !full);

        // ---- bucket ordinal of every record (buckets are contiguous: the input is sorted by prefix); fast attempt:
        // composite sort word = ordinal above the top fb raw bits, ob + fb <= 27 so that 13 index bits fit beside what
        // is left after the first 9-bit pass.  A tile with a single bucket (the usual case when buckets are longer than the
        // tile step) needs neither: it sorts on the raw bits as cut, shifted on the fly by the first pass.
        uint32_t nbuckets = 1;
        int ob = 0, fb = 0, pre = 0;
        if (one_bucket) {
            fb = min(min(kFinFastBits, rbits), a.fast_bits);
            pre = rbits - fb;
        } else {
            uint32_t cnt = 0;
            for (uint32_t j = 0; j < itn; ++j)
                if (first + j < n_loc) cnt += py[first + j];
            uint32_t o = block_exclusive_scan<THREADS>(cnt, scratch, &nbuckets);
            while (nbuckets > 1 && ((nbuckets - 1u) >> ob) != 0u) ++ob;
            fb = min(min(kFinFastBits - ob, rbits), a.fast_bits);
            for (uint32_t j = 0; j < itn; ++j) {
                if (first + j < n_loc) {
                    o += py[first + j];
                    py[first + j] = (uint16_t)(o - 1u);
                    if (!full) bx[first + j] = ((o - 1u) << fb) | (fb ? (bx[first + j] >> (rbits - fb)) : 0u);
                }
            }
            __syncthreads();
        }

        // ---- local sort; the final permutation lands in py
        uint32_t* cur = bx;
        uint32_t* oth = by;
        if (!full) {
            local_sort_bits<true, true>(&cur, &oth, ob + fb, n_loc, whist, scratch, py, pre);
            if (ob + fb == 0)                      // one bucket, no bits: identity
                for (uint32_t i = tid; i < n_loc; i += THREADS) cur[i] = i;
        } else {
            // every bit below the prefix, 18 at a time from the least significant up, cut out of the keys through the
            // current permutation; then the ordinal
            for (int gpos = 0; gpos < a.pfx_pos; gpos += 18) {
                const int gw = min(18, a.pfx_pos - gpos);
                for (uint32_t i = tid; i < n_loc; i += THREADS) {
                    const uint32_t r = cur[i] & 0x1fffu;
                    cur[i] = r | (key_get_field(gkeys[r], gpos, gw) << 13);
                }
                __syncthreads();
                local_sort_bits<false, false>(&cur, &oth, gw, n_loc, whist, scratch, nullptr);
            }
            if (ob > 0) {
                for (uint32_t i = tid; i < n_loc; i += THREADS) {
                    const uint32_t r = cur[i] & 0x1fffu;
                    cur[i] = r | ((uint32_t)py[r] << 13);
                }
                __syncthreads();
                local_sort_bits<false, false>(&cur, &oth, ob, n_loc, whist, scratch, nullptr);
            }
        }
        __syncthreads();
        // the final permutation (sorted position -> record) and its inverse; coefficients then reach sorted order through
        // the INVERSE permutation: the global read is coalesced (a gather would touch one 32-byte sector per 8-byte
        // coefficient), the permuted write goes to shared memory
        {
            uint16_t* inv = (uint16_t*)whist;      // the histograms are dead until the next pass
            for (uint32_t i = tid; i < n_loc; i += THREADS) {
                const uint32_t r = cur[i] & 0x1fffu;
                py[i] = (uint16_t)r;
                inv[r] = (uint16_t)i;
            }
            __syncthreads();
#pragma unroll 4
            for (uint32_t i = tid; i < n_loc; i += THREADS) scs[inv[i]] = gcoef[i];
            __syncthreads();
        }

        // ---- gather through the permutation: heads of runs of equal keys, sums since the last head, order check
        r = RunState();
        bool viol = false;
        {
            K kp;
            key_zero(kp);
            bool hp = false;
            if (first > 0 && first < n_loc) { kp = gkeys[py[first - 1]]; hp = true; }
#pragma unroll 2
            for (uint32_t j = 0; j < itn; ++j) {
                if (first + j < n_loc) {
                    const K kk = gkeys[py[first + j]];
                    const double c = scs[first + j];
                    const bool head = !hp || !key_eq(kk, kp);
                    viol |= hp && key_lt(kk, kp);
                    run_step(r, head, c, j, first + j, a.tol, scs);
                    kp = kk;
                    hp = true;
                }
            }
        }
        if (!__syncthreads_or(viol ? 1 : 0)) break;
        if (full) {                                // every bit was sorted on and the order is still wrong
            if (tid == 0) a.ctl->unsorted = 1u;
            break;
        }
        full = true;
        try_single = false;
        if (tid == 0) atomicAdd(&a.ctl->refinish, 1u);
    }

    finish_tail<K>(a, r, scs, scratch, first, n_loc, lo, tile, [&](uint32_t pos, uint32_t) { return gkeys[py[pos]]; });
}

template <typename K>
__global__ void __launch_bounds__(kFinThreads, kFinBlocksPerSM) finish_kernel(const __grid_constant__ FinishArgs a)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ uint32_t todo[kFinThreads], ntodo;
    if (a.ctl->overflow) return;                   // set by tile_bounds_kernel: the call will re-run on the LSD path
    const uint32_t count = a.ctl->fin_count;
    if (!a.behind_group) {
        // one block per tile, the grid sized for the most tiles that can own records (at most one per bucket): more of them
        // than that and the array is not sorted by prefix
        if (blockIdx.x == 0 && threadIdx.x == 0 && count > gridDim.x) a.ctl->unsorted = 1u;
        if (blockIdx.x < count) finish_tile<K>(a, smem_raw, a.worklist[blockIdx.x]);       // one load instead of three dependent ones
        return;
    }
    // Behind the group kernel: the blocks take runs of list entries by ticket, long runs first and shorter ones as the list
    // runs out (a run is 1/(2 gridDim.x) of what is left: a few thousand tickets in all, and the blocks finish together --
    // equal shares per block measured 8 % slower on a list that is all work, the sum of 111 tile times varies that much),
    // look at a run's descriptors with one load and finish the tiles the group kernel left: none at all on an input full of
    // like terms, all of them on one without.  No list of its own and no atomic per tile: 65,536 adds to one address cost
    // the group kernel 0.4-0.7 ms when they were tried.
    if (a.ctl->grp_left == 0u) return;             // the group kernel finished every tile
    uint32_t done = 0;
    __shared__ uint32_t run_lo, run_hi;
    while (true) {
        if (threadIdx.x == 0) {
            const uint32_t seen = *(volatile const uint32_t*)&a.ctl->fin_ticket;
            const uint32_t left = seen < count ? count - seen : 0u;
            const uint32_t len = min(max(left / (2u * gridDim.x), 1u), (uint32_t)kFinThreads);
            run_lo = atomicAdd(&a.ctl->fin_ticket, len);
            run_hi = run_lo + len;
            ntodo = 0u;
        }
        __syncthreads();
        const uint32_t r0 = run_lo, r1 = min(run_hi, count);
        if (r0 >= count) break;
        const uint32_t q = r0 + threadIdx.x;
        if (q < r1 && !(a.worklist[q].w & 2u)) todo[atomicAdd(&ntodo, 1u)] = q;     // (any order: tiles are independent)
        __syncthreads();
        const uint32_t n = ntodo;
        for (uint32_t j = 0; j < n; ++j) {
            finish_tile<K>(a, smem_raw, a.worklist[todo[j]]);
            __syncthreads();
        }
        done += n;
        __syncthreads();                           // (everybody has read the run and the count before thread 0 takes the next)
    }
    if (threadIdx.x == 0 && done) atomicAdd(&a.ctl->fin2_count, done);
}

// ------------------------------------------------------------------------------------- group kernel

// The sorting finish moves every RECORD through three counting-sort passes and then gathers every record's key again to
// find the runs.  When a tile holds few distinct keys (the paper's regime: like terms by the dozen; config 5:
// ten records per monomial) that is the wrong amount of work.  finish_group_kernel, tried first on every work-list tile:
//   G1  streams the keys once and looks each up in a shared-memory hash table (256 buckets of four slots, a 31-bit
//       fingerprint per slot: one 16-byte load shows a bucket; atomicCAS on the bucket's first empty slot, the winner parks
//       the full key and its record number); after a barrier every record compares its FULL key with the slot's -- a
//       fingerprint collision, an overlong probe sequence, more than 768 distinct keys, or more keys than grouping pays for
//       (group_pays) give the tile back: it stays unmarked in the work list and finish_kernel behind finishes it;
//   G2  puts the U distinct keys (not the records) in order: a 10-bit leading digit (prefix difference above the top key
//       bits below the prefix) bins them, and inside a bin -- one or two keys as a rule, more than 16 hand the tile on -- a
//       key's place is the number of smaller keys, full keys compared: exact, no order check needed;
//   G3  ONE stable counting pass of the records on their slot (per-warp rows of 1024 packed 16-bit counters, rank = old
//       value of the atomic), the bin scan walking the slots in KEY order: every record now knows its final sorted position;
//   G4  coefficients go to their sorted position (coalesced read, as before) and run heads into a bit mask -- no key gather;
//   then the shared tail (S3, S4).  Equal keys keep their input order exactly as through the stable sort, so the sums are
//   bit-identical to finish_kernel's (tests/test_gpu_bucket_path.py compares the two).
constexpr int kGrpSlots = 1024;
constexpr int kGrpMaxDistinct = 768;
constexpr int kGrpMaxProbe = 48;
constexpr int kGrpBPT = kGrpMaxDistinct / kFinThreads;      // slots per thread in the bin scan
constexpr int kGrpDigit = 10;           // bits of the distinct keys' leading digit
constexpr int kGrpMaxBin = 16;          // most distinct keys that may share a leading digit
constexpr int kGrpTilesPerBlock = 1;    // consecutive work-list entries a block finishes, one after the other

struct GroupSmem {
    static constexpr int NW = kFinThreads / 32;
    // region A, kFinCap * 8 bytes: [tags u32][keys 16 B][bins u32][order u16][perm u16] while the table lives, then the
    // counting rows [NW][kGrpSlots] u16 over the keys (perm still alive), then the sorted coefficients over all of it
    static constexpr size_t off_tags = 0;
    static constexpr size_t off_keys = off_tags + (size_t)kGrpSlots * 4;
    static constexpr size_t off_bins = off_keys + (size_t)kGrpSlots * 16;
    static constexpr size_t off_order = off_bins + (size_t)kGrpSlots * 4;
    static constexpr size_t off_perm = off_order + (size_t)kGrpSlots * 2;
    static constexpr size_t region_a = off_perm + (size_t)kGrpSlots * 2;
    static constexpr size_t off_rows = off_keys;
    static constexpr size_t off_ids = (size_t)kFinCap * 8;           // u16 per record: its slot; later the head bit mask
    static constexpr size_t off_rk = off_ids + (size_t)kFinCap * 2;  // u16 per record: rank, then sorted position; before that
                                                                     // [record that claimed the slot]
    static constexpr size_t off_rep = off_rk + (size_t)kFinCap * 2;  // u16 per distinct key, in key order: a record that holds it
    static constexpr size_t off_scratch = off_rep + (size_t)kGrpMaxDistinct * 2;
    static constexpr size_t bytes = off_scratch + 64 * 4;
};
static_assert(GroupSmem::region_a <= (size_t)kFinCap * 8, "the table lives where the sorted coefficients go");
static_assert((size_t)GroupSmem::NW * kGrpSlots * 2 <= (size_t)kGrpSlots * 16, "the counting rows take the place of the table's keys");
static_assert(kGrpSlots <= kFinCap && kGrpBPT * kFinThreads == kGrpMaxDistinct && kGrpMaxDistinct <= kGrpSlots, "group path sizes");
static_assert((1 << kGrpDigit) == kGrpSlots && kGrpSlots % kFinThreads == 0, "one bin per slot index, whole slots per thread");
static_assert((GroupSmem::bytes + 96 + 1024) * kFinBlocksPerSM <= 228 * 1024, "four blocks per SM");

// does grouping a tile of n records with (at least) u distinct keys cost less than sorting it?  (finish_group_kernel, set-up)
__device__ __forceinline__ bool group_pays(uint32_t n, uint32_t u) { return 10u * n > 8400u + 52u * u; }

// bucket and fingerprint of a key: x = a multiply-add mix of the key's 32-bit words; the bucket is x's top byte and the
// fingerprint a bijection of x (two keys of one bucket share a fingerprint only if they share x, or differ in the forced bit)
__device__ __forceinline__ uint32_t key_mix(uint64_t k) { return (uint32_t)k * 0x9E3779B1u + (uint32_t)(k >> 32) * 0x85EBCA77u; }
__device__ __forceinline__ uint32_t key_mix(const Key128& k)
{
    return (uint32_t)k.lo * 0x9E3779B1u + (uint32_t)(k.lo >> 32) * 0x85EBCA77u + (uint32_t)k.hi * 0xC2B2AE3Du + (uint32_t)(k.hi >> 32) * 0x27D4EB2Fu;
}
template <typename K>
__device__ __forceinline__ void key_hash(const K& k, uint32_t* bucket, uint32_t* fp)
{
    uint32_t x = key_mix(k);
    x ^= x >> 15;
    *bucket = (x * 0x2C1B3C6Du) >> (32 - 8);                  // kGrpSlots / 4 = 256 buckets of four slots
    *fp = ((x ^ (x >> 13)) * 0x297A2D39u) | 0x80000000u;      // never 0 = empty
}
static_assert(kGrpSlots / 4 == 256, "key_hash takes the bucket from eight bits");
// the key bits at positions >= pos as a number (the prefix has at most 48 bits)
__device__ __forceinline__ uint64_t key_prefix64(uint64_t k, int pos) { return k >> pos; }
__device__ __forceinline__ uint64_t key_prefix64(const Key128& k, int pos)
{
    if (pos >= 64) return k.hi >> (pos - 64);
    return pos == 0 ? k.lo : ((k.lo >> pos) | (k.hi << (64 - pos)));
}

template <typename K>
__global__ void __launch_bounds__(kFinThreads, kFinBlocksPerSM) finish_group_kernel(const __grid_constant__ FinishArgs a)
{
    constexpr int THREADS = kFinThreads, CAP = kFinCap, NW = THREADS / 32, SPT = kGrpSlots / THREADS;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    uint32_t* tags = (uint32_t*)(smem_raw + GroupSmem::off_tags);
    const uint4* tags4 = (const uint4*)tags;
    K* tkeys = (K*)(smem_raw + GroupSmem::off_keys);
    uint32_t* bins = (uint32_t*)(smem_raw + GroupSmem::off_bins);            // count of the distinct keys per leading digit, then (start | count << 16)
    uint16_t* order = (uint16_t*)(smem_raw + GroupSmem::off_order);          // slots grouped by leading digit
    uint16_t* perm = (uint16_t*)(smem_raw + GroupSmem::off_perm);            // slots in key order
    uint32_t* rows32 = (uint32_t*)(smem_raw + GroupSmem::off_rows);
    uint16_t* ids = (uint16_t*)(smem_raw + GroupSmem::off_ids);
    uint32_t* hb = (uint32_t*)(smem_raw + GroupSmem::off_ids);              // head bits by sorted position, once the slots are dead
    uint16_t* rk = (uint16_t*)(smem_raw + GroupSmem::off_rk);
    uint16_t* own = rk;                                                      // [kGrpSlots] record that claimed the slot
    uint16_t* rep = (uint16_t*)(smem_raw + GroupSmem::off_rep);
    uint32_t* scratch = (uint32_t*)(smem_raw + GroupSmem::off_scratch);      // [0..NW+1] scans, [48] largest prefix difference
    double* scs = (double*)smem_raw;

    const unsigned tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
    // A block takes kGrpTilesPerBlock consecutive entries of the work list, one after the other: still thousands of blocks for
    // the block scheduler to balance, but a call whose tiles are not worth grouping (grp_off, below) pays an eighth of the
    // block starts -- 65,536 blocks that only look at a flag and leave cost 0.2 ms.  (Persistent blocks that take tiles by ticket
    // and pull the NEXT tile's descriptor and records into L2 were measured too: 3.00 against 2.95 ms on config 5.)
    const uint32_t overflow = a.ctl->overflow, fin_count = a.ctl->fin_count;
    uint32_t off = a.ctl->grp_off;
    const uint32_t b0 = blockIdx.x * (uint32_t)kGrpTilesPerBlock;
    uint4* wls = (uint4*)(scratch + 16);           // the block's descriptors, one coalesced load
    if (tid < (unsigned)kGrpTilesPerBlock && b0 + tid < fin_count) wls[tid] = a.worklist[b0 + tid];
    if (overflow) return;                          // set by tile_bounds_kernel: the call will re-run on the LSD path
    if (blockIdx.x == 0 && tid == 0 && fin_count > a.max_list) a.ctl->unsorted = 1u;   // more bucket starts than buckets: not sorted by prefix
    __syncthreads();
    const uint32_t b_end = min(b0 + (uint32_t)kGrpTilesPerBlock, fin_count);
    uint32_t left_here = 0;                        // tiles this block leaves to the sorting kernel (thread 0 reports them)
    for (uint32_t b = b0; b < b_end; ++b) {
    const uint4 wl = wls[b - b0];
    const uint32_t tile = wl.x, lo = wl.y, hi = wl.z;
    const uint32_t n_loc = hi > lo ? min(hi - lo, (uint32_t)CAP) : 0u;
    const K* __restrict__ gkeys = (const K*)a.keys + lo;
    const double* __restrict__ gcoef = a.coefs + lo;
    const uint32_t itn = ((n_loc + THREADS - 1) / THREADS) | 1u;
    const uint32_t first = tid * itn;

    // Is grouping worth trying?  Measured on B200 (profiles/r2b_state.md; pooled 128-bit keys, tiles of 1526 and 3052 records,
    // 2 to 20 records per key; ms per 65,536 tiles): this kernel costs about 1.07 + 0.26 n/1000 + 3.3 U/1000 for a tile of n
    // records with U distinct keys, the sorting kernel about 0.65 + 0.81 n/1000 + 0.72 U/1000, so grouping pays when
    // n > 764 + 4.7 U (group_pays asks for 10 % more): never below about 840 records, and as U is known only from the look-ups,
    // every batch of 1024 records checks the keys met so far.  And not once most tiles so far were given back (an input
    // with few like terms): grp_off is sticky, the sorting kernel behind finds the tiles unmarked.
    // (the barrier: a block must not split over a flag that flips between its warps' loads)
    if (b > b0 && tid == 0) off = *(volatile const uint32_t*)&a.ctl->grp_off;
    const int leave = __syncthreads_or((a.no_group != 0 || off != 0u) ? 1 : 0);
    if (leave) { left_here += b_end - b; break; }
    if (!group_pays(n_loc, 0u)) ++left_here;
    else {
    bool bad = false;
    uint32_t U = 0;
    {
        for (uint32_t i = tid * 8u; i < n_loc; i += THREADS * 8u) asm volatile("prefetch.global.L2 [%0];" ::"l"(gkeys + i));
        for (uint32_t i = tid * 16u; i < n_loc; i += THREADS * 16u) asm volatile("prefetch.global.L2 [%0];" ::"l"(gcoef + i));
#pragma unroll
        for (int j = 0; j < SPT; ++j) { tags[tid + j * THREADS] = 0u; bins[tid + j * THREADS] = 0u; }
        if (tid < 8u) scratch[48 + tid] = 0u;      // [48] largest prefix difference, [51..55] keys met per batch
        __syncthreads();

        // ---- G1: every record finds or claims the slot of its key.  The table is 256 buckets of four tags: one 16-byte
        // load shows a bucket, a key takes the bucket's first empty slot (slots fill in order and never empty again, so two
        // records of one key cannot claim two slots).
        const K k0 = gkeys[0];
        const bool single = wl.w != 0u;            // first and last record share the prefix: one bucket if the array is sorted
        bool descending = false, early = false;
        uint32_t met = 0;
        for (uint32_t base = 0; base < n_loc; base += 4 * THREADS) {
            K k[4];
            uint32_t sl[4], nwon = 0;
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const uint32_t i = base + u * THREADS + tid;
                k[u] = k0;
                if (i < n_loc) k[u] = gkeys[i];
            }
            if (!single) {                         // prefix-order self-check (a one-bucket tile is checked on its distinct keys, G2)
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    const uint32_t i = base + u * THREADS + tid;
                    if (i > 0 && i < n_loc) {
                        const K kp = gkeys[i - 1];
                        descending |= key_prefix64(k[u], a.pfx_pos) < key_prefix64(kp, a.pfx_pos);
                    }
                }
            }
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const uint32_t i = base + u * THREADS + tid;
                sl[u] = 0u;
                if (i < n_loc) {
                    uint32_t b, fp, s = 0u;
                    key_hash(k[u], &b, &fp);
                    for (int tries = 0;; ++tries) {
                        const uint4 t = tags4[b];
                        int j = t.x == fp ? 0 : t.y == fp ? 1 : t.z == fp ? 2 : t.w == fp ? 3 : -1;
                        if (j >= 0) { s = 4u * b + (uint32_t)j; break; }
                        j = t.x == 0u ? 0 : t.y == 0u ? 1 : t.z == 0u ? 2 : t.w == 0u ? 3 : -1;
                        if (j >= 0) {
                            s = 4u * b + (uint32_t)j;
                            const uint32_t old = atomicCAS(&tags[s], 0u, fp);
                            if (old == 0u) { tkeys[s] = k[u]; own[s] = (uint16_t)i; ++nwon; break; }
                            if (old == fp) break;
                        } else b = (b + 1u) & (uint32_t)(kGrpSlots / 4 - 1);       // (a lost race looks at the same bucket again)
                        if (tries >= kGrpMaxProbe) { bad = true; break; }
                    }
                    sl[u] = s;
                    ids[i] = (uint16_t)s;
                }
            }
            if (nwon) atomicAdd(&scratch[51 + base / (4 * THREADS)], nwon);      // (a word per batch: final once the barrier is passed)
            __syncthreads();                       // the keys of every slot claimed so far are in place
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const uint32_t i = base + u * THREADS + tid;
                if (i < n_loc) bad |= !key_eq(tkeys[sl[u]], k[u]);
            }
            // distinct keys met so far: too many for grouping to pay?  (the same answer in every thread)
            met += scratch[51 + base / (4 * THREADS)];
            if (!group_pays(n_loc, met)) { early = true; break; }
        }
        if (descending) a.ctl->unsorted = 1u;      // the prefix passes were not stable (see sort.cu)
        bad |= early;

        // ---- G2: the distinct keys in order.  Leading digit = prefix difference above the top key bits below the prefix,
        // ten bits in all: a key's place is the start of its digit's bin plus the number of smaller keys in that bin (full
        // keys compared, so the order is exact; a bin of more than kGrpMaxBin keys hands the tile on)
        const uint64_t p0 = key_prefix64(k0, a.pfx_pos);
        K kk[SPT];
        uint32_t occ = 0, dmax = 0;
#pragma unroll
        for (int j = 0; j < SPT; ++j) {
            const uint32_t s = tid + j * THREADS;
            kk[j] = k0;
            if (tags[s] != 0u) {
                occ |= 1u << j;
                kk[j] = tkeys[s];
                const uint64_t d = key_prefix64(kk[j], a.pfx_pos) - p0;
                if (d >> kGrpDigit) bad = true;                       // prefixes too far apart for the digit (or not sorted)
                dmax = max(dmax, (uint32_t)d & (uint32_t)((1 << kGrpDigit) - 1));
            }
        }
        if (dmax) atomicMax(&scratch[48], dmax);
        if (single && dmax) bad = true;            // a second prefix inside a tile whose ends share theirs: not sorted by prefix
        bad = __syncthreads_or(bad ? 1 : 0) != 0;
        if (!bad) {
            dmax = scratch[48];
            int ob = 0;
            while ((dmax >> ob) != 0u) ++ob;
            const int fb = min(kGrpDigit - ob, a.pfx_pos);
            uint32_t dig[SPT], rnk[SPT];
#pragma unroll
            for (int j = 0; j < SPT; ++j) {
                dig[j] = 0u; rnk[j] = 0u;
                if (occ & (1u << j)) {
                    const uint32_t d = (uint32_t)(key_prefix64(kk[j], a.pfx_pos) - p0);
                    dig[j] = (d << fb) | (fb ? key_get_field(kk[j], a.pfx_pos - fb, fb) : 0u);
                    rnk[j] = atomicAdd(&bins[dig[j]], 1u);
                    bad |= rnk[j] >= (uint32_t)kGrpMaxBin;
                }
            }
            __syncthreads();
            {
                uint32_t c[SPT], sum = 0;
#pragma unroll
                for (int j = 0; j < SPT; ++j) { c[j] = bins[tid * SPT + j]; sum += c[j]; }
                uint32_t start = block_exclusive_scan<THREADS>(sum, scratch, &U);
#pragma unroll
                for (int j = 0; j < SPT; ++j) { bins[tid * SPT + j] = start | (c[j] << 16); start += c[j]; }
            }
            bad = __syncthreads_or(bad ? 1 : 0) != 0 || U > (uint32_t)kGrpMaxDistinct;
            if (!bad) {
#pragma unroll
                for (int j = 0; j < SPT; ++j)
                    if (occ & (1u << j)) order[(bins[dig[j]] & 0xffffu) + rnk[j]] = (uint16_t)(tid + j * THREADS);
                __syncthreads();
#pragma unroll
                for (int j = 0; j < SPT; ++j) {
                    if (occ & (1u << j)) {
                        const uint32_t s = tid + j * THREADS, bs = bins[dig[j]], start = bs & 0xffffu, cnt = bs >> 16;
                        uint32_t below = 0;
                        if (cnt > 1u)
                            for (uint32_t m = 0; m < cnt; ++m) {
                                const uint32_t s2 = order[start + m];
                                if (s2 != s) below += key_lt(tkeys[s2], kk[j]) ? 1u : 0u;
                            }
                        perm[start + below] = (uint16_t)s;
                        rep[start + below] = own[s];
                    }
                }
                __syncthreads();
            }
        }
    }
    if (bad) {
        // given back: the sorting kernel behind takes the tile.  Once at least 64 tiles and more than half of the tiles begun
        // (blocks start in order) came back -- an input with few like terms -- the rest no longer try.
        ++left_here;
        if (tid == 0) {
            const uint32_t f = atomicAdd(&a.ctl->grp_fail, 1u) + 1u;
            if (f >= 64u && 2u * f > b) a.ctl->grp_off = 1u;
        }
    } else {

    // ---- G3: one stable counting pass of the records on their slot; warp w owns the contiguous chunk [w*per, (w+1)*per)
    // and row w (see local_pass); the bins are scanned in KEY order
    const uint32_t per = (((n_loc + NW - 1) / NW) + 31u) & ~31u;
    const uint32_t wbeg = min(warp * per, n_loc), wend = min(wbeg + per, n_loc);
    {
        uint4* z = (uint4*)rows32;
#pragma unroll
        for (int j = 0; j < NW * kGrpSlots * 2 / 16 / THREADS; ++j) z[tid + j * THREADS] = make_uint4(0u, 0u, 0u, 0u);
    }
    __syncthreads();
    // Counter of (slot, warp): 16 bits, the eight warps of a slot side by side in one 16-byte group (the bin scan reads a
    // slot with one load), warps 2p and 2p + 1 sharing word (p + slot / 8) mod 4 of the group -- the rotation spreads one
    // warp's atomics over all 32 banks.
    static_assert(NW == 8, "eight 16-bit counters per 16-byte group");
    const uint32_t wpair = warp >> 1, wsh = (warp & 1u) * 16u;
    {
        for (uint32_t base = wbeg; base < wend; base += 64u) {
            const uint32_t i0 = base + lane, i1 = i0 + 32u;
            const uint32_t d0 = (i0 < wend) ? ids[i0] : 0u, d1 = (i1 < wend) ? ids[i1] : 0u;
            if (i0 < wend) rk[i0] = (uint16_t)(atomicAdd(&rows32[d0 * 4u + ((wpair + (d0 >> 3)) & 3u)], 1u << wsh) >> wsh);
            __syncwarp();
            if (i1 < wend) rk[i1] = (uint16_t)(atomicAdd(&rows32[d1 * 4u + ((wpair + (d1 >> 3)) & 3u)], 1u << wsh) >> wsh);
            __syncwarp();
        }
    }
    __syncthreads();
    {
        uint32_t c[kGrpBPT][NW], sl[kGrpBPT];
        uint32_t count = 0;
#pragma unroll
        for (int j = 0; j < kGrpBPT; ++j) {
            const uint32_t q = tid * kGrpBPT + j;
            sl[j] = q < U ? perm[q] : 0u;
            uint4 v = make_uint4(0u, 0u, 0u, 0u);
            if (q < U) v = ((const uint4*)rows32)[sl[j]];
            const uint32_t rot = (sl[j] >> 3) & 3u;                 // word (p + rot) mod 4 holds pair p
            if (rot & 1u) v = make_uint4(v.y, v.z, v.w, v.x);
            if (rot & 2u) v = make_uint4(v.z, v.w, v.x, v.y);
            c[j][0] = v.x & 0xffffu; c[j][1] = v.x >> 16; c[j][2] = v.y & 0xffffu; c[j][3] = v.y >> 16;
            c[j][4] = v.z & 0xffffu; c[j][5] = v.z >> 16; c[j][6] = v.w & 0xffffu; c[j][7] = v.w >> 16;
        }
#pragma unroll
        for (int j = 0; j < kGrpBPT; ++j)
#pragma unroll
            for (int w = 0; w < NW; ++w) { const uint32_t x = c[j][w]; c[j][w] = count; count += x; }
        uint32_t total;
        const uint32_t bin_start = block_exclusive_scan<THREADS>(count, scratch, &total);
#pragma unroll
        for (int j = 0; j < kGrpBPT; ++j) {
            const uint32_t q = tid * kGrpBPT + j;
            if (q < U) {
                // bit 15: this warp holds the key's first record (its rank-0 record is the head of the run)
                const uint32_t end = (j + 1 < kGrpBPT) ? c[j + 1][0] : count;
                bool seen = false;
                uint32_t h[NW];
#pragma unroll
                for (int w = 0; w < NW; ++w) {
                    const uint32_t nxt = (w + 1 < NW) ? c[j][w + 1] : end;
                    const bool has = nxt != c[j][w];
                    h[w] = (bin_start + c[j][w]) | ((has && !seen) ? 0x8000u : 0u);
                    seen |= has;
                }
                uint4 v = make_uint4(h[0] | (h[1] << 16), h[2] | (h[3] << 16), h[4] | (h[5] << 16), h[6] | (h[7] << 16));
                const uint32_t rot = (sl[j] >> 3) & 3u;             // back into the rotated order
                if (rot & 1u) v = make_uint4(v.w, v.x, v.y, v.z);
                if (rot & 2u) v = make_uint4(v.z, v.w, v.x, v.y);
                ((uint4*)rows32)[sl[j]] = v;
            }
        }
    }
    __syncthreads();
    // sorted position of every record (over its rank), bit 15 = head of its run
#pragma unroll 4
    for (uint32_t i = wbeg + lane; i < wend; i += 32u) {
        const uint32_t d = ids[i], r = rk[i];
        const uint32_t h = (rows32[d * 4u + ((wpair + (d >> 3)) & 3u)] >> wsh) & 0xffffu;
        rk[i] = (uint16_t)(((h & 0x1fffu) + r) | ((r == 0u) ? (h & 0x8000u) : 0u));
    }
    // the head bits take the place of the first 320 slot ids: when those all belong to warp 0's chunk, warp 0 clears them as
    // soon as it has read them
    if (per >= 320u) {
        if (warp == 0) {
            __syncwarp();
#pragma unroll
            for (int j = 0; j < 5; ++j) hb[lane + 32 * j] = 0u;
        }
    } else {
        __syncthreads();
        if (tid < 160u) hb[tid] = 0u;               // CAP / 32 words and the two a thread past the end may load
    }
    __syncthreads();

    // ---- G4: coefficients to their sorted position (coalesced global read), heads into the bit mask; eight loads in flight
    // per thread (four: +0.03 ms on config 5)
#pragma unroll 8
    for (uint32_t i = tid; i < n_loc; i += THREADS) {
        const uint32_t p = rk[i], pos = p & 0x1fffu;
        scs[pos] = gcoef[i];
        if (p & 0x8000u) atomicOr(&hb[pos >> 5], 1u << (pos & 31u));
    }
    __syncthreads();

    // ---- runs, sums since the last head, S4 for the runs that end inside the thread's stretch
    RunState r;
    {
        const uint32_t w0 = hb[first >> 5], w1 = hb[(first >> 5) + 1u];
        const uint32_t bits = __funnelshift_r(w0, w1, first & 31u);      // bit j: position first + j is a head
#pragma unroll 2
        for (uint32_t j = 0; j < itn; ++j)
            if (first + j < n_loc) run_step(r, ((bits >> j) & 1u) != 0u, scs[first + j], j, first + j, a.tol, scs);
    }
    finish_tail<K>(a, r, scs, scratch, first, n_loc, lo, tile, [&](uint32_t, uint32_t q) { return gkeys[rep[q]]; });
    if (tid == 0) a.worklist[b].w = wl.w | 2u;                 // done: the sorting kernel behind skips the tile
    }
    }
    __syncthreads();                               // the tail read what the next tile overwrites
    }
    if (tid == 0 && left_here) atomicAdd(&a.ctl->grp_left, left_here);
}

// ------------------------------------------------------------------------------- S4/S5 across tiles

// Exclusive scan of the tiles' survivor counts, in place, in two small kernels: per-chunk sums, then every block adds the
// sums of the chunks before it to the scan of its own chunk; tile_off[ntiles] = U'.
constexpr uint32_t kScanChunk = 1024u * 4u;

__global__ void __launch_bounds__(1024) tile_sum_kernel(const uint32_t* __restrict__ tile_cnt, uint32_t ntiles,
                                                        uint32_t* __restrict__ chunk_sum)
{
    __shared__ uint32_t scratch[34];
    const uint32_t base = blockIdx.x * kScanChunk;
    uint32_t sum = 0;
#pragma unroll
    for (uint32_t j = 0; j < 4; ++j) {
        const uint32_t t = base + j * 1024u + threadIdx.x;
        if (t < ntiles) sum += tile_cnt[t];
    }
    uint32_t total;
    (void)block_exclusive_scan<1024>(sum, scratch, &total);
    if (threadIdx.x == 0) chunk_sum[blockIdx.x] = total;
}

__global__ void __launch_bounds__(1024) tile_scan_kernel(uint32_t* __restrict__ tile_off, uint32_t ntiles,
                                                         const uint32_t* __restrict__ chunk_sum, Control* ctl,
                                                         int64_t* out_count_device)
{
    __shared__ uint32_t scratch[34];
    const unsigned tid = threadIdx.x;
    uint32_t before = 0;                           // survivors of the chunks before this block's (at most 1024 chunks)
    {
        uint32_t x = 0;
        for (uint32_t c = tid; c < blockIdx.x; c += 1024u) x += chunk_sum[c];
        (void)block_exclusive_scan<1024>(x, scratch, &before);
        __syncthreads();
    }
    const uint32_t base = blockIdx.x * kScanChunk;
    uint32_t v[4], sum = 0;
#pragma unroll
    for (uint32_t j = 0; j < 4; ++j) {
        const uint32_t t = base + tid * 4u + j;
        v[j] = t < ntiles ? tile_off[t] : 0u;
        sum += v[j];
    }
    uint32_t total;
    uint32_t excl = block_exclusive_scan<1024>(sum, scratch, &total) + before;
#pragma unroll
    for (uint32_t j = 0; j < 4; ++j) {
        const uint32_t t = base + tid * 4u + j;
        if (t < ntiles) tile_off[t] = excl;
        excl += v[j];
    }
    if (blockIdx.x == gridDim.x - 1 && tid == 0) {
        tile_off[ntiles] = before + total;
        ctl->survivors = before + total;
        if (out_count_device) *out_count_device = (int64_t)(before + total);
    }
}

// S5: one warp per work-list tile copies the tile's survivors to their final place (the tile's scanned offset) and unpacks
// the keys -- no search, consecutive lanes read and write consecutive terms.  Tiles without records are not on the list.
template <typename K>
__global__ void __launch_bounds__(256) emit_kernel(const __grid_constant__ EmitArgs a, const __grid_constant__ Plan plan)
{
    const uint32_t nlist = min(a.ctl->fin_count, a.max_list);
    const unsigned lane = lane_id();
    const uint32_t nwarps = gridDim.x * (blockDim.x >> 5);
    for (uint32_t q = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5); q < nlist; q += nwarps) {
        const uint4 wl = a.worklist[q];
        const uint32_t t = wl.x;
        const uint32_t off = a.tile_off[t], cnt = a.tile_off[t + 1] - off;
        const uint64_t src = wl.y;
        // four terms per lane in flight (all loads of a round first; a tile seldom holds more than a few hundred survivors):
        // 0.191 -> 0.163 ms on config 5, 1.67 -> 1.39 ms on 1e8 unpruned terms.  Eight tiles per block with all their
        // survivors spread evenly over the block's threads measured 0.173 / 1.42.
        for (uint32_t i0 = lane; i0 < cnt; i0 += 128u) {
            double sv[4];
            K kv[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const uint32_t i = i0 + 32u * u;
                sv[u] = 0.0;
                key_zero(kv[u]);
                if (i < cnt) { sv[u] = a.usums[src + i]; kv[u] = ((const K*)a.ukeys)[src + i]; }
            }
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const uint32_t i = i0 + 32u * u;
                const uint64_t o = (uint64_t)off + i;
                if (i < cnt && (int64_t)o < a.out_capacity) emit_term<K>(a, plan, o, sv[u], kv[u]);
            }
        }
    }
}

// ---------------------------------------------------------------------------------------- launchers

template <typename K>
static int launch_finish_t(const Plan& plan, int prefix_passes, int nfast, int fin_tile, int64_t n, const void* keys,
                           const double* coefs, double tol, void* ukeys, double* usums, CoefOut out_coef, void* out_exps,
                           int exp_bytes, int64_t out_capacity, uint32_t* tile_start, uint32_t* tile_state, uint4* worklist,
                           int group, uint32_t* chunk_sum, Control* ctl, int64_t* out_count_device,
                           cudaEvent_t after_tiles, cudaStream_t stream)
{
    const uint32_t ntiles = (uint32_t)((n + fin_tile - 1) / fin_tile);
    const int nlow = plan.npasses - prefix_passes;
    const int pfx_pos = plan.digit_pos[nlow];
    tile_bounds_kernel<K><<<(ntiles + 1 + 255) / 256, 256, 0, stream>>>((const K*)keys, (uint32_t)n, pfx_pos, (uint32_t)fin_tile,
                                                                       ntiles, tile_start, worklist, ctl);
    auto kern = finish_kernel<K>;
    constexpr size_t smem = FinishSmem::bytes;
    ensure_dynamic_smem(kern, (size_t)smem);
    FinishArgs a;
    a.keys = keys; a.coefs = coefs; a.n = (uint32_t)n; a.ntiles = ntiles; a.fin_tile = (uint32_t)fin_tile;
    a.tile_start = tile_start; a.tile_state = tile_state; a.worklist = worklist;
    a.pfx_pos = pfx_pos; a.fast_bits = nfast > 0 ? nfast * 8 : 32; a.tol = tol; a.ukeys = ukeys; a.usums = usums; a.ctl = ctl;
    a.behind_group = 0; a.max_list = 0; a.no_group = group == 2 ? 1 : 0;
    // a tile owns records only if a bucket starts in it: at most one tile per bucket, at most 2^T buckets
    const int T = plan.key_bits - pfx_pos;
    const uint32_t fin_blocks = (T < 31 && (1u << T) < ntiles) ? (1u << T) : ntiles;
    int launches = 5;
    if (group) {
        // every tile first through the group kernel; the tiles it leaves unmarked (few, or nearly all of them when the input
        // has too few like terms) through the sorting kernel, whose blocks then take runs of the list by ticket
        auto gkern = finish_group_kernel<K>;
        ensure_dynamic_smem(gkern, GroupSmem::bytes);
        a.max_list = fin_blocks;
        gkern<<<(fin_blocks + kGrpTilesPerBlock - 1) / kGrpTilesPerBlock, kFinThreads, GroupSmem::bytes, stream>>>(a);
        FinishArgs b = a;
        b.behind_group = 1;
        const uint32_t resident = (uint32_t)(sm_count() * kFinBlocksPerSM);
        kern<<<fin_blocks < resident ? fin_blocks : resident, kFinThreads, smem, stream>>>(b);
        ++launches;
    } else kern<<<fin_blocks, kFinThreads, smem, stream>>>(a);
    if (after_tiles) cudaEventRecord(after_tiles, stream);
    const uint32_t nchunks = (ntiles + kScanChunk - 1) / kScanChunk;
    tile_sum_kernel<<<nchunks, 1024, 0, stream>>>(tile_state, ntiles, chunk_sum);
    tile_scan_kernel<<<nchunks, 1024, 0, stream>>>(tile_state, ntiles, chunk_sum, ctl, out_count_device);
    EmitArgs e;
    e.ukeys = ukeys; e.usums = usums; e.ntiles = ntiles; e.tile_start = tile_start; e.tile_off = tile_state;
    e.out_coef = out_coef; e.out_exps = out_exps; e.exp_bytes = exp_bytes;
    e.wpr = row_words(plan.nvars, exp_bytes, out_exps);
    e.out_capacity = out_capacity;
    e.worklist = worklist; e.max_list = fin_blocks; e.ctl = ctl;
    int64_t blocks = ((int64_t)fin_blocks + 7) / 8;          // one warp per work-list tile, grid-stride
    if (blocks > sm_count() * 64) blocks = sm_count() * 64;
    if (blocks < 1) blocks = 1;
    emit_kernel<K><<<(unsigned)blocks, 256, 0, stream>>>(e, plan);
    return launches;
}

int launch_finish(const Plan& plan, int prefix_passes, int nfast, int fin_tile, int64_t n, const void* keys, const double* coefs,
                  double tol, void* ukeys, double* usums, CoefOut out_coef, void* out_exps, int exp_bytes, int64_t out_capacity,
                  uint32_t* tile_start, uint32_t* tile_state, uint4* worklist, int group, uint32_t* chunk_sum,
                  Control* ctl, int64_t* out_count_device, cudaEvent_t after_tiles, cudaStream_t stream)
{
    if (n <= 0 || prefix_passes < 1 || prefix_passes > plan.npasses || fin_tile < kFinMinTile || fin_tile >= kFinCap) return 0;
    if (plan.key_bytes == 8)
        return launch_finish_t<uint64_t>(plan, prefix_passes, nfast, fin_tile, n, keys, coefs, tol, ukeys, usums, out_coef, out_exps,
                                         exp_bytes, out_capacity, tile_start, tile_state, worklist, group, chunk_sum, ctl, out_count_device, after_tiles, stream);
    return launch_finish_t<Key128>(plan, prefix_passes, nfast, fin_tile, n, keys, coefs, tol, ukeys, usums, out_coef, out_exps,
                                   exp_bytes, out_capacity, tile_start, tile_state, worklist, group, chunk_sum, ctl, out_count_device, after_tiles, stream);
}

}  // namespace polylab
