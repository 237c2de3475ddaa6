// kernels.h -- host-side launchers of the polylab-b200 kernels (internal; the public ABI is
// include/polylab.h).  Every launcher enqueues on `stream`, returns the number of kernels it
// launched, and never synchronises.  Step names S0..S5, X1 are those of DESIGN.md.
#pragma once

#include "common.cuh"

namespace polylab {

// Tile sizes of the streaming kernels (records per thread block); also used by the workspace query.
constexpr int kSortThreads64 = 256;
constexpr int kSortThreads128 = 256;
constexpr int kSortItems64 = 16;    // 4096-record tiles of (u64 key, f64 coef)
constexpr int kSortThreads256 = 256;
constexpr int kSortItems256 = 8;    // 2048-record tiles of (256-bit key, f64 coef): 64 KB of staging, three blocks per SM
constexpr int kSortItems128 = 20;   // 5120-record tiles of (u128 key, f64 coef), two blocks per SM (swept on B200: 12x3 4.26, 16x2 4.08, 20x2 4.04, 24x2 4.74 ms for two passes of config 5)
constexpr int kReduceThreads = 256;
constexpr int kReduceItems = 9;     // odd: conflict-free blocked reads from shared memory
constexpr int kPruneThreads = 256;
constexpr int kPruneItems = 8;

constexpr int kFinBlocksPerSM = 4;
constexpr int kFinThreads = 256;    // bucket path (finish.cu): four blocks per SM (swept on B200: 512 x 8192 x 2 4.83 ms, 256 x 4608 x 4 4.29 ms)
constexpr int kFinCap = 4608;       // most records a finish tile can own (10 bytes of shared memory each); tile t owns the
                                    // buckets that start in positions [t*fin_tile, (t+1)*fin_tile), so a bucket may be
                                    // as long as kFinCap - fin_tile
constexpr int kFinDigit = 9;         // local sort: 9-bit digits, 512 bins
constexpr int kFinBins = 1 << kFinDigit;
constexpr int kFinFastBits = kFinDigit == 9 ? 27 : 2 * kFinDigit;   // sort bits of the first attempt
constexpr int kFinMaxMeanBucket = 3072;   // the planner partitions until N / 2^T is below this
constexpr int kFinMinTile = 512;    // smallest fin_tile the planner picks (workspace sizing)

// Number of SMs of the current device (grid sizing); queried once per device, 148 on a B200.
// records the text polylab_last_cuda_error returns (api.cu)
void note_cuda_error(cudaError_t e, const char* what);

inline int sm_count()
{
    static int cached[64] = {0};
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) dev = 0;
    if (cached[dev] == 0) {
        int n = 0;
        if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n <= 0) n = 148;
        cached[dev] = n;
    }
    return cached[dev];
}

// cudaFuncAttributeMaxDynamicSharedMemorySize is a per-DEVICE property of a kernel: set once per (kernel, device) -- a
// small table keyed by the kernel's address (many kernels share one function-pointer TYPE) -- instead of on every launch.
bool smem_attr_done(const void* kern, int dev, bool mark);
template <typename F>
inline void ensure_dynamic_smem(F kern, size_t bytes)
{
    int dev = 0;
    const bool known = cudaGetDevice(&dev) == cudaSuccess && dev >= 0 && dev < 64;
    if (known && smem_attr_done((const void*)kern, dev, false)) return;
    if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes) == cudaSuccess && known)
        smem_attr_done((const void*)kern, dev, true);
}

inline int sort_tile(int key_bytes)
{
    return key_bytes == 8 ? kSortThreads64 * kSortItems64 : key_bytes == 16 ? kSortThreads128 * kSortItems128 : kSortThreads256 * kSortItems256;
}
constexpr int kReduceTile = kReduceThreads * kReduceItems;
constexpr int kPruneTile = kPruneThreads * kPruneItems;

// S0: per-variable maxima of an exponent matrix into ctl->max_exp[which][v] (atomicMax).
int launch_bounds(const ExpView& ev, int64_t nterms, int nvars, Control* ctl, int which, cudaStream_t stream);

// S0 on a sample: 1184 evenly spaced segments of 512 rows.  The caller sizes the fields from the sampled maxima's bit
// lengths and relies on S1's range check to catch an exponent the sample missed (then S0 runs in full).
int launch_bounds_sample(const ExpView& ev, int64_t nterms, int nvars, Control* ctl, int which, cudaStream_t stream);

// Product with caller bounds: true maxima of both operands into ctl->max_exp (which must be zero), then
// max_a[v] + max_b[v] > emax -> ctl->status = POLYLAB_ERR_EXPONENT_RANGE (the exponent sums must fit exp_type, reading A8).
int launch_sum_range_check(const ExpView& ea, int64_t na, const ExpView& eb, int64_t nb, int nvars, uint32_t emax, Control* ctl,
                           cudaStream_t stream);

// fp32 -> fp64: out[i] = in[i] (the radix passes take fp64 coefficients only; see CoefIn in common.cuh).
int launch_widen(const void* in_f32, double* out, int64_t n, cudaStream_t stream);

// S1: pack rows into keys (key_bytes from the plan), check e <= plan.bound (-> ctl->status), and, when
// hist_digit >= 0, accumulate the histogram of that plan digit into ctl->hist[hist_digit] (the first pass's digit).
int launch_pack(const ExpView& ev, int64_t nterms, const Plan& plan, void* keys, Control* ctl, int hist_digit,
                cudaStream_t stream);

// Histogram of plan digit `hist_digit` over packed keys into ctl->hist[hist_digit].
int launch_key_hist(const Plan& plan, int hist_digit, int64_t n, const void* keys, Control* ctl, cudaStream_t stream);

// Can S1 be fused into the first radix pass for this exponent matrix?  (row-major, 16-byte aligned base, rows of 8 or 16 bytes)
bool rows_fusable(const ExpView& ev, int nvars);

// Histogram of plan digit `hist_digit` straight from such rows into ctl->hist[hist_digit] (no keys are written).
int launch_row_hist(const ExpView& ev, int64_t nterms, const Plan& plan, int hist_digit, Control* ctl, cudaStream_t stream);

// The same histogram over a sample: `nsegs` evenly spaced segments of `seg_rows` rows, into est[256] (zero before).
int launch_row_hist_sample(const ExpView& ev, int64_t nterms, const Plan& plan, int hist_digit, uint32_t* est, int nsegs, int seg_rows,
                           cudaStream_t stream);
int launch_slack_caps(const uint32_t* est, int64_t n, int64_t capacity, uint32_t* hist, uint32_t* cap, cudaStream_t stream);

// S1 for the test entry point: always writes (hi, lo) pairs.
int launch_pack_hilo(const ExpView& ev, int64_t nterms, const Plan& plan, uint64_t* out_hilo, Control* ctl,
                     cudaStream_t stream);

// X1: all products of packed operands: key = ka_i + kb_j, coef = fl(ca_i * cb_j); N = na*nb pairs written
// to keys/coefs (emission order: i*nb + j); histogram of plan digit `hist_digit` into ctl->hist[hist_digit].
int launch_expand_packed(const void* ka, CoefIn ca, int64_t na, const void* kb, CoefIn cb, int64_t nb,
                         const Plan& plan, void* keys, double* coefs, Control* ctl, int hist_digit, cudaStream_t stream);

// Raw product without keys (polylab_expand): rows a_i + b_j, coefficients fl(ca_i*cb_j).
int launch_expand_raw(const ExpView& ea, CoefIn ca, int64_t na, const ExpView& eb, CoefIn cb, int64_t nb,
                      int nvars, CoefOut out_coef, void* out_exps, Control* ctl_status, cudaStream_t stream);

// S2: one stable radix pass on plan digit `pass` of n (key, coef) pairs from (keys_in, coef_in) to (keys_out,
// coef_out); needs ctl->hist[pass].  `next` >= 0: also accumulate the histogram of plan digit `next` (the digit of
// the following pass) into ctl->hist[next].  `seq` = 0, 1, 2, ... counts the passes of the call: tile_state
// (ceil(n/tile) * 256 words) is zero before pass seq 0 and reused by every later pass (flag parity alternates).
// `rows` (rows_fusable() exponent matrix): S1 fused into the pass -- keys_in is ignored, the keys are packed in
// registers from the rows, range-checked into ctl->status; atomic ranking only.
// safe_rank: ballot-matching ranking (stable by construction); otherwise one shared atomic per record (see sort.cu).
// debug_unstable: test hook, reverses the lane order of the atomic kernel.
// `xs` (packed operands of a product): X1 fused into the pass -- keys_in / coef_in are ignored, record q = i*nb + j is
// formed in registers as (ka_i + kb_j, fl(ca_i * cb_j)); atomic ranking only.
// Slack bins: a pass given per-bin CAPACITIES instead of an exact histogram (`write`: ctl->hist[pass] holds them) lays its
// output out with holes and records the exact counts; the pass after it (`read`, `cap` = the same capacities) cuts its
// tiles per bin of that layout.  ctl->slack_overflow != 0 afterwards: a bin was too small, nothing valid was produced.
constexpr int kSlackExtraTiles = kRadix + 1;     // a pass that reads slack bins cuts its tiles per bin: at most this many more
struct SlackIO {
    bool write, read;
    const uint32_t* cap;        // DEVICE [256]
    uint2* tiles;               // DEVICE [tiles + kSlackExtraTiles]: the reading pass's tile descriptors
    uint32_t capacity;          // records the written buffers hold (>= the sum of the capacities)
};
struct ExpandSrc {
    const void* ka;
    CoefIn ca;
    int64_t na;
    const void* kb;
    CoefIn cb;
    int64_t nb;
};
int launch_sort_pass(const Plan& plan, int pass, int next, int seq, int64_t n, const void* keys_in, const double* coef_in,
                     void* keys_out, double* coef_out, uint32_t* tile_state, Control* ctl, bool safe_rank,
                     bool debug_unstable, cudaStream_t stream, const ExpView* rows = nullptr, const ExpandSrc* xs = nullptr,
                     const struct SlackIO* slack = nullptr);

// Histogram of plan digit `hist_digit` over the na*nb products of packed operands, without storing them.
int launch_expand_hist(const ExpandSrc& xs, const Plan& plan, int hist_digit, Control* ctl, cudaStream_t stream);

// S3: segmented sum over sorted pairs -> (ukeys[U], usums[U]) ascending, ctl->distinct = U; sets ctl->unsorted
// when a key is smaller than its predecessor.
// Scratch: tile_state/tile_heads/tile_hb [ntiles] uint32 (zeroed), tile_frag [ntiles] double, tile_cont [ntiles] uint8.
struct ReduceScratch {
    uint32_t* tile_state;
    uint32_t* tile_heads;
    uint32_t* tile_hb;
    double* tile_frag;
    uint8_t* tile_cont;
};
int launch_reduce(int key_bytes, int64_t n, const void* keys, CoefIn coefs, void* ukeys, double* usums,
                  const ReduceScratch& sc, Control* ctl, cudaStream_t stream);

// S4+S5: keep |s| > tol, order-preserving compaction, unpack into out_coef/out_exps (row-major, exp_bytes);
// ctl->survivors = U'.  max_units bounds U (grid sizing); tile_state: ceil(max_units/kPruneTile) words, zeroed.
int launch_prune_unpack(const Plan& plan, int64_t max_units, const void* ukeys, const double* usums, double tol,
                        CoefOut out_coef, void* out_exps, int exp_bytes, int64_t out_capacity, uint32_t* tile_state,
                        Control* ctl, int64_t* out_count_device, cudaStream_t stream, void* out_keys = nullptr);
// (out_keys != nullptr: packed output -- the survivors' KEYS go to out_keys[U'] instead of unpacked rows to out_exps)

// DEVICE_COUNT calls: *status_device = ctl->status, or POLYLAB_ERR_RETRY (and a zero count) when a self-check failed.
int launch_async_status(const Control* ctl, int32_t* status_device, int64_t* out_count_device, cudaStream_t stream);

// Bucket path (finish.cu): the pairs are sorted by their top `prefix_passes` plan digits; finish every bucket in
// shared memory and emit the simplified polynomial (S2 rest + S3 + S4 + S5).  (ukeys, usums): scratch for n pairs.
// tile_start, tile_state: ceil(n/fin_tile)+1 words each, tile_state zeroed; worklist: as many uint4; chunk_sum: ceil(tiles/4096) words.  after_tiles (optional): recorded
// between the finish kernel and the scan/emit kernels, for the stage timing.  Sets ctl->overflow (nothing emitted) when a bucket is too long,
// ctl->unsorted when the prefix order or the local order check fails, ctl->distinct, ctl->survivors.
// group: 1 = every tile goes through finish_group_kernel first (like terms grouped in a shared-memory hash table, only the
// distinct keys sorted), which marks the tiles it finished in the work list; the sorting finish_kernel behind it does the
// rest (ctl->fin2_count of them); 2 = test hook, the group kernel leaves every tile; 0 = sorting kernel only.
int launch_finish(const Plan& plan, int prefix_passes, int nfast, int fin_tile, int64_t n, const void* keys, const double* coefs,
                  double tol, void* ukeys, double* usums, CoefOut out_coef, void* out_exps, int exp_bytes, int64_t out_capacity,
                  uint32_t* tile_start, uint32_t* tile_state, uint4* worklist, int group, uint32_t* chunk_sum,
                  Control* ctl, int64_t* out_count_device, cudaEvent_t after_tiles, cudaStream_t stream);

// Small inputs (small.cu): S2 + S3 of at most small_cap() (key, coef) pairs in ONE thread block -- radix sort of a permutation
// in shared memory, segmented sum; (ukeys, usums)[U] ascending and ctl->distinct = U as launch_reduce leaves them (then
// launch_prune_unpack).  Sets ctl->unsorted if its atomic ranking turned out unstable.
// n_device (optional, DEVICE): the pair count is read on the device (clamped) instead of `n`.
constexpr int kSmallCap = 8192;          // 64-bit keys; 4096 for 128-bit keys, 2048 for 256-bit keys
inline int small_cap(int key_bytes) { return kSmallCap * 8 / key_bytes; }
int launch_block_sort_reduce(const Plan& plan, const void* keys, CoefIn coefs, const uint32_t* n_device, uint32_t n,
                             void* ukeys, double* usums, Control* ctl, cudaStream_t stream);

// Batched simplify (batch.cu): the records of all entries, keyed (entry, monomial).
struct BatchSeg {
    uint32_t start;         // number of the segment's first record
    uint32_t a0, na;        // terms [a0, a0 + na) of the packed operand A (or of the packed polynomial when nb == 0)
    uint32_t b0, nb;        // terms [b0, b0 + nb) of B: the segment holds the na * nb products; nb == 0: the na raw terms
    uint32_t entry;         // the polynomial (matrix entry) the segment's records belong to
};
int launch_batched_expand(const Plan& plan, const BatchSeg* segs, uint32_t nseg, int64_t n, const void* ka, CoefIn ca,
                          const void* kb, CoefIn cb, int entry_shift, void* keys, double* coefs, Control* ctl, cudaStream_t stream);
int launch_entry_count(int key_bytes, int key_bits, int64_t max_units, const void* ukeys, const double* usums, const Control* ctl, double tol,
                       int entry_shift, uint32_t* counts, cudaStream_t stream);

// Table path (table.cu): merge like terms in a dense or hash table before any sort.
struct __align__(16) TableSlot {
    uint64_t key1;          // packed key + 1; 0 = empty
    uint32_t ord;           // dense ordinal of the key, 0..U-1 (index into the accumulators)
    uint32_t meta;          // largest biased coefficient exponent seen + 1; 2048 = a non-finite coefficient; 0 = untouched
};
struct TableSrc {           // the N records: packed keys + coefficients, or (keys == nullptr) the products of packed operands
    const uint64_t* keys;
    CoefIn coef;
    const void* ka;
    CoefIn ca;
    const void* kb;
    CoefIn cb;
    uint32_t nb;
    uint32_t n;
};
struct TableArgs {
    TableSlot* slots;       // hash: [cmask + 1]
    uint32_t cmask;
    uint32_t limit;         // hash: most distinct keys before the path is abandoned
    uint32_t* meta;         // dense: [2^B]
    unsigned long long* acc_hi;   // [nord] fixed-point accumulators (two limbs of p bits)
    unsigned long long* acc_lo;
    uint32_t nord;          // dense: 2^B; hash: U (known after the insert pass)
    uint32_t nsm;           // set by launch_table_accum: ordinals below this are accumulated in shared memory
    int p;                  // limb width in bits
    Control* ctl;
};
constexpr int64_t kTableMaxTerms = (int64_t)1 << 26;      // the fixed-point error bound is derived for N <= 2^26 (table.cu)
constexpr int64_t kTableMinTerms = (int64_t)1 << 15;
constexpr int kTableDenseMaxBits = 22;
constexpr uint32_t kTableMaxDistinct = 1u << 20;
inline uint32_t table_dense_tile() { return 256u * 8u; }
int launch_table_insert(const TableSrc& src, const TableArgs& t, bool dense, cudaStream_t stream);
// S1 fused into the insert pass: contiguous row-major rows (ev.row_major_contiguous) -> keys[nterms] written, every record
// inserted, the range check into ctl->status and (hd >= 0) the histogram of plan digit hd into ctl->hist[hd] as launch_pack does.
int launch_table_insert_rows(const ExpView& ev, int64_t nterms, const Plan& plan, uint64_t* keys, CoefIn coef, const TableArgs& t,
                             bool dense, int hd, cudaStream_t stream);
int launch_table_accum(const TableSrc& src, const TableArgs& t, bool dense, cudaStream_t stream);
int launch_table_finalize(const TableArgs& t, uint64_t* ukeys, double* usums, cudaStream_t stream);
int launch_table_dense_emit(const TableArgs& t, const Plan& plan, double tol, CoefOut out_coef, void* out_exps, int exp_bytes,
                            int64_t out_capacity, uint32_t* tile_state, int64_t* out_count_device, cudaStream_t stream);

}  // namespace polylab
