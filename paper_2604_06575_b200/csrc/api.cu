// api.cu -- the C ABI of include/polylab.h: argument checks, the key-layout plan, workspace carving and
// the launch sequence  S0 bounds -> S1 pack -> (X1 expand) -> S2 radix passes -> S3 reduce -> S4/S5.
// No step of the path runs on the host; the host only sizes and launches.
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include "kernels.h"

#include <mutex>

namespace polylab {

// (kernel address -> devices on which its dynamic shared-memory limit has been raised); see ensure_dynamic_smem
bool smem_attr_done(const void* kern, int dev, bool mark)
{
    static std::mutex mu;
    static const void* keys[256];
    static unsigned long long masks[256];
    static int used = 0;
    std::lock_guard<std::mutex> lock(mu);
    for (int i = 0; i < used; ++i)
        if (keys[i] == kern) {
            if (mark) masks[i] |= 1ull << dev;
            return (masks[i] >> dev) & 1ull;
        }
    if (mark && used < 256) { keys[used] = kern; masks[used] = 1ull << dev; ++used; return true; }
    return false;
}

static thread_local char g_cuda_error[256] = "";

// internal return values of one attempt: the sorted-order check failed with the atomic-ranking kernels -> re-run with
// ballot ranking on the LSD path; a bucket of the bucket path was too long -> re-run on the LSD path
constexpr int kRetrySafeRank = -1000;
constexpr int kRetryNoBucket = -1001;
constexpr int kRetryExactBounds = -1002;       // an exponent exceeded the field sized from the sampled maxima
constexpr int kRetryExactHist = -1003;         // a slack bin sized from the sampled histogram was too small

struct Attempt {
    bool safe_rank;        // ballot-matching radix passes, LSD path only
    bool allow_bucket;     // may take the bucket path (finish.cu)
    bool exact_bounds;     // S0 reads every row (otherwise large inputs are sampled and S1's range check verifies)
    bool allow_table;      // may take the table path (table.cu); only the first attempt does
    bool exact_hist;       // the first prefix pass gets an exact histogram (otherwise large fused inputs use slack bins)
};

static bool cuda_failed(cudaError_t e, const char* what)
{
    if (e == cudaSuccess) return false;
    snprintf(g_cuda_error, sizeof g_cuda_error, "%s: %s", what, cudaGetErrorString(e));
    return true;
}
// (for static_ws.cu, whose set-up runs outside this file: the text polylab_last_cuda_error returns)
void note_cuda_error(cudaError_t e, const char* what) { cuda_failed(e, what); }
#define PL_CUDA(call)                                            \
    do {                                                         \
        if (cuda_failed((call), #call)) return POLYLAB_ERR_CUDA; \
    } while (0)

constexpr int64_t kSampleBoundsMinTerms = (int64_t)1 << 22;   // below this S0 reads every row

static inline size_t align_up(size_t x, size_t a = 256) { return (x + a - 1) / a * a; }
static inline int bitlen(uint64_t x) { int b = 0; while (x) { ++b; x >>= 1; } return b; }
static inline uint32_t exp_max_of(int exp_bytes) { return exp_bytes == 1 ? 0xffu : exp_bytes == 2 ? 0xffffu : 0xffffffffu; }

struct Opts {
    int exp_bytes;
    int coef_f32;          // coefficient arrays of the caller are fp32 (opts->coef_type)
    uint32_t flags;
    int64_t term_stride, var_stride;
    const uint32_t* max_exp_host;
    int32_t* status_device;
    polylab_stats* stats;
};

static int parse_opts(const polylab_opts* o, int nvars, Opts* out)
{
    Opts r;
    r.exp_bytes = 4; r.coef_f32 = 0; r.flags = 0; r.term_stride = nvars; r.var_stride = 1;
    r.max_exp_host = nullptr; r.status_device = nullptr; r.stats = nullptr;
    if (o) {
        if (o->exp_type != 0) {
            if (o->exp_type != POLYLAB_EXP_U8 && o->exp_type != POLYLAB_EXP_U16 && o->exp_type != POLYLAB_EXP_U32)
                return POLYLAB_ERR_INVALID_ARGUMENT;
            r.exp_bytes = o->exp_type;
        }
        r.flags = o->flags;
        if (o->coef_type != POLYLAB_COEF_F64 && o->coef_type != POLYLAB_COEF_F32) return POLYLAB_ERR_INVALID_ARGUMENT;
        r.coef_f32 = o->coef_type == POLYLAB_COEF_F32;
        if (o->term_stride != 0 || o->var_stride != 0) { r.term_stride = o->term_stride; r.var_stride = o->var_stride; }
        if (r.term_stride < 0 || r.var_stride < 0) return POLYLAB_ERR_INVALID_ARGUMENT;
        r.max_exp_host = o->max_exp_host;
        r.status_device = o->status_device;
        r.stats = o->stats;
    }
    if ((r.flags & POLYLAB_FLAG_DEVICE_COUNT) && !r.max_exp_host) return POLYLAB_ERR_INVALID_ARGUMENT;
    *out = r;
    return POLYLAB_OK;
}

static ExpView make_view(const void* base, const Opts& o, int nvars)
{
    ExpView v;
    v.base = base;
    v.term_stride = o.term_stride;
    v.var_stride = o.var_stride;
    v.exp_bytes = o.exp_bytes;
    v.row_major_contiguous = (o.term_stride == nvars && o.var_stride == 1 && ((uintptr_t)base % 16) == 0) ? 1 : 0;
    return v;
}

// Key layout from the per-variable maxima m_v of the rows that will be SORTED (for a product: max_a + max_b)
// and the bounds that INPUT rows must respect.  Variable 0 gets the most significant field (reading A1).
static int make_plan(int nvars, const uint64_t* m, const uint32_t* bound, Plan* plan)
{
    memset(plan, 0, sizeof *plan);
    plan->nvars = nvars;
    int bits = 0;
    for (int v = nvars - 1; v >= 0; --v) {
        const int w = bitlen(m[v]);
        if (w > 32) return POLYLAB_ERR_EXPONENT_RANGE;
        if (bits + w > 256) return POLYLAB_ERR_KEY_TOO_WIDE;
        plan->shift[v] = (uint8_t)(w ? bits : 0);
        plan->width[v] = (uint8_t)w;
        plan->bound[v] = bound[v];
        bits += w;
    }
    plan->key_bits = bits;
    plan->key_bytes = bits <= 64 ? 8 : bits <= 128 ? 16 : 32;
    // Digits: each 32-bit word of the key is split into ceil(bits_in_word / 8) digits of balanced width, so no digit
    // straddles a word (one shift + mask per digit) and the pass count is still ceil(B / 8).
    int P = 0;
    for (int w = 0; w * 32 < bits; ++w) {
        const int nb = bits - w * 32 < 32 ? bits - w * 32 : 32;
        const int pw = (nb + kRadixBits - 1) / kRadixBits;
        int pos = w * 32;
        for (int p = 0; p < pw; ++p) {
            const int dw = nb / pw + (p < nb % pw ? 1 : 0);
            plan->digit_pos[P] = (uint8_t)pos;
            plan->digit_bits[P] = (uint8_t)dw;
            pos += dw;
            ++P;
        }
    }
    plan->npasses = P;
    return POLYLAB_OK;
}

// ------------------------------------------------------------------------------ workspace carving

struct Layout {
    size_t control, sort_state, slack_tiles, red_state, red_heads, red_hb, red_frag, red_cont, prune_state, fin_state, fin_start, fin_wl, fin_chunks, zero_end;
    size_t tab_state, tab, tab_bytes;
    size_t keys[2], coefs[2], ka, kb, ca, cb, total;      // ca, cb: fp32 operand coefficients of a product, widened to fp64
};

// Table path (table.cu): the dense table indexes 2^B slots with the key itself (B <= 22 and no more slots than
// max(N, 65536)); the hash table has room for `limit` distinct keys at load <= 1/2.
static int64_t table_max_dense_slots(int64_t n)
{
    if (n > kTableMaxTerms) return 0;
    int64_t s = n > 65536 ? n : 65536;
    if (s > ((int64_t)1 << kTableDenseMaxBits)) s = (int64_t)1 << kTableDenseMaxBits;
    return s;
}
static uint32_t table_limit(int64_t n, bool forced)
{
    if (forced) return (uint32_t)(n < 1024 ? 1024 : n > 16384 ? 16384 : n);   // test hook: small inputs are never abandoned
    int64_t l = n / 4;
    if (l > (int64_t)kTableMaxDistinct) l = kTableMaxDistinct;
    return (uint32_t)(l < 1 ? 1 : l);
}
static uint32_t table_capacity(uint32_t limit)
{
    uint32_t c = 1024;
    while (c < 2u * limit) c <<= 1;
    return c;
}
static size_t table_hash_bytes(uint32_t limit) { return (size_t)table_capacity(limit) * sizeof(TableSlot) + (size_t)limit * 16 + 512; }
static size_t table_region_bytes(int64_t n)
{
    if (n < 1 || n > kTableMaxTerms) return 0;
    const size_t dense = (size_t)table_max_dense_slots(n) * 20 + 768;
    size_t hash = table_hash_bytes(table_limit(n, false));
    { const size_t f = table_hash_bytes(table_limit(n, true)); if (f > hash) hash = f; }
    return dense > hash ? dense : hash;
}

// Slack bins (sort.cu): from kSampleBoundsMinTerms terms on, the first prefix pass of a fused bucket-path call may take its
// bin capacities from a sampled histogram; its output then needs room for the sum of the capacities.
static int64_t slack_capacity(int64_t n) { return n >= kSampleBoundsMinTerms ? n + n / 8 + ((int64_t)1 << 21) : n; }

static Layout make_layout(int64_t n, int key_bytes, int64_t na, int64_t nb)
{
    Layout L;
    size_t off = 0;
    auto take = [&](size_t bytes) { const size_t o = off; off = align_up(off + bytes); return o; };
    const size_t sort_tiles = (size_t)((n + sort_tile(key_bytes) - 1) / sort_tile(key_bytes));
    const size_t red_tiles = (size_t)((n + kReduceTile - 1) / kReduceTile);
    const size_t prune_tiles = (size_t)((n + kPruneTile - 1) / kPruneTile);
    L.control = take(sizeof(Control));
    L.sort_state = take((sort_tiles + kSlackExtraTiles) * kRadix * sizeof(uint32_t));
    L.red_state = take(red_tiles * sizeof(uint32_t));
    L.prune_state = take(prune_tiles * sizeof(uint32_t));
    const size_t fin_tiles = (size_t)((n + kFinMinTile - 1) / kFinMinTile);
    L.fin_state = take((fin_tiles + 1) * sizeof(uint32_t));
    L.tab_state = take(((size_t)table_max_dense_slots(n) / table_dense_tile() + 2) * sizeof(uint32_t));
    L.zero_end = off;                                   // everything before this is zeroed per call
    L.tab_bytes = table_region_bytes(n);
    L.tab = take(L.tab_bytes);
    L.slack_tiles = take((sort_tiles + kSlackExtraTiles) * sizeof(uint2));     // (written in full by slack_tiles_kernel)
    L.fin_start = take((fin_tiles + 1) * sizeof(uint32_t));
    L.fin_wl = take((fin_tiles + 1) * sizeof(uint4));
    L.fin_chunks = take((fin_tiles / 4096 + 2) * sizeof(uint32_t));
    L.red_heads = take(red_tiles * sizeof(uint32_t));
    L.red_hb = take(red_tiles * sizeof(uint32_t));
    L.red_frag = take(red_tiles * sizeof(double));
    L.red_cont = take(red_tiles);
    // (the second buffers receive the first prefix pass, which may lay its bins out with slack: see slack_capacity)
    for (int i = 0; i < 2; ++i) L.keys[i] = take((size_t)(i ? slack_capacity(n) : n) * key_bytes);
    for (int i = 0; i < 2; ++i) L.coefs[i] = take((size_t)(i ? slack_capacity(n) : n) * sizeof(double));
    L.ka = take((size_t)na * key_bytes);
    L.kb = take((size_t)nb * key_bytes);
    L.ca = take((size_t)na * sizeof(double));
    L.cb = take((size_t)nb * sizeof(double));
    L.total = off;
    return L;
}

// Widest key a call can need: every variable's field is at most as wide as its exponent type (a product's sums must fit
// that type too), plus `extra_bits` (the entry field of a batched call).
static int max_key_bytes(int nvars, const polylab_opts* opts, int extra_bits = 0)
{
    const int es = (opts && opts->exp_type) ? opts->exp_type : 4;
    const int64_t bits = (int64_t)nvars * 8 * es + extra_bits;
    return bits <= 64 ? 8 : bits <= 128 ? 16 : 32;
}

static size_t worst_layout_bytes(int64_t n, int64_t na, int64_t nb, int widest_key_bytes = 32)
{
    size_t best = 0;
    for (int kb = 8; kb <= widest_key_bytes; kb *= 2) {
        const size_t t = make_layout(n, kb, na, nb).total;
        best = t > best ? t : best;
    }
    return best + 256;                                  // + slack to align the caller's base pointer
}

static void fill_stats(polylab_stats* st, const Plan& plan, int64_t n)
{
    if (!st) return;
    const int32_t launches = st->kernel_launches, fallback = st->rank_fallback, bfall = st->bucket_fallback, bretry = st->bounds_retry;
    const int32_t tfall = st->table_fallback, hretry = st->hist_retry;
    memset(st, 0, sizeof *st);
    st->table_fallback = tfall;
    st->hist_retry = hretry;
    st->kernel_launches = launches;
    st->rank_fallback = fallback;
    st->bucket_fallback = bfall;
    st->bounds_retry = bretry;
    st->key_bits = plan.key_bits;
    st->key_bytes = plan.key_bytes;
    st->sort_passes = plan.npasses;
    st->plan_digits = plan.npasses;
    for (int p = 0; p < plan.npasses; ++p) st->digit_bits[p] = plan.digit_bits[p];
    st->sort_terms = n;
    st->distinct = -1;
    st->survivors = -1;
}

// ------------------------------------------------------------------------------- stage timing

// Optional CUDA events between the steps (POLYLAB_FLAG_TIMING): recorded on the call's stream, read after
// the call's final synchronisation.  Events are created once per host thread.
struct Timing {
    bool on = false;
    cudaStream_t stream = nullptr;
    cudaEvent_t ev[POLYLAB_STAGE_COUNT + 1];
    void begin(bool enable, cudaStream_t s)
    {
        static thread_local cudaEvent_t pool[POLYLAB_STAGE_COUNT + 1];
        static thread_local bool made = false;
        on = enable;
        stream = s;
        if (!on) return;
        if (!made) {
            for (auto& e : pool) cudaEventCreate(&e);
            made = true;
        }
        for (int i = 0; i <= POLYLAB_STAGE_COUNT; ++i) ev[i] = pool[i];
        cudaEventRecord(ev[0], stream);
    }
    void mark(int stage) { if (on) cudaEventRecord(ev[stage + 1], stream); }     // end of `stage`
    void finish(polylab_stats* st)
    {
        if (!on || !st) return;
        for (int i = 0; i < POLYLAB_STAGE_COUNT; ++i) cudaEventElapsedTime(&st->stage_ms[i], ev[i], ev[i + 1]);
    }
};

// ------------------------------------------------------------------------------- bucket path plan

// How many of the most significant plan digits to partition on before finishing in shared memory (0 = LSD path).
// The buckets must average at most one finish tile; the path pays only when it replaces at least three LSD passes.
static int choose_prefix_passes(const Plan& plan, int64_t n, const Opts& o, const Attempt& at)
{
    const bool force = (o.flags & POLYLAB_FLAG_DEBUG_FORCE_BUCKET) != 0;
    if (!at.allow_bucket || at.safe_rank || (o.flags & POLYLAB_FLAG_NO_BUCKET)) return 0;
    const int P = plan.npasses;
    if (plan.key_bytes > 16) return 0;                  // finish.cu handles one- and two-word keys
    if (P < 1 || (!force && (P < 4 || n < (1 << 20)))) return 0;
    for (int k = 1; k <= P; ++k) {
        const int T = plan.key_bits - plan.digit_pos[P - k];
        if (T >= 40 || (n >> T) < kFinMaxMeanBucket) return (force || P - k >= 3) ? k : 0;
    }
    return 0;
}

// Room a finish tile leaves for its longest bucket: twice the mean bucket N / 2^T (duplicated monomials make bucket
// sizes much wider than Poisson), within [512, kFinCap - kFinMinTile]; the tile covers the other kFinCap - room positions.
static int bucket_room(const Plan& plan, int k, int64_t n)
{
    const int T = plan.key_bits - plan.digit_pos[plan.npasses - k];
    const int64_t mean = T >= 40 ? 0 : (n >> T);
    int64_t room = 2 * mean;
    if (room < 512) room = 512;
    if (room > kFinCap - kFinMinTile) room = kFinCap - kFinMinTile;
    return (int)room;
}

static int fast_digits(const Opts& o)
{
    const int dbg = (int)((o.flags >> POLYLAB_FLAG_DEBUG_NFAST_SHIFT) & 0xfu);
    return dbg;                    // 0 = no limit: as many bits below the prefix as fit the 27-bit composite sort word
}

// 1: tiles go through the group kernel first (finish.cu); 0: the sorting finish kernel only; 2: test hook, the group kernel
// runs and hands every tile on
static int finish_group_mode(const Opts& o)
{
    if (o.flags & POLYLAB_FLAG_NO_GROUP_FINISH) return 0;
    // (the fast-digits hook is about the sorting kernel's local sort: every tile must reach it)
    return ((o.flags & POLYLAB_FLAG_DEBUG_GROUP_HANDS_ON) || fast_digits(o) != 0) ? 2 : 1;
}

// After S1/X1 accumulated the histogram of the first prefix digit: do its bins predict buckets that fit a tile?
// (A necessary test only; tile_bounds_kernel has the last word.)  On rejection the LSD path needs digit 0's histogram.
static int bucket_precheck(const Plan& plan, int* k, int64_t n, unsigned char* ws, const Layout& L, const Opts& o,
                           int* launches, cudaStream_t stream, const ExpView* unpacked = nullptr, const ExpandSrc* xs = nullptr)
{
    // (an asynchronous call cannot read the histogram back: tile_bounds_kernel alone decides, through status_device)
    if (*k == 0 || (o.flags & (POLYLAB_FLAG_DEBUG_FORCE_BUCKET | POLYLAB_FLAG_DEVICE_COUNT))) return POLYLAB_OK;
    // (the rejection branch below is the only one that needs `unpacked`)
    Control* ctl = (Control*)(ws + L.control);
    const int P = plan.npasses, d = P - *k;
    uint32_t h[kRadix];
    PL_CUDA(cudaMemcpyAsync(h, ctl->hist[d], sizeof h, cudaMemcpyDeviceToHost, stream));
    PL_CUDA(cudaStreamSynchronize(stream));
    uint64_t mx = 0;
    for (int b = 0; b < kRadix; ++b) mx = h[b] > mx ? h[b] : mx;
    const int rest = plan.key_bits - plan.digit_pos[d] - plan.digit_bits[d];      // prefix bits above this digit
    if ((mx >> rest) <= (uint64_t)bucket_room(plan, *k, n) * 7 / 8) return POLYLAB_OK;
    *k = 0;
    if (o.stats) o.stats->bucket_fallback = 1;
    PL_CUDA(cudaMemsetAsync(ctl->hist[d], 0, sizeof h, stream));
    if (xs) *launches += launch_expand_hist(*xs, plan, 0, ctl, stream);                             // X1 stays in the first pass
    else if (unpacked) *launches += launch_pack(*unpacked, n, plan, ws + L.keys[0], ctl, 0, stream);   // S1 had been left to the first pass
    else *launches += launch_key_hist(plan, 0, n, ws + L.keys[0], ctl, stream);
    return POLYLAB_OK;
}

// ----------------------------------------------------------------------- shared tail of both paths

// keys/coefs of the N unsorted pairs are in (L.keys[0], coef0); digit-0 histogram is in ctl->hist[0].
struct Readback { int32_t status; uint32_t distinct, survivors, unsorted, overflow, refinish, fin_count, tab_count, tab_overflow, slack_overflow, fin2_count; };

// Bucket path: k stable passes over the top k digits, then finish.cu.  The pairs are in (L.keys[0], coef0) and the
// histogram of digit P-k is in ctl->hist[P-k].
static int bucket_sort_emit(const Plan& plan, int k, int64_t n, unsigned char* ws, const Layout& L, CoefIn coef0,
                            double tol, const Opts& o, CoefOut out_coef, void* out_exps, int64_t out_capacity,
                            int64_t* out_nterms, int* launches, Timing& tm, cudaStream_t stream, const ExpView* rows,
                            const ExpandSrc* xs, bool slack)
{
    Control* ctl = (Control*)(ws + L.control);
    void* kbuf[2] = {ws + L.keys[0], ws + L.keys[1]};
    double* cbuf[2] = {(double*)(ws + L.coefs[0]), (double*)(ws + L.coefs[1])};
    const int P = plan.npasses;
    if (coef0.f32) {                                     // the radix passes take fp64: widen into the buffer the first pass does not write
        *launches += launch_widen(coef0.p, cbuf[0], n, stream);
        coef0 = CoefIn(cbuf[0]);
    }
    for (int s = 0; s < k; ++s) {
        const double* cin = (s == 0) ? (const double*)coef0.p : cbuf[s & 1];
        const SlackIO sio = {slack && s == 0, slack && s == 1, ctl->slack_cap, (uint2*)(ws + L.slack_tiles), (uint32_t)slack_capacity(n)};
        *launches += launch_sort_pass(plan, P - k + s, s + 1 < k ? P - k + s + 1 : -1, s, n, kbuf[s & 1], cin, kbuf[(s + 1) & 1],
                                      cbuf[(s + 1) & 1], (uint32_t*)(ws + L.sort_state), ctl, false,
                                      (o.flags & POLYLAB_FLAG_DEBUG_UNSTABLE) != 0, stream, s == 0 ? rows : nullptr,
                                      s == 0 ? xs : nullptr, (slack && s < 2) ? &sio : nullptr);
    }
    tm.mark(POLYLAB_STAGE_SORT);
    *launches += launch_finish(plan, k, fast_digits(o), kFinCap - bucket_room(plan, k, n), n, kbuf[k & 1], cbuf[k & 1], tol,
                               kbuf[(k + 1) & 1], cbuf[(k + 1) & 1], out_coef, out_exps, o.exp_bytes, out_capacity,
                               (uint32_t*)(ws + L.fin_start), (uint32_t*)(ws + L.fin_state), (uint4*)(ws + L.fin_wl),
                               finish_group_mode(o), (uint32_t*)(ws + L.fin_chunks), ctl,
                               (o.flags & POLYLAB_FLAG_DEVICE_COUNT) ? out_nterms : nullptr,
                               tm.on ? tm.ev[POLYLAB_STAGE_REDUCE + 1] : nullptr, stream);      // REDUCE = tiles, PRUNE = scan + emit
    tm.mark(POLYLAB_STAGE_PRUNE);
    PL_CUDA(cudaGetLastError());
    if (o.flags & POLYLAB_FLAG_DEVICE_COUNT) {             // no read-back: the self-checks report through status_device
        *launches += launch_async_status(ctl, o.status_device, out_nterms, stream);
        if (o.stats) { o.stats->kernel_launches += *launches; o.stats->prefix_passes = k; o.stats->sort_passes = k; o.stats->hist_sampled = slack ? 1 : 0; }
        return POLYLAB_OK;
    }
    if (o.stats) o.stats->kernel_launches += *launches;
    Readback res;
    PL_CUDA(cudaMemcpyAsync(&res, &ctl->status, sizeof res, cudaMemcpyDeviceToHost, stream));
    PL_CUDA(cudaStreamSynchronize(stream));
    if (res.status == POLYLAB_ERR_EXPONENT_RANGE) return res.status;   // keys built from out-of-range exponents prove nothing below
    if (slack && res.slack_overflow) return kRetryExactHist;           // a sampled bin capacity was too small: nothing valid below
    if (res.overflow) return kRetryNoBucket;
    if (res.unsorted) return kRetrySafeRank;
    tm.finish(o.stats);
    if (o.stats) {
        o.stats->distinct = res.distinct; o.stats->survivors = res.survivors;
        o.stats->prefix_passes = k; o.stats->sort_passes = k; o.stats->refinish_tiles = (int32_t)res.refinish;
        o.stats->grouped_tiles = finish_group_mode(o) ? (int32_t)(res.fin_count - res.fin2_count) : 0;
        o.stats->hist_sampled = slack ? 1 : 0;
    }
    if (res.status != POLYLAB_OK) return res.status;
    *out_nterms = (int64_t)res.survivors;
    return (int64_t)res.survivors > out_capacity ? POLYLAB_ERR_OUTPUT_TOO_SMALL : POLYLAB_OK;
}

// At most kSmallCap pairs: one thread block does S2-S5 (small.cu).  The sort path's test hooks mean the multi-kernel path.
static bool small_eligible(int64_t n, const Plan& plan, const Opts& o)
{
    if (n > small_cap(plan.key_bytes) || (o.flags & (POLYLAB_FLAG_NO_SMALL | POLYLAB_FLAG_SAFE_RANK))) return false;
    return !(o.flags & (POLYLAB_FLAG_DEBUG_FORCE_BUCKET | POLYLAB_FLAG_DEBUG_UNSTABLE | (0xfu << POLYLAB_FLAG_DEBUG_NFAST_SHIFT)));
}

// Batched calls (batch.cu): after the segmented sum, count the survivors of every entry (the key's top field).
struct BatchOut { int entry_shift; uint32_t* counts; };

static int sort_reduce_emit(const Plan& plan, int k_bucket, int64_t n, unsigned char* ws, const Layout& L, CoefIn coef0,
                            double tol, const Opts& o, CoefOut out_coef, void* out_exps, int64_t out_capacity,
                            int64_t* out_nterms, int* launches, Timing& tm, bool safe_rank, cudaStream_t stream,
                            const ExpView* rows = nullptr, const ExpandSrc* xs = nullptr, const BatchOut* batch = nullptr,
                            void* packed_keys = nullptr, bool slack = false)
{
    if (k_bucket > 0)
        return bucket_sort_emit(plan, k_bucket, n, ws, L, coef0, tol, o, out_coef, out_exps, out_capacity, out_nterms, launches,
                                tm, stream, rows, xs, slack);
    Control* ctl = (Control*)(ws + L.control);
    void* kbuf[2] = {ws + L.keys[0], ws + L.keys[1]};
    double* cbuf[2] = {(double*)(ws + L.coefs[0]), (double*)(ws + L.coefs[1])};
    const int P = plan.npasses;
    const bool dev_count = (o.flags & POLYLAB_FLAG_DEVICE_COUNT) != 0;
    const bool small = xs == nullptr && !safe_rank && small_eligible(n, plan, o);   // (its ranking is the atomic one)
    if (small) {
        tm.mark(POLYLAB_STAGE_SORT);
        *launches += launch_block_sort_reduce(plan, kbuf[0], coef0, nullptr, (uint32_t)n, kbuf[1], cbuf[1], ctl, stream);
        if (batch) *launches += launch_entry_count(plan.key_bytes, plan.key_bits, n, kbuf[1], cbuf[1], ctl, tol, batch->entry_shift, batch->counts, stream);
        tm.mark(POLYLAB_STAGE_REDUCE);
        *launches += launch_prune_unpack(plan, n, kbuf[1], cbuf[1], tol, out_coef, out_exps, o.exp_bytes, out_capacity,
                                         (uint32_t*)(ws + L.prune_state), ctl, dev_count ? out_nterms : nullptr, stream, packed_keys);
        if (o.stats) { o.stats->small_path = 1; o.stats->sort_passes = 0; }
    } else {
        if (coef0.f32 && P > 0) {                        // the radix passes take fp64: widen into the buffer the first pass does not write
            *launches += launch_widen(coef0.p, cbuf[0], n, stream);
            coef0 = CoefIn(cbuf[0]);
        }
        for (int p = 0; p < P; ++p) {
            const double* cin = (p == 0) ? (const double*)coef0.p : cbuf[p & 1];
            *launches += launch_sort_pass(plan, p, p + 1 < P ? p + 1 : -1, p, n, kbuf[p & 1], cin, kbuf[(p + 1) & 1],
                                          cbuf[(p + 1) & 1], (uint32_t*)(ws + L.sort_state), ctl, safe_rank,
                                          (o.flags & POLYLAB_FLAG_DEBUG_UNSTABLE) != 0, stream, nullptr, p == 0 ? xs : nullptr);
        }
        tm.mark(POLYLAB_STAGE_SORT);
        const void* skeys = kbuf[P & 1];
        const CoefIn scoef = (P == 0) ? coef0 : CoefIn(cbuf[P & 1]);
        void* ukeys = kbuf[(P + 1) & 1];
        double* usums = cbuf[(P + 1) & 1];
        ReduceScratch sc;
        sc.tile_state = (uint32_t*)(ws + L.red_state);
        sc.tile_heads = (uint32_t*)(ws + L.red_heads);
        sc.tile_hb = (uint32_t*)(ws + L.red_hb);
        sc.tile_frag = (double*)(ws + L.red_frag);
        sc.tile_cont = (uint8_t*)(ws + L.red_cont);
        *launches += launch_reduce(plan.key_bytes, n, skeys, scoef, ukeys, usums, sc, ctl, stream);
        if (batch) *launches += launch_entry_count(plan.key_bytes, plan.key_bits, n, ukeys, usums, ctl, tol, batch->entry_shift, batch->counts, stream);
        tm.mark(POLYLAB_STAGE_REDUCE);
        *launches += launch_prune_unpack(plan, n, ukeys, usums, tol, out_coef, out_exps, o.exp_bytes, out_capacity,
                                         (uint32_t*)(ws + L.prune_state), ctl, dev_count ? out_nterms : nullptr, stream, packed_keys);
    }
    tm.mark(POLYLAB_STAGE_PRUNE);
    PL_CUDA(cudaGetLastError());
    if (o.stats) o.stats->kernel_launches += *launches;
    if (dev_count) {
        *launches += launch_async_status(ctl, o.status_device, out_nterms, stream);
        if (o.stats) o.stats->kernel_launches += 1;
        return POLYLAB_OK;
    }
    struct { int32_t status; uint32_t distinct, survivors, unsorted; } res;
    PL_CUDA(cudaMemcpyAsync(&res, &ctl->status, sizeof res, cudaMemcpyDeviceToHost, stream));
    PL_CUDA(cudaStreamSynchronize(stream));
    if (res.status == POLYLAB_ERR_EXPONENT_RANGE) return res.status;   // keys built from out-of-range exponents prove nothing below
    if (res.unsorted) return safe_rank ? (int)POLYLAB_ERR_INTERNAL : kRetrySafeRank;
    tm.finish(o.stats);
    if (o.stats) { o.stats->distinct = res.distinct; o.stats->survivors = res.survivors; }
    if (res.status != POLYLAB_OK) return res.status;
    *out_nterms = (int64_t)res.survivors;
    return (int64_t)res.survivors > out_capacity ? POLYLAB_ERR_OUTPUT_TOO_SMALL : POLYLAB_OK;
}

// ---------------------------------------------------------------------------------------- table path

static bool table_dense(const Plan& plan, int64_t n, const Opts& o)
{
    return !(o.flags & POLYLAB_FLAG_DEBUG_FORCE_HASH) && plan.key_bits <= kTableDenseMaxBits &&
           ((int64_t)1 << plan.key_bits) <= table_max_dense_slots(n);
}

static bool table_eligible(const Plan& plan, int64_t n, const Opts& o, const Attempt& at)
{
    if (!at.allow_table || at.safe_rank || (o.flags & (POLYLAB_FLAG_NO_TABLE | POLYLAB_FLAG_SAFE_RANK))) return false;
    // an asynchronous call cannot read the hash table's distinct count back; the dense table needs no read-back
    if ((o.flags & POLYLAB_FLAG_DEVICE_COUNT) && !table_dense(plan, n, o)) return false;
    // the sort path's test hooks mean the sort path
    if (o.flags & (POLYLAB_FLAG_DEBUG_FORCE_BUCKET | POLYLAB_FLAG_DEBUG_UNSTABLE | (0xfu << POLYLAB_FLAG_DEBUG_NFAST_SHIFT))) return false;
    if (plan.key_bytes != 8 || plan.key_bits > 63 || plan.npasses < 1 || n > kTableMaxTerms) return false;
    if (o.flags & POLYLAB_FLAG_DEBUG_FORCE_TABLE) return n <= ((int64_t)1 << 20);
    return n >= kTableMinTerms;
}

// Merges the N records of `src` in a table and emits the simplified polynomial.  *done = false: the table was abandoned
// (too many distinct monomials) and nothing was emitted -- the caller continues on the sort path.
// S1 fused into the table's insert pass (simplify, contiguous rows): the rows to pack and the digit whose histogram the sort
// path would need if the table is abandoned
struct FusedRows { const ExpView* ev; int hd; };

static int table_path(const Plan& plan, int64_t n, unsigned char* ws, const Layout& L, TableSrc src, double tol, const Opts& o,
                      CoefOut out_coef, void* out_exps, int64_t out_capacity, int64_t* out_nterms, int* launches, Timing& tm,
                      cudaStream_t stream, bool* done, void* packed_keys = nullptr, const FusedRows* fr = nullptr)
{
    *done = false;
    Control* ctl = (Control*)(ws + L.control);
    const bool forced = (o.flags & POLYLAB_FLAG_DEBUG_FORCE_TABLE) != 0;
    // (packed output -- an intermediate power -- goes through the hash table: its tail is the prune kernel, which can keep keys)
    const bool dense = !packed_keys && table_dense(plan, n, o);
    src.n = (uint32_t)n;
    TableArgs t;
    memset(&t, 0, sizeof t);
    t.ctl = ctl;
    int lg = 0;
    while (((int64_t)1 << lg) < n) ++lg;
    t.p = 62 - lg > 40 ? 40 : 62 - lg;                 // limb width: N terms of p bits never overflow 62 bits
    unsigned char* base = ws + L.tab;
    if (dense) {
        const size_t slots = (size_t)1 << plan.key_bits;
        t.nord = (uint32_t)slots;
        t.acc_hi = (unsigned long long*)base;
        t.acc_lo = t.acc_hi + slots;
        t.meta = (uint32_t*)(t.acc_lo + slots);
        PL_CUDA(cudaMemsetAsync(base, 0, slots * 20, stream));
    } else {
        t.limit = table_limit(n, forced);
        const uint32_t cap = table_capacity(t.limit);
        t.cmask = cap - 1u;
        t.slots = (TableSlot*)base;
        t.acc_hi = (unsigned long long*)(base + (size_t)cap * sizeof(TableSlot));
        t.acc_lo = t.acc_hi + t.limit;
        PL_CUDA(cudaMemsetAsync(base, 0, (size_t)cap * sizeof(TableSlot) + (size_t)t.limit * 16, stream));
    }
    if (fr) *launches += launch_table_insert_rows(*fr->ev, n, plan, (uint64_t*)(ws + L.keys[0]), src.coef, t, dense, fr->hd, stream);
    else *launches += launch_table_insert(src, t, dense, stream);
    struct Tail { int32_t status; uint32_t distinct, survivors, unsorted, overflow, refinish, fin_count, tab_count, tab_overflow; } res;
    if (!dense) {
        PL_CUDA(cudaMemcpyAsync(&res, &ctl->status, sizeof res, cudaMemcpyDeviceToHost, stream));
        PL_CUDA(cudaStreamSynchronize(stream));
        if (res.status == POLYLAB_ERR_EXPONENT_RANGE) { *done = true; return res.status; }
        if (res.tab_overflow || res.tab_count > t.limit) {
            if (o.stats) o.stats->table_fallback = 1;
            return POLYLAB_OK;
        }
        t.nord = res.tab_count;
    }
    *launches += launch_table_accum(src, t, dense, stream);
    *done = true;
    if (!dense) {
        // (key, sum)[U] -> the ordinary sort / prune / unpack over U records
        const int64_t U = t.nord;
        *launches += launch_table_finalize(t, (uint64_t*)(ws + L.keys[0]), (double*)(ws + L.coefs[0]), stream);
        if (!small_eligible(U, plan, o)) {
            PL_CUDA(cudaMemsetAsync(ctl->hist, 0, sizeof ctl->hist, stream));      // S1 counted the N records into one of them
            *launches += launch_key_hist(plan, 0, U, ws + L.keys[0], ctl, stream);
        }
        if (o.stats) { o.stats->table_path = 2; o.stats->sort_terms = n; }
        const int rc = sort_reduce_emit(plan, 0, U, ws, L, (const double*)(ws + L.coefs[0]), tol, o, out_coef, out_exps, out_capacity,
                                        out_nterms, launches, tm, false, stream, nullptr, nullptr, nullptr, packed_keys);
        return rc == kRetrySafeRank ? kRetrySafeRank : rc;
    }
    tm.mark(POLYLAB_STAGE_SORT);
    tm.mark(POLYLAB_STAGE_REDUCE);
    const bool dev_count = (o.flags & POLYLAB_FLAG_DEVICE_COUNT) != 0;
    *launches += launch_table_dense_emit(t, plan, tol, out_coef, out_exps, o.exp_bytes, out_capacity, (uint32_t*)(ws + L.tab_state),
                                         dev_count ? out_nterms : nullptr, stream);
    tm.mark(POLYLAB_STAGE_PRUNE);
    PL_CUDA(cudaGetLastError());
    if (dev_count) {
        *launches += launch_async_status(ctl, o.status_device, out_nterms, stream);
        if (o.stats) { o.stats->kernel_launches += *launches; o.stats->table_path = 1; o.stats->sort_passes = 0; }
        return POLYLAB_OK;
    }
    if (o.stats) o.stats->kernel_launches += *launches;
    PL_CUDA(cudaMemcpyAsync(&res, &ctl->status, sizeof res, cudaMemcpyDeviceToHost, stream));
    PL_CUDA(cudaStreamSynchronize(stream));
    if (res.status != POLYLAB_OK) return res.status;
    if (res.unsorted) return POLYLAB_ERR_INTERNAL;
    tm.finish(o.stats);
    if (o.stats) { o.stats->distinct = res.distinct; o.stats->survivors = res.survivors; o.stats->table_path = 1; o.stats->sort_passes = 0; }
    *out_nterms = (int64_t)res.survivors;
    return (int64_t)res.survivors > out_capacity ? POLYLAB_ERR_OUTPUT_TOO_SMALL : POLYLAB_OK;
}

static int deliver_zero(const Opts& o, int64_t* out_nterms, cudaStream_t stream)
{
    if (o.flags & POLYLAB_FLAG_DEVICE_COUNT) {
        PL_CUDA(cudaMemsetAsync(out_nterms, 0, sizeof(int64_t), stream));
        if (o.status_device) PL_CUDA(cudaMemsetAsync(o.status_device, 0, sizeof(int32_t), stream));
    } else *out_nterms = 0;
    if (o.stats) { memset(o.stats, 0, sizeof *o.stats); }
    return POLYLAB_OK;
}

static unsigned char* align_ptr(void* p) { return (unsigned char*)(((uintptr_t)p + 255) / 256 * 256); }

}  // namespace polylab

using namespace polylab;

// =============================================================================== entry points

extern "C" {

static int opts_exp_bytes(const polylab_opts* opts) { return (opts && opts->exp_type) ? opts->exp_type : 4; }
static size_t opts_coef_bytes(const polylab_opts* opts) { return (opts && opts->coef_type == POLYLAB_COEF_F32) ? 4 : 8; }

size_t polylab_simplify_workspace_bytes(int64_t nterms, int32_t nvars, const polylab_opts* opts)
{
    if (nterms < 0 || nvars < 1) return 0;
    return worst_layout_bytes(nterms, 0, 0, max_key_bytes(nvars, opts));
}

size_t polylab_mul_simplify_workspace_bytes(int64_t na, int64_t nb, int32_t nvars, const polylab_opts* opts)
{
    if (na < 0 || nb < 0 || nvars < 1) return 0;
    if (na > 0 && nb > 0 && na >= POLYLAB_MAX_TERMS / nb + 1) return 0;
    return worst_layout_bytes(na * nb, na, nb, max_key_bytes(nvars, opts));
}

static int simplify_once(const double* coef, const void* exps, int64_t nterms, int32_t nvars, double tol,
                         const polylab_opts* opts, double* out_coef, void* out_exps, int64_t out_capacity,
                         int64_t* out_nterms, void* workspace, size_t workspace_bytes, void* cuda_stream, const Attempt& at)
{
    cudaStream_t stream = (cudaStream_t)cuda_stream;
    if (nvars < 1 || nvars > POLYLAB_MAX_NVARS || nterms < 0 || nterms >= POLYLAB_MAX_TERMS) return POLYLAB_ERR_INVALID_ARGUMENT;
    if (!(tol >= 0.0) || isinf(tol) || !out_nterms || out_capacity < 0) return POLYLAB_ERR_INVALID_ARGUMENT;
    Opts o;
    int rc = parse_opts(opts, nvars, &o);
    if (rc != POLYLAB_OK) return rc;
    if (nterms == 0) return deliver_zero(o, out_nterms, stream);
    if (!coef || !exps || !workspace || (out_capacity > 0 && (!out_coef || !out_exps))) return POLYLAB_ERR_INVALID_ARGUMENT;

    unsigned char* ws = align_ptr(workspace);
    const size_t avail = workspace_bytes >= (size_t)(ws - (unsigned char*)workspace) ? workspace_bytes - (ws - (unsigned char*)workspace) : 0;
    if (avail < sizeof(Control)) return POLYLAB_ERR_WORKSPACE_TOO_SMALL;
    int launches = 0;
    const ExpView ev = make_view(exps, o, nvars);
    Control* ctl = (Control*)ws;             // Layout::control is offset 0 for every layout
    Timing tm;
    tm.begin((o.flags & POLYLAB_FLAG_TIMING) && o.stats && !(o.flags & POLYLAB_FLAG_DEVICE_COUNT), stream);

    // ---- S0: per-variable maxima (from the caller, or from the data with one read-back)
    uint64_t m[kMaxVars];
    uint32_t bound[kMaxVars];
    bool sampled = false;
    if (o.max_exp_host) {
        for (int v = 0; v < nvars; ++v) { m[v] = o.max_exp_host[v]; bound[v] = o.max_exp_host[v]; }
    } else {
        // Large inputs: maxima of a 0.3 % sample of the rows.  A field only needs the maximum's BIT LENGTH, so the bound is
        // widened to the field's capacity and S1's range check proves that no unsampled exponent exceeds it; if one does,
        // the call re-runs with S0 over every row.
        sampled = !at.exact_bounds && nterms >= kSampleBoundsMinTerms && !(o.flags & POLYLAB_FLAG_EXACT_BOUNDS);
        PL_CUDA(cudaMemsetAsync(ctl, 0, sizeof(Control), stream));
        launches += sampled ? launch_bounds_sample(ev, nterms, nvars, ctl, 0, stream) : launch_bounds(ev, nterms, nvars, ctl, 0, stream);
        uint32_t mh[kMaxVars];
        PL_CUDA(cudaMemcpyAsync(mh, ctl->max_exp[0], sizeof(uint32_t) * nvars, cudaMemcpyDeviceToHost, stream));
        PL_CUDA(cudaStreamSynchronize(stream));
        for (int v = 0; v < nvars; ++v) {
            const uint32_t mv = sampled ? (bitlen(mh[v]) >= 32 ? 0xffffffffu : (1u << bitlen(mh[v])) - 1u) : mh[v];
            m[v] = mv; bound[v] = mv;
        }
    }
    tm.mark(POLYLAB_STAGE_BOUNDS);
    Plan plan;
    rc = make_plan(nvars, m, bound, &plan);
    if (rc != POLYLAB_OK) return rc;
    fill_stats(o.stats, plan, nterms);
    if (o.stats) o.stats->bounds_sampled = sampled ? 1 : 0;

    const Layout L = make_layout(nterms, plan.key_bytes, 0, 0);
    if (avail < L.total) return POLYLAB_ERR_WORKSPACE_TOO_SMALL;
    PL_CUDA(cudaMemsetAsync(ws, 0, L.zero_end, stream));

    // ---- S1 (+ histogram of the first pass's digit), then the shared tail
    int k = choose_prefix_passes(plan, nterms, o, at);
    const bool try_table = table_eligible(plan, nterms, o, at);
    const bool fuse = !try_table && k > 0 && rows_fusable(ev, nvars) && !(o.flags & POLYLAB_FLAG_NO_FUSED_PACK);
    // table path over contiguous rows: S1 runs inside the table's insert pass
    const bool fuse_table = try_table && ev.row_major_contiguous && !(o.flags & POLYLAB_FLAG_NO_FUSED_PACK);
    const int pack_hd = plan.npasses > 0 ? (k ? plan.npasses - k : 0) : -1;
    // Slack bins: a large fused bucket-path call does not sweep the rows for the first prefix digit's exact histogram (0.5 ms
    // on 2e8 terms); it estimates the bins from a 1-2 % sample, gives each a capacity 7 sigma above its estimate, and the pass
    // itself verifies that no bin overran (else the call re-runs with the exact sweep: stats->hist_retry).
    bool slack = false;
    const bool slack_wanted = fuse && k >= 2 && nterms >= kSampleBoundsMinTerms && !at.exact_hist &&
                              !(o.flags & (POLYLAB_FLAG_EXACT_HIST | POLYLAB_FLAG_DEBUG_FORCE_BUCKET | POLYLAB_FLAG_DEBUG_UNSTABLE));
    if (slack_wanted) {
        const int d = plan.npasses - k;
        const int nsegs = sm_count() * 8;
        launches += launch_row_hist_sample(ev, nterms, plan, d, ctl->est, nsegs, 2048, stream);
        if (o.flags & POLYLAB_FLAG_DEVICE_COUNT) {
            // no read-back: capacities computed on the device; a bin that overruns (or a sample that does not fit the buffer)
            // surfaces as POLYLAB_ERR_RETRY in status_device.  (Without a status word the call took safe ranking: k == 0.)
            launches += launch_slack_caps(ctl->est, nterms, slack_capacity(nterms), ctl->hist[d], ctl->slack_cap, stream);
            slack = true;
        }
    }
    if (slack_wanted && !slack) {
        const int d = plan.npasses - k;
        uint32_t est[kRadix], cap[kRadix];
        PL_CUDA(cudaMemcpyAsync(est, ctl->est, sizeof est, cudaMemcpyDeviceToHost, stream));
        PL_CUDA(cudaStreamSynchronize(stream));
        uint64_t ssum = 0, cmax = 0;
        for (int b = 0; b < kRadix; ++b) { ssum += est[b]; cmax = est[b] > cmax ? est[b] : cmax; }
        if (ssum > 0) {
            const double f = (double)nterms / (double)ssum;
            double total = 0.0;
            for (int b = 0; b < kRadix; ++b) {
                const double c = (double)est[b];
                const double cb = ceil(f * (c + 7.0 * sqrt(c + 1.0) + 8.0) / 16.0) * 16.0;      // multiples of 16 records: keys and coefficients of a bin start on 128-byte lines
                cap[b] = cb > 4.0e9 ? 0xffffffffu : (uint32_t)cb;
                total += cb;
            }
            // the skew pre-check of bucket_precheck, on the estimate; and the capacities must fit the buffer
            const int rest = plan.key_bits - plan.digit_pos[d] - plan.digit_bits[d];
            const bool even = ((uint64_t)((double)cmax * f) >> rest) <= (uint64_t)bucket_room(plan, k, nterms) * 7 / 8;
            if (even && total <= (double)slack_capacity(nterms)) {
                PL_CUDA(cudaMemcpyAsync(ctl->hist[d], cap, sizeof cap, cudaMemcpyHostToDevice, stream));
                PL_CUDA(cudaMemcpyAsync(ctl->slack_cap, cap, sizeof cap, cudaMemcpyHostToDevice, stream));
                slack = true;
            }
        }
    }
    if (fuse_table || slack) { /* S1 runs inside the table's insert pass / the histogram is an estimate */ }
    else if (fuse) launches += launch_row_hist(ev, nterms, plan, plan.npasses - k, ctl, stream);      // S1 itself runs inside the first pass
    else launches += launch_pack(ev, nterms, plan, ws + L.keys[0], ctl, plan.npasses > 0 ? (k ? plan.npasses - k : 0) : -1, stream);
    if (try_table) {
        tm.mark(POLYLAB_STAGE_PACK);
        TableSrc src = TableSrc();
        src.keys = (const uint64_t*)(ws + L.keys[0]); src.coef = CoefIn(coef, o.coef_f32);
        bool done = false;
        const FusedRows fr = {&ev, pack_hd};
        rc = table_path(plan, nterms, ws, L, src, tol, o, CoefOut(out_coef, o.coef_f32), out_exps, out_capacity, out_nterms, &launches, tm, stream, &done,
                        nullptr, fuse_table ? &fr : nullptr);
        if (done || rc != POLYLAB_OK) return (rc == POLYLAB_ERR_EXPONENT_RANGE && sampled) ? kRetryExactBounds : rc;
    }
    if (!slack) {
        rc = bucket_precheck(plan, &k, nterms, ws, L, o, &launches, stream, fuse ? &ev : nullptr);
        if (rc != POLYLAB_OK) return rc;
    }
    tm.mark(POLYLAB_STAGE_PACK);
    rc = sort_reduce_emit(plan, k, nterms, ws, L, CoefIn(coef, o.coef_f32), tol, o, CoefOut(out_coef, o.coef_f32), out_exps, out_capacity, out_nterms, &launches, tm,
                          at.safe_rank, stream, (fuse && k > 0) ? &ev : nullptr, nullptr, nullptr, nullptr, slack);
    return (rc == POLYLAB_ERR_EXPONENT_RANGE && sampled) ? kRetryExactBounds : rc;
}

static bool wants_safe_rank(const polylab_opts* opts)
{
    // an asynchronous call without a status word could not report a failed self-check: it gets the ranking that needs none
    return opts && ((opts->flags & POLYLAB_FLAG_SAFE_RANK) || ((opts->flags & POLYLAB_FLAG_DEVICE_COUNT) && !opts->status_device));
}

// Runs `once(attempt)`; a failed self-check re-runs the call on a more conservative path (at most twice).
extern "C++" {
template <typename F>
static int run_attempts(const polylab_opts* opts, F once)
{
    if (opts && opts->stats) { opts->stats->kernel_launches = 0; opts->stats->rank_fallback = 0; opts->stats->bucket_fallback = 0; opts->stats->bounds_retry = 0; opts->stats->table_fallback = 0; opts->stats->hist_retry = 0; }
    Attempt at = {wants_safe_rank(opts), true, false, true, false};
    int rc = once(at);
    for (int tries = 0; tries < 4 && (rc == kRetryExactBounds || rc == kRetryNoBucket || rc == kRetrySafeRank || rc == kRetryExactHist); ++tries) {
        polylab_stats* st = opts ? opts->stats : nullptr;
        if (rc != kRetryExactBounds && rc != kRetryExactHist) at.allow_table = false;
        if (rc == kRetryExactHist) {
            if (st) st->hist_retry = 1;
            at.exact_hist = true;
        } else if (rc == kRetryExactBounds) {             // each retry only ever tightens the attempt, so three suffice
            if (st) st->bounds_retry = 1;
            at.exact_bounds = true;
        } else if (rc == kRetryNoBucket) {
            if (st) st->bucket_fallback = 1;
            at.allow_bucket = false;
        } else {
            if (st) st->rank_fallback = 1;
            at.safe_rank = true;
            at.allow_bucket = false;
        }
        rc = once(at);
    }
    if (rc == kRetryExactBounds || rc == kRetryNoBucket || rc == kRetrySafeRank || rc == kRetryExactHist) rc = POLYLAB_ERR_INTERNAL;
    return rc;
}
}  // extern "C++"

int polylab_simplify(const double* coef, const void* exps, int64_t nterms, int32_t nvars, double tol,
                     const polylab_opts* opts, double* out_coef, void* out_exps, int64_t out_capacity,
                     int64_t* out_nterms, void* workspace, size_t workspace_bytes, void* cuda_stream)
{
    return run_attempts(opts, [&](const Attempt& at) {
        return simplify_once(coef, exps, nterms, nvars, tol, opts, out_coef, out_exps, out_capacity, out_nterms, workspace,
                             workspace_bytes, cuda_stream, at);
    });
}

// X1 + S2..S5 of a product whose operands are PACKED (keys with the product's field layout + coefficients): table path, or
// X1 fused into the first radix pass, or materialised products for the one-block / ballot paths.  packed_keys != nullptr:
// the result stays packed -- keys to packed_keys[], sums to out_coef[] -- for the next product of a power.
static int product_tail(const Plan& plan, const ExpandSrc& xs, int k, unsigned char* ws, const Layout& L, double tol, const Opts& o,
                        CoefOut out_coef, void* out_exps, int64_t out_capacity, int64_t* out_nterms, int* launches, Timing& tm,
                        const Attempt& at, cudaStream_t stream, void* packed_keys)
{
    Control* ctl = (Control*)(ws + L.control);
    const int64_t n = xs.na * xs.nb;
    int rc;
    if (packed_keys) k = 0;                              // (the bucket path's emit kernel unpacks)
    if (table_eligible(plan, n, o, at)) {
        tm.mark(POLYLAB_STAGE_PACK);
        TableSrc src = TableSrc();
        src.ka = xs.ka; src.ca = xs.ca; src.kb = xs.kb; src.cb = xs.cb; src.nb = (uint32_t)xs.nb;
        bool done = false;
        rc = table_path(plan, n, ws, L, src, tol, o, out_coef, out_exps, out_capacity, out_nterms, launches, tm, stream, &done, packed_keys);
        if (done || rc != POLYLAB_OK) return rc;
    }
    // X1 runs inside the first radix pass (the products are formed in registers and never stored) unless the ballot
    // ranking kernel or the one-block path is taken or there is no pass at all; only the first digit's histogram is built up front
    const bool fuse = plan.npasses > 0 && !at.safe_rank && !(o.flags & POLYLAB_FLAG_NO_FUSED_PACK) && !small_eligible(n, plan, o);
    if (fuse) *launches += launch_expand_hist(xs, plan, k ? plan.npasses - k : 0, ctl, stream);
    else *launches += launch_expand_packed(xs.ka, xs.ca, xs.na, xs.kb, xs.cb, xs.nb, plan, ws + L.keys[0],
                                           (double*)(ws + L.coefs[0]), ctl, k ? plan.npasses - k : 0, stream);
    rc = bucket_precheck(plan, &k, n, ws, L, o, launches, stream, nullptr, fuse ? &xs : nullptr);
    if (rc != POLYLAB_OK) return rc;
    tm.mark(POLYLAB_STAGE_PACK);
    return sort_reduce_emit(plan, k, n, ws, L, (const double*)(ws + L.coefs[0]), tol, o, out_coef, out_exps, out_capacity,
                            out_nterms, launches, tm, at.safe_rank, stream, nullptr, fuse ? &xs : nullptr, nullptr, packed_keys);
}

static int mul_simplify_once(const polylab_poly* a, const polylab_poly* b, double tol, const polylab_opts* opts,
                             double* out_coef, void* out_exps, int64_t out_capacity, int64_t* out_nterms,
                             void* workspace, size_t workspace_bytes, void* cuda_stream, const Attempt& at)
{
    cudaStream_t stream = (cudaStream_t)cuda_stream;
    if (!a || !b || a->nvars != b->nvars) return POLYLAB_ERR_INVALID_ARGUMENT;
    const int nvars = a->nvars;
    const int64_t na = a->nterms, nb = b->nterms;
    if (nvars < 1 || nvars > POLYLAB_MAX_NVARS || na < 0 || nb < 0) return POLYLAB_ERR_INVALID_ARGUMENT;
    if (na > 0 && nb > 0 && na > (POLYLAB_MAX_TERMS - 1) / nb) return POLYLAB_ERR_INVALID_ARGUMENT;
    if (!(tol >= 0.0) || isinf(tol) || !out_nterms || out_capacity < 0) return POLYLAB_ERR_INVALID_ARGUMENT;
    Opts o;
    int rc = parse_opts(opts, nvars, &o);
    if (rc != POLYLAB_OK) return rc;
    const int64_t n = na * nb;
    if (n == 0) return deliver_zero(o, out_nterms, stream);
    if (!a->coef || !a->exps || !b->coef || !b->exps || !workspace || (out_capacity > 0 && (!out_coef || !out_exps)))
        return POLYLAB_ERR_INVALID_ARGUMENT;

    unsigned char* ws = align_ptr(workspace);
    const size_t avail = workspace_bytes >= (size_t)(ws - (unsigned char*)workspace) ? workspace_bytes - (ws - (unsigned char*)workspace) : 0;
    if (avail < sizeof(Control)) return POLYLAB_ERR_WORKSPACE_TOO_SMALL;
    int launches = 0;
    const ExpView eva = make_view(a->exps, o, nvars), evb = make_view(b->exps, o, nvars);
    Control* ctl = (Control*)ws;
    Timing tm;
    tm.begin((o.flags & POLYLAB_FLAG_TIMING) && o.stats && !(o.flags & POLYLAB_FLAG_DEVICE_COUNT), stream);

    // ---- S0 on both operands; the sorted rows are sums, so fields are sized for max_a + max_b
    uint64_t m[kMaxVars];
    uint32_t ba[kMaxVars], bb[kMaxVars];
    const uint32_t emax = exp_max_of(o.exp_bytes);
    bool check_sums = false;                  // caller bounds that allow a sum above exp_type's range: checked on the device
    if (o.max_exp_host) {
        for (int v = 0; v < nvars; ++v) {
            ba[v] = bb[v] = o.max_exp_host[v]; m[v] = 2ull * o.max_exp_host[v];
            check_sums |= m[v] > emax;
        }
    } else {
        PL_CUDA(cudaMemsetAsync(ctl, 0, sizeof(Control), stream));
        launches += launch_bounds(eva, na, nvars, ctl, 0, stream);
        launches += launch_bounds(evb, nb, nvars, ctl, 1, stream);
        uint32_t mh[2][kMaxVars];
        PL_CUDA(cudaMemcpyAsync(mh, ctl->max_exp, sizeof mh, cudaMemcpyDeviceToHost, stream));
        PL_CUDA(cudaStreamSynchronize(stream));
        for (int v = 0; v < nvars; ++v) {
            ba[v] = mh[0][v]; bb[v] = mh[1][v];
            m[v] = (uint64_t)mh[0][v] + mh[1][v];
            if (m[v] > emax) return POLYLAB_ERR_EXPONENT_RANGE;       // the sum must fit exp_type (reading A8)
        }
    }
    tm.mark(POLYLAB_STAGE_BOUNDS);
    Plan plan_a, plan_b;
    rc = make_plan(nvars, m, ba, &plan_a);
    if (rc != POLYLAB_OK) return rc;
    make_plan(nvars, m, bb, &plan_b);
    fill_stats(o.stats, plan_a, n);

    const Layout L = make_layout(n, plan_a.key_bytes, na, nb);
    if (avail < L.total) return POLYLAB_ERR_WORKSPACE_TOO_SMALL;
    PL_CUDA(cudaMemsetAsync(ws, 0, L.zero_end, stream));
    if (check_sums) launches += launch_sum_range_check(eva, na, evb, nb, nvars, emax, ctl, stream);

    // ---- S1 on the operands, X1 on packed keys (+ histogram of the first digit), then the shared tail
    int k = choose_prefix_passes(plan_a, n, o, at);
    launches += launch_pack(eva, na, plan_a, ws + L.ka, ctl, -1, stream);
    launches += launch_pack(evb, nb, plan_b, ws + L.kb, ctl, -1, stream);
    // X1 runs inside the first radix pass (the products are formed in registers and never stored) unless the ballot
    // ranking kernel is asked for or there is no pass at all; only the first digit's histogram is built up front
    CoefIn ca(a->coef, o.coef_f32), cb(b->coef, o.coef_f32);
    if (o.coef_f32) {                                    // two small arrays: every kernel downstream sees fp64 operands
        launches += launch_widen(a->coef, (double*)(ws + L.ca), na, stream) + launch_widen(b->coef, (double*)(ws + L.cb), nb, stream);
        ca = CoefIn((const double*)(ws + L.ca));
        cb = CoefIn((const double*)(ws + L.cb));
    }
    const ExpandSrc xs = {ws + L.ka, ca, na, ws + L.kb, cb, nb};
    return product_tail(plan_a, xs, k, ws, L, tol, o, CoefOut(out_coef, o.coef_f32), out_exps, out_capacity, out_nterms, &launches, tm, at, stream, nullptr);
}

int polylab_mul_simplify(const polylab_poly* a, const polylab_poly* b, double tol, const polylab_opts* opts,
                         double* out_coef, void* out_exps, int64_t out_capacity, int64_t* out_nterms,
                         void* workspace, size_t workspace_bytes, void* cuda_stream)
{
    return run_attempts(opts, [&](const Attempt& at) {
        return mul_simplify_once(a, b, tol, opts, out_coef, out_exps, out_capacity, out_nterms, workspace, workspace_bytes,
                                 cuda_stream, at);
    });
}

// ------------------------------------------------------------------------------- batched (N3)

// Plan of a batched call: make_plan over (entry, variables) -- the entry index is "variable -1", the most significant field --
// then the entry field is dropped from the variable tables (S5 unpacks variables only).
static int make_batched_plan(int nvars, const uint64_t* m, const uint32_t* bound, int64_t nentries, Plan* plan, int* entry_shift)
{
    uint64_t m2[kMaxVars];
    uint32_t b2[kMaxVars];
    m2[0] = nentries > 1 ? (uint64_t)(nentries - 1) : 1u;        // at least one bit, so that shifting by entry_shift is defined
    b2[0] = (uint32_t)m2[0];
    for (int v = 0; v < nvars; ++v) { m2[v + 1] = m[v]; b2[v + 1] = bound[v]; }
    Plan full;
    const int rc = make_plan(nvars + 1, m2, b2, &full);
    if (rc != POLYLAB_OK) return rc;
    *plan = full;
    plan->nvars = nvars;
    for (int v = 0; v < nvars; ++v) { plan->shift[v] = full.shift[v + 1]; plan->width[v] = full.width[v + 1]; plan->bound[v] = full.bound[v + 1]; }
    plan->shift[nvars] = 0; plan->width[nvars] = 0; plan->bound[nvars] = 0;
    *entry_shift = full.shift[0];
    return POLYLAB_OK;
}

static int batch_args_ok(const polylab_batch* p, const polylab_opts* opts)
{
    if (!p || p->nvars < 1 || p->nvars > POLYLAB_MAX_NVARS - 1 || p->nentries < 0 || p->nentries >= POLYLAB_MAX_TERMS) return 0;
    if (p->nentries > 0 && !p->offsets_host) return 0;
    if (opts && (opts->max_exp_host || (opts->flags & POLYLAB_FLAG_DEVICE_COUNT) || opts->term_stride != 0 || opts->var_stride != 0)) return 0;
    int64_t prev = 0;
    for (int64_t e = 0; e <= p->nentries && p->nentries > 0; ++e) {
        if (p->offsets_host[e] < prev || (e == 0 && p->offsets_host[0] != 0)) return 0;
        prev = p->offsets_host[e];
    }
    if (prev >= POLYLAB_MAX_TERMS) return 0;
    if (prev > 0 && (!p->coef || !p->exps)) return 0;
    return 1;
}

struct BatchLayout { size_t inner_bytes, segs, counts, total; };
static BatchLayout batch_layout(int64_t n, int64_t na, int64_t nb, int64_t nseg, int64_t nentries, int widest_key_bytes)
{
    BatchLayout B;
    B.inner_bytes = worst_layout_bytes(n, na, nb, widest_key_bytes);
    size_t off = align_up(B.inner_bytes);
    B.segs = off; off = align_up(off + (size_t)(nseg + 1) * sizeof(BatchSeg));
    B.counts = off; off = align_up(off + (size_t)(nentries + 1) * sizeof(uint32_t));
    B.total = off + 256;
    return B;
}

// The shared body: operands a (and b for products) are packed with one plan, the segments' records are materialised with
// the entry index on top, and the ordinary tail (one-block path or LSD passes, segmented sum, prune, unpack) runs once.
static int batched_run(const polylab_batch* a, const polylab_batch* b, const BatchSeg* segs_host, int64_t nseg, int64_t n,
                       int64_t nentries, double tol, const polylab_opts* opts, double* out_coef, void* out_exps, int64_t out_capacity,
                       int64_t* out_offsets_host, void* workspace, size_t workspace_bytes, void* cuda_stream, const Attempt& at)
{
    cudaStream_t stream = (cudaStream_t)cuda_stream;
    const int nvars = a->nvars;
    Opts o;
    int rc = parse_opts(opts, nvars, &o);
    if (rc != POLYLAB_OK) return rc;
    for (int64_t e = 0; e <= nentries; ++e) out_offsets_host[e] = 0;
    if (n == 0) { if (o.stats) memset(o.stats, 0, sizeof *o.stats); return POLYLAB_OK; }
    if (!workspace || (out_capacity > 0 && (!out_coef || !out_exps))) return POLYLAB_ERR_INVALID_ARGUMENT;
    const int64_t na = a->nentries ? a->offsets_host[a->nentries] : 0, nb = b ? (b->nentries ? b->offsets_host[b->nentries] : 0) : 0;
    unsigned char* ws = align_ptr(workspace);
    const size_t avail = workspace_bytes >= (size_t)(ws - (unsigned char*)workspace) ? workspace_bytes - (ws - (unsigned char*)workspace) : 0;
    const BatchLayout BL = batch_layout(n, na, nb, nseg, nentries, max_key_bytes(nvars, opts, 30));
    if (avail < BL.total - 256) return POLYLAB_ERR_WORKSPACE_TOO_SMALL;
    int launches = 0;
    Control* ctl = (Control*)ws;
    Timing tm;
    tm.begin((o.flags & POLYLAB_FLAG_TIMING) && o.stats, stream);
    const ExpView eva = make_view(a->exps, o, nvars);
    ExpView evb = eva;
    if (b) evb = make_view(b->exps, o, nvars);

    // ---- S0 over all terms of the operand(s); for products the fields are sized for max_a + max_b
    PL_CUDA(cudaMemsetAsync(ctl, 0, sizeof(Control), stream));
    launches += launch_bounds(eva, na, nvars, ctl, 0, stream);
    if (b) launches += launch_bounds(evb, nb, nvars, ctl, 1, stream);
    uint32_t mh[2][kMaxVars];
    PL_CUDA(cudaMemcpyAsync(mh, ctl->max_exp, sizeof mh, cudaMemcpyDeviceToHost, stream));
    PL_CUDA(cudaStreamSynchronize(stream));
    uint64_t m[kMaxVars];
    uint32_t ba[kMaxVars], bb[kMaxVars];
    const uint32_t emax = exp_max_of(o.exp_bytes);
    for (int v = 0; v < nvars; ++v) {
        ba[v] = mh[0][v]; bb[v] = b ? mh[1][v] : 0u;
        m[v] = (uint64_t)ba[v] + bb[v];
        if (m[v] > emax) return POLYLAB_ERR_EXPONENT_RANGE;           // a product's exponent sums must fit exp_type (A8)
    }
    tm.mark(POLYLAB_STAGE_BOUNDS);
    Plan plan_a, plan_b;
    int entry_shift = 0;
    rc = make_batched_plan(nvars, m, ba, nentries, &plan_a, &entry_shift);
    if (rc != POLYLAB_OK) return rc;
    make_batched_plan(nvars, m, bb, nentries, &plan_b, &entry_shift);
    fill_stats(o.stats, plan_a, n);

    const Layout L = make_layout(n, plan_a.key_bytes, na, nb);
    if (L.total > BL.inner_bytes) return POLYLAB_ERR_INTERNAL;
    PL_CUDA(cudaMemsetAsync(ws, 0, L.zero_end, stream));
    BatchSeg* segs = (BatchSeg*)(ws + BL.segs);
    uint32_t* counts = (uint32_t*)(ws + BL.counts);
    PL_CUDA(cudaMemcpyAsync(segs, segs_host, (size_t)nseg * sizeof(BatchSeg), cudaMemcpyHostToDevice, stream));
    PL_CUDA(cudaMemsetAsync(counts, 0, (size_t)(nentries + 1) * sizeof(uint32_t), stream));

    // ---- S1 on the operands (monomial fields only), then the records with the entry index on top (+ X1 for products)
    launches += launch_pack(eva, na, plan_a, ws + L.ka, ctl, -1, stream);
    if (b) launches += launch_pack(evb, nb, plan_b, ws + L.kb, ctl, -1, stream);
    launches += launch_batched_expand(plan_a, segs, (uint32_t)nseg, n, ws + L.ka, CoefIn(a->coef, o.coef_f32), b ? ws + L.kb : nullptr, b ? CoefIn(b->coef, o.coef_f32) : CoefIn(),
                                      entry_shift, ws + L.keys[0], (double*)(ws + L.coefs[0]), ctl, stream);
    tm.mark(POLYLAB_STAGE_PACK);
    const BatchOut bo = {entry_shift, counts};
    Opts o2 = o;
    o2.flags |= POLYLAB_FLAG_NO_BUCKET | POLYLAB_FLAG_NO_TABLE;
    int64_t total = 0;
    rc = sort_reduce_emit(plan_a, 0, n, ws, L, (const double*)(ws + L.coefs[0]), tol, o2, CoefOut(out_coef, o.coef_f32), out_exps, out_capacity, &total,
                          &launches, tm, at.safe_rank, stream, nullptr, nullptr, &bo);
    if (rc != POLYLAB_OK && rc != POLYLAB_ERR_OUTPUT_TOO_SMALL) return rc;
    // ---- offsets: prefix sums of the entries' survivor counts (nentries values, on the host)
    uint32_t* hc = (uint32_t*)malloc((size_t)(nentries + 1) * sizeof(uint32_t));
    if (!hc) return POLYLAB_ERR_INTERNAL;
    if (cuda_failed(cudaMemcpyAsync(hc, counts, (size_t)nentries * sizeof(uint32_t), cudaMemcpyDeviceToHost, stream), "copy of the entry counts") ||
        cuda_failed(cudaStreamSynchronize(stream), "cudaStreamSynchronize")) { free(hc); return POLYLAB_ERR_CUDA; }
    int64_t run = 0;
    for (int64_t e = 0; e < nentries; ++e) { out_offsets_host[e] = run; run += hc[e]; }
    out_offsets_host[nentries] = run;
    free(hc);
    if (run != total) return POLYLAB_ERR_INTERNAL;
    return rc;
}

size_t polylab_simplify_batched_workspace_bytes(int64_t nterms, int64_t nentries, int32_t nvars, const polylab_opts* opts)
{
    if (nterms < 0 || nentries < 0 || nterms >= POLYLAB_MAX_TERMS || nvars < 1) return 0;
    return batch_layout(nterms, nterms, 0, nentries, nentries, max_key_bytes(nvars, opts, 30)).total;
}

int polylab_simplify_batched(const polylab_batch* p, double tol, const polylab_opts* opts, double* out_coef, void* out_exps,
                             int64_t out_capacity, int64_t* out_offsets_host, void* workspace, size_t workspace_bytes, void* cuda_stream)
{
    if (!batch_args_ok(p, opts) || !(tol >= 0.0) || isinf(tol) || !out_offsets_host || out_capacity < 0) return POLYLAB_ERR_INVALID_ARGUMENT;
    const int64_t ne = p->nentries, n = ne ? p->offsets_host[ne] : 0;
    BatchSeg* segs = (BatchSeg*)malloc((size_t)(ne + 1) * sizeof(BatchSeg));
    if (!segs) return POLYLAB_ERR_INTERNAL;
    int64_t nseg = 0;
    for (int64_t e = 0; e < ne; ++e) {                               // one segment per non-empty entry: its raw terms
        const int64_t t0 = p->offsets_host[e], t1 = p->offsets_host[e + 1];
        if (t1 > t0) { const BatchSeg s = {(uint32_t)t0, (uint32_t)t0, (uint32_t)(t1 - t0), 0u, 0u, (uint32_t)e}; segs[nseg++] = s; }
    }
    const int rc = run_attempts(opts, [&](const Attempt& at) {
        return batched_run(p, nullptr, segs, nseg, n, ne, tol, opts, out_coef, out_exps, out_capacity, out_offsets_host, workspace,
                           workspace_bytes, cuda_stream, at);
    });
    free(segs);
    return rc;
}

size_t polylab_matmul_simplify_workspace_bytes(int64_t nproducts, int64_t a_nterms, int64_t b_nterms, int64_t m, int64_t k, int64_t n,
                                               int32_t nvars, const polylab_opts* opts)
{
    if (nproducts < 0 || nproducts >= POLYLAB_MAX_TERMS || a_nterms < 0 || b_nterms < 0 || m < 0 || k < 0 || n < 0 || nvars < 1) return 0;
    if (m * n >= POLYLAB_MAX_TERMS || (k > 0 && m * n > POLYLAB_MAX_TERMS / k)) return 0;
    return batch_layout(nproducts, a_nterms, b_nterms, m * n * k, m * n, max_key_bytes(nvars, opts, 30)).total;
}

int polylab_matmul_simplify(const polylab_batch* a, int32_t m, int32_t k, const polylab_batch* b, int32_t n, double tol,
                            const polylab_opts* opts, double* out_coef, void* out_exps, int64_t out_capacity, int64_t* out_offsets_host,
                            void* workspace, size_t workspace_bytes, void* cuda_stream)
{
    if (!batch_args_ok(a, opts) || !batch_args_ok(b, opts) || a->nvars != b->nvars || m < 0 || k < 0 || n < 0) return POLYLAB_ERR_INVALID_ARGUMENT;
    if (a->nentries != (int64_t)m * k || b->nentries != (int64_t)k * n) return POLYLAB_ERR_INVALID_ARGUMENT;
    if (!(tol >= 0.0) || isinf(tol) || !out_offsets_host || out_capacity < 0) return POLYLAB_ERR_INVALID_ARGUMENT;
    const int64_t ne = (int64_t)m * n;
    if (ne >= POLYLAB_MAX_TERMS || (k > 0 && ne > POLYLAB_MAX_TERMS / k)) return POLYLAB_ERR_INVALID_ARGUMENT;
    BatchSeg* segs = (BatchSeg*)malloc((size_t)(ne * k + 1) * sizeof(BatchSeg));
    if (!segs) return POLYLAB_ERR_INTERNAL;
    int64_t nseg = 0, nprod = 0;
    for (int i = 0; i < m; ++i)
        for (int j = 0; j < n; ++j)
            for (int l = 0; l < k; ++l) {                            // C(i,j) += A(i,l) * B(l,j): one segment of products
                const int64_t a0 = a->offsets_host[(int64_t)i * k + l], a1 = a->offsets_host[(int64_t)i * k + l + 1];
                const int64_t b0 = b->offsets_host[(int64_t)l * n + j], b1 = b->offsets_host[(int64_t)l * n + j + 1];
                const int64_t cnt = (a1 - a0) * (b1 - b0);
                if (cnt == 0) continue;
                if (nprod + cnt >= POLYLAB_MAX_TERMS) { free(segs); return POLYLAB_ERR_INVALID_ARGUMENT; }
                const BatchSeg s = {(uint32_t)nprod, (uint32_t)a0, (uint32_t)(a1 - a0), (uint32_t)b0, (uint32_t)(b1 - b0), (uint32_t)((int64_t)i * n + j)};
                segs[nseg++] = s;
                nprod += cnt;
            }
    const int rc = run_attempts(opts, [&](const Attempt& at) {
        return batched_run(a, b, segs, nseg, nprod, ne, tol, opts, out_coef, out_exps, out_capacity, out_offsets_host, workspace,
                           workspace_bytes, cuda_stream, at);
    });
    free(segs);
    return rc;
}

// ------------------------------------------------------------------------------- powers (N2)

// The powers stay PACKED between the products: S0 runs once on p, ONE key layout is sized for the final
// degree (field v holds power * max_v), p is packed once, and every intermediate power lives in the workspace as
// (keys, sums) -- no S5 -> S0 -> S1 round trip between products.  Products go left to right (q <- q * p): for the paper's
// dense p_d family binary powering forms MORE term products (p_4^4: 126^2 + 1287^2 = 1.67e6 against 126^2 + 1287*126 +
// 6188*126 = 0.96e6), and the product count, not the number of calls, is what the time follows.
struct PowLayout { size_t keys[2], coef[2], kp, cp, inner, inner_bytes, total; };

static PowLayout pow_layout(int64_t np, int nvars, int64_t cap, const polylab_opts* opts)
{
    PowLayout P;
    size_t off = 0;
    auto take = [&](size_t bytes) { const size_t o = off; off = align_up(off + bytes); return o; };
    const int kb = max_key_bytes(nvars, opts);
    for (int i = 0; i < 2; ++i) { P.keys[i] = take((size_t)cap * kb); P.coef[i] = take((size_t)cap * sizeof(double)); }
    P.kp = take((size_t)np * kb);
    P.cp = take((size_t)np * sizeof(double));
    P.inner_bytes = worst_layout_bytes(cap * np, 0, 0, kb);
    P.inner = take(P.inner_bytes);
    P.total = off + 256;
    return P;
}

size_t polylab_pow_simplify_workspace_bytes(int64_t nterms, int32_t nvars, int32_t power, int64_t out_capacity,
                                            const polylab_opts* opts)
{
    if (nterms < 0 || nvars < 1 || power < 0 || out_capacity < 0) return 0;
    if (power <= 1) return polylab_simplify_workspace_bytes(nterms, nvars, opts);
    const int64_t cap = out_capacity > nterms ? out_capacity : nterms;
    if (nterms > 0 && cap >= POLYLAB_MAX_TERMS / nterms) return 0;              // a product could exceed the term limit
    return pow_layout(nterms, nvars, cap, opts).total;
}

int polylab_pow_simplify(const polylab_poly* p, int32_t power, double tol, const polylab_opts* opts,
                         double* out_coef, void* out_exps, int64_t out_capacity, int64_t* out_nterms,
                         void* workspace, size_t workspace_bytes, void* cuda_stream)
{
    cudaStream_t stream = (cudaStream_t)cuda_stream;
    if (!p || power < 0 || !out_nterms || out_capacity < 0 || !(tol >= 0.0) || isinf(tol)) return POLYLAB_ERR_INVALID_ARGUMENT;
    const int nvars = p->nvars;
    const int64_t np = p->nterms;
    if (nvars < 1 || nvars > POLYLAB_MAX_NVARS || np < 0 || np >= POLYLAB_MAX_TERMS) return POLYLAB_ERR_INVALID_ARGUMENT;
    if (opts && (opts->max_exp_host || (opts->flags & POLYLAB_FLAG_DEVICE_COUNT) || opts->term_stride != 0 || opts->var_stride != 0))
        return POLYLAB_ERR_INVALID_ARGUMENT;
    const int es = opts_exp_bytes(opts);
    if (es != POLYLAB_EXP_U8 && es != POLYLAB_EXP_U16 && es != POLYLAB_EXP_U32) return POLYLAB_ERR_INVALID_ARGUMENT;
    if (power == 0) {                                    // p^0 = 1, also for the zero polynomial (the empty product)
        *out_nterms = 1;
        if (out_capacity < 1) return POLYLAB_ERR_OUTPUT_TOO_SMALL;
        if (!out_coef || !out_exps) return POLYLAB_ERR_INVALID_ARGUMENT;
        const double one = 1.0;
        const float onef = 1.0f;
        const bool f32 = opts && opts->coef_type == POLYLAB_COEF_F32;
        PL_CUDA(cudaMemcpyAsync(out_coef, f32 ? (const void*)&onef : (const void*)&one, f32 ? sizeof onef : sizeof one, cudaMemcpyHostToDevice, stream));
        PL_CUDA(cudaMemsetAsync(out_exps, 0, (size_t)nvars * es, stream));
        PL_CUDA(cudaStreamSynchronize(stream));
        return POLYLAB_OK;
    }
    if (power == 1 || np == 0)
        return polylab_simplify(p->coef, p->exps, np, nvars, tol, opts, out_coef, out_exps, out_capacity, out_nterms, workspace,
                                workspace_bytes, cuda_stream);
    if (!p->coef || !p->exps || !workspace || (out_capacity > 0 && (!out_coef || !out_exps))) return POLYLAB_ERR_INVALID_ARGUMENT;
    const int64_t cap = out_capacity > np ? out_capacity : np;
    if (cap >= POLYLAB_MAX_TERMS / np) return POLYLAB_ERR_INVALID_ARGUMENT;
    const PowLayout P = pow_layout(np, nvars, cap, opts);
    unsigned char* ws = align_ptr(workspace);
    if (workspace_bytes < (size_t)(ws - (unsigned char*)workspace) + P.total - 256) return POLYLAB_ERR_WORKSPACE_TOO_SMALL;
    Opts o;
    int rc = parse_opts(opts, nvars, &o);
    if (rc != POLYLAB_OK) return rc;
    unsigned char* iws = ws + P.inner;                   // the products' own workspace (256-byte aligned: every region is)
    Control* ctl = (Control*)iws;

    // ---- S0 once; the key layout of p^power: field v is sized for power * max_v, which must fit exp_type (reading A8)
    const ExpView ev = make_view(p->exps, o, nvars);
    PL_CUDA(cudaMemsetAsync(ctl, 0, sizeof(Control), stream));
    int launches0 = launch_bounds(ev, np, nvars, ctl, 0, stream);
    uint32_t mh[kMaxVars];
    PL_CUDA(cudaMemcpyAsync(mh, ctl->max_exp[0], sizeof(uint32_t) * nvars, cudaMemcpyDeviceToHost, stream));
    PL_CUDA(cudaStreamSynchronize(stream));
    uint64_t m[kMaxVars];
    const uint32_t emax = exp_max_of(es);
    for (int v = 0; v < nvars; ++v) {
        m[v] = (uint64_t)mh[v] * (uint64_t)power;
        if (m[v] > emax) return POLYLAB_ERR_EXPONENT_RANGE;
    }
    Plan plan;
    rc = make_plan(nvars, m, mh, &plan);
    if (rc != POLYLAB_OK) return rc;
    // ---- S1 once: p's keys in the final layout
    launches0 += launch_pack(ev, np, plan, ws + P.kp, ctl, -1, stream);

    const void* ak = ws + P.kp;                          // the running power q (packed): starts as p itself
    CoefIn pc(p->coef, o.coef_f32);
    if (o.coef_f32) {                                    // p's coefficients widened once; the powers' sums are fp64 anyway
        launches0 += launch_widen(p->coef, (double*)(ws + P.cp), np, stream);
        pc = CoefIn((const double*)(ws + P.cp));
    }
    CoefIn ac = pc;
    int64_t count = np;
    for (int step = 2; step <= power; ++step) {
        const bool last = step == power;
        const int64_t n = count * np;
        const Layout L = make_layout(n, plan.key_bytes, 0, 0);
        if (L.total > P.inner_bytes) return POLYLAB_ERR_INTERNAL;
        const ExpandSrc xs = {ak, ac, count, ws + P.kp, pc, np};
        void* pk = last ? nullptr : (void*)(ws + P.keys[step & 1]);
        const CoefOut oc = last ? CoefOut(out_coef, o.coef_f32) : CoefOut((double*)(ws + P.coef[step & 1]));
        int64_t produced = 0;
        rc = run_attempts(opts, [&](const Attempt& at) {
            cudaError_t e = cudaMemsetAsync(iws, 0, L.zero_end, stream);
            if (cuda_failed(e, "cudaMemsetAsync")) return (int)POLYLAB_ERR_CUDA;
            fill_stats(o.stats, plan, n);
            int launches = step == 2 ? launches0 : 0;
            Timing tm;
            tm.begin((o.flags & POLYLAB_FLAG_TIMING) && o.stats, stream);
            tm.mark(POLYLAB_STAGE_BOUNDS);
            return product_tail(plan, xs, choose_prefix_passes(plan, n, o, at), iws, L, last ? tol : 0.0, o, oc, last ? out_exps : nullptr,
                                last ? out_capacity : cap, &produced, &launches, tm, at, stream, pk);
        });
        if (rc != POLYLAB_OK) {
            if (rc == POLYLAB_ERR_OUTPUT_TOO_SMALL) *out_nterms = produced;
            return rc;
        }
        if (!last && produced > out_capacity) { *out_nterms = produced; return POLYLAB_ERR_OUTPUT_TOO_SMALL; }
        count = produced;
        ak = pk; ac = CoefIn((const double*)oc.p);
        if (count == 0) break;                           // the zero polynomial stays zero
    }
    *out_nterms = count;
    return POLYLAB_OK;
}

int polylab_expand(const polylab_poly* a, const polylab_poly* b, const polylab_opts* opts, double* out_coef,
                   void* out_exps, void* workspace, size_t workspace_bytes, void* cuda_stream)
{
    cudaStream_t stream = (cudaStream_t)cuda_stream;
    if (!a || !b || a->nvars != b->nvars) return POLYLAB_ERR_INVALID_ARGUMENT;
    const int nvars = a->nvars;
    const int64_t na = a->nterms, nb = b->nterms;
    if (nvars < 1 || nvars > POLYLAB_MAX_NVARS || na < 0 || nb < 0) return POLYLAB_ERR_INVALID_ARGUMENT;
    if (na > 0 && nb > 0 && na > (POLYLAB_MAX_TERMS - 1) / nb) return POLYLAB_ERR_INVALID_ARGUMENT;
    Opts o;
    int rc = parse_opts(opts, nvars, &o);
    if (rc != POLYLAB_OK) return rc;
    if (na * nb == 0) return POLYLAB_OK;
    if (!a->coef || !a->exps || !b->coef || !b->exps || !out_coef || !out_exps || !workspace) return POLYLAB_ERR_INVALID_ARGUMENT;
    unsigned char* ws = align_ptr(workspace);
    if (workspace_bytes < (size_t)(ws - (unsigned char*)workspace) + sizeof(Control)) return POLYLAB_ERR_WORKSPACE_TOO_SMALL;
    Control* ctl = (Control*)ws;
    PL_CUDA(cudaMemsetAsync(&ctl->status, 0, sizeof(int32_t), stream));
    launch_expand_raw(make_view(a->exps, o, nvars), CoefIn(a->coef, o.coef_f32), na, make_view(b->exps, o, nvars), CoefIn(b->coef, o.coef_f32), nb, nvars, CoefOut(out_coef, o.coef_f32),
                      out_exps, ctl, stream);
    PL_CUDA(cudaGetLastError());
    int32_t status = 0;
    PL_CUDA(cudaMemcpyAsync(&status, &ctl->status, sizeof status, cudaMemcpyDeviceToHost, stream));
    PL_CUDA(cudaStreamSynchronize(stream));
    return status;
}

int polylab_pack_keys(const void* exps, int64_t nterms, int32_t nvars, const polylab_opts* opts, uint64_t* out_keys,
                      int32_t* key_bits_host, void* workspace, size_t workspace_bytes, void* cuda_stream)
{
    cudaStream_t stream = (cudaStream_t)cuda_stream;
    if (nvars < 1 || nvars > POLYLAB_MAX_NVARS || nterms < 0 || nterms >= POLYLAB_MAX_TERMS) return POLYLAB_ERR_INVALID_ARGUMENT;
    Opts o;
    int rc = parse_opts(opts, nvars, &o);
    if (rc != POLYLAB_OK) return rc;
    if (nterms == 0) { if (key_bits_host) *key_bits_host = 0; return POLYLAB_OK; }
    if (!exps || !out_keys || !workspace) return POLYLAB_ERR_INVALID_ARGUMENT;
    unsigned char* ws = align_ptr(workspace);
    if (workspace_bytes < (size_t)(ws - (unsigned char*)workspace) + sizeof(Control)) return POLYLAB_ERR_WORKSPACE_TOO_SMALL;
    Control* ctl = (Control*)ws;
    const ExpView ev = make_view(exps, o, nvars);
    PL_CUDA(cudaMemsetAsync(ctl, 0, sizeof(Control), stream));
    uint64_t m[kMaxVars];
    uint32_t bound[kMaxVars];
    if (o.max_exp_host) {
        for (int v = 0; v < nvars; ++v) { m[v] = o.max_exp_host[v]; bound[v] = o.max_exp_host[v]; }
    } else {
        launch_bounds(ev, nterms, nvars, ctl, 0, stream);
        uint32_t mh[kMaxVars];
        PL_CUDA(cudaMemcpyAsync(mh, ctl->max_exp[0], sizeof(uint32_t) * nvars, cudaMemcpyDeviceToHost, stream));
        PL_CUDA(cudaStreamSynchronize(stream));
        for (int v = 0; v < nvars; ++v) { m[v] = mh[v]; bound[v] = mh[v]; }
    }
    Plan plan;
    rc = make_plan(nvars, m, bound, &plan);
    if (rc != POLYLAB_OK) return rc;
    if (key_bits_host) *key_bits_host = plan.key_bits;
    if (plan.key_bits > 128) return POLYLAB_ERR_KEY_TOO_WIDE;          // this entry point's output format is (hi, lo)
    plan.key_bytes = 16;
    launch_pack_hilo(ev, nterms, plan, out_keys, ctl, stream);
    PL_CUDA(cudaGetLastError());
    int32_t status = 0;
    PL_CUDA(cudaMemcpyAsync(&status, &ctl->status, sizeof status, cudaMemcpyDeviceToHost, stream));
    PL_CUDA(cudaStreamSynchronize(stream));
    return status;
}

// ------------------------------------------------------------------- host-buffer entry points

struct HostLayout { size_t coef, exps, out_coef, out_exps, inner, total; };

static HostLayout host_layout(int64_t n_in_terms, int64_t n_sort, int nvars, int exp_bytes, size_t inner_bytes)
{
    HostLayout H;
    size_t off = 0;
    auto take = [&](size_t bytes) { const size_t o = off; off = align_up(off + bytes); return o; };
    H.coef = take((size_t)n_in_terms * sizeof(double));
    H.exps = take((size_t)n_in_terms * nvars * exp_bytes);
    H.out_coef = take((size_t)n_sort * sizeof(double));
    H.out_exps = take((size_t)n_sort * nvars * exp_bytes);
    H.inner = take(inner_bytes);
    H.total = off + 256;
    return H;
}

size_t polylab_simplify_host_workspace_bytes(int64_t nterms, int32_t nvars, const polylab_opts* opts)
{
    if (nterms < 0 || nvars < 1) return 0;
    return host_layout(nterms, nterms, nvars, opts_exp_bytes(opts), polylab_simplify_workspace_bytes(nterms, nvars, opts)).total;
}

size_t polylab_mul_simplify_host_workspace_bytes(int64_t na, int64_t nb, int32_t nvars, const polylab_opts* opts)
{
    if (na < 0 || nb < 0 || nvars < 1) return 0;
    return host_layout(na + nb + 64, na * nb, nvars, opts_exp_bytes(opts), polylab_mul_simplify_workspace_bytes(na, nb, nvars, opts)).total;
}

static int host_opts_ok(const polylab_opts* opts, int nvars)
{
    if (!opts) return 1;
    if (opts->flags & POLYLAB_FLAG_DEVICE_COUNT) return 0;
    if ((opts->term_stride != 0 || opts->var_stride != 0) && !(opts->term_stride == nvars && opts->var_stride == 1)) return 0;
    return 1;
}

int polylab_simplify_host(const double* coef_host, const void* exps_host, int64_t nterms, int32_t nvars, double tol,
                          const polylab_opts* opts, double* out_coef_host, void* out_exps_host, int64_t out_capacity,
                          int64_t* out_nterms_host, void* device_workspace, size_t workspace_bytes, void* cuda_stream)
{
    cudaStream_t stream = (cudaStream_t)cuda_stream;
    if (nvars < 1 || nvars > POLYLAB_MAX_NVARS || nterms < 0 || nterms >= POLYLAB_MAX_TERMS || !out_nterms_host || out_capacity < 0)
        return POLYLAB_ERR_INVALID_ARGUMENT;
    if (!host_opts_ok(opts, nvars)) return POLYLAB_ERR_INVALID_ARGUMENT;
    if (nterms == 0) { *out_nterms_host = 0; return (tol >= 0.0) ? POLYLAB_OK : POLYLAB_ERR_INVALID_ARGUMENT; }
    if (!coef_host || !exps_host || !device_workspace) return POLYLAB_ERR_INVALID_ARGUMENT;
    const int es = opts_exp_bytes(opts);
    const size_t inner = polylab_simplify_workspace_bytes(nterms, nvars, opts);
    const HostLayout H = host_layout(nterms, nterms, nvars, es, inner);
    unsigned char* ws = align_ptr(device_workspace);
    if (workspace_bytes < (size_t)(ws - (unsigned char*)device_workspace) + H.total - 256) return POLYLAB_ERR_WORKSPACE_TOO_SMALL;
    const size_t cbytes = opts_coef_bytes(opts);
    PL_CUDA(cudaMemcpyAsync(ws + H.coef, coef_host, (size_t)nterms * cbytes, cudaMemcpyHostToDevice, stream));
    PL_CUDA(cudaMemcpyAsync(ws + H.exps, exps_host, (size_t)nterms * nvars * es, cudaMemcpyHostToDevice, stream));
    int64_t count = 0;
    const int rc = polylab_simplify((const double*)(ws + H.coef), ws + H.exps, nterms, nvars, tol, opts, (double*)(ws + H.out_coef),
                                    ws + H.out_exps, nterms, &count, ws + H.inner, inner, cuda_stream);
    if (rc != POLYLAB_OK) return rc;
    *out_nterms_host = count;
    const int64_t ncopy = count < out_capacity ? count : out_capacity;
    if (ncopy > 0) {
        if (!out_coef_host || !out_exps_host) return POLYLAB_ERR_INVALID_ARGUMENT;
        PL_CUDA(cudaMemcpyAsync(out_coef_host, ws + H.out_coef, (size_t)ncopy * cbytes, cudaMemcpyDeviceToHost, stream));
        PL_CUDA(cudaMemcpyAsync(out_exps_host, ws + H.out_exps, (size_t)ncopy * nvars * es, cudaMemcpyDeviceToHost, stream));
    }
    PL_CUDA(cudaStreamSynchronize(stream));
    return count > out_capacity ? POLYLAB_ERR_OUTPUT_TOO_SMALL : POLYLAB_OK;
}

int polylab_mul_simplify_host(const polylab_poly* a_host, const polylab_poly* b_host, double tol, const polylab_opts* opts,
                              double* out_coef_host, void* out_exps_host, int64_t out_capacity, int64_t* out_nterms_host,
                              void* device_workspace, size_t workspace_bytes, void* cuda_stream)
{
    cudaStream_t stream = (cudaStream_t)cuda_stream;
    if (!a_host || !b_host || a_host->nvars != b_host->nvars || !out_nterms_host || out_capacity < 0) return POLYLAB_ERR_INVALID_ARGUMENT;
    const int nvars = a_host->nvars;
    const int64_t na = a_host->nterms, nb = b_host->nterms;
    if (nvars < 1 || nvars > POLYLAB_MAX_NVARS || na < 0 || nb < 0) return POLYLAB_ERR_INVALID_ARGUMENT;
    if (na > 0 && nb > 0 && na > (POLYLAB_MAX_TERMS - 1) / nb) return POLYLAB_ERR_INVALID_ARGUMENT;
    if (!host_opts_ok(opts, nvars)) return POLYLAB_ERR_INVALID_ARGUMENT;
    const int64_t n = na * nb;
    if (n == 0) { *out_nterms_host = 0; return (tol >= 0.0) ? POLYLAB_OK : POLYLAB_ERR_INVALID_ARGUMENT; }
    if (!a_host->coef || !a_host->exps || !b_host->coef || !b_host->exps || !device_workspace) return POLYLAB_ERR_INVALID_ARGUMENT;
    const int es = opts_exp_bytes(opts);
    const size_t inner = polylab_mul_simplify_workspace_bytes(na, nb, nvars, opts);
    const HostLayout H = host_layout(na + nb + 64, n, nvars, es, inner);
    unsigned char* ws = align_ptr(device_workspace);
    if (workspace_bytes < (size_t)(ws - (unsigned char*)device_workspace) + H.total - 256) return POLYLAB_ERR_WORKSPACE_TOO_SMALL;
    // operand b sits behind operand a in the input slices, each 32-term aligned
    const int64_t nb_off = (na + 31) / 32 * 32;
    const size_t cbytes = opts_coef_bytes(opts);
    double* dca = (double*)(ws + H.coef);
    double* dcb = dca + nb_off;                          // (8-byte slots also when the coefficients are fp32)
    unsigned char* dea = ws + H.exps;
    unsigned char* deb = dea + (size_t)nb_off * nvars * es;
    PL_CUDA(cudaMemcpyAsync(dca, a_host->coef, (size_t)na * cbytes, cudaMemcpyHostToDevice, stream));
    PL_CUDA(cudaMemcpyAsync(dcb, b_host->coef, (size_t)nb * cbytes, cudaMemcpyHostToDevice, stream));
    PL_CUDA(cudaMemcpyAsync(dea, a_host->exps, (size_t)na * nvars * es, cudaMemcpyHostToDevice, stream));
    PL_CUDA(cudaMemcpyAsync(deb, b_host->exps, (size_t)nb * nvars * es, cudaMemcpyHostToDevice, stream));
    polylab_poly da = {dca, dea, na, nvars}, db = {dcb, deb, nb, nvars};
    int64_t count = 0;
    const int rc = polylab_mul_simplify(&da, &db, tol, opts, (double*)(ws + H.out_coef), ws + H.out_exps, n, &count, ws + H.inner,
                                        inner, cuda_stream);
    if (rc != POLYLAB_OK) return rc;
    *out_nterms_host = count;
    const int64_t ncopy = count < out_capacity ? count : out_capacity;
    if (ncopy > 0) {
        if (!out_coef_host || !out_exps_host) return POLYLAB_ERR_INVALID_ARGUMENT;
        PL_CUDA(cudaMemcpyAsync(out_coef_host, ws + H.out_coef, (size_t)ncopy * cbytes, cudaMemcpyDeviceToHost, stream));
        PL_CUDA(cudaMemcpyAsync(out_exps_host, ws + H.out_exps, (size_t)ncopy * nvars * es, cudaMemcpyDeviceToHost, stream));
    }
    PL_CUDA(cudaStreamSynchronize(stream));
    return count > out_capacity ? POLYLAB_ERR_OUTPUT_TOO_SMALL : POLYLAB_OK;
}

const char* polylab_status_string(int status)
{
    switch (status) {
    case POLYLAB_OK: return "ok";
    case POLYLAB_ERR_INVALID_ARGUMENT: return "invalid argument";
    case POLYLAB_ERR_KEY_TOO_WIDE: return "packed key wider than 256 bits";
    case POLYLAB_ERR_EXPONENT_RANGE: return "exponent out of range";
    case POLYLAB_ERR_WORKSPACE_TOO_SMALL: return "workspace too small";
    case POLYLAB_ERR_OUTPUT_TOO_SMALL: return "output capacity too small";
    case POLYLAB_ERR_CUDA: return "CUDA error";
    case POLYLAB_ERR_INTERNAL: return "internal error: sorted-order self-check failed";
    case POLYLAB_ERR_RETRY: return "asynchronous call: a self-check of the fast path failed, call again with POLYLAB_FLAG_SAFE_RANK";
    default: return "unknown status";
    }
}

const char* polylab_last_cuda_error(void) { return g_cuda_error; }
int polylab_version(void) { return POLYLAB_VERSION; }

}  // extern "C"
