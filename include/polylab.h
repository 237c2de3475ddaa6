/*
 * polylab.h -- C ABI of polylab-b200: simplification of sparse multivariate polynomials on one
 * NVIDIA B200 (sm_100a).  Plain pointers and sizes only; no C++ or torch types.
 *
 * Data model (the paper's): a polynomial is a coefficient vector plus an exponent matrix with one
 * row per monomial -- constructor MPOLY(n,coef,pow), /root/reference/PAPER.md:80 (Table 3) and
 * PAPER.md:97 (section 3.1).  Exponents are non-negative integers (alpha in N^n).
 * Variable identity is outside this ABI: operands of a product share nvars and column meaning
 * (the paper aligns variable spaces BEFORE an operation).
 *
 * Operations:
 *   simplify(p, zeroprec): "merges repeated monomials and removes coefficients below a user-chosen
 *     tolerance" (Table 4; Table 3).
 *   product of scalar polynomials (mtimes/times): every term of a times every
 *     term of b -- coefficient products and exponent sums -- then simplify (the paper's heavy
 *     workload simplify(p_d^3)).
 *
 * Result form (readings A1-A4): monomials strictly ascending in lexicographic order of
 * the exponent row with variable 0 (column 0) most significant -- the order of the paper's
 * transcripts PAPER.md:195-201 and PAPER.md:134; no duplicates; a merged monomial is kept iff
 * |sum| > tol (absolute, applied after merging; NaN sums are dropped); the zero polynomial is
 * *out_nterms = 0.
 *
 * Pointers: DEVICE unless the name or the comment says host.  The library allocates nothing and
 * frees nothing: inputs are const and never written, outputs and workspace are caller-owned and
 * must not overlap the inputs or each other.  All work is enqueued on `cuda_stream` (a cudaStream_t
 * passed as void*, NULL = legacy default stream).  Unless POLYLAB_FLAG_DEVICE_COUNT is set a call
 * synchronises that stream before returning (to deliver *out_nterms and the status).
 * Thread-safe for distinct workspaces.  Every function returns a polylab_status; nothing aborts.
 */
#ifndef POLYLAB_H
#define POLYLAB_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#if defined(__GNUC__)
#pragma GCC visibility push(default)
#endif

#define POLYLAB_VERSION 120          /* 0.1.2: polylab_stats.grouped_tiles, POLYLAB_FLAG_NO_GROUP_FINISH, the fast-digits test hook in flag bits 16..19 */
#define POLYLAB_MAX_NVARS 256        /* packed keys hold at most 256 bits (reading A9) */
#define POLYLAB_MAX_TERMS ((int64_t)1 << 30)   /* exclusive bound on nterms and on na*nb */
#define POLYLAB_SMALL_WORKSPACE_BYTES 65536    /* workspace of polylab_expand and polylab_pack_keys */

typedef enum {
    POLYLAB_OK = 0,
    POLYLAB_ERR_INVALID_ARGUMENT = 1,   /* null pointer with work to do, nvars < 1 or > MAX_NVARS, nterms < 0 or
                                           >= MAX_TERMS, tol NaN or < 0, unknown exp_type, nvars mismatch */
    POLYLAB_ERR_KEY_TOO_WIDE = 2,       /* sum over variables of bitlen(max exponent) > 256 (polylab_pack_keys: > 128) */
    POLYLAB_ERR_EXPONENT_RANGE = 3,     /* an exponent exceeds the caller's max_exp_host bound, or a product's
                                           exponent sum does not fit exp_type */
    POLYLAB_ERR_WORKSPACE_TOO_SMALL = 4,
    POLYLAB_ERR_OUTPUT_TOO_SMALL = 5,   /* survivors > out_capacity: *out_nterms = required size, the first
                                           out_capacity terms are written */
    POLYLAB_ERR_CUDA = 6,               /* a CUDA runtime call failed (see polylab_last_cuda_error) */
    POLYLAB_ERR_INTERNAL = 7,           /* the sorted-order self-check failed even with the ballot-ranking kernel */
    POLYLAB_ERR_RETRY = 8               /* only ever written to opts->status_device by a POLYLAB_FLAG_DEVICE_COUNT call: a
                                           self-check of the fast path failed (ranking order, bucket length, slack-bin size), nothing valid
                                           was emitted and the device count is 0 -- call again with POLYLAB_FLAG_SAFE_RANK |
                                           POLYLAB_FLAG_NO_BUCKET (or without POLYLAB_FLAG_DEVICE_COUNT, which retries itself) */
} polylab_status;

typedef enum { POLYLAB_EXP_U8 = 1, POLYLAB_EXP_U16 = 2, POLYLAB_EXP_U32 = 4 } polylab_exp_type;

/* Coefficient STORAGE type of every coefficient array a call is given or fills (coef, out_coef, polylab_poly.coef,
 * polylab_batch.coef; the prototypes say double*): POLYLAB_COEF_F32 is the paper's polylab_precision('set','single')
 * (Table 10) -- pass float arrays cast to the prototype's pointer type.  fp32 values
 * are widened when first loaded; products, sums and the prune comparison are fp64; a result is rounded to fp32 once,
 * when stored (so |stored - exact| <= 2^-24 |s| + the fp64 bound).  The prune predicate |s| > tol is applied to the fp64
 * sum, before that rounding. */
typedef enum { POLYLAB_COEF_F64 = 0, POLYLAB_COEF_F32 = 1 } polylab_coef_type;

enum {
    POLYLAB_FLAG_DEVICE_COUNT = 1u,  /* out_nterms is a DEVICE int64_t*; the call does not synchronise.
                                        Requires max_exp_host (no bounds read-back).  Data errors and failed self-checks
                                        are then reported only through the device status word opts->status_device
                                        (POLYLAB_ERR_EXPONENT_RANGE, POLYLAB_ERR_RETRY).  With a status word the call takes
                                        the same fast kernels as a synchronous one (atomic ranking, one-block path, bucket
                                        path, dense table; not the hash table, which needs a read-back); without one it ranks by
                                        ballot matching, whose order needs no check. */
    POLYLAB_FLAG_TIMING = 2u,        /* record CUDA events between the steps and fill stats->stage_ms
                                        (needs stats; ignored with POLYLAB_FLAG_DEVICE_COUNT) */
    POLYLAB_FLAG_SAFE_RANK = 4u,     /* rank records inside a radix pass by warp ballot matching (stable by
                                        construction) instead of one shared-memory atomic per record.  The
                                        atomic kernel is stable only because sm_100a returns the old values of
                                        one warp instruction's same-address atomics in lane order (measured, not
                                        documented); therefore the default path verifies the sorted order in the
                                        segmented-sum step and re-runs the call with this flag if the check
                                        fails (stats->rank_fallback = 1).  Implied by POLYLAB_FLAG_DEVICE_COUNT without
                                        opts->status_device, which could not report the check. */
    POLYLAB_FLAG_NO_BUCKET = 8u,     /* never take the bucket path: always sort with ceil(B/8) LSD passes.  By default a
                                        call with >= 2^20 terms and >= 4 digits first partitions the pairs on their
                                        most significant digit(s) and, if those spread the keys evenly enough for every
                                        bucket to fit shared memory, finishes sort + sum + prune + unpack on chip
                                        (stats->prefix_passes > 0); otherwise (stats->bucket_fallback = 1) it runs the
                                        LSD passes.  Both paths give the same result up to summation order.  Not
                                        taken with POLYLAB_FLAG_SAFE_RANK. */
    POLYLAB_FLAG_NO_FUSED_PACK = 16u, /* always run S1 (pack) and X1 (expand) as kernels of their own.  By default the first
                                        radix pass forms its keys in registers: from the exponent rows on the bucket path
                                        (contiguous rows of 8 or 16 bytes), from the packed operands for a product
                                        (the na*nb products are then never stored).  Same result, bit for bit. */
    POLYLAB_FLAG_EXACT_BOUNDS = 32u,  /* S0 always reads every exponent.  By default a simplify call with >= 2^22 terms and
                                        no max_exp_host takes the maxima of a sample of the rows, sizes the key fields by
                                        their bit lengths, and lets S1's range check verify every row; a violation
                                        re-runs the call with full bounds (stats->bounds_retry = 1).  Same result. */
    POLYLAB_FLAG_EXACT_HIST = 256u,   /* the bucket path always sweeps the rows for the exact histogram of its first prefix digit.  By
                                        default a fused call with >= 2^22 terms and two or more prefix passes estimates that
                                        histogram from a 1-2 % sample of the rows, lays the first pass's bins out with slack (7
                                        sigma above the estimate) and lets the pass itself verify that none overran
                                        (stats->hist_sampled = 1); an overrun re-runs the call with the sweep
                                        (stats->hist_retry = 1).  Same result, bit for bit.  A POLYLAB_FLAG_DEVICE_COUNT call
                                        with a status word sizes the bins on the device; an overrun is POLYLAB_ERR_RETRY there. */
    POLYLAB_FLAG_NO_GROUP_FINISH = 512u, /* bucket path: finish every tile with the sorting kernel.  By default a tile with enough records first
                                        tries to GROUP them: like terms are found through a shared-memory hash table (full keys
                                        compared), only the tile's distinct monomials are put in order, and one stable counting pass
                                        puts the records in order (stats->grouped_tiles).  A tile whose records-per-monomial ratio
                                        is too low for that to pay (about 6 at 3000 records), or with more than 768 distinct
                                        monomials, a fingerprint collision or an overlong probe sequence, is finished by the sorting
                                        kernel instead, and once most tiles are, the rest no longer try.  Same result, bit for bit. */
    POLYLAB_FLAG_NO_TABLE = 64u,      /* never take the table path.  By default a call with 2^15 <= N <= 2^26 terms whose key fits 63 bits
                                        first merges like terms in a table (the packed key itself as the index when 2^B slots
                                        are affordable, else a hash table) with order-independent fixed-point accumulators,
                                        and sorts only the U distinct monomials (stats->table_path = 1 dense, 2 hash).  If
                                        more than min(N/4, 2^20) distinct monomials turn up the call continues on the sort
                                        path (stats->table_fallback = 1).  Results obey the same parity rule; on this path
                                        they are also invariant under permutations of the input terms.  Not taken with
                                        POLYLAB_FLAG_SAFE_RANK; with POLYLAB_FLAG_DEVICE_COUNT only the dense table. */
    POLYLAB_FLAG_NO_SMALL = 128u,     /* never take the one-block path.  By default at most 8192 terms (or products, or distinct
                                        monomials left by the table path; 4096 with 128-bit keys) are sorted and summed by a
                                        single thread block in shared memory (stats->small_path = 1): two launches instead of
                                        a dozen.  Not taken with POLYLAB_FLAG_SAFE_RANK. */
    POLYLAB_FLAG_DEBUG_FORCE_TABLE = 0x10000000u,  /* test hook: take the table path at any size up to 2^20 terms (abandoned only beyond 16384 distinct monomials) */
    POLYLAB_FLAG_DEBUG_FORCE_HASH = 0x08000000u,   /* test hook: use the hash table even where the dense table applies */
    POLYLAB_FLAG_DEBUG_FORCE_BUCKET = 0x20000000u, /* test hook: take the bucket path whenever it is defined (any size, no
                                        skew pre-check), so that small tests reach it and its overflow fallback */
    POLYLAB_FLAG_DEBUG_GROUP_HANDS_ON = 0x04000000u, /* test hook: the bucket path's group kernel runs and hands every tile on to the
                                        sorting kernel */
    POLYLAB_FLAG_DEBUG_UNSTABLE = 0x40000000u  /* test hook: makes the atomic-ranking kernel unstable on purpose
                                        (reversed lane order) so that tests can exercise detection and fallback */
};
/* test hook: bits 16..19 of flags, when non-zero, override how many low digits the bucket path's first local sort
   attempt uses (default 3); 1 makes most tiles fail the order check and re-sort on every digit */
#define POLYLAB_FLAG_DEBUG_NFAST_SHIFT 16

/* indices into polylab_stats.stage_ms */
enum { POLYLAB_STAGE_BOUNDS = 0, POLYLAB_STAGE_PACK = 1, POLYLAB_STAGE_SORT = 2, POLYLAB_STAGE_REDUCE = 3,
       POLYLAB_STAGE_PRUNE = 4, POLYLAB_STAGE_COUNT = 5 };

/* Per-call statistics (HOST, optional): the plan that was chosen and what the pipeline saw. */
typedef struct polylab_stats {
    int32_t key_bits;        /* B = sum of field widths                                  */
    int32_t key_bytes;       /* W = 8, 16 or 32 (one, two or four 64-bit words)           */
    int32_t sort_passes;     /* P radix passes executed                                  */
    int32_t digit_bits[32];  /* width of each digit of the key, least significant first   */
    int64_t sort_terms;      /* N = terms that entered the sort (na*nb for a product)    */
    int64_t distinct;        /* U = distinct monomials before pruning (-1 with DEVICE_COUNT) */
    int64_t survivors;       /* U' (-1 with DEVICE_COUNT)                                */
    int32_t kernel_launches; /* kernels of this library launched by the call (both attempts after a fallback) */
    int32_t rank_fallback;   /* 1 if the sorted-order check failed and the call re-ran with SAFE_RANK */
    float stage_ms[8];       /* with POLYLAB_FLAG_TIMING: device time of S0 (incl. read-back), S1 (+X1),
                                S2 (all passes), S3, S4+S5; CUDA events on the call's stream.  On the bucket
                                path S2 = the prefix passes, S3 = tile bounds + the finish kernel (local sort, S3, S4 per tile)
                                and S4+S5 = the count scan + the emit/unpack kernel */
    int32_t prefix_passes;   /* > 0: the bucket path ran with this many prefix passes (then sort_passes == prefix_passes) */
    int32_t bucket_fallback; /* 1 if the bucket path was planned and abandoned (skewed digit histogram or a bucket
                                too long for a tile); the result then comes from the LSD path */
    int32_t refinish_tiles;  /* bucket path: tiles whose fast local sort failed the order check and re-sorted fully */
    int32_t plan_digits;     /* ceil(B/8): digits of the key layout = entries of digit_bits = LSD passes the plan needs */
    int32_t bounds_sampled;  /* 1 if S0 ran on a sample of the rows (see POLYLAB_FLAG_EXACT_BOUNDS) */
    int32_t bounds_retry;    /* 1 if the sampled bounds were violated and the call re-ran with full bounds */
    int32_t table_path;      /* 1: like terms were merged in a dense table (no sort at all); 2: in a hash table, and only the
                                distinct monomials were sorted (see POLYLAB_FLAG_NO_TABLE); 0: sort path */
    int32_t table_fallback;  /* 1 if the table path was tried and abandoned (too many distinct monomials) */
    int32_t small_path;      /* 1 if one thread block did the sort and the segmented sum (see POLYLAB_FLAG_NO_SMALL) */
    int32_t hist_sampled;    /* 1 if the first prefix pass took slack bins from a sampled histogram (POLYLAB_FLAG_EXACT_HIST) */
    int32_t hist_retry;      /* 1 if such a bin overran and the call re-ran with the exact histogram */
    int32_t grouped_tiles;   /* bucket path: tiles finished by grouping like terms in a hash table (POLYLAB_FLAG_NO_GROUP_FINISH) */
} polylab_stats;

/* Options; a zero-initialised struct (or a NULL pointer) means the defaults. */
typedef struct polylab_opts {
    int32_t exp_type;             /* polylab_exp_type of exps and out_exps; 0 = POLYLAB_EXP_U32          */
    uint32_t flags;               /* POLYLAB_FLAG_*                                                      */
    int64_t term_stride;          /* element (t,v) of an exponent matrix is at index                     */
    int64_t var_stride;           /*   t*term_stride + v*var_stride (in elements); both 0 = row-major    */
                                  /*   (nvars,1); MATLAB's column-major pow is (1,nterms).  Applies to   */
                                  /*   inputs; outputs are always row-major [out_capacity x nvars].      */
    const uint32_t* max_exp_host; /* HOST, nvars entries, optional: upper bounds on the exponents of     */
                                  /*   each variable (for a product: of EACH operand).  Skips the bounds */
                                  /*   kernel and its read-back; violations -> POLYLAB_ERR_EXPONENT_RANGE */
    int32_t* status_device;       /* DEVICE, optional: receives the polylab_status of data-dependent      */
                                  /*   checks (used with POLYLAB_FLAG_DEVICE_COUNT)                      */
    polylab_stats* stats;         /* HOST, optional                                                      */
    int32_t coef_type;            /* polylab_coef_type of every coefficient array of the call; 0 = fp64   */
} polylab_opts;

/* A read-only view of a polynomial: coef[nterms], exps[nterms x nvars] (strides from polylab_opts). */
typedef struct polylab_poly {
    const double* coef;
    const void* exps;
    int64_t nterms;
    int32_t nvars;
} polylab_poly;

/* Workspace sizes (bytes, worst case over all key layouts) for the device-pointer entry points. */
size_t polylab_simplify_workspace_bytes(int64_t nterms, int32_t nvars, const polylab_opts* opts);
size_t polylab_mul_simplify_workspace_bytes(int64_t na, int64_t nb, int32_t nvars, const polylab_opts* opts);

/*
 * simplify.  coef[nterms], exps[nterms x nvars] DEVICE inputs (may be unsorted, contain
 * duplicates, zeros, cancelling pairs).  Outputs: out_coef[out_capacity], out_exps[out_capacity x nvars]
 * (row-major, exp_type) DEVICE; *out_nterms HOST (DEVICE with POLYLAB_FLAG_DEVICE_COUNT) = number of
 * surviving monomials U'.  out_capacity = nterms always suffices.  nterms == 0 is valid (0 terms).
 * Steps: bounds -> pack exponent rows into 64/128-bit keys -> LSD radix sort of (key, coef) -> segmented
 * sum of equal keys -> prune |s| <= tol -> unpack survivors.
 */
int polylab_simplify(const double* coef, const void* exps, int64_t nterms, int32_t nvars, double tol,
                     const polylab_opts* opts,
                     double* out_coef, void* out_exps, int64_t out_capacity, int64_t* out_nterms,
                     void* workspace, size_t workspace_bytes, void* cuda_stream);

/*
 * simplify(a*b): forms all a->nterms * b->nterms products -- coefficient
 * fl(ca_i*cb_j) (one IEEE multiplication, never fused with the later sums) and exponent row a_i + b_j --
 * then merges them as polylab_simplify does.  out_capacity = na*nb always suffices.
 */
int polylab_mul_simplify(const polylab_poly* a, const polylab_poly* b, double tol,
                         const polylab_opts* opts,
                         double* out_coef, void* out_exps, int64_t out_capacity, int64_t* out_nterms,
                         void* workspace, size_t workspace_bytes, void* cuda_stream);

/*
 * simplify(p^power) -- the paper's mpower on a scalar polynomial (Table 1; the heavy workload
 * simplify(p_d^3)) -- by repeated products q <- simplify(q * p), left to right.  The bounds step runs
 * once on p, ONE key layout is sized for the final degree (field v holds power * max_v), p is packed once, and the
 * intermediate powers stay on the device as packed (key, sum) pairs inside the workspace: no unpack, no re-pack, no
 * re-upload between products.  Intermediates are merged with tolerance 0 (exact zeros dropped, reading A2); only the final
 * power is pruned with `tol`.  Every intermediate power must fit out_capacity terms, else POLYLAB_ERR_OUTPUT_TOO_SMALL with
 * *out_nterms = the size that was needed.  power >= 0: power 0 gives the constant polynomial 1, power 1 is
 * polylab_simplify.  p: DEVICE, row-major exponents (strides in opts are not supported here); opts->max_exp_host and
 * POLYLAB_FLAG_DEVICE_COUNT are not supported (POLYLAB_ERR_INVALID_ARGUMENT).  power * (largest exponent of a variable in
 * p) must fit exp_type, else POLYLAB_ERR_EXPONENT_RANGE.  opts->stats describes the last product.  The call synchronises
 * the stream once for the bounds and once per product (for the term count that sizes the next product's launches).
 */
size_t polylab_pow_simplify_workspace_bytes(int64_t nterms, int32_t nvars, int32_t power, int64_t out_capacity,
                                            const polylab_opts* opts);
int polylab_pow_simplify(const polylab_poly* p, int32_t power, double tol, const polylab_opts* opts,
                         double* out_coef, void* out_exps, int64_t out_capacity, int64_t* out_nterms,
                         void* workspace, size_t workspace_bytes, void* cuda_stream);

/*
 * Batched operations on polynomial MATRICES (Table 4: matrix mtimes, sum, prod; section 3.4;
 * the rows of Table 7, where per-entry launches make the paper's GPU backends lose to its CPU class).
 * A batch is many scalar polynomials over the same nvars variables stored back to back: entry e owns the terms
 * [offsets_host[e], offsets_host[e+1]) of (coef, exps); offsets_host is a HOST array of nentries + 1 non-decreasing values
 * starting at 0 (an entry may be empty: the zero polynomial).  A matrix is a batch in row-major entry order.
 * One call simplifies every entry: the entry index is the most significant field of the packed key, so a single sort /
 * segmented sum / prune / unpack serves them all.  Outputs: the simplified entries concatenated in entry order, each in
 * canonical monomial order, in out_coef[out_capacity] / out_exps[out_capacity x nvars] (DEVICE); out_offsets_host (HOST,
 * nentries + 1 values) receives where each entry starts (out_offsets_host[nentries] = total number of terms).  Survivors
 * beyond out_capacity -> POLYLAB_ERR_OUTPUT_TOO_SMALL with out_offsets_host filled in.  Exponents: row-major, opts->exp_type;
 * opts->max_exp_host, strides and POLYLAB_FLAG_DEVICE_COUNT are not supported (POLYLAB_ERR_INVALID_ARGUMENT); nvars <= 255.
 * The calls synchronise the stream.
 */
typedef struct polylab_batch {
    const double* coef;           /* DEVICE [offsets_host[nentries]]                     */
    const void* exps;             /* DEVICE [offsets_host[nentries] x nvars], row-major  */
    const int64_t* offsets_host;  /* HOST [nentries + 1]                                 */
    int64_t nentries;
    int32_t nvars;
} polylab_batch;

/* simplify every entry of a batch (for a matrix `sum` along a dimension: lay the summands of one result entry back to back) */
size_t polylab_simplify_batched_workspace_bytes(int64_t nterms, int64_t nentries, int32_t nvars, const polylab_opts* opts);
int polylab_simplify_batched(const polylab_batch* p, double tol, const polylab_opts* opts,
                             double* out_coef, void* out_exps, int64_t out_capacity, int64_t* out_offsets_host,
                             void* workspace, size_t workspace_bytes, void* cuda_stream);

/*
 * simplify(A*B) for polynomial matrices A (m x k) and B (k x n): entry (i, j) = sum over l of A(i,l)*B(l,j), every product
 * of scalar polynomials formed term by term (coefficient products rounded once, exponent sums) and all of them merged in
 * one pass.  The result has m*n entries, row-major.  nproducts = the sum over (i, j, l) of nterms(A(i,l)) * nterms(B(l,j)),
 * which must be < POLYLAB_MAX_TERMS; out_capacity = nproducts always suffices.
 */
size_t polylab_matmul_simplify_workspace_bytes(int64_t nproducts, int64_t a_nterms, int64_t b_nterms, int64_t m, int64_t k, int64_t n,
                                               int32_t nvars, const polylab_opts* opts);
int polylab_matmul_simplify(const polylab_batch* a, int32_t m, int32_t k, const polylab_batch* b, int32_t n, double tol,
                            const polylab_opts* opts, double* out_coef, void* out_exps, int64_t out_capacity,
                            int64_t* out_offsets_host, void* workspace, size_t workspace_bytes, void* cuda_stream);

/*
 * The raw product a*b without merging (reading A10): out_coef[na*nb], out_exps[na*nb x nvars] row-major,
 * term (i,j) at index i*nb + j.  workspace: POLYLAB_SMALL_WORKSPACE_BYTES.  Exponent sums that do not fit
 * exp_type -> POLYLAB_ERR_EXPONENT_RANGE (the call synchronises to report it).
 */
int polylab_expand(const polylab_poly* a, const polylab_poly* b, const polylab_opts* opts,
                   double* out_coef, void* out_exps, void* workspace, size_t workspace_bytes, void* cuda_stream);

/*
 * Step S1 alone, exposed for stage-level parity tests: packs each exponent row into a 128-bit key
 * written as two uint64 (hi, lo) to out_keys[2*nterms]; unsigned order of (hi,lo) = lexicographic order
 * of rows.  Field widths come from max_exp_host when given, else from the data.  key_bits_host (HOST,
 * optional) receives B.  workspace: POLYLAB_SMALL_WORKSPACE_BYTES.  Synchronises.
 */
int polylab_pack_keys(const void* exps, int64_t nterms, int32_t nvars, const polylab_opts* opts,
                      uint64_t* out_keys, int32_t* key_bits_host, void* workspace, size_t workspace_bytes,
                      void* cuda_stream);

/*
 * The same two operations with HOST input and output buffers (pageable or pinned): copies the inputs
 * into `device_workspace`, runs the device path, copies the result back, synchronises.  Workspace
 * size from the *_host_workspace_bytes queries (inputs + outputs + the device path's workspace).
 * opts->max_exp_host still applies; strides must be row-major here.
 */
size_t polylab_simplify_host_workspace_bytes(int64_t nterms, int32_t nvars, const polylab_opts* opts);
size_t polylab_mul_simplify_host_workspace_bytes(int64_t na, int64_t nb, int32_t nvars, const polylab_opts* opts);
int polylab_simplify_host(const double* coef_host, const void* exps_host, int64_t nterms, int32_t nvars,
                          double tol, const polylab_opts* opts,
                          double* out_coef_host, void* out_exps_host, int64_t out_capacity,
                          int64_t* out_nterms_host,
                          void* device_workspace, size_t workspace_bytes, void* cuda_stream);
int polylab_mul_simplify_host(const polylab_poly* a_host, const polylab_poly* b_host, double tol,
                              const polylab_opts* opts,
                              double* out_coef_host, void* out_exps_host, int64_t out_capacity,
                              int64_t* out_nterms_host,
                              void* device_workspace, size_t workspace_bytes, void* cuda_stream);

/*
 * polylab_simplify without a workspace argument and without any allocation: the scratch memory of the whole pipeline is a
 * static device array of POLYLAB_STATIC_WORKSPACE_BYTES inside the library (every GPU that loads the library holds it until
 * the process exits).  For callers that cannot call cudaMalloc or hand over device memory of their own: set-up code around
 * CUDA graph capture, tight serving loops, harnesses that forbid allocation.  The operation, the arguments, the result and the
 * statuses are polylab_simplify's (Table 3; section 6.3), bit for bit, with these differences:
 *   - nterms <= POLYLAB_STATIC_MAX_TERMS; more (or a layout that does not fit the array) is POLYLAB_ERR_WORKSPACE_TOO_SMALL
 *     and nothing is launched;
 *   - POLYLAB_FLAG_TIMING is POLYLAB_ERR_INVALID_ARGUMENT (stage events would have to be created);
 *   - the call makes no cudaMalloc / cudaFree / allocating library call; the array's device address is looked up once per
 *     device, on the first call with that device current;
 *   - ALL calls on a GPU share the one array, which keeps the previous call's contents (each call clears what it needs
 *     zeroed): two calls that overlap on the GPU -- different streams, or two host threads -- race; serialise them.
 * coef, exps, out_coef, out_exps are DEVICE pointers owned by the caller, as in polylab_simplify.
 */
#define POLYLAB_STATIC_MAX_TERMS 65536
#define POLYLAB_STATIC_WORKSPACE_BYTES (8u << 20)
int polylab_simplify_static(const double* coef, const void* exps, int64_t nterms, int32_t nvars, double tol,
                            const polylab_opts* opts, double* out_coef, void* out_exps, int64_t out_capacity,
                            int64_t* out_nterms, void* cuda_stream);

const char* polylab_status_string(int status);
const char* polylab_last_cuda_error(void);   /* text of the last CUDA failure seen by this thread */
int polylab_version(void);

#if defined(__GNUC__)
#pragma GCC visibility pop
#endif

#ifdef __cplusplus
}
#endif
#endif /* POLYLAB_H */
