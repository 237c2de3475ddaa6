// small.cu -- steps S2 and S3 of a SMALL input in one thread block: sort and segmented sum without a single trip through
// global memory in between; the runs then go through the ordinary prune / unpack kernel (S4, S5: reduce.cu), whose many
// blocks write the output rows far faster than one SM can (measured: 58 us of 104 for 7,680 rows of 10 bytes).  Used
// (a) for inputs of at most small_cap() terms, where the multi-kernel radix path is all launch latency (the paper's
// lightweight-operator regime, Table 7), and (b) as the tail of the table path (table.cu) when at most
// that many distinct monomials are left to put in canonical order.
//
// The block keeps the keys in shared memory and sorts a PERMUTATION of them, least significant plan digit first: warp w
// ranks the 1/32 of the positions it owns (one shared-memory atomic per record, order verified afterwards), a 256-bin
// scan over (warp, digit) counts gives every record its slot, and only 16-bit indices move.  A stable sort sums equal
// monomials in input order -- left to right inside a thread, by a fixed shuffle tree across threads (reading A6): a
// function of the layout only, bit-reproducible.  Measured and rejected: a bitonic network over 8192 pairs (91 stages *
// 164 KB of shared-memory traffic on ONE SM = 183 us); ballot-matching ranks (3x the instructions, and one block has one
// SM's four issue slots: 15k cycles per pass).
#include "kernels.h"

namespace polylab {

constexpr int kSmallThreads = 1024;

// Most pairs the one-block path takes: the keys twice (original order, sorted order; the first copy later holds the sorted
// coefficients) + two permutations + the (digit, warp) counters must fit 227 KB of shared memory.
template <typename K>
struct SmallSmem {
    static constexpr int CAP = kSmallCap * 8 / (int)sizeof(K);
    static constexpr int HROW = 33;                                          // counters of one digit: 32 warps + 1 pad (bank spread)
    static constexpr size_t off_a = 0;                                       // keys by original index, then sorted coefficients
    static constexpr size_t off_b = off_a + (size_t)CAP * sizeof(K);         // sorted keys
    static constexpr size_t off_p0 = off_b + (size_t)CAP * sizeof(K);        // permutation ping
    static constexpr size_t off_p1 = off_p0 + (size_t)CAP * 2;               // permutation pong
    static constexpr size_t off_hist = off_p1 + (size_t)CAP * 2;             // [256][33] u32: records of warp w with digit d
    static constexpr size_t off_bin = off_hist + (size_t)kRadix * HROW * 4;  // [256] u32: first slot of digit d
    static constexpr size_t bytes = off_bin + (size_t)kRadix * 4;
};

template <typename K>
__global__ void __launch_bounds__(kSmallThreads, 1) block_sort_reduce_kernel(const K* __restrict__ keys, CoefIn coefs,
                                                                           const uint32_t* n_device, uint32_t n_host,
                                                                           const __grid_constant__ Plan plan, K* __restrict__ ukeys,
                                                                           double* __restrict__ usums, Control* ctl)
{
    constexpr int T = kSmallThreads, NW = T / 32, CAP = SmallSmem<K>::CAP, MAXIT = CAP / T, HROW = SmallSmem<K>::HROW;
    static_assert(NW == 32, "one lane per warp in the counter scan");
    extern __shared__ __align__(16) unsigned char smem_raw[];
    K* ka = (K*)(smem_raw + SmallSmem<K>::off_a);
    K* sk = (K*)(smem_raw + SmallSmem<K>::off_b);
    double* sc = (double*)(smem_raw + SmallSmem<K>::off_a);
    uint16_t* pin = (uint16_t*)(smem_raw + SmallSmem<K>::off_p0);
    uint16_t* pout = (uint16_t*)(smem_raw + SmallSmem<K>::off_p1);
    uint32_t* wh = (uint32_t*)(smem_raw + SmallSmem<K>::off_hist);
    uint32_t* sbin = (uint32_t*)(smem_raw + SmallSmem<K>::off_bin);
    __shared__ uint32_t scratch[NW + 2];
    __shared__ uint32_t wagg_f[NW];
    __shared__ double wagg_v[NW];
    const unsigned tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
    const uint32_t n = n_device ? min(*n_device, (uint32_t)CAP) : n_host;
    if (n == 0) {
        if (tid == 0) ctl->distinct = 0;
        return;
    }
    for (uint32_t i = tid; i < n; i += T) {
        ka[i] = keys[i];
        pin[i] = (uint16_t)i;
    }
    // ---- S2: stable LSD radix sort of the permutation, one plan digit per pass.  Warp w owns positions [wbeg, wend); all its
    // loads of a pass are issued up front (the kernel is one block: latency, not bandwidth, is what it has to hide).
    const uint32_t per = (((n + NW - 1) / NW) + 31u) & ~31u;           // positions per warp, a multiple of 32
    const uint32_t wbeg = min(warp * per, n), wend = min(wbeg + per, n);
    constexpr uint32_t kNone = 0xffffffffu;
    for (int p = 0; p < plan.npasses; ++p) {
        const int dpos = plan.digit_pos[p];
        const uint32_t dmask = (1u << plan.digit_bits[p]) - 1u;
        for (uint32_t i = tid; i < (uint32_t)(kRadix * HROW); i += T) wh[i] = 0u;
        __syncthreads();                                               // counters zeroed, pin complete
        uint32_t rec[MAXIT], dig[MAXIT], rk[MAXIT];
#pragma unroll
        for (int u = 0; u < MAXIT; ++u) {
            const uint32_t i = wbeg + u * 32u + lane;
            rec[u] = i < wend ? pin[i] : 0u;
            dig[u] = i < wend ? key_digit(ka[rec[u]], dpos, dmask) : kNone;
        }
        // rank among the warp's records of the same digit: the old value of ONE shared-memory atomic per record.  Stable
        // because a warp instruction's same-address shared atomics return in lane order on sm_100a (measured,
        // profiles/r1b_shared_atomics.md; not documented): the run detection below verifies the order and raises
        // ctl->unsorted, upon which the call re-runs on the multi-kernel path (ballot matching here: 3x the instructions
        // of a block that has ONE SM's four issue slots)
#pragma unroll
        for (int u = 0; u < MAXIT; ++u) {
            rk[u] = 0u;
            if (dig[u] != kNone) rk[u] = atomicAdd(wh + dig[u] * HROW + warp, 1u);
            __syncwarp();
        }
        __syncthreads();
        // exclusive scan of every digit's counters over the warps (lane = source warp), eight digits per warp
        {
            uint32_t c[8], x[8];
#pragma unroll
            for (int q = 0; q < 8; ++q) { c[q] = wh[(warp * 8 + q) * HROW + lane]; x[q] = c[q]; }
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
#pragma unroll
                for (int q = 0; q < 8; ++q) {
                    const uint32_t y = __shfl_up_sync(kFullMask, x[q], o);
                    if (lane >= (unsigned)o) x[q] += y;
                }
            }
#pragma unroll
            for (int q = 0; q < 8; ++q) {
                wh[(warp * 8 + q) * HROW + lane] = x[q] - c[q];
                if (lane == 31) sbin[warp * 8 + q] = x[q];             // the digit's total
            }
        }
        __syncthreads();
        uint32_t total;
        const uint32_t bin_start = block_exclusive_scan<T>(tid < (unsigned)kRadix ? sbin[tid] : 0u, scratch, &total);
        __syncthreads();
        if (tid < (unsigned)kRadix) sbin[tid] = bin_start;
        __syncthreads();
#pragma unroll
        for (int u = 0; u < MAXIT; ++u)
            if (dig[u] != kNone) pout[sbin[dig[u]] + wh[dig[u] * HROW + warp] + rk[u]] = (uint16_t)rec[u];
        __syncthreads();
        uint16_t* t = pin; pin = pout; pout = t;
    }
    __syncthreads();
    for (uint32_t i = tid; i < n; i += T) sk[i] = ka[pin[i]];          // keys in sorted order
    __syncthreads();                                                   // the original-order keys are dead: their place takes
    for (uint32_t i = tid; i < n; i += T) sc[i] = coefs[pin[i]];       // the coefficients in sorted order
    __syncthreads();

    // ---- S3: runs of equal keys; thread t owns the `it` consecutive positions from t * it.  Run number r (= the ordinal of
    // its head) is written to (ukeys, usums)[r] by the thread in which it ENDS.
    // (an ODD number of positions per thread: the threads' strided shared-memory reads then spread over all banks; with the
    // even stride of 8 eight-byte keys they hit two bank groups 16 ways -- measured 36k of the kernel's 95k cycles)
    const uint32_t it = ((n + T - 1) / T) | 1u;
    const uint32_t first = tid * it;
    uint32_t hm = 0, nh = 0, nclosed = 0;
    double acc = 0.0;
    double csum[MAXIT + 1];
    bool descending = false;
#pragma unroll
    for (int j = 0; j < MAXIT + 1; ++j) {
        csum[j] = 0.0;
        if ((uint32_t)j < it && first + j < n) {
            bool head = true;
            if (first + j > 0) {
                const K kp = sk[first + j - 1], kk = sk[first + j];
                head = !key_eq(kk, kp);
                descending |= key_lt(kk, kp);
            }
            if (head) {
                if (first + j > 0) { csum[nclosed] = acc; ++nclosed; }     // the run that ends just before this head
                hm |= 1u << j; ++nh; acc = sc[first + j];
            } else acc = __dadd_rn(acc, sc[first + j]);
        }
    }
    if (descending) ctl->unsorted = 1u;                              // the atomic ranking was not stable: the caller re-runs
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
    SegPair carry;
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
    if (nclosed > 0) csum[0] = __dadd_rn(carry.v, csum[0]);          // the first run that ends here began in earlier threads
    uint32_t H;
    const uint32_t hb = block_exclusive_scan<T>(nh, scratch, &H);   // ordinal of this thread's first head
    {
        uint32_t c = 0;
        const uint32_t chm = (first == 0) ? (hm & ~1u) : hm;          // the heads that close a run
        // closing head number c of this thread has ordinal hb + c (+1 in the thread that owns position 0, whose first
        // head closes nothing); the run it closes is the one before it
        const uint32_t r0 = hb + ((first == 0 && (hm & 1u)) ? 1u : 0u);
        for (uint32_t m = chm; m != 0u; m &= m - 1u, ++c) {
            usums[r0 + c - 1u] = csum[c];
            ukeys[r0 + c - 1u] = sk[first + (__ffs(m) - 1) - 1];
        }
    }
    if (tid == T - 1) {
        usums[H - 1u] = incl.v;                                      // the run still open at the end
        ukeys[H - 1u] = sk[n - 1];
        ctl->distinct = H;
    }
}

template <typename K>
static int launch_block_sort_reduce_t(const Plan& plan, const void* keys, CoefIn coefs, const uint32_t* n_device, uint32_t n,
                                      void* ukeys, double* usums, Control* ctl, cudaStream_t stream)
{
    auto kern = block_sort_reduce_kernel<K>;
    ensure_dynamic_smem(kern, (size_t)SmallSmem<K>::bytes);
    kern<<<1, kSmallThreads, SmallSmem<K>::bytes, stream>>>((const K*)keys, coefs, n_device, n, plan, (K*)ukeys, usums, ctl);
    return 1;
}

int launch_block_sort_reduce(const Plan& plan, const void* keys, CoefIn coefs, const uint32_t* n_device, uint32_t n,
                             void* ukeys, double* usums, Control* ctl, cudaStream_t stream)
{
    if (plan.key_bytes == 8) return launch_block_sort_reduce_t<uint64_t>(plan, keys, coefs, n_device, n, ukeys, usums, ctl, stream);
    if (plan.key_bytes == 16) return launch_block_sort_reduce_t<Key128>(plan, keys, coefs, n_device, n, ukeys, usums, ctl, stream);
    return launch_block_sort_reduce_t<Key256>(plan, keys, coefs, n_device, n, ukeys, usums, ctl, stream);
}

}  // namespace polylab
