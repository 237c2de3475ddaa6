// batch.cu -- batched simplify: many independent polynomials -- the entries of a polynomial matrix --
// simplified by ONE pass of the pipeline.  The paper's polynomial matrices are arrays of scalar polynomials whose
// mtimes / sum / prod apply the scalar operations entry by entry (Table 4; section 3.4:
// A^2 for A = [x1 1; 0 x2]); these are the launch-bound rows where its GPU backends lose to the CPU (PAPER.md:560-563,
// Table 7).  Here the entry index becomes the MOST significant field of the packed key, above variable 0: one sort /
// segmented sum / prune / unpack then leaves the entries' simplified polynomials concatenated in entry order, each in
// canonical monomial order, and a count per entry gives the offsets.
//
// The records are described by SEGMENTS: segment s contributes to entry `entry` either the raw terms [a0, a0 + na) of a
// packed polynomial (nb == 0) or all na * nb products of terms [a0, a0 + na) of A with terms [b0, b0 + nb) of B (step X1;
// a matrix product's entry (i, j) has one segment per inner index l).  Record q finds its segment by binary search over
// the segments' first record numbers.
#include "kernels.h"

namespace polylab {

// the entry index is one more field of the key, above variable 0 (at most 30 bits: nentries < 2^30)
template <typename K> __device__ __forceinline__ K entry_key(K k, uint32_t entry, int shift) { key_or_field(k, entry, shift); return k; }
template <typename K> __device__ __forceinline__ uint32_t key_entry(const K& k, int shift, int width) { return key_get_field(k, shift, width); }

template <typename K>
__global__ void __launch_bounds__(256) batched_expand_kernel(const BatchSeg* __restrict__ segs, uint32_t nseg, uint32_t n,
                                                             const K* __restrict__ ka, CoefIn ca,
                                                             const K* __restrict__ kb, CoefIn cb,
                                                             int entry_shift, K* __restrict__ keys, double* __restrict__ coefs,
                                                             int dpos, uint32_t dmask, uint32_t* hist)
{
    __shared__ uint32_t sh[kRadix];
    for (int b = threadIdx.x; b < kRadix; b += blockDim.x) sh[b] = 0u;
    __syncthreads();
    for (uint32_t q = blockIdx.x * blockDim.x + threadIdx.x; q < n; q += gridDim.x * blockDim.x) {
        uint32_t lo = 0, hi = nseg;                      // the last segment whose first record is <= q
        while (hi - lo > 1u) {
            const uint32_t mid = (lo + hi) >> 1;
            if (__ldg(&segs[mid].start) <= q) lo = mid; else hi = mid;
        }
        const BatchSeg s = segs[lo];
        const uint32_t r = q - s.start;
        K key;
        double c;
        if (s.nb == 0u) {
            key = ka[s.a0 + r];
            c = ca[s.a0 + r];
        } else {
            const uint32_t i = r / s.nb, j = r - i * s.nb;
            key = key_add(ka[s.a0 + i], kb[s.b0 + j]);    // fields sized for max_a + max_b: no carry between them
            c = __dmul_rn(ca[s.a0 + i], cb[s.b0 + j]);    // one IEEE multiplication, never contracted
        }
        key = entry_key(key, s.entry, entry_shift);
        keys[q] = key;
        coefs[q] = c;
        if (dmask) atomicAdd(&sh[key_digit(key, dpos, dmask)], 1u);
    }
    __syncthreads();
    if (dmask)
        for (int b = threadIdx.x; b < kRadix; b += blockDim.x)
            if (sh[b]) atomicAdd(&hist[b], sh[b]);
}

int launch_batched_expand(const Plan& plan, const BatchSeg* segs, uint32_t nseg, int64_t n, const void* ka, CoefIn ca,
                          const void* kb, CoefIn cb, int entry_shift, void* keys, double* coefs, Control* ctl, cudaStream_t stream)
{
    if (n <= 0 || nseg == 0) return 0;
    int64_t blocks = (n + 1023) / 1024;
    if (blocks > sm_count() * 16) blocks = sm_count() * 16;
    const int dpos = plan.npasses ? plan.digit_pos[0] : 0;
    const uint32_t dmask = plan.npasses ? (1u << plan.digit_bits[0]) - 1u : 0u;
    if (plan.key_bytes == 8)
        batched_expand_kernel<uint64_t><<<(unsigned)blocks, 256, 0, stream>>>(segs, nseg, (uint32_t)n, (const uint64_t*)ka, ca, (const uint64_t*)kb,
                                                                            cb, entry_shift, (uint64_t*)keys, coefs, dpos, dmask, ctl->hist[0]);
    else if (plan.key_bytes == 16)
        batched_expand_kernel<Key128><<<(unsigned)blocks, 256, 0, stream>>>(segs, nseg, (uint32_t)n, (const Key128*)ka, ca, (const Key128*)kb, cb,
                                                                          entry_shift, (Key128*)keys, coefs, dpos, dmask, ctl->hist[0]);
    else
        batched_expand_kernel<Key256><<<(unsigned)blocks, 256, 0, stream>>>(segs, nseg, (uint32_t)n, (const Key256*)ka, ca, (const Key256*)kb, cb,
                                                                          entry_shift, (Key256*)keys, coefs, dpos, dmask, ctl->hist[0]);
    return 1;
}

// survivors per entry, from the merged (key, sum) list (the prune predicate of S4, reading A2)
template <typename K>
__global__ void __launch_bounds__(256) entry_count_kernel(const K* __restrict__ ukeys, const double* __restrict__ usums, const Control* ctl,
                                                          double tol, int entry_shift, int entry_bits, uint32_t* __restrict__ counts)
{
    const uint32_t U = ctl->distinct;
    for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < U; i += gridDim.x * blockDim.x)
        if (fabs(usums[i]) > tol) atomicAdd(&counts[key_entry(ukeys[i], entry_shift, entry_bits)], 1u);
}

int launch_entry_count(int key_bytes, int key_bits, int64_t max_units, const void* ukeys, const double* usums, const Control* ctl, double tol,
                       int entry_shift, uint32_t* counts, cudaStream_t stream)
{
    if (max_units <= 0) return 0;
    int64_t blocks = (max_units + 1023) / 1024;
    if (blocks > sm_count() * 8) blocks = sm_count() * 8;
    const int eb = key_bits - entry_shift;
    if (key_bytes == 8) entry_count_kernel<uint64_t><<<(unsigned)blocks, 256, 0, stream>>>((const uint64_t*)ukeys, usums, ctl, tol, entry_shift, eb, counts);
    else if (key_bytes == 16) entry_count_kernel<Key128><<<(unsigned)blocks, 256, 0, stream>>>((const Key128*)ukeys, usums, ctl, tol, entry_shift, eb, counts);
    else entry_count_kernel<Key256><<<(unsigned)blocks, 256, 0, stream>>>((const Key256*)ukeys, usums, ctl, tol, entry_shift, eb, counts);
    return 1;
}

}  // namespace polylab
