// pack.cu -- steps S0 (bounds), S1 (pack exponent rows into keys) and X1 (term-product expansion).
//
// S1: key_t = sum_v e_{t,v} << shift_v with variable 0 in the most significant field (
// the row order it must reproduce is the paper's transcript order).
// X1: all na*nb products of two polynomials -- coefficient products and exponent sums (mtimes/times,
// PAPER.md:117-118); on packed keys the exponent sum of every variable is ONE integer addition because
// the plan sizes each field for max_a + max_b (no carry between fields).
#include "kernels.h"

namespace polylab {

// ----------------------------------------------------------------------------------------------- S0

// Thread tid of the first VT = (THREADS / nvars) * nvars threads always meets variable tid % nvars, so
// the running maximum lives in a register; one shared and one global atomicMax per variable per block.
template <int THREADS>
__global__ void __launch_bounds__(THREADS) bounds_kernel(ExpView ev, int64_t nterms, int nvars, uint32_t* gmax)
{
    __shared__ uint32_t smax[kMaxVars];
    const int tid = threadIdx.x;
    if (tid < nvars) smax[tid] = 0u;
    __syncthreads();
    const int rows_per_iter = THREADS / nvars;
    if (tid < rows_per_iter * nvars) {
        const int v = tid % nvars, r = tid / nvars;
        const int64_t step = (int64_t)gridDim.x * rows_per_iter;
        uint32_t m = 0u;
        const int64_t voff = (int64_t)v * ev.var_stride;
#pragma unroll 8
        for (int64_t t = (int64_t)blockIdx.x * rows_per_iter + r; t < nterms; t += step)
            m = max(m, load_exp(ev.base, ev.exp_bytes, t * ev.term_stride + voff));
        if (m) atomicMax(&smax[v], m);
    }
    __syncthreads();
    if (tid < nvars && smax[tid]) atomicMax(&gmax[tid], smax[tid]);
}

// Contiguous row-major rows (16-byte aligned base): the matrix is read as a stream of 16-byte words.  The grid's
// sweep (gridDim * THREADS * 16 bytes) is a multiple of the row size, so byte lane i of a thread's word always
// holds the same variable and the running maximum is a lane-wise SIMD max (4 x u8 / 2 x u16 / 1 x u32 per
// 32-bit register).  One shared atomicMax per lane per thread at the end, one global per variable per block.
template <int THREADS, int ES>
__global__ void __launch_bounds__(THREADS) bounds_stream_kernel(const uint4* __restrict__ base, int64_t nbytes, int nvars,
                                                                uint32_t* gmax)
{
    __shared__ uint32_t smax[kMaxVars];
    const int tid = threadIdx.x;
    if (tid < nvars) smax[tid] = 0u;
    __syncthreads();
    const int64_t nwords = nbytes >> 4;                       // full 16-byte words; the tail is handled below
    const int64_t stride = (int64_t)gridDim.x * THREADS;
    const int64_t w0 = (int64_t)blockIdx.x * THREADS + tid;
    uint32_t m[4] = {0u, 0u, 0u, 0u};
    auto acc = [&](const uint4& q) {
        if (ES == 1) { m[0] = __vmaxu4(m[0], q.x); m[1] = __vmaxu4(m[1], q.y); m[2] = __vmaxu4(m[2], q.z); m[3] = __vmaxu4(m[3], q.w); }
        else if (ES == 2) { m[0] = __vmaxu2(m[0], q.x); m[1] = __vmaxu2(m[1], q.y); m[2] = __vmaxu2(m[2], q.z); m[3] = __vmaxu2(m[3], q.w); }
        else { m[0] = max(m[0], q.x); m[1] = max(m[1], q.y); m[2] = max(m[2], q.z); m[3] = max(m[3], q.w); }
    };
    int64_t w = w0;
    for (; w + 3 * stride < nwords; w += 4 * stride) {        // four independent 16-byte loads in flight
        const uint4 q0 = __ldg(base + w), q1 = __ldg(base + w + stride), q2 = __ldg(base + w + 2 * stride),
                    q3 = __ldg(base + w + 3 * stride);
        acc(q0); acc(q1); acc(q2); acc(q3);
    }
    for (; w < nwords; w += stride) acc(__ldg(base + w));
    // lane i of this thread's words is element (w0 * 16 / ES + i) of the stream, i.e. variable (that) % nvars
    const int64_t e0 = w0 * (16 / ES);
#pragma unroll
    for (int i = 0; i < 16 / ES; ++i) {
        uint32_t x;
        if (ES == 1) x = (m[i / 4] >> (8 * (i % 4))) & 0xffu;
        else if (ES == 2) x = (m[i / 2] >> (16 * (i % 2))) & 0xffffu;
        else x = m[i];
        if (x) atomicMax(&smax[(int)((e0 + i) % nvars)], x);
    }
    // tail: the last nbytes % 16 bytes, element by element
    if (blockIdx.x == 0) {
        const int64_t ne = nbytes / ES;
        for (int64_t e = nwords * (16 / ES) + tid; e < ne; e += THREADS) {
            const uint32_t x = load_exp(base, ES, e);
            if (x) atomicMax(&smax[(int)(e % nvars)], x);
        }
    }
    __syncthreads();
    if (tid < nvars && smax[tid]) atomicMax(&gmax[tid], smax[tid]);
}

// Maxima over a SAMPLE of the rows: block b sweeps rows [b*seg_stride, b*seg_stride + seg_rows).  Any strides.
template <int THREADS>
__global__ void __launch_bounds__(THREADS) bounds_sample_kernel(ExpView ev, int64_t nterms, int nvars, int64_t seg_stride,
                                                                int seg_rows, uint32_t* gmax)
{
    __shared__ uint32_t smax[kMaxVars];
    const int tid = threadIdx.x;
    if (tid < nvars) smax[tid] = 0u;
    __syncthreads();
    const int rows_per_iter = THREADS / nvars;
    if (tid < rows_per_iter * nvars) {
        const int v = tid % nvars, r = tid / nvars;
        const int64_t t0 = (int64_t)blockIdx.x * seg_stride;
        const int64_t t1 = min(nterms, t0 + seg_rows);
        uint32_t m = 0u;
        const int64_t voff = (int64_t)v * ev.var_stride;
#pragma unroll 4
        for (int64_t t = t0 + r; t < t1; t += rows_per_iter)
            m = max(m, load_exp(ev.base, ev.exp_bytes, t * ev.term_stride + voff));
        if (m) atomicMax(&smax[v], m);
    }
    __syncthreads();
    if (tid < nvars && smax[tid]) atomicMax(&gmax[tid], smax[tid]);
}

int launch_bounds_sample(const ExpView& ev, int64_t nterms, int nvars, Control* ctl, int which, cudaStream_t stream)
{
    if (nterms <= 0) return 0;
    const int kSegs = sm_count() * 8;
    constexpr int kSegRows = 512;
    bounds_sample_kernel<256><<<kSegs, 256, 0, stream>>>(ev, nterms, nvars, nterms / kSegs, kSegRows, ctl->max_exp[which]);
    return 1;
}

int launch_bounds(const ExpView& ev, int64_t nterms, int nvars, Control* ctl, int which, cudaStream_t stream)
{
    if (nterms <= 0) return 0;
    constexpr int T = 256;
    if (ev.row_major_contiguous) {
        // grid = k * (row bytes): the sweep of gridDim * T * 16 bytes is then a whole number of rows
        const int rb = nvars * ev.exp_bytes;
        const int64_t nbytes = nterms * rb;
        int64_t k = (nbytes / 16 + (int64_t)T * 8 - 1) / ((int64_t)T * 8) / rb;      // ~8 words per thread
        const int64_t kmax = (sm_count() * 16 + rb - 1) / rb;
        if (k > kmax) k = kmax;
        if (k < 1) k = 1;
        const unsigned blocks = (unsigned)(k * rb);
        const uint4* base = (const uint4*)ev.base;
        if (ev.exp_bytes == 1) bounds_stream_kernel<T, 1><<<blocks, T, 0, stream>>>(base, nbytes, nvars, ctl->max_exp[which]);
        else if (ev.exp_bytes == 2) bounds_stream_kernel<T, 2><<<blocks, T, 0, stream>>>(base, nbytes, nvars, ctl->max_exp[which]);
        else bounds_stream_kernel<T, 4><<<blocks, T, 0, stream>>>(base, nbytes, nvars, ctl->max_exp[which]);
        return 1;
    }
    const int rows_per_iter = T / nvars;
    int64_t blocks = (nterms + (int64_t)rows_per_iter * 16 - 1) / ((int64_t)rows_per_iter * 16);
    if (blocks > sm_count() * 16) blocks = sm_count() * 16;
    bounds_kernel<T><<<(unsigned)blocks, T, 0, stream>>>(ev, nterms, nvars, ctl->max_exp[which]);
    return 1;
}

// A product's exponent sums must fit exp_type (reading A8).  With bounds from the data the host checks max_a + max_b; with
// caller bounds (no read-back) the operands' true maxima are taken on the device and compared here.
__global__ void sum_range_check_kernel(Control* ctl, int nvars, uint32_t emax)
{
    const int v = blockIdx.x * blockDim.x + threadIdx.x;
    if (v < nvars && (uint64_t)ctl->max_exp[0][v] + ctl->max_exp[1][v] > emax) atomicMax(&ctl->status, (int)POLYLAB_ERR_EXPONENT_RANGE);
}

int launch_sum_range_check(const ExpView& ea, int64_t na, const ExpView& eb, int64_t nb, int nvars, uint32_t emax, Control* ctl,
                           cudaStream_t stream)
{
    int launches = launch_bounds(ea, na, nvars, ctl, 0, stream) + launch_bounds(eb, nb, nvars, ctl, 1, stream);
    sum_range_check_kernel<<<1, kMaxVars, 0, stream>>>(ctl, nvars, emax);
    return launches + 1;
}

// ----------------------------------------------------------------------------------------------- S1

// first-pass digit histogram of a block: shared atomics, flushed with one global reduction per non-empty bin
struct BlockHist {
    uint32_t* sh;
    __device__ void init(uint32_t* s) { sh = s; for (int b = threadIdx.x; b < kRadix; b += blockDim.x) sh[b] = 0u; }
    __device__ void add(uint32_t d) { atomicAdd(&sh[d], 1u); }
    __device__ void flush(uint32_t* g)
    {
        for (int b = threadIdx.x; b < kRadix; b += blockDim.x)
            if (sh[b]) atomicAdd(&g[b], sh[b]);
    }
};


// Rows contiguous in memory (row-major, 16-byte aligned base): each thread reads its row with the widest
// word WB (bytes) that divides the row size; ES = bytes per exponent.
template <typename K, int ES, int WB>
__global__ void __launch_bounds__(256) pack_rows_kernel(const uint8_t* __restrict__ base, int64_t nterms,
                                                        const __grid_constant__ Plan plan, K* __restrict__ keys,
                                                        Control* ctl, int hd)
{
    __shared__ uint32_t sh[kRadix];
    BlockHist bh;
    if (hd >= 0) { bh.init(sh); __syncthreads(); }
    const int rb = plan.nvars * ES;
    const int dpos = plan.digit_pos[hd >= 0 ? hd : 0];
    const uint32_t dmask = (1u << plan.digit_bits[hd >= 0 ? hd : 0]) - 1u;
    bool bad = false;
    for (int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; t < nterms; t += (int64_t)gridDim.x * blockDim.x) {
        const uint8_t* row = base + t * rb;
        K key;
        key_zero(key);
        for (int c = 0; c < rb; c += WB) {
            uint32_t w[WB >= 4 ? WB / 4 : 1];
            if (WB == 16) {
                const uint4 q = __ldg((const uint4*)(row + c));
                w[0] = q.x; w[WB >= 16 ? 1 : 0] = q.y; w[WB >= 16 ? 2 : 0] = q.z; w[WB >= 16 ? 3 : 0] = q.w;
            } else if (WB == 4) w[0] = __ldg((const uint32_t*)(row + c));
            else if (WB == 2) w[0] = __ldg((const uint16_t*)(row + c));
            else w[0] = __ldg(row + c);
            const int v0 = c / ES;
#pragma unroll
            for (int k = 0; k < WB / ES; ++k) {
                uint32_t e;
                if (ES == 4) e = w[k];
                else if (ES == 2) e = (w[k / 2] >> (16 * (k % 2))) & 0xffffu;
                else e = (w[k / 4] >> (8 * (k % 4))) & 0xffu;
                pack_field(key, e, v0 + k, plan, bad);
            }
        }
        keys[t] = key;
        if (hd >= 0) bh.add(key_digit(key, dpos, dmask));
    }
    if (bad) atomicMax(&ctl->status, (int)POLYLAB_ERR_EXPONENT_RANGE);
    if (hd >= 0) { __syncthreads(); bh.flush(ctl->hist[hd]); }
}

// Contiguous rows whose size is not a multiple of 16 bytes (10 one-byte variables, 6 two-byte ones, ...): a thread reading
// its own row would issue narrow, misaligned loads (five 2-byte loads for a 10-byte row).  Instead the block brings a tile
// of `tile_rows` consecutive rows into shared memory with aligned 16-byte asynchronous copies (cp.async), double-buffered:
// the next tile is in flight while every thread picks its rows of the current one out of shared memory.

template <typename K, int ES>
__global__ void __launch_bounds__(256) pack_rows_staged_kernel(const uint8_t* __restrict__ base, int64_t nterms, int tile_rows,
                                                               const __grid_constant__ Plan plan, K* __restrict__ keys,
                                                               Control* ctl, int hd)
{
    extern __shared__ __align__(16) unsigned char stage[];          // two buffers of tile_rows * row bytes + 16, each 16-byte aligned
    __shared__ uint32_t sh[kRadix];
    BlockHist bh;
    if (hd >= 0) { bh.init(sh); }
    const int rb = plan.nvars * ES;
    const int dpos = plan.digit_pos[hd >= 0 ? hd : 0];
    const uint32_t dmask = (1u << plan.digit_bits[hd >= 0 ? hd : 0]) - 1u;
    const int64_t nbytes = nterms * rb;
    const int bufsz = (tile_rows * rb + 16 + 15) & ~15;
    const int64_t step = (int64_t)gridDim.x * tile_rows;
    auto issue = [&](int buf, int64_t t0) {                          // rows [t0, t0 + tile_rows) -> stage + buf * bufsz
        if (t0 < nterms) {
            const int nr = (int)min((int64_t)tile_rows, nterms - t0);
            const int64_t b0 = t0 * rb, b1 = b0 + (int64_t)nr * rb, a0 = b0 & ~(int64_t)15;
            unsigned char* dst = stage + (size_t)buf * bufsz;
            for (int64_t off = a0 + 16 * (int64_t)threadIdx.x; off < b1; off += 16 * 256) {
                if (off + 16 <= nbytes) cp_async16(dst + (off - a0), base + off);
                else for (int64_t b = off; b < nbytes; ++b) dst[b - a0] = base[b];         // the array's last, partial word
            }
        }
        asm volatile("cp.async.commit_group;" ::: "memory");
    };
    bool bad = false;
    int64_t t0 = (int64_t)blockIdx.x * tile_rows;
    issue(0, t0);
    for (int it = 0; t0 < nterms; ++it, t0 += step) {
        const int cur = it & 1;
        issue(cur ^ 1, t0 + step);                                  // (the buffer was released by the barrier that ended the last round)
        asm volatile("cp.async.wait_group 1;" ::: "memory");
        __syncthreads();                                            // tile `cur` has landed for every thread
        const int nr = (int)min((int64_t)tile_rows, nterms - t0);
        const int64_t b0 = t0 * rb, a0 = b0 & ~(int64_t)15;
        const unsigned char* src = stage + (size_t)cur * bufsz + (b0 - a0);
        for (int r = threadIdx.x; r < nr; r += 256) {
            const unsigned char* row = src + (int64_t)r * rb;
            K key;
            key_zero(key);
            for (int v = 0; v < plan.nvars; ++v) {
                const uint32_t e = ES == 1 ? row[v] : ES == 2 ? ((const uint16_t*)row)[v] : ((const uint32_t*)row)[v];
                pack_field(key, e, v, plan, bad);
            }
            keys[t0 + r] = key;
            if (hd >= 0) bh.add(key_digit(key, dpos, dmask));
        }
        __syncthreads();                                            // tile `cur` has been read: its buffer may be refilled
    }
    asm volatile("cp.async.wait_group 0;" ::: "memory");
    if (bad) atomicMax(&ctl->status, (int)POLYLAB_ERR_EXPONENT_RANGE);
    if (hd >= 0) { __syncthreads(); bh.flush(ctl->hist[hd]); }
}

// Any strides / alignment: one element load per variable.
template <typename K>
__global__ void __launch_bounds__(256) pack_strided_kernel(ExpView ev, int64_t nterms, const __grid_constant__ Plan plan,
                                                           K* __restrict__ keys, Control* ctl, int hd)
{
    __shared__ uint32_t sh[kRadix];
    BlockHist bh;
    if (hd >= 0) { bh.init(sh); __syncthreads(); }
    const int dpos = plan.digit_pos[hd >= 0 ? hd : 0];
    const uint32_t dmask = (1u << plan.digit_bits[hd >= 0 ? hd : 0]) - 1u;
    bool bad = false;
    for (int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; t < nterms; t += (int64_t)gridDim.x * blockDim.x) {
        K key;
        key_zero(key);
        for (int v = 0; v < plan.nvars; ++v)
            pack_field(key, load_exp(ev.base, ev.exp_bytes, t * ev.term_stride + (int64_t)v * ev.var_stride), v, plan, bad);
        keys[t] = key;
        if (hd >= 0) bh.add(key_digit(key, dpos, dmask));
    }
    if (bad) atomicMax(&ctl->status, (int)POLYLAB_ERR_EXPONENT_RANGE);
    if (hd >= 0) { __syncthreads(); bh.flush(ctl->hist[hd]); }
}

template <typename K, int ES>
static void launch_pack_rows_es(int wb, unsigned blocks, const ExpView& ev, int64_t nterms, const Plan& plan, K* keys,
                                Control* ctl, int hd, cudaStream_t stream)
{
    const uint8_t* base = (const uint8_t*)ev.base;
    if (wb == 16) pack_rows_kernel<K, ES, 16><<<blocks, 256, 0, stream>>>(base, nterms, plan, keys, ctl, hd);
    else if (wb == 4) pack_rows_kernel<K, ES, 4><<<blocks, 256, 0, stream>>>(base, nterms, plan, keys, ctl, hd);
    else if (ES <= 2 && wb == 2) pack_rows_kernel<K, ES, (ES <= 2 ? 2 : 4)><<<blocks, 256, 0, stream>>>(base, nterms, plan, keys, ctl, hd);
    else pack_rows_kernel<K, ES, (ES == 1 ? 1 : ES)><<<blocks, 256, 0, stream>>>(base, nterms, plan, keys, ctl, hd);
}

template <typename K>
static int launch_pack_t(const ExpView& ev, int64_t nterms, const Plan& plan, K* keys, Control* ctl, int hd,
                         cudaStream_t stream)
{
    if (nterms <= 0) return 0;
    int64_t blocks = (nterms + 256 * 4 - 1) / (256 * 4);       // >= 4 rows per thread once the grid saturates
    if (blocks > sm_count() * 32) blocks = sm_count() * 32;
    if (blocks < 1) blocks = 1;
    if (ev.row_major_contiguous && (plan.nvars * ev.exp_bytes) % 16 != 0) {
        const int rb = plan.nvars * ev.exp_bytes;
        int tile_rows = 16384 / rb;                              // at most 16 KB of rows per tile, two tiles in shared memory
        tile_rows = tile_rows > 1024 ? 1024 : tile_rows < 32 ? 32 : tile_rows / 32 * 32;
        int64_t sblocks = (nterms + tile_rows - 1) / tile_rows;
        if (sblocks > sm_count() * 6) sblocks = sm_count() * 6;
        const size_t smem = 2 * (((size_t)tile_rows * rb + 16 + 15) & ~(size_t)15);
        const uint8_t* base = (const uint8_t*)ev.base;
        if (ev.exp_bytes == 1) pack_rows_staged_kernel<K, 1><<<(unsigned)sblocks, 256, smem, stream>>>(base, nterms, tile_rows, plan, keys, ctl, hd);
        else if (ev.exp_bytes == 2) pack_rows_staged_kernel<K, 2><<<(unsigned)sblocks, 256, smem, stream>>>(base, nterms, tile_rows, plan, keys, ctl, hd);
        else pack_rows_staged_kernel<K, 4><<<(unsigned)sblocks, 256, smem, stream>>>(base, nterms, tile_rows, plan, keys, ctl, hd);
    } else if (ev.row_major_contiguous) {
        const int rb = plan.nvars * ev.exp_bytes;
        const int wb = (rb % 16 == 0) ? 16 : (rb % 4 == 0) ? 4 : (rb % 2 == 0) ? 2 : 1;
        if (ev.exp_bytes == 1) launch_pack_rows_es<K, 1>(wb, (unsigned)blocks, ev, nterms, plan, keys, ctl, hd, stream);
        else if (ev.exp_bytes == 2) launch_pack_rows_es<K, 2>(wb, (unsigned)blocks, ev, nterms, plan, keys, ctl, hd, stream);
        else launch_pack_rows_es<K, 4>(wb, (unsigned)blocks, ev, nterms, plan, keys, ctl, hd, stream);
    } else {
        pack_strided_kernel<K><<<(unsigned)blocks, 256, 0, stream>>>(ev, nterms, plan, keys, ctl, hd);
    }
    return 1;
}

int launch_pack(const ExpView& ev, int64_t nterms, const Plan& plan, void* keys, Control* ctl, int hd,
                cudaStream_t stream)
{
    if (plan.key_bytes == 8) return launch_pack_t<uint64_t>(ev, nterms, plan, (uint64_t*)keys, ctl, hd, stream);
    if (plan.key_bytes == 16) return launch_pack_t<Key128>(ev, nterms, plan, (Key128*)keys, ctl, hd, stream);
    return launch_pack_t<Key256>(ev, nterms, plan, (Key256*)keys, ctl, hd, stream);
}

int launch_pack_hilo(const ExpView& ev, int64_t nterms, const Plan& plan, uint64_t* out_hilo, Control* ctl,
                     cudaStream_t stream)
{
    return launch_pack_t<Key128>(ev, nterms, plan, (Key128*)out_hilo, ctl, -1, stream);   // Key128 is (hi, lo)
}

// Histogram of digit `hd` over already packed keys into ctl->hist[hd] (used when the bucket path is rejected after
// S1 and the LSD passes need the histogram of digit 0 instead).
template <typename K>
__global__ void __launch_bounds__(256) key_hist_kernel(const K* __restrict__ keys, int64_t n, int dpos, uint32_t dmask,
                                                       uint32_t* hist)
{
    __shared__ uint32_t sh[kRadix];
    BlockHist bh;
    bh.init(sh);
    __syncthreads();
    for (int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; t < n; t += (int64_t)gridDim.x * blockDim.x)
        bh.add(key_digit(keys[t], dpos, dmask));
    __syncthreads();
    bh.flush(hist);
}

int launch_key_hist(const Plan& plan, int hd, int64_t n, const void* keys, Control* ctl, cudaStream_t stream)
{
    if (n <= 0 || hd < 0 || hd >= plan.npasses) return 0;
    int64_t blocks = (n + 256 * 8 - 1) / (256 * 8);
    if (blocks > sm_count() * 16) blocks = sm_count() * 16;
    const int dpos = plan.digit_pos[hd];
    const uint32_t dmask = (1u << plan.digit_bits[hd]) - 1u;
    if (plan.key_bytes == 8) key_hist_kernel<uint64_t><<<(unsigned)blocks, 256, 0, stream>>>((const uint64_t*)keys, n, dpos, dmask, ctl->hist[hd]);
    else if (plan.key_bytes == 16) key_hist_kernel<Key128><<<(unsigned)blocks, 256, 0, stream>>>((const Key128*)keys, n, dpos, dmask, ctl->hist[hd]);
    else key_hist_kernel<Key256><<<(unsigned)blocks, 256, 0, stream>>>((const Key256*)keys, n, dpos, dmask, ctl->hist[hd]);
    return 1;
}

// Histogram of plan digit `hd` straight from contiguous exponent rows of 8 or 16 bytes, without building the keys:
// only the variables whose fields overlap the digit contribute (at most 8).  Used when S1 is fused into the first
// radix pass of the bucket path (sort.cu), which needs this histogram before it can scatter.
struct DigitParts {
    int n;
    uint8_t var[8];
    int8_t lshift[8];       // contribution = min(e, emax) << lshift (lshift >= 0) or >> -lshift, then & mask
    uint32_t emax[8];       // the variable's bound: the fused pass clamps an out-of-range exponent the same way
    uint32_t mask;
};

template <int RB, int ES>
__global__ void __launch_bounds__(256) row_hist_kernel(const uint8_t* __restrict__ base, int64_t nterms, DigitParts dp,
                                                       uint32_t* hist)
{
    __shared__ uint32_t sh[kRadix];
    BlockHist bh;
    bh.init(sh);
    __syncthreads();
    // four rows per thread and iteration: all four loads are issued before the first is used
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    for (int64_t t0 = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; t0 < nterms; t0 += 4 * stride) {
        uint32_t w[4][RB / 4];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const int64_t t = t0 + u * stride;
            if (t < nterms) {
                if (RB == 16) {
                    const uint4 q = __ldg((const uint4*)(base + t * RB));
                    w[u][0] = q.x; w[u][RB / 4 > 1 ? 1 : 0] = q.y; w[u][RB / 4 > 2 ? 2 : 0] = q.z; w[u][RB / 4 > 3 ? 3 : 0] = q.w;
                } else {
                    const uint2 q = __ldg((const uint2*)(base + t * RB));
                    w[u][0] = q.x; w[u][RB / 4 > 1 ? 1 : 0] = q.y;
                }
            }
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            if (t0 + u * stride >= nterms) break;
            uint32_t d = 0;
            for (int i = 0; i < dp.n; ++i) {
                const int v = dp.var[i];
                uint32_t e;
                const int wi = ES == 4 ? v : ES == 2 ? (v >> 1) : (v >> 2);      // selects, not a dynamically indexed array
                uint32_t x = w[u][0];
                if (RB / 4 > 1 && wi == 1) x = w[u][RB / 4 > 1 ? 1 : 0];
                if (RB / 4 > 2 && wi == 2) x = w[u][RB / 4 > 2 ? 2 : 0];
                if (RB / 4 > 3 && wi == 3) x = w[u][RB / 4 > 3 ? 3 : 0];
                if (ES == 4) e = x;
                else if (ES == 2) e = (x >> (16 * (v & 1))) & 0xffffu;
                else e = (x >> (8 * (v & 3))) & 0xffu;
                e = min(e, dp.emax[i]);
                const int ls = dp.lshift[i];
                d |= ls >= 0 ? (e << ls) : (e >> -ls);
            }
            bh.add(d & dp.mask);
        }
    }
    __syncthreads();
    bh.flush(hist);
}

// The same histogram over a SAMPLE of the rows: block b reads rows [b * seg_stride, b * seg_stride + seg_rows).  The first
// prefix pass of the bucket path then lays its bins out with slack sized from this estimate (api.cu, sort.cu: slack bins)
// instead of waiting for a sweep over every row.
template <int RB, int ES>
__global__ void __launch_bounds__(256) row_hist_sample_kernel(const uint8_t* __restrict__ base, int64_t nterms, int64_t seg_stride,
                                                              int seg_rows, DigitParts dp, uint32_t* hist)
{
    __shared__ uint32_t sh[kRadix];
    BlockHist bh;
    bh.init(sh);
    __syncthreads();
    const int64_t t0 = (int64_t)blockIdx.x * seg_stride, t1 = min(nterms, t0 + seg_rows);
    for (int64_t t = t0 + threadIdx.x; t < t1; t += blockDim.x) {
        uint32_t w[RB / 4];
        if (RB == 16) {
            const uint4 q = __ldg((const uint4*)(base + t * RB));
            w[0] = q.x; w[RB / 4 > 1 ? 1 : 0] = q.y; w[RB / 4 > 2 ? 2 : 0] = q.z; w[RB / 4 > 3 ? 3 : 0] = q.w;
        } else {
            const uint2 q = __ldg((const uint2*)(base + t * RB));
            w[0] = q.x; w[RB / 4 > 1 ? 1 : 0] = q.y;
        }
        uint32_t d = 0;
        for (int i = 0; i < dp.n; ++i) {
            const int v = dp.var[i];
            const int wi = ES == 4 ? v : ES == 2 ? (v >> 1) : (v >> 2);
            uint32_t x = w[0];
            if (RB / 4 > 1 && wi == 1) x = w[RB / 4 > 1 ? 1 : 0];
            if (RB / 4 > 2 && wi == 2) x = w[RB / 4 > 2 ? 2 : 0];
            if (RB / 4 > 3 && wi == 3) x = w[RB / 4 > 3 ? 3 : 0];
            uint32_t e;
            if (ES == 4) e = x;
            else if (ES == 2) e = (x >> (16 * (v & 1))) & 0xffffu;
            else e = (x >> (8 * (v & 3))) & 0xffu;
            e = min(e, dp.emax[i]);
            const int ls = dp.lshift[i];
            d |= ls >= 0 ? (e << ls) : (e >> -ls);
        }
        bh.add(d & dp.mask);
    }
    __syncthreads();
    bh.flush(hist);
}

// Slack-bin capacities on the device, for calls that must not synchronise (POLYLAB_FLAG_DEVICE_COUNT): the same rule as the
// host applies in api.cu -- estimate scaled to N, plus 7 sigma of the sample count, plus 8 -- written as the first prefix
// digit's "histogram" and as the capacities the second pass reads.  If the sample is empty or the capacities do not fit the
// buffer, every capacity is 0: the pass then writes nothing and raises slack_overflow (-> POLYLAB_ERR_RETRY).
__global__ void __launch_bounds__(kRadix) slack_caps_kernel(const uint32_t* __restrict__ est, uint32_t n, uint64_t capacity,
                                                            uint32_t* __restrict__ hist, uint32_t* __restrict__ cap)
{
    __shared__ double part[kRadix / 32];
    __shared__ double bcast;
    const unsigned b = threadIdx.x, lane = b & 31u, warp = b >> 5;
    auto block_sum = [&](double x) -> double {
        for (int o = 16; o; o >>= 1) x += __shfl_xor_sync(kFullMask, x, o);
        __syncthreads();
        if (lane == 0) part[warp] = x;
        __syncthreads();
        if (b == 0) { double t = 0.0; for (int w = 0; w < kRadix / 32; ++w) t += part[w]; bcast = t; }
        __syncthreads();
        return bcast;
    };
    const double c = (double)est[b];
    const double ssum = block_sum(c);
    double cb = 0.0;
    if (ssum > 0.0) cb = ceil((double)n / ssum * (c + 7.0 * sqrt(c + 1.0) + 8.0) / 16.0) * 16.0;   // multiples of 16 records
    const double total = block_sum(cb);
    const uint32_t out = (ssum > 0.0 && total <= (double)capacity && cb < 4.0e9) ? (uint32_t)cb : 0u;
    const bool any_zero = __syncthreads_or(out == 0u ? 1 : 0) != 0;       // one unusable capacity voids all of them
    hist[b] = any_zero ? 0u : out;
    cap[b] = any_zero ? 0u : out;
}

int launch_slack_caps(const uint32_t* est, int64_t n, int64_t capacity, uint32_t* hist, uint32_t* cap, cudaStream_t stream)
{
    slack_caps_kernel<<<1, kRadix, 0, stream>>>(est, (uint32_t)n, (uint64_t)capacity, hist, cap);
    return 1;
}

bool rows_fusable(const ExpView& ev, int nvars)
{
    const int rb = nvars * ev.exp_bytes;
    return ev.row_major_contiguous && (rb == 8 || rb == 16);
}

static DigitParts digit_parts(const Plan& plan, int hd);

int launch_row_hist_sample(const ExpView& ev, int64_t nterms, const Plan& plan, int hd, uint32_t* est, int nsegs, int seg_rows, cudaStream_t stream)
{
    if (nterms <= 0 || !rows_fusable(ev, plan.nvars) || hd < 0 || hd >= plan.npasses || nsegs < 1) return 0;
    const DigitParts dp = digit_parts(plan, hd);
    const int rb = plan.nvars * ev.exp_bytes;
    const uint8_t* base = (const uint8_t*)ev.base;
    const int64_t seg_stride = nterms / nsegs > 0 ? nterms / nsegs : 1;
#define POLYLAB_RHS(RB, ES) row_hist_sample_kernel<RB, ES><<<(unsigned)nsegs, 256, 0, stream>>>(base, nterms, seg_stride, seg_rows, dp, est)
    if (rb == 16) { if (ev.exp_bytes == 1) POLYLAB_RHS(16, 1); else if (ev.exp_bytes == 2) POLYLAB_RHS(16, 2); else POLYLAB_RHS(16, 4); }
    else { if (ev.exp_bytes == 1) POLYLAB_RHS(8, 1); else if (ev.exp_bytes == 2) POLYLAB_RHS(8, 2); else POLYLAB_RHS(8, 4); }
#undef POLYLAB_RHS
    return 1;
}

static DigitParts digit_parts(const Plan& plan, int hd)
{
    DigitParts dp;
    dp.n = 0;
    const int dpos = plan.digit_pos[hd], dbits = plan.digit_bits[hd];
    dp.mask = (1u << dbits) - 1u;
    for (int v = 0; v < plan.nvars; ++v) {
        const int lo = plan.shift[v], hi = lo + plan.width[v];
        if (plan.width[v] == 0 || hi <= dpos || lo >= dpos + dbits) continue;
        dp.var[dp.n] = (uint8_t)v;
        dp.lshift[dp.n] = (int8_t)(lo - dpos);
        dp.emax[dp.n] = plan.bound[v];
        ++dp.n;
    }
    return dp;
}

int launch_row_hist(const ExpView& ev, int64_t nterms, const Plan& plan, int hd, Control* ctl, cudaStream_t stream)
{
    if (nterms <= 0 || !rows_fusable(ev, plan.nvars) || hd < 0 || hd >= plan.npasses) return 0;
    DigitParts dp;
    dp.n = 0;
    const int dpos = plan.digit_pos[hd], dbits = plan.digit_bits[hd];
    dp.mask = (1u << dbits) - 1u;
    for (int v = 0; v < plan.nvars; ++v) {
        const int lo = plan.shift[v], hi = lo + plan.width[v];
        if (plan.width[v] == 0 || hi <= dpos || lo >= dpos + dbits) continue;
        dp.var[dp.n] = (uint8_t)v;
        dp.lshift[dp.n] = (int8_t)(lo - dpos);
        dp.emax[dp.n] = plan.bound[v];
        ++dp.n;
    }
    const int rb = plan.nvars * ev.exp_bytes;
    int64_t blocks = (nterms + 256 * 8 - 1) / (256 * 8);
    if (blocks > sm_count() * 16) blocks = sm_count() * 16;
    const uint8_t* base = (const uint8_t*)ev.base;
    uint32_t* hist = ctl->hist[hd];
#define POLYLAB_RH(RB, ES) row_hist_kernel<RB, ES><<<(unsigned)blocks, 256, 0, stream>>>(base, nterms, dp, hist)
    if (rb == 16) { if (ev.exp_bytes == 1) POLYLAB_RH(16, 1); else if (ev.exp_bytes == 2) POLYLAB_RH(16, 2); else POLYLAB_RH(16, 4); }
    else { if (ev.exp_bytes == 1) POLYLAB_RH(8, 1); else if (ev.exp_bytes == 2) POLYLAB_RH(8, 2); else POLYLAB_RH(8, 4); }
#undef POLYLAB_RH
    return 1;
}

__global__ void __launch_bounds__(256) widen_kernel(const float* __restrict__ in, double* __restrict__ out, int64_t n)
{
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) out[i] = (double)in[i];
}

int launch_widen(const void* in_f32, double* out, int64_t n, cudaStream_t stream)
{
    if (n <= 0) return 0;
    int64_t blocks = (n + 1023) / 1024;
    if (blocks > sm_count() * 16) blocks = sm_count() * 16;
    widen_kernel<<<(unsigned)blocks, 256, 0, stream>>>((const float*)in_f32, out, n);
    return 1;
}

// ----------------------------------------------------------------------------------------------- X1

template <typename K>
__global__ void __launch_bounds__(256) expand_packed_kernel(const K* __restrict__ ka, CoefIn ca,
                                                            uint32_t na, const K* __restrict__ kb,
                                                            CoefIn cb, uint32_t nb,
                                                            K* __restrict__ keys, double* __restrict__ coefs, int dpos,
                                                            uint32_t dmask, uint32_t* hist)
{
    constexpr int ITEMS = 4;
    __shared__ uint32_t sh[kRadix];
    BlockHist bh;
    bh.init(sh);
    __syncthreads();
    const uint32_t n = na * nb;                                   // < 2^30, checked on the host
    const uint32_t q0 = blockIdx.x * (256u * ITEMS) + threadIdx.x;
#pragma unroll
    for (int k = 0; k < ITEMS; ++k) {
        const uint32_t q = q0 + k * 256u;
        if (q < n) {
            const uint32_t i = q / nb, j = q - i * nb;
            const K key = key_add(ka[i], kb[j]);
            keys[q] = key;
            coefs[q] = __dmul_rn(ca[i], cb[j]);                   // one IEEE multiplication, never contracted
            bh.add(key_digit(key, dpos, dmask));
        }
    }
    __syncthreads();
    bh.flush(hist);
}

int launch_expand_packed(const void* ka, CoefIn ca, int64_t na, const void* kb, CoefIn cb, int64_t nb,
                         const Plan& plan, void* keys, double* coefs, Control* ctl, int hd, cudaStream_t stream)
{
    const int64_t n = na * nb;
    if (n <= 0) return 0;
    const unsigned blocks = (unsigned)((n + 1023) / 1024);
    if (hd < 0 || hd >= plan.npasses) hd = 0;
    const int dpos = plan.npasses ? plan.digit_pos[hd] : 0;
    const uint32_t dmask = plan.npasses ? (1u << plan.digit_bits[hd]) - 1u : 0u;
    if (plan.key_bytes == 8)
        expand_packed_kernel<uint64_t><<<blocks, 256, 0, stream>>>((const uint64_t*)ka, ca, (uint32_t)na, (const uint64_t*)kb,
                                                                   cb, (uint32_t)nb, (uint64_t*)keys, coefs, dpos, dmask, ctl->hist[hd]);
    else if (plan.key_bytes == 16)
        expand_packed_kernel<Key128><<<blocks, 256, 0, stream>>>((const Key128*)ka, ca, (uint32_t)na, (const Key128*)kb, cb,
                                                                 (uint32_t)nb, (Key128*)keys, coefs, dpos, dmask, ctl->hist[hd]);
    else
        expand_packed_kernel<Key256><<<blocks, 256, 0, stream>>>((const Key256*)ka, ca, (uint32_t)na, (const Key256*)kb, cb,
                                                                 (uint32_t)nb, (Key256*)keys, coefs, dpos, dmask, ctl->hist[hd]);
    return 1;
}

// Histogram of one digit over all products, nothing stored (X1 fused into the first radix pass needs it up front).
template <typename K>
__global__ void __launch_bounds__(256) expand_hist_kernel(const K* __restrict__ ka, uint32_t na, const K* __restrict__ kb,
                                                          uint32_t nb, int dpos, uint32_t dmask, uint32_t* hist)
{
    __shared__ uint32_t sh[kRadix];
    BlockHist bh;
    bh.init(sh);
    __syncthreads();
    const uint32_t n = na * nb;
    for (uint32_t q = blockIdx.x * blockDim.x + threadIdx.x; q < n; q += gridDim.x * blockDim.x) {
        const uint32_t i = q / nb, j = q - i * nb;
        bh.add(key_digit(key_add(ka[i], kb[j]), dpos, dmask));
    }
    __syncthreads();
    bh.flush(hist);
}

int launch_expand_hist(const ExpandSrc& xs, const Plan& plan, int hd, Control* ctl, cudaStream_t stream)
{
    const int64_t n = xs.na * xs.nb;
    if (n <= 0 || hd < 0 || hd >= plan.npasses) return 0;
    int64_t blocks = (n + 256 * 8 - 1) / (256 * 8);
    if (blocks > sm_count() * 16) blocks = sm_count() * 16;
    const int dpos = plan.digit_pos[hd];
    const uint32_t dmask = (1u << plan.digit_bits[hd]) - 1u;
    if (plan.key_bytes == 8)
        expand_hist_kernel<uint64_t><<<(unsigned)blocks, 256, 0, stream>>>((const uint64_t*)xs.ka, (uint32_t)xs.na, (const uint64_t*)xs.kb,
                                                                          (uint32_t)xs.nb, dpos, dmask, ctl->hist[hd]);
    else if (plan.key_bytes == 16)
        expand_hist_kernel<Key128><<<(unsigned)blocks, 256, 0, stream>>>((const Key128*)xs.ka, (uint32_t)xs.na, (const Key128*)xs.kb,
                                                                        (uint32_t)xs.nb, dpos, dmask, ctl->hist[hd]);
    else
        expand_hist_kernel<Key256><<<(unsigned)blocks, 256, 0, stream>>>((const Key256*)xs.ka, (uint32_t)xs.na, (const Key256*)xs.kb,
                                                                        (uint32_t)xs.nb, dpos, dmask, ctl->hist[hd]);
    return 1;
}

// Raw product in (coef, exps) form, no keys: polylab_expand (reading A10).
__global__ void __launch_bounds__(256) expand_raw_kernel(ExpView ea, CoefIn ca, uint32_t na,
                                                         ExpView eb, CoefIn cb, uint32_t nb,
                                                         int nvars, CoefOut out_coef, void* out_exps,
                                                         int32_t* status)
{
    const uint32_t n = na * nb;
    const uint32_t emax = ea.exp_bytes == 1 ? 0xffu : ea.exp_bytes == 2 ? 0xffffu : 0xffffffffu;
    bool bad = false;
    for (uint32_t q = blockIdx.x * blockDim.x + threadIdx.x; q < n; q += gridDim.x * blockDim.x) {
        const uint32_t i = q / nb, j = q - i * nb;
        out_coef.store(q, __dmul_rn(ca[i], cb[j]));
        for (int v = 0; v < nvars; ++v) {
            const uint32_t x = load_exp(ea.base, ea.exp_bytes, (int64_t)i * ea.term_stride + (int64_t)v * ea.var_stride);
            const uint32_t y = load_exp(eb.base, eb.exp_bytes, (int64_t)j * eb.term_stride + (int64_t)v * eb.var_stride);
            const uint32_t s = x + y;
            bad |= (s < x) || (s > emax);
            store_exp(out_exps, ea.exp_bytes, (int64_t)q * nvars + v, s);
        }
    }
    if (bad) atomicMax(status, (int)POLYLAB_ERR_EXPONENT_RANGE);
}

int launch_expand_raw(const ExpView& ea, CoefIn ca, int64_t na, const ExpView& eb, CoefIn cb, int64_t nb,
                      int nvars, CoefOut out_coef, void* out_exps, Control* ctl_status, cudaStream_t stream)
{
    const int64_t n = na * nb;
    if (n <= 0) return 0;
    int64_t blocks = (n + 255) / 256;
    if (blocks > sm_count() * 32) blocks = sm_count() * 32;
    expand_raw_kernel<<<(unsigned)blocks, 256, 0, stream>>>(ea, ca, (uint32_t)na, eb, cb, (uint32_t)nb, nvars, out_coef,
                                                            out_exps, &ctl_status->status);
    return 1;
}

}  // namespace polylab
