// sph_sort.cu -- step a2 and the scans of a5: a stable least-significant-digit radix sort of (key, value)
// pairs and an inclusive scan with stream compaction, written for this path (no library call).
//
// The paper keeps its particles in space-filling-curve order (§1); here that order is
// produced on the device by sorting the 48-bit Morton keys.  One pass per 8-bit digit, three kernels per
// pass -- (1) per-tile digit histograms, (2) an exclusive scan of the histogram matrix, (3) a scatter that
// ranks the tile's keys stably (warp-wide ballots on the digit bits), orders the tile in shared memory and
// writes every digit's run of the tile to its place as one contiguous, coalesced piece.  HBM-bound:
// a pass reads the keys twice and the values once and writes both once (32 bytes per record).
#include "sph_internal.cuh"

namespace {

#define SORT_THREADS 256
#define SORT_WARPS (SORT_THREADS / 32)
#define SORT_ROUNDS 8                               // keys per thread (16 x 2 blocks/SM and 12 x 3 measured slower)
#define SORT_MINB 4                                 // resident blocks per SM the scatter kernel is compiled for
#define SORT_TILE (SORT_THREADS * SORT_ROUNDS)      // keys per block
#define SORT_RADIX 256
#define FULL 0xffffffffu

__device__ __forceinline__ unsigned lane_lt()
{
    unsigned m;
    asm("mov.u32 %0, %%lanemask_lt;" : "=r"(m));
    return m;
}

template <typename K>
__device__ __forceinline__ uint32_t digit_of(K key, int shift, uint32_t mask)
{
    return (uint32_t)(key >> shift) & mask;
}

// (1) histogram of the pass's digit over every tile: hist[d * tiles + tile]
template <typename K>
__global__ void __launch_bounds__(SORT_THREADS) k_sort_hist(const K *__restrict__ keys, uint32_t n, int shift, uint32_t mask,
                                                            uint32_t *__restrict__ hist, uint32_t tiles)
{
    __shared__ uint32_t sh[SORT_RADIX];
    const uint32_t tile = blockIdx.x, t0 = tile * SORT_TILE;
    sh[threadIdx.x] = 0;
    __syncthreads();
#pragma unroll 4
    for (int r = 0; r < SORT_ROUNDS; r++) {
        const uint32_t i = t0 + r * SORT_THREADS + threadIdx.x;
        if (i < n) atomicAdd(&sh[digit_of(keys[i], shift, mask)], 1u);
    }
    __syncthreads();
    hist[threadIdx.x * tiles + tile] = sh[threadIdx.x];
}

// (2) every digit's row of the histogram matrix becomes its exclusive prefix over the tiles (block d scans row d);
// the last block to finish turns the 256 row totals into base[d] = number of keys with a smaller digit.
// tot: 256 row totals followed by one counter that wraps back to 0 by itself (atomicInc).
__global__ void __launch_bounds__(SORT_THREADS) k_sort_scan(uint32_t *__restrict__ hist, uint32_t tiles, uint32_t *__restrict__ base,
                                                            uint32_t *__restrict__ tot)
{
    __shared__ uint32_t wt[SORT_WARPS];
    __shared__ bool last;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    uint32_t *row = hist + (size_t)blockIdx.x * tiles;
    // warp w owns a contiguous piece of the row and walks it 32 entries at a time (coalesced): first its sum ...
    const uint32_t per = ((tiles + SORT_WARPS - 1) / SORT_WARPS + 31u) & ~31u, i0 = warp * per, i1 = min(i0 + per, tiles);
    uint32_t s = 0;
    for (uint32_t i = i0 + lane; i < i1; i += 32) s += row[i];
    s = __reduce_add_sync(FULL, s);
    if (lane == 0) wt[warp] = s;
    __syncthreads();
    uint32_t run = 0, all = 0;
#pragma unroll
    for (int w = 0; w < SORT_WARPS; w++) {
        run += w < warp ? wt[w] : 0u;
        all += wt[w];
    }
    // ... then the exclusive prefix, chunk by chunk with a running carry
    for (uint32_t b = i0; b < i1; b += 32) {
        const uint32_t i = b + lane;
        const uint32_t v = i < i1 ? row[i] : 0u;
        uint32_t inc = v;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t t = __shfl_up_sync(FULL, inc, o);
            if (lane >= o) inc += t;
        }
        if (i < i1) row[i] = run + inc - v;
        run += __shfl_sync(FULL, inc, 31);
    }
    if (tid == 0) {
        tot[blockIdx.x] = all;
        __threadfence();
        last = atomicInc(&tot[SORT_RADIX], SORT_RADIX - 1) == SORT_RADIX - 1;
    }
    __syncthreads();
    if (!last) return;
    __threadfence();
    // exclusive scan of the 256 row totals (thread d holds total d)
    const uint32_t v = reinterpret_cast<volatile uint32_t *>(tot)[tid];
    uint32_t in2 = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const uint32_t t = __shfl_up_sync(FULL, in2, o);
        if (lane >= o) in2 += t;
    }
    __syncthreads();
    if (lane == 31) wt[warp] = in2;
    __syncthreads();
    uint32_t wb = 0;
#pragma unroll
    for (int w = 0; w < SORT_WARPS; w++) wb += w < warp ? wt[w] : 0u;
    base[tid] = wb + in2 - v;
}

// (3) stable scatter of one tile
template <typename K, bool HAS_VAL>
struct SortSmem {
    uint32_t wcnt[SORT_WARPS][SORT_RADIX]; // per warp: digit counts, then exclusive prefix over the warps
    uint32_t toff[SORT_RADIX];             // first position of the digit's run in the ordered tile
    uint32_t gpos[SORT_RADIX];             // global position of that run minus toff
    K keys[SORT_TILE];
    uint32_t vals[HAS_VAL ? SORT_TILE : 1];
};

template <typename K, bool HAS_VAL>
__global__ void __launch_bounds__(SORT_THREADS, SORT_MINB) k_sort_scatter(const K *__restrict__ kin, const uint32_t *__restrict__ vin,
                                                               K *__restrict__ kout, uint32_t *__restrict__ vout, uint32_t n,
                                                               int shift, uint32_t mask, const uint32_t *__restrict__ hist,
                                                               const uint32_t *__restrict__ base, uint32_t tiles)
{
    extern __shared__ __align__(16) unsigned char raw[];
    SortSmem<K, HAS_VAL> &S = *reinterpret_cast<SortSmem<K, HAS_VAL> *>(raw);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const uint32_t tile = blockIdx.x, t0 = tile * SORT_TILE;
    const uint32_t tn = min((uint32_t)SORT_TILE, n - t0);
    // rank inside the warp's chunk: the chunk is SORT_ROUNDS consecutive rows of 32 keys, row by row, lane by lane --
    // the order of the input, so equal digits keep their order (stable).  (All global loads of the block are issued
    // first, so that their latency overlaps the clearing of the counters.)
    K key[SORT_ROUNDS];
    uint32_t val[SORT_ROUNDS], rank[SORT_ROUNDS];
    const uint32_t w0 = warp * (32 * SORT_ROUNDS);
#pragma unroll
    for (int r = 0; r < SORT_ROUNDS; r++) {
        const uint32_t o = w0 + r * 32 + lane;
        const bool valid = o < tn;
        key[r] = valid ? kin[t0 + o] : (K)0;
        if (HAS_VAL) val[r] = valid ? vin[t0 + o] : 0u;
    }
    const uint32_t gbase = base[tid] + hist[(size_t)tid * tiles + tile]; // where this tile's run of digit tid starts
    for (int i = tid; i < SORT_WARPS * SORT_RADIX; i += SORT_THREADS) (&S.wcnt[0][0])[i] = 0;
    __syncthreads();
    // the lanes holding the same digit, from eight ballots (one per digit bit) -- measured faster than __match_any_sync
    // here (index build 1.54 instead of 1.63 ms at 10^7 keys: the match instruction's latency dominated the kernel);
    // all rounds' masks are computed before the first counter update, which is ordered through shared memory
    unsigned mm[SORT_ROUNDS];
#pragma unroll
    for (int r = 0; r < SORT_ROUNDS; r++) {
        const bool valid = w0 + r * 32 + lane < tn;
        const uint32_t d = valid ? digit_of(key[r], shift, mask) : 0u;
        const unsigned vm = __ballot_sync(FULL, valid);
        unsigned m = valid ? vm : ~vm; // (invalid lanes match one another only)
#pragma unroll
        for (int b = 0; b < 8; b++) {
            const bool bit = (d >> b) & 1u;
            const unsigned bb = __ballot_sync(FULL, bit);
            m &= bit ? bb : ~bb;
        }
        mm[r] = m;
    }
#pragma unroll
    for (int r = 0; r < SORT_ROUNDS; r++) {
        const bool valid = w0 + r * 32 + lane < tn;
        const uint32_t d = valid ? digit_of(key[r], shift, mask) : 0xffffffffu;
        const unsigned m = mm[r];
        const int leader = __ffs(m) - 1;
        uint32_t old = 0;
        if (lane == leader && valid) {
            old = S.wcnt[warp][d];
            S.wcnt[warp][d] = old + __popc(m);
        }
        old = __shfl_sync(FULL, old, leader);
        rank[r] = old + __popc(m & lane_lt());
        __syncwarp();
    }
    __syncthreads();
    // digit d (thread d): exclusive prefix over the warps, tile total, then the runs' offsets in the ordered tile
    {
        uint32_t acc = 0;
#pragma unroll
        for (int w = 0; w < SORT_WARPS; w++) {
            const uint32_t t = S.wcnt[w][tid];
            S.wcnt[w][tid] = acc;
            acc += t;
        }
        // exclusive scan of the 256 tile totals: warp scan + the 8 warp totals through toff[0..7] (reused below)
        uint32_t inc = acc;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t t = __shfl_up_sync(FULL, inc, o);
            if (lane >= o) inc += t;
        }
        __shared__ uint32_t wtot[SORT_WARPS];
        if (lane == 31) wtot[warp] = inc;
        __syncthreads();
        uint32_t wb = 0;
#pragma unroll
        for (int w = 0; w < SORT_WARPS; w++) wb += w < warp ? wtot[w] : 0u;
        const uint32_t off = wb + inc - acc;
        S.toff[tid] = off;
        S.gpos[tid] = gbase - off;
    }
    __syncthreads();
    // order the tile in shared memory
#pragma unroll
    for (int r = 0; r < SORT_ROUNDS; r++) {
        if (w0 + r * 32 + lane < tn) {
            const uint32_t d = digit_of(key[r], shift, mask);
            const uint32_t p = S.toff[d] + S.wcnt[warp][d] + rank[r];
            S.keys[p] = key[r];
            if (HAS_VAL) S.vals[p] = val[r];
        }
    }
    __syncthreads();
    // every digit's run of the tile goes to its place as one contiguous piece
    for (uint32_t i = tid; i < tn; i += SORT_THREADS) {
        const K k = S.keys[i];
        const uint32_t g = S.gpos[digit_of(k, shift, mask)] + i;
        kout[g] = k;
        if (HAS_VAL) vout[g] = S.vals[i];
    }
}

// ---- inclusive scan of 0/1 marks with compaction -----------------------------------------------------------------
#define SCAN_THREADS 256
#define SCAN_ITEMS 16
#define SCAN_TILE (SCAN_THREADS * SCAN_ITEMS)

__device__ __forceinline__ uint32_t block_exclusive(uint32_t v, uint32_t *total)
{
    __shared__ uint32_t wt[SCAN_THREADS / 32];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    uint32_t inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const uint32_t t = __shfl_up_sync(FULL, inc, o);
        if (lane >= o) inc += t;
    }
    if (lane == 31) wt[warp] = inc;
    __syncthreads();
    uint32_t wb = 0, tot = 0;
#pragma unroll
    for (int w = 0; w < SCAN_THREADS / 32; w++) {
        wb += w < warp ? wt[w] : 0u;
        tot += wt[w];
    }
    *total = tot;
    __syncthreads();
    return wb + inc - v;
}

__global__ void __launch_bounds__(SCAN_THREADS) k_scan_sums(const uint32_t *__restrict__ mark, uint32_t n, uint32_t *__restrict__ bsum)
{
    const uint32_t i0 = blockIdx.x * SCAN_TILE + threadIdx.x * SCAN_ITEMS;
    uint32_t s = 0;
#pragma unroll
    for (int k = 0; k < SCAN_ITEMS; k++) s += i0 + k < n ? mark[i0 + k] : 0u;
    uint32_t tot;
    block_exclusive(s, &tot);
    if (threadIdx.x == 0) bsum[blockIdx.x] = tot;
}

// exclusive scan of the block sums in place (one block), grand total to *count
__global__ void __launch_bounds__(SCAN_THREADS) k_scan_bsums(uint32_t *__restrict__ bsum, uint32_t nb, unsigned int *__restrict__ count)
{
    uint32_t carry = 0;
    for (uint32_t b = 0; b < nb; b += SCAN_THREADS) {
        const uint32_t i = b + threadIdx.x;
        const uint32_t v = i < nb ? bsum[i] : 0u;
        uint32_t tot;
        const uint32_t ex = block_exclusive(v, &tot);
        if (i < nb) bsum[i] = carry + ex;
        carry += tot;
    }
    if (threadIdx.x == 0) *count = carry;
}

// incl[i] = number of marks in [0, i] (if incl != NULL); the k-th marked position (k from 0) goes to start[k]
__global__ void __launch_bounds__(SCAN_THREADS) k_scan_apply(const uint32_t *__restrict__ mark, uint32_t n, const uint32_t *__restrict__ bsum,
                                                             uint32_t *__restrict__ incl, uint32_t *__restrict__ start)
{
    const uint32_t i0 = blockIdx.x * SCAN_TILE + threadIdx.x * SCAN_ITEMS;
    uint32_t m[SCAN_ITEMS], s = 0;
#pragma unroll
    for (int k = 0; k < SCAN_ITEMS; k++) {
        m[k] = i0 + k < n ? mark[i0 + k] : 0u;
        s += m[k];
    }
    uint32_t tot;
    uint32_t run = bsum[blockIdx.x] + block_exclusive(s, &tot);
#pragma unroll
    for (int k = 0; k < SCAN_ITEMS; k++) {
        if (i0 + k < n) {
            if (m[k]) start[run] = i0 + k;
            run += m[k];
            if (incl) incl[i0 + k] = run;
        }
    }
}

template <typename K, bool HAS_VAL>
int sort_impl(sph_ctx *ctx, K *keys, K *keys_alt, uint32_t *vals, uint32_t *vals_alt, int64_t n, int bits, int *in_alt)
{
    *in_alt = 0;
    if (n <= 1 || bits <= 0) return SPH_OK;
    cudaStream_t st = ctx->stream;
    const uint32_t tiles = (uint32_t)((n + SORT_TILE - 1) / SORT_TILE);
    const size_t need = (size_t)SORT_RADIX * tiles + 2 * SORT_RADIX + 1;
    if (need > ctx->sort_cap) {
        ctx->sort_cap = 0;
        if (ctx->sort_hist) cudaFree(ctx->sort_hist);
        ctx->sort_hist = nullptr;
        SPH_CUDA(ctx, cudaMalloc((void **)&ctx->sort_hist, (need + need / 4) * sizeof(uint32_t)));
        ctx->sort_cap = need + need / 4;
    }
    uint32_t *hist = ctx->sort_hist, *base = ctx->sort_hist + (size_t)SORT_RADIX * tiles, *tot = base + SORT_RADIX;
    SPH_CUDA(ctx, cudaMemsetAsync(tot + SORT_RADIX, 0, sizeof(uint32_t), st)); // the self-wrapping block counter
    auto kfn = k_sort_scatter<K, HAS_VAL>;
    const size_t dyn = sizeof(SortSmem<K, HAS_VAL>);
    SPH_CUDA(ctx, cudaFuncSetAttribute(kfn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)dyn));
    K *ki = keys, *ko = keys_alt;
    uint32_t *vi = vals, *vo = vals_alt;
    for (int shift = 0; shift < bits; shift += 8) {
        const uint32_t mask = bits - shift >= 8 ? 0xffu : (1u << (bits - shift)) - 1u;
        k_sort_hist<K><<<tiles, SORT_THREADS, 0, st>>>(ki, (uint32_t)n, shift, mask, hist, tiles);
        k_sort_scan<<<SORT_RADIX, SORT_THREADS, 0, st>>>(hist, tiles, base, tot);
        kfn<<<tiles, SORT_THREADS, dyn, st>>>(ki, vi, ko, vo, (uint32_t)n, shift, mask, hist, base, tiles);
        { K *t = ki; ki = ko; ko = t; }
        { uint32_t *t = vi; vi = vo; vo = t; }
        *in_alt ^= 1;
        ctx->launches += 3;
    }
    SPH_CUDA(ctx, cudaGetLastError());
    return SPH_OK;
}

} // namespace

int sph_sort_pairs_u64(sph_ctx *ctx, uint64_t *keys, uint64_t *keys_alt, uint32_t *vals, uint32_t *vals_alt, int64_t n, int bits,
                       int *in_alt)
{
    return sort_impl<uint64_t, true>(ctx, keys, keys_alt, vals, vals_alt, n, bits, in_alt);
}

int sph_sort_keys_u32(sph_ctx *ctx, uint32_t *keys, uint32_t *keys_alt, int64_t n, int bits, int *in_alt)
{
    return sort_impl<uint32_t, false>(ctx, keys, keys_alt, nullptr, nullptr, n, bits, in_alt);
}

int sph_scan_marks(sph_ctx *ctx, const uint32_t *mark, int64_t n, uint32_t *incl, uint32_t *start, unsigned int *count_dev)
{
    if (n <= 0) return SPH_OK;
    cudaStream_t st = ctx->stream;
    const uint32_t nb = (uint32_t)((n + SCAN_TILE - 1) / SCAN_TILE);
    if (nb > ctx->scan_cap) {
        ctx->scan_cap = 0;
        if (ctx->scan_bsum) cudaFree(ctx->scan_bsum);
        ctx->scan_bsum = nullptr;
        SPH_CUDA(ctx, cudaMalloc((void **)&ctx->scan_bsum, ((size_t)nb + nb / 4 + 64) * sizeof(uint32_t)));
        ctx->scan_cap = nb + nb / 4 + 64;
    }
    k_scan_sums<<<nb, SCAN_THREADS, 0, st>>>(mark, (uint32_t)n, ctx->scan_bsum);
    k_scan_bsums<<<1, SCAN_THREADS, 0, st>>>(ctx->scan_bsum, nb, count_dev);
    k_scan_apply<<<nb, SCAN_THREADS, 0, st>>>(mark, (uint32_t)n, ctx->scan_bsum, incl, start);
    ctx->launches += 3;
    SPH_CUDA(ctx, cudaGetLastError());
    return SPH_OK;
}

// ---- stream compaction of 0/1 flags as a public call, with and without allocation ----------------------------------
// sph_compact_flags: the scan + compaction above with the context's growable block-sum buffer (the path sph_kdk_step
// and the index build use).  sph_compact_flags_noalloc: the same three kernels with the block sums in the fixed
// file-scope device array below, for callers that must not allocate (CUDA graph capture, serving loops).
#define SPH_NOALLOC_BLOCKS 16384 // block sums: 64 KB of device memory per GPU that loads the library, until exit
#define SPH_NOALLOC_DEVICES 64
static_assert((int64_t)SPH_NOALLOC_BLOCKS * SCAN_TILE == SPH_COMPACT_NOALLOC_MAX, "include/sph.h states the limit");

static __device__ __align__(256) uint32_t g_noalloc_bsum[SPH_NOALLOC_BLOCKS];
// In host code g_noalloc_bsum is only a handle for the runtime, not a device address: the address is asked for once per
// device (with that device current) and kept here.
static uint32_t *g_noalloc_ptr[SPH_NOALLOC_DEVICES];

static int compact_args(sph_ctx *ctx, const char *who, int64_t n, const uint32_t *flags, const int32_t *ids_out, const uint32_t *count_dev)
{
    if (n < 0 || !count_dev || (n > 0 && (!flags || !ids_out))) return sph_fail(ctx, SPH_E_ARG, "%s: n < 0 or NULL array", who);
    if (n >= (int64_t)1 << 31) return sph_fail(ctx, SPH_E_ARG, "%s: n = %lld exceeds 2^31 - 1", who, (long long)n);
    return SPH_OK;
}

extern "C" int sph_compact_flags(sph_ctx *ctx, int64_t n, const uint32_t *flags, int32_t *ids_out, uint32_t *count_dev)
{
    if (!ctx) return SPH_E_ARG;
    int rc = compact_args(ctx, "sph_compact_flags", n, flags, ids_out, count_dev);
    if (rc) return rc;
    if (n == 0) {
        SPH_CUDA(ctx, cudaMemsetAsync(count_dev, 0, sizeof(uint32_t), ctx->stream));
        return SPH_OK;
    }
    return sph_scan_marks(ctx, flags, n, nullptr, reinterpret_cast<uint32_t *>(ids_out), count_dev);
}

extern "C" int sph_compact_flags_noalloc(sph_ctx *ctx, int64_t n, const uint32_t *flags, int32_t *ids_out, uint32_t *count_dev)
{
    if (!ctx) return SPH_E_ARG;
    int rc = compact_args(ctx, "sph_compact_flags_noalloc", n, flags, ids_out, count_dev);
    if (rc) return rc;
    if (n > (int64_t)SPH_COMPACT_NOALLOC_MAX)
        return sph_fail(ctx, SPH_E_ARG, "sph_compact_flags_noalloc: n = %lld exceeds SPH_COMPACT_NOALLOC_MAX = %lld (fixed scratch; use sph_compact_flags)",
                        (long long)n, (long long)SPH_COMPACT_NOALLOC_MAX);
    cudaStream_t st = ctx->stream;
    int dev = -1;
    SPH_CUDA(ctx, cudaGetDevice(&dev));
    if (dev < 0 || dev >= SPH_NOALLOC_DEVICES) return sph_fail(ctx, SPH_E_ARG, "sph_compact_flags_noalloc: device ordinal %d not supported", dev);
    if (!g_noalloc_ptr[dev]) { // set-up, once per device (racing first calls of two host threads store the same address)
        uint32_t *p = nullptr;
        SPH_CUDA(ctx, cudaGetSymbolAddress((void **)&p, g_noalloc_bsum));
        if (!p) return sph_fail(ctx, SPH_E_CUDA, "sph_compact_flags_noalloc: no device address for the scratch array");
        g_noalloc_ptr[dev] = p;
    }
    uint32_t *bsum = g_noalloc_ptr[dev];
    if (n == 0) { // (a 4-byte store by a kernel: cudaMemsetAsync would do, but this keeps the call to kernel launches only)
        k_scan_bsums<<<1, SCAN_THREADS, 0, st>>>(bsum, 0u, count_dev);
        ctx->launches++;
        SPH_CUDA(ctx, cudaGetLastError());
        return SPH_OK;
    }
    // nothing in the scratch has to start at zero: k_scan_sums writes entries [0, nb) before anything reads them, and
    // entries beyond nb (left by an earlier, larger call) are never read
    const uint32_t nb = (uint32_t)((n + SCAN_TILE - 1) / SCAN_TILE);
    k_scan_sums<<<nb, SCAN_THREADS, 0, st>>>(flags, (uint32_t)n, bsum);
    k_scan_bsums<<<1, SCAN_THREADS, 0, st>>>(bsum, nb, count_dev);
    k_scan_apply<<<nb, SCAN_THREADS, 0, st>>>(flags, (uint32_t)n, bsum, nullptr, reinterpret_cast<uint32_t *>(ids_out));
    ctx->launches += 3;
    SPH_CUDA(ctx, cudaGetLastError());
    return SPH_OK;
}
