// a4 (part): hand-written stable LSD radix sort of (key32, value32) pairs, 4 passes of 8 bits, no CUB
// (reordering methods "encode and sort rays"; encode+sort overhead).
// Per pass: (1) per-block digit histograms, (2) a two-level exclusive scan over the digit-major (digit, block) table,
// (3) stable scatter: blocks re-read their tile in order; inside a round of 256 keys the rank of a key among equal
// digits is (keys of that digit in earlier warps) + (earlier lanes of its warp, from __match_any_sync).
#include "crt_internal.h"

namespace {

constexpr int RS_THREADS = 256;
constexpr int RS_ITEMS = 16;
constexpr int RS_TILE = RS_THREADS * RS_ITEMS;
constexpr int RS_WARPS = RS_THREADS / 32;

__global__ void __launch_bounds__(RS_THREADS) rs_hist_kernel(const uint32_t* __restrict__ keys, int64_t n, int shift, uint32_t* __restrict__ hist, int n_blocks)
{
    __shared__ uint32_t h[256];
    h[threadIdx.x] = 0;
    __syncthreads();
    const int64_t base = (int64_t)blockIdx.x * RS_TILE;
#pragma unroll 4
    for (int it = 0; it < RS_ITEMS; ++it) {
        const int64_t i = base + it * RS_THREADS + threadIdx.x;
        if (i < n) atomicAdd(&h[(keys[i] >> shift) & 255u], 1u);
    }
    __syncthreads();
    hist[(size_t)threadIdx.x * n_blocks + blockIdx.x] = h[threadIdx.x];
}

// exclusive scan of the digit-major (digit, block) table, in two levels: block d scans row d (n_blocks counters, coalesced)
// in place and writes the row total; the scatter kernel turns the 256 totals into digit bases itself
__global__ void __launch_bounds__(256) rs_scan_kernel(uint32_t* __restrict__ hist, int n_blocks, uint32_t* __restrict__ totals)
{
    __shared__ uint32_t warp_sums[8];
    __shared__ uint32_t carry_s;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    uint32_t* row = hist + (size_t)blockIdx.x * n_blocks;
    if (tid == 0) carry_s = 0;
    __syncthreads();
    for (int base = 0; base < n_blocks; base += 256) {
        const int i = base + tid;
        const uint32_t v = i < n_blocks ? row[i] : 0u;
        uint32_t incl = v;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) { uint32_t t = __shfl_up_sync(0xffffffffu, incl, d); if (lane >= d) incl += t; }
        if (lane == 31) warp_sums[warp] = incl;
        __syncthreads();
        uint32_t off = carry_s;
        for (int w = 0; w < warp; ++w) off += warp_sums[w];
        if (i < n_blocks) row[i] = off + incl - v;
        __syncthreads();
        if (tid == 255) carry_s = off + incl;
        __syncthreads();
    }
    if (tid == 0) totals[blockIdx.x] = carry_s;
}

__global__ void __launch_bounds__(RS_THREADS) rs_scatter_kernel(const uint32_t* __restrict__ keys_in, const int32_t* __restrict__ vals_in, int64_t n, int shift,
                                                                const uint32_t* __restrict__ hist, int n_blocks, const uint32_t* __restrict__ totals,
                                                                uint32_t* __restrict__ keys_out, int32_t* __restrict__ vals_out)
{
    __shared__ uint32_t run[256];
    __shared__ uint32_t wcount[RS_WARPS][256];
    __shared__ uint32_t wsum[RS_WARPS];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    {   // digit base = exclusive scan of the 256 digit totals (thread = digit)
        const uint32_t v = totals[tid];
        uint32_t incl = v;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) { uint32_t t = __shfl_up_sync(0xffffffffu, incl, d); if (lane >= d) incl += t; }
        if (lane == 31) wsum[warp] = incl;
        __syncthreads();
        uint32_t off = 0;
        for (int w = 0; w < warp; ++w) off += wsum[w];
        run[tid] = off + incl - v + hist[(size_t)tid * n_blocks + blockIdx.x];
    }
#pragma unroll
    for (int w = 0; w < RS_WARPS; ++w) wcount[w][tid] = 0;
    __syncthreads();
    const int64_t base = (int64_t)blockIdx.x * RS_TILE;
    for (int it = 0; it < RS_ITEMS; ++it) {
        const int64_t i = base + it * RS_THREADS + tid;
        const bool valid = i < n;
        uint32_t key = 0; int32_t val = 0;
        if (valid) { key = keys_in[i]; val = vals_in[i]; }
        const uint32_t digit = valid ? ((key >> shift) & 255u) : 256u;
        const unsigned peers = __match_any_sync(0xffffffffu, digit);
        const unsigned rank = __popc(peers & ((1u << lane) - 1u));
        if (valid && rank == 0) wcount[warp][digit] = __popc(peers);
        __syncthreads();
        if (valid) {
            uint32_t off = run[digit] + rank;
            for (int w = 0; w < warp; ++w) off += wcount[w][digit];
            keys_out[off] = key; vals_out[off] = val;
        }
        __syncthreads();
        uint32_t tot = 0;
#pragma unroll
        for (int w = 0; w < RS_WARPS; ++w) { tot += wcount[w][tid]; wcount[w][tid] = 0; }
        run[tid] += tot;
        __syncthreads();
    }
}

inline size_t align256(size_t x) { return (x + 255) & ~(size_t)255; }

}  // namespace

size_t radix_sort_scratch_bytes(int64_t n)
{
    const int64_t blocks = (n + RS_TILE - 1) / RS_TILE;
    return 2 * align256((size_t)n * 4) + align256((size_t)blocks * 256 * 4) + align256(256 * 4) + 256;
}

crt_status launch_radix_sort(crt_ctx* ctx, const uint32_t* kin, const int32_t* vin, int64_t n, uint32_t* kout, int32_t* vout,
                             void* scratch, size_t scratch_bytes, cudaStream_t st)
{
    if (n == 0) return CRT_OK;
    if (n >= ((int64_t)1 << 31)) return crt_fail(ctx, CRT_ERR_UNSUPPORTED, "radix sort: n >= 2^31");
    if (scratch_bytes < radix_sort_scratch_bytes(n)) return crt_fail(ctx, CRT_ERR_INVALID_ARG, "radix sort: scratch too small");
    const int blocks = (int)((n + RS_TILE - 1) / RS_TILE);
    char* s = static_cast<char*>(scratch);
    uint32_t* ka = reinterpret_cast<uint32_t*>(s); s += align256((size_t)n * 4);
    int32_t* va = reinterpret_cast<int32_t*>(s); s += align256((size_t)n * 4);
    uint32_t* hist = reinterpret_cast<uint32_t*>(s); s += align256((size_t)blocks * 256 * 4);
    uint32_t* totals = reinterpret_cast<uint32_t*>(s);
    const uint32_t* src_k = kin; const int32_t* src_v = vin;
    for (int pass = 0; pass < 4; ++pass) {
        uint32_t* dst_k = (pass & 1) ? kout : ka; int32_t* dst_v = (pass & 1) ? vout : va;
        rs_hist_kernel<<<blocks, RS_THREADS, 0, st>>>(src_k, n, 8 * pass, hist, blocks);
        rs_scan_kernel<<<256, 256, 0, st>>>(hist, blocks, totals);
        rs_scatter_kernel<<<blocks, RS_THREADS, 0, st>>>(src_k, src_v, n, 8 * pass, hist, blocks, totals, dst_k, dst_v);
        src_k = dst_k; src_v = dst_v;
    }
    CRT_CHECK_LAUNCH(ctx, "radix_sort");
    return CRT_OK;
}
