// a4 (part): hand-written stable LSD radix sort of (key32, value32) pairs, 4 passes of 8 bits, no CUB
// (reordering methods "encode and sort rays"; encode+sort overhead).
// Per pass: (1) per-block digit histograms, (2) a two-level exclusive scan over the digit-major (digit, block) table,
// (3) stable scatter: warp-private running digit counters + __match_any_sync rank the keys of a tile with one block barrier,
// and the tile leaves through shared memory in output order (see rs_scatter_kernel).
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
    uint32_t k[RS_ITEMS];                 // all 16 loads in flight before the first shared-memory atomic
#pragma unroll
    for (int it = 0; it < RS_ITEMS; ++it) {
        const int64_t i = base + it * RS_THREADS + threadIdx.x;
        k[it] = i < n ? __ldg(keys + i) : 0u;
    }
#pragma unroll
    for (int it = 0; it < RS_ITEMS; ++it)
        if (base + it * RS_THREADS + threadIdx.x < n) atomicAdd(&h[(k[it] >> shift) & 255u], 1u);
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

// Stable scatter of one pass.  Warp w owns the w-th 512-key segment of the block's tile and walks it in 16 rounds of 32
// consecutive keys; the rank of a key among equal digits of its segment is a warp-PRIVATE running counter (no block barrier
// per round) plus the earlier lanes of its round (__match_any_sync).  After one barrier the counters give, per digit, the
// block-local start of each warp's run; keys and values are staged in shared memory in output order and then written out
// so that the keys of one digit leave as one contiguous run (about 16 keys = 64 bytes for a uniform digit) instead of as
// isolated 4-byte stores.  Order inside a digit = segment, round, lane = input order: the sort stays stable.
__global__ void __launch_bounds__(RS_THREADS, 4) rs_scatter_kernel(const uint32_t* __restrict__ keys_in, const int32_t* __restrict__ vals_in, int64_t n, int shift,
                                                                const uint32_t* __restrict__ hist, int n_blocks, const uint32_t* __restrict__ totals,
                                                                uint32_t* __restrict__ keys_out, int32_t* __restrict__ vals_out)
{
    __shared__ uint32_t gbase[256];               // global position of the block's first key of each digit
    __shared__ uint32_t lstart[257];              // block-local position of the first key of each digit (exclusive scan of the block's counts)
    __shared__ uint32_t wcount[RS_WARPS][256];    // per warp: keys of each digit in its segment; then: local start of the warp's run
    __shared__ uint32_t wsum[RS_WARPS];
    __shared__ uint32_t s_key[RS_TILE];
    __shared__ int32_t s_val[RS_TILE];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const unsigned lt = (1u << lane) - 1u;
    {   // digit base = exclusive scan of the 256 digit totals (thread = digit) + this block's offset inside the digit
        const uint32_t v = totals[tid];
        uint32_t incl = v;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) { uint32_t t = __shfl_up_sync(0xffffffffu, incl, d); if (lane >= d) incl += t; }
        if (lane == 31) wsum[warp] = incl;
        __syncthreads();
        uint32_t off = 0;
        for (int w = 0; w < warp; ++w) off += wsum[w];
        gbase[tid] = off + incl - v + hist[(size_t)tid * n_blocks + blockIdx.x];
    }
#pragma unroll
    for (int w = 0; w < RS_WARPS; ++w) wcount[w][tid] = 0;
    __syncthreads();
    const int64_t base = (int64_t)blockIdx.x * RS_TILE + (int64_t)warp * (RS_TILE / RS_WARPS);
    uint32_t key[RS_ITEMS]; uint32_t rank[RS_ITEMS];       // rank: rank inside the warp's segment | digit << 16
#pragma unroll
    for (int it = 0; it < RS_ITEMS; ++it) {
        const int64_t i = base + it * 32 + lane;
        key[it] = i < n ? keys_in[i] : 0u;
    }
    // The 16 rounds depend on each other only through the counter of their digit: the first lane of each digit class adds the
    // class size to the warp's counter with a shared-memory atomic (which returns the count of earlier rounds) and hands it to
    // its peers by shuffle, so the rounds pipeline instead of forming a read-sync-write chain.
#pragma unroll
    for (int it = 0; it < RS_ITEMS; ++it) {
        const bool valid = base + it * 32 + lane < n;
        const uint32_t digit = valid ? ((key[it] >> shift) & 255u) : 256u;
        const unsigned peers = __match_any_sync(0xffffffffu, digit);
        const int leader = __ffs(peers) - 1;
        uint32_t before = 0;
        if (valid && lane == leader) before = atomicAdd(&wcount[warp][digit], (uint32_t)__popc(peers));
        before = __shfl_sync(0xffffffffu, before, leader);
        rank[it] = valid ? ((before + __popc(peers & lt)) | (digit << 16)) : 0xffffffffu;
    }
    __syncthreads();
    {   // thread = digit: block count, exclusive scan over digits -> lstart; per-warp run starts
        uint32_t cnt = 0, run[RS_WARPS];
#pragma unroll
        for (int w = 0; w < RS_WARPS; ++w) { run[w] = cnt; cnt += wcount[w][tid]; }
        uint32_t incl = cnt;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) { uint32_t t = __shfl_up_sync(0xffffffffu, incl, d); if (lane >= d) incl += t; }
        __syncthreads();                                  // wsum is reused
        if (lane == 31) wsum[warp] = incl;
        __syncthreads();
        uint32_t off = 0;
        for (int w = 0; w < warp; ++w) off += wsum[w];
        const uint32_t start = off + incl - cnt;
        lstart[tid] = start;
        if (tid == 255) lstart[256] = start + cnt;
#pragma unroll
        for (int w = 0; w < RS_WARPS; ++w) wcount[w][tid] = start + run[w];
    }
    __syncthreads();
#pragma unroll
    for (int it = 0; it < RS_ITEMS; ++it) {
        if (rank[it] != 0xffffffffu) {
            const uint32_t pos = wcount[warp][rank[it] >> 16] + (rank[it] & 0xffffu);
            s_key[pos] = key[it]; s_val[pos] = vals_in[base + it * 32 + lane];
        }
    }
    __syncthreads();
    const uint32_t n_local = lstart[256];
    for (uint32_t j = tid; j < n_local; j += RS_THREADS) {
        const uint32_t k = s_key[j], digit = (k >> shift) & 255u;
        const uint32_t out = gbase[digit] + (j - lstart[digit]);
        keys_out[out] = k; vals_out[out] = s_val[j];
    }
}

constexpr size_t align256(size_t x) { return (x + 255) & ~(size_t)255; }

// ---- scratch of the entry point that allocates nothing (crt_radix_sort_pairs_noalloc) ------------------------------------------
// The same layout as the caller-provided scratch of launch_radix_sort (ping-pong keys, ping-pong values, the (digit, block) histogram
// table, the 256 digit totals), sized for CRT_RADIX_SORT_NOALLOC_MAX_N pairs, in a file-scope device array: 17.3 MB that every GPU
// which loads the library holds until the process exits.  In HOST code the name below is a host-side stand-in, not a device address;
// the address is resolved once per device by radix_sort_noalloc_setup (cudaGetSymbolAddress with that device current) and kept in
// g_rs_static_ptr.
constexpr int64_t RS_STATIC_MAX_N = (int64_t)1 << 21;          // 2,097,152 pairs: covers the 2,088,960 ray slots of a 1920x1080 frame (BASELINE config 2 / 5)
constexpr size_t RS_STATIC_BYTES = 2 * align256((size_t)RS_STATIC_MAX_N * 4) + align256((size_t)((RS_STATIC_MAX_N + RS_TILE - 1) / RS_TILE) * 256 * 4) + align256(256 * 4) + 256;
static __device__ __align__(256) unsigned char g_rs_static_scratch[RS_STATIC_BYTES];

constexpr int RS_MAX_DEVICES = 64;
void* g_rs_static_ptr[RS_MAX_DEVICES] = {};                     // device address of g_rs_static_scratch on each device (null: not resolved)
cudaError_t g_rs_static_err[RS_MAX_DEVICES] = {};               // why not

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

// Set-up of the no-allocation sort, once per device, called by crt_create with `device` current: resolves the device address of the
// static scratch array.  A failure is kept and reported by the entry point (crt_create itself does not depend on it).
void radix_sort_noalloc_setup(int device)
{
    if (device < 0 || device >= RS_MAX_DEVICES || g_rs_static_ptr[device]) return;
    void* p = nullptr;
    const cudaError_t e = cudaGetSymbolAddress(&p, g_rs_static_scratch);
    if (e == cudaSuccess && p) g_rs_static_ptr[device] = p;
    else { g_rs_static_err[device] = e == cudaSuccess ? cudaErrorInvalidSymbol : e; cudaGetLastError(); }
}

int64_t radix_sort_noalloc_max_n() { return RS_STATIC_MAX_N; }

// The sort of launch_radix_sort with the library's static scratch: no cudaMalloc, cudaFree or allocating library call on this path.
// Nothing in the scratch has to start at zero: every histogram entry, total and ping-pong element a pass reads was written earlier in
// the same call (rs_hist_kernel writes all 256 x n_blocks entries it later reads), so the previous call's contents are never read.
// All calls on a device share the one array: two calls whose kernels overlap on the GPU (different streams, or different contexts of
// one device) race; callers serialise them (one stream, or an event between them).
crt_status launch_radix_sort_noalloc(crt_ctx* ctx, const uint32_t* kin, const int32_t* vin, int64_t n, uint32_t* kout, int32_t* vout, cudaStream_t st)
{
    if (n == 0) return CRT_OK;
    if (n > RS_STATIC_MAX_N)
        return crt_fail(ctx, CRT_ERR_UNSUPPORTED, "radix_sort_pairs_noalloc: %lld pairs exceed the static scratch's maximum of %lld (use crt_radix_sort_pairs with caller scratch)",
                        (long long)n, (long long)RS_STATIC_MAX_N);
    const int dev = ctx->device;
    if (dev < 0 || dev >= RS_MAX_DEVICES || !g_rs_static_ptr[dev])
        return crt_fail(ctx, CRT_ERR_STATE, "radix_sort_pairs_noalloc: the static scratch's device address was not resolved at crt_create (%s)",
                        dev >= 0 && dev < RS_MAX_DEVICES ? cudaGetErrorString(g_rs_static_err[dev]) : "device index beyond the table");
    return launch_radix_sort(ctx, kin, vin, n, kout, vout, g_rs_static_ptr[dev], RS_STATIC_BYTES, st);
}
