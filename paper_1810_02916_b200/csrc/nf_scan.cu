// nf_scan.cu -- device-wide exclusive prefix sums (cell_offset).
// Three-phase scan: per-block reduce, recursive scan of block sums, per-block scan + offset.
#include "nf_common.cuh"

namespace {

constexpr int SCAN_THREADS = 256;
constexpr int SCAN_ITEMS = 16;
constexpr int SCAN_TILE = SCAN_THREADS * SCAN_ITEMS;

template <class TOut>
__device__ __forceinline__ TOut warp_inclusive(TOut v, int lane)
{
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        TOut n = __shfl_up_sync(0xffffffffu, v, d);
        if (lane >= d) v += n;
    }
    return v;
}

// block-wide exclusive scan of one value per thread; returns exclusive prefix, total in *total
template <class TOut>
__device__ __forceinline__ TOut block_exclusive(TOut v, TOut *total)
{
    __shared__ TOut warp_sums[SCAN_THREADS / 32];
    int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    TOut inc = warp_inclusive(v, lane);
    if (lane == 31) warp_sums[w] = inc;
    __syncthreads();
    if (w == 0) {
        TOut s = lane < SCAN_THREADS / 32 ? warp_sums[lane] : TOut(0);
        TOut si = warp_inclusive(s, lane);
        if (lane < SCAN_THREADS / 32) warp_sums[lane] = si - s;
        if (lane == SCAN_THREADS / 32 - 1) *total = si;
    }
    __syncthreads();
    TOut r = inc - v + warp_sums[w];
    __syncthreads();
    return r;
}

template <class TIn, class TOut>
__global__ void __launch_bounds__(SCAN_THREADS) k_scan_reduce(const TIn *__restrict__ in, size_t n, TOut *__restrict__ sums)
{
    __shared__ TOut total;
    size_t base = (size_t)blockIdx.x * SCAN_TILE;
    TOut s = 0;
#pragma unroll
    for (int k = 0; k < SCAN_ITEMS; k++) {
        size_t i = base + (size_t)k * SCAN_THREADS + threadIdx.x;
        if (i < n) s += (TOut)in[i];
    }
    block_exclusive<TOut>(s, &total);
    if (threadIdx.x == 0) sums[blockIdx.x] = total;
}

// in-place safe (in may alias out when TIn == TOut): all loads of a tile happen before its stores
template <class TIn, class TOut>
__global__ void __launch_bounds__(SCAN_THREADS) k_scan_apply(const TIn *in, size_t n, const TOut *__restrict__ block_offsets, TOut *out, int write_total)
{
    __shared__ TOut total;
    size_t base = (size_t)blockIdx.x * SCAN_TILE + (size_t)threadIdx.x * SCAN_ITEMS;
    TOut v[SCAN_ITEMS];
    TOut s = 0;
#pragma unroll
    for (int k = 0; k < SCAN_ITEMS; k++) {
        size_t i = base + k;
        v[k] = i < n ? (TOut)in[i] : TOut(0);
        s += v[k];
    }
    TOut ex = block_exclusive<TOut>(s, &total);
    TOut run = ex + (block_offsets ? block_offsets[blockIdx.x] : TOut(0));
#pragma unroll
    for (int k = 0; k < SCAN_ITEMS; k++) {
        size_t i = base + k;
        if (i < n) out[i] = run;
        run += v[k];
        if (write_total && i == n - 1) out[n] = run;  // out has n+1 entries
    }
}

template <class TIn, class TOut>
int scan_impl(nf_ctx *ctx, const TIn *in, TOut *out, size_t n, TOut *temp, cudaStream_t st, int write_total)
{
    if (n == 0) {
        if (write_total) NF_CUDA(ctx, cudaMemsetAsync(out, 0, sizeof(TOut), st));
        return NF_OK;
    }
    size_t nblk = (n + SCAN_TILE - 1) / SCAN_TILE;
    if (nblk == 1) {
        k_scan_apply<TIn, TOut><<<1, SCAN_THREADS, 0, st>>>(in, n, nullptr, out, write_total);
        NF_LAUNCHED(ctx);
        return NF_OK;
    }
    TOut *sums = temp;
    k_scan_reduce<TIn, TOut><<<(unsigned)nblk, SCAN_THREADS, 0, st>>>(in, n, sums);
    NF_LAUNCHED(ctx);
    NF_TRY((scan_impl<TOut, TOut>(ctx, sums, sums, nblk, temp + nf_align_up(nblk, 64), st, 0)));
    k_scan_apply<TIn, TOut><<<(unsigned)nblk, SCAN_THREADS, 0, st>>>(in, n, sums, out, write_total);
    NF_LAUNCHED(ctx);
    return NF_OK;
}

}  // namespace

size_t nf_scan_temp_elems(size_t n)
{
    size_t total = 0;
    while (n > (size_t)SCAN_TILE) {
        n = (n + SCAN_TILE - 1) / SCAN_TILE;
        total += nf_align_up(n, 64);
    }
    return total + 64;
}

int nf_exclusive_scan_u32(nf_ctx *ctx, const uint32_t *in, uint32_t *out, size_t n, uint32_t *temp, cudaStream_t st)
{
    return scan_impl<uint32_t, uint32_t>(ctx, in, out, n, temp, st, 0);
}

// out has n+1 entries: out[n] = total
int nf_exclusive_scan_u32_u64(nf_ctx *ctx, const uint32_t *in, uint64_t *out, size_t n, uint64_t *temp, cudaStream_t st)
{
    return scan_impl<uint32_t, uint64_t>(ctx, in, out, n, temp, st, 1);
}
