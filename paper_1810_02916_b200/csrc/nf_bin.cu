// nf_bin.cu -- cell assignment and STABLE counting sort by cell.
//
// PAPER.md:37 "the domain is decomposed into K^3 cubic cells, and every particle belongs to
// one cell"; :47 a slab spans all Y,Z at one X (x slowest, z fastest); :51 positions are
// stored as float32 offsets from the cell centre.
//
// Pipeline (all on the caller's stream):
//   keys      one thread per particle: float32 cell index per axis (bit-exact contract in
//             include/nf.h), key = (cx*K+cy)*K+cz
//   radix     LSD radix sort of (key, original index) with one digit per axis (cz, cy, cx),
//             each pass a stable counting sort over <= K bins: per-tile digit histogram,
//             device-wide scan, stable scatter with warp-level match/ballot ranking.
//             LSD + stable passes => ties keep input order => perm increases within a cell.
//   gather    sorted slot s: i = perm[s]; offset = x_i - centre(cell) -> float4; the first and last slot of
//             every run of equal keys give the cell's histogram (no atomics: cell_count = end - first)
//   scan      cell_offset = exclusive scan of cell_count (uint64)
//
// The sort is deterministic (no atomics decide an output position).
#include "nf_common.cuh"

namespace {

constexpr int RS_THREADS = 512;
constexpr int RS_WARPS = RS_THREADS / 32;
constexpr int RS_ROUNDS = 16;                       // rounds of 32 elements per warp
constexpr int RS_WARP_ELEMS = RS_ROUNDS * 32;       // 512
constexpr int RS_TILE = RS_WARPS * RS_WARP_ELEMS;   // 8192

// float32 cell index, include/nf.h contract: c = (int)floorf(x * invw) clamped to [0, K-1].
// __fmul_rn is never contracted into an FMA.
// "Out of range" is x outside [0, box) or NaN; an x just below box whose product rounds up to K
// is valid and silently clamped into cell K-1 (reading c9).
__device__ __forceinline__ int cell_index(float x, float invw, float box, int K, int *bad)
{
    float fl = floorf(__fmul_rn(x, invw));
    int b = !(x >= 0.0f && x < box);
    int c;
    if (!(fl >= 0.0f)) c = 0;
    else if (fl > (float)(K - 1)) c = K - 1;
    else c = (int)fl;
    *bad |= b;
    return c;
}

__global__ void __launch_bounds__(256) k_keys(const float *__restrict__ pos, int64_t N, int K, float invw, float box, int plane_cx,
                                              uint32_t *__restrict__ keys, unsigned long long *__restrict__ n_bad)
{
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    int bad = 0;
    if (i < N) {
        float x = pos[3 * i + 0], y = pos[3 * i + 1], z = pos[3 * i + 2];
        int cx = cell_index(x, invw, box, K, &bad);
        int cy = cell_index(y, invw, box, K, &bad);
        int cz = cell_index(z, invw, box, K, &bad);
        uint32_t key;
        if (plane_cx >= 0) {
            bad |= (cx != plane_cx);
            key = (uint32_t)cy * (uint32_t)K + (uint32_t)cz;
        } else {
            key = ((uint32_t)cx * (uint32_t)K + (uint32_t)cy) * (uint32_t)K + (uint32_t)cz;
        }
        keys[i] = key;
    }
    unsigned m = __ballot_sync(0xffffffffu, bad);
    if (m && (threadIdx.x & 31) == 0) atomicAdd(n_bad, (unsigned long long)__popc(m));
}

// digit of a key: (key / div) % K, by shift and mask when K is a power of two (sh < 32)
struct Digit {
    uint32_t div, K, sh, mask;     // sh = 32: general K
    uint32_t nbits;                // bits of a digit value, ceil(log2 K)
    __device__ __forceinline__ uint32_t operator()(uint32_t key) const { return sh < 32 ? (key >> sh) & mask : (key / div) % K; }
};

// Lanes of `act` holding the same digit as this lane: one ballot per digit bit (a warp "multi-split").  The same
// result as __match_any_sync, which is several times slower for ~30 distinct values per warp (measured: the
// scatter pass went from 17.5 ms to 13.3 ms on C4).
__device__ __forceinline__ unsigned same_digit_lanes(unsigned act, uint32_t d, uint32_t nbits)
{
    unsigned peers = act;
    for (uint32_t b = 0; b < nbits; b++) {
        const bool bit = (d >> b) & 1u;
        const unsigned m = __ballot_sync(0xffffffffu, bit);
        peers &= bit ? m : ~m;
    }
    return peers;
}

// per-tile digit histogram -> hist[digit * ntiles + tile]
// n_dev (nullable): the element count lives on the device (at most N); tiles past it count nothing
__global__ void __launch_bounds__(RS_THREADS) k_radix_hist(const uint32_t *__restrict__ keys, int64_t N, const uint32_t *__restrict__ n_dev,
                                                           Digit dg, uint32_t *__restrict__ hist, uint32_t ntiles)
{
    extern __shared__ uint32_t sh[];
    if (n_dev) N = min(N, (int64_t)*n_dev);
    const uint32_t K = dg.K;
    for (uint32_t d = threadIdx.x; d < K; d += RS_THREADS) sh[d] = 0;
    __syncthreads();
    int64_t base = (int64_t)blockIdx.x * RS_TILE;
#pragma unroll 4
    for (int k = 0; k < RS_TILE / RS_THREADS; k++) {
        int64_t i = base + (int64_t)k * RS_THREADS + threadIdx.x;
        if (i < N) atomicAdd(&sh[dg(keys[i])], 1u);
    }
    __syncthreads();
    for (uint32_t d = threadIdx.x; d < K; d += RS_THREADS) hist[(size_t)d * ntiles + blockIdx.x] = sh[d];
}

// Stable scatter of one tile of RS_TILE elements.  Warp w owns elements [tile*RS_TILE + w*512, +512)
// in index order.  Ranks come from warp match/ballot (no atomic decides a slot), the tile is first
// sorted by digit INTO SHARED MEMORY, and only then written out, so that every digit's run of the
// tile (RS_TILE / K elements on average) leaves as one contiguous, coalesced burst instead of
// 4-byte stores scattered over the whole array.  idx_in == nullptr means "identity" (first pass).
// shared: cnt[RS_WARPS][K] | gdelta[K] | wsum[RS_WARPS] | skey[RS_TILE] | sidx[RS_TILE]
__global__ void __launch_bounds__(RS_THREADS) k_radix_scatter(const uint32_t *__restrict__ keys_in, const uint32_t *__restrict__ idx_in,
                                                              int64_t N, const uint32_t *__restrict__ n_dev, Digit dg,
                                                              const uint32_t *__restrict__ hist_scanned, uint32_t ntiles,
                                                              uint32_t *__restrict__ keys_out, uint32_t *__restrict__ idx_out)
{
    extern __shared__ uint32_t sh[];
    if (n_dev) N = min(N, (int64_t)*n_dev);
    if ((int64_t)blockIdx.x * RS_TILE >= N) return;
    const uint32_t K = dg.K;
    uint32_t *gdelta = sh + (size_t)RS_WARPS * K;
    uint32_t *wsum = gdelta + K;
    uint32_t *skey = wsum + 32;
    uint32_t *sidx = skey + RS_TILE;
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const unsigned lt = (1u << lane) - 1u;
    for (uint32_t d = threadIdx.x; d < K * RS_WARPS; d += RS_THREADS) sh[d] = 0;
    __syncthreads();
    uint32_t *cnt = sh + (size_t)w * K;
    const int64_t tbase = (int64_t)blockIdx.x * RS_TILE;
    const int64_t wbase = tbase + (int64_t)w * RS_WARP_ELEMS;
    uint32_t key[RS_ROUNDS];
    unsigned peers[RS_ROUNDS];       // lanes of the round holding the same digit (0: element past N)
    // count pass
#pragma unroll
    for (int r = 0; r < RS_ROUNDS; r++) {
        int64_t i = wbase + r * 32 + lane;
        bool valid = i < N;
        key[r] = valid ? keys_in[i] : 0u;
        unsigned act = __ballot_sync(0xffffffffu, valid);
        const uint32_t d = dg(key[r]);
        peers[r] = same_digit_lanes(act, d, dg.nbits);
        if (!valid) peers[r] = 0u;
        if (valid && (peers[r] & lt) == 0) cnt[d] += __popc(peers[r]);  // leader = lowest lane of the group
        __syncwarp();
    }
    __syncthreads();
    // For every digit: exclusive scan across warps, then across digits (block scan of the digit
    // totals, RS_THREADS digits per sweep) -> cnt[w][d] = first slot of (warp, digit) within the
    // sorted tile; gdelta[d] = (global slot of the tile's first element of digit d) - (its tile slot).
    uint32_t carry = 0;
    for (uint32_t d0 = 0; d0 < K; d0 += RS_THREADS) {
        const uint32_t d = d0 + threadIdx.x;
        uint32_t tot = 0;
        if (d < K) {
#pragma unroll
            for (int ww = 0; ww < RS_WARPS; ww++) {
                uint32_t t = sh[(size_t)ww * K + d];
                sh[(size_t)ww * K + d] = tot;
                tot += t;
            }
        }
        uint32_t incl = tot;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            uint32_t v = __shfl_up_sync(0xffffffffu, incl, o);
            if (lane >= o) incl += v;
        }
        if (lane == 31) wsum[w] = incl;
        __syncthreads();
        uint32_t woff = 0, all = 0;
#pragma unroll
        for (int ww = 0; ww < RS_WARPS; ww++) {
            uint32_t t = wsum[ww];
            if (ww < w) woff += t;
            all += t;
        }
        const uint32_t dstart = carry + woff + incl - tot;
        if (d < K) {
#pragma unroll
            for (int ww = 0; ww < RS_WARPS; ww++) sh[(size_t)ww * K + d] += dstart;
            gdelta[d] = hist_scanned[(size_t)d * ntiles + blockIdx.x] - dstart;
        }
        carry += all;
        __syncthreads();
    }
    // rank pass: stable slot within the sorted tile, staged in shared memory
#pragma unroll
    for (int r = 0; r < RS_ROUNDS; r++) {
        int64_t i = wbase + r * 32 + lane;
        if (peers[r]) {
            const unsigned pr = peers[r];
            uint32_t d = dg(key[r]);
            int leader = __ffs(pr) - 1;
            uint32_t base = 0;
            if (lane == leader) {
                base = cnt[d];
                cnt[d] = base + __popc(pr);
            }
            base = __shfl_sync(pr, base, leader);
            uint32_t slot = base + __popc(pr & lt);
            skey[slot] = key[r];
            sidx[slot] = idx_in ? idx_in[i] : (uint32_t)i;
        }
        __syncwarp();
    }
    __syncthreads();
    // write out: consecutive tile slots of one digit go to consecutive global slots
    const int64_t rem = N - tbase;
    const uint32_t tile_n = rem < RS_TILE ? (uint32_t)rem : (uint32_t)RS_TILE;
    for (uint32_t s = threadIdx.x; s < tile_n; s += RS_THREADS) {
        const uint32_t k = skey[s];
        const uint32_t dst = s + gdelta[dg(k)];
        keys_out[dst] = k;
        idx_out[dst] = sidx[s];
    }
}

// gather positions into cell order and re-centre.  Offset contract:
// hw = 0.5f*(box/(float)K); centre = (float)(2c+1)*hw; o = x - centre (no FMA contraction).
constexpr int GA_PER = 4;              // sorted slots per thread: all their (random) position loads are in flight together

__global__ void __launch_bounds__(256) k_gather(const float *__restrict__ pos, const float *__restrict__ mass,
                                                const uint32_t *__restrict__ keys_sorted,
                                                const uint32_t *__restrict__ perm, int64_t N, int K, float hw, int plane_cx,
                                                float4 *__restrict__ pos_sorted, uint32_t *__restrict__ cell_first,
                                                uint32_t *__restrict__ cell_end)
{
    const int64_t s0 = (int64_t)blockIdx.x * (256 * GA_PER) + threadIdx.x;
    uint32_t key[GA_PER], idx[GA_PER];
    float x[GA_PER], y[GA_PER], z[GA_PER], m[GA_PER];
#pragma unroll
    for (int j = 0; j < GA_PER; j++) {
        const int64_t s = s0 + j * 256;
        key[j] = s < N ? keys_sorted[s] : 0u;
        idx[j] = s < N ? perm[s] : 0u;
    }
#pragma unroll
    for (int j = 0; j < GA_PER; j++) {
        const int64_t s = s0 + j * 256;
        if (s < N) {
            const float *pp = pos + 3 * (size_t)idx[j];
            x[j] = __ldg(pp + 0); y[j] = __ldg(pp + 1); z[j] = __ldg(pp + 2);
            m[j] = mass ? __ldg(mass + idx[j]) : 0.0f;           // the spare lane carries the particle's mass when one is given
        }
    }
#pragma unroll
    for (int j = 0; j < GA_PER; j++) {
        const int64_t s = s0 + j * 256;
        if (s >= N) continue;
        const uint32_t k = key[j];
        // histogram from the sorted keys: a run of equal keys is one cell
        const uint32_t prev = s > 0 ? keys_sorted[s - 1] : ~k, next = s + 1 < N ? keys_sorted[s + 1] : ~k;
        if (k != prev) cell_first[k] = (uint32_t)s;
        if (k != next) cell_end[k] = (uint32_t)(s + 1);
        const int cz = (int)(k % (uint32_t)K);
        const int cy = (int)((k / (uint32_t)K) % (uint32_t)K);
        const int cx = plane_cx >= 0 ? plane_cx : (int)(k / ((uint32_t)K * (uint32_t)K));
        float4 o;
        o.x = __fsub_rn(x[j], __fmul_rn((float)(2 * cx + 1), hw));
        o.y = __fsub_rn(y[j], __fmul_rn((float)(2 * cy + 1), hw));
        o.z = __fsub_rn(z[j], __fmul_rn((float)(2 * cz + 1), hw));
        o.w = m[j];
        pos_sorted[s] = o;
    }
}

// cell_count[c] = end - first (both zero for a cell no run belongs to)
__global__ void __launch_bounds__(256) k_cell_counts(uint32_t *__restrict__ cell_count, const uint32_t *__restrict__ cell_first, size_t ncell)
{
    const size_t c = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (c < ncell) cell_count[c] -= cell_first[c];
}

}  // namespace

size_t nf_bin_scratch_bytes(int64_t N, int K, bool plane)
{
    size_t n = (size_t)(N > 0 ? N : 1);
    size_t ntiles = (n + RS_TILE - 1) / RS_TILE;
    size_t ncell = plane ? (size_t)K * K : (size_t)K * K * K;
    size_t b = 0;
    b += 3 * nf_align_up(n * sizeof(uint32_t), 256);                 // keysA, keysB, idxB
    b += nf_align_up((size_t)K * ntiles * sizeof(uint32_t), 256);    // digit histograms
    b += nf_align_up(nf_scan_temp_elems((size_t)K * ntiles) * sizeof(uint32_t), 256);
    b += nf_align_up(nf_scan_temp_elems(ncell) * sizeof(uint64_t), 256);
    b += nf_align_up(ncell * sizeof(uint32_t), 256);                 // first slot of every cell's run
    return b + 4096;
}

// One stable LSD pass over (key, index) pairs by the digit (key >> shift) & (bins - 1), bins a power of two <= 1024.  The
// element count may live on the device (n_dev, at most n_max).  hist: bins * ceil(n_max / RS_TILE) words; tmp32: its scan temp.
size_t nf_radix_tiles(int64_t n_max) { return n_max > 0 ? ((size_t)n_max + RS_TILE - 1) / RS_TILE : 1; }
int nf_radix_pass(nf_ctx *ctx, const uint32_t *kin, const uint32_t *iin, int64_t n_max, const uint32_t *n_dev, uint32_t bins,
                  uint32_t shift, uint32_t *kout, uint32_t *iout, uint32_t *hist, uint32_t *tmp32, cudaStream_t st)
{
    if (n_max <= 0) return NF_OK;
    const size_t ntiles = nf_radix_tiles(n_max);
    Digit dg;
    dg.div = 1u << shift; dg.K = bins; dg.sh = shift; dg.mask = bins - 1;
    dg.nbits = 0;
    while ((1u << dg.nbits) < bins) dg.nbits++;
    const size_t sh_hist = (size_t)bins * sizeof(uint32_t);
    const size_t sh_scat = ((size_t)bins * RS_WARPS + (size_t)bins + 32 + 2 * (size_t)RS_TILE) * sizeof(uint32_t);
    k_radix_hist<<<(unsigned)ntiles, RS_THREADS, sh_hist, st>>>(kin, n_max, n_dev, dg, hist, (uint32_t)ntiles);
    NF_LAUNCHED(ctx);
    NF_TRY(nf_exclusive_scan_u32(ctx, hist, hist, (size_t)bins * ntiles, tmp32, st));
    NF_CUDA(ctx, cudaFuncSetAttribute(k_radix_scatter, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sh_scat));
    k_radix_scatter<<<(unsigned)ntiles, RS_THREADS, sh_scat, st>>>(kin, iin, n_max, n_dev, dg, hist, (uint32_t)ntiles, kout, iout);
    NF_LAUNCHED(ctx);
    return NF_OK;
}

// a1 alone: keys (cx*K+cy)*K+cz of N positions, no histogram; out-of-range particles counted in counters[0]
int nf_keys_impl(nf_ctx *ctx, const float *pos, int64_t N, int K, float box, uint32_t *keys, cudaStream_t st)
{
    if (N <= 0) return NF_OK;
    const float invw = (float)K / box;
    k_keys<<<(unsigned)(((size_t)N + 255) / 256), 256, 0, st>>>(pos, N, K, invw, box, -1, keys, ctx->counters);
    NF_LAUNCHED(ctx);
    return NF_OK;
}

int nf_bin_impl(nf_ctx *ctx, const float *pos, const float *mass, int64_t N, int K, float box, int plane_cx,
                float *pos_sorted, uint32_t *perm, uint32_t *cell_count, uint64_t *cell_offset,
                cudaStream_t st)
{
    const bool plane = plane_cx >= 0;
    const size_t ncell = plane ? (size_t)K * K : (size_t)K * K * K;
    const int npass = plane ? 2 : 3;
    const size_t n = (size_t)N;
    const size_t ntiles = n ? (n + RS_TILE - 1) / RS_TILE : 1;

    uint32_t *keysA = nf_scratch_take<uint32_t>(ctx, n ? n : 1);
    uint32_t *keysB = nf_scratch_take<uint32_t>(ctx, n ? n : 1);
    uint32_t *idxB = nf_scratch_take<uint32_t>(ctx, n ? n : 1);
    uint32_t *hist = nf_scratch_take<uint32_t>(ctx, (size_t)K * ntiles);
    uint32_t *tmp32 = nf_scratch_take<uint32_t>(ctx, nf_scan_temp_elems((size_t)K * ntiles));
    uint64_t *tmp64 = nf_scratch_take<uint64_t>(ctx, nf_scan_temp_elems(ncell));
    uint32_t *first = nf_scratch_take<uint32_t>(ctx, ncell);
    if (!keysA || !keysB || !idxB || !hist || !tmp32 || !tmp64 || !first) {
        NF_SET_ERR(ctx, "nf_bin: internal scratch arena too small");
        return NF_ERR_NOMEM;
    }

    NF_CUDA(ctx, cudaMemsetAsync(cell_count, 0, ncell * sizeof(uint32_t), st));
    if (N == 0) return nf_exclusive_scan_u32_u64(ctx, cell_count, cell_offset, ncell, tmp64, st);
    NF_CUDA(ctx, cudaMemsetAsync(first, 0, ncell * sizeof(uint32_t), st));
    {
        float invw = (float)K / box;
        k_keys<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(pos, N, K, invw, box, plane_cx, keysA, ctx->counters);
        NF_LAUNCHED(ctx);
    }

    // LSD passes: digit cz (div 1), cy (div K), cx (div K^2).  Destinations alternate so that
    // the last pass writes the index array into `perm`.
    const uint32_t *kin = keysA;
    const uint32_t *iin = nullptr;
    uint32_t div = 1;
    for (int p = 0; p < npass; p++) {
        bool to_perm = ((npass - 1 - p) % 2) == 0;
        uint32_t *kout = (kin == keysA) ? keysB : keysA;
        uint32_t *iout = to_perm ? perm : idxB;
        size_t sh_hist = (size_t)K * sizeof(uint32_t);
        size_t sh_scat = ((size_t)K * RS_WARPS + (size_t)K + 32 + 2 * (size_t)RS_TILE) * sizeof(uint32_t);
        Digit dg;
        dg.div = div; dg.K = (uint32_t)K; dg.sh = 32; dg.mask = (uint32_t)K - 1;
        if ((K & (K - 1)) == 0) { dg.sh = 0; while ((1u << dg.sh) < div) dg.sh++; }
        dg.nbits = 0;
        while ((1u << dg.nbits) < (uint32_t)K) dg.nbits++;
        k_radix_hist<<<(unsigned)ntiles, RS_THREADS, sh_hist, st>>>(kin, N, nullptr, dg, hist, (uint32_t)ntiles);
        NF_LAUNCHED(ctx);
        NF_TRY(nf_exclusive_scan_u32(ctx, hist, hist, (size_t)K * ntiles, tmp32, st));
        NF_CUDA(ctx, cudaFuncSetAttribute(k_radix_scatter, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sh_scat));
        k_radix_scatter<<<(unsigned)ntiles, RS_THREADS, sh_scat, st>>>(kin, iin, N, nullptr, dg, hist, (uint32_t)ntiles, kout, iout);
        NF_LAUNCHED(ctx);
        kin = kout;
        iin = iout;
        div *= (uint32_t)K;
    }
    float hw = 0.5f * (box / (float)K);
    k_gather<<<(unsigned)((n + 256 * GA_PER - 1) / (256 * GA_PER)), 256, 0, st>>>(pos, mass, kin, perm, N, K, hw, plane_cx,
                                                                                   reinterpret_cast<float4 *>(pos_sorted), first, cell_count);
    NF_LAUNCHED(ctx);
    k_cell_counts<<<(unsigned)((ncell + 255) / 256), 256, 0, st>>>(cell_count, first, ncell);
    NF_LAUNCHED(ctx);
    return nf_exclusive_scan_u32_u64(ctx, cell_count, cell_offset, ncell, tmp64, st);
}
