// nf_dense.cu -- in-cell spatial ordering of DENSE cells for the interaction kernel.
//
// PAPER.md:75 "the largest cell has over 200,000 particles" (the late-time, clustered state) and :107, where the paper
// reports its own slowdown there.  Inside such a cell every tile of sources holds pairs closer than eps to some of a
// task's sinks, so the whole own-cell sweep has to evaluate the min form of Eq. 2.  With the
// particles of the cell ordered along a space-filling curve (Hilbert's), 128 consecutive sinks and 446 consecutive sources are compact
// blobs, and a bounding box per 64 particles lets the kernel's producer PROVE that a (task, tile) pair holds no pair
// inside eps -- then the cheaper r^-3 sweep is exact (the two laws agree for r >= eps).
//
// Only the ENCODED copies (enc, enc_h: what the interaction kernel reads) are re-ordered; pos_sorted, perm and every
// output keep nf_bin's stable order.  `slot` maps an encoded position back to the sorted slot of its particle.
//
//   k_dense_mark     per cell: is it dense (>= NF_DENSE_N particles)?  rank and 64-aligned compact offset by two scans
//   k_dense_cells    which dense cells take part (capacity), their table by rank
//   k_dense_keys     per compact position: key = rank << 21 | 21-bit Hilbert index of the cell-centred offset, index = in-cell index
//   nf_radix_pass    4 stable LSD passes of 8 bits over the compact array (its length lives on the device)
//   k_dense_finish   encoded copies in the new order, slot map, one box per 64 compact positions
//
// Deterministic: ranks come from scans, the sort is stable, no atomic decides a position.
#include "nf_common.cuh"

namespace {

constexpr uint32_t PAD = 0xffffffffu;
constexpr uint32_t CURVE_BITS = 21, CURVE_MASK = (1u << CURVE_BITS) - 1;

using DenseCell = nf_dense_cell;

__device__ __forceinline__ uint32_t spread3(uint32_t v)      // 7 bits -> every third bit
{
    uint32_t r = 0;
#pragma unroll
    for (int b = 0; b < 7; b++) r |= ((v >> b) & 1u) << (3 * b);
    return r;
}

__global__ void __launch_bounds__(256) k_dense_mark(const uint64_t *__restrict__ off, size_t ncell, uint32_t *__restrict__ n64,
                                                    uint32_t *__restrict__ one)
{
    const size_t c = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= ncell) return;
    const uint64_t n = off[c + 1] - off[c];
    const bool d = n >= (uint64_t)NF_DENSE_N;
    n64[c] = d ? (uint32_t)((n + 63) & ~63ull) : 0u;
    one[c] = d ? 1u : 0u;
}

// 21-bit Hilbert index of a point of the 128^3 grid (J. Skilling, "Programming the Hilbert curve", AIP Conf. Proc. 707,
// 2004: the transpose construction, restated): consecutive indices are face-adjacent grid cells, so a run of consecutive
// particles is a compact blob -- a Morton run jumps across the cell wherever it crosses an octant boundary, and its
// bounding box with it.  Integer arithmetic only: part of the tree's definition (reading t2).
__device__ __forceinline__ uint32_t hilbert3(uint32_t x, uint32_t y, uint32_t z)
{
    uint32_t X[3] = {x, y, z};
    for (uint32_t Q = 64u; Q > 1u; Q >>= 1) {
        const uint32_t P = Q - 1u;
#pragma unroll
        for (int i = 0; i < 3; i++) {
            if (X[i] & Q) X[0] ^= P;                                    // invert the low bits of X[0]
            else { const uint32_t t = (X[0] ^ X[i]) & P; X[0] ^= t; X[i] ^= t; }   // exchange the low bits of X[0] and X[i]
        }
    }
    X[1] ^= X[0]; X[2] ^= X[1];                                       // Gray encode
    uint32_t t = 0;
    for (uint32_t Q = 64u; Q > 1u; Q >>= 1)
        if (X[2] & Q) t ^= Q - 1u;
    X[0] ^= t; X[1] ^= t; X[2] ^= t;
    return spread3(X[2]) | (spread3(X[1]) << 1) | (spread3(X[0]) << 2);
}

// one thread per cell.  coff / rank: exclusive scans of n64 / one.  A dense cell takes part while its rank and the end of its
// compact range stay below the limits (the cells that do form a prefix of the dense cells in cell order).
__global__ void __launch_bounds__(256) k_dense_cells(const uint64_t *__restrict__ off, size_t ncell, const uint32_t *__restrict__ n64,
                                                     const uint32_t *__restrict__ coff, const uint32_t *__restrict__ rank, uint32_t cap,
                                                     uint32_t *__restrict__ dinfo, DenseCell *__restrict__ dcell, uint32_t *__restrict__ nd)
{
    const size_t c = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= ncell) return;
    const uint32_t m = n64[c];
    const bool dense = m != 0 && rank[c] < (uint32_t)NF_DENSE_MAX_CELLS && (unsigned long long)coff[c] + m <= cap;
    dinfo[c] = dense ? (coff[c] >> 6) + 1u : 0u;
    if (!dense) return;
    DenseCell dc;
    dc.c0 = off[c]; dc.coff = coff[c]; dc.cell = (uint32_t)c; dc.n = (uint32_t)(off[c + 1] - off[c]); dc.pad = 0;
    dcell[rank[c]] = dc;
    atomicMax(nd, coff[c] + m);                  // integer: order-independent
    atomicAdd(nd + 1, 1u);                       // number of dense cells taken
}

// one thread per compact position: key = rank << 21 | Hilbert index of the cell-centred offset, index = in-cell index
__global__ void __launch_bounds__(256) k_dense_keys(const float4 *__restrict__ pos, const uint32_t *__restrict__ nd,
                                                    const DenseCell *__restrict__ dcell, uint32_t cap, float invw,
                                                    uint32_t *__restrict__ key, uint32_t *__restrict__ idx)
{
    const uint32_t n_d = nd[0], ndense = nd[1];
    for (uint32_t t = blockIdx.x * blockDim.x + threadIdx.x; t < n_d; t += gridDim.x * blockDim.x) {
        uint32_t lo = 0, hi = ndense;            // the dense cell this position belongs to: last rank with coff <= t
        while (hi - lo > 1) {
            const uint32_t mid = (lo + hi) >> 1;
            if (dcell[mid].coff <= t) lo = mid; else hi = mid;
        }
        const DenseCell dc = dcell[lo];
        const uint32_t j = t - dc.coff;
        uint32_t k = CURVE_MASK, i = PAD;       // padding sorts behind the cell's particles
        if (j < dc.n) {
            const float4 q = pos[dc.c0 + j];
            // every operation rounded to float32, no fused multiply-add: the order is part of the tree's definition
            // (reading t2) and the oracle takes the same decision in the same precision
            const int qx = min(127, max(0, (int)__fmul_rn(__fadd_rn(__fmul_rn(q.x, invw), 0.5f), 128.0f)));
            const int qy = min(127, max(0, (int)__fmul_rn(__fadd_rn(__fmul_rn(q.y, invw), 0.5f), 128.0f)));
            const int qz = min(127, max(0, (int)__fmul_rn(__fadd_rn(__fmul_rn(q.z, invw), 0.5f), 128.0f)));
            k = hilbert3((uint32_t)qx, (uint32_t)qy, (uint32_t)qz);
            i = j;
        }
        key[t] = (lo << CURVE_BITS) | k;
        idx[t] = i;
    }
    (void)cap;
}

// Cells of NF_DENSE_N particles or more that the ordering does NOT take (beyond its capacity; rare): nf_encode_impl left
// them out (skip_n), so their encoded copies are written here, in the binned order.  One warp per cell.
__global__ void __launch_bounds__(256) k_dense_left_out(const float4 *__restrict__ pos, const uint64_t *__restrict__ off, size_t ncell,
                                                        const uint32_t *__restrict__ dinfo, int K, float scale, float ws,
                                                        float4 *__restrict__ enc, float4 *__restrict__ enc_h)
{
    const size_t c = (size_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (c >= ncell) return;
    const uint64_t s0 = off[c], s1 = off[c + 1];
    if (s1 - s0 < (uint64_t)NF_DENSE_N || dinfo[c] != 0u) return;
    const int lane = threadIdx.x & 31;
    const int cz = (int)(c % (size_t)K);
    const float ez = ((float)(cz % NF_ZB) - 0.5f * (float)(NF_ZB - 1)) * ws;
    const float eh = ((float)((cz + NF_ZB / 2) % NF_ZB) - 0.5f * (float)(NF_ZB - 1)) * ws;
    for (uint64_t s = s0 + lane; s < s1; s += 32) {
        const float4 o = pos[s];
        const float x = o.x * scale, y = o.y * scale;
        enc[s] = make_float4(x, y, fmaf(o.z, scale, ez), o.w);
        enc_h[s] = make_float4(x, y, fmaf(o.z, scale, eh), o.w);
    }
}

// one warp per 64 compact positions (a "chunk"; cells start on chunk boundaries)
__global__ void __launch_bounds__(256) k_dense_finish(const float4 *__restrict__ pos, const uint32_t *__restrict__ key,
                                                      const uint32_t *__restrict__ idx, const uint32_t *__restrict__ nd,
                                                      const DenseCell *__restrict__ dcell, int K, float scale, float ws,
                                                      float4 *__restrict__ enc, float4 *__restrict__ enc_h,
                                                      uint32_t *__restrict__ slot, float *__restrict__ box, uint32_t nchunk_max)
{
    const int lane = threadIdx.x & 31;
    const uint32_t n_d = *nd;
    for (uint32_t ch = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5); ch < nchunk_max; ch += gridDim.x * (blockDim.x >> 5)) {
        const uint32_t t0 = ch * 64u;
        if (t0 >= n_d) return;
        const DenseCell dc = dcell[key[t0] >> CURVE_BITS];
        const int cz = (int)(dc.cell % (uint32_t)K);
        const float ez = ((float)(cz % NF_ZB) - 0.5f * (float)(NF_ZB - 1)) * ws;
        const float eh = ((float)((cz + NF_ZB / 2) % NF_ZB) - 0.5f * (float)(NF_ZB - 1)) * ws;
        float lo[3] = {3.0e38f, 3.0e38f, 3.0e38f}, hi[3] = {-3.0e38f, -3.0e38f, -3.0e38f};
#pragma unroll
        for (int h = 0; h < 2; h++) {
            const uint32_t t = t0 + 32u * h + lane;
            const uint32_t j = idx[t];
            uint32_t s = PAD;
            if (j != PAD) {
                const unsigned long long src = dc.c0 + j, dst = dc.c0 + (t - dc.coff);
                const float4 o = pos[src];
                const float x = o.x * scale, y = o.y * scale, z = o.z * scale;
                enc[dst] = make_float4(x, y, fmaf(o.z, scale, ez), o.w);
                enc_h[dst] = make_float4(x, y, fmaf(o.z, scale, eh), o.w);
                s = (uint32_t)src;
                lo[0] = fminf(lo[0], x); hi[0] = fmaxf(hi[0], x);
                lo[1] = fminf(lo[1], y); hi[1] = fmaxf(hi[1], y);
                lo[2] = fminf(lo[2], z); hi[2] = fmaxf(hi[2], z);
            }
            slot[t] = s;
        }
#pragma unroll
        for (int a = 0; a < 3; a++)
            for (int d = 16; d > 0; d >>= 1) {
                lo[a] = fminf(lo[a], __shfl_xor_sync(0xffffffffu, lo[a], d));
                hi[a] = fmaxf(hi[a], __shfl_xor_sync(0xffffffffu, hi[a], d));
            }
        if (lane == 0) {
            float *b = box + 6 * (size_t)ch;
            b[0] = lo[0]; b[1] = lo[1]; b[2] = lo[2]; b[3] = hi[0]; b[4] = hi[1]; b[5] = hi[2];
        }
    }
}

}  // namespace

// compact positions the ordering takes per call: room for every particle in 64-aligned cells (N + 64 per dense cell), at
// least 2^20 + 2^17, at most 2^28
uint32_t nf_dense_cap(int64_t N)
{
    const int64_t c = (N > (1 << 20) ? N : (1 << 20)) + 64ll * NF_DENSE_MAX_CELLS;
    return (uint32_t)(c < (1ll << 28) ? c : (1ll << 28)) & ~63u;
}

size_t nf_dense_scratch_bytes(int64_t N, size_t ncell)
{
    const size_t cap = nf_dense_cap(N);
    size_t b = 4 * nf_align_up(ncell * sizeof(uint32_t), 256);                                  // n64, one, coff, rank
    b += 2 * nf_align_up(nf_scan_temp_elems(ncell) * sizeof(uint32_t), 256);
    b += 3 * nf_align_up(cap * sizeof(uint32_t), 256);                                          // key ping-pong, one index buffer (the other is dslot)
    b += nf_align_up((size_t)NF_DENSE_MAX_CELLS * sizeof(DenseCell), 256) + 256;
    b += nf_align_up(256 * nf_radix_tiles(cap) * sizeof(uint32_t), 256);                        // digit histograms
    b += nf_align_up(nf_scan_temp_elems(256 * nf_radix_tiles(cap)) * sizeof(uint32_t), 256);
    return b + 4096;
}

int nf_dense_order_impl(nf_ctx *ctx, const nf_force_params &p, const float4 *pos, const uint64_t *off, size_t ncell, int64_t N,
                        float4 *enc, float4 *enc_h, uint32_t *dinfo, uint32_t *dslot, float *dbox, cudaStream_t st,
                        const nf_dense_keep *keep)
{
    const int K = p.K;
    const uint32_t cap = nf_dense_cap(N);
    uint32_t *n64 = nf_scratch_take<uint32_t>(ctx, ncell);
    uint32_t *one = nf_scratch_take<uint32_t>(ctx, ncell);
    uint32_t *coff = nf_scratch_take<uint32_t>(ctx, ncell);
    uint32_t *rank = nf_scratch_take<uint32_t>(ctx, ncell);
    uint32_t *stmp = nf_scratch_take<uint32_t>(ctx, nf_scan_temp_elems(ncell));
    uint32_t *keyA = nf_scratch_take<uint32_t>(ctx, cap), *keyB = nf_scratch_take<uint32_t>(ctx, cap);
    uint32_t *idxA = nf_scratch_take<uint32_t>(ctx, cap), *idxB = dslot;
    float *box = dbox;
    DenseCell *dcell = keep ? keep->dcell : nf_scratch_take<DenseCell>(ctx, NF_DENSE_MAX_CELLS);
    uint32_t *nd = keep ? keep->nd : nf_scratch_take<uint32_t>(ctx, 64);
    const size_t nt = nf_radix_tiles(cap);
    uint32_t *hist = nf_scratch_take<uint32_t>(ctx, 256 * nt);
    uint32_t *htmp = nf_scratch_take<uint32_t>(ctx, nf_scan_temp_elems(256 * nt));
    if (!n64 || !one || !coff || !rank || !dinfo || !stmp || !keyA || !keyB || !idxA || !idxB || !box || !dcell || !nd || !hist || !htmp) {
        NF_SET_ERR(ctx, "nf_forces: internal scratch arena too small (dense-cell ordering)");
        return NF_ERR_NOMEM;
    }
    float scale, ws;
    nf_encode_consts(p, &scale, &ws);
    NF_CUDA(ctx, cudaMemsetAsync(nd, 0, 2 * sizeof(uint32_t), st));
    k_dense_mark<<<(unsigned)((ncell + 255) / 256), 256, 0, st>>>(off, ncell, n64, one);
    NF_LAUNCHED(ctx);
    NF_TRY(nf_exclusive_scan_u32(ctx, n64, coff, ncell, stmp, st));
    NF_TRY(nf_exclusive_scan_u32(ctx, one, rank, ncell, stmp, st));
    k_dense_cells<<<(unsigned)((ncell + 255) / 256), 256, 0, st>>>(off, ncell, n64, coff, rank, cap, dinfo, dcell, nd);
    NF_LAUNCHED(ctx);
    k_dense_left_out<<<(unsigned)((ncell + 7) / 8), 256, 0, st>>>(pos, off, ncell, dinfo, K, scale, ws, enc, enc_h);
    NF_LAUNCHED(ctx);
    k_dense_keys<<<(unsigned)(cap / 256 < 148u * 8u ? (cap + 255) / 256 : 148u * 8u), 256, 0, st>>>(pos, nd, dcell, cap, (float)K / p.box, keyA, idxA);
    NF_LAUNCHED(ctx);
    NF_TRY(nf_radix_pass(ctx, keyA, idxA, cap, nd, 256, 0, keyB, idxB, hist, htmp, st));
    NF_TRY(nf_radix_pass(ctx, keyB, idxB, cap, nd, 256, 8, keyA, idxA, hist, htmp, st));
    NF_TRY(nf_radix_pass(ctx, keyA, idxA, cap, nd, 256, 16, keyB, idxB, hist, htmp, st));
    NF_TRY(nf_radix_pass(ctx, keyB, idxB, cap, nd, 256, 24, keyA, idxA, hist, htmp, st));
    const uint32_t nchunk = cap / 64;
    const unsigned grid = (unsigned)(nchunk / 8 < 148 * 16 ? (nchunk + 7) / 8 : 148 * 16);
    k_dense_finish<<<grid, 256, 0, st>>>(pos, keyA, idxA, nd, dcell, K, scale, ws, enc, enc_h, idxB, box, nchunk);
    NF_LAUNCHED(ctx);
    return NF_OK;
}
