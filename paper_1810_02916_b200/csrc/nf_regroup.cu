// nf_regroup.cu -- regrouping after the drift: the particles of one
// x-plane ("slab"), already kicked and drifted, are filed by the plane their NEW x
// coordinate maps to.  The third time-step criterion keeps every displacement below 80 % of a cell
// width ("particles drift by at most one slab per time step"), so a particle stays
// or moves to a neighbouring plane: the plane's arrays are rewritten as three stable segments
//     [ to plane-1 | stay | to plane+1 ]      (input order kept inside each segment)
// with their lengths, and the new content of plane d is  [ +1 segment of d-1 | stay of d | -1 of d+1 ].
//
//   k_regroup_count     code per particle (bit-exact cell formula of nf_bin) + per-block counts
//   (exclusive scan of the bin-major block counts: nf_scan.cu)
//   k_regroup_scatter   stable ranks from warp ballots, positions and velocities written out
// Deterministic: no atomic decides a slot.
#include "nf_common.cuh"

namespace {

constexpr int RG_THREADS = 256;
constexpr int RG_ROUNDS = 16;
constexpr int RG_TILE = RG_THREADS * RG_ROUNDS;

// 0: to plane-1, 1: stay, 2: to plane+1; bit 7: moved further than one plane (filed under the nearer neighbour)
__device__ __forceinline__ unsigned dest_code(float x, float invw, int K, int plane_cx)
{
    const float fl = floorf(__fmul_rn(x, invw));                 // the cell formula of include/nf.h (nf_bin)
    int c;
    if (!(fl >= 0.0f)) c = 0;
    else if (fl > (float)(K - 1)) c = K - 1;
    else c = (int)fl;
    const int rel = ((c - plane_cx) % K + K) % K;                // 0 stay, 1 up, K-1 down (K = 2: 1 is "up")
    if (rel == 0) return 1u;
    if (rel == 1) return 2u;
    if (rel == K - 1) return 0u;
    return (2 * rel <= K ? 2u : 0u) | 0x80u;
}

__global__ void __launch_bounds__(RG_THREADS) k_regroup_count(const float *__restrict__ pos, int64_t n, int K, float invw, int plane_cx,
                                                              unsigned char *__restrict__ code, uint32_t *__restrict__ blk_cnt,
                                                              uint32_t nblk, unsigned long long *__restrict__ n_bad)
{
    __shared__ uint32_t s_cnt[3];
    if (threadIdx.x < 3) s_cnt[threadIdx.x] = 0;
    __syncthreads();
    uint32_t c0 = 0, c1 = 0, c2 = 0, bad = 0;
    const int64_t base = (int64_t)blockIdx.x * RG_TILE;
#pragma unroll 4
    for (int r = 0; r < RG_ROUNDS; r++) {
        const int64_t i = base + (int64_t)r * RG_THREADS + threadIdx.x;
        if (i < n) {
            const unsigned d = dest_code(pos[3 * i], invw, K, plane_cx);
            code[i] = (unsigned char)(d & 3u);
            bad += d >> 7;
            c0 += (d & 3u) == 0u;
            c1 += (d & 3u) == 1u;
            c2 += (d & 3u) == 2u;
        }
    }
    for (int d = 16; d > 0; d >>= 1) {
        c0 += __shfl_xor_sync(0xffffffffu, c0, d);
        c1 += __shfl_xor_sync(0xffffffffu, c1, d);
        c2 += __shfl_xor_sync(0xffffffffu, c2, d);
        bad += __shfl_xor_sync(0xffffffffu, bad, d);
    }
    if ((threadIdx.x & 31) == 0) {            // integer adds: order-independent
        atomicAdd(&s_cnt[0], c0);
        atomicAdd(&s_cnt[1], c1);
        atomicAdd(&s_cnt[2], c2);
        if (bad) atomicAdd(n_bad, (unsigned long long)bad);
    }
    __syncthreads();
    if (threadIdx.x < 3) blk_cnt[(size_t)threadIdx.x * nblk + blockIdx.x] = s_cnt[threadIdx.x];
}

__global__ void __launch_bounds__(RG_THREADS) k_regroup_scatter(const float *__restrict__ pos, const float *__restrict__ vel,
                                                                const unsigned char *__restrict__ code, int64_t n,
                                                                const uint32_t *__restrict__ blk_off, uint32_t nblk,
                                                                float *__restrict__ pos_out, float *__restrict__ vel_out,
                                                                unsigned long long *__restrict__ seg_n)
{
    __shared__ uint32_t s_w[RG_THREADS / 32][3];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const unsigned lt = (1u << lane) - 1u;
    uint32_t run[3];
#pragma unroll
    for (int b = 0; b < 3; b++) run[b] = blk_off[(size_t)b * nblk + blockIdx.x];
    if (blockIdx.x == 0 && threadIdx.x == 0 && seg_n) {
        const uint32_t o1 = blk_off[nblk], o2 = blk_off[2 * (size_t)nblk];
        seg_n[0] = o1;
        seg_n[1] = o2 - o1;
        seg_n[2] = (unsigned long long)n - o2;
    }
    const int64_t base = (int64_t)blockIdx.x * RG_TILE;
    for (int r = 0; r < RG_ROUNDS; r++) {
        const int64_t i = base + (int64_t)r * RG_THREADS + threadIdx.x;
        const bool valid = i < n;
        const unsigned c = valid ? code[i] : 3u;
        const unsigned m0 = __ballot_sync(0xffffffffu, c == 0u), m1 = __ballot_sync(0xffffffffu, c == 1u),
                       m2 = __ballot_sync(0xffffffffu, c == 2u);
        if (lane == 0) { s_w[w][0] = __popc(m0); s_w[w][1] = __popc(m1); s_w[w][2] = __popc(m2); }
        __syncthreads();
        uint32_t before[3] = {0, 0, 0}, all[3] = {0, 0, 0};
#pragma unroll
        for (int ww = 0; ww < RG_THREADS / 32; ww++) {
#pragma unroll
            for (int b = 0; b < 3; b++) {
                const uint32_t t = s_w[ww][b];
                if (ww < w) before[b] += t;
                all[b] += t;
            }
        }
        if (valid) {
            const unsigned mine = c == 0u ? m0 : (c == 1u ? m1 : m2);
            const size_t dst = (size_t)run[c] + before[c] + __popc(mine & lt);
            const size_t s3 = 3 * (size_t)i, d3 = 3 * dst;
            pos_out[d3] = pos[s3]; pos_out[d3 + 1] = pos[s3 + 1]; pos_out[d3 + 2] = pos[s3 + 2];
            vel_out[d3] = vel[s3]; vel_out[d3 + 1] = vel[s3 + 1]; vel_out[d3 + 2] = vel[s3 + 2];
        }
#pragma unroll
        for (int b = 0; b < 3; b++) run[b] += all[b];
        __syncthreads();
    }
}

}  // namespace

size_t nf_regroup_scratch_bytes(int64_t N)
{
    const size_t n = (size_t)(N > 0 ? N : 1), nblk = (n + RG_TILE - 1) / RG_TILE;
    return nf_align_up(n, 256) + 2 * nf_align_up(3 * nblk * sizeof(uint32_t), 256) +
           nf_align_up(nf_scan_temp_elems(3 * nblk) * sizeof(uint32_t), 256) + 1024;
}

// pos, vel: the drifted particles of plane plane_cx (device, n x 3); pos_out, vel_out: the three segments;
// seg_n: 3 device counters (nullable).  Particles that moved further than one plane are counted in counters[0].
int nf_regroup_impl(nf_ctx *ctx, const float *pos, const float *vel, int64_t n, int K, float box, int plane_cx, float *pos_out,
                    float *vel_out, unsigned long long *seg_n, cudaStream_t st)
{
    if (n <= 0) {
        if (seg_n) NF_CUDA(ctx, cudaMemsetAsync(seg_n, 0, 3 * sizeof(unsigned long long), st));
        return NF_OK;
    }
    const size_t nblk = ((size_t)n + RG_TILE - 1) / RG_TILE;
    unsigned char *code = nf_scratch_take<unsigned char>(ctx, (size_t)n);
    uint32_t *cnt = nf_scratch_take<uint32_t>(ctx, 3 * nblk);
    uint32_t *off = nf_scratch_take<uint32_t>(ctx, 3 * nblk);
    uint32_t *tmp = nf_scratch_take<uint32_t>(ctx, nf_scan_temp_elems(3 * nblk));
    if (!code || !cnt || !off || !tmp) {
        NF_SET_ERR(ctx, "nf_regroup: internal scratch arena too small");
        return NF_ERR_NOMEM;
    }
    const float invw = (float)K / box;
    k_regroup_count<<<(unsigned)nblk, RG_THREADS, 0, st>>>(pos, n, K, invw, plane_cx, code, cnt, (uint32_t)nblk, ctx->counters);
    NF_LAUNCHED(ctx);
    NF_TRY(nf_exclusive_scan_u32(ctx, cnt, off, 3 * nblk, tmp, st));
    k_regroup_scatter<<<(unsigned)nblk, RG_THREADS, 0, st>>>(pos, vel, code, n, off, (uint32_t)nblk, pos_out, vel_out, seg_n);
    NF_LAUNCHED(ctx);
    return NF_OK;
}

extern "C" int nf_regroup_plane(nf_ctx *ctx, const float *pos_xyz, const float *vel_xyz, int64_t N, int K, float box, int plane_cx,
                                float *pos_out, float *vel_out, int64_t *seg_n, void *stream)
{
    if (!ctx) return NF_ERR_ARG;
    NF_ARG(ctx, N >= 0 && N < ((int64_t)1 << 32), "nf_regroup_plane: N = %lld out of range [0, 2^32)", (long long)N);
    NF_ARG(ctx, K >= 1 && K <= NF_MAX_K, "K = %d out of range [1, %d]", K, NF_MAX_K);
    NF_ARG(ctx, box > 0.0f && box < 3.0e38f, "box must be positive and finite");
    NF_ARG(ctx, plane_cx >= 0 && plane_cx < K, "plane_cx = %d outside [0, K)", plane_cx);
    NF_ARG(ctx, seg_n != nullptr, "nf_regroup_plane: seg_n must not be null");
    NF_ARG(ctx, N == 0 || (pos_xyz && vel_xyz && pos_out && vel_out), "nf_regroup_plane: null particle array with N > 0");
    NF_ARG(ctx, N == 0 || (pos_xyz != pos_out && vel_xyz != vel_out), "nf_regroup_plane: outputs must not alias the inputs");
    NF_CUDA(ctx, cudaSetDevice(ctx->device));
    NF_TRY(nf_scratch_reserve(ctx, nf_regroup_scratch_bytes(N)));
    nf_scratch_reset(ctx);
    cudaStream_t st = (cudaStream_t)stream;
    NF_CUDA(ctx, cudaMemsetAsync(ctx->counters, 0, sizeof(unsigned long long), st));
    NF_TRY(nf_regroup_impl(ctx, pos_xyz, vel_xyz, N, K, box, plane_cx, pos_out, vel_out, ctx->counters + 4, st));
    NF_CUDA(ctx, cudaMemcpyAsync(ctx->h_counters + 4, ctx->counters + 4, 3 * sizeof(unsigned long long), cudaMemcpyDeviceToHost, st));
    NF_CUDA(ctx, cudaMemcpyAsync(ctx->h_counters, ctx->counters, sizeof(unsigned long long), cudaMemcpyDeviceToHost, st));
    NF_CUDA(ctx, cudaStreamSynchronize(st));
    for (int b = 0; b < 3; b++) seg_n[b] = (int64_t)ctx->h_counters[4 + b];
    if (ctx->h_counters[0]) {
        NF_SET_ERR(ctx, "%lld particle(s) moved further than one plane (time-step criterion 3, PAPER.md:195)", (long long)ctx->h_counters[0]);
        return NF_ERR_RANGE;
    }
    return NF_OK;
}
