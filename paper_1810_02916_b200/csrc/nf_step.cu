// nf_step.cu -- the steps either side of the near-field force in the slab pipeline
// (SURVEY.md Sec. 8(f) ranks 2-3): kick + drift (Table 1 "Kick", "Drift") and the
// velocity reductions of the time-step criteria.
//
// k_kick_drift   v <- v + a*kick ; x <- wrap(x + v*drift)       elementwise, HBM-bound (36 B / particle)
// k_cell_vrms    per-cell rms speed in the cell order of nf_bin + global max |v_axis|
#include "nf_common.cuh"

namespace {

// One thread per coordinate (3N of them): fully coalesced 4-byte streams.
// float32 contract: two single-rounded fused multiply-adds, then one
// periodic wrap -- v1 = fma(a, kick, v); x1 = fma(v1, drift, x); x1 >= box: x1 - box; x1 < 0:
// x1 + box; a result that rounds to box itself becomes 0.
__global__ void __launch_bounds__(256) k_kick_drift(float *__restrict__ pos, float *__restrict__ vel, const float *__restrict__ acc,
                                                    size_t n3, float kick, float drift, float box)
{
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n3) return;
    const float v1 = __fmaf_rn(acc[i], kick, vel[i]);
    float x1 = __fmaf_rn(v1, drift, pos[i]);
    if (x1 >= box) x1 = __fsub_rn(x1, box);
    else if (x1 < 0.0f) x1 = __fadd_rn(x1, box);
    if (!(x1 < box)) x1 = 0.0f;
    vel[i] = v1;
    pos[i] = x1;
}

// One warp per cell: lanes stride over the cell's sorted slots, fixed-order shuffle reduction
// (deterministic).  vmax: integer atomicMax on the bits of a non-negative float (exact).
__global__ void __launch_bounds__(256) k_cell_vrms(const float *__restrict__ vel, const uint32_t *__restrict__ perm,
                                                   const uint64_t *__restrict__ off, size_t ncell, float *__restrict__ vrms,
                                                   float *__restrict__ vmax)
{
    const size_t c = (size_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (c >= ncell) return;
    const int lane = threadIdx.x & 31;
    const uint64_t s0 = off[c], s1 = off[c + 1];
    float sum = 0.f, mx = 0.f;
    for (uint64_t s = s0 + lane; s < s1; s += 32) {
        const size_t i = perm ? (size_t)perm[s] : (size_t)s;
        const float vx = vel[3 * i], vy = vel[3 * i + 1], vz = vel[3 * i + 2];
        sum += vx * vx + vy * vy + vz * vz;
        mx = fmaxf(mx, fmaxf(fabsf(vx), fmaxf(fabsf(vy), fabsf(vz))));
    }
    for (int d = 16; d > 0; d >>= 1) {
        sum += __shfl_xor_sync(0xffffffffu, sum, d);
        mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, d));
    }
    if (lane == 0) {
        if (vrms) vrms[c] = s1 > s0 ? sqrtf(sum / (float)(s1 - s0)) : 0.f;
        if (vmax && mx > 0.f) atomicMax(reinterpret_cast<unsigned int *>(vmax), __float_as_uint(mx));
    }
}

}  // namespace

int nf_kick_drift_impl(nf_ctx *ctx, float *pos, float *vel, const float *acc, int64_t N, float kick, float drift, float box,
                       cudaStream_t st)
{
    if (N <= 0) return NF_OK;
    const size_t n3 = 3 * (size_t)N;
    k_kick_drift<<<(unsigned)((n3 + 255) / 256), 256, 0, st>>>(pos, vel, acc, n3, kick, drift, box);
    NF_LAUNCHED(ctx);
    return NF_OK;
}

int nf_kick_drift(nf_ctx *ctx, float *pos_xyz, float *vel_xyz, const float *acc_xyz, int64_t N, float kick, float drift,
                  float box, void *stream)
{
    if (!ctx) return NF_ERR_ARG;
    NF_ARG(ctx, N >= 0, "nf_kick_drift: N < 0");
    NF_ARG(ctx, N == 0 || (pos_xyz && vel_xyz && acc_xyz), "nf_kick_drift: null particle array with N > 0");
    NF_ARG(ctx, box > 0.0f && box < 3.0e38f, "box must be positive and finite");
    NF_ARG(ctx, kick == kick && drift == drift && fabsf(kick) < 3.0e38f && fabsf(drift) < 3.0e38f, "kick and drift must be finite");
    NF_CUDA(ctx, cudaSetDevice(ctx->device));
    return nf_kick_drift_impl(ctx, pos_xyz, vel_xyz, acc_xyz, N, kick, drift, box, (cudaStream_t)stream);
}

int nf_cell_vrms(nf_ctx *ctx, const float *vel_xyz, const uint32_t *perm, const uint64_t *cell_offset, int64_t N, int K,
                 float *cell_vrms, float *vmax, void *stream)
{
    if (!ctx) return NF_ERR_ARG;
    NF_ARG(ctx, N >= 0 && K >= 1 && K <= NF_MAX_K, "nf_cell_vrms: bad N or K");
    NF_ARG(ctx, cell_offset != nullptr, "nf_cell_vrms: cell_offset must not be null");
    NF_ARG(ctx, N == 0 || vel_xyz, "nf_cell_vrms: null velocity array with N > 0");
    NF_ARG(ctx, cell_vrms || vmax, "nf_cell_vrms: no output requested");
    NF_CUDA(ctx, cudaSetDevice(ctx->device));
    cudaStream_t st = (cudaStream_t)stream;
    const size_t ncell = (size_t)K * K * K;
    if (vmax) NF_CUDA(ctx, cudaMemsetAsync(vmax, 0, sizeof(float), st));
    k_cell_vrms<<<(unsigned)((ncell + 7) / 8), 256, 0, st>>>(vel_xyz, perm, cell_offset, ncell, cell_vrms, vmax);
    NF_LAUNCHED(ctx);
    return NF_OK;
}
