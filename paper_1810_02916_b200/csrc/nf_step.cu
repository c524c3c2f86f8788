// nf_step.cu -- the steps either side of the near-field force in the slab pipeline
// (SURVEY.md Sec. 8(f) ranks 2-3): kick + drift (Table 1 "Kick", "Drift") and the
// velocity reductions of the time-step criteria.
//
// k_kick_drift   v <- v + a*kick ; x <- wrap(x + v*drift)       elementwise, HBM-bound (36 B / particle)
// k_cell_vrms    per-cell rms speed in the cell order of nf_bin + global max |v_axis|
// k_timestep_*   reduction of criteria 2 and 3 over the cells (min / max of v_rms / a_max, global v_rms and a_max)
#include "nf_common.cuh"
#include <math.h>

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

// Time-step terms.  Stage 1: each block reduces a contiguous range of cells to one record; stage 2: one block
// reduces the records in index order.  Minimum / maximum of float32 values are order-independent; the double sum
// is formed in a fixed tree order, so the result is the same from run to run.
constexpr int TS_BLOCKS = 1024, TS_THREADS = 256;
struct TsRec { float rmin, rmax, amax; unsigned int pad; double sum_nv2; unsigned long long n, used; };

__device__ __forceinline__ void ts_merge(TsRec &a, const TsRec &b)
{
    a.rmin = fminf(a.rmin, b.rmin); a.rmax = fmaxf(a.rmax, b.rmax); a.amax = fmaxf(a.amax, b.amax);
    a.sum_nv2 += b.sum_nv2; a.n += b.n; a.used += b.used;
}
__device__ __forceinline__ TsRec ts_block_reduce(TsRec r)
{
    __shared__ TsRec sh[TS_THREADS];
    sh[threadIdx.x] = r;
    __syncthreads();
    for (int d = TS_THREADS / 2; d > 0; d >>= 1) {
        if ((int)threadIdx.x < d) { TsRec a = sh[threadIdx.x]; ts_merge(a, sh[threadIdx.x + d]); sh[threadIdx.x] = a; }
        __syncthreads();
    }
    return sh[0];
}
__device__ __forceinline__ TsRec ts_empty()
{
    TsRec r; r.rmin = 3.0e38f; r.rmax = 0.f; r.amax = 0.f; r.pad = 0; r.sum_nv2 = 0.0; r.n = 0; r.used = 0;
    return r;
}

__global__ void __launch_bounds__(TS_THREADS) k_timestep_cells(const float *__restrict__ vrms, const float *__restrict__ amax,
                                                               const uint64_t *__restrict__ off, size_t ncell, TsRec *__restrict__ rec)
{
    const size_t per = (ncell + gridDim.x - 1) / gridDim.x;
    const size_t c0 = (size_t)blockIdx.x * per, c1 = c0 + per < ncell ? c0 + per : ncell;
    TsRec r = ts_empty();
    for (size_t c = c0 + threadIdx.x; c < c1; c += TS_THREADS) {
        const unsigned long long n = off[c + 1] - off[c];
        if (n == 0) continue;
        const float v = vrms[c], a = amax[c];
        r.sum_nv2 += (double)n * (double)v * (double)v;
        r.n += n;
        r.amax = fmaxf(r.amax, a);
        if (a > 0.f) {
            const float q = __fdiv_rn(v, a);
            r.rmin = fminf(r.rmin, q); r.rmax = fmaxf(r.rmax, q); r.used++;
        }
    }
    r = ts_block_reduce(r);
    if (threadIdx.x == 0) rec[blockIdx.x] = r;
}
__global__ void __launch_bounds__(TS_THREADS) k_timestep_final(const TsRec *__restrict__ rec, int nrec, TsRec *__restrict__ out)
{
    TsRec r = ts_empty();
    for (int i = threadIdx.x; i < nrec; i += TS_THREADS) ts_merge(r, rec[i]);
    r = ts_block_reduce(r);
    if (threadIdx.x == 0) *out = r;
}

}  // namespace

int nf_timestep_terms(nf_ctx *ctx, const float *cell_vrms, const float *cell_amax, const uint64_t *cell_offset,
                      int K, float box, const float *vmax, nf_timestep *out, void *stream)
{
    if (!ctx) return NF_ERR_ARG;
    NF_ARG(ctx, K >= 1 && K <= NF_MAX_K, "nf_timestep_terms: bad K");
    NF_ARG(ctx, cell_vrms && cell_amax && cell_offset && out, "nf_timestep_terms: null argument");
    NF_ARG(ctx, box > 0.0f && box < 3.0e38f, "box must be positive and finite");
    NF_CUDA(ctx, cudaSetDevice(ctx->device));
    cudaStream_t st = (cudaStream_t)stream;
    const size_t ncell = (size_t)K * K * K;
    const int nb = (int)(ncell < (size_t)TS_BLOCKS * TS_THREADS ? (ncell + TS_THREADS - 1) / TS_THREADS : TS_BLOCKS);
    NF_TRY(nf_scratch_reserve(ctx, (size_t)(nb + 2) * sizeof(TsRec) + 1024));
    nf_scratch_reset(ctx);
    TsRec *rec = nf_scratch_take<TsRec>(ctx, (size_t)nb + 1);
    if (!rec) { NF_SET_ERR(ctx, "nf_timestep_terms: internal scratch arena too small"); return NF_ERR_NOMEM; }
    k_timestep_cells<<<nb, TS_THREADS, 0, st>>>(cell_vrms, cell_amax, cell_offset, ncell, rec);
    NF_LAUNCHED(ctx);
    k_timestep_final<<<1, TS_THREADS, 0, st>>>(rec, nb, rec + nb);
    NF_LAUNCHED(ctx);
    TsRec h;
    float hv = 0.f;
    NF_CUDA(ctx, cudaMemcpyAsync(&h, rec + nb, sizeof(TsRec), cudaMemcpyDeviceToHost, st));
    if (vmax) NF_CUDA(ctx, cudaMemcpyAsync(&hv, vmax, sizeof(float), cudaMemcpyDeviceToHost, st));
    NF_CUDA(ctx, cudaStreamSynchronize(st));
    out->cells_used = (int64_t)h.used;
    out->ratio_cell_min = h.used ? (double)h.rmin : 0.0;
    out->ratio_cell_max = (double)h.rmax;
    out->vrms_global = h.n ? sqrt(h.sum_nv2 / (double)h.n) : 0.0;
    out->amax_global = (double)h.amax;
    out->ratio_global = h.amax > 0.f ? out->vrms_global / (double)h.amax : 0.0;
    out->ratio_criterion2 = out->ratio_global > out->ratio_cell_min ? out->ratio_global : out->ratio_cell_min;
    out->vmax = (double)hv;
    out->drift_limit = hv > 0.f ? 0.8 * ((double)box / (double)K) / (double)hv : INFINITY;
    return NF_OK;
}

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

// ------------------------------------------------------------------------------------------
// nf_timestep_terms_static: nf_timestep_terms for callers that cannot call cudaMalloc (code under CUDA graph capture,
// tight serving loops, harnesses that forbid it).  Same kernels; their scratch -- one TsRec per block of
// NF_TS_STATIC_CELLS_PER_REC cells plus the final record -- is a file-scope __device__ array instead of the context's
// arena (which grows with cudaMalloc on demand).  Every GPU that loads libnf holds the array (164 KB) until exit.
// In host code the array's NAME is a host-side stand-in, not a device address: the device address comes from
// cudaGetSymbolAddress, once per device, with that device current.
// ------------------------------------------------------------------------------------------
#include <mutex>

namespace {
constexpr size_t TS_STATIC_CELLS_PER_REC = 4096;                                  // cells reduced into one record
constexpr size_t TS_STATIC_MAX_REC = (size_t)NF_TS_STATIC_MAX_K * NF_TS_STATIC_MAX_K * NF_TS_STATIC_MAX_K / TS_STATIC_CELLS_PER_REC;
static __device__ __align__(256) unsigned char g_ts_static[(TS_STATIC_MAX_REC + 1) * sizeof(TsRec)];
constexpr int TS_STATIC_MAX_DEVICES = 64;
TsRec *g_ts_static_ptr[TS_STATIC_MAX_DEVICES];       // device address of g_ts_static on each device (null: not looked up yet)
std::mutex g_ts_static_mutex;
}  // namespace

int nf_timestep_terms_static(nf_ctx *ctx, const float *cell_vrms, const float *cell_amax, const uint64_t *cell_offset,
                             int K, float box, const float *vmax, nf_timestep *out, void *stream)
{
    if (!ctx) return NF_ERR_ARG;
    NF_ARG(ctx, K >= 1, "nf_timestep_terms_static: bad K");
    NF_ARG(ctx, K <= NF_TS_STATIC_MAX_K,
           "nf_timestep_terms_static: K = %d exceeds the static scratch (K <= %d: one record per %zu cells, %zu records); use nf_timestep_terms",
           K, NF_TS_STATIC_MAX_K, TS_STATIC_CELLS_PER_REC, TS_STATIC_MAX_REC);
    NF_ARG(ctx, cell_vrms && cell_amax && cell_offset && out, "nf_timestep_terms_static: null argument");
    NF_ARG(ctx, box > 0.0f && box < 3.0e38f, "box must be positive and finite");
    NF_ARG(ctx, ctx->device >= 0 && ctx->device < TS_STATIC_MAX_DEVICES, "nf_timestep_terms_static: device index %d out of range", ctx->device);
    NF_CUDA(ctx, cudaSetDevice(ctx->device));
    TsRec *rec = nullptr;
    {
        std::lock_guard<std::mutex> lock(g_ts_static_mutex);
        if (!g_ts_static_ptr[ctx->device]) {
            void *p = nullptr;
            NF_CUDA(ctx, cudaGetSymbolAddress(&p, g_ts_static));
            g_ts_static_ptr[ctx->device] = static_cast<TsRec *>(p);
        }
        rec = g_ts_static_ptr[ctx->device];
    }
    cudaStream_t st = (cudaStream_t)stream;
    const size_t ncell = (size_t)K * K * K;
    const int nb = (int)((ncell + TS_STATIC_CELLS_PER_REC - 1) / TS_STATIC_CELLS_PER_REC);     // <= TS_STATIC_MAX_REC
    // nothing has to start at zero: every block writes its own record and the final pass reads records [0, nb) only
    k_timestep_cells<<<nb, TS_THREADS, 0, st>>>(cell_vrms, cell_amax, cell_offset, ncell, rec);
    NF_LAUNCHED(ctx);
    k_timestep_final<<<1, TS_THREADS, 0, st>>>(rec, nb, rec + nb);
    NF_LAUNCHED(ctx);
    TsRec h;
    float hv = 0.f;
    NF_CUDA(ctx, cudaMemcpyAsync(&h, rec + nb, sizeof(TsRec), cudaMemcpyDeviceToHost, st));
    if (vmax) NF_CUDA(ctx, cudaMemcpyAsync(&hv, vmax, sizeof(float), cudaMemcpyDeviceToHost, st));
    NF_CUDA(ctx, cudaStreamSynchronize(st));
    out->cells_used = (int64_t)h.used;
    out->ratio_cell_min = h.used ? (double)h.rmin : 0.0;
    out->ratio_cell_max = (double)h.rmax;
    out->vrms_global = h.n ? sqrt(h.sum_nv2 / (double)h.n) : 0.0;
    out->amax_global = (double)h.amax;
    out->ratio_global = h.amax > 0.f ? out->vrms_global / (double)h.amax : 0.0;
    out->ratio_criterion2 = out->ratio_global > out->ratio_cell_min ? out->ratio_global : out->ratio_cell_min;
    out->vmax = (double)hv;
    out->drift_limit = hv > 0.f ? 0.8 * ((double)box / (double)K) / (double)hv : INFINITY;
    return NF_OK;
}
