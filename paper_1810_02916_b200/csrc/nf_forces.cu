// nf_forces.cu -- near-field interaction kernels.
//
// PAPER.md:37  every particle receives the direct pairwise sum of forces from all particles in
//              the cells within R of its own cell ((2R+1)^3 cells);
// PAPER.md:243 Eq. 2 compact spline, evaluated as min(10 - 15u + 6u^2, u^-3)/eps^3 (fn. 4, :239);
// PAPER.md:233 Eq. 1 Plummer;  PAPER.md:51 cell-centred float32 offsets.
//
// Two kernels:
//   k_forces_cell   -- general path (any K >= 2R+1): one block per sink cell, source cells
//                      staged through shared memory one at a time, sink shifted into each
//                      source cell's frame (d = o_j - (o_i - dc*w), the cell-centred form).
//   k_forces_pencil -- fast path (K >= 4R): see the block comment above it.
#include "nf_common.cuh"

namespace {

__device__ __forceinline__ float rsqrt_approx(float x)
{
    float y;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// Force-law constants in internal units.  Positions are multiplied by `scale` = 2^k (exact)
// with 2^k ~ 1/eps, so eps' = eps*scale lies in [2^-1/2, 2^1/2) and A, B, C are O(1..100)
// for every eps (SURVEY.md Sec. 7 hard part 4).  f(r') = min(A + r'^2 (C + B/r'), r'^-3).
struct ForceConsts {
    float A, B, C;      // 10/eps'^3, -15/eps'^4, 6/eps'^5   (spline)
    float r2_floor;     // addend of r'^2: tiny (spline; keeps r = 0 finite) or eps'^2 (Plummer)
    float eps2;         // eps'^2 (spline: below this the polynomial branch can win the min)
    float scale;        // 2^k
    float out_scale;    // Gm * scale^2: a = out_scale * sum f' d'
    int plummer;
};

// two-term compensated accumulation: (hi, lo) += x
__device__ __forceinline__ void comp_add(float &hi, float &lo, float x)
{
    float s = hi + x;
    float bb = s - hi;
    float err = (hi - (s - bb)) + (x - bb);
    hi = s;
    lo += err;
}

struct PlaneTable {
    const float4 *pos[1];  // flexible: n_planes entries follow in device memory
};

// ------------------------------------------------------------------------------------------
// General kernel.  grid = (K*K, sink planes); block = 128 threads; block handles sink cell
// (plane, cy, cz).  Sinks are processed 128 at a time, one per thread.
// ------------------------------------------------------------------------------------------
constexpr int CELL_THREADS = 128;

__global__ void __launch_bounds__(CELL_THREADS) k_forces_cell(const nf_plane_view *__restrict__ planes, nf_force_params p, ForceConsts fc)
{
    __shared__ float4 tile[CELL_THREADS];
    const int K = p.K, R = p.R;
    const int sink_plane = p.sink_lo + blockIdx.y;
    const int cyz = blockIdx.x;
    const int cy = cyz / K, cz = cyz % K;
    const nf_plane_view sp = planes[sink_plane];
    const uint64_t s0 = sp.off[cyz], s1 = sp.off[cyz + 1];
    if (s0 == s1) return;
    const float w = (p.box / (float)K) * fc.scale;

    for (uint64_t sb = s0; sb < s1; sb += CELL_THREADS) {
        const uint64_t si = sb + threadIdx.x;
        const bool active = si < s1;
        float4 me = active ? sp.pos[si] : make_float4(0.f, 0.f, 0.f, 0.f);
        const float xi = me.x * fc.scale, yi = me.y * fc.scale, zi = me.z * fc.scale;
        float ahx = 0.f, ahy = 0.f, ahz = 0.f, alx = 0.f, aly = 0.f, alz = 0.f;
        for (int dx = -R; dx <= R; dx++) {
            int px = sink_plane + dx;
            if (p.periodic_x) px = (px % p.n_planes + p.n_planes) % p.n_planes;
            else if (px < 0 || px >= p.n_planes) continue;
            const nf_plane_view qp = planes[px];
            const float xs = xi - (float)dx * w;  // sink in the source cell's frame
            for (int dy = -R; dy <= R; dy++) {
                const int qy = ((cy + dy) % K + K) % K;
                const float ys = yi - (float)dy * w;
                for (int dz = -R; dz <= R; dz++) {
                    const int qz = ((cz + dz) % K + K) % K;
                    const float zs = zi - (float)dz * w;
                    const uint64_t j0 = qp.off[qy * K + qz], j1 = qp.off[qy * K + qz + 1];
                    float ax = 0.f, ay = 0.f, az = 0.f;
                    for (uint64_t jb = j0; jb < j1; jb += CELL_THREADS) {
                        __syncthreads();
                        const uint64_t j = jb + threadIdx.x;
                        if (j < j1) {
                            float4 q = qp.pos[j];
                            tile[threadIdx.x] = make_float4(q.x * fc.scale, q.y * fc.scale, q.z * fc.scale, 0.f);
                        }
                        __syncthreads();
                        const int n = (int)min((uint64_t)CELL_THREADS, j1 - jb);
#pragma unroll 4
                        for (int t = 0; t < n; t++) {
                            const float4 q = tile[t];
                            const float ddx = q.x - xs, ddy = q.y - ys, ddz = q.z - zs;
                            float r2 = fmaf(ddz, ddz, fc.r2_floor);
                            r2 = fmaf(ddy, ddy, r2);
                            r2 = fmaf(ddx, ddx, r2);
                            const float ri = rsqrt_approx(r2);
                            float f = ri * ri * ri;
                            if (!fc.plummer) {
                                const float poly = fmaf(r2, fmaf(fc.B, ri, fc.C), fc.A);
                                f = fminf(poly, f);
                            }
                            ax = fmaf(f, ddx, ax);
                            ay = fmaf(f, ddy, ay);
                            az = fmaf(f, ddz, az);
                        }
                    }
                    comp_add(ahx, alx, ax);
                    comp_add(ahy, aly, ay);
                    comp_add(ahz, alz, az);
                }
            }
        }
        if (active && sp.acc) {
            const uint64_t o = sp.perm ? (uint64_t)sp.perm[si] : si;
            sp.acc[3 * o + 0] = (ahx + alx) * fc.out_scale;
            sp.acc[3 * o + 1] = (ahy + aly) * fc.out_scale;
            sp.acc[3 * o + 2] = (ahz + alz) * fc.out_scale;
        }
    }
}

// interactions: I = sum_c n_c * sum_{c' in N(c)} n_c' over a fully periodic K^3 box
__global__ void __launch_bounds__(256) k_interactions(const uint32_t *__restrict__ cnt, int K, int R, unsigned long long *out)
{
    const size_t ncell = (size_t)K * K * K;
    unsigned long long local = 0;
    for (size_t c = (size_t)blockIdx.x * blockDim.x + threadIdx.x; c < ncell; c += (size_t)gridDim.x * blockDim.x) {
        const unsigned long long n = cnt[c];
        if (n == 0) continue;
        const int cz = (int)(c % K), cy = (int)((c / K) % K), cx = (int)(c / ((size_t)K * K));
        unsigned long long m = 0;
        for (int dx = -R; dx <= R; dx++) {
            const int qx = ((cx + dx) % K + K) % K;
            for (int dy = -R; dy <= R; dy++) {
                const int qy = ((cy + dy) % K + K) % K;
                for (int dz = -R; dz <= R; dz++) {
                    const int qz = ((cz + dz) % K + K) % K;
                    m += cnt[((size_t)qx * K + qy) * K + qz];
                }
            }
        }
        local += n * m;
    }
    for (int d = 16; d > 0; d >>= 1) local += __shfl_down_sync(0xffffffffu, local, d);
    if ((threadIdx.x & 31) == 0 && local) atomicAdd(out, local);  // integer atomics: order-independent
}

__global__ void k_fill_planes(nf_plane_view *planes, int K, const float4 *pos, const uint64_t *off, const uint32_t *perm, float *acc)
{
    int cx = blockIdx.x * blockDim.x + threadIdx.x;
    if (cx >= K) return;
    nf_plane_view v;
    v.pos = pos;
    v.off = off + (size_t)cx * K * K;
    v.perm = perm;
    v.acc = acc;
    planes[cx] = v;
}

// ordered pairs for the sink planes of a plane table (counts from offset differences)
__global__ void __launch_bounds__(256) k_interactions_planes(const nf_plane_view *__restrict__ planes, nf_force_params p, unsigned long long *out)
{
    const int K = p.K, R = p.R;
    const int cyz = blockIdx.x * blockDim.x + threadIdx.x;
    const int sink_plane = p.sink_lo + blockIdx.y;
    unsigned long long local = 0;
    if (cyz < K * K) {
        const int cy = cyz / K, cz = cyz % K;
        const uint64_t *so = planes[sink_plane].off;
        const unsigned long long n = so[cyz + 1] - so[cyz];
        if (n) {
            unsigned long long m = 0;
            for (int dx = -R; dx <= R; dx++) {
                int px = sink_plane + dx;
                if (p.periodic_x) px = (px % p.n_planes + p.n_planes) % p.n_planes;
                else if (px < 0 || px >= p.n_planes) continue;
                const uint64_t *qo = planes[px].off;
                for (int dy = -R; dy <= R; dy++) {
                    const int qy = ((cy + dy) % K + K) % K;
                    for (int dz = -R; dz <= R; dz++) {
                        const int qz = ((cz + dz) % K + K) % K;
                        m += qo[qy * K + qz + 1] - qo[qy * K + qz];
                    }
                }
            }
            local = n * m;
        }
    }
    for (int d = 16; d > 0; d >>= 1) local += __shfl_down_sync(0xffffffffu, local, d);
    if ((threadIdx.x & 31) == 0 && local) atomicAdd(out, local);
}

ForceConsts make_consts(const nf_force_params &p)
{
    ForceConsts fc;
    int e;
    frexpf(p.eps, &e);                 // eps = m * 2^e, m in [0.5, 1)
    float scale = ldexpf(1.0f, -e);    // eps*scale in [0.5, 1)
    if (p.eps * scale < 0.70710678f) scale *= 2.0f;  // -> [0.7071, 1.4142)
    const double es = (double)p.eps * (double)scale;
    fc.scale = scale;
    fc.plummer = p.softening == NF_SOFT_PLUMMER;
    fc.A = (float)(10.0 / (es * es * es));
    fc.B = (float)(-15.0 / (es * es * es * es));
    fc.C = (float)(6.0 / (es * es * es * es * es));
    fc.eps2 = (float)(es * es);
    fc.r2_floor = fc.plummer ? fc.eps2 : 8.673617379884035e-19f;  // 2^-60
    fc.out_scale = (float)((double)p.Gm * (double)scale * (double)scale);
    return fc;
}

}  // namespace

size_t nf_forces_scratch_bytes(const nf_force_params &p)
{
    return nf_align_up((size_t)p.n_planes * sizeof(nf_plane_view), 256) + 4096;
}

int nf_fill_planes_full(nf_ctx *ctx, nf_plane_view *d_planes, int K, const float4 *pos, const uint64_t *off,
                        const uint32_t *perm, float *acc, cudaStream_t st)
{
    k_fill_planes<<<(K + 127) / 128, 128, 0, st>>>(d_planes, K, pos, off, perm, acc);
    NF_LAUNCHED(ctx);
    return NF_OK;
}

int nf_interactions_planes(nf_ctx *ctx, const nf_force_params &p, const nf_plane_view *d_planes, cudaStream_t st)
{
    const int n_sink_planes = p.sink_hi - p.sink_lo;
    if (n_sink_planes <= 0) return NF_OK;
    dim3 grid((unsigned)((p.K * p.K + 255) / 256), (unsigned)n_sink_planes);
    k_interactions_planes<<<grid, 256, 0, st>>>(d_planes, p, ctx->counters + 1);
    NF_LAUNCHED(ctx);
    return NF_OK;
}

int nf_forces_impl(nf_ctx *ctx, const nf_force_params &p, const nf_plane_view *d_planes,
                   cudaStream_t st, bool record_timing)
{
    if (record_timing) NF_CUDA(ctx, cudaEventRecord(ctx->ev_total0, st));
    const ForceConsts fc = make_consts(p);
    if (record_timing) NF_CUDA(ctx, cudaEventRecord(ctx->ev_kern0, st));
    const int n_sink_planes = p.sink_hi - p.sink_lo;
    if (n_sink_planes > 0) {
        dim3 grid((unsigned)(p.K * p.K), (unsigned)n_sink_planes);
        k_forces_cell<<<grid, CELL_THREADS, 0, st>>>(d_planes, p, fc);
        NF_LAUNCHED(ctx);
    }
    if (record_timing) {
        NF_CUDA(ctx, cudaEventRecord(ctx->ev_kern1, st));
        NF_CUDA(ctx, cudaEventRecord(ctx->ev_total1, st));
        ctx->forces_timed = true;
    }
    return NF_OK;
}

int nf_interactions_impl(nf_ctx *ctx, const uint32_t *cell_count, int K, int R, int64_t *out, cudaStream_t st)
{
    NF_CUDA(ctx, cudaMemsetAsync(ctx->counters + 1, 0, sizeof(unsigned long long), st));
    const size_t ncell = (size_t)K * K * K;
    unsigned blocks = (unsigned)min((size_t)ctx->sm_count * 8, (ncell + 255) / 256);
    k_interactions<<<blocks, 256, 0, st>>>(cell_count, K, R, ctx->counters + 1);
    NF_LAUNCHED(ctx);
    NF_CUDA(ctx, cudaMemcpyAsync(ctx->h_counters + 1, ctx->counters + 1, sizeof(unsigned long long), cudaMemcpyDeviceToHost, st));
    NF_CUDA(ctx, cudaStreamSynchronize(st));
    *out = (int64_t)ctx->h_counters[1];
    return NF_OK;
}
