// nf_forces.cu -- near-field interaction kernels.
//
// PAPER.md:37  every particle receives the direct pairwise sum of forces from all particles in
//              the cells within R of its own cell ((2R+1)^3 cells);
// PAPER.md:243 Eq. 2 compact spline, evaluated as min(10 - 15u + 6u^2, u^-3)/eps^3 (fn. 4, :239);
// PAPER.md:233 Eq. 1 Plummer;  PAPER.md:51 cell-centred float32 offsets.
//
// k_task_count / k_task_fill build the work list (chunks of <= 256 sinks of one cell);
// k_forces_tile is the interaction kernel (see the block comment above it).
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

// ------------------------------------------------------------------------------------------
// Packed FP32 (sm_100 FFMA2 / FADD2 / FMUL2): one 64-bit register holds the same quantity for
// TWO SINKS; the source coordinate is a scalar operand broadcast to both halves (ptxas emits
// the .F32 broadcast operand form, so no duplicating moves).  13 (spline) or 11 (r^-3 only)
// FMA-pipe instructions per source serve two interactions per lane.
// ------------------------------------------------------------------------------------------
typedef unsigned long long u64;
__device__ __forceinline__ u64 pk(float a, float b) { u64 r; asm("mov.b64 %0, {%1,%2};" : "=l"(r) : "f"(a), "f"(b)); return r; }
__device__ __forceinline__ void upk(u64 r, float &a, float &b) { asm("mov.b64 {%0,%1}, %2;" : "=f"(a), "=f"(b) : "l"(r)); }
__device__ __forceinline__ u64 fma2(u64 a, u64 b, u64 c) { u64 d; asm("fma.rn.ftz.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c)); return d; }
__device__ __forceinline__ u64 sub2(u64 a, u64 b) { u64 d; asm("sub.rn.ftz.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d; }
__device__ __forceinline__ u64 mul2(u64 a, u64 b) { u64 d; asm("mul.rn.ftz.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d; }

// One source against the lane's two sinks.  MODE 0: spline, min(poly, r^-3); 1: r^-3 only
// (valid when the cell separation guarantees r >= eps, or for Plummer where r2_floor = eps^2).
template <int MODE>
__device__ __forceinline__ void interact(const float4 q, const u64 xs, const u64 ys, const u64 zs, const ForceConsts &fc,
                                         u64 &ax, u64 &ay, u64 &az)
{
    const u64 dx = sub2(pk(q.x, q.x), xs), dy = sub2(pk(q.y, q.y), ys), dz = sub2(pk(q.z, q.z), zs);
    u64 r2 = fma2(dz, dz, pk(fc.r2_floor, fc.r2_floor));
    r2 = fma2(dy, dy, r2);
    r2 = fma2(dx, dx, r2);
    float r2a, r2b;
    upk(r2, r2a, r2b);
    const u64 ri = pk(rsqrt_approx(r2a), rsqrt_approx(r2b));
    u64 f = mul2(mul2(ri, ri), ri);
    if (MODE == 0) {
        const u64 poly = fma2(r2, fma2(pk(fc.B, fc.B), ri, pk(fc.C, fc.C)), pk(fc.A, fc.A));
        float pa, pb, fa, fb;
        upk(poly, pa, pb);
        upk(f, fa, fb);
        f = pk(fminf(pa, fa), fminf(pb, fb));
    }
    ax = fma2(f, dx, ax);
    ay = fma2(f, dy, ay);
    az = fma2(f, dz, az);
}

// q (a multiple of 4, >= 4) consecutive sources against the lane's two sinks; the loads of the
// next group of four are issued before the arithmetic of the current one.
template <int MODE>
__device__ __forceinline__ void run_sources(const float4 *__restrict__ src, int q, const u64 xs, const u64 ys, const u64 zs,
                                            const ForceConsts &fc, u64 &ax, u64 &ay, u64 &az)
{
    const float4 *end = src + q;
    float4 a0 = src[0], a1 = src[1], a2 = src[2], a3 = src[3];
    src += 4;
#pragma unroll 1
    while (src < end) {
        const float4 b0 = src[0], b1 = src[1], b2 = src[2], b3 = src[3];
        src += 4;
        interact<MODE>(a0, xs, ys, zs, fc, ax, ay, az);
        interact<MODE>(a1, xs, ys, zs, fc, ax, ay, az);
        interact<MODE>(a2, xs, ys, zs, fc, ax, ay, az);
        interact<MODE>(a3, xs, ys, zs, fc, ax, ay, az);
        a0 = b0; a1 = b1; a2 = b2; a3 = b3;
    }
    interact<MODE>(a0, xs, ys, zs, fc, ax, ay, az);
    interact<MODE>(a1, xs, ys, zs, fc, ax, ay, az);
    interact<MODE>(a2, xs, ys, zs, fc, ax, ay, az);
    interact<MODE>(a3, xs, ys, zs, fc, ax, ay, az);
}

// ------------------------------------------------------------------------------------------
// Work list.  A task is a chunk of <= TILE_SINKS consecutive sinks of ONE cell of a sink plane.
// ------------------------------------------------------------------------------------------
constexpr int TILE_T = 128;                 // threads per block
constexpr int TILE_SINKS = 2 * TILE_T;      // sinks per task at most (two per lane, one phase)
constexpr int TILE_CAP = 2048;              // float4 slots of the source buffer (32 KiB)

struct Task {
    uint32_t cyz;     // cell index within the plane, cy*K + cz
    uint16_t plane;   // sink plane (index into the plane table)
    uint16_t chunk;   // chunk of TILE_SINKS sinks within the cell
};

__global__ void __launch_bounds__(256) k_task_count(const nf_plane_view *__restrict__ planes, nf_force_params p, uint32_t *__restrict__ tc)
{
    const int cyz = blockIdx.x * blockDim.x + threadIdx.x;
    if (cyz >= p.K * p.K) return;
    const uint64_t *off = planes[p.sink_lo + blockIdx.y].off;
    const uint64_t n = off[cyz + 1] - off[cyz];
    tc[(size_t)blockIdx.y * p.K * p.K + cyz] = (uint32_t)((n + TILE_SINKS - 1) / TILE_SINKS);
}

// ctl[0] = work cursor (zeroed here), ctl[1] = number of tasks
__global__ void __launch_bounds__(256) k_task_fill(const uint32_t *__restrict__ tc, const uint32_t *__restrict__ to, nf_force_params p,
                                                   Task *__restrict__ tasks, uint32_t *__restrict__ ctl)
{
    const int cyz = blockIdx.x * blockDim.x + threadIdx.x;
    const int KK = p.K * p.K;
    if (cyz >= KK) return;
    const size_t c = (size_t)blockIdx.y * KK + cyz;
    const uint32_t n = tc[c], o = to[c];
    for (uint32_t k = 0; k < n; k++) {
        Task t;
        t.cyz = (uint32_t)cyz;
        t.plane = (uint16_t)(p.sink_lo + blockIdx.y);
        t.chunk = (uint16_t)k;
        tasks[o + k] = t;
    }
    if (cyz == KK - 1 && blockIdx.y == gridDim.y - 1) {
        ctl[0] = 0;
        ctl[1] = o + n;
    }
}

// ------------------------------------------------------------------------------------------
// Interaction kernel.  Persistent blocks of TILE_T threads pull tasks from the work list.
//
// Task = n <= 256 sinks of cell (plane, cy, cz).  Lane mapping: L = ceil(n/2) "sink lanes"
// each hold two sinks in packed registers; the P = floor(T/L) "phases" split every source run
// between them, so small cells still fill the block (lane use L*P/T).  For each of the
// (2R+1)^2 source columns (dx, dy) the 2R+1 cells cz-R..cz+R form one z-run (contiguous in
// memory because z is the fastest cell index; the periodic wrap splits it).  A run of m sources
// is staged into shared memory as P slices of q = roundup4(ceil(m/P)) slots, already multiplied
// by `scale` and with the z shift of its cell added, so that same-cell differences stay exact
// (PAPER.md:51); unused slots hold a far-away sentinel (zero force).  Several runs are staged
// per pass (as many as fit the buffer), then every phase sweeps its slice of each run.
// float32 partial sums per run, double outer sum over runs and phases; no atomics on floats.
// ------------------------------------------------------------------------------------------
template <int R>
struct TaskTab {
    static constexpr int W = 2 * R + 1;
    uint32_t start[W * W][W];    // first particle of each cell segment, relative to its plane's arrays
    int cum[W * W][W + 1];       // particles of the run before segment s; cum[r][W] = m_r
    int px[W * W];               // plane of the run (-1: outside the open chunk)
    int q[W * W];                // padded slice length of the run for this task's P
};

template <int R>
__global__ void __launch_bounds__(TILE_T, 6) k_forces_tile(const nf_plane_view *__restrict__ planes, const nf_force_params p, const ForceConsts fc,
                                                           const Task *__restrict__ tasks, uint32_t *__restrict__ ctl)
{
    constexpr int W = 2 * R + 1, NR = W * W;
    __shared__ __align__(16) float4 buf[TILE_CAP];
    __shared__ TaskTab<R> tab;
    __shared__ uint32_t s_task;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int K = p.K;
    const float w = (p.box / (float)K) * fc.scale;
    const float4 SENT = make_float4(1.0e15f, 1.0e15f, 1.0e15f, 0.f);   // r2 ~ 1e30: r^-3 flushes to zero
    const bool far_ok = !fc.plummer && w > 1.001f * sqrtf(fc.eps2);

    for (;;) {
        __syncthreads();
        if (tid == 0) s_task = atomicAdd(&ctl[0], 1u);
        __syncthreads();
        const uint32_t ti = s_task;
        if (ti >= ctl[1]) return;
        const Task task = tasks[ti];
        const int sink_plane = task.plane;
        const int cy = (int)(task.cyz / (uint32_t)K), cz = (int)(task.cyz % (uint32_t)K);
        const nf_plane_view sp = planes[sink_plane];
        const uint64_t c0 = sp.off[task.cyz], c1 = sp.off[task.cyz + 1];
        const uint64_t s0 = c0 + (uint64_t)task.chunk * TILE_SINKS;
        const int n = (int)min((uint64_t)TILE_SINKS, c1 - s0);
        const int L = (n + 1) >> 1;
        const int P = TILE_T / L;
        const int sl = tid % L, ph = tid / L;
        const bool active = ph < P;

        // ---- segment table of the task: (run, cell of the z-window) -> start, count ----
        for (int e = tid; e < NR * W; e += TILE_T) {
            const int r = e / W, s = e - r * W;
            const int dx = r / W - R, dy = r - (r / W) * W - R;
            int px = sink_plane + dx;
            if (p.periodic_x) px = (px % p.n_planes + p.n_planes) % p.n_planes;
            else if (px < 0 || px >= p.n_planes) px = -1;
            uint32_t st = 0;
            int cnt = 0;
            if (px >= 0) {
                const int qy = ((cy + dy) % K + K) % K, qz = ((cz + s - R) % K + K) % K;
                const uint64_t *qo = planes[px].off + (size_t)qy * K + qz;
                st = (uint32_t)qo[0];
                cnt = (int)(qo[1] - qo[0]);
            }
            tab.start[r][s] = st;
            tab.cum[r][s + 1] = cnt;      // counts first, prefix-summed below
            if (s == 0) tab.px[r] = px;
        }
        // the lane's two sinks (the second is a duplicate of the first when n is odd)
        const uint64_t i0 = s0 + 2 * (uint64_t)sl;
        const uint64_t i1 = (2 * sl + 1 < n) ? i0 + 1 : i0;
        const float4 m0 = sp.pos[i0], m1 = sp.pos[i1];
        const u64 xi = pk(m0.x * fc.scale, m1.x * fc.scale), yi = pk(m0.y * fc.scale, m1.y * fc.scale),
                  zi = pk(m0.z * fc.scale, m1.z * fc.scale);
        double ax0 = 0.0, ay0 = 0.0, az0 = 0.0, ax1 = 0.0, ay1 = 0.0, az1 = 0.0;
        __syncthreads();
        if (tid < NR) {
            int c = 0;
            tab.cum[tid][0] = 0;
#pragma unroll
            for (int s = 1; s <= W; s++) { c += tab.cum[tid][s]; tab.cum[tid][s] = c; }
            tab.q[tid] = ((c + P - 1) / P + 3) & ~3;
        }
        __syncthreads();

        // padded slice length of a run of m sources
        auto slice = [&](int m) { return ((m + P - 1) / P + 3) & ~3; };
        const int q_cap = (TILE_CAP / P) & ~3;            // longest slice the buffer can hold

        int r = 0, m_done = 0;                            // next run, sources of it already processed
        while (r < NR) {
            // ---- choose the pass: whole runs r..r_end-1, or one piece of an oversized run ----
            int r_end = r, slots = 0;
            bool piece = false;
            if (m_done == 0) {
                while (r_end < NR) {
                    const int need = P * tab.q[r_end];
                    if (slots + need > TILE_CAP) break;
                    slots += need;
                    r_end++;
                }
            }
            int mc = 0, qc = 0;
            if (r_end == r) {                             // run r does not fit: take P*q_cap sources of it
                piece = true;
                mc = min(tab.cum[r][W] - m_done, P * q_cap);
                qc = slice(mc);
                r_end = r + 1;
            }
            __syncthreads();                              // the previous pass is done with buf
            // ---- stage: one warp per cell segment, lanes over its particles ----
            {
                int base = 0;
                for (int rr = r; rr < r_end; rr++) {
                    const int m = piece ? mc : tab.cum[rr][W];
                    const int q = piece ? qc : tab.q[rr];
                    const int px = tab.px[rr];
                    if (m > 0) {
                        const float4 *__restrict__ qpos = planes[px].pos;
                        for (int sg = warp; sg < W; sg += TILE_T / 32) {
                            const int lo = tab.cum[rr][sg], hi = tab.cum[rr][sg + 1];
                            const int a = max(lo, m_done), b = min(hi, m_done + m);     // part of the segment in this pass
                            const uint32_t st = tab.start[rr][sg];
                            const float zsh = (float)(sg - R) * w;
                            for (int g = a + lane; g < b; g += 32) {
                                const float4 o = qpos[st + (uint32_t)(g - lo)];
                                buf[base + g - m_done] = make_float4(o.x * fc.scale, o.y * fc.scale, fmaf(o.z, fc.scale, zsh), 0.f);
                            }
                        }
                        for (int i = m + tid; i < P * q; i += TILE_T) buf[base + i] = SENT;
                    }
                    base += P * q;
                }
            }
            __syncthreads();
            // ---- compute: every phase sweeps its slice of each staged run ----
            if (active) {
                int base = 0;
                for (int rr = r; rr < r_end; rr++) {
                    const int m = piece ? mc : tab.cum[rr][W];
                    if (m == 0) continue;
                    const int q = piece ? qc : tab.q[rr];
                    const int dx = rr / W - R, dy = rr - (rr / W) * W - R;
                    const u64 xs = sub2(xi, pk((float)dx * w, (float)dx * w));   // sinks in the source column's frame
                    const u64 ys = sub2(yi, pk((float)dy * w, (float)dy * w));
                    const bool near = !fc.plummer && (!far_ok || (dx >= -1 && dx <= 1 && dy >= -1 && dy <= 1));
                    u64 ax = 0, ay = 0, az = 0;
                    const float4 *src = buf + base + ph * q;
                    if (near) run_sources<0>(src, q, xs, ys, zi, fc, ax, ay, az);
                    else run_sources<1>(src, q, xs, ys, zi, fc, ax, ay, az);
                    float a, b;
                    upk(ax, a, b); ax0 += (double)a; ax1 += (double)b;
                    upk(ay, a, b); ay0 += (double)a; ay1 += (double)b;
                    upk(az, a, b); az0 += (double)a; az1 += (double)b;
                    base += P * q;
                }
            }
            if (piece) {
                m_done += mc;
                if (m_done >= tab.cum[r][W]) { m_done = 0; r++; }
            } else {
                r = r_end;
            }
        }

        // ---- reduce the phases (fixed order), scale and write ----
        __syncthreads();
        double *red = reinterpret_cast<double *>(buf);       // [P][L][6] doubles <= 128*48 B = 6 KiB
        if (active) {
            double *d = red + ((size_t)ph * L + sl) * 6;
            d[0] = ax0; d[1] = ay0; d[2] = az0; d[3] = ax1; d[4] = ay1; d[5] = az1;
        }
        __syncthreads();
        for (int i = tid; i < n; i += TILE_T) {
            const int l = i >> 1, h = (i & 1) * 3;
            double sx = 0.0, sy = 0.0, sz = 0.0;
            for (int pp = 0; pp < P; pp++) {
                const double *d = red + ((size_t)pp * L + l) * 6 + h;
                sx += d[0]; sy += d[1]; sz += d[2];
            }
            if (sp.acc) {
                const uint64_t si = s0 + (uint64_t)i;
                const uint64_t o = sp.perm ? (uint64_t)sp.perm[si] : si;
                sp.acc[3 * o + 0] = (float)(sx * (double)fc.out_scale);
                sp.acc[3 * o + 1] = (float)(sy * (double)fc.out_scale);
                sp.acc[3 * o + 2] = (float)(sz * (double)fc.out_scale);
            }
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

static size_t n_sink_cells(const nf_force_params &p)
{
    const int n_sink_planes = p.sink_hi - p.sink_lo;
    return (size_t)(n_sink_planes > 0 ? n_sink_planes : 0) * p.K * p.K;
}
static size_t max_tasks(const nf_force_params &p)
{
    return n_sink_cells(p) + (size_t)(p.max_sinks > 0 ? p.max_sinks : 0) / TILE_SINKS + 1;
}

// scratch taken by nf_forces_impl (work list) plus room for a plane table of n_planes views
size_t nf_forces_scratch_bytes(const nf_force_params &p)
{
    const size_t nc = n_sink_cells(p);
    size_t b = nf_align_up((size_t)p.n_planes * sizeof(nf_plane_view), 256);
    b += 2 * nf_align_up(nc * sizeof(uint32_t), 256);                               // tc, to
    b += nf_align_up(nf_scan_temp_elems(nc) * sizeof(uint32_t), 256);               // scan temp
    b += nf_align_up(max_tasks(p) * sizeof(Task), 256);                             // tasks
    return b + 256 + 4096;
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

template <int R>
static int launch_tile(nf_ctx *ctx, const nf_force_params &p, const ForceConsts &fc, const nf_plane_view *d_planes,
                       const Task *tasks, uint32_t *ctl, cudaStream_t st)
{
    int occ = 0;
    NF_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_forces_tile<R>, TILE_T, 0));
    if (occ < 1) occ = 1;
    const size_t want = max_tasks(p);
    size_t blocks = (size_t)ctx->sm_count * occ;
    if (blocks > want) blocks = want;
    k_forces_tile<R><<<(unsigned)blocks, TILE_T, 0, st>>>(d_planes, p, fc, tasks, ctl);
    NF_LAUNCHED(ctx);
    return NF_OK;
}

int nf_forces_impl(nf_ctx *ctx, const nf_force_params &p, const nf_plane_view *d_planes,
                   cudaStream_t st, bool record_timing)
{
    if (record_timing) NF_CUDA(ctx, cudaEventRecord(ctx->ev_total0, st));
    const ForceConsts fc = make_consts(p);
    const int n_sink_planes = p.sink_hi - p.sink_lo;
    const size_t nc = n_sink_cells(p);
    uint32_t *tc = nf_scratch_take<uint32_t>(ctx, nc ? nc : 1);
    uint32_t *to = nf_scratch_take<uint32_t>(ctx, nc ? nc : 1);
    uint32_t *tmp = nf_scratch_take<uint32_t>(ctx, nf_scan_temp_elems(nc));
    Task *tasks = nf_scratch_take<Task>(ctx, max_tasks(p));
    uint32_t *ctl = nf_scratch_take<uint32_t>(ctx, 2);
    if (!tc || !to || !tmp || !tasks || !ctl) {
        NF_SET_ERR(ctx, "nf_forces: internal scratch arena too small");
        return NF_ERR_NOMEM;
    }
    if (n_sink_planes > 0) {
        // work list
        dim3 grid((unsigned)((p.K * p.K + 255) / 256), (unsigned)n_sink_planes);
        k_task_count<<<grid, 256, 0, st>>>(d_planes, p, tc);
        NF_LAUNCHED(ctx);
        NF_TRY(nf_exclusive_scan_u32(ctx, tc, to, nc, tmp, st));
        k_task_fill<<<grid, 256, 0, st>>>(tc, to, p, tasks, ctl);
        NF_LAUNCHED(ctx);
    }
    if (record_timing) NF_CUDA(ctx, cudaEventRecord(ctx->ev_kern0, st));
    if (n_sink_planes > 0) {
        switch (p.R) {
        case 0: NF_TRY(launch_tile<0>(ctx, p, fc, d_planes, tasks, ctl, st)); break;
        case 1: NF_TRY(launch_tile<1>(ctx, p, fc, d_planes, tasks, ctl, st)); break;
        case 2: NF_TRY(launch_tile<2>(ctx, p, fc, d_planes, tasks, ctl, st)); break;
        default: NF_TRY(launch_tile<3>(ctx, p, fc, d_planes, tasks, ctl, st)); break;
        }
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
