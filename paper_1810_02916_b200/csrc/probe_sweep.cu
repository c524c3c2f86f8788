// probe_sweep.cu -- the interaction kernel's sweep loops in isolation (a measuring tool, not part of libnf.so).
//
//     python -m paper_1810_02916_b200.build --probe     ->  paper_1810_02916_b200/probe_sweep
//     ./paper_1810_02916_b200/probe_sweep                (on a B200; prints one line per variant)
//
// What it answers ("Measured pipe facts"): how fast can the loop body of k_forces_warp run when nothing
// else happens -- tiles resident in shared memory, no staging, no work list?  One block per SM; every warp sweeps the
// same kind of tile `reps` times with four sinks per lane (two packed pairs), exactly the arithmetic of nf_forces.cu:
//   law 2: r^-3 only (MODE 2)      law 1: r^-3 + FMNMX3 tracking of the smallest r^2 (MODE 1)
//   law 0: the min form of Eq. 2, PAPER.md:243 / fn. 4 :239 (MODE 0)
//   gram : r^2 = |q|^2 + |s|^2 - 2 q.s with |q|^2 in the .w lane and sum f, sum f q accumulated (10 pipe instructions
//          instead of 11; NOT used by the library: same speed, worse accuracy across cell faces)
//   mufu : 2 = both rsqrt, 0 = none (timing only): what the MUFU costs
// Printed: interactions/s and the fraction of the FP32 roofline at 20 flop per interaction (SMs x 1965 MHz x 256).
#include <cstdio>
#include <cstdlib>
#include <cuda_runtime.h>
#include <stdint.h>

typedef unsigned long long u64;
__device__ __forceinline__ float rsqrt_approx(float x) { float y; asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float min3(float a, float b, float c) { float y; asm("min.ftz.f32 %0, %1, %2, %3;" : "=f"(y) : "f"(a), "f"(b), "f"(c)); return y; }
__device__ __forceinline__ u64 pk(float a, float b) { u64 r; asm("mov.b64 %0, {%1,%2};" : "=l"(r) : "f"(a), "f"(b)); return r; }
__device__ __forceinline__ void upk(u64 r, float &a, float &b) { asm("mov.b64 {%0,%1}, %2;" : "=f"(a), "=f"(b) : "l"(r)); }
__device__ __forceinline__ u64 fma2(u64 a, u64 b, u64 c) { u64 d; asm("fma.rn.ftz.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c)); return d; }
__device__ __forceinline__ void fma2_acc(u64 &acc, u64 a, u64 b) { asm("fma.rn.ftz.f32x2 %0, %1, %2, %0;" : "+l"(acc) : "l"(a), "l"(b)); }
__device__ __forceinline__ u64 sub2(u64 a, u64 b) { u64 d; asm("sub.rn.ftz.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d; }
__device__ __forceinline__ u64 add2(u64 a, u64 b) { u64 d; asm("add.rn.ftz.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d; }
__device__ __forceinline__ u64 mul2(u64 a, u64 b) { u64 d; asm("mul.rn.ftz.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d; }

struct FC { float A, B, C, r2_floor; };
enum { LAW_MIN = 0, LAW_TRACK = 1, LAW_R3 = 2, LAW_GRAM = 3 };

// one source against two of the lane's sinks
template <int LAW, int MUFU>
__device__ __forceinline__ void interact(const float4 q, const u64 xs, const u64 ys, const u64 zs, const u64 s2, const FC &fc, u64 &ax, u64 &ay,
                                         u64 &az, u64 &sf, float &rmin)
{
    if (LAW == LAW_GRAM) {      // xs, ys, zs hold -2 s;  s2 = |s|^2 + floor
        u64 r2 = add2(pk(q.w, q.w), s2);
        r2 = fma2(pk(q.z, q.z), zs, r2);
        r2 = fma2(pk(q.y, q.y), ys, r2);
        r2 = fma2(pk(q.x, q.x), xs, r2);
        float a, b;
        upk(r2, a, b);
        const u64 ri = MUFU == 2 ? pk(rsqrt_approx(a), rsqrt_approx(b)) : r2;
        const u64 f = mul2(mul2(ri, ri), ri);
        sf = add2(sf, f);
        fma2_acc(ax, f, pk(q.x, q.x));
        fma2_acc(ay, f, pk(q.y, q.y));
        fma2_acc(az, f, pk(q.z, q.z));
    } else {
        const u64 dx = sub2(pk(q.x, q.x), xs), dy = sub2(pk(q.y, q.y), ys), dz = sub2(pk(q.z, q.z), zs);
        u64 r2 = fma2(dz, dz, pk(fc.r2_floor, fc.r2_floor));
        r2 = fma2(dy, dy, r2);
        r2 = fma2(dx, dx, r2);
        float a, b;
        upk(r2, a, b);
        const u64 ri = MUFU == 2 ? pk(rsqrt_approx(a), rsqrt_approx(b)) : r2;
        u64 f = mul2(mul2(ri, ri), ri);
        if (LAW == LAW_MIN) {
            const u64 poly = fma2(r2, fma2(pk(fc.B, fc.B), ri, pk(fc.C, fc.C)), pk(fc.A, fc.A));
            float pa, pb, fa, fb;
            upk(poly, pa, pb);
            upk(f, fa, fb);
            f = pk(fminf(pa, fa), fminf(pb, fb));
        } else if (LAW == LAW_TRACK) {
            rmin = min3(rmin, a, b);
        }
        fma2_acc(ax, f, dx);
        fma2_acc(ay, f, dy);
        fma2_acc(az, f, dz);
    }
}

template <int LAW, int MUFU>
__device__ __forceinline__ void pair4(const float4 a0, const float4 a1, const u64 (&xs)[2], const u64 (&ys)[2], const u64 (&zs)[2],
                                      const u64 (&s2)[2], const FC &fc, u64 (&ax)[2], u64 (&ay)[2], u64 (&az)[2], u64 (&sf)[2], float &rmin)
{
    interact<LAW, MUFU>(a0, xs[0], ys[0], zs[0], s2[0], fc, ax[0], ay[0], az[0], sf[0], rmin);
    interact<LAW, MUFU>(a0, xs[1], ys[1], zs[1], s2[1], fc, ax[1], ay[1], az[1], sf[1], rmin);
    interact<LAW, MUFU>(a1, xs[0], ys[0], zs[0], s2[0], fc, ax[0], ay[0], az[0], sf[0], rmin);
    interact<LAW, MUFU>(a1, xs[1], ys[1], zs[1], s2[1], fc, ax[1], ay[1], az[1], sf[1], rmin);
}

// the sweep of nf_forces.cu: q sources (a multiple of 4 here), two register sets alternate, loads one pair ahead
template <int LAW, int MUFU>
__device__ __forceinline__ void sweep(const float4 *__restrict__ src, int q, const u64 (&xs)[2], const u64 (&ys)[2], const u64 (&zs)[2],
                                      const u64 (&s2)[2], const FC &fc, u64 (&ax)[2], u64 (&ay)[2], u64 (&az)[2], u64 (&sf)[2], float &rmin)
{
    const float4 *end = src + q;
    float4 a0 = src[0], a1 = src[1];
#pragma unroll 2
    do {
        const float4 b0 = src[2], b1 = src[3];
        pair4<LAW, MUFU>(a0, a1, xs, ys, zs, s2, fc, ax, ay, az, sf, rmin);
        a0 = src[4]; a1 = src[5];
        src += 4;
        pair4<LAW, MUFU>(b0, b1, xs, ys, zs, s2, fc, ax, ay, az, sf, rmin);
    } while (src < end);
}

constexpr int TILE = 520, MAX_WARPS = 16;

template <int LAW, int MUFU>
__global__ void __launch_bounds__(MAX_WARPS * 32, 1) k_probe(const float4 *__restrict__ g, int q, int reps, FC fc, float *out, int P)
{
    extern __shared__ float4 bufraw[];
    float4(*buf)[TILE] = reinterpret_cast<float4(*)[TILE]>(bufraw);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    for (int i = lane; i < TILE; i += 32) buf[warp][i] = g[(blockIdx.x * MAX_WARPS + warp) * TILE + i];
    __syncwarp();
    u64 xs[2], ys[2], zs[2], s2[2];
    for (int h = 0; h < 2; h++) {
        const float x0 = 0.01f * lane + h, x1 = 0.013f * lane - h, y0 = 0.02f * lane, y1 = 0.3f + h, z0 = 2.f + 0.01f * lane, z1 = 2.5f;
        if (LAW == LAW_GRAM) {
            xs[h] = pk(-2 * x0, -2 * x1); ys[h] = pk(-2 * y0, -2 * y1); zs[h] = pk(-2 * z0, -2 * z1);
            s2[h] = pk(x0 * x0 + y0 * y0 + z0 * z0, x1 * x1 + y1 * y1 + z1 * z1);
        } else {
            xs[h] = pk(x0, x1); ys[h] = pk(y0, y1); zs[h] = pk(z0, z1); s2[h] = 0;
        }
    }
    u64 gx[2] = {0, 0}, gy[2] = {0, 0}, gz[2] = {0, 0};
    for (int r = 0; r < reps; r++) {                   // one "tile" per repetition: sums from zero, added to the running sums
        u64 ax[2] = {0, 0}, ay[2] = {0, 0}, az[2] = {0, 0}, sf[2] = {0, 0};
        float rmin = 3e38f;
        sweep<LAW, MUFU>(buf[warp] + (lane / (32 / P)) * q, q, xs, ys, zs, s2, fc, ax, ay, az, sf, rmin);   // P phases read P slices
        for (int h = 0; h < 2; h++) {
            if (LAW == LAW_GRAM) { ax[h] = fma2(sf[h], xs[h], ax[h]); ay[h] = fma2(sf[h], ys[h], ay[h]); az[h] = fma2(sf[h], zs[h], az[h]); }
            gx[h] = add2(gx[h], ax[h]); gy[h] = add2(gy[h], ay[h]); gz[h] = add2(gz[h], az[h]);
        }
        if (LAW == LAW_TRACK && rmin < 0.f) gx[0] = 0;
    }
    float a, b, s = 0;
    for (int h = 0; h < 2; h++) { upk(gx[h], a, b); s += a + b; upk(gy[h], a, b); s += a + b; upk(gz[h], a, b); s += a + b; }
    out[blockIdx.x * MAX_WARPS * 32 + threadIdx.x] = s;
}

template <int LAW, int MUFU>
static void run(const char *name, const float4 *g, float *out, int sms, int warps, int P, int q)
{
    const FC fc{10.f, -15.f, 6.f, 1e-18f};
    const int reps = 800000 / q, smem = MAX_WARPS * TILE * 16;
    cudaFuncSetAttribute(k_probe<LAW, MUFU>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    k_probe<LAW, MUFU><<<sms, warps * 32, smem>>>(g, q, reps, fc, out, P);          // warm-up
    cudaDeviceSynchronize();
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    cudaEventRecord(e0);
    k_probe<LAW, MUFU><<<sms, warps * 32, smem>>>(g, q, reps, fc, out, P);
    cudaEventRecord(e1);
    cudaEventSynchronize(e1);
    float ms;
    cudaEventElapsedTime(&ms, e0, e1);
    const double inter = (double)sms * warps * 32 * 4.0 * q * reps, peak = sms * 1.965e9 * 256;
    printf("%-34s warps/SM %2d  phases %d  sources/sweep %3d  %8.3f ms  %.3e interactions/s  %5.1f %% of the FP32 roofline  [%s]\n", name, warps, P,
           q, ms, inter / (ms * 1e-3), 100 * 20 * inter / (ms * 1e-3) / peak, cudaGetErrorString(cudaGetLastError()));
}

int main()
{
    cudaDeviceProp p;
    cudaGetDeviceProperties(&p, 0);
    const int sms = p.multiProcessorCount;
    printf("%s, %d SMs; roofline = SMs x 1965 MHz x 256 flop, 20 flop per interaction\n", p.name, sms);
    const size_t n = (size_t)sms * MAX_WARPS * TILE;
    float4 *h = (float4 *)malloc(n * sizeof(float4));
    srand48(1);
    for (size_t i = 0; i < n; i++) {
        const float x = drand48() - 0.5f, y = drand48() - 0.5f, z = drand48() - 0.5f;
        h[i] = make_float4(x, y, z, x * x + y * y + z * z);
    }
    float4 *g;
    float *out;
    cudaMalloc(&g, n * sizeof(float4));
    cudaMemcpy(g, h, n * sizeof(float4), cudaMemcpyHostToDevice);
    cudaMalloc(&out, (size_t)sms * MAX_WARPS * 32 * 4);
    run<LAW_R3, 2>("MODE 2: r^-3 (11 pipe ops)", g, out, sms, 12, 1, 160);
    run<LAW_TRACK, 2>("MODE 1: r^-3 + FMNMX3 tracking", g, out, sms, 12, 1, 160);
    run<LAW_MIN, 2>("MODE 0: min form (13 pipe ops)", g, out, sms, 12, 1, 160);
    run<LAW_GRAM, 2>("Gram form r^-3 (10 pipe ops)", g, out, sms, 12, 1, 160);
    run<LAW_R3, 0>("MODE 2 without the rsqrt", g, out, sms, 12, 1, 160);
    run<LAW_GRAM, 0>("Gram form without the rsqrt", g, out, sms, 12, 1, 160);
    run<LAW_MIN, 0>("MODE 0 without the rsqrt", g, out, sms, 12, 1, 160);
    for (int w : {8, 16}) run<LAW_R3, 2>("MODE 2, other warp counts", g, out, sms, w, 1, 160);
    for (int P : {2, 4, 8}) run<LAW_R3, 2>("MODE 2, tile split over phases", g, out, sms, 12, P, 480 / P / 4 * 4);
    for (int q : {40, 80, 320, 480}) run<LAW_R3, 2>("MODE 2, other sweep lengths", g, out, sms, 12, 1, q);
    return 0;
}
