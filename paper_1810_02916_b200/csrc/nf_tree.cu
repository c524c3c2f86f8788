// nf_tree.cu -- tree near field for DENSE cells.
//
// PAPER.md:49 "Future versions of Abacus will employ trees in the near-field domain, especially for dense cells";
// PAPER.md:75 "the largest cell has over 200,000 particles".  The paper prints no algorithm; this file implements the
// one DESIGN.md states (readings t1-t6), the same one oracle/nf_tree.py follows on the CPU:
//
//   t1  dense cell = a cell of nf_dense.cu's in-cell ordering (>= NF_DENSE_N particles, within its capacity)
//   t2  its particles in Hilbert order of their cell-centred offsets (k_dense_keys)
//   t3  leaves = 16 consecutive particles (a quarter of a 64-particle "chunk" of the compact array), a node of level l =
//       8 nodes of level l-1, up to one root; a node carries the box of its particles' offsets, its mass and its centre of mass
//   t4  sink group = 64 consecutive particles of a cell (Hilbert order in a dense cell, binned order elsewhere) and
//       the box of their offsets
//   t5  a group walks the tree of every dense cell among its (2R+1)^3 neighbours from the root: a node is ACCEPTED when
//       the gap d between the two boxes and the node's diagonal s satisfy d^2 > eps^2 and s^2 < theta^2 d^2 (float32,
//       every operation rounded, no fused multiply-add: the oracle takes the same decisions bit for bit); accepted ->
//       one particle of the node's mass at its centre of mass, 1/r^2 law; else open it; a leaf that is not accepted
//       is summed particle by particle with the full softened law
//   t6  everything else (sources of cells that are not dense) stays with the interaction kernel, which skips the
//       dense source cells when p.tree is set
//
//   k_tree_layout    one thread: per dense cell the number of nodes of every level and where they start
//   k_tree_leaves    one warp per chunk: Hilbert-ordered copy of (offset, mass); box, mass, centre of mass of its four leaves
//   k_tree_level     level l from level l-1
//   k_tree_items     per cell: number of sink groups if any neighbour cell is dense (scanned into the work list)
//   k_tree_walk<1>   one warp per sink group: in how many parts it walks (t4: as a whole, or in parts when its box is out of
//                    proportion); scanned into the work list of (group, part) pairs
//   k_tree_walk<0>   one warp per (group, part): the walk of t5 with a bounded depth-first stack in shared memory; ADDS to acc
//   k_tree_amax      per-cell maximum of |a| from the final accelerations
//
// Deterministic: every sink belongs to one warp, which visits cells, nodes and particles in a fixed order; the only
// atomics are integer counters.
#include "nf_common.cuh"

namespace {

constexpr int LEAF = 16;                        // particles per leaf (t3); sink groups are 64 (t4)
constexpr int MAXLEV = 9;                       // 2^24 leaves at most (2^28 compact positions): 8 levels above them
constexpr uint32_t PAD = 0xffffffffu;
constexpr int WALK_WARPS = 8;
constexpr int STACK_CAP = 256 * MAXLEV + 64;    // depth-first over batches of 32 nodes: at most 8 * 32 pending per level
constexpr int LIST_CAP = 64;
constexpr float FILL = 1.0e15f;

// packed float32 pairs (the two sinks a lane holds): one instruction for both, as in the interaction kernel
typedef unsigned long long u64;
__device__ __forceinline__ u64 pk(float a, float b) { u64 r; asm("mov.b64 %0, {%1,%2};" : "=l"(r) : "f"(a), "f"(b)); return r; }
__device__ __forceinline__ void upk(u64 r, float &a, float &b) { asm("mov.b64 {%0,%1}, %2;" : "=f"(a), "=f"(b) : "l"(r)); }
__device__ __forceinline__ u64 fma2(u64 a, u64 b, u64 c) { u64 d; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c)); return d; }
__device__ __forceinline__ u64 sub2(u64 a, u64 b) { u64 d; asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d; }
__device__ __forceinline__ u64 add2(u64 a, u64 b) { u64 d; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d; }
// MUFU.RSQ alone: rsqrtf() without -ftz wraps it in a range fix-up for denormals (2 FSETP + 4 FMUL per pair); no argument here is one
__device__ __forceinline__ float rsq(float a) { float r; asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(a)); return r; }
__device__ __forceinline__ u64 mul2(u64 a, u64 b) { u64 d; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d; }

struct TreeCell {
    unsigned long long c0;        // first sorted slot of the cell
    uint32_t coff, n, nlev, pad;
    uint32_t base[MAXLEV];        // first node of level l
    uint32_t cnt[MAXLEV];         // nodes of level l
};

__global__ void k_tree_layout(const nf_dense_cell *__restrict__ dcell, const uint32_t *__restrict__ nd, TreeCell *__restrict__ tcell,
                              uint32_t *__restrict__ crank)
{
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    const uint32_t ndense = nd[1];
    uint32_t next = 0;
    for (uint32_t r = 0; r < ndense; r++) {
        const nf_dense_cell dc = dcell[r];
        TreeCell t;
        t.c0 = dc.c0; t.coff = dc.coff; t.n = dc.n; t.pad = 0;
        uint32_t m = (dc.n + (uint32_t)LEAF - 1u) / (uint32_t)LEAF;
        int l = 0;
        for (;; l++) {
            t.base[l] = next; t.cnt[l] = m;
            next += m;
            if (m == 1) break;
            m = (m + 7u) >> 3;
        }
        t.nlev = (uint32_t)l + 1u;
        for (int k = l + 1; k < MAXLEV; k++) { t.base[k] = 0; t.cnt[k] = 0; }
        tcell[r] = t;
        crank[dc.coff >> 6] = r;
    }
}

__global__ void k_tree_sentinel(float4 *sentinel)
{
    if (threadIdx.x < 2) sentinel[threadIdx.x] = make_float4(1.0e15f, 1.0e15f, 1.0e15f, 0.f);
}

__device__ __forceinline__ uint32_t cell_of_chunk(const TreeCell *__restrict__ tcell, uint32_t ndense, uint32_t t0)
{
    uint32_t lo = 0, hi = ndense;                 // last r with coff <= t0
    while (hi - lo > 1) {
        const uint32_t mid = (lo + hi) >> 1;
        if (tcell[mid].coff <= t0) lo = mid; else hi = mid;
    }
    return lo;
}

template <bool MASS>
__global__ void __launch_bounds__(256) k_tree_leaves(const float4 *__restrict__ pos, const uint32_t *__restrict__ dslot,
                                                     const uint32_t *__restrict__ nd, const TreeCell *__restrict__ tcell,
                                                     float4 *__restrict__ tpos, float4 *__restrict__ nlo, float4 *__restrict__ nhi,
                                                     float4 *__restrict__ ncom, uint32_t nchunk_max)
{
    const int lane = threadIdx.x & 31;
    const uint32_t n_d = nd[0], ndense = nd[1];
    for (uint32_t ch = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5); ch < nchunk_max; ch += gridDim.x * (blockDim.x >> 5)) {
        const uint32_t t0 = ch * 64u;
        if (t0 >= n_d) return;
        const uint32_t r = cell_of_chunk(tcell, ndense, t0);
        const uint32_t leaf0 = (t0 - tcell[r].coff) / (uint32_t)LEAF, nleaf = tcell[r].cnt[0], base = tcell[r].base[0];
        // positions t0 + 32 h + lane: lanes 0-15 / 16-31 of round h are leaf 2h / 2h + 1 of this chunk
#pragma unroll
        for (int h = 0; h < 2; h++) {
            float lo[3] = {3.0e38f, 3.0e38f, 3.0e38f}, hi[3] = {-3.0e38f, -3.0e38f, -3.0e38f};
            double sm = 0.0, sx = 0.0, sy = 0.0, sz = 0.0;
            const uint32_t t = t0 + 32u * h + lane;
            const uint32_t s = dslot[t];
            float4 o = make_float4(FILL, FILL, FILL, 0.f);        // padding: massless and far away (r^-3 flushes to zero)
            if (s != PAD) {
                o = pos[s];
                if (!MASS) o.w = 1.0f;
                lo[0] = hi[0] = o.x; lo[1] = hi[1] = o.y; lo[2] = hi[2] = o.z;
                sm = (double)o.w; sx = (double)o.w * (double)o.x; sy = (double)o.w * (double)o.y; sz = (double)o.w * (double)o.z;
            }
            tpos[t] = o;
#pragma unroll
            for (int d = 8; d > 0; d >>= 1) {            // within each half-warp: one leaf
#pragma unroll
                for (int a = 0; a < 3; a++) {
                    lo[a] = fminf(lo[a], __shfl_xor_sync(0xffffffffu, lo[a], d));
                    hi[a] = fmaxf(hi[a], __shfl_xor_sync(0xffffffffu, hi[a], d));
                }
                sm += __shfl_xor_sync(0xffffffffu, sm, d);
                sx += __shfl_xor_sync(0xffffffffu, sx, d);
                sy += __shfl_xor_sync(0xffffffffu, sy, d);
                sz += __shfl_xor_sync(0xffffffffu, sz, d);
            }
            const uint32_t leaf = leaf0 + 2u * h + (lane >> 4);
            if ((lane & 15) == 0 && leaf < nleaf) {
                const double inv = sm != 0.0 ? 1.0 / sm : 0.0;
                nlo[base + leaf] = make_float4(lo[0], lo[1], lo[2], (float)sm);
                nhi[base + leaf] = make_float4(hi[0], hi[1], hi[2], 0.f);
                ncom[base + leaf] = make_float4((float)(sx * inv), (float)(sy * inv), (float)(sz * inv), (float)sm);
            }
        }
    }
}

// blockIdx.y = dense cell (by rank), threads over the nodes of level l
__global__ void __launch_bounds__(128) k_tree_level(const uint32_t *__restrict__ nd, const TreeCell *__restrict__ tcell, int l,
                                                    float4 *__restrict__ nlo, float4 *__restrict__ nhi, float4 *__restrict__ ncom)
{
    const uint32_t r = blockIdx.y;
    if (r >= nd[1]) return;
    const TreeCell &T = tcell[r];
    if ((uint32_t)l >= T.nlev) return;
    const uint32_t cnt = T.cnt[l], ccnt = T.cnt[l - 1], base = T.base[l], cbase = T.base[l - 1];
    for (uint32_t k = blockIdx.x * blockDim.x + threadIdx.x; k < cnt; k += gridDim.x * blockDim.x) {
        float lo[3] = {3.0e38f, 3.0e38f, 3.0e38f}, hi[3] = {-3.0e38f, -3.0e38f, -3.0e38f};
        double sm = 0.0, sx = 0.0, sy = 0.0, sz = 0.0;
        for (uint32_t j = 8u * k; j < min(8u * k + 8u, ccnt); j++) {
            const float4 a = nlo[cbase + j], b = nhi[cbase + j], c = ncom[cbase + j];
            lo[0] = fminf(lo[0], a.x); lo[1] = fminf(lo[1], a.y); lo[2] = fminf(lo[2], a.z);
            hi[0] = fmaxf(hi[0], b.x); hi[1] = fmaxf(hi[1], b.y); hi[2] = fmaxf(hi[2], b.z);
            sm += (double)c.w; sx += (double)c.w * (double)c.x; sy += (double)c.w * (double)c.y; sz += (double)c.w * (double)c.z;
        }
        const double inv = sm != 0.0 ? 1.0 / sm : 0.0;
        nlo[base + k] = make_float4(lo[0], lo[1], lo[2], (float)sm);
        nhi[base + k] = make_float4(hi[0], hi[1], hi[2], 0.f);
        ncom[base + k] = make_float4((float)(sx * inv), (float)(sy * inv), (float)(sz * inv), (float)sm);
    }
}

// per cell: sink groups to walk = ceil(n / 64) if any of the (2R+1)^3 neighbour cells is dense, else 0 (element ncell: 0)
__global__ void __launch_bounds__(256) k_tree_items(const uint64_t *__restrict__ off, const uint32_t *__restrict__ dinfo, int K, int R,
                                                    size_t ncell, uint32_t *__restrict__ ng)
{
    const size_t c = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (c > ncell) return;
    uint32_t g = 0;
    if (c < ncell) {
        const uint64_t n = off[c + 1] - off[c];
        if (n > 0) {
            const int cz = (int)(c % K), cy = (int)((c / K) % K), cx = (int)(c / ((size_t)K * K));
            bool any = false;
            for (int dx = -R; dx <= R && !any; dx++)
                for (int dy = -R; dy <= R && !any; dy++)
                    for (int dz = -R; dz <= R; dz++) {
                        const int qx = ((cx + dx) % K + K) % K, qy = ((cy + dy) % K + K) % K, qz = ((cz + dz) % K + K) % K;
                        if (dinfo[((size_t)qx * K + qy) * K + qz]) { any = true; break; }
                    }
            if (any) g = (uint32_t)((n + 63) >> 6);
        }
    }
    ng[c] = g;
}

struct Part { float lo[3], hi[3]; unsigned long long mask; };   // sinks that walk together (bit 32 h + lane), and their box

struct WalkShared {
    Part part;                     // the part this item walks
    uint32_t stack[STACK_CAP];
    ulonglong2 list[2 * LIST_CAP]; // accepted nodes waiting to be evaluated: (x,x | y,y), (z,z | m,m) -- duplicated for the packed sweep
    ulonglong2 stage[2 * 64];      // the particles of up to four leaves, same layout
    uint32_t leaves[32];           // leaves opened by a batch; bit 31: every pair of the leaf is further apart than eps
};

__device__ __forceinline__ void put_dup(ulonglong2 *dst, const float4 q)
{
    dst[0] = make_ulonglong2(pk(q.x, q.x), pk(q.y, q.y));
    dst[1] = make_ulonglong2(pk(q.z, q.z), pk(q.w, q.w));
}

struct SweepConsts { u64 ie, ie3, six, m15, ten, eps2; };

// n sources against the lane's two sinks (PX, PY, PZ), sums formed from zero into LX, LY, LZ.
// LAW 0: m / r^2 (accepted nodes; leaves proven outside eps -- the spline equals it there, fn. 4)
// LAW 1: the spline of Eq. 2 as min(poly, r^-3);  LAW 2: Plummer, Eq. 1
template <int LAW>
__device__ __forceinline__ void sweep2(const ulonglong2 *__restrict__ src, uint32_t n, u64 PX, u64 PY, u64 PZ, const SweepConsts &C,
                                       u64 &LX, u64 &LY, u64 &LZ)
{
#pragma unroll 4
    for (uint32_t j = 0; j < n; j++) {
        const ulonglong2 xy = src[2 * j], zw = src[2 * j + 1];
        const u64 DX = sub2(xy.x, PX), DY = sub2(xy.y, PY), DZ = sub2(zw.x, PZ);
        u64 R2 = fma2(DZ, DZ, fma2(DY, DY, mul2(DX, DX)));
        if (LAW == 2) R2 = add2(R2, C.eps2);
        float a, b;
        upk(R2, a, b);
        if (LAW == 1) { a = fmaxf(a, 1.0e-30f); b = fmaxf(b, 1.0e-30f); }      // r = 0: the pair of a sink with itself
        const u64 RI = pk(rsq(a), rsq(b));
        u64 F = mul2(mul2(RI, RI), RI);
        if (LAW == 1) {
            const u64 U = mul2(mul2(R2, RI), C.ie);
            const u64 POLY = mul2(fma2(U, fma2(U, C.six, C.m15), C.ten), C.ie3);
            float f0, f1, p0, p1;
            upk(F, f0, f1); upk(POLY, p0, p1);
            F = pk(fminf(f0, p0), fminf(f1, p1));                               // fn. 4
        }
        F = mul2(F, zw.y);
        LX = fma2(F, DX, LX); LY = fma2(F, DY, LY); LZ = fma2(F, DZ, LZ);
    }
}

struct WalkParams {
    const float4 *pos; const uint64_t *off; const uint32_t *perm; const uint32_t *dinfo; const uint32_t *dslot;
    const TreeCell *tcell; const uint32_t *crank; const float4 *tpos; const float4 *nlo; const float4 *nhi; const float4 *ncom;
    const uint32_t *goff;          // exclusive scan of the groups per cell, ncell + 1 entries
    uint32_t *np;                  // parts per group (t4), written by the counting instance
    const uint32_t *poff;          // exclusive scan of np: the work list is over (group, part) pairs
    float *acc; unsigned long long *stats; uint32_t *cursor;
    size_t ncell; int K, R, plummer; float cw, eps, eps2, th2, Gm;
};

// COUNT: one warp per group, writes the number of parts the group walks in (t4) and nothing else.  Else: one warp per
// (group, part) pair pulled from a cursor -- a group that walks in up to 64 parts is up to 64 work items, not one item
// 19 walks long (that one item used to be the kernel's tail: SMs 63 % busy).
template <bool COUNT>
__global__ void __launch_bounds__(WALK_WARPS * 32, 2) k_tree_walk(const WalkParams P)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    WalkShared &S = reinterpret_cast<WalkShared *>(smem_raw)[threadIdx.x >> 5];
    const int lane = threadIdx.x & 31;
    const int K = P.K, R = P.R;
    const uint32_t n_groups = P.goff[P.ncell];
    const uint32_t n_items = COUNT ? n_groups : P.poff[n_groups];
    const float inv_eps = 1.0f / P.eps, inv_eps3 = inv_eps * inv_eps * inv_eps;
    const SweepConsts SC = {pk(inv_eps, inv_eps), pk(inv_eps3, inv_eps3), pk(6.0f, 6.0f), pk(-15.0f, -15.0f), pk(10.0f, 10.0f), pk(P.eps2, P.eps2)};
    unsigned long long st_node = 0, st_leaf = 0;
    for (uint32_t round = 0;; round++) {
        uint32_t item = 0;
        if (COUNT) item = (round * gridDim.x + blockIdx.x) * WALK_WARPS + (threadIdx.x >> 5);
        else {
            if (lane == 0) item = atomicAdd(P.cursor, 1u);
            item = __shfl_sync(0xffffffffu, item, 0);
        }
        if (item >= n_items) break;
        uint32_t grp = item, part_k = 0;
        if (!COUNT) {                            // the group of this item: last grp with poff[grp] <= item
            uint32_t lo_g = 0, hi_g = n_groups;
            while (hi_g - lo_g > 1) {
                const uint32_t mid = (lo_g + hi_g) >> 1;
                if (P.poff[mid] <= item) lo_g = mid; else hi_g = mid;
            }
            grp = lo_g; part_k = item - P.poff[lo_g];
        }
        // the cell of this group: last c with goff[c] <= grp
        size_t lo_c = 0, hi_c = P.ncell;
        while (hi_c - lo_c > 1) {
            const size_t mid = (lo_c + hi_c) >> 1;
            if (P.goff[mid] <= grp) lo_c = mid; else hi_c = mid;
        }
        const size_t c = lo_c;
        const uint32_t g = grp - P.goff[c];
        const int cz = (int)(c % K), cy = (int)((c / K) % K), cx = (int)(c / ((size_t)K * K));
        const uint64_t c0 = P.off[c], c1 = P.off[c + 1];
        const uint32_t own = P.dinfo[c];
        // t4: the group's sinks (two per lane) and their box
        uint64_t slot[2];
        float sx[2], sy[2], sz[2];
        bool valid[2];
        float glo[3] = {3.0e38f, 3.0e38f, 3.0e38f}, ghi[3] = {-3.0e38f, -3.0e38f, -3.0e38f};
#pragma unroll
        for (int h = 0; h < 2; h++) {
            const uint32_t t = 64u * g + 32u * h + lane;
            valid[h] = false; slot[h] = 0; sx[h] = sy[h] = sz[h] = 0.f;
            if (own) {
                const uint32_t s = P.dslot[(size_t)(own - 1u) * 64u + t];
                if (s != PAD) { valid[h] = true; slot[h] = s; }
            } else if (c0 + t < c1) { valid[h] = true; slot[h] = c0 + t; }
            if (valid[h]) {
                const float4 o = P.pos[slot[h]];
                sx[h] = o.x; sy[h] = o.y; sz[h] = o.z;
            }
        }
        // boxes of the four quarters (16 consecutive sinks: a half-warp of one round) and of the whole group
        float qlo[2][3], qhi[2][3];                  // this lane's quarter in round h
        const float mylo[2][3] = {{valid[0] ? sx[0] : 3.0e38f, valid[0] ? sy[0] : 3.0e38f, valid[0] ? sz[0] : 3.0e38f},
                                  {valid[1] ? sx[1] : 3.0e38f, valid[1] ? sy[1] : 3.0e38f, valid[1] ? sz[1] : 3.0e38f}};
        const float myhi[2][3] = {{valid[0] ? sx[0] : -3.0e38f, valid[0] ? sy[0] : -3.0e38f, valid[0] ? sz[0] : -3.0e38f},
                                  {valid[1] ? sx[1] : -3.0e38f, valid[1] ? sy[1] : -3.0e38f, valid[1] ? sz[1] : -3.0e38f}};
#pragma unroll
        for (int h = 0; h < 2; h++)
#pragma unroll
            for (int a = 0; a < 3; a++) {
                float l = mylo[h][a], u = myhi[h][a];
#pragma unroll
                for (int d = 8; d > 0; d >>= 1) {
                    l = fminf(l, __shfl_xor_sync(0xffffffffu, l, d));
                    u = fmaxf(u, __shfl_xor_sync(0xffffffffu, u, d));
                }
                qlo[h][a] = l; qhi[h][a] = u;
            }
        const uint32_t vm0 = __ballot_sync(0xffffffffu, valid[0]), vm1 = __ballot_sync(0xffffffffu, valid[1]);
        const unsigned long long vmask = (unsigned long long)vm0 | ((unsigned long long)vm1 << 32);
        // t4 (group_parts): the group walks as a whole unless its box is out of proportion to its quarters'
        uint32_t nparts = 0;
        {
            float blo[4][3], bhi[4][3], d2q[4];
            uint32_t cq[4];
            float lim = 3.0e38f;
            bool counted = false;
#pragma unroll
            for (int q = 0; q < 4; q++) {
                float s2 = 0.f;
#pragma unroll
                for (int a = 0; a < 3; a++) {
                    blo[q][a] = __shfl_sync(0xffffffffu, qlo[q >> 1][a], 16 * (q & 1));
                    bhi[q][a] = __shfl_sync(0xffffffffu, qhi[q >> 1][a], 16 * (q & 1));
                    const float e = __fsub_rn(bhi[q][a], blo[q][a]);
                    s2 = a == 0 ? __fmul_rn(e, e) : __fadd_rn(s2, __fmul_rn(e, e));
                }
                cq[q] = __popcll(vmask & (0xffffull << (16 * q)));
                d2q[q] = s2;
                if (cq[q] >= 8u) { lim = fminf(lim, s2); counted = true; }
            }
#pragma unroll
            for (int a = 0; a < 3; a++) {
                glo[a] = fminf(fminf(blo[0][a], blo[1][a]), fminf(blo[2][a], blo[3][a]));
                ghi[a] = fmaxf(fmaxf(bhi[0][a], bhi[1][a]), fmaxf(bhi[2][a], bhi[3][a]));
            }
            float d2g = 0.f;
#pragma unroll
            for (int a = 0; a < 3; a++) {
                const float e = __fsub_rn(ghi[a], glo[a]);
                d2g = a == 0 ? __fmul_rn(e, e) : __fadd_rn(d2g, __fmul_rn(e, e));
            }
            lim = __fmul_rn(9.0f, lim);
            if (!(counted && d2g > lim && P.th2 > 0.f)) {       // theta = 0 accepts nothing: no box matters, one walk
                if (lane == 0 && !COUNT) { Part &pt = S.part; pt.mask = vmask; for (int a = 0; a < 3; a++) { pt.lo[a] = glo[a]; pt.hi[a] = ghi[a]; } }
                nparts = 1;
            } else {
#pragma unroll
                for (int q = 0; q < 4; q++) {
                    if (cq[q] == 0) continue;
                    if (d2q[q] > lim) {                    // sink by sink
                        for (uint32_t i = 0; i < cq[q]; i++) {
                            const int src = 16 * (q & 1) + (int)i;
                            const float x = __shfl_sync(0xffffffffu, sx[q >> 1], src), y = __shfl_sync(0xffffffffu, sy[q >> 1], src),
                                        z = __shfl_sync(0xffffffffu, sz[q >> 1], src);
                            if (lane == 0 && !COUNT && nparts == part_k) { Part &pt = S.part; pt.mask = 1ull << (16 * q + i); pt.lo[0] = pt.hi[0] = x; pt.lo[1] = pt.hi[1] = y; pt.lo[2] = pt.hi[2] = z; }
                            nparts++;
                        }
                    } else {
                        if (lane == 0 && !COUNT && nparts == part_k) { Part &pt = S.part; pt.mask = vmask & (0xffffull << (16 * q)); for (int a = 0; a < 3; a++) { pt.lo[a] = blo[q][a]; pt.hi[a] = bhi[q][a]; } }
                        nparts++;
                    }
                }
            }
            __syncwarp();
        }
        if (COUNT) {
            if (lane == 0) P.np[grp] = nparts;
            __syncwarp();
            continue;
        }
        float ax[2] = {0.f, 0.f}, ay[2] = {0.f, 0.f}, az[2] = {0.f, 0.f};
        {
        const Part part = S.part;
#pragma unroll
        for (int a = 0; a < 3; a++) { glo[a] = part.lo[a]; ghi[a] = part.hi[a]; }
        const bool act[2] = {(bool)((part.mask >> lane) & 1ull), (bool)((part.mask >> (32 + lane)) & 1ull)};
        const uint32_t nsink = (uint32_t)__popcll(part.mask);
        for (int dx = -R; dx <= R; dx++)
            for (int dy = -R; dy <= R; dy++)
                for (int dz = -R; dz <= R; dz++) {
                    const int qx = ((cx + dx) % K + K) % K, qy = ((cy + dy) % K + K) % K, qz = ((cz + dz) % K + K) % K;
                    const uint32_t dd = P.dinfo[((size_t)qx * K + qy) * K + qz];
                    if (!dd) continue;
                    const TreeCell &T = P.tcell[P.crank[dd - 1u]];
                    const float sh[3] = {__fmul_rn((float)dx, P.cw), __fmul_rn((float)dy, P.cw), __fmul_rn((float)dz, P.cw)};
                    // the sinks in the frame of the source cell
                    float px[2], py[2], pz[2];
#pragma unroll
                    for (int h = 0; h < 2; h++) { px[h] = sx[h] - sh[0]; py[h] = sy[h] - sh[1]; pz[h] = sz[h] - sh[2]; }
                    const u64 PX = pk(px[0], px[1]), PY = pk(py[0], py[1]), PZ = pk(pz[0], pz[1]);
                    uint32_t sp = 0, nlist = 0;
                    if (lane == 0) S.stack[0] = (T.nlev - 1u) << 26;
                    sp = 1;
                    __syncwarp();
                    while (sp > 0 || nlist > 0) {
                        uint32_t nleaf = 0;
                        if (sp > 0) {
                            const uint32_t nb = min(32u, sp);
                            bool have = (uint32_t)lane < nb, acc_it = false, far_eps = false;
                            uint32_t l = 0, k = 0, node = 0;
                            if (have) {
                                const uint32_t e = S.stack[sp - 1u - lane];
                                l = e >> 26; k = e & 0x3ffffffu;
                                node = T.base[l] + k;
                                const float4 a = P.nlo[node], b = P.nhi[node];
                                const float nl[3] = {a.x, a.y, a.z}, nh[3] = {b.x, b.y, b.z};
                                float d2 = 0.f, s2 = 0.f;
#pragma unroll
                                for (int q = 0; q < 3; q++) {
                                    const float g1 = __fsub_rn(glo[q], __fadd_rn(nh[q], sh[q])), g2 = __fsub_rn(__fadd_rn(nl[q], sh[q]), ghi[q]);
                                    const float gp = fmaxf(fmaxf(g1, g2), 0.f);
                                    const float e1 = __fsub_rn(nh[q], nl[q]);
                                    d2 = q == 0 ? __fmul_rn(gp, gp) : __fadd_rn(d2, __fmul_rn(gp, gp));
                                    s2 = q == 0 ? __fmul_rn(e1, e1) : __fadd_rn(s2, __fmul_rn(e1, e1));
                                }
                                far_eps = d2 > P.eps2;
                                acc_it = far_eps && s2 < __fmul_rn(P.th2, d2);
                            }
                            sp -= nb;
                            __syncwarp();
                            // accepted nodes -> list
                            const uint32_t am = __ballot_sync(0xffffffffu, have && acc_it);
                            if (have && acc_it) put_dup(S.list + 2 * (nlist + __popc(am & ((1u << lane) - 1u))), P.ncom[node]);
                            nlist += __popc(am);
                            st_node += (unsigned long long)__popc(am) * nsink;
                            // opened leaves -> this batch's leaf list
                            const bool openl = have && !acc_it && l == 0;
                            const uint32_t lm = __ballot_sync(0xffffffffu, openl);
                            if (openl) S.leaves[__popc(lm & ((1u << lane) - 1u))] = k | (far_eps ? 1u << 31 : 0u);
                            nleaf = __popc(lm);
                            st_leaf += (unsigned long long)__reduce_add_sync(0xffffffffu, openl ? min((uint32_t)LEAF, T.n - (uint32_t)LEAF * k) : 0u) * nsink;
                            // opened nodes -> their children on the stack
                            const bool openn = have && !acc_it && l > 0;
                            uint32_t nch = 0;
                            if (openn) nch = min(8u, T.cnt[l - 1u] - 8u * k);
                            uint32_t incl = nch;
#pragma unroll
                            for (int d = 1; d < 32; d <<= 1) {
                                const uint32_t v = __shfl_up_sync(0xffffffffu, incl, d);
                                if (lane >= d) incl += v;
                            }
                            const uint32_t tot = __shfl_sync(0xffffffffu, incl, 31);
                            if (sp + tot > (uint32_t)STACK_CAP) __trap();      // cannot happen (see STACK_CAP)
                            // lane 0 held the top of the stack (the lowest level): its children go on top again, so that
                            // levels never increase towards the top and the stack stays within 256 entries per level
                            for (uint32_t j = 0; j < nch; j++) S.stack[sp + (tot - incl) + j] = ((l - 1u) << 26) | (8u * k + j);
                            sp += tot;
                            __syncwarp();
                        }
                        // the leaves opened by this batch, four at a time, particle by particle: the full softened law, or the
                        // bare m / r^2 where the boxes prove every pair of the leaf further apart than eps (the same values)
                        for (uint32_t i = 0; i < nleaf; i += 4) {
#pragma unroll
                            for (int rr = 0; rr < 2; rr++) {
                                const uint32_t li = i + 2u * rr + ((uint32_t)lane >> 4);
                                float4 q = make_float4(FILL, FILL, FILL, 0.f);           // massless filler
                                if (li < nleaf) q = P.tpos[(size_t)T.coff + (size_t)LEAF * (S.leaves[li] & 0x7fffffffu) + (lane & 15)];
                                put_dup(S.stage + 2 * (32 * rr + lane), q);
                            }
                            __syncwarp();
                            const uint32_t nl = min(4u, nleaf - i);
                            u64 LX = 0, LY = 0, LZ = 0;                                   // formed from zero, then added: shorter sums
                            for (uint32_t q4 = 0; q4 < nl; q4++) {
                                const ulonglong2 *src = S.stage + 2 * LEAF * q4;
                                if (P.plummer) sweep2<2>(src, LEAF, PX, PY, PZ, SC, LX, LY, LZ);
                                else if (S.leaves[i + q4] >> 31) sweep2<0>(src, LEAF, PX, PY, PZ, SC, LX, LY, LZ);
                                else sweep2<1>(src, LEAF, PX, PY, PZ, SC, LX, LY, LZ);
                            }
                            float lx[2], ly[2], lz[2];
                            upk(LX, lx[0], lx[1]); upk(LY, ly[0], ly[1]); upk(LZ, lz[0], lz[1]);
#pragma unroll
                            for (int h = 0; h < 2; h++) if (act[h]) { ax[h] += lx[h]; ay[h] += ly[h]; az[h] += lz[h]; }
                            __syncwarp();
                        }
                        // accepted nodes: evaluate when the list could not take another batch, or at the end of the walk
                        if (nlist > (uint32_t)(LIST_CAP - 32) || (sp == 0 && nlist > 0)) {
                            u64 LX = 0, LY = 0, LZ = 0;
                            if (P.plummer) sweep2<2>(S.list, nlist, PX, PY, PZ, SC, LX, LY, LZ);
                            else sweep2<0>(S.list, nlist, PX, PY, PZ, SC, LX, LY, LZ);
                            float lx[2], ly[2], lz[2];
                            upk(LX, lx[0], lx[1]); upk(LY, ly[0], ly[1]); upk(LZ, lz[0], lz[1]);
#pragma unroll
                            for (int h = 0; h < 2; h++) if (act[h]) { ax[h] += lx[h]; ay[h] += ly[h]; az[h] += lz[h]; }
                            nlist = 0;
                            __syncwarp();
                        }
                    }
                }
#pragma unroll
        for (int h = 0; h < 2; h++)
            if (valid[h] && act[h]) {
                const uint64_t o = P.perm ? (uint64_t)P.perm[slot[h]] : slot[h];
                P.acc[3 * o + 0] += P.Gm * ax[h];
                P.acc[3 * o + 1] += P.Gm * ay[h];
                P.acc[3 * o + 2] += P.Gm * az[h];
            }
        }   // the part
        __syncwarp();          // S.part is rewritten by the next item
    }
    for (int d = 16; d > 0; d >>= 1) {
        st_node += __shfl_xor_sync(0xffffffffu, st_node, d);
        st_leaf += __shfl_xor_sync(0xffffffffu, st_leaf, d);
    }
    if (lane == 0 && (st_node | st_leaf)) {
        atomicAdd(P.stats, st_node / 32ull);        // every lane carried the same count (integer atomics: order-independent)
        atomicAdd(P.stats + 1, st_leaf / 32ull);
    }
}

// one warp per cell: maximum of |a| over its particles, from the final accelerations
__global__ void __launch_bounds__(256) k_tree_amax(const uint64_t *__restrict__ off, const uint32_t *__restrict__ perm,
                                                   const float *__restrict__ acc, size_t ncell, float *__restrict__ amax)
{
    const size_t c = (size_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (c >= ncell) return;
    const int lane = threadIdx.x & 31;
    float m = 0.f;
    for (uint64_t s = off[c] + lane; s < off[c + 1]; s += 32) {
        const uint64_t o = perm ? (uint64_t)perm[s] : s;
        const float x = acc[3 * o], y = acc[3 * o + 1], z = acc[3 * o + 2];
        m = fmaxf(m, x * x + y * y + z * z);
    }
    for (int d = 16; d > 0; d >>= 1) m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, d));
    if (lane == 0) amax[c] = sqrtf(m);
}

size_t tree_groups_max(int64_t N, size_t ncell) { return (size_t)N / 64 + ncell + 1; }    // sum over cells of ceil(n / 64)
size_t tree_nodes_max(int64_t N) { return (size_t)(nf_dense_cap(N) / LEAF) * 8 / 7 + (size_t)MAXLEV * NF_DENSE_MAX_CELLS + 64; }

}  // namespace

size_t nf_tree_scratch_bytes(int64_t N, size_t ncell)
{
    const size_t cap = nf_dense_cap(N), nn = tree_nodes_max(N);
    size_t b = nf_align_up((size_t)NF_DENSE_MAX_CELLS * sizeof(nf_dense_cell), 256) + 256 + 256;      // kept by nf_dense, sentinel
    b += nf_align_up((size_t)NF_DENSE_MAX_CELLS * sizeof(TreeCell), 256) + nf_align_up(cap / 64 * sizeof(uint32_t), 256);
    b += nf_align_up(cap * sizeof(float4), 256) + 3 * nf_align_up(nn * sizeof(float4), 256);
    b += 2 * nf_align_up((ncell + 1) * sizeof(uint32_t), 256) + nf_align_up(nf_scan_temp_elems(ncell + 1) * sizeof(uint32_t), 256);
    const size_t ng = tree_groups_max(N, ncell) + 1;
    b += 2 * nf_align_up(ng * sizeof(uint32_t), 256) + nf_align_up(nf_scan_temp_elems(ng) * sizeof(uint32_t), 256);       // np, poff
    return b + 4096;
}

int nf_tree_sentinel(nf_ctx *ctx, float4 *sentinel, cudaStream_t st)
{
    k_tree_sentinel<<<1, 32, 0, st>>>(sentinel);
    NF_LAUNCHED(ctx);
    return NF_OK;
}

int nf_tree_forces_impl(nf_ctx *ctx, const nf_force_params &p, float theta, const float4 *pos, const uint64_t *off, const uint32_t *perm,
                        int64_t N, const uint32_t *dinfo, const uint32_t *dslot, const nf_dense_keep &keep, float *acc,
                        float *cell_amax, cudaStream_t st)
{
    const int K = p.K;
    const size_t ncell = (size_t)K * K * K;
    const size_t cap = nf_dense_cap(N), nn = tree_nodes_max(N);
    TreeCell *tcell = nf_scratch_take<TreeCell>(ctx, NF_DENSE_MAX_CELLS);
    uint32_t *crank = nf_scratch_take<uint32_t>(ctx, cap / 64);
    float4 *tpos = nf_scratch_take<float4>(ctx, cap);
    float4 *nlo = nf_scratch_take<float4>(ctx, nn), *nhi = nf_scratch_take<float4>(ctx, nn), *ncom = nf_scratch_take<float4>(ctx, nn);
    uint32_t *ng = nf_scratch_take<uint32_t>(ctx, ncell + 1), *goff = nf_scratch_take<uint32_t>(ctx, ncell + 1);
    uint32_t *stmp = nf_scratch_take<uint32_t>(ctx, nf_scan_temp_elems(ncell + 1));
    const size_t ngm = tree_groups_max(N, ncell) + 1;
    uint32_t *np = nf_scratch_take<uint32_t>(ctx, ngm), *poff = nf_scratch_take<uint32_t>(ctx, ngm);
    uint32_t *ptmp = nf_scratch_take<uint32_t>(ctx, nf_scan_temp_elems(ngm));
    if (!tcell || !crank || !tpos || !nlo || !nhi || !ncom || !ng || !goff || !stmp || !np || !poff || !ptmp) {
        NF_SET_ERR(ctx, "nf_forces_tree: internal scratch arena too small");
        return NF_ERR_NOMEM;
    }
    unsigned long long *stats = ctx->counters + 8;          // [8] node, [9] leaf interactions, [10] work cursor
    NF_CUDA(ctx, cudaMemsetAsync(stats, 0, 3 * sizeof(unsigned long long), st));
    k_tree_layout<<<1, 32, 0, st>>>(keep.dcell, keep.nd, tcell, crank);
    NF_LAUNCHED(ctx);
    const uint32_t nchunk = (uint32_t)(cap / 64);
    const unsigned grid = (unsigned)(nchunk / 8 < 148u * 16u ? (nchunk + 7) / 8 : 148u * 16u);
    if (p.softening & NF_MASS_W) k_tree_leaves<true><<<grid, 256, 0, st>>>(pos, dslot, keep.nd, tcell, tpos, nlo, nhi, ncom, nchunk);
    else k_tree_leaves<false><<<grid, 256, 0, st>>>(pos, dslot, keep.nd, tcell, tpos, nlo, nhi, ncom, nchunk);
    NF_LAUNCHED(ctx);
    // levels above the leaves: a cell of n particles has ceil(log8(n / 64)) of them; the box holds at most N particles
    int maxlev = 1;
    for (uint64_t m = ((uint64_t)N + LEAF - 1) / LEAF; m > 1; m = (m + 7) / 8) maxlev++;
    for (int l = 1; l < maxlev && l < MAXLEV; l++) {
        const uint64_t per = (((uint64_t)N + LEAF - 1) / LEAF >> (3 * l)) + 1;
        dim3 g((unsigned)((per + 127) / 128 < 64 ? (per + 127) / 128 : 64), NF_DENSE_MAX_CELLS);
        k_tree_level<<<g, 128, 0, st>>>(keep.nd, tcell, l, nlo, nhi, ncom);
        NF_LAUNCHED(ctx);
    }
    k_tree_items<<<(unsigned)((ncell + 1 + 255) / 256), 256, 0, st>>>(off, dinfo, K, p.R, ncell, ng);
    NF_LAUNCHED(ctx);
    NF_TRY(nf_exclusive_scan_u32(ctx, ng, goff, ncell + 1, stmp, st));
    WalkParams W;
    W.pos = pos; W.off = off; W.perm = perm; W.dinfo = dinfo; W.dslot = dslot; W.tcell = tcell; W.crank = crank; W.tpos = tpos;
    W.nlo = nlo; W.nhi = nhi; W.ncom = ncom; W.goff = goff; W.np = np; W.poff = poff; W.acc = acc; W.stats = stats;
    W.cursor = reinterpret_cast<uint32_t *>(stats + 2);
    W.ncell = ncell; W.K = K; W.R = p.R; W.plummer = (p.softening & NF_SOFT_LAW_MASK) == NF_SOFT_PLUMMER ? 1 : 0;
    W.cw = p.box / (float)K; W.eps = p.eps; W.eps2 = p.eps * p.eps; W.th2 = theta * theta; W.Gm = p.Gm;
    const size_t smem = sizeof(WalkShared) * WALK_WARPS;
    NF_CUDA(ctx, cudaFuncSetAttribute(k_tree_walk<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    NF_CUDA(ctx, cudaFuncSetAttribute(k_tree_walk<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    // parts per group, scanned: the walk's work list is over (group, part) pairs
    NF_CUDA(ctx, cudaMemsetAsync(np, 0, ngm * sizeof(uint32_t), st));
    const size_t cblocks = (ngm + WALK_WARPS - 1) / WALK_WARPS;
    k_tree_walk<true><<<(unsigned)(cblocks < (size_t)ctx->sm_count * 2 ? cblocks : (size_t)ctx->sm_count * 2), WALK_WARPS * 32, smem, st>>>(W);
    NF_LAUNCHED(ctx);
    NF_TRY(nf_exclusive_scan_u32(ctx, np, poff, ngm, ptmp, st));
    NF_CUDA(ctx, cudaEventRecord(ctx->ev_walk0, st));
    k_tree_walk<false><<<(unsigned)ctx->sm_count * 2, WALK_WARPS * 32, smem, st>>>(W);
    NF_LAUNCHED(ctx);
    NF_CUDA(ctx, cudaEventRecord(ctx->ev_walk1, st));
    ctx->tree_timed = true;
    if (cell_amax) {
        k_tree_amax<<<(unsigned)((ncell + 7) / 8), 256, 0, st>>>(off, perm, acc, ncell, cell_amax);
        NF_LAUNCHED(ctx);
    }
    return NF_OK;
}
