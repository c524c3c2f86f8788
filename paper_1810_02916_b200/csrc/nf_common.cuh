// nf_common.cuh -- context, error handling and scratch arena shared by the libnf sources.
// Part of the CUDA product path; shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>
#include <string.h>

#include "../../include/nf.h"

#define NF_VERSION_NUM 100

struct nf_ctx {
    int device;
    int sm_count;
    char err[512];
    // bump-allocated device scratch (grown on demand; growth synchronises the device)
    char *scratch;
    size_t scratch_bytes;
    size_t scratch_used;
    // small persistent device counters: [0] out-of-range particles, [1] interactions, [2] work cursor
    unsigned long long *counters;
    unsigned long long *h_counters;  // pinned host mirror
    // timing of the last nf_forces
    cudaEvent_t ev_total0, ev_kern0, ev_kern1, ev_total1;
    bool forces_timed;
    cudaEvent_t ev_walk0, ev_walk1;   // around the walk kernel of the last nf_forces_tree
    bool tree_timed;
    long long launches;  // kernels launched by this context since nf_create
    // slab streaming resources (created lazily)
    cudaStream_t s_h2d, s_d2h;
    void *slab_state;
    void *host_pipe;     // nf_forces_host_begin / _end (created lazily)
};

#define NF_SET_ERR(ctx, ...)                                        \
    do {                                                            \
        if (ctx) snprintf((ctx)->err, sizeof((ctx)->err), __VA_ARGS__); \
    } while (0)

#define NF_CUDA(ctx, call)                                                                   \
    do {                                                                                     \
        cudaError_t e__ = (call);                                                            \
        if (e__ != cudaSuccess) {                                                            \
            NF_SET_ERR(ctx, "CUDA error %d (%s) at %s:%d: %s", (int)e__, cudaGetErrorName(e__), \
                       __FILE__, __LINE__, cudaGetErrorString(e__));                         \
            return e__ == cudaErrorMemoryAllocation ? NF_ERR_NOMEM : NF_ERR_CUDA;            \
        }                                                                                    \
    } while (0)

// after every kernel launch: count it (nf_launch_count) and pick up launch errors
#define NF_LAUNCHED(ctx)                      \
    do {                                      \
        (ctx)->launches++;                    \
        NF_CUDA(ctx, cudaGetLastError());     \
    } while (0)

#define NF_ARG(ctx, cond, ...)           \
    do {                                 \
        if (!(cond)) {                   \
            NF_SET_ERR(ctx, __VA_ARGS__); \
            return NF_ERR_ARG;           \
        }                                \
    } while (0)

#define NF_TRY(call)              \
    do {                          \
        int rc__ = (call);        \
        if (rc__ != NF_OK) return rc__; \
    } while (0)

static inline size_t nf_align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

// Scratch arena: reset at the start of each API call, then carve.
int nf_scratch_reserve(nf_ctx *ctx, size_t bytes);  // ensure capacity (may sync + realloc)
static inline void nf_scratch_reset(nf_ctx *ctx) { ctx->scratch_used = 0; }
template <class T>
static inline T *nf_scratch_take(nf_ctx *ctx, size_t count)
{
    size_t off = nf_align_up(ctx->scratch_used, 256);
    size_t end = off + nf_align_up(count * sizeof(T), 256);
    if (end > ctx->scratch_bytes) return nullptr;
    ctx->scratch_used = end;
    return reinterpret_cast<T *>(ctx->scratch + off);
}

// ---- internal entry points shared between translation units ---------------------------
// exclusive scans (nf_scan.cu); temp must hold nf_scan_temp_elems(n) elements of the out type
size_t nf_scan_temp_elems(size_t n);
int nf_exclusive_scan_u32(nf_ctx *ctx, const uint32_t *in, uint32_t *out, size_t n, uint32_t *temp, cudaStream_t st);
int nf_exclusive_scan_u32_u64(nf_ctx *ctx, const uint32_t *in, uint64_t *out, size_t n, uint64_t *temp, cudaStream_t st);

// binning (nf_bin.cu).  plane_cx < 0: full box, keys (cx*K+cy)*K+cz over K^3 cells;
// plane_cx >= 0: one x-plane, keys cy*K+cz over K^2 cells, particles must have cx == plane_cx.
size_t nf_bin_scratch_bytes(int64_t N, int K, bool plane);
int nf_bin_impl(nf_ctx *ctx, const float *pos, const float *mass /* nullable */, int64_t N, int K, float box, int plane_cx,
                float *pos_sorted, uint32_t *perm, uint32_t *cell_count, uint64_t *cell_offset,
                cudaStream_t st);

int nf_keys_impl(nf_ctx *ctx, const float *pos, int64_t N, int K, float box, uint32_t *keys, cudaStream_t st);

// forces (nf_forces.cu).  A "plane table" describes the x-planes available as sources and
// sinks: plane p (0 <= p < n_planes) has its own cell-contiguous arrays.
struct nf_plane_view {
    const float4 *pos;        // sorted cell-centred offsets of this plane's particles
    const float4 *enc;        // the same particles, scaled and z-block-encoded (nf_encode_impl), blocks from cz = 0
    const float4 *enc_h;      // ... and with the z-blocks shifted by half a block
    const uint64_t *off;      // K*K+1 exclusive offsets within this plane's arrays
    const uint32_t *perm;     // nullable
    float *acc;               // output for this plane (n x 3), nullable for ghost planes
    float *amax;              // nullable: K*K per-cell maxima of |a| (zeroed by the caller; integer atomicMax on the float bits)
    // in-cell ordering of this plane's dense cells (nf_dense.cu); all null = none
    const uint32_t *dinfo;    // K*K words, 0 = cell not dense, else (compact offset of the cell / 64) + 1
    const uint32_t *dslot;    // compact position -> slot (within this plane's arrays) of the particle whose encoded copy sits there
    const float *dbox;        // per 64 compact positions: lo.xyz, hi.xyz of the scaled cell-centred offsets
};
struct nf_force_params {
    int K;            // cells per side in y and z
    int n_planes;     // number of x-planes in the table
    int periodic_x;   // 1: plane index wraps modulo n_planes (full box); 0: open
    int sink_lo, sink_hi;  // sink planes [lo, hi)
    int R;
    float eps, box, Gm;
    int softening;
    long long max_sinks;  // upper bound on the particles in the sink planes (sizes the work list)
    int dense;            // 1: some plane view carries the in-cell ordering of dense cells (selects the kernel instance with that logic)
    int tree;             // 1 (needs dense): the sources of dense cells are left to the tree near field (nf_tree.cu) -- the interaction kernel skips them
    const float4 *sentinel;   // tree: two far-away massless sources, the only tile of a task that has no other source left
};
size_t nf_forces_scratch_bytes(const nf_force_params &p);
// d_planes: DEVICE array of p.n_planes views (fill with nf_fill_planes_full or copy from pinned memory)
int nf_forces_impl(nf_ctx *ctx, const nf_force_params &p, const nf_plane_view *d_planes,
                   cudaStream_t st, bool record_timing);
// the full box seen as K planes sharing one set of arrays: plane cx starts at cell cx*K*K
int nf_fill_planes_full(nf_ctx *ctx, nf_plane_view *d_planes, int K, const float4 *pos, const float4 *enc, const float4 *enc_h,
                        const uint64_t *off, const uint32_t *perm, float *acc, float *cell_amax, const uint32_t *dinfo, const uint32_t *dslot,
                        const float *dbox, cudaStream_t st);
// enc[s], enc_h[s] = the two encoded copies of pos[s] for the ncell cells described by off (cell index % K = cz);
// they depend on p.eps, p.box, p.K
// skip_n > 0: cells of at least skip_n particles are left out -- the caller runs nf_dense_order_impl next, which encodes them
int nf_encode_impl(nf_ctx *ctx, const nf_force_params &p, const float4 *pos, const uint64_t *off, size_t ncell, float4 *enc,
                   float4 *enc_h, cudaStream_t st, uint32_t skip_n = 0);
// In-cell ordering of dense cells (nf_dense.cu), full box only.  Cells of at least NF_DENSE_N particles get their ENCODED
// copies (enc, enc_h: what the interaction kernel reads) re-ordered along a Hilbert curve inside the cell, with a box per 64
// particles, so that the kernel can prove most (task, tile) pairs free of pairs inside eps.  dinfo: K^3 words out.
// `off` describes ncell cells whose index modulo K is cz (the full box: K^3 cells; one plane: K^2).  Outputs: dinfo
// (ncell words), dslot (nf_dense_cap(N) words), dbox (nf_dense_cap(N) / 64 * 6 floats) -- caller-owned, they must live as
// long as the encoded copies; temporaries come from the arena (nf_dense_scratch_bytes).
constexpr int NF_ZB = 8;                // cells per z-block of the encoding (nf_forces.cu k_encode)
constexpr int NF_DENSE_N = 4096;
constexpr int NF_DENSE_MAX_CELLS = 2048;
uint32_t nf_dense_cap(int64_t N);
size_t nf_dense_scratch_bytes(int64_t N, size_t ncell);
// is the ordering taken for a set of N particles in ncell cells?  From the arguments alone (the same call always takes the same path)
static inline bool nf_dense_wanted(int64_t N, size_t ncell, int softening) { return N >= NF_DENSE_N && ((softening & NF_DENSE_ORDER) || (size_t)N / ncell >= 512); }
struct nf_dense_cell { unsigned long long c0; uint32_t coff, cell, n, pad; };   // first slot, compact offset (64-aligned), cell index, particles
// keep (nullable): where the caller wants the table of dense cells (NF_DENSE_MAX_CELLS entries, by rank) and two counters
// (compact length, number of dense cells) to outlive the call -- nf_tree.cu builds on them
struct nf_dense_keep { nf_dense_cell *dcell; uint32_t *nd; };
int nf_dense_order_impl(nf_ctx *ctx, const nf_force_params &p, const float4 *pos, const uint64_t *off, size_t ncell, int64_t N,
                        float4 *enc, float4 *enc_h, uint32_t *dinfo, uint32_t *dslot, float *dbox, cudaStream_t st,
                        const nf_dense_keep *keep = nullptr);
// Tree near field for dense cells (nf_tree.cu, readings t1-t6), whole box only.  Runs after the
// interaction kernel (which skipped the sources of dense cells: p.tree) and ADDS the dense cells' attraction to acc.
size_t nf_tree_scratch_bytes(int64_t N, size_t ncell);
int nf_tree_forces_impl(nf_ctx *ctx, const nf_force_params &p, float theta, const float4 *pos, const uint64_t *off, const uint32_t *perm,
                        int64_t N, const uint32_t *dinfo, const uint32_t *dslot, const nf_dense_keep &keep, float *acc,
                        float *cell_amax, cudaStream_t st);
// writes the two sentinel sources (p.sentinel); part of the tree path, launched before the interaction kernel
int nf_tree_sentinel(nf_ctx *ctx, float4 *sentinel, cudaStream_t st);
size_t nf_radix_tiles(int64_t n_max);
int nf_radix_pass(nf_ctx *ctx, const uint32_t *kin, const uint32_t *iin, int64_t n_max, const uint32_t *n_dev, uint32_t bins,
                  uint32_t shift, uint32_t *kout, uint32_t *iout, uint32_t *hist, uint32_t *tmp32, cudaStream_t st);
// encoding constants shared by nf_forces.cu and nf_dense.cu
void nf_encode_consts(const nf_force_params &p, float *scale, float *ws);
// once per context: uploads the task-split table
int nf_forces_init(nf_ctx *ctx);
// ordered pairs evaluated for the sink planes of a plane table (device result added to ctx->counters[1])
int nf_interactions_planes(nf_ctx *ctx, const nf_force_params &p, const nf_plane_view *d_planes, cudaStream_t st);
void nf_slab_state_free(nf_ctx *ctx);
void nf_host_pipe_free(nf_ctx *ctx);
// kick + drift launcher (nf_step.cu), also the epilogue of nf_stream_step_slabs
int nf_kick_drift_impl(nf_ctx *ctx, float *pos, float *vel, const float *acc, int64_t N, float kick, float drift, float box,
                       cudaStream_t st);
int nf_interactions_impl(nf_ctx *ctx, const uint32_t *cell_count, int K, int R, int64_t *out, cudaStream_t st);
// regrouping after the drift (nf_regroup.cu): [to plane-1 | stay | to plane+1], stable; scratch from the arena
size_t nf_regroup_scratch_bytes(int64_t N);
int nf_regroup_impl(nf_ctx *ctx, const float *pos, const float *vel, int64_t n, int K, float box, int plane_cx, float *pos_out,
                    float *vel_out, unsigned long long *seg_n, cudaStream_t st);
