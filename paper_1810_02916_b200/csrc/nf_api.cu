// nf_api.cu -- extern "C" entry points declared in include/nf.h (argument checks, scratch
// sizing, dispatch).  Every step of the path runs in the kernels of nf_bin.cu / nf_forces.cu.
#include <new>

#include "nf_common.cuh"

static const char *const k_no_ctx = "nf: null context";

struct HostPipe {                    // state of nf_forces_host_begin / _end
    int active, next;                // steps in flight (0..2); buffer pair of the next begin
    int64_t N;
    int K;
    size_t shared_at;                // arena offset where the part shared by all steps starts
    float *raw[2], *acc[2];          // doubled input / output buffers (arena)
    bool used[2];
    cudaEvent_t ev_h2d[2], ev_raw_free[2], ev_done[2], ev_d2h[2];
    unsigned long long *h_bad;       // pinned [2]: out-of-range count of each step
};

void nf_host_pipe_free(nf_ctx *ctx)
{
    HostPipe *hp = static_cast<HostPipe *>(ctx->host_pipe);
    if (!hp) return;
    for (int i = 0; i < 2; i++) {
        if (hp->ev_h2d[i]) cudaEventDestroy(hp->ev_h2d[i]);
        if (hp->ev_raw_free[i]) cudaEventDestroy(hp->ev_raw_free[i]);
        if (hp->ev_done[i]) cudaEventDestroy(hp->ev_done[i]);
        if (hp->ev_d2h[i]) cudaEventDestroy(hp->ev_d2h[i]);
    }
    if (hp->h_bad) cudaFreeHost(hp->h_bad);
    delete hp;
    ctx->host_pipe = nullptr;
}

int nf_scratch_reserve(nf_ctx *ctx, size_t bytes)
{
    if (bytes <= ctx->scratch_bytes) return NF_OK;
    NF_CUDA(ctx, cudaDeviceSynchronize());
    if (ctx->scratch) NF_CUDA(ctx, cudaFree(ctx->scratch));
    ctx->scratch = nullptr;
    ctx->scratch_bytes = 0;
    size_t want = nf_align_up(bytes + bytes / 16, 1 << 20);
    cudaError_t e = cudaMalloc((void **)&ctx->scratch, want);
    if (e != cudaSuccess) {
        cudaGetLastError();
        NF_SET_ERR(ctx, "cudaMalloc of %zu scratch bytes failed: %s", want, cudaGetErrorString(e));
        return NF_ERR_NOMEM;
    }
    ctx->scratch_bytes = want;
    return NF_OK;
}

extern "C" {

int nf_version(void) { return NF_VERSION_NUM; }

int nf_create(nf_ctx **out, int device)
{
    if (!out) return NF_ERR_ARG;
    *out = nullptr;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev) {
        cudaGetLastError();
        return NF_ERR_CUDA;
    }
    nf_ctx *ctx = new (std::nothrow) nf_ctx();
    if (!ctx) return NF_ERR_NOMEM;
    memset(ctx, 0, sizeof(*ctx));
    ctx->device = device;
    int rc = NF_OK;
    do {
        if (cudaSetDevice(device) != cudaSuccess) { rc = NF_ERR_CUDA; break; }
        if (cudaDeviceGetAttribute(&ctx->sm_count, cudaDevAttrMultiProcessorCount, device) != cudaSuccess) { rc = NF_ERR_CUDA; break; }
        if (cudaMalloc((void **)&ctx->counters, 16 * sizeof(unsigned long long)) != cudaSuccess) { rc = NF_ERR_NOMEM; break; }
        if (cudaMemset(ctx->counters, 0, 16 * sizeof(unsigned long long)) != cudaSuccess) { rc = NF_ERR_CUDA; break; }
        if (cudaMallocHost((void **)&ctx->h_counters, 16 * sizeof(unsigned long long)) != cudaSuccess) { rc = NF_ERR_NOMEM; break; }
        memset(ctx->h_counters, 0, 16 * sizeof(unsigned long long));
        if (cudaEventCreate(&ctx->ev_total0) != cudaSuccess || cudaEventCreate(&ctx->ev_kern0) != cudaSuccess ||
            cudaEventCreate(&ctx->ev_kern1) != cudaSuccess || cudaEventCreate(&ctx->ev_total1) != cudaSuccess ||
            cudaEventCreate(&ctx->ev_walk0) != cudaSuccess || cudaEventCreate(&ctx->ev_walk1) != cudaSuccess) { rc = NF_ERR_CUDA; break; }
        if (cudaStreamCreateWithFlags(&ctx->s_h2d, cudaStreamNonBlocking) != cudaSuccess ||
            cudaStreamCreateWithFlags(&ctx->s_d2h, cudaStreamNonBlocking) != cudaSuccess) { rc = NF_ERR_CUDA; break; }
        rc = nf_forces_init(ctx);
    } while (0);
    if (rc != NF_OK) {
        cudaGetLastError();
        nf_destroy(ctx);
        return rc;
    }
    *out = ctx;
    return NF_OK;
}

int nf_destroy(nf_ctx *ctx)
{
    if (!ctx) return NF_OK;
    cudaSetDevice(ctx->device);
    cudaDeviceSynchronize();
    if (ctx->scratch) cudaFree(ctx->scratch);
    if (ctx->counters) cudaFree(ctx->counters);
    if (ctx->h_counters) cudaFreeHost(ctx->h_counters);
    if (ctx->ev_total0) cudaEventDestroy(ctx->ev_total0);
    if (ctx->ev_kern0) cudaEventDestroy(ctx->ev_kern0);
    if (ctx->ev_kern1) cudaEventDestroy(ctx->ev_kern1);
    if (ctx->ev_total1) cudaEventDestroy(ctx->ev_total1);
    if (ctx->ev_walk0) cudaEventDestroy(ctx->ev_walk0);
    if (ctx->ev_walk1) cudaEventDestroy(ctx->ev_walk1);
    if (ctx->s_h2d) cudaStreamDestroy(ctx->s_h2d);
    if (ctx->s_d2h) cudaStreamDestroy(ctx->s_d2h);
    nf_slab_state_free(ctx);
    nf_host_pipe_free(ctx);
    cudaGetLastError();
    delete ctx;
    return NF_OK;
}

const char *nf_last_error(const nf_ctx *ctx) { return ctx ? ctx->err : k_no_ctx; }

static int check_common(nf_ctx *ctx, int64_t N, int K, float box)
{
    NF_ARG(ctx, N >= 0 && N < ((int64_t)1 << 32), "N = %lld out of range [0, 2^32)", (long long)N);
    NF_ARG(ctx, K >= 1 && K <= NF_MAX_K, "K = %d out of range [1, %d]", K, NF_MAX_K);
    NF_ARG(ctx, box > 0.0f && box < 3.0e38f, "box must be positive and finite");
    return NF_OK;
}

static size_t forces_scratch_full(int64_t N, int K)
{
    nf_force_params p{};
    p.K = K;
    p.n_planes = K;
    p.sink_lo = 0;
    p.sink_hi = K;
    p.max_sinks = N;
    return nf_forces_scratch_bytes(p) + 2 * nf_align_up((size_t)(N > 0 ? N : 1) * 16, 256);   // + the two encoded copies
}

static size_t dense_full_bytes(int64_t N, int K, int softening);

int nf_reserve(nf_ctx *ctx, int64_t maxN, int K)
{
    if (!ctx) return NF_ERR_ARG;
    NF_TRY(check_common(ctx, maxN, K, 1.0f));
    NF_CUDA(ctx, cudaSetDevice(ctx->device));
    size_t need = nf_bin_scratch_bytes(maxN, K, false);
    // (the in-cell ordering of dense cells is reserved for where it is automatic; a call that asks for it with
    // NF_DENSE_ORDER on a sparser box grows the arena once)
    size_t f = forces_scratch_full(maxN, K) + dense_full_bytes(maxN, K, 0);
    return nf_scratch_reserve(ctx, need > f ? need : f);
}

int nf_bin(nf_ctx *ctx, const float *pos_xyz, int64_t N, int K, float box, float *pos_sorted,
           uint32_t *perm, uint32_t *cell_count, uint64_t *cell_offset, void *stream)
{
    return nf_bin_m(ctx, pos_xyz, nullptr, N, K, box, pos_sorted, perm, cell_count, cell_offset, stream);
}

int nf_bin_m(nf_ctx *ctx, const float *pos_xyz, const float *mass, int64_t N, int K, float box, float *pos_sorted,
             uint32_t *perm, uint32_t *cell_count, uint64_t *cell_offset, void *stream)
{
    if (!ctx) return NF_ERR_ARG;
    NF_TRY(check_common(ctx, N, K, box));
    NF_ARG(ctx, cell_count && cell_offset, "nf_bin: cell_count / cell_offset must not be null");
    NF_ARG(ctx, N == 0 || (pos_xyz && pos_sorted && perm), "nf_bin: null particle array with N > 0");
    NF_ARG(ctx, ((uintptr_t)pos_sorted & 15) == 0, "nf_bin: pos_sorted must be 16-byte aligned");
    NF_CUDA(ctx, cudaSetDevice(ctx->device));
    NF_TRY(nf_scratch_reserve(ctx, nf_bin_scratch_bytes(N, K, false)));
    nf_scratch_reset(ctx);
    NF_CUDA(ctx, cudaMemsetAsync(ctx->counters, 0, sizeof(unsigned long long), (cudaStream_t)stream));
    return nf_bin_impl(ctx, pos_xyz, mass, N, K, box, -1, pos_sorted, perm, cell_count, cell_offset, (cudaStream_t)stream);
}

int nf_out_of_range(nf_ctx *ctx, int64_t *n, void *stream)
{
    if (!ctx) return NF_ERR_ARG;
    NF_ARG(ctx, n != nullptr, "nf_out_of_range: null output");
    NF_CUDA(ctx, cudaSetDevice(ctx->device));
    cudaStream_t st = (cudaStream_t)stream;
    NF_CUDA(ctx, cudaMemcpyAsync(ctx->h_counters, ctx->counters, sizeof(unsigned long long), cudaMemcpyDeviceToHost, st));
    NF_CUDA(ctx, cudaStreamSynchronize(st));
    *n = (int64_t)ctx->h_counters[0];
    if (*n) {
        NF_SET_ERR(ctx, "%lld particle(s) outside [0, box) were clamped into edge cells", (long long)*n);
        return NF_ERR_RANGE;
    }
    return NF_OK;
}

static int check_force_args(nf_ctx *ctx, int K, int R, float eps, float Gm, int softening)
{
    NF_ARG(ctx, R >= 0 && R <= NF_MAX_R, "R = %d out of range [0, %d]", R, NF_MAX_R);
    NF_ARG(ctx, K >= 2 * R + 1, "K = %d < 2R+1 = %d would list a neighbour cell twice", K, 2 * R + 1);
    NF_ARG(ctx, eps > 0.0f && eps < 3.0e38f, "eps must be positive and finite");
    NF_ARG(ctx, Gm == Gm && fabsf(Gm) < 3.0e38f, "Gm must be finite");
    const int law = softening & NF_SOFT_LAW_MASK;
    NF_ARG(ctx, (law == NF_SOFT_SPLINE || law == NF_SOFT_PLUMMER) && (softening & ~(NF_SOFT_LAW_MASK | NF_MASS_W | NF_DENSE_ORDER)) == 0,
           "unknown softening %d", softening);
    return NF_OK;
}

// Arena bytes of the in-cell ordering of dense cells for a whole box (temporaries + its three outputs), 0 when not taken
static size_t dense_full_bytes(int64_t N, int K, int softening)
{
    const size_t ncell = (size_t)K * K * K;
    if (!nf_dense_wanted(N, ncell, softening)) return 0;
    const size_t cap = nf_dense_cap(N);
    return nf_dense_scratch_bytes(N, ncell) + nf_align_up(ncell * 4, 256) + nf_align_up(cap * 4, 256) + nf_align_up(cap / 64 * 24, 256) + 1024;
}

// Encoded copies of a whole box, the in-cell ordering of its dense cells where it is wanted (nf_dense.cu; outputs taken
// from the arena), and the plane table.  Clears NF_DENSE_ORDER in p.softening and sets p.dense.
struct TreeHandles { uint32_t *dinfo, *dslot; nf_dense_keep keep; };
static int encode_full(nf_ctx *ctx, nf_force_params &p, const float4 *ps, const uint64_t *off, const uint32_t *perm, int64_t N,
                       float4 *enc, float4 *enc_h, nf_plane_view *d_planes, float *acc, float *cell_amax, cudaStream_t st,
                       TreeHandles *tree = nullptr)
{
    const int K = p.K;
    const size_t ncell = (size_t)K * K * K;
    const bool dense = nf_dense_wanted(N, ncell, p.softening | (tree ? NF_DENSE_ORDER : 0));
    p.softening &= ~NF_DENSE_ORDER;
    NF_TRY(nf_encode_impl(ctx, p, ps, off, ncell, enc, enc_h, st, dense ? NF_DENSE_N : 0));
    uint32_t *dinfo = nullptr, *dslot = nullptr;
    float *dbox = nullptr;
    if (dense) {
        const size_t cap = nf_dense_cap(N);
        dinfo = nf_scratch_take<uint32_t>(ctx, ncell);
        dslot = nf_scratch_take<uint32_t>(ctx, cap);
        dbox = nf_scratch_take<float>(ctx, cap / 64 * 6);
        if (!dinfo || !dslot || !dbox) { NF_SET_ERR(ctx, "nf_forces: internal scratch arena too small (dense-cell ordering)"); return NF_ERR_NOMEM; }
        nf_dense_keep keep{nullptr, nullptr};
        float4 *sentinel = nullptr;
        if (tree) {                                // nf_tree.cu builds on the table of dense cells; the kernel needs a sentinel tile
            keep.dcell = nf_scratch_take<nf_dense_cell>(ctx, NF_DENSE_MAX_CELLS);
            keep.nd = nf_scratch_take<uint32_t>(ctx, 64);
            sentinel = nf_scratch_take<float4>(ctx, 16);
            if (!keep.dcell || !keep.nd || !sentinel) { NF_SET_ERR(ctx, "nf_forces_tree: internal scratch arena too small"); return NF_ERR_NOMEM; }
        }
        const size_t mark = ctx->scratch_used;
        NF_TRY(nf_dense_order_impl(ctx, p, ps, off, ncell, N, enc, enc_h, dinfo, dslot, dbox, st, tree ? &keep : nullptr));
        ctx->scratch_used = mark;                  // its temporaries are dead once enqueued work is ordered: same stream
        p.dense = 1;
        if (tree) {
            NF_TRY(nf_tree_sentinel(ctx, sentinel, st));
            p.tree = 1; p.sentinel = sentinel;
            tree->dinfo = dinfo; tree->dslot = dslot; tree->keep = keep;
        }
    }
    // with the tree the per-cell maxima come from the final accelerations (nf_tree.cu), not from the kernel's epilogue
    return nf_fill_planes_full(ctx, d_planes, K, ps, enc, enc_h, off, perm, acc, p.tree ? nullptr : cell_amax, dinfo, dslot, dbox, st);
}

// nf_forces / nf_forces_ex / nf_forces_chunk: sinks are the particles of the x-planes [x_lo, x_hi)
static int forces_common(nf_ctx *ctx, const float *pos_sorted, const uint64_t *cell_offset, const uint32_t *perm, int64_t N, int K,
                         int R, float eps, float box, float Gm, int softening, int x_lo, int x_hi, float *acc_xyz, float *cell_amax,
                         void *stream, bool tree = false, float theta = 0.f)
{
    NF_TRY(check_common(ctx, N, K, box));
    NF_TRY(check_force_args(ctx, K, R, eps, Gm, softening));
    NF_ARG(ctx, cell_offset != nullptr, "nf_forces: cell_offset must not be null");
    NF_ARG(ctx, N == 0 || (pos_sorted && acc_xyz), "nf_forces: null particle array with N > 0");
    NF_ARG(ctx, ((uintptr_t)pos_sorted & 15) == 0, "nf_forces: pos_sorted must be 16-byte aligned");
    NF_ARG(ctx, 0 <= x_lo && x_lo <= x_hi && x_hi <= K, "sink plane range [%d, %d) is not inside [0, %d]", x_lo, x_hi, K);
    NF_CUDA(ctx, cudaSetDevice(ctx->device));
    if (N == 0 || x_lo == x_hi) {
        if (cell_amax) NF_CUDA(ctx, cudaMemsetAsync(cell_amax, 0, sizeof(float) * (size_t)K * K * K, (cudaStream_t)stream));
        return NF_OK;
    }
    nf_force_params p{};
    p.K = K; p.n_planes = K; p.periodic_x = 1; p.sink_lo = x_lo; p.sink_hi = x_hi;
    p.R = R; p.eps = eps; p.box = box; p.Gm = Gm; p.softening = softening; p.max_sinks = N;
    nf_scratch_reset(ctx);
    const size_t ncell = (size_t)K * K * K;
    tree = tree && N >= NF_DENSE_N;                    // no cell can be dense below that: the plain path
    NF_TRY(nf_scratch_reserve(ctx, forces_scratch_full(N, K) + dense_full_bytes(N, K, softening | (tree ? NF_DENSE_ORDER : 0)) +
                                       (tree ? nf_tree_scratch_bytes(N, ncell) : 0)));
    nf_plane_view *d_planes = nf_scratch_take<nf_plane_view>(ctx, (size_t)K);
    float4 *enc = nf_scratch_take<float4>(ctx, (size_t)N);
    float4 *enc_h = nf_scratch_take<float4>(ctx, (size_t)N);
    if (!d_planes || !enc || !enc_h) { NF_SET_ERR(ctx, "nf_forces: internal scratch arena too small"); return NF_ERR_NOMEM; }
    cudaStream_t st = (cudaStream_t)stream;
    const float4 *ps = reinterpret_cast<const float4 *>(pos_sorted);
    if (cell_amax) NF_CUDA(ctx, cudaMemsetAsync(cell_amax, 0, sizeof(float) * (size_t)K * K * K, st));
    TreeHandles th{};
    NF_TRY(encode_full(ctx, p, ps, cell_offset, perm, N, enc, enc_h, d_planes, acc_xyz, cell_amax, st, tree ? &th : nullptr));
    NF_TRY(nf_forces_impl(ctx, p, d_planes, st, true));
    if (tree) NF_TRY(nf_tree_forces_impl(ctx, p, theta, ps, cell_offset, perm, N, th.dinfo, th.dslot, th.keep, acc_xyz, cell_amax, st));
    return NF_OK;
}

int nf_forces_tree(nf_ctx *ctx, const float *pos_sorted, const uint64_t *cell_offset, const uint32_t *perm, int64_t N, int K, int R,
                   float eps, float box, float Gm, int softening, float theta, float *acc_xyz, float *cell_amax, void *stream)
{
    if (!ctx) return NF_ERR_ARG;
    NF_ARG(ctx, theta >= 0.0f && theta < 1.0f, "nf_forces_tree: theta = %g outside [0, 1)", (double)theta);
    return forces_common(ctx, pos_sorted, cell_offset, perm, N, K, R, eps, box, Gm, softening, 0, K, acc_xyz, cell_amax, stream, true, theta);
}

int nf_last_tree_timing(nf_ctx *ctx, float *walk_ms)
{
    if (!ctx) return NF_ERR_ARG;
    NF_ARG(ctx, walk_ms != nullptr, "nf_last_tree_timing: null output");
    NF_ARG(ctx, ctx->tree_timed, "nf_last_tree_timing: no nf_forces_tree has walked a tree on this context yet");
    NF_CUDA(ctx, cudaEventSynchronize(ctx->ev_walk1));
    NF_CUDA(ctx, cudaEventElapsedTime(walk_ms, ctx->ev_walk0, ctx->ev_walk1));
    return NF_OK;
}

int nf_tree_stats(nf_ctx *ctx, int64_t *node_interactions, int64_t *leaf_interactions, void *stream)
{
    if (!ctx) return NF_ERR_ARG;
    NF_ARG(ctx, node_interactions && leaf_interactions, "nf_tree_stats: null output");
    NF_CUDA(ctx, cudaSetDevice(ctx->device));
    cudaStream_t st = (cudaStream_t)stream;
    NF_CUDA(ctx, cudaMemcpyAsync(ctx->h_counters + 8, ctx->counters + 8, 2 * sizeof(unsigned long long), cudaMemcpyDeviceToHost, st));
    NF_CUDA(ctx, cudaStreamSynchronize(st));
    *node_interactions = (int64_t)ctx->h_counters[8];
    *leaf_interactions = (int64_t)ctx->h_counters[9];
    return NF_OK;
}

int nf_forces(nf_ctx *ctx, const float *pos_sorted, const uint64_t *cell_offset,
              const uint32_t *cell_count, const uint32_t *perm, int64_t N, int K, int R,
              float eps, float box, float Gm, int softening, float *acc_xyz, void *stream)
{
    return nf_forces_ex(ctx, pos_sorted, cell_offset, cell_count, perm, N, K, R, eps, box, Gm, softening, acc_xyz, nullptr, stream);
}

int nf_forces_ex(nf_ctx *ctx, const float *pos_sorted, const uint64_t *cell_offset,
                 const uint32_t *cell_count, const uint32_t *perm, int64_t N, int K, int R,
                 float eps, float box, float Gm, int softening, float *acc_xyz, float *cell_amax, void *stream)
{
    if (!ctx) return NF_ERR_ARG;
    (void)cell_count;     // accepted for symmetry with nf_bin's outputs; everything is derived from cell_offset
    return forces_common(ctx, pos_sorted, cell_offset, perm, N, K, R, eps, box, Gm, softening, 0, K, acc_xyz, cell_amax, stream);
}

int nf_forces_chunk(nf_ctx *ctx, const float *pos_sorted, const uint64_t *cell_offset, const uint32_t *perm, int64_t N, int K,
                    int R, float eps, float box, float Gm, int softening, int x_lo, int x_hi, float *acc_xyz, float *cell_amax,
                    void *stream)
{
    if (!ctx) return NF_ERR_ARG;
    return forces_common(ctx, pos_sorted, cell_offset, perm, N, K, R, eps, box, Gm, softening, x_lo, x_hi, acc_xyz, cell_amax, stream);
}

int nf_keys(nf_ctx *ctx, const float *pos_xyz, int64_t N, int K, float box, uint32_t *keys, void *stream)
{
    if (!ctx) return NF_ERR_ARG;
    NF_TRY(check_common(ctx, N, K, box));
    NF_ARG(ctx, N == 0 || (pos_xyz && keys), "nf_keys: null array with N > 0");
    NF_CUDA(ctx, cudaSetDevice(ctx->device));
    NF_CUDA(ctx, cudaMemsetAsync(ctx->counters, 0, sizeof(unsigned long long), (cudaStream_t)stream));
    return nf_keys_impl(ctx, pos_xyz, N, K, box, keys, (cudaStream_t)stream);
}

static size_t host_path_bytes(int64_t N, int K)
{
    const size_t n = (size_t)(N > 0 ? N : 1), ncell = (size_t)K * K * K;
    size_t b = nf_align_up(n * 12, 256) * 2 + nf_align_up(n * 16, 256) + 2 * nf_align_up(n * 4, 256) +
               nf_align_up(ncell * 4, 256) + nf_align_up((ncell + 1) * 8, 256);
    return b + nf_bin_scratch_bytes(N, K, false) + forces_scratch_full(N, K) + dense_full_bytes(N, K, NF_DENSE_ORDER) + 4096;
}

int nf_reserve_host(nf_ctx *ctx, int64_t maxN, int K)
{
    if (!ctx) return NF_ERR_ARG;
    NF_TRY(check_common(ctx, maxN, K, 1.0f));
    NF_CUDA(ctx, cudaSetDevice(ctx->device));
    return nf_scratch_reserve(ctx, host_path_bytes(maxN, K));
}

int nf_forces_host(nf_ctx *ctx, const float *pos_host, int64_t N, int K, int R, float eps,
                   float box, float Gm, int softening, float *acc_host, void *stream)
{
    if (!ctx) return NF_ERR_ARG;
    NF_ARG(ctx, (softening & NF_MASS_W) == 0, "nf_forces_host takes no masses (NF_MASS_W): use nf_forces_host_m");
    return nf_forces_host_m(ctx, pos_host, nullptr, N, K, R, eps, box, Gm, softening, acc_host, stream);
}

int nf_forces_host_m(nf_ctx *ctx, const float *pos_host, const float *mass_host, int64_t N, int K, int R, float eps,
                     float box, float Gm, int softening, float *acc_host, void *stream)
{
    if (!ctx) return NF_ERR_ARG;
    NF_TRY(check_common(ctx, N, K, box));
    NF_TRY(check_force_args(ctx, K, R, eps, Gm, softening));
    NF_ARG(ctx, N == 0 || (pos_host && acc_host), "nf_forces_host: null particle array with N > 0");
    NF_ARG(ctx, ((softening & NF_MASS_W) != 0) == (mass_host != nullptr) || N == 0, "nf_forces_host_m: NF_MASS_W must be set exactly when mass_host is given");
    NF_CUDA(ctx, cudaSetDevice(ctx->device));
    if (N == 0) return NF_OK;
    NF_TRY(nf_scratch_reserve(ctx, host_path_bytes(N, K)));
    nf_scratch_reset(ctx);
    const size_t n = (size_t)N, ncell = (size_t)K * K * K;
    float *raw = nf_scratch_take<float>(ctx, n * 3);
    float *acc = nf_scratch_take<float>(ctx, n * 3);
    float *sorted = nf_scratch_take<float>(ctx, n * 4);
    uint32_t *perm = nf_scratch_take<uint32_t>(ctx, n);
    float *mass = mass_host ? nf_scratch_take<float>(ctx, n) : nullptr;
    uint32_t *count = nf_scratch_take<uint32_t>(ctx, ncell);
    uint64_t *off = nf_scratch_take<uint64_t>(ctx, ncell + 1);
    nf_plane_view *d_planes = nf_scratch_take<nf_plane_view>(ctx, (size_t)K);
    float4 *enc = nf_scratch_take<float4>(ctx, n);
    float4 *enc_h = nf_scratch_take<float4>(ctx, n);
    if (!raw || !acc || !sorted || !perm || !count || !off || !d_planes || !enc || !enc_h || (mass_host && !mass)) {
        NF_SET_ERR(ctx, "nf_forces_host: internal scratch arena too small");
        return NF_ERR_NOMEM;
    }
    cudaStream_t st = (cudaStream_t)stream;
    NF_CUDA(ctx, cudaMemsetAsync(ctx->counters, 0, sizeof(unsigned long long), st));
    NF_CUDA(ctx, cudaMemcpyAsync(raw, pos_host, n * 12, cudaMemcpyHostToDevice, st));
    if (mass) NF_CUDA(ctx, cudaMemcpyAsync(mass, mass_host, n * 4, cudaMemcpyHostToDevice, st));
    NF_TRY(nf_bin_impl(ctx, raw, mass, N, K, box, -1, sorted, perm, count, off, st));
    nf_force_params p{};
    p.K = K; p.n_planes = K; p.periodic_x = 1; p.sink_lo = 0; p.sink_hi = K;
    p.R = R; p.eps = eps; p.box = box; p.Gm = Gm; p.softening = softening; p.max_sinks = N;
    NF_TRY(encode_full(ctx, p, reinterpret_cast<const float4 *>(sorted), off, perm, N, enc, enc_h, d_planes, acc, nullptr, st));
    NF_TRY(nf_forces_impl(ctx, p, d_planes, st, true));
    NF_CUDA(ctx, cudaMemcpyAsync(acc_host, acc, n * 12, cudaMemcpyDeviceToHost, st));
    NF_CUDA(ctx, cudaMemcpyAsync(ctx->h_counters, ctx->counters, sizeof(unsigned long long), cudaMemcpyDeviceToHost, st));
    NF_CUDA(ctx, cudaStreamSynchronize(st));
    if (ctx->h_counters[0]) {
        NF_SET_ERR(ctx, "%lld particle(s) outside [0, box) were clamped into edge cells", (long long)ctx->h_counters[0]);
        return NF_ERR_RANGE;
    }
    return NF_OK;
}

// ---- pipelined host path: two steps in flight -----------------------------------------------------
// Step s+1's H2D copy runs on the context's copy stream while step s computes, and step s's D2H copy runs
// while step s+1 computes (PAPER.md:69: the GPU work is overlapped with the transfers; :111 the paper's
// rate "includes PCIe bus transfer overheads").  Input and output buffers are doubled; everything else in
// the scratch arena is shared, because the compute parts of consecutive steps are ordered on one stream.
int nf_forces_host_begin(nf_ctx *ctx, const float *pos_host, int64_t N, int K, int R, float eps, float box, float Gm,
                         int softening, float *acc_host, void *stream)
{
    if (!ctx) return NF_ERR_ARG;
    NF_TRY(check_common(ctx, N, K, box));
    NF_TRY(check_force_args(ctx, K, R, eps, Gm, softening));
    NF_ARG(ctx, N > 0 && pos_host && acc_host, "nf_forces_host_begin: needs N > 0 and non-null host arrays");
    NF_ARG(ctx, (softening & NF_MASS_W) == 0, "nf_forces_host_begin takes no masses");
    NF_CUDA(ctx, cudaSetDevice(ctx->device));
    HostPipe *hp = static_cast<HostPipe *>(ctx->host_pipe);
    if (!hp) {
        hp = new (std::nothrow) HostPipe();
        if (!hp) { NF_SET_ERR(ctx, "host allocation failed"); return NF_ERR_NOMEM; }
        memset(hp, 0, sizeof(*hp));
        ctx->host_pipe = hp;
        for (int i = 0; i < 2; i++) {
            NF_CUDA(ctx, cudaEventCreateWithFlags(&hp->ev_h2d[i], cudaEventDisableTiming));
            NF_CUDA(ctx, cudaEventCreateWithFlags(&hp->ev_raw_free[i], cudaEventDisableTiming));
            NF_CUDA(ctx, cudaEventCreateWithFlags(&hp->ev_done[i], cudaEventDisableTiming));
            NF_CUDA(ctx, cudaEventCreateWithFlags(&hp->ev_d2h[i], cudaEventDisableTiming));
        }
        NF_CUDA(ctx, cudaMallocHost((void **)&hp->h_bad, 2 * sizeof(unsigned long long)));
    }
    NF_ARG(ctx, hp->active < 2, "nf_forces_host_begin: two steps are already in flight (call nf_forces_host_end)");
    const size_t n = (size_t)N, ncell = (size_t)K * K * K;
    if (hp->active == 0) {
        // doubled input / output + sorted, perm, cells, the two encoded copies + the larger of the binning scratch
        // and the work list (the work list overlays the binning scratch: same stream, binning is done by then)
        nf_force_params fp{};
        fp.K = K; fp.n_planes = K; fp.sink_lo = 0; fp.sink_hi = K; fp.max_sinks = N;
        const size_t wl = nf_forces_scratch_bytes(fp), bs = nf_bin_scratch_bytes(N, K, false);
        const size_t need = 4 * nf_align_up(n * 12, 256) + 3 * nf_align_up(n * 16, 256) + nf_align_up(n * 4, 256) +
                            nf_align_up(ncell * 4, 256) + nf_align_up((ncell + 1) * 8, 256) + (wl > bs ? wl : bs) +
                            dense_full_bytes(N, K, NF_DENSE_ORDER) + 8192;
        NF_TRY(nf_scratch_reserve(ctx, need));
        nf_scratch_reset(ctx);
        for (int i = 0; i < 2; i++) {
            hp->raw[i] = nf_scratch_take<float>(ctx, n * 3);
            hp->acc[i] = nf_scratch_take<float>(ctx, n * 3);
            hp->used[i] = false;
        }
        hp->shared_at = ctx->scratch_used;
        hp->N = N; hp->K = K; hp->next = 0;
        if (!hp->raw[1] || !hp->acc[1]) { NF_SET_ERR(ctx, "nf_forces_host_begin: internal scratch arena too small"); return NF_ERR_NOMEM; }
    } else {
        NF_ARG(ctx, hp->N == N && hp->K == K, "nf_forces_host_begin: N and K must not change while a step is in flight");
    }
    const int i = hp->next;
    cudaStream_t st = (cudaStream_t)stream;
    // the shared part of the arena, carved the same way every step
    ctx->scratch_used = hp->shared_at;
    float *sorted = nf_scratch_take<float>(ctx, n * 4);
    uint32_t *perm = nf_scratch_take<uint32_t>(ctx, n);
    uint32_t *count = nf_scratch_take<uint32_t>(ctx, ncell);
    uint64_t *off = nf_scratch_take<uint64_t>(ctx, ncell + 1);
    nf_plane_view *d_planes = nf_scratch_take<nf_plane_view>(ctx, (size_t)K);
    float4 *enc = nf_scratch_take<float4>(ctx, n);
    float4 *enc_h = nf_scratch_take<float4>(ctx, n);
    if (!sorted || !perm || !count || !off || !d_planes || !enc || !enc_h) {
        NF_SET_ERR(ctx, "nf_forces_host_begin: internal scratch arena too small");
        return NF_ERR_NOMEM;
    }
    // H2D on the copy stream, as soon as the binning that last read this input buffer is done
    if (hp->used[i]) NF_CUDA(ctx, cudaStreamWaitEvent(ctx->s_h2d, hp->ev_raw_free[i], 0));
    else {                                         // first use: order after prior work on the caller's stream
        NF_CUDA(ctx, cudaEventRecord(hp->ev_raw_free[i], st));
        NF_CUDA(ctx, cudaStreamWaitEvent(ctx->s_h2d, hp->ev_raw_free[i], 0));
    }
    NF_CUDA(ctx, cudaMemcpyAsync(hp->raw[i], pos_host, n * 12, cudaMemcpyHostToDevice, ctx->s_h2d));
    NF_CUDA(ctx, cudaEventRecord(hp->ev_h2d[i], ctx->s_h2d));
    // compute on the caller's stream
    NF_CUDA(ctx, cudaStreamWaitEvent(st, hp->ev_h2d[i], 0));
    if (hp->used[i]) NF_CUDA(ctx, cudaStreamWaitEvent(st, hp->ev_d2h[i], 0));     // acc[i] has been copied out
    NF_CUDA(ctx, cudaMemsetAsync(ctx->counters, 0, sizeof(unsigned long long), st));
    const size_t mark = ctx->scratch_used;
    NF_TRY(nf_bin_impl(ctx, hp->raw[i], nullptr, N, K, box, -1, sorted, perm, count, off, st));
    NF_CUDA(ctx, cudaEventRecord(hp->ev_raw_free[i], st));
    ctx->scratch_used = mark;                       // the work list may overlay the binning scratch
    nf_force_params p{};
    p.K = K; p.n_planes = K; p.periodic_x = 1; p.sink_lo = 0; p.sink_hi = K;
    p.R = R; p.eps = eps; p.box = box; p.Gm = Gm; p.softening = softening; p.max_sinks = N;
    NF_TRY(encode_full(ctx, p, reinterpret_cast<const float4 *>(sorted), off, perm, N, enc, enc_h, d_planes, hp->acc[i], nullptr, st));
    NF_TRY(nf_forces_impl(ctx, p, d_planes, st, true));
    NF_CUDA(ctx, cudaMemcpyAsync(hp->h_bad + i, ctx->counters, sizeof(unsigned long long), cudaMemcpyDeviceToHost, st));
    NF_CUDA(ctx, cudaEventRecord(hp->ev_done[i], st));
    // D2H on the other copy stream
    NF_CUDA(ctx, cudaStreamWaitEvent(ctx->s_d2h, hp->ev_done[i], 0));
    NF_CUDA(ctx, cudaMemcpyAsync(acc_host, hp->acc[i], n * 12, cudaMemcpyDeviceToHost, ctx->s_d2h));
    NF_CUDA(ctx, cudaEventRecord(hp->ev_d2h[i], ctx->s_d2h));
    hp->used[i] = true;
    hp->next = i ^ 1;
    hp->active++;
    return NF_OK;
}

int nf_forces_host_end(nf_ctx *ctx)
{
    if (!ctx) return NF_ERR_ARG;
    HostPipe *hp = static_cast<HostPipe *>(ctx->host_pipe);
    NF_ARG(ctx, hp && hp->active > 0, "nf_forces_host_end: no step in flight");
    NF_CUDA(ctx, cudaSetDevice(ctx->device));
    const int j = hp->active == 2 ? hp->next : (hp->next ^ 1);      // the oldest step in flight
    NF_CUDA(ctx, cudaEventSynchronize(hp->ev_d2h[j]));
    hp->active--;
    if (hp->h_bad[j]) {
        NF_SET_ERR(ctx, "%lld particle(s) outside [0, box) were clamped into edge cells", (long long)hp->h_bad[j]);
        return NF_ERR_RANGE;
    }
    return NF_OK;
}

int nf_interactions(nf_ctx *ctx, const uint32_t *cell_count, int K, int R, int64_t *interactions, void *stream)
{
    if (!ctx) return NF_ERR_ARG;
    NF_ARG(ctx, cell_count && interactions, "nf_interactions: null argument");
    NF_ARG(ctx, K >= 1 && K <= NF_MAX_K && R >= 0 && R <= NF_MAX_R && K >= 2 * R + 1, "nf_interactions: bad K / R");
    NF_CUDA(ctx, cudaSetDevice(ctx->device));
    return nf_interactions_impl(ctx, cell_count, K, R, interactions, (cudaStream_t)stream);
}

float nf_spline_equivalent_eps(float eps_plummer) { return 2.16f * eps_plummer; }

int nf_last_forces_timing(nf_ctx *ctx, float *kernel_ms, float *total_ms)
{
    if (!ctx) return NF_ERR_ARG;
    NF_ARG(ctx, ctx->forces_timed, "nf_last_forces_timing: no nf_forces call has been timed yet");
    NF_CUDA(ctx, cudaSetDevice(ctx->device));
    NF_CUDA(ctx, cudaEventSynchronize(ctx->ev_total1));
    if (kernel_ms) NF_CUDA(ctx, cudaEventElapsedTime(kernel_ms, ctx->ev_kern0, ctx->ev_kern1));
    if (total_ms) NF_CUDA(ctx, cudaEventElapsedTime(total_ms, ctx->ev_total0, ctx->ev_total1));
    return NF_OK;
}

int nf_launch_count(const nf_ctx *ctx, int64_t *launches)
{
    if (!ctx || !launches) return NF_ERR_ARG;
    *launches = (int64_t)ctx->launches;
    return NF_OK;
}

}  // extern "C"
