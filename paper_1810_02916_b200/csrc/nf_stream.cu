// nf_stream.cu -- nf_stream_slabs: the slab pipeline of PAPER.md:41 ("load a rolling window of
// slabs into memory, compute forces ... on the central slab, write out the trailing slab, and
// then load a slab at the leading edge") with the slabs held in pinned host memory
// instead of on disk.
//
// Three streams: H2D copies (ctx->s_h2d), kernels (the caller's stream), D2H copies
// (ctx->s_d2h), ordered by events.  A ring of W = 2R+1+LOOKAHEAD device slots holds the
// resident planes; each slot owns raw positions, cell-sorted offsets, perm, per-plane cell
// counts / offsets and the accelerations of the plane.
#include <new>
#include <vector>

#include "nf_common.cuh"

namespace {

constexpr int LOOKAHEAD = 2;  // "we allow Abacus to read ahead by a few slabs"

struct Slot {
    float *raw;        // n x 3
    float *sorted;     // n x 4
    float *enc;        // n x 4: scaled, z-block-encoded copy read by the interaction kernel
    float *enc_h;      // n x 4: the same with the z-blocks shifted by half a block
    uint32_t *perm;    // n
    uint32_t *count;   // K*K
    uint64_t *off;     // K*K + 1
    float *acc;        // n x 3
    float *vel;        // n x 3 (nf_stream_step_slabs only)
    float *part_pos;   // n x 3, n x 3 (nf_stream_step_regroup only): the drifted plane as [to plane-1 | stay | to plane+1]
    float *part_vel;
    // in-cell ordering of the plane's dense cells (nf_dense.cu), null when the pass does not take it
    uint32_t *dinfo;   // K*K
    uint32_t *dslot;   // nf_dense_cap(n)
    float *dbox;       // nf_dense_cap(n) / 64 * 6
};

// the kick + drift epilogue of nf_stream_step_slabs (null pointers: plain nf_stream_slabs)
struct StepArgs {
    const float *const *vel_host;     // P x nseg
    float *const *pos_out_host;       // P
    float *const *vel_out_host;       // P
    float kick, drift;
    int64_t *out_seg_n;               // non-null: regroup after the drift (nf_stream_step_regroup), P x 3 counts (host out)
};

// the planes of a pass: plane q is the concatenation of nseg host segments pos[q*nseg + k] of n[q*nseg + k] particles
struct PlaneIn {
    const float *const *pos;
    const int64_t *n;
    int nseg;
};

struct SlabState {
    char *mem = nullptr;
    size_t mem_bytes = 0;
    unsigned long long *d_segn = nullptr, *h_segn = nullptr;   // [P][3] segment lengths of the regrouped planes
    int segn_cap = 0;
    nf_plane_view *h_views = nullptr;  // pinned, [P+2R]
    nf_plane_view *d_views = nullptr;
    int views_cap = 0;
};

void free_state(SlabState *s)
{
    if (!s) return;
    if (s->mem) cudaFree(s->mem);
    if (s->h_views) cudaFreeHost(s->h_views);
    if (s->d_views) cudaFree(s->d_views);
    if (s->d_segn) cudaFree(s->d_segn);
    if (s->h_segn) cudaFreeHost(s->h_segn);
    delete s;
}

struct EventPool {
    std::vector<cudaEvent_t> ev;
    ~EventPool() { for (auto e : ev) cudaEventDestroy(e); }
    cudaEvent_t get(bool timing)
    {
        cudaEvent_t e = nullptr;
        if (cudaEventCreateWithFlags(&e, timing ? cudaEventDefault : cudaEventDisableTiming) != cudaSuccess) return nullptr;
        ev.push_back(e);
        return e;
    }
};

}  // namespace

void nf_slab_state_free(nf_ctx *ctx)
{
    free_state(static_cast<SlabState *>(ctx->slab_state));
    ctx->slab_state = nullptr;
}

static bool is_pinned(const void *p)
{
    cudaPointerAttributes at;
    cudaError_t e = cudaPointerGetAttributes(&at, p);
    if (e != cudaSuccess) { cudaGetLastError(); return false; }
    return at.type == cudaMemoryTypeHost;      // page-locked host memory; managed memory migrates and is refused
}

static int stream_run(nf_ctx *ctx, EventPool &pool, const PlaneIn &in,
                      int P, int K, int R, float eps, float box, int plane0, float Gm,
                      int softening, float *const *plane_acc_host, const StepArgs *step, nf_stream_stats *stats,
                      void *stream)
{
    if (!ctx) return NF_ERR_ARG;
    NF_ARG(ctx, in.pos && in.n && (plane_acc_host || step), "nf_stream_slabs: null pointer table");
    NF_ARG(ctx, P >= 1, "nf_stream_slabs: P must be >= 1");
    NF_ARG(ctx, K >= 1 && K <= NF_MAX_K, "K = %d out of range [1, %d]", K, NF_MAX_K);
    NF_ARG(ctx, R >= 0 && R <= NF_MAX_R, "R = %d out of range [0, %d]", R, NF_MAX_R);
    NF_ARG(ctx, K >= 2 * R + 1, "K = %d < 2R+1", K);
    NF_ARG(ctx, P <= K, "P = %d sink planes exceed K = %d", P, K);
    NF_ARG(ctx, eps > 0.0f && eps < 3.0e38f, "eps must be positive and finite");
    NF_ARG(ctx, box > 0.0f && box < 3.0e38f, "box must be positive and finite");
    NF_ARG(ctx, (softening & ~NF_DENSE_ORDER) == NF_SOFT_SPLINE || (softening & ~NF_DENSE_ORDER) == NF_SOFT_PLUMMER,
           "unknown softening %d (the slab stream carries no masses)", softening);
    const int NP = P + 2 * R, NS = in.nseg;
    const bool regroup = step && step->out_seg_n;
    NF_ARG(ctx, NS >= 1 && NS <= 3, "a plane has 1 to 3 host segments");
    std::vector<int64_t> plane_n_v(NP, 0);
    int64_t max_n = 1;
    NF_CUDA(ctx, cudaSetDevice(ctx->device));
    for (int q = 0; q < NP; q++) {
        for (int k = 0; k < NS; k++) {
            const int64_t nk = in.n[q * NS + k];
            NF_ARG(ctx, nk >= 0 && nk < ((int64_t)1 << 32), "plane %d, segment %d: particle count out of range", q, k);
            // host pointers must be pinned (page-locked): "Pinning memory"
            NF_ARG(ctx, nk == 0 || (in.pos[q * NS + k] && is_pinned(in.pos[q * NS + k])),
                   "plane_pos_host[%d] (segment %d) is null or not pinned host memory", q, k);
            plane_n_v[q] += nk;
        }
        NF_ARG(ctx, plane_n_v[q] < ((int64_t)1 << 32), "plane_n[%d] out of range", q);
        if (plane_n_v[q] > max_n) max_n = plane_n_v[q];
    }
    const int64_t *plane_n = plane_n_v.data();
    for (int p = 0; p < P; p++) {
        if (plane_n[R + p] == 0) continue;
        NF_ARG(ctx, !plane_acc_host || (plane_acc_host[p] && is_pinned(plane_acc_host[p])), "plane_acc_host[%d] is null or not pinned host memory", p);
        if (step) {
            for (int k = 0; k < NS; k++)
                NF_ARG(ctx, in.n[(R + p) * NS + k] == 0 || (step->vel_host[p * NS + k] && is_pinned(step->vel_host[p * NS + k])),
                       "plane_vel_host[%d] (segment %d) is null or not pinned host memory", p, k);
            NF_ARG(ctx, step->pos_out_host[p] && is_pinned(step->pos_out_host[p]), "plane_pos_out_host[%d] is null or not pinned host memory", p);
            NF_ARG(ctx, step->vel_out_host[p] && is_pinned(step->vel_out_host[p]), "plane_vel_out_host[%d] is null or not pinned host memory", p);
        }
    }

    cudaStream_t st = (cudaStream_t)stream;
    const int W = 2 * R + 1 + LOOKAHEAD;
    const size_t ncell = (size_t)K * K;

    // ---- device memory: ring slots + shared scratch for binning ----
    SlabState *S = static_cast<SlabState *>(ctx->slab_state);
    if (!S) {
        S = new (std::nothrow) SlabState();
        if (!S) { NF_SET_ERR(ctx, "host allocation failed"); return NF_ERR_NOMEM; }
        ctx->slab_state = S;
    }
    const size_t n = (size_t)max_n;
    // in-cell ordering of dense cells, plane by plane: asked for, or the fullest plane's mean occupancy says so
    const bool dense = nf_dense_wanted(max_n, ncell, softening);
    softening &= ~NF_DENSE_ORDER;
    const size_t dcap = dense ? nf_dense_cap(max_n) : 0;
    const size_t dense_bytes = dense ? nf_align_up(ncell * 4, 256) + nf_align_up(dcap * 4, 256) + nf_align_up(dcap / 64 * 24, 256) : 0;
    const size_t slot_bytes = dense_bytes + nf_align_up(n * 12, 256) + 3 * nf_align_up(n * 16, 256) + nf_align_up(n * 4, 256) +
                              nf_align_up(ncell * 4, 256) + nf_align_up((ncell + 1) * 8, 256) + nf_align_up(n * 12, 256) +
                              (step ? nf_align_up(n * 12, 256) : 0) + (regroup ? 2 * nf_align_up(n * 12, 256) : 0);
    const size_t need = slot_bytes * W;
    if (need > S->mem_bytes) {
        NF_CUDA(ctx, cudaDeviceSynchronize());
        if (S->mem) NF_CUDA(ctx, cudaFree(S->mem));
        S->mem = nullptr; S->mem_bytes = 0;
        cudaError_t e = cudaMalloc((void **)&S->mem, need);
        if (e != cudaSuccess) { cudaGetLastError(); NF_SET_ERR(ctx, "cudaMalloc of %zu bytes for the slab ring failed", need); return NF_ERR_NOMEM; }
        S->mem_bytes = need;
    }
    if (NP > S->views_cap) {
        NF_CUDA(ctx, cudaDeviceSynchronize());
        if (S->h_views) NF_CUDA(ctx, cudaFreeHost(S->h_views));
        if (S->d_views) NF_CUDA(ctx, cudaFree(S->d_views));
        S->h_views = nullptr; S->d_views = nullptr; S->views_cap = 0;
        NF_CUDA(ctx, cudaMallocHost((void **)&S->h_views, sizeof(nf_plane_view) * NP));
        NF_CUDA(ctx, cudaMalloc((void **)&S->d_views, sizeof(nf_plane_view) * NP));
        S->views_cap = NP;
    }
    nf_force_params fp{};
    fp.K = K; fp.n_planes = NP; fp.periodic_x = 0; fp.R = R; fp.eps = eps; fp.box = box; fp.Gm = Gm; fp.softening = softening;
    fp.sink_lo = 0; fp.sink_hi = 1; fp.max_sinks = max_n;     // one sink plane per nf_forces_impl call
    fp.dense = dense ? 1 : 0;
    if (regroup && P > S->segn_cap) {
        NF_CUDA(ctx, cudaDeviceSynchronize());
        if (S->d_segn) NF_CUDA(ctx, cudaFree(S->d_segn));
        if (S->h_segn) NF_CUDA(ctx, cudaFreeHost(S->h_segn));
        S->d_segn = nullptr; S->h_segn = nullptr; S->segn_cap = 0;
        NF_CUDA(ctx, cudaMalloc((void **)&S->d_segn, sizeof(unsigned long long) * 3 * P));
        NF_CUDA(ctx, cudaMallocHost((void **)&S->h_segn, sizeof(unsigned long long) * 3 * P));
        S->segn_cap = P;
    }
    // binning, the force work list and the regrouping of a plane take their scratch one after the other
    NF_TRY(nf_scratch_reserve(ctx, nf_bin_scratch_bytes(max_n, K, true) + nf_forces_scratch_bytes(fp) +
                                       (regroup ? nf_regroup_scratch_bytes(max_n) : 0) + (dense ? nf_dense_scratch_bytes(max_n, ncell) : 0)));

    std::vector<Slot> slots(W);
    for (int s = 0; s < W; s++) {
        char *b = S->mem + slot_bytes * s;
        slots[s].raw = (float *)b;                b += nf_align_up(n * 12, 256);
        slots[s].sorted = (float *)b;             b += nf_align_up(n * 16, 256);
        slots[s].enc = (float *)b;                b += nf_align_up(n * 16, 256);
        slots[s].enc_h = (float *)b;              b += nf_align_up(n * 16, 256);
        slots[s].perm = (uint32_t *)b;            b += nf_align_up(n * 4, 256);
        slots[s].count = (uint32_t *)b;           b += nf_align_up(ncell * 4, 256);
        slots[s].off = (uint64_t *)b;             b += nf_align_up((ncell + 1) * 8, 256);
        slots[s].acc = (float *)b;                b += nf_align_up(n * 12, 256);
        slots[s].vel = step ? (float *)b : nullptr;
        if (step) b += nf_align_up(n * 12, 256);
        slots[s].part_pos = regroup ? (float *)b : nullptr;
        if (regroup) b += nf_align_up(n * 12, 256);
        slots[s].part_vel = regroup ? (float *)b : nullptr;
        if (regroup) b += nf_align_up(n * 12, 256);
        slots[s].dinfo = dense ? (uint32_t *)b : nullptr;
        if (dense) b += nf_align_up(ncell * 4, 256);
        slots[s].dslot = dense ? (uint32_t *)b : nullptr;
        if (dense) b += nf_align_up(dcap * 4, 256);
        slots[s].dbox = dense ? (float *)b : nullptr;
    }
    // plane views (device pointers are fixed by the slot assignment q % W)
    for (int q = 0; q < NP; q++) {
        const Slot &sl = slots[q % W];
        S->h_views[q].pos = (const float4 *)sl.sorted;
        S->h_views[q].enc = (const float4 *)sl.enc;
        S->h_views[q].enc_h = (const float4 *)sl.enc_h;
        S->h_views[q].off = sl.off;
        S->h_views[q].perm = sl.perm;
        S->h_views[q].acc = sl.acc;
        S->h_views[q].amax = nullptr;
        S->h_views[q].dinfo = sl.dinfo;
        S->h_views[q].dslot = sl.dslot;
        S->h_views[q].dbox = sl.dbox;
    }
    NF_CUDA(ctx, cudaMemcpyAsync(S->d_views, S->h_views, sizeof(nf_plane_view) * NP, cudaMemcpyHostToDevice, st));
    NF_CUDA(ctx, cudaMemsetAsync(ctx->counters, 0, 2 * sizeof(unsigned long long), st));

    std::vector<cudaEvent_t> h2d0(NP), h2d1(NP), bin0(NP), bin1(NP), frc0(P), frc1(P), d2h0(P), d2h1(P);
    for (int q = 0; q < NP; q++) { h2d0[q] = pool.get(true); h2d1[q] = pool.get(true); bin0[q] = pool.get(true); bin1[q] = pool.get(true); }
    for (int p = 0; p < P; p++) { frc0[p] = pool.get(true); frc1[p] = pool.get(true); d2h0[p] = pool.get(true); d2h1[p] = pool.get(true); }
    cudaEvent_t ev_begin = pool.get(true), ev_end = pool.get(true), ev_ready = pool.get(false);
    for (auto e : pool.ev) if (!e) { NF_SET_ERR(ctx, "cudaEventCreate failed"); return NF_ERR_CUDA; }

    double vel_bytes = 0.0;
    NF_CUDA(ctx, cudaEventRecord(ev_ready, st));        // order the whole call after prior work on `stream`
    NF_CUDA(ctx, cudaStreamWaitEvent(ctx->s_h2d, ev_ready, 0));
    NF_CUDA(ctx, cudaStreamWaitEvent(ctx->s_d2h, ev_ready, 0));
    NF_CUDA(ctx, cudaEventRecord(ev_begin, ctx->s_h2d));

    for (int q = 0; q < NP; q++) {
        const Slot &sl = slots[q % W];
        // slot reuse: plane q-W lived here.  It was last read as a source by sink plane
        // (q-W)+R, and (if it was a sink) its accelerations were copied out by d2h1.
        const int prev = q - W;
        if (prev >= 0) {
            int last_sink = prev;  // chunk plane prev+R is the last sink that reads plane prev; its sink number is prev
            if (last_sink >= 0 && last_sink < P) NF_CUDA(ctx, cudaStreamWaitEvent(ctx->s_h2d, frc1[last_sink], 0));
            int own_sink = prev - R;
            if (own_sink >= 0 && own_sink < P) NF_CUDA(ctx, cudaStreamWaitEvent(ctx->s_h2d, d2h1[own_sink], 0));
        }
        NF_CUDA(ctx, cudaEventRecord(h2d0[q], ctx->s_h2d));
        size_t at = 0;
        for (int k = 0; k < NS; k++) {
            const size_t nk = (size_t)in.n[q * NS + k];
            if (nk == 0) continue;
            NF_CUDA(ctx, cudaMemcpyAsync(sl.raw + 3 * at, in.pos[q * NS + k], nk * 12, cudaMemcpyHostToDevice, ctx->s_h2d));
            if (step && q >= R && q < R + P) {
                NF_CUDA(ctx, cudaMemcpyAsync(sl.vel + 3 * at, step->vel_host[(q - R) * NS + k], nk * 12, cudaMemcpyHostToDevice, ctx->s_h2d));
                vel_bytes += (double)nk * 12.0;
            }
            at += nk;
        }
        NF_CUDA(ctx, cudaEventRecord(h2d1[q], ctx->s_h2d));

        NF_CUDA(ctx, cudaStreamWaitEvent(st, h2d1[q], 0));
        NF_CUDA(ctx, cudaEventRecord(bin0[q], st));
        nf_scratch_reset(ctx);
        const int cx = ((plane0 + q) % K + K) % K;
        // counters[0] accumulates out-of-range / wrong-plane particles over all planes
        NF_TRY(nf_bin_impl(ctx, sl.raw, nullptr, plane_n[q], K, box, cx, sl.sorted, sl.perm, sl.count, sl.off, st));
        NF_TRY(nf_encode_impl(ctx, fp, (const float4 *)sl.sorted, sl.off, ncell, (float4 *)sl.enc, (float4 *)sl.enc_h, st, dense ? NF_DENSE_N : 0));
        if (dense)
            NF_TRY(nf_dense_order_impl(ctx, fp, (const float4 *)sl.sorted, sl.off, ncell, plane_n[q], (float4 *)sl.enc, (float4 *)sl.enc_h,
                                       sl.dinfo, sl.dslot, sl.dbox, st));
        NF_CUDA(ctx, cudaEventRecord(bin1[q], st));

        const int sp = q - R;        // chunk plane whose neighbourhood is now complete
        const int p = sp - R;        // its sink number
        if (p >= 0 && p < P) {
            fp.sink_lo = sp; fp.sink_hi = sp + 1;
            NF_CUDA(ctx, cudaEventRecord(frc0[p], st));
            NF_TRY(nf_forces_impl(ctx, fp, S->d_views, st, false));
            NF_TRY(nf_interactions_planes(ctx, fp, S->d_views, st));
            const Slot &ss = slots[sp % W];
            // kick + drift of the sink plane in place: its raw positions were only the input of its own
            // binning (the later sink planes read the sorted / encoded copies), so they can move now
            if (step && plane_n[sp] > 0)
                NF_TRY(nf_kick_drift_impl(ctx, ss.raw, ss.vel, ss.acc, plane_n[sp], step->kick, step->drift, box, st));
            // ... and be filed by the plane they now belong to (three stable segments + their lengths)
            if (regroup)
                NF_TRY(nf_regroup_impl(ctx, ss.raw, ss.vel, plane_n[sp], K, box, ((plane0 + sp) % K + K) % K, ss.part_pos, ss.part_vel,
                                       S->d_segn + 3 * p, st));
            NF_CUDA(ctx, cudaEventRecord(frc1[p], st));
            NF_CUDA(ctx, cudaStreamWaitEvent(ctx->s_d2h, frc1[p], 0));
            NF_CUDA(ctx, cudaEventRecord(d2h0[p], ctx->s_d2h));
            if (plane_n[sp] > 0) {
                const size_t nb = (size_t)plane_n[sp] * 12;
                if (plane_acc_host) NF_CUDA(ctx, cudaMemcpyAsync(plane_acc_host[p], ss.acc, nb, cudaMemcpyDeviceToHost, ctx->s_d2h));
                if (step) {
                    NF_CUDA(ctx, cudaMemcpyAsync(step->pos_out_host[p], regroup ? ss.part_pos : ss.raw, nb, cudaMemcpyDeviceToHost, ctx->s_d2h));
                    NF_CUDA(ctx, cudaMemcpyAsync(step->vel_out_host[p], regroup ? ss.part_vel : ss.vel, nb, cudaMemcpyDeviceToHost, ctx->s_d2h));
                }
            }
            NF_CUDA(ctx, cudaEventRecord(d2h1[p], ctx->s_d2h));
        }
    }
    NF_CUDA(ctx, cudaStreamWaitEvent(st, d2h1[P - 1], 0));
    NF_CUDA(ctx, cudaEventRecord(ev_end, st));
    NF_CUDA(ctx, cudaMemcpyAsync(ctx->h_counters, ctx->counters, 2 * sizeof(unsigned long long), cudaMemcpyDeviceToHost, st));
    if (regroup) NF_CUDA(ctx, cudaMemcpyAsync(S->h_segn, S->d_segn, sizeof(unsigned long long) * 3 * P, cudaMemcpyDeviceToHost, st));
    NF_CUDA(ctx, cudaStreamSynchronize(st));
    NF_CUDA(ctx, cudaStreamSynchronize(ctx->s_d2h));
    NF_CUDA(ctx, cudaStreamSynchronize(ctx->s_h2d));

    if (regroup)
        for (int i = 0; i < 3 * P; i++) step->out_seg_n[i] = (int64_t)S->h_segn[i];
    if (stats) {
        memset(stats, 0, sizeof(*stats));
        float ms = 0.f;
        for (int q = 0; q < NP; q++) {
            stats->particles_in += plane_n[q];
            NF_CUDA(ctx, cudaEventElapsedTime(&ms, h2d0[q], h2d1[q])); stats->h2d_seconds += ms * 1e-3;
            NF_CUDA(ctx, cudaEventElapsedTime(&ms, bin0[q], bin1[q])); stats->kernel_seconds += ms * 1e-3;
        }
        for (int p = 0; p < P; p++) {
            stats->particles_out += plane_n[R + p];
            NF_CUDA(ctx, cudaEventElapsedTime(&ms, frc0[p], frc1[p])); stats->kernel_seconds += ms * 1e-3; stats->force_seconds += ms * 1e-3;
            NF_CUDA(ctx, cudaEventElapsedTime(&ms, d2h0[p], d2h1[p])); stats->d2h_seconds += ms * 1e-3;
        }
        NF_CUDA(ctx, cudaEventElapsedTime(&ms, ev_begin, ev_end)); stats->wall_seconds = ms * 1e-3;
        stats->h2d_bytes = 12.0 * (double)stats->particles_in + vel_bytes;
        stats->d2h_bytes = 12.0 * (double)stats->particles_out * ((plane_acc_host ? 1.0 : 0.0) + (step ? 2.0 : 0.0));
        stats->h2d_gbps = stats->h2d_seconds > 0 ? stats->h2d_bytes / stats->h2d_seconds * 1e-9 : 0.0;
        stats->d2h_gbps = stats->d2h_seconds > 0 ? stats->d2h_bytes / stats->d2h_seconds * 1e-9 : 0.0;
        stats->interactions = (int64_t)ctx->h_counters[1];
        stats->out_of_range = (int64_t)ctx->h_counters[0];
        const double copy_s = stats->h2d_seconds + stats->d2h_seconds;
        double hidden = copy_s > 0 ? 1.0 - (stats->wall_seconds - stats->kernel_seconds) / copy_s : 0.0;
        stats->overlap_fraction = hidden < 0 ? 0.0 : (hidden > 1 ? 1.0 : hidden);
    }
    if (ctx->h_counters[0]) {
        NF_SET_ERR(ctx, "%lld particle(s) outside [0, box), filed under the wrong plane (clamped into edge cells), or drifted further than one plane",
                   (long long)ctx->h_counters[0]);
        return NF_ERR_RANGE;
    }
    return NF_OK;
}

// Every path out of the pass -- also an error in the middle of it -- first waits for the three
// streams: copies already queued still read and write the caller's pinned buffers, and the events of
// the pool must not be destroyed while work that records or waits on them is pending (include/nf.h:
// "the library never retains a caller buffer past the call").
static int stream_impl(nf_ctx *ctx, const PlaneIn &in,
                       int P, int K, int R, float eps, float box, int plane0, float Gm,
                       int softening, float *const *plane_acc_host, const StepArgs *step, nf_stream_stats *stats,
                       void *stream)
{
    if (!ctx) return NF_ERR_ARG;
    EventPool pool;
    const int rc = stream_run(ctx, pool, in, P, K, R, eps, box, plane0, Gm, softening, plane_acc_host, step, stats, stream);
    if (rc != NF_OK && rc != NF_ERR_ARG) {
        cudaStreamSynchronize((cudaStream_t)stream);
        if (ctx->s_h2d) cudaStreamSynchronize(ctx->s_h2d);
        if (ctx->s_d2h) cudaStreamSynchronize(ctx->s_d2h);
        if (rc != NF_ERR_RANGE) cudaGetLastError();
    }
    return rc;
}

extern "C" int nf_stream_slabs(nf_ctx *ctx, const float *const *plane_pos_host, const int64_t *plane_n,
                               int P, int K, int R, float eps, float box, int plane0, float Gm,
                               int softening, float *const *plane_acc_host, nf_stream_stats *stats,
                               void *stream)
{
    if (!ctx) return NF_ERR_ARG;
    NF_ARG(ctx, plane_acc_host != nullptr, "nf_stream_slabs: null pointer table");
    const PlaneIn in{plane_pos_host, plane_n, 1};
    return stream_impl(ctx, in, P, K, R, eps, box, plane0, Gm, softening, plane_acc_host, nullptr, stats, stream);
}

extern "C" int nf_stream_step_slabs(nf_ctx *ctx, const float *const *plane_pos_host, const float *const *plane_vel_host,
                                    const int64_t *plane_n, int P, int K, int R, float eps, float box, int plane0,
                                    float Gm, int softening, float kick, float drift, float *const *plane_pos_out_host,
                                    float *const *plane_vel_out_host, float *const *plane_acc_host,
                                    nf_stream_stats *stats, void *stream)
{
    if (!ctx) return NF_ERR_ARG;
    NF_ARG(ctx, plane_vel_host && plane_pos_out_host && plane_vel_out_host, "nf_stream_step_slabs: null pointer table");
    NF_ARG(ctx, kick == kick && drift == drift && fabsf(kick) < 3.0e38f && fabsf(drift) < 3.0e38f, "kick and drift must be finite");
    StepArgs a{plane_vel_host, plane_pos_out_host, plane_vel_out_host, kick, drift, nullptr};
    const PlaneIn in{plane_pos_host, plane_n, 1};
    return stream_impl(ctx, in, P, K, R, eps, box, plane0, Gm, softening, plane_acc_host, &a, stats, stream);
}

extern "C" int nf_stream_step_regroup(nf_ctx *ctx, const float *const *seg_pos_host, const float *const *seg_vel_host,
                                      const int64_t *seg_n, int P, int K, int R, float eps, float box, int plane0, float Gm,
                                      int softening, float kick, float drift, float *const *plane_pos_out_host,
                                      float *const *plane_vel_out_host, int64_t *out_seg_n, float *const *plane_acc_host,
                                      nf_stream_stats *stats, void *stream)
{
    if (!ctx) return NF_ERR_ARG;
    NF_ARG(ctx, seg_vel_host && plane_pos_out_host && plane_vel_out_host && out_seg_n, "nf_stream_step_regroup: null pointer table");
    NF_ARG(ctx, kick == kick && drift == drift && fabsf(kick) < 3.0e38f && fabsf(drift) < 3.0e38f, "kick and drift must be finite");
    StepArgs a{seg_vel_host, plane_pos_out_host, plane_vel_out_host, kick, drift, out_seg_n};
    const PlaneIn in{seg_pos_host, seg_n, 3};
    return stream_impl(ctx, in, P, K, R, eps, box, plane0, Gm, softening, plane_acc_host, &a, stats, stream);
}
