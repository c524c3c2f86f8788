/*
 * nf.h -- C ABI of libnf: the near-field force of the Abacus N-body method on one B200.
 *
 * Source of every definition: arXiv:1810.02916, Sec. 2.1 "Method" and Sec. 4.3
 * "Softening".  Readings of points the paper leaves open are listed in DESIGN.md ("Readings").
 *
 *   - "the domain is decomposed into K^3 cubic cells, and every particle belongs to one
 *     cell"                                              -> nf_bin
 *   - "Particles in cells separated by fewer than near-field radius R cells (typically 2)
 *     interact via the near-field force, which we compute as a direct pairwise summation of
 *     1/r^2 forces (or some appropriately softened form)"; 2R+1 slabs are
 *     needed, i.e. the (2R+1)^3 neighbour cells          -> nf_forces
 *   - compact spline softening, Eq. 2; Plummer, Eq. 1
 *   - "positions are stored as offsets relative to cell centers"
 *   - the slab pipeline: "load a rolling window of slabs ... compute forces ... on the
 *     central slab, write out the trailing slab, and then load a slab at the leading edge"
 *     (PAPER.md:41), fed from pinned host memory        -> nf_stream_slabs
 *
 * Conventions
 *   - Plain C types only.  "dev" pointers are CUDA device pointers on the context's device,
 *     "host" pointers are host memory (pinned where stated).  `stream` is a cudaStream_t
 *     passed as void* (NULL = the legacy default stream).
 *   - The caller owns every input and output buffer.  The library never frees or retains a
 *     caller buffer past the stream-ordered work of the call that received it.  The context
 *     owns only scratch memory.
 *   - Every call returns an int status (NF_OK = 0).  Argument checks happen on the host
 *     before any launch.  No exceptions, no exit(), no output to stdout/stderr.
 *     nf_last_error() gives a human-readable detail for the last non-zero status.
 *   - nf_bin and nf_forces are asynchronous: they enqueue work on `stream` and return.
 *     They may synchronise only when scratch memory has to grow (avoid with nf_reserve).  Once the scratch is
 *     reserved they issue nothing but stream-ordered kernels, memsets and event records, so a step (nf_bin +
 *     nf_forces on fixed buffers) can be captured in a CUDA graph and replayed: worth 13 % of a step on the smallest
 *     config (32^3 particles), whose ~45 launches are otherwise latency-bound.
 *   - There is no CPU fallback anywhere in this library.
 *   - A context must not be used from two threads at once.  Its scratch arena is reused from call
 *     to call in stream order: issue the calls of one context on ONE stream (or order the streams
 *     yourself with events); use one context per concurrent stream.
 */
#ifndef NF_H
#define NF_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct nf_ctx nf_ctx;

enum {
    NF_OK = 0,
    NF_ERR_ARG = 1,    /* null pointer, N < 0, K < 2R+1, K > NF_MAX_K, R < 0, eps <= 0, box <= 0, ... */
    NF_ERR_NOMEM = 2,  /* device or host allocation failed */
    NF_ERR_CUDA = 3,   /* CUDA runtime error; nf_last_error() names it */
    NF_ERR_RANGE = 4   /* positions outside [0, box) were seen and clamped into the edge cell */
};

enum {
    NF_SOFT_SPLINE = 0, /* Eq. 2: F = [10 - 15u + 6u^2] r/eps^3 (u = r/eps < 1), r/r^3 beyond */
    NF_SOFT_PLUMMER = 1 /* Eq. 1: F = r/(r^2 + eps^2)^(3/2) */
};

/* Flag OR-ed into the `softening` argument of nf_forces / nf_forces_ex: sources carry their own
 * masses in the .w lane of pos_sorted (written by nf_bin_m) and `Gm` is then G alone:
 * a_i = G * sum_j m_j f(|d|) d.  The paper's runs use equal masses; SURVEY.md Sec. 8(f) rank 1. */
#define NF_MASS_W 0x100
/* Flag OR-ed into the `softening` argument of every force call (nf_forces*, nf_forces_host*, nf_stream_*): the box holds
 * cells of thousands of particles or more ("the largest cell has over 200,000 particles").  Such cells
 * (>= 4096 particles; up to 2048 of them and 2^28 particles per box, or per plane in the
 * slab stream) get their INTERNAL encoded copies ordered along a Hilbert curve inside the cell, with a bounding box per 64
 * particles, so that the kernel can prove most source tiles of a dense cell free of pairs inside eps and sweep them with
 * the bare 1/r^2 law instead of the min form of Eq. 2 -- exact, because the two agree for r >= eps (fn. 4).
 * No output changes its order or meaning; accelerations change in the last bits only (another summation order), and
 * remain bit-reproducible from call to call.  Taken automatically, flag or not, when the mean occupancy (N / K^3; in the
 * slab stream the fullest plane's n / K^2) is at least 512: the decision depends on the arguments alone. */
#define NF_DENSE_ORDER 0x200
#define NF_SOFT_LAW_MASK 0xff

#define NF_MAX_K 1024 /* K^3 must fit a uint32 key; radix digits are per-axis cell indices */
#define NF_MAX_R 3

/* Library version: major*10000 + minor*100 + patch. */
int nf_version(void);

/* Create / destroy a context on CUDA device `device`.  The context owns scratch memory
 * (sort keys, histograms, work lists, slab ring buffers) and internal streams/events. */
int nf_create(nf_ctx **out, int device);
int nf_destroy(nf_ctx *ctx);

/* Text for the last non-zero status returned on this context ("" if none).  The pointer is
 * valid until the next call on the context.  ctx may be NULL (returns a static string). */
const char *nf_last_error(const nf_ctx *ctx);

/* Pre-size scratch for up to maxN particles and K cells per side so that later nf_bin /
 * nf_forces calls with N <= maxN never allocate (and therefore never synchronise). */
int nf_reserve(nf_ctx *ctx, int64_t maxN, int K);

/*
 * nf_bin -- cell assignment + STABLE counting sort into cell-contiguous arrays.
 * (PAPER.md:37 cells; :41/:47 slab = all Y,Z at one X => x is the slowest index; :51 offsets.)
 *
 *   pos_xyz      dev in   N x 3 float32, global positions, each coordinate in [0, box)
 *   N            number of particles, 0 <= N < 2^32
 *   K            cells per side, 1 <= K <= NF_MAX_K
 *   box          periodic box length L > 0
 *   pos_sorted   dev out  N x 4 float32 (16-byte aligned): xyz = offset of the particle from
 *                         the centre of its own cell, w = 0 (reserved: mass)
 *   perm         dev out  N uint32: original index of the particle in each sorted slot
 *   cell_count   dev out  K^3 uint32, linear cell index (cx*K + cy)*K + cz (z fastest)
 *   cell_offset  dev out  K^3+1 uint64, exclusive prefix sum of cell_count
 *
 * Bit-exact contract, all in float32, no fused
 * multiply-add:  invw = (float)K / box;  c = (int)floorf(x * invw) clamped to [0, K-1];
 * hw = 0.5f * (box / (float)K);  centre = (float)(2c+1) * hw;  offset = x - centre.
 * Ties (same cell) keep their input order (perm increases within a cell), so the output is
 * unique.  Particles whose coordinate is outside [0, box) (or NaN) are clamped into the edge
 * cell and counted; read the count with nf_out_of_range().  A coordinate just below box whose
 * product x * invw rounds up to K is valid: it lands in cell K-1 and is not counted.
 */
int nf_bin(nf_ctx *ctx, const float *pos_xyz, int64_t N, int K, float box,
           float *pos_sorted, uint32_t *perm, uint32_t *cell_count, uint64_t *cell_offset,
           void *stream);

/* nf_bin_m -- nf_bin with per-particle masses: mass (dev in, N float32, caller's order, nullable)
 * is carried into the .w lane of pos_sorted (pos_sorted[s].w = mass[perm[s]]; 0 when mass is
 * NULL, which makes nf_bin_m identical to nf_bin).  Everything else as for nf_bin. */
int nf_bin_m(nf_ctx *ctx, const float *pos_xyz, const float *mass, int64_t N, int K, float box,
             float *pos_sorted, uint32_t *perm, uint32_t *cell_count, uint64_t *cell_offset,
             void *stream);

/* nf_keys -- the cell assignment alone: keys[i] =
 * (cx*K + cy)*K + cz of particle i by the bit-exact float32 formula of nf_bin, no histogram, no sort.
 * The x-plane ("slab") a particle is filed under is keys[i] / K^2.
 *   pos_xyz  dev in   N x 3 float32;   keys  dev out  N uint32.
 * Out-of-range particles are clamped and counted as for nf_bin (read with nf_out_of_range). */
int nf_keys(nf_ctx *ctx, const float *pos_xyz, int64_t N, int K, float box, uint32_t *keys, void *stream);

/* Synchronises `stream`, stores the number of out-of-range particles seen by the last nf_bin
 * (or nf_stream_slabs) on this context in *n, and returns NF_ERR_RANGE if it is non-zero. */
int nf_out_of_range(nf_ctx *ctx, int64_t *n, void *stream);

/*
 * nf_forces -- near-field accelerations for every particle (fully periodic box).
 *
 *   a_i = Gm * sum over the (2R+1)^3 periodic neighbour cells c' of cell(i), over j in c':
 *         f(|d|) d,   d = (o_j - o_i) + (c' - c) * w   (cell-centred offsets, w = box/K),
 *   f(r) = min(10 - 15u + 6u^2, u^-3) / eps^3, u = r/eps  (== Eq. 2, see fn. 4 PAPER.md:239),
 *   or the Plummer law.  Pairs with r = 0 (self, coincident particles) contribute zero.
 *   The periodic image of a source is fixed by the cell offset (reading c8).
 *
 *   pos_sorted, cell_offset   dev in   as written by nf_bin
 *   cell_count   dev in, may be NULL: kept in the signature beside nf_bin's other outputs; the
 *                current implementation derives every count from cell_offset and never reads it
 *   perm         dev in, nullable: if given, accelerations are written in the caller's
 *                original order (acc[perm[s]] = a of sorted slot s), else in sorted order
 *   N, K, box    as for nf_bin;  requires K >= 2R+1 (else a cell would be listed twice)
 *   R            near-field radius in cells, 0 <= R <= NF_MAX_R  (the paper uses 2)
 *   eps          softening length > 0: eps_s of Eq. 2, or eps_p of Eq. 1 (no 2.16 factor is
 *                applied inside the library; see nf_spline_equivalent_eps)
 *   Gm           G times the (equal) particle mass
 *   softening    NF_SOFT_SPLINE or NF_SOFT_PLUMMER, optionally | NF_MASS_W and | NF_DENSE_ORDER
 *   acc_xyz      dev out  N x 3 float32
 *
 * float32 in, float32 accumulate (per-tile partial sums formed from zero, added to a running
 * float32 sum over tiles visited in mirror-paired column order; the partial sums of the lanes that
 * share a sink are combined in double), float32 out.  Deterministic: no floating-point atomics;
 * the same inputs give the same bits.  Denormal float32 values are flushed to zero inside the
 * interaction kernel (not in nf_bin / nf_kick_drift, whose contracts are IEEE).
 *
 * Accuracy envelope ("Float32 envelope").  A pair inside one cell is formed from
 * exact differences of cell-centred offsets.  A pair that straddles a cell face is
 * formed from offsets shifted by whole cells in float32, which rounds at ~1e-7 w (w = box/K; up to
 * 2.4e-7 w in z), so such a pair at separation r carries a relative error of up to ~3e-7 w/r in its
 * force.  The north_star bar (1e-5 median, 1e-3 maximum of |da| / max(|a|, rms|a|)) therefore holds
 * when eps >= 4e-3 w and no structure narrower than ~5e-3 w sits on a cell face or corner; below
 * that the maximum error of face-straddling close pairs grows like 3e-7 w / min(r, eps) (an unsoftened
 * clump 1e-4 w wide planted on a corner reaches ~5e-3), while pairs inside one cell stay exact.
 * All five BASELINE configs (eps/w = 5e-3 .. 1e-2) and the paper's run (eps/w ~ 1.4e-2) are inside.
 * The library accepts any eps > 0; results outside the envelope are bounded as stated, not refused.
 *
 * If nf_out_of_range() reports clamped particles for the arrays passed here, accelerations of
 * particles in the edge cells are unspecified (the pruning of close-pair tests assumes every offset
 * lies within its cell): treat NF_ERR_RANGE as an error of the input, not as a warning.
 */
int nf_forces(nf_ctx *ctx, const float *pos_sorted, const uint64_t *cell_offset,
              const uint32_t *cell_count, const uint32_t *perm, int64_t N, int K, int R,
              float eps, float box, float Gm, int softening, float *acc_xyz, void *stream);

/*
 * nf_forces_ex -- nf_forces with the outputs the time-step criterion needs (PAPER.md:194, :207:
 * "TimeStepAccel times the maximum of v_rms/a_max computed within each cell"; SURVEY.md Sec. 8(f)
 * rank 2), reduced inside the interaction kernel's epilogue:
 *
 *   cell_amax   dev out, nullable  K^3 float32: max over the particles of each cell of |a_i|
 *               (2-norm of the float32 acceleration written to acc_xyz); 0 for empty cells.
 *               Exact and order-independent: an integer atomicMax on the float bit patterns.
 *   softening   may carry NF_MASS_W (per-particle source masses, see above)
 *
 * nf_forces(...) is nf_forces_ex(..., cell_amax = NULL, ...).
 */
int nf_forces_ex(nf_ctx *ctx, const float *pos_sorted, const uint64_t *cell_offset,
                 const uint32_t *cell_count, const uint32_t *perm, int64_t N, int K, int R,
                 float eps, float box, float Gm, int softening, float *acc_xyz,
                 float *cell_amax, void *stream);

/*
 * nf_forces_chunk -- nf_forces_ex for a device-resident CHUNK of the box: the multi-GPU slab
 * decomposition (PAPER.md:41 slabs, :81 "a parallel version of Abacus based on the existing slab
 * decomposition").  The arrays describe whatever particles this GPU holds,
 * binned by nf_bin over the full K^3 grid: its own x-planes [x_lo, x_hi) plus the R ghost planes
 * received from each x-neighbour; all other planes are simply empty.  Only particles of planes
 * [x_lo, x_hi) are sinks (acc_xyz rows of ghost particles are not written); every particle present is
 * a source for the sinks within R cells of it, with the usual periodic wrap in x, y and z -- so a
 * chunk touching the box edge takes its wrapped ghost planes with their stored coordinates.
 * Missing planes contribute nothing: x is open at the ends of what was supplied.
 *
 *   x_lo, x_hi   sink plane range, 0 <= x_lo <= x_hi <= K (ranges that wrap are two calls)
 *   cell_amax    nullable, K^3 float32 as for nf_forces_ex (zero outside the sink planes)
 *   everything else as for nf_forces_ex.  nf_forces_ex is nf_forces_chunk with [0, K).  A sink's acceleration does not depend on
 *   the range it is computed in, up to the last bits: the bits are the same as long as no task of the call is split over
 *   several work-list entries (small problems with few, long tasks), else equal within rounding.
 */
int nf_forces_chunk(nf_ctx *ctx, const float *pos_sorted, const uint64_t *cell_offset, const uint32_t *perm,
                    int64_t N, int K, int R, float eps, float box, float Gm, int softening, int x_lo, int x_hi,
                    float *acc_xyz, float *cell_amax, void *stream);

/*
 * nf_forces_tree -- nf_forces_ex with a TREE for the sources of dense cells ("Future versions of Abacus
 * will employ trees in the near-field domain, especially for dense cells"; "the largest cell has over
 * 200,000 particles").  The paper names the idea and prints no algorithm; the one built
 * here is stated in DESIGN.md (readings t1-t6) and followed step by step by oracle/nf_tree.py:
 *
 *   - a cell of >= 4096 particles is DENSE (the cells NF_DENSE_ORDER orders: at most 2048 of them and
 *     2^28 particles in 64-aligned sizes, taken in cell order; further ones are not dense);
 *   - its particles, in Hilbert order of their cell-centred offsets, form leaves of 16 and nodes of 8 children up to a
 *     root; a node has the bounding box of its particles, their mass and centre of mass;
 *   - sinks are taken 64 at a time (consecutive in their cell) with their bounding box -- a group whose box is more than
 *     three times wider (diagonal) than the tightest of its four quarters walks quarter by quarter, such a quarter sink by
 *     sink --; such a group meets each dense
 *     cell among its (2R+1)^3 neighbours by walking that cell's tree: a node whose box is further from the group's box
 *     than eps and than (its diagonal / theta) acts as ONE particle at its centre of mass (1/r^2); any other node is
 *     opened, and a leaf that is not accepted is summed particle by particle with the softened law of `softening`;
 *   - sources of cells that are not dense are summed directly, exactly as by nf_forces_ex.
 *
 *   theta       opening angle, 0 <= theta < 1.  theta = 0 accepts nothing: the result is the direct sum (nf_forces_ex up
 *               to summation order).  For theta > 0 the result is an APPROXIMATION: per accepted node the error is at
 *               most G M / D^2 * (1/(1-theta)^2 - 1 - 2 theta), D the distance to its centre of mass.
 *               Measured on one cell of 4x10^5 particles: theta = 0.5 is 8x faster than the direct sum and 3x10^-4 (median,
 *               north-star metric) away from it, theta = 0.7 13x and 7x10^-4; theta = 0 is 10x SLOWER than nf_forces_ex.
 *   everything else as for nf_forces_ex (NF_MASS_W allowed; NF_DENSE_ORDER implied).  cell_amax is computed from the
 *   final accelerations.  Asynchronous on `stream`; deterministic (bit-reproducible from call to call).
 *   The box must be whole (no chunk / slab / host variant).
 *
 * nf_tree_stats -- what the last nf_forces_tree on this context evaluated (synchronises `stream`):
 *   node_interactions  sum over (sink, accepted node) pairs
 *   leaf_interactions  sum over (sink, particle of an opened leaf) pairs
 * The walk's decisions are taken in float32 in a fixed order of rounded operations, so both counts are exact
 * properties of the input (the oracle reproduces them bit for bit).
 */
int nf_forces_tree(nf_ctx *ctx, const float *pos_sorted, const uint64_t *cell_offset, const uint32_t *perm, int64_t N,
                   int K, int R, float eps, float box, float Gm, int softening, float theta, float *acc_xyz,
                   float *cell_amax, void *stream);
int nf_tree_stats(nf_ctx *ctx, int64_t *node_interactions, int64_t *leaf_interactions, void *stream);
/* duration of the walk kernel of the last nf_forces_tree on this context (CUDA events on its stream; synchronises on the end event) */
int nf_last_tree_timing(nf_ctx *ctx, float *walk_ms);

/*
 * nf_kick_drift -- the leapfrog updates that follow the force in the slab pipeline (Table 1
 * "Kick", "Drift").  The paper gives no formula, so the
 * factors are the caller's (they absorb the cosmological prefactors of the time step):
 *
 *   v <- v + a * kick ;   x <- x + v * drift  (with the NEW v), wrapped once into [0, box)
 *
 * float32 contract, bit-reproducible: v1 = fma(a, kick, v) and x1 = fma(v1, drift, x), each a single
 * rounding; then x1 >= box: x1 - box; x1 < 0: x1 + box; a result equal to box becomes 0.  One wrap only:
 * the third time-step criterion keeps |v * drift| below 80 % of a cell width.
 *
 *   pos_xyz, vel_xyz   dev in/out  N x 3 float32 (updated in place)
 *   acc_xyz            dev in      N x 3 float32, same order
 */
int nf_kick_drift(nf_ctx *ctx, float *pos_xyz, float *vel_xyz, const float *acc_xyz, int64_t N,
                  float kick, float drift, float box, void *stream);

/*
 * nf_cell_vrms -- velocity reductions of the time-step criteria: the rms speed
 * within each cell (criterion 2 pairs it with the a_max of nf_forces_ex) and the largest velocity
 * component of any particle (criterion 3: "the step size times the maximum velocity must be less
 * than 80% of a cell width").
 *
 *   vel_xyz      dev in   N x 3 float32 in the caller's order (perm given) or in sorted order (perm NULL)
 *   perm, cell_offset     dev in   as written by nf_bin for the same particles
 *   cell_vrms    dev out, nullable  K^3 float32: sqrt(mean |v|^2) over the cell's particles, 0 if empty
 *   vmax         dev out, nullable  1 float32: max over particles and axes of |v_axis|
 */
int nf_cell_vrms(nf_ctx *ctx, const float *vel_xyz, const uint32_t *perm, const uint64_t *cell_offset,
                 int64_t N, int K, float *cell_vrms, float *vmax, void *stream);

/*
 * nf_timestep_terms -- the reduction of time-step criteria 2 and 3 from the per-cell
 * quantities nf_forces_ex (a_max) and nf_cell_vrms (v_rms, maximum velocity) return:
 *
 *   criterion 2  "the step size must be less than TimeStepAccel times the maximum of v_rms/a_max computed within
 *                each cell" (:194) ... "we also compute a global v_rms/a_max and use the maximum of the global and
 *                cell-based values.  This protects us from taking catastrophically small time steps as a result of
 *                abnormally cold cells" (:207).  A cold cell makes its own ratio SMALL, so the cell-based value that
 *                the global one guards against is the smallest ratio over cells (reading c19); the largest
 *                is returned too, for the literal reading.
 *   criterion 3  "the step size times the maximum velocity must be less than 80% of a cell width" (:195).
 *
 *   cell_vrms, cell_amax   dev in   K^3 float32 each (nf_cell_vrms / nf_forces_ex)
 *   cell_offset            dev in   K^3 + 1 uint64 (nf_bin): particle counts weight the global v_rms
 *   vmax                   dev in, nullable  1 float32 (nf_cell_vrms)
 *   out                    host out
 *
 * Cells that are empty or have a_max = 0 take no part in the cell ratios.  Each ratio is the float32 quotient
 * v_rms / a_max (round to nearest), so minimum and maximum are exact and order-independent; the global v_rms is
 * sqrt(sum_c n_c v_rms_c^2 / N) accumulated in double in a fixed order (deterministic).  Synchronises `stream`.
 * The caller multiplies by its own TimeStepAccel (eta) and combines with criterion 1.
 */
typedef struct nf_timestep {
    double ratio_cell_min;   /* min over cells of v_rms / a_max        (0 if no cell qualifies) */
    double ratio_cell_max;   /* max over cells of v_rms / a_max */
    double ratio_global;     /* global v_rms / global a_max            (0 if a_max = 0) */
    double ratio_criterion2; /* max(ratio_global, ratio_cell_min): the step is eta times this (reading c19) */
    double vrms_global, amax_global, vmax;
    double drift_limit;      /* criterion 3: 0.8 * (box / K) / vmax    (infinity if vmax = 0 or not given) */
    int64_t cells_used;      /* cells that entered the cell ratios */
} nf_timestep;
int nf_timestep_terms(nf_ctx *ctx, const float *cell_vrms, const float *cell_amax, const uint64_t *cell_offset,
                      int K, float box, const float *vmax, nf_timestep *out, void *stream);

/*
 * nf_timestep_terms_static -- nf_timestep_terms for callers that cannot call cudaMalloc (code under CUDA graph capture,
 * tight serving loops, harnesses that forbid it): it allocates nothing.  nf_timestep_terms takes its scratch (one
 * partial record per block of cells) from the context's arena, which grows with cudaMalloc on demand; this call keeps
 * the same scratch in a file-scope __device__ array of fixed size -- 4097 records of 40 bytes = 164 KB, which every GPU
 * that loads the library holds until the process exits -- and calls no cudaMalloc, cudaFree or allocating library
 * routine.  Same kernels, same arguments, same meaning of `out`; minimum, maximum and counts are identical to
 * nf_timestep_terms, the double sum behind vrms_global is formed over other block boundaries (equal within rounding).
 *
 *   K <= NF_TS_STATIC_MAX_K (256): one record per 4096 cells, 4096 records.  A larger K is NF_ERR_ARG with a message
 *   that says so; use nf_timestep_terms there.
 *   All calls, from every context and stream on a device, share the one array; it keeps the last call's contents
 *   (nothing needs clearing: every record read was written by the same call).  Calls that OVERLAP on the GPU race:
 *   issue them on one stream or order them yourself.  Synchronises `stream` (the result is returned to the host).
 */
#define NF_TS_STATIC_MAX_K 256
int nf_timestep_terms_static(nf_ctx *ctx, const float *cell_vrms, const float *cell_amax, const uint64_t *cell_offset,
                             int K, float box, const float *vmax, nf_timestep *out, void *stream);

/*
 * nf_forces_host -- the whole path from HOST buffers: H2D copy of the positions, nf_bin,
 * nf_forces, D2H copy of the accelerations (the paper's GPU rate "includes
 * PCIe bus transfer overheads").  All device buffers come from the context's scratch arena
 * (about 60 bytes per particle; pre-size with nf_reserve_host to avoid the first-call
 * allocation).
 *
 *   pos_host   host in   N x 3 float32 global positions (pinned memory recommended; pageable
 *                        memory works but the copies are then staged by the driver)
 *   acc_host   host out  N x 3 float32 accelerations in the caller's order
 *   other arguments as for nf_bin / nf_forces.
 *
 * The call returns after the D2H copy has completed (it synchronises `stream`).  Returns
 * NF_ERR_RANGE (after completing the computation) if positions outside [0, box) were clamped.
 * nf_forces_host takes equal masses only (NF_MASS_W is an NF_ERR_ARG here);
 * nf_forces_host_m adds   mass_host  host in, N float32 source masses in the caller's order, and
 * wants NF_MASS_W set in `softening` exactly when mass_host is non-NULL (Gm is then G).
 */
int nf_forces_host(nf_ctx *ctx, const float *pos_host, int64_t N, int K, int R, float eps,
                   float box, float Gm, int softening, float *acc_host, void *stream);
int nf_forces_host_m(nf_ctx *ctx, const float *pos_host, const float *mass_host, int64_t N, int K, int R,
                     float eps, float box, float Gm, int softening, float *acc_host, void *stream);
int nf_reserve_host(nf_ctx *ctx, int64_t maxN, int K);

/*
 * nf_forces_host_begin / nf_forces_host_end -- nf_forces_host as a two-deep pipeline, for callers with a
 * sequence of independent batches (or with step n+1's positions ready while step n is still running): the
 * H2D copy of step n+1 and the D2H copy of step n run on the context's copy streams BEHIND the kernels of the
 * step in between (PAPER.md:69 GPU work overlapped with the transfers; :111 the paper's rate "includes PCIe
 * bus transfer overheads"), so a steady stream of steps runs at the speed of the kernels alone.
 *
 *   begin  enqueues one whole step (H2D, nf_bin, nf_forces, D2H into acc_host) and returns at once; at most
 *          two steps may be in flight (a third begin is an NF_ERR_ARG).  pos_host and acc_host must be pinned
 *          for the copies to be asynchronous, and must stay valid and untouched until the matching end.
 *          Equal masses only.  N and K must not change while a step is in flight.
 *   end    waits for the OLDEST step in flight (its accelerations are then in its acc_host) and returns its
 *          status: NF_ERR_RANGE if positions outside [0, box) were clamped.
 *
 * Between a begin and its end no other call may be made on this context (the scratch arena is in use).
 * Device memory: about 112 bytes per particle (input and output buffers doubled).
 */
int nf_forces_host_begin(nf_ctx *ctx, const float *pos_host, int64_t N, int K, int R, float eps, float box,
                         float Gm, int softening, float *acc_host, void *stream);
int nf_forces_host_end(nf_ctx *ctx);

/* Number of ordered (sink, source) pairs nf_forces evaluates for these cell counts:
 * I = sum_c n_c * sum_{c' in N(c)} n_c'  (self pairs included, padding excluded; the
 * "pairwise interactions" of PAPER.md:107).  Computed on the device, synchronises `stream`,
 * result in *interactions (host). */
int nf_interactions(nf_ctx *ctx, const uint32_t *cell_count, int K, int R,
                    int64_t *interactions, void *stream);

/* eps_s = 2.16 eps_p: the spline softening with the same minimum pairwise
 * dynamical time as a Plummer softening eps_p.  Pure host helper. */
float nf_spline_equivalent_eps(float eps_plummer);

/* Statistics of one nf_stream_slabs call (all times in seconds, measured with CUDA events). */
typedef struct nf_stream_stats {
    int64_t particles_in;    /* particles copied host -> device (sink + ghost planes) */
    int64_t particles_out;   /* accelerations copied device -> host (sink planes) */
    int64_t interactions;    /* ordered pairs evaluated */
    int64_t out_of_range;    /* particles clamped (see nf_bin) or found in the wrong plane */
    double h2d_bytes, d2h_bytes;
    double h2d_seconds, d2h_seconds;      /* sum of the individual copies' durations */
    double kernel_seconds;                /* sum of bin + force kernel durations */
    double wall_seconds;                  /* first H2D start to last D2H end */
    double h2d_gbps, d2h_gbps;            /* bytes / copy seconds */
    double overlap_fraction;              /* 1 - (wall - kernel)/ (h2d + d2h seconds), clamped to [0,1] */
    double force_seconds;                 /* the part of kernel_seconds spent in work-list build + interaction kernel */
} nf_stream_stats;

/*
 * nf_stream_slabs -- the slab-ordered pass over P consecutive x-planes of
 * cells, from pinned host memory, with H2D / D2H copies on side streams overlapping the
 * kernels.
 *
 *   plane_pos_host  host in   P + 2R pointers (pinned = page-locked host memory, cudaMemoryTypeHost;
 *                             pageable or managed memory is refused with NF_ERR_ARG); plane q holds plane_n[q] x 3
 *                             float32 global positions of the particles whose x-cell index
 *                             is (plane0 + q) mod K; the first and last R planes are ghosts
 *                             (sources only)
 *   plane_n         host in   P + 2R particle counts
 *   P               number of sink planes, >= 1
 *   K               cells per side of the full box (y and z have K cells and are periodic
 *                   with period box; cell width w = box / K)
 *   R, eps, Gm, softening     as for nf_forces
 *   plane0          x-cell index of the first ghost plane, may be negative or wrap past K
 *                   (the plane index is taken modulo K; the caller supplies the wrapped
 *                   planes' particles with their stored coordinates in [0, box))
 *   plane_acc_host  host out  P pointers (pinned): plane_n[R+p] x 3 float32 accelerations of
 *                             sink plane p, in that plane's input order
 *   stats           host out, nullable
 *
 * x is open inside the chunk: only the P + 2R supplied planes act as sources.  Requires
 * K >= 2R+1 and P <= K (with P + 2R > K the ghost planes repeat sink planes of the other end of
 * the periodic box: pass the same arrays again).  Returns after the last D2H copy has completed
 * (the call synchronises, also on every error path, so no caller buffer is in use after it
 * returns); `stream` orders the call after prior work on that stream.
 * A particle outside [0, box) or filed under a plane other than the one its x coordinate maps to
 * (nf_keys / K^2) is clamped into its plane's edge cells and counted in stats->out_of_range; the
 * call then completes and returns NF_ERR_RANGE, and the accelerations of that pass are unspecified
 * near those particles (see the envelope note of nf_forces).
 */
int nf_stream_slabs(nf_ctx *ctx, const float *const *plane_pos_host, const int64_t *plane_n,
                    int P, int K, int R, float eps, float box, int plane0, float Gm,
                    int softening, float *const *plane_acc_host, nf_stream_stats *stats,
                    void *stream);

/*
 * nf_stream_step_slabs -- nf_stream_slabs with the Kick and Drift of the slab pipeline (Table 1,
 * PAPER.md:149-150) as a streaming epilogue: after the forces of a sink plane its particles are
 * kicked and drifted on the device (nf_kick_drift's float32 contract) and the NEW positions and
 * velocities are copied back instead of (or beside) the accelerations -- one pass over the chunk
 * per time step.
 *
 *   plane_vel_host       host in   P pointers (pinned): velocities of sink plane p, plane_n[R+p] x 3
 *   kick, drift          as for nf_kick_drift
 *   plane_pos_out_host   host out  P pointers (pinned): drifted positions of sink plane p, input order,
 *                                  wrapped into [0, box) -- a particle may have left its plane; this call
 *                                  leaves the filing to the caller, nf_stream_step_regroup does it in the stream
 *   plane_vel_out_host   host out  P pointers (pinned): kicked velocities
 *   plane_acc_host       host out, nullable table: the accelerations, as nf_stream_slabs writes them
 *   everything else as for nf_stream_slabs.
 */
int nf_stream_step_slabs(nf_ctx *ctx, const float *const *plane_pos_host, const float *const *plane_vel_host,
                         const int64_t *plane_n, int P, int K, int R, float eps, float box, int plane0,
                         float Gm, int softening, float kick, float drift, float *const *plane_pos_out_host,
                         float *const *plane_vel_out_host, float *const *plane_acc_host,
                         nf_stream_stats *stats, void *stream);

/*
 * nf_regroup_plane -- regrouping after the drift, one plane ("update particles on the central
 * slab, write out the trailing slab"; :195, :209 "particles drift by at most one slab per time step";
 * SURVEY.md Sec. 8(f) rank 3).  The drifted particles of x-plane plane_cx are rewritten as three STABLE
 * segments by the plane their new x coordinate maps to (the bit-exact cell formula of nf_bin / nf_keys):
 *
 *     [ now in plane_cx - 1 | still in plane_cx | now in plane_cx + 1 ]      (periodic in K; input order kept
 *                                                                             inside each segment)
 *   pos_xyz, vel_xyz   dev in   N x 3 float32, positions already wrapped into [0, box) (nf_kick_drift)
 *   pos_out, vel_out   dev out  N x 3 float32, must not alias the inputs
 *   seg_n              host out 3 segment lengths (they sum to N)
 *
 * The new content of plane d is then [ third segment of d-1 | second of d | first of d+1 ].  A particle that
 * moved further than one plane breaks time-step criterion 3: it is filed under the nearer neighbour and
 * counted, and the call returns NF_ERR_RANGE after completing.  Synchronises `stream` (it returns counts).
 */
int nf_regroup_plane(nf_ctx *ctx, const float *pos_xyz, const float *vel_xyz, int64_t N, int K, float box,
                     int plane_cx, float *pos_out, float *vel_out, int64_t *seg_n, void *stream);

/*
 * nf_stream_step_regroup -- nf_stream_step_slabs with the regrouping done in the stream as well, so that one
 * call is one whole time step of the slab pipeline and its output is directly the input of the
 * next call -- no host-side filing in between.
 *
 *   seg_pos_host   host in  (P + 2R) x 3 pinned pointers: plane q is the concatenation, in this order, of the
 *                           segments seg_pos_host[3q + 0..2] with seg_n[3q + 0..2] particles (empty segments
 *                           may be NULL).  A first step passes whole planes as {NULL, plane, NULL}; a later
 *                           step passes, for plane d, the three segments the previous step wrote:
 *                           {third segment of plane d-1's output, second of d's, first of d+1's}.
 *   seg_vel_host   host in  P x 3 pinned pointers: velocities of the sink planes, same segmentation
 *   seg_n          host in  (P + 2R) x 3 counts
 *   plane_pos_out_host, plane_vel_out_host
 *                  host out P pinned pointers, each with room for the plane's particles (sum of its 3 input
 *                           segments): the kicked and drifted particles of sink plane p as the three stable
 *                           segments of nf_regroup_plane
 *   out_seg_n      host out P x 3 segment lengths
 *   plane_acc_host host out, nullable table: accelerations in the plane's INPUT order (before regrouping)
 *   everything else as for nf_stream_step_slabs.  With P = K (ghost planes = the sink planes of the other end
 *   of the periodic box, passed again) the call steps the whole box.
 */
int nf_stream_step_regroup(nf_ctx *ctx, const float *const *seg_pos_host, const float *const *seg_vel_host,
                           const int64_t *seg_n, int P, int K, int R, float eps, float box, int plane0, float Gm,
                           int softening, float kick, float drift, float *const *plane_pos_out_host,
                           float *const *plane_vel_out_host, int64_t *out_seg_n, float *const *plane_acc_host,
                           nf_stream_stats *stats, void *stream);

/* Timing of the kernels of the last nf_forces call on this context (CUDA events recorded on
 * the call's stream around the interaction kernel).  Synchronises on the end event.
 * *kernel_ms = duration of the interaction kernel alone; *total_ms = whole nf_forces call
 * (work-list build + kernel + scale/un-permute).  Either pointer may be NULL. */
int nf_last_forces_timing(nf_ctx *ctx, float *kernel_ms, float *total_ms);

/* Number of CUDA kernels this context has launched since nf_create (memcpy / memset nodes are
 * not counted).  Host-side counter; does not synchronise.  Used by bench.py's gpu_launches. */
int nf_launch_count(const nf_ctx *ctx, int64_t *launches);

#ifdef __cplusplus
}
#endif
#endif /* NF_H */
