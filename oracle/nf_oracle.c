/*
 * nf_oracle.c -- CPU oracle for the Abacus near-field force (arXiv:1810.02916).
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may build, load or call it.
 * It shares no code, header, table or constant with the CUDA path under
 * paper_1810_02916_b200/csrc/ and neither includes the other.
 *
 * What it computes (the method reaches this result exactly, up to rounding:
 * "the near-field force is exact (up to machine precision)", PAPER.md:39;
 * "brute-force N^2 summation"):
 *
 *   - the domain is K^3 cubic cells and every particle belongs to one cell (Sec. 2.1);
 *   - particles in cells within near-field radius R cells of each other interact by a direct
 *     pairwise sum; "R slabs must be present on either side ... For R = 2, this
 *     means 5 slabs" fixes the neighbourhood as (2R+1)^3 cells, Chebyshev cell
 *     distance <= R inclusive (reading c1);
 *   - the pair force is the compact spline of Eq. 2 (Sec. 4.3.1):
 *         F(r) = [10 - 15(r/eps) + 6(r/eps)^2] r/eps^3   for r <  eps
 *         F(r) = r / r^3                                  for r >= eps
 *     and, as a variant, Plummer softening, Eq. 1: F = r/(r^2+eps_p^2)^(3/2).
 *
 * Everything floating-point is double precision, computed from the caller's float32 global
 * positions promoted to double -- except the cell assignment and the cell-centred offsets,
 * whose float32 formulas ARE the bit-exact contract.
 * Compile with -ffp-contract=off so that no multiply-add is fused.
 *
 * Pins (tests/test_oracle_pins.py): pair-centric brute force on tiny inputs, two-particle
 * closed forms inside and outside eps, C2 continuity at r = eps, the min identity of
 * footnote 4, antisymmetry / zero net force, symmetric lattice, power-of-two
 * rescaling, whole-cell translation, all-pairs direct sum for K = 2R+1.  Next rows: masses (mass-ratio
 * closed form, momentum, brute force with masses, linearity), per-cell a_max / v_rms (python-loop
 * definition), kick + drift (hand-worked exact cases, leapfrog invariant of the harmonic oscillator).
 * nfo_kick_drift: the paper names Kick and Drift but prints no formula, so its
 * parity is UNPINNED AGAINST THE PAPER; it is pinned to the textbook leapfrog only (reading c20).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* ---- cell assignment: "every particle belongs to one cell" ------------------
 * Float32 contract: invw = (float)K / box (one float32 division);
 * t = x * invw (one float32 multiply); c = (int)floorf(t), clamped to [0, K-1].
 * Returns 1 if x itself is outside [0, box) or NaN (reading c9).  An x just below
 * box whose product x*invw rounds up to K is a valid position: it is clamped into cell K-1 and
 * NOT reported. */
static int cell_of(float x, float invw, float box, int K, int *c_out)
{
    float t = x * invw;
    float fl = floorf(t);
    int bad = !(x >= 0.0f && x < box);
    int c;
    if (!(fl >= 0.0f)) c = 0;               /* negative or NaN */
    else if (fl > (float)(K - 1)) c = K - 1;
    else c = (int)fl;
    *c_out = c;
    return bad;
}

/* key = (cx*K + cy)*K + cz : x slowest (a slab is all Y,Z at one X), z fastest. */
int64_t nfo_keys(const float *pos, int64_t N, int K, float box, uint32_t *key)
{
    float invw = (float)K / box;
    int64_t nbad = 0;
    for (int64_t i = 0; i < N; i++) {
        int cx, cy, cz;
        int b = cell_of(pos[3 * i + 0], invw, box, K, &cx);
        b |= cell_of(pos[3 * i + 1], invw, box, K, &cy);
        b |= cell_of(pos[3 * i + 2], invw, box, K, &cz);
        key[i] = (uint32_t)(((int64_t)cx * K + cy) * K + cz);
        nbad += b;
    }
    return nbad;
}

/* ---- stable counting sort by cell key -------------------------------------------------
 * Outputs: cell_count[K^3], cell_offset[K^3+1] (exclusive prefix sum), perm[N] (original
 * index of each sorted slot; increasing within a cell = stable), pos_sorted[N][4]:
 * xyz = float32 offset from the particle's own cell centre ("positions are stored as
 * offsets relative to cell centers"), w = 0.
 * Offset contract: hw = 0.5f*(box/(float)K); centre = (float)(2c+1)*hw; o = x - centre,
 * each a single float32 operation.  Returns the number of out-of-range particles. */
int64_t nfo_bin(const float *pos, int64_t N, int K, float box,
                float *pos_sorted, uint32_t *perm, uint32_t *cell_count, uint64_t *cell_offset)
{
    int64_t ncell = (int64_t)K * K * K;
    uint32_t *key = (uint32_t *)malloc(sizeof(uint32_t) * (size_t)(N > 0 ? N : 1));
    int64_t nbad = nfo_keys(pos, N, K, box, key);
    memset(cell_count, 0, sizeof(uint32_t) * (size_t)ncell);
    for (int64_t i = 0; i < N; i++) cell_count[key[i]]++;
    cell_offset[0] = 0;
    for (int64_t c = 0; c < ncell; c++) cell_offset[c + 1] = cell_offset[c] + cell_count[c];
    uint64_t *cursor = (uint64_t *)malloc(sizeof(uint64_t) * (size_t)ncell);
    memcpy(cursor, cell_offset, sizeof(uint64_t) * (size_t)ncell);
    float w = box / (float)K;
    float hw = 0.5f * w;
    for (int64_t i = 0; i < N; i++) {           /* increasing i => stable */
        uint32_t k = key[i];
        uint64_t s = cursor[k]++;
        int cz = (int)(k % (uint32_t)K);
        int cy = (int)((k / (uint32_t)K) % (uint32_t)K);
        int cx = (int)(k / ((uint32_t)K * (uint32_t)K));
        float ctrx = (float)(2 * cx + 1) * hw;
        float ctry = (float)(2 * cy + 1) * hw;
        float ctrz = (float)(2 * cz + 1) * hw;
        pos_sorted[4 * s + 0] = pos[3 * i + 0] - ctrx;
        pos_sorted[4 * s + 1] = pos[3 * i + 1] - ctry;
        pos_sorted[4 * s + 2] = pos[3 * i + 2] - ctrz;
        pos_sorted[4 * s + 3] = 0.0f;
        perm[s] = (uint32_t)i;
    }
    free(cursor);
    free(key);
    return nbad;
}

/* ---- pair force laws, |F|/r as a function of r (so that F_vec = fr * d_vec) ------------- */

/* Eq. 2.  r > 0. */
double nfo_spline_over_r(double r, double eps)
{
    double u = r / eps;
    if (u < 1.0) return (10.0 - 15.0 * u + 6.0 * u * u) / (eps * eps * eps);
    return 1.0 / (r * r * r);
}

/* Eq. 1. */
double nfo_plummer_over_r(double r, double eps_p)
{
    double s = r * r + eps_p * eps_p;
    return 1.0 / (s * sqrt(s));
}

/* ---- near-field accelerations ---------------------------------------------------------
 * a_i = Gm * sum over the (2R+1)^3 periodic neighbour cells c' of cell(i), over j in c',
 *       of F(|d|)/|d| * d,   d = (x_j + n*box) - x_i   (attractive; reading c2),
 * where n in {-1,0,1} per axis is the periodic image selected by the CELL offset
 * (c' = (c + delta) mod K, n = floor((c + delta)/K); reading c8), not by minimum
 * image.  Pairs with r^2 == 0 (the self pair, coincident particles) contribute nothing:
 * Eq. 2 gives F = 10*0/eps^3 = 0 (reading c6).
 *
 * sink_idx: original indices of the sinks to evaluate (NULL = all N, in input order).
 * acc: n_sinks x 3 doubles, in the order of sink_idx.
 * softening: 0 = spline (Eq. 2, eps = eps_s), 1 = Plummer (Eq. 1, eps = eps_p).
 * mass: NULL = equal masses (the paper's case; Gm = G*m), else N float32 source
 *       masses in input order and a_i = Gm * sum_j m_j F d/|d| with Gm = G (SURVEY.md Sec. 8(f) rank 1:
 *       the pair force of PAPER.md:37 between unequal masses is G m_i m_j F, so the acceleration of i
 *       carries m_j).
 * Returns 0, or -1 on bad arguments (K < 2R+1 would list a cell twice). */
int nfo_forces_m(const float *pos, const float *mass, int64_t N, int K, int R, double eps, float box, double Gm,
                 const int64_t *sink_idx, int64_t n_sinks, int softening, int nthreads,
                 double *acc)
{
    if (K < 2 * R + 1 || R < 0 || !(eps > 0.0) || !(box > 0.0f) || N < 0) return -1;
    int64_t ncell = (int64_t)K * K * K;
    uint32_t *key = (uint32_t *)malloc(sizeof(uint32_t) * (size_t)(N > 0 ? N : 1));
    nfo_keys(pos, N, K, box, key);
    uint64_t *off = (uint64_t *)calloc((size_t)ncell + 1, sizeof(uint64_t));
    for (int64_t i = 0; i < N; i++) off[key[i] + 1]++;
    for (int64_t c = 0; c < ncell; c++) off[c + 1] += off[c];
    uint64_t *cursor = (uint64_t *)malloc(sizeof(uint64_t) * (size_t)ncell);
    memcpy(cursor, off, sizeof(uint64_t) * (size_t)ncell);
    /* cell-contiguous copies of the GLOBAL positions, promoted to double */
    double *X = (double *)malloc(sizeof(double) * 3 * (size_t)(N > 0 ? N : 1));
    double *M = mass ? (double *)malloc(sizeof(double) * (size_t)(N > 0 ? N : 1)) : NULL;
    for (int64_t i = 0; i < N; i++) {
        uint64_t s = cursor[key[i]]++;
        X[3 * s + 0] = (double)pos[3 * i + 0];
        X[3 * s + 1] = (double)pos[3 * i + 1];
        X[3 * s + 2] = (double)pos[3 * i + 2];
        if (M) M[s] = (double)mass[i];
    }
    free(cursor);
    if (sink_idx == NULL) n_sinks = N;
    double L = (double)box;
#ifdef _OPENMP
    if (nthreads > 0) omp_set_num_threads(nthreads);
#endif
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t s = 0; s < n_sinks; s++) {
        int64_t i = sink_idx ? sink_idx[s] : s;
        double xi = (double)pos[3 * i + 0], yi = (double)pos[3 * i + 1], zi = (double)pos[3 * i + 2];
        uint32_t k = key[i];
        int cz = (int)(k % (uint32_t)K);
        int cy = (int)((k / (uint32_t)K) % (uint32_t)K);
        int cx = (int)(k / ((uint32_t)K * (uint32_t)K));
        double ax = 0.0, ay = 0.0, az = 0.0;
        for (int dx = -R; dx <= R; dx++) {
            int gx = cx + dx;
            int nx = (gx < 0) ? -1 : (gx >= K ? 1 : 0);
            int sx = gx - nx * K;
            for (int dy = -R; dy <= R; dy++) {
                int gy = cy + dy;
                int ny = (gy < 0) ? -1 : (gy >= K ? 1 : 0);
                int sy = gy - ny * K;
                for (int dz = -R; dz <= R; dz++) {
                    int gz = cz + dz;
                    int nz = (gz < 0) ? -1 : (gz >= K ? 1 : 0);
                    int sz = gz - nz * K;
                    int64_t c2 = ((int64_t)sx * K + sy) * K + sz;
                    for (uint64_t j = off[c2]; j < off[c2 + 1]; j++) {
                        double ddx = (X[3 * j + 0] + nx * L) - xi;
                        double ddy = (X[3 * j + 1] + ny * L) - yi;
                        double ddz = (X[3 * j + 2] + nz * L) - zi;
                        double r2 = ddx * ddx + ddy * ddy + ddz * ddz;
                        if (r2 == 0.0) continue;
                        double r = sqrt(r2);
                        double f = softening ? nfo_plummer_over_r(r, eps)
                                             : nfo_spline_over_r(r, eps);
                        if (M) f *= M[j];
                        ax += f * ddx;
                        ay += f * ddy;
                        az += f * ddz;
                    }
                }
            }
        }
        acc[3 * s + 0] = Gm * ax;
        acc[3 * s + 1] = Gm * ay;
        acc[3 * s + 2] = Gm * az;
    }
    free(X);
    free(M);
    free(off);
    free(key);
    return 0;
}

int nfo_forces(const float *pos, int64_t N, int K, int R, double eps, float box, double Gm,
               const int64_t *sink_idx, int64_t n_sinks, int softening, int nthreads,
               double *acc)
{
    return nfo_forces_m(pos, NULL, N, K, R, eps, box, Gm, sink_idx, n_sinks, softening, nthreads, acc);
}

/* Per-cell maximum of |a| (2-norm), the quantity the time-step criterion takes "within each cell"
 * (PAPER.md:194, :207).  acc: N x 3 doubles in input order; key: the particles' cell keys;
 * amax: ncell doubles, 0 for empty cells.  The definition written out. */
void nfo_cell_amax(const double *acc, const uint32_t *key, int64_t N, int64_t ncell, double *amax)
{
    for (int64_t c = 0; c < ncell; c++) amax[c] = 0.0;
    for (int64_t i = 0; i < N; i++) {
        double a = sqrt(acc[3 * i] * acc[3 * i] + acc[3 * i + 1] * acc[3 * i + 1] + acc[3 * i + 2] * acc[3 * i + 2]);
        if (a > amax[key[i]]) amax[key[i]] = a;
    }
}

/* Number of ordered (sink, source) pairs the near field requires, self pairs included
 * (reading c13): I = sum_c n_c * sum_{c' in N(c)} n_c'.  If sink_plane_lo <=
 * cx < sink_plane_hi restricts the sinks to a range of x-planes (slab streaming), pass it;
 * otherwise pass 0, K. */
int64_t nfo_interactions(const uint32_t *cell_count, int K, int R, int sink_plane_lo, int sink_plane_hi)
{
    int64_t total = 0;
#pragma omp parallel for reduction(+ : total) schedule(static)
    for (int cx = sink_plane_lo; cx < sink_plane_hi; cx++) {
        for (int cy = 0; cy < K; cy++)
            for (int cz = 0; cz < K; cz++) {
                int64_t n = cell_count[((int64_t)cx * K + cy) * K + cz];
                if (n == 0) continue;
                int64_t m = 0;
                for (int dx = -R; dx <= R; dx++)
                    for (int dy = -R; dy <= R; dy++)
                        for (int dz = -R; dz <= R; dz++) {
                            int sx = ((cx + dx) % K + K) % K;
                            int sy = ((cy + dy) % K + K) % K;
                            int sz = ((cz + dz) % K + K) % K;
                            m += cell_count[((int64_t)sx * K + sy) * K + sz];
                        }
                total += n * m;
            }
    }
    return total;
}

/* ---- kick and drift (Table 1 "Kick", "Drift") -----------------------------
 * The paper names the two leapfrog updates but prints no formula; the factors are the caller's
 * (DESIGN.md "Kick and drift").  float32 contract, written out: v1 = fmaf(a, kick, v) -- velocity
 * first -- then x1 = fmaf(v1, drift, x) with the NEW velocity, each a single rounding (C99 fmaf),
 * then one periodic wrap into [0, box): x1 >= box -> x1 - box; x1 < 0 -> x1 + box; a result that
 * is not below box after that (x1 + box rounded up to box) -> 0.  Elementwise over the 3N
 * coordinates, in place. */
void nfo_kick_drift(float *pos, float *vel, const float *acc, int64_t N, float kick, float drift, float box)
{
    for (int64_t i = 0; i < 3 * N; i++) {
        float v1 = fmaf(acc[i], kick, vel[i]);
        float x1 = fmaf(v1, drift, pos[i]);
        if (x1 >= box) x1 = x1 - box;
        else if (x1 < 0.0f) x1 = x1 + box;
        if (!(x1 < box)) x1 = 0.0f;
        vel[i] = v1;
        pos[i] = x1;
    }
}

/* ---- velocity reductions of the time-step criteria -----------------------
 * vrms[c] = sqrt(mean over the particles of cell c of |v|^2), 0 for empty cells (criterion 2 uses
 * "v_rms/a_max computed within each cell"); *vmax = the largest |v_axis| of any particle
 * (criterion 3: "the step size times the maximum velocity must be less than 80% of a cell width";
 * cells are axis-aligned, so the component is what crosses a face -- DESIGN.md reading c18).
 * vel: N x 3 float32 in input order; key: the particles' cell keys.  All in double. */
void nfo_cell_vrms(const float *vel, const uint32_t *key, int64_t N, int64_t ncell, double *vrms, double *vmax)
{
    int64_t *cnt = (int64_t *)calloc((size_t)ncell, sizeof(int64_t));
    double m = 0.0;
    for (int64_t c = 0; c < ncell; c++) vrms[c] = 0.0;
    for (int64_t i = 0; i < N; i++) {
        double vx = vel[3 * i], vy = vel[3 * i + 1], vz = vel[3 * i + 2];
        vrms[key[i]] += vx * vx + vy * vy + vz * vz;
        cnt[key[i]]++;
        if (fabs(vx) > m) m = fabs(vx);
        if (fabs(vy) > m) m = fabs(vy);
        if (fabs(vz) > m) m = fabs(vz);
    }
    for (int64_t c = 0; c < ncell; c++) vrms[c] = cnt[c] ? sqrt(vrms[c] / (double)cnt[c]) : 0.0;
    *vmax = m;
    free(cnt);
}

int nfo_max_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
