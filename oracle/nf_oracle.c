/*
 * nf_oracle.c -- float64 CPU oracle for the Abacus near-field direct sum.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may build, load or call it.
 * It shares no code, header, table or constant with the CUDA path under
 * paper_2110_11398_b200/csrc/, and neither includes the other.
 *
 * What it computes (citations are lines of /root/reference/PAPER.md):
 *   - the box of side L is a cubic lattice of CPD^3 cells                 (sec. 3.1)
 *   - the near field of a particle is "the force arising from nearby cells",
 *     set by the near-field radius R
 *   - every pair appears in exactly one of near/far field, periodic images
 *     are kept, "no approximation of close particle pairs as non-periodic"
 *   - R = 2 in production
 *   - "sourced by particles in neighboring cells out to radius R ... computed by a
 *     direct, O(N^2) summation with a compact spline softening kernel"
 *   - the softening "returns to exactly the 1/r^2 form at a scale mildly larger than
 *     the softening length"; lengths are Plummer-equivalent
 *
 * The method reaches exactly a plain definition (a finite direct sum), so the oracle
 * is that definition written out: for every sink, a triple loop over the (2R+1)^3
 * periodic neighbour cells and a loop over the particles of each, in float64.
 * No blocking, no fusion, no reordering.  The only parallel construct is an OpenMP
 * "parallel for" over sinks, used so the timed CPU baseline uses the host's cores.
 *
 * Readings where the paper is silent (restated in DESIGN.md):
 *   C1  "radius R" is a cube: all cells with max-norm offset <= R.
 *   C2  PAPER.md does not print the spline.  Reading used:
 *         F(r) = r * (10 - 15u + 6u^2) / eps_s^3   for u = r/eps_s < 1,
 *         F(r) = r / r^3                           otherwise,
 *       i.e. r^-3 replaced inside eps_s by its 2nd-order Taylor expansion about eps_s.
 *       PARITY UNPINNED by the paper for the choice of this spline (its stated
 *       properties are pinned in tests/test_oracle_pins.py).
 *   C3  eps is the Plummer-equivalent length; eps_s = 2.16 * eps.  PARITY UNPINNED
 *       by the paper for the literal 2.16 (10^(1/3) = 2.154 from equal central
 *       force gradient is the pinned property).
 *   C4  G = 1, all masses 1, no cosmological prefactors.
 *   C5  r = 0 (self term, exactly coincident particles) contributes 0.
 *   C6  cell index = floor((double)x * ((double)cpd / L)), clamped to cpd-1.
 *   C7  the periodic image of a source is the one implied by the CELL offset.
 *   C9  within a cell, particles are ordered by ascending input index.
 *   C10 cell id = (cx*cpd + cy)*cpd + cz  (x slowest = slab index, z fastest).
 *   C11 positions outside [0, L) or non-finite are an error, not wrapped.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define NFO_OK          0
#define NFO_ERR_ARG    -1
#define NFO_ERR_DOMAIN -2
#define NFO_ERR_NOMEM  -3

/* number of threads the parallel loops will use (reported by the bench) */
int nfo_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

static int nfo_check_args(int cpd, double L, double eps, int R)
{
    if (cpd < 1 || R < 0 || !(L > 0.0) || !(eps >= 0.0)) return NFO_ERR_ARG;
    if (cpd < 2 * R + 1) return NFO_ERR_ARG;                 /* reading C8 */
    if ((double)cpd * cpd * cpd >= 4294967296.0) return NFO_ERR_ARG;
    return NFO_OK;
}

/* Softened pair kernel K(r): acceleration on the sink is d * K(|d|).  Reading C2/C3/C5. */
double nfo_kernel(double r, double eps)
{
    double eps_s = 2.16 * eps;
    if (r == 0.0) return 0.0;
    if (eps_s == 0.0 || r >= eps_s) return 1.0 / (r * r * r);
    double u = r / eps_s;
    return (10.0 - 15.0 * u + 6.0 * u * u) / (eps_s * eps_s * eps_s);
}

/*
 * O1-O3: cell ids, counts, exclusive offsets, stable permutation.
 *   pos    [n][3] float32, input order          (host)
 *   cid    [n]    out: cell id per particle
 *   count  [C]    out: particles per cell, C = cpd^3
 *   offset [C+1]  out: exclusive prefix sum, offset[C] = n
 *   perm   [n]    out: sorted slot s holds input particle perm[s]
 */
int nfo_bin(const float *pos, int64_t n, int cpd, double L,
            uint32_t *cid, uint32_t *count, uint32_t *offset, uint32_t *perm)
{
    if (nfo_check_args(cpd, L, 0.0, 0) != NFO_OK || n < 0 || n >= 4294967296LL) return NFO_ERR_ARG;
    int64_t C = (int64_t)cpd * cpd * cpd;
    memset(count, 0, (size_t)C * sizeof(uint32_t));
    double scale = (double)cpd / L;
    for (int64_t i = 0; i < n; i++) {
        int c[3];
        for (int d = 0; d < 3; d++) {
            double x = (double)pos[3 * i + d];
            if (!isfinite(x) || x < 0.0 || x >= L) return NFO_ERR_DOMAIN;
            int k = (int)floor(x * scale);
            if (k >= cpd) k = cpd - 1;
            c[d] = k;
        }
        uint32_t id = (uint32_t)(((int64_t)c[0] * cpd + c[1]) * cpd + c[2]);
        cid[i] = id;
        count[id]++;
    }
    uint32_t run = 0;
    for (int64_t k = 0; k < C; k++) { offset[k] = run; run += count[k]; }
    offset[C] = run;
    uint32_t *next = (uint32_t *)malloc((size_t)(C > 0 ? C : 1) * sizeof(uint32_t));
    if (!next) return NFO_ERR_NOMEM;
    memcpy(next, offset, (size_t)C * sizeof(uint32_t));
    for (int64_t i = 0; i < n; i++) perm[next[cid[i]]++] = (uint32_t)i;   /* ascending i: stable */
    free(next);
    return NFO_OK;
}

/*
 * The comparison law of the paper: "the commonly used Plummer softening based on the potential
 * 1/sqrt(r^2 + eps^2), which converges only quadratically to the correct large-scale force law"
 * (sec. 5.2).  Force on the sink: d * (r^2 + eps^2)^(-3/2); eps is the Plummer length itself.
 * r = 0 contributes 0 (d = 0); eps = 0 is the Newtonian law with the r = 0 convention of reading C5.
 */
double nfo_kernel_plummer(double r, double eps)
{
    if (r == 0.0) return 0.0;
    double s = r * r + eps * eps;
    return 1.0 / (s * sqrt(s));
}

/* Acceleration on input particle i (float64), by the definition O4.  kind 0: spline (the method), 1: Plummer. */
static void nfo_one_sink(const float *pos, int cpd, double L, double eps, int R, int kind,
                         const uint32_t *cid, const uint32_t *offset, const uint32_t *perm,
                         int64_t i, double *a_out)
{
    uint32_t id = cid[i];
    int cz = (int)(id % (uint32_t)cpd);
    int cy = (int)((id / (uint32_t)cpd) % (uint32_t)cpd);
    int cx = (int)(id / ((uint32_t)cpd * (uint32_t)cpd));
    double xi = (double)pos[3 * i + 0], yi = (double)pos[3 * i + 1], zi = (double)pos[3 * i + 2];
    double ax = 0.0, ay = 0.0, az = 0.0;
    for (int ox = -R; ox <= R; ox++)
    for (int oy = -R; oy <= R; oy++)
    for (int oz = -R; oz <= R; oz++) {
        int sx = cx + ox, sy = cy + oy, sz = cz + oz;
        double wx = 0.0, wy = 0.0, wz = 0.0;
        if (sx < 0) { sx += cpd; wx = -1.0; } else if (sx >= cpd) { sx -= cpd; wx = 1.0; }
        if (sy < 0) { sy += cpd; wy = -1.0; } else if (sy >= cpd) { sy -= cpd; wy = 1.0; }
        if (sz < 0) { sz += cpd; wz = -1.0; } else if (sz >= cpd) { sz -= cpd; wz = 1.0; }
        int64_t c2 = ((int64_t)sx * cpd + sy) * cpd + sz;
        for (uint32_t t = offset[c2]; t < offset[c2 + 1]; t++) {
            int64_t j = perm[t];
            double dx = (double)pos[3 * j + 0] - xi + wx * L;
            double dy = (double)pos[3 * j + 1] - yi + wy * L;
            double dz = (double)pos[3 * j + 2] - zi + wz * L;
            double r2 = dx * dx + dy * dy + dz * dz;
            if (r2 == 0.0) continue;
            double K = kind == 1 ? nfo_kernel_plummer(sqrt(r2), eps) : nfo_kernel(sqrt(r2), eps);
            ax += dx * K; ay += dy * K; az += dz * K;
        }
    }
    a_out[0] = ax; a_out[1] = ay; a_out[2] = az;
}

/*
 * O4: accelerations of selected sinks.
 *   sinks  [m] input indices of the sinks to evaluate, or NULL for all (then m must be n)
 *   acc    [m][3] float64 out, row k belongs to sinks[k] (or to input particle k if sinks==NULL)
 * The binning arrays must come from nfo_bin on the same pos/cpd/L.
 */
int nfo_accel_kind(const float *pos, int64_t n, int cpd, double L, double eps, int R, int kind,
                   const uint32_t *cid, const uint32_t *offset, const uint32_t *perm,
                   const int64_t *sinks, int64_t m, double *acc)
{
    if (kind != 0 && kind != 1) return NFO_ERR_ARG;
    if (nfo_check_args(cpd, L, eps, R) != NFO_OK || n < 0 || m < 0) return NFO_ERR_ARG;
    if (!sinks && m != n) return NFO_ERR_ARG;
    int bad = 0;
#pragma omp parallel for schedule(dynamic, 64) reduction(|:bad)
    for (int64_t k = 0; k < m; k++) {
        int64_t i = sinks ? sinks[k] : k;
        if (i < 0 || i >= n) { bad |= 1; continue; }
        nfo_one_sink(pos, cpd, L, eps, R, kind, cid, offset, perm, i, acc + 3 * k);
    }
    return bad ? NFO_ERR_ARG : NFO_OK;
}

int nfo_accel(const float *pos, int64_t n, int cpd, double L, double eps, int R,
              const uint32_t *cid, const uint32_t *offset, const uint32_t *perm,
              const int64_t *sinks, int64_t m, double *acc)
{
    return nfo_accel_kind(pos, n, cpd, L, eps, R, 0, cid, offset, perm, sinks, m, acc);
}

/*
 * Variant with per-particle masses (the paper's particles all have one mass, PAPER.md:27,117,
 * so this is the same direct sum of PAPER.md:349 with the source mass written out instead of set to 1, reading C4):
 *   a_i = sum_j m_j d_ij K(|d_ij|),  G = 1, the sink's own mass does not enter.
 * Written out on its own (not by calling nfo_one_sink) so that the unit-mass oracle stays as it was pinned;
 * mass [n] float32 in input order, converted to float64 like the positions.
 */
int nfo_accel_mass(const float *pos, const float *mass, int64_t n, int cpd, double L, double eps, int R, int kind,
                   const uint32_t *cid, const uint32_t *offset, const uint32_t *perm,
                   const int64_t *sinks, int64_t m, double *acc)
{
    if (kind != 0 && kind != 1) return NFO_ERR_ARG;
    if (nfo_check_args(cpd, L, eps, R) != NFO_OK || n < 0 || m < 0 || !mass) return NFO_ERR_ARG;
    if (!sinks && m != n) return NFO_ERR_ARG;
    int bad = 0;
#pragma omp parallel for schedule(dynamic, 64) reduction(|:bad)
    for (int64_t k = 0; k < m; k++) {
        int64_t i = sinks ? sinks[k] : k;
        if (i < 0 || i >= n) { bad |= 1; continue; }
        uint32_t id = cid[i];
        int cz = (int)(id % (uint32_t)cpd);
        int cy = (int)((id / (uint32_t)cpd) % (uint32_t)cpd);
        int cx = (int)(id / ((uint32_t)cpd * (uint32_t)cpd));
        double xi = (double)pos[3 * i + 0], yi = (double)pos[3 * i + 1], zi = (double)pos[3 * i + 2];
        double ax = 0.0, ay = 0.0, az = 0.0;
        for (int ox = -R; ox <= R; ox++)
        for (int oy = -R; oy <= R; oy++)
        for (int oz = -R; oz <= R; oz++) {
            int sx = cx + ox, sy = cy + oy, sz = cz + oz;
            double wx = 0.0, wy = 0.0, wz = 0.0;
            if (sx < 0) { sx += cpd; wx = -1.0; } else if (sx >= cpd) { sx -= cpd; wx = 1.0; }
            if (sy < 0) { sy += cpd; wy = -1.0; } else if (sy >= cpd) { sy -= cpd; wy = 1.0; }
            if (sz < 0) { sz += cpd; wz = -1.0; } else if (sz >= cpd) { sz -= cpd; wz = 1.0; }
            int64_t c2 = ((int64_t)sx * cpd + sy) * cpd + sz;
            for (uint32_t t = offset[c2]; t < offset[c2 + 1]; t++) {
                int64_t j = perm[t];
                double dx = (double)pos[3 * j + 0] - xi + wx * L;
                double dy = (double)pos[3 * j + 1] - yi + wy * L;
                double dz = (double)pos[3 * j + 2] - zi + wz * L;
                double r2 = dx * dx + dy * dy + dz * dz;
                if (r2 == 0.0) continue;
                double K = kind == 1 ? nfo_kernel_plummer(sqrt(r2), eps) : nfo_kernel(sqrt(r2), eps);
                double mK = (double)mass[j] * K;
                ax += dx * mK; ay += dy * mK; az += dz * mK;
            }
        }
        acc[3 * k + 0] = ax; acc[3 * k + 1] = ay; acc[3 * k + 2] = az;
    }
    return bad ? NFO_ERR_ARG : NFO_OK;
}

/*
 * Kernel density estimate, computed by the paper "as part of the near-field force computation":
 * "a kernel density estimate around all particles, using a weighting of 1 - r^2/b^2, where b is chosen
 * to be 40% of the interparticle spacing" (sec. 3.3).
 *   rho_i = sum_j max(0, 1 - r_ij^2 / b^2),  j over the particles of the (2R+1)^3 stencil cells of i,
 * periodic image implied by the cell offset (reading C7).  Readings:
 *   D1  the particle itself is part of the sum (weight 1 at r = 0), as is any coincident particle;
 *   D2  b must not exceed R cell widths, so that the stencil holds every particle within b and the sum is
 *       the plain periodic estimate (b = 0.4 spacings is 0.1 cell widths at the paper's 67 per cell).
 *   sinks/m as in nfo_accel; rho [m] float64 out.
 */
int nfo_density(const float *pos, int64_t n, int cpd, double L, double b, int R,
                const uint32_t *cid, const uint32_t *offset, const uint32_t *perm,
                const int64_t *sinks, int64_t m, double *rho)
{
    if (nfo_check_args(cpd, L, 0.0, R) != NFO_OK || n < 0 || m < 0 || !(b > 0.0)) return NFO_ERR_ARG;
    if (b > R * (L / cpd)) return NFO_ERR_ARG;
    if (!sinks && m != n) return NFO_ERR_ARG;
    int bad = 0;
#pragma omp parallel for schedule(dynamic, 64) reduction(|:bad)
    for (int64_t k = 0; k < m; k++) {
        int64_t i = sinks ? sinks[k] : k;
        if (i < 0 || i >= n) { bad |= 1; continue; }
        uint32_t id = cid[i];
        int cz = (int)(id % (uint32_t)cpd);
        int cy = (int)((id / (uint32_t)cpd) % (uint32_t)cpd);
        int cx = (int)(id / ((uint32_t)cpd * (uint32_t)cpd));
        double xi = (double)pos[3 * i + 0], yi = (double)pos[3 * i + 1], zi = (double)pos[3 * i + 2];
        double sum = 0.0;
        for (int ox = -R; ox <= R; ox++)
        for (int oy = -R; oy <= R; oy++)
        for (int oz = -R; oz <= R; oz++) {
            int sx = cx + ox, sy = cy + oy, sz = cz + oz;
            double wx = 0.0, wy = 0.0, wz = 0.0;
            if (sx < 0) { sx += cpd; wx = -1.0; } else if (sx >= cpd) { sx -= cpd; wx = 1.0; }
            if (sy < 0) { sy += cpd; wy = -1.0; } else if (sy >= cpd) { sy -= cpd; wy = 1.0; }
            if (sz < 0) { sz += cpd; wz = -1.0; } else if (sz >= cpd) { sz -= cpd; wz = 1.0; }
            int64_t c2 = ((int64_t)sx * cpd + sy) * cpd + sz;
            for (uint32_t t = offset[c2]; t < offset[c2 + 1]; t++) {
                int64_t j = perm[t];
                double dx = (double)pos[3 * j + 0] - xi + wx * L;
                double dy = (double)pos[3 * j + 1] - yi + wy * L;
                double dz = (double)pos[3 * j + 2] - zi + wz * L;
                double w = 1.0 - (dx * dx + dy * dy + dz * dz) / (b * b);
                if (w > 0.0) sum += w;
            }
        }
        rho[k] = sum;
    }
    return bad ? NFO_ERR_ARG : NFO_OK;
}

/*
 * Uncancelled magnitude of the direct sum (test metric, reading C13 of SURVEY.md 8(c) / DESIGN.md 2):
 *   S_i = sum_j m_j |d_ij| K(|d_ij|),   j over the same (2R+1)^3 stencil particles as the acceleration
 * (the sum the near field evaluates; here every term enters with its NORM, so nothing cancels).
 * |a_i| <= S_i always (triangle inequality); S_i = |a_i| when the sink has one source.  A float32 evaluation of
 * the sum carries an error proportional to S_i, not to |a_i|: where the pair forces cancel (lattices, planes,
 * harmonic cores) BASELINE.json's ratio |a_gpu - a_ref| / |a_ref| is ill-conditioned and the tests bound the
 * error by a multiple of S_i instead.
 * Written out on its own, like nfo_density, so that the pinned acceleration loops stay untouched.
 *   mass  [n] float32 or NULL (unit masses);  kind 0: spline, 1: Plummer;  scale [m] float64 out.
 */
int nfo_force_scale(const float *pos, const float *mass, int64_t n, int cpd, double L, double eps, int R, int kind,
                    const uint32_t *cid, const uint32_t *offset, const uint32_t *perm,
                    const int64_t *sinks, int64_t m, double *scale)
{
    if (kind != 0 && kind != 1) return NFO_ERR_ARG;
    if (nfo_check_args(cpd, L, eps, R) != NFO_OK || n < 0 || m < 0) return NFO_ERR_ARG;
    if (!sinks && m != n) return NFO_ERR_ARG;
    int bad = 0;
#pragma omp parallel for schedule(dynamic, 64) reduction(|:bad)
    for (int64_t k = 0; k < m; k++) {
        int64_t i = sinks ? sinks[k] : k;
        if (i < 0 || i >= n) { bad |= 1; continue; }
        uint32_t id = cid[i];
        int cz = (int)(id % (uint32_t)cpd);
        int cy = (int)((id / (uint32_t)cpd) % (uint32_t)cpd);
        int cx = (int)(id / ((uint32_t)cpd * (uint32_t)cpd));
        double xi = (double)pos[3 * i + 0], yi = (double)pos[3 * i + 1], zi = (double)pos[3 * i + 2];
        double sum = 0.0;
        for (int ox = -R; ox <= R; ox++)
        for (int oy = -R; oy <= R; oy++)
        for (int oz = -R; oz <= R; oz++) {
            int sx = cx + ox, sy = cy + oy, sz = cz + oz;
            double wx = 0.0, wy = 0.0, wz = 0.0;
            if (sx < 0) { sx += cpd; wx = -1.0; } else if (sx >= cpd) { sx -= cpd; wx = 1.0; }
            if (sy < 0) { sy += cpd; wy = -1.0; } else if (sy >= cpd) { sy -= cpd; wy = 1.0; }
            if (sz < 0) { sz += cpd; wz = -1.0; } else if (sz >= cpd) { sz -= cpd; wz = 1.0; }
            int64_t c2 = ((int64_t)sx * cpd + sy) * cpd + sz;
            for (uint32_t t = offset[c2]; t < offset[c2 + 1]; t++) {
                int64_t j = perm[t];
                double dx = (double)pos[3 * j + 0] - xi + wx * L;
                double dy = (double)pos[3 * j + 1] - yi + wy * L;
                double dz = (double)pos[3 * j + 2] - zi + wz * L;
                double r2 = dx * dx + dy * dy + dz * dz;
                if (r2 == 0.0) continue;
                double r = sqrt(r2);
                double K = kind == 1 ? nfo_kernel_plummer(r, eps) : nfo_kernel(r, eps);
                double mj = mass ? fabs((double)mass[j]) : 1.0;
                sum += mj * r * K;
            }
        }
        scale[k] = sum;
    }
    return bad ? NFO_ERR_ARG : NFO_OK;
}

/*
 * Exact number of ordered pair evaluations of the definition (self pairs included):
 * I = sum_c count[c] * sum_{c' in stencil(c)} count[c'].
 */
int64_t nfo_interactions(const uint32_t *count, int cpd, int R)
{
    if (cpd < 2 * R + 1) return -1;
    int64_t total = 0;
    for (int cx = 0; cx < cpd; cx++)
    for (int cy = 0; cy < cpd; cy++)
    for (int cz = 0; cz < cpd; cz++) {
        int64_t nc = count[((int64_t)cx * cpd + cy) * cpd + cz];
        if (nc == 0) continue;
        int64_t src = 0;
        for (int ox = -R; ox <= R; ox++)
        for (int oy = -R; oy <= R; oy++)
        for (int oz = -R; oz <= R; oz++) {
            int sx = (cx + ox + cpd) % cpd, sy = (cy + oy + cpd) % cpd, sz = (cz + oz + cpd) % cpd;
            src += count[((int64_t)sx * cpd + sy) * cpd + sz];
        }
        total += nc * src;
    }
    return total;
}
