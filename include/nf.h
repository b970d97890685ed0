/*
 * nf.h -- C-ABI boundary of the B200-native near-field direct gravity sum.
 *
 * The operation is the near-field half of the Abacus force split (arXiv:2110.11398; line numbers
 * are /root/reference/PAPER.md):
 *   - the periodic box of side L is a lattice of CPD^3 cubic cells, a slab is the CPD^2 cells at
 *     fixed x                                                         (sec. 3.1)
 *   - the near field of a particle is "the force arising from nearby cells", set by the near-field
 *     radius R; every pair is in exactly one of near/far field and periodic images are kept
 *
 *   - it is "sourced by particles in neighboring cells out to radius R" and "computed by a direct,
 *     O(N^2) summation with a compact spline softening kernel"        (R = 2: 347)
 *   - the softening law "returns to exactly the 1/r^2 form at a scale mildly larger than the
 *     softening length", lengths quoted Plummer-equivalent
 *
 * Every sink particle i receives   a_i = sum_j d_ij K(|d_ij|),   d_ij = x_j - x_i + w L,
 * over all particles j of the (2R+1)^3 periodic cells around its own cell (w in {-1,0,+1}^3 is the
 * box shift implied by the wrap of the CELL index), with G = 1, unit masses and
 *   K(r) = r^-3                          for r >= eps_s  (or eps = 0),
 *   K(r) = (10 - 15u + 6u^2)/eps_s^3     for u = r/eps_s < 1,      eps_s = 2.16 eps,
 *   K(0) = 0 (self term and exactly coincident particles).
 * PAPER.md does not print the spline; this is the documented reading (readings C2/C3).
 *
 * All pointers named *_dev are DEVICE pointers valid on the plan's CUDA device; *_host are HOST
 * pointers (pinned memory makes the copies asynchronous).  The library never frees or keeps caller
 * memory past the call unless stated.  No torch types cross this boundary.
 *
 * A plan belongs to the CUDA device that is current at its first nf_bin; later calls switch to that device for
 * their duration if another one is current.
 *
 * Return values: 0 = NF_OK, negative = error; nf_last_error() gives a thread-local message.
 * There is NO CPU fallback: without a CUDA device every compute call fails with NF_ERR_CUDA.
 */
#ifndef NF_H
#define NF_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

#define NF_OK            0
#define NF_ERR_ARG      -1   /* null pointer, n < 0, n + 3 cpd^3 >= 2^32, cpd < 2R+1, cpd^3 >= 2^32, L <= 0, eps < 0, R < 0 or R > 127 */
#define NF_ERR_DOMAIN   -2   /* a coordinate is non-finite or outside [0, L)  (reported by nf_bin) */
#define NF_ERR_STATE    -3   /* nf_accel before a successful nf_bin */
#define NF_ERR_NOMEM    -4   /* device allocation failed / caller workspace too small */
#define NF_ERR_CUDA     -5   /* any CUDA runtime failure, including "no device" */

typedef struct nf_plan nf_plan;     /* opaque; owns every internal device buffer */

typedef struct nf_stats {
    long long n;               /* particles last binned */
    long long cells;           /* cpd^3 */
    long long padded_slots;    /* slots of the cell-padded source arrays (>= n) */
    long long units;           /* work units (sink chunks) of the last binning */
    long long interactions;    /* exact ordered pair evaluations of the definition, self pairs included:
                                  sum_c n_c * sum_{c' in stencil(c)} n_c'  */
    float ms_bin;              /* device time of the last nf_bin   (CUDA events on the plan's stream) */
    float ms_accel;            /* device time of the last nf_accel (direct-sum kernel incl. fused scatter) */
    int   sm_count;            /* multiprocessors of the device */
    int   clock_khz;           /* cudaDevAttrClockRate (max SM clock) */
    int   accel_grid;          /* CTAs of the persistent direct-sum launch */
    int   accel_block;         /* threads per CTA */
    int   kernel_launches_bin; /* kernels launched by one nf_bin */
    int   kernel_launches_accel; /* kernels launched by one nf_accel: 1, or 2 when the binning holds dense and sparse windows */
    int   rebin_path;          /* last nf_rebin: 1 = incremental merge, 2 = sorted from scratch; 0 = none since nf_bin */
    long long rebin_movers;    /* particles that changed cell in the last incremental nf_rebin (-1: not counted) */
} nf_stats;

/*
 * nf_plan_create -- the problem statement of PAPER.md:337-349.
 *   cpd  cells per dimension (>= 2R+1 so that no cell appears twice in a stencil)
 *   L    box side (> 0), positions live in [0, L)
 *   eps  Plummer-equivalent softening length (>= 0; 0 = pure Newtonian)
 *   R    near-field radius in cells (>= 0 with cpd >= 2R+1; 2 in production; at most 127)
 * Host-only: validates, precomputes constants, allocates nothing of size O(n).
 * Returns NULL on error (see nf_last_error()).
 */
nf_plan *nf_plan_create(int cpd, double L, double eps, int R);

/*
 * nf_bin -- steps S1-S5: cell ids, per-cell counts, exclusive offsets, STABLE counting sort
 * (within a cell: ascending input index), cell-sorted source arrays, work-unit list.
 *   pos_dev  [n][3] float32, input order, device memory, read only
 *   n        0 <= n, n + 3 cpd^3 < 2^32.  n = 0 is a valid no-op.
 *            (the cell-padded source arrays are indexed with 32 bits: every non-empty cell adds up to 3 pad slots)
 * May be called repeatedly; each call invalidates the previous binning.  Enqueues on the plan's
 * stream and, as its LAST action, performs one 16-byte device-to-host read (the domain-error flag and the
 * number of work units) and therefore synchronises that stream before returning: the binning is complete
 * on return, nothing of it is still pending on the stream.
 * Errors: NF_ERR_ARG, NF_ERR_DOMAIN (no partial result promised), NF_ERR_NOMEM, NF_ERR_CUDA.
 */
int nf_bin(nf_plan *plan, const float *pos_dev, long long n);

/*
 * nf_rebin -- steps S1-S5 again for the SAME particles after they moved: the paper's pipeline
 * "reorders particles into their new cells" after every drift ("moving particles to their new cells",
 * PAPER.md:353; Table 6 "Finish" / "Merge New Particles"), and a drift is much shorter than a cell,
 * so nearly every particle stays where it was.
 *   pos_dev  [n][3] float32, device memory, the new positions in the SAME input order and with the same n as the
 *            last nf_bin / nf_rebin of this plan.
 * The result is by definition what nf_bin(plan, pos_dev, n) gives -- cell ids, counts, offsets and the stable
 * permutation are bit-identical to it (and to the oracle), hence so are the accelerations -- but no radix pass
 * runs: one pass over the input order finds the particles that changed cell, one pass over the old sorted order
 * merges each cell's stayers with its arrivals and rewrites the source arrays.  Falls back to the full sort when more
 * than a quarter of the particles moved, when ranking the arrivals (sum over the cells of arrivals^2) would cost more
 * than 16 n comparisons, or when the previous call saw more than 1/16 of the particles move (nf_stats.rebin_path / rebin_movers say which path ran).
 * Like nf_bin it resets the plan to unit masses and synchronises the stream once, as its last action.
 * Errors: NF_ERR_STATE (no valid binning: call nf_bin first, also after nf_set_sink_slabs / "window" / "heavy_first"),
 *         NF_ERR_ARG, NF_ERR_DOMAIN (the binning is invalid afterwards), NF_ERR_CUDA.
 */
int nf_rebin(nf_plan *plan, const float *pos_dev);

/*
 * nf_accel -- steps S6-S7: the direct sum over the cell stencil and the scatter to input order.
 *   acc_dev  [n][3] float32, device memory, OVERWRITTEN (not accumulated) with a_i for the
 *            positions last binned, row i = input particle i.
 * Asynchronous: returns after enqueueing on the plan's stream.
 * Errors: NF_ERR_STATE (no successful nf_bin), NF_ERR_ARG, NF_ERR_CUDA.
 */
int nf_accel(nf_plan *plan, float *acc_dev);

/*
 * nf_accel_density -- nf_accel plus the kernel density estimate the paper computes "as part of the near-field
 * force computation with minimal computational burden" (sec. 3.3), in the same pass:
 *   rho_i = sum_j max(0, 1 - r_ij^2 / b^2),   j over the same (2R+1)^3 stencil particles, the particle itself
 *   included (weight 1; reading D1).  The paper takes b = 0.4 interparticle spacings.
 *   acc_dev  [n][3] float32, as nf_accel
 *   rho_dev  [n] float32, device memory, OVERWRITTEN, row i = input particle i
 *   b        kernel radius in box units, 0 < b <= R cell widths (then the stencil holds every particle
 *            within b and the sum is the plain periodic estimate; reading D2), else NF_ERR_ARG
 * Asynchronous like nf_accel.  Errors: NF_ERR_STATE, NF_ERR_ARG, NF_ERR_CUDA.
 */
int nf_accel_density(nf_plan *plan, float *acc_dev, float *rho_dev, double b);

/*
 * nf_accel_kick -- nf_accel with the two steps that follow the near field in the paper's pipeline fused into
 * the kernel epilogue (no second pass over the accelerations):
 *   - the leapfrog kick  v_i += a_i * dt                      ("kicks the particle velocities")
 *   - the per-cell maximum particle acceleration max_i |a_i|  (the denominator of the timestep criterion,
 *     "the per-cell maximum particle acceleration")
 *   acc_dev        [n][3] float32 or NULL (accelerations not stored)
 *   vel_dev        [n][3] float32, input order, UPDATED IN PLACE with one float32 FMA per component, or NULL
 *   dt             kick factor (finite)
 *   amax_cell_dev  [cpd^3] float32, OVERWRITTEN: max over the particles of the cell of the Euclidean norm of the
 *                  float32 acceleration, 0 for an empty cell; or NULL
 * At least one of the three pointers must be non-NULL.  Asynchronous like nf_accel.
 * Errors: NF_ERR_STATE, NF_ERR_ARG, NF_ERR_CUDA.
 */
int nf_accel_kick(nf_plan *plan, float *acc_dev, float *vel_dev, double dt, float *amax_cell_dev);

/*
 * nf_set_masses -- per-particle SOURCE masses for the particles last binned (variant of SURVEY.md 8(f) NEXT 4;
 * the paper's particles all carry one mass, which is the default m = 1):
 *   a_i = sum_j m_j d_ij K(|d_ij|),  G = 1; the sink's own mass does not enter.
 * Every later nf_accel / nf_accel_density / nf_accel_kick on this binning uses them (the density estimate of
 * nf_accel_density stays the unweighted count-based sum of PAPER.md:387).
 *   mass_dev  DEVICE pointer, [n] float32 in input order (finite), read during the call's kernel, not retained;
 *             NULL = back to unit masses.
 * The masses are gathered into a plan-owned device array in the internal source layout (4 bytes per padded slot,
 * allocated at the first call, outside any lent workspace).  nf_bin resets the plan to unit masses: call
 * nf_set_masses after every nf_bin.  Asynchronous on the plan's stream.
 * Errors: NF_ERR_STATE (no binning), NF_ERR_NOMEM, NF_ERR_CUDA.
 */
int nf_set_masses(nf_plan *plan, const float *mass_dev);

/* nf_destroy -- frees everything the plan allocated (never a caller workspace).  NULL-safe. */
void nf_destroy(nf_plan *plan);

/*
 * nf_set_sink_slabs -- x-slab domain decomposition (the paper's parallel method: each node owns a contiguous
 * range of slabs and needs "R loaded slabs on either side").  After this call only the
 * particles whose cell has x index in {x_first, ..., x_first + n_slabs - 1} (mod cpd) are SINKS; every binned
 * particle is still a source.  A rank bins its own slabs plus the R halo slabs of each x-neighbour and gets
 * exactly the accelerations a whole-box plan would give its particles (bit for bit when both plans use the same
 * "window" and "quad_vote" options; the automatic window of small problems depends on the number of owned columns); rows of acc that belong to particles
 * outside the sink slabs are not written, and nf_stats.interactions counts the owned sinks only.
 * Takes effect at the next nf_bin (it invalidates the current binning).  Default: all slabs.
 * Errors: NF_ERR_ARG unless 0 <= x_first < cpd and 1 <= n_slabs <= cpd.
 */
int nf_set_sink_slabs(nf_plan *plan, int x_first, int n_slabs);

/*
 * The other half of the slab decomposition (one process per GPU; the transfers themselves are the caller's point-to-point
 * sends over NCCL / NVLink): everything that looks at particle data runs on the device, by the cell rule of nf_bin.
 *
 * nf_slab_histogram -- particles per x-slab of a position array.
 *   pos_dev [n][3] device, hist_host [cpd] host (OVERWRITTEN).  Synchronises.  NF_ERR_DOMAIN as nf_bin.
 * nf_slab_select -- stable compaction: the particles of pos_dev whose cell has x index in {x_first, ..., x_first +
 *   n_slabs - 1} (mod cpd), in their original relative order (so that the receiver's stable cell sort reproduces the
 *   order a whole-box plan sees inside every cell), copied device to device into
 *   out_dev [cap][3]; idx_out_dev [cap] (or NULL) receives their input indices (for payloads that travel with the
 *   particle, e.g. masses); *m_host = number selected.  NF_ERR_NOMEM if it exceeds cap.  Synchronises.
 * nf_get_slab_cost -- cost_host [cpd] (OVERWRITTEN): pair interactions per x-slab of the last binning, sum over the slab's
 *   cells of count x (particles in the cell's stencil) -- the scheduler's exact cost; 0 for slabs outside the sink slabs
 *   (their cells are sources only on this rank: the owner reports them).  Ranks add their vectors (all-reduce) to get the
 *   whole box.  Synchronises.  NF_ERR_STATE without a binning.
 * nf_slab_partition -- HOST ONLY, no device, no plan: world contiguous slab ranges first[r], count[r] covering 0..cpd-1,
 *   every rank at least one slab, minimising the largest range cost ("contiguous x-slabs balanced by
 *   interaction cost"; "a contiguous span of slabs").  cost == NULL: equal costs.  NF_ERR_ARG unless
 *   1 <= world <= cpd and every cost is finite and >= 0.
 */
int nf_slab_histogram(nf_plan *plan, const float *pos_dev, long long n, long long *hist_host);
/*
 * nf_slab_histogram_static -- nf_slab_histogram (same arguments, same result, same errors) for callers that cannot call
 * cudaMalloc: code under CUDA graph capture, tight serving loops, harnesses that forbid allocation.  The scratch of the
 * kernel (per-slab counters and the domain flag) is a file-scope device array of the library, not an allocation: the
 * call makes no cudaMalloc / cudaFree, calls no allocating library routine and uses no host heap.
 *   limit    cpd <= 1024 (the array holds 1024 slab counters + the flag: 8 KB, held by every GPU that loads the library
 *            until the process exits); a larger cpd -> NF_ERR_ARG with a message naming the limit.
 *   sharing  every call on a device uses the ONE array, which keeps the previous call's contents (the call clears what it
 *            uses first).  Calls that overlap on the same GPU -- other streams, other plans, other host threads -- RACE:
 *            the caller serialises them.  nf_slab_histogram has no such restriction.
 * Runs on the plan's device if it has one (bound at its first nf_bin), else on the current device.  Synchronises.
 */
int nf_slab_histogram_static(nf_plan *plan, const float *pos_dev, long long n, long long *hist_host);
int nf_slab_select(nf_plan *plan, const float *pos_dev, long long n, int x_first, int n_slabs, float *out_dev,
                   unsigned *idx_out_dev, long long cap, long long *m_host);
int nf_get_slab_cost(nf_plan *plan, double *cost_host);
int nf_slab_partition(const double *cost, int cpd, int world, int *first, int *count);

/* ---- host-buffer entry points (end-to-end path: the copies are part of the call) ------------- */

/* Copies pos_host [n][3] to a plan-owned device buffer (async if pinned) and runs nf_bin on it. */
int nf_bin_host(nf_plan *plan, const float *pos_host, long long n);
/* Runs nf_accel into a plan-owned device buffer and copies it to acc_host [n][3]; synchronises.
 * With restricted sink slabs the rows of particles outside them come back as zeros. */
int nf_accel_host(nf_plan *plan, float *acc_host);

/* ---- supporting exports (harness, tests; not part of the paper's problem statement) ---------- */

const char *nf_last_error(void);

/* CUDA stream (cudaStream_t as void*) all later calls enqueue on.  Default: the legacy stream 0. */
int nf_set_stream(nf_plan *plan, void *cuda_stream);

/* Bytes of workspace nf_bin needs for n particles on this plan. */
size_t nf_workspace_bytes(const nf_plan *plan, long long n);
/* Lend a device workspace (borrowed until nf_destroy or the next nf_set_workspace; 256-byte aligned).
 * Without it the plan allocates (and grows) its own with cudaMalloc. */
int nf_set_workspace(nf_plan *plan, void *dev_ptr, size_t bytes);

/*
 * Borrowed DEVICE pointers into the last binning (valid until the next nf_bin / nf_destroy):
 *   cell_id [n]      cell of input particle i, id = (cx*cpd + cy)*cpd + cz (x slowest, z fastest)
 *   count   [cpd^3]  particles per cell
 *   offset  [cpd^3+1] exclusive prefix sum of count, offset[cpd^3] = n
 *   perm    [n]      sorted slot s holds input particle perm[s]
 * Any output pointer may be NULL.
 */
int nf_get_binning(const nf_plan *plan, const unsigned **cell_id, const unsigned **count,
                   const unsigned **offset, const unsigned **perm);

/*
 * Borrowed DEVICE pointers to the internal source layout (for layout tests only):
 *   poff [cpd^3+1]  first slot of each cell in the padded arrays (cells padded to multiples of 4)
 *   x, y, z [padded_slots]  cell-corner-relative coordinates times *scale (a power of two);
 *                   pad slots hold a far-away dummy.
 */
int nf_get_layout(const nf_plan *plan, const unsigned **poff, const float **x, const float **y,
                  const float **z, double *scale);

/* Fills *out; synchronises the plan's stream (event times and the interaction count live on the device). */
int nf_get_stats(nf_plan *plan, nf_stats *out);

/*
 * Tuning knobs (integers).  Unknown key -> NF_ERR_ARG.
 *   "variant"      0 = packed f32x2 pair kernel (default), 1 = scalar FP32 kernel
 *   "fastpath"     1 = skip the spline on cells that cannot hold a pair closer than eps_s (default), 0 = never skip
 *   "heavy_first"  1 = schedule costly work units first (default), 0 = natural cell order
 *   "ctas_per_sm"  0 = occupancy-derived (default), >0 = cap
 *   "window"       sink slots (the particles of a z-column, every cell rounded up to an even count) per work unit: a multiple of 32 up to 512, rounded
 *                  up to whole sink groups of 64, or 0 (default) = 512, except for problems whose units would not fill the
 *                  grid of persistent CTAs, which get the longest of 512, 256, 128 and 64 that does.
 *                  The warps of a CTA that a short window leaves without sinks share the unit's stages.
 *                  Shorter windows give a small problem more work units, but every unit streams its whole stencil
 *                  again.  With 512-slot windows the remainder of a column is cut into 256 / 128 / fewer slots (sink
 *                  groups that divide the consumer warps).  Accelerations are bit-identical between plans only for equal
 *                  windows.  Takes effect at the next nf_bin.
 *   "flat_below"   windows whose cells hold fewer sink slots on average than this walk a lane's stencil run in one flat loop
 *                  (sparse cells: DESIGN.md 7); default 22, 0 = never.  Takes effect at the next nf_bin.  nf_bin sorts these
 *                  windows behind all the others and nf_accel runs them as a second launch (kernel_launches_accel = 2).
 *   "quad_vote"    -1 (default) = the direct-kernel instance that votes once per four sources in the spline-capable loop is
 *                  launched when the fullest cell of the binning holds more than 4096 particles (the halo cells of clustered
 *                  inputs spend nearly all their pairs in that loop); 0 = never, 1 = always.  The two instances agree to one ulp of the
 *                  pairs that sit within 0.1 % of eps_s (the spline's min is taken wherever the vote fired): bit-identical
 *                  results between plans (slab ranks against the whole box) need the same explicit setting.  The fused
 *                  nf_accel_density pass votes on max(eps_s, b): its forces agree with nf_accel's to that one ulp, not bit
 *                  for bit; nf_accel_kick runs the loops of nf_accel and returns its bits.
 *   "softening"    0 = the compact spline of the method (default); 1 = Plummer softening, force
 *                  d (r^2 + eps^2)^(-3/2) with eps the plan's length: the law the paper compares against
 *                  ("converges only quadratically to the correct large-scale force law")
 */
int nf_set_option(nf_plan *plan, const char *key, long long value);

#ifdef __cplusplus
}
#endif
#endif /* NF_H */
