// nf_direct.cu -- steps S6-S7 of the hot path: the near-field direct sum and the scatter to input order.
//
//   a_i = sum_j d_ij K(|d_ij|),  j over the particles of the (2R+1)^3 periodic cells around the cell of i
//   (sec. 3.1: "sourced by particles in neighboring cells out to radius R ... direct,
//   O(N^2) summation with a compact spline softening kernel"; periodic images kept).
//
// Design (sm_100a):
//   * a work unit is a WINDOW of <= kChunk consecutive sink slots of one z-column (cells are z-fastest, so a
//     column is one contiguous run of the sorted order; sink slots number its particles with every cell rounded
//     up to an even count): every warp holds 64 slots whatever the cell occupancy -- only the last slot of a
//     cell with an odd count is an idle sink;
//   * persistent CTAs, one producer warp + kConsumerWarps consumer warps, units pulled from an atomic
//     counter in heavy-first order;
//   * for each of the (2R+1)^2 neighbour columns the producer streams the z-run of cells [z0-R, z1+R] that the
//     window's sinks need into shared memory with TMA 1-D bulk copies (cp.async.bulk + mbarrier complete_tx)
//     through a kStages-deep ring, with a table of the cells (pieces) of the run;
//   * a lane whose sink sits in cell zc walks ITS OWN 2R+1 pieces zc-R..zc+R of the run (per-lane shared-memory
//     pointer), so no lane ever evaluates a pair outside its stencil; the order pairs the lanes of a warp by
//     source cell (step s takes the cell j with (j - z0 + R) mod (2R+1) == s), so lanes of neighbouring sink
//     cells read the same piece except in the one step where their stencils do not overlap;
//   * TWO sinks per lane in registers, an aligned pair of sink slots (always the same cell), packed as the two
//     halves of f32x2 operands; sources are read as LDS.128 of 4 x, 4 y, 4 z and every source is a scalar
//     broadcast against the sink pair: FADD2 / FFMA2 / FMUL2 (fma.rn.f32x2) do two interactions each, one
//     MUFU.RSQ per interaction.  Every shared-memory load, every piece lookup and every loop instruction of a
//     lane serves twice the interactions it would with one sink per lane;
//   * coordinates are cell-corner relative (exact); the periodic wrap and the cell-to-cell shift are one
//     constant per (sink cell, source cell) subtracted from the sink once per piece -- nothing periodic
//     in the pair loop;
//   * the spline is evaluated only where it can matter: a source cell whose nearest face is farther than eps_s
//     from every sink of the warp takes the pure Newtonian body; the others take min(r^2) over each quad of
//     sources, vote, and evaluate (C r + B) r + A and the min only when some lane has a pair inside eps_s;
//   * sparse windows (flat units: their cells hold few slots) walk a lane's 2R+1 stencil cells of a column as ONE run of
//     quads (flat loop); when the whole z-run of a neighbour column fits a stage the producer copies the run's padded
//     offsets instead of building a per-cell table (lean stage).  nf_bin sorts the flat units behind all the others and
//     nf_accel runs the two groups as two launches: the stepped units in instances compiled without the flat loop;
//   * FP32 FMA chain per (sink, source cell), partials added in FP64 in shared memory (two-level accumulation);
//   * the epilogue writes acc[perm[s]] directly (S7 fused, no sorted acceleration buffer).
#include "nf_internal.h"

#include <type_traits>

namespace nf {

enum { kFlagBegin = 1, kFlagEnd = 2, kFlagTerm = 4 };

struct __align__(16) Piece {   // one source cell (or a part of one) of the stage's z-run
    int    sm_off;             // first slot in the stage buffers (multiple of 4)
    int    nslots;             // multiple of 4; 0 = empty cell
    double czs;                // (corner_z(source cell) + box wrap) * scale
};

struct __align__(16) StageDesc {
    int      flags;
    int      npieces;
    int      j0;               // cell of pieces[0], as an index relative to z0 - R
    int      soft_mode;        // 2: spline body everywhere; 1: for |oz| <= 1 (column with |ox|,|oy| <= 1); 0: never
    float    dx, dy;           // sink shift of this column: d = x_src - (x_sink - shift), scaled units
    uint32_t v0;               // unit: first sink slot (voff numbering: cells rounded up to even counts)
    uint32_t nv;               //       sink slots
    uint32_t z0, z1;           //       first / last sink cell (z index)
    uint32_t colbase;          //       col * cpd
    int      oxy;              // column offset: (ox + 128) | (oy + 128) << 8
    int      flat;             // unit flag: sparse window, flat loop
    // lean stage (flat units whose whole z-run of a neighbour column fits the stage): no piece table; the stage carries the raw
    // padded offsets of the run's cells (ps[], bulk-copied like the coordinates) in up to three segments -- cells below the
    // periodic face, inside the box, above it -- and every consumer derives slots and z corners from them
    int      lean;
    struct Seg { int ncell, slot0, ps0, jw0; double wz; } seg[3];   // cells, first stage slot, index of the first cell's offset in ps[], wrapped z of the first cell, box wrap
    Piece    pieces[kMaxPieces];
};
constexpr int kLeanCells = 256;                 // longest z-run (cells) a lean stage describes
constexpr int kPsMax = kLeanCells + 3 * 8;      // + alignment slack of the three slices (each starts 16-byte aligned in global memory)

// Pipeline depth: 5 stages for the three coordinate arrays (the consumer warps of a split unit work on different
// stages at the same time: config 1 0.157 -> 0.137 ms against 3 stages, the large configs unchanged); the mass kernels
// stage a fourth array and keep 3 so that three CTAs still fit an SM.
template <int NARR> struct StagesFor { static constexpr int value = NARR == 3 ? kStages : kStagesMass; };

template <int NARR, bool FLAT = true>  // NARR 3: x, y, z;  4: + the source masses (nf_set_masses).  FLAT = false: no flat loop, no tables for it
struct __align__(128) SharedStorageT {
    static constexpr int kStages = StagesFor<NARR>::value;
    float buf[kStages][NARR][kTile + 4];  // x, y, z (, m) of the staged sources + one quad of dummies (never overwritten)
    StageDesc desc[kStages];
    unsigned long long full[kStages];
    unsigned long long empty[kStages];
    double quadz[FLAT ? kStages : 1][FLAT ? kTile / 4 + 1 : 1];   // flat loop: z corner (scaled, with box wrap) of the cell of every quad of the stage
    __align__(16) uint32_t ps[FLAT ? kStages : 1][FLAT ? kPsMax : 4];   // lean stages: padded offsets (poff) of the cells of the run, as copied
    double acc[kConsumerWarps][8][32];    // FP64 sums of every warp's sinks (x, y, z of sink A, x, y, z of sink B, rho A, rho B): kept here, not in
                                          // 16 registers per lane; the warps of a split unit add theirs up from here at the end of the unit
};

// ---- PTX helpers: mbarrier + TMA 1-D bulk copy ---------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(void *bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ bool mbar_try(uint32_t a, uint32_t parity)
{
    uint32_t ok;
    asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                 : "=r"(ok) : "r"(a), "r"(parity) : "memory");
    return ok != 0;
}
// A warp that has to wait (the producer running ahead, a consumer warp without sinks in a ragged window) backs
// off with nanosleep: a spinning try_wait loop costs issue slots that the working warps of the sub-partition need.
__device__ __forceinline__ void mbar_wait(void *bar, uint32_t parity)
{
    const uint32_t a = smem_u32(bar);
    if (mbar_try(a, parity)) return;
    while (!mbar_try(a, parity)) __nanosleep(kWaitSleepNs);
}
__device__ __forceinline__ void mbar_arrive(void *bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(void *bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void tma_load_1d(void *dst_smem, const void *src_gmem, uint32_t bytes, void *bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(dst_smem)), "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ float rsqrt_approx(float x)
{
    float y;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// ---- pair bodies -------------------------------------------------------------------------------
// A lane holds two sinks A, B; every float2 below is (value for A, value for B).  PACKED: f32x2 instructions (FADD2, FFMA2,
// FMUL2: two interactions each; a source coordinate enters as a scalar broadcast operand); otherwise scalar FP32 (variant 1).
constexpr float kSelfR2 = 2e-36f;   // r^2 of a pair at r = 0 is the offset `tiny` = 1e-36 (spline law); nothing else is below this
struct SoftCoef { float A, B, C, tiny, soft_r2, nb2, dens_r2; int plummer; float near_r2; };   // density: nb2 = -1/b^2, dens_r2 = b^2 (+ tiny, margin); near_r2 = max(soft_r2, dens_r2)

template <bool PACKED> __device__ __forceinline__ float2 add2(const float2 a, const float2 b)
{
    return PACKED ? __fadd2_rn(a, b) : make_float2(a.x + b.x, a.y + b.y);
}
template <bool PACKED> __device__ __forceinline__ float2 mul2(const float2 a, const float2 b)
{
    return PACKED ? __fmul2_rn(a, b) : make_float2(a.x * b.x, a.y * b.y);
}
template <bool PACKED> __device__ __forceinline__ float2 fma2(const float2 a, const float2 b, const float2 c)
{
    return PACKED ? __ffma2_rn(a, b, c) : make_float2(fmaf(a.x, b.x, c.x), fmaf(a.y, b.y, c.y));
}
__device__ __forceinline__ float2 bc(const float v) { return make_float2(v, v); }

// FP32 partial sums of one (sink pair, stage)
struct Partial {
    float2 x, y, z, rho;
    __device__ __forceinline__ void clear() { x = y = z = rho = make_float2(0.f, 0.f); }
};

constexpr uint32_t kFull = 0xffffffffu;
// -DNF_DEBUG_BOUNDS: every table index of the sparse path is checked on the device and a violation traps (the launch then
// fails with an error instead of reading or writing out of bounds); compute-sanitizer is not available on every box
#ifdef NF_DEBUG_BOUNDS
#define NF_CHECK(cond) do { if (!(cond)) __trap(); } while (0)
#else
#define NF_CHECK(cond) do { } while (0)
#endif
#ifndef NF_UNROLL_SOFT
#define NF_UNROLL_SOFT 2
#endif
constexpr int kUnrollSoft = NF_UNROLL_SOFT;   // unrolling of the spline-capable piece loop
#ifndef NF_UNROLL_TAIL
#define NF_UNROLL_TAIL 8
#endif
constexpr int kUnrollTail = NF_UNROLL_TAIL;   // unrolling of the ragged tail (whole pieces run there when a lane of the warp has none)
#ifndef NF_UNROLL_TAIL_QV
#define NF_UNROLL_TAIL_QV 4
#endif
constexpr int kUnrollTailQV = NF_UNROLL_TAIL_QV;   // the same in the quad-vote instances: the choice moves ptxas's register allocation of the
                                                   // whole kernel, and with 4 the quad-vote loop has 20 same-bank operand pairs instead of 25
                                                   // (config 4 +0.3 %, config 5 +0.5 %; the other instances lose 0.15 % with it)
constexpr int kTileAlloc = kTile + 4;          // + one quad of dummies that every lane may read past its piece
#ifndef NF_DENS_QV
#define NF_DENS_QV 1                           // fused density loops: one combined vote per quad (1) or two votes per two sources (0)
#endif
#ifndef NF_FLUSH_QUADS
#define NF_FLUSH_QUADS 6
#endif
constexpr int kFlushQuads = NF_FLUSH_QUADS;    // a step of at least this many quads ends its FP32 chain (24 sources per sink)

// Newtonian part of one source against the sink pair: d, r^2, 1/r and k = r^-3.  11 FP32-pipe lane-operations per
// interaction (3 add, 6 fma, 2 mul) plus one MUFU.RSQ; n = shift - sink, so d = source + n.
template <bool PACKED>
__device__ __forceinline__ void src_head(const float xs, const float ys, const float zs, const float2 nx, const float2 ny, const float2 nz,
                                         const float tiny, float2 &dx, float2 &dy, float2 &dz, float2 &r2, float2 &ri, float2 &k)
{
    dx = add2<PACKED>(nx, bc(xs)); dy = add2<PACKED>(ny, bc(ys)); dz = add2<PACKED>(nz, bc(zs));
    r2 = fma2<PACKED>(dz, dz, bc(tiny));
    r2 = fma2<PACKED>(dy, dy, r2);
    r2 = fma2<PACKED>(dx, dx, r2);
    ri.x = rsqrt_approx(r2.x);
    ri.y = rsqrt_approx(r2.y);
    k = mul2<PACKED>(mul2<PACKED>(ri, ri), ri);
}
template <bool PACKED>
__device__ __forceinline__ void src_spline(const float2 r2, const float2 ri, const SoftCoef &c, float2 &k)
{
    const float2 r = mul2<PACKED>(r2, ri);                  // t = (C r + B) r + A
    float2 t = fma2<PACKED>(r, bc(c.C), bc(c.B));
    t = fma2<PACKED>(t, r, bc(c.A));
    k.x = fminf(k.x, t.x);
    k.y = fminf(k.y, t.y);
}
// kernel density weights: rho += max(0, 1 - r^2/b^2)
template <bool PACKED>
__device__ __forceinline__ void src_density(const float2 r2, const SoftCoef &c, float2 &rho)
{
    float2 w = fma2<PACKED>(r2, bc(c.nb2), bc(1.0f));
    w.x = fmaxf(w.x, 0.0f);
    w.y = fmaxf(w.y, 0.0f);
    rho = add2<PACKED>(rho, w);
}
template <bool PACKED>
__device__ __forceinline__ void src_accum(const float2 k, const float2 dx, const float2 dy, const float2 dz, Partial &f)
{
    f.x = fma2<PACKED>(k, dx, f.x); f.y = fma2<PACKED>(k, dy, f.y); f.z = fma2<PACKED>(k, dz, f.z);
}

// Two sources against the sink pair of every lane (four interactions).  MODE 0: Newtonian.  MODE >= 1: exactly the lanes of
// `mask` must call it together (warp vote inside): the spline is evaluated only when some lane of the warp has one of these
// pairs inside eps_s -- a fraction of a percent of the calls at production density; otherwise the body is the Newtonian one
// plus three FMNMX, a vote and a branch.  MODE 2 adds the kernel density weight the same way (sources within b).
template <bool PACKED, int MODE, bool MASS>
__device__ __forceinline__ void duo(const float xa, const float ya, const float za, const float ma, const float xb, const float yb,
                                    const float zb, const float mb, const float2 nx, const float2 ny, const float2 nz,
                                    const SoftCoef &c, Partial &f, const uint32_t mask)
{
    float2 dxa, dya, dza, r2a, ria, ka, dxb, dyb, dzb, r2b, rib, kb;
    src_head<PACKED>(xa, ya, za, nx, ny, nz, c.tiny, dxa, dya, dza, r2a, ria, ka);
    src_head<PACKED>(xb, yb, zb, nx, ny, nz, c.tiny, dxb, dyb, dzb, r2b, rib, kb);
    if (MODE >= 1) {
        const float m = fminf(fminf(r2a.x, r2a.y), fminf(r2b.x, r2b.y));
        if (__any_sync(mask, m < c.soft_r2)) {
            src_spline<PACKED>(r2a, ria, c, ka);
            src_spline<PACKED>(r2b, rib, c, kb);
            if (MASS) {
                // with masses the capped k of the self pair (r^2 = tiny; the cap is 3e38 for eps = 0) times m could overflow to
                // inf and inf * 0 = NaN: the self pair and exactly coincident particles are dropped explicitly (reading C5)
                ka.x = r2a.x > kSelfR2 ? ka.x : 0.f; ka.y = r2a.y > kSelfR2 ? ka.y : 0.f;
                kb.x = r2b.x > kSelfR2 ? kb.x : 0.f; kb.y = r2b.y > kSelfR2 ? kb.y : 0.f;
            }
        }
        if (MODE == 2 && __any_sync(mask, m < c.dens_r2)) {     // some lane has one of these sources inside b
            if (c.plummer) {                  // the Plummer option puts eps^2 into r2: the weight needs the bare r^2
                r2a = fma2<PACKED>(dxa, dxa, fma2<PACKED>(dya, dya, mul2<PACKED>(dza, dza)));
                r2b = fma2<PACKED>(dxb, dxb, fma2<PACKED>(dyb, dyb, mul2<PACKED>(dzb, dzb)));
            }
            src_density<PACKED>(r2a, c, f.rho);
            src_density<PACKED>(r2b, c, f.rho);
        }
    }
    if (MASS) { ka = mul2<PACKED>(ka, bc(ma)); kb = mul2<PACKED>(kb, bc(mb)); }
    src_accum<PACKED>(ka, dxa, dya, dza, f);
    src_accum<PACKED>(kb, dxb, dyb, dzb, f);
}

// Four sources (one LDS.128 of x, y, z[, m]) against the sink pair of every lane: eight interactions.
template <bool PACKED, int MODE, bool MASS, bool QV = false>
__device__ __forceinline__ void quad(const float4 X, const float4 Y, const float4 Z, const float4 M, const float2 nx, const float2 ny,
                                     const float2 nz, const SoftCoef &c, Partial &f, const uint32_t mask = kFull)
{
    if (MODE == 0 || !QV) {
        duo<PACKED, MODE, MASS>(X.x, Y.x, Z.x, M.x, X.y, Y.y, Z.y, M.y, nx, ny, nz, c, f, mask);
        duo<PACKED, MODE, MASS>(X.z, Y.z, Z.z, M.z, X.w, Y.w, Z.w, M.w, nx, ny, nz, c, f, mask);
        return;
    }
    // QV (the kernel instance launched when the binning holds heavy cells, nf_api: the halo cells of the clustered configs
    // spend nearly all their interactions in this loop): ONE vote per quad.  The common path keeps d and k of the four
    // sources; the rare branch forms r^2 and 1/r again (the same bits: same inputs, same instructions).  Config 4 +2.9 %,
    // config 3 -1.2 % (16 bytes of spills at the 96-register budget) -- hence a separate instance, not the default.
    const float xs[4] = {X.x, X.y, X.z, X.w}, ys[4] = {Y.x, Y.y, Y.z, Y.w}, zs[4] = {Z.x, Z.y, Z.z, Z.w}, ms[4] = {M.x, M.y, M.z, M.w};
    float2 dx[4], dy[4], dz[4], k[4];
    float m = 3.0e38f;
#pragma unroll
    for (int j = 0; j < 4; j++) {
        float2 r2, ri;
        src_head<PACKED>(xs[j], ys[j], zs[j], nx, ny, nz, c.tiny, dx[j], dy[j], dz[j], r2, ri, k[j]);
        m = fminf(m, fminf(r2.x, r2.y));
    }
    // MODE 2 (the fused density pass): ONE vote for "some lane has one of these sources inside eps_s OR inside b"; the kernel
    // density radius b is several eps_s, so the spline gets a second vote inside the (already rare) branch.  Config 3: +7.2 %
    // -> +4.9 % over the force-only pass; config 4: +31 % -> +25 % (in the halo cores every quad has a source within b: an
    // unconditional density body for heavy pieces, without vote and recompute, measured the same 25 % -- the weight itself,
    // one FFMA2, two FMNMX and one FADD2 per two interactions, is what costs there).
    if (__any_sync(mask, m < (MODE == 2 ? c.near_r2 : c.soft_r2))) {
        const bool spline = MODE == 1 || __any_sync(mask, m < c.soft_r2);
#pragma unroll
        for (int j = 0; j < 4; j++) {
            float2 r2 = fma2<PACKED>(dz[j], dz[j], bc(c.tiny));
            r2 = fma2<PACKED>(dy[j], dy[j], r2);
            r2 = fma2<PACKED>(dx[j], dx[j], r2);
            if (spline) {
                float2 ri;
                ri.x = rsqrt_approx(r2.x);
                ri.y = rsqrt_approx(r2.y);
                src_spline<PACKED>(r2, ri, c, k[j]);
                if (MASS) {                    // see duo: drop r = 0 before the mass multiplies the capped k
                    k[j].x = r2.x > kSelfR2 ? k[j].x : 0.f;
                    k[j].y = r2.y > kSelfR2 ? k[j].y : 0.f;
                }
            }
            if (MODE == 2) {                   // weights of the lanes without a source inside b are exactly 0
                if (c.plummer)                 // the Plummer option puts eps^2 into r2: the weight needs the bare r^2
                    r2 = fma2<PACKED>(dx[j], dx[j], fma2<PACKED>(dy[j], dy[j], mul2<PACKED>(dz[j], dz[j])));
                src_density<PACKED>(r2, c, f.rho);
            }
        }
    }
#pragma unroll
    for (int j = 0; j < 4; j++) {
        if (MASS) k[j] = mul2<PACKED>(k[j], bc(ms[j]));
        src_accum<PACKED>(k[j], dx[j], dy[j], dz[j], f);
    }
}

// One step of a warp: every lane runs over ITS piece (n4 quads at px).  `live` = lanes that have a piece in this
// stage (n4 > 0), nmin / nmax = smallest / largest n4 among them.  The first loop is uniform over the live lanes;
// in the ragged tail a lane that has run out of sources is predicated off (Newtonian body) or reads the stage's
// dummy quad (coordinates 2^55: contributes exactly 0 to the force and to the density) so that the warp stays
// converged for the vote of the spline body.
template <bool PACKED, int MODE, bool MASS, bool QV = false, int UT = kUnrollTail>
__device__ __forceinline__ void piece_loop(const float4 *__restrict__ px, const int n4, const int nmin, const int nmax,
                                           const uint32_t live, const int jdummy, const float2 nx, const float2 ny, const float2 nz,
                                           const SoftCoef &c, Partial &f)
{
    const float4 *__restrict__ py = px + kTileAlloc / 4;
    const float4 *__restrict__ pz = py + kTileAlloc / 4;
    const float4 *__restrict__ pm = pz + kTileAlloc / 4;        // masses: read only with MASS
    const float4 one = make_float4(1.f, 1.f, 1.f, 1.f);
    if (n4 > 0) {
        if (MODE == 0) {
#pragma unroll 2
            for (int j = 0; j < nmin; j++) quad<PACKED, MODE, MASS>(px[j], py[j], pz[j], MASS ? pm[j] : one, nx, ny, nz, c, f);
        } else {
#pragma unroll kUnrollSoft
            for (int j = 0; j < nmin; j++) quad<PACKED, MODE, MASS, QV>(px[j], py[j], pz[j], MASS ? pm[j] : one, nx, ny, nz, c, f, live);
        }
    }
    __syncwarp();
#pragma unroll UT
    for (int j = nmin; j < nmax; j++) {
        if (MODE >= 1) {                              // the body votes: keep the warp converged
            const int jj = j < n4 ? j : jdummy;
            quad<PACKED, MODE, MASS, QV>(px[jj], py[jj], pz[jj], MASS ? pm[jj] : one, nx, ny, nz, c, f);
        } else if (j < n4) {
            quad<PACKED, MODE, MASS>(px[j], py[j], pz[j], MASS ? pm[j] : one, nx, ny, nz, c, f);
        }
    }
}

// ---- the kernel --------------------------------------------------------------------------------
struct AccelArgs {
    Consts k;
    const float *x, *y, *z;          // padded SoA sources (= sinks)
    const float *m;                  // padded SoA source masses (MASS kernels only; pads hold 0)
    const uint32_t *poff, *voff, *offset, *perm;
    const Unit *units;
    uint32_t n_units;
    uint32_t *counter;               // atomic work counter (zeroed before launch)
    float *acc;                      // [n][3] input order
    int fastpath;
    // kernel density estimate (DENS kernels only)
    float *rho;                      // [n] input order
    float dens_nb2;                  // -1 / b^2, scaled units
    float dens_thr2;                 // (b + rounding margin)^2: closer faces can hold a pair inside b
    int dens_mode;                   // 1: b < cell width, only touching cells whose face is within b; 2: every cell
    // fused epilogue: leapfrog kick and per-cell maximum acceleration; any may be NULL
    float *vel;                      // [n][3] input order, v += a * dt in float32
    float dt;
    uint32_t *amax;                  // [cpd^3] bit patterns of non-negative floats, zeroed before launch
};

// The producer warp runs in lockstep (all control flow is warp-uniform); lane 0 alone touches the
// descriptors, the barriers and the TMA unit.
template <int NARR, bool FLAT>
__device__ __forceinline__ void producer(const AccelArgs &a, SharedStorageT<NARR, FLAT> &sm, const int lane)
{
    constexpr int kStages = StagesFor<NARR>::value;
    const Consts &k = a.k;
    const int cpd = k.cpd, R = k.R;
    const bool lead = lane == 0;
    int stage = 0;
    uint32_t phase = 0;
    bool open = false, sealed = false;
    int fill = 0, np = 0, sflags = 0;
    uint32_t cp_g = 0, cp_s = 0, cp_n = 0;        // pending merged copy: global slot, stage slot, slots
    auto flush_copy = [&]() {
        if (cp_n && lead) {
            tma_load_1d(&sm.buf[stage][0][cp_s], a.x + cp_g, cp_n * 4u, &sm.full[stage]);
            tma_load_1d(&sm.buf[stage][1][cp_s], a.y + cp_g, cp_n * 4u, &sm.full[stage]);
            tma_load_1d(&sm.buf[stage][2][cp_s], a.z + cp_g, cp_n * 4u, &sm.full[stage]);
            if (NARR == 4) tma_load_1d(&sm.buf[stage][NARR - 1][cp_s], a.m + cp_g, cp_n * 4u, &sm.full[stage]);
        }
        cp_n = 0;
    };
    uint32_t extra_tx = 0;                        // bytes of the offset slices of a lean stage
    auto commit = [&](int extra) {
        flush_copy();
        __syncwarp();          // the table entries written by the other lanes are ordered before lane 0's releasing arrive
        if (lead) {
            sm.desc[stage].flags = sflags | extra;
            sm.desc[stage].npieces = np;
            mbar_arrive_expect_tx(&sm.full[stage], (uint32_t)fill * (4u * NARR) + extra_tx);
        }
        extra_tx = 0;
        if (++stage == kStages) { stage = 0; phase ^= 1u; }
        open = false; sealed = false;
    };
    for (;;) {
        uint32_t u = 0;
        if (lead) u = atomicAdd(a.counter, 1u);
        u = __shfl_sync(kFull, u, 0);
        if (u >= a.n_units) break;
        const Unit un = a.units[u];
        const int cx = (int)(un.col / (uint32_t)cpd), cy = (int)(un.col % (uint32_t)cpd);
        const int z0 = un.z0, z1 = un.z1;
        const double ocx = (double)(float)((double)cx * k.cell_w), ocy = (double)(float)((double)cy * k.cell_w);
        const int jlo = z0 - R, jhi = z1 + R;     // unwrapped z-run every neighbour column contributes
        bool first = true;
        for (int ox = -R; ox <= R; ox++) {
            int jx = cx + ox; double wx = 0.0;
            if (jx < 0) { jx += cpd; wx = -k.L; } else if (jx >= cpd) { jx -= cpd; wx = k.L; }
            const float Dx = (float)(((double)(float)((double)jx * k.cell_w) + wx - ocx) * k.scale);
            for (int oy = -R; oy <= R; oy++) {
                int jy = cy + oy; double wy = 0.0;
                if (jy < 0) { jy += cpd; wy = -k.L; } else if (jy >= cpd) { jy -= cpd; wy = k.L; }
                const float Dy = (float)(((double)(float)((double)jy * k.cell_w) + wy - ocy) * k.scale);
                const uint32_t row = ((uint32_t)jx * cpd + jy) * cpd;
                const int soft_mode = k.plummer ? 0 : !(k.fast_ok && a.fastpath) ? 2 : ((ox >= -1 && ox <= 1 && oy >= -1 && oy <= 1) ? 1 : 0);
                // Lean stage.  In a sparse window (flat unit) the per-cell table below costs the producer ~300 instructions per
                // 32 cells, one warp against eight: at 4-8 particles per cell the consumers waited for it 15-27 % of the time.
                // When the whole run of this column fits one stage the producer only reads the offsets at the ends of its (up
                // to three) segments, copies the coordinates and the offsets themselves, and the consumers do the rest.
                if (FLAT && un.flat && jhi - jlo + 1 <= kLeanCells) {
                    const int sa[3] = {jlo, max(jlo, 0), max(jlo, cpd)}, sb[3] = {min(jhi, -1), min(jhi, cpd - 1), jhi};
                    const int sh[3] = {cpd, 0, -cpd};
                    uint32_t v = 0;
                    {   // lanes 0..5 read the offsets at the two ends of the three segments (selects, no indexed local arrays)
                        const int q = lane >> 1;
                        const int qa = q == 0 ? sa[0] : (q == 1 ? sa[1] : sa[2]), qb = q == 0 ? sb[0] : (q == 1 ? sb[1] : sb[2]);
                        const int qs = q == 0 ? sh[0] : (q == 1 ? sh[1] : sh[2]);
                        if (lane < 6 && qa <= qb) v = __ldg(a.poff + row + (uint32_t)((lane & 1 ? qb + 1 : qa) + qs));
                    }
                    uint32_t g0[3], len[3];
#pragma unroll
                    for (int q = 0; q < 3; q++) {
                        g0[q] = __shfl_sync(kFull, v, 2 * q);
                        len[q] = __shfl_sync(kFull, v, 2 * q + 1) - g0[q];
                    }
                    const uint32_t total = len[0] + len[1] + len[2];
                    if (total == 0) continue;                     // an empty run never opens a stage
                    if (total <= (uint32_t)kTile) {
                        if (open) commit(0);
                        mbar_wait(&sm.empty[stage], phase ^ 1u);
                        open = true; sealed = true; fill = (int)total; np = jhi - jlo + 1;
                        sflags = first ? kFlagBegin : 0;
                        first = false;
                        if (lead) {
                            StageDesc &d = sm.desc[stage];
                            d.j0 = 0; d.soft_mode = soft_mode; d.dx = Dx; d.dy = Dy; d.oxy = (ox + 128) | ((oy + 128) << 8);
                            d.v0 = un.v0; d.nv = un.nv; d.flat = un.flat; d.z0 = (uint32_t)z0; d.z1 = (uint32_t)z1;
                            d.colbase = un.col * (uint32_t)cpd;
                            d.lean = 1;
                            uint32_t slot = 0, psb = 0;
#pragma unroll
                            for (int q = 0; q < 3; q++) {
                                const int nc = sa[q] <= sb[q] ? sb[q] - sa[q] + 1 : 0;
                                d.seg[q].ncell = nc; d.seg[q].slot0 = (int)slot; d.seg[q].jw0 = sa[q] + sh[q];
                                d.seg[q].wz = q == 0 ? -k.L : (q == 2 ? k.L : 0.0);
                                d.seg[q].ps0 = 0;
                                if (nc > 0) {
                                    const uint32_t e0 = row + (uint32_t)(sa[q] + sh[q]), al = e0 & ~3u;      // aligned superset of [e0, e0 + nc]
                                    const uint32_t cnt = (e0 + (uint32_t)nc + 1u - al + 3u) & ~3u;
                                    d.seg[q].ps0 = (int)(psb + (e0 - al));
                                    NF_CHECK(psb + cnt <= (uint32_t)kPsMax && slot + len[q] <= (uint32_t)kTile && (len[q] & 3u) == 0 && (g0[q] & 3u) == 0);
                                    tma_load_1d(&sm.ps[stage][psb], a.poff + al, cnt * 4u, &sm.full[stage]);
                                    extra_tx += cnt * 4u;
                                    psb += cnt;
                                    if (len[q]) {
                                        tma_load_1d(&sm.buf[stage][0][slot], a.x + g0[q], len[q] * 4u, &sm.full[stage]);
                                        tma_load_1d(&sm.buf[stage][1][slot], a.y + g0[q], len[q] * 4u, &sm.full[stage]);
                                        tma_load_1d(&sm.buf[stage][2][slot], a.z + g0[q], len[q] * 4u, &sm.full[stage]);
                                        if (NARR == 4) tma_load_1d(&sm.buf[stage][NARR - 1][slot], a.m + g0[q], len[q] * 4u, &sm.full[stage]);
                                    }
                                    slot += len[q];
                                }
                            }
                        }
                        continue;
                    }
                }
                for (int jb = jlo; jb <= jhi; jb += 32) {
                    // the warp fetches the padded offsets of up to 32 cells of the run at once
                    const int jl = jb + lane;
                    int jwl = jl;
                    if (jwl < 0) jwl += cpd; else if (jwl >= cpd) jwl -= cpd;
                    uint32_t P0 = 0, P1 = 0;
                    if (jl <= jhi) { P0 = __ldg(a.poff + row + jwl); P1 = __ldg(a.poff + row + jwl + 1); }
                    const int cnt = min(32, jhi - jb + 1);
                    // Fast path (all lanes in parallel): when the whole chunk of <= 32 cells fits the open stage, or a
                    // fresh one, every lane writes the table entry of its cell and lane 0 issues one merged copy per
                    // contiguous segment (a segment ends at the periodic z face).  Sparse regions, where a window of
                    // sinks spans dozens of cells, would otherwise serialise on the per-cell loop below.
                    {
                        const uint32_t nsl = lane < cnt ? P1 - P0 : 0u;
                        uint32_t inc = nsl;
#pragma unroll
                        for (int o = 1; o < 32; o <<= 1) {
                            const uint32_t up = __shfl_up_sync(kFull, inc, o);
                            if (lane >= o) inc += up;
                        }
                        const uint32_t total = __shfl_sync(kFull, inc, 31);
                        const uint32_t off = inc - nsl;
                        if (total == 0 && (!open || sealed)) continue;          // empty cells never open a stage
                        const bool can_append = open && !sealed && fill + (int)total <= kTile && np + cnt <= kMaxPieces;
                        const bool can_open = (int)total <= kTile && cnt <= kMaxPieces;
                        if (can_append || can_open) {
                            if (!can_append) {
                                if (open) commit(0);
                                mbar_wait(&sm.empty[stage], phase ^ 1u);
                                open = true; fill = 0; np = 0;
                                sflags = first ? kFlagBegin : 0;
                                first = false;
                                if (lead) {
                                    StageDesc &d = sm.desc[stage];
                                    d.lean = 0;
                                    d.j0 = jb - jlo; d.soft_mode = soft_mode; d.dx = Dx; d.dy = Dy; d.oxy = (ox + 128) | ((oy + 128) << 8);
                                    d.v0 = un.v0; d.nv = un.nv; d.flat = un.flat; d.z0 = (uint32_t)z0; d.z1 = (uint32_t)z1;
                                    d.colbase = un.col * (uint32_t)cpd;
                                }
                            }
                            if (lane < cnt) {
                                const double wz = jl < 0 ? -k.L : (jl >= cpd ? k.L : 0.0);
                                Piece &pc = sm.desc[stage].pieces[np + lane];
                                pc.sm_off = fill + (int)off; pc.nslots = (int)nsl;
                                pc.czs = ((double)(float)((double)jwl * k.cell_w) + wz) * k.scale;
                            }
                            uint32_t starts = __ballot_sync(kFull, lane < cnt && (lane == 0 || jwl == 0));
                            while (starts) {
                                const int b = __ffs(starts) - 1;
                                starts &= starts - 1;
                                const int e = starts ? __ffs(starts) - 1 : cnt;     // segment = lanes [b, e)
                                const uint32_t g0 = __shfl_sync(kFull, P0, b);
                                const uint32_t o0 = __shfl_sync(kFull, off, b);
                                const uint32_t len = __shfl_sync(kFull, inc, e - 1) - o0;
                                if (len == 0) continue;
                                const uint32_t s0 = (uint32_t)fill + o0;
                                if (cp_n && cp_g + cp_n == g0 && cp_s + cp_n == s0) cp_n += len;
                                else { flush_copy(); cp_g = g0; cp_s = s0; cp_n = len; }
                            }
                            np += cnt; fill += (int)total;
                            continue;
                        }
                    }
                    for (int q = 0; q < cnt; q++) {
                        uint32_t p0 = __shfl_sync(kFull, P0, q);
                        const uint32_t p1 = __shfl_sync(kFull, P1, q);
                        const bool empty = p0 == p1;
                        if (empty && (!open || sealed || fill == kTile || np == kMaxPieces)) continue;   // empty cells never open a stage
                        const int j = jb + q;
                        int jw = j; double wz = 0.0;
                        if (jw < 0) { jw += cpd; wz = -k.L; } else if (jw >= cpd) { jw -= cpd; wz = k.L; }
                        const double czs = ((double)(float)((double)jw * k.cell_w) + wz) * k.scale;
                        do {
                            if (open && (sealed || fill == kTile || np == kMaxPieces)) commit(0);
                            if (!open) {
                                if (empty) break;
                                mbar_wait(&sm.empty[stage], phase ^ 1u);
                                open = true; fill = 0; np = 0;
                                sflags = first ? kFlagBegin : 0;
                                first = false;
                                if (lead) {
                                    StageDesc &d = sm.desc[stage];
                                    d.lean = 0;
                                    d.j0 = j - jlo; d.soft_mode = soft_mode; d.dx = Dx; d.dy = Dy; d.oxy = (ox + 128) | ((oy + 128) << 8);
                                    d.v0 = un.v0; d.nv = un.nv; d.flat = un.flat; d.z0 = (uint32_t)z0; d.z1 = (uint32_t)z1;
                                    d.colbase = un.col * (uint32_t)cpd;
                                }
                            }
                            const uint32_t t = min(p1 - p0, (uint32_t)(kTile - fill));
                            if (lead) {
                                Piece &pc = sm.desc[stage].pieces[np];
                                pc.sm_off = fill; pc.nslots = (int)t; pc.czs = czs;
                            }
                            np++;
                            if (cp_n && cp_g + cp_n == p0 && cp_s + cp_n == (uint32_t)fill) cp_n += t;
                            else { flush_copy(); cp_g = p0; cp_s = (uint32_t)fill; cp_n = t; }
                            fill += (int)t; p0 += t;
                        } while (p0 < p1);
                    }
                }
                if (open) sealed = true;          // one neighbour column per stage
            }
        }
        commit(kFlagEnd);                         // the sinks' own cells are never empty, so a stage is open
    }
    mbar_wait(&sm.empty[stage], phase ^ 1u);
    if (lead) {
        sm.desc[stage].flags = kFlagTerm;
        sm.desc[stage].npieces = 0;
        mbar_arrive_expect_tx(&sm.full[stage], 0u);
    }
}

template <bool PACKED, bool DENS, bool EPI, bool MASS, bool QV, bool FLAT>
__device__ __forceinline__ void consumer(const AccelArgs &a, SharedStorageT<MASS ? 4 : 3, FLAT> &sm, const int warp, const int lane)
{
    const float dens_r2 = DENS ? -1.001f / a.dens_nb2 + a.k.tiny : 0.f;
    const SoftCoef coef = {a.k.A, a.k.B, a.k.C, a.k.tiny, a.k.soft_r2, DENS ? a.dens_nb2 : 0.f, dens_r2, a.k.plummer,
                           fmaxf(a.k.soft_r2, dens_r2)};
    constexpr int kStages = StagesFor<MASS ? 4 : 3>::value;
    const int nsteps = 2 * a.k.R + 1, R = a.k.R;
    int stage = 0;
    uint32_t phase = 0;
    float2 xi = make_float2(0.f, 0.f), yi = xi, zi = xi;         // the lane's two sinks (A, B): an aligned pair of sink slots
    double oczs = 0.0;
    double (*acc64)[32] = sm.acc[warp];                          // [8][32]: this warp's FP64 sums, one column per lane
    // A window of fewer than kChunk slots leaves consumer warps without sinks.  They take a share of the unit's stages
    // instead: with ng = ceil(np / 64) sink groups the kConsumerWarps / ng warps {g, g + ng, g + 2 ng, ...} hold the SAME
    // 64 slots, warp q of them computes the stages q, q + nsplit, ... of the unit, and the partial sums meet in shared
    // memory at the end of the unit, added in the fixed order q = 0, 1, ... (deterministic).  Small problems, whose units
    // cannot fill the machine, and the ragged last window of every column then keep all warps of the CTA busy.
    // one register: nsplit (warps sharing the sinks) | ng << 8 (sink groups) | q << 16 (this warp's share) | countdown << 24
    static_assert(kConsumerWarps <= 255, "the split state packs warp counts into 8-bit fields");
    uint32_t sp = 1u | ((uint32_t)kConsumerWarps << 8);
    int zrel = 0, zoff = 0;             // the lane's sink cell relative to z0, and zrel mod (2R+1)
    uint32_t slot = 0;                  // sorted slot (perm index) of sink A; sink B is slot + 1
    uint32_t cell = 0;                  // the lane's sink cell id
    uint32_t nreal = 0;                 // how many of the lane's two slots hold a particle to write (0, 1, 2)
    bool warp_on = false;
    for (;;) {
        mbar_wait(&sm.full[stage], phase);
        const StageDesc &d = sm.desc[stage];
        const int flags = d.flags;
        if (flags & kFlagTerm) break;
        if (flags & kFlagBegin) {
            const uint32_t nv = d.nv;
            const int ng = (int)((nv + (uint32_t)kGroup - 1u) / (uint32_t)kGroup), nsplit = kConsumerWarps / ng, q = warp / ng;
            sp = (uint32_t)nsplit | ((uint32_t)ng << 8) | ((uint32_t)q << 16) | ((uint32_t)q << 24);   // first stage of warp q: stage q
            const uint32_t kk = (uint32_t)((warp - q * ng) * kGroup + 2 * lane);
            warp_on = q < nsplit;
            const bool act = warp_on && kk < nv;
#pragma unroll
            for (int c = 0; c < (DENS ? 8 : 6); c++) acc64[c][lane] = 0.0;
            nreal = 0;
            if (warp_on) {
                // lanes past the end of a ragged window shadow its last pair (same pieces, nothing written)
                const uint32_t v = d.v0 + (act ? kk : nv - 2u);
                const uint32_t *vof = a.voff + d.colbase;
                int lo = (int)d.z0, hi = (int)d.z1;
                while (lo < hi) {                      // last cell of [z0, z1] whose first sink slot is <= v
                    const int mid = (lo + hi + 1) >> 1;
                    if (__ldg(vof + mid) <= v) lo = mid; else hi = mid - 1;
                }
                zrel = lo - (int)d.z0;
                zoff = zrel % nsteps;
                cell = d.colbase + (uint32_t)lo;
                const uint32_t r = v - __ldg(vof + lo);                                   // even: the pair (r, r + 1) of the cell
                const uint32_t o0 = __ldg(a.offset + cell), o1 = __ldg(a.offset + cell + 1);
                const uint32_t p = __ldg(a.poff + cell) + r;                              // its place in the padded source arrays
                slot = o0 + r;                                                            // r < count: the first of the pair is a particle
                if (act) nreal = slot + 1u < o1 ? 2u : 1u;
                const float2 X2 = __ldg(reinterpret_cast<const float2 *>(a.x + p));      // p is even: 8-byte aligned
                const float2 Y2 = __ldg(reinterpret_cast<const float2 *>(a.y + p));
                const float2 Z2 = __ldg(reinterpret_cast<const float2 *>(a.z + p));
                xi = X2; yi = Y2; zi = Z2;
                // the pad slot after the last particle of a cell with an odd count takes that particle's coordinates: it then
                // computes the same (unwritten) sums and never widens the gap tests below (a pad sits at 2^55)
                if (slot + 1u >= o1) { xi.y = xi.x; yi.y = yi.x; zi.y = zi.x; }
                oczs = (double)(float)((double)lo * a.k.cell_w) * a.k.scale;
            }
        }
        const bool mine = warp_on && (sp >> 24) == 0u;                  // countdown to this warp's next stage
        sp = mine ? (sp | (((sp & 255u) - 1u) << 24)) : sp - (1u << 24);
        if (mine) {
            const int np = d.npieces, soft_mode = d.soft_mode;
            const float2 nx = make_float2(d.dx - xi.x, d.dx - xi.y), ny = make_float2(d.dy - yi.x, d.dy - yi.y);   // shift - sink
            const int ibase = zrel - d.j0;
            // squared gap between the sinks and the neighbour column (0 for the own column): a cell whose
            // nearest face is farther than eps_s cannot hold a pair that needs the spline.  The smaller of the two sinks' gaps.
            float gxy2 = 0.f;
            const int ox = (d.oxy & 255) - 128, oy = (d.oxy >> 8) - 128;
            const bool near_col = ox >= -1 && ox <= 1 && oy >= -1 && oy <= 1;
            const bool gap_dens = DENS && a.dens_mode == 1 && near_col;
            if (soft_mode == 1 || gap_dens) {
                const float gx = ox < 0 ? fminf(xi.x, xi.y) : (ox > 0 ? a.k.w_scaled - fmaxf(xi.x, xi.y) : 0.f);
                const float gy = oy < 0 ? fminf(yi.x, yi.y) : (oy > 0 ? a.k.w_scaled - fmaxf(yi.x, yi.y) : 0.f);
                gxy2 = fmaf(gx, gx, gy * gy);
            }
            const float4 *sbase = reinterpret_cast<const float4 *>(&sm.buf[stage][0][0]);
            Partial f;
            f.clear();
            bool pending = true;
            auto flush = [&]() {                                        // FP32 chain -> FP64 sums (shared memory), chain restarts
                acc64[0][lane] += (double)f.x.x; acc64[1][lane] += (double)f.y.x; acc64[2][lane] += (double)f.z.x;
                acc64[3][lane] += (double)f.x.y; acc64[4][lane] += (double)f.y.y; acc64[5][lane] += (double)f.z.y;
                if (DENS) { acc64[6][lane] += (double)f.rho.x; acc64[7][lane] += (double)f.rho.y; }
                f.clear();
            };
            if (FLAT && d.flat) {
                // Sparse window (a handful of slots per cell): a lane's 2R+1 stencil cells of this column are ONE contiguous
                // run of quads in the stage, walked in one loop with the cell's z corner looked up per quad -- instead of
                // 2R+1 steps that each pay ~50 instructions of piece lookup and warp reductions for one or two quads.  Lanes
                // of different sink cells read different quads (a few shared-memory wavefronts per load, far from a limit
                // here).  Every consumer warp fills the table of the stages it works on (same values: no ordering needed).
                double *qz = sm.quadz[stage];
                const int ilo = max(ibase, 0), ihi = min(ibase + 2 * R, np - 1);
                // the warp fills the table for the cells ITS lanes walk (the runs of 64 consecutive sink slots: a dozen cells), not for
                // the whole stage; the warps write the same values where their ranges overlap
                const int wlo = __reduce_min_sync(kFull, ilo <= ihi ? ilo : np), whi = __reduce_max_sync(kFull, ilo <= ihi ? ihi : -1);   // none: [np, -1] is empty
                int qlo = 0, cnt = 0;
                if (d.lean) {
                    // cell i of the run: its segment, its slots from the copied offsets, its z corner by the producer's formula
                    const uint32_t *ps = sm.ps[stage];
                    const int n0 = d.seg[0].ncell, n01 = n0 + d.seg[1].ncell;
                    auto cell = [&](const int i, int &slot, int &nsl, double &czs) {
                        const int q = i < n0 ? 0 : (i < n01 ? 1 : 2), li = i - (q == 0 ? 0 : (q == 1 ? n0 : n01));
                        const StageDesc::Seg sg = d.seg[q];
                        NF_CHECK(i >= 0 && i < np && li >= 0 && li < sg.ncell && sg.ps0 >= 0 && sg.ps0 + li + 1 < kPsMax);
                        const uint32_t p0 = ps[sg.ps0 + li], p1 = ps[sg.ps0 + li + 1];
                        slot = sg.slot0 + (int)(p0 - ps[sg.ps0]); nsl = (int)(p1 - p0);
                        NF_CHECK(slot >= 0 && nsl >= 0 && slot + nsl <= kTile && (slot & 3) == 0 && (nsl & 3) == 0);
                        czs = ((double)(float)((double)(sg.jw0 + li) * a.k.cell_w) + sg.wz) * a.k.scale;
                    };
                    for (int i = wlo + lane; i <= whi; i += 32) {
                        int slot, nsl; double czs;
                        cell(i, slot, nsl, czs);
                        for (int q = slot >> 2, qe = (slot + nsl) >> 2; q < qe; q++) qz[q] = czs;
                    }
                    if (ilo <= ihi) {
                        int s0, n0s, s1, n1s; double c0;
                        cell(ilo, s0, n0s, c0);
                        cell(ihi, s1, n1s, c0);
                        qlo = s0 >> 2;
                        cnt = ((s1 + n1s) >> 2) - qlo;
                    }
                } else {
                    for (int i = wlo + lane; i <= whi; i += 32) {
                        NF_CHECK(i >= 0 && i < np && np <= kMaxPieces);
                        const Piece pc = d.pieces[i];
                        NF_CHECK(pc.sm_off >= 0 && pc.nslots >= 0 && pc.sm_off + pc.nslots <= kTile);
                        for (int q = pc.sm_off >> 2, qe = (pc.sm_off + pc.nslots) >> 2; q < qe; q++) qz[q] = pc.czs;
                    }
                    if (ilo <= ihi) {
                        const Piece pl = d.pieces[ilo], ph = d.pieces[ihi];
                        qlo = pl.sm_off >> 2;
                        cnt = ((ph.sm_off + ph.nslots) >> 2) - qlo;
                    }
                }
                if (lane == 0) qz[kTile / 4] = oczs;                 // the dummy quad: any finite corner
                __syncwarp();
                const int cmax = __reduce_max_sync(kFull, cnt);
                // near column: the spline-capable body (a vote per quad pair) only if some sink of the warp is within eps_s of the
                // column in x and y (the z gap is not looked at here: conservative); the corner columns almost never are
                const bool soft = soft_mode == 2 || (soft_mode == 1 && __any_sync(kFull, gxy2 < a.k.soft_thr2));
                const bool dens = DENS && (a.dens_mode == 2 || (gap_dens && __any_sync(kFull, gxy2 < a.dens_thr2)));
                const float4 *py0 = sbase + kTileAlloc / 4, *pz0 = py0 + kTileAlloc / 4, *pm0 = pz0 + kTileAlloc / 4;
                const float4 one = make_float4(1.f, 1.f, 1.f, 1.f);
                auto body = [&](auto mode) {
                    constexpr int MODE = decltype(mode)::value;
#pragma unroll 2
                    for (int it = 0; it < cmax; it++) {
                        const int q = it < cnt ? qlo + it : kTile / 4;
                        NF_CHECK(q >= 0 && q <= kTile / 4);
                        const float dzc = (float)(qz[q] - oczs);
                        const float2 nz = make_float2(dzc - zi.x, dzc - zi.y);
                        quad<PACKED, MODE, MASS, MODE == 2 && NF_DENS_QV>(sbase[q], py0[q], pz0[q], MASS ? pm0[q] : one, nx, ny, nz, coef, f);
                    }
                };
                if (DENS && dens) body(std::integral_constant<int, 2>());
                else if (soft)    body(std::integral_constant<int, 1>());
                else              body(std::integral_constant<int, 0>());
                __syncwarp();
            } else
            // Step s pairs the lanes of the warp by SOURCE cell: a lane takes the one cell j of its stencil with
            // (j - (z0 - R)) mod (2R+1) == s.  Lanes of different sink cells then read the same piece in all steps but
            // the few where the stencils do not overlap (cells j and j + 2R+1 share a step), so the piece lengths of
            // a step differ between lanes only there.
            for (int s = 0; s < nsteps; s++) {
                int t = s - zoff;                                   // offset of that cell from zc - R, in [0, 2R]
                t += t < 0 ? nsteps : 0;
                const int idx = ibase + t;                          // the lane's piece for cell zc - R + t
                const bool valid = (unsigned)idx < (unsigned)np;
                int n4 = 0, sm_off = 0;
                double czs = 0.0;
                if (valid) {
                    NF_CHECK(np <= kMaxPieces);
                    const Piece pc = d.pieces[idx];
                    n4 = pc.nslots >> 2; sm_off = pc.sm_off; czs = pc.czs;
                }
                const int nmax = __reduce_max_sync(kFull, n4);
                if (nmax == 0) continue;
                const int nmin = __reduce_min_sync(kFull, n4 > 0 ? n4 : 0x7fffffff);   // over the lanes that have a piece
                const uint32_t live = __ballot_sync(kFull, n4 > 0);
                const float dzc = (float)(czs - oczs);
                const float2 nz = make_float2(dzc - zi.x, dzc - zi.y);
                const float4 *px = sbase + (sm_off >> 2);
                const int jdummy = (kTile - sm_off) >> 2;           // the dummy quad, relative to px
                const int dt = t - R;
                bool soft = soft_mode == 2, dens = DENS && a.dens_mode == 2;
                if (soft_mode == 1 || gap_dens) {                   // warp-uniform; dt is per lane
                    const bool touching = n4 > 0 && dt >= -1 && dt <= 1;
                    const float gz = dt < 0 ? fminf(zi.x, zi.y) : (dt > 0 ? a.k.w_scaled - fmaxf(zi.x, zi.y) : 0.f);
                    const float gap2 = fmaf(gz, gz, gxy2);
                    if (soft_mode == 1) soft = __any_sync(kFull, touching && gap2 < a.k.soft_thr2);
                    if (gap_dens) dens = __any_sync(kFull, touching && gap2 < a.dens_thr2);
                }
                constexpr int UT = QV ? kUnrollTailQV : kUnrollTail;
                if (DENS && dens) piece_loop<PACKED, 2, MASS, NF_DENS_QV, UT>(px, n4, nmin, nmax, live, jdummy, nx, ny, nz, coef, f);
                else if (soft)    piece_loop<PACKED, 1, MASS, QV, UT>(px, n4, nmin, nmax, live, jdummy, nx, ny, nz, coef, f);
                else              piece_loop<PACKED, 0, MASS, false, UT>(px, n4, nmin, nmax, live, jdummy, nx, ny, nz, coef, f);
                // The FP32 chain of a sink runs over ONE source cell (one step), then joins the FP64 sums: on inputs whose
                // pair forces nearly cancel (config 2, a barely perturbed lattice) the rounding of a chain grows with its
                // length (error ~ 2^-24 x terms x |term| / sqrt 2), and chains of a whole stage (~350 sources) put the 99.9 %
                // quantile of the full particle set at 1.36e-5 (4.6e-6 with per-cell chains).  Steps of a few quads (sparse
                // cells) keep adding to the same chain.
                if (nmax >= kFlushQuads) { flush(); pending = false; } else pending = true;
            }
            if (pending) flush();
        }
        if ((flags & kFlagEnd) && (sp & 255u) > 1u) {          // warp-uniform, the same for every consumer warp of the CTA
            const int nsplit = (int)(sp & 255u), ng = (int)((sp >> 8) & 255u), q = (int)((sp >> 16) & 255u);
            asm volatile("bar.sync 1, %0;" ::"r"(32 * kConsumerWarps) : "memory");
            if (warp_on && q == 0) {
                for (int t = 1; t < nsplit; t++) {
                    const int w2 = warp + t * ng;
#pragma unroll
                    for (int c = 0; c < (DENS ? 8 : 6); c++) acc64[c][lane] += sm.acc[w2][c][lane];
                }
            }
            asm volatile("bar.sync 1, %0;" ::"r"(32 * kConsumerWarps) : "memory");   // the sums of the other warps may be zeroed for the next unit
        }
        if ((flags & kFlagEnd) && nreal && ((sp >> 16) & 255u) == 0u) {
            const double s2 = a.k.out_scale;
#pragma unroll
            for (int h = 0; h < 2; h++) {
                if ((uint32_t)h >= nreal) break;
                const size_t i = __ldg(a.perm + slot + h);
                const float fx = (float)(acc64[3 * h + 0][lane] * s2), fy = (float)(acc64[3 * h + 1][lane] * s2), fz = (float)(acc64[3 * h + 2][lane] * s2);
                if (!EPI || a.acc) { a.acc[3 * i + 0] = fx; a.acc[3 * i + 1] = fy; a.acc[3 * i + 2] = fz; }
                if (DENS) a.rho[i] = (float)acc64[6 + h][lane];
                if (EPI && a.vel) {                                   // kick: v += a dt (leapfrog)
                    a.vel[3 * i + 0] = fmaf(fx, a.dt, a.vel[3 * i + 0]);
                    a.vel[3 * i + 1] = fmaf(fy, a.dt, a.vel[3 * i + 1]);
                    a.vel[3 * i + 2] = fmaf(fz, a.dt, a.vel[3 * i + 2]);
                }
                if (EPI && a.amax)                             // per-cell max |a| of the timestep criterion
                    atomicMax(a.amax + cell, __float_as_uint(sqrtf(fmaf(fx, fx, fmaf(fy, fy, fz * fz)))));
            }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(&sm.empty[stage]);
        if (++stage == kStages) { stage = 0; phase ^= 1u; }
    }
}

// FLAT = false: an instance WITHOUT the flat loop and the lean stages, for the launch that holds no flat unit (nf_bin sorts
// them behind all the others): the stepped pair loops then keep the registers and uniform registers they had before the
// sparse path grew (with both in one instance ptxas re-loaded `tiny` and the spline coefficient from the constant bank
// inside the quad-vote loop: config 4 -1.6 %, config 5 -1.8 %).  A flat unit that reaches such an instance is still
// computed correctly, by the stepped loop.
template <bool PACKED, bool DENS, bool EPI, bool MASS, bool QV = false, bool FLAT = true>
__global__ void __launch_bounds__(kAccelThreads, kMinCtasPerSm) direct_kernel(const AccelArgs a)
{
    constexpr int NARR = MASS ? 4 : 3;
    constexpr int kStages = StagesFor<NARR>::value;
    extern __shared__ __align__(128) unsigned char smem_raw[];          // dynamic: stages above 48 KB need the opt-in
    SharedStorageT<NARR, FLAT> &sm = *reinterpret_cast<SharedStorageT<NARR, FLAT> *>(smem_raw);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid < kStages * NARR * 4)                                       // dummy quad: far-away coordinates, mass 0
        sm.buf[tid / (4 * NARR)][(tid / 4) % NARR][kTile + (tid & 3)] = (tid / 4) % NARR == 3 ? 0.f : kDummy;
    if (tid == 0) {
        for (int s = 0; s < kStages; s++) { mbar_init(&sm.full[s], 1); mbar_init(&sm.empty[s], kConsumerWarps); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    if (warp == kConsumerWarps) producer<NARR, FLAT>(a, sm, lane);
    else                        consumer<PACKED, DENS, EPI, MASS, QV, FLAT>(a, sm, warp, lane);
}

typedef void (*direct_fn)(const AccelArgs);
template <bool MASS>
static direct_fn pick_kernel_m(int variant, bool dens, bool epi)    // dens and epi are separate entry points
{
    if (variant == 0) return dens ? direct_kernel<true, true, false, MASS> : (epi ? direct_kernel<true, false, true, MASS> : direct_kernel<true, false, false, MASS>);
    return dens ? direct_kernel<false, true, false, MASS> : (epi ? direct_kernel<false, false, true, MASS> : direct_kernel<false, false, false, MASS>);
}
static direct_fn pick_kernel(int variant, bool dens, bool epi, bool mass = false, bool qv = false, bool noflat = false)
{
    // the instances without the flat loop exist for the packed force-only kernels with unit masses (plain and fused epilogue)
    if (noflat && variant == 0 && !dens && !mass) {
        if (qv) return epi ? direct_kernel<true, false, true, false, true, false> : direct_kernel<true, false, false, false, true, false>;
        return epi ? direct_kernel<true, false, true, false, false, false> : direct_kernel<true, false, false, false, false, false>;
    }
    // the quad-vote instances exist for the packed force-only kernels (plain and fused epilogue, with and without masses:
    // which pairs next to eps_s see the spline's min depends on the vote granularity, at the level of one ulp of that
    // pair, so the mass kernel must follow the plain one for "all masses 1 = the same bits")
    if (qv && variant == 0 && !dens) {
        if (mass) return epi ? direct_kernel<true, false, true, true, true> : direct_kernel<true, false, false, true, true>;
        return epi ? direct_kernel<true, false, true, false, true> : direct_kernel<true, false, false, false, true>;
    }
    return mass ? pick_kernel_m<true>(variant, dens, epi) : pick_kernel_m<false>(variant, dens, epi);
}
static size_t smem_bytes(bool mass, bool flat = true)
{
    if (!flat) return sizeof(SharedStorageT<3, false>);          // the instances without the flat loop are unit-mass kernels
    return mass ? sizeof(SharedStorageT<4>) : sizeof(SharedStorageT<3>);
}

int accel_max_ctas_per_sm(int variant)
{
    int nb = 0;
    direct_fn fn = pick_kernel(variant, false, false);
    cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_bytes(false));
    cudaError_t e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, fn, kAccelThreads, smem_bytes(false));
    if (e != cudaSuccess) { cudaGetLastError(); return 0; }
    return nb;
}

// rho == NULL: no density.  b is the density kernel radius in box units (validated by the caller).
// vel / amax_cell: optional fused epilogue (kick by dt, per-cell maximum acceleration).
int launch_accel(nf_plan *p, float *acc, float *rho, double b, float *vel, double dt, float *amax_cell)
{
    cudaStream_t st = p->stream;
    p->have_accel_time = false;
    p->launches_accel = 0;
    if (p->n == 0 || p->n_units == 0) return NF_OK;
    const bool dens = rho != nullptr;
    const bool mass = p->have_mass;
    p->quad_vote = p->quad_vote_opt >= 0 ? p->quad_vote_opt : (p->max_count > kQuadVoteAbove ? 1 : 0);
    const bool epi = vel != nullptr || amax_cell != nullptr;
    // nf_bin sorted the flat units (sparse windows) behind all the others: the stepped units go to an instance without the
    // flat loop, the flat units to the instance that has it (never the quad-vote one: heavy cells are not flat) -- two
    // launches, one after the other on the plan's stream.  Where no such instance exists (density, masses, scalar variant) or
    // the list is not partitioned (small problems, heavy_first = 0) one launch of the instance with both loops does it all.
    const bool split = p->n_flat >= 0 && p->heavy_first && p->variant == 0 && !dens && !mass;
    const long long n_step = split ? p->n_units - p->n_flat : p->n_units;
    direct_fn fns[2] = {pick_kernel(p->variant, dens, epi, mass, p->quad_vote != 0, split), pick_kernel(p->variant, dens, epi, mass, false, false)};
    long long first[2] = {0, n_step}, count[2] = {n_step, p->n_units - n_step}, grids[2] = {0, 0};
    const size_t smems[2] = {smem_bytes(mass, !split), smem_bytes(mass, true)};
    for (int l = 0; l < 2; l++) {
        if (count[l] <= 0) continue;
        int per_sm = 0;
        const size_t smem = smems[l];
        NF_CUDA_OK(cudaFuncSetAttribute(fns[l], cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, fns[l], kAccelThreads, smem) != cudaSuccess) { cudaGetLastError(); per_sm = 0; }
        if (per_sm <= 0) { set_error("direct_kernel cannot be resident on this device (occupancy query returned 0)"); return NF_ERR_CUDA; }
        if (p->ctas_per_sm > 0 && p->ctas_per_sm < per_sm) per_sm = p->ctas_per_sm;
        grids[l] = (long long)p->sm_count * per_sm;
        if (grids[l] > count[l]) grids[l] = count[l];
    }
    AccelArgs a;
    a.k = p->k;
    a.x = p->ws.x; a.y = p->ws.y; a.z = p->ws.z; a.m = mass ? p->mass_soa : nullptr;
    a.poff = p->ws.poff; a.voff = p->ws.voff; a.offset = p->ws.offset; a.perm = p->perm;
    const Unit *units = p->heavy_first ? p->ws.units_sorted : p->ws.units;
    a.acc = acc;
    a.fastpath = p->fastpath;
    a.rho = rho; a.dens_nb2 = 0.f; a.dens_thr2 = 0.f; a.dens_mode = 0;
    a.vel = vel; a.dt = (float)dt; a.amax = reinterpret_cast<uint32_t *>(amax_cell);
    if (dens) {
        const double bs = b * p->k.scale;                       // scaled units
        const double margin = 4.0 * 1.2e-7 * p->k.L * p->k.scale;   // as for the spline: float32 rounding of the coordinates
        a.dens_nb2 = (float)(-1.0 / (bs * bs));
        a.dens_thr2 = (float)((bs + margin) * (bs + margin) * 1.0001);
        a.dens_mode = (b <= 0.999 * p->k.cell_w) ? 1 : 2;
    }
    NF_CUDA_OK(cudaEventRecord(p->ev[2], st));
    NF_CUDA_OK(cudaMemsetAsync(&p->ws.scalars[1], 0, 4, st));        // the two work counters (scalars 1 and 9)
    NF_CUDA_OK(cudaMemsetAsync(&p->ws.scalars[9], 0, 4, st));
    if (amax_cell) NF_CUDA_OK(cudaMemsetAsync(amax_cell, 0, 4 * (size_t)p->k.ncells, st));
    p->accel_grid = 0;
    for (int l = 0; l < 2; l++) {
        if (count[l] <= 0) continue;
        a.units = units + first[l];
        a.n_units = (uint32_t)count[l];
        a.counter = &p->ws.scalars[l == 0 ? 1 : 9];
        fns[l]<<<(unsigned)grids[l], kAccelThreads, smems[l], st>>>(a);
        NF_CUDA_OK(cudaGetLastError());
        if (grids[l] > p->accel_grid) p->accel_grid = (int)grids[l];
        p->launches_accel++;
    }
    NF_CUDA_OK(cudaEventRecord(p->ev[3], st));
    p->have_accel_time = true;
    return NF_OK;
}

}  // namespace nf
