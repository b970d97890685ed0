// nf_direct.cu -- steps S6-S7 of the hot path: the near-field direct sum and the scatter to input order.
//
//   a_i = sum_j d_ij K(|d_ij|),  j over the particles of the (2R+1)^3 periodic cells around the cell of i
//   (sec. 3.1: "sourced by particles in neighboring cells out to radius R ... direct,
//   O(N^2) summation with a compact spline softening kernel"; periodic images kept).
//
// Design (sm_100a):
//   * persistent CTAs, one producer warp + kConsumerWarps consumer warps, work units (<= 128 sinks of one
//     cell) pulled from an atomic counter in heavy-first order;
//   * the producer streams each of the (2R+1)^2 z-pencils of the stencil into shared memory with TMA 1-D
//     bulk copies (cp.async.bulk + mbarrier complete_tx) through a kStages-deep ring; consumers never touch
//     global memory in the pair loop;
//   * one sink per lane in registers; sources are read as broadcast LDS.128 of 4 x, 4 y, 4 z and processed as
//     two packed pairs with FFMA2/FADD2/FMUL2 (fma.rn.f32x2), one MUFU.RSQ per interaction;
//   * coordinates are cell-corner relative (exact), the periodic wrap is a per-(sink cell, source cell)
//     constant subtracted from the sink once per piece -- nothing periodic in the pair loop;
//   * cells whose max-norm offset is >= 2 cannot hold a pair closer than eps_s (when eps_s <= cell width):
//     they take the pure Newtonian body (no spline, no min);
//   * FP32 FMA chain per (sink, source cell) piece, piece partials added in FP64 (two-level accumulation);
//   * the epilogue writes acc[perm[s]] directly (S7 fused, no sorted acceleration buffer).
#include "nf_internal.h"

namespace nf {

enum { kFlagBegin = 1, kFlagEnd = 2, kFlagTerm = 4 };

struct Piece {          // one source cell (or part of one) inside a stage
    int   sm_off;       // first slot in the stage buffers (multiple of 4)
    int   nslots;       // multiple of 4
    float dx, dy, dz;   // sink shift: d = x_src - (x_sink - shift), scaled cell-relative units
    int   soft;         // 1: spline + min body, 0: pure Newtonian body
};

struct StageDesc {
    int      flags;
    int      npieces;
    uint32_t sink_p0;   // padded slot of the unit's first sink
    uint32_t nsink;
    uint32_t out0;      // sorted (unpadded) slot of the unit's first sink -> perm index
    int      pad_[3];
    Piece    pieces[kMaxPieces];
};

struct __align__(128) SharedStorage {
    float sx[kStages][kTile];
    float sy[kStages][kTile];
    float sz[kStages][kTile];
    StageDesc desc[kStages];
    unsigned long long full[kStages];
    unsigned long long empty[kStages];
};

// ---- PTX helpers: mbarrier + TMA 1-D bulk copy ---------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(void *bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_wait(void *bar, uint32_t parity)
{
    const uint32_t a = smem_u32(bar);
    uint32_t ok;
    do {
        asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                     : "=r"(ok) : "r"(a), "r"(parity) : "memory");
    } while (!ok);
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
struct SoftCoef { float A, B, C, tiny; };

// two sources (packed) against one sink: 14 (soft) / 11 (Newtonian) FP32-pipe instructions per pair of
// interactions, plus 2 MUFU.RSQ and, soft only, 2 FMNMX.
template <bool SOFT>
__device__ __forceinline__ void interact2(const float2 X, const float2 Y, const float2 Z, const float2 nx, const float2 ny,
                                          const float2 nz, const SoftCoef &c, float2 &ax, float2 &ay, float2 &az)
{
    const float2 dx = __fadd2_rn(X, nx), dy = __fadd2_rn(Y, ny), dz = __fadd2_rn(Z, nz);
    float2 r2 = __ffma2_rn(dz, dz, make_float2(c.tiny, c.tiny));
    r2 = __ffma2_rn(dy, dy, r2);
    r2 = __ffma2_rn(dx, dx, r2);
    float2 ri;
    ri.x = rsqrt_approx(r2.x);
    ri.y = rsqrt_approx(r2.y);
    const float2 ri2 = __fmul2_rn(ri, ri);
    float2 k = __fmul2_rn(ri2, ri);
    if (SOFT) {
        const float2 r = __fmul2_rn(r2, ri);
        float2 t = __ffma2_rn(make_float2(c.C, c.C), r2, make_float2(c.A, c.A));
        t = __ffma2_rn(make_float2(c.B, c.B), r, t);
        k.x = fminf(k.x, t.x);
        k.y = fminf(k.y, t.y);
    }
    ax = __ffma2_rn(k, dx, ax);
    ay = __ffma2_rn(k, dy, ay);
    az = __ffma2_rn(k, dz, az);
}

// scalar body (variant 1): 14 / 11 FP32-pipe instructions per interaction
template <bool SOFT>
__device__ __forceinline__ void interact1(const float X, const float Y, const float Z, const float nx, const float ny,
                                          const float nz, const SoftCoef &c, float &ax, float &ay, float &az)
{
    const float dx = X + nx, dy = Y + ny, dz = Z + nz;
    const float r2 = fmaf(dx, dx, fmaf(dy, dy, fmaf(dz, dz, c.tiny)));
    const float ri = rsqrt_approx(r2);
    float k = ri * ri * ri;
    if (SOFT) {
        const float r = r2 * ri;
        const float t = fmaf(c.B, r, fmaf(c.C, r2, c.A));
        k = fminf(k, t);
    }
    ax = fmaf(k, dx, ax);
    ay = fmaf(k, dy, ay);
    az = fmaf(k, dz, az);
}

template <bool PACKED, bool SOFT>
__device__ __forceinline__ void piece_loop(const float4 *__restrict__ px, const float4 *__restrict__ py,
                                           const float4 *__restrict__ pz, const int n4, const float sxi, const float syi,
                                           const float szi, const SoftCoef &c, double &ax, double &ay, double &az)
{
    if (PACKED) {
        const float2 nx = make_float2(sxi, sxi), ny = make_float2(syi, syi), nz = make_float2(szi, szi);
        float2 fx = make_float2(0.f, 0.f), fy = fx, fz = fx;
#pragma unroll 2
        for (int j = 0; j < n4; j++) {
            const float4 X = px[j], Y = py[j], Z = pz[j];
            interact2<SOFT>(make_float2(X.x, X.y), make_float2(Y.x, Y.y), make_float2(Z.x, Z.y), nx, ny, nz, c, fx, fy, fz);
            interact2<SOFT>(make_float2(X.z, X.w), make_float2(Y.z, Y.w), make_float2(Z.z, Z.w), nx, ny, nz, c, fx, fy, fz);
        }
        ax += (double)fx.x + (double)fx.y;
        ay += (double)fy.x + (double)fy.y;
        az += (double)fz.x + (double)fz.y;
    } else {
        float fx0 = 0.f, fy0 = 0.f, fz0 = 0.f, fx1 = 0.f, fy1 = 0.f, fz1 = 0.f;
#pragma unroll 2
        for (int j = 0; j < n4; j++) {
            const float4 X = px[j], Y = py[j], Z = pz[j];
            interact1<SOFT>(X.x, Y.x, Z.x, sxi, syi, szi, c, fx0, fy0, fz0);
            interact1<SOFT>(X.y, Y.y, Z.y, sxi, syi, szi, c, fx1, fy1, fz1);
            interact1<SOFT>(X.z, Y.z, Z.z, sxi, syi, szi, c, fx0, fy0, fz0);
            interact1<SOFT>(X.w, Y.w, Z.w, sxi, syi, szi, c, fx1, fy1, fz1);
        }
        ax += (double)fx0 + (double)fx1;
        ay += (double)fy0 + (double)fy1;
        az += (double)fz0 + (double)fz1;
    }
}

// ---- the kernel --------------------------------------------------------------------------------
struct AccelArgs {
    Consts k;
    const float *x, *y, *z;          // padded SoA sources (= sinks)
    const uint32_t *poff, *offset, *perm;
    const Unit *units;
    uint32_t n_units;
    uint32_t *counter;               // atomic work counter (zeroed before launch)
    float *acc;                      // [n][3] input order
    int fastpath;
};

template <bool PACKED>
__global__ void __launch_bounds__(kAccelThreads) direct_kernel(const AccelArgs a)
{
    __shared__ SharedStorage sm;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;

    if (tid == 0) {
        for (int s = 0; s < kStages; s++) { mbar_init(&sm.full[s], 1); mbar_init(&sm.empty[s], kConsumerWarps); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    if (warp == kConsumerWarps) {
        // ================================ producer (one lane) ================================
        if (lane != 0) return;
        const Consts &k = a.k;
        const int cpd = k.cpd, R = k.R;
        int stage = 0;
        uint32_t phase = 0;
        bool open = false, sealed = false;
        int fill = 0, np = 0, sflags = 0;
        // pending merged copy
        uint32_t cp_g = 0, cp_s = 0, cp_n = 0;
        auto flush_copy = [&]() {
            if (cp_n) {
                tma_load_1d(&sm.sx[stage][cp_s], a.x + cp_g, cp_n * 4u, &sm.full[stage]);
                tma_load_1d(&sm.sy[stage][cp_s], a.y + cp_g, cp_n * 4u, &sm.full[stage]);
                tma_load_1d(&sm.sz[stage][cp_s], a.z + cp_g, cp_n * 4u, &sm.full[stage]);
                cp_n = 0;
            }
        };
        auto commit = [&](int extra) {
            flush_copy();
            sm.desc[stage].flags = sflags | extra;
            sm.desc[stage].npieces = np;
            mbar_arrive_expect_tx(&sm.full[stage], (uint32_t)fill * 12u);
            if (++stage == kStages) { stage = 0; phase ^= 1u; }
            open = false; sealed = false;
        };
        for (;;) {
            const uint32_t u = atomicAdd(a.counter, 1u);
            if (u >= a.n_units) break;
            const Unit un = a.units[u];
            const int cz = un.cell % cpd, cy = (un.cell / cpd) % cpd, cx = un.cell / (cpd * cpd);
            const uint32_t sink_p0 = __ldg(a.poff + un.cell) + un.k0;
            const uint32_t out0 = __ldg(a.offset + un.cell) + un.k0;
            const double ocx = (double)(float)((double)cx * k.cell_w), ocy = (double)(float)((double)cy * k.cell_w),
                         ocz = (double)(float)((double)cz * k.cell_w);
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
                    for (int oz = -R; oz <= R; oz++) {
                        int jz = cz + oz; double wz = 0.0;
                        if (jz < 0) { jz += cpd; wz = -k.L; } else if (jz >= cpd) { jz -= cpd; wz = k.L; }
                        uint32_t p0 = __ldg(a.poff + row + jz);
                        const uint32_t p1 = __ldg(a.poff + row + jz + 1);
                        if (p0 == p1) continue;
                        const float Dz = (float)(((double)(float)((double)jz * k.cell_w) + wz - ocz) * k.scale);
                        const int far = (ox > 1 || ox < -1 || oy > 1 || oy < -1 || oz > 1 || oz < -1);
                        const int soft = !(far && k.fast_ok && a.fastpath);
                        while (p0 < p1) {
                            if (open && (sealed || fill == kTile)) commit(0);
                            if (!open) {
                                mbar_wait(&sm.empty[stage], phase ^ 1u);
                                open = true; fill = 0; np = 0;
                                sflags = first ? kFlagBegin : 0;
                                first = false;
                                sm.desc[stage].sink_p0 = sink_p0;
                                sm.desc[stage].nsink = un.nk;
                                sm.desc[stage].out0 = out0;
                            }
                            const uint32_t t = min(p1 - p0, (uint32_t)(kTile - fill));
                            Piece &pc = sm.desc[stage].pieces[np++];
                            pc.sm_off = fill; pc.nslots = (int)t; pc.dx = Dx; pc.dy = Dy; pc.dz = Dz; pc.soft = soft;
                            if (cp_n && cp_g + cp_n == p0 && cp_s + cp_n == (uint32_t)fill) cp_n += t;
                            else { flush_copy(); cp_g = p0; cp_s = (uint32_t)fill; cp_n = t; }
                            fill += (int)t; p0 += t;
                        }
                    }
                    if (open) sealed = true;      // one z-pencil per stage
                }
            }
            commit(kFlagEnd);                     // the own cell is never empty, so a stage is open
        }
        mbar_wait(&sm.empty[stage], phase ^ 1u);
        sm.desc[stage].flags = kFlagTerm;
        sm.desc[stage].npieces = 0;
        mbar_arrive_expect_tx(&sm.full[stage], 0u);
        return;
    }

    // ==================================== consumers ====================================
    const SoftCoef coef = {a.k.A, a.k.B, a.k.C, a.k.tiny};
    int stage = 0;
    uint32_t phase = 0;
    float xi = 0.f, yi = 0.f, zi = 0.f;
    double ax = 0.0, ay = 0.0, az = 0.0;
    uint32_t nsink = 0, out0 = 0;
    for (;;) {
        mbar_wait(&sm.full[stage], phase);
        const StageDesc &d = sm.desc[stage];
        const int flags = d.flags;
        if (flags & kFlagTerm) break;
        if (flags & kFlagBegin) {
            nsink = d.nsink; out0 = d.out0;
            const uint32_t p = d.sink_p0 + (uint32_t)tid;
            const bool act = (uint32_t)tid < nsink;
            xi = act ? __ldg(a.x + p) : 0.f;
            yi = act ? __ldg(a.y + p) : 0.f;
            zi = act ? __ldg(a.z + p) : 0.f;
            ax = ay = az = 0.0;
        }
        if ((uint32_t)(warp * 32) < nsink) {
            const int np = d.npieces;
            for (int q = 0; q < np; q++) {
                const Piece pc = d.pieces[q];
                const float4 *px = reinterpret_cast<const float4 *>(&sm.sx[stage][pc.sm_off]);
                const float4 *py = reinterpret_cast<const float4 *>(&sm.sy[stage][pc.sm_off]);
                const float4 *pz = reinterpret_cast<const float4 *>(&sm.sz[stage][pc.sm_off]);
                const float sxi = pc.dx - xi, syi = pc.dy - yi, szi = pc.dz - zi;   // -(x_i - shift)
                if (pc.soft) piece_loop<PACKED, true>(px, py, pz, pc.nslots >> 2, sxi, syi, szi, coef, ax, ay, az);
                else         piece_loop<PACKED, false>(px, py, pz, pc.nslots >> 2, sxi, syi, szi, coef, ax, ay, az);
            }
        }
        if ((flags & kFlagEnd) && (uint32_t)tid < nsink) {
            const size_t i = __ldg(a.perm + out0 + tid);
            const double s2 = a.k.out_scale;
            a.acc[3 * i + 0] = (float)(ax * s2);
            a.acc[3 * i + 1] = (float)(ay * s2);
            a.acc[3 * i + 2] = (float)(az * s2);
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(&sm.empty[stage]);
        if (++stage == kStages) { stage = 0; phase ^= 1u; }
    }
}

int accel_max_ctas_per_sm(int variant)
{
    int nb = 0;
    cudaError_t e = variant == 0
        ? cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, direct_kernel<true>, kAccelThreads, 0)
        : cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, direct_kernel<false>, kAccelThreads, 0);
    if (e != cudaSuccess) { cudaGetLastError(); return 0; }
    return nb;
}

int launch_accel(nf_plan *p, float *acc)
{
    cudaStream_t st = p->stream;
    p->have_accel_time = false;
    p->launches_accel = 0;
    if (p->n == 0 || p->n_units == 0) return NF_OK;
    int per_sm = accel_max_ctas_per_sm(p->variant);
    if (per_sm <= 0) { set_error("direct_kernel cannot be resident on this device (occupancy query returned 0)"); return NF_ERR_CUDA; }
    if (p->ctas_per_sm > 0 && p->ctas_per_sm < per_sm) per_sm = p->ctas_per_sm;
    long long grid = (long long)p->sm_count * per_sm;
    if (grid > p->n_units) grid = p->n_units;
    AccelArgs a;
    a.k = p->k;
    a.x = p->ws.x; a.y = p->ws.y; a.z = p->ws.z;
    a.poff = p->ws.poff; a.offset = p->ws.offset; a.perm = p->perm;
    a.units = p->ws.units_sorted;
    a.n_units = (uint32_t)p->n_units;
    a.counter = &p->ws.scalars[1];
    a.acc = acc;
    a.fastpath = p->fastpath;
    NF_CUDA_OK(cudaEventRecord(p->ev[2], st));
    NF_CUDA_OK(cudaMemsetAsync(a.counter, 0, 4, st));
    if (p->variant == 0) direct_kernel<true><<<(unsigned)grid, kAccelThreads, 0, st>>>(a);
    else                 direct_kernel<false><<<(unsigned)grid, kAccelThreads, 0, st>>>(a);
    NF_CUDA_OK(cudaGetLastError());
    NF_CUDA_OK(cudaEventRecord(p->ev[3], st));
    p->have_accel_time = true;
    p->accel_grid = (int)grid;
    p->launches_accel = 1;
    return NF_OK;
}

}  // namespace nf
