// ubench_fp32_pipe.cu -- microbenchmark of the FP32 pipe of one B200 SM sub-partition for the instruction mix of the
// direct-sum pair body (where the "alu" roofline's attainable fraction comes from).  Not part of the
// library: a stand-alone program,
//     nvcc -gencode arch=compute_100a,code=sm_100a -O3 -std=c++17 -o ubench_fp32_pipe ubench_fp32_pipe.cu && ./ubench_fp32_pipe
// One CTA per SM, w warps per sub-partition (w = 1, 2, 4, 6, 8), every warp runs the same unrolled loop; cycles are read
// with clock64() per warp, the slowest warp counts.  "pipe-util" = FP32 lane-operations issued per cycle per lane
// (1 = the 128 lanes x 1 op/clk of the FP32 FMA peak); the two "body" rows also print the fraction of the 25-flop peak
// the pair body would reach if nothing else ran (11 FP32 lane-operations + 1 MUFU.RSQ per interaction).
// Results on B200: profiles/r2_ubench_fp32_pipe.md.
#include <cstdio>
#include <cstdlib>
#include <cuda_runtime.h>
#include <vector>

__device__ __forceinline__ float rsq(float x) { float y; asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }

#define ITER 2048

// MODE 0: 8 independent FFMA2 a += k*d (3 distinct pairs each)
// MODE 1: FFMA2 acc pattern: 4 groups x (ax += k dx; ay += k dy; az += k dz), k shared inside a group
// MODE 2: FFMA2 r2 = d*d + r2 (8 independent)
// MODE 3: FADD2 d = X + s(broadcast)  (8 independent)
// MODE 4: FMUL2 (8 independent)
// MODE 5: scalar FFMA 3 distinct (16 independent)
// MODE 6: full Newtonian body, source-packed (as in nf_direct.cu interact2), 2 quads per iteration, sources from registers
// MODE 7: full body, sink-packed: 2 sinks per lane, scalar sources
// MODE 8: full body scalar (interact1 MODE 0)
// MODE 9: MUFU.RSQ only (8 independent)
// MODE 10: as 6 but from shared memory (LDS.128 x3 per quad)
// MODE 11: as 7 but from shared memory
template <int MODE>
__global__ void __launch_bounds__(1024) ub(float *out, long long *cyc, int iters, float seed)
{
    __shared__ float4 sm[3 * 260];
    const int tid = threadIdx.x;
    for (int i = tid; i < 3 * 260; i += blockDim.x) sm[i] = make_float4(seed + i, seed * 2 + i, seed * 3 - i, seed + 0.5f * i);
    __syncthreads();
    float2 a[8], k[8], d[8];
#pragma unroll
    for (int i = 0; i < 8; i++) { a[i] = make_float2(seed + i, seed - i); k[i] = make_float2(1.0f + seed * i, 1.0f - seed * i); d[i] = make_float2(seed * 0.5f + i, seed * 0.25f + i); }
    float sx = seed * 7, sy = seed * 11, sz = seed * 13, tiny = 1e-30f;
    long long t0 = clock64();
    if (MODE == 0) {
        for (int it = 0; it < iters; it++) {
#pragma unroll
            for (int i = 0; i < 8; i++) a[i] = __ffma2_rn(k[i], d[i], a[i]);
        }
    } else if (MODE == 1) {
        for (int it = 0; it < iters; it++) {
#pragma unroll
            for (int g = 0; g < 4; g++) {
                const int s = (g & 1) * 3;
                a[s + 0] = __ffma2_rn(k[g], d[g], a[s + 0]);
                a[s + 1] = __ffma2_rn(k[g], d[g + 4], a[s + 1]);
                a[s + 2] = __ffma2_rn(k[g], k[g + 4], a[s + 2]);
            }
        }
    } else if (MODE == 2) {
        for (int it = 0; it < iters; it++) {
#pragma unroll
            for (int i = 0; i < 8; i++) a[i] = __ffma2_rn(d[i], d[i], a[i]);
        }
    } else if (MODE == 3) {
        for (int it = 0; it < iters; it++) {
#pragma unroll
            for (int i = 0; i < 8; i++) a[i] = __fadd2_rn(a[i], make_float2(sx, sx));
        }
    } else if (MODE == 4) {
        for (int it = 0; it < iters; it++) {
#pragma unroll
            for (int i = 0; i < 8; i++) a[i] = __fmul2_rn(a[i], k[i]);
        }
    } else if (MODE == 5) {
        for (int it = 0; it < iters; it++) {
#pragma unroll
            for (int i = 0; i < 8; i++) { a[i].x = fmaf(k[i].x, d[i].x, a[i].x); a[i].y = fmaf(k[i].y, d[i].y, a[i].y); }
        }
    } else if (MODE == 9) {
        for (int it = 0; it < iters; it++) {
#pragma unroll
            for (int i = 0; i < 8; i++) { a[i].x = rsq(a[i].x); }
        }
    } else if (MODE == 6 || MODE == 10) {
        float2 ax = a[0], ay = a[1], az = a[2];
        float4 X = make_float4(d[0].x, d[0].y, d[1].x, d[1].y), Y = make_float4(d[2].x, d[2].y, d[3].x, d[3].y), Z = make_float4(d[4].x, d[4].y, d[5].x, d[5].y);
        const float4 *px = sm, *py = sm + 260, *pz = sm + 520;
        for (int it = 0; it < iters; it++) {
#pragma unroll
            for (int q = 0; q < 2; q++) {
                if (MODE == 10) { const int j = (it * 2 + q) & 255; X = px[j]; Y = py[j]; Z = pz[j]; }
                else { X.x += 1.0f; Y.y += 1.0f; }       // keep the sources moving (cheap scalar ops)
#pragma unroll
                for (int h = 0; h < 2; h++) {
                    const float2 Xp = h ? make_float2(X.z, X.w) : make_float2(X.x, X.y);
                    const float2 Yp = h ? make_float2(Y.z, Y.w) : make_float2(Y.x, Y.y);
                    const float2 Zp = h ? make_float2(Z.z, Z.w) : make_float2(Z.x, Z.y);
                    const float2 dx = __fadd2_rn(Xp, make_float2(sx, sx)), dy = __fadd2_rn(Yp, make_float2(sy, sy)), dz = __fadd2_rn(Zp, make_float2(sz, sz));
                    float2 r2 = __ffma2_rn(dz, dz, make_float2(tiny, tiny));
                    r2 = __ffma2_rn(dy, dy, r2);
                    r2 = __ffma2_rn(dx, dx, r2);
                    float2 ri; ri.x = rsq(r2.x); ri.y = rsq(r2.y);
                    const float2 kk = __fmul2_rn(__fmul2_rn(ri, ri), ri);
                    ax = __ffma2_rn(kk, dx, ax); ay = __ffma2_rn(kk, dy, ay); az = __ffma2_rn(kk, dz, az);
                }
            }
        }
        a[0] = ax; a[1] = ay; a[2] = az;
    } else if (MODE == 7 || MODE == 11) {
        // two sinks per lane packed: (sA, sB); sources scalar
        float2 ax = a[0], ay = a[1], az = a[2];
        const float2 SX = make_float2(sx, sx + 1.f), SY = make_float2(sy, sy + 1.f), SZ = make_float2(sz, sz + 1.f);
        float4 X = make_float4(d[0].x, d[0].y, d[1].x, d[1].y), Y = make_float4(d[2].x, d[2].y, d[3].x, d[3].y), Z = make_float4(d[4].x, d[4].y, d[5].x, d[5].y);
        const float4 *px = sm, *py = sm + 260, *pz = sm + 520;
        for (int it = 0; it < iters; it++) {
            if (MODE == 11) { const int j = it & 255; X = px[j]; Y = py[j]; Z = pz[j]; }
            else { X.x += 1.0f; Y.y += 1.0f; }
#pragma unroll
            for (int h = 0; h < 4; h++) {
                const float xs = h == 0 ? X.x : h == 1 ? X.y : h == 2 ? X.z : X.w;
                const float ys = h == 0 ? Y.x : h == 1 ? Y.y : h == 2 ? Y.z : Y.w;
                const float zs = h == 0 ? Z.x : h == 1 ? Z.y : h == 2 ? Z.z : Z.w;
                const float2 dx = __fadd2_rn(SX, make_float2(xs, xs)), dy = __fadd2_rn(SY, make_float2(ys, ys)), dz = __fadd2_rn(SZ, make_float2(zs, zs));
                float2 r2 = __ffma2_rn(dz, dz, make_float2(tiny, tiny));
                r2 = __ffma2_rn(dy, dy, r2);
                r2 = __ffma2_rn(dx, dx, r2);
                float2 ri; ri.x = rsq(r2.x); ri.y = rsq(r2.y);
                const float2 kk = __fmul2_rn(__fmul2_rn(ri, ri), ri);
                ax = __ffma2_rn(kk, dx, ax); ay = __ffma2_rn(kk, dy, ay); az = __ffma2_rn(kk, dz, az);
            }
        }
        a[0] = ax; a[1] = ay; a[2] = az;
    } else if (MODE == 8) {
        float ax0 = a[0].x, ay0 = a[1].x, az0 = a[2].x, ax1 = a[0].y, ay1 = a[1].y, az1 = a[2].y;
        float4 X = make_float4(d[0].x, d[0].y, d[1].x, d[1].y), Y = make_float4(d[2].x, d[2].y, d[3].x, d[3].y), Z = make_float4(d[4].x, d[4].y, d[5].x, d[5].y);
        for (int it = 0; it < iters; it++) {
            X.x += 1.0f; Y.y += 1.0f;
#pragma unroll
            for (int h = 0; h < 4; h++) {
                const float xs = h == 0 ? X.x : h == 1 ? X.y : h == 2 ? X.z : X.w;
                const float ys = h == 0 ? Y.x : h == 1 ? Y.y : h == 2 ? Y.z : Y.w;
                const float zs = h == 0 ? Z.x : h == 1 ? Z.y : h == 2 ? Z.z : Z.w;
                const float dx = xs + sx, dy = ys + sy, dz = zs + sz;
                const float r2 = fmaf(dx, dx, fmaf(dy, dy, fmaf(dz, dz, tiny)));
                const float ri = rsq(r2);
                const float kk = ri * ri * ri;
                if (h & 1) { ax1 = fmaf(kk, dx, ax1); ay1 = fmaf(kk, dy, ay1); az1 = fmaf(kk, dz, az1); }
                else { ax0 = fmaf(kk, dx, ax0); ay0 = fmaf(kk, dy, ay0); az0 = fmaf(kk, dz, az0); }
            }
        }
        a[0] = make_float2(ax0, ax1); a[1] = make_float2(ay0, ay1); a[2] = make_float2(az0, az1);
    }
    long long t1 = clock64();
    float s = 0.f;
#pragma unroll
    for (int i = 0; i < 8; i++) s += a[i].x + a[i].y;
    out[blockIdx.x * blockDim.x + tid] = s;
    if ((tid & 31) == 0) cyc[(blockIdx.x * blockDim.x + tid) >> 5] = t1 - t0;
}

template <int MODE>
void run(const char *name, double lane_ops_per_iter, double inter_per_iter, int warps_per_smsp)
{
    const int threads = 128 * warps_per_smsp, blocks = 148;
    float *out; long long *cyc;
    cudaMalloc(&out, sizeof(float) * threads * blocks);
    cudaMalloc(&cyc, sizeof(long long) * threads * blocks / 32);
    ub<MODE><<<blocks, threads>>>(out, cyc, 64, 0.37f);
    cudaDeviceSynchronize();
    cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
    cudaEventRecord(e0);
    ub<MODE><<<blocks, threads>>>(out, cyc, ITER, 0.37f);
    cudaEventRecord(e1);
    cudaError_t err = cudaDeviceSynchronize();
    if (err != cudaSuccess) { printf("%s: %s\n", name, cudaGetErrorString(err)); exit(1); }
    float ms; cudaEventElapsedTime(&ms, e0, e1);
    std::vector<long long> h(threads * blocks / 32);
    cudaMemcpy(h.data(), cyc, sizeof(long long) * h.size(), cudaMemcpyDeviceToHost);
    double mean = 0; long long mx = 0;
    for (auto v : h) { mean += v; if (v > mx) mx = v; }
    mean /= h.size();
    // per SMSP: warps_per_smsp warps, each lane_ops_per_iter lane-ops per iteration per lane; the 32-lane pipe does 32 per cycle
    const double cyc_per_iter = (double)mx / ITER;
    const double pipe = warps_per_smsp * lane_ops_per_iter / cyc_per_iter;          // FP32 lane-ops per cycle per lane-slot (1 = peak)
    printf("%-34s w/smsp %2d  cycles/iter/warp %8.2f  pipe-util %.3f", name, warps_per_smsp, cyc_per_iter, pipe);
    if (inter_per_iter > 0) printf("  cycles per interaction per lane-slot %.2f  (25-flop frac %.3f)", cyc_per_iter / (warps_per_smsp * inter_per_iter), 25.0 / 2.0 * warps_per_smsp * inter_per_iter / cyc_per_iter);
    printf("  [%.3f ms]\n", ms);
    cudaFree(out); cudaFree(cyc);
}

int main()
{
    for (int w : {1, 2, 4, 6, 8}) {
        run<0>("FFMA2 3 distinct pairs", 16, 0, w);
        run<1>("FFMA2 acc pattern (k shared)", 24, 0, w);
        run<2>("FFMA2 d*d+r2", 16, 0, w);
        run<3>("FADD2 pair + scalar", 16, 0, w);
        run<4>("FMUL2", 16, 0, w);
        run<5>("FFMA scalar 3 distinct", 16, 0, w);
        run<9>("MUFU.RSQ (counted as 1 lane-op)", 8, 0, w);
        run<10>("body, 2 sources packed, 1 sink (LDS)", 88, 8, w);
        run<11>("body, 2 sinks packed, source bcast (LDS)", 88, 8, w);
        printf("\n");
    }
    return 0;
}
