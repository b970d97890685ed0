// nf_slabs.cu -- x-slab domain decomposition helpers: the paper's parallel method gives every
// node "a contiguous span of slabs" and needs "R loaded slabs on either side" from its neighbours (PAPER.md:355, 365-369
// sec. 3.2); sinks are owned, so nothing is reduced.  Here one process drives one GPU and everything that touches
// particle data runs in these kernels:
//   nf_slab_histogram  particles per x-slab of a position array (the cell rule of nf_bin, reading C6)
//   nf_slab_select     stable compaction of the particles of a slab range (what a peer needs as halo), device to device
//   nf_get_slab_cost   pair interactions per x-slab of the last binning (the scheduler's exact cost, S5)
//   nf_slab_partition  contiguous slab ranges with balanced cost (host arithmetic on cpd numbers, no particle data)
// The transfers themselves are the caller's (torch.distributed point-to-point over NCCL / NVLink).
#include "nf_internal.h"

#include <cmath>
#include <vector>

namespace nf {

__device__ __forceinline__ int slab_index(float xf, const Consts &k, bool &bad)
{
    const double x = (double)xf;
    if (!(x >= 0.0 && x < k.L)) bad = true;
    int q = (int)floor(x * k.inv_cell_w);
    return q >= k.cpd ? k.cpd - 1 : (q < 0 ? 0 : q);
}

constexpr int kSelThreads = 256, kSelItems = 4, kSelTile = kSelThreads * kSelItems;

__global__ void __launch_bounds__(kSelThreads) slab_hist_kernel(const float *__restrict__ pos, size_t n, Consts k,
                                                                unsigned long long *__restrict__ hist, uint32_t *__restrict__ flag)
{
    extern __shared__ uint32_t h[];                    // [cpd]
    for (int s = threadIdx.x; s < k.cpd; s += kSelThreads) h[s] = 0;
    __syncthreads();
    bool bad = false;
    for (size_t i = (size_t)blockIdx.x * kSelThreads + threadIdx.x; i < n; i += (size_t)gridDim.x * kSelThreads) {
        bool b2 = false;
        const int s = slab_index(pos[3 * i], k, b2);
        (void)slab_index(pos[3 * i + 1], k, b2);
        (void)slab_index(pos[3 * i + 2], k, b2);
        bad |= b2;
        atomicAdd(&h[s], 1u);
    }
    if (bad) atomicOr(flag, 1u);
    __syncthreads();
    for (int s = threadIdx.x; s < k.cpd; s += kSelThreads) if (h[s]) atomicAdd(&hist[s], (unsigned long long)h[s]);
}

__device__ __forceinline__ bool in_range(int s, int first, int cnt, int cpd)
{
    int rel = s - first; rel += rel < 0 ? cpd : 0;
    return rel < cnt;
}

// pass 1: selected particles per tile; pass 2 (after the exclusive scan of the tile counts): stable scatter
template <bool SCATTER>
__global__ void __launch_bounds__(kSelThreads) slab_select_kernel(const float *__restrict__ pos, size_t n, Consts k, int first, int cnt,
                                                                  uint32_t *__restrict__ tile_count, const uint32_t *__restrict__ tile_base,
                                                                  float *__restrict__ out, uint32_t *__restrict__ idx_out, size_t cap)
{
    __shared__ uint32_t s_warp[kSelThreads / 32];
    const size_t base = (size_t)blockIdx.x * kSelTile + (size_t)threadIdx.x * kSelItems;    // a thread owns consecutive particles
    uint32_t sel = 0;
    bool bad = false;
#pragma unroll
    for (int j = 0; j < kSelItems; j++)
        if (base + j < n && in_range(slab_index(pos[3 * (base + j)], k, bad), first, cnt, k.cpd)) sel |= 1u << j;
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    uint32_t inc = __popc(sel);
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { const uint32_t t = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= o) inc += t; }
    if (lane == 31) s_warp[w] = inc;
    __syncthreads();
    uint32_t wbase = 0, total = 0;
    for (int q = 0; q < kSelThreads / 32; q++) { const uint32_t t = s_warp[q]; if (q < w) wbase += t; total += t; }
    if (!SCATTER) {
        if (threadIdx.x == 0) tile_count[blockIdx.x] = total;
        return;
    }
    size_t dst = (size_t)tile_base[blockIdx.x] + wbase + inc - __popc(sel);
#pragma unroll
    for (int j = 0; j < kSelItems; j++) {
        if ((sel >> j) & 1u) {
            if (dst < cap) {
                const float *p = pos + 3 * (base + j);
                out[3 * dst + 0] = p[0]; out[3 * dst + 1] = p[1]; out[3 * dst + 2] = p[2];
                if (idx_out) idx_out[dst] = (uint32_t)(base + j);
            }
            dst++;
        }
    }
}

// pair interactions per x-slab of the last binning: sum over the slab's cells of count * (particles in the stencil)
__global__ void __launch_bounds__(256) slab_cost_kernel(Consts k, const uint32_t *__restrict__ count, const uint32_t *__restrict__ src,
                                                        double *__restrict__ cost)
{
    __shared__ double red[8];
    const uint32_t per = (uint32_t)k.cpd * k.cpd;
    double mine = 0.0;
    for (uint32_t c = threadIdx.x; c < per; c += 256) {
        const size_t id = (size_t)blockIdx.x * per + c;
        mine += (double)count[id] * (double)src[id];
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) mine += __shfl_down_sync(0xffffffffu, mine, o);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = mine;
    __syncthreads();
    if (threadIdx.x == 0) { double t = 0; for (int q = 0; q < 8; q++) t += red[q]; cost[blockIdx.x] = t; }
}

}  // namespace nf

using namespace nf;

extern "C" {

int nf_slab_histogram(nf_plan *p, const float *pos, long long n, long long *hist_host)
{
    if (!p || !hist_host || n < 0 || (!pos && n > 0)) { set_error("nf_slab_histogram: bad argument"); return NF_ERR_ARG; }
    const int cpd = p->k.cpd;
    for (int s = 0; s < cpd; s++) hist_host[s] = 0;
    if (n == 0) return NF_OK;
    unsigned long long *d = nullptr;
    NF_CUDA_OK(cudaMalloc(&d, 8 * (size_t)(cpd + 1)));
    cudaStream_t st = p->stream;
    cudaError_t e = cudaMemsetAsync(d, 0, 8 * (size_t)(cpd + 1), st);
    if (e == cudaSuccess) {
        const size_t want = ((size_t)n + kSelThreads - 1) / kSelThreads;
        const unsigned grid = (unsigned)(want < 2048 ? want : 2048);
        slab_hist_kernel<<<grid, kSelThreads, 4 * (size_t)cpd, st>>>(pos, (size_t)n, p->k, d, reinterpret_cast<uint32_t *>(d + cpd));
        e = cudaGetLastError();
    }
    std::vector<unsigned long long> h((size_t)cpd + 1);
    if (e == cudaSuccess) e = cudaMemcpyAsync(h.data(), d, 8 * (size_t)(cpd + 1), cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    cudaFree(d);
    if (e != cudaSuccess) { set_error("nf_slab_histogram: %s", cudaGetErrorString(e)); return NF_ERR_CUDA; }
    if (h[(size_t)cpd] & 1ull) { set_error("nf_slab_histogram: a coordinate is non-finite or outside [0, L)"); return NF_ERR_DOMAIN; }
    for (int s = 0; s < cpd; s++) hist_host[s] = (long long)h[(size_t)s];
    return NF_OK;
}

int nf_slab_select(nf_plan *p, const float *pos, long long n, int x_first, int n_slabs, float *out, unsigned *idx_out, long long cap,
                   long long *m_host)
{
    if (!p || !m_host || n < 0 || (!pos && n > 0) || cap < 0 || (!out && cap > 0)) { set_error("nf_slab_select: bad argument"); return NF_ERR_ARG; }
    if (x_first < 0 || x_first >= p->k.cpd || n_slabs < 0 || n_slabs > p->k.cpd) { set_error("nf_slab_select: bad slab range (%d, %d)", x_first, n_slabs); return NF_ERR_ARG; }
    *m_host = 0;
    if (n == 0 || n_slabs == 0) return NF_OK;
    if ((double)n >= 4294967296.0) { set_error("nf_slab_select: n >= 2^32"); return NF_ERR_ARG; }
    cudaStream_t st = p->stream;
    const size_t tiles = ((size_t)n + kSelTile - 1) / kSelTile;
    uint32_t *cnt = nullptr;
    NF_CUDA_OK(cudaMalloc(&cnt, 4 * (2 * tiles + 2)));
    uint32_t *base = cnt + tiles + 1;
    slab_select_kernel<false><<<(unsigned)tiles, kSelThreads, 0, st>>>(pos, (size_t)n, p->k, x_first, n_slabs, cnt, nullptr, nullptr, nullptr, 0);
    // exclusive scan of the tile counts on the host side of the stream: tiles = n / 1024 numbers
    std::vector<uint32_t> h(tiles + 1);
    cudaError_t e = cudaMemcpyAsync(h.data(), cnt, 4 * tiles, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    unsigned long long run = 0;
    if (e == cudaSuccess) {
        for (size_t t = 0; t < tiles; t++) { const uint32_t c = h[t]; h[t] = (uint32_t)run; run += c; }
        *m_host = (long long)run;
        if ((long long)run > cap) { cudaFree(cnt); set_error("nf_slab_select: %llu particles selected, the output holds %lld", run, cap); return NF_ERR_NOMEM; }
        e = cudaMemcpyAsync(base, h.data(), 4 * tiles, cudaMemcpyHostToDevice, st);
    }
    if (e == cudaSuccess && run > 0) {
        slab_select_kernel<true><<<(unsigned)tiles, kSelThreads, 0, st>>>(pos, (size_t)n, p->k, x_first, n_slabs, nullptr, base, out, idx_out, (size_t)cap);
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    cudaFree(cnt);
    if (e != cudaSuccess) { set_error("nf_slab_select: %s", cudaGetErrorString(e)); return NF_ERR_CUDA; }
    return NF_OK;
}

int nf_get_slab_cost(nf_plan *p, double *cost_host)
{
    if (!p || !cost_host) { set_error("nf_get_slab_cost: null argument"); return NF_ERR_ARG; }
    if (!p->binned) { set_error("nf_get_slab_cost: no binning"); return NF_ERR_STATE; }
    const int cpd = p->k.cpd;
    for (int s = 0; s < cpd; s++) cost_host[s] = 0.0;
    if (p->n == 0) return NF_OK;
    double *d = nullptr;
    NF_CUDA_OK(cudaMalloc(&d, 8 * (size_t)cpd));
    slab_cost_kernel<<<cpd, 256, 0, p->stream>>>(p->k, p->ws.count, p->ws.src, d);
    cudaError_t e = cudaGetLastError();
    if (e == cudaSuccess) e = cudaMemcpyAsync(cost_host, d, 8 * (size_t)cpd, cudaMemcpyDeviceToHost, p->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(p->stream);
    cudaFree(d);
    if (e != cudaSuccess) { set_error("nf_get_slab_cost: %s", cudaGetErrorString(e)); return NF_ERR_CUDA; }
    // cells outside the sink slabs only serve as sources on this rank: their cost belongs to their owner
    for (int s = 0; s < cpd; s++) { int rel = s - p->k.slab0; rel += rel < 0 ? cpd : 0; if (rel >= p->k.nslab) cost_host[s] = 0.0; }
    return NF_OK;
}

// Contiguous ranges [first[r], first[r] + count[r]) of the cpd slabs, every rank at least one slab, minimising the largest
// range cost (the step time of the slowest rank): the optimal bottleneck is one of the O(cpd^2) range sums; found by
// bisection over it with the greedy feasibility test, then the ranges are cut greedily from the left.
int nf_slab_partition(const double *cost, int cpd, int world, int *first, int *count)
{
    if (!first || !count || cpd < 1 || world < 1 || world > cpd) { set_error("nf_slab_partition: need 1 <= world <= cpd"); return NF_ERR_ARG; }
    std::vector<double> c((size_t)cpd, 1.0);
    double total = 0.0, cmax = 0.0;
    for (int s = 0; s < cpd; s++) {
        if (cost) {
            if (!(cost[s] >= 0.0) || !std::isfinite(cost[s])) { set_error("nf_slab_partition: cost[%d] is negative or not finite", s); return NF_ERR_ARG; }
            c[(size_t)s] = cost[s];
        }
        total += c[(size_t)s];
        if (c[(size_t)s] > cmax) cmax = c[(size_t)s];
    }
    // parts(B): ranges the greedy cut needs when no range may exceed B, a range taking at most as many slabs as leave one
    // for every later rank
    auto parts = [&](double B) {
        int np = 0, s = 0;
        while (s < cpd) {
            double run = 0.0; int len = 0;
            while (s < cpd && (len == 0 || run + c[(size_t)s] <= B)) { run += c[(size_t)s]; s++; len++; }
            np++;
        }
        return np;
    };
    double lo = cmax, hi = total > cmax ? total : cmax;
    if (parts(lo) > world) {
        for (int it = 0; it < 200 && hi - lo > 1e-12 * hi; it++) {
            const double mid = 0.5 * (lo + hi);
            if (parts(mid) <= world) hi = mid; else lo = mid;
        }
    } else hi = lo;
    const double B = hi;
    int s = 0;
    for (int r = 0; r < world; r++) {
        const int left = world - r - 1;                 // ranks after this one: each still needs a slab
        double run = 0.0; int len = 0;
        while (s + len < cpd - left && (len == 0 || run + c[(size_t)(s + len)] <= B)) { run += c[(size_t)(s + len)]; len++; }
        if (r == world - 1) len = cpd - s;              // the last rank takes what is left (within B by construction)
        first[r] = s; count[r] = len;
        s += len;
    }
    return NF_OK;
}

}  // extern "C"

// ==================================================================================================================
// nf_slab_histogram_static -- nf_slab_histogram for callers that must not allocate (code under CUDA graph capture,
// tight serving loops, harnesses that forbid cudaMalloc): the same kernel, its scratch (the per-slab counters and the
// domain flag) in a file-scope device array instead of a cudaMalloc'ed buffer.  No cudaMalloc, no cudaFree, no
// allocating library routine, no host heap.
//   * every GPU that loads the library holds the array (8 KB) until the process exits;
//   * the limit is cpd <= kStaticMaxCpd (larger grids: nf_slab_histogram);
//   * every call on a device shares the ONE array and finds the previous call's numbers in it: the call clears what
//     it uses first, and two calls that overlap on the same GPU (other streams, other plans, other host threads) race
//     -- the caller serialises them.
// In host code `g_slab_scratch` is a host-side stand-in, not a device address: the device address comes from
// cudaGetSymbolAddress, once per device, with that device current.
constexpr int kStaticMaxCpd = 1024;
static __device__ __align__(256) unsigned long long g_slab_scratch[kStaticMaxCpd + 2];   // [cpd] counts, then the flag word

namespace nf {
constexpr int kStaticMaxDevices = 64;
static unsigned long long *g_slab_scratch_ptr[kStaticMaxDevices];        // device address of g_slab_scratch on device i (0: not asked yet)

// the device address of the scratch on the CURRENT device (dev); not thread-safe against a first call on the same
// device from another host thread beyond both storing the same value
static int static_scratch(int dev, unsigned long long **out)
{
    if (dev < 0 || dev >= kStaticMaxDevices) { set_error("nf_slab_histogram_static: device %d outside [0, %d)", dev, kStaticMaxDevices); return NF_ERR_ARG; }
    if (!g_slab_scratch_ptr[dev]) {
        unsigned long long *ptr = nullptr;
        const cudaError_t e = cudaGetSymbolAddress((void **)&ptr, g_slab_scratch);
        if (e != cudaSuccess || !ptr) {
            cudaGetLastError();
            set_error("nf_slab_histogram_static: cudaGetSymbolAddress failed on device %d: %s", dev, cudaGetErrorString(e));
            return NF_ERR_CUDA;
        }
        g_slab_scratch_ptr[dev] = ptr;
    }
    *out = g_slab_scratch_ptr[dev];
    return NF_OK;
}
}  // namespace nf

extern "C" int nf_slab_histogram_static(nf_plan *p, const float *pos, long long n, long long *hist_host)
{
    if (!p || !hist_host || n < 0 || (!pos && n > 0)) { set_error("nf_slab_histogram_static: bad argument"); return NF_ERR_ARG; }
    const int cpd = p->k.cpd;
    if (cpd > kStaticMaxCpd) {
        set_error("nf_slab_histogram_static: cpd = %d exceeds the static scratch (at most %d slabs); use nf_slab_histogram", cpd, kStaticMaxCpd);
        return NF_ERR_ARG;
    }
    for (int s = 0; s < cpd; s++) hist_host[s] = 0;
    if (n == 0) return NF_OK;
    // the plan's device if it has one (bound at its first nf_bin), else the current one; current for the rest of the call
    int cur = -1, prev = -1;
    NF_CUDA_OK(cudaGetDevice(&cur));
    if (p->device >= 0 && p->device != cur) { NF_CUDA_OK(cudaSetDevice(p->device)); prev = cur; cur = p->device; }
    unsigned long long *d = nullptr;
    int rc = nf::static_scratch(cur, &d);
    unsigned long long flag = 0;
    cudaError_t e = cudaSuccess;
    if (rc == NF_OK) {
        cudaStream_t st = p->stream;
        e = cudaMemsetAsync(d, 0, 8 * (size_t)(cpd + 1), st);                   // the array keeps the last call's contents
        if (e == cudaSuccess) {
            const size_t want = ((size_t)n + kSelThreads - 1) / kSelThreads;
            const unsigned grid = (unsigned)(want < 2048 ? want : 2048);
            slab_hist_kernel<<<grid, kSelThreads, 4 * (size_t)cpd, st>>>(pos, (size_t)n, p->k, d, reinterpret_cast<uint32_t *>(d + cpd));
            e = cudaGetLastError();
        }
        // counts are below 2^63: the bits of unsigned long long ARE the caller's long long
        if (e == cudaSuccess) e = cudaMemcpyAsync(hist_host, d, 8 * (size_t)cpd, cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess) e = cudaMemcpyAsync(&flag, d + cpd, 8, cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    }
    if (prev >= 0) cudaSetDevice(prev);
    if (rc != NF_OK) return rc;
    if (e != cudaSuccess) { set_error("nf_slab_histogram_static: %s", cudaGetErrorString(e)); return NF_ERR_CUDA; }
    if (flag & 1ull) { set_error("nf_slab_histogram_static: a coordinate is non-finite or outside [0, L)"); return NF_ERR_DOMAIN; }
    return NF_OK;
}
