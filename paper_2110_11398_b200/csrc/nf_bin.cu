// nf_bin.cu -- steps S1-S5 of the hot path: cell ids, per-cell histogram, prefix
// sums, STABLE counting sort (LSD radix on the cell id, 8 bits per pass), gather into the
// cell-padded SoA source arrays, work-unit list with heavy-first order, exact interaction count.
//
// The paper's analogues are the CPU stages "Transpose Positions" and "Index Near Force Pencils"
// (Table 6), which repack positions and build the indexing
// structures for the GPU near-field work.  Here they are HBM-bound GPU passes (< 1 % of a step).
//
// Layout produced for the direct-sum kernel:
//   x[], y[], z[]  float32 SoA, cell-contiguous, cells in id order (x slowest, z fastest),
//                  each cell padded to a multiple of 4 slots (16-byte TMA granularity) with a dummy
//                  at 2^55 that contributes exactly 0;
//                  values are (pos - corner(cell)) * 2^k: cell-corner-relative, power-of-two scaled so
//                  the cell width is in [1,2).  Both steps are exact in float32 (Sterbenz), so no
//                  information of the input is lost and periodic wraps need no special case.
#include "nf_internal.h"

namespace nf {

// ------------------------------------------------------------------------------------------
// block-wide exclusive scan of one uint32 per thread (blockDim.x <= 1024, multiple of 32)
__device__ __forceinline__ uint32_t block_exclusive_scan(uint32_t v, uint32_t *total, uint32_t *smem /*[33]*/)
{
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = blockDim.x >> 5;
    uint32_t inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        uint32_t t = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += t;
    }
    if (lane == 31) smem[w] = inc;
    __syncthreads();
    if (w == 0) {
        uint32_t s = lane < nw ? smem[lane] : 0, si = s;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            uint32_t t = __shfl_up_sync(0xffffffffu, si, o);
            if (lane >= o) si += t;
        }
        smem[lane] = si - s;                 // exclusive warp base
        if (lane == 31) smem[32] = si;       // block total
    }
    __syncthreads();
    uint32_t res = smem[w] + inc - v;
    if (total) *total = smem[32];
    __syncthreads();
    return res;
}

// ---- three-kernel exclusive scan with an element transform -----------------------------------
struct OpId    { __device__ uint32_t operator()(uint32_t v) const { return v; } };
struct OpPad4  { __device__ uint32_t operator()(uint32_t v) const { return (v + 3u) & ~3u; } };

constexpr int kScanThreads = 256, kScanItems = 8, kScanTile = kScanThreads * kScanItems;

template <class Op>
__global__ void __launch_bounds__(kScanThreads) scan_reduce(const uint32_t *in, size_t n, uint32_t *bsum, Op op)
{
    __shared__ uint32_t sm[33];
    size_t base = (size_t)blockIdx.x * kScanTile + (size_t)threadIdx.x * kScanItems;
    uint32_t s = 0;
#pragma unroll
    for (int k = 0; k < kScanItems; k++) if (base + k < n) s += op(in[base + k]);
    uint32_t tot;
    block_exclusive_scan(s, &tot, sm);
    if (threadIdx.x == 0) bsum[blockIdx.x] = tot;
}

__global__ void __launch_bounds__(1024) scan_spine(uint32_t *bsum, uint32_t nb, uint32_t *total_out)
{
    __shared__ uint32_t sm[33];
    uint32_t carry = 0;
    for (uint32_t c0 = 0; c0 < nb; c0 += 1024) {
        uint32_t i = c0 + threadIdx.x;
        uint32_t v = i < nb ? bsum[i] : 0, tot;
        uint32_t ex = block_exclusive_scan(v, &tot, sm);
        if (i < nb) bsum[i] = carry + ex;
        carry += tot;
    }
    if (threadIdx.x == 0 && total_out) *total_out = carry;
}

// out[i] = exclusive prefix; out[n] = total when write_total (in may alias out)
template <class Op>
__global__ void __launch_bounds__(kScanThreads) scan_apply(const uint32_t *in, uint32_t *out, size_t n,
                                                            const uint32_t *bsum, Op op, int write_total)
{
    __shared__ uint32_t sm[33];
    size_t base = (size_t)blockIdx.x * kScanTile + (size_t)threadIdx.x * kScanItems;
    uint32_t v[kScanItems], s = 0;
#pragma unroll
    for (int k = 0; k < kScanItems; k++) { v[k] = (base + k < n) ? op(in[base + k]) : 0; s += v[k]; }
    uint32_t run = bsum[blockIdx.x] + block_exclusive_scan(s, nullptr, sm);
#pragma unroll
    for (int k = 0; k < kScanItems; k++) {
        if (base + k < n) {
            out[base + k] = run;
            run += v[k];
            if (write_total && base + k == n - 1) out[n] = run;
        }
    }
}

template <class Op>
static void exclusive_scan(const uint32_t *in, uint32_t *out, size_t n, uint32_t *tmp, Op op, int write_total,
                           uint32_t *total_out, cudaStream_t st, int *launches)
{
    if (n == 0) return;
    uint32_t nb = (uint32_t)((n + kScanTile - 1) / kScanTile);
    scan_reduce<<<nb, kScanThreads, 0, st>>>(in, n, tmp, op);
    scan_spine<<<1, 1024, 0, st>>>(tmp, nb, total_out);
    scan_apply<<<nb, kScanThreads, 0, st>>>(in, out, n, tmp, op, write_total);
    *launches += 3;
}

// ---- S1 + S2: cell id (float64 index formula, reading C6) and histogram ---------------------------
__global__ void __launch_bounds__(256) cellid_kernel(const float *__restrict__ pos, size_t n, Consts k,
                                                     uint32_t *__restrict__ cid, uint32_t *__restrict__ count,
                                                     uint32_t *__restrict__ scalars)
{
    size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const float *p = pos + 3 * i;
    int c[3];
    bool bad = false;
#pragma unroll
    for (int d = 0; d < 3; d++) {
        double x = (double)p[d];
        if (!(x >= 0.0 && x < k.L)) bad = true;        // also catches NaN; +-inf
        int q = (int)floor(x * k.inv_cell_w);
        q = q >= k.cpd ? k.cpd - 1 : (q < 0 ? 0 : q);
        c[d] = q;
    }
    uint32_t id = ((uint32_t)c[0] * k.cpd + c[1]) * k.cpd + c[2];
    cid[i] = id;
    if (bad) atomicOr(&scalars[0], 1u);
    atomicAdd(&count[id], 1u);
}

// ---- S4: stable LSD radix sort of (cell id, input index), 8 bits per pass ------------------------------
__global__ void __launch_bounds__(kSortThreads) radix_hist_kernel(const uint32_t *__restrict__ kin, size_t n, int shift,
                                                                  uint32_t *__restrict__ hist, uint32_t nblocks)
{
    __shared__ uint32_t h[256];
    h[threadIdx.x] = 0;
    __syncthreads();
    size_t base = (size_t)blockIdx.x * kSortTile;
#pragma unroll 4
    for (int r = 0; r < kSortItems; r++) {
        size_t e = base + (size_t)r * kSortThreads + threadIdx.x;
        if (e < n) atomicAdd(&h[(kin[e] >> shift) & 255u], 1u);
    }
    __syncthreads();
    hist[(size_t)threadIdx.x * nblocks + blockIdx.x] = h[threadIdx.x];
}

// Each warp owns a contiguous 512-key segment of the block's tile and ranks it in input order with
// match_any, so the scatter is stable: equal digits keep ascending input position (reading C9).
template <bool IOTA>
__global__ void __launch_bounds__(kSortThreads) radix_scatter_kernel(const uint32_t *__restrict__ kin, const uint32_t *__restrict__ vin,
                                                                     uint32_t *__restrict__ kout, uint32_t *__restrict__ vout,
                                                                     size_t n, int shift, const uint32_t *__restrict__ hist,
                                                                     uint32_t nblocks)
{
    __shared__ uint32_t cnt[kSortWarps][256];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    for (int q = threadIdx.x; q < kSortWarps * 256; q += kSortThreads) (&cnt[0][0])[q] = 0;
    __syncthreads();
    const size_t seg = (size_t)blockIdx.x * kSortTile + (size_t)w * (32 * kSortItems);
    uint32_t key[kSortItems], lr[kSortItems];
    const uint32_t lt = (1u << lane) - 1u;
#pragma unroll
    for (int r = 0; r < kSortItems; r++) {
        size_t e = seg + r * 32 + lane;
        bool valid = e < n;
        key[r] = valid ? kin[e] : 0u;
        uint32_t d = (key[r] >> shift) & 255u;
        uint32_t mask = __match_any_sync(0xffffffffu, valid ? d : (256u + lane));
        uint32_t old = valid ? cnt[w][d] : 0u;
        __syncwarp();
        if (valid && lane == __ffs(mask) - 1) cnt[w][d] = old + __popc(mask);
        __syncwarp();
        lr[r] = old + __popc(mask & lt);
    }
    __syncthreads();
    {
        const int d = threadIdx.x;                               // one digit per thread
        uint32_t run = hist[(size_t)d * nblocks + blockIdx.x];
#pragma unroll
        for (int ww = 0; ww < kSortWarps; ww++) { uint32_t c = cnt[ww][d]; cnt[ww][d] = run; run += c; }
    }
    __syncthreads();
#pragma unroll
    for (int r = 0; r < kSortItems; r++) {
        size_t e = seg + r * 32 + lane;
        if (e < n) {
            uint32_t d = (key[r] >> shift) & 255u;
            uint32_t dst = cnt[w][d] + lr[r];
            kout[dst] = key[r];
            vout[dst] = IOTA ? (uint32_t)e : vin[e];
        }
    }
}

// one pass; returns launches
static void radix_pass(const uint32_t *kin, const uint32_t *vin, uint32_t *kout, uint32_t *vout, size_t n, int shift,
                       bool iota, uint32_t *hist, uint32_t *scan_tmp, cudaStream_t st, int *launches)
{
    uint32_t nb = (uint32_t)((n + kSortTile - 1) / kSortTile);
    radix_hist_kernel<<<nb, kSortThreads, 0, st>>>(kin, n, shift, hist, nb);
    *launches += 1;
    exclusive_scan(hist, hist, (size_t)256 * nb, scan_tmp, OpId(), 0, nullptr, st, launches);
    if (iota) radix_scatter_kernel<true><<<nb, kSortThreads, 0, st>>>(kin, vin, kout, vout, n, shift, hist, nb);
    else      radix_scatter_kernel<false><<<nb, kSortThreads, 0, st>>>(kin, vin, kout, vout, n, shift, hist, nb);
    *launches += 1;
}

// ---- S4 (second half): gather into the padded, cell-relative, scaled SoA arrays -------------------------
__global__ void __launch_bounds__(256) gather_kernel(const float *__restrict__ pos, size_t n, Consts k,
                                                     const uint32_t *__restrict__ skey, const uint32_t *__restrict__ perm,
                                                     const uint32_t *__restrict__ offset, const uint32_t *__restrict__ poff,
                                                     float *__restrict__ X, float *__restrict__ Y, float *__restrict__ Z)
{
    size_t s = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= n) return;
    const uint32_t c = skey[s];
    const size_t i = perm[s];
    const uint32_t cz = c % k.cpd, cy = (c / k.cpd) % k.cpd, cx = c / (k.cpd * k.cpd);
    // corner origins are float32 values; pos - origin is exact (Sterbenz), the power-of-two scale too
    const float ox = (float)((double)cx * k.cell_w), oy = (float)((double)cy * k.cell_w), oz = (float)((double)cz * k.cell_w);
    const float sc = (float)k.scale;
    const uint32_t o0 = offset[c], o1 = offset[c + 1];
    const uint32_t p = poff[c] + (uint32_t)(s - o0);
    X[p] = (pos[3 * i + 0] - ox) * sc;
    Y[p] = (pos[3 * i + 1] - oy) * sc;
    Z[p] = (pos[3 * i + 2] - oz) * sc;
    if (s + 1 == o1) {
        const uint32_t pe = poff[c + 1];
        for (uint32_t q = p + 1; q < pe; q++) { X[q] = kDummy; Y[q] = kDummy; Z[q] = kDummy; }
    }
}

// ---- S5: stencil source counts, work units, cost keys, exact interaction count -------------------------------
// src[c] = particles in the (2R+1)^3 periodic stencil of cell c; interactions = sum_c count[c] * src[c].
__global__ void __launch_bounds__(256) cellcost_kernel(Consts k, const uint32_t *__restrict__ count,
                                                       uint32_t *__restrict__ src_out,
                                                       unsigned long long *__restrict__ interactions)
{
    __shared__ unsigned long long red[8];
    const uint32_t c = blockIdx.x * blockDim.x + threadIdx.x;
    unsigned long long mine = 0;
    if (c < k.ncells) {
        const int cpd = k.cpd, R = k.R;
        const int cz = c % cpd, cy = (c / cpd) % cpd, cx = c / (cpd * cpd);
        uint32_t src = 0;                        // <= n < 2^32
        for (int ox = -R; ox <= R; ox++) {
            int sx = cx + ox; sx += sx < 0 ? cpd : 0; sx -= sx >= cpd ? cpd : 0;
            for (int oy = -R; oy <= R; oy++) {
                int sy = cy + oy; sy += sy < 0 ? cpd : 0; sy -= sy >= cpd ? cpd : 0;
                const uint32_t row = ((uint32_t)sx * cpd + sy) * cpd;
                for (int oz = -R; oz <= R; oz++) {
                    int sz = cz + oz; sz += sz < 0 ? cpd : 0; sz -= sz >= cpd ? cpd : 0;
                    src += count[row + sz];
                }
            }
        }
        src_out[c] = src;
        int rel = cx - k.slab0; rel += rel < 0 ? cpd : 0;
        if (rel < k.nslab) mine = (unsigned long long)count[c] * src;      // sinks of the owned slabs only
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) mine += __shfl_down_sync(0xffffffffu, mine, o);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = mine;
    __syncthreads();
    if (threadIdx.x == 0) {
        unsigned long long t = 0;
        for (int w = 0; w < 8; w++) t += red[w];
        if (t) atomicAdd(interactions, t);
    }
}

// work units per z-column: windows of kChunk consecutive cell-sorted sinks
__global__ void __launch_bounds__(256) colunits_kernel(Consts k, const uint32_t *__restrict__ offset,
                                                       uint32_t *__restrict__ nunits)
{
    const uint32_t col = blockIdx.x * blockDim.x + threadIdx.x;
    if (col >= (uint32_t)(k.cpd * k.cpd)) return;
    const uint32_t ncol = offset[(size_t)(col + 1) * k.cpd] - offset[(size_t)col * k.cpd];
    int rel = (int)(col / (uint32_t)k.cpd) - k.slab0; rel += rel < 0 ? k.cpd : 0;
    nunits[col] = rel < k.nslab ? (ncol + kChunk - 1) / kChunk : 0u;            // columns outside the sink slabs: sources only
}

// One thread per column walks its cells once and emits the column's units with their cost keys.
__global__ void __launch_bounds__(128) units_kernel(Consts k, const uint32_t *__restrict__ offset,
                                                    const uint32_t *__restrict__ src, const uint32_t *__restrict__ ubase,
                                                    Unit *__restrict__ units, uint32_t *__restrict__ ukey)
{
    const uint32_t col = blockIdx.x * blockDim.x + threadIdx.x;
    if (col >= (uint32_t)(k.cpd * k.cpd)) return;
    const uint32_t *off = offset + (size_t)col * k.cpd;
    const uint32_t *sc = src + (size_t)col * k.cpd;
    int rel = (int)(col / (uint32_t)k.cpd) - k.slab0; rel += rel < 0 ? k.cpd : 0;
    if (rel >= k.nslab) return;
    const uint32_t c_begin = off[0], c_end = off[k.cpd];
    uint32_t u = ubase[col];
    int z = 0;
    for (uint32_t s0 = c_begin; s0 < c_end; s0 += kChunk, u++) {
        const uint32_t s1 = min(s0 + (uint32_t)kChunk, c_end);
        while (off[z + 1] <= s0) z++;                     // cell holding slot s0 (skips empty cells)
        Unit un;
        un.s0 = s0; un.col = col; un.ns = (uint16_t)(s1 - s0); un.z0 = (uint16_t)z; un.pad_ = 0;
        unsigned long long cost = 0;
        int zz = z;
        for (;;) {
            const uint32_t lo = max(off[zz], s0), hi = min(off[zz + 1], s1);
            cost += (unsigned long long)(hi - lo) * sc[zz];
            if (off[zz + 1] >= s1) break;
            zz++;
        }
        un.z1 = (uint16_t)zz;
        units[u] = un;
        ukey[u] = (uint32_t)__clzll((long long)cost);     // heavier -> smaller key
        z = zz;
    }
}

__global__ void __launch_bounds__(256) units_permute_kernel(const Unit *__restrict__ in, const uint32_t *__restrict__ order,
                                                            const uint32_t *__restrict__ n_units, Unit *__restrict__ out)
{
    uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < *n_units) out[i] = in[order[i]];
}

// ------------------------------------------------------------------------------------------
int launch_bin(nf_plan *p, const float *pos, long long n_ll)
{
    const size_t n = (size_t)n_ll;
    const Consts &k = p->k;
    Workspace &ws = p->ws;
    cudaStream_t st = p->stream;
    int L = 0;
    p->have_bin_time = false;
    p->n_units = 0;
    if (n == 0) { p->launches_bin = 0; p->perm = ws.valA; p->sorted_keys = ws.keyA; return NF_OK; }

    NF_CUDA_OK(cudaEventRecord(p->ev[0], st));
    NF_CUDA_OK(cudaMemsetAsync(ws.count, 0, 4 * (size_t)(k.ncells + 1), st));
    NF_CUDA_OK(cudaMemsetAsync(ws.scalars, 0, 4 * 64, st));
    NF_CUDA_OK(cudaMemsetAsync(ws.interactions, 0, 8, st));

    const unsigned nb256 = (unsigned)((n + 255) / 256);
    cellid_kernel<<<nb256, 256, 0, st>>>(pos, n, k, ws.cid, ws.count, ws.scalars);  L++;

    // prefix sums: offset (exported), padded offsets, unit bases
    exclusive_scan(ws.count, ws.offset, (size_t)k.ncells, ws.scan_tmp, OpId(), 1, nullptr, st, &L);
    exclusive_scan(ws.count, ws.poff, (size_t)k.ncells, ws.scan_tmp, OpPad4(), 1, &ws.scalars[3], st, &L);

    // stable sort by cell id
    int bits = 1;
    while (bits < 32 && (1ull << bits) < (unsigned long long)k.ncells) bits++;
    const int passes = (bits + 7) / 8;
    const uint32_t *kin = ws.cid, *vin = nullptr;
    uint32_t *kbuf[2] = {ws.keyA, ws.keyB}, *vbuf[2] = {ws.valA, ws.valB};
    for (int ps = 0; ps < passes; ps++) {
        radix_pass(kin, vin, kbuf[ps & 1], vbuf[ps & 1], n, 8 * ps, ps == 0, ws.radix_hist, ws.scan_tmp, st, &L);
        kin = kbuf[ps & 1]; vin = vbuf[ps & 1];
    }
    p->sort_passes = passes;
    p->sorted_keys = kin; p->perm = vin;
    uint32_t *free_key = kbuf[passes & 1], *free_val = vbuf[passes & 1];   // the pair not holding the result

    gather_kernel<<<nb256, 256, 0, st>>>(pos, n, k, p->sorted_keys, p->perm, ws.offset, ws.poff, ws.x, ws.y, ws.z);  L++;

    // stencil source counts + exact interaction count, units per column, units + heavy-first order: one
    // stable radix pass on the cost key (clz of the unit's interaction count, so heavier units come first
    // and equal keys keep column order).  The keys sit in the storage of units_sorted until the order is
    // known; the sort writes into the free particle-sort buffers.
    const unsigned nbc = (k.ncells + 255) / 256;
    const uint32_t ncols = (uint32_t)k.cpd * (uint32_t)k.cpd;
    uint32_t *ukey = (uint32_t *)ws.units_sorted;
    cellcost_kernel<<<nbc, 256, 0, st>>>(k, ws.count, ws.src, ws.interactions);  L++;
    colunits_kernel<<<(ncols + 255) / 256, 256, 0, st>>>(k, ws.offset, ws.ubase);  L++;
    exclusive_scan(ws.ubase, ws.ubase, (size_t)ncols, ws.scan_tmp, OpId(), 1, &ws.scalars[2], st, &L);
    units_kernel<<<(ncols + 127) / 128, 128, 0, st>>>(k, ws.offset, ws.src, ws.ubase, ws.units, ukey);  L++;
    NF_CUDA_OK(cudaGetLastError());

    // domain flag + unit count: the one documented synchronisation of nf_bin
    uint32_t sc[4];
    NF_CUDA_OK(cudaMemcpyAsync(sc, ws.scalars, sizeof(sc), cudaMemcpyDeviceToHost, st));
    NF_CUDA_OK(cudaStreamSynchronize(st));
    if (sc[0]) { set_error("nf_bin: a coordinate is non-finite or outside [0, L)"); return NF_ERR_DOMAIN; }
    const size_t nu = sc[2];
    p->n_units = (long long)nu;
    if (p->heavy_first && nu > 1) {
        radix_pass(ukey, nullptr, free_key, free_val, nu, 0, true, ws.radix_hist, ws.scan_tmp, st, &L);
        units_permute_kernel<<<(unsigned)((nu + 255) / 256), 256, 0, st>>>(ws.units, free_val, &ws.scalars[2], ws.units_sorted);  L++;
    } else if (nu > 0) {
        NF_CUDA_OK(cudaMemcpyAsync(ws.units_sorted, ws.units, sizeof(Unit) * nu, cudaMemcpyDeviceToDevice, st));
    }
    NF_CUDA_OK(cudaEventRecord(p->ev[1], st));
    NF_CUDA_OK(cudaGetLastError());
    p->have_bin_time = true;
    p->launches_bin = L;
    return NF_OK;
}

}  // namespace nf
