// nf_bin.cu -- steps S1-S5 of the hot path: cell ids, per-cell histogram, prefix
// sums, STABLE counting sort (LSD radix on the cell id, 1-3 passes of 8-11 bit digits), gather into the
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
struct OpPad2  { __device__ uint32_t operator()(uint32_t v) const { return (v + 1u) & ~1u; } };

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

// One block does the whole scan when it is short (small problems are bound by the number of launches of nf_bin):
// every thread owns kSmallItems consecutive elements; in may alias out.
constexpr int kSmallThreads = 1024, kSmallItems = 16, kSmallMax = kSmallThreads * kSmallItems;

template <class Op>
__device__ __forceinline__ void scan_small_body(const uint32_t *in, uint32_t *out, uint32_t n, Op op, int write_total,
                                                uint32_t *total_out, uint32_t *sm /*[33]*/)
{
    const uint32_t base = threadIdx.x * kSmallItems;
    uint32_t v[kSmallItems], s = 0;
#pragma unroll
    for (int k = 0; k < kSmallItems; k++) { v[k] = (base + k < n) ? op(in[base + k]) : 0; s += v[k]; }
    uint32_t tot;
    uint32_t run = block_exclusive_scan(s, &tot, sm);
#pragma unroll
    for (int k = 0; k < kSmallItems; k++)
        if (base + k < n) { out[base + k] = run; run += v[k]; }
    if (threadIdx.x == 0) {
        if (write_total) out[n] = tot;
        if (total_out) *total_out = tot;
    }
}

template <class Op>
__global__ void __launch_bounds__(kSmallThreads) scan_small(const uint32_t *in, uint32_t *out, uint32_t n, Op op, int write_total,
                                                            uint32_t *total_out)
{
    __shared__ uint32_t sm[33];
    scan_small_body(in, out, n, op, write_total, total_out, sm);
}

// Small problems are bound by the number of launches of nf_bin: the three prefix sums that follow the cell-id kernel
// (cell offsets, padded offsets, the digit histogram of the single sort pass) in one launch.
__global__ void __launch_bounds__(kSmallThreads) small_scans_kernel(const uint32_t *count, uint32_t *offset, uint32_t *poff, uint32_t *voff,
                                                                    uint32_t ncells, uint32_t *hist, uint32_t nhist, uint32_t *padded_total)
{
    __shared__ uint32_t sm[33];
    scan_small_body(count, offset, ncells, OpId(), 1, nullptr, sm);
    __syncthreads();
    scan_small_body(count, poff, ncells, OpPad4(), 1, padded_total, sm);
    __syncthreads();
    scan_small_body(count, voff, ncells, OpPad2(), 1, nullptr, sm);
    __syncthreads();
    scan_small_body(hist, hist, nhist, OpId(), 0, nullptr, sm);
}

template <class Op>
static void exclusive_scan(const uint32_t *in, uint32_t *out, size_t n, uint32_t *tmp, Op op, int write_total,
                           uint32_t *total_out, cudaStream_t st, int *launches)
{
    if (n == 0) return;
    if (n <= (size_t)kSmallMax) {
        scan_small<<<1, kSmallThreads, 0, st>>>(in, out, (uint32_t)n, op, write_total, total_out);
        *launches += 1;
        return;
    }
    uint32_t nb = (uint32_t)((n + kScanTile - 1) / kScanTile);
    scan_reduce<<<nb, kScanThreads, 0, st>>>(in, n, tmp, op);
    scan_spine<<<1, 1024, 0, st>>>(tmp, nb, total_out);
    scan_apply<<<nb, kScanThreads, 0, st>>>(in, out, n, tmp, op, write_total);
    *launches += 3;
}

// ---- S1 + S2: cell id (float64 index formula, reading C6), per-cell histogram, digit histogram of the first sort pass
// One block per sort tile (kSortTile particles), so that the block's digit counts are the column of the first
// pass's histogram matrix and the ids are not read again for it.
__global__ void __launch_bounds__(kSortThreads) cellid_kernel(const float *__restrict__ pos, size_t n, Consts k,
                                                              uint32_t *__restrict__ cid, uint32_t *__restrict__ count,
                                                              uint32_t *__restrict__ scalars, uint32_t digit_mask,
                                                              uint32_t *__restrict__ hist, uint32_t nblocks)
{
    __shared__ uint32_t h[1 << kSortMaxBits];
    for (uint32_t d = threadIdx.x; d <= digit_mask; d += kSortThreads) h[d] = 0;
    __syncthreads();
    const size_t base = (size_t)blockIdx.x * kSortTile;
    bool bad = false;
#pragma unroll 4
    for (int r = 0; r < kSortItems; r++) {
        const size_t i = base + (size_t)r * kSortThreads + threadIdx.x;
        if (i >= n) break;
        const float *p = pos + 3 * i;
        int c[3];
#pragma unroll
        for (int d = 0; d < 3; d++) {
            double x = (double)p[d];
            if (!(x >= 0.0 && x < k.L)) bad = true;        // also catches NaN; +-inf
            int q = (int)floor(x * k.inv_cell_w);
            q = q >= k.cpd ? k.cpd - 1 : (q < 0 ? 0 : q);
            c[d] = q;
        }
        const uint32_t id = ((uint32_t)c[0] * k.cpd + c[1]) * k.cpd + c[2];
        cid[i] = id;
        atomicAdd(&count[id], 1u);
        atomicAdd(&h[id & digit_mask], 1u);
    }
    if (bad) atomicOr(&scalars[0], 1u);
    __syncthreads();
    for (uint32_t d = threadIdx.x; d <= digit_mask; d += kSortThreads) hist[(size_t)d * nblocks + blockIdx.x] = h[d];
}

// ---- S4: stable LSD radix sort of (cell id, input index), 8-11 bits per pass, gather fused into the last pass -------
// n_dev != NULL: the number of keys lives on the device (the unit sort: nf_bin does not read it back before the sort; the
// grid is sized from the host-side bound and blocks past the end write empty histograms)
__global__ void __launch_bounds__(kSortThreads) radix_hist_kernel(const uint32_t *__restrict__ kin, size_t n, int shift,
                                                                  uint32_t digit_mask, uint32_t *__restrict__ hist,
                                                                  uint32_t nblocks, const uint32_t *__restrict__ n_dev)
{
    __shared__ uint32_t h[1 << kSortMaxBits];
    if (n_dev) n = *n_dev;
    for (uint32_t d = threadIdx.x; d <= digit_mask; d += kSortThreads) h[d] = 0;
    __syncthreads();
    const size_t base = (size_t)blockIdx.x * kSortTile;
#pragma unroll 4
    for (int r = 0; r < kSortItems; r++) {
        const size_t e = base + (size_t)r * kSortThreads + threadIdx.x;
        if (e < n) atomicAdd(&h[(kin[e] >> shift) & digit_mask], 1u);
    }
    __syncthreads();
    for (uint32_t d = threadIdx.x; d <= digit_mask; d += kSortThreads) hist[(size_t)d * nblocks + blockIdx.x] = h[d];
}

// What the last pass needs to write the cell-padded SoA source arrays instead of sorted keys (S4, second half):
// values are (pos - corner(cell)) * 2^k; both steps are exact in float32 (Sterbenz), see the file header.
struct GatherArgs {
    const float *pos;
    const uint32_t *offset, *poff;
    float *X, *Y, *Z;
    Consts k;
};

// One pass.  Each warp owns a contiguous 512-key segment of the block's tile and ranks it in input order with
// match_any, so the pass is stable: equal digits keep ascending input position (reading C9).  The tile is then put
// in digit order in shared memory so that consecutive threads write consecutive destinations.
//   IOTA: the values are the positions themselves (first pass);
//   LAST: the keys are whole cell ids in their final order: write perm and the padded SoA arrays, no keys.
// Lanes of the warp that hold the same BITS-bit digit as the caller (only valid lanes are counted; the result of an
// invalid lane is unused).  One ballot per bit: MATCH.ANY takes time in proportion to the number of distinct values
// in the warp, which for 9-11 bit digits of unsorted keys is nearly 32 (measured: half of the stall samples of a pass).
template <int BITS>
__device__ __forceinline__ uint32_t match_digit(const uint32_t d, const bool valid)
{
    uint32_t m = __ballot_sync(0xffffffffu, valid);
#pragma unroll
    for (int b = 0; b < BITS; b++) {
        const uint32_t bit = (d >> b) & 1u;
        m &= __ballot_sync(0xffffffffu, bit) ^ (bit - 1u);
    }
    return m;
}

constexpr int kRankBatch = 4;      // rounds of the ranking whose shared-memory atomics are in flight together

template <int BITS, bool IOTA, bool LAST>
__global__ void __launch_bounds__(kSortThreads, 2) radix_scatter_kernel(const uint32_t *__restrict__ kin, const uint32_t *__restrict__ vin,
                                                                        uint32_t *__restrict__ kout, uint32_t *__restrict__ vout,
                                                                        size_t n, int shift, const uint32_t *__restrict__ hist,
                                                                        uint32_t nblocks, const GatherArgs g,
                                                                        const uint32_t *__restrict__ n_dev)
{
    if (n_dev) n = *n_dev;
    constexpr int BINS = 1 << BITS;
    constexpr uint32_t MASK = BINS - 1;
    constexpr int DPT = BINS >= kSortThreads ? BINS / kSortThreads : 1;        // digits per thread in the scans
    extern __shared__ __align__(16) unsigned char sort_smem[];
    // [0, 64 KB): per-warp digit counters during ranking, then the reordered tile (keys, values)
    uint16_t (*cnt)[BINS] = reinterpret_cast<uint16_t (*)[BINS]>(sort_smem);
    uint32_t *skey = reinterpret_cast<uint32_t *>(sort_smem);
    uint32_t *sval = skey + kSortTile;
    uint32_t *lbase = sval + kSortTile;                    // first tile-local position of each digit
    uint32_t *gdelta = lbase + BINS;                       // global destination of the digit's first key - lbase
    uint32_t *scan_sm = gdelta + BINS;                     // [33]

    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    {
        uint32_t *z = reinterpret_cast<uint32_t *>(sort_smem);
        for (int q = threadIdx.x; q < kSortWarps * BINS / 2; q += kSortThreads) z[q] = 0;
    }
    const size_t tile0 = (size_t)blockIdx.x * kSortTile;
    if (tile0 >= n) return;                                // only with n_dev: the grid covers the host-side bound
    const size_t seg = tile0 + (size_t)w * (32 * kSortItems);
    uint32_t key[kSortItems], lr[kSortItems / 2];     // ranks / tile-local positions: two 16-bit values per register
#pragma unroll
    for (int r = 0; r < kSortItems / 2; r++) lr[r] = 0;
#pragma unroll
    for (int r = 0; r < kSortItems; r++) {
        const size_t e = seg + r * 32 + lane;
        key[r] = e < n ? kin[e] : 0u;
    }
    __syncthreads();
    // Rank of a key among the keys of its digit in the warp's segment: the lanes holding the digit are found with
    // match_any, the first of them adds their number to the warp's counter of the digit (two 16-bit counters per word;
    // a segment has 512 keys) and hands the old value to the others.  The rounds depend on each other only through
    // the order of the shared-memory atomics of the warp, so their latencies overlap.
    const uint32_t lt = (1u << lane) - 1u;
    uint32_t *cw = reinterpret_cast<uint32_t *>(sort_smem) + w * (BINS / 2);
#pragma unroll
    for (int h = 0; h < kSortItems; h += kRankBatch) {
        uint32_t m[kRankBatch], o[kRankBatch];
#pragma unroll
        for (int r = 0; r < kRankBatch; r++) {
            const bool valid = seg + (h + r) * 32 + lane < n;
            const uint32_t d = (key[h + r] >> shift) & MASK;
            m[r] = match_digit<BITS>(d, valid);
        }
#pragma unroll
        for (int r = 0; r < kRankBatch; r++) {
            const bool valid = seg + (h + r) * 32 + lane < n;
            const uint32_t d = (key[h + r] >> shift) & MASK;
            o[r] = 0;
            if (valid && (m[r] & lt) == 0) o[r] = atomicAdd(&cw[d >> 1], (uint32_t)__popc(m[r]) << ((d & 1u) * 16));
        }
#pragma unroll
        for (int r = 0; r < kRankBatch; r++) {
            const uint32_t d = (key[h + r] >> shift) & MASK;
            const uint32_t old = (__shfl_sync(0xffffffffu, o[r], __ffs(m[r]) - 1) >> ((d & 1u) * 16)) & 0xffffu;
            lr[(h + r) >> 1] |= (old + __popc(m[r] & lt)) << (((h + r) & 1) * 16);
        }
    }
    __syncthreads();
    {
        // per digit: exclusive scan over the warps; then the block-wide exclusive scan of the digit totals
        const int d0 = threadIdx.x * DPT;
        uint32_t tot[DPT], s = 0;
#pragma unroll
        for (int q = 0; q < DPT; q++) {
            uint32_t run = 0;
            if (d0 + q < BINS) {
#pragma unroll
                for (int ww = 0; ww < kSortWarps; ww++) { const uint32_t c = cnt[ww][d0 + q]; cnt[ww][d0 + q] = (uint16_t)run; run += c; }
            }
            tot[q] = run; s += run;
        }
        uint32_t ex = block_exclusive_scan(s, nullptr, scan_sm);
#pragma unroll
        for (int q = 0; q < DPT; q++) {
            if (d0 + q < BINS) {
                lbase[d0 + q] = ex;
                gdelta[d0 + q] = hist[(size_t)(d0 + q) * nblocks + blockIdx.x] - ex;
                ex += tot[q];
            }
        }
    }
    __syncthreads();
#pragma unroll
    for (int r = 0; r < kSortItems; r++) {
        const uint32_t d = (key[r] >> shift) & MASK;
        lr[r >> 1] += (lbase[d] + cnt[w][d]) << ((r & 1) * 16);     // tile-local position in digit order (< 8192)
    }
    __syncthreads();                                       // the counters are dead: their storage takes the tile
#pragma unroll
    for (int r = 0; r < kSortItems; r++) {
        const size_t e = seg + r * 32 + lane;
        const uint32_t lp = (lr[r >> 1] >> ((r & 1) * 16)) & 0xffffu;
        if (e < n) { skey[lp] = key[r]; sval[lp] = IOTA ? (uint32_t)e : vin[e]; }
    }
    __syncthreads();
    const uint32_t tile_n = (uint32_t)(n - tile0 < (size_t)kSortTile ? n - tile0 : (size_t)kSortTile);
    if (!LAST) {
#pragma unroll 4
        for (int r = 0; r < kSortItems; r++) {
            const uint32_t i = r * kSortThreads + threadIdx.x;
            if (i < tile_n) {
                const uint32_t c = skey[i];
                const uint32_t dst = gdelta[(c >> shift) & MASK] + i;
                kout[dst] = c;
                vout[dst] = sval[i];
            }
        }
    } else {
        // The 12 bytes of a particle sit anywhere in the input: the 96 floats of 32 consecutive sorted particles are
        // fetched by the warp as 3 loads in which adjacent lanes read adjacent floats of one particle (a request touches
        // ~14 sectors instead of 32) and handed to the owning lanes through shared memory.
        float *xyz = reinterpret_cast<float *>(scan_sm + 40) + w * 96;
        const Consts &k = g.k;
        const float sc = (float)k.scale;
        auto fetch = [&](int r, float (&f)[3]) {                       // the warp's loads of round r
            const uint32_t i0 = r * kSortThreads + w * 32;
#pragma unroll
            for (int j = 0; j < 3; j++) {
                const uint32_t flat = j * 32 + lane, q = flat / 3u, comp = flat - 3u * q;
                f[j] = (r < kSortItems && i0 + q < tile_n) ? __ldg(g.pos + 3 * (size_t)sval[i0 + q] + comp) : 0.f;
            }
        };
        float fa[3], fb[3];
        fetch(0, fa);
        fetch(1, fb);
        for (int r = 0; r < kSortItems; r++) {
            const uint32_t i0 = r * kSortThreads + w * 32;           // warp-uniform
            if (i0 >= tile_n) break;
            const uint32_t i = i0 + lane;
            const bool valid = i < tile_n;
            const uint32_t c = valid ? skey[i] : 0u, v = valid ? sval[i] : 0u;
#pragma unroll
            for (int j = 0; j < 3; j++) { xyz[j * 32 + lane] = fa[j]; fa[j] = fb[j]; }
            fetch(r + 2, fb);                                        // two rounds of loads stay in flight
            __syncwarp();
            if (valid) {
                const uint32_t dst = gdelta[(c >> shift) & MASK] + i;
                vout[dst] = v;
                const uint32_t cz = c % k.cpd, cy = (c / k.cpd) % k.cpd, cx = c / (k.cpd * k.cpd);
                // corner origins are float32 values; pos - origin is exact (Sterbenz), the power-of-two scale too
                const float ox = (float)((double)cx * k.cell_w), oy = (float)((double)cy * k.cell_w), oz = (float)((double)cz * k.cell_w);
                const uint32_t o0 = g.offset[c], o1 = g.offset[c + 1];
                const uint32_t p = g.poff[c] + (dst - o0);
                g.X[p] = (xyz[3 * lane + 0] - ox) * sc;
                g.Y[p] = (xyz[3 * lane + 1] - oy) * sc;
                g.Z[p] = (xyz[3 * lane + 2] - oz) * sc;
                if (dst + 1 == o1) {
                    const uint32_t pe = g.poff[c + 1];
                    for (uint32_t q = p + 1; q < pe; q++) { g.X[q] = kDummy; g.Y[q] = kDummy; g.Z[q] = kDummy; }
                }
            }
            __syncwarp();
        }
    }
}

template <int BITS>
static size_t scatter_smem_bytes() { return 8 * (size_t)kSortTile + 8 * ((size_t)1 << BITS) + 4 * 40 + 4 * 96 * kSortWarps; }

template <int BITS, bool IOTA, bool LAST>
static cudaError_t scatter_launch(const uint32_t *kin, const uint32_t *vin, uint32_t *kout, uint32_t *vout, size_t n, int shift,
                                  const uint32_t *hist, uint32_t nb, const GatherArgs &g, cudaStream_t st, const uint32_t *n_dev)
{
    static_assert(2 * kSortWarps * (1 << BITS) <= 8 * kSortTile, "the counters must fit the tile storage");
    auto fn = radix_scatter_kernel<BITS, IOTA, LAST>;
    const size_t smem = scatter_smem_bytes<BITS>();
    cudaError_t e = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    fn<<<nb, kSortThreads, smem, st>>>(kin, vin, kout, vout, n, shift, hist, nb, g, n_dev);
    return cudaGetLastError();
}

template <int BITS>
static cudaError_t scatter_dispatch(bool iota, bool last, const uint32_t *kin, const uint32_t *vin, uint32_t *kout, uint32_t *vout,
                                    size_t n, int shift, const uint32_t *hist, uint32_t nb, const GatherArgs &g, cudaStream_t st,
                                    const uint32_t *n_dev)
{
    if (iota) return last ? scatter_launch<BITS, true, true>(kin, vin, kout, vout, n, shift, hist, nb, g, st, n_dev)
                          : scatter_launch<BITS, true, false>(kin, vin, kout, vout, n, shift, hist, nb, g, st, n_dev);
    return last ? scatter_launch<BITS, false, true>(kin, vin, kout, vout, n, shift, hist, nb, g, st, n_dev)
                : scatter_launch<BITS, false, false>(kin, vin, kout, vout, n, shift, hist, nb, g, st, n_dev);
}

// One pass over n keys: digit histogram per tile (unless the caller already has it), its scan, the scatter.
// `last` (particle sort only) fuses the gather of `g` into the scatter.
static int radix_pass(const uint32_t *kin, const uint32_t *vin, uint32_t *kout, uint32_t *vout, size_t n, int shift, int bits,
                      bool iota, bool last, bool have_hist, const GatherArgs &g, uint32_t *hist, uint32_t *scan_tmp,
                      cudaStream_t st, int *launches, const uint32_t *n_dev = nullptr,   // n_dev: n is an upper bound, the count is on the device
                      bool hist_scanned = false)
{
    const uint32_t nb = (uint32_t)((n + kSortTile - 1) / kSortTile);
    const uint32_t bins = 1u << bits;
    if (!have_hist) {
        radix_hist_kernel<<<nb, kSortThreads, 0, st>>>(kin, n, shift, bins - 1u, hist, nb, n_dev);
        *launches += 1;
    }
    if (!hist_scanned) exclusive_scan(hist, hist, (size_t)bins * nb, scan_tmp, OpId(), 0, nullptr, st, launches);
    cudaError_t e;
    switch (bits) {
    case 8:  e = scatter_dispatch<8>(iota, last, kin, vin, kout, vout, n, shift, hist, nb, g, st, n_dev); break;
    case 9:  e = scatter_dispatch<9>(iota, last, kin, vin, kout, vout, n, shift, hist, nb, g, st, n_dev); break;
    case 10: e = scatter_dispatch<10>(iota, last, kin, vin, kout, vout, n, shift, hist, nb, g, st, n_dev); break;
    default: e = scatter_dispatch<11>(iota, last, kin, vin, kout, vout, n, shift, hist, nb, g, st, n_dev); break;
    }
    NF_CUDA_OK(e);
    *launches += 1;
    return NF_OK;
}

// ---- S5: stencil source counts, work units, cost keys, exact interaction count -------------------------------
// src[c] = particles in the (2R+1)^3 periodic stencil of cell c; interactions = sum_c count[c] * src[c].
__global__ void __launch_bounds__(256) cellcost_kernel(Consts k, const uint32_t *__restrict__ count,
                                                       uint32_t *__restrict__ src_out,
                                                       unsigned long long *__restrict__ interactions, uint32_t *__restrict__ max_count)
{
    __shared__ unsigned long long red[8];
    const uint32_t c = blockIdx.x * blockDim.x + threadIdx.x;
    unsigned long long mine = 0;
    uint32_t cmax = c < k.ncells ? count[c] : 0u;
    cmax = __reduce_max_sync(0xffffffffu, cmax);
    if ((threadIdx.x & 31) == 0 && cmax) atomicMax(max_count, cmax);
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

// work units per z-column: windows of k.chunk consecutive SINK slots (the particles of a column numbered with every cell
// rounded up to an even count, voff: a lane of the direct kernel holds an aligned pair of them, which never straddles two
// cells; only the last slot of a cell with an odd count is an idle sink).
// Length of the next window of a column that has `rem` slots left.  Whole windows of `chunk`; the remainder of a
// column with default windows is cut so that its sink groups (64 slots each) divide the consumer warps: 5-7 groups ->
// 256 slots (4 groups) first, 3 groups -> 128 slots (2 groups) first.  Every window then keeps all the warps of its CTA
// busy (the warps without sinks share the stages, nf_direct.cu); 3, 5, 6 or 7 groups would leave 2-3 of them idle.
__device__ __forceinline__ uint32_t window_len(uint32_t rem, uint32_t chunk)
{
    if (rem >= chunk) return chunk;
    if (chunk == (uint32_t)kChunk && (kConsumerWarps & (kConsumerWarps - 1)) == 0) {
        // the largest power of two of groups below a group count that is not one itself: 3 -> 2, 5..7 -> 4, 9..15 -> 8
        const uint32_t ng = (rem + (uint32_t)kGroup - 1u) / (uint32_t)kGroup;
        if (ng & (ng - 1u)) return (1u << (31 - __clz(ng))) * (uint32_t)kGroup;
    }
    return rem;
}
__device__ __forceinline__ uint32_t windows_in(uint32_t ncol, uint32_t chunk)
{
    uint32_t nw = ncol / chunk, rem = ncol - nw * chunk;
    while (rem) { rem -= window_len(rem, chunk); nw++; }
    return nw;
}

__global__ void __launch_bounds__(256) colunits_kernel(Consts k, const uint32_t *__restrict__ voff,
                                                       uint32_t *__restrict__ nunits)
{
    const uint32_t col = blockIdx.x * blockDim.x + threadIdx.x;
    if (col >= (uint32_t)(k.cpd * k.cpd)) return;
    const uint32_t ncol = voff[(size_t)(col + 1) * k.cpd] - voff[(size_t)col * k.cpd];
    int rel = (int)(col / (uint32_t)k.cpd) - k.slab0; rel += rel < 0 ? k.cpd : 0;
    nunits[col] = rel < k.nslab ? windows_in(ncol, (uint32_t)k.chunk) : 0u;      // columns outside the sink slabs: sources only
}

// One thread per column walks its cells once and emits the column's units with their cost keys.
// The sort key of a unit: clz of its interaction count (heavier -> smaller key, 0..64) with the flat flag above it, so that
// the one stable radix pass on the key also puts the flat units (sparse windows) behind all the others: nf_accel then runs
// the stepped units and the flat units as two launches of two kernel instances, each holding one loop structure only.
__global__ void __launch_bounds__(128) units_kernel(Consts k, const uint32_t *__restrict__ voff, const uint32_t *__restrict__ count,
                                                    const uint32_t *__restrict__ src, const uint32_t *__restrict__ ubase,
                                                    Unit *__restrict__ units, uint32_t *__restrict__ ukey, uint32_t *__restrict__ n_flat)
{
    const uint32_t col = blockIdx.x * blockDim.x + threadIdx.x;
    if (col >= (uint32_t)(k.cpd * k.cpd)) return;
    const uint32_t *off = voff + (size_t)col * k.cpd;
    const uint32_t *cn = count + (size_t)col * k.cpd;
    const uint32_t *sc = src + (size_t)col * k.cpd;
    int rel = (int)(col / (uint32_t)k.cpd) - k.slab0; rel += rel < 0 ? k.cpd : 0;
    if (rel >= k.nslab) return;
    const uint32_t c_begin = off[0], c_end = off[k.cpd];
    uint32_t u = ubase[col], nflat = 0;
    int z = 0;
    for (uint32_t s0 = c_begin, len = 0; s0 < c_end; s0 += len, u++) {
        len = window_len(c_end - s0, (uint32_t)k.chunk);
        const uint32_t s1 = s0 + len;
        while (off[z + 1] <= s0) z++;                     // cell holding slot s0 (skips empty cells)
        Unit un;
        un.v0 = s0; un.col = col; un.nv = (uint16_t)(s1 - s0); un.z0 = (uint16_t)z; un.flat = 0;
        unsigned long long cost = 0;                      // exact pair interactions of the window's real sinks
        int zz = z;
        for (;;) {
            const uint32_t lo = max(off[zz], s0), hi = min(off[zz] + cn[zz], s1);
            if (hi > lo) cost += (unsigned long long)(hi - lo) * sc[zz];
            if (off[zz + 1] >= s1) break;
            zz++;
        }
        un.z1 = (uint16_t)zz;
        // sparse: the cells the window touches hold few slots on average (all their slots, not the part inside the window: the
        // short last window of a dense column is not sparse)
        un.flat = (uint16_t)(off[zz + 1] - off[z] < (uint32_t)k.flat_below * (uint32_t)(zz - z + 1) ? 1 : 0);
        units[u] = un;
        ukey[u] = (uint32_t)__clzll((long long)cost) | ((uint32_t)un.flat << 7);     // heavier -> smaller key; flat units last
        nflat += un.flat;
        z = zz;
    }
    if (nflat) atomicAdd(n_flat, nflat);
}

__global__ void __launch_bounds__(256) units_permute_kernel(const Unit *__restrict__ in, const uint32_t *__restrict__ order,
                                                            const uint32_t *__restrict__ n_units, Unit *__restrict__ out)
{
    uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < *n_units) out[i] = in[order[i]];
}

// ---- optional source masses: mass[perm[s]] into the slot of sorted particle s in the padded SoA layout, pads 0 ------------
__global__ void __launch_bounds__(256) mass_gather_kernel(const float *__restrict__ mass, const uint32_t *__restrict__ perm,
                                                          const uint32_t *__restrict__ cid, const uint32_t *__restrict__ offset,
                                                          const uint32_t *__restrict__ poff, size_t n, float *__restrict__ M)
{
    const size_t s = (size_t)blockIdx.x * 256 + threadIdx.x;
    if (s >= n) return;
    const uint32_t i = perm[s], c = cid[i];
    const uint32_t p = poff[c] + ((uint32_t)s - offset[c]);
    M[p] = mass[i];
    if ((uint32_t)s + 1u == offset[c + 1])
        for (uint32_t q = p + 1; q < poff[c + 1]; q++) M[q] = 0.f;
}

int launch_set_masses(nf_plan *p, const float *mass)
{
    if (p->n == 0) return NF_OK;
    const size_t n = (size_t)p->n;
    mass_gather_kernel<<<(unsigned)((n + 255) / 256), 256, 0, p->stream>>>(mass, p->perm, p->ws.cid, p->ws.offset, p->ws.poff, n, p->mass_soa);
    NF_CUDA_OK(cudaGetLastError());
    return NF_OK;
}

// S5 of a small problem in ONE launch (one block): stencil counts and the exact interaction count, the units of every
// column, heavy-first order by a counting sort on the cost key (not stable: the order of equal keys only matters for L2
// locality, which a problem of this size has anyway; no result depends on the unit order).
constexpr int kSmallCells = 2048, kSmallUnits = 4096;
__global__ void __launch_bounds__(1024) small_units_kernel(Consts k, const uint32_t *__restrict__ count, const uint32_t *__restrict__ voff,
                                                           uint32_t *__restrict__ src_out, unsigned long long *__restrict__ interactions,
                                                           Unit *__restrict__ units, Unit *__restrict__ units_sorted,
                                                           uint32_t *__restrict__ scalars, int heavy_first)
{
    __shared__ uint32_t s_cnt[kSmallCells], s_src[kSmallCells], s_off[kSmallCells + 1], s_col[kSmallCells / 2 + 2], s_hist[66], s_cur[66];
    __shared__ unsigned char s_key[kSmallUnits];
    __shared__ unsigned long long s_inter;
    const int cpd = k.cpd, R = k.R;
    const uint32_t C = k.ncells, ncols = (uint32_t)cpd * cpd;
    uint32_t cmax = 0;
    for (uint32_t c = threadIdx.x; c < C; c += 1024) { s_cnt[c] = count[c]; cmax = max(cmax, s_cnt[c]); }
    cmax = __reduce_max_sync(0xffffffffu, cmax);
    if ((threadIdx.x & 31) == 0 && cmax) atomicMax(&scalars[7], cmax);
    for (uint32_t c = threadIdx.x; c <= C; c += 1024) s_off[c] = voff[c];
    if (threadIdx.x < 66) { s_hist[threadIdx.x] = 0; s_cur[threadIdx.x] = 0; }
    if (threadIdx.x == 0) s_inter = 0;
    __syncthreads();
    unsigned long long mine = 0;
    for (uint32_t c = threadIdx.x; c < C; c += 1024) {
        const int cz = c % cpd, cy = (c / cpd) % cpd, cx = c / (cpd * cpd);
        uint32_t src = 0;
        for (int ox = -R; ox <= R; ox++) {
            int sx = cx + ox; sx += sx < 0 ? cpd : 0; sx -= sx >= cpd ? cpd : 0;
            for (int oy = -R; oy <= R; oy++) {
                int sy = cy + oy; sy += sy < 0 ? cpd : 0; sy -= sy >= cpd ? cpd : 0;
                const uint32_t row = ((uint32_t)sx * cpd + sy) * cpd;
                for (int oz = -R; oz <= R; oz++) {
                    int sz = cz + oz; sz += sz < 0 ? cpd : 0; sz -= sz >= cpd ? cpd : 0;
                    src += s_cnt[row + sz];
                }
            }
        }
        s_src[c] = src;
        src_out[c] = src;
        int rel = cx - k.slab0; rel += rel < 0 ? cpd : 0;
        if (rel < k.nslab) mine += (unsigned long long)s_cnt[c] * src;      // sinks of the owned slabs only
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) mine += __shfl_down_sync(0xffffffffu, mine, o);     // one 64-bit shared atomic per warp, not per cell
    if ((threadIdx.x & 31) == 0 && mine) atomicAdd(&s_inter, mine);
    __syncthreads();
    for (uint32_t col = threadIdx.x; col < ncols; col += 1024) {
        const uint32_t ncol = s_off[(col + 1) * cpd] - s_off[col * cpd];
        int rel = (int)(col / (uint32_t)cpd) - k.slab0; rel += rel < 0 ? cpd : 0;
        s_col[col] = rel < k.nslab ? windows_in(ncol, (uint32_t)k.chunk) : 0u;
    }
    __syncthreads();
    if (threadIdx.x < 32) {                             // exclusive scan of the units per column by one warp
        uint32_t carry = 0;
        for (uint32_t c0 = 0; c0 < ncols; c0 += 32) {
            const uint32_t col = c0 + threadIdx.x;
            const uint32_t v = col < ncols ? s_col[col] : 0u;
            uint32_t inc = v;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) { const uint32_t t = __shfl_up_sync(0xffffffffu, inc, o); if ((int)threadIdx.x >= o) inc += t; }
            if (col < ncols) s_col[col] = carry + inc - v;
            carry += __shfl_sync(0xffffffffu, inc, 31);
        }
        if (threadIdx.x == 0) { s_col[ncols] = carry; scalars[2] = carry; *interactions = s_inter; }
    }
    __syncthreads();
    const uint32_t nu = s_col[ncols];
    for (uint32_t col = threadIdx.x; col < ncols; col += 1024) {
        if (s_col[col + 1] == s_col[col]) continue;
        const uint32_t *off = s_off + (size_t)col * cpd;
        const uint32_t *cn = s_cnt + (size_t)col * cpd, *sc = s_src + (size_t)col * cpd;
        const uint32_t c_begin = off[0], c_end = off[cpd];
        uint32_t u = s_col[col];
        int z = 0;
        for (uint32_t s0 = c_begin, len = 0; s0 < c_end; s0 += len, u++) {
            len = window_len(c_end - s0, (uint32_t)k.chunk);
            const uint32_t s1 = s0 + len;
            while (off[z + 1] <= s0) z++;
            Unit un;
            un.v0 = s0; un.col = col; un.nv = (uint16_t)(s1 - s0); un.z0 = (uint16_t)z; un.flat = 0;
            unsigned long long cost = 0;
            int zz = z;
            for (;;) {
                const uint32_t lo = max(off[zz], s0), hi = min(off[zz] + cn[zz], s1);
                if (hi > lo) cost += (unsigned long long)(hi - lo) * sc[zz];
                if (off[zz + 1] >= s1) break;
                zz++;
            }
            un.z1 = (uint16_t)zz;
            // sparse: the cells the window touches hold few slots on average (all their slots, not the part inside the window: the
        // short last window of a dense column is not sparse)
        un.flat = (uint16_t)(off[zz + 1] - off[z] < (uint32_t)k.flat_below * (uint32_t)(zz - z + 1) ? 1 : 0);
            units[u] = un;
            const uint32_t key = (uint32_t)__clzll((long long)cost);
            s_key[u] = (unsigned char)key;
            atomicAdd(&s_hist[key], 1u);
            z = zz;
        }
    }
    if (!heavy_first) return;
    __syncthreads();
    if (threadIdx.x < 32) {                             // exclusive scan of the 66 key counts
        uint32_t carry = 0;
        for (int c0 = 0; c0 < 66; c0 += 32) {
            const int q = c0 + (int)threadIdx.x;
            const uint32_t v = q < 66 ? s_hist[q] : 0u;
            uint32_t inc = v;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) { const uint32_t t = __shfl_up_sync(0xffffffffu, inc, o); if ((int)threadIdx.x >= o) inc += t; }
            if (q < 66) s_hist[q] = carry + inc - v;
            carry += __shfl_sync(0xffffffffu, inc, 31);
        }
    }
    __syncthreads();
    for (uint32_t u = threadIdx.x; u < nu; u += 1024) {
        const uint32_t key = s_key[u];
        units_sorted[s_hist[key] + atomicAdd(&s_cur[key], 1u)] = units[u];       // each thread re-reads the units it may not have written:
    }                                                                           // the __syncthreads above orders the global writes of the block
}

// ---- S5 on the stream: per-cell stencil counts + exact interaction count, units per column, units, heavy-first order.
// free_key / free_val: two n-sized scratch arrays for the unit sort.
static int launch_units(nf_plan *p, size_t n, uint32_t *free_key, uint32_t *free_val, int *Lp)
{
    const Consts &k = p->k;
    Workspace &ws = p->ws;
    cudaStream_t st = p->stream;
    int &L = *Lp;
    GatherArgs g{};
    // stencil source counts + exact interaction count, units per column, units + heavy-first order: one
    // stable radix pass on the cost key (clz of the unit's interaction count, so heavier units come first
    // and equal keys keep column order).  The keys sit in the storage of units_sorted until the order is
    // known; the sort writes into the free particle-sort buffers.
    const unsigned nbc = (k.ncells + 255) / 256;
    const uint32_t ncols = (uint32_t)k.cpd * (uint32_t)k.cpd;
    uint32_t *ukey = (uint32_t *)ws.units_sorted;
    cellcost_kernel<<<nbc, 256, 0, st>>>(k, ws.count, ws.src, ws.interactions, &ws.scalars[7]);  L++;
    colunits_kernel<<<(ncols + 255) / 256, 256, 0, st>>>(k, ws.voff, ws.ubase);  L++;
    exclusive_scan(ws.ubase, ws.ubase, (size_t)ncols, ws.scan_tmp, OpId(), 1, &ws.scalars[2], st, &L);
    units_kernel<<<(ncols + 127) / 128, 128, 0, st>>>(k, ws.voff, ws.count, ws.src, ws.ubase, ws.units, ukey, &ws.scalars[8]);  L++;
    NF_CUDA_OK(cudaGetLastError());

    // heavy-first order: the unit count stays on the device (scalars[2]); the sort's grids cover the host-side bound
    const size_t ncol_sink = (size_t)k.nslab * k.cpd;
    const size_t pmax = n + (n < (size_t)k.ncells ? n : (size_t)k.ncells);                // sink slots: every non-empty cell adds at most one
    const size_t umax = (n < ncol_sink ? n : ncol_sink) + pmax / (size_t)(k.chunk < kGroup ? kGroup : k.chunk) + 2 * ncol_sink + 2;
    const size_t ucap = (n < (size_t)ncols ? n : (size_t)ncols) + n / 16 + 2;            // what carve() reserved
    const size_t ub = umax < ucap ? umax : ucap;
    if (p->heavy_first) {
        const int rc = radix_pass(ukey, nullptr, free_key, free_val, ub, 0, kSortMinBits, true, false, false, g, ws.radix_hist,
                                  ws.scan_tmp, st, &L, &ws.scalars[2]);
        if (rc != NF_OK) return rc;
        units_permute_kernel<<<(unsigned)((ub + 255) / 256), 256, 0, st>>>(ws.units, free_val, &ws.scalars[2], ws.units_sorted);  L++;
    }
    return NF_OK;
}

// ------------------------------------------------------------------------------------------
int launch_bin(nf_plan *p, const float *pos, long long n_ll)
{
    const size_t n = (size_t)n_ll;
    // sink slots per work unit: the caller's window, else kChunk -- except for a problem so small that its units would not
    // fill the grid of persistent CTAs: there the longest of 512, 256, 128, 64 that still gives every CTA slot a unit (the
    // consumer warps of a short window share its stages, nf_direct.cu).
    p->k.chunk = kChunk;
    if (p->window > 0) p->k.chunk = p->window;
    else if (n_ll > 0) {
        const double cols = (double)p->k.nslab * p->k.cpd;
        const double per_col = 1.01 * (double)n_ll / ((double)p->k.cpd * p->k.cpd);      // sink slots, roughly
        const double slots = (double)p->sm_count * kMinCtasPerSm;
        int w = kChunk;
        while (w > kGroup && cols * std::ceil(per_col / w) < slots) w >>= 1;    // sink-group counts that divide the consumer warps
        p->k.chunk = w;
    }
    const Consts &k = p->k;
    Workspace &ws = p->ws;
    cudaStream_t st = p->stream;
    int L = 0;
    p->have_bin_time = false;
    p->n_units = 0;
    if (n == 0) { p->launches_bin = 0; p->perm = ws.valA; return NF_OK; }

    NF_CUDA_OK(cudaEventRecord(p->ev[0], st));
    // count, interactions and scalars are carved next to each other: one memset
    NF_CUDA_OK(cudaMemsetAsync(ws.count, 0, (size_t)((char *)(ws.scalars + 64) - (char *)ws.count), st));

    // stable sort by cell id: the first pass's digit histogram comes out of the cell-id kernel, the last pass writes
    // perm and the padded SoA arrays (no sorted keys are stored)
    int passes = 1, dbits = kSortMinBits;
    sort_plan((unsigned long long)k.ncells, &passes, &dbits);
    const uint32_t nbs = (uint32_t)((n + kSortTile - 1) / kSortTile);
    cellid_kernel<<<nbs, kSortThreads, 0, st>>>(pos, n, k, ws.cid, ws.count, ws.scalars, (1u << dbits) - 1u, ws.radix_hist, nbs);  L++;

    // A small problem is bound by the NUMBER of launches (config 1: 0.137 ms for ~20 of them, as long as its nf_accel):
    // one launch for the three prefix sums, one for the whole of S5 -- five stream operations in all.
    const size_t pmax_small = n + 3 * (n < (size_t)k.ncells ? n : (size_t)k.ncells);
    const bool small = passes == 1 && k.ncells <= (uint32_t)kSmallCells && ((size_t)nbs << dbits) <= (size_t)kSmallMax &&
                       pmax_small / kGroup + 3 * (size_t)k.cpd * k.cpd + 2 <= (size_t)kSmallUnits;
    // prefix sums: offset (exported), padded offsets, unit bases
    if (small) {
        small_scans_kernel<<<1, kSmallThreads, 0, st>>>(ws.count, ws.offset, ws.poff, ws.voff, k.ncells, ws.radix_hist, nbs << dbits, &ws.scalars[3]);  L++;
    } else {
        exclusive_scan(ws.count, ws.offset, (size_t)k.ncells, ws.scan_tmp, OpId(), 1, nullptr, st, &L);
        exclusive_scan(ws.count, ws.poff, (size_t)k.ncells, ws.scan_tmp, OpPad4(), 1, &ws.scalars[3], st, &L);
        exclusive_scan(ws.count, ws.voff, (size_t)k.ncells, ws.scan_tmp, OpPad2(), 1, nullptr, st, &L);
    }

    GatherArgs g;
    g.pos = pos; g.offset = ws.offset; g.poff = ws.poff; g.X = ws.x; g.Y = ws.y; g.Z = ws.z; g.k = k;
    const uint32_t *kin = ws.cid, *vin = nullptr;
    uint32_t *kbuf[2] = {ws.keyA, ws.keyB}, *vbuf[2] = {ws.valA, ws.valB};
    for (int ps = 0; ps < passes; ps++) {
        const int rc = radix_pass(kin, vin, kbuf[ps & 1], vbuf[ps & 1], n, dbits * ps, dbits, ps == 0, ps == passes - 1, ps == 0, g,
                                  ws.radix_hist, ws.scan_tmp, st, &L, nullptr, small);
        if (rc != NF_OK) return rc;
        kin = kbuf[ps & 1]; vin = vbuf[ps & 1];
    }
    p->sort_passes = passes;
    p->perm = vin;
    p->slotcell = nullptr;                                     // materialised by the first nf_rebin
    uint32_t *free_key = kbuf[passes & 1], *free_val = vbuf[passes & 1];   // the pair not holding the result

    if (small) {
        small_units_kernel<<<1, 1024, 0, st>>>(k, ws.count, ws.voff, ws.src, ws.interactions, ws.units, ws.units_sorted, ws.scalars,
                                               p->heavy_first);  L++;
    } else {
        const int rc = launch_units(p, n, free_key, free_val, &L);
        if (rc != NF_OK) return rc;
    }
    NF_CUDA_OK(cudaEventRecord(p->ev[1], st));
    NF_CUDA_OK(cudaGetLastError());
    // domain flag + unit count: the one documented synchronisation of nf_bin, at the END of the call -- nothing is
    // enqueued after it, so the binning is complete on return whatever stream the caller uses next
    uint32_t sc[16];
    NF_CUDA_OK(cudaMemcpyAsync(sc, ws.scalars, sizeof(sc), cudaMemcpyDeviceToHost, st));
    NF_CUDA_OK(cudaStreamSynchronize(st));
    if (sc[0]) { set_error("nf_bin: a coordinate is non-finite or outside [0, L)"); return NF_ERR_DOMAIN; }
    p->n_units = (long long)sc[2];
    p->max_count = sc[7];
    p->n_flat = small || !p->heavy_first ? -1 : (long long)sc[8];   // -1: the unit list is not partitioned (flat units anywhere)
    p->have_bin_time = true;
    p->launches_bin = L;
    return NF_OK;
}


// ==================================================================================================================
// Incremental re-binning (nf_rebin).  The paper's pipeline moves particles to their new cells
// after every drift ("reorders particles into their new cells"; "moving particles to their new cells",
// PAPER.md:353; Table 6 "Finish" / "Merge New Particles"), and a particle drifts much less than a
// cell per step, so almost every particle STAYS in its cell.  Result (cid, count, offset, perm, source arrays, units):
// exactly what nf_bin gives for the new positions -- the stable order inside a cell is ascending input index, so the
// new order of a cell is the merge of its stayers (already ascending in the old order) with its arrivals:
//     new slot of a stayer at old slot s, cell c, index i  =  G(s) + arr_off[c] + #{arrivals of c with index < i}
//     new slot of an arrival (c, i)                        =  arr_off[c] + #{arrivals of c with index < i} + G(s*)
// with G(s) = stayers among the old slots below s, arr_off = exclusive scan of the arrivals per cell, s* = first old
// slot of cell c whose index is >= i (or the end of the cell).  No radix pass: one pass over the input order (cell ids,
// movers), one pass over the old sorted order (G by a decoupled look-back, perm, gather into the source arrays).
__device__ __forceinline__ uint32_t cell_of(const float *p3, const Consts &k, bool &bad)
{
    int c[3];
#pragma unroll
    for (int d = 0; d < 3; d++) {
        const double x = (double)p3[d];
        if (!(x >= 0.0 && x < k.L)) bad = true;
        int q = (int)floor(x * k.inv_cell_w);
        q = q >= k.cpd ? k.cpd - 1 : (q < 0 ? 0 : q);
        c[d] = q;
    }
    return ((uint32_t)c[0] * k.cpd + c[1]) * k.cpd + c[2];
}

// pass 1, input order: new cell ids (reading C6), movers, count deltas, arrivals per cell.  A thread takes 4 consecutive
// particles: 48 contiguous bytes of positions as three 16-byte loads, the four old ids as one.
__global__ void __launch_bounds__(256) rebin_cellid_kernel(const float *__restrict__ pos, size_t n, Consts k, uint32_t *__restrict__ cid,
                                                           uint32_t *__restrict__ count, uint32_t *__restrict__ arr_count,
                                                           uint32_t *__restrict__ mover_list, uint32_t cap,
                                                           uint32_t *__restrict__ moverbits, uint32_t *__restrict__ scalars, int vec)
{
    __shared__ uint32_t s_cnt, s_base;
    if (threadIdx.x == 0) s_cnt = 0;
    __syncthreads();
    const size_t i0 = ((size_t)blockIdx.x * 256 + threadIdx.x) * 4;
    bool bad = false;
    uint32_t moved = 0;                                // bit j: particle i0 + j changed its cell
    uint32_t id[4] = {0, 0, 0, 0};
    if (vec && i0 + 4 <= n) {                          // vec: the caller's array is 16-byte aligned
        const float4 *p4 = reinterpret_cast<const float4 *>(pos + 3 * i0);           // 3 i0 floats = 48 (i0 / 4) bytes: 16-byte aligned
        const float4 v0 = __ldg(p4), v1 = __ldg(p4 + 1), v2 = __ldg(p4 + 2);
        const uint4 old = *reinterpret_cast<const uint4 *>(cid + i0);
        const float c[12] = {v0.x, v0.y, v0.z, v0.w, v1.x, v1.y, v1.z, v1.w, v2.x, v2.y, v2.z, v2.w};
        const uint32_t o[4] = {old.x, old.y, old.z, old.w};
#pragma unroll
        for (int j = 0; j < 4; j++) {
            id[j] = cell_of(c + 3 * j, k, bad);
            if (id[j] != o[j]) { moved |= 1u << j; atomicSub(&count[o[j]], 1u); }
        }
    } else {
        for (int j = 0; j < 4 && i0 + j < n; j++) {
            id[j] = cell_of(pos + 3 * (i0 + j), k, bad);
            const uint32_t old = cid[i0 + j];
            if (id[j] != old) { moved |= 1u << j; atomicSub(&count[old], 1u); }
        }
    }
    // the block reserves its share of the mover list with ONE global atomic (every mover adding to the same counter
    // serialises in L2: 160 000 movers cost 80 us that way)
    uint32_t local = 0;
    if (moved) local = atomicAdd(&s_cnt, (uint32_t)__popc(moved));
    __syncthreads();
    if (threadIdx.x == 0 && s_cnt) s_base = atomicAdd(&scalars[4], s_cnt);
    __syncthreads();
    if (moved) {
        uint32_t q = s_base + local;
#pragma unroll
        for (int j = 0; j < 4; j++) {
            if ((moved >> j) & 1u) {
                cid[i0 + j] = id[j];
                atomicAdd(&count[id[j]], 1u);
                atomicAdd(&arr_count[id[j]], 1u);
                if (q < cap) mover_list[q] = (uint32_t)(i0 + j);
                q++;
            }
        }
    }
    // 8 threads make one 32-bit word of the mover bitmap
    uint32_t word = moved << (4 * (threadIdx.x & 7));
    word |= __shfl_xor_sync(0xffffffffu, word, 1);
    word |= __shfl_xor_sync(0xffffffffu, word, 2);
    word |= __shfl_xor_sync(0xffffffffu, word, 4);
    if ((threadIdx.x & 7) == 0 && i0 < n) moverbits[i0 >> 5] = word;
    if (bad) atomicOr(&scalars[0], 1u);
}

// the movers grouped by their new cell (unordered inside a cell: the lists are short)
__global__ void __launch_bounds__(256) rebin_fill_kernel(const uint32_t *__restrict__ mover_list, uint32_t cap, const uint32_t *__restrict__ scalars,
                                                         const uint32_t *__restrict__ cid, const uint32_t *__restrict__ arr_off,
                                                         uint32_t *__restrict__ arr_cursor, uint32_t *__restrict__ arr_list)
{
    const uint32_t q = blockIdx.x * 256 + threadIdx.x;
    const uint32_t m = min(scalars[4], cap);
    if (q >= m) return;
    const uint32_t i = mover_list[q], c = cid[i];
    const uint32_t at = arr_off[c] + atomicAdd(&arr_cursor[c], 1u);
    if (at < cap) arr_list[at] = i;
}

// sum over the cells of (arrivals)^2: the ranking below compares every arrival of a cell with every other one
__global__ void __launch_bounds__(256) rebin_work_kernel(const uint32_t *__restrict__ arr_count, uint32_t ncells, unsigned long long *__restrict__ work)
{
    const uint32_t c = blockIdx.x * 256 + threadIdx.x;
    unsigned long long w = c < ncells ? (unsigned long long)arr_count[c] * arr_count[c] : 0ull;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) w += __shfl_down_sync(0xffffffffu, w, o);
    if ((threadIdx.x & 31) == 0 && w) atomicAdd(work, w);
}

// every cell's arrivals in ascending input index (the stable order): rank by comparison inside the (short) list
__global__ void __launch_bounds__(256) rebin_rank_kernel(const uint32_t *__restrict__ arr_list, uint32_t cap, uint32_t *__restrict__ scalars,
                                                         const unsigned long long *__restrict__ work, unsigned long long budget,
                                                         const uint32_t *__restrict__ cid, const uint32_t *__restrict__ arr_off,
                                                         const uint32_t *__restrict__ arr_count, uint32_t *__restrict__ arr_sorted)
{
    const uint32_t q = blockIdx.x * 256 + threadIdx.x;
    const uint32_t movers = scalars[4];
    if (movers > cap || *work > budget) { if (q == 0) atomicOr(&scalars[5], 1u); return; }
    if (q >= movers) return;
    const uint32_t i = arr_list[q], c = cid[i];
    const uint32_t a0 = arr_off[c], ac = arr_count[c];
    uint32_t rank = 0;
    for (uint32_t j = 0; j < ac; j++) rank += __ldg(arr_list + a0 + j) < i;
    arr_sorted[a0 + rank] = i;
}

// cell of every sorted slot (once after a full nf_bin; nf_rebin keeps it up to date afterwards)
__global__ void __launch_bounds__(256) slotcell_kernel(const uint32_t *__restrict__ offset, uint32_t ncells, size_t n, uint32_t *__restrict__ slotcell)
{
    const size_t s = (size_t)blockIdx.x * 256 + threadIdx.x;
    if (s >= n) return;
    uint32_t lo = 0, hi = ncells;                      // last c with offset[c] <= s
    while (lo + 1 < hi) {
        const uint32_t mid = (lo + hi) >> 1;
        if (__ldg(offset + mid) <= (uint32_t)s) lo = mid; else hi = mid;
    }
    slotcell[s] = lo;
}

struct RebinArgs {
    const float *pos;
    const uint32_t *perm_old, *slotcell_old, *cid, *moverbits, *arr_off, *arr_count, *arr_list, *offset_old, *offset_new, *poff;
    uint32_t *perm_new, *slotcell_new, *staybits, *wordprefix, *scalars;
    unsigned long long *tile_state;
    float *X, *Y, *Z;
    Consts k;
    size_t n;
    uint32_t cap;
};

// writes particle i (cell c, new sorted slot dst) into the padded SoA source arrays, with the pads after the cell's last particle
__device__ __forceinline__ void rebin_store(const RebinArgs &a, uint32_t c, uint32_t dst, float x, float y, float z)
{
    const Consts &k = a.k;
    const float sc = (float)k.scale;
    const uint32_t cz = c % k.cpd, cy = (c / k.cpd) % k.cpd, cx = c / (k.cpd * k.cpd);
    const float ox = (float)((double)cx * k.cell_w), oy = (float)((double)cy * k.cell_w), oz = (float)((double)cz * k.cell_w);
    const uint32_t o0 = a.offset_new[c], o1 = a.offset_new[c + 1];
    const uint32_t p = a.poff[c] + (dst - o0);
    a.X[p] = (x - ox) * sc;
    a.Y[p] = (y - oy) * sc;
    a.Z[p] = (z - oz) * sc;
    if (dst + 1 == o1) {
        const uint32_t pe = a.poff[c + 1];
        for (uint32_t q = p + 1; q < pe; q++) { a.X[q] = kDummy; a.Y[q] = kDummy; a.Z[q] = kDummy; }
    }
}

// pass 2, old sorted order: one block per tile of kSortTile slots, tiles taken in ticket order (look-back needs the
// earlier tiles to be running).  Each warp owns 512 consecutive slots, 32 per round: a round's ballot IS the stay word.
__global__ void __launch_bounds__(kSortThreads, 2) rebin_merge_kernel(const RebinArgs a)
{
    __shared__ uint32_t s_tile, s_base;
    __shared__ uint32_t s_warp[kSortWarps];
    __shared__ float s_xyz[kSortWarps][96];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    if (threadIdx.x == 0) s_tile = atomicAdd(&a.scalars[6], 1u);
    __syncthreads();
    const uint32_t tile = s_tile;
    const size_t tile0 = (size_t)tile * kSortTile, n = a.n;
    if (tile0 >= n) return;
    if (a.scalars[5]) return;                          // more movers than the merge handles: the host sorts from scratch
    const size_t seg = tile0 + (size_t)w * (32 * kSortItems);
    const uint32_t lt = (1u << lane) - 1u;
    uint32_t idx[kSortItems], cell[kSortItems], wd[kSortItems];
    uint32_t wtot = 0;
#pragma unroll
    for (int r = 0; r < kSortItems; r++) {
        const size_t e = seg + r * 32 + lane;
        const bool valid = e < n;
        idx[r] = valid ? a.perm_old[e] : 0u;
        cell[r] = valid ? a.slotcell_old[e] : 0u;
    }
#pragma unroll
    for (int r = 0; r < kSortItems; r++) {
        const size_t e = seg + r * 32 + lane;
        const bool stay = e < n && !((__ldg(a.moverbits + (idx[r] >> 5)) >> (idx[r] & 31u)) & 1u);
        wd[r] = __ballot_sync(0xffffffffu, stay);
        wtot += __popc(wd[r]);
        if (lane == 0 && seg + r * 32 < n) a.staybits[(seg + r * 32) >> 5] = wd[r];
    }
    if (lane == 0) s_warp[w] = wtot;
    __syncthreads();
    if (threadIdx.x == 0) {
        uint32_t run = 0;
        for (int q = 0; q < kSortWarps; q++) { const uint32_t t = s_warp[q]; s_warp[q] = run; run += t; }
        // decoupled look-back over the tiles: state = flag << 32 | value; flag 1: the tile's own count, 2: inclusive prefix
        volatile unsigned long long *st = a.tile_state;
        uint32_t base = 0;
        if (tile > 0) {
            st[tile] = (1ull << 32) | run;
            for (int t = (int)tile - 1;; t--) {
                unsigned long long v;
                do { v = st[t]; } while ((v >> 32) == 0ull);
                base += (uint32_t)v;
                if ((v >> 32) == 2ull) break;
            }
        }
        st[tile] = (2ull << 32) | (unsigned long long)(base + run);
        s_base = base;
    }
    __syncthreads();
    uint32_t run = s_base + s_warp[w];
    // the warp's three loads of a round: adjacent lanes read adjacent floats of one particle (12-byte gathers touch ~14
    // sectors per request instead of 32), handed to the owning lanes through shared memory
    auto fetch = [&](const uint32_t idr, const uint32_t wdr, float (&f)[3]) {
#pragma unroll
        for (int j = 0; j < 3; j++) {
            const uint32_t flat = j * 32 + lane, q = flat / 3u, comp = flat - 3u * q;
            const uint32_t iq = __shfl_sync(0xffffffffu, idr, q);
            f[j] = ((wdr >> q) & 1u) ? __ldg(a.pos + 3 * (size_t)iq + comp) : 0.f;
        }
    };
    constexpr int kAhead = 4;                          // rounds whose gathers are in flight together
#pragma unroll
    for (int r0 = 0; r0 < kSortItems; r0 += kAhead) {
        if (seg + r0 * 32 >= n) break;                 // warp-uniform
        float f[kAhead][3];
#pragma unroll
        for (int g = 0; g < kAhead; g++) fetch(idx[r0 + g], wd[r0 + g], f[g]);
#pragma unroll
        for (int g = 0; g < kAhead; g++) {
            const int r = r0 + g;
            if (seg + r * 32 >= n) break;
            if (lane == 0) a.wordprefix[(seg + r * 32) >> 5] = run;
#pragma unroll
            for (int j = 0; j < 3; j++) s_xyz[w][j * 32 + lane] = f[g][j];
            __syncwarp();
            if ((wd[r] >> lane) & 1u) {
                const uint32_t i = idx[r], c = cell[r];
                const uint32_t ac = __ldg(a.arr_count + c), a0 = __ldg(a.arr_off + c);
                uint32_t lo = 0, hi = ac;              // arrivals of the cell with a smaller index (the list is ascending)
                while (lo < hi) {
                    const uint32_t mid = (lo + hi) >> 1;
                    if (__ldg(a.arr_list + a0 + mid) < i) lo = mid + 1; else hi = mid;
                }
                const uint32_t dst = run + __popc(wd[r] & lt) + a0 + lo;
                a.perm_new[dst] = i;
                a.slotcell_new[dst] = c;
                rebin_store(a, c, dst, s_xyz[w][3 * lane + 0], s_xyz[w][3 * lane + 1], s_xyz[w][3 * lane + 2]);
            }
            __syncwarp();
            run += __popc(wd[r]);
        }
    }
}

// pass 2b: the arrivals
__global__ void __launch_bounds__(256) rebin_arrivals_kernel(const RebinArgs a)
{
    const uint32_t q = blockIdx.x * 256 + threadIdx.x;
    const uint32_t movers = a.scalars[4];
    if (a.scalars[5] || q >= movers) return;
    const uint32_t i = a.arr_list[q], c = a.cid[i];
    const uint32_t a0 = a.arr_off[c], rank = q - a0;               // the lists are sorted: the position is the rank
    uint32_t lo = a.offset_old[c], hi = a.offset_old[c + 1];       // first old slot of cell c with index >= i
    while (lo < hi) {
        const uint32_t mid = (lo + hi) >> 1;
        if (a.perm_old[mid] < i) lo = mid + 1; else hi = mid;
    }
    const uint32_t stayers_below = (size_t)lo < a.n ? a.wordprefix[lo >> 5] + __popc(a.staybits[lo >> 5] & ((1u << (lo & 31u)) - 1u))
                                                    : (uint32_t)a.n - movers;
    const uint32_t dst = a0 + rank + stayers_below;
    a.perm_new[dst] = i;
    a.slotcell_new[dst] = c;
    const float *p3 = a.pos + 3 * (size_t)i;
    rebin_store(a, c, dst, p3[0], p3[1], p3[2]);
}

int launch_rebin(nf_plan *p, const float *pos)
{
    const size_t n = (size_t)p->n;
    const Consts &k = p->k;
    Workspace &ws = p->ws;
    cudaStream_t st = p->stream;
    // particles that changed cell in the previous call: above 1/16 of them the merge costs more than the sort
    if (p->rebin_movers > (long long)(n / 16)) {
        p->rebin_movers = -1; p->rebin_path = 2;
        return launch_bin(p, pos, p->n);
    }
    int L = 0;
    p->have_bin_time = false;
    p->n_units = 0;
    const uint32_t cap = (uint32_t)(n / 4 + 32);
    const uint32_t *perm_old = p->perm;
    uint32_t *perm_new = perm_old == ws.valA ? ws.valB : ws.valA;
    NF_CUDA_OK(cudaEventRecord(p->ev[0], st));
    if (!p->slotcell) {
        slotcell_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(ws.offset, k.ncells, n, ws.keyA);  L++;
        p->slotcell = ws.keyA;
    }
    const uint32_t *slotcell_old = p->slotcell;
    uint32_t *slotcell_new = slotcell_old == ws.keyA ? ws.keyB : ws.keyA;
    NF_CUDA_OK(cudaMemsetAsync(ws.scalars, 0, 4 * 64, st));
    NF_CUDA_OK(cudaMemsetAsync(ws.interactions, 0, 16, st));
    NF_CUDA_OK(cudaMemsetAsync(ws.arr_count, 0, 4 * (size_t)(k.ncells + 1), st));
    NF_CUDA_OK(cudaMemsetAsync(ws.arr_cursor, 0, 4 * (size_t)(k.ncells + 1), st));
    const size_t ntiles = (n + kSortTile - 1) / kSortTile;
    NF_CUDA_OK(cudaMemsetAsync(ws.tile_state, 0, 8 * (ntiles + 1), st));
    rebin_cellid_kernel<<<(unsigned)((n + 1023) / 1024), 256, 0, st>>>(pos, n, k, ws.cid, ws.count, ws.arr_count, ws.mover_list, cap,
                                                                     ws.moverbits, ws.scalars, ((uintptr_t)pos & 15) == 0);  L++;
    exclusive_scan(ws.arr_count, ws.arr_off, (size_t)k.ncells, ws.scan_tmp, OpId(), 1, nullptr, st, &L);
    exclusive_scan(ws.count, ws.offset_new, (size_t)k.ncells, ws.scan_tmp, OpId(), 1, nullptr, st, &L);
    exclusive_scan(ws.count, ws.poff, (size_t)k.ncells, ws.scan_tmp, OpPad4(), 1, &ws.scalars[3], st, &L);
    exclusive_scan(ws.count, ws.voff, (size_t)k.ncells, ws.scan_tmp, OpPad2(), 1, nullptr, st, &L);
    rebin_fill_kernel<<<(cap + 255) / 256, 256, 0, st>>>(ws.mover_list, cap, ws.scalars, ws.cid, ws.arr_off, ws.arr_cursor, ws.arr_list);  L++;
    // the cells' arrival lists in ascending index: ranked by comparison, sum of (arrivals per cell)^2 operations, bounded by
    // 16 n (a 3e6-particle halo cell that exchanges 1 % of its members costs 9e8); beyond that the host sorts from scratch
    rebin_work_kernel<<<(k.ncells + 255) / 256, 256, 0, st>>>(ws.arr_count, k.ncells, ws.interactions + 1);  L++;
    rebin_rank_kernel<<<(cap + 255) / 256, 256, 0, st>>>(ws.arr_list, cap, ws.scalars, ws.interactions + 1, 16ull * n + 4096, ws.cid,
                                                         ws.arr_off, ws.arr_count, ws.mover_list);  L++;
    RebinArgs a;
    a.pos = pos; a.perm_old = perm_old; a.slotcell_old = slotcell_old; a.cid = ws.cid; a.moverbits = ws.moverbits;
    a.arr_off = ws.arr_off; a.arr_count = ws.arr_count; a.arr_list = ws.mover_list;      // sorted lists (the mover list's storage)
    a.offset_old = ws.offset; a.offset_new = ws.offset_new; a.poff = ws.poff;
    a.perm_new = perm_new; a.slotcell_new = slotcell_new; a.staybits = ws.staybits; a.wordprefix = ws.wordprefix;
    a.scalars = ws.scalars; a.tile_state = ws.tile_state; a.X = ws.x; a.Y = ws.y; a.Z = ws.z; a.k = k; a.n = n; a.cap = cap;
    rebin_merge_kernel<<<(unsigned)ntiles, kSortThreads, 0, st>>>(a);  L++;
    rebin_arrivals_kernel<<<(cap + 255) / 256, 256, 0, st>>>(a);  L++;
    NF_CUDA_OK(cudaGetLastError());
    NF_CUDA_OK(cudaMemcpyAsync(ws.offset, ws.offset_new, 4 * (size_t)(k.ncells + 1), cudaMemcpyDeviceToDevice, st));
    p->perm = perm_new;
    p->slotcell = slotcell_new;
    // the old perm / slot-cell arrays are free now: scratch of the unit sort
    { const int rc = launch_units(p, n, const_cast<uint32_t *>(slotcell_old), const_cast<uint32_t *>(perm_old), &L); if (rc != NF_OK) return rc; }
    NF_CUDA_OK(cudaEventRecord(p->ev[1], st));
    NF_CUDA_OK(cudaGetLastError());
    uint32_t sc[16];
    NF_CUDA_OK(cudaMemcpyAsync(sc, ws.scalars, sizeof(sc), cudaMemcpyDeviceToHost, st));   // the call's one synchronisation, at its end
    NF_CUDA_OK(cudaStreamSynchronize(st));
    if (sc[0]) { set_error("nf_rebin: a coordinate is non-finite or outside [0, L)"); return NF_ERR_DOMAIN; }
    p->rebin_movers = (long long)sc[4];
    if (sc[5] || sc[4] > cap) {                       // more movers (or arrivals into one cell) than the merge handles: sort from scratch
        p->rebin_path = 2;
        return launch_bin(p, pos, p->n);
    }
    p->rebin_path = 1;
    p->n_units = (long long)sc[2];
    p->max_count = sc[7];
    p->n_flat = !p->heavy_first ? -1 : (long long)sc[8];
    p->have_bin_time = true;
    p->launches_bin = L;
    return NF_OK;
}

}  // namespace nf
