// nf_api.cu -- the C-ABI of include/nf.h: plan life cycle, workspace, streams, introspection.
// Host logic only; the kernels live in nf_bin.cu (S1-S5) and nf_direct.cu (S6-S7).
#include "nf_internal.h"

#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <new>

namespace nf {

static thread_local char g_err[512] = "";

void set_error(const char *fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
}

static inline size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

// Carve the arena.  Called with base == NULL to get the size only.
size_t carve(Workspace &ws, void *base, long long n, int cpd)
{
    size_t off = 0;
    char *b = (char *)base;
    auto take = [&](size_t bytes) -> void * {
        void *p = b ? (void *)(b + off) : nullptr;
        off = align_up(off + bytes, 256);
        return p;
    };
    const size_t N = (size_t)(n > 0 ? n : 0);
    const size_t C = (size_t)cpd * cpd * cpd;
    const size_t nonempty = N < C ? N : C;
    const size_t pmax = N + 3 * nonempty + 8;
    const size_t ncol = (size_t)cpd * cpd;
    const size_t umax = (N < ncol ? N : ncol) + N / 16 + 2;    // every column ends with one ragged window; the others hold >= 64 of the <= 4 N padded slots
    const size_t nsort = (N + 1 > umax ? N + 1 : umax);          // the unit order reuses the sort buffers
    int sort_passes = 1, sort_bits = kSortMinBits;
    sort_plan((unsigned long long)C, &sort_passes, &sort_bits);
    const size_t hist_particles = ((size_t)1 << sort_bits) * ((N + kSortTile - 1) / kSortTile + 1);
    const size_t hist_units = ((size_t)1 << kSortMinBits) * ((umax + kSortTile - 1) / kSortTile + 1);
    const size_t hist_items = hist_particles > hist_units ? hist_particles : hist_units;
    const size_t scan_items = (hist_items > C + 2 ? hist_items : C + 2);
    ws.cid  = (uint32_t *)take(4 * (N + 1));
    ws.keyA = (uint32_t *)take(4 * nsort);
    ws.keyB = (uint32_t *)take(4 * nsort);
    ws.valA = (uint32_t *)take(4 * nsort);
    ws.valB = (uint32_t *)take(4 * nsort);
    ws.radix_hist = (uint32_t *)take(4 * hist_items);
    ws.count  = (uint32_t *)take(4 * (C + 1));                  // count, interactions, scalars: zeroed by ONE memset (nf_bin.cu)
    ws.interactions = (unsigned long long *)take(8 * 4);
    ws.scalars      = (uint32_t *)take(4 * 64);
    ws.offset = (uint32_t *)take(4 * (C + 2));
    ws.poff   = (uint32_t *)take(4 * (C + 2));
    ws.voff   = (uint32_t *)take(4 * (C + 2));
    ws.ubase  = (uint32_t *)take(4 * (C + 2));
    ws.src    = (uint32_t *)take(4 * (C + 1));
    ws.scan_tmp = (uint32_t *)take(4 * (scan_items / 2048 + 4096));
    ws.x = (float *)take(4 * pmax);
    ws.y = (float *)take(4 * pmax);
    ws.z = (float *)take(4 * pmax);
    ws.units        = (Unit *)take(sizeof(Unit) * umax);
    ws.units_sorted = (Unit *)take(sizeof(Unit) * umax);
    ws.bucket_hist  = (uint32_t *)take(4 * 256);
    ws.offset_new = (uint32_t *)take(4 * (C + 2));
    ws.arr_count  = (uint32_t *)take(4 * (C + 2));
    ws.arr_off    = (uint32_t *)take(4 * (C + 2));
    ws.arr_cursor = (uint32_t *)take(4 * (C + 2));
    ws.mover_list = (uint32_t *)take(4 * (N / 4 + 64));
    ws.arr_list   = (uint32_t *)take(4 * (N / 4 + 64));
    ws.moverbits  = (uint32_t *)take(4 * (N / 32 + 2));
    ws.staybits   = (uint32_t *)take(4 * (N / 32 + 2));
    ws.wordprefix = (uint32_t *)take(4 * (N / 32 + 2));
    ws.tile_state = (unsigned long long *)take(8 * (N / kSortTile + 2));
    ws.bytes = off;
    return off;
}

static int ensure_device(nf_plan *p)
{
    if (p->device >= 0) return NF_OK;
    int dev = 0, cnt = 0;
    cudaError_t e = cudaGetDeviceCount(&cnt);
    if (e != cudaSuccess || cnt == 0) {
        set_error("no CUDA device available (%s); this library has no CPU fallback",
                  e == cudaSuccess ? "device count 0" : cudaGetErrorString(e));
        return NF_ERR_CUDA;
    }
    NF_CUDA_OK(cudaGetDevice(&dev));
    NF_CUDA_OK(cudaDeviceGetAttribute(&p->sm_count, cudaDevAttrMultiProcessorCount, dev));
    NF_CUDA_OK(cudaDeviceGetAttribute(&p->clock_khz, cudaDevAttrClockRate, dev));
    for (int i = 0; i < 4; i++) NF_CUDA_OK(cudaEventCreate(&p->ev[i]));
    p->device = dev;
    return NF_OK;
}

static int ensure_workspace(nf_plan *p, long long n)
{
    Workspace tmp;
    size_t need = carve(tmp, nullptr, n, p->k.cpd);
    if (p->arena && p->arena_bytes >= need) {
        if (p->ws_n != n) { carve(p->ws, p->arena, n, p->k.cpd); p->ws_n = n; }
        return NF_OK;
    }
    if (p->arena && !p->arena_owned) {
        set_error("caller workspace too small: have %zu bytes, need %zu", p->arena_bytes, need);
        return NF_ERR_NOMEM;
    }
    if (p->arena) { cudaFree(p->arena); p->arena = nullptr; p->arena_bytes = 0; }
    void *a = nullptr;
    cudaError_t e = cudaMalloc(&a, need);
    if (e != cudaSuccess) {
        cudaGetLastError();
        set_error("cudaMalloc of %zu workspace bytes failed: %s", need, cudaGetErrorString(e));
        return NF_ERR_NOMEM;
    }
    p->arena = a; p->arena_bytes = need; p->arena_owned = true;
    carve(p->ws, p->arena, n, p->k.cpd);
    p->ws_n = n;
    return NF_OK;
}

static int ensure_stage(nf_plan *p, long long n)
{
    size_t need = (size_t)(n > 0 ? n : 1) * 3 * sizeof(float);
    if (p->stage_cap >= need) return NF_OK;
    if (p->pos_stage) cudaFree(p->pos_stage);
    if (p->acc_stage) cudaFree(p->acc_stage);
    p->pos_stage = p->acc_stage = nullptr; p->stage_cap = 0;
    if (cudaMalloc(&p->pos_stage, need) != cudaSuccess || cudaMalloc(&p->acc_stage, need) != cudaSuccess) {
        cudaGetLastError();
        set_error("cudaMalloc of host-path staging buffers (2 x %zu bytes) failed", need);
        return NF_ERR_NOMEM;
    }
    p->stage_cap = need;
    return NF_OK;
}

// A plan lives on the device that was current at its first nf_bin; later calls made while another device is current
// switch to it for the duration of the call.
struct DeviceGuard {
    int prev = -1;
    explicit DeviceGuard(const nf_plan *p)
    {
        int cur = -1;
        if (p && p->device >= 0 && cudaGetDevice(&cur) == cudaSuccess && cur != p->device && cudaSetDevice(p->device) == cudaSuccess)
            prev = cur;
    }
    ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};

// Softening constants of the pair bodies.  kind 0: the compact spline (readings C2/C3); kind 1: Plummer.
static int set_softening(nf_plan *p, int kind)
{
    Consts &k = p->k;
    const double eps = p->eps, L = k.L;
    const double es = 2.16 * eps * k.scale;       // spline radius in scaled units
    k.w_scaled = (float)(k.cell_w * k.scale);
    if (kind == 1 && eps > 0.0) {
        // d (r^2 + eps^2)^-3/2: the Newtonian body with eps^2 in place of the tiny r^2 offset; the spline never
        // applies (t = 3e38 >= k, and no r^2 is below soft_r2 = 0)
        const double ep = eps * k.scale;
        k.plummer = 1;
        k.tiny = (float)(ep * ep);
        k.A = 3.0e38f; k.B = 0.f; k.C = 0.f;
        k.fast_ok = 1; k.soft_thr2 = 0.f; k.soft_r2 = 0.f;
        return NF_OK;
    }
    k.plummer = 0;
    k.tiny = 1e-36f;
    if (eps == 0.0) {
        k.A = 3.0e38f; k.B = 0.f; k.C = 0.f;      // min(r^-3, 3e38): only r = 0 is capped, and 3e38 * 0 = 0
    } else {
        const double A = 10.0 / (es * es * es), B = -15.0 / (es * es * es * es), C = 6.0 / (es * es * es * es * es);
        if (!(std::fabs(C) < 1e37) || !(std::fabs(B) < 1e37) || !(A < 1e37)) {
            set_error("eps = %g is too small relative to the cell width %g for float32 spline coefficients; use eps = 0", eps, k.cell_w);
            return NF_ERR_ARG;
        }
        k.A = (float)A; k.B = (float)B; k.C = (float)C;
    }
    k.fast_ok = (2.16 * eps <= 0.999 * k.cell_w) ? 1 : 0;
    // cell-relative coordinates carry the float32 rounding of the position and of the corner: <= 2^-23 L each
    const double margin = 4.0 * 1.2e-7 * L * k.scale;
    const double thr = es + margin;
    k.soft_thr2 = (float)(thr * thr * 1.0001);
    k.soft_r2 = (float)(es * es * 1.001 + 1e-30);     // eps = 0: only r = 0 (r^2 = tiny) is below it
    return NF_OK;
}

}  // namespace nf

using namespace nf;

extern "C" {

const char *nf_last_error(void) { return g_err; }

nf_plan *nf_plan_create(int cpd, double L, double eps, int R)
{
    if (R < 0 || R > kMaxR) { set_error("R = %d outside [0, %d]", R, kMaxR); return nullptr; }
    if (cpd < 2 * R + 1) { set_error("cpd = %d < 2R+1 = %d: a cell would appear twice in a stencil", cpd, 2 * R + 1); return nullptr; }
    if ((double)cpd * cpd * cpd >= 4294967296.0) { set_error("cpd^3 >= 2^32"); return nullptr; }
    if (!(L > 0.0) || !std::isfinite(L)) { set_error("L must be positive and finite"); return nullptr; }
    if (!(eps >= 0.0) || !std::isfinite(eps)) { set_error("eps must be >= 0 and finite"); return nullptr; }
    nf_plan *p = new (std::nothrow) nf_plan();
    if (!p) { set_error("out of host memory"); return nullptr; }
    memset(p, 0, sizeof(*p));
    Consts &k = p->k;
    k.cpd = cpd; k.R = R; k.ncells = (uint32_t)cpd * cpd * cpd;
    k.slab0 = 0; k.nslab = cpd; k.chunk = kChunk; k.flat_below = kFlatBelow;
    k.L = L; k.cell_w = L / cpd; k.inv_cell_w = (double)cpd / L;
    int e2 = 0;
    (void)std::frexp(k.cell_w, &e2);              // cell_w = m 2^e2, m in [0.5, 1)
    k.scale = std::ldexp(1.0, 1 - e2);            // cell_w * scale in [1, 2)
    k.out_scale = k.scale * k.scale;
    p->eps = eps;
    if (set_softening(p, 0) != NF_OK) { delete p; return nullptr; }
    p->device = -1;
    p->stream = 0;
    p->ws_n = -1;
    p->variant = 0; p->fastpath = 1; p->heavy_first = 1; p->ctas_per_sm = 0; p->window = 0; p->quad_vote_opt = -1;
    g_err[0] = 0;
    return p;
}

void nf_destroy(nf_plan *p)
{
    if (!p) return;
    if (p->arena && p->arena_owned) cudaFree(p->arena);
    if (p->pos_stage) cudaFree(p->pos_stage);
    if (p->acc_stage) cudaFree(p->acc_stage);
    if (p->mass_soa) cudaFree(p->mass_soa);
    if (p->device >= 0) for (int i = 0; i < 4; i++) cudaEventDestroy(p->ev[i]);
    delete p;
}

int nf_set_stream(nf_plan *p, void *s)
{
    if (!p) { set_error("null plan"); return NF_ERR_ARG; }
    p->stream = (cudaStream_t)s;
    return NF_OK;
}

size_t nf_workspace_bytes(const nf_plan *p, long long n)
{
    if (!p || n < 0) return 0;
    Workspace tmp;
    return carve(tmp, nullptr, n, p->k.cpd);
}

int nf_set_workspace(nf_plan *p, void *dev_ptr, size_t bytes)
{
    if (!p) { set_error("null plan"); return NF_ERR_ARG; }
    if (dev_ptr && ((uintptr_t)dev_ptr & 255)) { set_error("workspace must be 256-byte aligned"); return NF_ERR_ARG; }
    if (p->arena && p->arena_owned) cudaFree(p->arena);
    p->arena = dev_ptr; p->arena_bytes = dev_ptr ? bytes : 0; p->arena_owned = false;
    p->ws_n = -1; p->binned = false;
    return NF_OK;
}

int nf_set_sink_slabs(nf_plan *p, int x_first, int n_slabs)
{
    if (!p) { set_error("null plan"); return NF_ERR_ARG; }
    if (x_first < 0 || x_first >= p->k.cpd || n_slabs < 1 || n_slabs > p->k.cpd) {
        set_error("sink slabs: need 0 <= x_first < cpd and 1 <= n_slabs <= cpd (got %d, %d)", x_first, n_slabs);
        return NF_ERR_ARG;
    }
    p->k.slab0 = x_first; p->k.nslab = n_slabs;
    p->binned = false;                       // the work units depend on it
    return NF_OK;
}

int nf_bin(nf_plan *p, const float *pos, long long n)
{    DeviceGuard guard(p);

    if (!p) { set_error("null plan"); return NF_ERR_ARG; }
    p->binned = false;
    p->have_mass = false;                                       // masses belong to one binning
    if (n < 0) { set_error("n < 0"); return NF_ERR_ARG; }
    if ((double)n + 3.0 * p->k.ncells + 16.0 >= 4294967296.0) { set_error("n + 3 cpd^3 >= 2^32"); return NF_ERR_ARG; }
    if (!pos && n > 0) { set_error("null pos"); return NF_ERR_ARG; }
    int rc = ensure_device(p);
    if (rc) return rc;
    rc = ensure_workspace(p, n);
    if (rc) return rc;
    p->rebin_movers = -1; p->rebin_path = 0;
    rc = launch_bin(p, pos, n);
    if (rc) return rc;
    p->n = n; p->binned = true;
    return NF_OK;
}

int nf_rebin(nf_plan *p, const float *pos)
{    DeviceGuard guard(p);

    if (!p) { set_error("null plan"); return NF_ERR_ARG; }
    if (!p->binned) { set_error("nf_rebin called before a successful nf_bin (options that change the work units need a fresh nf_bin)"); return NF_ERR_STATE; }
    if (!pos && p->n > 0) { set_error("null pos"); return NF_ERR_ARG; }
    p->binned = false;
    p->have_mass = false;                                       // masses belong to one binning
    if (p->n == 0) { p->binned = true; return NF_OK; }
    const int rc = launch_rebin(p, pos);
    if (rc) return rc;
    p->binned = true;
    return NF_OK;
}

int nf_set_masses(nf_plan *p, const float *mass)
{    DeviceGuard guard(p);

    if (!p) { set_error("null plan"); return NF_ERR_ARG; }
    if (!p->binned) { set_error("nf_set_masses called before a successful nf_bin"); return NF_ERR_STATE; }
    if (!mass) { p->have_mass = false; return NF_OK; }          // back to unit masses
    const size_t N = (size_t)p->n, C = (size_t)p->k.ncells;
    const size_t need = 4 * (N + 3 * (N < C ? N : C) + 8);      // padded slots: every non-empty cell adds at most 3
    if (p->mass_cap < need) {
        if (p->mass_soa) cudaFree(p->mass_soa);
        p->mass_soa = nullptr; p->mass_cap = 0;
        if (cudaMalloc(&p->mass_soa, need) != cudaSuccess) {
            cudaGetLastError();
            set_error("cudaMalloc of %zu bytes for the source masses failed", need);
            return NF_ERR_NOMEM;
        }
        p->mass_cap = need;
    }
    const int rc = launch_set_masses(p, mass);
    if (rc) return rc;
    p->have_mass = true;
    return NF_OK;
}

int nf_accel(nf_plan *p, float *acc)
{    DeviceGuard guard(p);

    if (!p) { set_error("null plan"); return NF_ERR_ARG; }
    if (!p->binned) { set_error("nf_accel called before a successful nf_bin"); return NF_ERR_STATE; }
    if (!acc && p->n > 0) { set_error("null acc"); return NF_ERR_ARG; }
    return launch_accel(p, acc, nullptr, 0.0, nullptr, 0.0, nullptr);
}

int nf_accel_density(nf_plan *p, float *acc, float *rho, double b)
{    DeviceGuard guard(p);

    if (!p) { set_error("null plan"); return NF_ERR_ARG; }
    if (!p->binned) { set_error("nf_accel_density called before a successful nf_bin"); return NF_ERR_STATE; }
    if ((!acc || !rho) && p->n > 0) { set_error("null acc or rho"); return NF_ERR_ARG; }
    if (!(b > 0.0) || !std::isfinite(b) || b > p->k.R * p->k.cell_w) {
        set_error("density radius b = %g must be in (0, R cell widths = %g]: the stencil must hold every particle within b",
                  b, p->k.R * p->k.cell_w);
        return NF_ERR_ARG;
    }
    if (p->n == 0) return NF_OK;
    return launch_accel(p, acc, rho, b, nullptr, 0.0, nullptr);
}

int nf_accel_kick(nf_plan *p, float *acc, float *vel, double dt, float *amax_cell)
{    DeviceGuard guard(p);

    if (!p) { set_error("null plan"); return NF_ERR_ARG; }
    if (!p->binned) { set_error("nf_accel_kick called before a successful nf_bin"); return NF_ERR_STATE; }
    if (!acc && !vel && !amax_cell) { set_error("nf_accel_kick: acc, vel and amax_cell are all null"); return NF_ERR_ARG; }
    if (!std::isfinite(dt)) { set_error("dt must be finite"); return NF_ERR_ARG; }
    if (p->n == 0) {
        if (amax_cell) NF_CUDA_OK(cudaMemsetAsync(amax_cell, 0, 4 * (size_t)p->k.ncells, p->stream));
        return NF_OK;
    }
    return launch_accel(p, acc, nullptr, 0.0, vel, dt, amax_cell);
}

int nf_bin_host(nf_plan *p, const float *pos_host, long long n)
{    DeviceGuard guard(p);

    if (!p) { set_error("null plan"); return NF_ERR_ARG; }
    p->binned = false;
    if (n < 0 || (!pos_host && n > 0)) { set_error("bad pos_host / n"); return NF_ERR_ARG; }
    int rc = ensure_device(p);
    if (rc) return rc;
    rc = ensure_stage(p, n);
    if (rc) return rc;
    if (n > 0) NF_CUDA_OK(cudaMemcpyAsync(p->pos_stage, pos_host, (size_t)n * 12, cudaMemcpyHostToDevice, p->stream));
    return nf_bin(p, p->pos_stage, n);
}

int nf_accel_host(nf_plan *p, float *acc_host)
{    DeviceGuard guard(p);

    if (!p) { set_error("null plan"); return NF_ERR_ARG; }
    if (!p->binned) { set_error("nf_accel_host called before a successful nf_bin"); return NF_ERR_STATE; }
    if (!acc_host && p->n > 0) { set_error("null acc_host"); return NF_ERR_ARG; }
    int rc = ensure_stage(p, p->n);
    if (rc) return rc;
    if (p->k.nslab < p->k.cpd && p->n > 0)        // rows outside the sink slabs are not computed: hand back zeros
        NF_CUDA_OK(cudaMemsetAsync(p->acc_stage, 0, (size_t)p->n * 12, p->stream));
    rc = launch_accel(p, p->acc_stage, nullptr, 0.0, nullptr, 0.0, nullptr);
    if (rc) return rc;
    if (p->n > 0) NF_CUDA_OK(cudaMemcpyAsync(acc_host, p->acc_stage, (size_t)p->n * 12, cudaMemcpyDeviceToHost, p->stream));
    NF_CUDA_OK(cudaStreamSynchronize(p->stream));
    return NF_OK;
}

int nf_get_binning(const nf_plan *p, const unsigned **cell_id, const unsigned **count,
                   const unsigned **offset, const unsigned **perm)
{
    if (!p) { set_error("null plan"); return NF_ERR_ARG; }
    if (!p->binned) { set_error("no binning"); return NF_ERR_STATE; }
    if (cell_id) *cell_id = p->ws.cid;
    if (count) *count = p->ws.count;
    if (offset) *offset = p->ws.offset;
    if (perm) *perm = p->perm;
    return NF_OK;
}

int nf_get_layout(const nf_plan *p, const unsigned **poff, const float **x, const float **y,
                  const float **z, double *scale)
{
    if (!p) { set_error("null plan"); return NF_ERR_ARG; }
    if (!p->binned) { set_error("no binning"); return NF_ERR_STATE; }
    if (poff) *poff = p->ws.poff;
    if (x) *x = p->ws.x;
    if (y) *y = p->ws.y;
    if (z) *z = p->ws.z;
    if (scale) *scale = p->k.scale;
    return NF_OK;
}

int nf_get_stats(nf_plan *p, nf_stats *out)
{    DeviceGuard guard(p);

    if (!p || !out) { set_error("null argument"); return NF_ERR_ARG; }
    memset(out, 0, sizeof(*out));
    out->cells = p->k.ncells;
    out->accel_block = kAccelThreads;
    if (p->device < 0) return NF_OK;
    out->sm_count = p->sm_count; out->clock_khz = p->clock_khz;
    out->accel_grid = p->accel_grid;
    out->kernel_launches_bin = p->launches_bin;
    out->kernel_launches_accel = p->launches_accel;
    out->rebin_path = p->rebin_path; out->rebin_movers = p->rebin_movers;
    NF_CUDA_OK(cudaStreamSynchronize(p->stream));
    if (p->binned) {
        out->n = p->n;
        uint32_t sc[4] = {0, 0, 0, 0};
        unsigned long long inter = 0;
        if (p->n > 0) {
            NF_CUDA_OK(cudaMemcpy(sc, p->ws.scalars, sizeof(sc), cudaMemcpyDeviceToHost));
            NF_CUDA_OK(cudaMemcpy(&inter, p->ws.interactions, 8, cudaMemcpyDeviceToHost));
        }
        out->units = sc[2]; out->padded_slots = sc[3]; out->interactions = (long long)inter;
    }
    if (p->have_bin_time) NF_CUDA_OK(cudaEventElapsedTime(&out->ms_bin, p->ev[0], p->ev[1]));
    if (p->have_accel_time) NF_CUDA_OK(cudaEventElapsedTime(&out->ms_accel, p->ev[2], p->ev[3]));
    return NF_OK;
}

int nf_set_option(nf_plan *p, const char *key, long long v)
{
    if (!p || !key) { set_error("null argument"); return NF_ERR_ARG; }
    if (!strcmp(key, "variant") && (v == 0 || v == 1)) { p->variant = (int)v; return NF_OK; }
    if (!strcmp(key, "fastpath") && (v == 0 || v == 1)) { p->fastpath = (int)v; return NF_OK; }
    if (!strcmp(key, "heavy_first") && (v == 0 || v == 1)) { p->heavy_first = (int)v; p->binned = false; return NF_OK; }
    if (!strcmp(key, "softening") && (v == 0 || v == 1)) {
        // 0: the spline of the method; 1: the Plummer comparison law.  eps = 0 is Newtonian either way.
        return set_softening(p, (int)v);
    }
    if (!strcmp(key, "ctas_per_sm") && v >= 0 && v <= 32) { p->ctas_per_sm = (int)v; return NF_OK; }
    if (!strcmp(key, "quad_vote") && v >= -1 && v <= 1) { p->quad_vote_opt = (int)v; return NF_OK; }
    if (!strcmp(key, "flat_below") && v >= 0 && v <= 1024) { p->k.flat_below = (int)v; p->binned = false; return NF_OK; }
    if (!strcmp(key, "window") && v >= 0 && v % 32 == 0 && v <= kChunk) {
        p->window = (int)((v + kGroup - 1) / kGroup * kGroup);     // whole sink groups of 64 slots
        p->binned = false; return NF_OK;
    }
    set_error("unknown option or bad value: %s = %lld", key, v);
    return NF_ERR_ARG;
}

}  // extern "C"
