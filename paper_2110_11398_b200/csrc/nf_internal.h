// nf_internal.h -- plan state and kernel launchers shared by the three translation units of
// libnf_b200.so.  Nothing here is shared with oracle/.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>
#include <stddef.h>

#include "../../include/nf.h"

namespace nf {

// ---- compile-time shape of the direct-sum kernel -------------------------------------------
constexpr int kMaxR          = 127;               // the column offset travels as a biased byte; cpd >= 2R+1 is the real limit
#ifndef NF_CONSUMER_WARPS
#define NF_CONSUMER_WARPS 8
#endif
#ifndef NF_TILE
#define NF_TILE 1024
#endif
#ifndef NF_STAGES
#define NF_STAGES 5
#endif
#ifndef NF_STAGES_MASS
#define NF_STAGES_MASS 3
#endif
#ifndef NF_MIN_CTAS
#define NF_MIN_CTAS 2
#endif
constexpr int kConsumerWarps = NF_CONSUMER_WARPS; // consumer warps per CTA
constexpr int kGroup         = 64;                // sink slots per warp: every lane holds TWO sinks (an aligned pair of padded slots)
constexpr int kChunk         = kGroup * kConsumerWarps;   // max sink slots per work unit (a window of one z-column): 512
constexpr int kTile          = NF_TILE;           // source slots per pipeline stage (multiple of 4)
constexpr int kStages        = NF_STAGES;         // TMA pipeline depth (three staged arrays)
constexpr int kStagesMass    = NF_STAGES_MASS;    //   with the fourth array of the mass kernels
#ifndef NF_MAX_PIECES
#define NF_MAX_PIECES 40
#endif
constexpr int kMaxPieces     = NF_MAX_PIECES;     // source cells (table entries) per stage
#ifndef NF_QUAD_VOTE_ABOVE
#define NF_QUAD_VOTE_ABOVE 4096
#endif
constexpr unsigned kQuadVoteAbove = NF_QUAD_VOTE_ABOVE;   // fullest cell above this: launch the quad-vote instance of the direct kernel
#ifndef NF_FLAT_BELOW
#define NF_FLAT_BELOW 22
#endif
constexpr int kFlatBelow     = NF_FLAT_BELOW;     // default of the "flat_below" option (padded slots per spanned cell)
constexpr int kAccelThreads  = 32 * (kConsumerWarps + 1);   // + 1 producer warp
constexpr int kMinCtasPerSm  = NF_MIN_CTAS;       // register budget: 65536 / (kMinCtasPerSm * kAccelThreads) per thread
#ifndef NF_WAIT_SLEEP_NS
#define NF_WAIT_SLEEP_NS 400
#endif
constexpr unsigned kWaitSleepNs = NF_WAIT_SLEEP_NS;  // back-off of a waiting warp between mbarrier polls
constexpr float kDummy       = 36028797018963968.0f;        // 2^55: pad-slot coordinate, contributes exactly 0

// ---- radix sort shape ----------------------------------------------------------------------
constexpr int kSortWarps   = 16;
constexpr int kSortThreads = 32 * kSortWarps;
constexpr int kSortItems   = 16;                          // keys per thread
constexpr int kSortTile    = kSortThreads * kSortItems;   // 8192 keys per block
constexpr int kSortMinBits = 8, kSortMaxBits = 11;        // digit width of one pass

// LSD passes and digit width for keys below `nkeys` (cell ids: nkeys = cpd^3): as few passes as 11-bit digits allow,
// the bits spread evenly over them (18 bits: 2 x 9; 21: 2 x 11; 24: 3 x 8)
inline void sort_plan(unsigned long long nkeys, int *passes, int *digit_bits)
{
    int bits = 1;
    while (bits < 32 && (1ull << bits) < nkeys) bits++;
    const int np = (bits + kSortMaxBits - 1) / kSortMaxBits;
    int b = (bits + np - 1) / np;
    if (b < kSortMinBits) b = kSortMinBits;
    *passes = np; *digit_bits = b;
}

struct Unit {            // one work unit: a window of <= kChunk consecutive SINK slots of one z-column.  Sink slots number the
                         // particles of a column with every cell rounded up to an EVEN count (voff): a lane of the direct kernel
                         // holds an aligned pair of them, which never straddles two cells; the odd cell's last slot is an idle sink
    uint32_t v0;         // first sink slot (index into the voff numbering), even
    uint32_t col;        // column id cx * cpd + cy
    uint16_t nv;         // sink slots in the window, even
    uint16_t z0, z1;     // first and last cell (z index) that hold a slot of the window
    uint16_t flat;       // 1: sparse window (few slots per cell): the direct kernel walks a lane's stencil run in one flat loop
};

struct Workspace {       // carved out of one arena; all 256-byte aligned
    uint32_t *cid, *keyA, *keyB, *valA, *valB;   // [n]
    uint32_t *radix_hist;                         // [bins * sort_blocks], digit-major
    uint32_t *count, *offset, *poff, *ubase;      // [C], [C+1], [C+1], [cpd^2+1] (unit base per column)
    uint32_t *voff;                               // [C+1] sink-slot offsets: exclusive scan of the counts rounded up to even
    uint32_t *src;                                // [C] particles in the stencil of each cell
    uint32_t *scan_tmp;                           // block sums
    float *x, *y, *z;                             // [P_max]
    Unit *units, *units_sorted;                   // [U_max]
    uint32_t *bucket_hist;                        // [64] + cursor
    unsigned long long *interactions;             // [1]
    uint32_t *scalars;                            // [64]: 0 error flag, 1 unit counter, 2 n_units, 3 padded total,
                                                  //       4 movers of the last nf_rebin, 5 rebin fallback flag, 6 look-back ticket,
                                                  //       7 particles in the fullest cell, 8 flat units, 9 unit counter of the
                                                  //       second launch of nf_accel
    // incremental re-binning (nf_rebin)
    uint32_t *offset_new;                         // [C+2]
    uint32_t *arr_count, *arr_off, *arr_cursor;   // [C+2] arrivals per cell, their exclusive scan, fill cursors
    uint32_t *mover_list, *arr_list;              // [n/4 + 64] input indices of the movers; the same grouped by new cell
    uint32_t *moverbits;                          // [n/32 + 2] bit i: particle i changed its cell
    uint32_t *staybits, *wordprefix;              // [n/32 + 2] by OLD sorted slot: stays in its cell; stayers before the word
    unsigned long long *tile_state;               // [n/8192 + 2] decoupled look-back of the merge pass
    size_t bytes;
};

struct Consts {          // everything the kernels need about the problem, by value
    int cpd, R;
    int chunk;                      // sink slots per work unit (window of one z-column), 64..kChunk
    int flat_below;                 // windows whose cells hold fewer sink slots on average than this take the flat loop (0: none)
    int slab0, nslab;               // sink slabs: cells with x index in {slab0, ..., slab0 + nslab - 1} mod cpd (default: all)
    uint32_t ncells;
    double L, cell_w, inv_cell_w;   // inv_cell_w = cpd / L
    double scale;                   // power of two with cell_w*scale in [1,2)
    float A, B, C;                  // spline in scaled units: t(r) = A + B r + C r^2
    float tiny;
    int plummer;                    // 1: Plummer law d (r^2 + eps^2)^-3/2 (tiny = eps^2, no spline anywhere)
    int fast_ok;                    // eps_s <= 0.999 cell_w: cells with max-norm offset >= 2 are pure Newtonian
    double out_scale;               // scale^2
    float w_scaled;                 // cell width in scaled units, in [1,2)
    float soft_r2;                  // eps_s^2 (scaled, with a 0.1 % margin): pairs below it take the spline
    float soft_thr2;                // (eps_s + rounding margin)^2 in scaled units: closer faces need the spline body
};

}  // namespace nf

struct nf_plan {
    nf::Consts k;
    double eps;
    int device;
    int sm_count, clock_khz;
    cudaStream_t stream;
    // workspace
    void *arena;  size_t arena_bytes;  bool arena_owned;
    nf::Workspace ws;
    long long ws_n;                 // n the carve-up was made for (-1 = none)
    // state of the last binning
    long long n;  bool binned;
    long long n_units;
    long long n_flat;               // flat units, sorted behind all the others in units_sorted; -1: the list is not partitioned
    int sort_passes;
    const uint32_t *perm;
    const uint32_t *slotcell;       // cell of every sorted slot (nf_rebin keeps it; NULL after a full nf_bin until first needed)
    long long rebin_movers;         // particles that changed cell in the last nf_rebin (-1: unknown)
    int rebin_path;                 // 0: none yet, 1: incremental, 2: full sort
    // optional source masses (nf_set_masses): padded SoA like ws.x, plan-owned, outside the arena
    float *mass_soa; size_t mass_cap; bool have_mass;
    // host-buffer path
    float *pos_stage; float *acc_stage; size_t stage_cap;   // device staging for *_host calls
    // options
    int variant, fastpath, heavy_first, ctas_per_sm, window;
    int quad_vote_opt;              // option "quad_vote": -1 automatic (heavy cells), 0 never, 1 always
    int quad_vote;                  // the choice for the current binning
    unsigned max_count;             // particles in the fullest cell of the current binning
    // stats
    cudaEvent_t ev[4];
    bool have_bin_time, have_accel_time;
    int accel_grid, launches_bin, launches_accel;
};

namespace nf {
void set_error(const char *fmt, ...);
size_t carve(Workspace &ws, void *base, long long n, int cpd);   // base may be NULL (size only)
int  launch_bin(nf_plan *p, const float *pos, long long n);             // S1-S5 (nf_bin.cu)
int  launch_rebin(nf_plan *p, const float *pos);                        // S1-S5 for moved particles of the same set (nf_bin.cu)
int  launch_set_masses(nf_plan *p, const float *mass);                  // masses of the binned particles -> padded SoA (nf_bin.cu)
int  launch_accel(nf_plan *p, float *acc, float *rho, double b, float *vel, double dt, float *amax_cell);   // S6-S7 (nf_direct.cu)
int  accel_max_ctas_per_sm(int variant);
}
#define NF_CUDA_OK(call)                                                                        \
    do {                                                                                        \
        cudaError_t e_ = (call);                                                                \
        if (e_ != cudaSuccess) {                                                                \
            nf::set_error("%s failed: %s (%s:%d)", #call, cudaGetErrorString(e_), __FILE__, __LINE__); \
            return NF_ERR_CUDA;                                                                 \
        }                                                                                       \
    } while (0)
