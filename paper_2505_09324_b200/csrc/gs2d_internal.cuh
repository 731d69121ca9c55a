// gs2d_internal.cuh -- context layout, launch helpers and device records shared by the
// CUDA translation units of libgs2d.  Product code: nothing here is used by oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "gs2d.h"

namespace gs2d {

constexpr int TILE = 16;          // 16x16 screen tiles (BASELINE.json north_star)
constexpr int TILE_PX = TILE * TILE;

// Device record of one Gaussian, written by the preprocess kernel and gathered by the
// rasterizers.  With kappa = sqrt(0.5 * log2(e)):
//   i1 = kappa / l1,  i3 = kappa / l3,  k = -kappa * l2 / (l1 * l3)
//   u = dx * i1,  v = dy * i3 + dx * k,   exp(-sigma) = exp2(-(u*u + v*v))
// which is sigma = 1/2 d^T Sigma^-1 d in the whitened coordinates L^-1 d
// (Eq. 1 gives Sigma = L L^T; DESIGN.md §5 "record").
struct __align__(16) Rec {
    float mux, muy, i1, k;   // lo
    float i3, cr, cg, cb;    // hi : premultiplied colour c' = o * rgb
};

// Per-tile statistics produced by the forward kernel in "stats" mode.
struct __align__(8) TileStats {
    double sq_raw;    // sum (C - T)^2      unclamped, valid pixels x 3 channels
    double sq_clamp;  // sum (clamp(C) - T)^2
    double abs_clamp; // sum |T - clamp(C)|
};

// Device-side status word bits (latched, read by synchronising calls).
constexpr unsigned FLAG_CAPACITY = 1u;
constexpr unsigned FLAG_NONFINITE = 2u;

// Backward work item: entries [begin, begin+count) of `list`, all of tile `tile`.
constexpr int BWD_CHUNK = 32;     // list entries per backward work item
constexpr int BIN_COPIES = 8;     // private copies of the per-tile counters (gs2d_bin.cu)

struct DeviceState {
    unsigned int flags;          // FLAG_*
    int first_nonfinite_iter;    // 1-based, 0 = none
    int n_pairs;                 // P of the last binning (may exceed capacity)
    int n_active;                // result of the last active count
    int n_items;                 // backward work items of the last binning
    int pad1;
    int n_class[4];              // tiles per forward-order class ([0] unused: class 0 is the rest)
    unsigned int item_cursor;    // backward: dynamic work fetch (reset by the scan kernel)
    unsigned int pad0;
    unsigned long long pair_cursor;  // preprocess: running pair count (reset by the scan kernel)
    unsigned long long big_cursor;   // preprocess: overflow pair slots claimed by large rectangles
    double loss_sum;             // reduced sq_raw of the last stats reduction
    double sq_clamp_sum;
    unsigned long long total_in; // ROI init: total inside weight
    unsigned long long total_out;
};

}  // namespace gs2d

struct gs_ctx {
    gs_config cfg;
    int TX, TY, T;
    int device;
    int sm_count;
    long long cap_pairs;

    // binning scratch
    gs2d::Rec *rec;          // [N_max]
    short4 *rect;            // [N_max] tx0,ty0,tx1,ty1 (tx1 < tx0 when culled)
    int *tile_count;         // [BIN_COPIES*T] zero between binnings
    int *range;              // [T+1]
    int *copy_base;          // [BIN_COPIES*T] first list slot of each counter copy's entries
    int *item_off;           // [T+1] first backward work item of each tile
    int *tile_order;         // [4*T] per-class tile lists (class c at c*T); forward walks class 3 first
    unsigned long long *scan_agg;  // [3*ceil(T/256)] scan aggregates + epoch flags
    unsigned scan_epoch;     // stamps the flags of the current binning
    int *list;               // [cap_pairs] Gaussian ids, tile-major, ascending id inside a tile
    int *pair_rank;          // [N_max*32 + cap_pairs] Gaussian-major: arrival rank of the pair inside its tile
    int *pair_base;          // [N_max] overflow slot of Gaussians whose rectangle exceeds 32 tiles
    int2 *items;             // [cap_items] backward work items (tile, chunk index)
    long long cap_items;
    int bwd_grid;            // persistent grid of the backward kernel (0 = not yet queried)
    // raster scratch
    float4 *gtile;           // [T*256] tile-major dL/dC (lazy)
    float *acc;              // [N_max*8] gradient moments, zero between iterations
    gs2d::TileStats *tile_stats;  // [T]
    unsigned char *tile_flag;     // [T]
    float *image_scratch;    // [H*W*3] (lazy; host-buffer entry points)
    // fit scratch
    float *bias_corr;        // [2*max_iters] (lazy, grown on demand)
    int bias_corr_cap;
    float *host_params;      // [N_max*9] device copy for *_host entry points (lazy)
    float *host_frame;       // [H*W*3]
    float *host_m, *host_v;  // [N_max*9]
    float *grad_scratch;     // [N_max*9] (lazy)
    // ROI init scratch (lazy)
    int *roi_grey;           // [H*W]
    unsigned long long *roi_cin, *roi_cout;  // [H*W] inclusive prefix sums
    unsigned long long *roi_blk;             // block sums
    // device state + pinned mirror
    gs2d::DeviceState *dstate;
    gs2d::DeviceState *hstate;  // pinned
    int last_n;                 // n of the last binning
};

namespace gs2d {

void set_cuda_error(cudaError_t e, const char *where);
#define GS_CUDA_TRY(expr)                                   \
    do {                                                    \
        cudaError_t _e = (expr);                            \
        if (_e != cudaSuccess) {                            \
            gs2d::set_cuda_error(_e, #expr);                \
            return GS_ERR_CUDA;                             \
        }                                                   \
    } while (0)

inline int ceil_div(long long a, long long b) { return (int)((a + b - 1) / b); }

// --- launchers implemented in the .cu files (all asynchronous on `s`) ---
// gs2d_bin.cu
// sort: also run the standalone per-tile sort (callers that do not follow up with a forward
// pass, which sorts its own tile on entry).  ev (nullable): 4 events recorded before each of
// preprocess / scan / fill and after fill.
int launch_binning(gs_ctx *c, const gs_params &p, cudaStream_t s, bool sort, cudaEvent_t *ev = nullptr);
// gs2d_raster.cu
enum ForwardMode { FWD_IMAGE = 0, FWD_IMAGE_CLAMP = 1, FWD_FIT = 2, FWD_STATS = 3 };
// sorts each tile's list segment on entry and emits the backward work items
int launch_forward(gs_ctx *c, ForwardMode mode, float *image_out, const float *target, int iter, cudaStream_t s);
int launch_backward(gs_ctx *c, cudaStream_t s);
int launch_repack_grad(gs_ctx *c, const float *dL_dimage, cudaStream_t s);
int launch_reduce_stats(gs_ctx *c, cudaStream_t s);
int ensure_fit_scratch(gs_ctx *c);
// gs2d_optim.cu
int launch_grad_finalize(gs_ctx *c, const gs_params &p, const gs_params &g, cudaStream_t s);
int launch_adam(gs_ctx *c, const gs_params &p, const gs_params *grad /*null: from acc*/, const gs_adam_state &st,
                const float lr[4], float beta1, float beta2, float eps, float bc1, float bc2,
                const unsigned char *active, cudaStream_t s);
// gs2d_select.cu
int launch_select(gs_ctx *c, float tau, unsigned char *active_out, int n, cudaStream_t s);
int launch_tile_resid(gs_ctx *c, double *resid_out, cudaStream_t s);
// gs2d_init.cu
int run_init_roi(gs_ctx *c, const float *frame, const unsigned char *mask, int n, unsigned long long seed,
                 float s_min, float s_max, const gs_params &out, cudaStream_t s);

}  // namespace gs2d
