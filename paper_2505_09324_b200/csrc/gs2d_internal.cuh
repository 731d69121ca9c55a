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

// Backward work item: entries [32 k, 32 k + 32) of the list of tile `tile`.
constexpr int BWD_CHUNK = 32;     // list entries per backward work item

// Device-side counters.  Everything a binning produces is double-buffered by the parity of
// the binning epoch, so that the kernel that consumes epoch e can reset the slot of epoch
// e + 1 while nobody else touches it (no memset launches inside the fit loop).
struct DeviceState {
    unsigned int flags;              // FLAG_* (latched until a synchronising call reads them)
    int first_nonfinite_iter;        // 1-based, 0 = none
    int n_active;                    // result of the last active count
    int pad0;
    unsigned long long pair_total[2];  // [epoch & 1] P = number of (tile, Gaussian) pairs (may exceed capacity)
    int tile_ovf[2];                 // [epoch & 1] != 0: some tile received more than tile_cap entries
    int n_items[2];                  // [epoch & 1] backward work items emitted by the sort stage
    unsigned int item_cursor[2];     // [epoch & 1] backward: dynamic work fetch
    int n_class[3][4];               // [forward launch % 3][class] tiles per forward-order class
    double loss_sum;                 // reduced sq_raw of the last stats reduction
    double sq_clamp_sum;
    unsigned long long total_in;     // ROI init: total inside weight
    unsigned long long total_out;
};

// What a kernel needs to bin one Gaussian (k_bin and the fused Adam kernel).
struct BinArgs {
    float cutoff;
    int W, H, TX, TY;
    int tile_cap;                    // bucket capacity per tile
    int slot;                        // binning epoch & 1
    Rec *rec;                        // [N]
    int *tile_count;                 // [2][T] by epoch parity; the slot's half is zero before the binning
    int *bucket;                     // [T * tile_cap] Gaussian ids, arrival order
    DeviceState *st;
};

// What the per-tile sort stage (the prologue of the forward kernel, or k_sort_tiles) needs.
struct TileArgs {
    int *tile_count;                 // [2][T] by epoch parity: the slot's half is read, the other zeroed
    int *tile_n;                     // [T] list length of the tile (written here)
    int *bucket;                     // [T * tile_cap] sorted in place
    int2 *items;                     // backward work items (appended here when emit != 0)
    int tile_cap;
    int slot;                        // binning epoch & 1
    int emit;                        // emit backward work items
    long long cap_pairs;
    DeviceState *st;
};

}  // namespace gs2d

struct gs_ctx {
    gs_config cfg;
    int TX, TY, T;
    int device;
    int sm_count;
    long long cap_pairs;

    // binning scratch: one bucket of tile_cap ids per tile (gs2d_bin.cu)
    gs2d::Rec *rec;          // [N_max]
    int *tile_count;         // [2][T] arrivals per tile, by epoch parity (the consumer of epoch e zeroes half e+1)
    int *tile_n;             // [T] list length per tile of the last sorted binning
    int *bucket;             // [T * tile_cap] Gaussian ids; ascending inside a tile after the sort stage
    int tile_cap;
    int *tile_order;         // [3][4*T] forward launch order: per-class tile lists (class c at c*T)
    unsigned fwd_launches;   // forward launches so far (selects the order buffer)
    unsigned epoch;          // binning epoch (selects the DeviceState slots)
    int2 *items;             // [cap_items] backward work items (tile, chunk index)
    long long cap_items;
    int bwd_grid;            // persistent grid of the backward kernel (0 = not yet queried)
    // "fresh" bins: a binning whose sort stage has not run yet, and the arrays it was made from
    bool fresh;
    bool sorted;             // the buckets of the last consumed binning are in canonical order
    const float *fresh_mu;
    int fresh_n;
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
// Makes sure the context holds fresh (unsorted) bins of `p`: a no-op when the previous fused
// Adam step of the same arrays left them behind, a k_bin launch otherwise.
int ensure_bins(gs_ctx *c, const gs_params &p, cudaStream_t s);
void discard_fresh_bins(gs_ctx *c, cudaStream_t s);      // drop bins nobody will consume
BinArgs bin_args(gs_ctx *c, bool next_epoch);            // next_epoch: start a new binning epoch
TileArgs tile_args(gs_ctx *c, bool emit);
int launch_sort_tiles(gs_ctx *c, cudaStream_t s);        // consume fresh bins, or sort buckets consumed unsorted
int launch_compact(gs_ctx *c, int *range_out, int *list_out, cudaStream_t s);
// gs2d_raster.cu
enum ForwardMode { FWD_IMAGE = 0, FWD_IMAGE_CLAMP = 1, FWD_FIT = 2, FWD_STATS = 3 };
// consumes the fresh bins: sorts each tile's bucket on entry and (FWD_FIT) emits the backward work items
int launch_forward(gs_ctx *c, ForwardMode mode, float *image_out, const float *target, int iter, cudaStream_t s);
int launch_backward(gs_ctx *c, cudaStream_t s);
int launch_repack_grad(gs_ctx *c, const float *dL_dimage, cudaStream_t s);
int launch_reduce_stats(gs_ctx *c, cudaStream_t s);
int ensure_fit_scratch(gs_ctx *c);
// gs2d_optim.cu
int launch_grad_finalize(gs_ctx *c, const gs_params &p, const gs_params &g, cudaStream_t s);
// grad == null: gradients from the moment accumulator (fit loop); rebin: also bin the updated
// parameters for the next iteration (leaves fresh bins of `p` in the context)
int launch_adam(gs_ctx *c, const gs_params &p, const gs_params *grad, const gs_adam_state &st, const float lr[4],
                float beta1, float beta2, float eps, float bc1, float bc2, const unsigned char *active, bool rebin,
                cudaStream_t s);
// gs2d_select.cu
int launch_select(gs_ctx *c, float tau, unsigned char *active_out, int n, cudaStream_t s);
int launch_tile_resid(gs_ctx *c, double *resid_out, cudaStream_t s);
// gs2d_init.cu
int run_init_roi(gs_ctx *c, const float *frame, const unsigned char *mask, int n, unsigned long long seed,
                 float s_min, float s_max, const gs_params &out, cudaStream_t s);

}  // namespace gs2d
