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
struct __align__(32) Rec {
    float mux, muy, i1, k;   // lo
    float i3, cr, cg, cb;    // hi : premultiplied colour c' = o * rgb
};

// Packed binary32 arithmetic of the rasterizers (sm_100: FFMA2 / FMUL2 / FADD2 on a register pair).
// One issue slot does the work of two; each half rounds exactly as the scalar instruction would.
// A lane holds its 8 pixel rows as 4 pairs (rows 2k, 2k + 1); a per-Gaussian scalar doubled with
// dup2() is the instruction's broadcast operand, not a register copy.
#ifdef __CUDACC__
__device__ __forceinline__ float2 dup2(float a) { return make_float2(a, a); }
// row offsets of the four pairs: in constant memory, so that they are operands of the instruction
// (written as literals they are rebuilt in uniform registers inside every loop iteration)
static __constant__ float2 c_rowpair[4] = {{0.0f, 1.0f}, {2.0f, 3.0f}, {4.0f, 5.0f}, {6.0f, 7.0f}};
#endif

// Per-tile statistics produced by the forward kernel in "stats" mode.
struct __align__(8) TileStats {
    double sq_raw;    // sum (C - T)^2      unclamped, valid pixels x 3 channels
    double sq_clamp;  // sum (clamp(C) - T)^2
    double abs_clamp; // sum |T - clamp(C)|
    int n_valid;      // pixels the sums run over: the tile's pixels inside the frame (and inside the ROI, c-16)
    int pad;
};

// Device-side status word bits (latched, read by synchronising calls).
constexpr unsigned FLAG_CAPACITY = 1u;
constexpr unsigned FLAG_NONFINITE = 2u;

// The binning stores, per (tile, Gaussian) pair, the Gaussian's id in the tile's bucket (tile_cap slots);
// arrivals beyond the bucket go to one shared SPILL list of (tile, id) entries that every consumer of the
// binning also walks for its overflowing tiles (a slow path: no tile length is a capacity error).  Records
// live once per Gaussian (rec[N]) and are gathered by id.
constexpr int REC_F4 = 2;         // float4 per record

// Tile classes by list length (scheduling only): class c holds the tiles with 16 c <= n < 16 c + 16
// (the last one everything longer).  Every kernel that consumes a binning files the tile under its
// class for the NEXT launch, which walks the classes longest lists first: no long tile starts
// late, the kernel has no tail.  Inside a class the order is arrival order.  The fit kernel works on
// the tiles of classes >= TEAM_CLASS with a whole CTA, on the others with one warp each.
constexpr int FIT_CHUNK = 64;     // bucket records per shared-memory buffer of the fit kernel
constexpr int NCLS = 16;
constexpr int TEAM_CLASS = FIT_CHUNK / 16;  // n >= FIT_CHUNK
__host__ __device__ __forceinline__ int tile_class(int n) { return n >= 16 * NCLS ? NCLS - 1 : (n >> 4); }

// Device-side counters.  Everything a binning produces is double-buffered by the parity of
// the binning epoch, so that the kernel that consumes epoch e can reset the slot of epoch
// e + 1 while nobody else touches it (no memset launches inside the fit loop).
struct DeviceState {
    unsigned int flags;              // FLAG_* (latched until a synchronising call reads them)
    int first_nonfinite_iter;        // 1-based, 0 = none
    int n_active;                    // result of the last active count
    int pad0;
    unsigned long long pair_total[2];  // [epoch & 1] P = number of (tile, Gaussian) pairs (may exceed capacity)
    int tile_ovf[2];                 // [epoch & 1] != 0: the spill list overflowed
    unsigned int spill_count[2];     // [epoch & 1] arrivals beyond their tile's bucket (may exceed spill_cap)
    int n_class[3][NCLS];            // [consumer launch % 3][class] tiles per class
    unsigned int cursor_team[3];     // [consumer launch % 3] fit kernel: next class-3 tile
    unsigned int cursor_warp[3];     // [consumer launch % 3] fit kernel: next tile of classes 2, 1, 0
    double loss_sum;                 // reduced sq_raw of the last stats reduction
    double sq_clamp_sum;
    unsigned long long total_in;     // ROI init: total inside weight
    unsigned long long total_out;
    unsigned long long roi_pixels;   // gs_set_roi: |M|
};

// Quantisation-aware training (DESIGN.md §3 c-14): the uniform quantisers of the 9
// parameter columns (mu_x, mu_y, l1, l2, l3, r, g, b, o).  on == 0: everything passes through.
struct QuantDev {
    int on;
    int levels[9];  // largest index (2^bits - 1); 0 = this column is not quantised
    float lo[9], step[9], inv_step[9];
};
// quantise-dequantise of one value, single-rounded binary32 (the oracle's definition):
//   idx = clamp(rint((x - lo) * inv_step), 0, levels);  x_q = lo + idx * step
__device__ __forceinline__ float fake_quant(const QuantDev &q, int j, float x) {
    if (!q.on || q.levels[j] == 0) return x;
    float i = rintf(__fmul_rn(__fsub_rn(x, q.lo[j]), q.inv_step[j]));
    i = fminf(fmaxf(i, 0.0f), (float)q.levels[j]);
    return __fadd_rn(q.lo[j], __fmul_rn(i, q.step[j]));
}

// What a kernel needs to bin one Gaussian (k_bin and the fused Adam kernel).
struct BinArgs {
    float cutoff;
    int W, H, TX, TY;
    int tile_cap;                    // bucket capacity per tile
    int slot;                        // binning epoch & 1
    Rec *rec;                        // [N]
    int *tile_count;                 // [2][T] by epoch parity; the slot's half is zero before the binning
    int *bucket;                     // [T * tile_cap] Gaussian ids, arrival order
    int2 *spill;                     // [spill_cap] (tile, id) of the arrivals beyond tile_cap
    int spill_cap;
    const unsigned char *active;     // [N] mask of a selective binning (mode != 0)
    int mode;                        // which Gaussians are listed: 0 all, 1 those with active[i] != 0, 2 those with active[i] == 0
    DeviceState *st;
    QuantDev q;                      // records and rectangles are made from the quantised parameters
    int4 *pair_info;                 // deterministic mode (else null): [N] per Gaussian (first pair slot, x0 | y0 << 16,
                                     // rectangle width, number of pairs) of this binning
};

// What the per-tile sort stage (the prologue of the forward kernel, or k_sort_tiles) needs.
struct TileArgs {
    int *tile_count;                 // [2][T] by epoch parity: the slot's half is read, the other zeroed
    int *tile_n;                     // [T] list length of the tile (written here)
    int *bucket;                     // [T * tile_cap] sorted in place
    int tile_cap;
    const int2 *spill;               // [spill_cap] (tile, id) beyond the buckets
    int spill_cap;
    int slot;                        // binning epoch & 1
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
    int2 *spill;             // [spill_cap] (tile, id) arrivals beyond a tile's bucket
    int spill_cap;
    int *tile_order;         // [3][NCLS*T] consumer launch order: per-class tile lists (class c at c*T)
    unsigned fwd_launches;   // consumer launches so far (selects the order buffer)
    unsigned epoch;          // binning epoch (selects the DeviceState slots)
    int fit_grid;            // persistent grid of the fit kernel (0 = not yet queried)
    alignas(64) unsigned char image_map[128];  // CUtensorMap of the image the fit kernel last read
    const float *image_map_ptr;
    bool image_map_ok;
    // "fresh" bins: a binning whose sort stage has not run yet, and the arrays it was made from
    bool fresh;
    bool sorted;             // the buckets of the last consumed binning are in canonical order
    const float *fresh_mu;
    int fresh_n;
    const unsigned char *fresh_active;  // mask and mode of the fresh bins (BinArgs::mode)
    int fresh_mode;
    // selective refit (P-frames): frame minus the render of the FROZEN Gaussians, the target the active ones are
    // fitted against (lazy), and what it was made from
    float *bg_target;
    const float *bg_frame, *bg_mu;
    const unsigned char *bg_active;
    int bg_n;
    bool bg_valid;
    // raster scratch
    float *acc;              // [N_max*8] gradient moments, zero between iterations
    // deterministic mode (gs_set_deterministic): every (tile, Gaussian) pair owns a slot of 8 moments, numbered per
    // Gaussian in tile order; the optimiser sums a Gaussian's slots in that order instead of reading atomics' sums
    bool deterministic;
    int4 *pair_info;         // [N_max] (lazy) first slot, rectangle origin and width, pair count of the last binning
    float *pair_mom;         // [cap_pairs*8] (lazy)
    gs2d::TileStats *tile_stats;  // [T]
    unsigned char *tile_flag;     // [T]
    float *image_scratch;    // [H*W*3] (lazy; host-buffer entry points)
    // fit scratch
    float *host_params;      // [N_max*9] device copy for *_host entry points (lazy)
    float *host_m, *host_v;  // [N_max*9]
    // ROI init scratch (lazy)
    int *roi_grey;           // [H*W]
    unsigned long long *roi_cin, *roi_cout;  // [H*W] inclusive prefix sums
    unsigned long long *roi_blk;             // block sums
    gs2d::QuantDev quant;         // gs_set_quantization (on == 0: off)
    // gs_set_roi (DESIGN.md §3 c-16): loss, PSNR and residuals over the ROI's pixels only (null: the whole frame)
    const unsigned char *roi;     // [H,W] caller-owned
    long long roi_count;          // |M|
    const unsigned char *bg_roi;  // ROI the derived fit target was made with
    unsigned char *sel_changed;   // [2][H*W] change map and its dilation (lazy; gs2d_select.cu)
    unsigned char *sel_active;    // [max_gaussians] P-frame mask of gs_encode_gop when the caller keeps none (lazy)
    // superpixel initialiser scratch (lazy, grown on demand; gs2d_superpixel.cu)
    void *sp_buf[7];
    size_t sp_bytes[7];
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
// mode / active: BinArgs::mode (0: every Gaussian is listed)
int ensure_bins(gs_ctx *c, const gs_params &p, cudaStream_t s, const unsigned char *active = nullptr, int mode = 0);
void discard_fresh_bins(gs_ctx *c, cudaStream_t s);      // drop bins nobody will consume
BinArgs bin_args(gs_ctx *c, bool next_epoch, const unsigned char *active = nullptr, int mode = 0);  // next_epoch: start a new binning epoch
TileArgs tile_args(gs_ctx *c);
int launch_sort_tiles(gs_ctx *c, cudaStream_t s);        // consume fresh bins, or sort buckets consumed unsorted
int launch_presort_tiles(gs_ctx *c, cudaStream_t s);     // fresh bins into canonical order, not consumed (deterministic mode)
int ensure_pair_slots(gs_ctx *c);                        // deterministic mode: allocate pair_info / pair_mom
int launch_compact(gs_ctx *c, int *range_out, int *list_out, cudaStream_t s);
// gs2d_raster.cu
enum ForwardMode { FWD_IMAGE = 0, FWD_IMAGE_CLAMP = 1, FWD_STATS = 3 };
// consumes the fresh bins: sorts each tile's bucket on entry
int launch_forward(gs_ctx *c, ForwardMode mode, float *image_out, const float *target, cudaStream_t s);
int launch_reduce_stats(gs_ctx *c, cudaStream_t s);
// gs2d_fit.cu
// FIT_LOSS: forward + L2 loss + backward of one fit iteration against `image` (the target frame);
// FIT_GRAD: backward only, `image` is dL/dimage.  Consumes the fresh bins; gradient moments -> acc.
enum FitMode { FIT_LOSS = 0, FIT_GRAD = 1 };
int launch_fit_tiles(gs_ctx *c, FitMode mode, const float *image, int iter, cudaStream_t s);
// out[i] = a[i] - out[i] over n floats (the selective-refit target: frame minus the frozen Gaussians' render)
int launch_sub_from(const float *a, float *out, size_t n, cudaStream_t s);
// out = src where the ROI byte is non-zero (non-finite values there become +Inf: they must poison the loss), NaN
// elsewhere (src may be out): the fit kernel skips NaN targets (c-16)
int launch_mask_target(const float *src, const unsigned char *roi, float *out, size_t npix, cudaStream_t s);
int launch_roi_count(gs_ctx *c, const unsigned char *roi, cudaStream_t s);  // -> dstate->roi_pixels
// gs2d_optim.cu
int launch_grad_finalize(gs_ctx *c, const gs_params &p, const gs_params &g, cudaStream_t s);
int launch_fake_quantize(gs_ctx *c, const gs_params &p, const gs_params &out, const QuantDev &q, cudaStream_t s);
// grad == null: gradients from the moment accumulator (fit loop); rebin: also bin the updated
// parameters for the next iteration (leaves fresh bins of `p` in the context)
int launch_adam(gs_ctx *c, const gs_params &p, const gs_params *grad, const gs_adam_state &st, const float lr[4],
                float beta1, float beta2, float eps, float bc1, float bc2, const unsigned char *active, bool rebin,
                cudaStream_t s);
// gs2d_select.cu
int launch_select(gs_ctx *c, float tau, unsigned char *active_out, int n, cudaStream_t s);
int launch_tile_resid(gs_ctx *c, double *resid_out, cudaStream_t s);
int launch_tile_sq(gs_ctx *c, double *tile_sq_out, cudaStream_t s);
// pixel-granular selection: `render` is the clamped render of the binned parameters (unused with changed_in)
int launch_select_pixels(gs_ctx *c, const float *frame, const float *render, float tau, float thr, int dilate,
                         const unsigned char *changed_in, unsigned char *changed_out, unsigned char *active_out, int n,
                         cudaStream_t s);  // (the context's ROI restricts the change map)
// gs2d_superpixel.cu
int run_init_superpixel(gs_ctx *c, const float *frame, const unsigned char *mask, int n_segments, int compactness,
                        int kmeans_iters, const gs_params &out, int *labels_out, int *n_out_host, cudaStream_t s);
// gs2d_init.cu
int run_init_roi(gs_ctx *c, const float *frame, const unsigned char *mask, int n, unsigned long long seed,
                 float s_min, float s_max, const gs_params &out, cudaStream_t s);

}  // namespace gs2d
