/*
 * gs2d.h -- C-ABI of the B200-native hot path of the 2D Gaussian Splatting ROI
 * video codec of arXiv 2505.09324 ("PAPER.md"; gaps read as DESIGN.md §3 says).
 *
 * The library is hand-written CUDA for sm_100a.  There is no CPU fallback: every
 * entry point that computes returns GS_ERR_CUDA when no device is usable.
 *
 * Conventions (all entry points)
 *   - Images are HWC float32, [H][W][3], nominally in [0,1]; pixel (x,y) has its
 *     centre at (x+0.5, y+0.5), origin top-left.  Masks are uint8 [H][W],
 *     non-zero = inside.
 *   - A Gaussian has 9 stored scalars (Eq. 1; DESIGN.md §3 #2):
 *     mu[2], the Cholesky factor l = (l1,l2,l3) of its covariance
 *     Sigma = L L^T with L = [[l1,0],[l2,l3]], colour rgb[3], opacity o.
 *     The blended colour is c' = o * rgb.
 *   - Unless a name ends in _host, every pointer is a caller-owned DEVICE pointer
 *     (16-byte aligned, e.g. a torch tensor's data_ptr()).  The library never
 *     frees or reallocates caller memory.  gs_ctx owns scratch only.
 *   - `stream` is a cudaStream_t passed as void* (NULL = the legacy default
 *     stream).  gs_render, gs_render_backward, gs_adam_step, gs_decode and
 *     gs_fit_steps are asynchronous on it.  gs_init_roi, gs_encode_iframe,
 *     gs_encode_pframe, gs_get_bins, gs_status and every *_host call
 *     synchronise the stream once before returning.
 *   - Every call returns a gs_status code.  No exception crosses the ABI.
 *     Conditions that only the device can see (pair-list capacity exceeded,
 *     non-finite loss) are latched in the context and returned by the next
 *     synchronising call or by gs_status().
 *   - A context is not thread-safe: one host thread and one stream at a time.
 */
#ifndef GS2D_H
#define GS2D_H

#ifdef __cplusplus
extern "C" {
#endif

enum gs_status_code {
    GS_OK = 0,
    GS_ERR_INVALID_ARGUMENT = -1,  /* null or misaligned pointer, n < 1, dims <= 0, n > max_gaussians */
    GS_ERR_INVALID_PARAMETER = -2, /* reserved: non-finite / singular Gaussians are culled, not rejected    */
    GS_ERR_EMPTY_MASK = -3,        /* gs_init_roi with an all-zero ROI                        */
    GS_ERR_CAPACITY = -4,          /* P > max_pairs, or more entries beyond the tiles' buckets than the spill list
                                      holds (see gs_config.max_pairs); outputs not written                  */
    GS_ERR_NONFINITE = -5,         /* loss became non-finite; the iteration is in the report  */
    GS_ERR_CUDA = -6,              /* CUDA runtime error (gs_last_cuda_error has the text)                  */
    GS_ERR_UNSUPPORTED = -7        /* tile != 16, frame wider/taller than 65535 tiles                       */
};

typedef struct gs_ctx gs_ctx; /* opaque: scratch buffers sized from gs_config */

typedef struct {
    int width, height;     /* frame size in pixels                                         */
    int tile;              /* must be 16 (BASELINE.json north_star: 16x16 screen tiles)    */
    float cutoff;          /* k: footprint = k marginal standard deviations; default 3.0   */
    float l_min;           /* projection floor for l1, l3 after an Adam step; default 0.1  */
    int max_gaussians;     /* capacity N_max                                               */
    long long max_pairs;   /* capacity: total number P of (tile, Gaussian) pairs of a binning.  Every tile owns a
                              bucket of max(512, 4 * (max_pairs / T + 1)) ids (never more than
                              min(max_gaussians, max_pairs)), T = number of tiles; entries beyond a tile's bucket
                              go to ONE shared spill list of max(4096, max_pairs / 4) entries that every consumer
                              walks for its overflowing tiles (a slow path, not an error).  GS_ERR_CAPACITY is
                              raised by P > max_pairs or by an overflow of the spill list.  Device memory:
                              16 bytes per unit of max_pairs (4-byte ids; records live once per Gaussian)   */
} gs_config;

typedef struct {
    float *mu;      /* [n,2]                         */
    float *chol;    /* [n,3]  l1,l2,l3               */
    float *rgb;     /* [n,3]                         */
    float *opacity; /* [n]                           */
    int n;
} gs_params; /* also the shape of a gradient: d/dmu, d/dchol, d/drgb, d/dopacity */

typedef struct {
    float *m; /* [n,9] first moments, columns (mu_x, mu_y, l1, l2, l3, r, g, b, o) */
    float *v; /* [n,9] second moments                                              */
} gs_adam_state;

typedef struct {
    int iters;
    float lr[4]; /* mu, chol, rgb, opacity */
    float beta1, beta2, eps;
    int resume;  /* gs_fit_steps only (0 elsewhere).  Non-zero: the call may START from the tile bins that
                    the previous gs_fit_steps(resume != 0) on this context left for the same parameter
                    arrays, and LEAVES the bins of its result for the next such call (its last Adam kernel
                    bins the updated parameters).  The caller thereby promises not to modify the parameter
                    arrays between two resumed calls.  A resumed call that CONTINUES a fit (t0 > 1) right after
                    the previous gs_fit_steps also keeps that call's derived fit target (frame minus the frozen
                    Gaussians' render, ROI mask applied) when frame, active and ROI pointers are the same: their
                    CONTENTS must then be unchanged too.  A call with t0 == 1 starts a fit: it re-reads frame,
                    mask and ROI, and any other entry point called in between drops both the bins and the
                    target.  0: the call bins what it is given and leaves nothing behind.             */
} gs_fit_opts;

typedef struct {
    double final_loss;        /* mean squared error of the UNCLAMPED render (DESIGN.md §3 #8) */
    double psnr;              /* 10 log10(1/MSE) of the clamped render, 99 dB ceiling         */
    int iters_run;
    int first_nonfinite_iter; /* 1-based; 0 = none                                            */
    int n_active;             /* Gaussians that were free to move                             */
    long long n_pairs;        /* P of the last binning                                        */
} gs_fit_report;

typedef struct {
    float decay;        /* learning rates are multiplied by `decay` at each milestone (0.5)        */
    float milestone[2]; /* fractions of opts->iters (0.6, 0.85): iteration i (0-based) runs with
                           lr * decay^(number of j with i >= floor(milestone[j] * iters + 0.5)), in double       */
    float target_psnr;  /* early stop: after every check_every-th iteration the PSNR of the clamped
                           render is evaluated; the fit stops once it is >= target_psnr.  <= 0: never            */
    int check_every;    /* >= 1 when target_psnr > 0                                                             */
} gs_fit_schedule;

typedef struct {
    /* Uniform quantisers of the 9 parameter columns (mu_x, mu_y, l1, l2, l3, r, g, b, o)
       ("distinct quantization strategies to the three attributes ... mean, cholesky and color"; SPEC.md:378-400:
       16 / 6 / 8 bits).  levels[j] = largest index (2^bits - 1), 0 = column j passes through.  A value x becomes
           lo[j] + step[j] * clamp(rint((x - lo[j]) * inv_step[j]), 0, levels[j])
       in single-rounded binary32, ties to even (DESIGN.md §3 c-14).  step and inv_step are given by the caller
       (step = (hi - lo) / levels, inv_step = levels / (hi - lo), each rounded once). */
    int levels[9];
    float lo[9], step[9], inv_step[9];
} gs_quant_spec;

/* ---- context ---------------------------------------------------------------------------- */

/* Allocates scratch for frames of cfg->width x cfg->height, up to max_gaussians
 * Gaussians and max_pairs (tile, Gaussian) pairs (see gs_config.max_pairs for the bucket
 * space).  Errors: INVALID_ARGUMENT, UNSUPPORTED, CUDA. */
int gs_create(const gs_config *cfg, gs_ctx **out);
int gs_destroy(gs_ctx *ctx);

/* ROI-restricted loss (the codec encodes "only the region of interest"; "mean squared error
 * over masked pixels", :286 masked PSNR, :326 change map inside the ROI; DESIGN.md §3 c-16).  While an ROI is set on
 * the context, with M its non-zero pixels: every fit (gs_fit_steps, gs_encode_*) minimises
 * sum_{p in M, ch} (C - T)^2 / (3 |M|), gs_loss_psnr and the fit reports give loss and PSNR over M,
 * gs_pframe_select averages a tile's residual over its ROI pixels (a tile without any is never changed), and the
 * change map of gs_pframe_select_pixels is restricted to M before the dilation.  Renders and gs_render_backward are
 * unaffected.  roi_mask: device uint8 [H][W], caller-owned, must stay valid and unchanged while it is set; NULL:
 * off (the whole frame, the default).  Synchronises `stream` once (it counts |M|).  Errors: INVALID_ARGUMENT, EMPTY_MASK (an all-zero mask; the setting is
 * left unchanged), CUDA. */
int gs_set_roi(gs_ctx *ctx, const unsigned char *roi_mask, void *stream);

/* Bit-reproducible fits (SPEC.md "Determinism": the same job and seed give the same Gaussians; DESIGN.md §3
 * "Determinism").  By default a fit is reproducible to rounding only: tile lists are summed in the arrival order of
 * the binning's counting atomics, and the gradient moments of a Gaussian meet in binary32 atomics.  With on = 1,
 * (1) every tile's list is brought into ascending id order before the fit kernel sums it, and every tile is scheduled
 * by its current list length (one more launch per iteration), (2) the backward pass stores the 8 moments of every (tile, Gaussian) pair in the pair's own slot
 * (slots are numbered per Gaussian in row-major tile order) and the optimiser adds a Gaussian's slots in that
 * order: no floating-point atomics anywhere.  gs_fit_steps, gs_encode_* and gs_render_backward then return the
 * same bits from the same inputs, whatever the call pattern and the context's history -- unless a tile lists more Gaussians than its bucket holds
 * (gs_config.max_pairs): entries in the shared spill list keep their arrival order.  Costs 32 bytes of device
 * memory per unit of max_pairs and ~10 % of the iteration.
 * Errors: INVALID_ARGUMENT, CUDA (allocation). */
int gs_set_deterministic(gs_ctx *ctx, int on);

/* Synchronises `stream`, then returns and clears the latched device-side status
 * (GS_OK, GS_ERR_CAPACITY or GS_ERR_NONFINITE).  Reading a non-finite latch re-arms the context:
 * later fits update their parameters again. */
int gs_status(gs_ctx *ctx, void *stream);
/* Text of the last CUDA error seen by this library in this process ("" if none). */
const char *gs_last_cuda_error(void);

/* Quantisation-aware training ("quantization is integrated directly into the Gaussian
 * optimization process"; "parameters pass through simulated quantize-dequantize with
 * straight-through gradients before rendering"; DESIGN.md §3 c-14).  While a spec is
 * set on the context, every binning makes its records and tile rectangles from the quantised parameters --
 * renders, fits, statistics and selections see them -- and the chain rule of the backward pass is evaluated
 * there, the gradient going straight through to the caller's raw parameters, which Adam updates.  NULL: off. */
int gs_set_quantization(gs_ctx *ctx, const gs_quant_spec *spec);
/* Post-training quantise-dequantise of a parameter set (out may alias in).  Asynchronous. */
int gs_fake_quantize(gs_ctx *ctx, gs_params in, const gs_quant_spec *spec, gs_params out, void *stream);

/* ---- the seven calls of BASELINE.json's north_star ---------------------------------------- */

/* Content-aware ROI initialiser (BASELINE.json configs[1],[2]; stands in for the
 * paper's matting + superpixel initialiser; DESIGN.md §3 c-8).
 * floor(7n/10) Gaussians are placed inside the ROI with probability proportional
 * to an integer Sobel-magnitude weight, the rest uniformly outside it (all
 * inside if the ROI covers the frame).  Colours are copied from `frame`,
 * opacity = 1, scales log-uniform in [s_min, s_max] px, rotation U[0,pi).
 * Random numbers: SplitMix64 finaliser of seed + (8 i + k + 1) * 0x9E3779B97F4A7C15
 * for Gaussian i, stream k (0 pixel, 1 jitter x, 2 jitter y, 3 s1, 4 s2, 5 angle).
 * frame [H,W,3] float32, roi_mask [H,W] uint8, out.{mu,chol,rgb,opacity} with
 * out.n = n.  Sampled pixels, positions and colours are bit-exact with the oracle.
 * Errors: INVALID_ARGUMENT, EMPTY_MASK, CUDA. */
int gs_init_roi(gs_ctx *ctx, const float *frame, const unsigned char *roi_mask, int n, unsigned long long seed,
                float s_min, float s_max, gs_params out, void *stream);

/* The paper's content-aware I-frame initialiser (the ROI is "segmented into N
 * superpixel segments using a K-means clustering-based superpixel algorithm"; "Gaussian means are
 * computed as the center of each superpixel, the Cholesky decomposition is derived from the
 * covariance matrix of each segment, and the RGB colors are calculated as the average pixel color";
 * SPEC.md:182-200 reads it as SLIC; the integer-exact reading is DESIGN.md §3 c-11):
 *   - the ROI's bounding box is cut into GX x GY about-square cells (pixel offset * G / box size,
 *     integer division), GX the largest value for which at most n_segments cells hold ROI pixels
 *     (bisection); one cluster per occupied cell, seeded at its ROI pixel nearest the cell centre;
 *   - kmeans_iters rounds of: every ROI pixel joins, among the clusters of the 3 x 3 cells around
 *     its cell, the one minimising  S2 |d colour|^2 + compactness^2 |d position|^2  (S2 = cell area;
 *     features in 1/16 units, colours quantised to 8 bits, 64-bit integers, ties to the smaller
 *     index); centres become rounded integer means;
 *   - one Gaussian per non-empty cluster, in cell order: mu = mean pixel centre, Sigma = covariance
 *     of the member pixels as unit squares (point covariance + I/12), l = chol(Sigma), colour =
 *     mean colour, opacity 1.
 * out.{mu,chol,rgb,opacity} need room for n_segments rows; *n_out_host (HOST) receives the number
 * K <= n_segments written.  labels_out [H,W] int32 (nullable): the pixel's Gaussian, -1 outside
 * the ROI.  Labels are bit-exact with the oracle.  Synchronises.
 * Errors: INVALID_ARGUMENT, EMPTY_MASK, CUDA. */
int gs_init_superpixel(gs_ctx *ctx, const float *frame, const unsigned char *roi_mask, int n_segments,
                       int compactness, int kmeans_iters, gs_params out, int *labels_out, int *n_out_host,
                       void *stream);

/* Tile binning + forward rasterisation (Eq. 2; DESIGN.md §3 c-2, c-3):
 *   C(p) = sum over the Gaussians n listed in the 16x16 tile of p of  o_n rgb_n exp(-sigma_n(p)),
 *   sigma_n = 1/2 d^T Sigma_n^-1 d,  d = p - mu_n.
 * image_out [H,W,3]; clamp != 0 clamps to [0,1] (display / PSNR / decode), clamp = 0
 * gives the raw sum the loss is defined on.  Non-finite or singular (l1 l3 = 0)
 * Gaussians and Gaussians whose footprint misses the frame are skipped.
 * Errors: INVALID_ARGUMENT now; CAPACITY latched (image_out then left untouched). */
int gs_render(gs_ctx *ctx, gs_params params, float *image_out, int clamp, void *stream);

/* Backward pass of gs_render with clamp = 0 ("differentiable";
 * DESIGN.md §3 c-5): given dL/dimage [H,W,3], writes the per-Gaussian gradients
 * of L with respect to mu, l, rgb and opacity into grad_out (same shapes as
 * params; every row is written, zeros for culled Gaussians).  List membership is
 * treated as constant.  The call re-bins `params` itself, so it never depends on
 * an earlier gs_render.  Accumulation over tiles uses fp32 atomics: results are
 * reproducible to rounding, not bit for bit. */
int gs_render_backward(gs_ctx *ctx, gs_params params, const float *dL_dimage, gs_params grad_out, void *stream);

/* One fused Adam step with active mask and projection (DESIGN.md §3 c-6):
 *   m <- b1 m + (1-b1) g ; v <- b2 v + (1-b2) g^2
 *   theta <- theta - lr_group (m/(1-b1^t)) / (sqrt(v/(1-b2^t)) + eps)
 * then l1 <- max(l1, l_min), l3 <- max(l3, l_min).  t >= 1 is the step index.
 * active: [n] uint8 or NULL (= all active).  Where active[i] = 0 the parameters
 * and both moments of Gaussian i are bit-identical afterwards. */
int gs_adam_step(gs_ctx *ctx, gs_params params, gs_params grad, gs_adam_state state, const float lr[4], float beta1,
                 float beta2, float eps, int t, const unsigned char *active, void *stream);

/* I-frame fit (DESIGN.md §3 c-7): zeroes the Adam moments, then
 * opts->iters iterations of  bin -> render -> L2 loss -> backward -> Adam  on
 * `inout` in place, then one more bin + render for the report.  frame [H,W,3].
 * Errors: INVALID_ARGUMENT, CAPACITY, NONFINITE (report->first_nonfinite_iter), CUDA. */
int gs_encode_iframe(gs_ctx *ctx, const float *frame, gs_params inout, gs_adam_state state, const gs_fit_opts *opts,
                     gs_fit_report *report, void *stream);

/* gs_encode_iframe with the paper's "dynamic learning rate scheduler" (unspecified there,
 * read as SPEC.md:267-275's two-step decay) and early stop at a target PSNR (PAPER.md:163 counts
 * "iterations for 30 PSNR").  SURVEY.md §8(f) next #4; DESIGN.md §3 c-12.  The schedule is
 * host-side: the learning rates are per-launch arguments of the Adam kernel; a PSNR check is one
 * statistics render and one 4-byte read.  report->iters_run is the number of iterations done. */
int gs_encode_iframe_sched(gs_ctx *ctx, const float *frame, gs_params inout, gs_adam_state state,
                           const gs_fit_opts *opts, const gs_fit_schedule *sched, gs_fit_report *report, void *stream);

/* P-frame encode (BASELINE.json configs[3]; DESIGN.md §3 c-9):
 * render `inout` (the previous frame's Gaussians), mark the 16x16 tiles whose
 * mean absolute residual against `frame` (clamped render, valid pixels, 3
 * channels) is > tau, set active_out[i] = 1 for every Gaussian listed in a marked
 * tile, then refit only those for opts->iters iterations (full-frame loss,
 * moments zeroed).  Unselected Gaussians are bit-identical afterwards.  Empty
 * selection: nothing changes and iters_run = 0.  active_out [n] uint8. */
int gs_encode_pframe(gs_ctx *ctx, const float *frame, gs_params inout, gs_adam_state state, float tau,
                     const gs_fit_opts *opts, unsigned char *active_out, gs_fit_report *report, void *stream);

/* Pixel-granular P-frame selection, the paper's own wording ("isolating pixels that exceed a
 * user-defined change threshold ... locate all Gaussians that influence the changing pixels"; SPEC.md:303-341;
 * SURVEY.md §8(f) next #2; DESIGN.md §3 c-13):
 *   pixel changed iff max over channels |frame - clamped render of `params`| > tau (strict), optionally dilated by
 *   one pixel (dilate != 0); Gaussian n influences pixel p iff n is listed in p's tile and exp(-sigma_n(p)) >=
 *   influence_eps (in (0,1); SPEC.md:358 default 0.01), a decision taken in single-rounded binary32 on the
 *   kappa-scaled whitened form (u = dx i1, v = dy i3 + dx k, u u + v v <= log2(1/eps)); active_out[i] = 1 iff i
 *   influences a changed pixel.
 * changed_in [H,W] uint8 (nullable): use this change map instead of computing one; changed_out (nullable) receives
 * the map used.  *n_active_host (HOST) the count.  Synchronises. */
int gs_pframe_select_pixels(gs_ctx *ctx, const float *frame, gs_params params, float tau, float influence_eps,
                            int dilate, const unsigned char *changed_in, unsigned char *changed_out,
                            unsigned char *active_out, int *n_active_host, void *stream);

/* gs_encode_pframe with the pixel-granular selection above in place of the tile-residual rule. */
int gs_encode_pframe_pixels(gs_ctx *ctx, const float *frame, gs_params inout, gs_adam_state state, float tau,
                            float influence_eps, int dilate, const gs_fit_opts *opts, unsigned char *active_out,
                            gs_fit_report *report, void *stream);

/* ---- GoP loop over a sequence ----------- */

typedef struct {
    int gop_length;          /* K >= 1.  Frame f (0-based) is an I-frame iff f % K == 0, else a P-frame that starts
                                from frame f-1's fitted Gaussians ("a GoP length of 4 results in an
                                I-frame every four P-frames" is read as SPEC.md:439, 487 reads it: [I,P,P,P,I,...];
                                K = 1: every frame is an I-frame)                                               */
    int init;                /* I-frame initialiser: 0 = gs_init_roi, 1 = gs_init_superpixel                    */
    int n;                   /* init 0: Gaussians per frame; init 1: segments asked for (the frame gets <= n)    */
    unsigned long long seed; /* init 0: I-frame f draws with seed + f                                           */
    float s_min, s_max;      /* init 0                                                                          */
    int compactness, kmeans_iters; /* init 1                                                                    */
    gs_fit_opts iframe;      /* I-frame fit: iterations, learning rates, Adam constants (resume ignored)        */
    gs_fit_schedule sched;   /* I-frame schedule / early stop (decay 1, target_psnr 0: plain gs_encode_iframe)   */
    gs_fit_opts pframe;      /* P-frame refit                                                                   */
    int pixel_select;        /* P-frame selection: 0 = tile-residual rule (gs_encode_pframe), 1 = pixel-granular
                                (gs_encode_pframe_pixels with influence_eps, dilate)                            */
    float tau, influence_eps;
    int dilate;
} gs_gop_opts;

typedef struct {
    int type;          /* 0 = I-frame, 1 = P-frame                  */
    int n;             /* Gaussians of the frame's parameter set     */
    gs_fit_report fit; /* as the single-frame calls report it        */
} gs_frame_report;

/* Encodes n_frames frames in order, one GoP after the other, each frame by the single-frame calls above
 * (I: initialiser + gs_encode_iframe_sched; P: selection + masked refit of the previous frame's set), and keeps a
 * snapshot of every frame's fitted parameter set.
 *   frames, roi_masks : HOST arrays of n_frames DEVICE pointers ([H,W,3] float32 / [H,W] uint8); roi_masks[f] is
 *                       read for I-frames only (may be NULL elsewhere).
 *   work, state       : device scratch with room for opts->n rows (work.n is ignored): the running set and its moments.
 *   out               : HOST array of n_frames gs_params whose device arrays have room for opts->n rows; out[f]
 *                       receives frame f's set (device-to-device copies) and out[f].n its size.
 *   active_out        : device [n_frames][opts->n] uint8, nullable: row f = the Gaussians refitted for P-frame f
 *                       (every Gaussian of the set for I-frames; zeros past out[f].n).
 *   reports           : HOST [n_frames], nullable.
 * Stops at the first frame whose call fails and returns its code (reports[f].type is then set, later entries are
 * untouched).  Synchronises.  Errors: those of the single-frame calls. */
int gs_encode_gop(gs_ctx *ctx, const float *const *frames, const unsigned char *const *roi_masks, int n_frames,
                  const gs_gop_opts *opts, gs_params work, gs_adam_state state, gs_params *out,
                  unsigned char *active_out, gs_frame_report *reports, void *stream);

/* Decode = one binning + one forward render, clamped to [0,1]; no gradient pass
 * (SPEC.md:490-498, 512).  Same as gs_render(..., clamp = 1). */
int gs_decode(gs_ctx *ctx, gs_params params, float *image_out, void *stream);

/* ---- decode without any device allocation ------------------------------------------------- */

#define GS_STATIC_MAX_GAUSSIANS 16384 /* Gaussians per call                                              */
#define GS_STATIC_MAX_TILES 4096      /* ceil(W/16) * ceil(H/16) per call: e.g. 1024 x 1024 or 1280 x 720 */
#define GS_STATIC_TILE_CAP 256        /* Gaussians listed in any one tile                                 */

/* gs_decode for callers that are not allowed to allocate device memory.  Every other call needs a gs_ctx, and
 * gs_create fills one with cudaMalloc.  That is unusable for a host application that has handed the whole GPU to its
 * own memory pools (a cudaMalloc from a library then fails or breaks the host's budget), for a real-time loop that
 * cannot take the device-wide synchronisation cudaMalloc / cudaFree imply, and for processes in which allocation is
 * forbidden once start-up is over.  This call takes no context: its scratch (records, per-tile counters and id
 * buckets, about 4.5 MiB) is a fixed-size array inside the library image, and it calls neither cudaMalloc nor
 * cudaFree nor any allocating library routine.
 *   params, image_out : DEVICE pointers owned by the caller, as for gs_decode (mu 8-byte aligned, the others 4);
 *                       image_out [height][width][3] float32 receives the render clamped to [0,1].
 *   width, height     : frame size; cutoff: footprint in marginal standard deviations (gs_config.cutoff; 3.0).
 *   stream            : a stream of the CURRENT device (the scratch address is looked up for cudaGetDevice()).
 * Same operation as gs_decode (PAPER.md:50-52 Eq. 2, :152): same culling, tile rectangles, canonical list order and
 * per-pixel arithmetic; agreement with gs_decode is tested to the 1e-4 pixel tolerance of the render tests.
 * Limits: params.n <= GS_STATIC_MAX_GAUSSIANS, tiles <= GS_STATIC_MAX_TILES, and no tile may list more than
 * GS_STATIC_TILE_CAP Gaussians.  A job beyond the first two returns GS_ERR_CAPACITY before any GPU work; a tile
 * beyond the third returns GS_ERR_CAPACITY after the call, with image_out left untouched.  Nothing is ever truncated.
 * The scratch array exists once per GPU, is resident on every GPU that loads the library until the process ends, and
 * is shared by all calls: it keeps the previous call's contents (this call clears the counters and the overflow flag
 * it depends on itself), and two calls whose GPU work overlaps on one device -- two streams, or two host threads --
 * race on it, so callers must serialise them.  The first call on each device looks the array's device address up
 * (cudaGetSymbolAddress, which may load the module); make that first call at start-up, before any stream capture.
 * Synchronises `stream` (it reads the overflow flag back).
 * Errors: INVALID_ARGUMENT (null / misaligned pointer, n < 1, dims < 1, cutoff not positive and finite),
 * CAPACITY (see above), UNSUPPORTED (device ordinal >= 64), CUDA. */
int gs_decode_static(gs_params params, int width, int height, float cutoff, float *image_out, void *stream);

/* ---- loop pieces and parity accessors ------------------------------------------------------ */

/* `iters` fit iterations starting at Adam step index t0 (>= 1) WITHOUT zeroing the
 * moments, without the final render and without synchronising: the body of
 * gs_encode_iframe, exposed so that a caller (bench.py) can time the loop with
 * CUDA events.  active may be NULL.  An iteration is two kernels: fit-tiles (forward
 * rasterizer + L2 loss gradient + backward pass, fused per tile) and Adam (+ chain rule,
 * + binning of the updated parameters for the next iteration); only the first iteration
 * of a call that does not resume (opts->resume) runs the standalone binning kernel. */
int gs_fit_steps(gs_ctx *ctx, const float *frame, gs_params inout, gs_adam_state state, const gs_fit_opts *opts,
                 int t0, const unsigned char *active, void *stream);

/* One fit iteration (as gs_fit_steps with iters = 1, resume = 1, Adam step index t) with a
 * CUDA event recorded on `stream` between the kernels.  ms_out_host[3] (HOST) receives the
 * elapsed milliseconds of: bin (standalone binning; ~0 when the previous step left its bins),
 * fit (forward + loss + backward), adam (+chain rule, +binning of the result).  With an active mask or an ROI the
 * derived fit target (one render of the frozen Gaussians and a subtraction; rebuilt when t == 1, else kept as
 * gs_fit_opts.resume describes) is made BEFORE the first event and is in none of the three times.
 * Synchronises.  For bench.py's per-kernel roofline numbers. */
int gs_profile_fit_step(gs_ctx *ctx, const float *frame, gs_params inout, gs_adam_state state,
                        const gs_fit_opts *opts, int t, const unsigned char *active, float *ms_out_host,
                        void *stream);

/* gs_decode with a CUDA event recorded on `stream` between its two kernels: ms_out_host[2] (HOST) receives
 * the elapsed milliseconds of the binning kernel and of the render kernel.  Synchronises.  For bench.py's
 * per-kernel roofline numbers of the decode path ("real-time decoding"). */
int gs_profile_decode(gs_ctx *ctx, gs_params params, float *image_out, float *ms_out_host, void *stream);

/* P-frame selection only (steps 1-4 of gs_encode_pframe).  tile_resid_out [T]
 * float64 (nullable), tile_flag_out [T] uint8 (nullable), active_out [n] uint8;
 * *n_active_host receives the count (host pointer).  Synchronises. */
int gs_pframe_select(gs_ctx *ctx, const float *frame, gs_params params, float tau, double *tile_resid_out,
                     unsigned char *tile_flag_out, unsigned char *active_out, int *n_active_host, void *stream);

/* Loss of DESIGN.md §3 c-4 for `params` against `frame`: bin + render + reduce.
 * Host outputs: *loss_host = mean((C-T)^2) unclamped, *psnr_host on the clamped
 * render.  Synchronises. */
int gs_loss_psnr(gs_ctx *ctx, const float *frame, gs_params params, double *loss_host, double *psnr_host,
                 void *stream);

/* Parity accessor: per tile, sum over its valid pixels and 3 channels of (C - T)^2 (unclamped), as the LAST
 * kernel that compared a render with a target left it -- the forward half of the fit kernel (gs_fit_steps,
 * gs_encode_*) or the statistics render (gs_loss_psnr, gs_pframe_select).  tile_sq_out: device, [T] float64.
 * Asynchronous on `stream`.  (Eq. 2; DESIGN.md §3 c-4.) */
int gs_get_tile_loss(gs_ctx *ctx, double *tile_sq_out, void *stream);

/* Canonical bins of the LAST binning done by this context (any call above that
 * renders; after a resumed gs_fit_steps: the bins of its result -- of its ACTIVE Gaussians only when that call
 * had an active mask, since a selective refit bins nothing else), compacted on
 * demand from the per-tile buckets: range_out [T+1] int32 = exclusive prefix of per-tile counts,
 * list_out [cap_list] int32 = Gaussian ids ordered by tile id, then by Gaussian
 * id ascending; *P_host = number of pairs (host pointer).  list_out may be NULL.
 * T = ceil(W/16) * ceil(H/16), tile id = ty * ceil(W/16) + tx.  Device outputs;
 * synchronises.  Errors: CAPACITY if P > cap_list (P is still reported). */
int gs_get_bins(gs_ctx *ctx, int *range_out, int *list_out, long long cap_list, long long *P_host, void *stream);

/* ---- host-buffer entry points (end-to-end measurements; all synchronise) ------------------- */

/* As gs_decode, but params.* and image_out are HOST pointers (pinned memory makes
 * the copies asynchronous): H2D of 9n floats, render, D2H of 3WH floats. */
int gs_decode_host(gs_ctx *ctx, gs_params params_host, float *image_out_host, void *stream);

/* As gs_encode_iframe, but frame_host, inout_host.* are HOST pointers; the Adam
 * moments live in context scratch.  H2D of the frame and 9n floats, the fit,
 * D2H of 9n floats. */
int gs_encode_iframe_host(gs_ctx *ctx, const float *frame_host, gs_params inout_host, const gs_fit_opts *opts,
                          gs_fit_report *report, void *stream);

#ifdef __cplusplus
}
#endif
#endif /* GS2D_H */
