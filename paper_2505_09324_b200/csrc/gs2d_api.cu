// gs2d_api.cu -- the extern "C" boundary declared in include/gs2d.h: argument checks,
// context scratch, and the host-side loops that sequence the kernels.  No arithmetic of the
// method lives here except the Adam bias corrections 1 - beta^t (computed in double).
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <new>

#include "gs2d_internal.cuh"

namespace gs2d {

static char g_cuda_error[512] = "";

void set_cuda_error(cudaError_t e, const char *where) {
    snprintf(g_cuda_error, sizeof g_cuda_error, "%s: %s (%s)", cudaGetErrorName(e), cudaGetErrorString(e), where);
}

// The kernels move the [n,3] / [n,9] arrays as float4 slabs and mu as float2: every parameter array must
// be 16-byte aligned (include/gs2d.h, "Layouts"); a sliced view that is not is rejected here, not faulted on.
static bool aligned16(const void *p) { return ((size_t)p & 15u) == 0; }
static bool params_ok(const gs_ctx *c, const gs_params &p) {
    return c && p.mu && p.chol && p.rgb && p.opacity && p.n >= 1 && p.n <= c->cfg.max_gaussians &&
           ((size_t)p.mu & 7u) == 0 && aligned16(p.chol) && aligned16(p.rgb) && ((size_t)p.opacity & 3u) == 0;
}
// host arrays (the *_host entry points copy them with cudaMemcpyAsync: no alignment beyond float)
static bool host_params_ok(const gs_ctx *c, const gs_params &p) {
    return c && p.mu && p.chol && p.rgb && p.opacity && p.n >= 1 && p.n <= c->cfg.max_gaussians;
}
static bool state_ok(const gs_adam_state &st) { return st.m && st.v && aligned16(st.m) && aligned16(st.v); }
// images are read / written as float4 row segments when the width allows it
static bool image_ok(const gs_ctx *c, const float *img) { return img && (c->cfg.width % 4 != 0 || aligned16(img)); }

static int read_state(gs_ctx *c, cudaStream_t s) {
    GS_CUDA_TRY(cudaMemcpyAsync(c->hstate, c->dstate, sizeof(DeviceState), cudaMemcpyDeviceToHost, s));
    GS_CUDA_TRY(cudaStreamSynchronize(s));
    return GS_OK;
}

// Returns and clears the latched device flags (after a synchronising read_state).
static int consume_flags(gs_ctx *c, cudaStream_t s) {
    unsigned f = c->hstate->flags;
    if (f) {
        // flags and first_nonfinite_iter are adjacent: a consumed non-finite latch no longer stops the updates
        // of later fits on this context (the Adam kernel skips its step while first_nonfinite_iter != 0)
        GS_CUDA_TRY(cudaMemsetAsync(&c->dstate->flags, 0, (f & FLAG_NONFINITE) ? 2 * sizeof(unsigned) : sizeof(unsigned), s));
        GS_CUDA_TRY(cudaStreamSynchronize(s));
    }
    if (f & FLAG_CAPACITY) return GS_ERR_CAPACITY;
    if (f & FLAG_NONFINITE) return GS_ERR_NONFINITE;
    return GS_OK;
}

// P of the binning the context last ran (valid after read_state)
static long long host_pairs(const gs_ctx *c) {
    const unsigned long long P = c->hstate->pair_total[c->epoch & 1u];
    return P > 0x7fffffffffffffffull ? 0x7fffffffffffffffll : (long long)P;
}

// Selective refit (P-frames): the frozen Gaussians do not change during the refit, so their
// image B is rendered ONCE and the active Gaussians are fitted against frame - B:
//     C_all - T = (C_active + B) - T = C_active - (T - B)
// Every iteration then bins, rasterises and differentiates the active Gaussians only: its cost follows the
// active fraction.  Leaves the target in c->bg_target.  It is reused only by a resumed gs_fit_steps /
// gs_profile_fit_step that CONTINUES a fit (step index > 1) on the same arrays, mask and ROI with no other entry point
// called in between: pointer identity says nothing about contents, so every other public call drops it
// (drop_fit_target) and a fit that starts at step 1 always rebuilds it.
static int selective_target(gs_ctx *c, const float *frame, const gs_params &p, const unsigned char *active, bool reuse,
                            cudaStream_t s, const float **target) {
    const size_t n3 = 3 * (size_t)c->cfg.width * (size_t)c->cfg.height;
    if (!c->bg_target) GS_CUDA_TRY(cudaMalloc(&c->bg_target, sizeof(float) * n3));
    *target = c->bg_target;
    if (reuse && c->bg_valid && c->bg_frame == frame && c->bg_active == active && c->bg_mu == p.mu && c->bg_n == p.n &&
        c->bg_roi == c->roi)
        return GS_OK;
    int rc;
    if (active) {
        discard_fresh_bins(c, s);
        if ((rc = ensure_bins(c, p, s, active, 2))) return rc;  // the frozen Gaussians only
        if ((rc = launch_forward(c, FWD_IMAGE, c->bg_target, nullptr, s))) return rc;
        if ((rc = launch_sub_from(frame, c->bg_target, n3, s))) return rc;
    }
    // c-16: target values outside the ROI become NaN, which the fit kernel's loss skips
    if (c->roi && (rc = launch_mask_target(active ? c->bg_target : frame, c->roi, c->bg_target, n3 / 3, s))) return rc;
    c->bg_roi = c->roi;
    c->bg_frame = frame;
    c->bg_active = active;
    c->bg_mu = p.mu;
    c->bg_n = p.n;
    c->bg_valid = true;
    return GS_OK;
}

static inline void drop_fit_target(gs_ctx *c) { c->bg_valid = false; }

// The fit loop: an iteration is fit-tiles (forward + loss + backward, fused per tile) -> Adam(+binning
// of the updated parameters).  Only the first iteration needs a standalone k_bin, and not even that when the
// context still holds the bins the previous loop left for the same arrays.  leave_bins: the last
// Adam step also bins (for a following render, or for a resumed gs_fit_steps).
// active (nullable): selective refit -- frozen Gaussians untouched by Adam and absent from the lists.
static int fit_loop(gs_ctx *c, const float *frame, const gs_params &p, const gs_adam_state &st, const gs_fit_opts *o,
                    int t0, const unsigned char *active, bool leave_bins, cudaStream_t s, bool reuse_target = false) {
    int rc = GS_OK;
    const float *target = frame;
    if ((active || c->roi) && o->iters > 0 && (rc = selective_target(c, frame, p, active, reuse_target, s, &target)))
        return rc;
    for (int k = 0; k < o->iters; ++k) {
        const int t = t0 + k;
        if ((rc = ensure_bins(c, p, s, active, 1))) return rc;
        if ((rc = launch_fit_tiles(c, FIT_LOSS, target, t, s))) return rc;
        const float bc1 = (float)(1.0 - pow((double)o->beta1, (double)t));
        const float bc2 = (float)(1.0 - pow((double)o->beta2, (double)t));
        const bool rebin = leave_bins || k + 1 < o->iters;
        if ((rc = launch_adam(c, p, nullptr, st, o->lr, o->beta1, o->beta2, o->eps, bc1, bc2, active, rebin, s)))
            return rc;
    }
    return GS_OK;
}

// bin + stats forward + reduction; fills the host mirror.  Synchronises.
static int final_stats(gs_ctx *c, const float *frame, const gs_params &p, cudaStream_t s) {
    int rc;
    drop_fit_target(c);  // (every encode ends here: its derived target is not kept for later calls)
    if ((rc = ensure_bins(c, p, s))) return rc;
    if ((rc = launch_forward(c, FWD_STATS, nullptr, frame, s))) return rc;
    if ((rc = launch_reduce_stats(c, s))) return rc;
    return read_state(c, s);
}

static void fill_report(gs_ctx *c, gs_fit_report *r, int iters_run, int n_active) {
    if (!r) return;
    const double n = c->roi ? 3.0 * (double)c->roi_count : 3.0 * (double)c->cfg.width * (double)c->cfg.height;
    r->final_loss = c->hstate->loss_sum / n;
    double mse = c->hstate->sq_clamp_sum / n;
    double ps = mse > 0.0 ? 10.0 * log10(1.0 / mse) : 99.0;
    r->psnr = ps > 99.0 ? 99.0 : ps;
    r->iters_run = iters_run;
    r->first_nonfinite_iter = c->hstate->first_nonfinite_iter;
    r->n_active = n_active;
    r->n_pairs = host_pairs(c);
}

}  // namespace gs2d

using namespace gs2d;

extern "C" {

const char *gs_last_cuda_error(void) { return g_cuda_error; }

int gs_create(const gs_config *cfg, gs_ctx **out) {
    if (!cfg || !out) return GS_ERR_INVALID_ARGUMENT;
    *out = nullptr;
    if (cfg->width <= 0 || cfg->height <= 0 || cfg->max_gaussians < 1 || cfg->max_pairs < 1)
        return GS_ERR_INVALID_ARGUMENT;
    if (!(cfg->cutoff > 0.0f) || !isfinite(cfg->cutoff) || !isfinite(cfg->l_min)) return GS_ERR_INVALID_ARGUMENT;
    if (cfg->tile != TILE) return GS_ERR_UNSUPPORTED;
    const int TX = ceil_div(cfg->width, TILE), TY = ceil_div(cfg->height, TILE);
    if (TX > 32767 || TY > 32767 || (long long)TX * TY > (1 << 26)) return GS_ERR_UNSUPPORTED;
    if (cfg->max_pairs > 0x7fffffffLL - 1024) return GS_ERR_UNSUPPORTED;
    if ((long long)cfg->width * cfg->height > (1LL << 29)) return GS_ERR_UNSUPPORTED;
    int dev = 0;
    GS_CUDA_TRY(cudaGetDevice(&dev));
    cudaDeviceProp prop;
    GS_CUDA_TRY(cudaGetDeviceProperties(&prop, dev));

    gs_ctx *c = new (std::nothrow) gs_ctx;
    if (!c) return GS_ERR_INVALID_ARGUMENT;
    memset(c, 0, sizeof *c);
    c->cfg = *cfg;
    c->TX = TX;
    c->TY = TY;
    c->T = TX * TY;
    c->device = dev;
    c->sm_count = prop.multiProcessorCount;
    c->cap_pairs = cfg->max_pairs;
    const size_t N = (size_t)cfg->max_gaussians, T = (size_t)c->T, P = (size_t)cfg->max_pairs;
    // bucket capacity per tile: 4x the mean capacity max_pairs / T, at least 512, never more than a
    // tile can legitimately receive (one entry per Gaussian, at most max_pairs in total)
    {
        long long cap = 4 * ((long long)P / (long long)T + 1);
        if (cap < 512) cap = 512;
        const long long most = (long long)(N < P ? N : P);
        if (cap > most) cap = most;
        cap = (cap + 31) / 32 * 32;
        if ((long long)T * cap > 0x7fffffffLL * 4) {
            delete c;
            return GS_ERR_UNSUPPORTED;
        }
        c->tile_cap = (int)cap;
    }
#define GS_ALLOC(ptr, bytes)                                  \
    do {                                                      \
        cudaError_t _e = cudaMalloc((void **)&(ptr), (bytes)); \
        if (_e != cudaSuccess) {                              \
            set_cuda_error(_e, "cudaMalloc " #ptr);           \
            gs_destroy(c);                                    \
            return GS_ERR_CUDA;                               \
        }                                                     \
    } while (0)
    GS_ALLOC(c->rec, sizeof(Rec) * N);
    GS_ALLOC(c->tile_count, sizeof(int) * T * 2);
    GS_ALLOC(c->tile_n, sizeof(int) * T);
    GS_ALLOC(c->bucket, sizeof(int) * T * (size_t)c->tile_cap);
    c->spill_cap = (int)((P / 4 > 4096 ? P / 4 : 4096));
    GS_ALLOC(c->spill, sizeof(int2) * (size_t)c->spill_cap);
    GS_ALLOC(c->tile_order, sizeof(int) * T * NCLS * 3);
    GS_ALLOC(c->acc, sizeof(float) * 8 * N);
    GS_ALLOC(c->tile_stats, sizeof(TileStats) * T);
    GS_ALLOC(c->tile_flag, T);
    GS_ALLOC(c->dstate, sizeof(DeviceState));
#undef GS_ALLOC
    cudaError_t e = cudaMallocHost((void **)&c->hstate, sizeof(DeviceState));
    if (e == cudaSuccess) e = cudaMemset(c->tile_count, 0, sizeof(int) * T * 2);
    if (e == cudaSuccess) e = cudaMemset(c->tile_n, 0, sizeof(int) * T);
    if (e == cudaSuccess) e = cudaMemset(c->acc, 0, sizeof(float) * 8 * N);
    if (e == cudaSuccess) {
        // forward launch 0 walks the identity order: every tile in class 0
        DeviceState init;
        memset(&init, 0, sizeof init);
        init.n_class[0][0] = c->T;
        e = cudaMemcpy(c->dstate, &init, sizeof init, cudaMemcpyHostToDevice);
    }
    if (e == cudaSuccess) {
        int *ident = new (std::nothrow) int[T];
        if (!ident) e = cudaErrorMemoryAllocation;
        else {
            for (size_t i = 0; i < T; ++i) ident[i] = (int)i;
            e = cudaMemcpy(c->tile_order, ident, sizeof(int) * T, cudaMemcpyHostToDevice);
            delete[] ident;
        }
    }
    if (e == cudaSuccess) e = cudaDeviceSynchronize();
    if (e != cudaSuccess) {
        set_cuda_error(e, "gs_create init");
        gs_destroy(c);
        return GS_ERR_CUDA;
    }
    memset(c->hstate, 0, sizeof(DeviceState));
    *out = c;
    return GS_OK;
}

int gs_set_roi(gs_ctx *c, const unsigned char *roi_mask, void *stream) {
    if (!c) return GS_ERR_INVALID_ARGUMENT;
    c->bg_valid = false;
    if (!roi_mask) {
        c->roi = nullptr;
        c->roi_count = 0;
        return GS_OK;
    }
    cudaStream_t s = (cudaStream_t)stream;
    int rc;
    if ((rc = launch_roi_count(c, roi_mask, s))) return rc;
    if ((rc = read_state(c, s))) return rc;
    if (c->hstate->roi_pixels == 0) return GS_ERR_EMPTY_MASK;
    c->roi = roi_mask;
    c->roi_count = (long long)c->hstate->roi_pixels;
    return GS_OK;
}

int gs_set_deterministic(gs_ctx *c, int on) {
    if (!c || (on != 0 && on != 1)) return GS_ERR_INVALID_ARGUMENT;
    if (on) {
        const int rc = ensure_pair_slots(c);
        if (rc) return rc;
    }
    c->deterministic = on != 0;
    c->fresh_mu = nullptr;  // bins made under the previous setting are not reused
    return GS_OK;
}

int gs_destroy(gs_ctx *c) {
    if (!c) return GS_OK;
    void *dev[] = {c->rec,        c->tile_count, c->tile_n,        c->bucket,     c->spill,      c->tile_order,
                   c->acc,        c->pair_info,  c->pair_mom,   c->tile_stats,    c->tile_flag,  c->image_scratch,
                   c->host_params, c->host_m,    c->host_v,
                   c->roi_grey,   c->roi_cin,    c->roi_cout,      c->roi_blk,    c->dstate};
    for (void *p : dev)
        if (p) cudaFree(p);
    for (void *p : c->sp_buf)
        if (p) cudaFree(p);
    if (c->sel_changed) cudaFree(c->sel_changed);
    if (c->sel_active) cudaFree(c->sel_active);
    if (c->bg_target) cudaFree(c->bg_target);
    if (c->hstate) cudaFreeHost(c->hstate);
    delete c;
    return GS_OK;
}

static bool quant_from_spec(const gs_quant_spec *q, QuantDev *d) {
    memset(d, 0, sizeof *d);
    if (!q) return true;
    for (int j = 0; j < 9; ++j) {
        if (q->levels[j] < 0 || q->levels[j] > 65535) return false;
        if (q->levels[j] > 0 && (!(q->step[j] > 0.0f) || !(q->inv_step[j] > 0.0f) || !isfinite(q->lo[j]))) return false;
        d->levels[j] = q->levels[j];
        d->lo[j] = q->lo[j];
        d->step[j] = q->step[j];
        d->inv_step[j] = q->inv_step[j];
    }
    d->on = 1;
    return true;
}

int gs_set_quantization(gs_ctx *c, const gs_quant_spec *spec) {
    if (!c) return GS_ERR_INVALID_ARGUMENT;
    QuantDev d;
    if (!quant_from_spec(spec, &d)) return GS_ERR_INVALID_ARGUMENT;
    c->quant = d;
    c->fresh_mu = nullptr;  // bins made under the previous setting are not reused
    c->bg_valid = false;
    return GS_OK;
}

int gs_fake_quantize(gs_ctx *c, gs_params p, const gs_quant_spec *spec, gs_params out, void *stream) {
    out.n = p.n;
    if (!params_ok(c, p) || !params_ok(c, out) || !spec) return GS_ERR_INVALID_ARGUMENT;
    QuantDev d;
    if (!quant_from_spec(spec, &d)) return GS_ERR_INVALID_ARGUMENT;
    discard_fresh_bins(c, (cudaStream_t)stream);
    drop_fit_target(c);
    return launch_fake_quantize(c, p, out, d, (cudaStream_t)stream);
}

int gs_status(gs_ctx *c, void *stream) {
    if (!c) return GS_ERR_INVALID_ARGUMENT;
    cudaStream_t s = (cudaStream_t)stream;
    int rc = read_state(c, s);
    if (rc) return rc;
    return consume_flags(c, s);
}

int gs_init_roi(gs_ctx *c, const float *frame, const unsigned char *roi_mask, int n, unsigned long long seed,
                float s_min, float s_max, gs_params out, void *stream) {
    out.n = n;
    if (!frame || !roi_mask || !params_ok(c, out)) return GS_ERR_INVALID_ARGUMENT;
    if (!(s_min > 0.0f) || !(s_max >= s_min) || !isfinite(s_max)) return GS_ERR_INVALID_ARGUMENT;
    discard_fresh_bins(c, (cudaStream_t)stream);  // `out` is overwritten: bins left for it are stale
    c->bg_valid = false;
    return run_init_roi(c, frame, roi_mask, n, seed, s_min, s_max, out, (cudaStream_t)stream);
}

int gs_init_superpixel(gs_ctx *c, const float *frame, const unsigned char *roi_mask, int n_segments, int compactness,
                       int kmeans_iters, gs_params out, int *labels_out, int *n_out_host, void *stream) {
    out.n = n_segments;
    if (!frame || !roi_mask || !params_ok(c, out) || !n_out_host) return GS_ERR_INVALID_ARGUMENT;
    if (compactness < 0 || compactness > 4096 || kmeans_iters < 0) return GS_ERR_INVALID_ARGUMENT;
    discard_fresh_bins(c, (cudaStream_t)stream);
    c->bg_valid = false;
    return run_init_superpixel(c, frame, roi_mask, n_segments, compactness, kmeans_iters, out, labels_out, n_out_host,
                               (cudaStream_t)stream);
}

int gs_render(gs_ctx *c, gs_params p, float *image_out, int clamp, void *stream) {
    if (!params_ok(c, p) || !image_ok(c, image_out)) return GS_ERR_INVALID_ARGUMENT;
    cudaStream_t s = (cudaStream_t)stream;
    discard_fresh_bins(c, s);  // bins left by a resumable gs_fit_steps are not trusted across calls
    drop_fit_target(c);        // nor is its derived fit target
    int rc = ensure_bins(c, p, s);
    if (rc) return rc;
    return launch_forward(c, clamp ? FWD_IMAGE_CLAMP : FWD_IMAGE, image_out, nullptr, s);
}

int gs_decode(gs_ctx *c, gs_params p, float *image_out, void *stream) { return gs_render(c, p, image_out, 1, stream); }

int gs_render_backward(gs_ctx *c, gs_params p, const float *dL_dimage, gs_params g, void *stream) {
    g.n = p.n;
    if (!params_ok(c, p) || !params_ok(c, g) || !dL_dimage) return GS_ERR_INVALID_ARGUMENT;
    cudaStream_t s = (cudaStream_t)stream;
    int rc;
    discard_fresh_bins(c, s);
    drop_fit_target(c);
    if ((rc = ensure_bins(c, p, s))) return rc;
    if ((rc = launch_fit_tiles(c, FIT_GRAD, dL_dimage, 0, s))) return rc;
    return launch_grad_finalize(c, p, g, s);
}

int gs_adam_step(gs_ctx *c, gs_params p, gs_params grad, gs_adam_state st, const float lr[4], float beta1, float beta2,
                 float eps, int t, const unsigned char *active, void *stream) {
    grad.n = p.n;
    if (!params_ok(c, p) || !params_ok(c, grad) || !state_ok(st) || !lr || t < 1) return GS_ERR_INVALID_ARGUMENT;
    const float bc1 = (float)(1.0 - pow((double)beta1, (double)t));
    const float bc2 = (float)(1.0 - pow((double)beta2, (double)t));
    // the parameters change in place: bins a resumable gs_fit_steps left for these arrays are stale now
    discard_fresh_bins(c, (cudaStream_t)stream);
    c->bg_valid = false;
    return launch_adam(c, p, &grad, st, lr, beta1, beta2, eps, bc1, bc2, active, false, (cudaStream_t)stream);
}

int gs_fit_steps(gs_ctx *c, const float *frame, gs_params p, gs_adam_state st, const gs_fit_opts *o, int t0,
                 const unsigned char *active, void *stream) {
    if (!params_ok(c, p) || !frame || !state_ok(st) || !o || o->iters < 0 || t0 < 1) return GS_ERR_INVALID_ARGUMENT;
    cudaStream_t s = (cudaStream_t)stream;
    // bins of a selective binning list the Gaussians the MASK selected when they were made: a fit that starts
    // (t0 == 1) reads the mask as it is now
    if (!o->resume || (t0 == 1 && c->fresh && c->fresh_mode != 0)) discard_fresh_bins(c, s);
    // a fit that starts at t0 = 1 is a new fit: a non-finite latch of an earlier one must not stop its updates
    if (t0 == 1) GS_CUDA_TRY(cudaMemsetAsync(&c->dstate->first_nonfinite_iter, 0, sizeof(int), s));
    // the derived fit target (frame - render(frozen), ROI mask) is kept only while a resumed fit continues: a call
    // that starts a fit (t0 == 1) rebuilds it from the frame, mask and ROI as they are now
    const bool keep_target = o->resume != 0 && t0 > 1;
    if (!keep_target) drop_fit_target(c);
    return fit_loop(c, frame, p, st, o, t0, active, o->resume != 0, s, keep_target);
}

int gs_profile_fit_step(gs_ctx *c, const float *frame, gs_params p, gs_adam_state st, const gs_fit_opts *o, int t,
                        const unsigned char *active, float *ms_out_host, void *stream) {
    if (!params_ok(c, p) || !frame || !state_ok(st) || !o || t < 1 || !ms_out_host) return GS_ERR_INVALID_ARGUMENT;
    cudaStream_t s = (cudaStream_t)stream;
    int rc;
    // the derived target of a masked / ROI step is built (t == 1) or reused (t > 1) BEFORE the first event: the
    // one-off frozen render and subtraction are not part of the three times reported
    const float *target = frame;
    if (t == 1) drop_fit_target(c);
    if ((active || c->roi) && (rc = selective_target(c, frame, p, active, true, s, &target))) return rc;
    cudaEvent_t ev[4] = {nullptr, nullptr, nullptr, nullptr};
    for (int i = 0; i < 4; ++i) {
        const cudaError_t ce = cudaEventCreate(&ev[i]);
        if (ce != cudaSuccess) {
            for (int j = 0; j < i; ++j) cudaEventDestroy(ev[j]);
            set_cuda_error(ce, "cudaEventCreate");
            return GS_ERR_CUDA;
        }
    }
    cudaEventRecord(ev[0], s);
    rc = ensure_bins(c, p, s, active, 1);  // nothing to do when the previous profiled step left its bins
    cudaEventRecord(ev[1], s);
    if (!rc) rc = launch_fit_tiles(c, FIT_LOSS, target, t, s);
    cudaEventRecord(ev[2], s);
    const float bc1 = (float)(1.0 - pow((double)o->beta1, (double)t));
    const float bc2 = (float)(1.0 - pow((double)o->beta2, (double)t));
    if (!rc) rc = launch_adam(c, p, nullptr, st, o->lr, o->beta1, o->beta2, o->eps, bc1, bc2, active, true, s);
    cudaEventRecord(ev[3], s);
    cudaError_t e = cudaStreamSynchronize(s);
    for (int i = 0; i < 3 && e == cudaSuccess; ++i) e = cudaEventElapsedTime(&ms_out_host[i], ev[i], ev[i + 1]);
    for (int i = 0; i < 4; ++i) cudaEventDestroy(ev[i]);
    if (e != cudaSuccess) {
        set_cuda_error(e, "gs_profile_fit_step");
        return GS_ERR_CUDA;
    }
    return rc;
}

int gs_profile_decode(gs_ctx *c, gs_params p, float *image_out, float *ms_out_host, void *stream) {
    if (!params_ok(c, p) || !image_ok(c, image_out) || !ms_out_host) return GS_ERR_INVALID_ARGUMENT;
    cudaStream_t s = (cudaStream_t)stream;
    cudaEvent_t ev[3] = {nullptr, nullptr, nullptr};
    for (int i = 0; i < 3; ++i) {
        const cudaError_t ce = cudaEventCreate(&ev[i]);
        if (ce != cudaSuccess) {
            for (int j = 0; j < i; ++j) cudaEventDestroy(ev[j]);
            set_cuda_error(ce, "cudaEventCreate");
            return GS_ERR_CUDA;
        }
    }
    discard_fresh_bins(c, s);
    drop_fit_target(c);
    cudaEventRecord(ev[0], s);
    int rc = ensure_bins(c, p, s);
    cudaEventRecord(ev[1], s);
    if (!rc) rc = launch_forward(c, FWD_IMAGE_CLAMP, image_out, nullptr, s);
    cudaEventRecord(ev[2], s);
    cudaError_t e = cudaStreamSynchronize(s);
    for (int i = 0; i < 2 && e == cudaSuccess; ++i) e = cudaEventElapsedTime(&ms_out_host[i], ev[i], ev[i + 1]);
    for (int i = 0; i < 3; ++i) cudaEventDestroy(ev[i]);
    if (e != cudaSuccess) {
        set_cuda_error(e, "gs_profile_decode");
        return GS_ERR_CUDA;
    }
    return rc;
}

int gs_loss_psnr(gs_ctx *c, const float *frame, gs_params p, double *loss_host, double *psnr_host, void *stream) {
    if (!params_ok(c, p) || !frame) return GS_ERR_INVALID_ARGUMENT;
    cudaStream_t s = (cudaStream_t)stream;
    discard_fresh_bins(c, s);
    int rc = final_stats(c, frame, p, s);
    if (rc) return rc;
    gs_fit_report r;
    fill_report(c, &r, 0, 0);
    if (loss_host) *loss_host = r.final_loss;
    if (psnr_host) *psnr_host = r.psnr;
    return consume_flags(c, s);
}

int gs_encode_iframe(gs_ctx *c, const float *frame, gs_params p, gs_adam_state st, const gs_fit_opts *o,
                     gs_fit_report *report, void *stream) {
    if (!params_ok(c, p) || !frame || !state_ok(st) || !o || o->iters < 0) return GS_ERR_INVALID_ARGUMENT;
    cudaStream_t s = (cudaStream_t)stream;
    GS_CUDA_TRY(cudaMemsetAsync(st.m, 0, sizeof(float) * 9 * (size_t)p.n, s));
    GS_CUDA_TRY(cudaMemsetAsync(st.v, 0, sizeof(float) * 9 * (size_t)p.n, s));
    GS_CUDA_TRY(cudaMemsetAsync(&c->dstate->first_nonfinite_iter, 0, sizeof(int), s));
    discard_fresh_bins(c, s);
    int rc = fit_loop(c, frame, p, st, o, 1, nullptr, true, s);
    if (rc) return rc;
    if ((rc = final_stats(c, frame, p, s))) return rc;
    int nf = c->hstate->first_nonfinite_iter;
    fill_report(c, report, nf ? nf - 1 : o->iters, p.n);
    return consume_flags(c, s);
}

int gs_encode_iframe_sched(gs_ctx *c, const float *frame, gs_params p, gs_adam_state st, const gs_fit_opts *o,
                           const gs_fit_schedule *sc, gs_fit_report *report, void *stream) {
    if (!params_ok(c, p) || !frame || !state_ok(st) || !o || o->iters < 0 || !sc) return GS_ERR_INVALID_ARGUMENT;
    if (sc->target_psnr > 0.0f && sc->check_every < 1) return GS_ERR_INVALID_ARGUMENT;
    cudaStream_t s = (cudaStream_t)stream;
    GS_CUDA_TRY(cudaMemsetAsync(st.m, 0, sizeof(float) * 9 * (size_t)p.n, s));
    GS_CUDA_TRY(cudaMemsetAsync(st.v, 0, sizeof(float) * 9 * (size_t)p.n, s));
    GS_CUDA_TRY(cudaMemsetAsync(&c->dstate->first_nonfinite_iter, 0, sizeof(int), s));
    discard_fresh_bins(c, s);
    int rc, done = 0;
    bool have_stats = false;
    const float *target = frame;
    if (c->roi && o->iters > 0 && (rc = selective_target(c, frame, p, nullptr, false, s, &target))) return rc;
    for (int k = 1; k <= o->iters; ++k) {
        double scale = 1.0;
        for (int j = 0; j < 2; ++j)
            if ((double)(k - 1) >= floor((double)sc->milestone[j] * (double)o->iters + 0.5)) scale *= (double)sc->decay;
        float lr[4];
        for (int j = 0; j < 4; ++j) lr[j] = (float)((double)o->lr[j] * scale);
        if ((rc = ensure_bins(c, p, s))) return rc;
        if ((rc = launch_fit_tiles(c, FIT_LOSS, target, k, s))) return rc;
        const float bc1 = (float)(1.0 - pow((double)o->beta1, (double)k));
        const float bc2 = (float)(1.0 - pow((double)o->beta2, (double)k));
        if ((rc = launch_adam(c, p, nullptr, st, lr, o->beta1, o->beta2, o->eps, bc1, bc2, nullptr, true, s))) return rc;
        done = k;
        have_stats = false;
        if (sc->target_psnr > 0.0f && k % sc->check_every == 0) {
            if ((rc = final_stats(c, frame, p, s))) return rc;
            have_stats = true;
            gs_fit_report r;
            fill_report(c, &r, k, p.n);
            if (c->hstate->first_nonfinite_iter || r.psnr >= (double)sc->target_psnr) break;
        }
    }
    if (!have_stats && (rc = final_stats(c, frame, p, s))) return rc;
    const int nf = c->hstate->first_nonfinite_iter;
    fill_report(c, report, nf ? nf - 1 : done, p.n);
    return consume_flags(c, s);
}

int gs_pframe_select(gs_ctx *c, const float *frame, gs_params p, float tau, double *tile_resid_out,
                     unsigned char *tile_flag_out, unsigned char *active_out, int *n_active_host, void *stream) {
    if (!params_ok(c, p) || !frame || !active_out) return GS_ERR_INVALID_ARGUMENT;
    cudaStream_t s = (cudaStream_t)stream;
    int rc;
    discard_fresh_bins(c, s);
    drop_fit_target(c);
    if ((rc = ensure_bins(c, p, s))) return rc;
    if ((rc = launch_forward(c, FWD_STATS, nullptr, frame, s))) return rc;
    if ((rc = launch_reduce_stats(c, s))) return rc;
    if ((rc = launch_select(c, tau, active_out, p.n, s))) return rc;
    if (tile_resid_out && (rc = launch_tile_resid(c, tile_resid_out, s))) return rc;
    if (tile_flag_out)
        GS_CUDA_TRY(cudaMemcpyAsync(tile_flag_out, c->tile_flag, (size_t)c->T, cudaMemcpyDeviceToDevice, s));
    if ((rc = read_state(c, s))) return rc;
    if (n_active_host) *n_active_host = c->hstate->n_active;
    return consume_flags(c, s);
}

int gs_pframe_select_pixels(gs_ctx *c, const float *frame, gs_params p, float tau, float influence_eps, int dilate,
                            const unsigned char *changed_in, unsigned char *changed_out, unsigned char *active_out,
                            int *n_active_host, void *stream) {
    if (!params_ok(c, p) || !frame || !active_out) return GS_ERR_INVALID_ARGUMENT;
    if (!(influence_eps > 0.0f) || !(influence_eps < 1.0f)) return GS_ERR_INVALID_ARGUMENT;
    cudaStream_t s = (cudaStream_t)stream;
    const float thr = (float)log2(1.0 / (double)influence_eps);
    int rc;
    discard_fresh_bins(c, s);
    drop_fit_target(c);
    if ((rc = ensure_bins(c, p, s))) return rc;
    if (changed_in) {
        if ((rc = launch_sort_tiles(c, s))) return rc;  // only the lists are needed
    } else {
        if (!c->image_scratch)
            GS_CUDA_TRY(cudaMalloc(&c->image_scratch, sizeof(float) * 3 * (size_t)c->cfg.width * c->cfg.height));
        if ((rc = launch_forward(c, FWD_IMAGE_CLAMP, c->image_scratch, nullptr, s))) return rc;
    }
    if ((rc = launch_select_pixels(c, frame, c->image_scratch, tau, thr, dilate, changed_in, changed_out, active_out,
                                   p.n, s)))
        return rc;
    if ((rc = read_state(c, s))) return rc;
    if (n_active_host) *n_active_host = c->hstate->n_active;
    return consume_flags(c, s);
}

int gs_encode_pframe_pixels(gs_ctx *c, const float *frame, gs_params p, gs_adam_state st, float tau,
                            float influence_eps, int dilate, const gs_fit_opts *o, unsigned char *active_out,
                            gs_fit_report *report, void *stream) {
    if (!params_ok(c, p) || !frame || !state_ok(st) || !o || o->iters < 0 || !active_out)
        return GS_ERR_INVALID_ARGUMENT;
    cudaStream_t s = (cudaStream_t)stream;
    int n_active = 0;
    int rc = gs_pframe_select_pixels(c, frame, p, tau, influence_eps, dilate, nullptr, nullptr, active_out, &n_active,
                                     stream);
    if (rc) return rc;
    if (n_active == 0) {  // nothing changed: report the state as it is
        if ((rc = final_stats(c, frame, p, s))) return rc;
        fill_report(c, report, 0, 0);
        return consume_flags(c, s);
    }
    GS_CUDA_TRY(cudaMemsetAsync(st.m, 0, sizeof(float) * 9 * (size_t)p.n, s));
    GS_CUDA_TRY(cudaMemsetAsync(st.v, 0, sizeof(float) * 9 * (size_t)p.n, s));
    GS_CUDA_TRY(cudaMemsetAsync(&c->dstate->first_nonfinite_iter, 0, sizeof(int), s));
    if ((rc = fit_loop(c, frame, p, st, o, 1, active_out, true, s))) return rc;
    if ((rc = final_stats(c, frame, p, s))) return rc;
    int nf = c->hstate->first_nonfinite_iter;
    fill_report(c, report, nf ? nf - 1 : o->iters, n_active);
    return consume_flags(c, s);
}

int gs_encode_pframe(gs_ctx *c, const float *frame, gs_params p, gs_adam_state st, float tau, const gs_fit_opts *o,
                     unsigned char *active_out, gs_fit_report *report, void *stream) {
    if (!params_ok(c, p) || !frame || !state_ok(st) || !o || o->iters < 0 || !active_out)
        return GS_ERR_INVALID_ARGUMENT;
    cudaStream_t s = (cudaStream_t)stream;
    int n_active = 0;
    int rc = gs_pframe_select(c, frame, p, tau, nullptr, nullptr, active_out, &n_active, stream);
    if (rc) return rc;
    if (n_active == 0) {  // nothing changed: the stats of the selection render are the report
        fill_report(c, report, 0, 0);
        return GS_OK;
    }
    GS_CUDA_TRY(cudaMemsetAsync(st.m, 0, sizeof(float) * 9 * (size_t)p.n, s));
    GS_CUDA_TRY(cudaMemsetAsync(st.v, 0, sizeof(float) * 9 * (size_t)p.n, s));
    GS_CUDA_TRY(cudaMemsetAsync(&c->dstate->first_nonfinite_iter, 0, sizeof(int), s));
    // selective refit: only the selected Gaussians are binned and fitted, against frame - render(frozen)
    if ((rc = fit_loop(c, frame, p, st, o, 1, active_out, true, s))) return rc;
    if ((rc = final_stats(c, frame, p, s))) return rc;
    int nf = c->hstate->first_nonfinite_iter;
    fill_report(c, report, nf ? nf - 1 : o->iters, n_active);
    return consume_flags(c, s);
}

// GoP loop: host-side composition of the single-frame calls; the frame-type rule is f % K.
int gs_encode_gop(gs_ctx *c, const float *const *frames, const unsigned char *const *roi_masks, int n_frames,
                  const gs_gop_opts *o, gs_params work, gs_adam_state st, gs_params *out, unsigned char *active_out,
                  gs_frame_report *reports, void *stream) {
    if (!c || !frames || !o || !out || n_frames < 0 || o->gop_length < 1 || o->n < 1 || o->n > c->cfg.max_gaussians)
        return GS_ERR_INVALID_ARGUMENT;
    if (!work.mu || !work.chol || !work.rgb || !work.opacity || !state_ok(st)) return GS_ERR_INVALID_ARGUMENT;
    if (o->init != 0 && o->init != 1) return GS_ERR_INVALID_ARGUMENT;
    cudaStream_t s = (cudaStream_t)stream;
    const bool plain = o->sched.decay == 1.0f && !(o->sched.target_psnr > 0.0f);
    int n_cur = 0;
    for (int f = 0; f < n_frames; ++f) {
        if (!frames[f] || !out[f].mu || !out[f].chol || !out[f].rgb || !out[f].opacity) return GS_ERR_INVALID_ARGUMENT;
        const bool is_i = f % o->gop_length == 0;
        gs_frame_report rep;
        memset(&rep, 0, sizeof rep);
        rep.type = is_i ? 0 : 1;
        if (reports) reports[f].type = rep.type;
        unsigned char *act = active_out ? active_out + (size_t)f * (size_t)o->n : nullptr;
        int rc;
        if (is_i) {
            if (!roi_masks || !roi_masks[f]) return GS_ERR_INVALID_ARGUMENT;
            work.n = o->n;
            if (o->init == 0) {
                rc = gs_init_roi(c, frames[f], roi_masks[f], o->n, o->seed + (unsigned long long)f, o->s_min, o->s_max,
                                 work, stream);
                n_cur = o->n;
            } else {
                rc = gs_init_superpixel(c, frames[f], roi_masks[f], o->n, o->compactness, o->kmeans_iters, work, nullptr,
                                        &n_cur, stream);
            }
            if (rc) return rc;
            work.n = n_cur;
            rc = plain ? gs_encode_iframe(c, frames[f], work, st, &o->iframe, &rep.fit, stream)
                       : gs_encode_iframe_sched(c, frames[f], work, st, &o->iframe, &o->sched, &rep.fit, stream);
            if (rc) return rc;
            if (act) {
                GS_CUDA_TRY(cudaMemsetAsync(act, 1, (size_t)n_cur, s));
                if (n_cur < o->n) GS_CUDA_TRY(cudaMemsetAsync(act + n_cur, 0, (size_t)(o->n - n_cur), s));
            }
        } else {
            work.n = n_cur;
            unsigned char *sel = act ? act : c->sel_active;
            if (!sel) {  // no caller buffer: a context-owned one, allocated on first use
                GS_CUDA_TRY(cudaMalloc(&c->sel_active, (size_t)c->cfg.max_gaussians));
                sel = c->sel_active;
            }
            rc = o->pixel_select ? gs_encode_pframe_pixels(c, frames[f], work, st, o->tau, o->influence_eps, o->dilate,
                                                           &o->pframe, sel, &rep.fit, stream)
                                 : gs_encode_pframe(c, frames[f], work, st, o->tau, &o->pframe, sel, &rep.fit, stream);
            if (rc) return rc;
            if (act && n_cur < o->n) GS_CUDA_TRY(cudaMemsetAsync(act + n_cur, 0, (size_t)(o->n - n_cur), s));
        }
        rep.n = n_cur;
        out[f].n = n_cur;
        const size_t nn = (size_t)n_cur * sizeof(float);
        GS_CUDA_TRY(cudaMemcpyAsync(out[f].mu, work.mu, 2 * nn, cudaMemcpyDeviceToDevice, s));
        GS_CUDA_TRY(cudaMemcpyAsync(out[f].chol, work.chol, 3 * nn, cudaMemcpyDeviceToDevice, s));
        GS_CUDA_TRY(cudaMemcpyAsync(out[f].rgb, work.rgb, 3 * nn, cudaMemcpyDeviceToDevice, s));
        GS_CUDA_TRY(cudaMemcpyAsync(out[f].opacity, work.opacity, nn, cudaMemcpyDeviceToDevice, s));
        if (reports) reports[f] = rep;
    }
    GS_CUDA_TRY(cudaStreamSynchronize(s));
    return GS_OK;
}

int gs_get_tile_loss(gs_ctx *c, double *tile_sq_out, void *stream) {
    if (!c || !tile_sq_out) return GS_ERR_INVALID_ARGUMENT;
    return launch_tile_sq(c, tile_sq_out, (cudaStream_t)stream);
}

int gs_get_bins(gs_ctx *c, int *range_out, int *list_out, long long cap_list, long long *P_host, void *stream) {
    if (!c || !range_out || !P_host) return GS_ERR_INVALID_ARGUMENT;
    cudaStream_t s = (cudaStream_t)stream;
    int rc = read_state(c, s);
    if (rc) return rc;
    // a binning nobody has consumed yet (left by a resumable gs_fit_steps), or buckets that a fit
    // iteration consumed without sorting: bring them into the canonical order now
    const bool was_fresh = c->fresh;
    if ((rc = launch_sort_tiles(c, s))) return rc;
    if (was_fresh && (rc = read_state(c, s))) return rc;
    const long long P = host_pairs(c);
    *P_host = P;
    if (P > c->cap_pairs || c->hstate->tile_ovf[c->epoch & 1u]) return GS_ERR_CAPACITY;
    if (list_out && P > cap_list) return GS_ERR_CAPACITY;
    if ((rc = launch_compact(c, range_out, list_out, s))) return rc;
    GS_CUDA_TRY(cudaStreamSynchronize(s));
    return GS_OK;
}

// ---- host-buffer entry points ------------------------------------------------------------

static int ensure_host_scratch(gs_ctx *c, bool fit) {
    const size_t N = (size_t)c->cfg.max_gaussians, px = (size_t)c->cfg.width * c->cfg.height * 3;
    if (!c->host_params) GS_CUDA_TRY(cudaMalloc(&c->host_params, sizeof(float) * (9 * N + 16)));
    if (!c->image_scratch) GS_CUDA_TRY(cudaMalloc(&c->image_scratch, sizeof(float) * px));
    if (fit) {
        if (!c->host_m) GS_CUDA_TRY(cudaMalloc(&c->host_m, sizeof(float) * 9 * N));
        if (!c->host_v) GS_CUDA_TRY(cudaMalloc(&c->host_v, sizeof(float) * 9 * N));
    }
    return GS_OK;
}

static gs_params device_view(gs_ctx *c, int n) {
    gs_params d;
    auto up4 = [](size_t x) { return (x + 3) & ~(size_t)3; };  // every array 16-byte aligned
    d.mu = c->host_params;
    d.chol = d.mu + up4(2 * (size_t)n);
    d.rgb = d.chol + up4(3 * (size_t)n);
    d.opacity = d.rgb + up4(3 * (size_t)n);
    d.n = n;
    return d;
}

static int copy_params(gs_ctx *c, const gs_params &h, const gs_params &d, cudaMemcpyKind kind, cudaStream_t s) {
    const size_t n = (size_t)h.n;
    const bool up = kind == cudaMemcpyHostToDevice;
    GS_CUDA_TRY(cudaMemcpyAsync(up ? d.mu : h.mu, up ? h.mu : d.mu, sizeof(float) * 2 * n, kind, s));
    GS_CUDA_TRY(cudaMemcpyAsync(up ? d.chol : h.chol, up ? h.chol : d.chol, sizeof(float) * 3 * n, kind, s));
    GS_CUDA_TRY(cudaMemcpyAsync(up ? d.rgb : h.rgb, up ? h.rgb : d.rgb, sizeof(float) * 3 * n, kind, s));
    GS_CUDA_TRY(cudaMemcpyAsync(up ? d.opacity : h.opacity, up ? h.opacity : d.opacity, sizeof(float) * n, kind, s));
    return GS_OK;
}

int gs_decode_host(gs_ctx *c, gs_params ph, float *image_out_host, void *stream) {
    if (!host_params_ok(c, ph) || !image_out_host) return GS_ERR_INVALID_ARGUMENT;
    cudaStream_t s = (cudaStream_t)stream;
    int rc = ensure_host_scratch(c, false);
    if (rc) return rc;
    gs_params d = device_view(c, ph.n);
    if ((rc = copy_params(c, ph, d, cudaMemcpyHostToDevice, s))) return rc;
    if ((rc = gs_render(c, d, c->image_scratch, 1, stream))) return rc;
    GS_CUDA_TRY(cudaMemcpyAsync(image_out_host, c->image_scratch,
                                sizeof(float) * 3 * (size_t)c->cfg.width * c->cfg.height, cudaMemcpyDeviceToHost, s));
    if ((rc = read_state(c, s))) return rc;
    return consume_flags(c, s);
}

int gs_encode_iframe_host(gs_ctx *c, const float *frame_host, gs_params ph, const gs_fit_opts *o, gs_fit_report *report,
                          void *stream) {
    if (!host_params_ok(c, ph) || !frame_host || !o) return GS_ERR_INVALID_ARGUMENT;
    cudaStream_t s = (cudaStream_t)stream;
    int rc = ensure_host_scratch(c, true);
    if (rc) return rc;
    gs_params d = device_view(c, ph.n);
    GS_CUDA_TRY(cudaMemcpyAsync(c->image_scratch, frame_host, sizeof(float) * 3 * (size_t)c->cfg.width * c->cfg.height,
                                cudaMemcpyHostToDevice, s));
    if ((rc = copy_params(c, ph, d, cudaMemcpyHostToDevice, s))) return rc;
    gs_adam_state st = {c->host_m, c->host_v};
    rc = gs_encode_iframe(c, c->image_scratch, d, st, o, report, stream);
    if (rc && rc != GS_ERR_NONFINITE) return rc;
    int rc2 = copy_params(c, ph, d, cudaMemcpyDeviceToHost, s);
    if (rc2) return rc2;
    GS_CUDA_TRY(cudaStreamSynchronize(s));
    return rc;
}

}  // extern "C"
