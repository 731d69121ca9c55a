// gs2d_raster.cu -- the render kernel: forward rasterizer for images, decode and statistics
// (SURVEY.md §8 rows a5, a12 and the residual statistics of a11; DESIGN.md §5 "render").
// The fit iteration's forward + loss + backward live in gs2d_fit.cu.
//
// One CTA of 64 threads (2 warps) per 16x16 tile.  The tile's list is sorted by id first
// (bit-reproducible images), then split between the two warps; a lane owns one column x eight
// rows and walks its warp's share, the records gathered through shared memory in double-buffered
// batches of 32 per warp.  Per Gaussian and lane the whitened coordinates are set up once (6 FP32
// instructions + 2 LDS) for 8 pixels, each of which costs 2 FFMA + 1 MUFU.EX2 + 3 FFMA; the two
// partial images are added in a fixed order.
#include "gs2d_internal.cuh"
#include "gs2d_sort.cuh"

namespace gs2d {

__device__ __forceinline__ float ex2_neg(float p) {  // 2^(-p), MUFU.EX2
    float w;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(w) : "f"(-p));
    return w;
}

constexpr int FWD_THREADS = 64;
constexpr int FWD_BATCH = 32;  // records staged per warp and batch (one per lane)

static_assert(FWD_THREADS == SORT_CTA_THREADS, "the forward CTA sorts its own tile");

template <int MODE>
__global__ void __launch_bounds__(FWD_THREADS)
    k_forward(TileArgs ta, const int *__restrict__ order_cur, int *__restrict__ order_next, int ord_cur, int ord_next,
              const Rec *__restrict__ rec, int W, int H, int TX, float *__restrict__ image_out,
              const float *__restrict__ target, TileStats *__restrict__ tile_stats,
              const unsigned char *__restrict__ roi) {
    __shared__ float4 s_rec[2][2][FWD_BATCH * 2];          // [warp][buffer]
    __shared__ __align__(16) float s_io[TILE * TILE * 3];  // one tile of HWC rows: warp 1's partial, then the result

    DeviceState *st = ta.st;
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const int T = gridDim.x;
    // (class sizes read straight from global memory: uniform addresses keep t and n uniform)
    const int t = tile_of_position(order_cur, T, st->n_class[ord_cur], (int)blockIdx.x);
    const int tx = t % TX, ty = t / TX;

    // lane = column x 8 rows: rows 8 hf .. 8 hf + 7 of the tile
    const int cx = lane & 15, hf = lane >> 4;
    const int gx = tx * TILE + cx, gy0 = ty * TILE + 8 * hf;
    float px = (float)gx + 0.5f;
    float py0 = (float)gy0 + 0.5f;
    // (a shuffle from the own lane: opaque to ptxas, which otherwise rematerialises both conversions
    // inside the list loop)
    px = __shfl_sync(0xffffffffu, px, lane);
    py0 = __shfl_sync(0xffffffffu, py0, lane);

    // target pixels (statistics: warp 0 owns the whole tile at the end), fetched before the sort so that
    // their latency is hidden
    float T_[8][3];
    bool in_roi[8];  // (c-16: with an ROI the statistics run over its pixels only)
#pragma unroll
    for (int i = 0; i < 8; ++i) in_roi[i] = true;
    if (MODE == FWD_STATS && wid == 0) {
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            const bool valid = gx < W && gy0 + i < H;
            const size_t off = ((size_t)(gy0 + i) * W + gx) * 3;
#pragma unroll
            for (int ch = 0; ch < 3; ++ch) T_[i][ch] = valid ? __ldg(target + off + ch) : 0.0f;
            if (roi) in_roi[i] = valid && __ldg(roi + (size_t)(gy0 + i) * W + gx) != 0;
        }
    }

    // consumer stage of the binning: the list is brought into the canonical order (ascending id),
    // so that images are bit-reproducible
    // (the warp-wide max of a value all lanes share: tells the compiler that n is warp-uniform,
    // which keeps the list loops on uniform registers and branches)
    // Programmatic dependent launch: this grid may have started while the binning kernel was still running (its CTAs
    // trigger at their start); everything above touches nothing the binning writes.  From here on its results are
    // complete and visible.
    asm volatile("griddepcontrol.wait;" ::: "memory");
    const int n = __reduce_max_sync(0xffffffffu, tile_count_of(ta, T, t));
    if (n > 1) cta_sort_tile(ta.bucket + (size_t)t * ta.tile_cap, min(n, ta.tile_cap), tid);
    // bookkeeping of thread 0, right before the kernel returns: the tile's published length and its
    // place in the NEXT launch's order.  (Late on purpose: the atomic's latency is off the critical
    // path, and stores issued before the list loops make the compiler treat n as divergent, which
    // costs the loops their uniform branches -- measured 96 -> 124 us on the 1080p x 70k decode.)
    auto finish = [&]() {
        if (tid == 0) {
            tile_publish(ta, T, t, n);
            tile_file(st, order_next, T, ord_cur, ord_next, t, n);
        }
    };
    if (n < 0) {  // capacity exceeded: leave outputs untouched
        finish();
        return;
    }
    // The sorted list is split between the two warps (fixed split: the sums stay reproducible); warp 0,
    // which has just sorted the list alone, takes the smaller share.  Every lane walks its warp's share
    // for its 8 pixels: per Gaussian the set-up is paid once per 8 pixels.
    const int nm = min(n, ta.tile_cap);  // the bucket's part of the list
    const int n0 = (nm * 9) / 20;
    int cnt = wid == 0 ? n0 : nm - n0;
    const int *list = ta.bucket + (size_t)t * ta.tile_cap + (wid == 0 ? 0 : n0);

    float2 Cp[4][3];  // the lane's 8 rows as 4 pairs (rows 2k, 2k + 1): packed arithmetic
#pragma unroll
    for (int k = 0; k < 4; ++k) Cp[k][0] = Cp[k][1] = Cp[k][2] = make_float2(0.0f, 0.0f);

    // One pass over the bucket's part of the list; a tile that lists more than its bucket holds (slow path) comes
    // round again for its spilled entries, collected from the spill list into shared memory (the image staging
    // area, free until the end) up to 766 at a time, sorted and split between the warps like the first segment.
    // Up to 766 spilled entries the image stays bit-reproducible; beyond, batches follow the list's arrival order.
    int sp_start = 0;
    for (;;) {
        float4 nlo = make_float4(0.f, 0.f, 0.f, 0.f), nhi = nlo;
        if (lane < cnt) {
            const int gid = list[lane];
            nlo = reinterpret_cast<const float4 *>(rec)[(size_t)gid * 2];
            nhi = reinterpret_cast<const float4 *>(rec)[(size_t)gid * 2 + 1];
        }
        int buf = 0;
        for (int b0 = 0; b0 < cnt; b0 += FWD_BATCH, buf ^= 1) {
            const int bn = min(FWD_BATCH, cnt - b0);
            float4 *sr = s_rec[wid][buf];
            sr[2 * lane] = nlo;
            sr[2 * lane + 1] = nhi;
            __syncwarp();  // batch visible; the warp is done with the batch before the previous one
            if (b0 + FWD_BATCH + lane < cnt) {
                const int gid = list[b0 + FWD_BATCH + lane];
                nlo = reinterpret_cast<const float4 *>(rec)[(size_t)gid * 2];
                nhi = reinterpret_cast<const float4 *>(rec)[(size_t)gid * 2 + 1];
            } else {
                nlo = make_float4(0.f, 0.f, 0.f, 0.f);
                nhi = nlo;
            }
            // entries past the end of the share are null records (zero colour): the walk is unrolled
            // by two without a remainder loop
#pragma unroll 2
            for (int j = 0; j < ((bn + 1) & ~1); ++j) {
                const float4 lo = sr[2 * j], hi = sr[2 * j + 1];
                const float dx = px - lo.x, dy0 = py0 - lo.y;
                const float u = dx * lo.z;
                const float2 uu = dup2(u * u);
                const float2 v0 = dup2(fmaf(dx, lo.w, dy0 * hi.x));
                const float2 hx = dup2(hi.x), cr = dup2(hi.y), cg = dup2(hi.z), cb = dup2(hi.w);
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    const float2 v = __ffma2_rn(hx, c_rowpair[k], v0);
                    const float2 p = __ffma2_rn(v, v, uu);
                    const float2 w = make_float2(ex2_neg(p.x), ex2_neg(p.y));
                    Cp[k][0] = __ffma2_rn(w, cr, Cp[k][0]);
                    Cp[k][1] = __ffma2_rn(w, cg, Cp[k][1]);
                    Cp[k][2] = __ffma2_rn(w, cb, Cp[k][2]);
                }
            }
        }
        if (n <= ta.tile_cap) break;
        int *s_ids = reinterpret_cast<int *>(s_io);
        __syncthreads();  // the previous segment has been walked
        if (wid == 0) {
            const int c = spill_collect(ta.spill, spill_size(ta), t, sp_start, s_ids, TILE * TILE * 3 - 2, lane);
            if (lane == 0) s_ids[TILE * TILE * 3 - 2] = c;
        }
        __syncthreads();
        const int c = s_ids[TILE * TILE * 3 - 2];
        if (c == 0) break;
        if (c > 1) cta_sort_tile(s_ids, c, tid);
        cnt = wid == 0 ? c / 2 : c - c / 2;
        list = s_ids + (wid == 0 ? 0 : c / 2);
    }
    if (n > ta.tile_cap) __syncthreads();  // (the staging area is reused below)
    float C[8][3];
#pragma unroll
    for (int i = 0; i < 8; ++i)
#pragma unroll
        for (int ch = 0; ch < 3; ++ch) C[i][ch] = (i & 1) ? Cp[i >> 1][ch].y : Cp[i >> 1][ch].x;

    // warp 1's partial image -> shared memory; warp 0 adds its own ON TOP (first half + second half:
    // a fixed order) and owns the tile from here
    if (wid == 1) {
#pragma unroll
        for (int i = 0; i < 8; ++i)
#pragma unroll
            for (int ch = 0; ch < 3; ++ch) s_io[(8 * hf + i) * 48 + cx * 3 + ch] = C[i][ch];
    }
    __syncthreads();
    if (wid == 0) {
#pragma unroll
        for (int i = 0; i < 8; ++i)
#pragma unroll
            for (int ch = 0; ch < 3; ++ch) C[i][ch] += s_io[(8 * hf + i) * 48 + cx * 3 + ch];
    }

    if (MODE == FWD_IMAGE || MODE == FWD_IMAGE_CLAMP) {
        const bool vec_rows = (W % 4 == 0) && (tx * TILE + TILE <= W);
        if (wid == 0) {
            if (MODE == FWD_IMAGE_CLAMP) {
#pragma unroll
                for (int i = 0; i < 8; ++i)
#pragma unroll
                    for (int ch = 0; ch < 3; ++ch) C[i][ch] = fminf(fmaxf(C[i][ch], 0.0f), 1.0f);
            }
            if (vec_rows) {  // stage the tile (each lane overwrites exactly the cells it has just read)
#pragma unroll
                for (int i = 0; i < 8; ++i)
#pragma unroll
                    for (int ch = 0; ch < 3; ++ch) s_io[(8 * hf + i) * 48 + cx * 3 + ch] = C[i][ch];
            } else {
#pragma unroll
                for (int i = 0; i < 8; ++i)
                    if (gx < W && gy0 + i < H) {
                        const size_t off = ((size_t)(gy0 + i) * W + gx) * 3;
                        image_out[off] = C[i][0];
                        image_out[off + 1] = C[i][1];
                        image_out[off + 2] = C[i][2];
                    }
            }
        }
        if (vec_rows) {  // both warps write 192-byte row segments as float4
            __syncthreads();
            const int rows = min(TILE, H - ty * TILE);
#pragma unroll
            for (int k = 0; k < 3; ++k) {
                const int e = tid + k * FWD_THREADS;  // 192 float4 per tile
                const int r = e / 12, c4 = e - r * 12;
                if (r < rows) {
                    const float4 v = reinterpret_cast<const float4 *>(s_io)[e];
                    const size_t off = ((size_t)(ty * TILE + r) * W + (size_t)tx * TILE) * 3;
                    reinterpret_cast<float4 *>(image_out + off)[c4] = v;
                }
            }
        }
        finish();
        return;
    }

    if (MODE == FWD_STATS) {
        if (wid == 0) {
            float sq_raw = 0.0f, sq_cl = 0.0f, ab_cl = 0.0f;
            int nv = 0;
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                if (gx < W && gy0 + i < H && in_roi[i]) {
                    ++nv;
                    const float d0 = C[i][0] - T_[i][0], d1 = C[i][1] - T_[i][1], d2 = C[i][2] - T_[i][2];
                    sq_raw += fmaf(d0, d0, fmaf(d1, d1, d2 * d2));
                    const float e0 = fminf(fmaxf(C[i][0], 0.0f), 1.0f) - T_[i][0],
                                e1 = fminf(fmaxf(C[i][1], 0.0f), 1.0f) - T_[i][1],
                                e2 = fminf(fmaxf(C[i][2], 0.0f), 1.0f) - T_[i][2];
                    sq_cl += fmaf(e0, e0, fmaf(e1, e1, e2 * e2));
                    ab_cl += (fabsf(e0) + fabsf(e1)) + fabsf(e2);
                }
            }
            // fixed butterfly over the 32 lanes: reproducible; fp64 from here (tiles are summed in fp64)
            double a = (double)sq_raw, b = (double)sq_cl, c = (double)ab_cl;
#pragma unroll
            for (int d = 16; d > 0; d >>= 1) {
                a += __shfl_xor_sync(0xffffffffu, a, d);
                b += __shfl_xor_sync(0xffffffffu, b, d);
                c += __shfl_xor_sync(0xffffffffu, c, d);
            }
            nv = __reduce_add_sync(0xffffffffu, nv);
            if (lane == 0) {
                tile_stats[t].n_valid = nv;
                tile_stats[t].sq_raw = a;
                tile_stats[t].sq_clamp = b;
                tile_stats[t].abs_clamp = c;
            }
        }
        finish();
    }
}

// Fixed-order reduction of the per-tile statistics (one CTA): deterministic loss / PSNR sums.
__global__ void __launch_bounds__(1024) k_reduce_stats(const TileStats *__restrict__ ts, int T, DeviceState *st) {
    __shared__ double s_a[1024], s_b[1024];
    int tid = threadIdx.x;
    double a = 0.0, b = 0.0;
    for (int i = tid; i < T; i += 1024) {
        a += ts[i].sq_raw;
        b += ts[i].sq_clamp;
    }
    s_a[tid] = a;
    s_b[tid] = b;
    __syncthreads();
    for (int d = 512; d > 0; d >>= 1) {
        if (tid < d) {
            s_a[tid] += s_a[tid + d];
            s_b[tid] += s_b[tid + d];
        }
        __syncthreads();
    }
    if (tid == 0) {
        st->loss_sum = s_a[0];
        st->sq_clamp_sum = s_b[0];
    }
}

int launch_forward(gs_ctx *c, ForwardMode mode, float *image_out, const float *target, cudaStream_t s) {
    const int W = c->cfg.width, H = c->cfg.height;
    const TileArgs ta = tile_args(c);
    const int oc = (int)(c->fwd_launches % 3u), on = (int)((c->fwd_launches + 1u) % 3u);
    ++c->fwd_launches;
    const int *order_cur = c->tile_order + (size_t)oc * NCLS * c->T;
    int *order_next = c->tile_order + (size_t)on * NCLS * c->T;
    // launched as a programmatic dependent of the kernel before it in the stream: behind k_bin (which triggers
    // early) the launch latency and the prologue of this grid overlap the binning's tail
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)c->T);
    cfg.blockDim = dim3(FWD_THREADS);
    cfg.dynamicSmemBytes = 0;
    cfg.stream = s;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    const unsigned char *roi = mode == FWD_STATS ? c->roi : nullptr;
    const Rec *rec = c->rec;
    const int TXv = c->TX;
    TileStats *tstats = c->tile_stats;
#define GS_FWD(M)                                                                                                    \
    GS_CUDA_TRY(cudaLaunchKernelEx(&cfg, k_forward<M>, ta, order_cur, (int *)order_next, oc, on, rec, W, H, TXv, image_out, \
                                   target, tstats, roi))
    switch (mode) {
        case FWD_IMAGE: GS_FWD(FWD_IMAGE); break;
        case FWD_IMAGE_CLAMP: GS_FWD(FWD_IMAGE_CLAMP); break;
        case FWD_STATS: GS_FWD(FWD_STATS); break;
    }
#undef GS_FWD
    c->fresh = false;  // the bins are consumed
    c->sorted = true;
    GS_CUDA_TRY(cudaGetLastError());
    return GS_OK;
}

int launch_reduce_stats(gs_ctx *c, cudaStream_t s) {
    k_reduce_stats<<<1, 1024, 0, s>>>(c->tile_stats, c->T, c->dstate);
    GS_CUDA_TRY(cudaGetLastError());
    return GS_OK;
}

}  // namespace gs2d
