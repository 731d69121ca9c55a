// gs2d_raster.cu -- forward rasterizer, loss gradient, backward pass
// (DESIGN.md §5 "forward", "backward").
//
// Forward  : one CTA of 256 threads per 16x16 tile.  The CTA is four "list-split" groups of
//            64 threads; a group owns the whole tile (thread = one column x four rows) and
//            every fourth Gaussian of the tile's list, staged through shared memory in
//            batches of 128 records.  The four partial images are added in a fixed order.
//            Per Gaussian and thread the whitened coordinates are set up once (6 FP32
//            instructions) and each of the 4 pixels costs 2 FP32 + 1 MUFU.EX2 + 3 FFMA.
// Backward : one THREAD per (tile, Gaussian) pair walks the tile's 256 pixels and keeps the 8
//            gradient moments in registers: no cross-thread reduction at all, two 16-byte
//            vector atomics per pair.  Equal work per thread, so a plain grid-stride loop
//            balances the SMs whatever the tile-list lengths are.
#include "gs2d_internal.cuh"

namespace gs2d {

__device__ __forceinline__ float ex2_neg(float p) {  // 2^(-p), MUFU.EX2
    float w;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(w) : "f"(-p));
    return w;
}

constexpr int FWD_THREADS = 256;
constexpr int FWD_BATCH = 128;  // records staged per batch
constexpr int FWD_GROUPS = 4;

__device__ __forceinline__ double block_sum_256(double v, double *s_warp, int tid) {
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) v += __shfl_xor_sync(0xffffffffu, v, d);
    if ((tid & 31) == 0) s_warp[tid >> 5] = v;
    __syncthreads();
    double r = 0.0;
    if (tid == 0) {
#pragma unroll
        for (int w = 0; w < FWD_THREADS / 32; ++w) r += s_warp[w];
    }
    __syncthreads();
    return r;  // valid on thread 0
}

template <int MODE>
__global__ void __launch_bounds__(FWD_THREADS)
    k_forward(const int *__restrict__ range, const int *__restrict__ list, const Rec *__restrict__ rec, int W, int H,
              int TX, float *__restrict__ image_out, const float *__restrict__ target, float4 *__restrict__ gtile,
              TileStats *__restrict__ tile_stats, float g_scale, int iter, DeviceState *st, long long cap) {
    __shared__ float4 s_rec[FWD_BATCH * 2];
    __shared__ float s_part[FWD_GROUPS][3][TILE_PX];
    __shared__ __align__(16) float s_io[TILE * TILE * 3];  // one tile of HWC rows
    __shared__ float4 s_g[TILE * 17];
    __shared__ double s_warp[FWD_THREADS / 32];

    if ((long long)st->n_pairs > cap) return;  // capacity exceeded: leave outputs untouched
    const int t = blockIdx.x, tid = threadIdx.x;
    const int tx = t % TX, ty = t / TX;
    const int start = range[t], n = range[t + 1] - start;

    const int g = tid >> 6, q = tid & 63;
    const int cx = q & 15, yq = q >> 4;
    const float px = (float)(tx * TILE + cx) + 0.5f;
    const float py0 = (float)(ty * TILE + 4 * yq) + 0.5f;

    float C[4][3];
#pragma unroll
    for (int i = 0; i < 4; ++i) C[i][0] = C[i][1] = C[i][2] = 0.0f;

    for (int b0 = 0; b0 < n; b0 += FWD_BATCH) {
        const int bn = min(FWD_BATCH, n - b0);
        if (b0 > 0) __syncthreads();  // previous batch fully consumed
        if (tid < bn * 2) {
            int gid = list[start + b0 + (tid >> 1)];
            s_rec[tid] = reinterpret_cast<const float4 *>(rec)[(size_t)gid * 2 + (tid & 1)];
        }
        __syncthreads();
#pragma unroll 2
        for (int j = g; j < bn; j += FWD_GROUPS) {
            const float4 lo = s_rec[2 * j], hi = s_rec[2 * j + 1];
            const float dx = px - lo.x, dy0 = py0 - lo.y;
            const float u = dx * lo.z;
            const float uu = u * u;
            const float v0 = fmaf(dx, lo.w, dy0 * hi.x);
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                const float v = fmaf(hi.x, (float)i, v0);
                const float w = ex2_neg(fmaf(v, v, uu));
                C[i][0] = fmaf(w, hi.y, C[i][0]);
                C[i][1] = fmaf(w, hi.z, C[i][1]);
                C[i][2] = fmaf(w, hi.w, C[i][2]);
            }
        }
    }

    // fixed-order sum of the four partial images; afterwards thread `tid` owns one pixel
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        s_part[g][0][i * 64 + q] = C[i][0];
        s_part[g][1][i * 64 + q] = C[i][1];
        s_part[g][2][i * 64 + q] = C[i][2];
    }
    __syncthreads();
    float c0 = ((s_part[0][0][tid] + s_part[1][0][tid]) + s_part[2][0][tid]) + s_part[3][0][tid];
    float c1 = ((s_part[0][1][tid] + s_part[1][1][tid]) + s_part[2][1][tid]) + s_part[3][1][tid];
    float c2 = ((s_part[0][2][tid] + s_part[1][2][tid]) + s_part[2][2][tid]) + s_part[3][2][tid];
    // slot tid = i*64 + q  ->  pixel column q&15, row 4*(q>>4) + i
    const int lx = q & 15, ly = 4 * (q >> 4) + g;  // here g = tid>>6 plays the role of i
    const int gx = tx * TILE + lx, gy = ty * TILE + ly;
    const bool valid = gx < W && gy < H;
    const bool vec_rows = (W % 4 == 0) && (tx * TILE + TILE <= W);
    const int rows = min(TILE, H - ty * TILE);

    if (MODE == FWD_IMAGE || MODE == FWD_IMAGE_CLAMP) {
        if (MODE == FWD_IMAGE_CLAMP) {
            c0 = fminf(fmaxf(c0, 0.0f), 1.0f);
            c1 = fminf(fmaxf(c1, 0.0f), 1.0f);
            c2 = fminf(fmaxf(c2, 0.0f), 1.0f);
        }
        if (vec_rows) {  // stage the tile and write 192-byte row segments as float4
            s_io[ly * 48 + lx * 3 + 0] = c0;
            s_io[ly * 48 + lx * 3 + 1] = c1;
            s_io[ly * 48 + lx * 3 + 2] = c2;
            __syncthreads();
            if (tid < 192) {
                int r = tid / 12, c4 = tid - r * 12;
                if (r < rows) {
                    float4 v = reinterpret_cast<const float4 *>(s_io)[r * 12 + c4];
                    size_t off = ((size_t)(ty * TILE + r) * W + (size_t)tx * TILE) * 3;
                    reinterpret_cast<float4 *>(image_out + off)[c4] = v;
                }
            }
        } else if (valid) {
            size_t off = ((size_t)gy * W + gx) * 3;
            image_out[off] = c0;
            image_out[off + 1] = c1;
            image_out[off + 2] = c2;
        }
        return;
    }

    // FIT / STATS: fetch the target tile
    float t0 = 0.0f, t1 = 0.0f, t2 = 0.0f;
    if (vec_rows) {
        if (tid < 192) {
            int r = tid / 12, c4 = tid - r * 12;
            if (r < rows) {
                size_t off = ((size_t)(ty * TILE + r) * W + (size_t)tx * TILE) * 3;
                reinterpret_cast<float4 *>(s_io)[r * 12 + c4] = reinterpret_cast<const float4 *>(target + off)[c4];
            }
        }
        __syncthreads();
        if (valid) {
            t0 = s_io[ly * 48 + lx * 3 + 0];
            t1 = s_io[ly * 48 + lx * 3 + 1];
            t2 = s_io[ly * 48 + lx * 3 + 2];
        }
    } else if (valid) {
        size_t off = ((size_t)gy * W + gx) * 3;
        t0 = target[off];
        t1 = target[off + 1];
        t2 = target[off + 2];
    }

    if (MODE == FWD_FIT) {
        // loss on the unclamped sum (DESIGN.md §3 c-4); G = dL/dC = 2 (C - T) / (3 W H)
        float d0 = valid ? c0 - t0 : 0.0f, d1 = valid ? c1 - t1 : 0.0f, d2 = valid ? c2 - t2 : 0.0f;
        s_g[lx * 17 + ly] = make_float4(d0 * g_scale, d1 * g_scale, d2 * g_scale, 0.0f);
        float sq = fmaf(d0, d0, fmaf(d1, d1, d2 * d2));
        double tot = block_sum_256((double)sq, s_warp, tid);  // also orders s_g
        gtile[(size_t)t * TILE_PX + tid] = s_g[(tid >> 4) * 17 + (tid & 15)];  // [t][x*16+y]
        if (tid == 0) {
            tile_stats[t].sq_raw = tot;
            if (!isfinite(tot)) {
                atomicOr(&st->flags, FLAG_NONFINITE);
                atomicCAS(&st->first_nonfinite_iter, 0, iter);
            }
        }
        return;
    }

    if (MODE == FWD_STATS) {
        float sq_raw = 0.0f, sq_cl = 0.0f, ab_cl = 0.0f;
        if (valid) {
            float d0 = c0 - t0, d1 = c1 - t1, d2 = c2 - t2;
            sq_raw = fmaf(d0, d0, fmaf(d1, d1, d2 * d2));
            float e0 = fminf(fmaxf(c0, 0.0f), 1.0f) - t0, e1 = fminf(fmaxf(c1, 0.0f), 1.0f) - t1,
                  e2 = fminf(fmaxf(c2, 0.0f), 1.0f) - t2;
            sq_cl = fmaf(e0, e0, fmaf(e1, e1, e2 * e2));
            ab_cl = (fabsf(e0) + fabsf(e1)) + fabsf(e2);
        }
        double a = block_sum_256((double)sq_raw, s_warp, tid);
        double b = block_sum_256((double)sq_cl, s_warp, tid);
        double c = block_sum_256((double)ab_cl, s_warp, tid);
        if (tid == 0) {
            tile_stats[t].sq_raw = a;
            tile_stats[t].sq_clamp = b;
            tile_stats[t].abs_clamp = c;
        }
    }
}

// ---------------------------------------------------------------------------------------------
// Backward: thread per (tile, Gaussian) pair.  With s = w * (c' . G) and the kappa-scaled
// whitened coordinates (u, v) of the record, the thread accumulates
//   R_ch = sum w G_ch,  Su = sum s u,  Sv = sum s v,  Suu = sum s u^2,  Suv = sum s u v,
//   Svv = sum s v^2
// over the 256 pixels of its tile (pixels outside the frame carry G = 0) and adds them to
// acc[gid][8].  The chain rule to (mu, l, rgb, o) is applied once per Gaussian afterwards
// (gs2d_optim.cu).  u is constant along a tile column, so the inner loop runs down a column.
constexpr int BWD_THREADS = 128;

__global__ void __launch_bounds__(BWD_THREADS)
    k_backward(const int *__restrict__ list, const int *__restrict__ pair_tile, const Rec *__restrict__ rec,
               const float4 *__restrict__ gtile, int TX, float *__restrict__ acc, const DeviceState *__restrict__ st,
               long long cap) {
    const int P = st->n_pairs;
    if ((long long)P > cap) return;
    for (int p = blockIdx.x * BWD_THREADS + threadIdx.x; p < P; p += gridDim.x * BWD_THREADS) {
        const int gid = list[p], t = pair_tile[p];
        const int tx = t % TX, ty = t / TX;
        const float4 lo = reinterpret_cast<const float4 *>(rec)[(size_t)gid * 2];
        const float4 hi = reinterpret_cast<const float4 *>(rec)[(size_t)gid * 2 + 1];
        const float4 *__restrict__ G = gtile + (size_t)t * TILE_PX;
        const float dy0 = ((float)(ty * TILE) + 0.5f) - lo.y;
        const float vy0 = dy0 * hi.x;
        const float dx0 = ((float)(tx * TILE) + 0.5f) - lo.x;
        float Rr = 0.f, Rg = 0.f, Rb = 0.f, Su = 0.f, Sv = 0.f, Suu = 0.f, Suv = 0.f, Svv = 0.f;
#pragma unroll 1
        for (int x = 0; x < TILE; ++x) {
            const float dx = dx0 + (float)x;
            const float u = dx * lo.z;
            const float uu = u * u;
            const float v0 = fmaf(dx, lo.w, vy0);
            float A0 = 0.f, A1 = 0.f, A2 = 0.f;
#pragma unroll
            for (int y = 0; y < TILE; ++y) {
                const float4 gq = G[x * TILE + y];
                const float v = fmaf(hi.x, (float)y, v0);
                const float w = ex2_neg(fmaf(v, v, uu));
                const float qd = fmaf(hi.w, gq.z, fmaf(hi.z, gq.y, hi.y * gq.x));
                const float s = w * qd;
                Rr = fmaf(w, gq.x, Rr);
                Rg = fmaf(w, gq.y, Rg);
                Rb = fmaf(w, gq.z, Rb);
                A0 += s;
                const float sv = s * v;
                A1 += sv;
                A2 = fmaf(sv, v, A2);
            }
            Su = fmaf(u, A0, Su);
            Suu = fmaf(uu, A0, Suu);
            Sv += A1;
            Suv = fmaf(u, A1, Suv);
            Svv += A2;
        }
        float4 *dst = reinterpret_cast<float4 *>(acc + (size_t)gid * 8);
        atomicAdd(dst, make_float4(Rr, Rg, Rb, Su));
        atomicAdd(dst + 1, make_float4(Sv, Suu, Suv, Svv));
    }
}

// dL/dimage [H,W,3] -> tile-major float4 [t][x*16+y], zero outside the frame
__global__ void __launch_bounds__(256) k_repack_grad(const float *__restrict__ dL, int W, int H, int TX,
                                                     float4 *__restrict__ gtile) {
    __shared__ float4 s_g[TILE * 17];
    const int t = blockIdx.x, tid = threadIdx.x;
    const int tx = t % TX, ty = t / TX;
    const int lx = tid & 15, ly = tid >> 4;
    const int gx = tx * TILE + lx, gy = ty * TILE + ly;
    float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
    if (gx < W && gy < H) {
        size_t off = ((size_t)gy * W + gx) * 3;
        v = make_float4(dL[off], dL[off + 1], dL[off + 2], 0.f);
    }
    s_g[lx * 17 + ly] = v;
    __syncthreads();
    gtile[(size_t)t * TILE_PX + tid] = s_g[(tid >> 4) * 17 + (tid & 15)];
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

int ensure_fit_scratch(gs_ctx *c) {
    if (!c->gtile) GS_CUDA_TRY(cudaMalloc(&c->gtile, sizeof(float4) * (size_t)c->T * TILE_PX));
    return GS_OK;
}

int launch_forward(gs_ctx *c, ForwardMode mode, float *image_out, const float *target, int iter, cudaStream_t s) {
    const int W = c->cfg.width, H = c->cfg.height;
    const float g_scale = (float)(2.0 / (3.0 * (double)W * (double)H));
#define GS_FWD(M)                                                                                              \
    k_forward<M><<<c->T, FWD_THREADS, 0, s>>>(c->range, c->list, c->rec, W, H, c->TX, image_out, target,      \
                                              c->gtile, c->tile_stats, g_scale, iter, c->dstate, c->cap_pairs)
    switch (mode) {
        case FWD_IMAGE: GS_FWD(FWD_IMAGE); break;
        case FWD_IMAGE_CLAMP: GS_FWD(FWD_IMAGE_CLAMP); break;
        case FWD_FIT: GS_FWD(FWD_FIT); break;
        case FWD_STATS: GS_FWD(FWD_STATS); break;
    }
#undef GS_FWD
    GS_CUDA_TRY(cudaGetLastError());
    return GS_OK;
}

int launch_backward(gs_ctx *c, cudaStream_t s) {
    long long want = (c->cap_pairs + BWD_THREADS - 1) / BWD_THREADS;
    long long full = (long long)c->sm_count * 16;
    int grid = (int)(want < full ? (want > 0 ? want : 1) : full);
    k_backward<<<grid, BWD_THREADS, 0, s>>>(c->list, c->pair_tile, c->rec, c->gtile, c->TX, c->acc, c->dstate,
                                            c->cap_pairs);
    GS_CUDA_TRY(cudaGetLastError());
    return GS_OK;
}

int launch_repack_grad(gs_ctx *c, const float *dL_dimage, cudaStream_t s) {
    k_repack_grad<<<c->T, 256, 0, s>>>(dL_dimage, c->cfg.width, c->cfg.height, c->TX, c->gtile);
    GS_CUDA_TRY(cudaGetLastError());
    return GS_OK;
}

int launch_reduce_stats(gs_ctx *c, cudaStream_t s) {
    k_reduce_stats<<<1, 1024, 0, s>>>(c->tile_stats, c->T, c->dstate);
    GS_CUDA_TRY(cudaGetLastError());
    return GS_OK;
}

}  // namespace gs2d
