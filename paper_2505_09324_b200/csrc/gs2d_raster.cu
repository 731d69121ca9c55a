// gs2d_raster.cu -- forward rasterizer, loss gradient, backward pass
// (DESIGN.md §5 "forward", "backward").
//
// Forward  : one CTA of 64 threads (2 warps) per 16x16 tile.  A thread owns one column x four
//            rows; the tile's list is walked once by every thread (no list split, hence no
//            cross-thread summation), with the records gathered through shared memory in
//            double-buffered batches of 64 (the next batch is fetched into registers while the
//            current one is consumed).  Per Gaussian and thread the whitened coordinates are
//            set up once (5 FP32 instructions) and each of the 4 pixels costs 2 FFMA +
//            1 MUFU.EX2 + 3 FFMA.  The epilogue fuses the L2 loss and dL/dC (a6).
// Backward : one WARP per work item (tile, chunk of <= 32 list entries).  The warp keeps the
//            tile's dL/dC in registers (lane = column, 16 rows x 3 channels), each half-warp
//            walks one Gaussian at a time over the 16 columns, and the 8 gradient moments are
//            reduced over the 16 lanes with a transposing butterfly (30 instructions) before
//            one 32-byte vector of fp32 atomics per (tile, Gaussian).  No memory access in the
//            inner loop.  Work items are fetched dynamically, so list lengths do not matter.
#include "gs2d_internal.cuh"
#include "gs2d_sort.cuh"

namespace gs2d {

__device__ __forceinline__ float ex2_neg(float p) {  // 2^(-p), MUFU.EX2
    float w;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(w) : "f"(-p));
    return w;
}

constexpr int FWD_THREADS = 64;
constexpr int FWD_BATCH = 64;  // records staged per batch (one per thread)

static_assert(FWD_THREADS == SORT_CTA_THREADS, "the forward CTA sorts its own tile");

// sum over the 64 threads of the CTA: fp32 inside a warp (<= 32 terms), fp64 across warps/tiles
__device__ __forceinline__ double block_sum_64(float v, double *s_warp, int tid) {
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) v += __shfl_xor_sync(0xffffffffu, v, d);
    if ((tid & 31) == 0) s_warp[tid >> 5] = (double)v;
    __syncthreads();
    double r = s_warp[0] + s_warp[1];
    __syncthreads();
    return r;
}

// Tile classes for the forward launch order (longest lists first, so that no long tile starts
// late and the kernel has no tail): class 3 >= 256 entries, 2 >= 96, 1 >= 32, 0 the rest.
// The order a launch walks is the one the PREVIOUS forward launch of the context recorded
// (list lengths drift slowly from one iteration to the next); it only affects scheduling.
__device__ __forceinline__ int tile_class(int n) { return n >= 256 ? 3 : (n >= 96 ? 2 : (n >= 32 ? 1 : 0)); }

template <int MODE>
__global__ void __launch_bounds__(FWD_THREADS)
    k_forward(TileArgs ta, const int *__restrict__ order_cur, int *__restrict__ order_next, int ord_cur, int ord_next,
              const Rec *__restrict__ rec, int W, int H, int TX, float *__restrict__ image_out,
              const float *__restrict__ target, float4 *__restrict__ gtile, TileStats *__restrict__ tile_stats,
              float g_scale, int iter) {
    __shared__ float4 s_rec[2][FWD_BATCH * 2];
    __shared__ __align__(16) float s_io[TILE * TILE * 3];  // one tile of HWC rows
    __shared__ double s_warp[FWD_THREADS / 32];

    DeviceState *st = ta.st;
    const int tid = threadIdx.x;
    const int T = gridDim.x;
    int t;
    {
        int bi = blockIdx.x;
        const int n3 = st->n_class[ord_cur][3], n2 = st->n_class[ord_cur][2], n1 = st->n_class[ord_cur][1];
        int cls = 3;
        if (bi >= n3) {
            bi -= n3;
            cls = 2;
            if (bi >= n2) {
                bi -= n2;
                cls = 1;
                if (bi >= n1) {
                    bi -= n1;
                    cls = 0;
                }
            }
        }
        t = order_cur[(size_t)cls * T + bi];
    }
    const int tx = t % TX, ty = t / TX;

    const int cx = tid & 15, yq = tid >> 4;
    const int gx = tx * TILE + cx, gy0 = ty * TILE + 4 * yq;
    const float px = (float)gx + 0.5f;
    const float py0 = (float)gy0 + 0.5f;

    // target pixels of this thread, fetched before the sort so that their latency is hidden
    float T_[4][3];
    if (MODE == FWD_FIT || MODE == FWD_STATS) {
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const bool valid = gx < W && gy0 + i < H;
            const size_t off = ((size_t)(gy0 + i) * W + gx) * 3;
#pragma unroll
            for (int ch = 0; ch < 3; ++ch) T_[i][ch] = valid ? __ldg(target + off + ch) : 0.0f;
        }
    }

    // consumer stage of the binning.  Renders (image / statistics) sum in the canonical order
    // (ascending id: bit-reproducible images); a fit iteration skips the sort -- its gradients
    // are accumulated with float atomics anyway, and nothing else reads the order.
    int item_base;
    const int n = tile_begin(ta, T, t, tid, MODE != FWD_FIT, item_base);
    // bookkeeping of thread 0, run right before the kernel returns (the atomics' latencies are
    // then off the critical path): the tile's backward work items, and its place in the NEXT
    // launch's order
    auto finish = [&]() {
        if (tid != 0) return;
        if (MODE == FWD_FIT && n > 0) emit_items(ta, t, n, item_base);
        const int cls = tile_class(n);
        const int pos = atomicAdd(&st->n_class[ord_next][cls], 1);
        order_next[(size_t)cls * T + pos] = t;
        if (blockIdx.x == 0) {  // the third order buffer is idle: reset it for the launch after next
            const int o3 = 3 - ord_cur - ord_next;
#pragma unroll
            for (int k = 0; k < 4; ++k) st->n_class[o3][k] = 0;
        }
    };
    if (n < 0) {  // capacity exceeded: leave outputs untouched
        finish();
        return;
    }
    const int *list = ta.bucket + (size_t)t * ta.tile_cap;
    constexpr int start = 0;

    float C[4][3];
#pragma unroll
    for (int i = 0; i < 4; ++i) C[i][0] = C[i][1] = C[i][2] = 0.0f;

    float4 nlo = make_float4(0.f, 0.f, 0.f, 0.f), nhi = nlo;
    if (tid < n) {
        const int gid = list[start + tid];
        nlo = reinterpret_cast<const float4 *>(rec)[(size_t)gid * 2];
        nhi = reinterpret_cast<const float4 *>(rec)[(size_t)gid * 2 + 1];
    }
    int buf = 0;
    for (int b0 = 0; b0 < n; b0 += FWD_BATCH, buf ^= 1) {
        const int bn = min(FWD_BATCH, n - b0);
        s_rec[buf][2 * tid] = nlo;
        s_rec[buf][2 * tid + 1] = nhi;
        __syncthreads();  // batch visible; everybody is done with the batch before the previous one
        if (b0 + FWD_BATCH + tid < n) {
            const int gid = list[start + b0 + FWD_BATCH + tid];
            nlo = reinterpret_cast<const float4 *>(rec)[(size_t)gid * 2];
            nhi = reinterpret_cast<const float4 *>(rec)[(size_t)gid * 2 + 1];
        } else {
            nlo = make_float4(0.f, 0.f, 0.f, 0.f);
            nhi = nlo;
        }
        const float4 *sr = s_rec[buf];
        // entries past the end of the list are null records (zero colour): the walk is unrolled
        // by two without a remainder loop
#pragma unroll 2
        for (int j = 0; j < ((bn + 1) & ~1); ++j) {
            const float4 lo = sr[2 * j], hi = sr[2 * j + 1];
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

    if (MODE == FWD_IMAGE || MODE == FWD_IMAGE_CLAMP) {
        if (MODE == FWD_IMAGE_CLAMP) {
#pragma unroll
            for (int i = 0; i < 4; ++i)
#pragma unroll
                for (int ch = 0; ch < 3; ++ch) C[i][ch] = fminf(fmaxf(C[i][ch], 0.0f), 1.0f);
        }
        const bool vec_rows = (W % 4 == 0) && (tx * TILE + TILE <= W);
        if (vec_rows) {  // stage the tile and write 192-byte row segments as float4
#pragma unroll
            for (int i = 0; i < 4; ++i)
#pragma unroll
                for (int ch = 0; ch < 3; ++ch) s_io[(4 * yq + i) * 48 + cx * 3 + ch] = C[i][ch];
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
        } else {
#pragma unroll
            for (int i = 0; i < 4; ++i)
                if (gx < W && gy0 + i < H) {
                    const size_t off = ((size_t)(gy0 + i) * W + gx) * 3;
                    image_out[off] = C[i][0];
                    image_out[off + 1] = C[i][1];
                    image_out[off + 2] = C[i][2];
                }
        }
        finish();
        return;
    }

    if (MODE == FWD_FIT) {
        // loss on the unclamped sum (DESIGN.md §3 c-4); G = dL/dC = 2 (C - T) / (3 W H), stored
        // tile-major [t][y*16+x] as float4, zero outside the frame
        float sq = 0.0f;
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const bool valid = gx < W && gy0 + i < H;
            const float d0 = valid ? C[i][0] - T_[i][0] : 0.0f, d1 = valid ? C[i][1] - T_[i][1] : 0.0f,
                        d2 = valid ? C[i][2] - T_[i][2] : 0.0f;
            sq += fmaf(d0, d0, fmaf(d1, d1, d2 * d2));
            gtile[(size_t)t * TILE_PX + (4 * yq + i) * TILE + cx] =
                make_float4(d0 * g_scale, d1 * g_scale, d2 * g_scale, 0.0f);
        }
        const double tot = block_sum_64(sq, s_warp, tid);
        if (tid == 0) {
            tile_stats[t].sq_raw = tot;
            if (!isfinite(tot)) {
                atomicOr(&st->flags, FLAG_NONFINITE);
                atomicCAS(&st->first_nonfinite_iter, 0, iter);
            }
        }
        finish();
        return;
    }

    if (MODE == FWD_STATS) {
        float sq_raw = 0.0f, sq_cl = 0.0f, ab_cl = 0.0f;
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            if (gx < W && gy0 + i < H) {
                const float d0 = C[i][0] - T_[i][0], d1 = C[i][1] - T_[i][1], d2 = C[i][2] - T_[i][2];
                sq_raw += fmaf(d0, d0, fmaf(d1, d1, d2 * d2));
                const float e0 = fminf(fmaxf(C[i][0], 0.0f), 1.0f) - T_[i][0],
                            e1 = fminf(fmaxf(C[i][1], 0.0f), 1.0f) - T_[i][1],
                            e2 = fminf(fmaxf(C[i][2], 0.0f), 1.0f) - T_[i][2];
                sq_cl += fmaf(e0, e0, fmaf(e1, e1, e2 * e2));
                ab_cl += (fabsf(e0) + fabsf(e1)) + fabsf(e2);
            }
        }
        const double a = block_sum_64(sq_raw, s_warp, tid);
        const double b = block_sum_64(sq_cl, s_warp, tid);
        const double c = block_sum_64(ab_cl, s_warp, tid);
        if (tid == 0) {
            tile_stats[t].sq_raw = a;
            tile_stats[t].sq_clamp = b;
            tile_stats[t].abs_clamp = c;
        }
        finish();
    }
}

// ---------------------------------------------------------------------------------------------
// Backward.  With s = w * (c' . G) and the kappa-scaled whitened coordinates (u, v) of the
// record, a half-warp accumulates for one Gaussian, lane = tile column,
//   R_ch = sum_y w G_ch,   A1 = sum_y s v,   A2 = sum_y s v^2      (A0 = sum_y s = c' . R)
// and forms its column's share of the 8 moments
//   (R_r, R_g, R_b, Su = u A0, Sv = A1, Suu = u^2 A0, Suv = u A1, Svv = A2),
// which the butterfly sums over the 16 columns.  Pixels outside the frame carry G = 0.  The
// chain rule to (mu, l, rgb, o) is applied once per Gaussian afterwards (gs2d_optim.cu).
constexpr int BWD_WARPS = 4;
constexpr int BWD_THREADS = BWD_WARPS * 32;

__global__ void __launch_bounds__(BWD_THREADS)
    k_backward(const int2 *__restrict__ items, const int *__restrict__ tile_n, const int *__restrict__ bucket,
               int tile_cap, int slot, const Rec *__restrict__ rec, const float4 *__restrict__ gtile, int TX,
               float *__restrict__ acc, DeviceState *st, long long cap) {
    __shared__ float4 s_rec[BWD_WARPS][BWD_CHUNK * 2];
    __shared__ int s_gid[BWD_WARPS][BWD_CHUNK];
    if (st->pair_total[slot] > (unsigned long long)cap || st->tile_ovf[slot] != 0) return;
    const int n_items = st->n_items[slot];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int cx = lane & 15, half = lane >> 4;
    const unsigned full = 0xffffffffu;
    float4 *srec = s_rec[wid];
    int *sgid = s_gid[wid];

    for (;;) {
        int item = 0;
        if (lane == 0) item = (int)atomicAdd(&st->item_cursor[slot], 1u);
        item = __shfl_sync(full, item, 0);
        if (item >= n_items) break;
        const int2 it = items[item];
        const int t = it.x;
        const int tx = t % TX, ty = t / TX;
        const int *list = bucket + (size_t)t * tile_cap + it.y * BWD_CHUNK;
        const int cnt = min(BWD_CHUNK, tile_n[t] - it.y * BWD_CHUNK);

        // records of this chunk -> shared memory (one entry per lane)
        if (lane < cnt) {
            const int gid = list[lane];
            sgid[lane] = gid;
            srec[2 * lane] = reinterpret_cast<const float4 *>(rec)[(size_t)gid * 2];
            srec[2 * lane + 1] = reinterpret_cast<const float4 *>(rec)[(size_t)gid * 2 + 1];
        }
        // dL/dC of this lane's column, all 16 rows
        float G[TILE][3];
        const float4 *__restrict__ gt = gtile + (size_t)t * TILE_PX + cx;
#pragma unroll
        for (int y = 0; y < TILE; ++y) {
            const float4 g = gt[y * TILE];
            G[y][0] = g.x;
            G[y][1] = g.y;
            G[y][2] = g.z;
        }
        __syncwarp();

        const float px = (float)(tx * TILE + cx) + 0.5f;
        const float py0 = (float)(ty * TILE) + 0.5f;
        for (int j0 = 0; j0 < cnt; j0 += 2) {
            const int j = j0 + half;
            const bool live = j < cnt;
            const int jj = live ? j : j0;  // the idle half-warp repeats its neighbour's entry and drops the result
            const float4 lo = srec[2 * jj], hi = srec[2 * jj + 1];
            const float dx = px - lo.x;
            const float u = dx * lo.z;
            const float uu = u * u;
            const float v0 = fmaf(dx, lo.w, (py0 - lo.y) * hi.x);
            float Rr = 0.f, Rg = 0.f, Rb = 0.f, A1 = 0.f, A2 = 0.f;
#pragma unroll
            for (int y = 0; y < TILE; ++y) {
                const float v = fmaf(hi.x, (float)y, v0);
                const float w = ex2_neg(fmaf(v, v, uu));
                const float q = fmaf(hi.w, G[y][2], fmaf(hi.z, G[y][1], hi.y * G[y][0]));
                const float s = w * q;
                Rr = fmaf(w, G[y][0], Rr);
                Rg = fmaf(w, G[y][1], Rg);
                Rb = fmaf(w, G[y][2], Rb);
                const float sv = s * v;
                A1 += sv;
                A2 = fmaf(sv, v, A2);
            }
            const float A0 = fmaf(hi.w, Rb, fmaf(hi.z, Rg, hi.y * Rr));
            // moments of this column: m0..m7 = Rr, Rg, Rb, Su, Sv, Suu, Suv, Svv
            const float m0 = Rr, m1 = Rg, m2 = Rb, m3 = u * A0, m4 = A1, m5 = uu * A0, m6 = u * A1, m7 = A2;
            // transposing butterfly over the 16 lanes of the half-warp
            const bool b8 = lane & 8, b4 = lane & 4, b2 = lane & 2;
            float r0 = (b8 ? m4 : m0) + __shfl_xor_sync(full, b8 ? m0 : m4, 8);
            float r1 = (b8 ? m5 : m1) + __shfl_xor_sync(full, b8 ? m1 : m5, 8);
            float r2 = (b8 ? m6 : m2) + __shfl_xor_sync(full, b8 ? m2 : m6, 8);
            float r3 = (b8 ? m7 : m3) + __shfl_xor_sync(full, b8 ? m3 : m7, 8);
            float q0 = (b4 ? r2 : r0) + __shfl_xor_sync(full, b4 ? r0 : r2, 4);
            float q1 = (b4 ? r3 : r1) + __shfl_xor_sync(full, b4 ? r1 : r3, 4);
            float p0 = (b2 ? q1 : q0) + __shfl_xor_sync(full, b2 ? q0 : q1, 2);
            p0 += __shfl_xor_sync(full, p0, 1);
            // lane (bit0 = 0) holds moment index 4*b8 + 2*b4 + b2
            if (live && !(lane & 1)) {
                const int idx = ((lane >> 3) & 1) * 4 + ((lane >> 2) & 1) * 2 + ((lane >> 1) & 1);
                atomicAdd(acc + (size_t)sgid[jj] * 8 + idx, p0);
            }
        }
        __syncwarp();  // the chunk's records are dead; the next item may overwrite them
    }
}

// dL/dimage [H,W,3] -> tile-major float4 [t][y*16+x], zero outside the frame
__global__ void __launch_bounds__(256) k_repack_grad(const float *__restrict__ dL, int W, int H, int TX,
                                                     float4 *__restrict__ gtile) {
    const int t = blockIdx.x, tid = threadIdx.x;
    const int tx = t % TX, ty = t / TX;
    const int lx = tid & 15, ly = tid >> 4;
    const int gx = tx * TILE + lx, gy = ty * TILE + ly;
    float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
    if (gx < W && gy < H) {
        size_t off = ((size_t)gy * W + gx) * 3;
        v = make_float4(dL[off], dL[off + 1], dL[off + 2], 0.f);
    }
    gtile[(size_t)t * TILE_PX + tid] = v;
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
    const TileArgs ta = tile_args(c, mode == FWD_FIT);
    const int oc = (int)(c->fwd_launches % 3u), on = (int)((c->fwd_launches + 1u) % 3u);
    ++c->fwd_launches;
    const int *order_cur = c->tile_order + (size_t)oc * 4 * c->T;
    int *order_next = c->tile_order + (size_t)on * 4 * c->T;
#define GS_FWD(M)                                                                                                    \
    k_forward<M><<<c->T, FWD_THREADS, 0, s>>>(ta, order_cur, order_next, oc, on, c->rec, W, H, c->TX, image_out, target, \
                                              c->gtile, c->tile_stats, g_scale, iter)
    switch (mode) {
        case FWD_IMAGE: GS_FWD(FWD_IMAGE); break;
        case FWD_IMAGE_CLAMP: GS_FWD(FWD_IMAGE_CLAMP); break;
        case FWD_FIT: GS_FWD(FWD_FIT); break;
        case FWD_STATS: GS_FWD(FWD_STATS); break;
    }
#undef GS_FWD
    c->fresh = false;  // the bins are consumed
    c->sorted = mode != FWD_FIT;
    GS_CUDA_TRY(cudaGetLastError());
    return GS_OK;
}

int launch_backward(gs_ctx *c, cudaStream_t s) {
    if (c->bwd_grid == 0) {
        int per_sm = 0;
        GS_CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_backward, BWD_THREADS, 0));
        c->bwd_grid = c->sm_count * (per_sm > 0 ? per_sm : 1);
    }
    k_backward<<<c->bwd_grid, BWD_THREADS, 0, s>>>(c->items, c->tile_n, c->bucket, c->tile_cap, (int)(c->epoch & 1u),
                                                   c->rec, c->gtile, c->TX, c->acc, c->dstate, c->cap_pairs);
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
