// gs2d_superpixel.cu -- the paper's content-aware I-frame initialiser (the ROI is
// "segmented into N superpixel segments using a K-means clustering-based superpixel algorithm";
// mean, covariance and mean colour of every segment become one Gaussian; SPEC.md:182-200 reads it
// as SLIC).  SURVEY.md §8(f) NEXT #1; the reading is DESIGN.md §3 c-11.
//
// The whole segmentation is integer arithmetic (features in 1/16 units, 64-bit distances, rounded
// integer means), so labels are bit-exact with the oracle and independent of the order in which
// the atomics land:
//   k_sp_bbox     ROI pixel count and bounding box
//   k_sp_cells    which cells of a GX x GY grid over the bounding box hold ROI pixels, and how many (K)
//   k_sp_seed     per cell: the ROI pixel nearest its centre (64-bit atomicMin on distance:index)
//   k_sp_centres  initial centres from the seeds / rounded means from the sums
//   k_sp_assign   per ROI pixel: nearest of the <= 9 clusters around its cell; feature sums
//   k_sp_index    one CTA: non-empty clusters -> output indices (exclusive scan)
//   k_sp_stats    per ROI pixel: output label; exact segment sums (dyadic values in fp64 atomics)
//   k_sp_gauss    per segment: mu, Sigma = covariance + I/12, l = chol(Sigma), mean colour
#include "gs2d_internal.cuh"

namespace gs2d {

struct SpGrid {
    int W, H, x0, y0, bw, bh, GX, GY;  // bounding box origin and size; cell grid
};
// cell of pixel (x, y): integer division of the offset scaled by the grid (DESIGN.md §3 c-11)
__device__ __forceinline__ int sp_cx(const SpGrid &g, int x) { return (int)(((long long)(x - g.x0) * g.GX) / g.bw); }
__device__ __forceinline__ int sp_cy(const SpGrid &g, int y) { return (int)(((long long)(y - g.y0) * g.GY) / g.bh); }

struct SpState {  // device-side results the host reads back
    unsigned long long area;
    int x0, y0, x1, y1;
    int K;      // occupied cells
    int n_out;  // non-empty clusters
};

constexpr unsigned long long SP_NONE = ~0ull;

__device__ __forceinline__ int sp_q255(float v) { return (int)floorf(__fadd_rn(__fmul_rn(255.0f, v), 0.5f)); }

__global__ void __launch_bounds__(256) k_sp_bbox(const unsigned char *__restrict__ mask, int W, int H, SpState *st) {
    int x0 = W, y0 = H, x1 = -1, y1 = -1;
    unsigned cnt = 0;
    for (size_t p = (size_t)blockIdx.x * blockDim.x + threadIdx.x; p < (size_t)W * H; p += (size_t)gridDim.x * blockDim.x)
        if (mask[p]) {
            const int y = (int)(p / W), x = (int)(p - (size_t)y * W);
            ++cnt;
            x0 = min(x0, x);
            x1 = max(x1, x);
            y0 = min(y0, y);
            y1 = max(y1, y);
        }
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) {
        cnt += __shfl_xor_sync(0xffffffffu, cnt, d);
        x0 = min(x0, __shfl_xor_sync(0xffffffffu, x0, d));
        y0 = min(y0, __shfl_xor_sync(0xffffffffu, y0, d));
        x1 = max(x1, __shfl_xor_sync(0xffffffffu, x1, d));
        y1 = max(y1, __shfl_xor_sync(0xffffffffu, y1, d));
    }
    if ((threadIdx.x & 31) == 0 && cnt) {
        atomicAdd(&st->area, (unsigned long long)cnt);
        atomicMin(&st->x0, x0);
        atomicMin(&st->y0, y0);
        atomicMax(&st->x1, x1);
        atomicMax(&st->y1, y1);
    }
}

__global__ void __launch_bounds__(256) k_sp_cells(const unsigned char *__restrict__ mask, SpGrid g,
                                                  unsigned long long *__restrict__ best, SpState *st) {
    const int bw = g.bw, bh = g.bh;
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= (size_t)bw * bh) return;
    const int y = g.y0 + (int)(i / bw), x = g.x0 + (int)(i % bw);
    if (!mask[(size_t)y * g.W + x]) return;
    const int k = sp_cy(g, y) * g.GX + sp_cx(g, x);
    // best[k]: SP_NONE = empty cell; the first ROI pixel that arrives marks it (above any seed key)
    if (best[k] == SP_NONE && atomicExch(&best[k], SP_NONE - 1) == SP_NONE) atomicAdd(&st->K, 1);
}

__global__ void __launch_bounds__(256) k_sp_seed(const unsigned char *__restrict__ mask, SpGrid g,
                                                 unsigned long long *__restrict__ best) {
    const int bw = g.bw, bh = g.bh;
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= (size_t)bw * bh) return;
    const int y = g.y0 + (int)(i / bw), x = g.x0 + (int)(i % bw);
    if (!mask[(size_t)y * g.W + x]) return;
    const int cx = sp_cx(g, x), cy = sp_cy(g, y);
    // first and last pixel offset of the cell along each axis; e = twice the offset from the cell centre
    const long long lox = ((long long)cx * bw + g.GX - 1) / g.GX, hix = ((long long)(cx + 1) * bw + g.GX - 1) / g.GX - 1;
    const long long loy = ((long long)cy * bh + g.GY - 1) / g.GY, hiy = ((long long)(cy + 1) * bh + g.GY - 1) / g.GY - 1;
    const long long ex = 2 * (x - g.x0) - lox - hix, ey = 2 * (y - g.y0) - loy - hiy;
    const unsigned long long key = ((unsigned long long)(ex * ex + ey * ey) << 32) | (unsigned)((size_t)y * g.W + x);
    atomicMin(&best[cy * g.GX + cx], key);  // nearest the cell centre, ties to the smallest pixel index
}

// init != 0: centres from the seed pixels; else: rounded means of the sums (clusters without
// pixels keep their centre), and the sums are cleared for the next pass
__global__ void __launch_bounds__(256) k_sp_centres(const float *__restrict__ frame, SpGrid g, int C, int init,
                                                    const unsigned long long *__restrict__ best,
                                                    int *__restrict__ cen, unsigned long long *__restrict__ sum) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= C) return;
    if (init) {
        if (best[k] == SP_NONE) return;
        const size_t p = (size_t)(best[k] & 0xffffffffull);
        const int y = (int)(p / g.W), x = (int)(p - (size_t)y * g.W);
        cen[5 * k] = 16 * x + 8;
        cen[5 * k + 1] = 16 * y + 8;
#pragma unroll
        for (int c = 0; c < 3; ++c) cen[5 * k + 2 + c] = 16 * sp_q255(frame[3 * p + c]);
    } else {
        const unsigned long long n = sum[6 * k + 5];
        if (n > 0)
#pragma unroll
            for (int j = 0; j < 5; ++j) cen[5 * k + j] = (int)((sum[6 * k + j] + n / 2) / n);
    }
#pragma unroll
    for (int j = 0; j < 6; ++j) sum[6 * k + j] = 0ull;
}

__global__ void __launch_bounds__(256) k_sp_assign(const float *__restrict__ frame, const unsigned char *__restrict__ mask,
                                                   SpGrid g, long long S2, long long M2,
                                                   const unsigned long long *__restrict__ best,
                                                   const int *__restrict__ cen, int *__restrict__ label,
                                                   unsigned long long *__restrict__ sum) {
    const int bw = g.bw, bh = g.bh;
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    const bool in_box = i < (size_t)bw * bh;
    const int y = g.y0 + (int)((in_box ? i : 0) / bw), x = g.x0 + (int)((in_box ? i : 0) % bw);
    const size_t p = (size_t)y * g.W + x;
    const bool roi = in_box && mask[p];
    int f[5] = {16 * x + 8, 16 * y + 8, 0, 0, 0};
    if (roi)
#pragma unroll
        for (int c = 0; c < 3; ++c) f[2 + c] = 16 * sp_q255(frame[3 * p + c]);
    const int cx = sp_cx(g, x), cy = sp_cy(g, y);
    long long bd = 0;
    int bk = -1;
    if (roi)
    for (int dy = -1; dy <= 1; ++dy)
        for (int dx = -1; dx <= 1; ++dx) {  // ascending k: a tie keeps the smaller index
            const int ux = cx + dx, uy = cy + dy;
            if (ux < 0 || uy < 0 || ux >= g.GX || uy >= g.GY) continue;
            const int k = uy * g.GX + ux;
            if (best[k] == SP_NONE) continue;
            const long long ddx = f[0] - cen[5 * k], ddy = f[1] - cen[5 * k + 1], dr = f[2] - cen[5 * k + 2],
                            dg = f[3] - cen[5 * k + 3], db = f[4] - cen[5 * k + 4];
            const long long D = S2 * (dr * dr + dg * dg + db * db) + M2 * (ddx * ddx + ddy * ddy);
            if (bk < 0 || D < bd) {
                bd = D;
                bk = k;
            }
        }
    if (roi) label[p] = bk;
    // feature sums, aggregated over the lanes of the warp that chose the same cluster (neighbouring
    // pixels mostly do): one leader adds the group's 32-bit partial sums (features < 2^17, 32 lanes)
    const unsigned peers = __match_any_sync(0xffffffffu, bk);
    const int lane = threadIdx.x & 31;
    const bool leader = (__ffs(peers) - 1) == lane;
#pragma unroll
    for (int j = 0; j < 5; ++j) {
        const unsigned v = __reduce_add_sync(peers, (unsigned)f[j]);
        if (leader && bk >= 0) atomicAdd(&sum[6 * bk + j], (unsigned long long)v);
    }
    if (leader && bk >= 0) atomicAdd(&sum[6 * bk + 5], (unsigned long long)__popc(peers));
}

// out_index[k] = rank of cluster k among the non-empty ones (or -1); one CTA
__global__ void __launch_bounds__(1024) k_sp_index(int C, const unsigned long long *__restrict__ sum,
                                                   int *__restrict__ out_index, SpState *st) {
    __shared__ int s_w[32];
    __shared__ int s_carry;
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    if (tid == 0) s_carry = 0;
    __syncthreads();
    for (int b0 = 0; b0 < C; b0 += 1024) {
        const int k = b0 + tid;
        const int v = (k < C && sum[6 * k + 5] > 0) ? 1 : 0;
        int x = v;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const int o = __shfl_up_sync(0xffffffffu, x, d);
            if (lane >= d) x += o;
        }
        if (lane == 31) s_w[wid] = x;
        __syncthreads();
        if (wid == 0) {
            int w = s_w[lane], yv = w;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                const int o = __shfl_up_sync(0xffffffffu, yv, d);
                if (lane >= d) yv += o;
            }
            s_w[lane] = yv - w;
        }
        __syncthreads();
        const int carry = s_carry;
        if (k < C) out_index[k] = v ? carry + s_w[wid] + x - 1 : -1;
        __syncthreads();
        if (tid == 1023) s_carry = carry + s_w[wid] + x;
        __syncthreads();
    }
    if (tid == 0) st->n_out = s_carry;
}

// Segment sums relative to the cluster's centre (1/16 units): every addend is a small dyadic
// number, so the fp64 atomics are exact and order-independent.
//   stats[g][0..8] = sum dx, sum dy, sum dx^2, sum dx dy, sum dy^2, sum fix16(r, g, b), count
__global__ void __launch_bounds__(256) k_sp_stats(const float *__restrict__ frame, const unsigned char *__restrict__ mask,
                                                  int W, int H, const int *__restrict__ label,
                                                  const int *__restrict__ out_index, const int *__restrict__ cen,
                                                  double *__restrict__ stats, int *__restrict__ labels_out) {
    const size_t p = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= (size_t)W * H) return;
    if (!mask[p]) {
        if (labels_out) labels_out[p] = -1;
        return;
    }
    const int k = label[p], g = out_index[k];
    if (labels_out) labels_out[p] = g;
    const int y = (int)(p / W), x = (int)(p - (size_t)y * W);
    const double dx = (double)(16 * x + 8 - cen[5 * k]) * 0.0625, dy = (double)(16 * y + 8 - cen[5 * k + 1]) * 0.0625;
    double *s = stats + 9 * (size_t)g;
    atomicAdd(s + 0, dx);
    atomicAdd(s + 1, dy);
    atomicAdd(s + 2, dx * dx);
    atomicAdd(s + 3, dx * dy);
    atomicAdd(s + 4, dy * dy);
#pragma unroll
    for (int c = 0; c < 3; ++c) atomicAdd(s + 5 + c, floor(65536.0 * (double)frame[3 * p + c] + 0.5));
    atomicAdd(s + 8, 1.0);
}

__global__ void __launch_bounds__(256) k_sp_gauss(int C, const int *__restrict__ out_index, const int *__restrict__ cen,
                                                  const double *__restrict__ stats, float *__restrict__ mu,
                                                  float *__restrict__ chol, float *__restrict__ rgb,
                                                  float *__restrict__ opacity) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= C) return;
    const int g = out_index[k];
    if (g < 0) return;
    const double *s = stats + 9 * (size_t)g;
    const double n = s[8];
    const double ex = s[0] / n, ey = s[1] / n;  // mean offset from the centre
    const double sxx = s[2] / n - ex * ex + 1.0 / 12.0, sxy = s[3] / n - ex * ey, syy = s[4] / n - ey * ey + 1.0 / 12.0;
    const double l1 = sqrt(sxx), l2 = sxy / l1, l3 = sqrt(syy - l2 * l2);
    mu[2 * g] = (float)((double)cen[5 * k] * 0.0625 + ex);
    mu[2 * g + 1] = (float)((double)cen[5 * k + 1] * 0.0625 + ey);
    chol[3 * g] = (float)l1;
    chol[3 * g + 1] = (float)l2;
    chol[3 * g + 2] = (float)l3;
#pragma unroll
    for (int c = 0; c < 3; ++c) rgb[3 * g + c] = (float)(s[5 + c] / (65536.0 * n));
    opacity[g] = 1.0f;
}

// Host side.
int run_init_superpixel(gs_ctx *c, const float *frame, const unsigned char *mask, int n_segments, int compactness,
                        int kmeans_iters, const gs_params &out, int *labels_out, int *n_out_host, cudaStream_t s) {
    const int W = c->cfg.width, H = c->cfg.height;
    const size_t npx = (size_t)W * H;
    // scratch is owned by the context and grows on demand (cudaMalloc / cudaFree per call cost more than
    // the kernels)
    auto grow = [&](int slot, size_t bytes) -> void * {
        if (c->sp_bytes[slot] < bytes) {
            if (c->sp_buf[slot]) cudaFree(c->sp_buf[slot]);
            c->sp_buf[slot] = nullptr;
            c->sp_bytes[slot] = 0;
            if (cudaMalloc(&c->sp_buf[slot], bytes) != cudaSuccess) return nullptr;
            c->sp_bytes[slot] = bytes;
        }
        return c->sp_buf[slot];
    };
    SpState *dst = (SpState *)grow(0, sizeof(SpState));
    if (!dst) return GS_ERR_CUDA;
    SpState h;
    h.area = 0ull;
    h.x0 = W;
    h.y0 = H;
    h.x1 = -1;
    h.y1 = -1;
    h.K = 0;
    h.n_out = 0;
    int rc = GS_OK;
    unsigned long long *best = nullptr, *sum = nullptr;
    int *cen = nullptr, *label = nullptr, *out_index = nullptr;
    double *stats = nullptr;
    auto cleanup = [&]() {};
#define SP_TRY(expr)                                  \
    do {                                              \
        cudaError_t _e = (expr);                      \
        if (_e != cudaSuccess) {                      \
            set_cuda_error(_e, #expr);                \
            cleanup();                                \
            return GS_ERR_CUDA;                       \
        }                                             \
    } while (0)
    SP_TRY(cudaMemcpyAsync(dst, &h, sizeof h, cudaMemcpyHostToDevice, s));
    k_sp_bbox<<<c->sm_count * 8, 256, 0, s>>>(mask, W, H, dst);
    SP_TRY(cudaMemcpyAsync(&h, dst, sizeof h, cudaMemcpyDeviceToHost, s));
    SP_TRY(cudaStreamSynchronize(s));
    if (h.area == 0ull) {
        cleanup();
        return GS_ERR_EMPTY_MASK;
    }
    SpGrid g;
    g.W = W;
    g.H = H;
    g.x0 = h.x0;
    g.y0 = h.y0;
    const int bw = h.x1 - h.x0 + 1, bh = h.y1 - h.y0 + 1;
    g.bw = bw;
    g.bh = bh;
    const size_t nbox = (size_t)bw * bh;
    const int box_blocks = ceil_div((long long)nbox, 256);
    best = (unsigned long long *)grow(1, sizeof(unsigned long long) * nbox);  // GX GY <= bw bh for every grid tried
    if (!best) return GS_ERR_CUDA;
    auto grid_of = [&](int gx) {
        g.GX = gx;
        const long long gy = ((long long)2 * gx * bh + bw) / (2LL * bw);
        g.GY = gy < 1 ? 1 : (int)gy;
    };
    auto occupied = [&](int gx, int &K) -> int {  // marks best[] for the grid and counts its occupied cells
        grid_of(gx);
        GS_CUDA_TRY(cudaMemsetAsync(best, 0xff, sizeof(unsigned long long) * (size_t)g.GX * g.GY, s));
        GS_CUDA_TRY(cudaMemsetAsync(&dst->K, 0, sizeof(int), s));
        k_sp_cells<<<box_blocks, 256, 0, s>>>(mask, g, best, dst);
        GS_CUDA_TRY(cudaMemcpyAsync(&K, &dst->K, sizeof(int), cudaMemcpyDeviceToHost, s));
        GS_CUDA_TRY(cudaStreamSynchronize(s));
        return GS_OK;
    };
    // bisection for the largest GX whose grid has at most n_segments occupied cells (lo = 0: not even GX = 1)
    int lo = 0, hi = bw, K = 0;
    while (lo < hi) {
        const int mid = (lo + hi + 1) / 2;
        if (occupied(mid, K)) {
            cleanup();
            return GS_ERR_CUDA;
        }
        if (K <= n_segments) lo = mid;
        else hi = mid - 1;
    }
    if (lo >= 1) {
        if (occupied(lo, K)) {
            cleanup();
            return GS_ERR_CUDA;
        }
    } else {  // the ROI is so elongated that even one column of cells exceeds n_segments: one cell
        g.GX = g.GY = 1;
        SP_TRY(cudaMemsetAsync(best, 0xff, sizeof(unsigned long long), s));
        SP_TRY(cudaMemsetAsync(&dst->K, 0, sizeof(int), s));
        k_sp_cells<<<box_blocks, 256, 0, s>>>(mask, g, best, dst);
    }
    const int C = g.GX * g.GY;
    sum = (unsigned long long *)grow(2, sizeof(unsigned long long) * 6 * (size_t)C);
    cen = (int *)grow(3, sizeof(int) * 5 * (size_t)C);
    label = (int *)grow(4, sizeof(int) * npx);
    out_index = (int *)grow(5, sizeof(int) * (size_t)C);
    stats = (double *)grow(6, sizeof(double) * 9 * (size_t)n_segments);
    if (!sum || !cen || !label || !out_index || !stats) return GS_ERR_CUDA;
    k_sp_seed<<<box_blocks, 256, 0, s>>>(mask, g, best);
    k_sp_centres<<<ceil_div(C, 256), 256, 0, s>>>(frame, g, C, 1, best, cen, sum);
    long long S2 = ((long long)bw * bh) / ((long long)g.GX * g.GY);  // the cell area: SLIC's grid step squared
    if (S2 < 1) S2 = 1;
    const long long M2 = (long long)compactness * compactness;
    for (int it = 0; it <= kmeans_iters; ++it) {  // the last pass only assigns: labels of the final centres
        k_sp_assign<<<box_blocks, 256, 0, s>>>(frame, mask, g, S2, M2, best, cen, label, sum);
        if (it < kmeans_iters) k_sp_centres<<<ceil_div(C, 256), 256, 0, s>>>(frame, g, C, 0, best, cen, sum);
    }
    k_sp_index<<<1, 1024, 0, s>>>(C, sum, out_index, dst);
    SP_TRY(cudaMemsetAsync(stats, 0, sizeof(double) * 9 * (size_t)n_segments, s));
    k_sp_stats<<<ceil_div((long long)npx, 256), 256, 0, s>>>(frame, mask, W, H, label, out_index, cen, stats, labels_out);
    k_sp_gauss<<<ceil_div(C, 256), 256, 0, s>>>(C, out_index, cen, stats, out.mu, out.chol, out.rgb, out.opacity);
    SP_TRY(cudaGetLastError());
    SP_TRY(cudaMemcpyAsync(&h.n_out, &dst->n_out, sizeof(int), cudaMemcpyDeviceToHost, s));
    SP_TRY(cudaStreamSynchronize(s));
#undef SP_TRY
    if (n_out_host) *n_out_host = h.n_out;
    cleanup();
    return rc;
}

}  // namespace gs2d
