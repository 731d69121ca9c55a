// gs2d_init.cu -- content-aware ROI initialiser (BASELINE.json
// configs[1], [2]; DESIGN.md §3 c-8).  It stands in for the paper's matting + superpixel
// initialiser: Gaussians go where the frame has detail.
//
//   k_roi_grey      q_ch = floor(255 x_ch + 0.5) (two single-rounded binary32 ops), grey = sum
//   k_roi_blocksum  integer Sobel weights per pixel, per-chunk sums (inside, outside)
//   k_roi_scanblk   one CTA: exclusive scan of the chunk sums, totals
//   k_roi_prefix    inclusive 64-bit prefix sums c_in[p], c_out[p] in row-major pixel order
//   k_roi_sample    per Gaussian: counter-based draw, upper-bound search, parameters
#include "gs2d_internal.cuh"

namespace gs2d {

constexpr int ROI_CHUNK = 2048;  // pixels per CTA in the two weight passes
constexpr int ROI_THREADS = 256;
constexpr int ROI_IPT = ROI_CHUNK / ROI_THREADS;

__global__ void __launch_bounds__(256) k_roi_grey(const float *__restrict__ frame, int npx, int *__restrict__ grey) {
    int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= npx) return;
    int s = 0;
#pragma unroll
    for (int ch = 0; ch < 3; ++ch) {
        float t = __fmul_rn(255.0f, frame[3 * (size_t)p + ch]);
        float r = __fadd_rn(t, 0.5f);
        s += (int)floorf(r);
    }
    grey[p] = s;
}

__device__ __forceinline__ int clampi(int v, int lo, int hi) { return v < lo ? lo : (v > hi ? hi : v); }

// weight = isqrt(gx^2 + gy^2) + 1 inside the ROI (3x3 Sobel on grey, clamp-to-edge), 0 outside;
// outside weight = 1 per non-ROI pixel.
__device__ __forceinline__ void roi_weight(const int *__restrict__ grey, const unsigned char *__restrict__ mask, int W,
                                           int H, int p, unsigned &w_in, unsigned &w_out) {
    if (!mask[p]) {
        w_in = 0;
        w_out = 1;
        return;
    }
    int y = p / W, x = p - y * W;
    int xm = clampi(x - 1, 0, W - 1), xp = clampi(x + 1, 0, W - 1);
    int ym = clampi(y - 1, 0, H - 1), yp = clampi(y + 1, 0, H - 1);
#define GR(yy, xx) grey[(size_t)(yy) * W + (xx)]
    int gx = (GR(ym, xp) + 2 * GR(y, xp) + GR(yp, xp)) - (GR(ym, xm) + 2 * GR(y, xm) + GR(yp, xm));
    int gy = (GR(yp, xm) + 2 * GR(yp, x) + GR(yp, xp)) - (GR(ym, xm) + 2 * GR(ym, x) + GR(ym, xp));
#undef GR
    long long m2 = (long long)gx * gx + (long long)gy * gy;
    long long r = (long long)sqrt((double)m2);
    while (r * r > m2) --r;
    while ((r + 1) * (r + 1) <= m2) ++r;
    w_in = (unsigned)r + 1u;
    w_out = 0;
}

__device__ __forceinline__ unsigned long long block_excl_scan_u64(unsigned long long v, unsigned long long *s_warp,
                                                                  unsigned long long &total) {
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    unsigned long long incl = v;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        unsigned long long o = __shfl_up_sync(0xffffffffu, incl, d);
        if (lane >= d) incl += o;
    }
    if (lane == 31) s_warp[wid] = incl;
    __syncthreads();
    if (wid == 0) {
        unsigned long long w = lane < (int)(blockDim.x >> 5) ? s_warp[lane] : 0ull, s = w;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            unsigned long long o = __shfl_up_sync(0xffffffffu, s, d);
            if (lane >= d) s += o;
        }
        s_warp[lane] = s - w;
        if (lane == 31) s_warp[32] = s;
    }
    __syncthreads();
    unsigned long long ex = s_warp[wid] + incl - v;
    total = s_warp[32];
    __syncthreads();
    return ex;
}

__global__ void __launch_bounds__(ROI_THREADS) k_roi_blocksum(const int *__restrict__ grey,
                                                              const unsigned char *__restrict__ mask, int W, int H,
                                                              unsigned long long *__restrict__ blk) {
    __shared__ unsigned long long s_warp[33];
    const int npx = W * H;
    int base = blockIdx.x * ROI_CHUNK + threadIdx.x * ROI_IPT;
    unsigned long long a = 0, b = 0;
    for (int i = 0; i < ROI_IPT; ++i) {
        int p = base + i;
        if (p < npx) {
            unsigned wi, wo;
            roi_weight(grey, mask, W, H, p, wi, wo);
            a += wi;
            b += wo;
        }
    }
    unsigned long long ta, tb;
    block_excl_scan_u64(a, s_warp, ta);
    block_excl_scan_u64(b, s_warp, tb);
    if (threadIdx.x == 0) {
        blk[2 * blockIdx.x] = ta;
        blk[2 * blockIdx.x + 1] = tb;
    }
}

__global__ void __launch_bounds__(1024) k_roi_scanblk(unsigned long long *__restrict__ blk, int nblk, DeviceState *st) {
    __shared__ unsigned long long s_warp[33];
    int ipt = (nblk + 1023) / 1024;
    int b = threadIdx.x * ipt, e = min(b + ipt, nblk);
    for (int k = 0; k < 2; ++k) {
        unsigned long long local = 0;
        for (int i = b; i < e; ++i) local += blk[2 * i + k];
        unsigned long long total;
        unsigned long long run = block_excl_scan_u64(local, s_warp, total);
        for (int i = b; i < e; ++i) {
            unsigned long long c = blk[2 * i + k];
            blk[2 * i + k] = run;
            run += c;
        }
        if (threadIdx.x == 0) {
            if (k == 0) st->total_in = total;
            else st->total_out = total;
        }
    }
}

__global__ void __launch_bounds__(ROI_THREADS) k_roi_prefix(const int *__restrict__ grey,
                                                            const unsigned char *__restrict__ mask, int W, int H,
                                                            const unsigned long long *__restrict__ blk,
                                                            unsigned long long *__restrict__ cin,
                                                            unsigned long long *__restrict__ cout) {
    __shared__ unsigned long long s_warp[33];
    const int npx = W * H;
    int base = blockIdx.x * ROI_CHUNK + threadIdx.x * ROI_IPT;
    unsigned wi[ROI_IPT], wo[ROI_IPT];
    unsigned long long a = 0, b = 0;
#pragma unroll
    for (int i = 0; i < ROI_IPT; ++i) {
        int p = base + i;
        wi[i] = wo[i] = 0;
        if (p < npx) roi_weight(grey, mask, W, H, p, wi[i], wo[i]);
        a += wi[i];
        b += wo[i];
    }
    unsigned long long ta, tb;
    unsigned long long ra = block_excl_scan_u64(a, s_warp, ta) + blk[2 * blockIdx.x];
    unsigned long long rb = block_excl_scan_u64(b, s_warp, tb) + blk[2 * blockIdx.x + 1];
#pragma unroll
    for (int i = 0; i < ROI_IPT; ++i) {
        int p = base + i;
        ra += wi[i];
        rb += wo[i];
        if (p < npx) {
            cin[p] = ra;  // inclusive
            cout[p] = rb;
        }
    }
}

// Counter-based generator: SplitMix64 finaliser of seed + (8 i + k + 1) * golden (gs2d.h).
__device__ __forceinline__ unsigned long long rnd64(unsigned long long seed, unsigned long long i,
                                                    unsigned long long k) {
    unsigned long long z = seed + (8ull * i + k + 1ull) * 0x9E3779B97F4A7C15ull;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
    return z ^ (z >> 31);
}

__global__ void __launch_bounds__(256)
    k_roi_sample(int N, int N_in, unsigned long long seed, const float *__restrict__ frame, int W, int npx,
                 const unsigned long long *__restrict__ cin, const unsigned long long *__restrict__ cout,
                 unsigned long long total_in, unsigned long long total_out, float s_min, float s_max,
                 float *__restrict__ mu, float *__restrict__ chol, float *__restrict__ rgb,
                 float *__restrict__ opacity) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const bool inside = i < N_in;
    const unsigned long long *__restrict__ c = inside ? cin : cout;
    const unsigned long long total = inside ? total_in : total_out;
    const unsigned long long target = rnd64(seed, (unsigned long long)i, 0) % total;
    int lo = 0, hi = npx - 1;  // first p with c[p] > target
    while (lo < hi) {
        int mid = lo + (hi - lo) / 2;
        if (c[mid] > target) hi = mid;
        else lo = mid + 1;
    }
    const int p = lo;
    const int y = p / W, x = p - y * W;
    // 24 random bits -> [0,1) exactly representable; jitter in [-0.5, 0.5)
    const float jx = __fsub_rn(__fmul_rn((float)(rnd64(seed, i, 1) >> 40), 5.9604644775390625e-8f), 0.5f);
    const float jy = __fsub_rn(__fmul_rn((float)(rnd64(seed, i, 2) >> 40), 5.9604644775390625e-8f), 0.5f);
    mu[2 * i] = __fadd_rn((float)x + 0.5f, jx);
    mu[2 * i + 1] = __fadd_rn((float)y + 0.5f, jy);
    rgb[3 * i] = frame[3 * (size_t)p];
    rgb[3 * i + 1] = frame[3 * (size_t)p + 1];
    rgb[3 * i + 2] = frame[3 * (size_t)p + 2];
    opacity[i] = 1.0f;
    const float u1 = (float)(rnd64(seed, i, 3) >> 40) * 5.9604644775390625e-8f;
    const float u2 = (float)(rnd64(seed, i, 4) >> 40) * 5.9604644775390625e-8f;
    const float u3 = (float)(rnd64(seed, i, 5) >> 40) * 5.9604644775390625e-8f;
    const float ls = logf(s_max / s_min);
    const float s1 = s_min * expf(u1 * ls), s2 = s_min * expf(u2 * ls);
    float st, ct;
    sincosf(3.14159265358979323846f * u3, &st, &ct);
    // Sigma = R diag(s1^2, s2^2) R^T and its Cholesky factor; det Sigma = (s1 s2)^2 = (l1 l3)^2
    const float S11 = ct * ct * s1 * s1 + st * st * s2 * s2;
    const float S12 = ct * st * ((s1 - s2) * (s1 + s2));
    const float l1 = sqrtf(S11);
    chol[3 * i] = l1;
    chol[3 * i + 1] = S12 / l1;
    chol[3 * i + 2] = s1 * s2 / l1;
}

int run_init_roi(gs_ctx *c, const float *frame, const unsigned char *mask, int n, unsigned long long seed, float s_min,
                 float s_max, const gs_params &out, cudaStream_t s) {
    const int W = c->cfg.width, H = c->cfg.height, npx = W * H;
    const int nblk = ceil_div(npx, ROI_CHUNK);
    if (!c->roi_grey) {
        GS_CUDA_TRY(cudaMalloc(&c->roi_grey, sizeof(int) * (size_t)npx));
        GS_CUDA_TRY(cudaMalloc(&c->roi_cin, sizeof(unsigned long long) * (size_t)npx));
        GS_CUDA_TRY(cudaMalloc(&c->roi_cout, sizeof(unsigned long long) * (size_t)npx));
        GS_CUDA_TRY(cudaMalloc(&c->roi_blk, sizeof(unsigned long long) * 2 * (size_t)nblk));
    }
    k_roi_grey<<<ceil_div(npx, 256), 256, 0, s>>>(frame, npx, c->roi_grey);
    k_roi_blocksum<<<nblk, ROI_THREADS, 0, s>>>(c->roi_grey, mask, W, H, c->roi_blk);
    k_roi_scanblk<<<1, 1024, 0, s>>>(c->roi_blk, nblk, c->dstate);
    k_roi_prefix<<<nblk, ROI_THREADS, 0, s>>>(c->roi_grey, mask, W, H, c->roi_blk, c->roi_cin, c->roi_cout);
    GS_CUDA_TRY(cudaGetLastError());
    // the totals decide the split and the empty-ROI error: one small read-back
    GS_CUDA_TRY(cudaMemcpyAsync(c->hstate, c->dstate, sizeof(DeviceState), cudaMemcpyDeviceToHost, s));
    GS_CUDA_TRY(cudaStreamSynchronize(s));
    const unsigned long long tin = c->hstate->total_in, tout = c->hstate->total_out;
    if (tin == 0) return GS_ERR_EMPTY_MASK;
    int N_in = (int)((7LL * n) / 10);
    if (tout == 0) N_in = n;  // no outside pixels: all inside
    k_roi_sample<<<ceil_div(n, 256), 256, 0, s>>>(n, N_in, seed, frame, W, npx, c->roi_cin, c->roi_cout, tin, tout,
                                                  s_min, s_max, out.mu, out.chol, out.rgb, out.opacity);
    GS_CUDA_TRY(cudaGetLastError());
    GS_CUDA_TRY(cudaStreamSynchronize(s));
    return GS_OK;
}

}  // namespace gs2d
