// gs2d_select.cu -- P-frame selection (
// BASELINE.json configs[3]; DESIGN.md §3 c-9).  Runs after a FWD_STATS forward pass:
//   r_t = abs_clamp_t / (3 * valid pixels of tile t);  tile changed iff r_t > tau (strict)
//   active[n] = 1 iff n is listed in at least one changed tile.
#include "gs2d_internal.cuh"
#include "gs2d_sort.cuh"

namespace gs2d {

__global__ void __launch_bounds__(256) k_flag_tiles(const TileStats *__restrict__ ts, int T, int TX, int W, int H,
                                                    double tau, unsigned char *__restrict__ tile_flag) {
    int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= T) return;
    const int nv = ts[t].n_valid;  // the tile's pixels inside the frame (and the ROI): a tile without any never changes
    double r = nv > 0 ? ts[t].abs_clamp / (double)(3 * nv) : 0.0;
    tile_flag[t] = r > tau ? 1 : 0;
}

__global__ void __launch_bounds__(256) k_tile_resid(const TileStats *__restrict__ ts, int T, int TX, int W, int H,
                                                    double *__restrict__ resid) {
    int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= T) return;
    const int nv = ts[t].n_valid;
    resid[t] = nv > 0 ? ts[t].abs_clamp / (double)(3 * nv) : 0.0;
}

// one warp per tile: the lanes stride over the list of a changed tile
__global__ void __launch_bounds__(256) k_mark_active(int T, const int *__restrict__ tile_n, TileArgs a,
                                                     const unsigned char *__restrict__ tile_flag,
                                                     unsigned char *__restrict__ active) {
    const int t = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (t >= T || !tile_flag[t]) return;
    const int n = tile_n[t];  // 0 when the binning exceeded a capacity
    const int *list = a.bucket + (size_t)t * a.tile_cap;
    for (int p = threadIdx.x & 31; p < min(n, a.tile_cap); p += 32) active[list[p]] = 1;  // every writer stores the same value
    if (n > a.tile_cap) {  // the tile's entries beyond its bucket
        const int S = spill_size(a);
        for (int e = threadIdx.x & 31; e < S; e += 32) {
            const int2 v = a.spill[e];
            if (v.x == t) active[v.y] = 1;
        }
    }
}

__global__ void __launch_bounds__(1024) k_count_active(const unsigned char *__restrict__ active, int N,
                                                       DeviceState *st) {
    __shared__ int s_c[1024];
    int tid = threadIdx.x, c = 0;
    for (int i = tid; i < N; i += 1024) c += active[i] ? 1 : 0;
    s_c[tid] = c;
    __syncthreads();
    for (int d = 512; d > 0; d >>= 1) {
        if (tid < d) s_c[tid] += s_c[tid + d];
        __syncthreads();
    }
    if (tid == 0) st->n_active = s_c[0];
}

int launch_select(gs_ctx *c, float tau, unsigned char *active_out, int n, cudaStream_t s) {
    GS_CUDA_TRY(cudaMemsetAsync(active_out, 0, (size_t)n, s));
    k_flag_tiles<<<ceil_div(c->T, 256), 256, 0, s>>>(c->tile_stats, c->T, c->TX, c->cfg.width, c->cfg.height,
                                                     (double)tau, c->tile_flag);
    k_mark_active<<<ceil_div(c->T, 8), 256, 0, s>>>(c->T, c->tile_n, tile_args(c), c->tile_flag, active_out);
    k_count_active<<<1, 1024, 0, s>>>(active_out, n, c->dstate);
    GS_CUDA_TRY(cudaGetLastError());
    return GS_OK;
}

// ---- pixel-granular selection (DESIGN.md §3 c-13) ----------
// changed[p] = max over channels |frame - clamped render| > tau (strict)
__global__ void __launch_bounds__(256) k_change_map(const float *__restrict__ frame, const float *__restrict__ render,
                                                    size_t npix, float tau, unsigned char *__restrict__ changed,
                                                    const unsigned char *__restrict__ roi) {
    const size_t p = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= npix) return;
    if (roi && roi[p] == 0) {  // c-16: only ROI pixels can change
        changed[p] = 0;
        return;
    }
    float r = 0.0f;
#pragma unroll
    for (int ch = 0; ch < 3; ++ch) r = fmaxf(r, fabsf(frame[3 * p + ch] - render[3 * p + ch]));
    changed[p] = r > tau ? 1 : 0;
}

// dilation by one pixel (3x3, inside the frame)
__global__ void __launch_bounds__(256) k_dilate(const unsigned char *__restrict__ in, int W, int H,
                                                unsigned char *__restrict__ out) {
    const size_t p = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= (size_t)W * H) return;
    const int y = (int)(p / W), x = (int)(p - (size_t)y * W);
    unsigned char f = 0;
    for (int dy = -1; dy <= 1; ++dy)
        for (int dx = -1; dx <= 1; ++dx) {
            const int yy = y + dy, xx = x + dx;
            if (yy >= 0 && yy < H && xx >= 0 && xx < W) f |= in[(size_t)yy * W + xx];
        }
    out[p] = f ? 1 : 0;
}

// One CTA per tile: the tile's changed pixels as a 256-bit mask; every list entry is tested against
// them until one is influenced.  The decision exp(-sigma) >= eps (DESIGN.md §3 c-13) is taken on the record's
// kappa-scaled whitened form in single-rounded binary32:
//   u = dx i1;  v = dy i3 + dx k;  arg = u u + v v;  influence iff arg <= thr = log2(1 / eps)
// (the oracle decides in float64; the two differ only for weights within rounding of eps)
__global__ void __launch_bounds__(64) k_select_pixels(const unsigned char *__restrict__ changed, int W, int H, int TX,
                                                      const int *__restrict__ tile_n, TileArgs a,
                                                      const Rec *__restrict__ rec, float thr,
                                                      unsigned char *__restrict__ active) {
    __shared__ unsigned s_ch[8];
    const int t = blockIdx.x, tid = threadIdx.x;
    const int tx = t % TX, ty = t / TX;
    if (tid < 8) s_ch[tid] = 0u;
    __syncthreads();
    unsigned bits = 0u;  // this thread's 4 pixels: row tid / 4, columns 4 (tid % 4) ...
    const int ly = tid >> 2, lx0 = (tid & 3) * 4;
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const int x = tx * TILE + lx0 + i, y = ty * TILE + ly;
        if (x < W && y < H && changed[(size_t)y * W + x]) bits |= 1u << i;
    }
    if (bits) atomicOr(&s_ch[(ly * TILE + lx0) >> 5], bits << ((ly * TILE + lx0) & 31));
    __syncthreads();
    unsigned any = 0u;
#pragma unroll
    for (int w = 0; w < 8; ++w) any |= s_ch[w];
    if (!any) return;
    const int n = tile_n[t];
    const int *list = a.bucket + (size_t)t * a.tile_cap;
    auto test = [&](int gid) {
        if (active[gid]) return;  // (a stale 0 only costs the test again)
        const float4 lo = reinterpret_cast<const float4 *>(rec)[(size_t)gid * 2];
        const float i3 = reinterpret_cast<const float *>(rec)[(size_t)gid * 8 + 4];
        bool hit = false;
        for (int w = 0; w < 8 && !hit; ++w) {
            unsigned m = s_ch[w];
            while (m) {
                const int b = __ffs(m) - 1;
                m &= m - 1;
                const int e = w * 32 + b;
                const float px = (float)(tx * TILE + (e & 15)) + 0.5f, py = (float)(ty * TILE + (e >> 4)) + 0.5f;
                const float dx = __fsub_rn(px, lo.x), dy = __fsub_rn(py, lo.y);
                const float u = __fmul_rn(dx, lo.z);
                const float v = __fadd_rn(__fmul_rn(dy, i3), __fmul_rn(dx, lo.w));
                const float arg = __fadd_rn(__fmul_rn(u, u), __fmul_rn(v, v));
                if (arg <= thr) {
                    hit = true;
                    break;
                }
            }
        }
        if (hit) active[gid] = 1;  // every writer stores the same value
    };
    for (int j = tid; j < min(n, a.tile_cap); j += 64) test(list[j]);
    if (n > a.tile_cap) {  // the tile's entries beyond its bucket
        const int S = spill_size(a);
        for (int e = tid; e < S; e += 64) {
            const int2 v = a.spill[e];
            if (v.x == t) test(v.y);
        }
    }
}

int launch_select_pixels(gs_ctx *c, const float *frame, const float *render, float tau, float thr, int dilate,
                         const unsigned char *changed_in, unsigned char *changed_out, unsigned char *active_out, int n,
                         cudaStream_t s) {
    const int W = c->cfg.width, H = c->cfg.height;
    const size_t npix = (size_t)W * H;
    const unsigned char *changed = changed_in;
    if (!changed_in) {
        if (!c->sel_changed) GS_CUDA_TRY(cudaMalloc(&c->sel_changed, 2 * npix));
        unsigned char *raw = c->sel_changed, *dil = c->sel_changed + npix;
        k_change_map<<<ceil_div((long long)npix, 256), 256, 0, s>>>(frame, render, npix, tau, raw, c->roi);
        if (dilate) k_dilate<<<ceil_div((long long)npix, 256), 256, 0, s>>>(raw, W, H, dil);
        changed = dilate ? dil : raw;
    }
    if (changed_out && changed_out != changed)
        GS_CUDA_TRY(cudaMemcpyAsync(changed_out, changed, npix, cudaMemcpyDeviceToDevice, s));
    GS_CUDA_TRY(cudaMemsetAsync(active_out, 0, (size_t)n, s));
    k_select_pixels<<<c->T, 64, 0, s>>>(changed, W, H, c->TX, c->tile_n, tile_args(c), c->rec, thr, active_out);
    k_count_active<<<1, 1024, 0, s>>>(active_out, n, c->dstate);
    GS_CUDA_TRY(cudaGetLastError());
    return GS_OK;
}

__global__ void __launch_bounds__(256) k_tile_sq(const TileStats *__restrict__ ts, int T, double *__restrict__ out) {
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t < T) out[t] = ts[t].sq_raw;
}

int launch_tile_sq(gs_ctx *c, double *out, cudaStream_t s) {
    k_tile_sq<<<ceil_div(c->T, 256), 256, 0, s>>>(c->tile_stats, c->T, out);
    GS_CUDA_TRY(cudaGetLastError());
    return GS_OK;
}

int launch_tile_resid(gs_ctx *c, double *resid_out, cudaStream_t s) {
    k_tile_resid<<<ceil_div(c->T, 256), 256, 0, s>>>(c->tile_stats, c->T, c->TX, c->cfg.width, c->cfg.height,
                                                     resid_out);
    GS_CUDA_TRY(cudaGetLastError());
    return GS_OK;
}

}  // namespace gs2d
