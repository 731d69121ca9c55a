// gs2d_select.cu -- P-frame selection (
// BASELINE.json configs[3]; DESIGN.md §3 c-9).  Runs after a FWD_STATS forward pass:
//   r_t = abs_clamp_t / (3 * valid pixels of tile t);  tile changed iff r_t > tau (strict)
//   active[n] = 1 iff n is listed in at least one changed tile.
#include "gs2d_internal.cuh"

namespace gs2d {

__global__ void __launch_bounds__(256) k_flag_tiles(const TileStats *__restrict__ ts, int T, int TX, int W, int H,
                                                    double tau, unsigned char *__restrict__ tile_flag) {
    int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= T) return;
    int tx = t % TX, ty = t / TX;
    int vw = min(TILE, W - tx * TILE), vh = min(TILE, H - ty * TILE);
    double r = ts[t].abs_clamp / (double)(3 * vw * vh);
    tile_flag[t] = r > tau ? 1 : 0;
}

__global__ void __launch_bounds__(256) k_tile_resid(const TileStats *__restrict__ ts, int T, int TX, int W, int H,
                                                    double *__restrict__ resid) {
    int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= T) return;
    int tx = t % TX, ty = t / TX;
    int vw = min(TILE, W - tx * TILE), vh = min(TILE, H - ty * TILE);
    resid[t] = ts[t].abs_clamp / (double)(3 * vw * vh);
}

// one warp per tile: the lanes stride over the list of a changed tile
__global__ void __launch_bounds__(256) k_mark_active(int T, const int *__restrict__ tile_n,
                                                     const int *__restrict__ bucket, int tile_cap,
                                                     const unsigned char *__restrict__ tile_flag,
                                                     unsigned char *__restrict__ active) {
    const int t = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (t >= T || !tile_flag[t]) return;
    const int n = tile_n[t];  // 0 when the binning exceeded a capacity
    const int *list = bucket + (size_t)t * tile_cap;
    for (int p = threadIdx.x & 31; p < n; p += 32) active[list[p]] = 1;  // every writer stores the same value
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
    k_mark_active<<<ceil_div(c->T, 8), 256, 0, s>>>(c->T, c->tile_n, c->bucket, c->tile_cap, c->tile_flag, active_out);
    k_count_active<<<1, 1024, 0, s>>>(active_out, n, c->dstate);
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
