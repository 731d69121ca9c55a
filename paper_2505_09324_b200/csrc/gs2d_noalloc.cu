// gs2d_noalloc.cu -- gs_decode_static: the decode render (binning + clamped forward rasterisation, PAPER.md:152,
// Eq. 2 at PAPER.md:50-52; the same operation as gs_decode) for callers that must not allocate device memory.
//
// Who needs this.  Every other entry point works on a gs_ctx, and gs_create builds that context with a dozen
// cudaMalloc calls.  Some hosts of a decoder cannot afford a single one:
//   - a player or inference server that reserved the whole GPU for its own memory pools at start-up, so that a
//     cudaMalloc made by a plug-in library simply fails (or eats into a budget somebody else planned);
//   - a real-time playback loop that shares the GPU with other streams: cudaMalloc and cudaFree synchronise the
//     whole device, so an allocation made on the decode thread stalls every other stream's work in flight;
//   - code that runs under an "allocation forbidden" rule after initialisation (safety-certified or sandboxed
//     processes in which the allocator entry points are blocked once the pipeline is armed).
// For them the scratch of one decode -- the per-Gaussian records, the per-tile arrival counters and the per-tile id
// buckets -- lives in ONE file-scope device array of fixed size, below.  The caller brings inputs and the output
// image, nothing else; the call makes no cudaMalloc, cudaFree or other allocating runtime call.
//
// The price, stated once:
//   - limits: at most GS_STATIC_MAX_GAUSSIANS Gaussians, GS_STATIC_MAX_TILES 16x16 tiles (about one megapixel) and
//     GS_STATIC_TILE_CAP Gaussians listed in any one tile; larger jobs are refused with an error code, never
//     truncated;
//   - the array (about 4.5 MiB) is part of the library image: every GPU on which the process uses libgs2d holds it
//     from the moment the module is loaded there until the process exits, whether or not this entry point is called;
//   - there is ONE array per device, shared by every call from every thread.  It still holds what the previous call
//     left; each call clears the parts that must start at zero (counters, overflow flag) itself.  Two calls whose
//     GPU work overlaps on one device (different streams, or different host threads) race on it: callers serialise.
//
// Set-up.  In host code the array's name is only a handle for the runtime, not a device address, so the address the
// kernels receive is looked up with cudaGetSymbolAddress -- once per device, with that device current, on the first
// call made for that device.  That first call may load the module and should therefore be made during start-up,
// before any stream capture begins.  Later calls on the same device reuse the cached address.
//
// The kernels here are deliberately plain (one thread per Gaussian for the binning, one 2-warp CTA per tile for the
// render, the same record, rectangle rule, canonical list order and per-pixel arithmetic as k_bin / k_forward) and
// share only header-level device helpers with the context path; no existing kernel or launcher is touched.
#include <math.h>

#include <mutex>

#include "gs2d_bin.cuh"
#include "gs2d_sort.cuh"

namespace gs2d {
namespace {

constexpr int NA_MAX_N = GS_STATIC_MAX_GAUSSIANS;
constexpr int NA_MAX_T = GS_STATIC_MAX_TILES;
constexpr int NA_CAP = GS_STATIC_TILE_CAP;
static_assert(NA_CAP <= SORT_REG_MAX, "a bucket is sorted by one warp in registers");

// layout of the static scratch (byte offsets, each a multiple of 256)
constexpr size_t NA_OFF_FLAG = 0;                                              // unsigned: != 0 = a bucket overflowed
constexpr size_t NA_OFF_COUNT = 256;                                           // int [NA_MAX_T] arrivals per tile
constexpr size_t NA_OFF_REC = NA_OFF_COUNT + sizeof(int) * NA_MAX_T;           // Rec [NA_MAX_N]
constexpr size_t NA_OFF_BUCKET = NA_OFF_REC + sizeof(Rec) * NA_MAX_N;          // int [NA_MAX_T][NA_CAP] Gaussian ids
constexpr size_t NA_BYTES = NA_OFF_BUCKET + sizeof(int) * (size_t)NA_MAX_T * NA_CAP;
static_assert(NA_OFF_REC % 256 == 0 && NA_OFF_BUCKET % 256 == 0, "sub-arrays keep the 256-byte alignment");

// The scratch itself.  Host code must never pass `g_static_scratch` to a kernel: see static_scratch_of().
static __device__ __align__(256) unsigned char g_static_scratch[NA_BYTES];

constexpr int NA_MAX_DEVICES = 64;
std::mutex g_setup_lock;
unsigned char *g_scratch_addr[NA_MAX_DEVICES];  // device address of g_static_scratch on device d (null: not looked up yet)

// Device address of the scratch array on the CURRENT device `dev`; looked up on first use (thread-safe).
cudaError_t static_scratch_of(int dev, unsigned char **out) {
    std::lock_guard<std::mutex> hold(g_setup_lock);
    if (!g_scratch_addr[dev]) {
        unsigned char *ptr = nullptr;
        const cudaError_t e = cudaGetSymbolAddress((void **)&ptr, g_static_scratch);
        if (e != cudaSuccess) return e;
        g_scratch_addr[dev] = ptr;
    }
    *out = g_scratch_addr[dev];
    return cudaSuccess;
}

// Record, tile rectangle and bucket arrivals of one Gaussian per thread (the arithmetic of bin_cta).
__global__ void __launch_bounds__(128)
    k_static_bin(const float2 *__restrict__ mu, const float *__restrict__ chol, const float *__restrict__ rgb,
                 const float *__restrict__ opacity, int n, float cutoff, int W, int H, int TX, int TY,
                 Rec *__restrict__ rec, int *__restrict__ count, int *__restrict__ bucket,
                 unsigned *__restrict__ flag) {
    const int gid = blockIdx.x * blockDim.x + threadIdx.x;
    if (gid >= n) return;
    const float2 m = mu[gid];
    const float l1 = chol[3 * gid], l2 = chol[3 * gid + 1], l3 = chol[3 * gid + 2];
    const float cr = rgb[3 * gid], cg = rgb[3 * gid + 1], cb = rgb[3 * gid + 2], o = opacity[gid];
    int x0, y0, x1, y1;
    tile_rect(m.x, m.y, l1, l2, l3, cutoff, W, H, TX, TY, x0, y0, x1, y1);
    const float i1 = KAPPA / l1, i3 = KAPPA / l3;
    float4 *dst = reinterpret_cast<float4 *>(rec + gid);
    dst[0] = make_float4(m.x, m.y, i1, -l2 * i1 / l3);
    dst[1] = make_float4(i3, o * cr, o * cg, o * cb);
    for (int ty = y0; ty <= y1; ++ty)
        for (int tx = x0; tx <= x1; ++tx) {
            const int t = ty * TX + tx;
            const int slot = atomicAdd(count + t, 1);
            if (slot < NA_CAP) bucket[(size_t)t * NA_CAP + slot] = gid;
            else *flag = 1u;  // every writer stores the same value
        }
}

__device__ __forceinline__ float na_ex2_neg(float p) {  // 2^(-p), MUFU.EX2
    float w;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(w) : "f"(-p));
    return w;
}

// One CTA of 64 threads per tile: the tile's bucket is sorted by id, split between the two warps in the fixed
// proportion of k_forward, each lane sums its column x 8 rows over its warp's share, warp 0 adds warp 1's partial
// image to its own, clamps to [0,1] and the CTA writes the tile.  Nothing is written if a bucket overflowed.
__global__ void __launch_bounds__(SORT_CTA_THREADS)
    k_static_forward(const Rec *__restrict__ rec, const int *__restrict__ count, int *__restrict__ bucket,
                     const unsigned *__restrict__ flag, int W, int H, int TX, float *__restrict__ image_out) {
    __shared__ __align__(16) float s_io[TILE * TILE * 3];
    if (*flag != 0u) return;  // (uniform over the grid)
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const int t = blockIdx.x, tx = t % TX, ty = t / TX;
    const int cx = lane & 15, hf = lane >> 4;
    const int gx = tx * TILE + cx, gy0 = ty * TILE + 8 * hf;
    const float px = (float)gx + 0.5f, py0 = (float)gy0 + 0.5f;

    const int n = count[t];
    int *seg = bucket + (size_t)t * NA_CAP;
    cta_sort_tile(seg, n, tid);  // ends with a barrier
    const int n0 = (n * 9) / 20;
    const int cnt = wid == 0 ? n0 : n - n0;
    const int *list = seg + (wid == 0 ? 0 : n0);

    float2 Cp[4][3];
#pragma unroll
    for (int k = 0; k < 4; ++k) Cp[k][0] = Cp[k][1] = Cp[k][2] = make_float2(0.0f, 0.0f);
    for (int j = 0; j < cnt; ++j) {
        const int gid = list[j];  // (uniform over the warp: a broadcast load)
        const float4 lo = __ldg(reinterpret_cast<const float4 *>(rec) + (size_t)gid * 2);
        const float4 hi = __ldg(reinterpret_cast<const float4 *>(rec) + (size_t)gid * 2 + 1);
        const float dx = px - lo.x, dy0 = py0 - lo.y;
        const float u = dx * lo.z;
        const float2 uu = dup2(u * u);
        const float2 v0 = dup2(fmaf(dx, lo.w, dy0 * hi.x));
        const float2 hx = dup2(hi.x), cr = dup2(hi.y), cg = dup2(hi.z), cb = dup2(hi.w);
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            const float2 v = __ffma2_rn(hx, c_rowpair[k], v0);
            const float2 p = __ffma2_rn(v, v, uu);
            const float2 w = make_float2(na_ex2_neg(p.x), na_ex2_neg(p.y));
            Cp[k][0] = __ffma2_rn(w, cr, Cp[k][0]);
            Cp[k][1] = __ffma2_rn(w, cg, Cp[k][1]);
            Cp[k][2] = __ffma2_rn(w, cb, Cp[k][2]);
        }
    }
    float Cv[8][3];
#pragma unroll
    for (int i = 0; i < 8; ++i)
#pragma unroll
        for (int ch = 0; ch < 3; ++ch) Cv[i][ch] = (i & 1) ? Cp[i >> 1][ch].y : Cp[i >> 1][ch].x;
    if (wid == 1) {
#pragma unroll
        for (int i = 0; i < 8; ++i)
#pragma unroll
            for (int ch = 0; ch < 3; ++ch) s_io[(8 * hf + i) * 48 + cx * 3 + ch] = Cv[i][ch];
    }
    __syncthreads();
    if (wid == 0) {  // first share + second share, clamped; each lane overwrites exactly the cells it has just read
#pragma unroll
        for (int i = 0; i < 8; ++i)
#pragma unroll
            for (int ch = 0; ch < 3; ++ch) {
                const int e = (8 * hf + i) * 48 + cx * 3 + ch;
                s_io[e] = fminf(fmaxf(Cv[i][ch] + s_io[e], 0.0f), 1.0f);
            }
    }
    __syncthreads();
    // the CTA writes the tile's rows: 48 consecutive floats per row, clipped at the frame's edges
    const int rows = min(TILE, H - ty * TILE), cols3 = 3 * min(TILE, W - tx * TILE);
    for (int e = tid; e < TILE * 48; e += SORT_CTA_THREADS) {
        const int r = e / 48, c = e - r * 48;
        if (r < rows && c < cols3) image_out[((size_t)(ty * TILE + r) * W + (size_t)tx * TILE) * 3 + c] = s_io[e];
    }
}

}  // namespace
}  // namespace gs2d

using namespace gs2d;

extern "C" int gs_decode_static(gs_params p, int width, int height, float cutoff, float *image_out, void *stream) {
    if (!p.mu || !p.chol || !p.rgb || !p.opacity || !image_out || p.n < 1 || width < 1 || height < 1 ||
        !(cutoff > 0.0f) || !isfinite(cutoff))
        return GS_ERR_INVALID_ARGUMENT;
    if (((size_t)p.mu & 7u) || ((size_t)p.chol & 3u) || ((size_t)p.rgb & 3u) || ((size_t)p.opacity & 3u) ||
        ((size_t)image_out & 3u))
        return GS_ERR_INVALID_ARGUMENT;
    const long long TX = (width + TILE - 1) / TILE, TY = (height + TILE - 1) / TILE;
    // beyond the static scratch: refused, not truncated
    if (p.n > NA_MAX_N || TX * TY > NA_MAX_T) return GS_ERR_CAPACITY;

    cudaStream_t s = (cudaStream_t)stream;
    int dev = -1;
    GS_CUDA_TRY(cudaGetDevice(&dev));
    if (dev < 0 || dev >= NA_MAX_DEVICES) return GS_ERR_UNSUPPORTED;
    unsigned char *base = nullptr;
    {
        const cudaError_t e = static_scratch_of(dev, &base);  // first call on this device: cudaGetSymbolAddress
        if (e != cudaSuccess) {
            set_cuda_error(e, "cudaGetSymbolAddress(g_static_scratch)");
            return GS_ERR_CUDA;
        }
    }
    unsigned *flag = reinterpret_cast<unsigned *>(base + NA_OFF_FLAG);
    int *count = reinterpret_cast<int *>(base + NA_OFF_COUNT);
    Rec *rec = reinterpret_cast<Rec *>(base + NA_OFF_REC);
    int *bucket = reinterpret_cast<int *>(base + NA_OFF_BUCKET);
    const int T = (int)(TX * TY);

    // the previous call's counters and flag are still there: clear what this call counts into
    GS_CUDA_TRY(cudaMemsetAsync(base, 0, NA_OFF_COUNT + sizeof(int) * (size_t)T, s));
    k_static_bin<<<(p.n + 127) / 128, 128, 0, s>>>(reinterpret_cast<const float2 *>(p.mu), p.chol, p.rgb, p.opacity,
                                                   p.n, cutoff, width, height, (int)TX, (int)TY, rec, count, bucket,
                                                   flag);
    GS_CUDA_TRY(cudaGetLastError());
    k_static_forward<<<T, SORT_CTA_THREADS, 0, s>>>(rec, count, bucket, flag, width, height, (int)TX, image_out);
    GS_CUDA_TRY(cudaGetLastError());
    unsigned overflow = 0u;
    GS_CUDA_TRY(cudaMemcpyAsync(&overflow, flag, sizeof overflow, cudaMemcpyDeviceToHost, s));
    GS_CUDA_TRY(cudaStreamSynchronize(s));
    return overflow ? GS_ERR_CAPACITY : GS_OK;
}
