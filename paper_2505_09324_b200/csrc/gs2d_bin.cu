// gs2d_bin.cu -- tile binning (DESIGN.md §5 "binning").
//
//   k_preprocess  per Gaussian: record, tile rectangle (single-rounded binary32 rule,
//                 DESIGN.md §3 c-2), and a count per covered tile (RED into tile_count)
//   k_scan_tiles  one CTA: exclusive prefix of tile_count -> range[T+1], cursor[T]; P
//   k_fill        per Gaussian: claim a slot in every covered tile's segment
//   k_sort_tiles  per tile: sort the segment by Gaussian id (canonical order)
//
// This is a one-digit radix (counting) sort of the (tile, Gaussian) pairs with the tile id
// as the digit, followed by a segmented sort that restores the stable order inside each
// digit; it replaces the multi-pass LSD radix sort north_star sketches.
#include "gs2d_internal.cuh"

namespace gs2d {

// sqrt(0.5 * log2(e)) : folds the 1/2 of sigma and the change of base into the record
constexpr float KAPPA = 0.84932180028801904f;
constexpr int SMALL_RECT = 8;       // rectangles up to this many tiles are walked by their own thread
constexpr int SORT_SMEM_MAX = 2048; // longest segment sorted in shared memory

// Tile rectangle of one Gaussian: DESIGN.md §3 c-2.  Every operation is binary32,
// round-to-nearest, one rounding each; the *_rn intrinsics are never contracted into FMAs.
__device__ __forceinline__ bool tile_rect(float mux, float muy, float l1, float l2, float l3, float k, int W, int H,
                                          int TX, int TY, short4 &r) {
    r = make_short4(0, 0, -1, -1);
    if (!(isfinite(mux) && isfinite(muy) && isfinite(l1) && isfinite(l2) && isfinite(l3))) return false;
    if (l1 == 0.0f || l3 == 0.0f) return false;
    float rx = __fmul_rn(k, fabsf(l1));
    float s22 = __fadd_rn(__fmul_rn(l2, l2), __fmul_rn(l3, l3));
    float ry = __fmul_rn(k, __fsqrt_rn(s22));
    float lo_x = __fsub_rn(mux, rx), hi_x = __fadd_rn(mux, rx);
    float lo_y = __fsub_rn(muy, ry), hi_y = __fadd_rn(muy, ry);
    if (hi_x < 0.0f || lo_x >= (float)W || hi_y < 0.0f || lo_y >= (float)H) return false;
    // NaN extents (k or the products overflowed to inf - inf) fail every comparison above; cull them
    if (!(lo_x == lo_x && hi_x == hi_x && lo_y == lo_y && hi_y == hi_y)) return false;
    float fx0 = fmaxf(0.0f, floorf(__fmul_rn(lo_x, 0.0625f)));
    float fx1 = fminf((float)(TX - 1), floorf(__fmul_rn(hi_x, 0.0625f)));
    float fy0 = fmaxf(0.0f, floorf(__fmul_rn(lo_y, 0.0625f)));
    float fy1 = fminf((float)(TY - 1), floorf(__fmul_rn(hi_y, 0.0625f)));
    r = make_short4((short)(int)fx0, (short)(int)fy0, (short)(int)fx1, (short)(int)fy1);
    return true;
}

// Walk the tiles of this thread's rectangle; rectangles larger than SMALL_RECT tiles are
// walked by the whole warp, one rectangle at a time, so that one fat Gaussian does not
// serialise thousands of atomics on one lane.  f(tile_id, gaussian_id).
template <typename F>
__device__ __forceinline__ void for_each_tile(short4 r, int n, int TX, F f) {
    const unsigned full = 0xffffffffu;
    int w = r.z - r.x + 1, h = r.w - r.y + 1;
    int cnt = (w > 0 && h > 0) ? w * h : 0;
    if (cnt > 0 && cnt <= SMALL_RECT) {
        for (int ty = r.y; ty <= r.w; ++ty)
            for (int tx = r.x; tx <= r.z; ++tx) f(ty * TX + tx, n);
    }
    unsigned big = __ballot_sync(full, cnt > SMALL_RECT);
    int lane = threadIdx.x & 31;
    while (big) {
        int src = __ffs(big) - 1;
        big &= big - 1;
        int x0 = __shfl_sync(full, (int)r.x, src), y0 = __shfl_sync(full, (int)r.y, src);
        int ww = __shfl_sync(full, w, src), tot = __shfl_sync(full, cnt, src);
        int nn = __shfl_sync(full, n, src);
        for (int i = lane; i < tot; i += 32) {
            int dy = i / ww, dx = i - dy * ww;
            f((y0 + dy) * TX + (x0 + dx), nn);
        }
    }
}

__global__ void __launch_bounds__(256) k_preprocess(int N, const float2 *__restrict__ mu, const float *__restrict__ chol,
                                                    const float *__restrict__ rgb, const float *__restrict__ opacity,
                                                    float cutoff, int W, int H, int TX, int TY, Rec *__restrict__ rec,
                                                    short4 *__restrict__ rect, int *__restrict__ tile_count) {
    int n = blockIdx.x * blockDim.x + threadIdx.x;
    short4 r = make_short4(0, 0, -1, -1);
    if (n < N) {
        float2 m = mu[n];
        float l1 = chol[3 * n], l2 = chol[3 * n + 1], l3 = chol[3 * n + 2];
        float o = opacity[n];
        tile_rect(m.x, m.y, l1, l2, l3, cutoff, W, H, TX, TY, r);
        float i1 = KAPPA / l1, i3 = KAPPA / l3;
        float4 lo = make_float4(m.x, m.y, i1, -l2 * i1 / l3);
        float4 hi = make_float4(i3, o * rgb[3 * n], o * rgb[3 * n + 1], o * rgb[3 * n + 2]);
        float4 *dst = reinterpret_cast<float4 *>(rec + n);
        dst[0] = lo;
        dst[1] = hi;
        rect[n] = r;
    }
    for_each_tile(r, n, TX, [&](int t, int) { atomicAdd(tile_count + t, 1); });
}

// One CTA of 1024 threads.  Thread i owns a contiguous run of `ipt` tiles.
__global__ void __launch_bounds__(1024) k_scan_tiles(int T, int *__restrict__ tile_count, int *__restrict__ range,
                                                     int *__restrict__ cursor, long long cap, DeviceState *st) {
    __shared__ int warp_tot[32];
    int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    int ipt = (T + 1023) / 1024;
    int b = tid * ipt, e = min(b + ipt, T);
    int local = 0;
    for (int i = b; i < e; ++i) local += tile_count[i];
    int incl = local;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        int o = __shfl_up_sync(0xffffffffu, incl, d);
        if (lane >= d) incl += o;
    }
    if (lane == 31) warp_tot[wid] = incl;
    __syncthreads();
    if (wid == 0) {
        int v = warp_tot[lane], s = v;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            int o = __shfl_up_sync(0xffffffffu, s, d);
            if (lane >= d) s += o;
        }
        warp_tot[lane] = s - v;  // exclusive
    }
    __syncthreads();
    int run = warp_tot[wid] + incl - local;
    for (int i = b; i < e; ++i) {
        int c = tile_count[i];
        range[i] = run;
        cursor[i] = run;
        tile_count[i] = 0;  // ready for the next binning
        run += c;
    }
    if (tid == 1023) {  // the last thread's running total is P
        // threads whose run is empty still carry the correct prefix
        range[T] = run;
        st->n_pairs = run;
        if ((long long)run > cap) atomicOr(&st->flags, FLAG_CAPACITY);
    }
}

__global__ void __launch_bounds__(256) k_fill(int N, const short4 *__restrict__ rect, int TX, int *__restrict__ cursor,
                                              int *__restrict__ list, int *__restrict__ pair_tile, long long cap,
                                              const DeviceState *__restrict__ st) {
    if ((long long)st->n_pairs > cap) return;  // capacity exceeded: nothing downstream runs
    int n = blockIdx.x * blockDim.x + threadIdx.x;
    short4 r = n < N ? rect[n] : make_short4(0, 0, -1, -1);
    for_each_tile(r, n, TX, [&](int t, int g) {
        int pos = atomicAdd(cursor + t, 1);
        list[pos] = g;
        pair_tile[pos] = t;
    });
}

// Bitonic network in which every comparator puts the smaller key at the lower index (the
// first step of each merge mirrors the upper half).  Positions >= n behave as +infinity and
// are never touched, so any n works without padding.  `a` may be shared or global memory.
template <int THREADS>
__device__ __forceinline__ void bitonic_all_up(int *a, int n, int tid) {
    int m = 1;
    while (m < n) m <<= 1;
    int half_m = m >> 1;
    for (int k = 2; k <= m; k <<= 1) {
        int half = k >> 1;
        for (int i = tid; i < half_m; i += THREADS) {  // mirror step
            int blk = i / half, off = i - blk * half;
            int lo = blk * k + off, hi = blk * k + k - 1 - off;
            if (hi < n) {
                int x = a[lo], y = a[hi];
                if (x > y) {
                    a[lo] = y;
                    a[hi] = x;
                }
            }
        }
        __syncthreads();
        for (int j = half >> 1; j > 0; j >>= 1) {
            for (int i = tid; i < half_m; i += THREADS) {
                int lo = ((i / j) * (j << 1)) + (i % j), hi = lo + j;
                if (hi < n) {
                    int x = a[lo], y = a[hi];
                    if (x > y) {
                        a[lo] = y;
                        a[hi] = x;
                    }
                }
            }
            __syncthreads();
        }
    }
}

constexpr int SORT_THREADS = 128;

__global__ void __launch_bounds__(SORT_THREADS) k_sort_tiles(const int *__restrict__ range, int *list, long long cap,
                                                             const DeviceState *__restrict__ st) {
    __shared__ int s_ids[SORT_SMEM_MAX];
    if ((long long)st->n_pairs > cap) return;
    int t = blockIdx.x, tid = threadIdx.x;
    int start = range[t], n = range[t + 1] - start;
    if (n <= 1) return;
    int *seg = list + start;
    if (n <= 32) {  // one warp, registers only
        if (tid >= 32) return;
        int v = tid < n ? seg[tid] : 0x7fffffff;
#pragma unroll
        for (int k = 2; k <= 32; k <<= 1) {
#pragma unroll
            for (int j = k >> 1; j > 0; j >>= 1) {
                int o = __shfl_xor_sync(0xffffffffu, v, j);
                bool keep_min = ((tid & j) == 0) == ((tid & k) == 0);
                v = keep_min ? min(v, o) : max(v, o);
            }
        }
        if (tid < n) seg[tid] = v;
        return;
    }
    if (n <= SORT_SMEM_MAX) {
        for (int i = tid; i < n; i += SORT_THREADS) s_ids[i] = seg[i];
        __syncthreads();
        bitonic_all_up<SORT_THREADS>(s_ids, n, tid);
        for (int i = tid; i < n; i += SORT_THREADS) seg[i] = s_ids[i];
        return;
    }
    bitonic_all_up<SORT_THREADS>(seg, n, tid);  // degenerate tiles: in place in global memory
}

int launch_binning(gs_ctx *c, const gs_params &p, cudaStream_t s, cudaEvent_t *ev) {
    int N = p.n;
    int blocks = ceil_div(N, 256);
    if (ev) cudaEventRecord(ev[0], s);
    k_preprocess<<<blocks, 256, 0, s>>>(N, reinterpret_cast<const float2 *>(p.mu), p.chol, p.rgb, p.opacity,
                                        c->cfg.cutoff, c->cfg.width, c->cfg.height, c->TX, c->TY, c->rec, c->rect,
                                        c->tile_count);
    if (ev) cudaEventRecord(ev[1], s);
    k_scan_tiles<<<1, 1024, 0, s>>>(c->T, c->tile_count, c->range, c->cursor, c->cap_pairs, c->dstate);
    if (ev) cudaEventRecord(ev[2], s);
    k_fill<<<blocks, 256, 0, s>>>(N, c->rect, c->TX, c->cursor, c->list, c->pair_tile, c->cap_pairs, c->dstate);
    if (ev) cudaEventRecord(ev[3], s);
    k_sort_tiles<<<c->T, SORT_THREADS, 0, s>>>(c->range, c->list, c->cap_pairs, c->dstate);
    if (ev) cudaEventRecord(ev[4], s);
    c->last_n = N;
    GS_CUDA_TRY(cudaGetLastError());
    return GS_OK;
}

}  // namespace gs2d
