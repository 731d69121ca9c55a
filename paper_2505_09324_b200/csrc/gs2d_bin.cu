// gs2d_bin.cu -- tile binning (DESIGN.md §5 "binning").
//
// A binning is a one-digit counting sort of the (tile, Gaussian) pairs with the tile id as the
// digit, done in ONE pass: every tile owns a bucket of tile_cap ids, and the counting atomic
// of an arrival returns its slot in the bucket.  There is no scan and no fill pass.  The
// canonical order inside a tile (ascending Gaussian id, DESIGN.md §3 c-2) is restored by the
// consumer of the bins that needs it: the per-tile sort stage (gs2d_sort.cuh), the prologue of
// the render kernel.  The fit kernel sums in arrival order and streams the 48-byte bucket
// records that the binning stores beside the ids.  The canonical CSR form (range[T+1], list[P]) exists only on demand
// (gs_get_bins): k_compact_*.
//
//   k_bin           per Gaussian: record, tile rectangle (single-rounded binary32 rule), arrivals
//   k_sort_tiles    the consumer stage alone (paths that do not run the forward kernel), or only
//                   the sort of buckets that a fit iteration consumed unsorted
//   k_compact_scan  one CTA: exclusive prefix of tile_n -> range[T+1]
//   k_compact_copy  one warp per tile: bucket -> list[range[t] ...)
//
// Inside the fit loop k_bin does not run at all: the fused Adam kernel bins the parameters it
// has just updated (gs2d_optim.cu), so an iteration is forward, backward, Adam.
#include "gs2d_bin.cuh"
#include "gs2d_sort.cuh"

namespace gs2d {

__global__ void __launch_bounds__(256)
    k_bin(int N, const float2 *__restrict__ mu, const float *__restrict__ chol, const float *__restrict__ rgb,
          const float *__restrict__ opacity, BinArgs a) {
    __shared__ BinSmem<256> s_bin;
    // the render kernel behind this one may be scheduled from now on (it waits for this grid's completion before
    // it reads anything written here: gs2d_raster.cu)
    asm volatile("griddepcontrol.launch_dependents;");
    const int n = blockIdx.x * blockDim.x + threadIdx.x;
    const bool valid = n < N;
    float2 m = make_float2(0.f, 0.f);
    float l1 = 0.f, l2 = 0.f, l3 = 0.f, r = 0.f, g = 0.f, b = 0.f, o = 0.f;
    if (valid) {
        m = mu[n];
        l1 = chol[3 * n];
        l2 = chol[3 * n + 1];
        l3 = chol[3 * n + 2];
        r = rgb[3 * n];
        g = rgb[3 * n + 1];
        b = rgb[3 * n + 2];
        o = opacity[n];
    }
    bin_cta<256>(a, s_bin, valid, n, m.x, m.y, l1, l2, l3, r, g, b, o);
}

// consume == 1: the consumer stage of a fresh binning (count -> tile_n, sort);
// consume == 0: only sort the id buckets that the fit kernel consumed without sorting;
// consume == 2: only sort the id buckets of a FRESH binning, which stays fresh (deterministic mode: the fit
//               kernel then sums every list in ascending id order).
// (The launch order of the next consumer is left as it is: this kernel files no tiles.)
__global__ void __launch_bounds__(SORT_CTA_THREADS) k_sort_tiles(TileArgs a, int consume, int *refile_order, int refile_oc) {
    const int t = blockIdx.x, tid = threadIdx.x;
    int n;
    if (!consume) {
        n = a.tile_n[t];
    } else if (consume == 2) {  // the arrivals of a fresh binning, not consumed (the fit kernel will)
        n = max(tile_count_of(a, gridDim.x, t), 0);
        // ... and the tile is filed under the class of its CURRENT length for the launch that follows (the class counters
        // of that launch were zeroed by the host): whether a tile is fitted by a team or by one warp -- two
        // different orders of summation -- then depends on its list, not on what the context did before
        if (tid == 0 && refile_order) {
            const int cls = tile_class(n);
            const int pos = atomicAdd(&a.st->n_class[refile_oc][cls], 1);
            refile_order[(size_t)cls * gridDim.x + pos] = t;
        }
    } else {
        n = tile_count_of(a, gridDim.x, t);
        if (tid == 0) tile_publish(a, gridDim.x, t, n);
    }
    if (n > 1) cta_sort_tile(a.bucket + (size_t)t * a.tile_cap, min(n, a.tile_cap), tid);  // (the bucket's part)
}

// range[t] = exclusive prefix of tile_n (one CTA walks the tiles in chunks of 1024)
__global__ void __launch_bounds__(1024) k_compact_scan(const int *__restrict__ tile_n, int T, int *__restrict__ range) {
    __shared__ int s_w[32];
    __shared__ int s_carry;
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    if (tid == 0) s_carry = 0;
    __syncthreads();
    for (int b0 = 0; b0 < T; b0 += 1024) {
        const int e = b0 + tid;
        const int v = e < T ? tile_n[e] : 0;
        int x = v;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const int o = __shfl_up_sync(0xffffffffu, x, d);
            if (lane >= d) x += o;
        }
        if (lane == 31) s_w[wid] = x;
        __syncthreads();
        if (wid == 0) {
            int w = s_w[lane], y = w;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                const int o = __shfl_up_sync(0xffffffffu, y, d);
                if (lane >= d) y += o;
            }
            s_w[lane] = y - w;  // exclusive over the warps
        }
        __syncthreads();
        const int carry = s_carry;
        if (e < T) range[e] = carry + s_w[wid] + x - v;
        __syncthreads();
        if (tid == 1023) s_carry = carry + s_w[wid] + x;
        __syncthreads();
    }
    if (tid == 0) range[T] = s_carry;
}

// one warp per tile: the bucket's (sorted) ids, then the tile's spilled ids, unsorted
__global__ void __launch_bounds__(256) k_compact_copy(int T, const int *__restrict__ tile_n,
                                                      const int *__restrict__ range, TileArgs a,
                                                      int *__restrict__ list) {
    const int t = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5), lane = threadIdx.x & 31;
    if (t >= T) return;
    const int n = tile_n[t], o = range[t], nm = min(n, a.tile_cap);
    const int *src = a.bucket + (size_t)t * a.tile_cap;
    for (int i = lane; i < nm; i += 32) list[o + i] = src[i];
    if (n > nm) {
        const int S = spill_size(a);
        int at = o + nm;
        for (int e0 = 0; e0 < S; e0 += 32) {
            const int e = e0 + lane;
            int2 v = make_int2(-1, -1);
            if (e < S) v = a.spill[e];
            const bool hit = v.x == t;
            const unsigned m = __ballot_sync(0xffffffffu, hit);
            if (hit) list[at + __popc(m & ((1u << lane) - 1u))] = v.y;
            at += __popc(m);
        }
    }
}
// tiles with spilled entries: their list segment is brought into ascending order as a whole
__global__ void __launch_bounds__(SORT_CTA_THREADS) k_compact_sort_spilled(const int *__restrict__ tile_n,
                                                                          const int *__restrict__ range, int tile_cap,
                                                                          int *__restrict__ list) {
    const int t = blockIdx.x, n = tile_n[t];
    if (n <= tile_cap) return;
    bitonic_all_up<SORT_CTA_THREADS>(list + range[t], n, threadIdx.x);
}

BinArgs bin_args(gs_ctx *c, bool next_epoch, const unsigned char *active, int mode) {
    if (next_epoch) ++c->epoch;
    BinArgs a;
    a.cutoff = c->cfg.cutoff;
    a.W = c->cfg.width;
    a.H = c->cfg.height;
    a.TX = c->TX;
    a.TY = c->TY;
    a.tile_cap = c->tile_cap;
    a.slot = (int)(c->epoch & 1u);
    a.rec = c->rec;
    a.tile_count = c->tile_count;
    a.bucket = c->bucket;
    a.spill = c->spill;
    a.spill_cap = c->spill_cap;
    a.active = active;
    a.mode = active ? mode : 0;
    a.st = c->dstate;
    a.q = c->quant;
    a.pair_info = c->deterministic ? c->pair_info : nullptr;
    return a;
}

TileArgs tile_args(gs_ctx *c) {
    TileArgs a;
    a.tile_count = c->tile_count;
    a.tile_n = c->tile_n;
    a.bucket = c->bucket;
    a.tile_cap = c->tile_cap;
    a.spill = c->spill;
    a.spill_cap = c->spill_cap;
    a.slot = (int)(c->epoch & 1u);
    a.cap_pairs = c->cap_pairs;
    a.st = c->dstate;
    return a;
}

void discard_fresh_bins(gs_ctx *c, cudaStream_t s) {
    if (!c->fresh) return;
    // nobody consumed the arrivals: clear them and the epoch's counters, and give the epoch back
    const int slot = (int)(c->epoch & 1u);
    cudaMemsetAsync(c->tile_count + (size_t)slot * c->T, 0, sizeof(int) * (size_t)c->T, s);
    cudaMemsetAsync(&c->dstate->pair_total[slot], 0, sizeof(unsigned long long), s);
    cudaMemsetAsync(&c->dstate->tile_ovf[slot], 0, sizeof(int), s);
    cudaMemsetAsync(&c->dstate->spill_count[slot], 0, sizeof(unsigned), s);
    --c->epoch;
    c->fresh = false;
}

int ensure_bins(gs_ctx *c, const gs_params &p, cudaStream_t s, const unsigned char *active, int mode) {
    if (!active) mode = 0;
    if (c->fresh && c->fresh_mu == p.mu && c->fresh_n == p.n && c->fresh_mode == mode &&
        (mode == 0 || c->fresh_active == active))
        return GS_OK;
    discard_fresh_bins(c, s);
    const BinArgs a = bin_args(c, true, active, mode);
    k_bin<<<ceil_div(p.n, 256), 256, 0, s>>>(p.n, reinterpret_cast<const float2 *>(p.mu), p.chol, p.rgb, p.opacity, a);
    GS_CUDA_TRY(cudaGetLastError());
    c->fresh = true;
    c->fresh_mu = p.mu;
    c->fresh_n = p.n;
    c->fresh_active = active;
    c->fresh_mode = mode;
    return GS_OK;
}

int launch_sort_tiles(gs_ctx *c, cudaStream_t s) {
    if (c->fresh) {
        k_sort_tiles<<<c->T, SORT_CTA_THREADS, 0, s>>>(tile_args(c), 1, nullptr, 0);
        c->fresh = false;
        c->sorted = true;
    } else if (!c->sorted) {
        k_sort_tiles<<<c->T, SORT_CTA_THREADS, 0, s>>>(tile_args(c), 0, nullptr, 0);
        c->sorted = true;
    }
    GS_CUDA_TRY(cudaGetLastError());
    return GS_OK;
}

int launch_presort_tiles(gs_ctx *c, cudaStream_t s) {
    if (!c->fresh) return GS_OK;
    const int oc = (int)(c->fwd_launches % 3u);  // the order buffer the next consumer launch reads
    GS_CUDA_TRY(cudaMemsetAsync(&c->dstate->n_class[oc][0], 0, sizeof(int) * NCLS, s));
    k_sort_tiles<<<c->T, SORT_CTA_THREADS, 0, s>>>(tile_args(c), 2, c->tile_order + (size_t)oc * NCLS * c->T, oc);
    GS_CUDA_TRY(cudaGetLastError());
    return GS_OK;
}

int ensure_pair_slots(gs_ctx *c) {
    if (!c->pair_info) GS_CUDA_TRY(cudaMalloc(&c->pair_info, sizeof(int4) * (size_t)c->cfg.max_gaussians));
    if (!c->pair_mom) GS_CUDA_TRY(cudaMalloc(&c->pair_mom, sizeof(float) * 8 * (size_t)c->cap_pairs));
    return GS_OK;
}

int launch_compact(gs_ctx *c, int *range_out, int *list_out, cudaStream_t s) {
    k_compact_scan<<<1, 1024, 0, s>>>(c->tile_n, c->T, range_out);
    if (list_out)
    {
        k_compact_copy<<<ceil_div(c->T, 8), 256, 0, s>>>(c->T, c->tile_n, range_out, tile_args(c), list_out);
        k_compact_sort_spilled<<<c->T, SORT_CTA_THREADS, 0, s>>>(c->tile_n, range_out, c->tile_cap, list_out);
    }
    GS_CUDA_TRY(cudaGetLastError());
    return GS_OK;
}

}  // namespace gs2d
