// gs2d_bin.cu -- tile binning (DESIGN.md §5 "binning").
//
//   k_preprocess  per Gaussian: record, tile rectangle (single-rounded binary32 rule,
//                 DESIGN.md §3 c-2); one counting atomic per covered tile whose RETURN value is
//                 the pair's arrival rank inside its tile (kept Gaussian-major in pair_rank)
//   k_scan_tiles  one CTA: exclusive prefix of tile_count -> range[T+1]; P; the backward work
//                 items (tile, chunk of BWD_CHUNK entries); the list of over-long tiles
//   k_fill        per Gaussian: list[range[t] + rank] = id   (no atomics)
//   k_sort_tiles  per tile: sort the segment by Gaussian id (canonical order); one warp per
//                 tile with the keys in registers, a CTA-wide network for over-long tiles
//
// This is a one-digit radix (counting) sort of the (tile, Gaussian) pairs with the tile id
// as the digit, followed by a segmented sort that restores the stable order inside each
// digit; it replaces the multi-pass LSD radix sort north_star sketches.
#include "gs2d_internal.cuh"
#include "gs2d_sort.cuh"

namespace gs2d {

// sqrt(0.5 * log2(e)) : folds the 1/2 of sigma and the change of base into the record
constexpr float KAPPA = 0.84932180028801904f;
constexpr int SMALL_RECT = 32;      // rectangles up to this many tiles are walked by their own thread
constexpr int RECT_BATCH = 8;       // independent atomics / loads in flight per thread

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

// Walk the tiles of a rectangle.  Pair i of Gaussian n (i = dy * w + dx, row-major inside the
// rectangle) lives in slot base + i of the Gaussian-major pair arrays.  Rectangles of up to
// SMALL_RECT tiles are walked by their own thread in batches of RECT_BATCH, so that a batch of
// independent atomics (or loads) is in flight before the first result is consumed; larger
// rectangles are walked by the whole warp, one rectangle at a time, so that one fat Gaussian
// does not serialise thousands of operations on one lane.
//   produce(tile, gaussian) -> int          (the atomic or the load)
//   consume(slot, tile, gaussian, value)    (the dependent store)
template <typename FP, typename FC>
__device__ __forceinline__ void for_each_pair(short4 r, int n, unsigned long long base, int TX, FP produce,
                                              FC consume) {
    const unsigned full = 0xffffffffu;
    const int w = r.z - r.x + 1, h = r.w - r.y + 1;
    const int cnt = (w > 0 && h > 0) ? w * h : 0;
    if (cnt > 0 && cnt <= SMALL_RECT) {
        int tx = r.x, ty = r.y;
        for (int i0 = 0; i0 < cnt; i0 += RECT_BATCH) {
            int val[RECT_BATCH], til[RECT_BATCH];
#pragma unroll
            for (int j = 0; j < RECT_BATCH; ++j) {
                til[j] = ty * TX + tx;
                if (i0 + j < cnt) val[j] = produce(til[j], n);
                if (++tx > r.z) {
                    tx = r.x;
                    ++ty;
                }
            }
#pragma unroll
            for (int j = 0; j < RECT_BATCH; ++j)
                if (i0 + j < cnt) consume(base + (unsigned long long)(i0 + j), til[j], n, val[j]);
        }
    }
    unsigned big = __ballot_sync(full, cnt > SMALL_RECT);
    const int lane = threadIdx.x & 31;
    while (big) {
        const int src = __ffs(big) - 1;
        big &= big - 1;
        const int x0 = __shfl_sync(full, (int)r.x, src), y0 = __shfl_sync(full, (int)r.y, src);
        const int ww = __shfl_sync(full, w, src), tot = __shfl_sync(full, cnt, src);
        const int nn = __shfl_sync(full, n, src);
        const unsigned long long bb = __shfl_sync(full, base, src);
        for (int i = lane; i < tot; i += 32) {
            const int dy = i / ww, dx = i - dy * ww;
            const int t = (y0 + dy) * TX + (x0 + dx);
            consume(bb + (unsigned long long)i, t, nn, produce(t, nn));
        }
    }
}

__global__ void __launch_bounds__(256)
    k_preprocess(int N, const float2 *__restrict__ mu, const float *__restrict__ chol, const float *__restrict__ rgb,
                 const float *__restrict__ opacity, float cutoff, int W, int H, int TX, int TY, int T,
                 Rec *__restrict__ rec,
                 short4 *__restrict__ rect, int *__restrict__ tile_count, int *__restrict__ pair_rank,
                 unsigned *__restrict__ pair_base, long long cap, DeviceState *st) {
    const int n = blockIdx.x * blockDim.x + threadIdx.x;
    const int lane = threadIdx.x & 31;
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
    // pair slots, Gaussian-major: rectangles of up to SMALL_RECT tiles own the fixed slots
    // [n * SMALL_RECT, ...); larger ones claim a range of the overflow region with one atomic
    const int w = r.z - r.x + 1, h = r.w - r.y + 1;
    const unsigned cnt = (w > 0 && h > 0) ? (unsigned)(w * h) : 0u;
    unsigned tot = cnt;
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) tot += __shfl_xor_sync(0xffffffffu, tot, d);
    if (lane == 0 && tot > 0) atomicAdd(&st->pair_cursor, (unsigned long long)tot);  // exact P (a RED)
    const unsigned long long small_region = (unsigned long long)N * SMALL_RECT;
    unsigned long long base = (unsigned long long)n * SMALL_RECT;
    if (cnt > SMALL_RECT) {
        const unsigned long long o = atomicAdd(&st->big_cursor, (unsigned long long)cnt);
        base = small_region + o;
        pair_base[n] = (unsigned)(o < 0xffffffffull ? o : 0xffffffffull);
    }
    const unsigned long long ucap = small_region + (unsigned long long)cap;  // overflow fits whenever P <= cap
    // BIN_COPIES private copies of the per-tile counters (one per CTA residue) keep the
    // same-address atomic chains of crowded tiles short
    int *my_count = tile_count + (size_t)(blockIdx.x % BIN_COPIES) * T;
    for_each_pair(
        r, n, base, TX, [&](int t, int) { return atomicAdd(my_count + t, 1); },
        [&](unsigned long long slot, int, int, int rank) {
            if (slot < ucap) pair_rank[slot] = rank;
        });
}

// Tile classes for the forward launch order (longest lists first, so that no long tile starts
// late and the kernel has no tail): class 3 >= 256 entries, 2 >= 96, 1 >= 32, 0 the rest.
__device__ __forceinline__ int tile_class(int n) { return n >= 256 ? 3 : (n >= 96 ? 2 : (n >= 32 ? 1 : 0)); }

__device__ __forceinline__ unsigned long long warp_incl_scan_u64(unsigned long long v, int lane) {
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        unsigned long long o = __shfl_up_sync(0xffffffffu, v, d);
        if (lane >= d) v += o;
    }
    return v;
}

// Multi-CTA scan over the tiles, one tile per thread, 256 tiles per CTA, in one pass: every CTA
// reduces its tiles, publishes the packed aggregate with an epoch-stamped flag, and sums the
// aggregates of all CTAs before it (a warp polls 32 predecessors at a time).  CTAs are
// dispatched in blockIdx order, so every predecessor is running or done: no deadlock.
// Two packed 64-bit words: (list entries | backward items << 32) and the three class counters
// (21 bits each; T < 2^21 or the order is the identity).  Class c tiles are appended to their
// own order list; the forward kernel walks the lists from class 3 down.
constexpr int SCAN_THREADS = 256;

__device__ __forceinline__ unsigned long long ld_volatile_u64(const unsigned long long *p) {
    unsigned long long v;
    asm volatile("ld.volatile.global.u64 %0, [%1];" : "=l"(v) : "l"(p));
    return v;
}

__global__ void __launch_bounds__(SCAN_THREADS)
    k_scan_tiles(int T, int *__restrict__ tile_count, int *__restrict__ range, int *__restrict__ copy_base,
                 int *__restrict__ item_off, int *__restrict__ tile_order, unsigned long long *scan_agg,
                 unsigned epoch, long long cap, DeviceState *st) {
    __shared__ unsigned long long s_w1[SCAN_THREADS / 32], s_w2[SCAN_THREADS / 32];
    __shared__ unsigned long long s_pre1, s_pre2;
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const int b = blockIdx.x, nb = gridDim.x;
    const int e = b * SCAN_THREADS + tid;
    const bool ordered = T < (1 << 21);
    int cnt[BIN_COPIES];
    int n = 0;
#pragma unroll
    for (int c = 0; c < BIN_COPIES; ++c) {
        cnt[c] = e < T ? tile_count[(size_t)c * T + e] : 0;
        n += cnt[c];
    }
    const int ni = (n + BWD_CHUNK - 1) / BWD_CHUNK;
    const int cl = tile_class(n);
    const unsigned long long v1 = ((unsigned long long)(unsigned)ni << 32) | (unsigned)n;
    const unsigned long long v2 = (cl == 0 || !ordered) ? 0ull : (1ull << (21 * (cl - 1)));
    const unsigned long long x1 = warp_incl_scan_u64(v1, lane), x2 = warp_incl_scan_u64(v2, lane);
    if (lane == 31) {
        s_w1[wid] = x1;
        s_w2[wid] = x2;
    }
    __syncthreads();
    if (wid == 0) {
        // block aggregate -> global, stamped with this binning's epoch
        const unsigned long long a1 = lane < SCAN_THREADS / 32 ? s_w1[lane] : 0ull;
        const unsigned long long a2 = lane < SCAN_THREADS / 32 ? s_w2[lane] : 0ull;
        const unsigned long long i1 = warp_incl_scan_u64(a1, lane), i2 = warp_incl_scan_u64(a2, lane);
        if (lane < SCAN_THREADS / 32) {
            s_w1[lane] = i1 - a1;  // exclusive over the warps
            s_w2[lane] = i2 - a2;
        }
        const unsigned long long tot1 = __shfl_sync(0xffffffffu, i1, 31), tot2 = __shfl_sync(0xffffffffu, i2, 31);
        if (lane == 0) {
            scan_agg[3 * b] = tot1;
            scan_agg[3 * b + 1] = tot2;
            __threadfence();
            atomicExch(&scan_agg[3 * b + 2], (unsigned long long)epoch);
        }
        // sum of the aggregates of CTAs 0..b-1
        unsigned long long p1 = 0ull, p2 = 0ull;
        for (int j0 = b - 1; j0 >= 0; j0 -= 32) {
            const int j = j0 - lane;
            if (j >= 0) {
                while (ld_volatile_u64(&scan_agg[3 * j + 2]) != (unsigned long long)epoch) {
                }
                __threadfence();
                p1 += ld_volatile_u64(&scan_agg[3 * j]);
                p2 += ld_volatile_u64(&scan_agg[3 * j + 1]);
            }
        }
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) {
            p1 += __shfl_xor_sync(0xffffffffu, p1, d);
            p2 += __shfl_xor_sync(0xffffffffu, p2, d);
        }
        if (lane == 0) {
            s_pre1 = p1;
            s_pre2 = p2;
            if (b == nb - 1) {  // the last CTA knows the totals
                const unsigned long long t1 = p1 + tot1, t2 = p2 + tot2;
                const unsigned long long P = st->pair_cursor;  // exact even when the packed low word wrapped
                range[T] = (int)(unsigned)(t1 & 0xffffffffull);
                item_off[T] = (int)(t1 >> 32);
                st->n_pairs = P > 0x7fffffffull ? 0x7fffffff : (int)P;
                st->n_items = (int)(t1 >> 32);
                st->n_class[1] = (int)(t2 & 0x1fffffull);
                st->n_class[2] = (int)((t2 >> 21) & 0x1fffffull);
                st->n_class[3] = (int)((t2 >> 42) & 0x1fffffull);
                st->pair_cursor = 0ull;
                st->big_cursor = 0ull;
                st->item_cursor = 0u;
                if (P > (unsigned long long)cap) atomicOr(&st->flags, FLAG_CAPACITY);
            }
        }
    }
    __syncthreads();
    if (e >= T) return;
    const unsigned long long e1 = s_pre1 + s_w1[wid] + x1 - v1, e2 = s_pre2 + s_w2[wid] + x2 - v2;  // exclusive
    int run = (int)(unsigned)(e1 & 0xffffffffull);
    range[e] = run;
    item_off[e] = (int)(e1 >> 32);
#pragma unroll
    for (int c = 0; c < BIN_COPIES; ++c) {
        tile_count[(size_t)c * T + e] = 0;  // ready for the next binning
        copy_base[(size_t)c * T + e] = run;
        run += cnt[c];
    }
    // per-class order lists: class c occupies tile_order[c*T ...)
    const unsigned p1 = (unsigned)(e2 & 0x1fffffull), p2 = (unsigned)((e2 >> 21) & 0x1fffffull),
                   p3 = (unsigned)((e2 >> 42) & 0x1fffffull);
    if (ordered) {
        const unsigned pos = cl == 3 ? p3 : (cl == 2 ? p2 : (cl == 1 ? p1 : (unsigned)e - p1 - p2 - p3));
        tile_order[(size_t)cl * T + pos] = e;
    } else {
        tile_order[e] = e;  // class 0 holds every tile; n_class[1..3] are zero because v2 is masked below
    }
}

__global__ void __launch_bounds__(256) k_fill(int N, const short4 *__restrict__ rect, int TX, int T,
                                              const int *__restrict__ copy_base, const int *__restrict__ pair_rank,
                                              const unsigned *__restrict__ pair_base, int *__restrict__ list,
                                              long long cap, const DeviceState *__restrict__ st) {
    if ((long long)st->n_pairs > cap) return;  // capacity exceeded: nothing downstream runs
    const int n = blockIdx.x * blockDim.x + threadIdx.x;
    const short4 r = n < N ? rect[n] : make_short4(0, 0, -1, -1);
    unsigned long long base = (unsigned long long)n * SMALL_RECT;
    if (r.z >= r.x && r.w >= r.y && (r.z - r.x + 1) * (r.w - r.y + 1) > SMALL_RECT)
        base = (unsigned long long)N * SMALL_RECT + pair_base[n];
    const int *my_base = copy_base + (size_t)(blockIdx.x % BIN_COPIES) * T;  // same CTA shape as k_preprocess
    for_each_pair(
        r, n, base, TX, [&](int t, int) { return my_base[t]; },
        [&](unsigned long long slot, int, int g, int start) { list[start + pair_rank[slot]] = g; });
}

// The standalone per-tile sort (paths that do not run the forward kernel, which otherwise sorts
// its own tile on entry): one CTA of SORT_CTA_THREADS per tile, see cta_sort_tile().
__global__ void __launch_bounds__(SORT_CTA_THREADS)
    k_sort_tiles(const int *__restrict__ range, int *list, const int *__restrict__ item_off, int2 *__restrict__ items,
                 long long cap, const DeviceState *__restrict__ st) {
    if ((long long)st->n_pairs > cap) return;
    const int t = blockIdx.x;
    const int start = range[t], n = range[t + 1] - start;
    cta_sort_tile(list + start, n, threadIdx.x);
    emit_items(t, n, item_off, items, threadIdx.x);
}

int launch_binning(gs_ctx *c, const gs_params &p, cudaStream_t s, bool sort, cudaEvent_t *ev) {
    int N = p.n;
    int blocks = ceil_div(N, 256);
    if (ev) cudaEventRecord(ev[0], s);
    k_preprocess<<<blocks, 256, 0, s>>>(N, reinterpret_cast<const float2 *>(p.mu), p.chol, p.rgb, p.opacity,
                                        c->cfg.cutoff, c->cfg.width, c->cfg.height, c->TX, c->TY, c->T, c->rec,
                                        c->rect, c->tile_count, c->pair_rank,
                                        reinterpret_cast<unsigned *>(c->pair_base), c->cap_pairs, c->dstate);
    if (ev) cudaEventRecord(ev[1], s);
    k_scan_tiles<<<ceil_div(c->T, SCAN_THREADS), SCAN_THREADS, 0, s>>>(c->T, c->tile_count, c->range, c->copy_base,
                                                                       c->item_off, c->tile_order, c->scan_agg,
                                                                       ++c->scan_epoch, c->cap_pairs, c->dstate);
    if (ev) cudaEventRecord(ev[2], s);
    k_fill<<<blocks, 256, 0, s>>>(N, c->rect, c->TX, c->T, c->copy_base, c->pair_rank,
                                  reinterpret_cast<const unsigned *>(c->pair_base), c->list, c->cap_pairs, c->dstate);
    if (ev) cudaEventRecord(ev[3], s);
    if (sort)
        k_sort_tiles<<<c->T, SORT_CTA_THREADS, 0, s>>>(c->range, c->list, c->item_off, c->items, c->cap_pairs,
                                                       c->dstate);
    c->last_n = N;
    GS_CUDA_TRY(cudaGetLastError());
    return GS_OK;
}

}  // namespace gs2d
