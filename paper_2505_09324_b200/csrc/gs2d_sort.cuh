// gs2d_sort.cuh -- per-tile sort of a list segment by Gaussian id (the canonical order of
// DESIGN.md §3 c-2) and emission of the tile's backward work items.  Used on entry by the
// forward kernel (gs2d_raster.cu) and by the standalone k_sort_tiles (gs2d_bin.cu).
#pragma once
#include "gs2d_internal.cuh"

namespace gs2d {

constexpr int SORT_CTA_THREADS = 64;  // = the forward kernel's CTA
constexpr int SORT_REG_MAX = 512;     // longest segment sorted by one warp in registers

// Bitonic sorting network over KPL*32 keys held KPL per lane; logical element e = i*32 + lane
// (striped, so that loads and stores of a segment are coalesced).  Padding keys are INT_MAX.
template <int KPL>
__device__ __forceinline__ void warp_sort_segment(int *seg, int n, int lane) {
    int v[KPL];
#pragma unroll
    for (int i = 0; i < KPL; ++i) {
        const int e = i * 32 + lane;
        v[i] = e < n ? seg[e] : 0x7fffffff;
    }
#pragma unroll
    for (int k = 2; k <= KPL * 32; k <<= 1) {
#pragma unroll
        for (int j = k >> 1; j > 0; j >>= 1) {
            if (j >= 32) {  // both keys in this lane: registers i and i ^ (j/32)
                const int dj = j >> 5;
#pragma unroll
                for (int i = 0; i < KPL; ++i) {
                    const int p = i ^ dj;
                    if (p > i) {
                        const bool asc = (((i * 32) & k) == 0);
                        const int a = v[i], b = v[p];
                        const bool sw = asc ? (a > b) : (a < b);
                        v[i] = sw ? b : a;
                        v[p] = sw ? a : b;
                    }
                }
            } else {
#pragma unroll
                for (int i = 0; i < KPL; ++i) {
                    const int o = __shfl_xor_sync(0xffffffffu, v[i], j);
                    const bool asc = k < 32 ? ((lane & k) == 0) : (((i * 32) & k) == 0);
                    const bool keep_min = ((lane & j) == 0) == asc;
                    v[i] = keep_min ? min(v[i], o) : max(v[i], o);
                }
            }
        }
    }
#pragma unroll
    for (int i = 0; i < KPL; ++i) {
        const int e = i * 32 + lane;
        if (e < n) seg[e] = v[i];
    }
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


// Sort seg[0..n) ascending; all SORT_CTA_THREADS threads of the CTA must call it.  Segments of
// up to SORT_REG_MAX ids are sorted by warp 0 in registers; longer (degenerate) ones by the
// whole CTA in place in global memory.  Ends with a barrier: the sorted segment is visible to
// the CTA.
__device__ __forceinline__ void cta_sort_tile(int *seg, int n, int tid) {
    if (n > SORT_REG_MAX) {
        bitonic_all_up<SORT_CTA_THREADS>(seg, n, tid);
        return;  // bitonic_all_up ends with a barrier
    }
    if (n > 1 && tid < 32) {
        if (n <= 32) warp_sort_segment<1>(seg, n, tid);
        else if (n <= 64) warp_sort_segment<2>(seg, n, tid);
        else if (n <= 128) warp_sort_segment<4>(seg, n, tid);
        else if (n <= 256) warp_sort_segment<8>(seg, n, tid);
        else warp_sort_segment<16>(seg, n, tid);
    }
    __syncthreads();
}

// Consumer side of a binning, for tile t, called by all SORT_CTA_THREADS threads of the CTA:
// reads the tile's arrival count, publishes the list length in tile_n, zeroes the tile's counter
// of the OTHER epoch parity (the one the next binning will count into; nobody reads it now, so
// no barrier is needed), optionally sorts the bucket into the canonical order (ascending id) and
// reserves the tile's backward work items.  Returns the list length, or -1 when the binning
// exceeded a capacity (nothing downstream may write).  With sort == true it ends with a barrier
// (the sorted bucket is visible to the CTA); without, it has no barrier at all.
//   item_base (thread 0 only): first slot of the tile's items; write them with emit_items() --
//   late in the kernel, so that the atomic's latency is off the critical path.
__device__ __forceinline__ int tile_begin(const TileArgs &a, int T, int t, int tid, bool sort, int &item_base) {
    const int n_raw = a.tile_count[(size_t)a.slot * T + t];
    const bool bad = a.st->pair_total[a.slot] > (unsigned long long)a.cap_pairs || a.st->tile_ovf[a.slot] != 0;
    const int n = bad ? -1 : n_raw;
    item_base = 0;
    if (tid == 0) {
        a.tile_count[(size_t)(a.slot ^ 1) * T + t] = 0;
        a.tile_n[t] = n < 0 ? 0 : n;
        if (a.emit && n > 0) item_base = atomicAdd(&a.st->n_items[a.slot], (n + BWD_CHUNK - 1) / BWD_CHUNK);
        if (t == 0) {  // the other epoch's slots are idle now: reset them for the next binning
            a.st->pair_total[a.slot ^ 1] = 0ull;
            a.st->tile_ovf[a.slot ^ 1] = 0;
            a.st->n_items[a.slot ^ 1] = 0;
            a.st->item_cursor[a.slot ^ 1] = 0u;
            if (bad) atomicOr(&a.st->flags, FLAG_CAPACITY);
        }
    }
    if (n > 0 && sort) cta_sort_tile(a.bucket + (size_t)t * a.tile_cap, n, tid);
    return n;
}

// Backward work items of tile t: (t, k) for every chunk k of BWD_CHUNK list entries (thread 0).
__device__ __forceinline__ void emit_items(const TileArgs &a, int t, int n, int item_base) {
    const int ni = (n + BWD_CHUNK - 1) / BWD_CHUNK;
    for (int k = 0; k < ni; ++k) a.items[item_base + k] = make_int2(t, k);
}

}  // namespace gs2d
