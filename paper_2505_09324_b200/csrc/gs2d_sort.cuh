// gs2d_sort.cuh -- per-tile sort of a list segment by Gaussian id (the canonical order of
// DESIGN.md §3 c-2) and the bookkeeping every consumer of a binning does per tile.  Used by the
// render kernel (gs2d_raster.cu), the fit kernel (gs2d_fit.cu) and k_sort_tiles (gs2d_bin.cu).
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

// Consumer side of a binning, for tile t: reads the tile's arrival count and tells whether the
// binning exceeded a capacity (then nothing downstream may write).  Any thread may call it.
__device__ __forceinline__ int tile_count_of(const TileArgs &a, int T, int t) {
    const int n_raw = a.tile_count[(size_t)a.slot * T + t];
    const bool bad = a.st->pair_total[a.slot] > (unsigned long long)a.cap_pairs || a.st->tile_ovf[a.slot] != 0;
    return bad ? -1 : n_raw;
}

// Number of valid entries of the spill list of the binning a consumer works on.
__device__ __forceinline__ int spill_size(const TileArgs &a) {
    return (int)min(a.st->spill_count[a.slot], (unsigned)a.spill_cap);
}

// Ids of tile t among spill[start, S): collected by one WARP into out[0, max_out) in list order (the order is
// the arrival order of the binning).  Scans 32 entries per step, stops when fewer than 32 free slots remain or
// the list ends; `start` is advanced past what was scanned.  Returns the number collected.
__device__ __forceinline__ int spill_collect(const int2 *__restrict__ spill, int S, int t, int &start, int *out,
                                             int max_out, int lane) {
    const unsigned lt = (1u << lane) - 1u;
    int cnt = 0;
    while (start < S && cnt + 32 <= max_out) {
        const int e = start + lane;
        int2 v = make_int2(-1, -1);
        if (e < S) v = spill[e];
        const bool hit = v.x == t;
        const unsigned m = __ballot_sync(0xffffffffu, hit);
        if (hit) out[cnt + __popc(m & lt)] = v.y;
        cnt += __popc(m);
        start += 32;
    }
    __syncwarp();
    return cnt;
}

// Bookkeeping of the consumer of tile t, ONE thread per tile: publishes the list length in tile_n,
// zeroes the tile's counter of the OTHER epoch parity (the one the next binning will count into;
// nobody reads it now), and -- the thread that owns tile 0 -- resets the other epoch's counters
// and latches the capacity flag.
__device__ __forceinline__ void tile_publish(const TileArgs &a, int T, int t, int n) {
    a.tile_count[(size_t)(a.slot ^ 1) * T + t] = 0;
    a.tile_n[t] = n < 0 ? 0 : n;
    if (t == 0) {
        a.st->pair_total[a.slot ^ 1] = 0ull;
        a.st->tile_ovf[a.slot ^ 1] = 0;
        a.st->spill_count[a.slot ^ 1] = 0u;
        if (n < 0) atomicOr(&a.st->flags, FLAG_CAPACITY);
    }
}

// Files tile t under its class for the NEXT consumer launch (ONE thread per tile); the owner of
// tile 0 also resets the idle third of the triple-buffered launch state.  `pos` is the value of
// atomicAdd(&st->n_class[ord_next][tile_class(n)], 1), which the caller may have issued long
// before (its latency is then off the critical path).
__device__ __forceinline__ void tile_file_at(DeviceState *st, int *order_next, int T, int ord_cur, int ord_next,
                                             int t, int n, int pos) {
    order_next[(size_t)tile_class(n < 0 ? 0 : n) * T + pos] = t;
    if (t == 0) {
        const int o3 = 3 - ord_cur - ord_next;
#pragma unroll
        for (int k = 0; k < NCLS; ++k) st->n_class[o3][k] = 0;
        st->cursor_team[o3] = 0u;
        st->cursor_warp[o3] = 0u;
    }
}
__device__ __forceinline__ void tile_file(DeviceState *st, int *order_next, int T, int ord_cur, int ord_next, int t,
                                          int n) {
    const int pos = atomicAdd(&st->n_class[ord_next][tile_class(n < 0 ? 0 : n)], 1);
    tile_file_at(st, order_next, T, ord_cur, ord_next, t, n, pos);
}

// Position q of the launch order -> tile id: classes are walked longest lists first.  cnt[NCLS] are
// the class sizes of the launch (shared memory or registers).
__device__ __forceinline__ int tile_of_position(const int *order_cur, int T, const int *cnt, int q) {
    int cls = NCLS - 1;
#pragma unroll
    for (int k = NCLS - 1; k > 0; --k) {  // branch-free: values stay on the uniform datapath
        const int c = cnt[k];
        const bool go = cls == k && q >= c;
        q = go ? q - c : q;
        cls = go ? k - 1 : cls;
    }
    return order_cur[(size_t)cls * T + q];
}

}  // namespace gs2d
