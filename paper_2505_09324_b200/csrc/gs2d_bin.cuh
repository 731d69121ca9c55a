// gs2d_bin.cuh -- binning of ONE Gaussian into the per-tile buckets (SURVEY.md §8 rows
// a1-a3; DESIGN.md §3 c-2, §5 "binning").  Shared by the standalone k_bin (gs2d_bin.cu) and
// by the fused Adam kernel (gs2d_optim.cu), which bins the parameters it has just updated
// so that the next iteration starts at its forward pass.
#pragma once
#include "gs2d_internal.cuh"

namespace gs2d {

// sqrt(0.5 * log2(e)) : folds the 1/2 of sigma and the change of base into the record
constexpr float KAPPA = 0.84932180028801904f;

// Tile rectangle of one Gaussian: DESIGN.md §3 c-2.  Every operation is binary32,
// round-to-nearest, one rounding each; the *_rn intrinsics are never contracted into FMAs.
// Returns false (and an empty rectangle) for culled Gaussians.
__device__ __forceinline__ bool tile_rect(float mux, float muy, float l1, float l2, float l3, float k, int W, int H,
                                          int TX, int TY, int &x0, int &y0, int &x1, int &y1) {
    x0 = y0 = 0;
    x1 = y1 = -1;
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
    x0 = (int)fx0;
    y0 = (int)fy0;
    x1 = (int)fx1;
    y1 = (int)fy1;
    return true;
}

// One arrival of Gaussian `gid` in tile `t`: the counting atomic's return value is the slot in the tile's
// bucket; arrivals beyond the bucket go to the shared spill list.
__device__ __forceinline__ int bucket_claim(const BinArgs &a, int t) {
    return atomicAdd(a.tile_count + (size_t)a.slot * (a.TX * a.TY) + t, 1);
}
__device__ __forceinline__ void bucket_store(const BinArgs &a, int t, int slot, int gid) {
    if (slot < a.tile_cap) {
        a.bucket[(size_t)t * a.tile_cap + slot] = gid;
    } else {
        const unsigned ss = atomicAdd(&a.st->spill_count[a.slot], 1u);
        if (ss < (unsigned)a.spill_cap) a.spill[ss] = make_int2(t, gid);
        else a.st->tile_ovf[a.slot] = 1;  // every writer stores the same value
    }
}

// Shared memory of a CTA that bins THREADS Gaussians together.
template <int THREADS>
struct BinSmem {
    int gid[THREADS], x0[THREADS], y0[THREADS], w[THREADS];
    int off[THREADS + 1];          // exclusive prefix of the rectangle sizes
    int wsum[THREADS / 32];
    int base;                      // deterministic mode: slot of the CTA's first pair
};

constexpr int PAIR_BATCH = 6;  // independent counting atomics in flight per thread

// Records (rec[gid], once per Gaussian) + tile rectangles + bucket arrivals of THREADS Gaussians, one per thread (valid == false:
// an idle thread).  ALL threads of the CTA must call this together.  The (tile, Gaussian) pairs of
// the CTA are numbered by a prefix sum over the rectangle sizes and dealt out to the threads
// round-robin, so that every thread has the same number of arrivals whatever the rectangles are
// (one fat Gaussian is walked by the whole CTA), and a batch of PAIR_BATCH independent counting
// atomics is in flight per thread before the first slot is consumed.
template <int THREADS>
__device__ __forceinline__ void bin_cta(const BinArgs &a, BinSmem<THREADS> &sm, bool valid, int gid, float mux,
                                        float muy, float l1, float l2, float l3, float cr, float cg, float cb,
                                        float o) {
    const unsigned full = 0xffffffffu;
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    int x0 = 0, y0 = 0, x1 = -1, y1 = -1;
    float4 r0 = make_float4(0.f, 0.f, 0.f, 0.f), r1 = r0;
    if (a.q.on) {  // QAT: the render sees the quantised parameters (straight-through in the backward pass)
        mux = fake_quant(a.q, 0, mux), muy = fake_quant(a.q, 1, muy);
        l1 = fake_quant(a.q, 2, l1), l2 = fake_quant(a.q, 3, l2), l3 = fake_quant(a.q, 4, l3);
        cr = fake_quant(a.q, 5, cr), cg = fake_quant(a.q, 6, cg), cb = fake_quant(a.q, 7, cb);
        o = fake_quant(a.q, 8, o);
    }
    if (valid) {
        // a selective binning lists only the active (mode 1) or only the frozen (mode 2) Gaussians
        if (a.mode == 0 || (a.active[gid] != 0) == (a.mode == 1))
            tile_rect(mux, muy, l1, l2, l3, a.cutoff, a.W, a.H, a.TX, a.TY, x0, y0, x1, y1);
        const float i1 = KAPPA / l1, i3 = KAPPA / l3;
        r0 = make_float4(mux, muy, i1, -l2 * i1 / l3);
        r1 = make_float4(i3, o * cr, o * cg, o * cb);
        float4 *dst = reinterpret_cast<float4 *>(a.rec + gid);
        dst[0] = r0;
        dst[1] = r1;
    }
    const int w = x1 - x0 + 1, h = y1 - y0 + 1;
    const int cnt = (w > 0 && h > 0) ? w * h : 0;
    sm.gid[tid] = gid;
    sm.x0[tid] = x0;
    sm.y0[tid] = y0;
    sm.w[tid] = w > 0 ? w : 1;
    // inclusive prefix sum of cnt over the CTA
    int incl = cnt;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const int v = __shfl_up_sync(full, incl, d);
        if (lane >= d) incl += v;
    }
    if (lane == 31) sm.wsum[wid] = incl;
    __syncthreads();
    int before = 0;
#pragma unroll
    for (int k = 0; k < THREADS / 32; ++k) before += k < wid ? sm.wsum[k] : 0;
    sm.off[tid + 1] = before + incl;
    if (tid == 0) sm.off[0] = 0;
    __syncthreads();
    const int total = sm.off[THREADS];
    // exact P; the value before the addition is the slot of the CTA's first pair (any order of the CTAs will do:
    // a Gaussian's slots are contiguous and in tile order whatever the base)
    unsigned long long cta_base = 0ull;
    if (tid == 0 && total > 0) cta_base = atomicAdd(&a.st->pair_total[a.slot], (unsigned long long)total);

    for (int base = 0; base < total; base += THREADS * PAIR_BATCH) {
        int til[PAIR_BATCH], slot[PAIR_BATCH], own[PAIR_BATCH];
#pragma unroll
        for (int j = 0; j < PAIR_BATCH; ++j) {
            const int p = base + j * THREADS + tid;
            own[j] = -1;
            if (p < total) {
                int lo = 0, hi = THREADS;  // the Gaussian g with off[g] <= p < off[g + 1]
#pragma unroll
                for (int it = THREADS; it > 1; it >>= 1) {
                    const int mid = (lo + hi) >> 1;
                    if (sm.off[mid] <= p) lo = mid;
                    else hi = mid;
                }
                const int i = p - sm.off[lo], ww = sm.w[lo];
                const int dy = i / ww, dx = i - dy * ww;
                own[j] = lo;
                til[j] = (sm.y0[lo] + dy) * a.TX + sm.x0[lo] + dx;
                slot[j] = bucket_claim(a, til[j]);
            }
        }
#pragma unroll
        for (int j = 0; j < PAIR_BATCH; ++j)
            if (own[j] >= 0) bucket_store(a, til[j], slot[j], sm.gid[own[j]]);
    }
    if (a.pair_info) {  // (uniform over the grid)
        if (tid == 0) sm.base = (int)min(cta_base, 0x7fffffffull);
        __syncthreads();
        if (valid) a.pair_info[gid] = make_int4(sm.base + sm.off[tid], x0 | (y0 << 16), w > 0 ? w : 1, cnt);
    }
}

}  // namespace gs2d
