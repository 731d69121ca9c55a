// gs2d_bin.cuh -- binning of ONE Gaussian into the per-tile buckets (SURVEY.md §8 rows
// a1-a3; DESIGN.md §3 c-2, §5 "binning").  Shared by the standalone k_bin (gs2d_bin.cu) and
// by the fused Adam kernel (gs2d_optim.cu), which bins the parameters it has just updated
// so that the next iteration starts at its forward pass.
#pragma once
#include "gs2d_internal.cuh"

namespace gs2d {

// sqrt(0.5 * log2(e)) : folds the 1/2 of sigma and the change of base into the record
constexpr float KAPPA = 0.84932180028801904f;
constexpr int SMALL_RECT = 32;  // rectangles up to this many tiles are walked by their own thread
constexpr int RECT_BATCH = 8;   // independent atomics in flight per thread

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

// One arrival of Gaussian `gid` in tile `t`: the counting atomic's return value is the slot; the
// slot receives the id (canonical lists, P-frame selection) and the 48-byte bucket record (fit kernel).
__device__ __forceinline__ int bucket_claim(const BinArgs &a, int t) {
    return atomicAdd(a.tile_count + (size_t)a.slot * (a.TX * a.TY) + t, 1);
}
__device__ __forceinline__ void bucket_store(const BinArgs &a, int t, int slot, int gid, const float4 &r0,
                                             const float4 &r1, const float4 &r2) {
    if (slot < a.tile_cap) {
        const size_t e = (size_t)t * a.tile_cap + slot;
        a.bucket[e] = gid;
        if (a.bucket_rec) {  // only binnings made for the fit kernel carry the records
            float4 *dst = reinterpret_cast<float4 *>(a.bucket_rec + e);
            dst[0] = r0;
            dst[1] = r1;
            dst[2] = r2;
        }
    } else {
        a.st->tile_ovf[a.slot] = 1;  // every writer stores the same value
    }
}

// Record + tile rectangle + bucket arrivals of Gaussian `gid` (valid == false: an idle lane).
// ALL 32 lanes of the warp must call this together.  Rectangles of up to SMALL_RECT tiles are
// walked by their own lane in batches of RECT_BATCH, so that a batch of independent atomics is
// in flight before the first result is consumed; larger rectangles are walked by the whole
// warp, one rectangle at a time, so that one fat Gaussian does not serialise thousands of
// atomics on one lane.
__device__ __forceinline__ void bin_gaussian(const BinArgs &a, bool valid, int gid, float mux, float muy, float l1,
                                             float l2, float l3, float cr, float cg, float cb, float o) {
    const unsigned full = 0xffffffffu;
    const int lane = threadIdx.x & 31;
    int x0 = 0, y0 = 0, x1 = -1, y1 = -1;
    float4 r0 = make_float4(0.f, 0.f, 0.f, 0.f), r1 = r0, r2 = r0;
    if (valid) {
        tile_rect(mux, muy, l1, l2, l3, a.cutoff, a.W, a.H, a.TX, a.TY, x0, y0, x1, y1);
        const float i1 = KAPPA / l1, i3 = KAPPA / l3;
        r0 = make_float4(mux, muy, i1, -l2 * i1 / l3);
        r1 = make_float4(i3, o * cr, o * cg, o * cb);
        const float i3sq = i3 * i3;
        r2 = make_float4(exp2f(-2.0f * i3sq), -2.0f * i3, -i3sq, __int_as_float(gid));
        float4 *dst = reinterpret_cast<float4 *>(a.rec + gid);
        dst[0] = r0;
        dst[1] = r1;
    }
    const int w = x1 - x0 + 1, h = y1 - y0 + 1;
    const int cnt = (w > 0 && h > 0) ? w * h : 0;
    // exact P, one RED per warp
    unsigned tot = (unsigned)cnt;
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) tot += __shfl_xor_sync(full, tot, d);
    if (lane == 0 && tot > 0) atomicAdd(&a.st->pair_total[a.slot], (unsigned long long)tot);

    if (cnt > 0 && cnt <= SMALL_RECT) {
        int tx = x0, ty = y0;
        for (int i0 = 0; i0 < cnt; i0 += RECT_BATCH) {
            int slot[RECT_BATCH], til[RECT_BATCH];
#pragma unroll
            for (int j = 0; j < RECT_BATCH; ++j) {
                til[j] = ty * a.TX + tx;
                if (i0 + j < cnt) slot[j] = bucket_claim(a, til[j]);
                if (++tx > x1) {
                    tx = x0;
                    ++ty;
                }
            }
#pragma unroll
            for (int j = 0; j < RECT_BATCH; ++j)
                if (i0 + j < cnt) bucket_store(a, til[j], slot[j], gid, r0, r1, r2);
        }
    }
    unsigned big = __ballot_sync(full, cnt > SMALL_RECT);
    while (big) {
        const int src = __ffs(big) - 1;
        big &= big - 1;
        const int bx0 = __shfl_sync(full, x0, src), by0 = __shfl_sync(full, y0, src);
        const int ww = __shfl_sync(full, w, src), tt = __shfl_sync(full, cnt, src);
        const int g = __shfl_sync(full, gid, src);
        float4 s0, s1, s2;
        s0.x = __shfl_sync(full, r0.x, src), s0.y = __shfl_sync(full, r0.y, src);
        s0.z = __shfl_sync(full, r0.z, src), s0.w = __shfl_sync(full, r0.w, src);
        s1.x = __shfl_sync(full, r1.x, src), s1.y = __shfl_sync(full, r1.y, src);
        s1.z = __shfl_sync(full, r1.z, src), s1.w = __shfl_sync(full, r1.w, src);
        s2.x = __shfl_sync(full, r2.x, src), s2.y = __shfl_sync(full, r2.y, src);
        s2.z = __shfl_sync(full, r2.z, src), s2.w = __shfl_sync(full, r2.w, src);
        for (int i = lane; i < tt; i += 32) {
            const int dy = i / ww, dx = i - dy * ww;
            const int t = (by0 + dy) * a.TX + (bx0 + dx);
            bucket_store(a, t, bucket_claim(a, t), g, s0, s1, s2);
        }
    }
}

}  // namespace gs2d
