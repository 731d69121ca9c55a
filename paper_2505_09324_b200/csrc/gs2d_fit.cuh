// gs2d_fit.cuh -- the fit kernel's plumbing (gs2d_fit.cu): the PTX wrappers for mbarriers and bulk / tensor copies,
// the kernel arguments and tile geometry.  (A tensor-core formulation of the same kernel shared this header in
// round 2; it lost 175 us to 97 us and was retired in round 3 -- DESIGN.md §9b keeps the account.)
#pragma once
#include <cuda.h>  // CUtensorMap (types only: the encoder is fetched through the runtime, no -lcuda)

#include "gs2d_internal.cuh"
#include "gs2d_sort.cuh"

namespace gs2d {

// ---- PTX: mbarrier + bulk copies ------------------------------------------------------------
__device__ __forceinline__ unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long *bar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long *bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long *bar, unsigned parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(smem_u32(bar)),
        "r"(parity)
        : "memory");
}
// global -> shared bulk copy (16-byte aligned, size a multiple of 16), completes on `bar`
__device__ __forceinline__ void bulk_g2s(void *dst, const void *src, unsigned bytes, unsigned long long *bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     smem_u32(dst)),
                 "l"(src), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}

// one 48-float x 16-row box of the [H][3W] image at (column element c0, row c1) -> shared memory;
// out-of-frame elements arrive as zeros, the barrier always receives the full 3072 bytes
__device__ __forceinline__ void tma_tile_g2s(void *dst, const CUtensorMap *map, int c0, int c1,
                                             unsigned long long *bar) {
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];" ::"r"(
            smem_u32(dst)),
        "l"(map), "r"(c0), "r"(c1), "r"(smem_u32(bar))
        : "memory");
}

// 16 bytes global -> shared, asynchronous (LDGSTS); completion through cp_async_arrive on an mbarrier
__device__ __forceinline__ void cp_async16(void *smem_dst, const void *gsrc) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem_u32(smem_dst)), "l"(gsrc) : "memory");
}
// one arrival on `bar` (counted in its initial count) once all earlier cp.async of this thread have landed
__device__ __forceinline__ void cp_async_arrive(unsigned long long *bar) {
    asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}

__device__ __forceinline__ float fit_ex2_neg(float p) {  // 2^(-p), MUFU.EX2
    float w;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(w) : "f"(-p));
    return w;
}

struct FitArgs {
    TileArgs ta;
    const int *order_cur;
    int *order_next;
    int ord_cur, ord_next;
    const Rec *rec;          // [N] records, gathered by id
    const int *bucket;       // [T * tile_cap] their Gaussian ids
    const float *image;  // target frame or dL/dimage, [H,W,3]
    int W, H, TX, T;
    unsigned long long tx_magic;  // ceil(2^40 / TX): t / TX = (t * tx_magic) >> 40 for t < 2^26, TX < 2^15
    int tma_rows;        // the image has a tensor map (W % 4 == 0, 16-byte aligned base): tiles by TMA
    float g_scale;       // 2 / (3 W H); with an ROI 2 / (3 |M|)
    long long team_small_pairs;  // launches with fewer pairs fit lists of >= 32 entries as teams (k_fit_tiles)
    int roi_on;          // c-16: target values outside the ROI arrive as NaN and carry no loss
    int iter;
    float *acc;          // [N,8] gradient moments
    const int4 *pair_info;   // deterministic mode (else null): per Gaussian (first slot, x0 | y0 << 16, width, pairs)
    float *pair_mom;         // ... and the [P,8] moment slots of the (tile, Gaussian) pairs
    TileStats *tile_stats;
};

// Geometry of a tile seen by one lane.
struct TileGeo {
    int t, tx, ty;
    int rows;            // valid rows of the tile
    float px, py0;       // this lane's column centre, centre of the tile's first row
};
__device__ __forceinline__ TileGeo tile_geo(const FitArgs &a, int t, int lane) {
    TileGeo g;
    g.t = t;
    g.ty = (int)(((unsigned long long)(unsigned)t * a.tx_magic) >> 40);
    g.tx = t - g.ty * a.TX;
    g.rows = min(TILE, a.H - g.ty * TILE);
    g.px = (float)(g.tx * TILE + (lane & 15)) + 0.5f;
    g.py0 = (float)(g.ty * TILE) + 0.5f;
    return g;
}

constexpr unsigned ROWS_BYTES = TILE_PX * 3 * sizeof(float);

}  // namespace gs2d
