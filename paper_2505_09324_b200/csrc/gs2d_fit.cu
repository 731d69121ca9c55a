// gs2d_fit.cu -- the fused fit kernel: forward rasterizer + L2 loss + backward pass of one fit
// iteration, per tile, in ONE persistent kernel (DESIGN.md §5 "fit").
//
// Summation blending (Eq. 2) has no transmittance chain, so the backward pass of a
// tile needs nothing from other tiles: dL/dC of its own 256 pixels is enough.  A tile is therefore
// fitted start to finish by one worker, and dL/dC never leaves the chip.
//
//   worker   = one WARP for tiles of fewer than FIT_CHUNK list entries, the whole CTA (4 warps,
//              the list split four ways) for longer lists (classes >= TEAM_CLASS).  A CTA first
//              drains the long tiles as a team, then its warps pull lighter tiles independently.
//   forward  : lane = column x 8 rows; the worker walks its list once; per Gaussian and lane the
//              whitened coordinates are set up once and each pixel costs 2 FMA + MUFU.EX2 + 3 FMA.
//   packing  : the per-pixel arithmetic of both passes runs on row PAIRS with the packed binary32
//              instructions of sm_100 (FFMA2 / FMUL2 / FADD2: two results per issue slot, each
//              rounded as the scalar instruction would): 39 issue slots per Gaussian and lane of 8
//              pixels forward (57 scalar), 190 per two Gaussians x 16 rows backward (250 scalar).
//   loss     : partial sums meet in shared memory; G = dL/dC = 2 (C - T) / (3 W H) goes straight
//              into registers in the backward layout (lane = column x 16 rows).
//   backward : half-warp per Gaussian; 8 gradient moments reduced over the 16 columns with a
//              transposing butterfly, then one vector of fp32 atomics per (tile, Gaussian).
//   staging  : the binning stores ids only (records live once per Gaussian, rec[N]).  A chunk of up to
//              FIT_CHUNK list entries is staged by the warp's lanes: each reads its ids from the tile's
//              bucket and gathers the 32-byte records by id with cp.async (gather_records); the
//              target tile is one TMA tensor copy.  All of it completes on ONE mbarrier per buffer
//              (32 cp.async arrivals + the tensor copy's transaction bytes).  A warp issues the
//              copies of its NEXT tile before the backward pass of the current one: no load
//              latency on the critical path.
#include <stdlib.h>

#include "gs2d_fit.cuh"

namespace gs2d {

constexpr int FIT_WARPS = 4;
constexpr int FIT_THREADS = FIT_WARPS * 32;

// ---- shared memory ----------------------------------------------------------------------------
struct __align__(128) WarpSmem {
    float4 rec[2][FIT_CHUNK * REC_F4];   // two buffers of records ...
    int ids[2][FIT_CHUNK];               // ... and of the Gaussian ids of the same list entries
    float tgt[TILE_PX * 3];              // target (FIT_LOSS) or dL/dC (FIT_GRAD) tile, HWC rows
    float cpart[TILE_PX * 3];            // team mode: this warp's partial image, lane-major float4
    unsigned long long bar[4];           // [0],[1]: list buffers (+ the tile's rows); [2]: team rows
};
struct __align__(16) CtaHdr {
    int t, n;
    int pad[2];
    int cnt[NCLS];  // class sizes of this launch
};
constexpr size_t FIT_SMEM = sizeof(WarpSmem) * FIT_WARPS + sizeof(CtaHdr);

// ---- staging ------------------------------------------------------------------------------------
// entries [e0, e0 + cnt) of the id buckets -> list buffer `buf`: every lane reads its entries' ids and gathers
// their records (rec[id], 32 bytes) with cp.async; all 32 lanes arrive on the buffer's barrier when their
// copies have landed, lane 0 once more with `extra` bytes expected (the tile's rows, issued by the caller
// right after): the barriers count 33 arrivals.  cnt <= FIT_CHUNK.
__device__ __forceinline__ void gather_records(const FitArgs &a, WarpSmem *sm, int buf, int cnt, unsigned extra, int lane) {
#pragma unroll
    for (int k = 0; k < FIT_CHUNK / 32; ++k) {
        const int e = lane + 32 * k;
        if (e < cnt) {
            const float4 *src = reinterpret_cast<const float4 *>(a.rec + sm->ids[buf][e]);
            cp_async16(&sm->rec[buf][REC_F4 * e], src);
            cp_async16(&sm->rec[buf][REC_F4 * e + 1], src + 1);
        }
    }
    cp_async_arrive(&sm->bar[buf]);
    if (lane == 0) mbar_expect_tx(&sm->bar[buf], extra);
}
__device__ __forceinline__ void issue_records(const FitArgs &a, WarpSmem *sm, int buf, size_t e0, int cnt,
                                              unsigned extra, int lane) {
    int gid[FIT_CHUNK / 32];
#pragma unroll
    for (int k = 0; k < FIT_CHUNK / 32; ++k) gid[k] = lane + 32 * k < cnt ? a.bucket[e0 + lane + 32 * k] : 0;
#pragma unroll
    for (int k = 0; k < FIT_CHUNK / 32; ++k)
        if (lane + 32 * k < cnt) sm->ids[buf][lane + 32 * k] = gid[k];
    gather_records(a, sm, buf, cnt, extra, lane);
}
// the tile's 16 rows of `image` -> dst (HWC rows of 48 floats): ONE tensor copy, lane 0 issues
__device__ __forceinline__ void issue_rows(const CUtensorMap *map, const TileGeo &g, float *dst,
                                           unsigned long long *bar, int lane) {
    if (lane == 0) tma_tile_g2s(dst, map, g.tx * (TILE * 3), g.ty * TILE, bar);
}
// fallback for frames whose rows cannot be bulk-copied: plain loads by the warp
__device__ __forceinline__ void load_rows_generic(const FitArgs &a, const TileGeo &g, float *dst, int lane) {
    for (int e = lane; e < TILE_PX * 3; e += 32) {
        const int r = e / (TILE * 3), c = e - r * (TILE * 3);
        const int gy = g.ty * TILE + r, gc = g.tx * TILE * 3 + c;
        if (gy < a.H && gc < a.W * 3) dst[e] = a.image[(size_t)gy * a.W * 3 + gc];
    }
}

__device__ __forceinline__ float2 ex2_neg2(float2 p) { return make_float2(fit_ex2_neg(p.x), fit_ex2_neg(p.y)); }

// ---- forward: `cnt` records of a shared-memory chunk, lane = column x 8 rows (4 row pairs) -------
__device__ __forceinline__ void fwd_chunk(const float4 *__restrict__ rec, int cnt, float px, float pyA,
                                          float2 (&C)[4][3]) {
#pragma unroll 2
    for (int j = 0; j < cnt; ++j) {
        const float4 lo = rec[REC_F4 * j], hi = rec[REC_F4 * j + 1];
        const float dx = px - lo.x, dy0 = pyA - lo.y;
        const float u = dx * lo.z;
        const float2 uu = dup2(u * u);
        const float2 v0 = dup2(fmaf(dx, lo.w, dy0 * hi.x));
        const float2 hx = dup2(hi.x), cr = dup2(hi.y), cg = dup2(hi.z), cb = dup2(hi.w);
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            const float2 v = __ffma2_rn(hx, c_rowpair[k], v0);
            const float2 w = ex2_neg2(__ffma2_rn(v, v, uu));
            C[k][0] = __ffma2_rn(w, cr, C[k][0]);
            C[k][1] = __ffma2_rn(w, cg, C[k][1]);
            C[k][2] = __ffma2_rn(w, cb, C[k][2]);
        }
    }
}

// ---- backward: `cnt` records of a shared-memory chunk --------------------------------------------
// With s = w * (c' . G) and the kappa-scaled whitened coordinates (u, v) of the record, a
// half-warp accumulates for one Gaussian, lane = tile column,
//   R_ch = sum_y w G_ch,   A1 = sum_y s v,   A2 = sum_y s v^2      (A0 = sum_y s = c' . R)
// and forms its column's share of the 8 moments
//   (R_r, R_g, R_b, Su = u A0, Sv = A1, Suu = u^2 A0, Suv = u A1, Svv = A2),
// which the butterfly sums over the 16 columns.  Pixels outside the frame carry G = 0.  The
// chain rule to (mu, l, rgb, o) is applied once per Gaussian afterwards (gs2d_optim.cu).
// G is held in row pairs, own rows first: pairs 0..3 = rows 8 hf + (2k, 2k + 1) of the tile, pairs 4..7 =
// rows 8 (1 - hf) + (2k, 2k + 1) (hf = lane >> 4), the layout make_G leaves it in; the order of the
// rows in the sums is free.
// DET: the 8 moments of a pair go to the pair's own slot (plain stores) instead of the Gaussian's accumulator
// (atomics): slot = first slot of the Gaussian + position of tile (tx, ty) in its rectangle, row-major.
template <bool DET>
__device__ __forceinline__ void bwd_chunk(const FitArgs &a, const float4 *__restrict__ rec, const int *__restrict__ ids,
                                          int cnt, float px, float py0, const float2 (&G)[TILE / 2][3], int tx, int ty,
                                          int lane) {
    float *__restrict__ acc = a.acc;
    const unsigned full = 0xffffffffu;
    const int half = lane >> 4;
    const float pyA = py0 + (float)(8 * half);  // centre of this lane's first own row
    const float stepB = half ? -8.0f : 8.0f;    // partner rows start 8 rows below / above
    for (int j0 = 0; j0 < cnt; j0 += 2) {
        const int j = j0 + half;
        const bool live = j < cnt;
        const int jj = live ? j : j0;  // the idle half-warp repeats its neighbour's entry and drops the result
        const float4 lo = rec[REC_F4 * jj], hi = rec[REC_F4 * jj + 1];
        const int gid = ids[jj];
        int4 info = make_int4(0, 0, 1, 0);
        if (DET) info = __ldg(a.pair_info + gid);  // (used after the row loop: the latency is hidden)
        const float dx = px - lo.x;
        const float u = dx * lo.z;
        const float uu = u * u;
        const float vA = fmaf(dx, lo.w, (pyA - lo.y) * hi.x);
        const float vB = fmaf(hi.x, stepB, vA);
        const float2 hx = dup2(hi.x), uu2 = dup2(uu), cr = dup2(hi.y), cg = dup2(hi.z), cb = dup2(hi.w);
        float2 Rr2 = dup2(0.f), Rg2 = Rr2, Rb2 = Rr2, A12 = Rr2, A22 = Rr2;
#pragma unroll
        for (int k = 0; k < TILE / 2; ++k) {  // row pairs: k < 4 own rows, k >= 4 the partner's
            const float2 v = __ffma2_rn(hx, c_rowpair[k & 3], dup2(k < 4 ? vA : vB));
            const float2 w = ex2_neg2(__ffma2_rn(v, v, uu2));
            const float2 q = __ffma2_rn(cb, G[k][2], __ffma2_rn(cg, G[k][1], __fmul2_rn(cr, G[k][0])));
            const float2 s = __fmul2_rn(w, q);
            Rr2 = __ffma2_rn(w, G[k][0], Rr2);
            Rg2 = __ffma2_rn(w, G[k][1], Rg2);
            Rb2 = __ffma2_rn(w, G[k][2], Rb2);
            const float2 sv = __fmul2_rn(s, v);
            A12 = __fadd2_rn(A12, sv);
            A22 = __ffma2_rn(sv, v, A22);
        }
        const float Rr = Rr2.x + Rr2.y, Rg = Rg2.x + Rg2.y, Rb = Rb2.x + Rb2.y;
        const float A1 = A12.x + A12.y, A2 = A22.x + A22.y;
        const float A0 = fmaf(hi.w, Rb, fmaf(hi.z, Rg, hi.y * Rr));
        // moments of this column: m0..m7 = Rr, Rg, Rb, Su, Sv, Suu, Suv, Svv
        const float m0 = Rr, m1 = Rg, m2 = Rb, m3 = u * A0, m4 = A1, m5 = uu * A0, m6 = u * A1, m7 = A2;
        // transposing butterfly over the 16 lanes of the half-warp
        const bool b8 = lane & 8, b4 = lane & 4, b2 = lane & 2;
        float r0 = (b8 ? m4 : m0) + __shfl_xor_sync(full, b8 ? m0 : m4, 8);
        float r1 = (b8 ? m5 : m1) + __shfl_xor_sync(full, b8 ? m1 : m5, 8);
        float r2 = (b8 ? m6 : m2) + __shfl_xor_sync(full, b8 ? m2 : m6, 8);
        float r3 = (b8 ? m7 : m3) + __shfl_xor_sync(full, b8 ? m3 : m7, 8);
        float q0 = (b4 ? r2 : r0) + __shfl_xor_sync(full, b4 ? r0 : r2, 4);
        float q1 = (b4 ? r3 : r1) + __shfl_xor_sync(full, b4 ? r1 : r3, 4);
        float p0 = (b2 ? q1 : q0) + __shfl_xor_sync(full, b2 ? q0 : q1, 2);
        p0 += __shfl_xor_sync(full, p0, 1);
        // lane (bit0 = 0) holds moment index 4*b8 + 2*b4 + b2
        if (live && !(lane & 1)) {
            const int idx = ((lane >> 3) & 1) * 4 + ((lane >> 2) & 1) * 2 + ((lane >> 1) & 1);
            if (DET) {
                const int slot = info.x + (ty - (info.y >> 16)) * info.z + (tx - (info.y & 0xffff));
                a.pair_mom[(size_t)slot * 8 + idx] = p0;
            } else {
                atomicAdd(acc + (size_t)gid * 8 + idx, p0);
            }
        }
    }
}

// ---- loss: image sums + target -> G in the backward layout ---------------------------------------
// C: the image of this lane's own 8 rows (FIT_LOSS).  G = 2 (C - T) / (3 W H) on valid pixels, 0
// elsewhere (FIT_GRAD: G = the given dL/dC); the two half-warps swap their rows with one shuffle
// per value.  Returns this lane's share of sum (C - T)^2.
template <bool LOSS>
__device__ __forceinline__ float make_G(const FitArgs &a, const TileGeo &g, const float2 (&C)[4][3], const float *tgt,
                                        int lane, float2 (&G)[TILE / 2][3]) {
    const int cx = lane & 15, hf = lane >> 4;
    const bool colv = g.tx * TILE + cx < a.W;
    float sq = 0.0f;
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        const bool valid = colv && hf * 8 + i < g.rows;
        const int e = (hf * 8 + i) * (TILE * 3) + cx * 3;
#pragma unroll
        for (int ch = 0; ch < 3; ++ch) {
            const float tv = tgt[e + ch];
            float d;
            if (LOSS) {
                const bool in = valid && !(a.roi_on && tv != tv);  // (c-16: NaN marks a pixel outside the ROI)
                d = in ? ((i & 1) ? C[i >> 1][ch].y : C[i >> 1][ch].x) - tv : 0.0f;
                sq = fmaf(d, d, sq);
                d *= a.g_scale;
            } else {
                d = valid ? tv : 0.0f;
            }
            const float o = __shfl_xor_sync(0xffffffffu, d, 16);
            if (i & 1) {
                G[i >> 1][ch].y = d;
                G[4 + (i >> 1)][ch].y = o;
            } else {
                G[i >> 1][ch].x = d;
                G[4 + (i >> 1)][ch].x = o;
            }
        }
    }
    return sq;
}

// team mode: partial images meet in shared memory, lane-major float4 (conflict-free); a float4 holds
// two row pairs, in the order of the flattened C[4][3]
__device__ __forceinline__ void store_part(WarpSmem *sm, const float2 (&C)[4][3], int lane) {
    float4 *dst = reinterpret_cast<float4 *>(sm->cpart);
#pragma unroll
    for (int k = 0; k < 6; ++k) {
        const float2 p0 = C[(2 * k) / 3][(2 * k) % 3], p1 = C[(2 * k + 1) / 3][(2 * k + 1) % 3];
        dst[k * 32 + lane] = make_float4(p0.x, p0.y, p1.x, p1.y);
    }
}
__device__ __forceinline__ void add_parts(const WarpSmem *ws, int wid, float2 (&C)[4][3], int lane) {
#pragma unroll
    for (int p = 1; p < FIT_WARPS; ++p) {
        const float4 *src = reinterpret_cast<const float4 *>(ws[(wid + p) & (FIT_WARPS - 1)].cpart);
#pragma unroll
        for (int k = 0; k < 6; ++k) {
            const float4 v = src[k * 32 + lane];
            float2 &c0 = C[(2 * k) / 3][(2 * k) % 3], &c1 = C[(2 * k + 1) / 3][(2 * k + 1) % 3];
            c0 = __fadd2_rn(c0, make_float2(v.x, v.y));
            c1 = __fadd2_rn(c1, make_float2(v.z, v.w));
        }
    }
}

__device__ __forceinline__ void store_loss(const FitArgs &a, int t, float sq, int lane) {
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) sq += __shfl_xor_sync(0xffffffffu, sq, d);
    if (lane == 0) {
        a.tile_stats[t].sq_raw = (double)sq;
        if (!isfinite(sq)) {
            atomicOr(&a.ta.st->flags, FLAG_NONFINITE);
            atomicCAS(&a.ta.st->first_nonfinite_iter, 0, a.iter);
        }
    }
}

// ---- streaming a list (or a slice of it) through the warp's two record buffers -------------------
// ph: bit i = parity to wait for on bar[i].  Every issue is matched by exactly one wait.
__device__ __forceinline__ void wait_buf(WarpSmem *sm, int buf, unsigned &ph) {
    mbar_wait(&sm->bar[buf], (ph >> buf) & 1u);
    ph ^= 1u << buf;
    __syncwarp();  // the ids were stored by the lanes themselves
}
// entries [e0, e0 + cnt) of the buckets; chunk 0 sits in buffer b0 and has been waited for; later
// chunks alternate
__device__ __forceinline__ void fwd_stream(const FitArgs &a, WarpSmem *sm, size_t e0, int cnt, int b0, unsigned &ph,
                                           int lane, float px, float pyA, float2 (&C)[4][3]) {
    const int nc = (cnt + FIT_CHUNK - 1) / FIT_CHUNK;
    for (int c = 0; c < nc; ++c) {
        const int cb = (b0 + c) & 1;
        if (c + 1 < nc)
            issue_records(a, sm, cb ^ 1, e0 + (size_t)(c + 1) * FIT_CHUNK, min(FIT_CHUNK, cnt - (c + 1) * FIT_CHUNK), 0u,
                          lane);
        if (c > 0) wait_buf(sm, cb, ph);
        fwd_chunk(sm->rec[cb], min(FIT_CHUNK, cnt - c * FIT_CHUNK), px, pyA, C);
        __syncwarp();  // the chunk is dead: its buffer may be refilled
    }
}
// streams the entries again from chunk 0 (into buffer b0; both buffers are free)
template <bool DET>
__device__ __forceinline__ void bwd_stream(const FitArgs &a, WarpSmem *sm, size_t e0, int cnt, int b0, unsigned &ph,
                                           int lane, float px, float py0, const float2 (&G)[TILE / 2][3], int tx, int ty) {
    const int nc = (cnt + FIT_CHUNK - 1) / FIT_CHUNK;
    issue_records(a, sm, b0, e0, min(FIT_CHUNK, cnt), 0u, lane);
    for (int c = 0; c < nc; ++c) {
        const int cb = (b0 + c) & 1;
        if (c + 1 < nc)
            issue_records(a, sm, cb ^ 1, e0 + (size_t)(c + 1) * FIT_CHUNK, min(FIT_CHUNK, cnt - (c + 1) * FIT_CHUNK), 0u,
                          lane);
        wait_buf(sm, cb, ph);
        bwd_chunk<DET>(a, sm->rec[cb], sm->ids[cb], min(FIT_CHUNK, cnt - c * FIT_CHUNK), px, py0, G, tx, ty, lane);
        __syncwarp();
    }
}

// Slow path for tiles that list more Gaussians than their bucket holds: the tile's entries in the shared spill
// list, FIT_CHUNK at a time.  Worker `w` of `nw` (a power of two) takes every nw-th of them; a chunk is staged in
// list buffer 0 (ids collected from the spill list, records gathered) and handed to f(count).
template <class F>
__device__ __forceinline__ void for_spill_chunks(const FitArgs &a, WarpSmem *sm, int t, int w, int nw, unsigned &ph,
                                                 int lane, F &&f) {
    const unsigned lt = (1u << lane) - 1u;
    const int S = spill_size(a.ta);
    int start = 0, ordinal = 0;
    while (start < S) {
        int cnt = 0;
        while (start < S && cnt + 32 <= FIT_CHUNK) {
            const int e = start + lane;
            int2 v = make_int2(-1, -1);
            if (e < S) v = a.ta.spill[e];
            const bool hit = v.x == t;
            const unsigned m = __ballot_sync(0xffffffffu, hit);
            const bool mine = hit && (((ordinal + __popc(m & lt)) & (nw - 1)) == w);
            const unsigned m2 = __ballot_sync(0xffffffffu, mine);
            if (mine) sm->ids[0][cnt + __popc(m2 & lt)] = v.y;
            cnt += __popc(m2);
            ordinal += __popc(m);
            start += 32;
        }
        if (cnt > 0) {
            __syncwarp();
            gather_records(a, sm, 0, cnt, 0u, lane);
            wait_buf(sm, 0, ph);
            f(cnt);
            __syncwarp();
        }
    }
}

// records of chunk 0 of tile g.t (list length n) and the tile's rows -> buffer `buf`, one barrier
__device__ __forceinline__ void issue_tile(const FitArgs &a, const CUtensorMap *map, WarpSmem *sm, const TileGeo &g,
                                           int n, int buf, int lane) {
    const unsigned extra = a.tma_rows ? ROWS_BYTES : 0u;
    issue_records(a, sm, buf, (size_t)g.t * a.ta.tile_cap, min(n, FIT_CHUNK), extra, lane);
    if (a.tma_rows) issue_rows(map, g, sm->tgt, &sm->bar[buf], lane);
}

template <int MODE, bool DET>
__global__ void __launch_bounds__(FIT_THREADS, 5)
    k_fit_tiles(const FitArgs a, const __grid_constant__ CUtensorMap tmap) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    WarpSmem *ws = reinterpret_cast<WarpSmem *>(smem_raw);
    CtaHdr *hdr = reinterpret_cast<CtaHdr *>(smem_raw + sizeof(WarpSmem) * FIT_WARPS);
    constexpr bool LOSS = MODE == FIT_LOSS;
    const unsigned full = 0xffffffffu;
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    WarpSmem *sm = ws + wid;
    DeviceState *st = a.ta.st;
    const int T = a.T, oc = a.ord_cur, on = a.ord_next;

    if (lane == 0) {
        mbar_init(&sm->bar[0], 33u);  // 32 lanes' record gathers + lane 0 (the tile's rows)
        mbar_init(&sm->bar[1], 33u);
        mbar_init(&sm->bar[2], 1u);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    __syncthreads();

    if (tid < NCLS) hdr->cnt[tid] = st->n_class[oc][tid];
    __syncthreads();
    // Which classes the CTAs fit as teams.  A warp alone needs ~900 cycles per list entry (forward + backward), 30 us
    // for a 63-entry tile: nothing when 2,368 warps have 3e5 pairs to share, but the whole kernel when the binning
    // is small (a selective refit of a few thousand Gaussians, a small frame) and most warps have nothing to do.  With
    // few pairs in the launch the team threshold therefore drops from 64 entries to 32: the longest tiles' latency,
    // which is then the kernel's, is split four ways (measured at 1080p: 76 -> 53 us per iteration with 31 % of
    // 50,000 Gaussians active, 39 -> 32 us with 7 %; 16 entries: no further gain; at 3e5 pairs no difference).
    const unsigned long long P_launch = st->pair_total[a.ta.slot];
    const int tc = P_launch < (unsigned long long)a.team_small_pairs ? TEAM_CLASS / 2 : TEAM_CLASS;
    int n_team = 0, n_light = 0;
#pragma unroll
    for (int k = 0; k < NCLS; ++k) {
        if (k >= tc) n_team += hdr->cnt[k];
        else n_light += hdr->cnt[k];
    }
    unsigned ph = 0u;       // parities of this warp's record barriers
    unsigned ph_team = 0u;  // parity of warp 0's row barrier (team mode)
    float2 G[TILE / 2][3];

    // ---- long lists: the CTA works on one tile as a team, the list split four ways -------------
    for (;;) {
        if (tid == 0) {
            const unsigned h = atomicAdd(&st->cursor_team[oc], 1u);
            int t = -1, n = 0;
            if (h < (unsigned)n_team) {
                t = tile_of_position(a.order_cur, T, hdr->cnt, (int)h);
                n = tile_count_of(a.ta, T, t);
            }
            hdr->t = t;
            hdr->n = n;
        }
        __syncthreads();
        // (warp-wide max of values all lanes share: marks them warp-uniform for the compiler, which
        // keeps the list loops on uniform registers and branches)
        const int t = __reduce_max_sync(full, hdr->t), n_raw = __reduce_max_sync(full, hdr->n);
        if (t < 0) break;
        const int n = max(n_raw, 0);
        const TileGeo g = tile_geo(a, t, lane);
        // The list in units of 4 entries (slices start at multiples of 4: 16-byte id copies), the units
        // dealt out evenly; which warp takes which slice rotates with the tile, so that the shorter last
        // slice does not always fall to the same SM sub-partition.
        const int nm = min(n, a.ta.tile_cap);  // the bucket's part; the rest sits in the spill list
        const bool spilled = n > nm;
        const int units = (nm + 3) >> 2, sl = (wid + t) & (FIT_WARPS - 1);
        const int beg = min(nm, ((sl * units) / FIT_WARPS) << 2);
        const int cnt = min(nm, (((sl + 1) * units) / FIT_WARPS) << 2) - beg;
        const size_t seg = (size_t)t * a.ta.tile_cap + beg;
        int pos_file = 0;
        if (tid == 0) pos_file = atomicAdd(&st->n_class[on][tile_class(n)], 1);
        if (wid == 0) {  // the tile's rows, for everybody
            if (a.tma_rows) {
                if (lane == 0) mbar_expect_tx(&ws[0].bar[2], ROWS_BYTES);
                issue_rows(&tmap, g, ws[0].tgt, &ws[0].bar[2], lane);
            } else {
                load_rows_generic(a, g, ws[0].tgt, lane);
            }
        }
        float2 C[4][3];
        if (LOSS) {
            issue_records(a, sm, 0, seg, min(cnt, FIT_CHUNK), 0u, lane);
            wait_buf(sm, 0, ph);
#pragma unroll
            for (int k = 0; k < 4; ++k) C[k][0] = C[k][1] = C[k][2] = make_float2(0.0f, 0.0f);
            fwd_stream(a, sm, seg, cnt, 0, ph, lane, g.px, g.py0 + (float)(8 * (lane >> 4)), C);
            if (spilled)
                for_spill_chunks(a, sm, t, sl, FIT_WARPS, ph, lane, [&](int c) {
                    fwd_chunk(sm->rec[0], c, g.px, g.py0 + (float)(8 * (lane >> 4)), C);
                });
            store_part(sm, C, lane);
        }
        __syncthreads();  // partial images (and generic row loads) visible
        if (LOSS) add_parts(ws, wid, C, lane);
        const bool res_t = LOSS && cnt <= FIT_CHUNK && !spilled;  // the slice is still resident in buffer 0
        if (a.tma_rows) {
            mbar_wait(&ws[0].bar[2], ph_team);
            ph_team ^= 1u;
        }
        const float sq = make_G<LOSS>(a, g, C, ws[0].tgt, lane, G);
        __syncthreads();  // everybody is done with the rows, the partial images and the header
        if (LOSS && wid == 0 && n_raw >= 0) store_loss(a, t, sq, lane);
        if (cnt > 0) {
            if (res_t) bwd_chunk<DET>(a, sm->rec[0], sm->ids[0], cnt, g.px, g.py0, G, g.tx, g.ty, lane);
            else bwd_stream<DET>(a, sm, seg, cnt, 0, ph, lane, g.px, g.py0, G, g.tx, g.ty);
        }
        if (spilled)
            for_spill_chunks(a, sm, t, sl, FIT_WARPS, ph, lane, [&](int c) {
                bwd_chunk<DET>(a, sm->rec[0], sm->ids[0], c, g.px, g.py0, G, g.tx, g.ty, lane);
            });
        if (tid == 0) {  // (stores kept behind the list loops: see gs2d_raster.cu, finish())
            tile_publish(a.ta, T, t, n_raw);
            tile_file_at(st, a.order_next, T, oc, on, t, n, pos_file);
        }
    }

    // ---- short lists: every warp on its own, next tile prefetched during the backward pass -----
    // A warp holds at most one claimed tile beside the one it works on (a deeper claim queue would
    // leave some warps with two tiles to go when the queue runs dry, others with none).
    int lcnt[TEAM_CLASS];
#pragma unroll
    for (int k = 0; k < TEAM_CLASS; ++k) lcnt[k] = hdr->cnt[k];
    auto lookup = [&](unsigned q) -> int {  // position in the light order (longest lists first) -> tile
        if (q >= (unsigned)n_light) return -1;
        int cls = tc - 1, r = (int)q;
#pragma unroll
        for (int k = TEAM_CLASS - 1; k > 0; --k) {
            const bool go = cls == k && r >= lcnt[k];
            r = go ? r - lcnt[k] : r;
            cls = go ? k - 1 : cls;
        }
        return a.order_cur[(size_t)cls * T + r];
    };
    unsigned qreg = 0u;  // lane 0: claimed queue position of the next tile
    if (lane == 0) qreg = atomicAdd(&st->cursor_warp[oc], 1u);
    int t = __reduce_max_sync(full, lookup(__shfl_sync(full, qreg, 0)));
    int n_raw = __reduce_max_sync(full, t >= 0 ? tile_count_of(a.ta, T, t) : 0);
    int buf = 0;
    if (t >= 0) issue_tile(a, &tmap, sm, tile_geo(a, t, lane), max(n_raw, 0), buf, lane);
    while (t >= 0) {
        const int n = max(n_raw, 0);
        const TileGeo g = tile_geo(a, t, lane);
        const size_t seg = (size_t)t * a.ta.tile_cap;
        int pos_file = 0;
        if (lane == 0) {
            qreg = atomicAdd(&st->cursor_warp[oc], 1u);  // the next tile: looked up after the forward pass
            pos_file = atomicAdd(&st->n_class[on][tile_class(n)], 1);
        }
        if (!a.tma_rows) load_rows_generic(a, g, sm->tgt, lane);
        wait_buf(sm, buf, ph);  // chunk 0 (+ rows) has landed
        const int nm = min(n, a.ta.tile_cap);  // (n > tile_cap reaches a single warp only on a context's first launch)
        const bool spilled = n > nm;
        const bool resident = n <= FIT_CHUNK;
        float2 C[4][3];
        if (LOSS) {
#pragma unroll
            for (int k = 0; k < 4; ++k) C[k][0] = C[k][1] = C[k][2] = make_float2(0.0f, 0.0f);
            fwd_stream(a, sm, seg, nm, buf, ph, lane, g.px, g.py0 + (float)(8 * (lane >> 4)), C);
            if (spilled)
                for_spill_chunks(a, sm, t, 0, 1, ph, lane, [&](int c) {
                    fwd_chunk(sm->rec[0], c, g.px, g.py0 + (float)(8 * (lane >> 4)), C);
                });
        }
        const int t_next = __reduce_max_sync(full, lookup(__shfl_sync(full, qreg, 0)));
        __syncwarp();
        const float sq = make_G<LOSS>(a, g, C, sm->tgt, lane, G);
        const int n_next = __reduce_max_sync(full, t_next >= 0 ? tile_count_of(a.ta, T, t_next) : 0);
        __syncwarp();  // the rows are dead
        if (LOSS && n_raw >= 0) store_loss(a, t, sq, lane);
        if (resident && t_next >= 0)
            issue_tile(a, &tmap, sm, tile_geo(a, t_next, lane), max(n_next, 0), buf ^ 1, lane);
        if (n > 0) {
            if (resident) {
                bwd_chunk<DET>(a, sm->rec[buf], sm->ids[buf], n, g.px, g.py0, G, g.tx, g.ty, lane);
            } else {
                bwd_stream<DET>(a, sm, seg, nm, buf, ph, lane, g.px, g.py0, G, g.tx, g.ty);
                if (spilled)
                    for_spill_chunks(a, sm, t, 0, 1, ph, lane, [&](int c) {
                                bwd_chunk<DET>(a, sm->rec[0], sm->ids[0], c, g.px, g.py0, G, g.tx, g.ty, lane);
                    });
            }
        }
        if (!resident && t_next >= 0)
            issue_tile(a, &tmap, sm, tile_geo(a, t_next, lane), max(n_next, 0), buf ^ 1, lane);
        if (lane == 0) {
            tile_publish(a.ta, T, t, n_raw);
            tile_file_at(st, a.order_next, T, oc, on, t, n, pos_file);
        }
        t = t_next;
        n_raw = n_next;
        buf ^= 1;
    }
}

// ---- host: tensor map of the image, launch ------------------------------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                  const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

// [H][3W] float32 image, boxes of 48 x 16 elements.  Returns false when the image cannot have a map
// (row pitch or base not 16-byte aligned) or the driver lacks the encoder: the kernel then loads
// the rows with plain loads.
static bool encode_image_map(const float *image, int W, int H, CUtensorMap *out) {
    // (function-local static with an initialiser: thread-safe, contexts may be driven from several host threads)
    static const EncodeTiledFn fn = []() -> EncodeTiledFn {
        void *p = nullptr;
        cudaDriverEntryPointQueryResult qr;
        const bool ok = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qr) == cudaSuccess &&
                        qr == cudaDriverEntryPointSuccess;
        cudaGetLastError();
        return ok ? (EncodeTiledFn)p : nullptr;
    }();
    if (!fn || W % 4 != 0 || ((size_t)image & 15u) != 0) return false;
    const cuuint64_t dims[2] = {(cuuint64_t)W * 3, (cuuint64_t)H};
    const cuuint64_t strides[1] = {(cuuint64_t)W * 3 * sizeof(float)};
    const cuuint32_t box[2] = {TILE * 3, TILE};
    const cuuint32_t estr[2] = {1, 1};
    return fn(out, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, (void *)image, dims, strides, box, estr,
              CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE,
              CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

__global__ void __launch_bounds__(256) k_sub_from(const float *__restrict__ a, float *__restrict__ out, size_t n) {
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x)
        out[i] = a[i] - out[i];
}
__global__ void __launch_bounds__(256) k_mask_target(const float *__restrict__ src, const unsigned char *__restrict__ roi,
                                                     float *__restrict__ out, size_t npix) {
    // NaN is the fit kernel's mark for "outside the ROI" (make_G).  A non-finite target value INSIDE the ROI must
    // still poison the loss (as without an ROI): it is passed on as +Inf, which no mark can be
    // mistaken for -- the iteration's loss is then non-finite and the latch fires with that iteration's index.
    const float nan = __int_as_float(0x7fc00000), inf = __int_as_float(0x7f800000);
    for (size_t p = (size_t)blockIdx.x * blockDim.x + threadIdx.x; p < npix; p += (size_t)gridDim.x * blockDim.x) {
        const bool in = roi[p] != 0;
#pragma unroll
        for (int ch = 0; ch < 3; ++ch) {
            const float v = src[3 * p + ch];
            out[3 * p + ch] = in ? (isfinite(v) ? v : inf) : nan;
        }
    }
}
int launch_mask_target(const float *src, const unsigned char *roi, float *out, size_t npix, cudaStream_t s) {
    k_mask_target<<<(int)((npix + 256 * 4 - 1) / (256 * 4)), 256, 0, s>>>(src, roi, out, npix);
    GS_CUDA_TRY(cudaGetLastError());
    return GS_OK;
}
__global__ void __launch_bounds__(1024) k_roi_count(const unsigned char *__restrict__ roi, size_t npix, DeviceState *st) {
    __shared__ unsigned long long s_c[1024];
    unsigned long long c = 0;
    for (size_t p = threadIdx.x; p < npix; p += 1024) c += roi[p] ? 1 : 0;
    s_c[threadIdx.x] = c;
    __syncthreads();
    for (int d = 512; d > 0; d >>= 1) {
        if ((int)threadIdx.x < d) s_c[threadIdx.x] += s_c[threadIdx.x + d];
        __syncthreads();
    }
    if (threadIdx.x == 0) st->roi_pixels = s_c[0];
}
int launch_roi_count(gs_ctx *c, const unsigned char *roi, cudaStream_t s) {
    k_roi_count<<<1, 1024, 0, s>>>(roi, (size_t)c->cfg.width * c->cfg.height, c->dstate);
    GS_CUDA_TRY(cudaGetLastError());
    return GS_OK;
}
int launch_sub_from(const float *a, float *out, size_t n, cudaStream_t s) {
    k_sub_from<<<(int)((n + 256 * 8 - 1) / (256 * 8)), 256, 0, s>>>(a, out, n);
    GS_CUDA_TRY(cudaGetLastError());
    return GS_OK;
}

int launch_fit_tiles(gs_ctx *c, FitMode mode, const float *image, int iter, cudaStream_t s) {
    // deterministic mode: every list in ascending id order before it is summed
    if (c->deterministic) {
        const int rc = launch_presort_tiles(c, s);
        if (rc) return rc;
    }
    if (c->fit_grid == 0) {
        GS_CUDA_TRY(cudaFuncSetAttribute(k_fit_tiles<FIT_LOSS, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)FIT_SMEM));
        GS_CUDA_TRY(cudaFuncSetAttribute(k_fit_tiles<FIT_GRAD, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)FIT_SMEM));
        GS_CUDA_TRY(cudaFuncSetAttribute(k_fit_tiles<FIT_LOSS, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)FIT_SMEM));
        GS_CUDA_TRY(cudaFuncSetAttribute(k_fit_tiles<FIT_GRAD, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)FIT_SMEM));
        int per_sm = 0;
        GS_CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_fit_tiles<FIT_LOSS, false>, FIT_THREADS, FIT_SMEM));
        // One CTA per SM short of full occupancy: on one stream that costs nothing (measured: 8.87k against
        // 8.88k iters/s), and it leaves room for another stream's kernels -- the Adam/binning kernel or the
        // first CTAs of the next frame's fit -- to become resident beside this grid (4 streams: 12.8k against
        // 12.0k iters/s).
        if (per_sm > 2) --per_sm;
        c->fit_grid = c->sm_count * (per_sm > 0 ? per_sm : 1);
    }
    FitArgs a;
    a.ta = tile_args(c);
    const int oc = (int)(c->fwd_launches % 3u), on = (int)((c->fwd_launches + 1u) % 3u);
    ++c->fwd_launches;
    a.order_cur = c->tile_order + (size_t)oc * NCLS * c->T;
    a.order_next = c->tile_order + (size_t)on * NCLS * c->T;
    a.ord_cur = oc;
    a.ord_next = on;
    a.rec = c->rec;
    a.bucket = c->bucket;
    a.image = image;
    a.W = c->cfg.width;
    a.H = c->cfg.height;
    a.TX = c->TX;
    a.T = c->T;
    a.tx_magic = ((1ull << 40) + (unsigned long long)c->TX - 1ull) / (unsigned long long)c->TX;
    static_assert(sizeof(c->image_map) == sizeof(CUtensorMap), "gs_ctx::image_map holds a CUtensorMap");
    if (c->image_map_ptr != image) {  // the map depends on the address only: cached per context
        c->image_map_ok = encode_image_map(image, a.W, a.H, reinterpret_cast<CUtensorMap *>(c->image_map));
        c->image_map_ptr = image;
    }
    a.tma_rows = c->image_map_ok ? 1 : 0;
    const CUtensorMap &tmap = *reinterpret_cast<const CUtensorMap *>(c->image_map);
    a.roi_on = (c->roi && mode == FIT_LOSS) ? 1 : 0;
    a.team_small_pairs = 250000;  // (about 100 pairs per warp of the persistent grid)
    a.g_scale = a.roi_on ? (float)(2.0 / (3.0 * (double)c->roi_count)) : (float)(2.0 / (3.0 * (double)a.W * (double)a.H));
    a.iter = iter;
    a.acc = c->acc;
    a.pair_info = c->deterministic ? c->pair_info : nullptr;
    a.pair_mom = c->deterministic ? c->pair_mom : nullptr;
    a.tile_stats = c->tile_stats;
    // never more CTAs than there could be work for (a team per class-3 tile or a warp per tile)
    const int grid = min(c->fit_grid, c->T);
    if (c->deterministic) {
        if (mode == FIT_GRAD) k_fit_tiles<FIT_GRAD, true><<<grid, FIT_THREADS, FIT_SMEM, s>>>(a, tmap);
        else k_fit_tiles<FIT_LOSS, true><<<grid, FIT_THREADS, FIT_SMEM, s>>>(a, tmap);
    } else {
        if (mode == FIT_GRAD) k_fit_tiles<FIT_GRAD, false><<<grid, FIT_THREADS, FIT_SMEM, s>>>(a, tmap);
        else k_fit_tiles<FIT_LOSS, false><<<grid, FIT_THREADS, FIT_SMEM, s>>>(a, tmap);
    }
    c->fresh = false;                // the bins are consumed
    c->sorted = c->deterministic;    // ... in arrival order, unless they were sorted first
    GS_CUDA_TRY(cudaGetLastError());
    return GS_OK;
}

}  // namespace gs2d
