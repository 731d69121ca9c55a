// gs2d_fit_tc.cu -- the fit kernel on the 5th-generation tensor cores (tcgen05 / TMEM): forward
// rasterizer + L2 loss + backward pass of one fit iteration, per tile.
//
// Per tile, Eq. 2 and its gradient ARE dense contractions once the weights
//     w[n][p] = exp(-sigma_n(p)),   n = list entry, p = pixel of the tile (256)
// are written down as a matrix W:
//     forward   C[p][ch]      = sum_n W[n][p] c'[n][ch]                 (K = list entries)
//     backward  M[n][ch][k]   = sum_p W[n][p] G[p][ch] phi_k(p)         (K = 256 pixels)
// with phi = (1, x, y, x^2, xy, y^2) in pixel coordinates relative to the tile centre.  The eight gradient
// moments of a (tile, Gaussian) pair (DESIGN.md §3 c-5) are linear in M: contract the channels with c'
// (s = w c'.G), then move the polynomial moments from the tile centre to the Gaussian's whitened
// coordinates -- ~60 flops per PAIR instead of 12 FP32 operations per PIXEL-pair.  What is left for the
// CUDA cores per pixel-pair is the exponent (2 FMA), one MUFU.EX2 and the conversion of w to the tensor
// cores' operand format, ONCE for both passes (W stays in shared memory between them).
//
// Precision: the tensor cores take binary16 operands and accumulate in binary32.  Every operand is
// split into a binary16 head and a binary16 tail (x = hi + lo exactly to 2^-22 relative), and all
// four partial products hi*hi + hi*lo + lo*hi + lo*lo are accumulated: the results carry binary32
// accuracy (pixels to ~1e-6, well inside the 1e-4 bar).  The tails cost no extra instructions on the
// tensor side where the M dimension was padding anyway: W's 64 tail rows ride in the upper half of
// the M = 128 operand, c' tails in unused N columns.
//
//   operand layouts (no swizzle; "core matrix" = 8 rows x 16 bytes; verified on B200)
//     W   [32 pixel octets][16 row groups][8 rows][8 pixels] binary16; row groups 0-7 = heads of list
//         entries 0-63, 8-15 = their tails.  ONE buffer serves both passes: as the MN-major A operand
//         of the forward product (M = pixels, K = entries) and as the K-major A operand of the backward
//         product (M = entries, K = pixels).
//     Cb  [8 entry groups][2 column groups][8 entries][8 columns]: (c'_hi rgb, c'_lo rgb, 0, 0 | 0...) x 2^6
//     Bm  [32 pixel octets][6 column groups][8 pixels][8 columns]: G[p][ch] phi_k(p) scaled per tile, heads in
//         column groups 0-2, tails in 3-5 (one N = 48 operand: W is read from shared memory once per K step)
//   accumulators in TMEM: forward D [128 pixels x 16] x 2 halves, backward D [128 rows x 48]
//
// One CTA of 8 warps works on one tile at a time; two CTAs per SM, so that one CTA's tensor-core
// phase overlaps the other's CUDA-core phase.  Lists longer than 64 entries go through the W buffer
// in chunks: the forward product accumulates over the chunks, the backward pass revisits them.
#include <cuda_fp16.h>
#include <stdio.h>

#include "gs2d_fit.cuh"

namespace gs2d {

constexpr int TC_THREADS = 256;
constexpr int TC_CHUNK = 64;                    // list entries per W buffer
constexpr unsigned W_PG = 2048;                 // bytes per pixel octet of W: 16 row groups x 128
constexpr unsigned W_BYTES = 32 * W_PG;         // 64 KB
constexpr unsigned W_TAIL = 1024;               // tails: row groups 8..15
constexpr unsigned BM_KG = 768;                 // bytes per pixel octet of the moment operand: 6 column groups x 128
constexpr unsigned BM_BYTES = 32 * BM_KG;       // (column groups 0-2 heads, 3-5 tails: N = 48)
constexpr unsigned BM_TAIL = 384;
// Products that accumulate into the same tensor-memory tile are executed one after the other at the full
// pipeline latency (~100 cycles each, whatever N is); the K steps are therefore dealt to independent accumulators
// that the epilogues add up: forward 4 x [128 x 16] (pixel half x {heads, tails}), backward 4 x [128 x 48].
constexpr unsigned TMEM_COLS = 256;
constexpr unsigned TM_FWD = 0;                  // + 16 * (2 * half + part)
constexpr unsigned TM_BWD = 64;                 // + 48 * (K step & 3)
constexpr unsigned CB_KG = 256;                 // bytes per entry group of the colour operand: 2 column groups x 128
constexpr unsigned CB_BYTES = 8 * CB_KG;
constexpr float W_SCALE_LOG2 = 10.0f;           // W holds 2^10 w   (binary16 normal range down to w = 6e-8)
constexpr float C_SCALE = 64.0f;                // Cb holds 2^6 c'
constexpr float FWD_UNSCALE = 1.0f / (1024.0f * 64.0f);
constexpr int E_STRIDE = 20;                    // floats per row of the tail scratch

struct __align__(128) TcSmem {
    unsigned char W[W_BYTES];
    unsigned char Bm[BM_BYTES];
    unsigned char Cb[CB_BYTES];
    float4 rec[2][TC_CHUNK * REC_F4];
    int ids[2][TC_CHUNK];
    float tgt[TILE_PX * 3];
    float escr[64 * E_STRIDE];                  // backward accumulator rows of the tails
    unsigned long long bar_rec[2], bar_mma;
    unsigned tmem_base;
    int t_next, n_next;
    int cnt[NCLS];
    float red_sq[8];
    unsigned red_max[8];
};

// ---- tcgen05 wrappers ---------------------------------------------------------------------------
__device__ __forceinline__ unsigned long long smem_desc(unsigned addr, unsigned lbo, unsigned sbo) {
    // no swizzle; LBO = byte distance of core matrices adjacent in K, SBO = adjacent in M / N
    return (unsigned long long)((addr >> 4) & 0x3fffu) | ((unsigned long long)((lbo >> 4) & 0x3fffu) << 16) |
           ((unsigned long long)((sbo >> 4) & 0x3fffu) << 32) | (1ull << 46);
}
__host__ __device__ constexpr unsigned instr_desc_f16(int M, int N, int a_mn_major, int b_mn_major) {
    // binary16 operands, binary32 accumulator
    return (1u << 4) | ((unsigned)a_mn_major << 15) | ((unsigned)b_mn_major << 16) | ((unsigned)(N >> 3) << 17) |
           ((unsigned)(M >> 4) << 24);
}
__device__ __forceinline__ void umma_f16(unsigned d_tmem, unsigned long long da, unsigned long long db, unsigned idesc,
                                         unsigned accumulate) {
    asm volatile(
        "{\n.reg .pred p;\nsetp.ne.b32 p, %4, 0;\n"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n}\n" ::"r"(d_tmem),
        "l"(da), "l"(db), "r"(idesc), "r"(accumulate)
        : "memory");
}
__device__ __forceinline__ void umma_commit(unsigned long long *bar) {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar))
                 : "memory");
}
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void proxy_fence() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void tmem_ld8(unsigned taddr, float (&r)[8]) {
    unsigned u[8];
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                 : "=r"(u[0]), "=r"(u[1]), "=r"(u[2]), "=r"(u[3]), "=r"(u[4]), "=r"(u[5]), "=r"(u[6]), "=r"(u[7])
                 : "r"(taddr));
#pragma unroll
    for (int i = 0; i < 8; ++i) r[i] = __uint_as_float(u[i]);
}
__device__ __forceinline__ void tmem_ld_wait() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }

// bounded wait: a tensor-core or copy completion that never arrives is a bug, not a hang
__device__ __forceinline__ void mbar_wait_bounded(unsigned long long *bar, unsigned parity) {
    unsigned ok = 0;
    const long long t0 = clock64();
    while (!ok) {
        asm volatile("{\n.reg .pred p;\nmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\nselp.u32 %0, 1, 0, p;\n}\n"
                     : "=r"(ok)
                     : "r"(smem_u32(bar)), "r"(parity)
                     : "memory");
        if (!ok && clock64() - t0 > 4000000000ll) __trap();
    }
}

__device__ __forceinline__ unsigned pack_h2(__half2 h) { return *reinterpret_cast<unsigned *>(&h); }
// x (two values) -> binary16 heads and tails: head = rn16(x), tail = rn16(x - head)
__device__ __forceinline__ void split_h2(float2 x, unsigned &hi, unsigned &lo) {
    const __half2 h = __floats2half2_rn(x.x, x.y);
    const float2 hf = __half22float2(h);
    const __half2 l = __floats2half2_rn(x.x - hf.x, x.y - hf.y);
    hi = pack_h2(h);
    lo = pack_h2(l);
}

// ---- W: weights of `cnt` list entries at the 256 pixels of the tile -> shared memory ---------------
// work item = (entry m, pixel octet o), an octet = 8 rows of one column; the items are dealt out evenly,
// consecutive threads taking consecutive entries of one octet (16-byte stores of a quarter-warp are contiguous)
__device__ __forceinline__ void gen_W(unsigned char *W, const float4 *__restrict__ rec, int cnt, float px0, float py0,
                                      int tid) {
    const int cp8 = (cnt + 7) & ~7;
    const int step_o = TC_THREADS / cp8, step_m = TC_THREADS - step_o * cp8;
    int o = tid / cp8, m = tid - o * cp8;
    while (o < 32) {
        // two items per round, in one basic block (independent chains: the MUFU and conversion latencies overlap)
        int mm[2], oo[2];
        bool ok[2];
#pragma unroll
        for (int s = 0; s < 2; ++s) {
            mm[s] = m;
            oo[s] = o;
            ok[s] = o < 32 && m < cnt;
            m += step_m;
            o += step_o;
            if (m >= cp8) {
                m -= cp8;
                ++o;
            }
        }
        float4 lo[2], hi[2];
#pragma unroll
        for (int s = 0; s < 2; ++s) {
            const int mi = min(mm[s], cnt - 1);
            lo[s] = rec[REC_F4 * mi];       // (mux, muy, i1, k)
            hi[s] = rec[REC_F4 * mi + 1];   // (i3, c'r, c'g, c'b)
        }
        float2 uu[2], v0[2];
#pragma unroll
        for (int s = 0; s < 2; ++s) {
            const int x = oo[s] & 15, h = (oo[s] >> 4) & 1;
            const float dx = (px0 + (float)x) - lo[s].x;
            const float u = dx * lo[s].z;
            uu[s] = dup2(fmaf(u, u, -W_SCALE_LOG2));  // 2^-(u^2 + v^2 - 10) = 2^10 w
            v0[s] = dup2(fmaf(dx, lo[s].w, ((py0 + (float)(8 * h)) - lo[s].y) * hi[s].x));
        }
        unsigned wh[2][4], wl[2][4];
#pragma unroll
        for (int k = 0; k < 4; ++k)
#pragma unroll
            for (int s = 0; s < 2; ++s) {
                const float2 v = __ffma2_rn(dup2(hi[s].x), c_rowpair[k], v0[s]);
                const float2 p = __ffma2_rn(v, v, uu[s]);
                split_h2(make_float2(fit_ex2_neg(p.x), fit_ex2_neg(p.y)), wh[s][k], wl[s][k]);
            }
#pragma unroll
        for (int s = 0; s < 2; ++s)
            if (ok[s]) {
                unsigned char *dst = W + (unsigned)oo[s] * W_PG + (mm[s] >> 3) * 128 + (mm[s] & 7) * 16;
                *reinterpret_cast<uint4 *>(dst) = make_uint4(wh[s][0], wh[s][1], wh[s][2], wh[s][3]);
                *reinterpret_cast<uint4 *>(dst + W_TAIL) = make_uint4(wl[s][0], wl[s][1], wl[s][2], wl[s][3]);
            }
    }
}

// ---- Cb: premultiplied colours of the chunk's entries (heads | tails in columns 0-2 | 3-5) ---------
__device__ __forceinline__ void gen_Cb(unsigned char *Cb, const float4 *__restrict__ rec, int cnt, int tid) {
    if (tid >= TC_CHUNK) return;
    uint4 v = make_uint4(0u, 0u, 0u, 0u);
    if (tid < cnt) {
        const float4 hi = rec[REC_F4 * tid + 1];
        unsigned h01, l01, h2x, l2x;
        split_h2(make_float2(hi.y * C_SCALE, hi.z * C_SCALE), h01, l01);
        split_h2(make_float2(hi.w * C_SCALE, 0.0f), h2x, l2x);
        // columns: 0 1 2 = heads r g b, 3 4 5 = tails r g b
        v.x = h01;
        v.y = (h2x & 0xffffu) | (l01 << 16);
        v.z = (l01 >> 16) | (l2x << 16);
    }
    *reinterpret_cast<uint4 *>(Cb + (tid >> 3) * CB_KG + (tid & 7) * 16) = v;
}

// Base descriptors (thread 0's registers): a step along an operand adds (bytes >> 4) to the address field.
struct TcDesc {
    unsigned long long w_mn, w_k, cb, bm;
};
__device__ __forceinline__ TcDesc make_descs(const TcSmem *sm) {
    TcDesc d;
    d.w_mn = smem_desc(smem_u32(sm->W), 128u, W_PG);   // forward A: M = pixels (octets W_PG apart), K = entries
    d.w_k = smem_desc(smem_u32(sm->W), W_PG, 128u);    // backward A: M = rows (heads, tails), K = pixels
    d.cb = smem_desc(smem_u32(sm->Cb), CB_KG, 128u);
    d.bm = smem_desc(smem_u32(sm->Bm), BM_KG, 128u);
    return d;
}
// forward product of one chunk: D_f[half][part] (+)= W^T (part: heads / tails) x Cb
__device__ __forceinline__ void issue_forward(const TcDesc &d, unsigned tmem, int cnt, bool first_chunk) {
    constexpr unsigned IDESC = instr_desc_f16(128, 16, 1, 1);
    const int ks = (cnt + 15) >> 4;
#pragma unroll
    for (int j = 0; j < 4; ++j)
        if (j < ks) {
#pragma unroll
            for (int h = 0; h < 2; ++h)
#pragma unroll
                for (int part = 0; part < 2; ++part)
                    umma_f16(tmem + TM_FWD + 16u * (unsigned)(2 * h + part),
                             d.w_mn + (((unsigned)(16 * h) * W_PG + (unsigned)(part * 8 + 2 * j) * 128u) >> 4),
                             d.cb + (((unsigned)j * 2u * CB_KG) >> 4), IDESC, (j == 0 && first_chunk) ? 0u : 1u);
        }
}
// backward product of one chunk: D_b[j & 3] += [W heads; W tails] x [Bm heads | Bm tails] over K step j
__device__ __forceinline__ void issue_backward(const TcDesc &d, unsigned tmem) {
    constexpr unsigned IDESC = instr_desc_f16(128, 48, 0, 1);
#pragma unroll
    for (int j = 0; j < 16; ++j)
        umma_f16(tmem + TM_BWD + 48u * (unsigned)(j & 3), d.w_k + (((unsigned)j * 2u * W_PG) >> 4),
                 d.bm + (((unsigned)j * 2u * BM_KG) >> 4), IDESC, j < 4 ? 0u : 1u);
}

// ids of list entries [e0, e0 + cnt) of tile t -> buffer `buf` (+ the tile's rows when with_rows); one thread.
// The records are gathered by id by the threads once the ids have landed (stage_records).
__device__ __forceinline__ void tc_issue_chunk(const FitArgs &a, const CUtensorMap *map, TcSmem *sm, int t, int e0, int cnt,
                                               int buf, bool with_rows, const TileGeo &g) {
    const unsigned ibytes = (unsigned)((cnt + 3) & ~3) * 4u;  // (buckets are padded to multiples of 32 ids)
    const unsigned extra = (with_rows && a.tma_rows) ? ROWS_BYTES : 0u;
    mbar_expect_tx(&sm->bar_rec[buf], ibytes + extra);
    if (cnt > 0) bulk_g2s(sm->ids[buf], a.bucket + (size_t)t * a.ta.tile_cap + e0, ibytes, &sm->bar_rec[buf]);
    if (extra) tma_tile_g2s(sm->tgt, map, g.tx * (TILE * 3), g.ty * TILE, &sm->bar_rec[buf]);
}

#ifdef TC_PROFILE
#define TCP_DECL long long tcp_t = clock64(), tcp_acc[10] = {0,0,0,0,0,0,0,0,0,0}; int tcp_tiles = 0, tcp_pairs = 0;
#define TCP(i) do { const long long now_ = clock64(); tcp_acc[i] += now_ - tcp_t; tcp_t = now_; } while (0)
#else
#define TCP_DECL
#define TCP(i)
#endif

// records of the chunk whose ids sit in buffer `buf` -> the buffer's record array (all threads; ends with a barrier)
__device__ __forceinline__ void stage_records(const FitArgs &a, TcSmem *sm, int buf, int cnt, int tid) {
    if (tid < cnt) {
        const float4 *src = reinterpret_cast<const float4 *>(a.rec + sm->ids[buf][tid]);
        sm->rec[buf][REC_F4 * tid] = src[0];
        sm->rec[buf][REC_F4 * tid + 1] = src[1];
    }
    __syncthreads();
}

template <int MODE>
__global__ void __launch_bounds__(TC_THREADS, 2)
    k_fit_tc(const FitArgs a, const __grid_constant__ CUtensorMap tmap) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    TcSmem *sm = reinterpret_cast<TcSmem *>(smem_raw);
    constexpr bool LOSS = MODE == FIT_LOSS;
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    DeviceState *st = a.ta.st;
    const int T = a.T, oc = a.ord_cur, on = a.ord_next;

    // ---- set-up: barriers, tensor memory, operand buffers zeroed (what the products read must be finite)
    if (tid == 0) {
        mbar_init(&sm->bar_rec[0], 1u);
        mbar_init(&sm->bar_rec[1], 1u);
        mbar_init(&sm->bar_mma, 1u);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    if (wid == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 256;" ::"r"(smem_u32(&sm->tmem_base))
                     : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    {
        uint4 *z = reinterpret_cast<uint4 *>(sm->W);
        constexpr int NZ = (int)((W_BYTES + BM_BYTES + CB_BYTES) / 16);
        for (int i = tid; i < NZ; i += TC_THREADS) z[i] = make_uint4(0u, 0u, 0u, 0u);
    }
    if (tid < NCLS) sm->cnt[tid] = st->n_class[oc][tid];
    proxy_fence();
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const unsigned tmem = sm->tmem_base;
    unsigned ph_rec = 0u, ph_mma = 0u;  // parities to wait for
    int rb = 0;                         // record buffer of the next chunk visit

    // Two single-thread roles: thread 0 issues the tensor-core products; thread QT (warp 7) owns the tile
    // queue, the copies and the per-tile bookkeeping.  QT works while everybody waits for the backward
    // products: its dependent global accesses (claim -> launch order -> list length) cost no time there.
    constexpr int QT = TC_THREADS - 32;
    TcDesc dsc = {};
    bool bad = false;      // the binning exceeded a capacity: nothing downstream may write
    int tq = -1, nq = 0;   // QT: the tile after the current one, resolved
    const int *tcount = a.ta.tile_count + (size_t)a.ta.slot * T;
    auto claim = [&](int &tt, int &nn) {
        const unsigned q = atomicAdd(&st->cursor_team[oc], 1u);
        tt = -1;
        nn = 0;
        if (q < (unsigned)T) {
            tt = tile_of_position(a.order_cur, T, sm->cnt, (int)q);
            nn = bad ? -1 : tcount[tt];
        }
    };
    if (tid == 0) dsc = make_descs(sm);
    if (tid == QT) {
        bad = st->pair_total[a.ta.slot] > (unsigned long long)a.ta.cap_pairs || st->tile_ovf[a.ta.slot] != 0;
        int t0, n0;
        claim(t0, n0);
        if (t0 >= 0) tc_issue_chunk(a, &tmap, sm, t0, 0, min(max(n0, 0), TC_CHUNK), rb, true, tile_geo(a, t0, 0));
        sm->t_next = t0;
        sm->n_next = n0;
        claim(tq, nq);
    }
    __syncthreads();
    int t = sm->t_next, n_raw = sm->n_next;
    TCP_DECL

    while (t >= 0) {
        // (this kernel has no slow path for entries beyond a tile's bucket: such a tile is a capacity error here)
        const int n = min(max(n_raw, 0), a.ta.tile_cap);
        if (tid == QT && n_raw > a.ta.tile_cap) atomicOr(&st->flags, FLAG_CAPACITY);
        const int nc = (n + TC_CHUNK - 1) / TC_CHUNK;
        const TileGeo g = tile_geo(a, t, 0);
        const float px0 = (float)(g.tx * TILE) + 0.5f, py0 = (float)(g.ty * TILE) + 0.5f;
        // QT, once per tile, while the others wait for the backward products (or right after the loss when there
        // are none): hand over the next tile and start its copies, file this tile, resolve the tile after next
        auto qt_window = [&]() {
            sm->t_next = tq;
            sm->n_next = nq;
            if (tq >= 0) tc_issue_chunk(a, &tmap, sm, tq, 0, min(max(nq, 0), TC_CHUNK), rb ^ 1, true, tile_geo(a, tq, 0));
            const int pos_file = atomicAdd(&st->n_class[on][tile_class(n)], 1);
            tile_publish(a.ta, T, t, n_raw);
            tile_file_at(st, a.order_next, T, oc, on, t, n, pos_file);
            claim(tq, nq);
        };
        // ---- forward: W of every chunk, C accumulated in tensor memory --------------------------
        // (chunk 0's barrier also carries the tile's rows; with nc == 0 it carries only them)
        int rb_last = rb;  // buffer that holds the records of the chunk W currently holds
        bool idle = false;
        for (int c = 0; c < max(nc, 1); ++c) {
            const int cnt = min(TC_CHUNK, n - c * TC_CHUNK);  // 0 when the list is empty
            TCP(0);
            mbar_wait_bounded(&sm->bar_rec[rb], (ph_rec >> rb) & 1u);
            TCP(1);
            ph_rec ^= 1u << rb;
            rb_last = rb;
            if (tid == QT) {  // the next visit's records: the next forward chunk, else the first backward revisit
                if (c + 1 < nc)
                    tc_issue_chunk(a, &tmap, sm, t, (c + 1) * TC_CHUNK, min(TC_CHUNK, n - (c + 1) * TC_CHUNK), rb ^ 1, false, g);
                else if (nc > 1)
                    tc_issue_chunk(a, &tmap, sm, t, (nc - 2) * TC_CHUNK, TC_CHUNK, rb ^ 1, false, g);
            }
            stage_records(a, sm, rb, cnt, tid);
            if (cnt > 0) {
                gen_W(sm->W, sm->rec[rb], cnt, px0, py0, tid);
                if (LOSS) gen_Cb(sm->Cb, sm->rec[rb], cnt, tid);
                proxy_fence();
                tc_fence_before();
                __syncthreads();
                TCP(2);
                if (LOSS) {
                    if (tid == 0) {
                        tc_fence_after();
                        issue_forward(dsc, tmem, cnt, c == 0);
                        umma_commit(&sm->bar_mma);
                    }
                    TCP(3);
                    // W is rewritten by the next chunk, D_f read by the loss: both wait for the products
                    mbar_wait_bounded(&sm->bar_mma, ph_mma);
                    ph_mma ^= 1u;
                    tc_fence_after();
                    TCP(4);
                }
            }
            if (c + 1 < nc) rb ^= 1;
        }
        if (!a.tma_rows && !idle) {
            for (int e = tid; e < TILE_PX * 3; e += TC_THREADS) {
                const int r = e / (TILE * 3), cc = e - r * (TILE * 3);
                const int gy = g.ty * TILE + r, gc = g.tx * TILE * 3 + cc;
                sm->tgt[e] = (gy < a.H && gc < a.W * 3) ? a.image[(size_t)gy * a.W * 3 + gc] : 0.0f;
            }
            __syncthreads();
        }

        // ---- loss: this thread's pixel q = tid: column x, row y ----------------------------------
        float fscale = 1.0f;  // what the backward accumulators must be multiplied with
        if (!idle) {
            const int x = (tid >> 3) & 15, y = 8 * (tid >> 7) + (tid & 7);
            const bool valid = g.tx * TILE + x < a.W && y < g.rows;
            float e[3] = {0.0f, 0.0f, 0.0f};
            float sq = 0.0f;
            if (LOSS) {
                float d[8] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
                if (nc > 0) {  // this pixel half's two accumulators: x W heads, x W tails
                    float d2[8];
                    const unsigned ta = tmem + ((unsigned)((wid & 3) * 32) << 16) + TM_FWD + 32u * (unsigned)(wid >> 2);
                    tmem_ld8(ta, d);
                    tmem_ld8(ta + 16u, d2);
                    tmem_ld_wait();
#pragma unroll
                    for (int i = 0; i < 6; ++i) d[i] += d2[i];
                }
#pragma unroll
                for (int ch = 0; ch < 3; ++ch) {
                    const float cv = (d[ch] + d[3 + ch]) * FWD_UNSCALE;
                    e[ch] = valid ? cv - sm->tgt[y * (TILE * 3) + x * 3 + ch] : 0.0f;
                    sq = fmaf(e[ch], e[ch], sq);
                }
            } else {
#pragma unroll
                for (int ch = 0; ch < 3; ++ch) e[ch] = valid ? sm->tgt[y * (TILE * 3) + x * 3 + ch] : 0.0f;
            }
            // tile-wide max |e| (power-of-two scale of the moment operand) and sum of squares
            unsigned am = __float_as_uint(fmaxf(fmaxf(fabsf(e[0]), fabsf(e[1])), fabsf(e[2])));
            am = __reduce_max_sync(0xffffffffu, am);
#pragma unroll
            for (int dlt = 16; dlt > 0; dlt >>= 1) sq += __shfl_xor_sync(0xffffffffu, sq, dlt);
            if (lane == 0) {
                sm->red_max[wid] = am;
                sm->red_sq[wid] = sq;
            }
            tc_fence_before();
            __syncthreads();
            unsigned amax = 0u;
            float sqt = 0.0f;
#pragma unroll
            for (int k = 0; k < 8; ++k) {
                amax = max(amax, sm->red_max[k]);
                sqt += sm->red_sq[k];
            }
            if (LOSS && tid == 0 && n_raw >= 0) {
                a.tile_stats[t].sq_raw = (double)sqt;
                if (!isfinite(sqt)) {
                    atomicOr(&st->flags, FLAG_NONFINITE);
                    atomicCAS(&st->first_nonfinite_iter, 0, a.iter);
                }
            }
            // scale 2^k with max|e| 2^k in [128, 256): |e phi| 2^k < 256 * 56.25 stays in binary16 range
            int ex = (int)((amax >> 23) & 255u) - 127;
            ex = amax == 0u ? 0 : min(max(ex, -100), 100);
            const float s_up = __uint_as_float((unsigned)(7 - ex + 127) << 23);
            fscale = __uint_as_float((unsigned)(ex - 7 - 10 + 127) << 23) * (LOSS ? a.g_scale : 1.0f);
            if (n > 0) {
                // ---- Bm: row of this pixel: e[ch] phi_k, k = (1, xc, yc, xc^2, xc yc, yc^2) ------------
                const float xc = (float)x - 7.5f, yc = (float)y - 7.5f;
                const float ph[6] = {1.0f, xc, yc, xc * xc, xc * yc, yc * yc};
                unsigned bh[12], bl[12];
#pragma unroll
                for (int j = 0; j < 9; ++j) {  // columns 2j, 2j + 1 of 18 = ch * 6 + k
                    const int c0 = (2 * j) / 6, k0 = (2 * j) % 6, c1 = (2 * j + 1) / 6, k1 = (2 * j + 1) % 6;
                    split_h2(make_float2(e[c0] * s_up * ph[k0], e[c1] * s_up * ph[k1]), bh[j], bl[j]);
                }
                bh[9] = bh[10] = bh[11] = bl[9] = bl[10] = bl[11] = 0u;
                unsigned char *row = sm->Bm + (tid >> 3) * BM_KG + (tid & 7) * 16;
#pragma unroll
                for (int gq = 0; gq < 3; ++gq) {
                    *reinterpret_cast<uint4 *>(row + gq * 128) = make_uint4(bh[4 * gq], bh[4 * gq + 1], bh[4 * gq + 2], bh[4 * gq + 3]);
                    *reinterpret_cast<uint4 *>(row + BM_TAIL + gq * 128) =
                        make_uint4(bl[4 * gq], bl[4 * gq + 1], bl[4 * gq + 2], bl[4 * gq + 3]);
                }
                proxy_fence();
            }
            __syncthreads();  // Bm complete; the rows are dead
        }
        TCP(5);

        // ---- backward: chunks revisited from the last (whose W is still resident) to the first --------
        if (!idle && n > 0) {
            for (int c = nc - 1; c >= 0; --c) {
                const int cnt = min(TC_CHUNK, n - c * TC_CHUNK);
                if (c != nc - 1) {
                    rb ^= 1;
                    mbar_wait_bounded(&sm->bar_rec[rb], (ph_rec >> rb) & 1u);
                    ph_rec ^= 1u << rb;
                    rb_last = rb;
                    if (tid == QT && c > 0) tc_issue_chunk(a, &tmap, sm, t, (c - 1) * TC_CHUNK, TC_CHUNK, rb ^ 1, false, g);
                    stage_records(a, sm, rb, cnt, tid);
                    gen_W(sm->W, sm->rec[rb], cnt, px0, py0, tid);
                    proxy_fence();
                    tc_fence_before();
                    __syncthreads();
                }
                TCP(6);
                if (tid == 0) {
                    tc_fence_after();
                    issue_backward(dsc, tmem);
                    umma_commit(&sm->bar_mma);
                }
                if (tid == QT && c == 0) qt_window();  // the other record buffer and the rows are free
                TCP(7);
                mbar_wait_bounded(&sm->bar_mma, ph_mma);
                ph_mma ^= 1u;
                tc_fence_after();
                TCP(8);
                // accumulator rows: lanes 0-63 heads, 64-127 tails of entry (lane & 63); 18 columns used
                float dv[24];
                if (wid < 4) {
                    const unsigned ta = tmem + ((unsigned)(wid * 32) << 16) + TM_BWD;
#pragma unroll
                    for (int i = 0; i < 24; ++i) dv[i] = 0.0f;
#pragma unroll
                    for (int acc = 0; acc < 4; ++acc) {
                        float r8[8], s8[8];
#pragma unroll
                        for (int q8 = 0; q8 < 3; ++q8) {  // columns 0-23: x Bm heads, 24-47: x Bm tails
                            tmem_ld8(ta + 48u * acc + 8u * q8, r8);
                            tmem_ld8(ta + 48u * acc + 24u + 8u * q8, s8);
                            tmem_ld_wait();
#pragma unroll
                            for (int i = 0; i < 8; ++i) dv[8 * q8 + i] += r8[i] + s8[i];
                        }
                    }
                    if (tid >= 64) {
                        float4 *dst = reinterpret_cast<float4 *>(sm->escr + (tid - 64) * E_STRIDE);
#pragma unroll
                        for (int i = 0; i < 5; ++i) dst[i] = make_float4(dv[4 * i], dv[4 * i + 1], dv[4 * i + 2], dv[4 * i + 3]);
                    }
                }
                tc_fence_before();
                __syncthreads();
                if (tid < cnt) {
                    const int gid = sm->ids[rb_last][tid];
                    {
                        const float4 *src = reinterpret_cast<const float4 *>(sm->escr + tid * E_STRIDE);
#pragma unroll
                        for (int i = 0; i < 5; ++i) {
                            const float4 v = src[i];
                            dv[4 * i] += v.x;
                            dv[4 * i + 1] += v.y;
                            dv[4 * i + 2] += v.z;
                            dv[4 * i + 3] += v.w;
                        }
                        const float4 lo = sm->rec[rb_last][REC_F4 * tid], hi = sm->rec[rb_last][REC_F4 * tid + 1];
                        // polynomial moments of s = w (c'.G) about the tile centre
                        float S[6];
#pragma unroll
                        for (int k = 0; k < 6; ++k) S[k] = fscale * fmaf(hi.w, dv[12 + k], fmaf(hi.z, dv[6 + k], hi.y * dv[k]));
                        const float mx = lo.x - (float)(g.tx * TILE + 8), my = lo.y - (float)(g.ty * TILE + 8);
                        // ... about the Gaussian's centre: d = (xc - mx, yc - my)
                        const float Ax = fmaf(-mx, S[0], S[1]), Ay = fmaf(-my, S[0], S[2]);
                        const float Axx = fmaf(mx, fmaf(mx, S[0], -2.0f * S[1]), S[3]);
                        const float Axy = fmaf(mx, fmaf(my, S[0], -S[2]), fmaf(-my, S[1], S[4]));
                        const float Ayy = fmaf(my, fmaf(my, S[0], -2.0f * S[2]), S[5]);
                        // ... in the record's whitened coordinates u = i1 dx, v = i3 dy + k dx
                        const float i1 = lo.z, kk = lo.w, i3 = hi.x;
                        const float m0 = fscale * dv[0], m1 = fscale * dv[6], m2 = fscale * dv[12];
                        const float m3 = i1 * Ax;
                        const float m4 = fmaf(i3, Ay, kk * Ax);
                        const float m5 = i1 * i1 * Axx;
                        const float m6 = i1 * fmaf(i3, Axy, kk * Axx);
                        const float m7 = fmaf(i3 * i3, Ayy, fmaf(2.0f * i3 * kk, Axy, kk * kk * Axx));
                        float *dst = a.acc + (size_t)gid * 8;
                        asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(dst), "f"(m0), "f"(m1), "f"(m2),
                                     "f"(m3)
                                     : "memory");
                        asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(dst + 4), "f"(m4), "f"(m5),
                                     "f"(m6), "f"(m7)
                                     : "memory");
                    }
                }
                __syncthreads();  // the scratch rows and the record buffer are free
                TCP(9);
            }
        } else if (tid == QT) {
            qt_window();
        }
        __syncthreads();  // t_next / n_next visible (written before the backward pass; read here)
#ifdef TC_PROFILE
        ++tcp_tiles; tcp_pairs += n;
#endif
        t = sm->t_next;
        n_raw = sm->n_next;
        rb ^= 1;
        __syncthreads();  // ... and not overwritten before everybody has read them
    }

#ifdef TC_PROFILE
    if (tid == 0 && (blockIdx.x == 0 || blockIdx.x == 77) && a.iter == 7)
        printf("cta %d tiles %d pairs %d | recwait0 %lld recwait %lld genW %lld fwdissue %lld fwdwait %lld loss+Bm %lld pre-bwd %lld bwdissue %lld bwdwait %lld epiE %lld\n",
               (int)blockIdx.x, tcp_tiles, tcp_pairs, tcp_acc[0], tcp_acc[1], tcp_acc[2], tcp_acc[3], tcp_acc[4], tcp_acc[5], tcp_acc[6], tcp_acc[7], tcp_acc[8], tcp_acc[9]);
#endif
    tc_fence_before();
    __syncthreads();
    if (wid == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 256;" ::"r"(tmem) : "memory");
}

int launch_fit_tc(gs_ctx *c, const FitArgs &a, const CUtensorMap &tmap, FitMode mode, cudaStream_t s) {
    static bool attr_done = false;
    const int smem = (int)sizeof(TcSmem) + 128;
    if (!attr_done) {
        GS_CUDA_TRY(cudaFuncSetAttribute(k_fit_tc<FIT_LOSS>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
        GS_CUDA_TRY(cudaFuncSetAttribute(k_fit_tc<FIT_GRAD>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
        attr_done = true;
    }
    const int grid = min(2 * c->sm_count, c->T);
    if (mode == FIT_GRAD) k_fit_tc<FIT_GRAD><<<grid, TC_THREADS, smem, s>>>(a, tmap);
    else k_fit_tc<FIT_LOSS><<<grid, TC_THREADS, smem, s>>>(a, tmap);
    GS_CUDA_TRY(cudaGetLastError());
    return GS_OK;
}

}  // namespace gs2d
