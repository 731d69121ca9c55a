// gs2d_optim.cu -- gradient finalisation and the fused Adam / mask / projection kernel
// (DESIGN.md §3 c-5, c-6; §5 "optimiser").
#include "gs2d_bin.cuh"

namespace gs2d {

// 1/kappa and 1/kappa^2 with kappa = sqrt(0.5 log2 e): undo the scaling of the record's
// whitened coordinates.
constexpr float INV_KAPPA = 1.17740100225250890f;   // sqrt(2 ln 2)
constexpr float INV_KAPPA2 = 1.38629436111989062f;  // 2 ln 2

// Chain rule from the 8 accumulated moments of one Gaussian to its 9 gradients.
// The backward kernel accumulated, with s' = w (c'.G) and kappa-scaled (u', v'):
//   lo = (R_r, R_g, R_b, sum s' u'),  hi = (sum s' v', sum s' u'^2, sum s' u' v', sum s' v'^2).
// With s = -s' (dC/dsigma = -C) and unscaled u, v (DESIGN.md §3 c-5, whitened form):
//   dL/dmu_x = sum s (-u/l1 + v l2/(l1 l3))      dL/dmu_y = sum s (-v/l3)
//   dL/dl1   = sum s (-u^2/l1 + u v l2/(l1 l3))  dL/dl2 = sum s (-u v/l3)   dL/dl3 = sum s (-v^2/l3)
//   dL/drgb_ch = o R_ch                           dL/do = sum_ch rgb_ch R_ch
__device__ __forceinline__ void moments_to_grad(float4 lo, float4 hi, float l1, float l2, float l3, float r, float g,
                                                float b, float o, float *out) {
    const bool ok = isfinite(l1) && isfinite(l2) && isfinite(l3) && l1 != 0.0f && l3 != 0.0f;
    if (!ok) {
#pragma unroll
        for (int j = 0; j < 9; ++j) out[j] = 0.0f;
        return;
    }
    const float Su = -lo.w * INV_KAPPA, Sv = -hi.x * INV_KAPPA;
    const float Suu = -hi.y * INV_KAPPA2, Suv = -hi.z * INV_KAPPA2, Svv = -hi.w * INV_KAPPA2;
    const float i1 = 1.0f / l1, i3 = 1.0f / l3;
    const float c = l2 * i1 * i3;
    out[0] = fmaf(Sv, c, -Su * i1);
    out[1] = -Sv * i3;
    out[2] = fmaf(Suv, c, -Suu * i1);
    out[3] = -Suv * i3;
    out[4] = -Svv * i3;
    out[5] = o * lo.x;
    out[6] = o * lo.y;
    out[7] = o * lo.z;
    out[8] = fmaf(b, lo.z, fmaf(g, lo.y, r * lo.x));
}

// Deterministic mode: the moments of Gaussian n are the sum of its pairs' slots, in slot (= tile) order.  `ok` is
// false when the binning the slots belong to exceeded a capacity (nothing was written then).
struct PairSlots {
    const int4 *info;   // [N] (first slot, x0 | y0 << 16, width, pairs); null: the atomics' accumulator is used
    const float *mom;   // [P,8]
    int slot;           // epoch parity of that binning
    long long cap_pairs;
};
__device__ __forceinline__ void sum_pair_slots(const PairSlots &ps, const DeviceState *st, int n, float4 &lo, float4 &hi) {
    lo = make_float4(0.f, 0.f, 0.f, 0.f);
    hi = lo;
    const bool ok = st->pair_total[ps.slot] <= (unsigned long long)ps.cap_pairs && st->tile_ovf[ps.slot] == 0;
    if (!ok) return;
    const int4 info = ps.info[n];
    const float4 *src = reinterpret_cast<const float4 *>(ps.mom) + 2 * (size_t)info.x;
    for (int k = 0; k < info.w; ++k) {
        const float4 a = src[2 * k], b = src[2 * k + 1];
        lo.x += a.x, lo.y += a.y, lo.z += a.z, lo.w += a.w;
        hi.x += b.x, hi.y += b.y, hi.z += b.z, hi.w += b.w;
    }
}

__global__ void __launch_bounds__(256)
    k_grad_finalize(int N, const float *__restrict__ mu, const float *__restrict__ chol, const float *__restrict__ rgb,
                    const float *__restrict__ opacity, float *__restrict__ acc, float *__restrict__ g_mu,
                    float *__restrict__ g_chol, float *__restrict__ g_rgb, float *__restrict__ g_op, QuantDev q,
                    PairSlots ps, const DeviceState *__restrict__ st) {
    int n = blockIdx.x * blockDim.x + threadIdx.x;
    if (n >= N) return;
    float4 lo, hi;
    if (ps.info) {
        sum_pair_slots(ps, st, n, lo, hi);
    } else {
        float4 *a = reinterpret_cast<float4 *>(acc + (size_t)n * 8);
        lo = a[0], hi = a[1];
        a[0] = make_float4(0.f, 0.f, 0.f, 0.f);  // acc is zero between passes
        a[1] = make_float4(0.f, 0.f, 0.f, 0.f);
    }
    float out[9];
    // (QAT: the gradient is taken where the render was evaluated, at the quantised parameters)
    moments_to_grad(lo, hi, fake_quant(q, 2, chol[3 * n]), fake_quant(q, 3, chol[3 * n + 1]),
                    fake_quant(q, 4, chol[3 * n + 2]), fake_quant(q, 5, rgb[3 * n]), fake_quant(q, 6, rgb[3 * n + 1]),
                    fake_quant(q, 7, rgb[3 * n + 2]), fake_quant(q, 8, opacity[n]), out);
    g_mu[2 * n] = out[0];
    g_mu[2 * n + 1] = out[1];
    g_chol[3 * n] = out[2];
    g_chol[3 * n + 1] = out[3];
    g_chol[3 * n + 2] = out[4];
    g_rgb[3 * n] = out[5];
    g_rgb[3 * n + 1] = out[6];
    g_rgb[3 * n + 2] = out[7];
    g_op[n] = out[8];
}

struct AdamArgs {
    float lr[4];
    float beta1, beta2, eps, ibc1, ibc2, l_min;  // ibc = 1 / (1 - beta^t)
};

__device__ __forceinline__ float fast_sqrt(float x) {
    float r;
    asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}

// FROM_ACC = true : gradients come from the moment accumulator (fit loop; a8 fused into a9),
//                   which is zeroed for the next iteration; the step is skipped once a
//                   non-finite loss has been latched (the oracle's loop stops there).
// FROM_ACC = false: gradients are the caller's arrays (gs_adam_step).
// One CTA owns ADAM_THREADS consecutive Gaussians.  The [n,9] moment arrays and the [n,3]
// parameter arrays are moved between global and shared memory with coalesced float4 / float
// accesses of the CTA's contiguous slab; each thread then works on its own Gaussian out of
// shared memory (odd strides 9 and 3: no bank conflicts).
constexpr int ADAM_THREADS = 128;  // Gaussians per CTA
// Threads per CTA: the second half does no Adam arithmetic; it doubles the copies and the counting atomics in
// flight (the kernel is latency-bound at ~10 warps per SM: one thread per Gaussian is too few)
constexpr int ADAM_CTA = 256;

// global -> shared copy of the CTA's slab with cp.async (LDGSTS): every 16-byte piece of every array is in flight
// before the first one is waited for.  (Written as load-then-store loops the pieces went one DRAM round trip after
// the other -- the store of piece i stalls on its load before the load of piece i + 1 issues: 19 of the kernel's 22 us.)
__device__ __forceinline__ void cp_async16(void *smem_dst, const void *gsrc) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"((unsigned)__cvta_generic_to_shared(smem_dst)), "l"(gsrc)
                 : "memory");
}
__device__ __forceinline__ void cp_async4(void *smem_dst, const void *gsrc) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"((unsigned)__cvta_generic_to_shared(smem_dst)), "l"(gsrc)
                 : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }
template <int PER, bool VEC>
__device__ __forceinline__ void slab_load(float *s, const float *__restrict__ g, int n0, int cnt, int tid) {
    const float *src = g + (size_t)n0 * PER;
    const int tot = cnt * PER;
    if (VEC && cnt == ADAM_THREADS) {
#pragma unroll
        for (int i = tid; i < ADAM_THREADS * PER / 4; i += ADAM_CTA)
            cp_async16(reinterpret_cast<float4 *>(s) + i, reinterpret_cast<const float4 *>(src) + i);
    } else {
        for (int i = tid; i < tot; i += ADAM_CTA) cp_async4(s + i, src + i);
    }
}
template <int PER, bool VEC>
__device__ __forceinline__ void slab_store(float *__restrict__ g, const float *s, int n0, int cnt, int tid) {
    float *dst = g + (size_t)n0 * PER;
    const int tot = cnt * PER;
    if (VEC && cnt == ADAM_THREADS) {
        for (int i = tid; i < ADAM_THREADS * PER / 4; i += ADAM_CTA)
            reinterpret_cast<float4 *>(dst)[i] = reinterpret_cast<const float4 *>(s)[i];
    } else {
        for (int i = tid; i < tot; i += ADAM_CTA) dst[i] = s[i];
    }
}

// REBIN: after the update the kernel bins the parameters it holds (updated or frozen) for the
// next iteration -- record, tile rectangle and bucket arrivals of gs2d_bin.cuh -- so that the
// next iteration starts at its forward pass.
template <bool FROM_ACC, bool REBIN>
__global__ void __launch_bounds__(ADAM_CTA)
    k_adam(int N, float *__restrict__ mu, float *__restrict__ chol, float *__restrict__ rgb,
           float *__restrict__ opacity, float *__restrict__ m, float *__restrict__ v, float *__restrict__ acc,
           const float *__restrict__ g_mu, const float *__restrict__ g_chol, const float *__restrict__ g_rgb,
           const float *__restrict__ g_op, AdamArgs a, const unsigned char *__restrict__ active,
           const DeviceState *__restrict__ st, BinArgs ba, PairSlots ps) {
    __shared__ __align__(16) float s_m[ADAM_THREADS * 9], s_v[ADAM_THREADS * 9];
    __shared__ __align__(16) float s_chol[ADAM_THREADS * 3], s_rgb[ADAM_THREADS * 3];
    __shared__ __align__(16) float s_gc[FROM_ACC ? 4 : ADAM_THREADS * 3], s_gr[FROM_ACC ? 4 : ADAM_THREADS * 3];
    __shared__ BinSmem<REBIN ? ADAM_CTA : 32> s_bin;
    const int tid = threadIdx.x;
    const int n0 = blockIdx.x * ADAM_THREADS;
    const int cnt = min(ADAM_THREADS, N - n0);
    const int n = n0 + tid;
    const bool mine = tid < cnt;

    float4 lo = make_float4(0.f, 0.f, 0.f, 0.f), hi = lo;
    if (FROM_ACC) {
        if (mine && !ps.info) {
            float4 *ac = reinterpret_cast<float4 *>(acc + (size_t)n * 8);
            lo = ac[0];
            hi = ac[1];
            ac[0] = make_float4(0.f, 0.f, 0.f, 0.f);
            ac[1] = make_float4(0.f, 0.f, 0.f, 0.f);
        }
    }
    // once a non-finite loss has been latched the updates stop (the oracle's loop stops there)
    const bool dead = FROM_ACC && st->first_nonfinite_iter != 0;  // uniform over the grid
    slab_load<9, true>(s_m, m, n0, cnt, tid);
    slab_load<9, true>(s_v, v, n0, cnt, tid);
    slab_load<3, true>(s_chol, chol, n0, cnt, tid);
    slab_load<3, true>(s_rgb, rgb, n0, cnt, tid);
    if (!FROM_ACC) {
        slab_load<3, true>(s_gc, g_chol, n0, cnt, tid);
        slab_load<3, true>(s_gr, g_rgb, n0, cnt, tid);
    }
    // deterministic mode: the slots of this Gaussian's pairs, in order (read before the re-binning below replaces
    // this Gaussian's entry of the pair table)
    if (FROM_ACC && ps.info && mine) sum_pair_slots(ps, st, n, lo, hi);
    float2 pm = make_float2(0.f, 0.f), gm = pm;
    float po = 0.f, go = 0.f;
    bool act = false;
    if (mine) {
        pm = reinterpret_cast<const float2 *>(mu)[n];
        po = opacity[n];
        act = (active ? active[n] != 0 : true) && !dead;
        if (!FROM_ACC) {
            gm = reinterpret_cast<const float2 *>(g_mu)[n];
            go = g_op[n];
        }
    }
    cp_async_wait_all();
    __syncthreads();

    float th[9];
#pragma unroll
    for (int j = 0; j < 9; ++j) th[j] = 0.0f;
    if (mine) {
        th[0] = pm.x;
        th[1] = pm.y;
        th[2] = s_chol[3 * tid];
        th[3] = s_chol[3 * tid + 1];
        th[4] = s_chol[3 * tid + 2];
        th[5] = s_rgb[3 * tid];
        th[6] = s_rgb[3 * tid + 1];
        th[7] = s_rgb[3 * tid + 2];
        th[8] = po;
    }
    if (mine && act) {  // frozen Gaussians: parameters and moments untouched
        float g[9];
        if (FROM_ACC) {
            // QAT: chain rule at the quantised parameters the render saw; the gradient goes straight
            // through to the raw parameters
            moments_to_grad(lo, hi, fake_quant(ba.q, 2, th[2]), fake_quant(ba.q, 3, th[3]), fake_quant(ba.q, 4, th[4]),
                            fake_quant(ba.q, 5, th[5]), fake_quant(ba.q, 6, th[6]), fake_quant(ba.q, 7, th[7]),
                            fake_quant(ba.q, 8, th[8]), g);
        } else {
            g[0] = gm.x;
            g[1] = gm.y;
            g[2] = s_gc[3 * tid];
            g[3] = s_gc[3 * tid + 1];
            g[4] = s_gc[3 * tid + 2];
            g[5] = s_gr[3 * tid];
            g[6] = s_gr[3 * tid + 1];
            g[7] = s_gr[3 * tid + 2];
            g[8] = go;
        }
        const float omb1 = 1.0f - a.beta1, omb2 = 1.0f - a.beta2;
#pragma unroll
        for (int j = 0; j < 9; ++j) {
            const float lr = a.lr[j < 2 ? 0 : (j < 5 ? 1 : (j < 8 ? 2 : 3))];
            float mj = fmaf(a.beta1, s_m[9 * tid + j], omb1 * g[j]);
            float vj = fmaf(a.beta2, s_v[9 * tid + j], omb2 * g[j] * g[j]);
            s_m[9 * tid + j] = mj;
            s_v[9 * tid + j] = vj;
            // (bias corrections as reciprocals, MUFU square root and reciprocal: a few ulp, against
            // a step tolerance of 1e-4 relative -- DESIGN.md §3 tolerances)
            const float mhat = mj * a.ibc1, vhat = vj * a.ibc2;
            th[j] -= __fdividef(lr * mhat, fast_sqrt(vhat) + a.eps);
        }
        th[2] = fmaxf(th[2], a.l_min);  // projection: l1, l3 >= l_min (DESIGN.md §3 #3)
        th[4] = fmaxf(th[4], a.l_min);
        reinterpret_cast<float2 *>(mu)[n] = make_float2(th[0], th[1]);
        s_chol[3 * tid] = th[2];
        s_chol[3 * tid + 1] = th[3];
        s_chol[3 * tid + 2] = th[4];
        s_rgb[3 * tid] = th[5];
        s_rgb[3 * tid + 1] = th[6];
        s_rgb[3 * tid + 2] = th[7];
        opacity[n] = th[8];
    }
    __syncthreads();
    // untouched rows are written back with the values that were read: bit-identical
    if (!dead) {
        slab_store<9, true>(m, s_m, n0, cnt, tid);
        slab_store<9, true>(v, s_v, n0, cnt, tid);
        slab_store<3, true>(chol, s_chol, n0, cnt, tid);
        slab_store<3, true>(rgb, s_rgb, n0, cnt, tid);
    }
    if (REBIN)
        bin_cta<ADAM_CTA>(ba, reinterpret_cast<BinSmem<ADAM_CTA> &>(s_bin), mine, n, th[0], th[1], th[2], th[3],
                              th[4], th[5], th[6], th[7], th[8]);
}

__global__ void __launch_bounds__(256)
    k_fake_quantize(int N, const float *__restrict__ mu, const float *__restrict__ chol, const float *__restrict__ rgb,
                    const float *__restrict__ opacity, float *__restrict__ o_mu, float *__restrict__ o_chol,
                    float *__restrict__ o_rgb, float *__restrict__ o_op, QuantDev q) {
    const int n = blockIdx.x * blockDim.x + threadIdx.x;
    if (n >= N) return;
    o_mu[2 * n] = fake_quant(q, 0, mu[2 * n]);
    o_mu[2 * n + 1] = fake_quant(q, 1, mu[2 * n + 1]);
#pragma unroll
    for (int j = 0; j < 3; ++j) {
        o_chol[3 * n + j] = fake_quant(q, 2 + j, chol[3 * n + j]);
        o_rgb[3 * n + j] = fake_quant(q, 5 + j, rgb[3 * n + j]);
    }
    o_op[n] = fake_quant(q, 8, opacity[n]);
}

// the slot table of the binning the context last ran (deterministic mode; info == null otherwise)
static PairSlots pair_slots(const gs_ctx *c) {
    PairSlots ps;
    ps.info = c->deterministic ? c->pair_info : nullptr;
    ps.mom = c->pair_mom;
    ps.slot = (int)(c->epoch & 1u);
    ps.cap_pairs = c->cap_pairs;
    return ps;
}

int launch_fake_quantize(gs_ctx *c, const gs_params &p, const gs_params &out, const QuantDev &q, cudaStream_t s) {
    k_fake_quantize<<<ceil_div(p.n, 256), 256, 0, s>>>(p.n, p.mu, p.chol, p.rgb, p.opacity, out.mu, out.chol, out.rgb,
                                                      out.opacity, q);
    GS_CUDA_TRY(cudaGetLastError());
    return GS_OK;
}

int launch_grad_finalize(gs_ctx *c, const gs_params &p, const gs_params &g, cudaStream_t s) {
    k_grad_finalize<<<ceil_div(p.n, 256), 256, 0, s>>>(p.n, p.mu, p.chol, p.rgb, p.opacity, c->acc, g.mu, g.chol,
                                                      g.rgb, g.opacity, c->quant, pair_slots(c), c->dstate);
    GS_CUDA_TRY(cudaGetLastError());
    return GS_OK;
}

int launch_adam(gs_ctx *c, const gs_params &p, const gs_params *grad, const gs_adam_state &st, const float lr[4],
                float beta1, float beta2, float eps, float bc1, float bc2, const unsigned char *active, bool rebin,
                cudaStream_t s) {
    AdamArgs a;
    for (int i = 0; i < 4; ++i) a.lr[i] = lr[i];
    a.beta1 = beta1;
    a.beta2 = beta2;
    a.eps = eps;
    a.ibc1 = (float)(1.0 / (double)bc1);
    a.ibc2 = (float)(1.0 / (double)bc2);
    a.l_min = c->cfg.l_min;
    const int blocks = ceil_div(p.n, ADAM_THREADS);
    if (grad) {
        k_adam<false, false><<<blocks, ADAM_CTA, 0, s>>>(p.n, p.mu, p.chol, p.rgb, p.opacity, st.m, st.v, nullptr,
                                                             grad->mu, grad->chol, grad->rgb, grad->opacity, a, active,
                                                             c->dstate, BinArgs{}, PairSlots{});
    } else if (rebin) {
        discard_fresh_bins(c, s);  // (never fresh here: the forward pass of this iteration consumed them)
        const PairSlots ps = pair_slots(c);  // of the binning the backward pass has just consumed
        // selective refit: only the active Gaussians are listed (the frozen ones live in the fit target)
        const BinArgs ba = bin_args(c, true, active, 1);
        k_adam<true, true><<<blocks, ADAM_CTA, 0, s>>>(p.n, p.mu, p.chol, p.rgb, p.opacity, st.m, st.v, c->acc,
                                                           nullptr, nullptr, nullptr, nullptr, a, active, c->dstate, ba,
                                                           ps);
        c->fresh = true;
        c->fresh_mu = p.mu;
        c->fresh_n = p.n;
        c->fresh_active = active;
        c->fresh_mode = active ? 1 : 0;
    } else {
        BinArgs bq{};
        bq.q = c->quant;  // (no binning here, but the chain rule needs the quantisers)
        k_adam<true, false><<<blocks, ADAM_CTA, 0, s>>>(p.n, p.mu, p.chol, p.rgb, p.opacity, st.m, st.v, c->acc,
                                                            nullptr, nullptr, nullptr, nullptr, a, active, c->dstate,
                                                            bq, pair_slots(c));
    }
    GS_CUDA_TRY(cudaGetLastError());
    return GS_OK;
}

}  // namespace gs2d
