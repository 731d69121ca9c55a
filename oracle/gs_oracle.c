/*
 * gs_oracle.c -- ORACLE.  TEST INFRASTRUCTURE ONLY.
 *
 * A plain, slow, float64 CPU restatement of the hot path of the 2D Gaussian
 * Splatting ROI video codec of arXiv 2505.09324 (reference text: PAPER.md; the
 * readings of its gaps: SURVEY.md §8(c), restated in DESIGN.md §3).  It exists so
 * that the CUDA library under paper_2505_09324_b200/ can be checked against
 * something that can be read against the paper by eye.  It shares no code,
 * header, table or helper with the CUDA path and must never be imported by it.
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
 * reference legs may load this file.
 *
 * What is exact and what is not: the method is an iteration (Adam fit) around a
 * tile-truncated sum (Eq. 2 restricted to each 16x16 tile's list), so the oracle
 * follows the algorithm step by step in the paper's notation:
 *
 *   c-1  Sigma = L L^T, L = [[l1,0],[l2,l3]]                     PAPER.md:38-43 Eq. 1
 *   c-2  binning rule in single-rounded binary32 (bit-exact)
 *   c-3  C_i = sum_{n in list(tile(i))} c'_n exp(-sigma_n)         PAPER.md:50-52 Eq. 2
 *        sigma_n = 1/2 d^T Sigma^-1 d, evaluated in whitened form SPEC.md:152
 *   c-4  L = mean((C-T)^2), G = dL/dC, PSNR on the clamped image
 *   c-5  analytic gradients, whitened per-pixel form
 *   c-6  Adam + active mask + projection l1,l3 >= l_min
 *   c-7  fit loop
 *   c-8  ROI-weighted initialiser                                 BASELINE.json configs[1]
 *   c-9  P-frame tile-residual selection + masked refit
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): SPEC.md worked values, the closed
 * form  sum_p c' exp(-sigma) = 2 pi sqrt(det Sigma) c', scipy's multivariate
 * normal pdf, torch autograd (float64) on a dense restatement of Eq. 2, central
 * finite differences, torch.optim.Adam, brute-force binning / selection.
 * Unpinned readings (free choices): l_min projection value,
 * zeroing of Adam state per frame, the full-frame P-frame loss region.
 *
 * Everything floating point is double except (i) the binning rule, which is
 * DEFINED as a sequence of single-rounded binary32 operations so that it can be
 * compared bit for bit (compile with -ffp-contract=off), and (ii) the few
 * binary32 steps of the ROI initialiser that are defined the same way.
 *
 * OpenMP is used only as "for each tile" / "for each Gaussian" over independent
 * outputs; there is no blocking, fusion or reordering of the arithmetic.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define TILE 16

static int g_threads = 0; /* 0 = OpenMP default */

void gso_set_threads(int n) { g_threads = n; }
int gso_get_threads(void) {
#ifdef _OPENMP
    return g_threads > 0 ? g_threads : omp_get_max_threads();
#else
    return 1;
#endif
}
#ifdef _OPENMP
#define NTHREADS() (g_threads > 0 ? g_threads : omp_get_max_threads())
#else
#define NTHREADS() 1
#endif

/* ------------------------------------------------------------------ c-1 */

/* Sigma = L L^T (Eq. 1).  S = {S11, S12, S21, S22}. */
void gso_cov_from_chol(const double *l, double *S) {
    double l1 = l[0], l2 = l[1], l3 = l[2];
    S[0] = l1 * l1;
    S[1] = l1 * l2;
    S[2] = l1 * l2;
    S[3] = l2 * l2 + l3 * l3;
}

/* Sigma^-1 = [[a,b],[b,c]] in closed form from l. */
void gso_inverse_cov(const double *l, double *abc) {
    double l1 = l[0], l2 = l[1], l3 = l[2];
    abc[0] = (l2 * l2 + l3 * l3) / (l1 * l1 * l3 * l3);
    abc[1] = -l2 / (l1 * l3 * l3);
    abc[2] = 1.0 / (l3 * l3);
}

/* sigma = 1/2 d^T Sigma^-1 d through the whitened coordinates
 * (u,v) = L^-1 d :  u = dx/l1, v = (dy - l2 u)/l3, sigma = (u^2+v^2)/2. */
static inline double sigma_whitened(double dx, double dy, double l1, double l2, double l3,
                                    double *u_out, double *v_out) {
    double u = dx / l1;
    double v = (dy - l2 * u) / l3;
    if (u_out) *u_out = u;
    if (v_out) *v_out = v;
    return 0.5 * (u * u + v * v);
}

double gso_sigma(double dx, double dy, const double *l) {
    return sigma_whitened(dx, dy, l[0], l[1], l[2], 0, 0);
}

/* ------------------------------------------------------------------ c-2 */

/* Tile rectangle of one Gaussian.  Every operation is binary32, round to
 * nearest, one rounding each (no fused multiply-add).  Returns 1 if culled.
 *   rx = k|l1| ; ry = k sqrt(l2*l2 + l3*l3)
 *   lo = mu - r ; hi = mu + r
 *   culled iff an input is non-finite, l1 = 0, l3 = 0,
 *              hi_x < 0, lo_x >= W, hi_y < 0 or lo_y >= H
 *   tx0 = max(0, floor(lo_x/16)), tx1 = min(TX-1, floor(hi_x/16)); same in y. */
static int tile_rect_f32(float mux, float muy, float l1, float l2, float l3, float k,
                         int W, int H, int *r /* tx0,ty0,tx1,ty1 */) {
    int TX = (W + TILE - 1) / TILE, TY = (H + TILE - 1) / TILE;
    r[0] = r[1] = 0;
    r[2] = r[3] = -1;
    if (!isfinite(mux) || !isfinite(muy) || !isfinite(l1) || !isfinite(l2) || !isfinite(l3)) return 1;
    if (l1 == 0.0f || l3 == 0.0f) return 1;
    float rx = k * fabsf(l1);
    float p22 = l2 * l2;
    float p33 = l3 * l3;
    float s22 = p22 + p33;
    float ry = k * sqrtf(s22);
    float lo_x = mux - rx, hi_x = mux + rx;
    float lo_y = muy - ry, hi_y = muy + ry;
    if (hi_x < 0.0f || lo_x >= (float)W || hi_y < 0.0f || lo_y >= (float)H) return 1;
    float fx0 = fmaxf(0.0f, floorf(lo_x * 0.0625f));
    float fx1 = fminf((float)(TX - 1), floorf(hi_x * 0.0625f));
    float fy0 = fmaxf(0.0f, floorf(lo_y * 0.0625f));
    float fy1 = fminf((float)(TY - 1), floorf(hi_y * 0.0625f));
    r[0] = (int)fx0;
    r[1] = (int)fy0;
    r[2] = (int)fx1;
    r[3] = (int)fy1;
    return 0;
}

/* Pixel footprint half-widths, reported for the pins. */
void gso_footprint_halfwidths(const double *l, double cutoff, float *rx_ry) {
    float l1 = (float)l[0], l2 = (float)l[1], l3 = (float)l[2], k = (float)cutoff;
    rx_ry[0] = k * fabsf(l1);
    float p22 = l2 * l2, p33 = l3 * l3;
    float s22 = p22 + p33;
    rx_ry[1] = k * sqrtf(s22);
}

/* rect4[n] = {tx0,ty0,tx1,ty1} (tx1 < tx0 when culled).  Parameters are rounded
 * to binary32 first: that is the precision the rule is defined in. */
static void all_rects(int W, int H, int N, const double *mu, const double *chol, double cutoff, int *rect4) {
    for (int n = 0; n < N; ++n)
        tile_rect_f32((float)mu[2 * n], (float)mu[2 * n + 1], (float)chol[3 * n], (float)chol[3 * n + 1],
                      (float)chol[3 * n + 2], (float)cutoff, W, H, rect4 + 4 * n);
}

/* Canonical bins: range[T+1] exclusive prefix of per-tile counts, list[P] by tile
 * id ascending then Gaussian id ascending.  list may be NULL (count only).
 * Returns 0, or -1 if cap < P. */
int gso_bin(int W, int H, int N, const double *mu, const double *chol, double cutoff,
            int *rect4, int *range, int *list, long long cap, long long *P_out) {
    int TX = (W + TILE - 1) / TILE, TY = (H + TILE - 1) / TILE, T = TX * TY;
    all_rects(W, H, N, mu, chol, cutoff, rect4);
    long long *cnt = (long long *)calloc((size_t)T + 1, sizeof(long long));
    for (int n = 0; n < N; ++n) {
        const int *r = rect4 + 4 * n;
        for (int ty = r[1]; ty <= r[3]; ++ty)
            for (int tx = r[0]; tx <= r[2]; ++tx) cnt[ty * TX + tx]++;
    }
    long long acc = 0;
    for (int t = 0; t < T; ++t) {
        range[t] = (int)acc;
        acc += cnt[t];
    }
    range[T] = (int)acc;
    *P_out = acc;
    if (list) {
        if (cap < acc) {
            free(cnt);
            return -1;
        }
        for (int t = 0; t < T; ++t) cnt[t] = range[t];
        for (int n = 0; n < N; ++n) { /* ascending n => ascending id inside every tile */
            const int *r = rect4 + 4 * n;
            for (int ty = r[1]; ty <= r[3]; ++ty)
                for (int tx = r[0]; tx <= r[2]; ++tx) list[cnt[ty * TX + tx]++] = n;
        }
    }
    free(cnt);
    return 0;
}

/* ------------------------------------------------------------------ c-3 */

typedef struct {
    int W, H, TX, TY, T, N;
    int *rect4, *range, *list;
} bins_t;

static int make_bins(bins_t *b, int W, int H, int N, const double *mu, const double *chol, double cutoff) {
    b->W = W;
    b->H = H;
    b->N = N;
    b->TX = (W + TILE - 1) / TILE;
    b->TY = (H + TILE - 1) / TILE;
    b->T = b->TX * b->TY;
    b->rect4 = (int *)malloc(sizeof(int) * 4 * (size_t)(N > 0 ? N : 1));
    b->range = (int *)malloc(sizeof(int) * ((size_t)b->T + 1));
    long long P = 0;
    gso_bin(W, H, N, mu, chol, cutoff, b->rect4, b->range, NULL, 0, &P);
    b->list = (int *)malloc(sizeof(int) * (size_t)(P > 0 ? P : 1));
    return gso_bin(W, H, N, mu, chol, cutoff, b->rect4, b->range, b->list, P, &P);
}
static void free_bins(bins_t *b) {
    free(b->rect4);
    free(b->range);
    free(b->list);
}

/* Eq. 2 for one pixel over an id list (ascending id); c' = o*c. */
static inline void pixel_sum(double px, double py, const int *ids, int cnt, int dense_N, const double *mu,
                             const double *chol, const double *rgb, const double *op, double *C) {
    double c0 = 0.0, c1 = 0.0, c2 = 0.0;
    int m = ids ? cnt : dense_N;
    for (int j = 0; j < m; ++j) {
        int n = ids ? ids[j] : j;
        double dx = px - mu[2 * n], dy = py - mu[2 * n + 1];
        double sg = sigma_whitened(dx, dy, chol[3 * n], chol[3 * n + 1], chol[3 * n + 2], 0, 0);
        double w = exp(-sg);
        double o = op[n];
        c0 += (o * rgb[3 * n + 0]) * w;
        c1 += (o * rgb[3 * n + 1]) * w;
        c2 += (o * rgb[3 * n + 2]) * w;
    }
    C[0] = c0;
    C[1] = c1;
    C[2] = c2;
}

/* Render, UNCLAMPED (the loss sees the unclamped sum).
 * dense = 0: every pixel sums the Gaussians in its tile's list.
 * dense = 1: every pixel sums all N Gaussians (closed forms, finite differences).
 * tiles/ntiles: if tiles != NULL only those tile ids are rendered, the rest of
 * image is left untouched. */
int gso_render(int W, int H, int N, const double *mu, const double *chol, const double *rgb, const double *op,
               int dense, double cutoff, const int *tiles, int ntiles, double *image) {
    bins_t b;
    memset(&b, 0, sizeof b);
    b.TX = (W + TILE - 1) / TILE;
    b.TY = (H + TILE - 1) / TILE;
    b.T = b.TX * b.TY;
    if (!dense) make_bins(&b, W, H, N, mu, chol, cutoff);
    int nt = tiles ? ntiles : b.T;
#pragma omp parallel for schedule(dynamic, 1) num_threads(NTHREADS())
    for (int k = 0; k < nt; ++k) {
        int t = tiles ? tiles[k] : k;
        int tx = t % b.TX, ty = t / b.TX;
        const int *ids = dense ? NULL : b.list + b.range[t];
        int cnt = dense ? 0 : b.range[t + 1] - b.range[t];
        for (int y = ty * TILE; y < ty * TILE + TILE && y < H; ++y)
            for (int x = tx * TILE; x < tx * TILE + TILE && x < W; ++x)
                pixel_sum(x + 0.5, y + 0.5, ids, cnt, N, mu, chol, rgb, op, image + 3 * ((size_t)y * W + x));
    }
    if (!dense) free_bins(&b);
    return 0;
}

/* ------------------------------------------------------------------ c-4 */

/* L = (1/(3WH)) sum (C-T)^2 on the unclamped C; G = dL/dC = 2(C-T)/(3WH). */
double gso_loss(int W, int H, const double *image, const float *target, double *G) {
    size_t n = (size_t)W * H * 3;
    double inv = 1.0 / (double)n;
    double acc = 0.0;
    for (size_t i = 0; i < n; ++i) {
        double d = image[i] - (double)target[i];
        acc += d * d;
        if (G) G[i] = 2.0 * d * inv;
    }
    return acc * inv;
}

/* PSNR = 10 log10(1/MSE) on clamp(C,0,1); 99 dB ceiling. */
double gso_psnr(int W, int H, const double *image, const float *target) {
    size_t n = (size_t)W * H * 3;
    double acc = 0.0;
    for (size_t i = 0; i < n; ++i) {
        double c = image[i] < 0.0 ? 0.0 : (image[i] > 1.0 ? 1.0 : image[i]);
        double d = c - (double)target[i];
        acc += d * d;
    }
    double mse = acc / (double)n;
    if (!(mse > 0.0)) return 99.0;
    double p = 10.0 * log10(1.0 / mse);
    return p > 99.0 ? 99.0 : p;
}

/* ------------------------------------------------------------------ c-5 */

/* Gradients of  sum_p sum_ch G_ch(p) C_ch(p)  with respect to the 9 scalars of
 * each Gaussian, layout grad[n] = (mu_x, mu_y, l1, l2, l3, r, g, b, o).
 * Per pixel, whitened form:  w = exp(-sigma), q = sum_ch c'_ch G_ch, s = -w q
 *   d sigma/d mu_x = -u/l1 + v l2/(l1 l3)      d sigma/d mu_y = -v/l3
 *   d sigma/d l1   = -u^2/l1 + u v l2/(l1 l3)  d sigma/d l2 = -u v/l3
 *   d sigma/d l3   = -v^2/l3
 *   dL/d theta = sum_p s d sigma/d theta ; dL/dc_ch = o sum_p w G_ch ;
 *   dL/do = sum_p w sum_ch c_ch G_ch.
 * List membership is treated as constant (almost-everywhere derivative).
 * Summation domain of Gaussian n: the valid pixels of every tile of its rectangle
 * (dense = 1: every pixel).  gsub/nsub: restrict to a subset of Gaussians (the
 * other rows of grad are left untouched). */
int gso_backward(int W, int H, int N, const double *mu, const double *chol, const double *rgb, const double *op,
                 const double *G, int dense, double cutoff, const int *gsub, int nsub, double *grad) {
    int TX = (W + TILE - 1) / TILE, TY = (H + TILE - 1) / TILE;
    int *rect4 = (int *)malloc(sizeof(int) * 4 * (size_t)(N > 0 ? N : 1));
    all_rects(W, H, N, mu, chol, cutoff, rect4);
    int cnt = gsub ? nsub : N;
#pragma omp parallel for schedule(dynamic, 16) num_threads(NTHREADS())
    for (int k = 0; k < cnt; ++k) {
        int n = gsub ? gsub[k] : k;
        double *g = grad + 9 * (size_t)n;
        for (int j = 0; j < 9; ++j) g[j] = 0.0;
        int r[4] = {rect4[4 * n], rect4[4 * n + 1], rect4[4 * n + 2], rect4[4 * n + 3]};
        if (dense) {
            r[0] = 0;
            r[1] = 0;
            r[2] = TX - 1;
            r[3] = TY - 1;
            if (chol[3 * n] == 0.0 || chol[3 * n + 2] == 0.0) continue;
        }
        double l1 = chol[3 * n], l2 = chol[3 * n + 1], l3 = chol[3 * n + 2];
        double o = op[n], cr = rgb[3 * n], cg = rgb[3 * n + 1], cb = rgb[3 * n + 2];
        for (int ty = r[1]; ty <= r[3]; ++ty)
            for (int tx = r[0]; tx <= r[2]; ++tx)
                for (int y = ty * TILE; y < ty * TILE + TILE && y < H; ++y)
                    for (int x = tx * TILE; x < tx * TILE + TILE && x < W; ++x) {
                        const double *Gp = G + 3 * ((size_t)y * W + x);
                        double dx = (x + 0.5) - mu[2 * n], dy = (y + 0.5) - mu[2 * n + 1];
                        double u, v;
                        double sg = sigma_whitened(dx, dy, l1, l2, l3, &u, &v);
                        double w = exp(-sg);
                        double q = (o * cr) * Gp[0] + (o * cg) * Gp[1] + (o * cb) * Gp[2];
                        double s = -w * q;
                        g[0] += s * (-u / l1 + v * l2 / (l1 * l3));
                        g[1] += s * (-v / l3);
                        g[2] += s * (-u * u / l1 + u * v * l2 / (l1 * l3));
                        g[3] += s * (-u * v / l3);
                        g[4] += s * (-v * v / l3);
                        g[5] += o * w * Gp[0];
                        g[6] += o * w * Gp[1];
                        g[7] += o * w * Gp[2];
                        g[8] += w * (cr * Gp[0] + cg * Gp[1] + cb * Gp[2]);
                    }
    }
    free(rect4);
    return 0;
}

/* ------------------------------------------------------------------ c-6 */

/* One Adam step (torch.optim.Adam convention, no weight decay, no amsgrad):
 *   m <- b1 m + (1-b1) g ; v <- b2 v + (1-b2) g^2
 *   theta <- theta - lr_group (m/(1-b1^t)) / (sqrt(v/(1-b2^t)) + eps)
 * groups: mu (lr[0]), chol (lr[1]), rgb (lr[2]), opacity (lr[3]).
 * active[n] = 0: parameters and moments of n untouched.  Afterwards
 * l1 <- max(l1, l_min), l3 <- max(l3, l_min).  m, v, grad are [N,9] in the
 * gradient layout. */
void gso_adam(int N, double *mu, double *chol, double *rgb, double *op, const double *grad, double *m, double *v,
              const double *lr, double b1, double b2, double eps, int t, const unsigned char *active,
              double l_min) {
    double bc1 = 1.0 - pow(b1, (double)t), bc2 = 1.0 - pow(b2, (double)t);
    for (int n = 0; n < N; ++n) {
        if (active && !active[n]) continue;
        double *theta[9] = {mu + 2 * n,       mu + 2 * n + 1,  chol + 3 * n,    chol + 3 * n + 1, chol + 3 * n + 2,
                            rgb + 3 * n,      rgb + 3 * n + 1, rgb + 3 * n + 2, op + n};
        const double group_lr[9] = {lr[0], lr[0], lr[1], lr[1], lr[1], lr[2], lr[2], lr[2], lr[3]};
        for (int j = 0; j < 9; ++j) {
            double g = grad[9 * (size_t)n + j];
            double *mj = m + 9 * (size_t)n + j, *vj = v + 9 * (size_t)n + j;
            *mj = b1 * (*mj) + (1.0 - b1) * g;
            *vj = b2 * (*vj) + (1.0 - b2) * g * g;
            double mhat = *mj / bc1, vhat = *vj / bc2;
            *theta[j] -= group_lr[j] * mhat / (sqrt(vhat) + eps);
        }
        if (chol[3 * n] < l_min) chol[3 * n] = l_min;
        if (chol[3 * n + 2] < l_min) chol[3 * n + 2] = l_min;
    }
}

/* ------------------------------------------------------------------ c-7 */

/* Fit loop.  Moments are zeroed and t restarts at 1.  Iteration k: bin(theta_k)
 * -> C -> L, G -> gradients -> theta_{k+1}.  After the last iteration one more
 * bin + render gives final loss and PSNR.  loss_trace (nullable) has iters+1
 * entries: the loss seen by each iteration, then the final loss.
 * first_nonfinite: 1-based iteration whose loss was not finite, else 0. */
int gso_fit_roi(int W, int H, int N, double *mu, double *chol, double *rgb, double *op, double *m, double *v,
                const float *target, const unsigned char *roi, int iters, const double *lr, double b1, double b2,
                double eps, const unsigned char *active, double l_min, double cutoff, double *loss_trace,
                double *final_loss, double *psnr, int *first_nonfinite);
int gso_fit(int W, int H, int N, double *mu, double *chol, double *rgb, double *op, double *m, double *v,
            const float *target, int iters, const double *lr, double b1, double b2, double eps,
            const unsigned char *active, double l_min, double cutoff, double *loss_trace, double *final_loss,
            double *psnr, int *first_nonfinite) {
    return gso_fit_roi(W, H, N, mu, chol, rgb, op, m, v, target, NULL, iters, lr, b1, b2, eps, active, l_min, cutoff,
                       loss_trace, final_loss, psnr, first_nonfinite);
}

/* ------------------------------------------------------------------ c-16 */

/* ROI-restricted loss (the paper's codec encodes "only the region of interest"; SPEC.md:260
 * "mean squared error over masked pixels", :283, :286 "early-stop metric is masked PSNR"; DESIGN.md §3 c-16).
 * With M the set of pixels whose mask byte is non-zero:
 *     L = (1 / (3 |M|)) sum_{p in M} sum_ch (C - T)^2   on the unclamped C;
 *     G = dL/dC = 2 (C - T) / (3 |M|) inside M, 0 outside;
 *     PSNR = 10 log10(1 / MSE) of the clamped image over M, 99 dB ceiling.
 * roi == NULL is c-4 (every pixel).  An empty ROI has no loss: the functions return NaN. */
long long gso_roi_count(int W, int H, const unsigned char *roi) {
    long long c = 0;
    for (size_t p = 0; p < (size_t)W * H; ++p) c += roi[p] ? 1 : 0;
    return c;
}
double gso_loss_roi(int W, int H, const double *image, const float *target, const unsigned char *roi, double *G) {
    if (!roi) return gso_loss(W, H, image, target, G);
    const long long cnt = gso_roi_count(W, H, roi);
    if (cnt == 0) return NAN;
    const double inv = 1.0 / (3.0 * (double)cnt);
    double acc = 0.0;
    for (size_t p = 0; p < (size_t)W * H; ++p)
        for (int ch = 0; ch < 3; ++ch) {
            const size_t i = 3 * p + ch;
            const double d = image[i] - (double)target[i];
            if (roi[p]) acc += d * d;
            if (G) G[i] = roi[p] ? 2.0 * d * inv : 0.0;
        }
    return acc * inv;
}
double gso_psnr_roi(int W, int H, const double *image, const float *target, const unsigned char *roi) {
    if (!roi) return gso_psnr(W, H, image, target);
    const long long cnt = gso_roi_count(W, H, roi);
    if (cnt == 0) return NAN;
    double acc = 0.0;
    for (size_t p = 0; p < (size_t)W * H; ++p)
        if (roi[p])
            for (int ch = 0; ch < 3; ++ch) {
                const size_t i = 3 * p + ch;
                const double c = image[i] < 0.0 ? 0.0 : (image[i] > 1.0 ? 1.0 : image[i]);
                const double d = c - (double)target[i];
                acc += d * d;
            }
    const double mse = acc / (3.0 * (double)cnt);
    if (!(mse > 0.0)) return 99.0;
    const double ps = 10.0 * log10(1.0 / mse);
    return ps > 99.0 ? 99.0 : ps;
}

/* The c-7 loop with the loss of c-16 (roi == NULL: c-4, the loop every other function of this file calls). */
int gso_fit_roi(int W, int H, int N, double *mu, double *chol, double *rgb, double *op, double *m, double *v,
                const float *target, const unsigned char *roi, int iters, const double *lr, double b1, double b2,
                double eps, const unsigned char *active, double l_min, double cutoff, double *loss_trace,
                double *final_loss, double *psnr, int *first_nonfinite) {
    size_t npx = (size_t)W * H * 3;
    double *image = (double *)malloc(sizeof(double) * npx);
    double *G = (double *)malloc(sizeof(double) * npx);
    double *grad = (double *)malloc(sizeof(double) * 9 * (size_t)N);
    memset(m, 0, sizeof(double) * 9 * (size_t)N);
    memset(v, 0, sizeof(double) * 9 * (size_t)N);
    *first_nonfinite = 0;
    for (int k = 1; k <= iters; ++k) {
        gso_render(W, H, N, mu, chol, rgb, op, 0, cutoff, NULL, 0, image);
        double L = gso_loss_roi(W, H, image, target, roi, G);
        if (loss_trace) loss_trace[k - 1] = L;
        if (!isfinite(L) && *first_nonfinite == 0) {
            *first_nonfinite = k;
            break;
        }
        gso_backward(W, H, N, mu, chol, rgb, op, G, 0, cutoff, NULL, 0, grad);
        gso_adam(N, mu, chol, rgb, op, grad, m, v, lr, b1, b2, eps, k, active, l_min);
    }
    gso_render(W, H, N, mu, chol, rgb, op, 0, cutoff, NULL, 0, image);
    *final_loss = gso_loss_roi(W, H, image, target, roi, NULL);
    if (loss_trace) loss_trace[iters] = *final_loss;
    *psnr = gso_psnr_roi(W, H, image, target, roi);
    free(image);
    free(G);
    free(grad);
    return 0;
}

/* ------------------------------------------------------------------ c-8 */

/* Counter-based generator: SplitMix64 finaliser applied to
 * seed + (8 i + k + 1) * 0x9E3779B97F4A7C15  (sample i, stream k in 0..7). */
static uint64_t rnd64(uint64_t seed, uint64_t i, uint64_t k) {
    uint64_t z = seed + (8u * i + k + 1u) * 0x9E3779B97F4A7C15ULL;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
    return z ^ (z >> 31);
}
uint64_t gso_rnd64(uint64_t seed, uint64_t i, uint64_t k) { return rnd64(seed, i, k); }

static inline int clampi(int v, int lo, int hi) { return v < lo ? lo : (v > hi ? hi : v); }

/* Integer sampling weights: q_ch = floor(255 x_ch + 0.5) in two
 * single-rounded binary32 operations, grey = q_r+q_g+q_b, 3x3 Sobel with
 * clamp-to-edge borders, weight = isqrt(gx^2+gy^2) + 1 inside the ROI.
 * w_in[p] (0 outside the ROI) and w_out[p] (1 outside the ROI, 0 inside). */
void gso_roi_weights(int W, int H, const float *frame, const unsigned char *mask, int *w_in, int *w_out) {
    int *grey = (int *)malloc(sizeof(int) * (size_t)W * H);
    for (size_t p = 0; p < (size_t)W * H; ++p) {
        int s = 0;
        for (int ch = 0; ch < 3; ++ch) {
            float t = 255.0f * frame[3 * p + ch];
            float r = t + 0.5f;
            s += (int)floorf(r);
        }
        grey[p] = s;
    }
    for (int y = 0; y < H; ++y)
        for (int x = 0; x < W; ++x) {
            size_t p = (size_t)y * W + x;
            if (!mask[p]) {
                w_in[p] = 0;
                w_out[p] = 1;
                continue;
            }
            int xm = clampi(x - 1, 0, W - 1), xp = clampi(x + 1, 0, W - 1);
            int ym = clampi(y - 1, 0, H - 1), yp = clampi(y + 1, 0, H - 1);
#define GR(yy, xx) grey[(size_t)(yy) * W + (xx)]
            int gx = (GR(ym, xp) + 2 * GR(y, xp) + GR(yp, xp)) - (GR(ym, xm) + 2 * GR(y, xm) + GR(yp, xm));
            int gy = (GR(yp, xm) + 2 * GR(yp, x) + GR(yp, xp)) - (GR(ym, xm) + 2 * GR(ym, x) + GR(ym, xp));
#undef GR
            long long m2 = (long long)gx * gx + (long long)gy * gy;
            long long r = (long long)floor(sqrt((double)m2));
            while (r * r > m2) --r;
            while ((r + 1) * (r + 1) <= m2) ++r;
            w_in[p] = (int)r + 1;
            w_out[p] = 0;
        }
    free(grey);
}

/* ROI-weighted initialiser.  Returns 0, -3 for an empty ROI, -1 for bad args.
 * pix_out (nullable) receives the sampled row-major pixel index of each Gaussian.
 * Outputs are binary32: position, colour copy and opacity bit-exact by
 * definition; l computed in double here then rounded (the CUDA path evaluates
 * exp/sin/cos in binary32; parity 1e-5 relative). */
int gso_init_roi(int W, int H, const float *frame, const unsigned char *mask, int N, uint64_t seed, double s_min,
                 double s_max, float *mu, float *chol, float *rgb, float *op, long long *pix_out) {
    if (W <= 0 || H <= 0 || N < 1 || !(s_min > 0.0) || !(s_max >= s_min)) return -1;
    size_t np = (size_t)W * H;
    int *w_in = (int *)malloc(sizeof(int) * np), *w_out = (int *)malloc(sizeof(int) * np);
    gso_roi_weights(W, H, frame, mask, w_in, w_out);
    uint64_t *c_in = (uint64_t *)malloc(sizeof(uint64_t) * np), *c_out = (uint64_t *)malloc(sizeof(uint64_t) * np);
    uint64_t a = 0, b = 0;
    for (size_t p = 0; p < np; ++p) { /* inclusive prefix sums, row-major */
        a += (uint64_t)w_in[p];
        b += (uint64_t)w_out[p];
        c_in[p] = a;
        c_out[p] = b;
    }
    int rc = 0;
    if (a == 0) {
        rc = -3; /* empty ROI */
    } else {
        int N_in = (int)((7LL * N) / 10);
        if (b == 0) N_in = N; /* no outside pixels: all inside */
        const double PI = 3.14159265358979323846;
        for (int i = 0; i < N; ++i) {
            const uint64_t *c = i < N_in ? c_in : c_out;
            uint64_t total = i < N_in ? a : b;
            uint64_t target = rnd64(seed, (uint64_t)i, 0) % total;
            size_t lo = 0, hi = np - 1; /* first p with c[p] > target */
            while (lo < hi) {
                size_t mid = lo + (hi - lo) / 2;
                if (c[mid] > target) hi = mid;
                else lo = mid + 1;
            }
            size_t p = lo;
            int x = (int)(p % (size_t)W), y = (int)(p / (size_t)W);
            float jx = (float)(rnd64(seed, (uint64_t)i, 1) >> 40) * 0x1p-24f - 0.5f; /* exact in binary32 */
            float jy = (float)(rnd64(seed, (uint64_t)i, 2) >> 40) * 0x1p-24f - 0.5f;
            float cxp = (float)x + 0.5f, cyp = (float)y + 0.5f; /* exact */
            mu[2 * i] = cxp + jx;                               /* one rounding */
            mu[2 * i + 1] = cyp + jy;
            rgb[3 * i] = frame[3 * p];
            rgb[3 * i + 1] = frame[3 * p + 1];
            rgb[3 * i + 2] = frame[3 * p + 2];
            op[i] = 1.0f;
            double u1 = (double)(rnd64(seed, (uint64_t)i, 3) >> 40) * 0x1p-24;
            double u2 = (double)(rnd64(seed, (uint64_t)i, 4) >> 40) * 0x1p-24;
            double u3 = (double)(rnd64(seed, (uint64_t)i, 5) >> 40) * 0x1p-24;
            double ls = log(s_max / s_min);
            double s1 = s_min * exp(u1 * ls), s2 = s_min * exp(u2 * ls), th = PI * u3;
            double ct = cos(th), st = sin(th);
            /* Sigma = R diag(s1^2, s2^2) R^T, then its Cholesky factor */
            double S11 = ct * ct * s1 * s1 + st * st * s2 * s2;
            double S12 = ct * st * (s1 * s1 - s2 * s2);
            double S22 = st * st * s1 * s1 + ct * ct * s2 * s2;
            double l1 = sqrt(S11), l2 = S12 / l1, l3 = sqrt(S22 - l2 * l2);
            chol[3 * i] = (float)l1;
            chol[3 * i + 1] = (float)l2;
            chol[3 * i + 2] = (float)l3;
            if (pix_out) pix_out[i] = (long long)p;
        }
    }
    free(w_in);
    free(w_out);
    free(c_in);
    free(c_out);
    return rc;
}

/* ------------------------------------------------------------------ c-9 */

/* P-frame selection:
 *  1 bin + render the previous Gaussians, clamp to [0,1]
 *  2 r_t = mean over the tile's valid pixels and 3 channels of |frame - render|
 *  3 tile changed iff r_t > tau (strict)
 *  4 active[n] = 1 iff n is in the list of at least one changed tile */
int gso_pframe_select(int W, int H, int N, const double *mu, const double *chol, const double *rgb,
                      const double *op, const float *frame, double tau, double cutoff, double *tile_resid,
                      unsigned char *tile_flag, unsigned char *active, int *n_active) {
    size_t npx = (size_t)W * H * 3;
    double *image = (double *)malloc(sizeof(double) * npx);
    gso_render(W, H, N, mu, chol, rgb, op, 0, cutoff, NULL, 0, image);
    bins_t b;
    make_bins(&b, W, H, N, mu, chol, cutoff);
    memset(active, 0, (size_t)N);
    for (int t = 0; t < b.T; ++t) {
        int tx = t % b.TX, ty = t / b.TX;
        double acc = 0.0;
        long long cnt = 0;
        for (int y = ty * TILE; y < ty * TILE + TILE && y < H; ++y)
            for (int x = tx * TILE; x < tx * TILE + TILE && x < W; ++x)
                for (int ch = 0; ch < 3; ++ch) {
                    size_t i = 3 * ((size_t)y * W + x) + ch;
                    double c = image[i] < 0.0 ? 0.0 : (image[i] > 1.0 ? 1.0 : image[i]);
                    acc += fabs((double)frame[i] - c);
                    ++cnt;
                }
        double r = acc / (double)cnt;
        if (tile_resid) tile_resid[t] = r;
        unsigned char f = r > tau ? 1 : 0;
        if (tile_flag) tile_flag[t] = f;
        if (f)
            for (int j = b.range[t]; j < b.range[t + 1]; ++j) active[b.list[j]] = 1;
    }
    int na = 0;
    for (int n = 0; n < N; ++n) na += active[n];
    *n_active = na;
    free_bins(&b);
    free(image);
    return 0;
}

/* c-9 with an ROI (c-16): r_t = mean of |frame - render| over the tile's ROI pixels and 3 channels; a tile without
 * ROI pixels has r_t = 0 and is never changed.  roi == NULL: c-9. */
int gso_pframe_select_roi(int W, int H, int N, const double *mu, const double *chol, const double *rgb,
                          const double *op, const float *frame, const unsigned char *roi, double tau, double cutoff,
                          double *tile_resid, unsigned char *tile_flag, unsigned char *active, int *n_active) {
    if (!roi)
        return gso_pframe_select(W, H, N, mu, chol, rgb, op, frame, tau, cutoff, tile_resid, tile_flag, active, n_active);
    size_t npx = (size_t)W * H * 3;
    double *image = (double *)malloc(sizeof(double) * npx);
    gso_render(W, H, N, mu, chol, rgb, op, 0, cutoff, NULL, 0, image);
    bins_t b;
    make_bins(&b, W, H, N, mu, chol, cutoff);
    memset(active, 0, (size_t)N);
    for (int t = 0; t < b.T; ++t) {
        int tx = t % b.TX, ty = t / b.TX;
        double acc = 0.0;
        long long cnt = 0;
        for (int y = ty * TILE; y < ty * TILE + TILE && y < H; ++y)
            for (int x = tx * TILE; x < tx * TILE + TILE && x < W; ++x) {
                if (!roi[(size_t)y * W + x]) continue;
                for (int ch = 0; ch < 3; ++ch) {
                    size_t i = 3 * ((size_t)y * W + x) + ch;
                    double c = image[i] < 0.0 ? 0.0 : (image[i] > 1.0 ? 1.0 : image[i]);
                    acc += fabs((double)frame[i] - c);
                    ++cnt;
                }
            }
        double r = cnt > 0 ? acc / (double)cnt : 0.0;
        if (tile_resid) tile_resid[t] = r;
        unsigned char f = r > tau ? 1 : 0;
        if (tile_flag) tile_flag[t] = f;
        if (f)
            for (int j = b.range[t]; j < b.range[t + 1]; ++j) active[b.list[j]] = 1;
    }
    int na = 0;
    for (int n = 0; n < N; ++n) na += active[n];
    *n_active = na;
    free_bins(&b);
    free(image);
    return 0;
}

/* P-frame encode: select, then (if anything is active) the c-7 loop with that
 * fixed mask, full-frame loss, moments zeroed.  Empty selection: parameters are
 * returned untouched and zero iterations run. */
int gso_encode_pframe(int W, int H, int N, double *mu, double *chol, double *rgb, double *op, double *m, double *v,
                      const float *frame, double tau, int iters, const double *lr, double b1, double b2,
                      double eps, double l_min, double cutoff, unsigned char *active, int *n_active,
                      int *iters_run, double *final_loss, double *psnr, int *first_nonfinite) {
    gso_pframe_select(W, H, N, mu, chol, rgb, op, frame, tau, cutoff, NULL, NULL, active, n_active);
    *iters_run = 0;
    *first_nonfinite = 0;
    if (*n_active == 0) {
        size_t npx = (size_t)W * H * 3;
        double *image = (double *)malloc(sizeof(double) * npx);
        gso_render(W, H, N, mu, chol, rgb, op, 0, cutoff, NULL, 0, image);
        *final_loss = gso_loss(W, H, image, frame, NULL);
        *psnr = gso_psnr(W, H, image, frame);
        free(image);
        return 0;
    }
    gso_fit(W, H, N, mu, chol, rgb, op, m, v, frame, iters, lr, b1, b2, eps, active, l_min, cutoff, NULL, final_loss,
            psnr, first_nonfinite);
    *iters_run = iters;
    return 0;
}

/* ---------------------------------------------------------------------------------------------
 * c-11  Superpixel initialiser (the paper's content-aware I-frame initialisation, PAPER.md:66-68:
 *       "segmented into N superpixel segments using a K-means clustering-based superpixel
 *       algorithm ... Gaussian means are computed as the center of each superpixel, the Cholesky
 *       decomposition is derived from the covariance matrix of each segment, and the RGB colors
 *       are calculated as the average pixel color"; SPEC.md:182-200 instantiates it as SLIC).
 *
 * The reading (DESIGN.md §3 c-11) is stated in INTEGER arithmetic so that labels are exact:
 *   features of ROI pixel (x, y), in 1/16 units:  X = 16 x + 8, Y = 16 y + 8 (the pixel centre),
 *     R, G, B = 16 * floor(255 v + 0.5)  (v the binary32 frame value, two single-rounded ops)
 *   grid: the ROI's bounding box (x0, y0)-(x1, y1), bw x bh pixels, is cut into GX x GY cells,
 *     GY = max(1, round(GX bh / bw)) (cells about square), pixel (x, y) lying in cell
 *     cx = (x - x0) GX / bw, cy = (y - y0) GY / bh (integer division).  GX is the largest value in
 *     [1, bw] -- found by bisection, K taken as non-decreasing in GX -- for which the number K of
 *     cells that hold an ROI pixel is <= N ("segmented into N superpixel segments": the
 *     count should approach N); if even GX = 1 gives K > N the grid is 1 x 1.  Cluster
 *     k = cy * GX + cx is the cell (cx, cy); cells without ROI pixels have no cluster.
 *     S2 = max(1, bw bh / (GX GY)) is the cell area (the square of SLIC's grid step).
 *   seed of a cell: its ROI pixel nearest the cell centre: with lo, hi the first and last pixel
 *     offset of the cell along x, ex = 2 (x - x0) - lo - hi (same in y), d = ex^2 + ey^2, ties to
 *     the smallest row-major pixel index; the initial centre is that pixel.
 *   iteration (kmeans_iters times): every ROI pixel takes, among the clusters of the 3 x 3 cells
 *     around its own cell, the one minimising
 *         D = S2 (dR^2 + dG^2 + dB^2) + m^2 (dX^2 + dY^2)       (64-bit integers; m = compactness)
 *     ties to the smallest k; then every cluster's centre becomes the rounded mean of its pixels,
 *     (sum + count/2) / count per feature; a cluster that lost all pixels keeps its centre.
 *   Gaussians: clusters with pixels, in ascending k: mu = mean pixel centre; Sigma = covariance of
 *     the member pixels seen as unit squares = point covariance + I/12 (the SPEC.md:198 example:
 *     a 10 x 10 square gives 100/12 = 8.25 + 1/12); l = chol(Sigma); colour = mean of
 *     floor(65536 v + 0.5)/65536; opacity 1.
 * labels_out[H*W]: index of the pixel's Gaussian in the output, -1 outside the ROI.
 * Returns the number of Gaussians (<= N), or -1 bad argument, -3 empty ROI. */
static inline int q255(float v) { return (int)floorf(255.0f * v + 0.5f); }

int gso_init_superpixel(int W, int H, const float *frame, const unsigned char *mask, int N, int m_compact, int iters,
                        float *mu_out, float *chol_out, float *rgb_out, float *op_out, int *labels_out,
                        int *S_out) {
    if (W <= 0 || H <= 0 || N < 1 || m_compact < 0 || iters < 0) return -1;
    long long A = 0;
    int x0 = W, y0 = H, x1 = -1, y1 = -1;
    for (int y = 0; y < H; ++y)
        for (int x = 0; x < W; ++x)
            if (mask[(size_t)y * W + x]) {
                ++A;
                if (x < x0) x0 = x;
                if (x > x1) x1 = x;
                if (y < y0) y0 = y;
                if (y > y1) y1 = y;
            }
    if (A == 0) return -3;
    const int bw = x1 - x0 + 1, bh = y1 - y0 + 1;
    int GX = 1, GY = 1, K = 0;
    unsigned char *has = (unsigned char *)malloc((size_t)bw * bh);
    /* bisection for the largest GX whose grid has at most N occupied cells */
    int lo = 0, hi = bw; /* lo = 0: "not even GX = 1" */
    while (lo < hi) {
        const int mid = (lo + hi + 1) / 2;
        const int gy = (int)(((long long)2 * mid * bh + bw) / (2LL * bw)) > 1 ? (int)(((long long)2 * mid * bh + bw) / (2LL * bw)) : 1;
        memset(has, 0, (size_t)mid * gy);
        int k = 0;
        for (int y = y0; y <= y1; ++y)
            for (int x = x0; x <= x1; ++x)
                if (mask[(size_t)y * W + x]) {
                    unsigned char *h = &has[(size_t)(((long long)(y - y0) * gy) / bh) * mid + ((long long)(x - x0) * mid) / bw];
                    if (!*h) {
                        *h = 1;
                        ++k;
                    }
                }
        if (k <= N) lo = mid;
        else hi = mid - 1;
    }
    if (lo >= 1) {
        GX = lo;
        GY = (int)(((long long)2 * GX * bh + bw) / (2LL * bw));
        if (GY < 1) GY = 1;
    }
    memset(has, 0, (size_t)GX * GY);
    for (int y = y0; y <= y1; ++y)
        for (int x = x0; x <= x1; ++x)
            if (mask[(size_t)y * W + x]) {
                unsigned char *h = &has[(size_t)(((long long)(y - y0) * GY) / bh) * GX + ((long long)(x - x0) * GX) / bw];
                if (!*h) {
                    *h = 1;
                    ++K;
                }
            }
    if (S_out) {
        S_out[0] = GX;
        S_out[1] = GY;
    }
    const int C = GX * GY;
    long long (*cen)[5] = (long long (*)[5])calloc((size_t)C, sizeof *cen);
    long long (*sum)[6] = (long long (*)[6])calloc((size_t)C, sizeof *sum);
    long long *best = (long long *)malloc(sizeof(long long) * (size_t)C);
    int *label = (int *)malloc(sizeof(int) * (size_t)W * H);
    for (int k = 0; k < C; ++k) best[k] = -1;
    /* seeds */
    for (int y = y0; y <= y1; ++y)
        for (int x = x0; x <= x1; ++x) {
            if (!mask[(size_t)y * W + x]) continue;
            const int cx = (int)(((long long)(x - x0) * GX) / bw), cy = (int)(((long long)(y - y0) * GY) / bh);
            const int k = cy * GX + cx;
            const long long lox = ((long long)cx * bw + GX - 1) / GX, hix = ((long long)(cx + 1) * bw + GX - 1) / GX - 1;
            const long long loy = ((long long)cy * bh + GY - 1) / GY, hiy = ((long long)(cy + 1) * bh + GY - 1) / GY - 1;
            const long long ex = 2 * (x - x0) - lox - hix, ey = 2 * (y - y0) - loy - hiy;
            const long long d = ex * ex + ey * ey;
            const long long idx = (long long)y * W + x;
            /* row-major scan: a later pixel replaces the seed only if strictly nearer */
            if (best[k] < 0 || d < (best[k] >> 32)) {
                best[k] = (d << 32) | idx;
                const float *px = frame + ((size_t)y * W + x) * 3;
                cen[k][0] = 16 * x + 8;
                cen[k][1] = 16 * y + 8;
                cen[k][2] = 16 * q255(px[0]);
                cen[k][3] = 16 * q255(px[1]);
                cen[k][4] = 16 * q255(px[2]);
            }
        }
    const long long S2 = ((long long)bw * bh) / ((long long)GX * GY) > 1 ? ((long long)bw * bh) / ((long long)GX * GY) : 1;
    const long long M2 = (long long)m_compact * m_compact;
    for (int it = 0; it <= iters; ++it) { /* the last pass only assigns: labels of the final centres */
        memset(sum, 0, sizeof(*sum) * (size_t)C);
        for (int y = 0; y < H; ++y)
            for (int x = 0; x < W; ++x) {
                const size_t p = (size_t)y * W + x;
                if (!mask[p]) {
                    label[p] = -1;
                    continue;
                }
                const float *px = frame + p * 3;
                const long long f[5] = {16 * x + 8, 16 * y + 8, 16 * q255(px[0]), 16 * q255(px[1]), 16 * q255(px[2])};
                const int cx = (int)(((long long)(x - x0) * GX) / bw), cy = (int)(((long long)(y - y0) * GY) / bh);
                long long bd = -1;
                int bk = -1;
                for (int dy = -1; dy <= 1; ++dy)
                    for (int dx = -1; dx <= 1; ++dx) {
                        const int ux = cx + dx, uy = cy + dy;
                        if (ux < 0 || uy < 0 || ux >= GX || uy >= GY) continue;
                        const int k = uy * GX + ux;
                        if (!has[k]) continue;
                        const long long ddx = f[0] - cen[k][0], ddy = f[1] - cen[k][1], dr = f[2] - cen[k][2],
                                        dg = f[3] - cen[k][3], db = f[4] - cen[k][4];
                        const long long D = S2 * (dr * dr + dg * dg + db * db) + M2 * (ddx * ddx + ddy * ddy);
                        if (bk < 0 || D < bd || (D == bd && k < bk)) {
                            bd = D;
                            bk = k;
                        }
                    }
                label[p] = bk;
                for (int j = 0; j < 5; ++j) sum[bk][j] += f[j];
                sum[bk][5] += 1;
            }
        if (it == iters) break;
        for (int k = 0; k < C; ++k)
            if (sum[k][5] > 0)
                for (int j = 0; j < 5; ++j) cen[k][j] = (sum[k][j] + sum[k][5] / 2) / sum[k][5];
    }
    /* Gaussians from the segments */
    int *out_index = (int *)malloc(sizeof(int) * (size_t)C);
    int n_out = 0;
    for (int k = 0; k < C; ++k) out_index[k] = sum[k][5] > 0 ? n_out++ : -1;
    double (*st)[8] = (double (*)[8])calloc((size_t)(n_out > 0 ? n_out : 1), sizeof *st);
    for (int y = 0; y < H; ++y)
        for (int x = 0; x < W; ++x) {
            const size_t p = (size_t)y * W + x;
            if (label[p] < 0) {
                if (labels_out) labels_out[p] = -1;
                continue;
            }
            const int g = out_index[label[p]];
            if (labels_out) labels_out[p] = g;
            const double X = x + 0.5, Y = y + 0.5;
            const float *px = frame + p * 3;
            st[g][0] += X;
            st[g][1] += Y;
            st[g][2] += X * X;
            st[g][3] += X * Y;
            st[g][4] += Y * Y;
            for (int c = 0; c < 3; ++c) st[g][5 + c] += floor(65536.0 * (double)px[c] + 0.5);
        }
    for (int k = 0; k < C; ++k) {
        const int g = out_index[k];
        if (g < 0) continue;
        const double n = (double)sum[k][5];
        const double mx = st[g][0] / n, my = st[g][1] / n;
        const double sxx = st[g][2] / n - mx * mx + 1.0 / 12.0, sxy = st[g][3] / n - mx * my,
                     syy = st[g][4] / n - my * my + 1.0 / 12.0;
        const double l1 = sqrt(sxx), l2 = sxy / l1, l3 = sqrt(syy - l2 * l2);
        mu_out[2 * g] = (float)mx;
        mu_out[2 * g + 1] = (float)my;
        chol_out[3 * g] = (float)l1;
        chol_out[3 * g + 1] = (float)l2;
        chol_out[3 * g + 2] = (float)l3;
        for (int c = 0; c < 3; ++c) rgb_out[3 * g + c] = (float)(st[g][5 + c] / (65536.0 * n));
        op_out[g] = 1.0f;
    }
    free(has);
    free(cen);
    free(sum);
    free(best);
    free(label);
    free(out_index);
    free(st);
    return n_out;
}

/* ---------------------------------------------------------------------------------------------
 * c-13  Pixel-granular P-frame selection ("isolating pixels that exceed a
 *       user-defined change threshold. For these identified pixels, the metadata from the
 *       reference frame is utilized to locate all Gaussians that influence the changing pixels";
 *       SPEC.md:303-341).  SURVEY.md §8(f) next #2; DESIGN.md §3 c-13.
 *   1 bin and render the previous Gaussians, clamp to [0,1]                       (as c-9)
 *   2 pixel changed iff max over channels |frame - render| > tau (strict)
 *     optionally dilated by one pixel (3x3, inside the frame)
 *   3 Gaussian n influences pixel p iff n is listed in p's tile and exp(-sigma_n(p)) >= eps
 *     (default eps 0.01), sigma in float64 through the whitened coordinates of c-1
 *     (sigma_whitened, the function the render uses).  No binary32 arithmetic, no scaled record:
 *     the decision is the definition written out.
 *   4 active[n] = 1 iff n influences at least one changed pixel.
 * wmax_out (nullable): per Gaussian the LARGEST exp(-sigma) over the changed pixels of its listed
 * tiles (0 when there is none), so that a parity test can tell a knife-edge decision (wmax within
 * rounding of eps: a binary32 implementation may legitimately fall on either side) from a wrong one.
 * changed_in (nullable): use this change map instead of steps 1-2 (parity tests feed both sides
 * the same map).  changed_out, resid_out (max-channel residual per pixel): nullable. */
int gso_pframe_select_pixels(int W, int H, int N, const double *mu, const double *chol, const double *rgb,
                             const double *op, const float *frame, double tau, double eps, int dilate, double cutoff,
                             const unsigned char *changed_in, unsigned char *changed_out, double *resid_out,
                             unsigned char *active, double *wmax_out, int *n_active) {
    const size_t npix = (size_t)W * H;
    unsigned char *changed = (unsigned char *)calloc(npix, 1);
    if (changed_in) {
        memcpy(changed, changed_in, npix);
    } else {
        double *image = (double *)malloc(sizeof(double) * npix * 3);
        gso_render(W, H, N, mu, chol, rgb, op, 0, cutoff, NULL, 0, image);
        unsigned char *raw = (unsigned char *)calloc(npix, 1);
        for (size_t p = 0; p < npix; ++p) {
            double r = 0.0;
            for (int ch = 0; ch < 3; ++ch) {
                double c = image[3 * p + ch];
                c = c < 0.0 ? 0.0 : (c > 1.0 ? 1.0 : c);
                double d = fabs((double)frame[3 * p + ch] - c);
                if (d > r) r = d;
            }
            if (resid_out) resid_out[p] = r;
            raw[p] = r > tau ? 1 : 0;
        }
        for (int y = 0; y < H; ++y)
            for (int x = 0; x < W; ++x) {
                unsigned char f = raw[(size_t)y * W + x];
                if (dilate && !f)
                    for (int dy = -1; dy <= 1 && !f; ++dy)
                        for (int dx = -1; dx <= 1 && !f; ++dx) {
                            int yy = y + dy, xx = x + dx;
                            if (yy >= 0 && yy < H && xx >= 0 && xx < W && raw[(size_t)yy * W + xx]) f = 1;
                        }
                changed[(size_t)y * W + x] = f;
            }
        free(raw);
        free(image);
    }
    if (changed_out) memcpy(changed_out, changed, npix);
    bins_t b;
    make_bins(&b, W, H, N, mu, chol, cutoff);
    memset(active, 0, (size_t)N);
    double *wmax = (double *)calloc((size_t)(N > 0 ? N : 1), sizeof(double));
    for (int t = 0; t < b.T; ++t) {
        const int tx = t % b.TX, ty = t / b.TX;
        for (int j = b.range[t]; j < b.range[t + 1]; ++j) {
            const int n = b.list[j];
            const double l1 = chol[3 * n], l2 = chol[3 * n + 1], l3 = chol[3 * n + 2];
            for (int y = ty * TILE; y < ty * TILE + TILE && y < H; ++y)
                for (int x = tx * TILE; x < tx * TILE + TILE && x < W; ++x) {
                    if (!changed[(size_t)y * W + x]) continue;
                    const double dx = ((double)x + 0.5) - mu[2 * n], dy = ((double)y + 0.5) - mu[2 * n + 1];
                    const double w = exp(-sigma_whitened(dx, dy, l1, l2, l3, 0, 0));
                    if (w > wmax[n]) wmax[n] = w;
                }
        }
    }
    for (int n = 0; n < N; ++n) active[n] = wmax[n] >= eps ? 1 : 0;
    if (wmax_out) memcpy(wmax_out, wmax, sizeof(double) * (size_t)N);
    free(wmax);
    int na = 0;
    for (int n = 0; n < N; ++n) na += active[n];
    *n_active = na;
    free_bins(&b);
    free(changed);
    return 0;
}
