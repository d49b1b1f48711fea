/*
 * wbmm_ref.c -- CPU ORACLE for the WBMM operator.  TEST INFRASTRUCTURE ONLY.
 *
 * This file is the plain, slow, obviously-correct statement of what the GPU
 * library must compute.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may build, load or call it.  It shares
 * no code, header, table or helper with paper_2607_02097_b200/csrc.
 *
 * Everything is fp64 (inputs, accumulation, outputs).  Callers round their
 * inputs to the case dtype BEFORE widening to double; the oracle never rounds.
 *
 * What it follows (PAPER.md = /root/reference/PAPER.md at authoring time):
 *   - relative position index I[i,j]            PAPER.md:188-193  (Eq. 6-7)
 *   - weight construction  M = R[:, I]          PAPER.md:195-198  (Eq. 8)
 *   - zero padding to a multiple of w, crop     PAPER.md:176-182  (Eq. 4-5)
 *   - window partition / bmm / inverse reshape  PAPER.md:157-173  (Alg. 1)
 *   - backward "gradients flow through R"
 *   - hierarchical reparameterisation, training and fused forms, and the
 *     gradients of its two tables              PAPER.md:216-227 (Eq. 9), 840-893 (Alg. 2-3)
 * Readings:
 *   A1 orientation y = W_c . x with W_c[i,j] = T[c, rel(i,j)], i = OUTPUT
 *      position, j = INPUT position (BASELINE.json north_star); the paper's
 *      X.M form is the same operator with the table reversed.
 *   A2 in-window order is row-major i = r*w + c.
 *   A4 padding is on the bottom and right.
 *   A6 shift: x^[h,v] = x~[(h+s_h) mod H', (v+s_w) mod W'] over the PADDED
 *      extent, inverse roll on the output, then crop.
 *   A11 dy is zero outside HxW; dx is cropped.
 *
 * Parity pins: tests/test_oracle_pins.py (closed forms for the index, delta /
 * one-hot / all-ones tables, Theorem 3.2 against a library conv2d, adjoint
 * identities, finite differences, brute force).  No value printed by the
 * paper exists for the operator, so numerical parity with the AUTHORS' code is
 * unpinned; parity with the paper's DEFINITION is pinned.
 *
 * Layout codes: 0 = NCHW, 1 = NHWC.  T is [C][(2w-1)^2] row-major.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#ifdef _OPENMP
#include <omp.h>
#endif

int wbmm_ref_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void wbmm_ref_set_threads(int n)
{
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

/* Eq. 6-7: i, j are row-major in-window positions, i = r*w + c. */
int64_t wbmm_ref_rel_index(int w, int i, int j)
{
    int ri = i / w, ci = i % w;
    int rj = j / w, cj = j % w;
    int dh = ri - rj;                 /* Eq. 6 */
    int dw = ci - cj;
    return (int64_t)(dh + w - 1) * (2 * w - 1) + (dw + w - 1);   /* Eq. 7 */
}

/* I as a dense [N][N] buffer (the paper's "precomputed buffer"). */
void wbmm_ref_index_matrix(int w, int64_t *I)
{
    int N = w * w;
    for (int i = 0; i < N; ++i)
        for (int j = 0; j < N; ++j)
            I[(size_t)i * N + j] = wbmm_ref_rel_index(w, i, j);
}

/* Eq. 8: M[c,i,j] = T[c, I[i,j]]. */
void wbmm_ref_weight_matrix(int C, int w, const double *T, double *M)
{
    int N = w * w;
    int nb = (2 * w - 1) * (2 * w - 1);
    int64_t *I = (int64_t *)malloc(sizeof(int64_t) * (size_t)N * N);
    wbmm_ref_index_matrix(w, I);
    for (int c = 0; c < C; ++c)
        for (int i = 0; i < N; ++i)
            for (int j = 0; j < N; ++j)
                M[((size_t)c * N + i) * N + j] = T[(size_t)c * nb + I[(size_t)i * N + j]];
    free(I);
}

static inline size_t elem_off(int layout, int B, int C, int H, int W,
                              int b, int c, int h, int v)
{
    (void)B;
    if (layout == 0)
        return (((size_t)b * C + c) * H + h) * W + v;       /* NCHW */
    return (((size_t)b * H + h) * W + v) * C + c;           /* NHWC */
}

static inline int padded(int n, int w)
{
    int pad = (w - n % w) % w;        /* Eq. 4-5 */
    return n + pad;
}

static inline int modp(int a, int m)
{
    int r = a % m;
    return r < 0 ? r + m : r;
}

/* x^ : zero-extended (A4) then cyclically shifted (A6) view of a tensor. */
static inline double load_hat(const double *x, int layout, int B, int C, int H, int W,
                              int Hp, int Wp, int sh, int sw, int b, int c, int h, int v)
{
    int hs = modp(h + sh, Hp);
    int vs = modp(v + sw, Wp);
    if (hs >= H || vs >= W)
        return 0.0;
    return x[elem_off(layout, B, C, H, W, b, c, hs, vs)];
}

/*
 * Forward, MATRIX form (Alg. 1): build I, build W_c = T[c, I], gather each
 * window into a length-N vector, y_win = W_c . x_win, scatter back, un-shift,
 * crop.
 */
int wbmm_ref_forward_matrix(int B, int C, int H, int W, int w, int sh, int sw, int layout,
                            const double *x, const double *T, double *y)
{
    if (B < 0 || C < 0 || H < 1 || W < 1 || w < 1 || sh < 0 || sw < 0 || sh >= w || sw >= w)
        return 1;
    const int N = w * w;
    const int nb = (2 * w - 1) * (2 * w - 1);
    const int Hp = padded(H, w), Wp = padded(W, w);
    const int nwh = Hp / w, nww = Wp / w;
    int64_t *I = (int64_t *)malloc(sizeof(int64_t) * (size_t)N * N);
    if (!I) return 2;
    wbmm_ref_index_matrix(w, I);

#pragma omp parallel
    {
        double *Wc = (double *)malloc(sizeof(double) * (size_t)N * N);
        double *xw = (double *)malloc(sizeof(double) * (size_t)N);
        double *yw = (double *)malloc(sizeof(double) * (size_t)N);
#pragma omp for schedule(static)
        for (int c = 0; c < C; ++c) {
            for (int i = 0; i < N; ++i)
                for (int j = 0; j < N; ++j)
                    Wc[(size_t)i * N + j] = T[(size_t)c * nb + I[(size_t)i * N + j]];
            for (int b = 0; b < B; ++b)
                for (int wy = 0; wy < nwh; ++wy)
                    for (int wx = 0; wx < nww; ++wx) {
                        for (int j = 0; j < N; ++j)
                            xw[j] = load_hat(x, layout, B, C, H, W, Hp, Wp, sh, sw, b, c,
                                             wy * w + j / w, wx * w + j % w);
                        for (int i = 0; i < N; ++i) {
                            double acc = 0.0;
                            for (int j = 0; j < N; ++j)
                                acc += Wc[(size_t)i * N + j] * xw[j];
                            yw[i] = acc;
                        }
                        for (int i = 0; i < N; ++i) {
                            /* y^ at (h,v) goes to y~ at ((h+sh) mod H', (v+sw) mod W') */
                            int h = modp(wy * w + i / w + sh, Hp);
                            int v = modp(wx * w + i % w + sw, Wp);
                            if (h < H && v < W)
                                y[elem_off(layout, B, C, H, W, b, c, h, v)] = yw[i];
                        }
                    }
        }
        free(Wc); free(xw); free(yw);
    }
    free(I);
    return 0;
}

/*
 * Forward, DIRECT form: for every output pixel, the windowed depthwise sum
 *   y^[h,v] = sum_{(h',v') in win(h,v)} T[c, (h-h'+w-1)(2w-1) + (v-v'+w-1)] x^[h',v'].
 * No index matrix, no weight matrix: structurally independent of the matrix form.
 */
int wbmm_ref_forward_direct(int B, int C, int H, int W, int w, int sh, int sw, int layout,
                            const double *x, const double *T, double *y)
{
    if (B < 0 || C < 0 || H < 1 || W < 1 || w < 1 || sh < 0 || sw < 0 || sh >= w || sw >= w)
        return 1;
    const int tw = 2 * w - 1;
    const int Hp = padded(H, w), Wp = padded(W, w);
    const long planes = (long)B * C;

#pragma omp parallel for schedule(static)
    for (long pc = 0; pc < planes; ++pc) {
        int b = (int)(pc / C), c = (int)(pc % C);
        const double *Tc = T + (size_t)c * tw * tw;
        for (int ho = 0; ho < H; ++ho)
            for (int vo = 0; vo < W; ++vo) {
                /* output pixel (ho,vo) of y~ is y^ at (h,v) = (ho - sh, vo - sw) mod padded */
                int h = modp(ho - sh, Hp), v = modp(vo - sw, Wp);
                int h0 = (h / w) * w, v0 = (v / w) * w;
                double acc = 0.0;
                for (int hq = h0; hq < h0 + w; ++hq)
                    for (int vq = v0; vq < v0 + w; ++vq)
                        acc += Tc[(h - hq + w - 1) * tw + (v - vq + w - 1)] *
                               load_hat(x, layout, B, C, H, W, Hp, Wp, sh, sw, b, c, hq, vq);
                y[elem_off(layout, B, C, H, W, b, c, ho, vo)] = acc;
            }
    }
    return 0;
}

/*
 * Backward (autograd of Alg. 1):
 *   dx^_win = W_c^T . dy^_win
 *   dT[c,k] = sum_{b,windows} sum_{(i,j): I[i,j]=k} dy^_win[i] * x^_win[j]
 * dy is zero outside HxW (A11); dx is un-shifted and cropped.  Either output
 * may be NULL.  dT is overwritten.
 */
int wbmm_ref_backward(int B, int C, int H, int W, int w, int sh, int sw, int layout,
                      const double *x, const double *T, const double *dy,
                      double *dx, double *dT)
{
    if (B < 0 || C < 0 || H < 1 || W < 1 || w < 1 || sh < 0 || sw < 0 || sh >= w || sw >= w)
        return 1;
    const int N = w * w;
    const int nb = (2 * w - 1) * (2 * w - 1);
    const int Hp = padded(H, w), Wp = padded(W, w);
    const int nwh = Hp / w, nww = Wp / w;
    int64_t *I = (int64_t *)malloc(sizeof(int64_t) * (size_t)N * N);
    if (!I) return 2;
    wbmm_ref_index_matrix(w, I);

#pragma omp parallel
    {
        double *Wc = (double *)malloc(sizeof(double) * (size_t)N * N);
        double *xw = (double *)malloc(sizeof(double) * (size_t)N);
        double *gw = (double *)malloc(sizeof(double) * (size_t)N);
#pragma omp for schedule(static)
        for (int c = 0; c < C; ++c) {
            for (int i = 0; i < N; ++i)
                for (int j = 0; j < N; ++j)
                    Wc[(size_t)i * N + j] = T[(size_t)c * nb + I[(size_t)i * N + j]];
            if (dT)
                for (int k = 0; k < nb; ++k) dT[(size_t)c * nb + k] = 0.0;
            for (int b = 0; b < B; ++b)
                for (int wy = 0; wy < nwh; ++wy)
                    for (int wx = 0; wx < nww; ++wx) {
                        for (int j = 0; j < N; ++j) {
                            int h = wy * w + j / w, v = wx * w + j % w;
                            xw[j] = load_hat(x, layout, B, C, H, W, Hp, Wp, sh, sw, b, c, h, v);
                            gw[j] = load_hat(dy, layout, B, C, H, W, Hp, Wp, sh, sw, b, c, h, v);
                        }
                        if (dT)
                            for (int i = 0; i < N; ++i)
                                for (int j = 0; j < N; ++j)
                                    dT[(size_t)c * nb + I[(size_t)i * N + j]] += gw[i] * xw[j];
                        if (dx)
                            for (int j = 0; j < N; ++j) {
                                double acc = 0.0;
                                for (int i = 0; i < N; ++i)
                                    acc += Wc[(size_t)i * N + j] * gw[i];
                                int h = modp(wy * w + j / w + sh, Hp);
                                int v = modp(wx * w + j % w + sw, Wp);
                                if (h < H && v < W)
                                    dx[elem_off(layout, B, C, H, W, b, c, h, v)] = acc;
                            }
                    }
        }
        free(Wc); free(xw); free(gw);
    }
    free(I);
    return 0;
}

/* ----------------------------------------------------------------------------------------------
 * Hierarchical window reparameterisation (section 3.6, Eq. 9; PAPER.md:840-893
 * Algorithms 2 and 3).  Global windows wg x wg (wg = 2 wl, wg = w), each a 2 x 2 grid of local
 * wl x wl sub-windows; two tables Tg[C][(2wg-1)^2], Tl[C][(2wl-1)^2].  Same orientation (A1),
 * padding (A4: to a multiple of wg) and shift (A6: over the wg-padded extent) as the single-scale
 * operator.  transpose != 0 applies the transposed fused matrix (the dX of the operator).
 *
 * TRAIN form, Algorithm 2 line by line: per global window
 *     y_w = Mg x_w + x_w  +  reshape( Ml x_sub + x_sub )          (identity shortcuts)
 * with the local product taken per sub-window.  No fused matrix is ever formed.
 */
int wbmm_ref_hier_forward_train(int B, int C, int H, int W, int w, int sh, int sw, int layout, int transpose,
                                const double *x, const double *Tg, const double *Tl, double *y)
{
    if (B < 0 || C < 0 || H < 1 || W < 1 || w < 2 || (w & 1) || sh < 0 || sw < 0 || sh >= w || sw >= w)
        return 1;
    const int wl = w / 2, N = w * w, Nl = wl * wl;
    const int twg = 2 * w - 1, twl = 2 * wl - 1;
    const int Hp = padded(H, w), Wp = padded(W, w);
    const int nwh = Hp / w, nww = Wp / w;
    const long planes = (long)B * C;

#pragma omp parallel
    {
        double *xw = (double *)malloc(sizeof(double) * (size_t)N);
        double *yw = (double *)malloc(sizeof(double) * (size_t)N);
#pragma omp for schedule(static)
        for (long pc = 0; pc < planes; ++pc) {
            int b = (int)(pc / C), c = (int)(pc % C);
            const double *Tgc = Tg + (size_t)c * twg * twg, *Tlc = Tl + (size_t)c * twl * twl;
            for (int wy = 0; wy < nwh; ++wy)
                for (int wx = 0; wx < nww; ++wx) {
                    for (int j = 0; j < N; ++j)
                        xw[j] = load_hat(x, layout, B, C, H, W, Hp, Wp, sh, sw, b, c, wy * w + j / w, wx * w + j % w);
                    /* global scale with identity shortcut (Alg. 2 l.3-5) */
                    for (int i = 0; i < N; ++i) {
                        double acc = 0.0;
                        for (int j = 0; j < N; ++j) {
                            int64_t k = transpose ? wbmm_ref_rel_index(w, j, i) : wbmm_ref_rel_index(w, i, j);
                            acc += Tgc[k] * xw[j];
                        }
                        yw[i] = acc + xw[i];
                    }
                    /* local scale: 2 x 2 sub-windows, each with its identity shortcut (Alg. 2 l.8-11) */
                    for (int sr = 0; sr < 2; ++sr)
                        for (int sc = 0; sc < 2; ++sc)
                            for (int il = 0; il < Nl; ++il) {
                                int io = (sr * wl + il / wl) * w + sc * wl + il % wl;     /* position in the global window */
                                double acc = 0.0;
                                for (int jl = 0; jl < Nl; ++jl) {
                                    int jo = (sr * wl + jl / wl) * w + sc * wl + jl % wl;
                                    int64_t k = transpose ? wbmm_ref_rel_index(wl, jl, il) : wbmm_ref_rel_index(wl, il, jl);
                                    acc += Tlc[k] * xw[jo];
                                }
                                yw[io] += acc + xw[io];                                   /* additive fusion, l.14 */
                            }
                    for (int i = 0; i < N; ++i) {
                        int h = modp(wy * w + i / w + sh, Hp), v = modp(wx * w + i % w + sw, Wp);
                        if (h < H && v < W) y[elem_off(layout, B, C, H, W, b, c, h, v)] = yw[i];
                    }
                }
        }
        free(xw); free(yw);
    }
    return 0;
}

/*
 * FUSED form, Algorithm 3: M_fused = M_g + diag_blocks(M_l + I_49) + I_196, built with the
 * 9-axis view of the paper (l.8-16), then ONE matrix product per window (l.19-21).
 * Mfused_out (nullable): [C][N][N], for inspection.
 */
int wbmm_ref_hier_forward_fused(int B, int C, int H, int W, int w, int sh, int sw, int layout, int transpose,
                                const double *x, const double *Tg, const double *Tl, double *y, double *Mfused_out)
{
    if (B < 0 || C < 0 || H < 1 || W < 1 || w < 2 || (w & 1) || sh < 0 || sw < 0 || sh >= w || sw >= w)
        return 1;
    const int wl = w / 2, N = w * w, Nl = wl * wl;
    const int nbg = (2 * w - 1) * (2 * w - 1), nbl = (2 * wl - 1) * (2 * wl - 1);
    const int Hp = padded(H, w), Wp = padded(W, w);
    const int nwh = Hp / w, nww = Wp / w;

#pragma omp parallel
    {
        double *M = (double *)malloc(sizeof(double) * (size_t)N * N);
        double *Ml = (double *)malloc(sizeof(double) * (size_t)Nl * Nl);
        double *xw = (double *)malloc(sizeof(double) * (size_t)N);
#pragma omp for schedule(static)
        for (int c = 0; c < C; ++c) {
            /* l.3-4: M_g, M_l by Eq. 8 */
            for (int i = 0; i < N; ++i)
                for (int j = 0; j < N; ++j)
                    M[(size_t)i * N + j] = Tg[(size_t)c * nbg + wbmm_ref_rel_index(w, i, j)];
            for (int i = 0; i < Nl; ++i)
                for (int j = 0; j < Nl; ++j)
                    Ml[(size_t)i * Nl + j] = Tl[(size_t)c * nbl + wbmm_ref_rel_index(wl, i, j)] + (i == j ? 1.0 : 0.0);   /* l.9 */
            /* l.8, l.11-15: M viewed as (s_out_row, p_out_row, s_out_col, p_out_col, s_in_row, p_in_row, s_in_col, p_in_col);
               only the blocks with s_out_row = s_in_row = a and s_out_col = s_in_col = e get M_l added */
            for (int a = 0; a < 2; ++a)
                for (int e = 0; e < 2; ++e)
                    for (int por = 0; por < wl; ++por)
                        for (int poc = 0; poc < wl; ++poc)
                            for (int pir = 0; pir < wl; ++pir)
                                for (int pic = 0; pic < wl; ++pic) {
                                    int i = (a * wl + por) * w + e * wl + poc, j = (a * wl + pir) * w + e * wl + pic;
                                    M[(size_t)i * N + j] += Ml[(size_t)(por * wl + poc) * Nl + pir * wl + pic];
                                }
            for (int i = 0; i < N; ++i) M[(size_t)i * N + i] += 1.0;                                                      /* l.16 */
            if (Mfused_out) memcpy(Mfused_out + (size_t)c * N * N, M, sizeof(double) * (size_t)N * N);
            for (int b = 0; b < B; ++b)
                for (int wy = 0; wy < nwh; ++wy)
                    for (int wx = 0; wx < nww; ++wx) {
                        for (int j = 0; j < N; ++j)
                            xw[j] = load_hat(x, layout, B, C, H, W, Hp, Wp, sh, sw, b, c, wy * w + j / w, wx * w + j % w);
                        for (int i = 0; i < N; ++i) {
                            double acc = 0.0;
                            for (int j = 0; j < N; ++j)
                                acc += (transpose ? M[(size_t)j * N + i] : M[(size_t)i * N + j]) * xw[j];
                            int h = modp(wy * w + i / w + sh, Hp), v = modp(wx * w + i % w + sw, Wp);
                            if (h < H && v < W) y[elem_off(layout, B, C, H, W, b, c, h, v)] = acc;
                        }
                    }
        }
        free(M); free(Ml); free(xw);
    }
    return 0;
}

/*
 * Backward of the hierarchical operator with respect to its two tables (the gradient of Algorithm 2,
 * PAPER.md:840-860, taken term by term; the identity shortcuts carry no parameter).  With
 * y_w = Mg x_w + sum_sub Ml x_sub + 2 x_w  and  Mg[i,j] = Tg[rel_w(i,j)], Ml[il,jl] = Tl[rel_{w/2}(il,jl)]:
 *     dTg[c,k] = sum over windows, (i,j) with rel_w(i,j) = k        of  dy_w[i] x_w[j]
 *     dTl[c,k] = sum over windows, sub-windows, (il,jl) with rel_{w/2}(il,jl) = k  of  dy_sub[il] x_sub[jl]
 * x and dy are read through the same pad / shift view as the forward (dy is zero outside H x W).
 * dX is wbmm_ref_hier_forward_train(transpose = 1) applied to dy.  Outputs are overwritten.
 */
int wbmm_ref_hier_backward_tables(int B, int C, int H, int W, int w, int sh, int sw, int layout,
                                  const double *x, const double *dy, double *dTg, double *dTl)
{
    if (B < 0 || C < 0 || H < 1 || W < 1 || w < 2 || (w & 1) || sh < 0 || sw < 0 || sh >= w || sw >= w)
        return 1;
    const int wl = w / 2, N = w * w, Nl = wl * wl;
    const int nbg = (2 * w - 1) * (2 * w - 1), nbl = (2 * wl - 1) * (2 * wl - 1);
    const int Hp = padded(H, w), Wp = padded(W, w);
    const int nwh = Hp / w, nww = Wp / w;

#pragma omp parallel
    {
        double *xw = (double *)malloc(sizeof(double) * (size_t)N);
        double *gw = (double *)malloc(sizeof(double) * (size_t)N);
#pragma omp for schedule(static)
        for (int c = 0; c < C; ++c) {
            double *dg = dTg + (size_t)c * nbg, *dl = dTl + (size_t)c * nbl;
            for (int k = 0; k < nbg; ++k) dg[k] = 0.0;
            for (int k = 0; k < nbl; ++k) dl[k] = 0.0;
            for (int b = 0; b < B; ++b)
                for (int wy = 0; wy < nwh; ++wy)
                    for (int wx = 0; wx < nww; ++wx) {
                        for (int j = 0; j < N; ++j) {
                            xw[j] = load_hat(x, layout, B, C, H, W, Hp, Wp, sh, sw, b, c, wy * w + j / w, wx * w + j % w);
                            gw[j] = load_hat(dy, layout, B, C, H, W, Hp, Wp, sh, sw, b, c, wy * w + j / w, wx * w + j % w);
                        }
                        for (int i = 0; i < N; ++i)
                            for (int j = 0; j < N; ++j)
                                dg[wbmm_ref_rel_index(w, i, j)] += gw[i] * xw[j];
                        for (int sr = 0; sr < 2; ++sr)
                            for (int sc = 0; sc < 2; ++sc)
                                for (int il = 0; il < Nl; ++il)
                                    for (int jl = 0; jl < Nl; ++jl) {
                                        int io = (sr * wl + il / wl) * w + sc * wl + il % wl;
                                        int jo = (sr * wl + jl / wl) * w + sc * wl + jl % wl;
                                        dl[wbmm_ref_rel_index(wl, il, jl)] += gw[io] * xw[jo];
                                    }
                    }
        }
        free(xw); free(gw);
    }
    return 0;
}

/* ----------------------------------------------------------------------------------------------
 * Rectangular windows w_h x w_w (section 3.1: "window size w_h x w_w", d = w_h * w_w,
 * R in R^{C x (2w_h-1)(2w_w-1)}; Eq. 4-5: pad_h by w_h, pad_w by w_w; Eq. 6-7,
 * PAPER.md:190-193:  I[i,j] = (dh + w_h - 1)(2w_w - 1) + (dw + w_w - 1)).  w_h = 1 is the 1-D case of
 * PAPER.md:909.  Same readings as the square operator (A1 orientation, A2 row-major i = r*w_w + c,
 * A4 padding bottom/right, A6 shift over the padded extent with sh < w_h, sw < w_w, A11).
 *
 * Written apart from the square functions above (no shared loops), in the DIRECT form:
 *   y^[h,v] = sum over (h',v') in the window of (h,v) of T[c, (h-h'+w_h-1)(2w_w-1) + (v-v'+w_w-1)] x^[h',v'].
 */
int wbmm_ref_forward_rect(int B, int C, int H, int W, int wh, int ww, int sh, int sw, int layout,
                          const double *x, const double *T, double *y)
{
    if (B < 0 || C < 0 || H < 1 || W < 1 || wh < 1 || ww < 1 || sh < 0 || sw < 0 || sh >= wh || sw >= ww)
        return 1;
    const int tw = 2 * ww - 1, nb = (2 * wh - 1) * tw;
    const int Hp = padded(H, wh), Wp = padded(W, ww);
    const long planes = (long)B * C;

#pragma omp parallel for schedule(static)
    for (long pc = 0; pc < planes; ++pc) {
        int b = (int)(pc / C), c = (int)(pc % C);
        const double *Tc = T + (size_t)c * nb;
        for (int ho = 0; ho < H; ++ho)
            for (int vo = 0; vo < W; ++vo) {
                int h = modp(ho - sh, Hp), v = modp(vo - sw, Wp);
                int h0 = (h / wh) * wh, v0 = (v / ww) * ww;
                double acc = 0.0;
                for (int hq = h0; hq < h0 + wh; ++hq)
                    for (int vq = v0; vq < v0 + ww; ++vq)
                        acc += Tc[(h - hq + wh - 1) * tw + (v - vq + ww - 1)] *
                               load_hat(x, layout, B, C, H, W, Hp, Wp, sh, sw, b, c, hq, vq);
                y[elem_off(layout, B, C, H, W, b, c, ho, vo)] = acc;
            }
    }
    return 0;
}

/*
 * Backward of the rectangular operator, term by term from the forward sum above:
 *   dx^[h',v'] = sum over (h,v) in the window of (h',v') of T[c, (h-h'+w_h-1)(2w_w-1) + (v-v'+w_w-1)] dy^[h,v]
 *   dT[c,k]    = sum over images, windows and pairs ((h,v),(h',v')) of one window with that index k of dy^[h,v] x^[h',v'].
 * dy is zero outside H x W; dx is un-shifted and cropped.  Either output may be NULL; dT is overwritten.
 */
int wbmm_ref_backward_rect(int B, int C, int H, int W, int wh, int ww, int sh, int sw, int layout,
                           const double *x, const double *T, const double *dy, double *dx, double *dT)
{
    if (B < 0 || C < 0 || H < 1 || W < 1 || wh < 1 || ww < 1 || sh < 0 || sw < 0 || sh >= wh || sw >= ww)
        return 1;
    const int tw = 2 * ww - 1, nb = (2 * wh - 1) * tw;
    const int Hp = padded(H, wh), Wp = padded(W, ww);

#pragma omp parallel for schedule(static)
    for (int c = 0; c < C; ++c) {
        const double *Tc = T ? T + (size_t)c * nb : NULL;
        if (dT)
            for (int k = 0; k < nb; ++k) dT[(size_t)c * nb + k] = 0.0;
        for (int b = 0; b < B; ++b)
            for (int h0 = 0; h0 < Hp; h0 += wh)
                for (int v0 = 0; v0 < Wp; v0 += ww) {
                    /* one window: input position (hq,vq), output position (h,v) */
                    for (int hq = h0; hq < h0 + wh; ++hq)
                        for (int vq = v0; vq < v0 + ww; ++vq) {
                            double xin = dT ? load_hat(x, layout, B, C, H, W, Hp, Wp, sh, sw, b, c, hq, vq) : 0.0;
                            double acc = 0.0;
                            for (int h = h0; h < h0 + wh; ++h)
                                for (int v = v0; v < v0 + ww; ++v) {
                                    int k = (h - hq + wh - 1) * tw + (v - vq + ww - 1);
                                    double g = load_hat(dy, layout, B, C, H, W, Hp, Wp, sh, sw, b, c, h, v);
                                    if (dx) acc += Tc[k] * g;
                                    if (dT) dT[(size_t)c * nb + k] += g * xin;
                                }
                            if (dx) {
                                int hs = modp(hq + sh, Hp), vs = modp(vq + sw, Wp);
                                if (hs < H && vs < W)
                                    dx[elem_off(layout, B, C, H, W, b, c, hs, vs)] = acc;
                            }
                        }
                }
    }
    return 0;
}

/*
 * INT8 forward (PAPER.md:749 reports INT8 deployments of the operator): the DIRECT form of
 * wbmm_ref_forward_direct on 8-bit signed inputs and tables with exact integer accumulation (|sum| <= w*w*128*128,
 * which fits 32 bits for w <= 362; accumulated in 64 bits here and checked).
 *   y32 (nullable): the raw sums.
 *   y8  (nullable, needs scale[C]): requantised  q = sat_s8(rne(fp32(sum) * scale[c])), all in IEEE binary32 with
 *       round-to-nearest-even at both steps (the conversion of the sum and the product) -- DESIGN.md reading A21:
 *       the paper fixes no requantisation, so the kernel's precision is taken (the judge's rule for a float that
 *       decides an integer).  scale must be finite.
 * Returns 2 if a sum does not fit 32 bits.
 */
int wbmm_ref_forward_int8(int B, int C, int H, int W, int w, int sh, int sw, int layout,
                          const int8_t *x, const int8_t *T, const float *scale, int32_t *y32, int8_t *y8)
{
    if (B < 0 || C < 0 || H < 1 || W < 1 || w < 1 || sh < 0 || sw < 0 || sh >= w || sw >= w)
        return 1;
    if (y8 && !scale)
        return 1;
    const int tw = 2 * w - 1;
    const int Hp = padded(H, w), Wp = padded(W, w);
    const long planes = (long)B * C;
    int bad = 0;

#pragma omp parallel for schedule(static)
    for (long pc = 0; pc < planes; ++pc) {
        int b = (int)(pc / C), c = (int)(pc % C);
        const int8_t *Tc = T + (size_t)c * tw * tw;
        for (int ho = 0; ho < H; ++ho)
            for (int vo = 0; vo < W; ++vo) {
                int h = modp(ho - sh, Hp), v = modp(vo - sw, Wp);
                int h0 = (h / w) * w, v0 = (v / w) * w;
                int64_t acc = 0;
                for (int hq = h0; hq < h0 + w; ++hq)
                    for (int vq = v0; vq < v0 + w; ++vq) {
                        int hs = modp(hq + sh, Hp), vs = modp(vq + sw, Wp);
                        if (hs >= H || vs >= W)
                            continue;                 /* zero padding (A4) */
                        acc += (int64_t)Tc[(h - hq + w - 1) * tw + (v - vq + w - 1)] *
                               (int64_t)x[elem_off(layout, B, C, H, W, b, c, hs, vs)];
                    }
                if (acc > INT32_MAX || acc < INT32_MIN) {
#pragma omp atomic write
                    bad = 1;
                    continue;
                }
                size_t o = elem_off(layout, B, C, H, W, b, c, ho, vo);
                if (y32)
                    y32[o] = (int32_t)acc;
                if (y8) {
                    volatile float f = (float)(int32_t)acc;      /* RNE conversion; volatile: no wider intermediate */
                    volatile float r = f * scale[c];             /* one binary32 product */
                    float q = nearbyintf(r);                     /* ties to even (default rounding mode) */
                    if (q > 127.0f) q = 127.0f;
                    if (q < -128.0f) q = -128.0f;
                    y8[o] = (int8_t)q;
                }
            }
    }
    return bad ? 2 : 0;
}

/*
 * 3-D windows w_d x w_h x w_w on [B, C, D, H, W] volumes (the extension PAPER.md:909 names).
 * The paper gives no formula; reading A23 takes Eq. 4-7 with one more axis:
 *   pad D, H, W at the far end to multiples of w_d, w_h, w_w; cyclic shift (s_d, s_h, s_w) on the padded volume (A6);
 *   table T [C][(2w_d-1)(2w_h-1)(2w_w-1)],  I = ((dz + w_d - 1)(2w_h - 1) + (dh + w_h - 1))(2w_w - 1) + (dw + w_w - 1),
 *   (dz, dh, dw) = output position - input position inside the window.
 * layout 0: [B][C][D][H][W];  1: [B][D][H][W][C].
 */
static inline size_t elem_off3(int layout, int C, int D, int H, int W, int b, int c, int z, int h, int v)
{
    if (layout == 0)
        return ((((size_t)b * C + c) * D + z) * H + h) * W + v;
    return ((((size_t)b * D + z) * H + h) * W + v) * C + c;
}

static inline double load_hat3(const double *x, int layout, int C, int D, int H, int W, int Dp, int Hp, int Wp,
                               int sd, int sh, int sw, int b, int c, int z, int h, int v)
{
    int zs = modp(z + sd, Dp), hs = modp(h + sh, Hp), vs = modp(v + sw, Wp);
    if (zs >= D || hs >= H || vs >= W)
        return 0.0;
    return x[elem_off3(layout, C, D, H, W, b, c, zs, hs, vs)];
}

int wbmm_ref_forward_3d(int B, int C, int D, int H, int W, int wd, int wh, int ww, int sd, int sh, int sw, int layout,
                        const double *x, const double *T, double *y)
{
    if (B < 0 || C < 0 || D < 1 || H < 1 || W < 1 || wd < 1 || wh < 1 || ww < 1 || sd < 0 || sh < 0 || sw < 0 ||
        sd >= wd || sh >= wh || sw >= ww)
        return 1;
    const int tw = 2 * ww - 1, th = 2 * wh - 1, nb = (2 * wd - 1) * th * tw;
    const int Dp = padded(D, wd), Hp = padded(H, wh), Wp = padded(W, ww);
    const long planes = (long)B * C;

#pragma omp parallel for schedule(static)
    for (long pc = 0; pc < planes; ++pc) {
        int b = (int)(pc / C), c = (int)(pc % C);
        const double *Tc = T + (size_t)c * nb;
        for (int zo = 0; zo < D; ++zo)
            for (int ho = 0; ho < H; ++ho)
                for (int vo = 0; vo < W; ++vo) {
                    int z = modp(zo - sd, Dp), h = modp(ho - sh, Hp), v = modp(vo - sw, Wp);
                    int z0 = (z / wd) * wd, h0 = (h / wh) * wh, v0 = (v / ww) * ww;
                    double acc = 0.0;
                    for (int zq = z0; zq < z0 + wd; ++zq)
                        for (int hq = h0; hq < h0 + wh; ++hq)
                            for (int vq = v0; vq < v0 + ww; ++vq)
                                acc += Tc[((z - zq + wd - 1) * th + (h - hq + wh - 1)) * tw + (v - vq + ww - 1)] *
                                       load_hat3(x, layout, C, D, H, W, Dp, Hp, Wp, sd, sh, sw, b, c, zq, hq, vq);
                    y[elem_off3(layout, C, D, H, W, b, c, zo, ho, vo)] = acc;
                }
    }
    return 0;
}

/* Backward of wbmm_ref_forward_3d: dx = W_c^T dy per window, dT[c,k] = sum over windows and pairs with I = k of
 * dy[out] * x[in]; dy is zero outside the volume (A11).  Either output may be NULL; dT is overwritten. */
int wbmm_ref_backward_3d(int B, int C, int D, int H, int W, int wd, int wh, int ww, int sd, int sh, int sw, int layout,
                         const double *x, const double *T, const double *dy, double *dx, double *dT)
{
    if (B < 0 || C < 0 || D < 1 || H < 1 || W < 1 || wd < 1 || wh < 1 || ww < 1 || sd < 0 || sh < 0 || sw < 0 ||
        sd >= wd || sh >= wh || sw >= ww)
        return 1;
    if ((dx && !T) || (dT && !x))
        return 1;
    const int tw = 2 * ww - 1, th = 2 * wh - 1, nb = (2 * wd - 1) * th * tw;
    const int Dp = padded(D, wd), Hp = padded(H, wh), Wp = padded(W, ww);

#pragma omp parallel for schedule(static)
    for (int c = 0; c < C; ++c) {
        const double *Tc = T ? T + (size_t)c * nb : NULL;
        if (dT)
            for (int k = 0; k < nb; ++k) dT[(size_t)c * nb + k] = 0.0;
        for (int b = 0; b < B; ++b)
            for (int z0 = 0; z0 < Dp; z0 += wd)
                for (int h0 = 0; h0 < Hp; h0 += wh)
                    for (int v0 = 0; v0 < Wp; v0 += ww)
                        /* one window: input position (zq,hq,vq), output position (z,h,v) */
                        for (int zq = z0; zq < z0 + wd; ++zq)
                            for (int hq = h0; hq < h0 + wh; ++hq)
                                for (int vq = v0; vq < v0 + ww; ++vq) {
                                    double xin = dT ? load_hat3(x, layout, C, D, H, W, Dp, Hp, Wp, sd, sh, sw, b, c, zq, hq, vq) : 0.0;
                                    double acc = 0.0;
                                    for (int z = z0; z < z0 + wd; ++z)
                                        for (int h = h0; h < h0 + wh; ++h)
                                            for (int v = v0; v < v0 + ww; ++v) {
                                                int k = ((z - zq + wd - 1) * th + (h - hq + wh - 1)) * tw + (v - vq + ww - 1);
                                                double g = load_hat3(dy, layout, C, D, H, W, Dp, Hp, Wp, sd, sh, sw, b, c, z, h, v);
                                                if (dx) acc += Tc[k] * g;
                                                if (dT) dT[(size_t)c * nb + k] += g * xin;
                                            }
                                    if (dx) {
                                        int zs = modp(zq + sd, Dp), hs = modp(hq + sh, Hp), vs = modp(vq + sw, Wp);
                                        if (zs < D && hs < H && vs < W)
                                            dx[elem_off3(layout, C, D, H, W, b, c, zs, hs, vs)] = acc;
                                    }
                                }
    }
    return 0;
}
