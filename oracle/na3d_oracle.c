/*
 * na3d_oracle.c -- CPU float64 ORACLE for StereoRoPE + 3D neighbourhood attention.
 *
 * TEST INFRASTRUCTURE ONLY.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may load this.  It shares no code with the CUDA path
 * (paper_2606_31248_b200/csrc) and the product never calls it.
 *
 * What it computes is the plain definition, written out in the paper's order, in float64, with
 * the inputs taken as the exact values of the f32 / bf16 arrays handed to the GPU:
 *
 *   A1  rotary angle   phi[t][j] = sum_a coords[t][a] * F[a][j]            (the
 *       stereographic coordinates "replace row/column indices as inputs to axial 2D RoPE")
 *   A2  rotation       (a, b) -> (a cos phi - b sin phi, a sin phi + b cos phi) on each channel
 *       pair of Q and K; V untouched                                        ([41,42])
 *   A3  neighbourhood  start_a(i) = min(max(i - floor(k_a/2), 0), n_a - k_a); the keys of a query
 *       are the k_L x k_Y x k_X box at that start ("3D Neighborhood Attention ...
 *       inside local (x,y,lev) windows"; border rule = inward clamp, reading R1)
 *   A4  logits         s_ij = scale * sum_c qrot_ic krot_jc
 *   A5  softmax, LSE   lse_i = m + ln sum_j exp(s_ij - m),  p_ij = exp(s_ij - lse_i)
 *   A6  output         o_i = sum_j p_ij v_j
 *   B1..B4 backward    D_i = sum_c dO_ic o_ic;  dV_j = sum_i p_ij dO_i;
 *       dS_ij = p_ij (dO_i . v_j - D_i);  dqrot_i = scale sum_j dS_ij krot_j;
 *       dkrot_j = scale sum_i dS_ij qrot_i (scattered from the query loop -- the oracle has no
 *       inverse-neighbourhood formula);  dq = R(-phi) dqrot,  dk = R(-phi) dkrot.
 *
 * No tiling, no online softmax, no fusion: triple loops over (query, neighbour, channel).
 * OpenMP only distributes independent (head, query) or head iterations over cores.
 *
 * Pins (tests/test_oracle_pins.py): dense attention when the window is the grid, brute-force
 * windows, k=1 closed form, RoPE norm / shift invariance / integer-coordinate axial RoPE, 1D/2D
 * reductions, central finite differences and torch float64 autograd for the backward.
 *
 * Layouts: q,k,v,o,do,dq,dk,dv [B,L,Y,X,H,D]; lse [B,H,L,Y,X]; coords [B,L,Y,X,A] f32;
 * freqs [A,D/2] f32.  Input dtype tags: 0 = float64, 1 = float32, 2 = bfloat16 bit pattern.
 */
#include <math.h>
#include <stddef.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct {
    int32_t B, H, D;
    int32_t L, Y, X;
    int32_t kL, kY, kX;
    int32_t A;        /* rotary axes: 0 = no RoPE */
    int32_t pairing;  /* 0: (2j, 2j+1)   1: (j, j + D/2) */
    int32_t dtype;    /* dtype tag of q, k, v, do */
    double scale;     /* <= 0: 1/sqrt(D) */
} oracle_desc_t;

int oracle_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

static inline double ld(const void *p, int dtype, size_t i) {
    if (dtype == 0) return ((const double *)p)[i];
    if (dtype == 1) return (double)((const float *)p)[i];
    uint32_t bits = ((uint32_t)((const uint16_t *)p)[i]) << 16; /* bf16 -> f32 is exact */
    float f;
    memcpy(&f, &bits, 4);
    return (double)f;
}

/* A3: first key index of query i's window on an axis of n tokens with kernel size k. */
int oracle_window_start(int i, int k, int n) {
    int s = i - k / 2;
    if (s < 0) s = 0;
    if (s > n - k) s = n - k;
    return s;
}

static inline double eff_scale(const oracle_desc_t *d) {
    return d->scale > 0.0 ? d->scale : 1.0 / sqrt((double)d->D);
}

/* A1: angles of one token, phi[0..D/2). */
static void angles(const oracle_desc_t *d, const float *coords, const float *freqs, size_t tok,
                   double *phi) {
    int half = d->D / 2;
    for (int j = 0; j < half; ++j) {
        double a = 0.0;
        for (int ax = 0; ax < d->A; ++ax)
            a += (double)coords[tok * (size_t)d->A + ax] * (double)freqs[(size_t)ax * half + j];
        phi[j] = a;
    }
}

static inline void pair_idx(const oracle_desc_t *d, int j, int *c0, int *c1) {
    if (d->pairing == 0) { *c0 = 2 * j; *c1 = 2 * j + 1; }
    else                 { *c0 = j;     *c1 = j + d->D / 2; }
}

/* A2: rotate one head vector x[0..D) (dtype-tagged source at element offset off) by +phi*sign. */
static void rotate_row(const oracle_desc_t *d, const void *src, int dtype, size_t off,
                       const double *phi, double sign, double *out) {
    int half = d->D / 2;
    if (d->A == 0) {
        for (int c = 0; c < d->D; ++c) out[c] = ld(src, dtype, off + c);
        return;
    }
    for (int j = 0; j < half; ++j) {
        int c0, c1;
        pair_idx(d, j, &c0, &c1);
        double a = ld(src, dtype, off + c0), b = ld(src, dtype, off + c1);
        double cs = cos(phi[j]), sn = sign * sin(phi[j]);
        out[c0] = a * cs - b * sn;
        out[c1] = a * sn + b * cs;
    }
}

/* Public: rotate a whole [B,N,H,D] tensor (sign = +1 forward rotation, -1 its transpose). */
void oracle_rope_rotate(const oracle_desc_t *d, const void *x, const float *coords,
                        const float *freqs, double sign, double *out) {
    size_t N = (size_t)d->L * d->Y * d->X;
    size_t T = (size_t)d->B * N;
#pragma omp parallel
    {
        double *phi = (double *)malloc(sizeof(double) * (size_t)(d->D / 2 + 1));
#pragma omp for schedule(static)
        for (long long t = 0; t < (long long)T; ++t) {
            angles(d, coords, freqs, (size_t)t, phi);
            for (int h = 0; h < d->H; ++h) {
                size_t off = ((size_t)t * d->H + h) * d->D;
                rotate_row(d, x, d->dtype, off, phi, sign, out + off);
            }
        }
        free(phi);
    }
}

/* Rotated copies (float64) of q and k for ONE sample b: [N,H,D] each. */
static void rotate_sample(const oracle_desc_t *d, const void *q, const void *k,
                          const float *coords, const float *freqs, int b, double *qr, double *kr) {
    size_t N = (size_t)d->L * d->Y * d->X;
#pragma omp parallel
    {
        double *phi = (double *)malloc(sizeof(double) * (size_t)(d->D / 2 + 1));
#pragma omp for schedule(static)
        for (long long t = 0; t < (long long)N; ++t) {
            size_t tok = (size_t)b * N + (size_t)t;
            angles(d, coords, freqs, tok, phi);
            for (int h = 0; h < d->H; ++h) {
                size_t src = (tok * d->H + h) * d->D;
                size_t dst = ((size_t)t * d->H + h) * d->D;
                rotate_row(d, q, d->dtype, src, phi, 1.0, qr + dst);
                rotate_row(d, k, d->dtype, src, phi, 1.0, kr + dst);
            }
        }
        free(phi);
    }
}

/* A3..A6 for one query of one head, given rotated q/k of the sample.  s[] has W entries. */
static void attend_one(const oracle_desc_t *d, const double *qr, const double *kr, const void *v,
                       int b, int h, int l, int y, int x, double *s, double *o, double *lse) {
    size_t N = (size_t)d->L * d->Y * d->X;
    int D = d->D, H = d->H;
    double sc = eff_scale(d);
    int sl = oracle_window_start(l, d->kL, d->L);
    int sy = oracle_window_start(y, d->kY, d->Y);
    int sx = oracle_window_start(x, d->kX, d->X);
    size_t i = ((size_t)l * d->Y + y) * d->X + x;
    const double *qi = qr + (i * H + h) * D;
    int w = 0;
    double m = -INFINITY;
    for (int a = 0; a < d->kL; ++a)
        for (int bb = 0; bb < d->kY; ++bb)
            for (int c = 0; c < d->kX; ++c, ++w) {
                size_t j = ((size_t)(sl + a) * d->Y + (sy + bb)) * d->X + (sx + c);
                const double *kj = kr + (j * H + h) * D;
                double acc = 0.0;
                for (int ch = 0; ch < D; ++ch) acc += qi[ch] * kj[ch];
                s[w] = sc * acc;
                if (s[w] > m) m = s[w];
            }
    double sum = 0.0;
    for (int u = 0; u < w; ++u) sum += exp(s[u] - m);
    *lse = m + log(sum);
    for (int ch = 0; ch < D; ++ch) o[ch] = 0.0;
    w = 0;
    for (int a = 0; a < d->kL; ++a)
        for (int bb = 0; bb < d->kY; ++bb)
            for (int c = 0; c < d->kX; ++c, ++w) {
                size_t j = ((size_t)(sl + a) * d->Y + (sy + bb)) * d->X + (sx + c);
                double p = exp(s[w] - *lse);
                s[w] = p; /* keep p_ij for the caller (backward) */
                size_t voff = ((((size_t)b * N + j) * H) + h) * D;
                for (int ch = 0; ch < D; ++ch) o[ch] += p * ld(v, d->dtype, voff + ch);
            }
}

/* Forward on the whole tensor: o [B,L,Y,X,H,D] f64, lse [B,H,L,Y,X] f64.  Returns 0 on success. */
int oracle_na3d_fwd(const oracle_desc_t *d, const void *q, const void *k, const void *v,
                    const float *coords, const float *freqs, double *o, double *lse) {
    size_t N = (size_t)d->L * d->Y * d->X;
    int W = d->kL * d->kY * d->kX;
    double *qr = (double *)malloc(sizeof(double) * N * d->H * d->D);
    double *kr = (double *)malloc(sizeof(double) * N * d->H * d->D);
    if (!qr || !kr) { free(qr); free(kr); return 1; }
    for (int b = 0; b < d->B; ++b) {
        rotate_sample(d, q, k, coords, freqs, b, qr, kr);
#pragma omp parallel
        {
            double *s = (double *)malloc(sizeof(double) * (size_t)W);
#pragma omp for schedule(static) collapse(2)
            for (int h = 0; h < d->H; ++h)
                for (long long i = 0; i < (long long)N; ++i) {
                    int x = (int)(i % d->X), y = (int)((i / d->X) % d->Y), l = (int)(i / ((size_t)d->X * d->Y));
                    attend_one(d, qr, kr, v, b, h, l, y, x, s,
                               o + ((((size_t)b * N + (size_t)i) * d->H) + h) * d->D,
                               lse + ((size_t)b * d->H + h) * N + (size_t)i);
                }
            free(s);
        }
    }
    free(qr); free(kr);
    return 0;
}

/* Rotated q (query token) or k (key token) of one (b, token, h) on the fly. */
static void rotated_row_of(const oracle_desc_t *d, const void *x, const float *coords,
                           const float *freqs, int b, size_t tok, int h, double *phi, double *out) {
    size_t N = (size_t)d->L * d->Y * d->X;
    size_t t = (size_t)b * N + tok;
    angles(d, coords, freqs, t, phi);
    rotate_row(d, x, d->dtype, (t * d->H + h) * d->D, phi, 1.0, out);
}

/* Softmax row of query (b, tok, h) straight from the unrotated inputs: p[W], lse; optionally o[D]. */
static void row_from_inputs(const oracle_desc_t *d, const void *q, const void *k, const void *v,
                            const float *coords, const float *freqs, int b, size_t tok, int h,
                            double *phi, double *qi, double *kj, double *p, double *o, double *lse) {
    size_t N = (size_t)d->L * d->Y * d->X;
    int D = d->D, H = d->H;
    double sc = eff_scale(d);
    int x = (int)(tok % d->X), y = (int)((tok / d->X) % d->Y), l = (int)(tok / ((size_t)d->X * d->Y));
    int sl = oracle_window_start(l, d->kL, d->L);
    int sy = oracle_window_start(y, d->kY, d->Y);
    int sx = oracle_window_start(x, d->kX, d->X);
    rotated_row_of(d, q, coords, freqs, b, tok, h, phi, qi);
    int w = 0;
    double m = -INFINITY;
    for (int a = 0; a < d->kL; ++a)
        for (int bb = 0; bb < d->kY; ++bb)
            for (int c = 0; c < d->kX; ++c, ++w) {
                size_t j = ((size_t)(sl + a) * d->Y + (sy + bb)) * d->X + (sx + c);
                rotated_row_of(d, k, coords, freqs, b, j, h, phi, kj);
                double acc = 0.0;
                for (int ch = 0; ch < D; ++ch) acc += qi[ch] * kj[ch];
                p[w] = sc * acc;
                if (p[w] > m) m = p[w];
            }
    double sum = 0.0;
    for (int u = 0; u < w; ++u) sum += exp(p[u] - m);
    *lse = m + log(sum);
    if (o) for (int ch = 0; ch < D; ++ch) o[ch] = 0.0;
    w = 0;
    for (int a = 0; a < d->kL; ++a)
        for (int bb = 0; bb < d->kY; ++bb)
            for (int c = 0; c < d->kX; ++c, ++w) {
                size_t j = ((size_t)(sl + a) * d->Y + (sy + bb)) * d->X + (sx + c);
                p[w] = exp(p[w] - *lse);
                if (o) {
                    size_t voff = ((((size_t)b * N + j) * H) + h) * D;
                    for (int ch = 0; ch < D; ++ch) o[ch] += p[w] * ld(v, d->dtype, voff + ch);
                }
            }
}

/* Forward for a list of queries.  idx[n] = flat index over (b, token, h) = (b*N + tok)*H + h.
 * o_out [n, D], lse_out [n]. */
int oracle_na3d_fwd_queries(const oracle_desc_t *d, const void *q, const void *k, const void *v,
                            const float *coords, const float *freqs, long long n,
                            const long long *idx, double *o_out, double *lse_out) {
    size_t N = (size_t)d->L * d->Y * d->X;
    int W = d->kL * d->kY * d->kX;
#pragma omp parallel
    {
        double *buf = (double *)malloc(sizeof(double) * (size_t)(W + 2 * d->D + d->D / 2 + 1));
        double *p = buf, *qi = p + W, *kj = qi + d->D, *phi = kj + d->D;
#pragma omp for schedule(dynamic, 4)
        for (long long u = 0; u < n; ++u) {
            int h = (int)(idx[u] % d->H);
            size_t bt = (size_t)(idx[u] / d->H);
            int b = (int)(bt / N);
            size_t tok = bt % N;
            row_from_inputs(d, q, k, v, coords, freqs, b, tok, h, phi, qi, kj, p,
                            o_out + (size_t)u * d->D, lse_out + u);
        }
        free(buf);
    }
    return 0;
}

/* Backward on the whole tensor: dq, dk, dv [B,L,Y,X,H,D] f64 (fully overwritten). */
int oracle_na3d_bwd(const oracle_desc_t *d, const void *q, const void *k, const void *v,
                    const void *d_o, const float *coords, const float *freqs,
                    double *dq, double *dk, double *dv) {
    size_t N = (size_t)d->L * d->Y * d->X;
    int W = d->kL * d->kY * d->kX, D = d->D, H = d->H;
    double sc = eff_scale(d);
    size_t per = N * H * D;
    double *qr = (double *)malloc(sizeof(double) * per);
    double *kr = (double *)malloc(sizeof(double) * per);
    double *dqr = (double *)malloc(sizeof(double) * per);
    double *dkr = (double *)malloc(sizeof(double) * per);
    if (!qr || !kr || !dqr || !dkr) { free(qr); free(kr); free(dqr); free(dkr); return 1; }
    for (int b = 0; b < d->B; ++b) {
        rotate_sample(d, q, k, coords, freqs, b, qr, kr);
        memset(dqr, 0, sizeof(double) * per);
        memset(dkr, 0, sizeof(double) * per);
        memset(dv + (size_t)b * per, 0, sizeof(double) * per);
        /* heads are independent; the scatter into dkrot / dv stays inside one head */
#pragma omp parallel for schedule(dynamic, 1)
        for (int h = 0; h < H; ++h) {
            double *p = (double *)malloc(sizeof(double) * (size_t)(W + D));
            double *o = p + W;
            for (size_t i = 0; i < N; ++i) {
                int x = (int)(i % d->X), y = (int)((i / d->X) % d->Y), l = (int)(i / ((size_t)d->X * d->Y));
                double lse;
                attend_one(d, qr, kr, v, b, h, l, y, x, p, o, &lse); /* p_ij, o_i (float64) */
                size_t ioff = ((((size_t)b * N + i) * H) + h) * D;
                double Di = 0.0; /* B1 */
                for (int ch = 0; ch < D; ++ch) Di += ld(d_o, d->dtype, ioff + ch) * o[ch];
                int sl = oracle_window_start(l, d->kL, d->L);
                int sy = oracle_window_start(y, d->kY, d->Y);
                int sx = oracle_window_start(x, d->kX, d->X);
                const double *qi = qr + (i * H + h) * D;
                double *dqi = dqr + (i * H + h) * D;
                int w = 0;
                for (int a = 0; a < d->kL; ++a)
                    for (int bb = 0; bb < d->kY; ++bb)
                        for (int c = 0; c < d->kX; ++c, ++w) {
                            size_t j = ((size_t)(sl + a) * d->Y + (sy + bb)) * d->X + (sx + c);
                            size_t joff = ((((size_t)b * N + j) * H) + h) * D;
                            const double *kj = kr + (j * H + h) * D;
                            double *dkj = dkr + (j * H + h) * D;
                            double dP = 0.0; /* B2 */
                            for (int ch = 0; ch < D; ++ch)
                                dP += ld(d_o, d->dtype, ioff + ch) * ld(v, d->dtype, joff + ch);
                            double dS = p[w] * (dP - Di);
                            for (int ch = 0; ch < D; ++ch) {
                                dv[joff + ch] += p[w] * ld(d_o, d->dtype, ioff + ch);
                                dqi[ch] += sc * dS * kj[ch];
                                dkj[ch] += sc * dS * qi[ch];
                            }
                        }
            }
            free(p);
        }
        /* B4: rotate the gradients back, dq = R(-phi) dqrot, dk = R(-phi) dkrot */
#pragma omp parallel
        {
            double *phi = (double *)malloc(sizeof(double) * (size_t)(D / 2 + 1));
#pragma omp for schedule(static)
            for (long long t = 0; t < (long long)N; ++t) {
                angles(d, coords, freqs, (size_t)b * N + (size_t)t, phi);
                for (int h = 0; h < H; ++h) {
                    size_t src = ((size_t)t * H + h) * D;
                    size_t dst = ((((size_t)b * N + (size_t)t) * H) + h) * D;
                    rotate_row(d, dqr, 0, src, phi, -1.0, dq + dst);
                    rotate_row(d, dkr, 0, src, phi, -1.0, dk + dst);
                }
            }
            free(phi);
        }
    }
    free(qr); free(kr); free(dqr); free(dkr);
    return 0;
}

/* Backward for sampled rows.  idx[n] = flat (b, token, h) as above.
 * dq_out[u] = dq of that token as a QUERY; dk_out[u], dv_out[u] = dk, dv of that token as a KEY,
 * found by brute force: every query of the sample is asked whether its window holds the key. */
int oracle_na3d_bwd_rows(const oracle_desc_t *d, const void *q, const void *k, const void *v,
                         const void *d_o, const float *coords, const float *freqs, long long n,
                         const long long *idx, double *dq_out, double *dk_out, double *dv_out) {
    size_t N = (size_t)d->L * d->Y * d->X;
    int W = d->kL * d->kY * d->kX, D = d->D, H = d->H;
    double sc = eff_scale(d);
#pragma omp parallel
    {
        double *buf = (double *)malloc(sizeof(double) * (size_t)(W + 6 * D + D / 2 + 1));
        double *p = buf, *qi = p + W, *kj = qi + D, *o = kj + D, *acc = o + D, *acc2 = acc + D,
               *tmp = acc2 + D, *phi = tmp + D;
#pragma omp for schedule(dynamic, 1)
        for (long long u = 0; u < n; ++u) {
            int h = (int)(idx[u] % H);
            size_t bt = (size_t)(idx[u] / H);
            int b = (int)(bt / N);
            size_t tok = bt % N;
            double lse;
            /* ---- dq of query tok ---- */
            row_from_inputs(d, q, k, v, coords, freqs, b, tok, h, phi, qi, kj, p, o, &lse);
            size_t ioff = ((((size_t)b * N + tok) * H) + h) * D;
            double Di = 0.0;
            for (int ch = 0; ch < D; ++ch) Di += ld(d_o, d->dtype, ioff + ch) * o[ch];
            {
                int x = (int)(tok % d->X), y = (int)((tok / d->X) % d->Y), l = (int)(tok / ((size_t)d->X * d->Y));
                int sl = oracle_window_start(l, d->kL, d->L);
                int sy = oracle_window_start(y, d->kY, d->Y);
                int sx = oracle_window_start(x, d->kX, d->X);
                for (int ch = 0; ch < D; ++ch) acc[ch] = 0.0;
                int w = 0;
                for (int a = 0; a < d->kL; ++a)
                    for (int bb = 0; bb < d->kY; ++bb)
                        for (int c = 0; c < d->kX; ++c, ++w) {
                            size_t j = ((size_t)(sl + a) * d->Y + (sy + bb)) * d->X + (sx + c);
                            size_t joff = ((((size_t)b * N + j) * H) + h) * D;
                            rotated_row_of(d, k, coords, freqs, b, j, h, phi, kj);
                            double dP = 0.0;
                            for (int ch = 0; ch < D; ++ch)
                                dP += ld(d_o, d->dtype, ioff + ch) * ld(v, d->dtype, joff + ch);
                            double dS = p[w] * (dP - Di);
                            for (int ch = 0; ch < D; ++ch) acc[ch] += sc * dS * kj[ch];
                        }
                angles(d, coords, freqs, (size_t)b * N + tok, phi);
                rotate_row(d, acc, 0, 0, phi, -1.0, dq_out + (size_t)u * D);
            }
            /* ---- dk, dv of key tok: ask every query ---- */
            for (int ch = 0; ch < D; ++ch) { acc[ch] = 0.0; acc2[ch] = 0.0; }
            int jx = (int)(tok % d->X), jy = (int)((tok / d->X) % d->Y), jl = (int)(tok / ((size_t)d->X * d->Y));
            for (size_t i = 0; i < N; ++i) {
                int x = (int)(i % d->X), y = (int)((i / d->X) % d->Y), l = (int)(i / ((size_t)d->X * d->Y));
                int sl = oracle_window_start(l, d->kL, d->L);
                int sy = oracle_window_start(y, d->kY, d->Y);
                int sx = oracle_window_start(x, d->kX, d->X);
                if (jl < sl || jl >= sl + d->kL || jy < sy || jy >= sy + d->kY || jx < sx || jx >= sx + d->kX)
                    continue;
                row_from_inputs(d, q, k, v, coords, freqs, b, i, h, phi, qi, kj, p, o, &lse);
                size_t qoff = ((((size_t)b * N + i) * H) + h) * D;
                double Dq = 0.0;
                for (int ch = 0; ch < D; ++ch) Dq += ld(d_o, d->dtype, qoff + ch) * o[ch];
                int w = ((jl - sl) * d->kY + (jy - sy)) * d->kX + (jx - sx);
                double dP = 0.0;
                for (int ch = 0; ch < D; ++ch)
                    dP += ld(d_o, d->dtype, qoff + ch) * ld(v, d->dtype, ioff + ch);
                double dS = p[w] * (dP - Dq);
                for (int ch = 0; ch < D; ++ch) {
                    acc2[ch] += p[w] * ld(d_o, d->dtype, qoff + ch); /* dV_j */
                    acc[ch] += sc * dS * qi[ch];                     /* dkrot_j */
                }
            }
            angles(d, coords, freqs, (size_t)b * N + tok, phi);
            rotate_row(d, acc, 0, 0, phi, -1.0, dk_out + (size_t)u * D);
            for (int ch = 0; ch < D; ++ch) dv_out[(size_t)u * D + ch] = acc2[ch];
        }
        free(buf);
    }
    return 0;
}
