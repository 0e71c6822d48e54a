/*
 * optflow_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, fp64 CPU statement of the dense optical-flow solve of arxiv/paper_1306_2461
 * (Gautier & Aider): a local, iterative, gradient-based, windowed-SSD Gauss-Newton registration of
 * the Lucas-Kanade family (sec. 2.4) run coarse-to-fine over an image pyramid from a
 * zero initial guess, `iterations` times per level, with an
 * interrogation window of radius R.  The paper prints no solver equation; the step
 * list is BASELINE.json:5 (north_star) and every point the paper leaves open follows the reading
 * D1..D23 of SURVEY.md 8(c), restated in DESIGN.md "Readings of the paper".
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * load this file.  It shares no code, header, table or constant with the CUDA path
 * (paper_1306_2461_b200/csrc) and neither includes the other.
 *
 * Conventions: images are H rows x W columns, row-major doubles, pixel (x,y) = (column,row),
 * integer pixel centres; flow (u,v) in pixels with  I2(x+u, y+v) ~= I1(x,y)  (D1, D2).
 * Every step reads the previous step's complete output (no in-place hazards).  The only concession
 * to speed is `#pragma omp parallel for` over image rows.
 *
 * Pins (tests/test_oracle_pins.py, -m "not gpu"): identical images -> exactly zero; band-limited
 * sub-pixel shift to 0.02 px; linear ramp closed form u = d/(1+eps/2) in one iteration; swap ->
 * negation; window sums vs brute force on 32x32; transpose / mirror / gain-offset invariances;
 * reduction to textbook Lucas-Kanade (scipy uniform_filter); integer shift; pyramid and upsample
 * exactness on constants and ramps; eq. 1 behaviour; monotone error vs iterations
 * (Table 1 trend); oracle_equalise (eq. 2): zero local mean / unit local variance,
 * gain-offset invariance, flat image -> 0, agreement with scipy uniform_filter in the interior.
 * Masks (f4, readings M1-M5 above oracle_mask_downsample): all-ones mask == no mask bit for bit; ramp
 * still exact in one iteration at every fluid pixel; the sums equal brute-force sums of mask*product;
 * image content deep under the mask does not reach any fluid vector; mask pyramid vs a Python loop.
 * No function here is "parity unpinned".
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>

#define ORACLE_WINDOW_BOX 0
#define ORACLE_WINDOW_GAUSSIAN 1

static int clampi(int i, int lo, int hi) { return i < lo ? lo : (i > hi ? hi : i); }

/* Window weight w(t), |t| <= R.  D11: box w = 1; Gaussian w(t) = exp(-t^2/(2 sigma^2)), sigma = R/3,
 * unnormalised (the solve is scale-free). */
double oracle_window_weight(int t, int R, int window_type)
{
    if (window_type == ORACLE_WINDOW_GAUSSIAN) {
        double sigma = (double)R / 3.0;
        return exp(-(double)(t * t) / (2.0 * sigma * sigma));
    }
    return 1.0;
}

/* O2 / D4, D5: one pyramid step ("reduced in size by a factor of 4"; Fig. 3).
 * W' = (W+1)/2, H' = (H+1)/2; k = [1 4 6 4 1]/16; rows first, then columns; indices clamped.
 *   T(y,X) = sum_i k_i P(y, clamp(2X+i, 0, W-1));   D(Y,X) = sum_j k_j T(clamp(2Y+j, 0, H-1), X)  */
void oracle_downsample(const double *src, int W, int H, double *dst)
{
    static const double k[5] = {1.0 / 16.0, 4.0 / 16.0, 6.0 / 16.0, 4.0 / 16.0, 1.0 / 16.0};
    int Wd = (W + 1) / 2, Hd = (H + 1) / 2;
    double *T = (double *)malloc(sizeof(double) * (size_t)H * Wd);
#pragma omp parallel for
    for (int y = 0; y < H; ++y)
        for (int X = 0; X < Wd; ++X) {
            double s = 0.0;
            for (int i = -2; i <= 2; ++i) s += k[i + 2] * src[(size_t)y * W + clampi(2 * X + i, 0, W - 1)];
            T[(size_t)y * Wd + X] = s;
        }
#pragma omp parallel for
    for (int Y = 0; Y < Hd; ++Y)
        for (int X = 0; X < Wd; ++X) {
            double s = 0.0;
            for (int j = -2; j <= 2; ++j) s += k[j + 2] * T[(size_t)clampi(2 * Y + j, 0, H - 1) * Wd + X];
            dst[(size_t)Y * Wd + X] = s;
        }
    free(T);
}

/* O4 hand-down / D6 ("used as an initial estimate ... in the next pair of images"):
 * fine(x,y) = 2 * bilinear(coarse; x/2, y/2) in the geometry coarse X <-> fine 2X.
 *   x0 = x>>1, fx = (x&1)/2, x1 = min(x0+1, Wc-1); same in y. */
void oracle_upsample_flow(const double *coarse, int Wc, int Hc, double *fine, int W, int H)
{
#pragma omp parallel for
    for (int y = 0; y < H; ++y) {
        int y0 = y >> 1, y1 = y0 + 1 < Hc ? y0 + 1 : Hc - 1;
        double fy = (y & 1) * 0.5;
        for (int x = 0; x < W; ++x) {
            int x0 = x >> 1, x1 = x0 + 1 < Wc ? x0 + 1 : Wc - 1;
            double fx = (x & 1) * 0.5;
            double top = (1.0 - fx) * coarse[(size_t)y0 * Wc + x0] + fx * coarse[(size_t)y0 * Wc + x1];
            double bot = (1.0 - fx) * coarse[(size_t)y1 * Wc + x0] + fx * coarse[(size_t)y1 * Wc + x1];
            fine[(size_t)y * W + x] = 2.0 * ((1.0 - fy) * top + fy * bot);
        }
    }
}

/* O4.a / D8: bilinear warp of I2 by the dense field, I2w(x,y) = I2(x+u, y+v); integer part of the
 * displacement added to the integer pixel index, indices clamped to the image. */
void oracle_warp(const double *I2, const double *u, const double *v, int W, int H, double *I2w)
{
#pragma omp parallel for
    for (int y = 0; y < H; ++y)
        for (int x = 0; x < W; ++x) {
            size_t k = (size_t)y * W + x;
            double fu = floor(u[k]), fv = floor(v[k]);
            double ax = u[k] - fu, ay = v[k] - fv;
            /* guard the int conversion against absurd displacements (cannot occur with D15) */
            if (fu > 1e9) fu = 1e9; if (fu < -1e9) fu = -1e9;
            if (fv > 1e9) fv = 1e9; if (fv < -1e9) fv = -1e9;
            long X = (long)x + (long)fu, Y = (long)y + (long)fv;
            int xa = (int)(X < 0 ? 0 : (X > W - 1 ? W - 1 : X));
            int xb = (int)(X + 1 < 0 ? 0 : (X + 1 > W - 1 ? W - 1 : X + 1));
            int ya = (int)(Y < 0 ? 0 : (Y > H - 1 ? H - 1 : Y));
            int yb = (int)(Y + 1 < 0 ? 0 : (Y + 1 > H - 1 ? H - 1 : Y + 1));
            double top = (1.0 - ax) * I2[(size_t)ya * W + xa] + ax * I2[(size_t)ya * W + xb];
            double bot = (1.0 - ax) * I2[(size_t)yb * W + xa] + ax * I2[(size_t)yb * W + xb];
            I2w[k] = (1.0 - ay) * top + ay * bot;
        }
}

/* O4.b / D9: central differences [-1/2, 0, 1/2] of I1 (unwarped), indices clamped at the borders. */
void oracle_gradients(const double *I1, int W, int H, double *Ix, double *Iy)
{
#pragma omp parallel for
    for (int y = 0; y < H; ++y)
        for (int x = 0; x < W; ++x) {
            int xm = x > 0 ? x - 1 : 0, xp = x < W - 1 ? x + 1 : W - 1;
            int ym = y > 0 ? y - 1 : 0, yp = y < H - 1 ? y + 1 : H - 1;
            Ix[(size_t)y * W + x] = (I1[(size_t)y * W + xp] - I1[(size_t)y * W + xm]) / 2.0;
            Iy[(size_t)y * W + x] = (I1[(size_t)yp * W + x] - I1[(size_t)ym * W + x]) / 2.0;
        }
}

/* O4.e / D11, D12 -- THE DEFINITION: S(x,y) = sum_{dy=-R..R} sum_{dx=-R..R} w(dx) w(dy) f(x+dx,y+dy),
 * terms outside the image omitted, no renormalisation. */
void oracle_window_sum_direct(const double *f, int W, int H, int R, int window_type, double *out)
{
#pragma omp parallel for
    for (int y = 0; y < H; ++y)
        for (int x = 0; x < W; ++x) {
            double s = 0.0;
            for (int dy = -R; dy <= R; ++dy) {
                int yy = y + dy;
                if (yy < 0 || yy >= H) continue;
                for (int dx = -R; dx <= R; ++dx) {
                    int xx = x + dx;
                    if (xx < 0 || xx >= W) continue;
                    s += oracle_window_weight(dx, R, window_type) * oracle_window_weight(dy, R, window_type) *
                         f[(size_t)yy * W + xx];
                }
            }
            out[(size_t)y * W + x] = s;
        }
}

/* The same sum in the order the north_star names it (BASELINE.json:5: "horizontal window sum ...
 * vertical window sum"): rows, then columns.  Pinned against brute force on 32x32 inputs. */
void oracle_window_sum(const double *f, int W, int H, int R, int window_type, double *out)
{
    double *w = (double *)malloc(sizeof(double) * (size_t)(2 * R + 1));
    double *h = (double *)malloc(sizeof(double) * (size_t)W * H);
    for (int t = -R; t <= R; ++t) w[t + R] = oracle_window_weight(t, R, window_type);
#pragma omp parallel for
    for (int y = 0; y < H; ++y)
        for (int x = 0; x < W; ++x) {
            double s = 0.0;
            for (int dx = -R; dx <= R; ++dx) {
                int xx = x + dx;
                if (xx < 0 || xx >= W) continue;
                s += w[dx + R] * f[(size_t)y * W + xx];
            }
            h[(size_t)y * W + x] = s;
        }
#pragma omp parallel for
    for (int y = 0; y < H; ++y)
        for (int x = 0; x < W; ++x) {
            double s = 0.0;
            for (int dy = -R; dy <= R; ++dy) {
                int yy = y + dy;
                if (yy < 0 || yy >= H) continue;
                s += w[dy + R] * h[(size_t)yy * W + x];
            }
            out[(size_t)y * W + x] = s;
        }
    free(h);
    free(w);
}

/* One Gauss-Newton iteration at one level (O4.a-g; "iterative Gauss-Newton scheme to minimize a
 * sum of squared difference criterion"; step list BASELINE.json:5).
 *   c. It = I2w - I1 - Ix*u - Iy*v            (expansion about the dense field, D10)
 *   d. Ix^2, Ix*Iy, Iy^2, Ix*It, Iy*It
 *   e. window sums -> a, b, c, p, q
 *   f. tr = a + c;  tr <= 0: valid = 0, no update.  Else lam = eps*tr/2, A = a+lam, C = c+lam,
 *      D = A*C - b^2, rp = -(p + a*u + b*v), rq = -(q + b*u + c*v),
 *      du = (C*rp - b*rq)/D, dv = (A*rq - b*rp)/D, each clamped to +-max_step   (D14, D15)
 *   g. u += du, v += dv
 * u, v are updated in place at the end.  sums5 (optional) receives a,b,c,p,q as 5 planes; valid
 * (optional) the validity bytes; det (optional) the undamped a*c - b^2.
 * direct_sums != 0 uses oracle_window_sum_direct instead of the two-pass form. */
void oracle_iteration_masked(const double *I1, const double *I2, const unsigned char *mask, int W, int H, int R,
                             int window_type, double eps, double max_step, double *u, double *v, double *sums5,
                             unsigned char *valid, double *det, int direct_sums)
{
    size_t N = (size_t)W * H;
    double *I2w = (double *)malloc(sizeof(double) * N);
    double *Ix = (double *)malloc(sizeof(double) * N);
    double *Iy = (double *)malloc(sizeof(double) * N);
    double *prod = (double *)malloc(sizeof(double) * N * 5);
    double *S = (double *)malloc(sizeof(double) * N * 5);

    oracle_warp(I2, u, v, W, H, I2w);
    oracle_gradients(I1, W, H, Ix, Iy);
#pragma omp parallel for
    for (long k = 0; k < (long)N; ++k) {
        double It = I2w[k] - I1[k] - Ix[k] * u[k] - Iy[k] * v[k];
        prod[0 * N + k] = Ix[k] * Ix[k];
        prod[1 * N + k] = Ix[k] * Iy[k];
        prod[2 * N + k] = Iy[k] * Iy[k];
        prod[3 * N + k] = Ix[k] * It;
        prod[4 * N + k] = Iy[k] * It;
        if (mask && !mask[k])                       /* M2: an obstacle pixel has zero weight in every window sum */
            for (int f = 0; f < 5; ++f) prod[f * N + k] = 0.0;
    }
    for (int f = 0; f < 5; ++f) {
        if (direct_sums) oracle_window_sum_direct(prod + f * N, W, H, R, window_type, S + f * N);
        else oracle_window_sum(prod + f * N, W, H, R, window_type, S + f * N);
    }
#pragma omp parallel for
    for (long k = 0; k < (long)N; ++k) {
        double a = S[0 * N + k], b = S[1 * N + k], c = S[2 * N + k], p = S[3 * N + k], q = S[4 * N + k];
        double tr = a + c, du = 0.0, dv = 0.0;
        unsigned char ok = 0;
        if (tr > 0.0) {
            ok = 1;
            double lam = eps * tr / 2.0;
            double A = a + lam, C = c + lam, D = A * C - b * b;
            double rp = -(p + a * u[k] + b * v[k]);
            double rq = -(q + b * u[k] + c * v[k]);
            du = (C * rp - b * rq) / D;
            dv = (A * rq - b * rp) / D;
            if (du > max_step) du = max_step; if (du < -max_step) du = -max_step;
            if (dv > max_step) dv = max_step; if (dv < -max_step) dv = -max_step;
        }
        u[k] += du;
        v[k] += dv;
        if (valid) valid[k] = ok;
        if (det) det[k] = a * c - b * b;
        if (mask && !mask[k]) {                     /* M3: no vector over an obstacle */
            u[k] = 0.0; v[k] = 0.0;
            if (valid) valid[k] = 0;
            if (det) det[k] = 0.0;
        }
    }
    if (sums5) memcpy(sums5, S, sizeof(double) * N * 5);
    free(S); free(prod); free(Iy); free(Ix); free(I2w);
}

void oracle_iteration(const double *I1, const double *I2, int W, int H, int R, int window_type,
                      double eps, double max_step, double *u, double *v, double *sums5,
                      unsigned char *valid, double *det, int direct_sums)
{
    oracle_iteration_masked(I1, I2, NULL, W, H, R, window_type, eps, max_step, u, v, sums5, valid, det, direct_sums);
}

/* NEXT item f4: masks over obstacles and side walls ("using masks to avoid
 * computations over obstacles or side walls").  The paper gives no more than that sentence; readings:
 *   M1 the mask is one byte per level-0 pixel, non-zero = fluid (computed), 0 = obstacle;
 *   M2 an obstacle pixel has zero weight in every window sum (its five products are dropped);
 *   M3 an obstacle pixel carries no vector: u = v = 0, valid = 0, det = 0, at every level and at every
 *      moment of the solve (after each update and after the hand-down);
 *   M4 level l+1 pixel (X,Y) is fluid iff at least one of its in-image children (2X..2X+1, 2Y..2Y+1) is;
 *   M5 the images themselves are not altered (the pyramid filter, the gradients and the warp read
 *      obstacle pixels as they are).
 * This function is M4. */
void oracle_mask_downsample(const unsigned char *src, int W, int H, unsigned char *dst)
{
    int Wd = (W + 1) / 2, Hd = (H + 1) / 2;
    for (int Y = 0; Y < Hd; ++Y)
        for (int X = 0; X < Wd; ++X) {
            int any = 0;
            for (int dy = 0; dy < 2; ++dy)
                for (int dx = 0; dx < 2; ++dx) {
                    int x = 2 * X + dx, y = 2 * Y + dy;
                    if (x < W && y < H && src[(size_t)y * W + x]) any = 1;
                }
            dst[(size_t)Y * Wd + X] = (unsigned char)any;
        }
}

/* The whole solve O1..O5.  I1, I2: level-0 images as doubles (exact conversion of the integer
 * frames, no scaling, D17).  levels >= 1 counts the base image (D3).  Outputs: u, v (level 0),
 * valid and det (optional) from the last iteration of level 0.
 * level_u / level_v (optional): arrays of `levels` pointers, each receiving that level's final field.
 * Returns 0, or -1 on bad arguments (coarsest level smaller than the window). */
int oracle_solve_masked(const double *I1, const double *I2, const unsigned char *mask, int W, int H, int levels,
                        int R, int iterations, int window_type, double eps, double max_step, double *u, double *v,
                        unsigned char *valid, double *det, double **level_u, double **level_v,
                        int direct_sums)
{
    if (W < 1 || H < 1 || levels < 1 || levels > 16 || R < 1 || iterations < 1) return -1;
    int Ws[16], Hs[16];
    Ws[0] = W; Hs[0] = H;
    for (int l = 1; l < levels; ++l) { Ws[l] = (Ws[l - 1] + 1) / 2; Hs[l] = (Hs[l - 1] + 1) / 2; }
    if (Ws[levels - 1] < 2 * R + 1 || Hs[levels - 1] < 2 * R + 1) return -1;

    double *P1[16], *P2[16];
    P1[0] = (double *)I1; P2[0] = (double *)I2;
    for (int l = 1; l < levels; ++l) {
        P1[l] = (double *)malloc(sizeof(double) * (size_t)Ws[l] * Hs[l]);
        P2[l] = (double *)malloc(sizeof(double) * (size_t)Ws[l] * Hs[l]);
        oracle_downsample(P1[l - 1], Ws[l - 1], Hs[l - 1], P1[l]);
        oracle_downsample(P2[l - 1], Ws[l - 1], Hs[l - 1], P2[l]);
    }
    unsigned char *M[16];                 /* mask == NULL: no mask at any level */
    M[0] = (unsigned char *)mask;
    for (int l = 1; l < levels; ++l) {
        M[l] = NULL;
        if (mask) {
            M[l] = (unsigned char *)malloc((size_t)Ws[l] * Hs[l]);
            oracle_mask_downsample(M[l - 1], Ws[l - 1], Hs[l - 1], M[l]);
        }
    }
    double *uc = NULL, *vc = NULL;        /* field of the level just finished */
    for (int l = levels - 1; l >= 0; --l) {
        size_t N = (size_t)Ws[l] * Hs[l];
        double *ul = (double *)calloc(N, sizeof(double));   /* O3: zero initial guess */
        double *vl = (double *)calloc(N, sizeof(double));
        if (l < levels - 1) {
            oracle_upsample_flow(uc, Ws[l + 1], Hs[l + 1], ul, Ws[l], Hs[l]);
            oracle_upsample_flow(vc, Ws[l + 1], Hs[l + 1], vl, Ws[l], Hs[l]);
            free(uc); free(vc);
            if (M[l])                                       /* M3 */
                for (size_t k = 0; k < N; ++k)
                    if (!M[l][k]) { ul[k] = 0.0; vl[k] = 0.0; }
        }
        for (int n = 0; n < iterations; ++n)
            oracle_iteration_masked(P1[l], P2[l], M[l], Ws[l], Hs[l], R, window_type, eps, max_step, ul, vl, NULL,
                                    (l == 0) ? valid : NULL, (l == 0) ? det : NULL, direct_sums);
        if (level_u && level_u[l]) memcpy(level_u[l], ul, sizeof(double) * N);
        if (level_v && level_v[l]) memcpy(level_v[l], vl, sizeof(double) * N);
        uc = ul; vc = vl;
    }
    memcpy(u, uc, sizeof(double) * (size_t)W * H);
    memcpy(v, vc, sizeof(double) * (size_t)W * H);
    free(uc); free(vc);
    for (int l = 1; l < levels; ++l) { free(P1[l]); free(P2[l]); free(M[l]); }
    return 0;
}

int oracle_solve(const double *I1, const double *I2, int W, int H, int levels, int R, int iterations,
                 int window_type, double eps, double max_step, double *u, double *v,
                 unsigned char *valid, double *det, double **level_u, double **level_v,
                 int direct_sums)
{
    return oracle_solve_masked(I1, I2, NULL, W, H, levels, R, iterations, window_type, eps, max_step, u, v,
                               valid, det, level_u, level_v, direct_sums);
}

/* NEXT item f1: local equalisation pre-filter, eq. 2 of the paper:
 *     In(x,y) = ( I(x,y) - mean(x,y) ) / sqrt( mean_of_squares(x,y) - mean(x,y)^2 )
 * "where [the bar] is a local mean for a given radius.  We choose a radius of 5 pixels."  The printed
 * denominator is garbled (D19); this is the zero-mean, unit-local-standard-deviation reading the text
 * gives ("the mean intensity value is subtracted ... and divided by the local intensity standard
 * deviation").  Readings: E1 the local mean is the plain average over the (2r+1)^2 box; E2 at the
 * borders over the in-image part of the box (divided by the number of pixels actually summed), so
 * a constant image has zero mean-removed value everywhere; E3 where the local variance is not
 * positive (flat neighbourhood) the output is 0; E4 no rescaling afterwards (the solve is gain and
 * offset invariant); E5 applied to both images before the pyramid.
 * Plain double loops over the window, no running sums. */
void oracle_equalise(const double *src, int W, int H, int r, double *dst)
{
#pragma omp parallel for
    for (int y = 0; y < H; ++y)
        for (int x = 0; x < W; ++x) {
            double s = 0.0, s2 = 0.0;
            int n = 0;
            for (int dy = -r; dy <= r; ++dy)
                for (int dx = -r; dx <= r; ++dx) {
                    int xx = x + dx, yy = y + dy;
                    if (xx < 0 || xx >= W || yy < 0 || yy >= H) continue;
                    double v = src[(size_t)yy * W + xx];
                    s += v;
                    s2 += v * v;
                    ++n;
                }
            double mean = s / n;
            double num = n * s2 - s * s;              /* n^2 * variance: exact for integer images */
            dst[(size_t)y * W + x] = num > 0.0 ? (src[(size_t)y * W + x] - mean) / (sqrt(num) / n) : 0.0;
        }
}

int oracle_num_threads(void)
{
#ifdef _OPENMP
    extern int omp_get_max_threads(void);
    return omp_get_max_threads();
#else
    return 1;
#endif
}
