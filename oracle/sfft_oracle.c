/*
 * sfft_oracle.c -- plain, slow, obviously-correct CPU reference for the SFFT
 * subtraction hot path.  TEST INFRASTRUCTURE ONLY: nothing on the product path may
 * call, link or import this file (only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs do).  It shares no code with the
 * CUDA library.
 *
 * What it computes (BASELINE.json north_star; SURVEY.md section 8(c) "Oracle" items 1-5;
 * the paper itself only names the method: "Saccadic Fast Fourier
 * Transform (SFFT) method for difference imaging", "flexible delta basis
 * function", "Apply SFFT subtraction"):
 *
 *     D = S - (R (*) K(x,y)) - B(x,y)
 *
 *  K: L x L delta-basis kernel whose coefficients vary as a 2-D polynomial of degree
 *  DK; B: background polynomial of degree DB.  The coefficients are the linear
 *  least-squares solution of  min || vec(m.S) - A c ||_2  where
 *    column (t,u,v) of A is the image (x,y) -> T_t((x-u) mod nx, (y-v) mod ny),
 *        T_t = xt^i yt^j (m.R),  t <-> (i,j), i+j <= DK,
 *    column s of A is P_s = xt^p yt^q, s <-> (p,q), p+q <= DB   (not masked),
 *  with xt = (2x+1-nx)/nx, yt = (2y+1-ny)/ny  (readings C2, C3, C4, C6, C7).
 *
 *  G = A^T A and h = A^T b are assembled BY DIRECT PIXEL SUMMATION of shifted,
 *  polynomial-weighted products (north_star: "assembles A^T A and A^T b by direct
 *  pixel summation"), the system is solved by textbook Cholesky, and the model is
 *  convolved in real space.  No FFT anywhere in this file.
 *
 * Precision: FP64; every image row is summed in FP64 and rows are combined in
 * long double, so the oracle's own error is << 1e-10.
 *
 * Index conventions (SURVEY.md 8(b) "Coefficient layout"):
 *   w = (L-1)/2, NK = (DK+1)(DK+2)/2, NB = (DB+1)(DB+2)/2, n = L*L*NK + NB
 *   index(t,u,v) = t*L*L + (v+w)*L + (u+w),   index(s) = NK*L*L + s
 *   (i,j) order: total degree ascending, then j ascending: (0,0),(1,0),(0,1),(2,0),...
 *
 * Pins: tests/test_oracle_pins.py (P1..P11 of SURVEY.md 8(c)); every exported
 * function below is pinned there -- none is "parity unpinned".
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define ORACLE_OK 0
#define ORACLE_ERR_INVALID_ARG (-1)
#define ORACLE_ERR_ALLOC (-2)
#define ORACLE_ERR_NOT_SPD (-5)

/* reading C9: pivot of the unit-diagonal (equilibrated) matrix at or below this => NOT_SPD */
#define ORACLE_PIVOT_MIN 1e-12

static int imod(int a, int n) { int r = a % n; return r < 0 ? r + n : r; }

int oracle_num_poly(int deg) { return (deg + 1) * (deg + 2) / 2; }

int oracle_num_unknowns(int L, int DK, int DB) {
    return L * L * oracle_num_poly(DK) + oracle_num_poly(DB);
}

/* t -> (i,j): total degree ascending, then j ascending (reading C4) */
void oracle_poly_index(int t, int *i, int *j) {
    int d = 0;
    while (t > d) { t -= d + 1; d++; }
    *j = t; *i = d - t;
}

/* centred pixel coordinate (reading C3) */
double oracle_coord(int x, int n) { return (2.0 * x + 1.0 - n) / (double)n; }

static double ipow(double b, int e) { double r = 1.0; while (e-- > 0) r *= b; return r; }

/* out(x,y) = xt(x)^i * yt(y)^j * (mask ? mask(x,y) : 1) * img(x,y)   [north_star (a)] */
void oracle_weighted_image(const double *img, const uint8_t *mask, int nx, int ny,
                           int i, int j, double *out) {
#pragma omp parallel for schedule(static)
    for (int y = 0; y < ny; y++) {
        double wy = ipow(oracle_coord(y, ny), j);
        for (int x = 0; x < nx; x++) {
            size_t k = (size_t)y * nx + x;
            double m = mask ? (mask[k] ? 1.0 : 0.0) : 1.0;
            out[k] = ipow(oracle_coord(x, nx), i) * wy * m * img[k];
        }
    }
}

/* out(x,y) = xt(x)^p * yt(y)^q  (background basis image P_s; never masked, C7) */
void oracle_poly_image(int nx, int ny, int p, int q, double *out) {
    for (int y = 0; y < ny; y++)
        for (int x = 0; x < nx; x++)
            out[(size_t)y * nx + x] = ipow(oracle_coord(x, nx), p) * ipow(oracle_coord(y, ny), q);
}

/* circular cross-correlation at one lag, by direct summation (SURVEY.md 8 "Notation"):
 *   X(a,b)[du,dv] = sum_{x,y} a(x,y) * b((x+du) mod nx, (y+dv) mod ny)               */
double oracle_lag_sum(const double *a, const double *b, int nx, int ny, int du, int dv) {
    long double total = 0.0L;
    int s = imod(du, nx); /* x2 = x + s for x < nx - s, else x + s - nx */
#pragma omp parallel for schedule(static) reduction(+ : total)
    for (int y = 0; y < ny; y++) {
        const double *ar = a + (size_t)y * nx;
        const double *br = b + (size_t)imod(y + dv, ny) * nx;
        double acc = 0.0;
        int split = nx - s;
#pragma omp simd reduction(+ : acc)
        for (int x = 0; x < split; x++) acc += ar[x] * br[x + s];
#pragma omp simd reduction(+ : acc)
        for (int x = split; x < nx; x++) acc += ar[x] * br[x + s - nx];
        total += (long double)acc;
    }
    return (double)total;
}

/* plain sum of products (lag 0 shortcut-free helper for Phi and Delta) */
static double dot_images(const double *a, const double *b, int nx, int ny) {
    return oracle_lag_sum(a, b, nx, ny, 0, 0);
}

/* Assemble G (n x n, full, symmetric) and h (n) by one direct sum per (pair, lag).
 * Because the boundary is circular (C6), G[(t,u,v),(t',u',v')] depends only on
 * (t,t',u-u',v-v'):  = X(T_t,T_t')[u-u', v-v'];  G[(t,u,v),s] = X(T_t,P_s)[u,v];
 * G[s,s'] = sum P_s P_s';  h[(t,u,v)] = X(T_t, m.S)[u,v];  h[s] = sum P_s (m.S)
 * (SURVEY.md 8(a) rows a2, a3).  The lower triangle is computed, then mirrored
 * (A^T A is symmetric by construction); tests pin the shortcut against the dense
 * A^T A of oracle_build_system_dense (pin P4).                                     */
int oracle_build_system(const double *S, const double *R, const uint8_t *mask,
                        int nx, int ny, int L, int DK, int DB, double *G, double *h) {
    if (!S || !R || !G || !h || L < 1 || (L & 1) == 0 || DK < 0 || DB < 0 ||
        nx < 2 * L - 1 || ny < 2 * L - 1)
        return ORACLE_ERR_INVALID_ARG;
    const int w = (L - 1) / 2, NK = oracle_num_poly(DK), NB = oracle_num_poly(DB);
    const int LL = L * L, n = LL * NK + NB;
    const size_t npix = (size_t)nx * ny;
    double *T = (double *)malloc(sizeof(double) * npix * NK);
    double *P = (double *)malloc(sizeof(double) * npix * NB);
    double *Sf = (double *)malloc(sizeof(double) * npix);
    const int W2 = 2 * L - 1; /* lags -2w..2w */
    double *lag = (double *)malloc(sizeof(double) * W2 * W2);
    if (!T || !P || !Sf || !lag) { free(T); free(P); free(Sf); free(lag); return ORACLE_ERR_ALLOC; }

    for (int t = 0; t < NK; t++) {
        int i, j; oracle_poly_index(t, &i, &j);
        oracle_weighted_image(R, mask, nx, ny, i, j, T + npix * t);
    }
    for (int s = 0; s < NB; s++) {
        int p, q; oracle_poly_index(s, &p, &q);
        oracle_poly_image(nx, ny, p, q, P + npix * s);
    }
    oracle_weighted_image(S, mask, nx, ny, 0, 0, Sf);
    memset(G, 0, sizeof(double) * (size_t)n * n);

    /* kernel-kernel blocks: rows (t,u,v) >= cols (t',u',v') */
    for (int t = 0; t < NK; t++)
        for (int tp = 0; tp <= t; tp++) {
            /* lag (du,dv) = (u-u', v-v'); for t == tp only lags with (dv,du) >= (0,0)
             * lexicographically occur in the lower triangle */
            memset(lag, 0, sizeof(double) * W2 * W2);
            for (int dv = -2 * w; dv <= 2 * w; dv++)
                for (int du = -2 * w; du <= 2 * w; du++)
                    if (t != tp || dv > 0 || (dv == 0 && du >= 0))
                        lag[(dv + 2 * w) * W2 + (du + 2 * w)] =
                            oracle_lag_sum(T + npix * t, T + npix * tp, nx, ny, du, dv);
            for (int v = -w; v <= w; v++)
                for (int u = -w; u <= w; u++)
                    for (int vp = -w; vp <= w; vp++)
                        for (int up = -w; up <= w; up++) {
                            int r = t * LL + (v + w) * L + (u + w);
                            int c = tp * LL + (vp + w) * L + (up + w);
                            if (r < c) continue;
                            /* G[r,c] = sum_p T_t(p-(u,v)) T_t'(p-(u',v'))
                             *        = sum_q T_t(q) T_t'(q + (u-u', v-v'))            */
                            G[(size_t)r * n + c] = lag[(v - vp + 2 * w) * W2 + (u - up + 2 * w)];
                        }
        }
    /* kernel-background blocks and right-hand side */
    for (int t = 0; t < NK; t++)
        for (int v = -w; v <= w; v++)
            for (int u = -w; u <= w; u++) {
                int r = t * LL + (v + w) * L + (u + w);
                for (int s = 0; s < NB; s++) /* sum_p T_t(p-(u,v)) P_s(p) = X(T_t,P_s)[u,v] */
                    G[(size_t)(NK * LL + s) * n + r] =
                        oracle_lag_sum(T + npix * t, P + npix * s, nx, ny, u, v);
                h[r] = oracle_lag_sum(T + npix * t, Sf, nx, ny, u, v);
            }
    for (int s = 0; s < NB; s++) {
        for (int sp = 0; sp <= s; sp++)
            G[(size_t)(NK * LL + s) * n + NK * LL + sp] = dot_images(P + npix * s, P + npix * sp, nx, ny);
        h[NK * LL + s] = dot_images(P + npix * s, Sf, nx, ny);
    }
    for (int r = 0; r < n; r++)
        for (int c = r + 1; c < n; c++) G[(size_t)r * n + c] = G[(size_t)c * n + r];
    free(T); free(P); free(Sf); free(lag);
    return ORACLE_OK;
}

/* Explicit dense design matrix A (npix x n, row-major), for tiny images only (pin P4). */
int oracle_design_matrix(const double *R, const uint8_t *mask, int nx, int ny,
                         int L, int DK, int DB, double *A) {
    if (!R || !A || L < 1 || (L & 1) == 0) return ORACLE_ERR_INVALID_ARG;
    const int w = (L - 1) / 2, NK = oracle_num_poly(DK), NB = oracle_num_poly(DB);
    const int LL = L * L, n = LL * NK + NB;
    const size_t npix = (size_t)nx * ny;
    double *T = (double *)malloc(sizeof(double) * npix);
    if (!T) return ORACLE_ERR_ALLOC;
    for (int t = 0; t < NK; t++) {
        int i, j; oracle_poly_index(t, &i, &j);
        oracle_weighted_image(R, mask, nx, ny, i, j, T);
        for (int v = -w; v <= w; v++)
            for (int u = -w; u <= w; u++) {
                int c = t * LL + (v + w) * L + (u + w);
                for (int y = 0; y < ny; y++)
                    for (int x = 0; x < nx; x++)
                        A[((size_t)y * nx + x) * n + c] =
                            T[(size_t)imod(y - v, ny) * nx + imod(x - u, nx)];
            }
    }
    for (int s = 0; s < NB; s++) {
        int p, q; oracle_poly_index(s, &p, &q);
        for (int y = 0; y < ny; y++)
            for (int x = 0; x < nx; x++)
                A[((size_t)y * nx + x) * n + NK * LL + s] =
                    ipow(oracle_coord(x, nx), p) * ipow(oracle_coord(y, ny), q);
    }
    free(T);
    return ORACLE_OK;
}

/* G = A^T A, h = A^T b from the explicit A, no lag shortcut (pin P4, tiny only). */
int oracle_build_system_dense(const double *S, const double *R, const uint8_t *mask,
                              int nx, int ny, int L, int DK, int DB, double *G, double *h) {
    const int n = oracle_num_unknowns(L, DK, DB);
    const size_t npix = (size_t)nx * ny;
    double *A = (double *)malloc(sizeof(double) * npix * n);
    if (!A) return ORACLE_ERR_ALLOC;
    int rc = oracle_design_matrix(R, mask, nx, ny, L, DK, DB, A);
    if (rc) { free(A); return rc; }
    for (int r = 0; r < n; r++) {
        for (int c = 0; c < n; c++) {
            long double acc = 0.0L;
            for (size_t k = 0; k < npix; k++) acc += (long double)A[k * n + r] * A[k * n + c];
            G[(size_t)r * n + c] = (double)acc;
        }
        long double acc = 0.0L;
        for (size_t k = 0; k < npix; k++) {
            double m = mask ? (mask[k] ? 1.0 : 0.0) : 1.0;
            acc += (long double)A[k * n + r] * (m * S[k]);
        }
        h[r] = (double)acc;
    }
    free(A);
    return ORACLE_OK;
}

/* Textbook (unblocked, scalar) Cholesky solve of G c = h after symmetric diagonal
 * equilibration Gt = D^-1/2 G D^-1/2 (reading C9).
 * Lfac (n x n, optional) receives the lower factor of Gt.                          */
int oracle_solve(const double *G, const double *h, int n, double *c, double *Lfac) {
    if (!G || !h || !c || n < 1) return ORACLE_ERR_INVALID_ARG;
    double *A = (double *)malloc(sizeof(double) * (size_t)n * n);
    double *d = (double *)malloc(sizeof(double) * n);
    double *y = (double *)malloc(sizeof(double) * n);
    if (!A || !d || !y) { free(A); free(d); free(y); return ORACLE_ERR_ALLOC; }
    int rc = ORACLE_OK;
    for (int i = 0; i < n; i++) {
        double g = G[(size_t)i * n + i];
        if (!(g > 0.0)) { rc = ORACLE_ERR_NOT_SPD; goto done; }
        d[i] = 1.0 / sqrt(g);
    }
    for (int i = 0; i < n; i++)
        for (int j = 0; j <= i; j++) A[(size_t)i * n + j] = d[i] * G[(size_t)i * n + j] * d[j];
    /* Cholesky-Banachiewicz, row by row */
    for (int i = 0; i < n; i++)
        for (int j = 0; j <= i; j++) {
            double s = A[(size_t)i * n + j];
            for (int k = 0; k < j; k++) s -= A[(size_t)i * n + k] * A[(size_t)j * n + k];
            if (i == j) {
                if (!(s > ORACLE_PIVOT_MIN)) { rc = ORACLE_ERR_NOT_SPD; goto done; }
                A[(size_t)i * n + i] = sqrt(s);
            } else {
                A[(size_t)i * n + j] = s / A[(size_t)j * n + j];
            }
        }
    for (int i = 0; i < n; i++) { /* L y = D^-1/2 h */
        double s = d[i] * h[i];
        for (int k = 0; k < i; k++) s -= A[(size_t)i * n + k] * y[k];
        y[i] = s / A[(size_t)i * n + i];
    }
    for (int i = n - 1; i >= 0; i--) { /* L^T z = y ; c = D^-1/2 z */
        double s = y[i];
        for (int k = i + 1; k < n; k++) s -= A[(size_t)k * n + i] * c[k];
        c[i] = s / A[(size_t)i * n + i];
    }
    for (int i = 0; i < n; i++) c[i] *= d[i];
    if (Lfac)
        for (int i = 0; i < n; i++)
            for (int j = 0; j < n; j++) Lfac[(size_t)i * n + j] = j <= i ? A[(size_t)i * n + j] : 0.0;
done:
    free(A); free(d); free(y);
    return rc;
}

/* Model value at one output pixel, real-space:
 *   M(x,y) = sum_t sum_{u,v} a_{t,u,v} xt(xs)^i yt(ys)^j R(xs,ys),
 *   (xs,ys) = ((x-u) mod nx, (y-v) mod ny);  UNMASKED R (reading C7).              */
static double model_pixel(const double *R, int nx, int ny, int L, int DK,
                          const double *c, int x, int y) {
    const int w = (L - 1) / 2, NK = oracle_num_poly(DK), LL = L * L;
    long double acc = 0.0L;
    for (int v = -w; v <= w; v++) {
        int ys = imod(y - v, ny);
        double yt = oracle_coord(ys, ny);
        for (int u = -w; u <= w; u++) {
            int xs = imod(x - u, nx);
            double xt = oracle_coord(xs, nx);
            double r = R[(size_t)ys * nx + xs];
            double k = 0.0; /* local kernel value K(u,v; xs,ys) = sum_t a_t xt^i yt^j */
            for (int t = 0; t < NK; t++) {
                int i, j; oracle_poly_index(t, &i, &j);
                k += c[t * LL + (v + w) * L + (u + w)] * ipow(xt, i) * ipow(yt, j);
            }
            acc += (long double)(k * r);
        }
    }
    return (double)acc;
}

static double background_pixel(int nx, int ny, int L, int DK, int DB, const double *c, int x, int y) {
    const int NK = oracle_num_poly(DK), NB = oracle_num_poly(DB), LL = L * L;
    double xt = oracle_coord(x, nx), yt = oracle_coord(y, ny), b = 0.0;
    for (int s = 0; s < NB; s++) {
        int p, q; oracle_poly_index(s, &p, &q);
        b += c[NK * LL + s] * ipow(xt, p) * ipow(yt, q);
    }
    return b;
}

/* D = S - M - B over the whole image, real space [north_star (d)] */
int oracle_subtract(const double *S, const double *R, int nx, int ny, int L, int DK, int DB,
                    const double *c, double *D) {
    if (!S || !R || !c || !D || (L & 1) == 0) return ORACLE_ERR_INVALID_ARG;
#pragma omp parallel for schedule(dynamic, 4)
    for (int y = 0; y < ny; y++)
        for (int x = 0; x < nx; x++)
            D[(size_t)y * nx + x] = S[(size_t)y * nx + x] - model_pixel(R, nx, ny, L, DK, c, x, y) -
                                    background_pixel(nx, ny, L, DK, DB, c, x, y);
    return ORACLE_OK;
}

/* D at a list of pixels only (full-size parity on sampled outputs) */
int oracle_subtract_at(const double *S, const double *R, int nx, int ny, int L, int DK, int DB,
                       const double *c, const int *xs, const int *ys, int npts, double *Dout) {
    if (!S || !R || !c || !xs || !ys || !Dout || (L & 1) == 0) return ORACLE_ERR_INVALID_ARG;
#pragma omp parallel for schedule(dynamic, 16)
    for (int k = 0; k < npts; k++) {
        int x = xs[k], y = ys[k];
        Dout[k] = S[(size_t)y * nx + x] - model_pixel(R, nx, ny, L, DK, c, x, y) -
                  background_pixel(nx, ny, L, DK, DB, c, x, y);
    }
    return ORACLE_OK;
}

/* One entry of G (or of h when col < 0) by its definition as a direct sum; used to
 * check sampled entries at sizes where assembling all of G takes minutes.
 * Twork: caller-provided scratch of 3*nx*ny doubles.                                */
int oracle_system_entry(const double *S, const double *R, const uint8_t *mask,
                        int nx, int ny, int L, int DK, int DB, int row, int col,
                        double *Twork, double *out) {
    const int w = (L - 1) / 2, NK = oracle_num_poly(DK), LL = L * L;
    const int n = oracle_num_unknowns(L, DK, DB);
    const size_t npix = (size_t)nx * ny;
    if (row < 0 || row >= n || col >= n || !Twork || !out) return ORACLE_ERR_INVALID_ARG;
    double *A = Twork, *B = Twork + npix;
    int du = 0, dv = 0, su = 0, sv = 0;
    /* image for `row`, un-shifted, and its shift (u,v) */
    if (row < NK * LL) {
        int t = row / LL, i, j; oracle_poly_index(t, &i, &j);
        sv = (row % LL) / L - w; su = (row % LL) % L - w;
        oracle_weighted_image(R, mask, nx, ny, i, j, A);
    } else {
        int p, q; oracle_poly_index(row - NK * LL, &p, &q);
        oracle_poly_image(nx, ny, p, q, A);
    }
    if (col < 0) {
        oracle_weighted_image(S, mask, nx, ny, 0, 0, B);
    } else if (col < NK * LL) {
        int t = col / LL, i, j; oracle_poly_index(t, &i, &j);
        dv = (col % LL) / L - w; du = (col % LL) % L - w;
        oracle_weighted_image(R, mask, nx, ny, i, j, B);
    } else {
        int p, q; oracle_poly_index(col - NK * LL, &p, &q);
        oracle_poly_image(nx, ny, p, q, B);
    }
    /* sum_p A(p-(su,sv)) B(p-(du,dv)) = sum_q A(q) B(q + (su-du, sv-dv)) */
    *out = oracle_lag_sum(A, B, nx, ny, su - du, sv - dv);
    return ORACLE_OK;
}
