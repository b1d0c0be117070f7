/*
 * oracle.c -- plain, slow, float64 CPU restatement of the background + detection hot path of
 * arxiv 2502.10783 ("Image Pre-Processing Framework for Time-Domain Astronomy in the Artificial
 * Intelligence Era"), written from the paper text only.
 *
 * THIS IS TEST INFRASTRUCTURE.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may build, load or call it.  It shares no code, header, table or helper with
 * the CUDA library under paper_2502_10783_b200/ and neither includes the other.
 *
 * Every step is the definition (or the paper's procedure) written out, one pass per step, no
 * blocking, fusion or reordering.  OpenMP is used only over independent outer units (meshes, rows).
 * Input pixels are float32, promoted exactly to float64.  Readings of points where the paper is
 * silent or garbled are the A1..A22 readings of SURVEY.md section 8(c), repeated in DESIGN.md.
 *
 * Pins (tests/test_oracle_*.py, `-m "not gpu"`): O1 numpy median/mean/std special case, closed-form
 * truncated-Gaussian recurrence, hand-made outlier mesh, brute-force masked loop; O2
 * scipy.ndimage.generic_filter(nanmedian); O3 scipy.ndimage.zoom(order=3, mode='reflect',
 * grid_mode=True); O4 Gaussian tail fraction; O5 exhaustive 4x4 masks vs transitive closure,
 * scipy.ndimage.label partitions; O6 analytic Gaussian flux/centroid/moments, hand-made components.
 * No function here is "parity unpinned".
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

/* ------------------------------------------------------------------------------------------------
 * O1  per-mesh sigma-clipped statistics and background estimators.
 * PAPER.md:67 (rectangular sub-regions, default 64x64), :69-76 (eqs. 1-4), :78 ("determine the upper
 * and lower limits based on the calculated central value and the specified sigma range, exclude data
 * outside these limits, and recalculate ... Once the maximum number of iterations is reached or the
 * data stabilizes, the background value for each sub-region is obtained").
 * Readings: A1 even-N median = mean of the two middle values; A2/A4 estimator =
 * median_factor*median - mean_factor*mean; A5 centre = median, spread = population std about the
 * mean; A6 inclusive bounds; A7 final statistics recomputed on the survivors; A8 ddof 0; A9 partial
 * edge meshes are their own mesh; A12 optional skew guard.
 * ---------------------------------------------------------------------------------------------- */
static int cmp_double(const void *a, const void *b) {
    double x = *(const double *)a, y = *(const double *)b;
    return (x > y) - (x < y);
}

/* eq. 1: median of S[0..n); scratch has room for n doubles */
static double median_of(const double *S, int n, double *scratch) {
    memcpy(scratch, S, (size_t)n * sizeof(double));
    qsort(scratch, (size_t)n, sizeof(double), cmp_double);
    if (n % 2 == 1) return scratch[(n - 1) / 2];            /* I_{(N+1)/2}, 1-based */
    return 0.5 * (scratch[n / 2 - 1] + scratch[n / 2]);      /* (I_{N/2} + I_{N/2+1}) / 2 */
}

/* eq. 2 */
static double mean_of(const double *S, int n) {
    double s = 0.0;
    for (int i = 0; i < n; ++i) s += S[i];
    return s / (double)n;
}

/* population standard deviation about the mean (two pass) */
static double std_of(const double *S, int n, double mu) {
    double s = 0.0;
    for (int i = 0; i < n; ++i) s += (S[i] - mu) * (S[i] - mu);
    return sqrt(s / (double)n);
}

void o1_mesh_stats(const float *img, int H, int W, int mh, int mw, double k_c, int iters,
                   double median_factor, double mean_factor, int skew_guard,
                   double *bkg_mesh, double *rms_mesh, int32_t *n_kept,
                   double *median_mesh, double *mean_mesh, int32_t *rounds_mesh) {
    int ny = (H + mh - 1) / mh, nx = (W + mw - 1) / mw;
#pragma omp parallel for schedule(dynamic, 1)
    for (int m = 0; m < ny * nx; ++m) {
        int j = m / nx, i = m % nx;
        int y0 = j * mh, y1 = (j + 1) * mh < H ? (j + 1) * mh : H;
        int x0 = i * mw, x1 = (i + 1) * mw < W ? (i + 1) * mw : W;
        int cap = (y1 - y0) * (x1 - x0);
        double *S = (double *)malloc((size_t)cap * sizeof(double));
        double *T = (double *)malloc((size_t)cap * sizeof(double));
        int n = 0;
        for (int y = y0; y < y1; ++y)
            for (int x = x0; x < x1; ++x) S[n++] = (double)img[(size_t)y * W + x];
        int rounds = 0;
        for (int it = 0; it < iters; ++it) {
            double med = median_of(S, n, T);
            double mu = mean_of(S, n);
            double sd = std_of(S, n, mu);
            double lo = med - k_c * sd, hi = med + k_c * sd;
            int n2 = 0;
            for (int q = 0; q < n; ++q)
                if (S[q] >= lo && S[q] <= hi) n2++;
            if (n2 == n || n2 == 0) break;
            n2 = 0;
            for (int q = 0; q < n; ++q)
                if (S[q] >= lo && S[q] <= hi) S[n2++] = S[q];
            n = n2;
            rounds++;
        }
        double med = median_of(S, n, T);
        double mu = mean_of(S, n);
        double sd = std_of(S, n, mu);
        double bkg = median_factor * med - mean_factor * mu;   /* eqs. 1-4 as one formula */
        if (skew_guard) {                                      /* A12 */
            if (sd == 0.0) bkg = mu;
            else if (fabs(mu - med) / sd >= 0.3) bkg = med;
        }
        bkg_mesh[m] = bkg;
        rms_mesh[m] = sd;
        n_kept[m] = n;
        if (median_mesh) median_mesh[m] = med;
        if (mean_mesh) mean_mesh[m] = mu;
        if (rounds_mesh) rounds_mesh[m] = rounds;
        free(S);
        free(T);
    }
}

/* ------------------------------------------------------------------------------------------------
 * O2  median filter of the mesh grid.  PAPER.md:80 ("we apply a median filter to the estimated
 * background values").  Readings: A11 both grids use it; A13 window truncated at the grid border.
 * ---------------------------------------------------------------------------------------------- */
void o2_grid_median(const double *grid, int ny, int nx, int fh, int fw, double *out) {
    double *win = (double *)malloc((size_t)fh * fw * sizeof(double));
    double *tmp = (double *)malloc((size_t)fh * fw * sizeof(double));
    for (int j = 0; j < ny; ++j)
        for (int i = 0; i < nx; ++i) {
            int n = 0;
            for (int dj = -(fh / 2); dj <= fh / 2; ++dj)
                for (int di = -(fw / 2); di <= fw / 2; ++di) {
                    int jj = j + dj, ii = i + di;
                    if (jj < 0 || jj >= ny || ii < 0 || ii >= nx) continue;
                    win[n++] = grid[jj * nx + ii];
                }
            out[j * nx + i] = median_of(win, n, tmp);
        }
    free(win);
    free(tmp);
}

/* ------------------------------------------------------------------------------------------------
 * O3  cubic B-spline interpolation of the filtered grid to full resolution.  PAPER.md:80 ("we employ
 * spline interpolation to scale the refined background values back").  Reading A14: order 3, samples
 * at mesh centres, half-sample-symmetric boundary (c[-1]=c[0], c[n]=c[n-1]).
 * ---------------------------------------------------------------------------------------------- */

/* Solve the n x n system  (c[k-1] + 4 c[k] + c[k+1]) / 6 = f[k]  with c[-1]=c[0], c[n]=c[n-1] by dense
 * Gaussian elimination with partial pivoting (no band tricks). */
static void solve_spline_line(const double *f, int n, double *c) {
    double *A = (double *)calloc((size_t)n * (n + 1), sizeof(double));
    for (int k = 0; k < n; ++k) {
        int km = k - 1 < 0 ? 0 : k - 1;
        int kp = k + 1 > n - 1 ? n - 1 : k + 1;
        A[k * (n + 1) + km] += 1.0 / 6.0;
        A[k * (n + 1) + k] += 4.0 / 6.0;
        A[k * (n + 1) + kp] += 1.0 / 6.0;
        A[k * (n + 1) + n] = f[k];
    }
    for (int col = 0; col < n; ++col) {
        int piv = col;
        for (int r = col + 1; r < n; ++r)
            if (fabs(A[r * (n + 1) + col]) > fabs(A[piv * (n + 1) + col])) piv = r;
        if (piv != col)
            for (int q = 0; q <= n; ++q) {
                double t = A[col * (n + 1) + q];
                A[col * (n + 1) + q] = A[piv * (n + 1) + q];
                A[piv * (n + 1) + q] = t;
            }
        for (int r = col + 1; r < n; ++r) {
            double m = A[r * (n + 1) + col] / A[col * (n + 1) + col];
            if (m == 0.0) continue;
            for (int q = col; q <= n; ++q) A[r * (n + 1) + q] -= m * A[col * (n + 1) + q];
        }
    }
    for (int r = n - 1; r >= 0; --r) {
        double s = A[r * (n + 1) + n];
        for (int q = r + 1; q < n; ++q) s -= A[r * (n + 1) + q] * c[q];
        c[r] = s / A[r * (n + 1) + r];
    }
    free(A);
}

/* separable: along y (columns) first, then along x (rows) */
void o3_spline_coeffs(const double *grid, int ny, int nx, double *coef) {
    double *f = (double *)malloc((size_t)(ny > nx ? ny : nx) * sizeof(double));
    double *c = (double *)malloc((size_t)(ny > nx ? ny : nx) * sizeof(double));
    for (int i = 0; i < nx; ++i) {
        for (int j = 0; j < ny; ++j) f[j] = grid[j * nx + i];
        solve_spline_line(f, ny, c);
        for (int j = 0; j < ny; ++j) coef[j * nx + i] = c[j];
    }
    for (int j = 0; j < ny; ++j) {
        for (int i = 0; i < nx; ++i) f[i] = coef[j * nx + i];
        solve_spline_line(f, nx, c);
        for (int i = 0; i < nx; ++i) coef[j * nx + i] = c[i];
    }
    free(f);
    free(c);
}

/* cubic B-spline basis */
static double beta3(double t) {
    t = fabs(t);
    if (t < 1.0) return (4.0 - 6.0 * t * t + 3.0 * t * t * t) / 6.0;
    if (t < 2.0) return (2.0 - t) * (2.0 - t) * (2.0 - t) / 6.0;
    return 0.0;
}

/* half-sample-symmetric reflection of an index into [0, n): -1->0, -2->1, n->n-1, n+1->n-2 */
static int reflect_index(int k, int n) {
    int p = 2 * n;
    k %= p;
    if (k < 0) k += p;
    return k < n ? k : p - 1 - k;
}

void o3_spline_eval(const double *coef, int ny, int nx, int H, int W, int mh, int mw, double *out) {
#pragma omp parallel for schedule(static)
    for (int y = 0; y < H; ++y) {
        double v = ((double)y + 0.5) / (double)mh - 0.5;
        int j0 = (int)floor(v);
        for (int x = 0; x < W; ++x) {
            double u = ((double)x + 0.5) / (double)mw - 0.5;
            int i0 = (int)floor(u);
            double s = 0.0;
            for (int dj = -1; dj <= 2; ++dj)
                for (int di = -1; di <= 2; ++di)
                    s += beta3(v - (double)(j0 + dj)) * beta3(u - (double)(i0 + di)) *
                         coef[reflect_index(j0 + dj, ny) * nx + reflect_index(i0 + di, nx)];
            out[(size_t)y * W + x] = s;
        }
    }
}

/* ------------------------------------------------------------------------------------------------
 * O3b/O4  subtraction and threshold.  PAPER.md:61-65 (removal = subtraction), :153 ("identify pixels
 * whose flux exceeds a specified main threshold").  Reading A15: strict '>' of sub against
 * k_d * rms map, with an rms > 0 guard.  fragile = pixels within 1e-5*rms of the threshold
 * (BASELINE.json north_star: catalogues must agree except for such pixels).
 * ---------------------------------------------------------------------------------------------- */
void o4_subtract_threshold(const float *img, const double *bkg64, const double *rms64, int H, int W,
                           double k_d, double *sub64, float *sub32, uint8_t *mask, uint8_t *fragile) {
#pragma omp parallel for schedule(static)
    for (int y = 0; y < H; ++y)
        for (int x = 0; x < W; ++x) {
            size_t p = (size_t)y * W + x;
            double s = (double)img[p] - bkg64[p];
            double thr = k_d * rms64[p];
            if (sub64) sub64[p] = s;
            if (sub32) sub32[p] = (float)s;
            if (mask) mask[p] = (rms64[p] > 0.0 && s > thr) ? 1 : 0;
            if (fragile) fragile[p] = (fabs(s - thr) <= 1e-5 * rms64[p]) ? 1 : 0;
        }
}

/* ------------------------------------------------------------------------------------------------
 * O5  8-connected component labelling.  PAPER.md:153 ("These pixels are then connected to form source
 * candidates").  Reading A16: 8-connectivity.  Raster scan; each unlabelled foreground pixel seeds a
 * flood fill that writes label = 1 + (y*W + x) of the seed -- the seed of a raster scan is the
 * minimum raster index of its component.  Background 0.
 * ---------------------------------------------------------------------------------------------- */
void o5_label(const uint8_t *mask, int H, int W, int32_t *labels) {
    size_t P = (size_t)H * W;
    memset(labels, 0, P * sizeof(int32_t));
    int32_t *stack = (int32_t *)malloc(P * sizeof(int32_t));
    for (size_t seed = 0; seed < P; ++seed) {
        if (!mask[seed] || labels[seed]) continue;
        int32_t lab = (int32_t)seed + 1;
        size_t top = 0;
        stack[top++] = (int32_t)seed;
        labels[seed] = lab;
        while (top) {
            int32_t p = stack[--top];
            int y = p / W, x = p % W;
            for (int dy = -1; dy <= 1; ++dy)
                for (int dx = -1; dx <= 1; ++dx) {
                    int yy = y + dy, xx = x + dx;
                    if ((dy == 0 && dx == 0) || yy < 0 || yy >= H || xx < 0 || xx >= W) continue;
                    size_t q = (size_t)yy * W + xx;
                    if (mask[q] && !labels[q]) {
                        labels[q] = lab;
                        stack[top++] = (int32_t)q;
                    }
                }
        }
    }
    free(stack);
}

/* ------------------------------------------------------------------------------------------------
 * O6  per-component reduction.  PAPER.md:153 ("calculate peak values and total flux for each
 * candidate source"), :159 (isophotal photometry = sum over the component's pixels).  Readings A18
 * (intensity-weighted, 0-based pixel-centre coordinates, raw central moments), A19 (npix >= min_area),
 * A20 (labels keep all components; only the catalogue is filtered).  I = sub (float32 as the
 * interface materialises it, promoted to float64).  Two passes: sums and centroid, then central
 * moments about that centroid.  Output ascending label.
 * ---------------------------------------------------------------------------------------------- */
typedef struct {
    int32_t label, npix, xmin, xmax, ymin, ymax, xpeak, ypeak;
    double peak, flux, x, y, x2, y2, xy;
} o6_source;

int64_t o6_reduce(const int32_t *labels, const float *sub, int H, int W, int min_area,
                  o6_source *out, int64_t capacity) {
    size_t P = (size_t)H * W;
    int64_t ncomp = 0;
    for (size_t p = 0; p < P; ++p)
        if (labels[p] == (int32_t)p + 1) ncomp++;
    int32_t *slot_of = (int32_t *)malloc(P * sizeof(int32_t));   /* indexed by root pixel */
    o6_source *acc = (o6_source *)calloc((size_t)(ncomp ? ncomp : 1), sizeof(o6_source));
    double *sx = (double *)calloc((size_t)(ncomp ? ncomp : 1), sizeof(double));
    double *sy = (double *)calloc((size_t)(ncomp ? ncomp : 1), sizeof(double));
    int64_t next = 0;
    for (size_t p = 0; p < P; ++p) {
        int32_t lab = labels[p];
        if (!lab) continue;
        int y = (int)(p / W), x = (int)(p % W);
        double I = (double)sub[p];
        o6_source *a;
        if (lab == (int32_t)p + 1) {                 /* root: first pixel of its component in raster order */
            slot_of[p] = (int32_t)next;
            a = &acc[next++];
            a->label = lab; a->npix = 0; a->flux = 0.0;
            a->xmin = a->xmax = x; a->ymin = a->ymax = y;
            a->peak = I; a->xpeak = x; a->ypeak = y;
        } else {
            a = &acc[slot_of[lab - 1]];
        }
        a->npix++;
        a->flux += I;
        sx[a - acc] += I * (double)x;
        sy[a - acc] += I * (double)y;
        if (x < a->xmin) a->xmin = x;
        if (x > a->xmax) a->xmax = x;
        if (y < a->ymin) a->ymin = y;
        if (y > a->ymax) a->ymax = y;
        if (I > a->peak) { a->peak = I; a->xpeak = x; a->ypeak = y; }   /* ties keep the smallest raster index */
    }
    for (int64_t s = 0; s < ncomp; ++s) {
        acc[s].x = sx[s] / acc[s].flux;
        acc[s].y = sy[s] / acc[s].flux;
    }
    for (size_t p = 0; p < P; ++p) {
        int32_t lab = labels[p];
        if (!lab) continue;
        o6_source *a = &acc[slot_of[lab - 1]];
        double I = (double)sub[p];
        double dx = (double)(p % W) - a->x, dy = (double)(p / W) - a->y;
        a->x2 += I * dx * dx;
        a->y2 += I * dy * dy;
        a->xy += I * dx * dy;
    }
    int64_t nout = 0;
    for (int64_t s = 0; s < ncomp; ++s) {
        if (acc[s].npix < min_area) continue;
        acc[s].x2 /= acc[s].flux;
        acc[s].y2 /= acc[s].flux;
        acc[s].xy /= acc[s].flux;
        if (nout < capacity) out[nout] = acc[s];
        nout++;
    }
    free(slot_of); free(acc); free(sx); free(sy);
    return nout;
}

int o6_source_size(void) { return (int)sizeof(o6_source); }
