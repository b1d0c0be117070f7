// K2: median filter of the background and RMS mesh grids, then cubic-B-spline prefilter (step a2).
// PAPER.md:80 ("we apply a median filter to the estimated background values ... Following the smoothing
// process, we employ spline interpolation").  Grid-sized work (<= a few thousand cells per frame): one
// CTA per (frame, grid), float64 throughout.  Readings A11 (both grids), A13 (window truncated at the
// border), A14 (order 3, half-sample-symmetric ends: c[-1]=c[0], c[n]=c[n-1]).
#include "common.cuh"

namespace {

constexpr int K2_NT = 256;

// Window median of cell (j, i) by rank counting (no per-thread array: a dynamically indexed local array
// lives in local memory, which made the first version of this kernel 120 us for 1332 cells).
// Rank of element a = #(v < v_a) + #(v == v_a with smaller window index); ranks are a permutation of 0..n-1.
__device__ double window_median(const double *g, int ny, int nx, int j, int i, int fh, int fw) {
    const int j0 = max(0, j - fh / 2), j1 = min(ny - 1, j + fh / 2);
    const int i0 = max(0, i - fw / 2), i1 = min(nx - 1, i + fw / 2);
    const int ww = i1 - i0 + 1, n = (j1 - j0 + 1) * ww;
    const int k_lo = (n - 1) / 2, k_hi = n / 2;
    double lo = 0.0, hi = 0.0;
    for (int a = 0; a < n; ++a) {
        const double va = g[(j0 + a / ww) * nx + i0 + a % ww];
        int rank = 0;
        for (int b = 0; b < n; ++b) {
            const double vb = g[(j0 + b / ww) * nx + i0 + b % ww];
            rank += (vb < va || (vb == va && b < a)) ? 1 : 0;
        }
        if (rank == k_lo) lo = va;
        if (rank == k_hi) hi = va;
    }
    return (n & 1) ? lo : 0.5 * (lo + hi);
}

// Solve (c[k-1] + 4 c[k] + c[k+1]) / 6 = f[k], c[-1]=c[0], c[n]=c[n-1], along a strided line, in place
// (Thomas algorithm; the matrix is strictly diagonally dominant).  cp[k], im[k] are the forward-sweep
// factors, which depend on n only and are shared by every line of that length.
__device__ void spline_factors(double *cp, double *im, int n) {
    const double a = 1.0 / 6.0;
    double m = 5.0 / 6.0;
    im[0] = 1.0 / m;
    cp[0] = a / m;
    for (int k = 1; k < n; ++k) {
        const double bk = (k == n - 1) ? 5.0 / 6.0 : 4.0 / 6.0;
        m = bk - a * cp[k - 1];
        cp[k] = a / m;
        im[k] = 1.0 / m;
    }
}
__device__ void spline_line(double *f, const double *cp, const double *im, int n, int stride) {
    if (n == 1) return;   // (c0 + 4 c0 + c0)/6 = f0
    const double a = 1.0 / 6.0;
    double prev = f[0] * im[0];
    f[0] = prev;
    for (int k = 1; k < n; ++k) {
        prev = (f[(size_t)k * stride] - a * prev) * im[k];
        f[(size_t)k * stride] = prev;
    }
    for (int k = n - 2; k >= 0; --k) {
        prev = f[(size_t)k * stride] - cp[k] * prev;
        f[(size_t)k * stride] = prev;
    }
}

// One CTA per (frame, grid).  The grid is staged in shared memory when it fits (K2_SMEM_CELLS cells);
// otherwise the same code runs on global memory (scratch = 2 * ny * nx doubles per (frame, grid)... the
// raw grid is read in place and the coefficient array is the working array).
constexpr int K2_SMEM_CELLS = 2560;

__global__ void __launch_bounds__(K2_NT) k2_filter_prefilter(const double *bkg_raw, const double *rms_raw, int ny,
                                                             int nx, int fh, int fw, float *bkg_mesh,
                                                             float *rms_mesh, double *bkg_coef, double *rms_coef,
                                                             double *scratch) {
    __shared__ double s_raw[K2_SMEM_CELLS], s_work[K2_SMEM_CELLS];
    __shared__ double s_cp[2][128], s_im[2][128];
    const int frame = blockIdx.x, which = blockIdx.y;
    const size_t goff = (size_t)frame * ny * nx;
    const double *raw = (which ? rms_raw : bkg_raw) + goff;
    float *mesh = which ? rms_mesh : bkg_mesh;
    double *coef = (which ? rms_coef : bkg_coef) + goff;
    const int cells = ny * nx;
    const bool in_smem = cells <= K2_SMEM_CELLS && ny <= 128 && nx <= 128;
    double *fac = scratch + ((size_t)frame * 2 + which) * k2_scratch_per_grid(ny, nx);   // global factors otherwise
    double *cp_y = in_smem ? s_cp[0] : fac, *im_y = in_smem ? s_im[0] : fac + ny;
    double *cp_x = in_smem ? s_cp[1] : fac + 2 * ny, *im_x = in_smem ? s_im[1] : fac + 2 * ny + nx;
    const double *src = raw;
    double *work = coef;
    if (in_smem) {
        for (int c = threadIdx.x; c < cells; c += K2_NT) s_raw[c] = raw[c];
        src = s_raw;
        work = s_work;
    }
    if (threadIdx.x == 0) spline_factors(cp_y, im_y, ny);
    if (threadIdx.x == 32) spline_factors(cp_x, im_x, nx);
    __syncthreads();
    for (int c = threadIdx.x; c < cells; c += K2_NT) {
        const double med = window_median(src, ny, nx, c / nx, c % nx, fh, fw);
        work[c] = med;
        if (mesh) mesh[goff + c] = (float)med;
    }
    __syncthreads();
    for (int i = threadIdx.x; i < nx; i += K2_NT) spline_line(work + i, cp_y, im_y, ny, nx);   // along y
    __syncthreads();
    for (int j = threadIdx.x; j < ny; j += K2_NT) spline_line(work + (size_t)j * nx, cp_x, im_x, nx, 1);
    if (in_smem) {
        __syncthreads();
        for (int c = threadIdx.x; c < cells; c += K2_NT) coef[c] = s_work[c];
    }
}

}  // namespace

int k2_launch(bd_ctx *ctx, const double *d_bkg_raw, const double *d_rms_raw, int B, int ny, int nx, int fh, int fw,
              float *d_bkg_mesh, float *d_rms_mesh, double *d_bkg_coef, double *d_rms_coef, double *d_scratch,
              cudaStream_t st) {
    dim3 grid(B, 2);
    k2_filter_prefilter<<<grid, K2_NT, 0, st>>>(d_bkg_raw, d_rms_raw, ny, nx, fh, fw, d_bkg_mesh, d_rms_mesh,
                                               d_bkg_coef, d_rms_coef, d_scratch);
    BD_CUDA_CHECK(ctx, cudaGetLastError());
    return BD_OK;
}
