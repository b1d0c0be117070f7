// K2: median filter of the background and RMS mesh grids, then cubic-B-spline prefilter (step a2).
// PAPER.md:80 ("we apply a median filter to the estimated background values ... Following the smoothing
// process, we employ spline interpolation").  Grid-sized work (<= a few thousand cells per frame): one
// CTA per (frame, grid), float64 throughout.  Readings A11 (both grids), A13 (window truncated at the
// border), A14 (order 3, half-sample-symmetric ends: c[-1]=c[0], c[n]=c[n-1]).
#include "common.cuh"

namespace {

constexpr int K2_NT = 256;
constexpr int K2_MAXWIN = 121;   // 11 x 11

// Solve (c[k-1] + 4 c[k] + c[k+1]) / 6 = f[k], c[-1]=c[0], c[n]=c[n-1], along a strided line, in place.
// Thomas algorithm; `cp` is scratch with the same stride.  The matrix is strictly diagonally dominant.
__device__ void spline_line(double *f, double *cp, int n, int stride) {
    if (n == 1) return;   // (c0 + 4 c0 + c0)/6 = f0
    const double a = 1.0 / 6.0;
    double b0 = 5.0 / 6.0;
    cp[0] = a / b0;
    f[0] = f[0] / b0;
    for (int k = 1; k < n; ++k) {
        double bk = (k == n - 1) ? 5.0 / 6.0 : 4.0 / 6.0;
        double m = bk - a * cp[(size_t)(k - 1) * stride];
        cp[(size_t)k * stride] = a / m;
        f[(size_t)k * stride] = (f[(size_t)k * stride] - a * f[(size_t)(k - 1) * stride]) / m;
    }
    for (int k = n - 2; k >= 0; --k)
        f[(size_t)k * stride] -= cp[(size_t)k * stride] * f[(size_t)(k + 1) * stride];
}

__global__ void __launch_bounds__(K2_NT) k2_filter_prefilter(const double *bkg_raw, const double *rms_raw, int ny,
                                                             int nx, int fh, int fw, float *bkg_mesh,
                                                             float *rms_mesh, double *bkg_coef, double *rms_coef,
                                                             double *scratch) {
    const int frame = blockIdx.x, which = blockIdx.y;
    const size_t goff = (size_t)frame * ny * nx;
    const double *raw = (which ? rms_raw : bkg_raw) + goff;
    float *mesh = which ? rms_mesh : bkg_mesh;
    double *coef = (which ? rms_coef : bkg_coef) + goff;
    double *cp = scratch + ((size_t)frame * 2 + which) * ny * nx;

    // median filter -> coef (used as the working array of the prefilter)
    for (int c = threadIdx.x; c < ny * nx; c += K2_NT) {
        int j = c / nx, i = c % nx;
        double win[K2_MAXWIN];
        int n = 0;
        for (int dj = -(fh / 2); dj <= fh / 2; ++dj)
            for (int di = -(fw / 2); di <= fw / 2; ++di) {
                int jj = j + dj, ii = i + di;
                if (jj < 0 || jj >= ny || ii < 0 || ii >= nx) continue;
                double v = raw[jj * nx + ii];
                int k = n++;
                while (k > 0 && win[k - 1] > v) { win[k] = win[k - 1]; --k; }   // insertion sort
                win[k] = v;
            }
        double med = (n & 1) ? win[(n - 1) / 2] : 0.5 * (win[n / 2 - 1] + win[n / 2]);
        coef[c] = med;
        if (mesh) mesh[goff + c] = (float)med;
    }
    __syncthreads();
    for (int i = threadIdx.x; i < nx; i += K2_NT) spline_line(coef + i, cp + i, ny, nx);   // along y
    __syncthreads();
    for (int j = threadIdx.x; j < ny; j += K2_NT) spline_line(coef + (size_t)j * nx, cp + (size_t)j * nx, nx, 1);
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
