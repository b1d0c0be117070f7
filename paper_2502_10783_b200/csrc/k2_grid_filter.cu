// K2: median filter of the background and RMS mesh grids, then cubic-B-spline prefilter (step a2).
// PAPER.md:80 ("we apply a median filter to the estimated background values ... Following the smoothing
// process, we employ spline interpolation").  Grid-sized work (<= a few thousand cells per frame), float64
// throughout: K2a = one warp per cell (window median), K2b = one CTA per (frame, grid) (prefilter).  Readings A11 (both grids), A13 (window truncated at the
// border), A14 (order 3, half-sample-symmetric ends: c[-1]=c[0], c[n]=c[n-1]).
#include "common.cuh"

namespace {

constexpr int K2_NT = 256;          // threads per CTA, both kernels
constexpr int K2_MAXWIN = 121;      // 11 x 11, the largest window check_params admits

// ---- K2a: window medians, one WARP per (frame, grid, cell) ------------------------------------------------
// Rank counting: rank of element a = #(v < v_a) + #(v == v_a with smaller window index); the ranks are a
// permutation of 0..n-1, so exactly one lane holds rank (n-1)/2 and one holds rank n/2 (A13: even count ->
// mean of the two middle values).  The window sits in shared memory; lane l owns elements l, l+32, ...
// (The first version ran the whole grid in one CTA with every thread counting ranks for its own cells:
// 316 us for the 2 x 1332 cells of config 3.)
__global__ void __launch_bounds__(K2_NT) k2a_window_median(const double *bkg_raw, const double *rms_raw, int B, int ny,
                                                           int nx, int fh, int fw, float *bkg_mesh, float *rms_mesh,
                                                           double *bkg_work, double *rms_work) {
    __shared__ double win[K2_NT / 32][K2_MAXWIN + 7];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int cells = ny * nx;
    const long long item = (long long)blockIdx.x * (K2_NT / 32) + warp;   // (frame, which, cell)
    if (item >= 2ll * B * cells) return;
    const int c = (int)(item % cells);
    const int which = (int)((item / cells) & 1);
    const int frame = (int)(item / (2ll * cells));
    const size_t goff = (size_t)frame * cells;
    const double *g = (which ? rms_raw : bkg_raw) + goff;
    const int j = c / nx, i = c - j * nx;
    const int j0 = max(0, j - fh / 2), j1 = min(ny - 1, j + fh / 2);
    const int i0 = max(0, i - fw / 2), i1 = min(nx - 1, i + fw / 2);
    const int ww = i1 - i0 + 1, n = (j1 - j0 + 1) * ww;
    double *w = win[warp];
    bd_pdl_wait();      // launched programmatically dependent on K1: the raw grids are read from here on
    bd_pdl_trigger();
    for (int a = lane; a < n; a += 32) w[a] = __ldg(g + (size_t)(j0 + a / ww) * nx + i0 + a % ww);
    __syncwarp();
    const int k_lo = (n - 1) / 2, k_hi = n / 2;
    double lo = 0.0, hi = 0.0;
    for (int a = lane; a < n; a += 32) {
        const double va = w[a];
        int rank = 0;
        for (int b = 0; b < n; ++b) {
            const double vb = w[b];
            rank += (vb < va || (vb == va && b < a)) ? 1 : 0;
        }
        if (rank == k_lo) lo = va;
        if (rank == k_hi) hi = va;
    }
    // exactly one lane holds each of lo, hi (the others hold 0.0): an exact "sum"
#pragma unroll
    for (int o = 16; o; o >>= 1) {
        lo += __shfl_xor_sync(0xffffffffu, lo, o);
        hi += __shfl_xor_sync(0xffffffffu, hi, o);
    }
    if (lane == 0) {
        const double med = (n & 1) ? lo : 0.5 * (lo + hi);
        (which ? rms_work : bkg_work)[goff + c] = med;
        float *mesh = which ? rms_mesh : bkg_mesh;
        if (mesh) mesh[goff + c] = (float)med;
    }
}

// Windows of at most 9 cells (the 3 x 3 filter of configs 1, 2, 4, 5): one THREAD per (frame, grid, cell), the window in
// registers, the same rank rule.  (A warp per cell is 131 072 warps for the 64 frames of config 4: 53 us.)
__global__ void __launch_bounds__(K2_NT) k2a_window_median_small(const double *bkg_raw, const double *rms_raw, int B, int ny,
                                                                 int nx, int fh, int fw, float *bkg_mesh, float *rms_mesh,
                                                                 double *bkg_work, double *rms_work) {
    const int cells = ny * nx;
    const long long item = (long long)blockIdx.x * K2_NT + threadIdx.x;   // (frame, which, cell)
    if (item >= 2ll * B * cells) return;
    const int c = (int)(item % cells);
    const int which = (int)((item / cells) & 1);
    const int frame = (int)(item / (2ll * cells));
    const size_t goff = (size_t)frame * cells;
    const int j = c / nx, i = c - j * nx;
    const int j0 = max(0, j - fh / 2), j1 = min(ny - 1, j + fh / 2);
    const int i0 = max(0, i - fw / 2), i1 = min(nx - 1, i + fw / 2);
    const int ww = i1 - i0 + 1, n = (j1 - j0 + 1) * ww;
    bd_pdl_wait();
    bd_pdl_trigger();
    const double *g = (which ? rms_raw : bkg_raw) + goff;
    double w[9];
#pragma unroll
    for (int a = 0; a < 9; ++a) w[a] = a < n ? __ldg(g + (size_t)(j0 + a / ww) * nx + i0 + a % ww) : 0.0;
    const int k_lo = (n - 1) / 2, k_hi = n / 2;
    double lo = 0.0, hi = 0.0;
#pragma unroll
    for (int a = 0; a < 9; ++a) {
        int rank = 0;
#pragma unroll
        for (int b = 0; b < 9; ++b) rank += (b < n && (w[b] < w[a] || (w[b] == w[a] && b < a))) ? 1 : 0;
        if (a < n && rank == k_lo) lo = w[a];
        if (a < n && rank == k_hi) hi = w[a];
    }
    const double med = (n & 1) ? lo : 0.5 * (lo + hi);
    (which ? rms_work : bkg_work)[goff + c] = med;
    float *mesh = which ? rms_mesh : bkg_mesh;
    if (mesh) mesh[goff + c] = (float)med;
}

// ---- K2f: invalid cells (NaN: background variants, reading B3) take the median of the VALID cells of the smallest square
// window (2r+1)^2, r = 1, 2, ..., truncated at the grid border, that holds one; both grids, read from the unfilled grids.
// One thread per cell.  The window of radius r - 1 held no valid cell, so the valid cells of the window of radius r all lie
// on its outer RING (Chebyshev distance exactly r, 8r cells before truncation): only the ring is scanned, and the rank
// counting (as in K2a) runs over the ring's valid cells.  A grid that is mostly or wholly invalid therefore costs
// O(max(ny, nx)^2) loads per cell, not the O(max(ny, nx)^3) + O(window^2) of rescanning whole windows.
// Ring cell t in [0, 8r): top row, bottom row (2r + 1 cells each), then the left and right columns without their corners.
__device__ __forceinline__ bool k2f_ring_cell(int t, int r, int j, int i, int ny, int nx, int *jj, int *ii) {
    const int w = 2 * r + 1;
    int dj, di;
    if (t < 2 * w) { dj = t < w ? -r : r; di = (t < w ? t : t - w) - r; }
    else { const int u = t - 2 * w, h = w - 2; di = u < h ? -r : r; dj = (u < h ? u : u - h) - r + 1; }
    *jj = j + dj; *ii = i + di;
    return *jj >= 0 && *jj < ny && *ii >= 0 && *ii < nx;
}
// median of g over the valid (gv not NaN) cells of the ring, n > 0 of them; ties: any order gives the same value
__device__ double k2f_ring_median(const double *g, const double *gv, int ny, int nx, int j, int i, int r, int n) {
    const int k_lo = (n - 1) / 2, k_hi = n / 2;
    double lo = 0.0, hi = 0.0;
    for (int a = 0; a < 8 * r; ++a) {
        int ja, ia;
        if (!k2f_ring_cell(a, r, j, i, ny, nx, &ja, &ia) || isnan(gv[(size_t)ja * nx + ia])) continue;
        const double va = g[(size_t)ja * nx + ia];
        int rank = 0;
        for (int b = 0; b < 8 * r; ++b) {
            int jb, ib;
            if (!k2f_ring_cell(b, r, j, i, ny, nx, &jb, &ib) || isnan(gv[(size_t)jb * nx + ib])) continue;
            const double vb = g[(size_t)jb * nx + ib];
            rank += (vb < va || (vb == va && b < a)) ? 1 : 0;
        }
        if (rank == k_lo) lo = va;
        if (rank == k_hi) hi = va;
    }
    return (n & 1) ? lo : 0.5 * (lo + hi);
}
// grid = (ceil(cells / K2_NT), B): a block's cells belong to one frame.  A block that holds an invalid cell first scans its
// frame's grid for ANY valid cell (cells / K2_NT loads per thread, from L2): a frame without one is written as 0 straight
// away instead of every cell walking all its rings to the far corner.
__global__ void __launch_bounds__(K2_NT) k2f_fill_invalid(const double *bkg_raw, const double *rms_raw, int B, int ny, int nx,
                                                          double *bkg_out, double *rms_out, uint8_t *valid) {
    const int cells = ny * nx;
    const int c = blockIdx.x * K2_NT + threadIdx.x;
    const size_t goff = (size_t)blockIdx.y * cells;
    const double *gb = bkg_raw + goff, *gr = rms_raw + goff;
    const bool mine = c < cells;
    const double vb = mine ? gb[c] : 0.0;
    const bool inv = mine && isnan(vb);
    if (mine && !inv) {
        bkg_out[goff + c] = vb; rms_out[goff + c] = gr[c];
        if (valid) valid[goff + c] = 1;
    }
    if (!__syncthreads_or(inv ? 1 : 0)) return;
    int any = 0;
    for (int k = threadIdx.x; k < cells; k += K2_NT) any |= isnan(gb[k]) ? 0 : 1;
    any = __syncthreads_or(any);
    if (!inv) return;
    if (valid) valid[goff + c] = 0;
    const int j = c / nx, i = c - j * nx;
    double fb = 0.0, fr = 0.0;
    const int rmax = any ? max(max(j, ny - 1 - j), max(i, nx - 1 - i)) : 0;   // the ring of this radius reaches the farthest corner
    for (int r = 1; r <= rmax; ++r) {
        int n = 0;
        for (int t = 0; t < 8 * r; ++t) {
            int jj, ii;
            if (k2f_ring_cell(t, r, j, i, ny, nx, &jj, &ii)) n += isnan(gb[(size_t)jj * nx + ii]) ? 0 : 1;
        }
        if (n > 0) {
            fb = k2f_ring_median(gb, gb, ny, nx, j, i, r, n);
            fr = k2f_ring_median(gr, gb, ny, nx, j, i, r, n);
            break;
        }
    }
    bkg_out[goff + c] = fb; rms_out[goff + c] = fr;
}

// ---- K2b: cubic-B-spline prefilter ------------------------------------------------------------------------
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

// One CTA per (frame, grid), in place on the coefficient array (which K2a filled with the filtered grid).
// The grid is staged in (dynamic) shared memory when it fits (up to K2_SMEM_DOUBLES cells incl. the row padding: 144 x 144;
// padded rows so that the x sweep, where thread j walks row j, is free of bank conflicts); otherwise the same code runs on
// global memory (126 us instead of ~15 for the 96 x 96 grid of config 5, which the first, 4096-cell limit sent there).
constexpr int K2_SMEM_DOUBLES = 20736 + 144;
constexpr int K2_SMEM_LINE = 160;   // longest line whose Thomas factors sit in shared memory

__host__ __device__ inline bool k2b_in_smem(int ny, int nx) { return ny * (nx | 1) <= K2_SMEM_DOUBLES && ny <= K2_SMEM_LINE && nx <= K2_SMEM_LINE; }

__global__ void __launch_bounds__(K2_NT) k2b_spline_prefilter(int ny, int nx, double *bkg_coef, double *rms_coef,
                                                              double *scratch) {
    extern __shared__ double s_work[];
    __shared__ double s_cp[2][K2_SMEM_LINE], s_im[2][K2_SMEM_LINE];
    const int frame = blockIdx.x, which = blockIdx.y;
    const size_t goff = (size_t)frame * ny * nx;
    double *coef = (which ? rms_coef : bkg_coef) + goff;
    const int cells = ny * nx;
    const int pitch = nx | 1;   // odd pitch
    const bool in_smem = k2b_in_smem(ny, nx);
    double *fac = scratch + ((size_t)frame * 2 + which) * k2_scratch_per_grid(ny, nx);   // global factors otherwise
    double *cp_y = in_smem ? s_cp[0] : fac, *im_y = in_smem ? s_im[0] : fac + ny;
    double *cp_x = in_smem ? s_cp[1] : fac + 2 * ny, *im_x = in_smem ? s_im[1] : fac + 2 * ny + nx;
    if (threadIdx.x == K2_NT - 32) spline_factors(cp_y, im_y, ny);   // (depend on the grid shape only: computed while K2a drains)
    if (threadIdx.x == K2_NT - 64) spline_factors(cp_x, im_x, nx);
    bd_pdl_wait();
    double *work = coef;
    int wp = nx;
    if (in_smem) {
        for (int c = threadIdx.x; c < cells; c += K2_NT) s_work[(c / nx) * pitch + c % nx] = coef[c];
        work = s_work;
        wp = pitch;
    }
    __syncthreads();
    for (int i = threadIdx.x; i < nx; i += K2_NT) spline_line(work + i, cp_y, im_y, ny, wp);   // along y
    __syncthreads();
    for (int j = threadIdx.x; j < ny; j += K2_NT) spline_line(work + (size_t)j * wp, cp_x, im_x, nx, 1);
    if (in_smem) {
        __syncthreads();
        for (int c = threadIdx.x; c < cells; c += K2_NT) coef[c] = s_work[(c / nx) * pitch + c % nx];
    }
}

}  // namespace

int k2f_launch(bd_ctx *ctx, const double *d_bkg_raw, const double *d_rms_raw, int B, int ny, int nx, double *d_bkg_filled,
               double *d_rms_filled, uint8_t *d_valid, cudaStream_t st) {
    const dim3 grid((unsigned)((ny * nx + K2_NT - 1) / K2_NT), (unsigned)B);   // B <= 65535 (check_frame)
    k2f_fill_invalid<<<grid, K2_NT, 0, st>>>(d_bkg_raw, d_rms_raw, B, ny, nx, d_bkg_filled, d_rms_filled, d_valid);
    BD_CUDA_CHECK(ctx, cudaGetLastError());
    return BD_OK;
}

int k2_launch(bd_ctx *ctx, const double *d_bkg_raw, const double *d_rms_raw, int B, int ny, int nx, int fh, int fw,
              float *d_bkg_mesh, float *d_rms_mesh, double *d_bkg_coef, double *d_rms_coef, double *d_scratch,
              cudaStream_t st) {
    const long long items = 2ll * B * ny * nx;
    const unsigned nblk = (unsigned)((items + K2_NT / 32 - 1) / (K2_NT / 32));
    if (fh * fw <= 9)
        BD_CUDA_CHECK(ctx, bd_launch_pdl(k2a_window_median_small, dim3((unsigned)((items + K2_NT - 1) / K2_NT)), dim3(K2_NT), 0, st, d_bkg_raw,
                                         d_rms_raw, B, ny, nx, fh, fw, d_bkg_mesh, d_rms_mesh, d_bkg_coef, d_rms_coef));
    else
        BD_CUDA_CHECK(ctx, bd_launch_pdl(k2a_window_median, dim3(nblk), dim3(K2_NT), 0, st, d_bkg_raw, d_rms_raw, B, ny, nx, fh, fw, d_bkg_mesh,
                                         d_rms_mesh, d_bkg_coef, d_rms_coef));
    dim3 grid(B, 2);
    const size_t smem_b = k2b_in_smem(ny, nx) ? (size_t)ny * (nx | 1) * sizeof(double) : 0;
    BD_CUDA_CHECK(ctx, cudaFuncSetAttribute(k2b_spline_prefilter, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(K2_SMEM_DOUBLES * sizeof(double))));
    BD_CUDA_CHECK(ctx, bd_launch_pdl(k2b_spline_prefilter, grid, dim3(K2_NT), smem_b, st, ny, nx, d_bkg_coef, d_rms_coef, d_scratch));
    BD_CUDA_CHECK(ctx, cudaGetLastError());
    return BD_OK;
}

// ---- bd_grid_filter_spline_static: step a2 for callers that may not allocate device memory --------------------------
// bd_grid_filter_spline takes its Thomas-factor scratch from a workspace the caller cudaMalloc'ed.  Some callers have no
// allocator to ask: a plug-in running inside a host application that handed it a fixed set of device buffers and forbids
// further allocation, a real-time acquisition loop that must not enter the driver's allocator (it can block for
// milliseconds and synchronise the device), or code running after the application has committed all of its memory.  For
// them the same two kernels run with the scratch in the array below, which is part of the library's image: the driver
// reserves it on every GPU that loads libbkgdet, when the module is loaded, and releases it at process exit.
//
// The array name is only a handle on the host; the device address comes from cudaGetSymbolAddress, asked once per device
// with that device current (the entry point binds ctx's device first) and kept in k2_static_addr[].
constexpr size_t K2_STATIC_DOUBLES = BD_GRID_STATIC_MAX_DOUBLES;   // bkgdet.h: 32768 doubles = 256 KiB
constexpr int K2_STATIC_MAX_DEVICES = 64;
static __device__ __align__(256) double k2_static_scratch[K2_STATIC_DOUBLES];

#include <mutex>
static std::mutex k2_static_mutex;
static double *k2_static_addr[K2_STATIC_MAX_DEVICES];   // device address of k2_static_scratch on device i, or null: not asked yet

// Device address of the array on ctx's device (which must be current).  The first call per device asks the runtime.
static int k2_static_scratch_ptr(bd_ctx *ctx, double **out) {
    if (ctx->device < 0 || ctx->device >= K2_STATIC_MAX_DEVICES)
        return bd_set_error(ctx, BD_EUNSUPPORTED, "bd_grid_filter_spline_static: device ordinal %d is beyond the %d the table holds",
                            ctx->device, K2_STATIC_MAX_DEVICES);
    std::lock_guard<std::mutex> lock(k2_static_mutex);
    if (!k2_static_addr[ctx->device]) {
        double *p = nullptr;
        BD_CUDA_CHECK(ctx, cudaGetSymbolAddress((void **)&p, k2_static_scratch));
        if (!p) return bd_set_error(ctx, BD_ECUDA, "cudaGetSymbolAddress returned a null address for the static scratch array");
        k2_static_addr[ctx->device] = p;
    }
    *out = k2_static_addr[ctx->device];
    return BD_OK;
}

extern "C" int bd_grid_filter_spline_static(bd_ctx *ctx, const double *d_bkg_raw, const double *d_rms_raw, int B, int ny, int nx,
                                            int filt_h, int filt_w, float *d_bkg_mesh, float *d_rms_mesh, double *d_bkg_coef,
                                            double *d_rms_coef, void *cuda_stream) {
    if (!ctx) return BD_EINVAL;
    if (!d_bkg_raw || !d_rms_raw || !d_bkg_coef || !d_rms_coef) return bd_set_error(ctx, BD_EINVAL, "null pointer");
    if (B <= 0 || ny <= 0 || nx <= 0 || B > 65535) return bd_set_error(ctx, BD_EINVAL, "bad grid shape");
    if (filt_h < 1 || filt_w < 1 || !(filt_h & 1) || !(filt_w & 1) || filt_h > 11 || filt_w > 11)
        return bd_set_error(ctx, BD_EINVAL, "filter size must be odd and in 1..11");
    const size_t need = 2 * (size_t)B * k2_scratch_per_grid(ny, nx);   // doubles; the same count bd_grid_filter_spline asks for
    if (need > K2_STATIC_DOUBLES)
        return bd_set_error(ctx, BD_EWORKSPACE,
                            "bd_grid_filter_spline_static: B=%d grids of %d x %d cells need 4*B*(ny+nx) = %zu doubles of scratch, the "
                            "built-in array holds %zu (%zu bytes); split the batch or use bd_grid_filter_spline with a workspace",
                            B, ny, nx, need, K2_STATIC_DOUBLES, K2_STATIC_DOUBLES * sizeof(double));
    BD_BIND_DEVICE(ctx);
    double *scratch = nullptr;
    const int rc = k2_static_scratch_ptr(ctx, &scratch);
    if (rc) return rc;
    // Nothing in the array has to start at zero: every (frame, grid) block of the prefilter writes its own factors
    // before it reads them, so whatever the previous call left behind is simply overwritten.
    return k2_launch(ctx, d_bkg_raw, d_rms_raw, B, ny, nx, filt_h, filt_w, d_bkg_mesh, d_rms_mesh, d_bkg_coef, d_rms_coef, scratch,
                     (cudaStream_t)cuda_stream);
}
