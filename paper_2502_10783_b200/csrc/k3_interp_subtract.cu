// K3: fused cubic-B-spline evaluation of the background and RMS coefficient grids, subtraction,
// RMS-map emission and threshold-mask generation (step a3).  PAPER.md:80 ("we employ spline
// interpolation to scale the refined background values back"), :61-65 (removal), :153 (threshold scan).
//
// HBM-bound streaming pass: 4 B/px read, up to 13 B/px written.  A CTA owns a strip of 1024 columns x
// `rows` rows; one thread owns 4 consecutive columns (one float4) and walks down the strip with K3_R row
// loads in flight.
//
// Arithmetic.  With h_d(y) = sum_r beta3(v - j0 - r) c[R(j0+r)][R(i0+d)] (the y-collapsed coefficients of the
// four grid columns i0-1..i0+2 that a pixel of grid cell i0 sees) the spline value is sum_d wx_d h_d, and
// because the cubic B-spline weights are a partition of unity (sum_d wx_d = 1 exactly),
//     bkg = h_0 + sum_{d != 0} wx_d (h_d - h_0).
// The CTA first builds, in float64, a shared-memory table with one entry per (row, i0): h_0 split into a
// float32 hi/lo pair, the three differences h_d - h_0 (a few ADU: float32 carries them to ~1e-6 ADU) and
// the four y-collapsed RMS coefficients.  A pixel then costs 3 + 4 float32 FMAs with the x-weights its
// thread keeps in registers, and sub = (img - hi) - (lo + sum) -- the first difference is exact for sky
// pixels (Sterbenz), so the result agrees with the float64 definition to ~1e-6 ADU although no float64
// instruction runs per pixel.  (The float32 ulp at ~1000 ADU, 6e-5, would not be good enough for the
// 1e-5*sigma mask agreement if bkg itself were accumulated in float32.)
#include "common.cuh"
#include "spline_eval.cuh"

namespace {

constexpr int K3_NT = 256;   // threads per CTA
constexpr int K3_PX = 4;     // pixels per thread per row (one float4)
#ifndef K3_ROWS_IN_FLIGHT
#define K3_ROWS_IN_FLIGHT 8
#endif
#ifndef K3_MIN_CTAS
#define K3_MIN_CTAS 2
#endif
#ifndef K3_STRIP_ROWS
#define K3_STRIP_ROWS 32
#endif
constexpr int K3_R = K3_ROWS_IN_FLIGHT;   // rows whose loads are in flight per thread
constexpr int K3_ENT = SPL_ENT;   // floats per table entry (48 B: three 128-bit shared loads)
constexpr int K3_TABLE_BYTES = 40 * 1024;

struct K3Args {
    const float *img;
    const double *bcoef, *rcoef;
    float *sub, *bkg, *rms;
    uint8_t *mask;
    int H, W, mh, mw, ny, nx, rows_per_cta, n_i0_max;
    float k_d;
};

// UNIFORM: mesh_w % 8 == 0, so the cell boundary (between columns mw*k + mw/2 - 1 and mw*k + mw/2) falls on a
// multiple of 4 and the four columns of a thread lie in the same grid cell i0.
template <bool UNIFORM>
__global__ void __launch_bounds__(K3_NT, K3_MIN_CTAS) k3_interp_subtract(K3Args a) {
    extern __shared__ __align__(16) float table[];   // [rows][n_i0][K3_ENT]

    const int frame = blockIdx.z;
    const int y_begin = blockIdx.y * a.rows_per_cta;
    const int y_end = min(y_begin + a.rows_per_cta, a.H);
    const int xc0 = blockIdx.x * K3_NT * K3_PX;
    const int xc1 = min(xc0 + K3_NT * K3_PX, a.W) - 1;
    const int x0 = xc0 + threadIdx.x * K3_PX;
    const size_t frame_off = (size_t)frame * a.H * a.W;
    const double *bc = a.bcoef + (size_t)frame * a.ny * a.nx;
    const double *rc = a.rcoef + (size_t)frame * a.ny * a.nx;
    const int i0_first = spl_cell_of(xc0, a.mw);
    const int n_i0 = spl_cell_of(xc1, a.mw) - i0_first + 1;

    // ---- table: one entry per (row, i0) --------------------------------------------------------------
    const int n_ent = (y_end - y_begin) * n_i0;
    for (int e = threadIdx.x; e < n_ent; e += K3_NT) {
        const int r = e / n_i0, ii = e - r * n_i0;
        spl_table_entry(bc, rc, a.ny, a.nx, a.mh, y_begin + r, i0_first + ii, table + (size_t)e * K3_ENT);
    }
    __syncthreads();
    if (x0 >= a.W) return;

    // ---- per-thread x weights (float64 -> float32) and table column ------------------------------------
    float wx[K3_PX][4];
    int ent_off[K3_PX];
#pragma unroll
    for (int q = 0; q < K3_PX; ++q) {
        const int i0 = spl_cell_of(x0 + q, a.mw);
        spl_x_weights(x0 + q, a.mw, i0, wx[q]);
        ent_off[q] = (i0 - i0_first) * K3_ENT;
    }
    const int row_stride = n_i0 * K3_ENT;

    const float *img = a.img + frame_off + x0;
    for (int yb = y_begin; yb < y_end; yb += K3_R) {
        float4 pix[K3_R];
#pragma unroll
        for (int r = 0; r < K3_R; ++r)
            if (yb + r < y_end) pix[r] = __ldcs(reinterpret_cast<const float4 *>(img + (size_t)(yb + r) * a.W));
#pragma unroll
        for (int r = 0; r < K3_R; ++r) {
            const int y = yb + r;
            if (y >= y_end) break;
            const float *trow = table + (size_t)(y - y_begin) * row_stride;
            const float in[4] = {pix[r].x, pix[r].y, pix[r].z, pix[r].w};
            float o_sub[4], o_bkg[4], o_rms[4];
            uint32_t mbits = 0;
            float4 t0, t1;
            float t8;
            if (UNIFORM) {
                const float *t = trow + ent_off[0];
                t0 = *reinterpret_cast<const float4 *>(t);
                t1 = *reinterpret_cast<const float4 *>(t + 4);
                t8 = t[8];
            }
#pragma unroll
            for (int q = 0; q < K3_PX; ++q) {
                if (!UNIFORM) {
                    const float *t = trow + ent_off[q];
                    t0 = *reinterpret_cast<const float4 *>(t);
                    t1 = *reinterpret_cast<const float4 *>(t + 4);
                    t8 = t[8];
                }
                const bool fg = spl_pixel(t0, t1, t8, wx[q], in[q], a.k_d, o_sub[q], o_bkg[q], o_rms[q]);
                mbits |= (fg ? 1u : 0u) << (8 * q);
            }
            const size_t off = frame_off + (size_t)y * a.W + x0;
            if (a.sub) __stcs(reinterpret_cast<float4 *>(a.sub + off), make_float4(o_sub[0], o_sub[1], o_sub[2], o_sub[3]));
            if (a.bkg) __stcs(reinterpret_cast<float4 *>(a.bkg + off), make_float4(o_bkg[0], o_bkg[1], o_bkg[2], o_bkg[3]));
            if (a.rms) __stcs(reinterpret_cast<float4 *>(a.rms + off), make_float4(o_rms[0], o_rms[1], o_rms[2], o_rms[3]));
            if (a.mask) __stcs(reinterpret_cast<uint32_t *>(a.mask + off), mbits);
        }
    }
}

}  // namespace

int k3_launch(bd_ctx *ctx, const float *d_img, int B, int H, int W, int mh, int mw, const double *d_bkg_coef,
              const double *d_rms_coef, double detect_k, float *d_sub, float *d_bkg, float *d_rms, uint8_t *d_mask,
              cudaStream_t st) {
    K3Args a;
    a.img = d_img; a.bcoef = d_bkg_coef; a.rcoef = d_rms_coef;
    a.sub = d_sub; a.bkg = d_bkg; a.rms = d_rms; a.mask = d_mask;
    a.H = H; a.W = W; a.mh = mh; a.mw = mw;
    a.ny = (H + mh - 1) / mh; a.nx = (W + mw - 1) / mw;
    a.k_d = (float)detect_k;
    const int cols = K3_NT * K3_PX;
    const int col_blocks = (W + cols - 1) / cols;
    // grid cells a 1024-column strip can touch; the table (rows x cells x 48 B) bounds the strip height
    a.n_i0_max = (cols < W ? cols : W) / mw + 2;
    int rows = K3_TABLE_BYTES / (a.n_i0_max * K3_ENT * (int)sizeof(float));
    if (rows > K3_STRIP_ROWS) rows = K3_STRIP_ROWS;
    if (rows >= K3_R) rows = rows / K3_R * K3_R;
    if (rows < 1) return bd_set_error(ctx, BD_EUNSUPPORTED, "mesh width %d too small for the interpolation kernel", mw);
    if (rows > H) rows = H;
    a.rows_per_cta = rows;
    dim3 grid(col_blocks, (H + rows - 1) / rows, B);
    size_t smem = (size_t)rows * a.n_i0_max * K3_ENT * sizeof(float);
    if (mw % 8 == 0) k3_interp_subtract<true><<<grid, K3_NT, smem, st>>>(a);
    else k3_interp_subtract<false><<<grid, K3_NT, smem, st>>>(a);
    BD_CUDA_CHECK(ctx, cudaGetLastError());
    return BD_OK;
}
