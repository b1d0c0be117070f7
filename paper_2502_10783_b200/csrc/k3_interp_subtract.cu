// K3: fused cubic-B-spline evaluation of the background and RMS coefficient grids, subtraction,
// RMS-map emission and threshold-mask generation (step a3).  PAPER.md:80 ("we employ spline
// interpolation to scale the refined background values back"), :61-65 (removal), :153 (threshold scan).
//
// HBM-bound streaming pass: 4 B/px read, up to 13 B/px written.  One thread owns 4 consecutive columns
// and walks down a strip of rows.  For its columns it keeps, in registers, the four x-collapsed spline
// coefficients g_r(x) = sum_di beta3(u - i0 - di) * c[R(j0-1+r)][R(i0+di)], r = 0..3, for both grids; a
// pixel then costs 4 FMAs per map with the row's y-weights (uniform over the CTA, from shared memory).
// The background and the threshold comparison are evaluated in float64 (the float32 ulp at ~1000 ADU is
// comparable to the 1e-5*sigma agreement the catalogue needs); the RMS map in float32.
#include "common.cuh"

namespace {

constexpr int K3_NT = 256;   // threads per CTA
constexpr int K3_PX = 4;     // pixels per thread per row (one float4)
constexpr int K3_R = 4;      // rows whose loads are in flight per thread

__device__ __forceinline__ void bspline_weights(double t, double w[4]) {
    // beta3 at distances 1+t, t, 1-t, 2-t  (t in [0,1))
    double omt = 1.0 - t;
    w[0] = omt * omt * omt / 6.0;
    w[1] = (4.0 - 6.0 * t * t + 3.0 * t * t * t) / 6.0;
    w[2] = (4.0 - 6.0 * omt * omt + 3.0 * omt * omt * omt) / 6.0;
    w[3] = t * t * t / 6.0;
}

__device__ __forceinline__ int reflect_idx(int k, int n) {   // half-sample symmetric: -1->0, n->n-1, period 2n
    int p = 2 * n;
    k %= p;
    if (k < 0) k += p;
    return k < n ? k : p - 1 - k;
}

struct K3Args {
    const float *img;
    const double *bcoef, *rcoef;
    float *sub, *bkg, *rms;
    uint8_t *mask;
    int H, W, mh, mw, ny, nx, rows_per_cta;
    double k_d;
};

__global__ void __launch_bounds__(K3_NT, 2) k3_interp_subtract(K3Args a) {
    extern __shared__ double smem_d[];
    double *wy_tab = smem_d;                                   // [rows_per_cta][4]
    int *j0_tab = (int *)(wy_tab + (size_t)a.rows_per_cta * 4);   // [rows_per_cta]

    const int frame = blockIdx.z;
    const int y_begin = blockIdx.y * a.rows_per_cta;
    const int y_end = min(y_begin + a.rows_per_cta, a.H);
    const int x0 = (blockIdx.x * K3_NT + threadIdx.x) * K3_PX;
    const size_t frame_off = (size_t)frame * a.H * a.W;
    const double *bc = a.bcoef + (size_t)frame * a.ny * a.nx;
    const double *rc = a.rcoef + (size_t)frame * a.ny * a.nx;

    for (int r = threadIdx.x; r < y_end - y_begin; r += K3_NT) {
        double v = ((double)(y_begin + r) + 0.5) / (double)a.mh - 0.5;
        double fl = floor(v);
        double w[4];
        bspline_weights(v - fl, w);
        wy_tab[r * 4 + 0] = w[0]; wy_tab[r * 4 + 1] = w[1]; wy_tab[r * 4 + 2] = w[2]; wy_tab[r * 4 + 3] = w[3];
        j0_tab[r] = (int)fl;
    }
    __syncthreads();
    if (x0 >= a.W) return;

    // x-collapse of one grid row (reflected) for this thread's 4 columns, both grids
    auto collapse = [&](int jrow, double gb_out[K3_PX], float gr_out[K3_PX]) {
        const double *brow = bc + (size_t)reflect_idx(jrow, a.ny) * a.nx;
        const double *rrow = rc + (size_t)reflect_idx(jrow, a.ny) * a.nx;
#pragma unroll
        for (int q = 0; q < K3_PX; ++q) {
            double u = ((double)(x0 + q) + 0.5) / (double)a.mw - 0.5;
            double fl = floor(u);
            int i0 = (int)fl;
            double w[4];
            bspline_weights(u - fl, w);
            double sb = 0.0, sr = 0.0;
#pragma unroll
            for (int d = 0; d < 4; ++d) {
                int ci = reflect_idx(i0 - 1 + d, a.nx);
                sb = fma(w[d], __ldg(brow + ci), sb);
                sr = fma(w[d], __ldg(rrow + ci), sr);
            }
            gb_out[q] = sb;
            gr_out[q] = (float)sr;
        }
    };

    double gb[4][K3_PX];
    float gr[4][K3_PX];
    int cur_j0 = j0_tab[0];
#pragma unroll
    for (int r = 0; r < 4; ++r) collapse(cur_j0 - 1 + r, gb[r], gr[r]);

    const float kdf_guard = 0.0f;
    for (int yb = y_begin; yb < y_end; yb += K3_R) {
        float4 pix[K3_R];
#pragma unroll
        for (int r = 0; r < K3_R; ++r) {
            int y = yb + r;
            if (y < y_end)
                pix[r] = __ldcs(reinterpret_cast<const float4 *>(a.img + frame_off + (size_t)y * a.W + x0));
        }
#pragma unroll
        for (int r = 0; r < K3_R; ++r) {
            int y = yb + r;
            if (y >= y_end) break;
            int j0 = j0_tab[y - y_begin];
            if (j0 != cur_j0) {   // uniform over the CTA: entered a new mesh row, slide the 4-row window
#pragma unroll
                for (int q = 0; q < K3_PX; ++q) {
                    gb[0][q] = gb[1][q]; gb[1][q] = gb[2][q]; gb[2][q] = gb[3][q];
                    gr[0][q] = gr[1][q]; gr[1][q] = gr[2][q]; gr[2][q] = gr[3][q];
                }
                cur_j0 = j0;
                collapse(cur_j0 + 2, gb[3], gr[3]);
            }
            const double4 wy01 = *reinterpret_cast<const double4 *>(wy_tab + (size_t)(y - y_begin) * 4);
            const double wy[4] = {wy01.x, wy01.y, wy01.z, wy01.w};
            const float wyf[4] = {(float)wy01.x, (float)wy01.y, (float)wy01.z, (float)wy01.w};
            const float in[4] = {pix[r].x, pix[r].y, pix[r].z, pix[r].w};
            float o_sub[4], o_bkg[4], o_rms[4];
            uint32_t mbits = 0;
#pragma unroll
            for (int q = 0; q < K3_PX; ++q) {
                double b = wy[0] * gb[0][q];
                b = fma(wy[1], gb[1][q], b);
                b = fma(wy[2], gb[2][q], b);
                b = fma(wy[3], gb[3][q], b);
                float s = wyf[0] * gr[0][q];
                s = fmaf(wyf[1], gr[1][q], s);
                s = fmaf(wyf[2], gr[2][q], s);
                s = fmaf(wyf[3], gr[3][q], s);
                double d = (double)in[q] - b;
                o_sub[q] = (float)d;
                o_bkg[q] = (float)b;
                o_rms[q] = s;
                bool fg = (s > kdf_guard) && (d > a.k_d * (double)s);
                mbits |= (fg ? 1u : 0u) << (8 * q);
            }
            size_t off = frame_off + (size_t)y * a.W + x0;
            __stcs(reinterpret_cast<float4 *>(a.sub + off), make_float4(o_sub[0], o_sub[1], o_sub[2], o_sub[3]));
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
    a.k_d = detect_k;
    // rows per CTA: aim for >= 8 CTAs per SM over the launch so the tail is short, but keep strips long
    // enough (>= 16 rows) that the 16 collapse FMAs/px at the strip start are amortised.
    int col_blocks = (W + K3_NT * K3_PX - 1) / (K3_NT * K3_PX);
    long want_ctas = (long)ctx->num_sms * 16;
    int rows = (int)(((long)H * col_blocks * B + want_ctas - 1) / want_ctas);
    rows = (rows + K3_R - 1) / K3_R * K3_R;
    if (rows < 16) rows = 16;
    if (rows > 128) rows = 128;
    a.rows_per_cta = rows;
    dim3 grid(col_blocks, (H + rows - 1) / rows, B);
    size_t smem = (size_t)rows * 4 * sizeof(double) + (size_t)rows * sizeof(int);
    k3_interp_subtract<<<grid, K3_NT, smem, st>>>(a);
    BD_CUDA_CHECK(ctx, cudaGetLastError());
    return BD_OK;
}
