// K11: bilinear reprojection of a frame through an affine matrix (second half).
// PAPER.md:114 ("we use the affine matrix to obtain the coordinate mapping between the source image and the resulting image.
// For each pixel in the source image, the pixel value in the resulting image is calculated through bilinear interpolation
// based on the four neighboring pixels").  The FIT of the matrix is out of scope: the matrix is an input.  Readings R1-R6
// (DESIGN.md): A is the forward map source -> result; the result PULLS: result(x', y') = bilinear sample of the source at
// A^-1 (x', y'); a neighbour outside the source is `fill`; a matrix without an inverse gives a frame of `fill`.
//
// A gather with unit-stride output: 4 B/px read (every source pixel is needed once; its re-use by the 4 result pixels around
// it is served by L1 / L2) + 4 B/px written = 8 B/px, HBM-bound.  One thread per 4 consecutive result pixels of a row (one
// 16-byte store), thread blocks of 16 x 16 threads = tiles of 64 x 16 result pixels, so that a block's footprint in the
// source is a compact (rotated) patch.  The inverse matrix is formed once per block in float64; source coordinates are float64
// FMAs (float32 has 1e-3 px of rounding at x = 9000), the fractional parts and the blend are float32.
#include "common.cuh"

namespace {

constexpr int K11_TX = 16, K11_TY = 16;   // threads per block; 4 pixels per thread along x

struct K11Args {
    const float *src;
    const double *affine;   // [B][6]
    float *out;
    int Hs, Ws, Hd, Wd;
    float fill;
};

__device__ __forceinline__ float k11_sample(const float *__restrict__ f, int Hs, int Ws, double xs, double ys, float fill) {
    // all four neighbours outside (or coordinates not finite): exactly fill
    if (!(xs > -1.0 && xs < (double)Ws && ys > -1.0 && ys < (double)Hs)) return fill;
    const int x0 = __double2int_rd(xs), y0 = __double2int_rd(ys);
    const float fx = (float)(xs - (double)x0), fy = (float)(ys - (double)y0);
    float v00, v01, v10, v11;
    if (x0 >= 0 && x0 + 1 < Ws && y0 >= 0 && y0 + 1 < Hs) {
        const float *p = f + (size_t)y0 * Ws + x0;
        v00 = __ldg(p); v01 = __ldg(p + 1); v10 = __ldg(p + Ws); v11 = __ldg(p + Ws + 1);
    } else {
        const bool xa = x0 >= 0, xb = x0 + 1 < Ws, ya = y0 >= 0, yb = y0 + 1 < Hs;
        v00 = (xa && ya) ? __ldg(f + (size_t)y0 * Ws + x0) : fill;
        v01 = (xb && ya) ? __ldg(f + (size_t)y0 * Ws + x0 + 1) : fill;
        v10 = (xa && yb) ? __ldg(f + (size_t)(y0 + 1) * Ws + x0) : fill;
        v11 = (xb && yb) ? __ldg(f + (size_t)(y0 + 1) * Ws + x0 + 1) : fill;
    }
    const float top = fmaf(fx, v01 - v00, v00), bot = fmaf(fx, v11 - v10, v10);
    return fmaf(fy, bot - top, top);
}

// Persistent blocks: block b of a frame takes tiles b, b + gridDim.x, ... (row-major over the result), so the float64
// inversion of the matrix (a chain of divisions one thread performs while the block waits) is paid once per block.
__global__ void __launch_bounds__(K11_TX *K11_TY, 4) k11_reproject(K11Args a, int tiles_x, int tiles) {
    __shared__ double s_inv[6];
    __shared__ int s_ok;
    const int frame = blockIdx.z;
    if (threadIdx.x == 0 && threadIdx.y == 0) {
        const double *A = a.affine + (size_t)frame * 6;
        const double a0 = A[0], a1 = A[1], a2 = A[2], a3 = A[3], a4 = A[4], a5 = A[5];
        const double det = a0 * a4 - a1 * a3;
        const bool ok = isfinite(det) && det != 0.0 && isfinite(a2) && isfinite(a5);   // R5
        if (ok) {
            const double i0 = a4 / det, i1 = -a1 / det, i3 = -a3 / det, i4 = a0 / det;
            s_inv[0] = i0; s_inv[1] = i1; s_inv[2] = -(i0 * a2 + i1 * a5);
            s_inv[3] = i3; s_inv[4] = i4; s_inv[5] = -(i3 * a2 + i4 * a5);
        }
        s_ok = ok ? 1 : 0;
    }
    __syncthreads();
    const bool ok = s_ok != 0;
    const double i0 = s_inv[0], i1 = s_inv[1], i2 = s_inv[2], i3 = s_inv[3], i4 = s_inv[4], i5 = s_inv[5];
    const float *f = a.src + (size_t)frame * a.Hs * a.Ws;
    const int Hs = a.Hs, Ws = a.Ws;
    const float dxf = (float)(i0 - 1.0), dyf = (float)i3;   // step of the fractions from one result pixel to the next along x
    int ty = blockIdx.x / tiles_x, tx = blockIdx.x - ty * tiles_x;
    for (int t = blockIdx.x; t < tiles; t += gridDim.x, tx += gridDim.x) {
        while (tx >= tiles_x) { tx -= tiles_x; ++ty; }
        const int xd = (tx * K11_TX + threadIdx.x) * 4, yd = ty * K11_TY + threadIdx.y;
        if (xd >= a.Wd || yd >= a.Hd) continue;
        float4 o = make_float4(a.fill, a.fill, a.fill, a.fill);
        if (ok) {
            const double bx = fma(i1, (double)yd, i2), by = fma(i4, (double)yd, i5);
            // float64 only for the first of the four pixels; the other three step by (i0 - 1, i3) in float32 from its fractions.
            // While all eight fractions stay inside [0, 1] the four pixels read source columns x0 .. x0 + 4 of rows y0, y0 + 1
            // (the usual case of an alignment: rotation of a fraction of a degree, scale within 1e-3 of 1).  A fraction that
            // float32 puts at 1 where float64 says 0 of the next pixel gives the same value (the interpolant is continuous);
            // the float32 steps add <= 1.2e-7 px to the 6e-8 px of the rounded fraction itself.
            const double xs0 = fma(i0, (double)xd, bx), ys0 = fma(i3, (double)xd, by);
            const int x0 = __double2int_rd(xs0), y0 = __double2int_rd(ys0);   // saturating; NaN -> 0 with NaN fractions
            const float fx0 = (float)(xs0 - (double)x0), fy0 = (float)(ys0 - (double)y0);
            float fx[4], fy[4];
#pragma unroll
            for (int q = 0; q < 4; ++q) { fx[q] = fmaf((float)q, dxf, fx0); fy[q] = fmaf((float)q, dyf, fy0); }
            // (the fractions are linear in q: inside [0, 1] at both ends means inside for all four; NaN fails the comparisons)
            const bool fast = x0 >= 0 && x0 <= Ws - 5 && y0 >= 0 && y0 <= Hs - 2 && fx0 >= 0.0f && fy0 >= 0.0f &&
                              fx[3] >= 0.0f && fx[3] <= 1.0f && fy[3] >= 0.0f && fy[3] <= 1.0f;
            // (A variant that kept quads straddling two source rows on this path by loading a third row was measured and was
            //  slower: 0.231 against 0.216 ms on the 9216 x 9232 frame -- profiles/r3_k11_reproject.md.)
            float r[4];
            if (fast) {
                // two aligned 16-byte loads per row cover columns x0 .. x0 + 4 whatever x0 mod 4 is
                const int base = x0 & ~3, off = x0 & 3;
                const float4 *p0 = reinterpret_cast<const float4 *>(f + (size_t)y0 * Ws + base);
                const float4 *p1 = reinterpret_cast<const float4 *>(f + (size_t)(y0 + 1) * Ws + base);
                const float4 u0 = __ldg(p0), u1 = __ldg(p0 + 1), w0 = __ldg(p1), w1 = __ldg(p1 + 1);
                // element off + j of the 8 loaded pixels, j = 0..4: shift by (off & 1), then by (off & 2)
                const bool s1 = off & 1, s2 = off & 2;
                const float ur[8] = {u0.x, u0.y, u0.z, u0.w, u1.x, u1.y, u1.z, u1.w}, wr[8] = {w0.x, w0.y, w0.z, w0.w, w1.x, w1.y, w1.z, w1.w};
                float ua[7], wa[7], tp[5], bt[5];
#pragma unroll
                for (int j = 0; j < 7; ++j) { ua[j] = s1 ? ur[j + 1] : ur[j]; wa[j] = s1 ? wr[j + 1] : wr[j]; }
#pragma unroll
                for (int j = 0; j < 5; ++j) { tp[j] = s2 ? ua[j + 2] : ua[j]; bt[j] = s2 ? wa[j + 2] : wa[j]; }
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    const float top = fmaf(fx[q], tp[q + 1] - tp[q], tp[q]), bot = fmaf(fx[q], bt[q + 1] - bt[q], bt[q]);
                    r[q] = fmaf(fy[q], bot - top, top);
                }
            } else {
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    const double x = (double)(xd + q);
                    r[q] = k11_sample(f, Hs, Ws, fma(i0, x, bx), fma(i3, x, by), a.fill);
                }
            }
            o = make_float4(r[0], r[1], r[2], r[3]);
        }
        *reinterpret_cast<float4 *>(a.out + ((size_t)frame * a.Hd + yd) * a.Wd + xd) = o;
    }
}

}  // namespace

int k11_launch(bd_ctx *ctx, const float *d_src, int B, int Hs, int Ws, const double *d_affine, float fill, float *d_out, int Hd,
               int Wd, cudaStream_t st) {
    K11Args a{d_src, d_affine, d_out, Hs, Ws, Hd, Wd, fill};
    const int tiles_x = (Wd / 4 + K11_TX - 1) / K11_TX, tiles_y = (Hd + K11_TY - 1) / K11_TY;
    const long long tiles = (long long)tiles_x * tiles_y;   // < 2^31 / 1024 (check_frame)
    const long long per_frame = (4ll * ctx->num_sms + B - 1) / B;   // the 4 resident blocks per SM of the launch bounds, over the whole batch
    const dim3 grid((unsigned)(tiles < per_frame ? tiles : per_frame), 1, B);
    k11_reproject<<<grid, dim3(K11_TX, K11_TY), 0, st>>>(a, tiles_x, (int)tiles);
    BD_CUDA_CHECK(ctx, cudaGetLastError());
    return BD_OK;
}
