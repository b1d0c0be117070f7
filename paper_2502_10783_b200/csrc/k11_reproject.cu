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

__global__ void __launch_bounds__(K11_TX *K11_TY) k11_reproject(K11Args a) {
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
    const int xd = (blockIdx.x * K11_TX + threadIdx.x) * 4, yd = blockIdx.y * K11_TY + threadIdx.y;
    if (xd >= a.Wd || yd >= a.Hd) return;
    float4 o = make_float4(a.fill, a.fill, a.fill, a.fill);
    if (s_ok) {
        const float *f = a.src + (size_t)frame * a.Hs * a.Ws;
        const double i0 = s_inv[0], i3 = s_inv[3];
        const double bx = fma(s_inv[1], (double)yd, s_inv[2]), by = fma(s_inv[4], (double)yd, s_inv[5]);
        float r[4];
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            const double x = (double)(xd + q);
            r[q] = k11_sample(f, a.Hs, a.Ws, fma(i0, x, bx), fma(i3, x, by), a.fill);
        }
        o = make_float4(r[0], r[1], r[2], r[3]);
    }
    *reinterpret_cast<float4 *>(a.out + ((size_t)frame * a.Hd + yd) * a.Wd + xd) = o;
}

}  // namespace

int k11_launch(bd_ctx *ctx, const float *d_src, int B, int Hs, int Ws, const double *d_affine, float fill, float *d_out, int Hd,
               int Wd, cudaStream_t st) {
    K11Args a{d_src, d_affine, d_out, Hs, Ws, Hd, Wd, fill};
    const dim3 grid((Wd / 4 + K11_TX - 1) / K11_TX, (Hd + K11_TY - 1) / K11_TY, B);
    k11_reproject<<<grid, dim3(K11_TX, K11_TY), 0, st>>>(a);
    BD_CUDA_CHECK(ctx, cudaGetLastError());
    return BD_OK;
}
