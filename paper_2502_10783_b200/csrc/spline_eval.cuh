// Cubic-B-spline evaluation shared by K3 (k3_interp_subtract) and the fused tile kernel of k45_detect.cu, so that
// both produce bit-identical bkg / rms / sub / mask values.  PAPER.md:80 (spline interpolation back to full
// resolution), :61-65 (removal), :153 (threshold); readings A14, A15.
//
// With h_d(y) = sum_r beta3(v - j0 - r) c[R(j0+r)][R(i0+d)] (the y-collapsed coefficients of the four grid columns
// i0-1..i0+2 that a pixel of grid cell i0 sees) the spline value is sum_d wx_d h_d, and because the weights are a
// partition of unity,  bkg = h_0' + sum_{d != 1} wx_d (h_d - h_1)  with h_1 split into a float32 hi/lo pair.
// One table entry per (row, i0), built in float64: {hi, lo, e_-1, e_+1, e_+2, r_-1, r_0, r_+1, r_+2} (12 floats,
// 48 B); a pixel then costs 3 + 4 float32 FMAs and  sub = (img - hi) - (lo + sum)  -- the first difference is exact
// for sky pixels (Sterbenz), so sub agrees with the float64 definition to ~1e-6 ADU.
#pragma once
#include <stdint.h>

constexpr int SPL_ENT = 12;   // floats per table entry

__device__ __forceinline__ void bspline_weights(double t, double w[4]) {
    // beta3 at distances 1+t, t, 1-t, 2-t  (t in [0,1)); multiplications by 1/6 instead of divisions (a float64
    // division is ~40 instructions, and the fused tile kernel evaluates these weights 5 times per thread per tile)
    const double s = 1.0 / 6.0, omt = 1.0 - t;
    w[0] = omt * omt * omt * s;
    w[1] = (4.0 - 6.0 * t * t + 3.0 * t * t * t) * s;
    w[2] = (4.0 - 6.0 * omt * omt + 3.0 * omt * omt * omt) * s;
    w[3] = t * t * t * s;
}

__device__ __forceinline__ int reflect_idx(int k, int n) {   // half-sample symmetric: -1->0, n->n-1, period 2n
    if (k >= 0 && k < n) return k;   // the common case, without the integer modulo (~30 instructions)
    int p = 2 * n;
    k %= p;
    if (k < 0) k += p;
    return k < n ? k : p - 1 - k;
}

// floor((x + 0.5)/m - 0.5) with exact integer arithmetic: floor((2x + 1 - m) / (2 m))
__device__ __forceinline__ int spl_cell_of(int x, int m) {
    int num = 2 * x + 1 - m, den = 2 * m;
    return num >= 0 ? num / den : -((-num + den - 1) / den);
}

// table entry of an image row (cell j0, y-weights wy) and grid cell i0
__device__ __forceinline__ void spl_table_entry_w(const double *bc, const double *rc, int ny, int nx, int j0, const double wy[4],
                                                  int i0, float *t) {
    double hb[4] = {0, 0, 0, 0}, hr[4] = {0, 0, 0, 0};
#pragma unroll
    for (int rr = 0; rr < 4; ++rr) {
        const size_t row = (size_t)reflect_idx(j0 - 1 + rr, ny) * nx;
#pragma unroll
        for (int d = 0; d < 4; ++d) {
            const int ci = reflect_idx(i0 - 1 + d, nx);
            hb[d] = fma(wy[rr], __ldg(bc + row + ci), hb[d]);
            hr[d] = fma(wy[rr], __ldg(rc + row + ci), hr[d]);
        }
    }
    const float hi = (float)hb[1];
    t[0] = hi;
    t[1] = (float)(hb[1] - (double)hi);
    t[2] = (float)(hb[0] - hb[1]);
    t[3] = (float)(hb[2] - hb[1]);
    t[4] = (float)(hb[3] - hb[1]);
    t[5] = (float)hr[0]; t[6] = (float)hr[1]; t[7] = (float)hr[2]; t[8] = (float)hr[3];
}
// y-weights of image row y (cell j0 = spl_cell_of(y, mh))
__device__ __forceinline__ void spl_y_weights(int y, int mh, int j0, double wy[4]) {
    bspline_weights(((double)y + 0.5) * (1.0 / (double)mh) - 0.5 - (double)j0, wy);
}
__device__ __forceinline__ void spl_table_entry(const double *bc, const double *rc, int ny, int nx, int mh, int y, int i0,
                                                float *t) {
    const int j0 = spl_cell_of(y, mh);
    double wy[4];
    spl_y_weights(y, mh, j0, wy);
    spl_table_entry_w(bc, rc, ny, nx, j0, wy, i0, t);
}

// float32 x-weights of image column x (cell i0 = spl_cell_of(x, mw))
__device__ __forceinline__ void spl_x_weights(int x, int mw, int i0, float wx[4]) {
    double w[4];
    bspline_weights(((double)x + 0.5) * (1.0 / (double)mw) - 0.5 - (double)i0, w);
    wx[0] = (float)w[0]; wx[1] = (float)w[1]; wx[2] = (float)w[2]; wx[3] = (float)w[3];
}

// The threshold rule of the library (A15), in ONE place: float32 product, float32 compare, on the float32 sub / rms values the
// interface materialises.  K3, the fused tile kernel and the mask-less path of detect_sources (k_make_mask) all call it,
// so the three routes give the same mask bit for bit whatever detect_k is (k_d = (float)detect_k).
__device__ __forceinline__ bool spl_above(float sub, float rms, float k_d) { return (rms > 0.0f) && (sub > __fmul_rn(k_d, rms)); }

// one pixel: t0 = {hi, lo, e_-1, e_+1}, t1 = {e_+2, r_-1, r_0, r_+1}, t8 = r_+2
__device__ __forceinline__ bool spl_pixel(const float4 &t0, const float4 &t1, float t8, const float wx[4], float in, float k_d,
                                          float &o_sub, float &o_bkg, float &o_rms) {
    float rel = wx[0] * t0.z;
    rel = fmaf(wx[2], t0.w, rel);
    rel = fmaf(wx[3], t1.x, rel);
    rel += t0.y;
    float s = wx[0] * t1.y;
    s = fmaf(wx[1], t1.z, s);
    s = fmaf(wx[2], t1.w, s);
    s = fmaf(wx[3], t8, s);
    const float d = (in - t0.x) - rel;
    o_sub = d;
    o_bkg = t0.x + rel;
    o_rms = s;
    return spl_above(d, s, k_d);
}
