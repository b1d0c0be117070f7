// K6: aperture and auto (Kron-like) photometry per catalogue object.
// PAPER.md:159 ("we calculate the flux of each object using several established methods, such as: aperture photometry,
// isophotal photometry and auto photometry ... Each GPU thread is assigned to measure a single object").
// Isophotal photometry is the `flux` of detect_sources; the paper gives neither formula nor constants for the other two:
// readings A23-A27 (the conventions of the method the paper adapts).
//
// The paper gives an object to one thread; here an object is one WARP: the lanes stride over the pixels of the aperture's
// bounding box (coalesced rows of `sub` and `rms`), float64 partial sums per lane, one xor-shuffle tree -- a fixed order,
// so the results are bit-reproducible.  Every comparison that decides whether a pixel counts (distance against the rim,
// sub-pixel samples, ellipse radius) is evaluated with explicitly rounded float64 products and sums (no FMA contraction):
// the same pixels count as in the float64 definition.
#include "common.cuh"

namespace {

struct K6Args {
    const float *sub, *rms;
    const bd_source *cat;
    const int64_t *n_sources;
    int64_t cap;
    int B, H, W;
    bd_phot_params p;
    bd_phot *out;
};

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
__device__ __forceinline__ int warp_sum_i(int v) {
#pragma unroll
    for (int o = 16; o; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
// x*x + y*y without contraction
__device__ __forceinline__ double sq2(double x, double y) { return __dadd_rn(__dmul_rn(x, x), __dmul_rn(y, y)); }

__global__ void __launch_bounds__(256) k6_photometry(K6Args a) {
    __shared__ long long s_total;
    const int lane = threadIdx.x & 31;
    if (threadIdx.x == 0) {
        long long t = 0;
        for (int f = 0; f < a.B; ++f) t += a.n_sources[f];
        s_total = t < a.cap ? t : a.cap;
    }
    __syncthreads();
    const long long total = s_total;
    const int H = a.H, W = a.W;
    const size_t HW = (size_t)H * W;
    const long long warps = (long long)gridDim.x * (blockDim.x >> 5);
    for (long long i = (long long)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5); i < total; i += warps) {
        const bd_source s = a.cat[i];
        const float *sub = a.sub + (size_t)s.frame * HW, *rms = a.rms + (size_t)s.frame * HW;
        const double xc = s.x, yc = s.y;
        int flags = 0;
        // ---- A23: circular aperture with sub-pixel sampling of the rim ------------------------------------------
        double f_ap = 0.0, a_ap = 0.0, v_ap = 0.0;
        {
            const double r = a.p.r_aper, half = r + 1.0, r_in = r - 0.75, r_out = r + 0.75, rr = __dmul_rn(r, r);
            const int x_lo = (int)floor(xc - half), x_hi = (int)ceil(xc + half);
            const int y_lo = (int)floor(yc - half), y_hi = (int)ceil(yc + half);
            const int bw = x_hi - x_lo + 1, n = bw * (y_hi - y_lo + 1), sp = a.p.subpix;
            int out_w = 0;
            for (int k = lane; k < n; k += 32) {
                const int yy = y_lo + k / bw, xx = x_lo + k % bw;
                const double dx = (double)xx - xc, dy = (double)yy - yc;
                const double d = sqrt(sq2(dx, dy));
                double w = 0.0;
                if (d < r_in) w = 1.0;
                else if (d <= r_out) {
                    int cnt = 0;
                    for (int iy = 0; iy < sp; ++iy) {
                        const double ey = dy + (((double)iy + 0.5) / (double)sp - 0.5);
                        for (int ix = 0; ix < sp; ++ix) {
                            const double ex = dx + (((double)ix + 0.5) / (double)sp - 0.5);
                            cnt += sq2(ex, ey) <= rr ? 1 : 0;
                        }
                    }
                    w = (double)cnt / (double)(sp * sp);
                }
                if (w > 0.0) {
                    if (xx < 0 || xx >= W || yy < 0 || yy >= H) out_w = 1;
                    else {
                        const double I = (double)__ldg(sub + (size_t)yy * W + xx), q = (double)__ldg(rms + (size_t)yy * W + xx);
                        f_ap += w * I; a_ap += w; v_ap += w * (q * q);
                    }
                }
            }
            f_ap = warp_sum(f_ap); a_ap = warp_sum(a_ap); v_ap = warp_sum(v_ap);
            if (__any_sync(0xffffffffu, out_w)) flags |= 1;
        }
        // ---- A24: ellipse metric from the second moments ----------------------------------------------------------
        double x2 = s.x2, y2 = s.y2;
        const double xy = s.xy;
        if (__dsub_rn(__dmul_rn(x2, y2), __dmul_rn(xy, xy)) < 0.00694) { x2 = x2 + 1.0 / 12.0; y2 = y2 + 1.0 / 12.0; }
        const double det = __dsub_rn(__dmul_rn(x2, y2), __dmul_rn(xy, xy));
        const double cxx = y2 / det, cyy = x2 / det, cxy = __dmul_rn(-2.0, xy) / det;
        const double sx2 = sqrt(x2), sy2 = sqrt(y2);
        // sums over the pixels with ellipse radius <= R: S0 = sum I, S1 = sum r I, V = sum rms^2, N = count
        auto ellipse_sums = [&](double R, double &S0, double &S1, double &V, int &N) {
            const double hx = __dmul_rn(R, sx2), hy = __dmul_rn(R, sy2);
            int x_lo = (int)floor(xc - hx), x_hi = (int)ceil(xc + hx), y_lo = (int)floor(yc - hy), y_hi = (int)ceil(yc + hy);
            if (x_lo < 0 || x_hi > W - 1 || y_lo < 0 || y_hi > H - 1) flags |= 2;
            x_lo = max(x_lo, 0); x_hi = min(x_hi, W - 1); y_lo = max(y_lo, 0); y_hi = min(y_hi, H - 1);
            S0 = 0.0; S1 = 0.0; V = 0.0; N = 0;
            if (x_hi < x_lo || y_hi < y_lo) return;
            const int bw = x_hi - x_lo + 1;
            const long long n = (long long)bw * (y_hi - y_lo + 1);
            for (long long k = lane; k < n; k += 32) {
                const int yy = y_lo + (int)(k / bw), xx = x_lo + (int)(k % bw);
                const double dx = (double)xx - xc, dy = (double)yy - yc;
                const double r2 = __dadd_rn(__dadd_rn(__dmul_rn(__dmul_rn(cxx, dx), dx), __dmul_rn(__dmul_rn(cyy, dy), dy)),
                                            __dmul_rn(__dmul_rn(cxy, dx), dy));
                const double rad = sqrt(fmax(r2, 0.0));
                if (rad <= R) {
                    const double I = (double)__ldg(sub + (size_t)yy * W + xx), q = (double)__ldg(rms + (size_t)yy * W + xx);
                    S0 += I; S1 += rad * I; V += q * q; ++N;
                }
            }
            S0 = warp_sum(S0); S1 = warp_sum(S1); V = warp_sum(V); N = warp_sum_i(N);
        };
        // ---- A25: Kron radius ----------------------------------------------------------------------------------------
        double S0, S1, V;
        int N;
        ellipse_sums(a.p.kron_search, S0, S1, V, N);
        double kron = a.p.kron_min_radius;
        if (S0 > 0.0 && S1 > 0.0) kron = fmax(__dmul_rn(a.p.kron_factor, S1) / S0, a.p.kron_min_radius);
        // ---- A26: auto flux --------------------------------------------------------------------------------------------
        ellipse_sums(kron, S0, S1, V, N);
        if (lane == 0) {
            bd_phot o;
            o.flux_aper = f_ap; o.fluxerr_aper = sqrt(v_ap); o.area_aper = a_ap;
            o.kron_radius = kron; o.flux_auto = S0; o.fluxerr_auto = sqrt(V);
            o.npix_auto = N; o.flags = flags;
            a.out[i] = o;
        }
    }
}

}  // namespace

int k6_launch(bd_ctx *ctx, const float *d_sub, const float *d_rms, int B, int H, int W, const bd_source *d_cat,
              const int64_t *d_n_sources, int64_t cat_capacity, const bd_phot_params *p, bd_phot *d_phot, cudaStream_t st) {
    K6Args a;
    a.sub = d_sub; a.rms = d_rms; a.cat = d_cat; a.n_sources = d_n_sources; a.cap = cat_capacity;
    a.B = B; a.H = H; a.W = W; a.p = *p; a.out = d_phot;
    long long blocks = (cat_capacity + 7) / 8;
    const long long max_blocks = (long long)ctx->num_sms * 16;
    if (blocks > max_blocks) blocks = max_blocks;
    if (blocks < 1) blocks = 1;
    k6_photometry<<<(unsigned)blocks, 256, 0, st>>>(a);
    BD_CUDA_CHECK(ctx, cudaGetLastError());
    return BD_OK;
}
