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

constexpr int K6_LARGE_PX = 4096;   // search boxes larger than this go to the CTA-per-object kernel

struct K6Args {
    const float *sub, *rms;
    const bd_source *cat;
    const int64_t *n_sources;
    int64_t cap;
    int B, H, W;
    bd_phot_params p;
    bd_phot *out;
    uint32_t *large_count;   // workspace: number of queued large objects, then their indices
    uint32_t *large_list;
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

// A24: ellipse metric of an object (1/12 added to the moments of degenerate objects)
struct Ellipse { double xc, yc, cxx, cyy, cxy, sx2, sy2; bool ok; };
__device__ __forceinline__ Ellipse make_ellipse(const bd_source &s) {
    Ellipse e;
    double x2 = s.x2, y2 = s.y2;
    const double xy = s.xy;
    if (__dsub_rn(__dmul_rn(x2, y2), __dmul_rn(xy, xy)) < 0.00694) { x2 = x2 + 1.0 / 12.0; y2 = y2 + 1.0 / 12.0; }
    const double det = __dsub_rn(__dmul_rn(x2, y2), __dmul_rn(xy, xy));
    e.xc = s.x; e.yc = s.y;
    // A28: a record with a non-finite centroid or moments, or moments that define no ellipse, is not measured
    e.ok = isfinite(s.x) && isfinite(s.y) && isfinite(x2) && isfinite(y2) && isfinite(xy) && det > 0.0 && x2 > 0.0 && y2 > 0.0;
    e.cxx = y2 / det; e.cyy = x2 / det; e.cxy = __dmul_rn(-2.0, xy) / det;
    e.sx2 = sqrt(x2); e.sy2 = sqrt(y2);
    return e;
}
// bounding box of the ellipse of radius R, clipped to the frame; returns false if it is empty; `cut` = it was clipped
struct Box { int x_lo, x_hi, y_lo, y_hi; };
__device__ __forceinline__ bool ellipse_box(const Ellipse &e, double R, int H, int W, Box &b, bool &cut) {
    const double hx = __dmul_rn(R, e.sx2), hy = __dmul_rn(R, e.sy2);
    b.x_lo = (int)floor(e.xc - hx); b.x_hi = (int)ceil(e.xc + hx); b.y_lo = (int)floor(e.yc - hy); b.y_hi = (int)ceil(e.yc + hy);
    cut = b.x_lo < 0 || b.x_hi > W - 1 || b.y_lo < 0 || b.y_hi > H - 1;
    b.x_lo = max(b.x_lo, 0); b.x_hi = min(b.x_hi, W - 1); b.y_lo = max(b.y_lo, 0); b.y_hi = min(b.y_hi, H - 1);
    return b.x_hi >= b.x_lo && b.y_hi >= b.y_lo;
}
__device__ __forceinline__ long long box_area(const Box &b) { return (long long)(b.x_hi - b.x_lo + 1) * (b.y_hi - b.y_lo + 1); }
// this thread's share (pixels t, t + nt, ... of the box) of  S0 = sum I, S1 = sum r I, V = sum rms^2, N = count  over r <= R
// (32-bit pixel indices: the box lies inside the frame and H*W < 2^31 is enforced at the boundary)
__device__ __forceinline__ void ellipse_partial(const Ellipse &e, const Box &b, double R, const float *sub, const float *rms, int W,
                                                int t, int nt, double &S0, double &S1, double &V, int &N) {
    S0 = 0.0; S1 = 0.0; V = 0.0; N = 0;
    const int bw = b.x_hi - b.x_lo + 1;
    const int n = (int)box_area(b);
    for (int k = t; k < n; k += nt) {
        const int row = k / bw;
        const int yy = b.y_lo + (int)row, xx = b.x_lo + (int)(k - row * bw);
        const double dx = (double)xx - e.xc, dy = (double)yy - e.yc;
        const double r2 = __dadd_rn(__dadd_rn(__dmul_rn(__dmul_rn(e.cxx, dx), dx), __dmul_rn(__dmul_rn(e.cyy, dy), dy)),
                                    __dmul_rn(__dmul_rn(e.cxy, dx), dy));
        const double rad = sqrt(fmax(r2, 0.0));
        if (rad <= R) {
            const double I = (double)__ldg(sub + (size_t)yy * W + xx), q = (double)__ldg(rms + (size_t)yy * W + xx);
            S0 += I; S1 += rad * I; V += q * q; ++N;
        }
    }
}
__device__ __forceinline__ double kron_radius_of(const bd_phot_params &p, double S0, double S1) {   // A25
    if (S0 > 0.0 && S1 > 0.0) return fmax(__dmul_rn(p.kron_factor, S1) / S0, p.kron_min_radius);
    return p.kron_min_radius;
}

__device__ __forceinline__ long long k6_total(const K6Args &a, long long *s_total) {
    if (threadIdx.x == 0) {
        long long t = 0;
        for (int f = 0; f < a.B; ++f) t += a.n_sources[f];
        *s_total = t < a.cap ? t : a.cap;
    }
    __syncthreads();
    return *s_total;
}

// one warp per object: aperture photometry of every object, auto photometry of the objects with a small search box
__global__ void __launch_bounds__(256) k6_photometry(K6Args a) {
    __shared__ long long s_total;
    const int lane = threadIdx.x & 31;
    const long long total = k6_total(a, &s_total);
    const int H = a.H, W = a.W;
    const size_t HW = (size_t)H * W;
    const long long warps = (long long)gridDim.x * (blockDim.x >> 5);
    for (long long i = (long long)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5); i < total; i += warps) {
        const bd_source s = a.cat[i];
        const float *sub = a.sub + (size_t)s.frame * HW, *rms = a.rms + (size_t)s.frame * HW;
        const double xc = s.x, yc = s.y;
        int flags = 0;
        const Ellipse e = make_ellipse(s);
        if (!e.ok) {   // A28: degenerate record
            if (lane == 0) {
                bd_phot o;
                o.flux_aper = 0.0; o.fluxerr_aper = 0.0; o.area_aper = 0.0; o.kron_radius = 0.0; o.flux_auto = 0.0; o.fluxerr_auto = 0.0;
                o.npix_auto = 0; o.flags = 4;
                a.out[i] = o;
            }
            continue;
        }
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
        // ---- A24-A26: ellipse, Kron radius, auto flux ------------------------------------------------------------------
        Box b;
        bool cut;
        double S0 = 0.0, S1 = 0.0, V = 0.0, kron = a.p.kron_min_radius;
        int N = 0;
        bool ok = ellipse_box(e, a.p.kron_search, H, W, b, cut);
        const bool large = ok && box_area(b) > K6_LARGE_PX;
        if (large) {   // measured by k6_photometry_large; the aperture part is final
            if (lane == 0) a.large_list[atomicAdd(a.large_count, 1u)] = (uint32_t)i;
        } else {
            if (cut) flags |= 2;
            if (ok) {
                ellipse_partial(e, b, a.p.kron_search, sub, rms, W, lane, 32, S0, S1, V, N);
                S0 = warp_sum(S0); S1 = warp_sum(S1);
            }
            kron = kron_radius_of(a.p, S0, S1);
            S0 = 0.0; V = 0.0; N = 0;
            ok = ellipse_box(e, kron, H, W, b, cut);
            if (cut) flags |= 2;
            if (ok) {
                ellipse_partial(e, b, kron, sub, rms, W, lane, 32, S0, S1, V, N);
                S0 = warp_sum(S0); V = warp_sum(V); N = warp_sum_i(N);
            }
        }
        if (lane == 0) {
            bd_phot o;
            o.flux_aper = f_ap; o.fluxerr_aper = sqrt(v_ap); o.area_aper = a_ap;
            o.kron_radius = kron; o.flux_auto = S0; o.fluxerr_auto = sqrt(V);
            o.npix_auto = N; o.flags = flags;
            a.out[i] = o;
        }
    }
}

// one CTA per queued large object: the same sums, threads striding over the box, per-warp partials combined in warp order
__device__ __forceinline__ void block_sum4(double *sm, double &S0, double &S1, double &V, int &N) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = blockDim.x >> 5;
    S0 = warp_sum(S0); S1 = warp_sum(S1); V = warp_sum(V); N = warp_sum_i(N);
    __syncthreads();
    if (lane == 0) { sm[warp * 4 + 0] = S0; sm[warp * 4 + 1] = S1; sm[warp * 4 + 2] = V; sm[warp * 4 + 3] = (double)N; }
    __syncthreads();
    S0 = 0.0; S1 = 0.0; V = 0.0;
    double n = 0.0;
    for (int w = 0; w < nw; ++w) { S0 += sm[w * 4 + 0]; S1 += sm[w * 4 + 1]; V += sm[w * 4 + 2]; n += sm[w * 4 + 3]; }
    N = (int)n;
}
__global__ void __launch_bounds__(256) k6_photometry_large(K6Args a) {
    __shared__ double sm[8 * 4];
    const int H = a.H, W = a.W;
    const size_t HW = (size_t)H * W;
    const uint32_t n_large = *a.large_count;
    for (uint32_t j = blockIdx.x; j < n_large; j += gridDim.x) {
        const uint32_t i = a.large_list[j];
        const bd_source s = a.cat[i];
        const float *sub = a.sub + (size_t)s.frame * HW, *rms = a.rms + (size_t)s.frame * HW;
        const Ellipse e = make_ellipse(s);
        Box b;
        bool cut;
        int flags = 0, N = 0;
        double S0 = 0.0, S1 = 0.0, V = 0.0;
        if (ellipse_box(e, a.p.kron_search, H, W, b, cut)) ellipse_partial(e, b, a.p.kron_search, sub, rms, W, threadIdx.x, blockDim.x, S0, S1, V, N);
        if (cut) flags |= 2;
        block_sum4(sm, S0, S1, V, N);
        const double kron = kron_radius_of(a.p, S0, S1);
        S0 = 0.0; S1 = 0.0; V = 0.0; N = 0;
        if (ellipse_box(e, kron, H, W, b, cut)) ellipse_partial(e, b, kron, sub, rms, W, threadIdx.x, blockDim.x, S0, S1, V, N);
        if (cut) flags |= 2;
        block_sum4(sm, S0, S1, V, N);
        if (threadIdx.x == 0) {
            bd_phot *o = a.out + i;
            o->kron_radius = kron; o->flux_auto = S0; o->fluxerr_auto = sqrt(V); o->npix_auto = N; o->flags |= flags;
        }
    }
}

}  // namespace

size_t k6_workspace_bytes(int64_t cat_capacity) { return 256 + (size_t)(cat_capacity > 0 ? cat_capacity : 1) * sizeof(uint32_t); }

int k6_launch(bd_ctx *ctx, const float *d_sub, const float *d_rms, int B, int H, int W, const bd_source *d_cat,
              const int64_t *d_n_sources, int64_t cat_capacity, const bd_phot_params *p, bd_phot *d_phot, void *d_ws,
              size_t ws_bytes, cudaStream_t st) {
    if (ws_bytes < k6_workspace_bytes(cat_capacity))
        return bd_set_error(ctx, BD_EWORKSPACE, "photometry workspace: need %zu bytes, got %zu", k6_workspace_bytes(cat_capacity), ws_bytes);
    K6Args a;
    a.sub = d_sub; a.rms = d_rms; a.cat = d_cat; a.n_sources = d_n_sources; a.cap = cat_capacity;
    a.B = B; a.H = H; a.W = W; a.p = *p; a.out = d_phot;
    a.large_count = (uint32_t *)d_ws;
    a.large_list = (uint32_t *)((char *)d_ws + 256);
    BD_CUDA_CHECK(ctx, cudaMemsetAsync(a.large_count, 0, sizeof(uint32_t), st));
    long long blocks = (cat_capacity + 7) / 8;
    const long long max_blocks = (long long)ctx->num_sms * 16;
    if (blocks > max_blocks) blocks = max_blocks;
    if (blocks < 1) blocks = 1;
    k6_photometry<<<(unsigned)blocks, 256, 0, st>>>(a);
    k6_photometry_large<<<ctx->num_sms * 4, 256, 0, st>>>(a);
    BD_CUDA_CHECK(ctx, cudaGetLastError());
    return BD_OK;
}
