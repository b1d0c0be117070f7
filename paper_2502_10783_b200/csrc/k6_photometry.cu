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

constexpr int K6_LARGE_PX = 4096;     // search boxes larger than this go to the CTA-per-object kernel,
constexpr int K6_HUGE_PX = 1 << 18;   // larger than this to the grid-wide kernels (k6h_*): chunks of the box over all CTAs
constexpr int K6H_CHUNK = 1 << 14;    // pixels of a box one CTA sums at a time (grows when the units would exceed K6H_MAX_UNITS)
constexpr int K6H_MAX_UNITS = 1 << 16;

struct K6Args {
    const float *sub, *rms;
    const bd_source *cat;
    const int64_t *n_sources;
    int64_t cap;
    int B, H, W;
    bd_phot_params p;
    bd_phot *out;
    uint32_t *large_count;   // workspace: [0] number of queued large objects, [1] of huge ones, [2] units, [3] chunk size
    uint32_t *large_list;
    uint32_t *huge_list;     // [cap]
    uint32_t *huge_first;    // [cap + 1] first unit of every huge object (exclusive prefix of its chunk count)
    double *huge_kron;       // [cap] Kron radius after the first pass
    double *huge_part;       // [K6H_MAX_UNITS][4] per-unit partial sums
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
// rad <= R with rad = sqrt(max(r2, 0)) rounded to nearest  <=>  r2 <= r2_limit(R): the largest double whose rounded square
// root does not exceed R (sqrt is monotone, so the limit is R*R up to a couple of ulps, found by stepping).  The per-pixel
// test is then one comparison, with the SAME membership as the definition's; the root is taken for members only.
__device__ __forceinline__ double r2_limit(double R) {
    double t = __dmul_rn(R, R);
    for (int k = 0; k < 4 && sqrt(t) > R; ++k) t = __longlong_as_double(__double_as_longlong(t) - 1);
    for (int k = 0; k < 4; ++k) {
        const double u = __longlong_as_double(__double_as_longlong(t) + 1);
        if (sqrt(u) <= R) t = u; else break;
    }
    return t;
}
// this thread's share (pixels k0 + t, k0 + t + nt, ... < k1 of the box) of  S0 = sum I, S1 = sum r I, V = sum rms^2,
// N = count  over r <= R (T = r2_limit(R)).  NEED_R: S1 is wanted (the first pass).
// (32-bit pixel indices: the box lies inside the frame and H*W < 2^31 is enforced at the boundary)
template <bool NEED_R>
__device__ __forceinline__ void ellipse_partial(const Ellipse &e, const Box &b, double T, const float *sub, const float *rms, int W,
                                                int k0, int k1, int t, int nt, double &S0, double &S1, double &V, int &N) {
    S0 = 0.0; S1 = 0.0; V = 0.0; N = 0;
    const int bw = b.x_hi - b.x_lo + 1;
    for (int k = k0 + t; k < k1; k += nt) {
        const int row = k / bw;
        const int yy = b.y_lo + (int)row, xx = b.x_lo + (int)(k - row * bw);
        const double dx = (double)xx - e.xc, dy = (double)yy - e.yc;
        const double r2 = __dadd_rn(__dadd_rn(__dmul_rn(__dmul_rn(e.cxx, dx), dx), __dmul_rn(__dmul_rn(e.cyy, dy), dy)),
                                    __dmul_rn(__dmul_rn(e.cxy, dx), dy));
        if (r2 <= T) {
            const double I = (double)__ldg(sub + (size_t)yy * W + xx);
            S0 += I; ++N;
            if (NEED_R) S1 += sqrt(fmax(r2, 0.0)) * I;
            else { const double q = (double)__ldg(rms + (size_t)yy * W + xx); V += q * q; }
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
    const double T_search = r2_limit(a.p.kron_search);
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
        // objects with more than K6_LARGE_PX pixels in either box are measured by k6_photometry_large / the k6h_* kernels
        // (which redo both passes); the aperture part is final
        auto defer = [&](long long area) {
            if (lane != 0) return;
            // (at most K6H_MAX_UNITS / 2 huge objects, so that their chunks fit the partial-sum table; the rest, if a frame
            //  ever has that many, are measured by one CTA each like the large ones)
            bool huge = area > K6_HUGE_PX;
            if (huge) {
                const uint32_t k = atomicAdd(a.large_count + 1, 1u);
                if (k < (uint32_t)(K6H_MAX_UNITS / 2)) a.huge_list[k] = (uint32_t)i;
                else huge = false;
            }
            if (!huge) a.large_list[atomicAdd(a.large_count, 1u)] = (uint32_t)i;
        };
        if (ok && box_area(b) > K6_LARGE_PX) {
            defer(box_area(b));
        } else {
            if (ok) {
                ellipse_partial<true>(e, b, T_search, sub, rms, W, 0, (int)box_area(b), lane, 32, S0, S1, V, N);
                S0 = warp_sum(S0); S1 = warp_sum(S1);
            }
            kron = kron_radius_of(a.p, S0, S1);
            S0 = 0.0; V = 0.0; N = 0;
            bool cut2;
            const bool ok2 = ellipse_box(e, kron, H, W, b, cut2);
            if (ok2 && box_area(b) > K6_LARGE_PX) {
                // a faint object whose flux sum inside the search ellipse is nearly zero gets an arbitrarily large Kron radius
                // (A25 has no upper limit): its second box can be the whole frame
                defer(box_area(b));
                kron = a.p.kron_min_radius;
            } else {
                if (cut || cut2) flags |= 2;
                if (ok2) {
                    ellipse_partial<false>(e, b, r2_limit(kron), sub, rms, W, 0, (int)box_area(b), lane, 32, S0, S1, V, N);
                    S0 = warp_sum(S0); V = warp_sum(V); N = warp_sum_i(N);
                }
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
        if (ellipse_box(e, a.p.kron_search, H, W, b, cut))
            ellipse_partial<true>(e, b, r2_limit(a.p.kron_search), sub, rms, W, 0, (int)box_area(b), threadIdx.x, blockDim.x, S0, S1, V, N);
        if (cut) flags |= 2;
        block_sum4(sm, S0, S1, V, N);
        const double kron = kron_radius_of(a.p, S0, S1);
        S0 = 0.0; S1 = 0.0; V = 0.0; N = 0;
        const bool ok2 = ellipse_box(e, kron, H, W, b, cut);
        if (ok2 && box_area(b) > K6_HUGE_PX) {   // second box huge: the grid-wide kernels (launched next) take the object over
            __shared__ uint32_t s_slot;
            if (threadIdx.x == 0) s_slot = atomicAdd(a.large_count + 1, 1u);
            __syncthreads();
            const uint32_t k = s_slot;
            __syncthreads();
            if (k < (uint32_t)(K6H_MAX_UNITS / 2)) {
                if (threadIdx.x == 0) a.huge_list[k] = i;
                continue;
            }
        }
        if (ok2)
            ellipse_partial<false>(e, b, r2_limit(kron), sub, rms, W, 0, (int)box_area(b), threadIdx.x, blockDim.x, S0, S1, V, N);
        if (cut) flags |= 2;
        block_sum4(sm, S0, S1, V, N);
        if (threadIdx.x == 0) {
            bd_phot *o = a.out + i;
            o->kron_radius = kron; o->flux_auto = S0; o->fluxerr_auto = sqrt(V); o->npix_auto = N; o->flags |= flags;
        }
    }
}

// ---- huge objects (search box > K6_HUGE_PX pixels: the saturated stars of a crowded field, whose Kron ellipses cover
// megapixels): the box is cut into chunks of `chunk` consecutive pixels (row-major over the box) that ALL CTAs of the grid
// share; per-chunk partial sums go to the workspace and are combined per object in chunk order, so the result does not
// depend on which CTA summed which chunk.  PASS 0: first-moment radius inside kron_search; PASS 1: sums inside kron_radius.
template <int PASS>
__device__ __forceinline__ bool k6h_box(const K6Args &a, uint32_t j, const Ellipse &e, Box &b, bool &cut) {
    const double R = PASS == 0 ? a.p.kron_search : a.huge_kron[j];
    return ellipse_box(e, R, a.H, a.W, b, cut);
}

template <int PASS>
__global__ void __launch_bounds__(256) k6h_plan(K6Args a) {
    __shared__ unsigned long long s_area;
    const uint32_t n = min(a.large_count[1], (uint32_t)(K6H_MAX_UNITS / 2));
    if (threadIdx.x == 0) s_area = 0ull;
    __syncthreads();
    unsigned long long mine = 0;
    for (uint32_t j = threadIdx.x; j < n; j += blockDim.x) {
        const bd_source s = a.cat[a.huge_list[j]];
        const Ellipse e = make_ellipse(s);
        Box b;
        bool cut;
        const long long area = k6h_box<PASS>(a, j, e, b, cut) ? box_area(b) : 0;
        a.huge_first[j] = (uint32_t)area;   // (H*W < 2^31)
        mine += (unsigned long long)area;
    }
    atomicAdd(&s_area, mine);
    __syncthreads();
    if (threadIdx.x == 0) {
        // units = sum ceil(area / chunk) <= total / chunk + n <= K6H_MAX_UNITS  (n <= K6H_MAX_UNITS / 2 by construction)
        unsigned long long chunk = (s_area + K6H_MAX_UNITS / 2 - 1) / (K6H_MAX_UNITS / 2);
        if (chunk < (unsigned long long)K6H_CHUNK) chunk = K6H_CHUNK;
        uint32_t run = 0;
        for (uint32_t j = 0; j < n; ++j) {
            const uint32_t area = a.huge_first[j];
            a.huge_first[j] = run;
            run += (uint32_t)((area + chunk - 1) / chunk);
        }
        a.huge_first[n] = run;
        a.large_count[2] = run;
        a.large_count[3] = (uint32_t)chunk;
    }
}

template <int PASS>
__global__ void __launch_bounds__(256) k6h_partial(K6Args a) {
    __shared__ double sm[8 * 4];
    const uint32_t n = min(a.large_count[1], (uint32_t)(K6H_MAX_UNITS / 2)), units = a.large_count[2], chunk = a.large_count[3];
    const size_t HW = (size_t)a.H * a.W;
    for (uint32_t u = blockIdx.x; u < units; u += gridDim.x) {
        uint32_t lo = 0, hi = n;            // the object whose unit range holds u
        while (hi - lo > 1) { const uint32_t mid = (lo + hi) >> 1; if (a.huge_first[mid] <= u) lo = mid; else hi = mid; }
        const uint32_t j = lo, c = u - a.huge_first[j];
        const bd_source s = a.cat[a.huge_list[j]];
        const Ellipse e = make_ellipse(s);
        Box b;
        bool cut;
        double S0 = 0.0, S1 = 0.0, V = 0.0;
        int N = 0;
        if (k6h_box<PASS>(a, j, e, b, cut)) {
            const long long area = box_area(b);
            const long long k0 = (long long)c * chunk, k1 = k0 + chunk < area ? k0 + chunk : area;
            const float *sub = a.sub + (size_t)s.frame * HW, *rms = a.rms + (size_t)s.frame * HW;
            const double T = r2_limit(PASS == 0 ? a.p.kron_search : a.huge_kron[j]);
            ellipse_partial<PASS == 0>(e, b, T, sub, rms, a.W, (int)k0, (int)k1, threadIdx.x, blockDim.x, S0, S1, V, N);
        }
        block_sum4(sm, S0, S1, V, N);
        if (threadIdx.x == 0) {
            double *p = a.huge_part + (size_t)u * 4;
            p[0] = S0; p[1] = S1; p[2] = V; p[3] = (double)N;
        }
        __syncthreads();
    }
}

template <int PASS>
__global__ void __launch_bounds__(256) k6h_combine(K6Args a) {
    const uint32_t n = min(a.large_count[1], (uint32_t)(K6H_MAX_UNITS / 2));
    for (uint32_t j = blockIdx.x * blockDim.x + threadIdx.x; j < n; j += gridDim.x * blockDim.x) {
        const uint32_t i = a.huge_list[j];
        double S0 = 0.0, S1 = 0.0, V = 0.0, N = 0.0;
        for (uint32_t u = a.huge_first[j]; u < a.huge_first[j + 1]; ++u) {
            const double *p = a.huge_part + (size_t)u * 4;
            S0 += p[0]; S1 += p[1]; V += p[2]; N += p[3];
        }
        const bd_source s = a.cat[i];
        const Ellipse e = make_ellipse(s);
        Box b;
        bool cut;
        k6h_box<PASS>(a, j, e, b, cut);
        bd_phot *o = a.out + i;
        if (cut) o->flags |= 2;
        if (PASS == 0) {
            a.huge_kron[j] = kron_radius_of(a.p, S0, S1);
        } else {
            o->kron_radius = a.huge_kron[j]; o->flux_auto = S0; o->fluxerr_auto = sqrt(V); o->npix_auto = (int)N;
        }
    }
}

}  // namespace

size_t k6_workspace_bytes(int64_t cat_capacity) {
    const size_t cap = (size_t)(cat_capacity > 0 ? cat_capacity : 1);
    // counters, large list, huge list, huge first-unit prefix, huge Kron radii, per-unit partial sums
    return 256 + bd_align_up(cap * 4, 256) * 2 + bd_align_up((cap + 1) * 4, 256) + bd_align_up(cap * 8, 256) + (size_t)K6H_MAX_UNITS * 4 * sizeof(double);
}

int k6_launch(bd_ctx *ctx, const float *d_sub, const float *d_rms, int B, int H, int W, const bd_source *d_cat,
              const int64_t *d_n_sources, int64_t cat_capacity, const bd_phot_params *p, bd_phot *d_phot, void *d_ws,
              size_t ws_bytes, cudaStream_t st) {
    if (ws_bytes < k6_workspace_bytes(cat_capacity))
        return bd_set_error(ctx, BD_EWORKSPACE, "photometry workspace: need %zu bytes, got %zu", k6_workspace_bytes(cat_capacity), ws_bytes);
    K6Args a;
    a.sub = d_sub; a.rms = d_rms; a.cat = d_cat; a.n_sources = d_n_sources; a.cap = cat_capacity;
    a.B = B; a.H = H; a.W = W; a.p = *p; a.out = d_phot;
    const size_t cap = (size_t)(cat_capacity > 0 ? cat_capacity : 1);
    char *w = (char *)d_ws;
    a.large_count = (uint32_t *)w; w += 256;
    a.large_list = (uint32_t *)w; w += bd_align_up(cap * 4, 256);
    a.huge_list = (uint32_t *)w; w += bd_align_up(cap * 4, 256);
    a.huge_first = (uint32_t *)w; w += bd_align_up((cap + 1) * 4, 256);
    a.huge_kron = (double *)w; w += bd_align_up(cap * 8, 256);
    a.huge_part = (double *)w;
    BD_CUDA_CHECK(ctx, cudaMemsetAsync(a.large_count, 0, 4 * sizeof(uint32_t), st));
    long long blocks = (cat_capacity + 7) / 8;
    const long long max_blocks = (long long)ctx->num_sms * 16;
    if (blocks > max_blocks) blocks = max_blocks;
    if (blocks < 1) blocks = 1;
    k6_photometry<<<(unsigned)blocks, 256, 0, st>>>(a);
    k6_photometry_large<<<ctx->num_sms * 4, 256, 0, st>>>(a);
    k6h_plan<0><<<1, 256, 0, st>>>(a);
    k6h_partial<0><<<ctx->num_sms * 8, 256, 0, st>>>(a);
    k6h_combine<0><<<8, 256, 0, st>>>(a);
    k6h_plan<1><<<1, 256, 0, st>>>(a);
    k6h_partial<1><<<ctx->num_sms * 8, 256, 0, st>>>(a);
    k6h_combine<1><<<8, 256, 0, st>>>(a);
    BD_CUDA_CHECK(ctx, cudaGetLastError());
    return BD_OK;
}
