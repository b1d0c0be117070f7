// K10: cleaning of the (deblended) catalogue (second half).
// PAPER.md:157 ("determine if the current object can be merged with any adjacent objects based on predefined criteria.
// If the analysis indicates that merging is appropriate, the current object is flagged as a false detection ... a
// parallel operation to remove the marked pixels").  The paper gives no criteria: readings D9-D12.
//
// The definition compares every object with every other one.  Here the influence of an object j is bounded: the zone
// test r_j^2 <= clean_zone^2 rho_j^2 confines the objects it can suppress to the bounding box of an ellipse about its
// centroid.  The objects are binned by centroid into 32-pixel cells (count, scan, scatter); one warp per object j walks
// the cell rows its box covers (the cells of a row are contiguous in the scattered list) and evaluates the pair test of
// D11 for the objects i found there, in float64 and in the operation order of the definition (explicitly rounded
// products and sums where a comparison without a fragile band depends on them).  Every decision is taken on the input
// catalogue, so the pairs are independent; a flag is a plain store.  The survivors are ranked with the bitmap scan of
// kept_rank.cuh over the record index (catalogue order is kept) and the pixels of the false detections are erased from
// the label map, one warp per flagged record over its bounding box.
#include "common.cuh"

namespace {

typedef unsigned long long u64;

#include "kept_rank.cuh"

constexpr int CELL = 32;

struct CRec {   // per catalogue record, 96 bytes
    double x, y, x2, y2, xy, D;      // centroid, shape (D9)
    double A, alpha, zone2, t;       // profile (D10), squared zone radius in r^2 units, threshold
    double flux, mean;               // flux, flux / npix
};

struct CWs {
    uint32_t *counters;      // [64]
    uint32_t *keptbits;      // one bit per record
    uint32_t *blkcnt, *blkprefix;
    uint32_t *cellcnt, *cellprefix, *cellcur;
    int32_t *cellitems;      // [cap]
    CRec *crec;              // [cap]
    uint8_t *flag;           // [cap]
    size_t ncell, NBk, zero_bytes, total;
    int ncx, ncy;
};

size_t carve(CWs &w, void *base, int B, int H, int W, int64_t cap) {
    w.ncx = (W + CELL - 1) / CELL;
    w.ncy = (H + CELL - 1) / CELL;
    w.ncell = (size_t)B * w.ncx * w.ncy;
    w.NBk = ((size_t)cap + 4095) / 4096;
    size_t off = 0;
    auto take = [&](size_t bytes) { size_t o = off; off = bd_align_up(off + bytes, 256); return (char *)base + o; };
    w.counters = (uint32_t *)take(64 * sizeof(uint32_t));
    w.keptbits = (uint32_t *)take((((size_t)cap + 31) / 32 + 32) * sizeof(uint32_t));
    w.blkcnt = (uint32_t *)take((w.NBk + 8) * sizeof(uint32_t));
    w.cellcnt = (uint32_t *)take((w.ncell + 8) * sizeof(uint32_t));
    w.cellcur = (uint32_t *)take((w.ncell + 8) * sizeof(uint32_t));
    w.flag = (uint8_t *)take((size_t)cap);
    w.zero_bytes = (size_t)((char *)w.flag - (char *)w.counters) + (size_t)cap;
    w.blkprefix = (uint32_t *)take((w.NBk + 8) * sizeof(uint32_t));
    w.cellprefix = (uint32_t *)take((w.ncell + 8) * sizeof(uint32_t));
    w.cellitems = (int32_t *)take((size_t)cap * sizeof(int32_t));
    w.crec = (CRec *)take((size_t)cap * sizeof(CRec));
    w.total = off;
    return off;
}

struct CArgs {
    const float *rms;
    int32_t *labels;
    const bd_source *cat;
    const int64_t *n_in;
    int64_t cap_in, cap_out;
    int B, H, W;
    float kf;
    double beta, zone;
    CWs w;
};

__device__ __forceinline__ long long c_total(const CArgs &a) {
    long long t = 0;
    for (int f = 0; f < a.B; ++f) t += a.n_in[f];
    return t < a.cap_in ? t : a.cap_in;
}

__device__ __forceinline__ size_t cell_of(const CArgs &a, int frame, double x, double y) {
    int cx = (int)floor(x / CELL), cy = (int)floor(y / CELL);
    cx = min(max(cx, 0), a.w.ncx - 1);
    cy = min(max(cy, 0), a.w.ncy - 1);
    return ((size_t)frame * a.w.ncy + cy) * a.w.ncx + cx;
}

// D9, D10: shape and profile of every record; bin count by centroid
__global__ void __launch_bounds__(256) k10_prepare(CArgs a) {
    const long long total = c_total(a);
    const size_t HW = (size_t)a.H * a.W;
    const double PI = 3.141592653589793;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (long long)gridDim.x * blockDim.x) {
        const bd_source s = a.cat[i];
        CRec c;
        double x2 = s.x2, y2 = s.y2;
        const double xy = s.xy;
        double D = __dsub_rn(__dmul_rn(x2, y2), __dmul_rn(xy, xy));
        if (D < 0.00694) {
            x2 = x2 + 1.0 / 12.0;
            y2 = y2 + 1.0 / 12.0;
            D = __dsub_rn(__dmul_rn(x2, y2), __dmul_rn(xy, xy));
        }
        c.x = s.x; c.y = s.y; c.x2 = x2; c.y2 = y2; c.xy = xy; c.D = D;
        c.t = __dmul_rn((double)a.kf, (double)__ldg(a.rms + (size_t)s.frame * HW + (size_t)s.ypeak * a.W + s.xpeak));
        c.flux = s.flux;
        c.mean = s.flux / (double)s.npix;
        c.A = 0.0; c.alpha = 0.0; c.zone2 = -1.0;   // zone2 < 0: influences nobody
        if (D > 0.0 && c.t > 0.0) {
            const double sD = sqrt(D);
            const double A = s.flux / __dmul_rn(__dmul_rn(2.0, PI), sD);
            if (A > c.t) {
                const double rho2 = (double)s.npix / __dmul_rn(PI, sD);
                c.A = A;
                c.alpha = (pow(A / c.t, 1.0 / a.beta) - 1.0) / rho2;
                c.zone2 = __dmul_rn(__dmul_rn(a.zone, a.zone), rho2);
            }
        }
        a.w.crec[i] = c;
        if (isfinite(s.x) && isfinite(s.y)) atomicAdd(&a.w.cellcnt[cell_of(a, s.frame, s.x, s.y)], 1u);
    }
}

__global__ void __launch_bounds__(256) k10_scatter(CArgs a) {
    const long long total = c_total(a);
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (long long)gridDim.x * blockDim.x) {
        const bd_source s = a.cat[i];
        if (!(isfinite(s.x) && isfinite(s.y))) continue;
        const size_t c = cell_of(a, s.frame, s.x, s.y);
        a.w.cellitems[a.w.cellprefix[c] + atomicAdd(&a.w.cellcur[c], 1u)] = (int32_t)i;
    }
}

// D11: one warp per neighbour j
__global__ void __launch_bounds__(256) k10_flags(CArgs a) {
    const long long total = c_total(a);
    const int lane = threadIdx.x & 31;
    const long long warps = (long long)gridDim.x * (blockDim.x >> 5);
    for (long long j = (long long)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5); j < total; j += warps) {
        const CRec cj = a.w.crec[j];
        if (!(cj.zone2 >= 0.0) || !isfinite(cj.x) || !isfinite(cj.y)) continue;
        const int frame = a.cat[j].frame, label_j = a.cat[j].label;
        // bounding box of { r_j^2 <= zone2 }: |dx| <= sqrt(zone2 x2), |dy| <= sqrt(zone2 y2)  (+ a safety margin)
        const double hx = sqrt(cj.zone2 * cj.x2) * (1.0 + 1e-9) + 1e-6, hy = sqrt(cj.zone2 * cj.y2) * (1.0 + 1e-9) + 1e-6;
        const int cx0 = min(max((int)floor((cj.x - hx) / CELL), 0), a.w.ncx - 1), cx1 = min(max((int)floor((cj.x + hx) / CELL), 0), a.w.ncx - 1);
        const int cy0 = min(max((int)floor((cj.y - hy) / CELL), 0), a.w.ncy - 1), cy1 = min(max((int)floor((cj.y + hy) / CELL), 0), a.w.ncy - 1);
        for (int cy = cy0; cy <= cy1; ++cy) {
            const size_t c0 = ((size_t)frame * a.w.ncy + cy) * a.w.ncx;
            const uint32_t k0 = a.w.cellprefix[c0 + cx0], k1 = a.w.cellprefix[c0 + cx1 + 1];
            for (uint32_t k = k0 + lane; k < k1; k += 32) {
                const int i = a.w.cellitems[k];
                if (i == j) continue;
                const CRec ci = a.w.crec[i];
                const bool brighter = cj.flux > ci.flux || (cj.flux == ci.flux && label_j < a.cat[i].label);
                if (!brighter) continue;
                const double dx = ci.x - cj.x, dy = ci.y - cj.y;
                // (y2 dx dx + x2 dy dy - 2 xy dx dy) / D, in the definition's operation order
                const double q = __dsub_rn(__dadd_rn(__dmul_rn(__dmul_rn(cj.y2, dx), dx), __dmul_rn(__dmul_rn(cj.x2, dy), dy)),
                                           __dmul_rn(__dmul_rn(__dmul_rn(2.0, cj.xy), dx), dy));
                const double r2 = q / cj.D;
                if (!(r2 <= cj.zone2)) continue;
                const double Ij = cj.A * pow(1.0 + cj.alpha * r2, -a.beta);
                if (ci.mean - Ij <= ci.t) a.w.flag[i] = 1;
            }
        }
    }
}

// survivors -> bit per record index, block counts.  One warp owns 32 consecutive records = one bitmap word: a plain store and
// one atomic per warp (the first version's per-record atomics on ~100 block counters took 190 us on config 5).
__global__ void __launch_bounds__(256) k10_mark(CArgs a) {
    const long long total = c_total(a);
    const int lane = threadIdx.x & 31;
    const long long nwords = (total + 31) >> 5, warps = ((long long)gridDim.x * blockDim.x) >> 5;
    for (long long w = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5; w < nwords; w += warps) {
        const long long i = w * 32 + lane;
        const bool keep = i < total && !a.w.flag[i];
        const uint32_t bits = __ballot_sync(0xffffffffu, keep);
        if (lane == 0 && bits) {
            a.w.keptbits[w] = bits;
            atomicAdd(&a.w.blkcnt[(w * 32) >> RB_SHIFT], (uint32_t)__popc(bits));
        }
    }
}

// compaction in catalogue order, per-frame counts, flags for the caller; false detections leave the label map (D12)
__global__ void __launch_bounds__(256) k10_emit_erase(CArgs a, bd_source *out, int64_t *n_out, uint8_t *flags_out) {
    const long long total = c_total(a);
    const long long t0 = (long long)blockIdx.x * blockDim.x + threadIdx.x, stride = (long long)gridDim.x * blockDim.x;
    if (t0 < a.B) {
        long long off0 = 0;
        for (int f = 0; f < t0; ++f) off0 += a.n_in[f];
        long long off1 = off0 + a.n_in[t0];
        off0 = min(off0, total); off1 = min(off1, total);
        n_out[t0] = (int64_t)kept_rank(a.w.keptbits, a.w.blkprefix, (size_t)off1) - (int64_t)kept_rank(a.w.keptbits, a.w.blkprefix, (size_t)off0);
    }
    for (long long i = t0; i < total; i += stride) {
        const uint8_t fl = a.w.flag[i];
        if (flags_out) flags_out[i] = fl;
        if (fl || !out) continue;
        const uint32_t rank = kept_rank(a.w.keptbits, a.w.blkprefix, (size_t)i);
        if ((int64_t)rank < a.cap_out) out[rank] = a.cat[i];
    }
    const int lane = threadIdx.x & 31;
    const size_t HW = (size_t)a.H * a.W;
    const long long warps = stride >> 5;
    for (long long i = t0 >> 5; i < total; i += warps) {
        if (!a.w.flag[i]) continue;
        const bd_source s = a.cat[i];
        int32_t *L = a.labels + (size_t)s.frame * HW;
        const int bw = s.xmax - s.xmin + 1, n = bw * (s.ymax - s.ymin + 1);
        for (int k = lane; k < n; k += 32) {
            const int yy = k / bw, xx = k - yy * bw;
            int32_t *q = L + (size_t)(s.ymin + yy) * a.W + s.xmin + xx;
            if (*q == s.label) *q = 0;
        }
    }
}

}  // namespace

size_t k10_workspace_bytes(int B, int H, int W, int64_t cap_in) {
    CWs w;
    return carve(w, nullptr, B, H, W, cap_in) + 256;
}

int k10_launch(bd_ctx *ctx, const float *d_rms, int B, int H, int W, double detect_k, const bd_deblend_params *p, int32_t *d_labels,
               const bd_source *d_cat_in, const int64_t *d_n_in, int64_t cap_in, bd_source *d_cat_out, int64_t cap_out,
               int64_t *d_n_out, uint8_t *d_flags, void *d_ws, size_t ws_bytes, cudaStream_t st) {
    CArgs a;
    memset(&a, 0, sizeof(a));
    char *base = (char *)bd_align_up((size_t)d_ws, 256);
    const size_t need = carve(a.w, base, B, H, W, cap_in);
    if ((size_t)(base - (char *)d_ws) + need > ws_bytes)
        return bd_set_error(ctx, BD_EWORKSPACE, "clean workspace: need %zu bytes, got %zu", need + 256, ws_bytes);
    a.rms = d_rms; a.labels = d_labels; a.cat = d_cat_in; a.n_in = d_n_in; a.cap_in = cap_in; a.cap_out = cap_out;
    a.B = B; a.H = H; a.W = W; a.kf = (float)detect_k; a.beta = p->clean_param; a.zone = p->clean_zone;
    BD_CUDA_CHECK(ctx, cudaMemsetAsync(a.w.counters, 0, a.w.zero_bytes, st));
    const int nb = ctx->num_sms * 8;
    k10_prepare<<<nb, 256, 0, st>>>(a);
    k5s_scan_blocks<<<1, 1024, 0, st>>>(a.w.cellcnt, a.w.ncell, a.w.cellprefix, a.w.counters + 1);
    k10_scatter<<<nb, 256, 0, st>>>(a);
    k10_flags<<<nb, 256, 0, st>>>(a);
    k10_mark<<<nb, 256, 0, st>>>(a);
    k5s_scan_blocks<<<1, 1024, 0, st>>>(a.w.blkcnt, a.w.NBk, a.w.blkprefix, a.w.counters + 2);
    const int nbe = nb * 256 >= B ? nb : (B + 255) / 256;
    k10_emit_erase<<<nbe, 256, 0, st>>>(a, d_cat_out, d_n_out, d_flags);
    BD_CUDA_CHECK(ctx, cudaGetLastError());
    return BD_OK;
}
