// K4 + K5: 8-connected component labelling and per-component reduction (steps a4, a5).
// PAPER.md:153 ("identify pixels whose flux exceeds a specified main threshold. These pixels are then
// connected to form source candidates ... calculate peak values and total flux for each candidate"),
// :159 (isophotal photometry).  Readings A16 (8-connectivity), A18-A20 (moments, min_area, label map).
//
// The paper scans with one thread per pixel and reduces with Thrust.  Here:
//   K4a  tile-local union-find in shared memory (128x32-pixel tiles, union by minimum index with
//        atomicMin), written out as parent pointers = 1 + raster index, plus a root bitmap;
//   K4b  seam merge: the pixel pairs that straddle tile borders are united in global memory
//        (atomicMin on the label array); a root that gets linked clears its bit;
//   scan of the root bitmap -> every root's rank in raster order (the catalogue order);
//   K4c  flatten every pixel to its root (= minimum raster index of the component) and count areas
//        by root rank;
//   scan of (area >= min_area) -> catalogue slot of every kept root;
//   K5b  accumulate flux, first and second moments (float64 atomics, coordinates relative to the root
//        pixel), peak (64-bit atomicMax on value|~index) and bounding box of kept components only;
//   K5c  finalise records in slot order = ascending (frame, label).
// Labels are bit-exact by construction; the float sums depend on atomic order (not bit-reproducible).
#include "common.cuh"

namespace {

typedef unsigned long long u64;

constexpr int TW = 128, TH = 32, K4_NT = 256;
constexpr int SCAN_NT = 256, SCAN_PER = 16, SCAN_ELEMS = SCAN_NT * SCAN_PER;

struct Acc {
    double f, sx, sy, sxx, syy, sxy;
    u64 peak;   // (ordered key of sub << 32) | (0xFFFFFFFF - raster index): atomicMax -> max value, ties -> min index
    u64 root;   // global pixel index of the root
    int xmin, xmax, ymin, ymax;
};

struct Ws {
    uint32_t *counters;     // [0] n_roots, [1] n_kept
    uint8_t *maskbuf;       // [P] (only when the caller gave no mask)
    uint32_t *rootbits;     // [NW+1]
    uint32_t *rootprefix;   // [NW+1]
    uint32_t *scanpart;     // [..]
    int32_t *area;          // [maxroots]
    uint32_t *keptprefix;   // [maxroots+1]
    Acc *acc;               // [cap]
    size_t P, NW, maxroots, npart;
    size_t total;
};

size_t carve(Ws &w, void *base, int B, int H, int W, int64_t cap) {
    size_t P = (size_t)B * H * W;
    w.P = P;
    w.NW = (P + 31) / 32;
    w.maxroots = (size_t)B * ((H + 1) / 2) * ((W + 1) / 2);
    size_t nscan = (w.NW + 1 > w.maxroots ? w.NW + 1 : w.maxroots);
    w.npart = (nscan + SCAN_ELEMS - 1) / SCAN_ELEMS + 2;
    size_t off = 0;
    auto take = [&](size_t bytes) { size_t o = off; off = bd_align_up(off + bytes, 256); return (char *)base + o; };
    w.counters = (uint32_t *)take(64 * sizeof(uint32_t));
    w.maskbuf = (uint8_t *)take(P);
    w.rootbits = (uint32_t *)take((w.NW + 1) * sizeof(uint32_t));
    w.rootprefix = (uint32_t *)take((w.NW + 2) * sizeof(uint32_t));
    w.scanpart = (uint32_t *)take(w.npart * sizeof(uint32_t));
    w.area = (int32_t *)take(w.maxroots * sizeof(int32_t));
    w.keptprefix = (uint32_t *)take((w.maxroots + 1) * sizeof(uint32_t));
    w.acc = (Acc *)take((size_t)(cap > 0 ? cap : 1) * sizeof(Acc));
    w.total = off;
    return off;
}

// ------------------------------------------------------------------------------------------------ mask
__global__ void k_make_mask(const float *sub, const float *rms, size_t n4, double k_d, uint8_t *mask) {
    size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n4) return;
    float4 s = reinterpret_cast<const float4 *>(sub)[i], r = reinterpret_cast<const float4 *>(rms)[i];
    uint32_t m = 0;
    m |= (r.x > 0.f && (double)s.x > k_d * (double)r.x) ? 1u : 0u;
    m |= (r.y > 0.f && (double)s.y > k_d * (double)r.y) ? 1u << 8 : 0u;
    m |= (r.z > 0.f && (double)s.z > k_d * (double)r.z) ? 1u << 16 : 0u;
    m |= (r.w > 0.f && (double)s.w > k_d * (double)r.w) ? 1u << 24 : 0u;
    reinterpret_cast<uint32_t *>(mask)[i] = m;
}

// ------------------------------------------------------------------------------------------------ K4a
__device__ __forceinline__ uint32_t sm_find(volatile uint32_t *parent, uint32_t x) {
    uint32_t p = parent[x];
    while (p != x) { x = p; p = parent[x]; }
    return x;
}
__device__ __noinline__ void sm_union(uint32_t *parent, uint32_t a, uint32_t b) {
    for (;;) {
        a = sm_find(parent, a);
        b = sm_find(parent, b);
        if (a == b) return;
        if (a < b) { uint32_t t = a; a = b; b = t; }
        uint32_t old = atomicMin(&parent[a], b);
        if (old == a) return;
        a = old;
    }
}

__global__ void __launch_bounds__(K4_NT) k4a_tile_label(const uint8_t *mask, int H, int W, int32_t *labels,
                                                        uint32_t *rootbits, int aligned32) {
    __shared__ uint32_t sm_mask[TH][TW / 4 + 1];
    __shared__ uint32_t parent[TH * TW];
    const int frame = blockIdx.z;
    const int x0 = blockIdx.x * TW, y0 = blockIdx.y * TH;
    const size_t fbase = (size_t)frame * H * W;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int rx0 = lane * 4;
    const bool col_ok = (x0 + rx0) < W;

#pragma unroll
    for (int k = 0; k < TH / 8; ++k) {
        int ry = warp + 8 * k;
        uint32_t m = 0;
        if (col_ok && (y0 + ry) < H) {
            m = __ldcs(reinterpret_cast<const uint32_t *>(mask + fbase + (size_t)(y0 + ry) * W + x0 + rx0));
            m = ((((m & 0x7F7F7F7Fu) + 0x7F7F7F7Fu) | m) & 0x80808080u) >> 7;   // bytes -> 0/1
        }
        sm_mask[ry][lane] = m;
#pragma unroll
        for (int q = 0; q < 4; ++q) parent[ry * TW + rx0 + q] = ry * TW + rx0 + q;
    }
    __syncthreads();

    auto fg = [&](int ry, int rx) -> uint32_t {
        if (ry < 0 || rx < 0 || rx >= TW) return 0u;
        return (sm_mask[ry][rx >> 2] >> (8 * (rx & 3))) & 1u;
    };
    // not unrolled on purpose: the unrolled body (16 pixels x 4 inlined union loops) was 85 KB of SASS and
    // the kernel was instruction-fetch bound (ncu: 65% stall_no_inst)
#pragma unroll 1
    for (int k = 0; k < TH / 8; ++k) {
        int ry = warp + 8 * k;
        uint32_t m = sm_mask[ry][lane];
        if (!m) continue;
#pragma unroll 1
        for (int q = 0; q < 4; ++q) {
            if (!((m >> (8 * q)) & 1u)) continue;
            int rx = rx0 + q;
            uint32_t p = ry * TW + rx;
            uint32_t w = fg(ry, rx - 1), a = fg(ry - 1, rx - 1), b = fg(ry - 1, rx), c = fg(ry - 1, rx + 1);
            if (w) sm_union(parent, p, p - 1);
            if (b) { if (!w) sm_union(parent, p, p - TW); }
            else {
                if (a && !w) sm_union(parent, p, p - TW - 1);
                if (c) sm_union(parent, p, p - TW + 1);
            }
        }
    }
    __syncthreads();

#pragma unroll 1
    for (int k = 0; k < TH / 8; ++k) {
        int ry = warp + 8 * k;
        bool row_ok = col_ok && (y0 + ry) < H;
        uint32_t m = sm_mask[ry][lane];
        int out[4];
        uint32_t nib = 0;
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            out[q] = 0;
            if ((m >> (8 * q)) & 1u) {
                uint32_t p = ry * TW + rx0 + q;
                uint32_t r = sm_find(parent, p);
                out[q] = (y0 + (int)(r / TW)) * W + x0 + (int)(r % TW) + 1;
                if (r == p) nib |= 1u << q;
            }
        }
        size_t g = fbase + (size_t)(y0 + ry) * W + x0 + rx0;
        if (row_ok) __stcg(reinterpret_cast<int4 *>(labels + g), make_int4(out[0], out[1], out[2], out[3]));
        if (aligned32) {
            uint32_t word = nib << (4 * (lane & 7));
            word |= __shfl_xor_sync(0xffffffffu, word, 1);
            word |= __shfl_xor_sync(0xffffffffu, word, 2);
            word |= __shfl_xor_sync(0xffffffffu, word, 4);
            if (row_ok && (lane & 7) == 0) rootbits[g >> 5] = word;
        } else if (row_ok && nib) {
            atomicOr(&rootbits[g >> 5], nib << (g & 31));
        }
    }
}

// ------------------------------------------------------------------------------------------------ K4b
__device__ __forceinline__ int g_find(const int32_t *L, int a) {
    for (;;) {
        int p = __ldcg(L + a) - 1;
        if (p == a) return a;
        a = p;
    }
}
__device__ __forceinline__ void g_union(int32_t *L, uint32_t *rootbits, size_t fbase, int a, int b) {
    for (;;) {
        a = g_find(L, a);
        b = g_find(L, b);
        if (a == b) return;
        if (a < b) { int t = a; a = b; b = t; }
        int old = atomicMin(L + a, b + 1);
        if (old == a + 1) {   // a was a root and now hangs under b
            size_t g = fbase + (size_t)a;
            atomicAnd(&rootbits[g >> 5], ~(1u << (g & 31)));
            return;
        }
        a = old - 1;
    }
}

// horizontal seams: row y = k*TH (k >= 1) against row y-1, all x
__global__ void k4b_seam_h(const uint8_t *mask, int H, int W, int32_t *labels, uint32_t *rootbits) {
    const int frame = blockIdx.z, seam = blockIdx.y + 1;
    const int y = seam * TH;
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    if (y >= H || x >= W) return;
    const size_t fbase = (size_t)frame * H * W;
    const uint8_t *m = mask + fbase;
    if (!m[(size_t)y * W + x]) return;
    int32_t *L = labels + fbase;
    const int p = y * W + x;
    const uint8_t *up = m + (size_t)(y - 1) * W;
    bool b = up[x], a = x > 0 && up[x - 1], c = x + 1 < W && up[x + 1];
    if (b) g_union(L, rootbits, fbase, p, p - W);
    else {
        if (a) g_union(L, rootbits, fbase, p, p - W - 1);
        if (c) g_union(L, rootbits, fbase, p, p - W + 1);
    }
}

// vertical seams: columns x-1 | x with x = k*TW (k >= 1), all y; the 2x2 block (y-1..y) x (x-1..x)
__global__ void k4b_seam_v(const uint8_t *mask, int H, int W, int32_t *labels, uint32_t *rootbits) {
    const int frame = blockIdx.z, seam = blockIdx.y + 1;
    const int x = seam * TW;
    const int y = blockIdx.x * blockDim.x + threadIdx.x;
    if (x >= W || y >= H) return;
    const size_t fbase = (size_t)frame * H * W;
    const uint8_t *m = mask + fbase;
    int32_t *L = labels + fbase;
    const bool m10 = m[(size_t)y * W + x - 1], m11 = m[(size_t)y * W + x];
    if (!m10 && !m11) return;
    const bool m00 = y > 0 && m[(size_t)(y - 1) * W + x - 1], m01 = y > 0 && m[(size_t)(y - 1) * W + x];
    const int p = y * W + x;
    if (m10 && m11) g_union(L, rootbits, fbase, p, p - 1);
    if (m11 && m00 && !m01) g_union(L, rootbits, fbase, p, p - W - 1);
    if (m10 && m01 && !m00) g_union(L, rootbits, fbase, p - 1, p - W);
}

// ------------------------------------------------------------------------------------------------ scans
// MODE 0: popc(bits[i]), i < n (host n).  MODE 1: (area[i] >= min_area), i < *n_dev.
struct ScanArgs {
    const uint32_t *bits;
    const int32_t *area;
    const uint32_t *n_dev;
    size_t n;
    int min_area;
    uint32_t *out;        // [n+1] exclusive prefix, out[n] = total
    uint32_t *part;
    uint32_t *total_out;
};
template <int MODE>
__device__ __forceinline__ uint32_t scan_load(const ScanArgs &a, size_t i, size_t n) {
    if (i >= n) return 0;
    if (MODE == 0) return __popc(a.bits[i]);
    return a.area[i] >= a.min_area ? 1u : 0u;
}
template <int MODE>
__global__ void __launch_bounds__(SCAN_NT) scan_reduce(ScanArgs a) {
    __shared__ uint32_t red[SCAN_NT / 32];
    const size_t n = MODE == 0 ? a.n : (size_t)*a.n_dev;
    const size_t b0 = (size_t)blockIdx.x * SCAN_ELEMS;
    uint32_t s = 0;
    if (b0 < n)
        for (int k = 0; k < SCAN_PER; ++k) s += scan_load<MODE>(a, b0 + (size_t)k * SCAN_NT + threadIdx.x, n);
    for (int o = 16; o; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        uint32_t t = 0;
        for (int w = 0; w < SCAN_NT / 32; ++w) t += red[w];
        a.part[blockIdx.x] = t;
    }
}
__global__ void __launch_bounds__(1024) scan_top(uint32_t *part, size_t nblk, uint32_t *total_out) {
    __shared__ uint32_t red[32];
    __shared__ uint32_t carry_s;
    if (threadIdx.x == 0) carry_s = 0;
    __syncthreads();
    for (size_t base = 0; base < nblk; base += 1024) {
        size_t i = base + threadIdx.x;
        uint32_t v = i < nblk ? part[i] : 0, incl = v;
        const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
        for (int o = 1; o < 32; o <<= 1) { uint32_t t = __shfl_up_sync(0xffffffffu, incl, o); if (lane >= o) incl += t; }
        if (lane == 31) red[warp] = incl;
        __syncthreads();
        uint32_t wbase = 0;
        for (int w = 0; w < warp; ++w) wbase += red[w];
        uint32_t carry = carry_s;
        if (i < nblk) part[i] = carry + wbase + incl - v;
        __syncthreads();
        if (threadIdx.x == 1023) carry_s = carry + wbase + incl;
        __syncthreads();
    }
    if (threadIdx.x == 0) *total_out = carry_s;
}
template <int MODE>
__global__ void __launch_bounds__(SCAN_NT) scan_apply(ScanArgs a) {
    __shared__ uint32_t red[SCAN_NT / 32];
    const size_t n = MODE == 0 ? a.n : (size_t)*a.n_dev;
    const size_t b0 = (size_t)blockIdx.x * SCAN_ELEMS;
    if (b0 > n) return;
    // thread t owns SCAN_PER consecutive elements
    const size_t t0 = b0 + (size_t)threadIdx.x * SCAN_PER;
    uint32_t v[SCAN_PER], local = 0;
#pragma unroll
    for (int k = 0; k < SCAN_PER; ++k) { v[k] = scan_load<MODE>(a, t0 + k, n); local += v[k]; }
    uint32_t incl = local;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (int o = 1; o < 32; o <<= 1) { uint32_t t = __shfl_up_sync(0xffffffffu, incl, o); if (lane >= o) incl += t; }
    if (lane == 31) red[warp] = incl;
    __syncthreads();
    uint32_t run = a.part[blockIdx.x] + incl - local;
    for (int w = 0; w < warp; ++w) run += red[w];
#pragma unroll
    for (int k = 0; k < SCAN_PER; ++k) {
        if (t0 + k <= n) a.out[t0 + k] = run;   // also writes out[n] = total
        run += v[k];
    }
}

// ------------------------------------------------------------------------------------------------ K4c / K5
__device__ __forceinline__ uint32_t root_rank(const uint32_t *rootbits, const uint32_t *rootprefix, size_t g) {
    return __ldg(rootprefix + (g >> 5)) + __popc(__ldg(rootbits + (g >> 5)) & ((1u << (g & 31)) - 1u));
}

__global__ void k_zero_area(int32_t *area, const uint32_t *n_roots) {
    size_t n = *n_roots;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) area[i] = 0;
}

// flatten to roots + area count; one thread per 4 pixels
__global__ void __launch_bounds__(256) k4c_flatten_count(int32_t *labels, int H, int W, size_t n4_per_frame,
                                                         const uint32_t *rootbits, const uint32_t *rootprefix,
                                                         int32_t *area) {
    const int frame = blockIdx.y;
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n4_per_frame) return;
    const size_t fbase = (size_t)frame * H * W;
    int32_t *L = labels + fbase;
    int4 v = __ldcg(reinterpret_cast<const int4 *>(L) + i);
    if (!(v.x | v.y | v.z | v.w)) return;
    int l[4] = {v.x, v.y, v.z, v.w};
    bool changed = false;
    int prev_root = -1;
    uint32_t prev_id = 0;
    int run = 0;
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        if (!l[q]) continue;
        int r = g_find(L, l[q] - 1);
        if (r + 1 != l[q]) { l[q] = r + 1; changed = true; }
        if (r == prev_root) { ++run; continue; }
        if (run) atomicAdd(&area[prev_id], run);
        prev_root = r;
        prev_id = root_rank(rootbits, rootprefix, fbase + (size_t)r);
        run = 1;
    }
    if (run) atomicAdd(&area[prev_id], run);
    if (changed) __stcg(reinterpret_cast<int4 *>(L) + i, make_int4(l[0], l[1], l[2], l[3]));
}

__global__ void k_init_acc(Acc *acc, const uint32_t *n_kept, int64_t cap) {
    size_t n = *n_kept;
    if ((int64_t)n > cap) n = (size_t)cap;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        Acc a;
        a.f = a.sx = a.sy = a.sxx = a.syy = a.sxy = 0.0;
        a.peak = 0; a.root = 0;
        a.xmin = 0x7FFFFFFF; a.ymin = 0x7FFFFFFF; a.xmax = -1; a.ymax = -1;
        acc[i] = a;
    }
}

__global__ void k_frame_counts(const uint32_t *rootbits, const uint32_t *rootprefix, const uint32_t *keptprefix,
                               int B, size_t HW, int64_t *n_sources) {
    int f = blockIdx.x * blockDim.x + threadIdx.x;
    if (f >= B) return;
    uint32_t r0 = root_rank(rootbits, rootprefix, (size_t)f * HW), r1 = root_rank(rootbits, rootprefix, (size_t)(f + 1) * HW);
    n_sources[f] = (int64_t)(keptprefix[r1] - keptprefix[r0]);
}

struct Part {   // a thread's running partial for one slot
    double f, sx, sy, sxx, syy, sxy;
    u64 peak;
    int xmin, xmax, ymin, ymax;
};
__device__ __forceinline__ void flush_part(Acc *acc, uint32_t slot, const Part &p) {
    Acc *a = acc + slot;
    atomicAdd(&a->f, p.f);
    atomicAdd(&a->sx, p.sx);
    atomicAdd(&a->sy, p.sy);
    atomicAdd(&a->sxx, p.sxx);
    atomicAdd(&a->syy, p.syy);
    atomicAdd(&a->sxy, p.sxy);
    atomicMax(&a->peak, p.peak);
    atomicMin(&a->xmin, p.xmin);
    atomicMax(&a->xmax, p.xmax);
    atomicMin(&a->ymin, p.ymin);
    atomicMax(&a->ymax, p.ymax);
}

__global__ void __launch_bounds__(256) k5b_accumulate(const int32_t *labels, const float *sub, int H, int W,
                                                      size_t n4_per_frame, const uint32_t *rootbits,
                                                      const uint32_t *rootprefix, const int32_t *area,
                                                      const uint32_t *keptprefix, int min_area, Acc *acc, int64_t cap) {
    const int frame = blockIdx.y;
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n4_per_frame) return;
    const size_t fbase = (size_t)frame * H * W;
    int4 v = __ldcs(reinterpret_cast<const int4 *>(labels + fbase) + i);
    if (!(v.x | v.y | v.z | v.w)) return;
    const int l[4] = {v.x, v.y, v.z, v.w};
    const float4 sv = __ldcs(reinterpret_cast<const float4 *>(sub + fbase) + i);
    const float I4[4] = {sv.x, sv.y, sv.z, sv.w};
    const int p0 = (int)(i * 4);
    const int y = p0 / W, x0 = p0 - y * W;

    int prev_root = -1;
    bool have = false;
    uint32_t slot = 0;
    int xr = 0, yr = 0;
    Part part;
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        if (!l[q]) continue;
        const int r = l[q] - 1;
        if (r != prev_root) {
            if (have) flush_part(acc, slot, part);
            prev_root = r;
            have = false;
            uint32_t id = root_rank(rootbits, rootprefix, fbase + (size_t)r);
            if (__ldg(area + id) >= min_area) {
                slot = __ldg(keptprefix + id);
                if ((int64_t)slot < cap) {
                    have = true;
                    yr = r / W; xr = r - yr * W;
                    part.f = part.sx = part.sy = part.sxx = part.syy = part.sxy = 0.0;
                    part.peak = 0;
                    part.xmin = 0x7FFFFFFF; part.ymin = 0x7FFFFFFF; part.xmax = -1; part.ymax = -1;
                }
            }
        }
        if (!have) continue;
        const int x = x0 + q;
        if (p0 + q == r) acc[slot].root = (u64)(fbase + (size_t)r);
        const double I = (double)I4[q], dx = (double)(x - xr), dy = (double)(y - yr);
        part.f += I;
        part.sx = fma(I, dx, part.sx);
        part.sy = fma(I, dy, part.sy);
        part.sxx = fma(I * dx, dx, part.sxx);
        part.syy = fma(I * dy, dy, part.syy);
        part.sxy = fma(I * dx, dy, part.sxy);
        u64 pk = ((u64)f32_to_key(I4[q]) << 32) | (u64)(0xFFFFFFFFu - (uint32_t)(p0 + q));
        part.peak = pk > part.peak ? pk : part.peak;
        part.xmin = min(part.xmin, x); part.xmax = max(part.xmax, x);
        part.ymin = min(part.ymin, y); part.ymax = max(part.ymax, y);
    }
    if (have) flush_part(acc, slot, part);
}

__global__ void k5c_finalize(const Acc *acc, const uint32_t *n_kept, int64_t cap, const int32_t *area,
                             const uint32_t *rootbits, const uint32_t *rootprefix, size_t HW, int W, bd_source *cat) {
    size_t n = *n_kept;
    if ((int64_t)n > cap) n = (size_t)cap;
    size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    Acc a = acc[i];
    bd_source s;
    const size_t g = (size_t)a.root;
    const int frame = (int)(g / HW);
    const int r = (int)(g - (size_t)frame * HW);
    const int yr = r / W, xr = r - yr * W;
    s.frame = frame;
    s.label = r + 1;
    s.npix = area[root_rank(rootbits, rootprefix, g)];
    s.xmin = a.xmin; s.xmax = a.xmax; s.ymin = a.ymin; s.ymax = a.ymax;
    const uint32_t pidx = 0xFFFFFFFFu - (uint32_t)(a.peak & 0xFFFFFFFFull);
    s.ypeak = (int)(pidx / (uint32_t)W);
    s.xpeak = (int)(pidx - (uint32_t)s.ypeak * (uint32_t)W);
    s.peak = key_to_f32((uint32_t)(a.peak >> 32));
    s.flux = a.f;
    const double mx = a.sx / a.f, my = a.sy / a.f;
    s.x = (double)xr + mx;
    s.y = (double)yr + my;
    s.x2 = a.sxx / a.f - mx * mx;
    s.y2 = a.syy / a.f - my * my;
    s.xy = a.sxy / a.f - mx * my;
    cat[i] = s;
}

}  // namespace

size_t k45_workspace_bytes(int B, int H, int W, int64_t cat_capacity) {
    Ws w;
    return carve(w, nullptr, B, H, W, cat_capacity) + 256;
}

int k45_launch(bd_ctx *ctx, const float *d_sub, const float *d_rms, const uint8_t *d_mask, int B, int H, int W,
               double detect_k, int min_area, int32_t *d_labels, bd_source *d_cat, int64_t cat_capacity,
               int64_t *d_n_sources, void *d_ws, size_t ws_bytes, cudaStream_t st) {
    Ws w;
    char *base = (char *)bd_align_up((size_t)d_ws, 256);
    size_t need = carve(w, base, B, H, W, cat_capacity);
    if ((size_t)(base - (char *)d_ws) + need > ws_bytes)
        return bd_set_error(ctx, BD_EWORKSPACE, "detect workspace: need %zu bytes, got %zu", need + 256, ws_bytes);
    const size_t HW = (size_t)H * W, P = w.P;
    const size_t n4f = HW / 4;

    const uint8_t *mask = d_mask;
    if (!mask) {
        size_t n4 = P / 4;
        k_make_mask<<<(unsigned)((n4 + 255) / 256), 256, 0, st>>>(d_sub, d_rms, n4, detect_k, w.maskbuf);
        mask = w.maskbuf;
    }
    const int aligned32 = (W % 32 == 0 && HW % 32 == 0) ? 1 : 0;
    if (aligned32) BD_CUDA_CHECK(ctx, cudaMemsetAsync(w.rootbits + w.NW, 0, sizeof(uint32_t), st));
    else BD_CUDA_CHECK(ctx, cudaMemsetAsync(w.rootbits, 0, (w.NW + 1) * sizeof(uint32_t), st));

    dim3 tg((W + TW - 1) / TW, (H + TH - 1) / TH, B);
    k4a_tile_label<<<tg, K4_NT, 0, st>>>(mask, H, W, d_labels, w.rootbits, aligned32);
    if (tg.y > 1) {
        dim3 g((W + 255) / 256, tg.y - 1, B);
        k4b_seam_h<<<g, 256, 0, st>>>(mask, H, W, d_labels, w.rootbits);
    }
    if (tg.x > 1) {
        dim3 g((H + 127) / 128, tg.x - 1, B);
        k4b_seam_v<<<g, 128, 0, st>>>(mask, H, W, d_labels, w.rootbits);
    }
    // rank of every root in raster order
    {
        ScanArgs a = {};
        a.bits = w.rootbits; a.n = w.NW + 1; a.out = w.rootprefix; a.part = w.scanpart; a.total_out = w.counters + 0;
        size_t nblk = (a.n + SCAN_ELEMS) / SCAN_ELEMS;
        scan_reduce<0><<<(unsigned)nblk, SCAN_NT, 0, st>>>(a);
        scan_top<<<1, 1024, 0, st>>>(w.scanpart, nblk, a.total_out);
        scan_apply<0><<<(unsigned)nblk, SCAN_NT, 0, st>>>(a);
    }
    k_zero_area<<<ctx->num_sms * 8, 256, 0, st>>>(w.area, w.counters + 0);
    {
        dim3 g((unsigned)((n4f + 255) / 256), B);
        k4c_flatten_count<<<g, 256, 0, st>>>(d_labels, H, W, n4f, w.rootbits, w.rootprefix, w.area);
    }
    // catalogue slot of every kept root
    {
        ScanArgs a = {};
        a.area = w.area; a.n_dev = w.counters + 0; a.min_area = min_area; a.out = w.keptprefix; a.part = w.scanpart;
        a.total_out = w.counters + 1;
        size_t nblk = (w.maxroots + SCAN_ELEMS) / SCAN_ELEMS;
        scan_reduce<1><<<(unsigned)nblk, SCAN_NT, 0, st>>>(a);
        scan_top<<<1, 1024, 0, st>>>(w.scanpart, nblk, a.total_out);
        scan_apply<1><<<(unsigned)nblk, SCAN_NT, 0, st>>>(a);
    }
    k_frame_counts<<<(B + 127) / 128, 128, 0, st>>>(w.rootbits, w.rootprefix, w.keptprefix, B, HW, d_n_sources);
    if (cat_capacity > 0 && d_cat) {
        k_init_acc<<<ctx->num_sms * 4, 256, 0, st>>>(w.acc, w.counters + 1, cat_capacity);
        dim3 g((unsigned)((n4f + 255) / 256), B);
        k5b_accumulate<<<g, 256, 0, st>>>(d_labels, d_sub, H, W, n4f, w.rootbits, w.rootprefix, w.area, w.keptprefix,
                                           min_area, w.acc, cat_capacity);
        size_t maxrec = (size_t)(cat_capacity < (int64_t)w.maxroots ? cat_capacity : (int64_t)w.maxroots);
        k5c_finalize<<<(unsigned)((maxrec + 255) / 256), 256, 0, st>>>(w.acc, w.counters + 1, cat_capacity, w.area,
                                                                       w.rootbits, w.rootprefix, HW, W, d_cat);
    }
    BD_CUDA_CHECK(ctx, cudaGetLastError());
    return BD_OK;
}
