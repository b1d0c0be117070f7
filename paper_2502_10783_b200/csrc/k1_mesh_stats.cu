// K1: per-mesh iterative sigma-clipped statistics (step a1).  PAPER.md:67 (rectangular sub-regions),
// :69-76 (eqs. 1-4), :78 ("determine the upper and lower limits based on the calculated central value and
// the specified sigma range, exclude data outside these limits, and recalculate the central value and
// standard deviation ... Once the maximum number of iterations is reached or the data stabilizes ...").
//
// The paper gives one GPU *thread* per sub-region.  Here a mesh is owned by a team of C CTAs (a
// thread-block cluster; C = 1 when the mesh fits one CTA's shared memory): each CTA stages a slab of the
// mesh's rows in shared memory with one TMA bulk-tensor load, so HBM sees each pixel once (4 B/px).
//
// What the clipping loop needs.  The survivors of every round are the pixels in a value interval [LO, HI]
// (LO = max of the lower bounds so far, HI = min of the upper bounds).  A round needs (1) n, sum(x-p),
// sum((x-p)^2) over [LO, HI] and the count below LO -- float64 sums against float64 bounds, so the survivor
// set is the float64 definition's -- and (2) two order statistics of the WHOLE mesh.
//
// Fast path (two sweeps of the slab, whatever the number of rounds).  While the TMA load is in flight every
// CTA reads the same small lattice sample of the mesh from global memory and sorts it (bitonic).  Sample
// quantiles give a key bracket [ka, kb] that contains the median rank and a conservative core interval
// [A, B] = q50 -+ c*(q50 - q16) that every clipping bound of the paper's loop stays outside of.
//   sweep 1: float64 core sums over [A, B]; count of "tail" pixels outside it; a 64-bin histogram of the
//            bracket with PER-THREAD byte counters (plain load/add/store: no shared-memory atomics, which
//            run at ~1/clk/SM), reduced with dp4a; team-wide totals through distributed shared memory;
//   sweep 2: gather the pixels of a window of bins around the median rank (<= 2048) and the tail pixels.
// Rank 0 of the team collects both lists through DSMEM, the other CTAs exit.  It sorts the window once
// (every round's median is then a table lookup) and runs the rounds on the tail list alone:
//   n = n_core + #tail in [lo, hi],  sums = core sums + tail sums.
// Any assumption that fails (bound enters the core, median rank leaves the window, tail list overflow,
// degenerate sample) sends the mesh to the
// Slow path (general, one CTA): a sweep per round plus a radix select that descends 64-bin histograms from
// the key range of [mean - sd, mean + sd] (the median lies within one standard deviation of the mean).
// It reads the slab from shared memory when C = 1 and the mesh from global memory (L2) otherwise.
#include <cooperative_groups.h>

#include "common.cuh"

namespace cg = cooperative_groups;

namespace {

constexpr int K1_NBIN = 64;        // histogram bins per level
constexpr int K1_T1 = 512;         // slow path: stop refining when the target bin holds <= this many pixels
constexpr int K1_LISTCAP = 4096;   // candidate window capacity (team total) with >= 512 threads; 2048 with 256
constexpr int K1_MAXWARPS = 16;
constexpr int K1_MAXC = 8;
#ifndef K1_FAST_MIN
#define K1_FAST_MIN 4096
#endif
constexpr int K1_FAST_MIN_PX = K1_FAST_MIN;   // smallest mesh for the fast path (measured: 64x64 meshes gain 25 % from it;
                                       // the dead slab of a 64x64 mesh, 16 KiB, exactly holds the sort arrays)

#ifdef K1_TIMING
__device__ unsigned long long g_k1_t[16];
#define K1_T(i) do { if (tid == 0) { const long long t_ = clock64(); atomicAdd(&g_k1_t[i], (unsigned long long)(t_ - t_prev)); t_prev = t_; } } while (0)
#else
#define K1_T(i) do { } while (0)
#endif
__device__ unsigned long long g_k1_slow_meshes;   // diagnostic: meshes that took the slow path
__device__ unsigned long long g_k1_reason[8];     // diagnostic: why (1 sample, 2 tails, 3 rank/bin, 4 window, 5 round window, 6 bound)

struct K1Args {
    const float *img;
    int B, H, W, mh, mw, ny, nx;
    int slab_rows, use_tma, tailcap, allow_fast;
    int stream;          // no slab: the sweeps read the mesh from global memory (second sweep: L2)
    int slab_bytes;      // shared memory reserved in front of Smem (the slab, or room for the sort arrays)
    double k_c;
    int iters, skew_guard;
    double median_factor, mean_factor;
    double *bkg_raw, *rms_raw, *median, *mean;
    int32_t *n_kept;
    const uint32_t *list_count, *list;   // list mode (C == 1): the meshes to do are list[0 .. *list_count), grid-stride
    // background variants (readings B1, B2, B6): bad-pixel mask [B,H,W] (non-zero = excluded) and the validity rules
    const uint8_t *bad;
    int min_valid;
    double max_masked_frac, max_reject_frac;
    int32_t *n_valid;
};

struct Xch {   // one CTA's contribution to the team-wide totals (peers read it through DSMEM)
    double s1, s2;
    int n_core, n_tail;
    uint32_t below, m_cand, m_tail, pad;
    uint32_t cnt[K1_NBIN];
};

struct SampleX {   // one CTA's sample statistics (peers read them through DSMEM)
    double q50, q16;
    double lo3, hi3;     // sample quantiles 3 standard deviations either side of 0.5 (averaged over a team of >= 4)
    uint32_t ka, kb;     // keys of the quantiles 6 standard deviations either side (used as they are otherwise)
    int valid, pad;
};

struct Smem {   // fixed-size part of shared memory; follows the slab
    alignas(16) unsigned long long mbar;
    SampleX sx;
    Xch xch;
    Xch tot;
    double red_d[2][2][K1_MAXWARPS];   // [slot set][quantity][warp], see block_reduce_stats
    int red_i[2][2][K1_MAXWARPS];
    uint32_t red_u[K1_MAXWARPS];
    uint32_t win_b0, win_b1;
    uint32_t list[K1_LISTCAP];   // candidate keys: this CTA's during the gather; the team's (sorted) at rank 0
    // the work area follows: sample keys -> per-thread byte histograms -> tail pixels
};

// bytes of Smem in use: with fewer than 512 threads only the first 2048 entries of list[] (the last member) are used, and
// the work area starts right after them
__host__ __device__ inline size_t k1_smem_fixed_bytes(int threads) {
    const size_t cut = threads >= 512 ? 0 : (size_t)(K1_LISTCAP - 2048) * sizeof(uint32_t);
    return (sizeof(Smem) - cut + 127) & ~(size_t)127;
}

template <int C>
struct Team {
    __device__ static void sync() {
        if constexpr (C == 1) __syncthreads();
        else cg::this_cluster().sync();
    }
    __device__ static unsigned rank() {
        if constexpr (C == 1) return 0;
        else return cg::this_cluster().block_rank();
    }
    template <typename T>
    __device__ static T *remote(T *p, unsigned r) {
        if constexpr (C == 1) return p;
        else return cg::this_cluster().map_shared_rank(p, r);
    }
};

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

// Sweep primitives on precomputed shared-memory addresses, predicated instead of branched (the compiler's version
// of `if (t <= span) col[(t >> shift) * nt] += 1` re-derived tid, the shared base and blockDim for every pixel and
// wrapped it in BSSY/BSYNC: ~75 instructions per pixel over the two sweeps).
// byte counter of bin (t >> shift), column `col_s` (= this thread's), row pitch nt:  if (t <= span) ++counter
__device__ __forceinline__ void k1_hist_inc(uint32_t col_s, uint32_t t, uint32_t span, int shift, int nt) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t.reg .u32 a, v;\n\t"
        "setp.le.u32 p, %1, %2;\n\t"
        "shr.u32 a, %1, %3;\n\t"
        "mad.lo.u32 a, a, %4, %0;\n\t"
        "@p ld.shared.u8 v, [a];\n\t"
        "@p add.u32 v, v, 1;\n\t"
        "@p st.shared.u8 [a], v;\n\t}"
        ::"r"(col_s), "r"(t), "r"(span), "r"(shift), "r"(nt)
        : "memory");
}
// if (t <= span) { *addr = k; addr += 4; }
__device__ __forceinline__ void k1_push_u32_if_le(uint32_t &addr, uint32_t t, uint32_t span, uint32_t k) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "setp.le.u32 p, %1, %2;\n\t"
        "@p st.shared.u32 [%0], %3;\n\t"
        "@p add.u32 %0, %0, 4;\n\t}"
        : "+r"(addr)
        : "r"(t), "r"(span), "r"(k)
        : "memory");
}
// if (!(lo <= e && e <= hi)) { *addr = e; addr += 4; }
__device__ __forceinline__ void k1_push_f32_if_outside(uint32_t &addr, float e, float lo, float hi) {
    asm volatile(
        "{\n\t.reg .pred p, q;\n\t"
        "setp.ge.f32 p, %1, %2;\n\t"
        "setp.le.and.f32 q, %1, %3, p;\n\t"
        "@!q st.shared.f32 [%0], %1;\n\t"
        "@!q add.u32 %0, %0, 4;\n\t}"
        : "+r"(addr)
        : "f"(e), "f"(lo), "f"(hi)
        : "memory");
}

// ---- warp-wide helpers (also used by k1w_warp_mesh.cuh) -----------------------------------------------------
__device__ __forceinline__ double kw_sum(double v) {
#pragma unroll
    for (int o = 16; o; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
__device__ __forceinline__ int kw_sum(int v) { return __reduce_add_sync(0xffffffffu, v); }

// ascending bitonic sort of 256 keys held 8 per lane, element e = lane * 8 + r
__device__ __forceinline__ void kw_sort256(uint32_t (&x)[8], int lane) {
#pragma unroll
    for (int k = 2; k <= 256; k <<= 1) {
#pragma unroll
        for (int j = k >> 1; j > 0; j >>= 1) {
            if (j >= 8) {
                const int lm = j >> 3;
                const bool keep_min = ((lane & lm) == 0) == (((lane * 8) & k) == 0);
#pragma unroll
                for (int r = 0; r < 8; ++r) {
                    const uint32_t y = __shfl_xor_sync(0xffffffffu, x[r], lm);
                    x[r] = keep_min ? min(x[r], y) : max(x[r], y);
                }
            } else {
#pragma unroll
                for (int r = 0; r < 8; ++r) {
                    const int p = r ^ j;
                    if (p > r) {
                        const bool up = ((lane * 8 + r) & k) == 0;
                        const uint32_t lo = min(x[r], x[p]), hi = max(x[r], x[p]);
                        x[r] = up ? lo : hi;
                        x[p] = up ? hi : lo;
                    }
                }
            }
        }
    }
}

// ---- block-wide reductions (result valid in every thread) -------------------------------------------------
// ONE barrier per call: every warp leaves its partial in the slot set `ph & 1`, and after the barrier every thread adds
// the (<= 16) partials itself, in warp order -- the same bits in every thread.  The slot sets alternate from call to
// call (ph counts the calls; all threads of the CTA make the same calls), so a set is rewritten only after a later
// call's barrier, when nobody reads it any more.  (The first version used three barriers and a second shuffle tree per
// call; with a call per clipping round that was 25 k cycles per mesh.)
__device__ __forceinline__ void block_reduce_stats(Smem &s, int &ph, double &s1, double &s2, int &n_in, int &n_below) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = blockDim.x >> 5, set = ph & 1;
    ++ph;
#pragma unroll
    for (int o = 16; o; o >>= 1) {
        s1 += __shfl_xor_sync(0xffffffffu, s1, o);
        s2 += __shfl_xor_sync(0xffffffffu, s2, o);
    }
    n_in = __reduce_add_sync(0xffffffffu, n_in);
    n_below = __reduce_add_sync(0xffffffffu, n_below);
    if (lane == 0) { s.red_d[set][0][warp] = s1; s.red_d[set][1][warp] = s2; s.red_i[set][0][warp] = n_in; s.red_i[set][1][warp] = n_below; }
    __syncthreads();
    // lane l takes the partial of warp l & 15; a xor tree over 16 lanes (the same in both halves of every warp)
    const int w = lane & 15;
    s1 = w < nw ? s.red_d[set][0][w] : 0.0; s2 = w < nw ? s.red_d[set][1][w] : 0.0;
    n_in = w < nw ? s.red_i[set][0][w] : 0; n_below = w < nw ? s.red_i[set][1][w] : 0;
#pragma unroll
    for (int o = 8; o; o >>= 1) {
        s1 += __shfl_xor_sync(0xffffffffu, s1, o);
        s2 += __shfl_xor_sync(0xffffffffu, s2, o);
        n_in += __shfl_xor_sync(0xffffffffu, n_in, o);
        n_below += __shfl_xor_sync(0xffffffffu, n_below, o);
    }
}

template <bool MIN>
__device__ uint32_t block_reduce_u32(Smem &s, uint32_t v) {   // MIN ? min : sum
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = blockDim.x >> 5;
#pragma unroll
    for (int o = 16; o; o >>= 1) {
        uint32_t t = __shfl_xor_sync(0xffffffffu, v, o);
        v = MIN ? min(v, t) : v + t;
    }
    if (lane == 0) s.red_u[warp] = v;
    __syncthreads();
    v = MIN ? 0xFFFFFFFFu : 0u;
    for (int w = 0; w < nw; ++w) v = MIN ? min(v, s.red_u[w]) : v + s.red_u[w];
    __syncthreads();
    return v;
}

// exclusive block scan of v; returns this thread's offset, total in `total`
__device__ uint32_t block_scan_excl(Smem &s, uint32_t v, uint32_t &total) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = blockDim.x >> 5;
    uint32_t incl = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        uint32_t t = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += t;
    }
    if (lane == 31) s.red_u[warp] = incl;
    __syncthreads();
    uint32_t base = 0;
    total = 0;
    for (int w = 0; w < nw; ++w) { if (w < warp) base += s.red_u[w]; total += s.red_u[w]; }
    __syncthreads();
    return base + incl - v;
}

// in-place ascending bitonic sort of a[0..n), n a power of two; all threads of the CTA call it
__device__ void bitonic_sort(uint32_t *a, int n) {
    for (int k = 2; k <= n; k <<= 1) {
        for (int j = k >> 1; j > 0; j >>= 1) {
            for (int t = threadIdx.x; t < (n >> 1); t += blockDim.x) {
                const int i = ((t & ~(j - 1)) << 1) | (t & (j - 1));   // index with bit j clear
                const int p = i | j;
                const uint32_t x = a[i], y = a[p];
                const bool up = (i & k) == 0;
                if ((x > y) == up) { a[i] = y; a[p] = x; }
            }
            __syncthreads();
        }
    }
}

// reduce the per-thread byte columns hist8[bin][thread] to per-bin totals out[bin] (needs nt % 64 == 0)
__device__ void reduce_byte_hist(const uint8_t *hist8, int nt, uint32_t *out) {
    const int tid = threadIdx.x;
    const int G = nt / K1_NBIN, b = tid / G, g = tid - b * G;   // G threads per bin, nt/4 words per bin
    const uint32_t *row = reinterpret_cast<const uint32_t *>(hist8) + (size_t)b * (nt / 4);
    uint32_t acc = 0;
#pragma unroll
    for (int j = 0; j < 16; ++j) acc = __dp4a(row[j * G + g], 0x01010101u, acc);
    for (int o = G >> 1; o; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    if (g == 0) out[b] = acc;
}

// Which bin of cnt[0..64) holds 0-based rank r (r < sum cnt)?  Every warp computes it redundantly (lane l owns
// bins 2l, 2l+1).  Returns false if r is not covered.  `excl0`/`c0`/`c1` are left for prefix queries.
struct BinHit { uint32_t b, pre, cnt; uint32_t excl, c0, c1; };
__device__ bool locate_bin(const uint32_t *cnt, uint32_t r, BinHit &h) {
    const int lane = threadIdx.x & 31;
    const uint32_t c0 = cnt[2 * lane], c1 = cnt[2 * lane + 1];
    uint32_t incl = c0 + c1;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        uint32_t t = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += t;
    }
    const uint32_t excl = incl - c0 - c1;
    const bool mine0 = r >= excl && r < excl + c0, mine1 = r >= excl + c0 && r < incl;
    const uint32_t bal = __ballot_sync(0xffffffffu, mine0 || mine1);
    h.excl = excl; h.c0 = c0; h.c1 = c1;
    if (bal == 0) return false;
    const int src = __ffs(bal) - 1;
    h.b = __shfl_sync(0xffffffffu, 2 * lane + (mine1 ? 1 : 0), src);
    h.pre = __shfl_sync(0xffffffffu, mine1 ? excl + c0 : excl, src);
    h.cnt = __shfl_sync(0xffffffffu, mine1 ? c1 : c0, src);
    return true;
}
// exclusive prefix of bin b, from the registers locate_bin left
__device__ __forceinline__ uint32_t bin_prefix(const BinHit &h, uint32_t b) {
    const int lane = threadIdx.x & 31;
    return __shfl_sync(0xffffffffu, (b & 1) ? h.excl + h.c0 : h.excl, (int)(b >> 1));
}

// thread 0: grow a window of bins around b while it holds <= K1_LISTCAP pixels
__device__ void grow_window(Smem &s, const uint32_t *cnt, int nb, uint32_t b, uint32_t cntb, uint32_t cap) {
    int b0 = (int)b, b1 = (int)b;
    uint32_t tot = cntb;
    // later rounds clip mostly positive outliers (sources, hot pixels), which moves the median rank DOWN:
    // two bins on the low side for every bin on the high side
    for (int g = 0; g < K1_NBIN; ++g) {
        bool grew = false;
        for (int rep = 0; rep < 2; ++rep)
            if (b0 - 1 >= 0 && tot + cnt[b0 - 1] <= cap) { --b0; tot += cnt[b0]; grew = true; }
        if (b1 + 1 < nb && tot + cnt[b1 + 1] <= cap) { ++b1; tot += cnt[b1]; grew = true; }
        if (!grew) break;
    }
    s.win_b0 = b0; s.win_b1 = b1;
}

// Counting sort of the candidate keys list[0..m) (all in [kga, kga + gspan]) into sorted[0..m): K1_FB fine bins
// by key, shared-memory atomics on m <= 2048 elements only, then an insertion sort inside the (tiny) bins that
// hold more than one key.  fcur is scratch [K1_FB].
#ifndef K1_FB_DIV
#define K1_FB_DIV 1
#endif
// fine bins of the counting sort: listcap / K1_FB_DIV are used.  The per-bin insertion sort (one thread per bin) was
// 15 k cycles per mesh with 4-6 keys per bin; with as many bins as candidates it is ~1.4 keys per bin on continuous
// data, and bins of equal keys (integer-valued frames) are skipped
struct SortArea {   // carved from a dead region of shared memory: 2 * listcap words
    uint32_t *sorted;   // [listcap]
    uint32_t *fcur;     // [listcap]
};
__device__ __forceinline__ uint32_t k1_listcap() { return blockDim.x >= 512 ? (uint32_t)K1_LISTCAP : 2048u; }
__device__ __forceinline__ SortArea make_sort_area(void *base) {
    SortArea a;
    a.sorted = reinterpret_cast<uint32_t *>(base);
    a.fcur = a.sorted + k1_listcap();   // [listcap] fine-bin cursors
    return a;
}
__device__ void sort_candidates(Smem &s, const uint32_t *list, uint32_t m, uint32_t kga, uint32_t gspan, const SortArea &srt) {
    const int tid = threadIdx.x, nt = blockDim.x, lane = tid & 31;
#ifdef K1_TIMING
    long long c_ = clock64();
#define K1_TS(i) do { if (tid == 0) { const long long t_ = clock64(); atomicAdd(&g_k1_t[i], (unsigned long long)(t_ - c_)); c_ = t_; } } while (0)
#else
#define K1_TS(i) do { } while (0)
#endif
    int fshift = 0;
    while ((gspan >> fshift) >= k1_listcap() / K1_FB_DIV) ++fshift;
    const int nfb = (int)(gspan >> fshift) + 1;
    for (int i = tid; i < nfb; i += nt) srt.fcur[i] = 0;
    __syncthreads();
    K1_TS(11);
    for (uint32_t i = tid; i < m; i += nt) atomicAdd(&srt.fcur[(list[i] - kga) >> fshift], 1u);
    __syncthreads();
    K1_TS(12);
    {   // exclusive scan of fcur[0..nfb), in place
        const int per = (nfb + nt - 1) / nt, f0 = tid * per;
        uint32_t local = 0;
        for (int k = 0; k < per; ++k) if (f0 + k < nfb) local += srt.fcur[f0 + k];
        uint32_t inc = local;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            uint32_t t = __shfl_up_sync(0xffffffffu, inc, o);
            if (lane >= o) inc += t;
        }
        if (lane == 31) s.red_u[tid >> 5] = inc;
        __syncthreads();
        uint32_t run = inc - local;
        for (int w = 0; w < (tid >> 5); ++w) run += s.red_u[w];
        for (int k = 0; k < per; ++k) {
            if (f0 + k >= nfb) break;
            const uint32_t c = srt.fcur[f0 + k];
            srt.fcur[f0 + k] = run;
            run += c;
        }
    }
    __syncthreads();
    K1_TS(13);
    for (uint32_t i = tid; i < m; i += nt) {
        const uint32_t k = list[i];
        srt.sorted[atomicAdd(&srt.fcur[(k - kga) >> fshift], 1u)] = k;
    }
    __syncthreads();
    K1_TS(14);
    if (fshift > 0) {   // fcur[f] is now the end of bin f = the start of bin f + 1
        for (int f = tid; f < nfb; f += nt) {
            const uint32_t lo = f ? srt.fcur[f - 1] : 0u, hi = srt.fcur[f];
            if (hi - lo < 2) continue;
            if (hi - lo > 4) {   // a bin of equal keys (integer-valued frames: hundreds of copies) needs no sorting
                uint32_t kmin = 0xFFFFFFFFu, kmax = 0;
                for (uint32_t i = lo; i < hi; ++i) { const uint32_t k = srt.sorted[i]; kmin = min(kmin, k); kmax = max(kmax, k); }
                if (kmin == kmax) continue;
            }
            for (uint32_t i = lo + 1; i < hi; ++i) {
                const uint32_t k = srt.sorted[i];
                uint32_t j = i;
                while (j > lo && srt.sorted[j - 1] > k) { srt.sorted[j] = srt.sorted[j - 1]; --j; }
                srt.sorted[j] = k;
            }
        }
        __syncthreads();
    }
    K1_TS(15);
}

// ---- pixel source of the slow path: the slab in shared memory (C = 1) or the mesh in global memory ---------
struct MeshSrc {
    const float *slab;   // non-null: n_slab valid pixels packed (TMA rows are full width, so packed) in shared memory
    int n_slab;
    const float *g;      // else: top-left pixel of the mesh in global memory, row pitch W
    int W, vh, vw;
    bool vec4;           // rows of g are 16-byte aligned and vw % 4 == 0
    const uint8_t *bad;  // non-null (then slab is null): mask of the mesh, same geometry as g; masked pixels are skipped
};

// Apply f(float) to every pixel of the mesh.  The assignment of pixels to threads is the same on every call
// (the per-thread byte histograms rely on that).
template <typename F>
__device__ __forceinline__ void for_each_px(const MeshSrc &m, F f) {
    const int tid = threadIdx.x, nt = blockDim.x;
    if (m.slab) {
        const float4 *s4 = reinterpret_cast<const float4 *>(m.slab);
        const int n4 = m.n_slab >> 2, n_tail = m.n_slab & 3;
        for (int i = tid; i < n4; i += nt) {
            const float4 v = s4[i];
            f(v.x); f(v.y); f(v.z); f(v.w);
        }
        if (tid < n_tail) f(m.slab[(n4 << 2) + tid]);
    } else {
        if (m.vec4) {   // thread t owns the 128-bit words t, t + nt, ... of the mesh; 4 loads in flight
            const int f4_row = m.vw >> 2, n_f4 = m.vh * f4_row;
            const int dr = nt / f4_row, dc = nt - dr * f4_row;
            for (int i0 = tid; i0 < n_f4; i0 += nt * 4) {
                float4 v[4];
                const float4 *pv[4];
                int r = i0 / f4_row, c = i0 - r * f4_row;
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    pv[k] = reinterpret_cast<const float4 *>(m.g + (size_t)r * m.W) + c;
                    if (i0 + k * nt < n_f4) v[k] = __ldg(pv[k]);
                    r += dr; c += dc;
                    if (c >= f4_row) { c -= f4_row; ++r; }
                }
#pragma unroll
                for (int k = 0; k < 4; ++k)
                    if (i0 + k * nt < n_f4) {
                        if (m.bad) {   // 4 mask bytes of the same 4 pixels (the mask has the frame's geometry)
                            const size_t off = reinterpret_cast<const float *>(pv[k]) - m.g;
                            const uint32_t mb = __ldg(reinterpret_cast<const uint32_t *>(m.bad + off));
                            if (!(mb & 0x000000FFu)) f(v[k].x);
                            if (!(mb & 0x0000FF00u)) f(v[k].y);
                            if (!(mb & 0x00FF0000u)) f(v[k].z);
                            if (!(mb & 0xFF000000u)) f(v[k].w);
                        } else { f(v[k].x); f(v[k].y); f(v[k].z); f(v[k].w); }
                    }
            }
        } else {
            const int lane = tid & 31, warp = tid >> 5, nw = nt >> 5;
            for (int r = warp; r < m.vh; r += nw) {
                const float *row = m.g + (size_t)r * m.W;
                const uint8_t *brow = m.bad ? m.bad + (size_t)r * m.W : nullptr;
                for (int c = lane; c < m.vw; c += 32)
                    if (!brow || !__ldg(brow + c)) f(__ldg(row + c));
            }
        }
    }
}

// ---- slow path: one CTA, general -------------------------------------------------------------------------
// Leaves the final statistics of the survivors in med/mu/sd/n.
__device__ __noinline__ void k1_slow_path(const MeshSrc &src, Smem &s, int &ph, uint8_t *hist8, int n_tot, double k_c, int iters,
                                          double &med, double &mu, double &sd, int &n_out, int &n_valid_out) {
    const int tid = threadIdx.x, nt = blockDim.x;
    const SortArea srt = make_sort_area(hist8);
    const uint32_t listcap = k1_listcap();
    // pivot of the round-0 sums: any pixel of the mesh would do for correctness; take the mean of a few
    double pivot;
    {
        double t1 = 0;
        int c = 0, z = 0;
        double z2 = 0;
        for_each_px(src, [&](float e) { t1 += (double)e; ++c; });
        block_reduce_stats(s, ph, t1, z2, c, z);
        n_tot = c;   // with a bad-pixel mask: the pixels that are left (B1)
        if (n_tot == 0) { n_out = 0; n_valid_out = 0; return; }
        pivot = t1 / (double)n_tot;
    }
    n_valid_out = n_tot;
    double s1, s2;
    {
        double t1 = 0, t2 = 0;
        int z0 = 0, z1 = 0;
        for_each_px(src, [&](float e) { const double d = (double)e - pivot; t1 += d; t2 = fma(d, d, t2); });
        block_reduce_stats(s, ph, t1, t2, z0, z1);
        s1 = t1; s2 = t2;
    }

    int mode = 0;                                   // 0 none, 1 sorted list, 2 single key
    uint32_t list_off = 0, list_m = 0;              // mode 1: ranks [list_off, list_off + list_m) are srt.sorted[]
    uint32_t sel_key = 0, sel_lo = 0, sel_hi = 0;   // mode 2: ranks [sel_lo, sel_hi) all have key sel_key

    // Build the window for 0-based rank `want` of the whole mesh, searching keys [ka, kb] (must contain it).
    auto build = [&](uint32_t want, uint32_t ka, uint32_t kb) {
        uint32_t off = 0;
        bool top = true;
        for (;;) {
            const uint32_t span = kb - ka;
            int shift = 0;
            while ((span >> shift) >= (uint32_t)K1_NBIN) ++shift;
            for (int i = tid; i < (K1_NBIN * nt) / 16; i += nt) reinterpret_cast<uint4 *>(hist8)[i] = make_uint4(0, 0, 0, 0);
            __syncthreads();
            uint32_t below = 0;
            uint8_t *col = hist8 + tid;
            for_each_px(src, [&](float e) {
                const uint32_t k = f32_to_key(e);
                const uint32_t t = k - ka;
                if (t <= span) col[(t >> shift) * nt] += 1;
                else if (top && k < ka) ++below;
            });
            __syncthreads();
            reduce_byte_hist(hist8, nt, s.tot.cnt);
            if (top) { below = block_reduce_u32<false>(s, below); off = below; }
            else __syncthreads();
            top = false;
            BinHit h;
            if (!locate_bin(s.tot.cnt, want - off, h)) {   // cannot happen for a range that brackets the rank
                ka = 0; kb = 0xFFFFFFFFu; off = 0; top = true;
                __syncthreads();
                continue;
            }
            if (shift == 0) {   // the bin is a single key
                mode = 2; sel_key = ka + h.b; sel_lo = off + h.pre; sel_hi = sel_lo + h.cnt;
                __syncthreads();
                return;
            }
            if (h.cnt > (uint32_t)K1_T1) {   // descend
                off += h.pre;
                ka = ka + (h.b << shift);
                kb = min(kb, ka + ((1u << shift) - 1u));
                __syncthreads();
                continue;
            }
            if (tid == 0) grow_window(s, s.tot.cnt, (int)(span >> shift) + 1, h.b, h.cnt, listcap);
            __syncthreads();
            const uint32_t b0 = s.win_b0, b1 = s.win_b1;
            const uint32_t pre0 = bin_prefix(h, b0);
            const uint32_t kga = ka + (b0 << shift);
            const uint32_t kgb = min(kb, ka + (((b1 + 1) << shift) - 1u));
            uint32_t mycnt = 0;
            for (uint32_t bb = b0; bb <= b1; ++bb) mycnt += col[bb * nt];
            uint32_t m;
            uint32_t pos = block_scan_excl(s, mycnt, m);
            const uint32_t gspan = kgb - kga;
            for_each_px(src, [&](float e) {
                const uint32_t k = f32_to_key(e);
                if (k - kga <= gspan) s.list[pos++] = k;
            });
            __syncthreads();
            sort_candidates(s, s.list, m, kga, gspan, srt);   // the histogram is dead: the sort arrays alias it
            mode = 1; list_off = off + pre0; list_m = m;
            return;
        }
    };

    // smallest key strictly greater than `key` in the mesh (only asked when one exists)
    auto next_key = [&](uint32_t key) -> uint32_t {
        uint32_t best = 0xFFFFFFFFu;
        for_each_px(src, [&](float e) { const uint32_t k = f32_to_key(e); if (k > key) best = min(best, k); });
        return block_reduce_u32<true>(s, best);
    };

    double LO = -INFINITY, HI = INFINITY;
    int n = n_tot, n_below = 0;
    for (int round = 0;; ++round) {
        const double inv_n = 1.0 / (double)n;
        const double m1 = s1 * inv_n;
        mu = pivot + m1;
        const double var = s2 * inv_n - m1 * m1;
        sd = var > 0.0 ? sqrt(var) : 0.0;
        const uint32_t k0 = (uint32_t)(n_below + (n - 1) / 2);
        const bool two = (n & 1) == 0;
        uint32_t key_a, key_b;
        for (;;) {
            if (mode == 2 && k0 >= sel_lo && k0 < sel_hi) {
                key_a = sel_key;
                key_b = (!two || k0 + 1 < sel_hi) ? sel_key : next_key(sel_key);
                break;
            }
            if (mode == 1 && k0 >= list_off && k0 < list_off + list_m) {
                const uint32_t j = k0 - list_off;
                key_a = srt.sorted[j];
                key_b = !two ? key_a : (j + 1 < list_m ? srt.sorted[j + 1] : next_key(key_a));
                break;
            }
            // the median of a set lies within one population standard deviation of its mean
            const double w = sd * (1.0 + 1e-9) + 1e-300;
            const uint32_t ka = f32_to_key(__double2float_rd(mu - w)), kb = f32_to_key(__double2float_ru(mu + w));
            __syncthreads();
            build(k0, ka, kb);
        }
        med = 0.5 * ((double)key_to_f32(key_a) + (double)key_to_f32(key_b));
        if (round >= iters) break;
        const double lo = fmax(LO, med - k_c * sd), hi = fmin(HI, med + k_c * sd);
        // survivors of [lo, hi]; sums about the new pivot (= current median: inside the surviving interval, so
        // the one-pass variance loses no digits -- and is exactly 0 when all survivors are equal)
        double t1 = 0, t2 = 0;
        int c_in = 0, c_below = 0;
        for_each_px(src, [&](float e) {
            const double x = (double)e;
            if (x < lo) ++c_below;
            else if (x <= hi) {
                const double d = x - med;
                ++c_in;
                t1 += d;
                t2 = fma(d, d, t2);
            }
        });
        block_reduce_stats(s, ph, t1, t2, c_in, c_below);
        if (c_in == n || c_in == 0) break;   // stable (A7) or would empty the set: keep the current statistics
        LO = lo; HI = hi;
        n = c_in; n_below = c_below; s1 = t1; s2 = t2;
        pivot = med;
    }
    n_out = n;
}

// 8 x 8 lattice points x 4 consecutive pixels of the mesh rows [row0, row0 + rows), read from global memory by one warp,
// sorted in its registers, left in samp[0..256).  Not inlined: its registers must not count against the sweeps'.
__device__ __noinline__ void k1_sample_sort_warp(const float *mesh_ptr, int W, int row0, int rows, int vw, uint32_t *samp) {
    const int lane = threadIdx.x & 31;
    uint32_t xs[8];
#pragma unroll
    for (int r = 0; r < 8; ++r) {
        const int e = r * 32 + lane, pt = e >> 2, q = e & 3, i = pt >> 3, j = pt & 7;
        const int y = row0 + ((2 * i + 1) * rows) / 16;
        const int x = min((((2 * j + 1) * vw) / 16) & ~3, vw - 4) + q;
        xs[r] = f32_to_key(__ldg(mesh_ptr + (size_t)y * W + x));
    }
    kw_sort256(xs, lane);
#pragma unroll
    for (int r = 0; r < 8; ++r) samp[lane * 8 + r] = xs[r];
    __syncwarp();
}

// ---- the kernel ------------------------------------------------------------------------------------------
template <int C, bool LIST>
#ifndef K1_MINB
#define K1_MINB 2
#endif
#ifndef K1_U
#define K1_U 4
#endif
__global__ void __launch_bounds__(C == 1 ? 512 : 1024, C == 1 ? K1_MINB : 1) k1_mesh_stats(const __grid_constant__ CUtensorMap tmap, K1Args a) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    float *slab = reinterpret_cast<float *>(smem_raw);   // [slab_rows * mw], 128-B aligned for TMA
    const size_t slab_bytes = (size_t)a.slab_bytes;
    Smem &s = *reinterpret_cast<Smem *>(smem_raw + slab_bytes);
    unsigned char *area = smem_raw + slab_bytes + k1_smem_fixed_bytes((int)blockDim.x);
    uint8_t *hist8 = area;                                  // [K1_NBIN][nt] byte counters
    uint32_t *samp = reinterpret_cast<uint32_t *>(area);    // sample keys (before the histogram)
    float *tail = reinterpret_cast<float *>(area);          // tail pixels (after the histogram)

    const unsigned rank = Team<C>::rank();
    int ph = 0;   // call counter of block_reduce_stats
    unsigned it = blockIdx.x / C;
    [[maybe_unused]] const unsigned n_work = LIST ? *a.list_count : 0u;
    do {   // one pass, except in list mode (C == 1): grid-stride over the worklist
    if constexpr (LIST) { if (it >= n_work) break; }
    const int mesh = LIST ? (int)a.list[it] : (int)it;
    const int frame = mesh / (a.ny * a.nx);
    const int mj = (mesh / a.nx) % a.ny, mi = mesh % a.nx;
    const int y0 = mj * a.mh, x0 = mi * a.mw;
    const int vh = min(a.mh, a.H - y0), vw = min(a.mw, a.W - x0);       // valid part of the mesh
    const int row0 = (int)rank * a.slab_rows;                           // first mesh row of this CTA's slab
    const int my_rows = max(0, min(a.slab_rows, vh - row0));
    const int n_c = my_rows * vw;                                       // valid pixels in this slab, a prefix
    const int n_tot = vh * vw;
    const float *mesh_ptr = a.img + (size_t)frame * a.H * a.W + (size_t)y0 * a.W + x0;
    const int tid = threadIdx.x, nt = blockDim.x;
#ifdef K1_TIMING
    long long t_prev = clock64();
#endif

    // ---- stage the slab ---------------------------------------------------------------------------------
    const bool stream = C == 1 && (a.stream || a.bad);   // with a mask every sweep reads global memory (general path)
    const bool tma = a.use_tma && vw == a.mw && !stream;
    if (tma && tid == 0) {
        uint32_t bar = smem_u32(&s.mbar);
        asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(bar));
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        uint32_t bytes = (uint32_t)((size_t)a.slab_rows * a.mw * sizeof(float));
        asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
        // rows past H are zero-filled by TMA; they lie beyond the n_c prefix and are never read
        asm volatile(
            "cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes"
            " [%0], [%1, {%2, %3, %4}], [%5];" ::"r"(smem_u32(slab)),
            "l"(&tmap), "r"(x0), "r"(y0 + row0), "r"(frame), "r"(bar)
            : "memory");
    }

    // ---- lattice sample of this CTA's slab rows (read from global while the TMA load is in flight), sorted ---
    bool fast = a.allow_fast && !a.bad && n_tot >= K1_FAST_MIN_PX && vw >= 16;
    constexpr int M_S = 256, G_S = 8;   // 8 x 8 lattice points x 4 consecutive pixels
    if (fast && my_rows > 0) {
        if constexpr (C == 1) {   // one warp sorts the sample in registers: no block barrier (the CTA-wide bitonic sort
            if (tid < 32) k1_sample_sort_warp(mesh_ptr, a.W, row0, my_rows, vw, samp);   // of 256 keys was 36 barriers, 8.5 k cycles)
        } else {
            for (int e = tid; e < M_S; e += nt) {
                const int pt = e >> 2, q = e & 3;
                const int i = pt / G_S, j = pt - i * G_S;
                const int y = row0 + ((2 * i + 1) * my_rows) / (2 * G_S);
                const int x = min((((2 * j + 1) * vw) / (2 * G_S)) & ~3, vw - 4) + q;
                samp[e] = f32_to_key(__ldg(mesh_ptr + (size_t)y * a.W + x));
            }
            __syncthreads();
            K1_T(0);
            bitonic_sort(samp, M_S);
        }
        K1_T(1);
    }
    // sample quantiles, averaged over the team -> pivot, core interval [A, B], median bracket [ka, kb]
    double pivot = 0.0;
    float A_f = 0.f, B_f = 0.f;
    uint32_t ka = 0, kb = 0;
    if (fast) {
        if (tid == 0) {
            s.sx.valid = my_rows > 0 ? 1 : 0;
            if (my_rows > 0) {
                s.sx.q50 = (double)key_to_f32(samp[M_S / 2]);
                s.sx.q16 = (double)key_to_f32(samp[(M_S * 16) / 100]);
                s.sx.ka = samp[M_S / 2 - 48];   // +-6 standard deviations of a 256-sample quantile near 0.5
                s.sx.kb = samp[M_S / 2 + 48];
                s.sx.lo3 = (double)key_to_f32(samp[M_S / 2 - 24]);
                s.sx.hi3 = (double)key_to_f32(samp[M_S / 2 + 24]);
            }
        }
        Team<C>::sync();   // #0 (a plain barrier when C = 1)
        double q50 = 0, q16 = 0, lo3 = 0, hi3 = 0;
        int nv = 0;
        ka = 0xFFFFFFFFu; kb = 0;
        for (unsigned r = 0; r < (unsigned)C; ++r) {   // rank order: the same bits on every CTA
            const SampleX *o = Team<C>::remote(&s.sx, r);
            if (!o->valid) continue;
            ++nv; q50 += o->q50; q16 += o->q16; lo3 += o->lo3; hi3 += o->hi3; ka = min(ka, o->ka); kb = max(kb, o->kb);
        }
        q50 /= (double)nv; q16 /= (double)nv;
        if (nv >= 4) {   // the average of >= 4 independent 3-sigma quantiles is a 6-sigma bracket, half as wide
            ka = f32_to_key(__double2float_rd(lo3 / (double)nv));
            kb = f32_to_key(__double2float_ru(hi3 / (double)nv));
        }
        const double sig = q50 - q16;                 // lower side: sources and hot pixels are positive
        const double c = nv >= 4 ? 2.2 : 2.0;         // the averaged estimate is less noisy
        pivot = q50;
        A_f = (float)(pivot - c * sig);
        B_f = (float)(pivot + c * sig);
        if (!(sig > 0.0) || ka >= kb || !((double)A_f < pivot) || !((double)B_f > pivot)) {
            fast = false;
            if (tid == 0 && rank == 0) atomicAdd(&g_k1_reason[1], 1ull);
        }
    }
    __syncthreads();   // the sample is dead: the work area becomes the byte histogram

    K1_T(2);
    if (tma) {
        uint32_t bar = smem_u32(&s.mbar), done = 0;
        while (!done) {
            asm volatile(
                "{ .reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], 0; selp.u32 %0, 1, 0, p; }"
                : "=r"(done)
                : "r"(bar)
                : "memory");
        }
    } else if (!stream && (C == 1 || fast)) {   // plain loader: valid pixels packed row-major
        for (int i = tid; i < n_c; i += nt) {
            int r = i / vw, c = i - r * vw;
            slab[i] = mesh_ptr[(size_t)(row0 + r) * a.W + c];
        }
        __syncthreads();
    }

    const float4 *slab4 = reinterpret_cast<const float4 *>(slab);
    const int n4 = n_c >> 2, n_tail4 = n_c & 3;
#define K1_SWEEP(BODY)                                                    \
    {                                                                     \
        for (int i_ = tid; i_ < n4; i_ += nt) {                           \
            const float4 v_ = slab4[i_];                                  \
            { const float e = v_.x; BODY }                                \
            { const float e = v_.y; BODY }                                \
            { const float e = v_.z; BODY }                                \
            { const float e = v_.w; BODY }                                \
        }                                                                 \
        if (tid < n_tail4) { const float e = slab[(n4 << 2) + tid]; BODY }\
    }

    // The same sweep over global memory (stream mode): thread t owns the 128-bit words t, t + nt, ... of the mesh,
    // 8 loads in flight.  The assignment of pixels to threads is the same on every sweep.
    const int f4_row = vw >> 2, n_f4 = vh * f4_row;
#define K1_SWEEP_G(BODY)                                                                          \
    {                                                                                             \
        const int dr_ = nt / f4_row, dc_ = nt - dr_ * f4_row;                                     \
        for (int i0_ = tid; i0_ < n_f4; i0_ += nt * K1_U) {                                          \
            float4 v_[K1_U];                                                                         \
            int r_ = i0_ / f4_row, c_ = i0_ - r_ * f4_row;                                        \
            _Pragma("unroll") for (int k_ = 0; k_ < K1_U; ++k_) {                                    \
                if (i0_ + k_ * nt < n_f4)                                                         \
                    v_[k_] = __ldg(reinterpret_cast<const float4 *>(mesh_ptr + (size_t)r_ * a.W) + c_); \
                r_ += dr_; c_ += dc_;                                                             \
                if (c_ >= f4_row) { c_ -= f4_row; ++r_; }                                         \
            }                                                                                     \
            _Pragma("unroll") for (int k_ = 0; k_ < K1_U; ++k_) {                                    \
                if (i0_ + k_ * nt < n_f4) {                                                       \
                    { const float e = v_[k_].x; BODY }                                            \
                    { const float e = v_[k_].y; BODY }                                            \
                    { const float e = v_[k_].z; BODY }                                            \
                    { const float e = v_[k_].w; BODY }                                            \
                }                                                                                 \
            }                                                                                     \
        }                                                                                         \
    }
#define K1_SWEEP_ANY(BODY)                      \
    {                                           \
        if (stream) K1_SWEEP_G(BODY)            \
        else K1_SWEEP(BODY)                     \
    }

    double med = 0, mu = 0, sd = 0;
    int n_final = n_tot, n_valid = n_tot;
    bool done_fast = false;
    bool slab_dirty = false;   // the fast path reuses the slab for its sort arrays

    if (fast) {
        // ---- sweep 1: core sums, tail count, bracket histogram ---------------------------------------------
        const uint32_t span = kb - ka;
        const int shift = max(0, 26 - __clz(span));   // smallest shift with (span >> shift) < K1_NBIN = 64
        for (int i = tid; i < (K1_NBIN * nt) / 16; i += nt) reinterpret_cast<uint4 *>(hist8)[i] = make_uint4(0, 0, 0, 0);
        __syncthreads();
        double t1 = 0, t2 = 0;
        int c_core = 0, c_tail = 0;
        uint32_t below = 0;
        uint8_t *col = hist8 + tid;
        K1_T(3);
        const uint32_t col_s = smem_u32(col);
        // A bracket of non-negative floats (every sky level): key - ka = bits - bits(ka) for the pixels that can fall into
        // it, a negative pixel's difference exceeds any span (bits >= 2^31 > bits(kb)), and "below the bracket" is a
        // signed compare of the raw bits -- the order-preserving key (3 instructions per pixel) is not needed.
        const bool pos = ka >= 0x80000000u;
        const uint32_t ka_bits = ka ^ 0x80000000u;
        if (pos) {
            K1_SWEEP_ANY({
                const uint32_t bits = __float_as_uint(e);
                k1_hist_inc(col_s, bits - ka_bits, span, shift, nt);
                below += (int)bits < (int)ka_bits ? 1u : 0u;
                const double d = (double)e - pivot;
                if (e >= A_f && e <= B_f) {
                    t1 += d;
                    t2 = fma(d, d, t2);
                    ++c_core;
                }
            })
        } else {
            K1_SWEEP_ANY({
                const uint32_t k = f32_to_key(e);
                k1_hist_inc(col_s, k - ka, span, shift, nt);
                below += k < ka ? 1u : 0u;
                const double d = (double)e - pivot;
                if (e >= A_f && e <= B_f) {
                    t1 += d;
                    t2 = fma(d, d, t2);
                    ++c_core;
                }
            })
        }
        {   // pixels this thread swept (the assignment of K1_SWEEP / K1_SWEEP_G): the tail count needs no counter of its own
            const int my_px = stream ? (tid < n_f4 ? ((n_f4 - tid + nt - 1) / nt) * 4 : 0)
                                     : (tid < n4 ? ((n4 - tid + nt - 1) / nt) * 4 : 0) + (tid < n_tail4 ? 1 : 0);
            c_tail = my_px - c_core;
        }
        __syncthreads();
        reduce_byte_hist(hist8, nt, s.xch.cnt);
        below = block_reduce_u32<false>(s, below);
        {
            int ct = c_tail;
            block_reduce_stats(s, ph, t1, t2, c_core, ct);
            if (tid == 0) { s.xch.s1 = t1; s.xch.s2 = t2; s.xch.n_core = c_core; s.xch.n_tail = ct; s.xch.below = below; }
        }
        K1_T(4);
        Team<C>::sync();   // #1: every CTA's xch is published
        K1_T(5);
        if (tid == 0) {
            double q1 = 0, q2 = 0;
            int nc = 0, ntl = 0;
            uint32_t bl = 0;
            for (unsigned r = 0; r < (unsigned)C; ++r) {   // rank order: every CTA computes the same bits
                const Xch *o = Team<C>::remote(&s.xch, r);
                q1 += o->s1; q2 += o->s2; nc += o->n_core; ntl += o->n_tail; bl += o->below;
            }
            s.tot.s1 = q1; s.tot.s2 = q2; s.tot.n_core = nc; s.tot.n_tail = ntl; s.tot.below = bl;
        }
        if (tid >= 32 && tid < 32 + K1_NBIN) {
            const int b = tid - 32;
            uint32_t t = 0;
            for (unsigned r = 0; r < (unsigned)C; ++r) t += Team<C>::remote(&s.xch, r)->cnt[b];
            s.tot.cnt[b] = t;
        }
        __syncthreads();
        const double s1c = s.tot.s1, s2c = s.tot.s2;
        const int n_core = s.tot.n_core, n_tail_tot = s.tot.n_tail;
        const uint32_t off = s.tot.below;
        // ---- window of bins around the round-0 median rank ----------------------------------------------
        const uint32_t k_first = (uint32_t)((n_tot - 1) / 2);
        BinHit h;
        bool ok = n_tail_tot <= a.tailcap && n_core > 0 && k_first >= off;
        ok = locate_bin(s.tot.cnt, k_first - off, h) && ok;   // (all lanes run the shuffles)
        if (tid == 0 && rank == 0) {
            if (!(n_tail_tot <= a.tailcap)) atomicAdd(&g_k1_reason[2], 1ull);
            else if (!ok) atomicAdd(&g_k1_reason[3], 1ull);
            else if (h.cnt > k1_listcap()) atomicAdd(&g_k1_reason[4], 1ull);
        }
        ok = ok && h.cnt <= k1_listcap();
        uint32_t m_tot = 0, list_off = 0, kga = 0, gspan = 0;
        if (ok) {
            if (tid == 0) grow_window(s, s.tot.cnt, (int)(span >> shift) + 1, h.b, h.cnt, k1_listcap());
            __syncthreads();
            const uint32_t b0 = s.win_b0, b1 = s.win_b1;
            list_off = off + bin_prefix(h, b0);
            kga = ka + (b0 << shift);
            const uint32_t kgb = min(kb, ka + (((b1 + 1) << shift) - 1u));
            gspan = kgb - kga;
            // ---- sweep 2: gather window candidates and tail pixels ---------------------------------------
            uint32_t mycnt = 0;
            for (uint32_t bb = b0; bb <= b1; ++bb) mycnt += col[bb * nt];
            uint32_t packed_tot;
            const uint32_t packed = block_scan_excl(s, mycnt | ((uint32_t)c_tail << 16), packed_tot);
            uint32_t pos_c = packed & 0xFFFFu, pos_t = packed >> 16;   // (the scan's barriers: histogram is dead)
            K1_T(6);
            uint32_t addr_c = smem_u32(&s.list[pos_c]), addr_t = smem_u32(&tail[pos_t]);
            if (pos) {   // (kga >= ka: the window is a bracket of non-negative floats too)
                const uint32_t kga_bits = kga ^ 0x80000000u;
                K1_SWEEP_ANY({
                    const uint32_t bits = __float_as_uint(e);
                    k1_push_u32_if_le(addr_c, bits - kga_bits, gspan, bits ^ 0x80000000u);
                    k1_push_f32_if_outside(addr_t, e, A_f, B_f);
                })
            } else {
                K1_SWEEP_ANY({
                    k1_push_u32_if_le(addr_c, f32_to_key(e) - kga, gspan, f32_to_key(e));
                    k1_push_f32_if_outside(addr_t, e, A_f, B_f);
                })
            }
            if (tid == 0) { s.xch.m_cand = packed_tot & 0xFFFFu; s.xch.m_tail = packed_tot >> 16; }
        }
        K1_T(7);
        Team<C>::sync();   // #2: lists published (or: everybody is done reading the peers' xch)
        if (!ok) {
            fast = false;
        } else {
            m_tot = s.xch.m_cand;
            uint32_t mt_tot = s.xch.m_tail;
            if constexpr (C > 1) {
                if (rank == 0) {
                    for (unsigned r = 1; r < (unsigned)C; ++r) {
                        const Xch *o = Team<C>::remote(&s.xch, r);
                        const uint32_t mr = o->m_cand, tr = o->m_tail;
                        const uint32_t *lsrc = Team<C>::remote(s.list, r);
                        const float *tsrc = Team<C>::remote(tail, r);
                        for (uint32_t i = tid; i < mr; i += nt) s.list[m_tot + i] = lsrc[i];
                        for (uint32_t i = tid; i < tr; i += nt) tail[mt_tot + i] = tsrc[i];
                        m_tot += mr; mt_tot += tr;
                    }
                }
                Team<C>::sync();   // #3: rank 0 has copied; peers may leave
                if (rank != 0) return;
            }
            __syncthreads();
            const SortArea srt = make_sort_area(slab);   // the slab is dead from here on
            slab_dirty = true;
            K1_T(8);
            sort_candidates(s, s.list, m_tot, kga, gspan, srt);
            K1_T(9);
            // ---- clipping rounds on the tail list (all warps: with two CTAs per SM a round run by one warp alone leaves the
            //      SM idle -- measured 0.51 ms against 0.33 ms; one barrier per round, see block_reduce_stats) ------------
            const double A_d = (double)A_f, B_d = (double)B_f;
            auto tail_stats = [&](double lo, double hi, double &q1, double &q2, int &c_in, int &c_below) {
                q1 = 0; q2 = 0; c_in = 0; c_below = 0;
                for (uint32_t i = tid; i < mt_tot; i += nt) {
                    const double x = (double)tail[i];
                    if (x < lo) ++c_below;
                    else if (x <= hi) {
                        const double d = x - pivot;
                        ++c_in;
                        q1 += d;
                        q2 = fma(d, d, q2);
                    }
                }
                block_reduce_stats(s, ph, q1, q2, c_in, c_below);
            };
            double LO = -INFINITY, HI = INFINITY, q1, q2;
            int c_in, c_below;
            tail_stats(LO, HI, q1, q2, c_in, c_below);
            int n = n_core + c_in, n_below = c_below;
            double s1 = s1c + q1, s2 = s2c + q2;
            done_fast = true;
            for (int round = 0;; ++round) {
                const double inv_n = 1.0 / (double)n;
                const double m1 = s1 * inv_n;
                mu = pivot + m1;
                const double var = s2 * inv_n - m1 * m1;
                sd = var > 0.0 ? sqrt(var) : 0.0;
                const uint32_t k0 = (uint32_t)(n_below + (n - 1) / 2);
                const bool two = (n & 1) == 0;
                if (k0 < list_off || k0 + (two ? 1u : 0u) >= list_off + m_tot) {
                    done_fast = false;
                    if (tid == 0) atomicAdd(&g_k1_reason[5], 1ull);
                    break;
                }
                const uint32_t j = k0 - list_off;
                const uint32_t key_a = srt.sorted[j], key_b = two ? srt.sorted[j + 1] : key_a;
                med = 0.5 * ((double)key_to_f32(key_a) + (double)key_to_f32(key_b));
                n_final = n;
                if (round >= a.iters) break;
                const double lo = fmax(LO, med - a.k_c * sd), hi = fmin(HI, med + a.k_c * sd);
                if (!(lo <= A_d && hi >= B_d)) {   // a bound entered the core
                    done_fast = false;
                    if (tid == 0) atomicAdd(&g_k1_reason[6], 1ull);
                    break;
                }
                tail_stats(lo, hi, q1, q2, c_in, c_below);
                const int n_new = n_core + c_in;
                if (n_new == n) break;   // stable (A7); n_new > 0 because the core survives
                LO = lo; HI = hi;
                n = n_new; n_below = c_below; s1 = s1c + q1; s2 = s2c + q2;
            }
        }
    }
#undef K1_SWEEP_ANY
#undef K1_SWEEP_G
#undef K1_SWEEP
    if constexpr (C > 1) {
        if (!fast) {   // nothing was exchanged yet (or everybody passed #2): the peers have no further part
            if (rank != 0) return;
        }
    }

    if (!done_fast) {
        if (tid == 0) atomicAdd(&g_k1_slow_meshes, 1ull);
        MeshSrc src;
        src.slab = (C == 1 && !slab_dirty && !stream) ? slab : nullptr;
        src.n_slab = n_c;
        src.g = mesh_ptr; src.W = a.W; src.vh = vh; src.vw = vw;
        src.bad = a.bad ? a.bad + (mesh_ptr - a.img) : nullptr;
        src.vec4 = (vw % 4 == 0) && (a.mw % 4 == 0) && (a.W % 4 == 0);
        __syncthreads();
        k1_slow_path(src, s, ph, hist8, n_tot, a.k_c, a.iters, med, mu, sd, n_final, n_valid);
    }

    K1_T(10);
    if (tid == 0) {
        double bkg = a.median_factor * med - a.mean_factor * mu;
        if (a.skew_guard) {
            if (sd == 0.0) bkg = mu;
            else if (fabs(mu - med) / sd >= 0.3) bkg = med;
        }
        // B2, B6: too few valid pixels, too much of the mesh masked, or too much of it rejected -> invalid (NaN)
        const int n_px = vh * vw;
        if (n_valid < 1 || n_valid < a.min_valid || (double)(n_px - n_valid) > a.max_masked_frac * (double)n_px ||
            (double)(n_valid - n_final) > a.max_reject_frac * (double)n_valid) {
            const double nan = __longlong_as_double(0x7FF8000000000000ll);
            bkg = nan; sd = nan; med = nan; mu = nan; n_final = 0;
        }
        if (a.bkg_raw) a.bkg_raw[mesh] = bkg;
        if (a.rms_raw) a.rms_raw[mesh] = sd;
        if (a.median) a.median[mesh] = med;
        if (a.mean) a.mean[mesh] = mu;
        if (a.n_kept) a.n_kept[mesh] = n_final;
        if (a.n_valid) a.n_valid[mesh] = n_valid;
    }
    if constexpr (LIST) { __syncthreads(); it += gridDim.x; }   // the next mesh reuses the shared memory
    else break;
    } while (true);
}

#include "k1w_warp_mesh.cuh"

}  // namespace

// ---- host side ------------------------------------------------------------------------------------------
static size_t k1_smem_bytes(int slab_rows, int mw, int threads) {
    size_t area = (size_t)K1_NBIN * threads;   // byte histograms; also holds the sample (<= 4 KiB) and the tails,
    const size_t sort_bytes = 2 * (size_t)(threads >= 512 ? K1_LISTCAP : 2048) * sizeof(uint32_t);
    if (area < sort_bytes) area = sort_bytes;   // and the general path's sort arrays
    return bd_align_up((size_t)slab_rows * mw * sizeof(float), 128) + k1_smem_fixed_bytes(threads) + area + 128;
}

// what one thread of a lone CTA sees of the whole mesh when it walks it row by row in global memory (slow path)
static size_t k1_rowwalk_per_thread(int mesh_h, int mesh_w, int threads) {
    const int nw = threads / 32;
    const size_t rows_w = (size_t)(mesh_h + nw - 1) / nw;
    if (mesh_w % 4 == 0) return ((size_t)mesh_h * (mesh_w / 4) + threads - 1) / threads * 4;   // flattened 128-bit words
    return rows_w * (size_t)((mesh_w + 31) / 32);
}

int k1_plan(const bd_ctx *ctx, int mesh_h, int mesh_w, K1Plan *plan) {
#ifndef K1_SOFT_KB
#define K1_SOFT_KB 48
#endif
    const size_t soft = K1_SOFT_KB * 1024;
    plan->stream = 0;
    // (1) The mesh fits one CTA's slab (<= 48 KiB; a 64 KiB slab leaves room for one CTA per SM only and was 30 % slower
    //     than stream mode on 128x128 meshes): slab mode, one TMA load, every sweep in shared memory.
    // (2) Larger meshes with mesh_w % 4 == 0: stream mode -- one CTA per mesh, no slab; the two sweeps of the fast
    //     path read global memory (the second one from L2) with 8 x 128-bit loads in flight per thread.  (The first
    //     version gave such a mesh to a cluster of 4 CTAs with DSMEM exchanges: 570 us on config 3, two thirds of
    //     the instructions being per-mesh overhead replicated in every CTA, and rank 0 finishing alone.)
    // (3) Otherwise: a cluster of 2..8 CTAs, each with a slab of rows (plain loader), slabs up to the opt-in limit.
    const size_t mesh_bytes = (size_t)mesh_h * mesh_w * sizeof(float);
    if (mesh_bytes > soft && mesh_w % 4 == 0) {
        for (int threads = 512; threads <= 512; threads *= 2) {
            const size_t n_f4 = (size_t)mesh_h * (mesh_w / 4);
            size_t per_thread = (n_f4 + threads - 1) / threads * 4;
            const size_t walk = k1_rowwalk_per_thread(mesh_h, mesh_w, threads);
            if (walk > per_thread) per_thread = walk;
            const size_t slab_bytes = bd_align_up(2 * K1_LISTCAP * sizeof(uint32_t), 128);   // sort arrays
            const size_t area = 56 * 1024;   // byte histograms (32 KiB), then up to 14336 tail pixels
            const size_t smem = slab_bytes + k1_smem_fixed_bytes(threads) + area + 128;
            if (per_thread <= 255 && smem <= ctx->smem_optin) {
                plan->cluster = 1;
                plan->slab_rows = mesh_h;
                plan->smem_bytes = smem;
                plan->slab_bytes = slab_bytes;
                plan->threads = threads;
                plan->tailcap = (int)(area / sizeof(float));
                plan->use_tma = 0;
                plan->stream = 1;
                return BD_OK;
            }
        }
    }
    for (int pass = 0; pass < 2; ++pass) {
        for (int c = 1; c <= K1_MAXC; c *= 2) {
            int rows = (mesh_h + c - 1) / c;
            size_t px = (size_t)rows * mesh_w;
            size_t slab = px * sizeof(float);
#ifndef K1_SMALL_NT
#define K1_SMALL_NT 128
#endif
            int threads = px >= 16384 ? 512 : (px > 4096 ? 256 : K1_SMALL_NT);   // small meshes: more, smaller CTAs per SM
            size_t smem = k1_smem_bytes(rows, mesh_w, threads);
            bool ok = pass == 0 ? slab <= soft : true;
            // byte counters: what one thread can see of (a) its slab, (b) the whole mesh read from global
            // memory by a lone CTA (slow path of a team), must stay <= 255 per bin
            size_t per_thread = px / threads + 5;
            const size_t walk = k1_rowwalk_per_thread(mesh_h, mesh_w, threads);
            if (walk > per_thread) per_thread = walk;
            if (ok && smem <= ctx->smem_optin && per_thread <= 255) {
                plan->cluster = c;
                plan->slab_rows = rows;
                plan->smem_bytes = smem;
                plan->slab_bytes = bd_align_up((size_t)rows * mesh_w * sizeof(float), 128);
                plan->threads = threads;
                plan->tailcap = K1_NBIN * threads / 4;
                plan->use_tma = (mesh_w % 4 == 0 && mesh_w <= 256 && rows <= 256) ? 1 : 0;
                return BD_OK;
            }
        }
    }
    return BD_EUNSUPPORTED;
}

template <int C, bool LIST = false>
static cudaError_t k1_launch_c(const CUtensorMap &tmap, const K1Args &a, const K1Plan &plan, int n_ctas, cudaStream_t st) {
    const int n_mesh = n_ctas;
    cudaError_t e = cudaFuncSetAttribute(k1_mesh_stats<C, LIST>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)plan.smem_bytes);
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(k1_mesh_stats<C, LIST>, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
    if (e != cudaSuccess) return e;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)n_mesh * C);
    cfg.blockDim = dim3(plan.threads);
    cfg.dynamicSmemBytes = plan.smem_bytes;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = C;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = C > 1 ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, k1_mesh_stats<C, LIST>, tmap, a);
}

size_t k1_workspace_bytes(int B, int ny, int nx) { return 256 + (size_t)B * ny * nx * sizeof(uint32_t); }

int k1_launch(bd_ctx *ctx, const float *d_img, int B, int H, int W, const bd_bkg_params *p, double *d_bkg_raw,
              double *d_rms_raw, double *d_median, double *d_mean, int32_t *d_n_kept, void *d_ws, cudaStream_t st,
              const uint8_t *d_bad, const bd_bkgx_params *px, int32_t *d_n_valid) {
    K1Plan plan;
    int rc = k1_plan(ctx, p->mesh_h, p->mesh_w, &plan);
    if (rc != BD_OK) return bd_set_error(ctx, rc, "mesh %dx%d is too large for the statistics kernel", p->mesh_h, p->mesh_w);
    K1Args a;
    a.img = d_img; a.B = B; a.H = H; a.W = W; a.mh = p->mesh_h; a.mw = p->mesh_w;
    a.ny = (H + a.mh - 1) / a.mh; a.nx = (W + a.mw - 1) / a.mw;
    a.slab_rows = plan.slab_rows; a.use_tma = plan.use_tma; a.tailcap = plan.tailcap;
    a.stream = plan.stream; a.slab_bytes = (int)plan.slab_bytes;
    a.allow_fast = ctx->k1_force_slow ? 0 : 1;
    a.k_c = p->clip_sigma; a.iters = p->clip_iters; a.skew_guard = p->skew_guard;
    a.median_factor = p->median_factor; a.mean_factor = p->mean_factor;
    a.bkg_raw = d_bkg_raw; a.rms_raw = d_rms_raw; a.median = d_median; a.mean = d_mean; a.n_kept = d_n_kept;
    a.list_count = nullptr; a.list = nullptr;
    const bool variants = d_bad || px;   // mask or validity rules: every mesh takes the general path
    a.bad = d_bad; a.n_valid = d_n_valid;
    a.min_valid = px ? px->min_valid_px : 0;
    a.max_masked_frac = px ? px->max_masked_frac : 1.0;
    a.max_reject_frac = px ? px->max_reject_frac : 1.0;
    if (d_bad) { a.allow_fast = 0; a.use_tma = 0; plan.use_tma = 0; }
    const int n_mesh = B * a.ny * a.nx;

    // Small meshes (the paper's default 64x64 and anything else up to 4096 pixels with mesh_w % 4 == 0): one warp per mesh
    // (k1w_warp_mesh.cuh); the meshes it cannot finish go through the general path of k1_mesh_stats<1> in list mode.
    const bool warp_mode = !variants && a.allow_fast && p->mesh_w % 4 == 0 && (long long)p->mesh_h * p->mesh_w <= 4096 &&
                           (long long)p->mesh_h * p->mesh_w >= KW_MIN_PX && p->mesh_w >= 16 && plan.cluster == 1 && d_ws;
    if (warp_mode) {
        K1WArgs w;
        w.img = d_img; w.B = B; w.H = H; w.W = W; w.mh = a.mh; w.mw = a.mw; w.ny = a.ny; w.nx = a.nx;
        w.use_tma = (ctx->encode_tiled && a.mw <= 256 && a.mh <= 256) ? 1 : 0;
        w.k_c = a.k_c; w.iters = a.iters; w.skew_guard = a.skew_guard; w.median_factor = a.median_factor; w.mean_factor = a.mean_factor;
        w.bkg_raw = d_bkg_raw; w.rms_raw = d_rms_raw; w.median = d_median; w.mean = d_mean; w.n_kept = d_n_kept;
        w.fb_count = (uint32_t *)d_ws; w.fb_list = (uint32_t *)((char *)d_ws + 256);
        CUtensorMap tm;
        memset(&tm, 0, sizeof(tm));
        if (w.use_tma) {
            cuuint64_t dims[3] = {(cuuint64_t)W, (cuuint64_t)H, (cuuint64_t)B};
            cuuint64_t strides[2] = {(cuuint64_t)W * sizeof(float), (cuuint64_t)W * H * sizeof(float)};
            cuuint32_t box[3] = {(cuuint32_t)a.mw, (cuuint32_t)a.mh, 1};
            cuuint32_t estr[3] = {1, 1, 1};
            CUresult r = ctx->encode_tiled(&tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, (void *)d_img, dims, strides, box, estr,
                                           CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                                           CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
            if (r != CUDA_SUCCESS) return bd_set_error(ctx, BD_ECUDA, "cuTensorMapEncodeTiled failed (%d)", (int)r);
        }
        BD_CUDA_CHECK(ctx, cudaMemsetAsync(w.fb_count, 0, sizeof(uint32_t), st));
        BD_CUDA_CHECK(ctx, cudaFuncSetAttribute(k1w_warp_mesh, cudaFuncAttributeMaxDynamicSharedMemorySize, KW_SMEM));
        BD_CUDA_CHECK(ctx, cudaFuncSetAttribute(k1w_warp_mesh, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared));
        k1w_warp_mesh<<<(unsigned)n_mesh, 32, KW_SMEM, st>>>(tm, w);
        BD_CUDA_CHECK(ctx, cudaGetLastError());
        // the leftovers: general path, slab filled by the plain loader, a few persistent CTAs over the worklist
        a.allow_fast = 0; a.use_tma = 0;
        a.list_count = w.fb_count; a.list = w.fb_list;
        plan.use_tma = 0;
        CUtensorMap none;
        memset(&none, 0, sizeof(none));
        const int n_ctas = n_mesh < ctx->num_sms * 2 ? n_mesh : ctx->num_sms * 2;
        BD_CUDA_CHECK(ctx, (k1_launch_c<1, true>(none, a, plan, n_ctas, st)));
        return BD_OK;
    }

    CUtensorMap tmap;
    memset(&tmap, 0, sizeof(tmap));
    if (plan.use_tma) {
        if (!ctx->encode_tiled) return bd_set_error(ctx, BD_ECUDA, "cuTensorMapEncodeTiled entry point unavailable");
        cuuint64_t dims[3] = {(cuuint64_t)W, (cuuint64_t)H, (cuuint64_t)B};
        cuuint64_t strides[2] = {(cuuint64_t)W * sizeof(float), (cuuint64_t)W * H * sizeof(float)};
        cuuint32_t box[3] = {(cuuint32_t)a.mw, (cuuint32_t)plan.slab_rows, 1};
        cuuint32_t estr[3] = {1, 1, 1};
        CUresult r = ctx->encode_tiled(&tmap, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, (void *)d_img, dims, strides, box, estr,
                                       CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                                       CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (r != CUDA_SUCCESS) return bd_set_error(ctx, BD_ECUDA, "cuTensorMapEncodeTiled failed (%d)", (int)r);
    }
    cudaError_t e;
    switch (plan.cluster) {
        case 1: e = k1_launch_c<1>(tmap, a, plan, n_mesh, st); break;
        case 2: e = k1_launch_c<2>(tmap, a, plan, n_mesh, st); break;
        case 4: e = k1_launch_c<4>(tmap, a, plan, n_mesh, st); break;
        default: e = k1_launch_c<8>(tmap, a, plan, n_mesh, st); break;
    }
    BD_CUDA_CHECK(ctx, e);
    return BD_OK;
}

// diagnostics (not part of include/bkgdet.h): number of meshes that took the slow path since the last reset
extern "C" int bd_debug_k1_slow_meshes(unsigned long long *out, int reset) {
    unsigned long long v = 0, z = 0;
    if (cudaMemcpyFromSymbol(&v, g_k1_slow_meshes, sizeof(v)) != cudaSuccess) return BD_ECUDA;
    if (reset && cudaMemcpyToSymbol(g_k1_slow_meshes, &z, sizeof(z)) != cudaSuccess) return BD_ECUDA;
    if (out) *out = v;
    return BD_OK;
}
extern "C" int bd_debug_k1_reasons(unsigned long long *out8, int reset) {
    unsigned long long z[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    if (cudaMemcpyFromSymbol(out8, g_k1_reason, sizeof(z)) != cudaSuccess) return BD_ECUDA;
    if (reset && cudaMemcpyToSymbol(g_k1_reason, z, sizeof(z)) != cudaSuccess) return BD_ECUDA;
    return BD_OK;
}
// diagnostics: force every mesh through the slow path (tests exercise both)
extern "C" int bd_debug_k1_force_slow(bd_ctx *ctx, int on) {
    if (!ctx) return BD_EINVAL;
    ctx->k1_force_slow = on ? 1 : 0;
    return BD_OK;
}

#ifdef K1_TIMING
extern "C" int bd_debug_k1_timing(unsigned long long *out16, int reset) {
    unsigned long long z[16] = {0};
    if (cudaMemcpyFromSymbol(out16, g_k1_t, sizeof(z)) != cudaSuccess) return BD_ECUDA;
    if (reset && cudaMemcpyToSymbol(g_k1_t, z, sizeof(z)) != cudaSuccess) return BD_ECUDA;
    return BD_OK;
}
#endif
