// K9: multi-threshold deblending of the source candidates.
// PAPER.md:155 ("calculate multi-level deblending thresholds.  At each threshold level, the algorithm re-evaluates
// objects and splits them as necessary, constructing a binary tree structure rooted in the original source candidate ...
// traversed from bottom to top ... pruning ... based on rigorous intensity and spatial criteria", one candidate per
// thread block).  The paper gives no constants or formulas: readings D1-D8.
//
// The paper re-labels a candidate at every level.  Here a candidate is labelled ONCE, incrementally: its pixels are
// counting-sorted by their level (the highest threshold they exceed) and the levels are walked from the top threshold
// down with one union-find that only ever grows (union by minimum index, so a root is its component's first pixel in
// raster order, which is the label the definition gives the node).  Walking the levels downwards IS the bottom-to-top
// traversal of the tree: when a level has been united, the roots that lost their root status during it are exactly the
// children that merged, so every node's decision (D5) is taken from per-root counters the moment its level is complete:
//   st[r]   = number of objects node r resolves into (0: the component is not a node, fewer than min_area pixels);
//   T[R]   += st[c] for a child that resolves into >= 2, += 1 for a single child with flux > min_cont * candidate flux;
//   st[R]   = max(T[R], 1): T[R] >= 2 means the node splits, and its single significant children are final objects
//             ("frozen": frz[child root] = the child's level).
// The work per level is proportional to the pixels that enter at that level plus the roots that merge, not to the
// candidate.  Candidates that resolve into one object (nearly all) end there.  For the others a second walk repeats the
// unions and, at every level that holds a frozen node, hands the node's pixels their object; the remaining pixels join by
// synchronous growth (D7) driven by a frontier list (only the unassigned neighbours of the pixels assigned in the last
// round are looked at); a last raster pass over the box writes the new labels (1 + minimum raster index of the object,
// D8) and reduces the objects' records (npix, flux, moments, peak, bbox: the quantities of step a5) with a segmented
// warp reduction and one set of atomics per (warp, object).
// Five tiers run the same code, chosen by the cells of the candidate's bounding box plus a one-pixel border: <= 112 and
// <= 256 cells: one WARP's job with every array in shared memory (32 resp. 16 warps per SM); <= 1536 and <= 5120: one
// thread block, arrays in shared memory; larger boxes: one thread block, arrays in the workspace, indexed by frame
// coordinates (candidates are disjoint, so the frame-sized arrays serve all of
// them at once and cannot overflow).  Label maps are bit-exact by construction; node fluxes are float64 atomics (order
// dependent in the last bits: decisions within 1e-9 of the contrast limit may differ from the definition).
#include <limits.h>

#include "common.cuh"

namespace {

typedef unsigned long long u64;

#include "kept_rank.cuh"

constexpr int DB_MAXT = 64;            // n_thresh <= 64
constexpr int CAP_TINY = 112, CAP_WARP = 256, CAP_MID = 1536, CAP_BIG = 5120;   // pixels of the box and its border per tier
constexpr int WARPS_PER_CTA = 8;
constexpr int T_QUEUED = 0x40000000, T_SELFSIG = 0x20000000, T_SUM = 0x1FFFFFFF;

struct ORec {   // 96 bytes: one object of a split candidate; sums are about the object's key pixel
    double f, sx, sy, sxx, syy, sxy;
    u64 peak;          // (ordered key of sub << 32) | (0xFFFFFFFF - raster index in frame)
    int32_t key;       // raster index (in the frame) of the first pixel of the object's node
    int32_t frame;
    int32_t npix;
    int32_t xmin, xmax, ymin, ymax;
    int32_t omin;      // minimum raster index of the object's pixels: label - 1
    int32_t pad[2];
};
static_assert(sizeof(ORec) == 96, "ORec must be 96 bytes");

// counters[] slots
enum { C_TIER0 = 0 /* 5 tiers */, C_CUR0 = 8, C_POOL = 16, C_SEG = 18 /* u64: [18], [19] */, C_NCOUNT = 64 };
constexpr int N_TIERS = 5;   // 0 tiny warp, 1 warp, 2 mid block, 3 big block, 4 workspace

struct DbWs {
    uint32_t *counters;
    int32_t *lists;        // [N_TIERS][cap_in]
    uint8_t *state;        // [cap_in] 1 = the candidate was split (its record is replaced by pool records)
    uint32_t *keptbits, *blkcnt, *blkprefix;
    ORec *pool;            // [cap_out]
    // global tier, frame-sized
    int32_t *par, *accn, *st, *T, *obj, *order, *lost, *touched;
    double *accf;
    int8_t *lvl;
    uint8_t *frz;
    size_t P, NWk, NB, zero_bytes, total;
};

size_t carve(DbWs &w, void *base, int B, int H, int W, int64_t cap_in, int64_t cap_out) {
    const size_t P = (size_t)B * H * W;
    w.P = P;
    w.NWk = (P + 31) / 32 + 32;
    w.NB = (P + 4095) / 4096;
    size_t off = 0;
    auto take = [&](size_t bytes) { size_t o = off; off = bd_align_up(off + bytes, 256); return (char *)base + o; };
    w.counters = (uint32_t *)take(C_NCOUNT * sizeof(uint32_t));
    w.keptbits = (uint32_t *)take(w.NWk * sizeof(uint32_t));
    w.blkcnt = (uint32_t *)take((w.NB + 8) * sizeof(uint32_t));
    w.zero_bytes = (size_t)((char *)w.blkcnt - (char *)w.counters) + (w.NB + 1) * sizeof(uint32_t);
    w.blkprefix = (uint32_t *)take((w.NB + 8) * sizeof(uint32_t));
    w.lists = (int32_t *)take(5 * (size_t)cap_in * sizeof(int32_t));
    w.state = (uint8_t *)take((size_t)cap_in);
    w.pool = (ORec *)take((size_t)cap_out * sizeof(ORec));
    w.par = (int32_t *)take(P * 4); w.accn = (int32_t *)take(P * 4); w.st = (int32_t *)take(P * 4); w.T = (int32_t *)take(P * 4);
    w.obj = (int32_t *)take(P * 4); w.order = (int32_t *)take(P * 4); w.lost = (int32_t *)take(P * 4); w.touched = (int32_t *)take(P * 4);
    w.accf = (double *)take(P * 8);
    w.lvl = (int8_t *)take(P); w.frz = (uint8_t *)take(P);
    w.total = off;
    return off;
}

struct DbArgs {
    const float *sub, *rms;
    int32_t *labels;
    const bd_source *cat;
    const int64_t *n_in;
    int64_t cap_in, cap_out;
    int B, H, W;
    float kf;            // detect_k as the float32 the mask used
    int min_area, nthr, log2n;
    double min_cont;
    DbWs w;
};

__device__ __forceinline__ long long db_total(const DbArgs &a) {
    long long t = 0;
    for (int f = 0; f < a.B; ++f) t += a.n_in[f];
    return t < a.cap_in ? t : a.cap_in;
}

__device__ __forceinline__ void mark_kept(const DbWs &w, size_t g) {
    atomicOr(&w.keptbits[g >> 5], 1u << (g & 31));
    atomicAdd(&w.blkcnt[g >> RB_SHIFT], 1u);
}

// D2: t_0 of a candidate = (float32 k) * (float32 rms at its peak pixel), an exact float64 product
__device__ __forceinline__ double cand_t0(const DbArgs &a, const bd_source &s) {
    const float r = __ldg(a.rms + (size_t)s.frame * a.H * a.W + (size_t)s.ypeak * a.W + s.xpeak);
    return __dmul_rn((double)a.kf, (double)r);
}

// ------------------------------------------------------------------------------------------------ classify
__global__ void __launch_bounds__(256) k9_classify(DbArgs a) {
    const long long total = db_total(a);
    const size_t HW = (size_t)a.H * a.W;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (long long)gridDim.x * blockDim.x) {
        const bd_source s = a.cat[i];
        const double t0 = cand_t0(a, s);
        a.w.state[i] = 0;
        // D2: not deblended (or too small to hold two nodes; or a box beyond the 15 + 16 bits of a packed (row, column) entry,
        // which no frame with H * W < 2^31 and a sane aspect ratio produces)
        if (!((double)s.peak > t0) || s.npix < 2 * max(a.min_area, 1) || s.xmax - s.xmin >= 65535 || s.ymax - s.ymin >= 32767) {
            mark_kept(a.w, (size_t)s.frame * HW + (size_t)(s.label - 1));
            continue;
        }
        const long long area = (long long)(s.xmax - s.xmin + 3) * (s.ymax - s.ymin + 3);   // the box and its one-pixel border
        const int tier = area <= CAP_TINY ? 0 : area <= CAP_WARP ? 1 : area <= CAP_MID ? 2 : area <= CAP_BIG ? 3 : 4;
        // one atomic per (warp, tier) instead of one per candidate on four hot counters
        const uint32_t peers = __match_any_sync(__activemask(), tier);
        const int leader = __ffs(peers) - 1;
        uint32_t base = 0;
        if ((int)(threadIdx.x & 31) == leader) base = atomicAdd(&a.w.counters[C_TIER0 + tier], (uint32_t)__popc(peers));
        base = __shfl_sync(peers, base, leader);
        const uint32_t k = base + (uint32_t)__popc(peers & ((1u << (threadIdx.x & 31)) - 1u));
        a.w.lists[(size_t)tier * a.cap_in + k] = (int32_t)i;
    }
}

// ------------------------------------------------------------------------------------------------ one candidate
struct DbCtl {   // per group (warp or block), shared memory
    double t[DB_MAXT];
    int hist[DB_MAXT], start[DB_MAXT], cur[DB_MAXT];
    u64 frzmask;
    int n_lost, n_old, n_touched, n_f[2], nslot, item, pool_base, pool_ok;
    long long seg;
};

struct DbArr {
    int32_t *par, *accn, *st, *T, *obj, *order, *lost, *touched;
    double *accf;
    int8_t *lvl;
    uint8_t *frz;
};

struct WarpGroup {
    int lane;
    __device__ __forceinline__ int tid() const { return lane; }
    __device__ __forceinline__ int size() const { return 32; }
    __device__ __forceinline__ void sync() const { __syncwarp(); }
    __device__ __forceinline__ int warp() const { return 0; }
    __device__ __forceinline__ int nwarps() const { return 1; }
};
struct BlockGroup {
    __device__ __forceinline__ int tid() const { return threadIdx.x; }
    __device__ __forceinline__ int size() const { return blockDim.x; }
    __device__ __forceinline__ void sync() const { __syncthreads(); }
    __device__ __forceinline__ int warp() const { return threadIdx.x >> 5; }
    __device__ __forceinline__ int nwarps() const { return blockDim.x >> 5; }
};

// loads of arrays other threads of the group update with atomics: past L1 in the global tier
template <bool GL, class T>
__device__ __forceinline__ T ldv(const T *p) {
    if (GL) return __ldcg(p);
    return *p;
}

template <bool GL>
struct Geo {
    int L, x0, y0, bw, bh, W, pitch, base;
    const float *sub;        // this frame
    const int32_t *lab;      // this frame
    __device__ __forceinline__ void coords(int a, int &ly, int &lx) const { const int rel = a - base; ly = rel / pitch; lx = rel - ly * pitch; }
    __device__ __forceinline__ int fidx(int ly, int lx) const { return (y0 + ly) * W + x0 + lx; }
    __device__ __forceinline__ int aidx(int ly, int lx) const { return base + ly * pitch + lx; }
};

template <bool GL>
__device__ __forceinline__ bool db_member(const Geo<GL> &g, const DbArr &A, int q) {
    if (GL) return g.lab[q] == g.L;
    return A.lvl[q] >= 0;
}
template <bool GL>
__device__ __forceinline__ bool db_active(const Geo<GL> &g, const DbArr &A, int q, int level) {
    if (GL) return g.lab[q] == g.L && A.lvl[q] >= level;
    return A.lvl[q] >= level;
}

template <bool GL>
__device__ __forceinline__ int db_find(int32_t *par, int x) {
    int p = ldv<GL>(par + x);
    while (p != x) {
        const int gp = ldv<GL>(par + p);
        if (gp != p) par[x] = gp;   // path halving (a non-root only ever moves towards its root)
        x = p;
        p = gp;
    }
    return x;
}

// union by minimum index; a root that is hooked goes into the lost list (exactly once in its life)
template <bool GL, bool TRACK>
__device__ __forceinline__ void db_unite(int32_t *par, int a, int b, int32_t *lost, int *n_lost, const int8_t *lvl, int level, int *n_old) {
    while (true) {
        a = db_find<GL>(par, a);
        b = db_find<GL>(par, b);
        if (a == b) return;
        if (a < b) { const int t = a; a = b; b = t; }
        const int old = atomicCAS(&par[a], a, b);
        if (old == a) {
            if (TRACK) {
                lost[atomicAdd(n_lost, 1)] = a;
                if (lvl[a] > level) atomicAdd(n_old, 1);   // a component of the level above merges: a tree decision is due
            }
            return;
        }
        a = old;
    }
}


// the 8 neighbours of pixel p = (ly, lx): f(q, dy, dx)
template <bool GL, class F>
__device__ __forceinline__ void db_for_neighbours(const Geo<GL> &geo, int p, int ly, int lx, F f) {
#pragma unroll
    for (int dy = -1; dy <= 1; ++dy) {
        if (GL && (ly + dy < 0 || ly + dy >= geo.bh)) continue;
#pragma unroll
        for (int dx = -1; dx <= 1; ++dx) {
            if (dy == 0 && dx == 0) continue;
            if (GL && (lx + dx < 0 || lx + dx >= geo.bw)) continue;
            f(p + dy * geo.pitch + dx, dy, dx);
        }
    }
}
// an entry of the level-sorted list: (row << 16) | column of the box; -> array index
template <bool GL>
__device__ __forceinline__ int db_entry(const Geo<GL> &geo, int packed, int &ly, int &lx) {
    ly = packed >> 16; lx = packed & 0xFFFF;
    return geo.aidx(ly, lx);
}

template <bool GL, bool TRACK, class G>
__device__ __forceinline__ void db_unite_level(const G &g, const Geo<GL> &geo, const DbArr &A, DbCtl *C, int level, int beg, int end) {
    for (int k = beg + g.tid(); k < end; k += g.size()) {
        int ly, lx;
        const int p = db_entry<GL>(geo, A.order[k], ly, lx);
        db_for_neighbours<GL>(geo, p, ly, lx, [&](int q, int, int) {
            if (db_active<GL>(geo, A, q, level)) db_unite<GL, TRACK>(A.par, p, q, A.lost, &C->n_lost, A.lvl, level, &C->n_old);
        });
    }
}

__device__ __forceinline__ int db_contrib(int st, double flux, double min_flux) {
    return st >= 2 ? st : (st == 1 && flux > min_flux ? 1 : 0);
}

// segmented warp reduction of one object's share of 32 consecutive box pixels
struct PixAcc {
    double f, sx, sy, sxx, syy, sxy;
    u64 peak;
    int npix, xmin, xmax, ymin, ymax, omin;
};
__device__ __forceinline__ void pix_reduce(PixAcc &v) {
#pragma unroll
    for (int o = 16; o; o >>= 1) {
        v.f += __shfl_xor_sync(0xffffffffu, v.f, o);
        v.sx += __shfl_xor_sync(0xffffffffu, v.sx, o);
        v.sy += __shfl_xor_sync(0xffffffffu, v.sy, o);
        v.sxx += __shfl_xor_sync(0xffffffffu, v.sxx, o);
        v.syy += __shfl_xor_sync(0xffffffffu, v.syy, o);
        v.sxy += __shfl_xor_sync(0xffffffffu, v.sxy, o);
        const u64 pk = __shfl_xor_sync(0xffffffffu, v.peak, o);
        v.peak = pk > v.peak ? pk : v.peak;
        v.npix += __shfl_xor_sync(0xffffffffu, v.npix, o);
        v.xmin = min(v.xmin, __shfl_xor_sync(0xffffffffu, v.xmin, o));
        v.xmax = max(v.xmax, __shfl_xor_sync(0xffffffffu, v.xmax, o));
        v.ymin = min(v.ymin, __shfl_xor_sync(0xffffffffu, v.ymin, o));
        v.ymax = max(v.ymax, __shfl_xor_sync(0xffffffffu, v.ymax, o));
        v.omin = min(v.omin, __shfl_xor_sync(0xffffffffu, v.omin, o));
    }
}

// Deblends candidate `ci`.  A: the group's arrays (shared memory, or the frame-sized workspace arrays offset to the
// candidate's frame).  Every thread of the group calls it with the same arguments.
template <bool GL, class G>
__device__ void db_candidate(const G &g, const DbArgs &a, const DbArr &A0, DbCtl *C, int ci) {
    const bd_source s = a.cat[ci];
    const int W = a.W;
    const size_t HW = (size_t)a.H * W;
    const size_t fo = (size_t)s.frame * HW;
    Geo<GL> geo;
    geo.L = s.label; geo.x0 = s.xmin; geo.y0 = s.ymin; geo.bw = s.xmax - s.xmin + 1; geo.bh = s.ymax - s.ymin + 1; geo.W = W;
    // shared tiers: the box sits inside a one-pixel border of inactive cells (lvl = -1), so the 8 neighbour tests of a
    // pixel need no bounds checks; workspace tier: frame coordinates, neighbours are tested against the box
    geo.pitch = GL ? W : geo.bw + 2;
    geo.base = GL ? s.ymin * W + s.xmin : geo.pitch + 1;
    geo.sub = a.sub + fo;
    geo.lab = a.labels + fo;
    int32_t *labels = a.labels + fo;
    const int nbox = geo.bw * geo.bh, nthr = a.nthr, min_area = a.min_area;
    const int tid = g.tid(), nt = g.size();
    DbArr A = A0;
    if (GL) {   // frame-sized arrays: this frame's part
        A.par += fo; A.accn += fo; A.st += fo; A.T += fo; A.obj += fo; A.accf += fo; A.lvl += fo; A.frz += fo;
    }

    // ---- thresholds (D2) and the list segment of the global tier ------------------------------------------------
    if (tid == 0) {
        const double t0 = cand_t0(a, s);
        double q = __ddiv_rn((double)s.peak, t0);
        for (int m = 0; m < a.log2n; ++m) q = __dsqrt_rn(q);
        C->t[0] = t0;
        for (int i = 1; i < nthr; ++i) C->t[i] = __dmul_rn(C->t[i - 1], q);
        C->frzmask = 0ull;
        C->nslot = 0;
        if (GL) C->seg = (long long)atomicAdd(reinterpret_cast<u64 *>(a.w.counters + C_SEG), (u64)s.npix);
    }
    for (int i = tid; i < DB_MAXT; i += nt) C->hist[i] = 0;
    g.sync();
    if (GL) { A.order += C->seg; A.lost += C->seg; A.touched += C->seg; }
    const double min_flux = __dmul_rn(a.min_cont, s.flux);   // D4 (the candidate's flux is the O6 flux of the record)

    // ---- levels of the member pixels, counting sort by level (descending) ---------------------------------------
    if (!GL) {   // the border of inactive cells: rows -1 and bh, columns -1 and bw
        for (int k = tid; k < geo.pitch; k += nt) { A.lvl[k] = -1; A.lvl[(geo.bh + 1) * geo.pitch + k] = -1; }
        for (int k = tid; k < geo.bh; k += nt) { A.lvl[(k + 1) * geo.pitch] = -1; A.lvl[(k + 1) * geo.pitch + geo.bw + 1] = -1; }
    }
    for (int k = tid; k < nbox; k += nt) {
        const int ly = k / geo.bw, lx = k - ly * geo.bw;
        const int f = geo.fidx(ly, lx), p = geo.aidx(ly, lx);
        if (labels[f] == geo.L) {
            const double v = (double)__ldg(geo.sub + f);
            int lo = 0;
#pragma unroll
            for (int step = DB_MAXT / 2; step; step >>= 1)
                if (lo + step < nthr && v > C->t[lo + step]) lo += step;
            A.lvl[p] = (int8_t)lo;
            A.frz[p] = 0;
            A.obj[p] = 0;
            atomicAdd(&C->hist[lo], 1);
        } else if (!GL) {
            A.lvl[p] = -1;
        }
    }
    g.sync();
    if (tid == 0) {
        int run = 0;
        for (int i = nthr - 1; i >= 0; --i) { C->start[i] = run; C->cur[i] = run; run += C->hist[i]; }
    }
    g.sync();
    for (int k = tid; k < nbox; k += nt) {
        const int ly = k / geo.bw, lx = k - ly * geo.bw;
        const int p = geo.aidx(ly, lx);
        const bool mem = GL ? labels[geo.fidx(ly, lx)] == geo.L : A.lvl[p] >= 0;
        if (mem) A.order[atomicAdd(&C->cur[A.lvl[p]], 1)] = (ly << 16) | lx;
    }
    g.sync();
    const int npix = C->start[0] + C->hist[0];

    // ---- pass 1: the tree decisions, from the top level down ------------------------------------------------------
    for (int i = nthr - 1; i >= 0; --i) {
        const int cnt = C->hist[i];
        if (!cnt) continue;
        const int beg = C->start[i], end = beg + cnt;
        for (int k = beg + tid; k < end; k += nt) {
            int ly, lx;
            const int p = db_entry<GL>(geo, A.order[k], ly, lx);
            A.par[p] = p;
            A.accn[p] = 1;
            A.accf[p] = (double)__ldg(geo.sub + geo.fidx(ly, lx));
            A.st[p] = min_area <= 1 ? 1 : 0;
            A.T[p] = 0;
        }
        if (tid == 0) { C->n_lost = 0; C->n_old = 0; C->n_touched = 0; }
        g.sync();
        db_unite_level<GL, true>(g, geo, A, C, i, beg, end);
        g.sync();
        const int nl = C->n_lost;
        if (nl == 0) {   // nothing merged: the new pixels are isolated at this level and finalised by their initialisation
            continue;
        }
        if (C->n_old == 0) {
            // Only pixels of this level were hooked: no component of the level above merged, so no node gains a child other
            // than its own former self and every st[] of a node stays what it was (T = the self contribution: st for a
            // split node, at most 1 otherwise).  What can change is that a component reaches min_area and becomes a node.
            for (int k = tid; k < nl; k += nt) {
                const int c = A.lost[k];
                const int R = db_find<GL>(A.par, c);
                atomicAdd(&A.accn[R], A.accn[c]);
                atomicAdd(&A.accf[R], A.accf[c]);
            }
            g.sync();
            for (int k = tid; k < nl; k += nt) {
                const int R = db_find<GL>(A.par, A.lost[k]);
                if (A.st[R] == 0 && ldv<GL>(A.accn + R) >= min_area) A.st[R] = 1;
            }
            g.sync();
            continue;
        }
        // children report to the root they ended under
        for (int k = tid; k < nl; k += nt) {
            const int c = A.lost[k];
            const int R = db_find<GL>(A.par, c);
            // (a pixel that entered at this very level was no component of the level above: it is no child)
            const int con = A.lvl[c] > i ? db_contrib(A.st[c], A.accf[c], min_flux) : 0;
            const int old = atomicOr(&A.T[R], T_QUEUED);
            if (!(old & T_QUEUED)) A.touched[atomicAdd(&C->n_touched, 1)] = R;
            if (con) atomicAdd(&A.T[R], con);
        }
        g.sync();
        const int ntc = C->n_touched;
        // a root that existed before this level is a child of its own new node
        for (int k = tid; k < ntc; k += nt) {
            const int R = A.touched[k];
            if (A.lvl[R] > i) {
                const int sr = A.st[R];
                const int t = ldv<GL>(A.T + R);
                if (sr >= 2) A.T[R] = t + sr;
                else if (sr == 1 && ldv<GL>(A.accf + R) > min_flux) A.T[R] = (t + 1) | T_SELFSIG;
            }
        }
        g.sync();
        for (int k = tid; k < nl; k += nt) {
            const int c = A.lost[k];
            const int R = db_find<GL>(A.par, c);
            atomicAdd(&A.accn[R], A.accn[c]);
            atomicAdd(&A.accf[R], A.accf[c]);
        }
        g.sync();
        for (int k = tid; k < ntc; k += nt) {
            const int R = A.touched[k];
            const int t = ldv<GL>(A.T + R);
            const int sum = t & T_SUM;
            const int ns = ldv<GL>(A.accn + R) >= min_area ? max(sum, 1) : 0;
            if (ns >= 2 && (t & T_SELFSIG)) {
                A.frz[R] = (uint8_t)(i + 1);
                atomicOr(&C->frzmask, 1ull << (i + 1));
            }
            A.st[R] = ns;
            A.T[R] = 0;
        }
        g.sync();
        for (int k = tid; k < nl; k += nt) {
            const int c = A.lost[k];
            if (A.lvl[c] > i && A.st[c] == 1 && A.accf[c] > min_flux) {
                const int R = db_find<GL>(A.par, c);
                if (A.st[R] >= 2) {
                    A.frz[c] = (uint8_t)(i + 1);
                    atomicOr(&C->frzmask, 1ull << (i + 1));
                }
            }
        }
        g.sync();
    }
    const int first = GL ? geo.L - 1 : geo.aidx((geo.L - 1) / W - geo.y0, (geo.L - 1) % W - geo.x0);
    const int nobj = A.st[first];
    if (nobj < 2) {   // D6: unchanged
        if (tid == 0) mark_kept(a.w, fo + (size_t)(geo.L - 1));
        g.sync();
        return;
    }

    // ---- pass 2: the pixels of the frozen nodes get their object (key = array index of the node's root + 1) --------
    const u64 fm = C->frzmask;
    const int jmin = __ffsll((long long)fm) - 1;
    for (int i = nthr - 1; i >= jmin; --i) {
        const int cnt = C->hist[i];
        const int beg = C->start[i], end = beg + cnt;
        if (cnt) {
            for (int k = beg + tid; k < end; k += nt) { int ly, lx; const int p = db_entry<GL>(geo, A.order[k], ly, lx); A.par[p] = p; }
            g.sync();
            db_unite_level<GL, false>(g, geo, A, C, i, beg, end);
            g.sync();
        }
        if ((fm >> i) & 1ull) {
            for (int k = tid; k < end; k += nt) {
                int ly, lx;
                const int p = db_entry<GL>(geo, A.order[k], ly, lx);
                const int r = db_find<GL>(A.par, p);
                if (A.frz[r] == i) A.obj[p] = r + 1;
            }
            g.sync();
        }
    }

    // ---- object slots, record pool --------------------------------------------------------------------------------
    for (int k = tid; k < npix; k += nt) {
        int ly, lx;
        const int p = db_entry<GL>(geo, A.order[k], ly, lx);
        if (A.frz[p]) A.st[p] = atomicAdd(&C->nslot, 1);
    }
    g.sync();
    if (tid == 0) {
        const uint32_t base = atomicAdd(&a.w.counters[C_POOL], (uint32_t)C->nslot);
        C->pool_base = (int)base;
        C->pool_ok = (long long)base + C->nslot <= a.cap_out ? 1 : 0;
        C->n_f[0] = 0; C->n_f[1] = 0;
    }
    g.sync();
    const bool pool_ok = C->pool_ok != 0;
    ORec *pool = a.w.pool + C->pool_base;

    // ---- D7: synchronous growth from a frontier -------------------------------------------------------------------
    int32_t *qr = A.T, *pend = A.accn, *F[2] = {A.lost, A.touched};
    for (int k = tid; k < npix; k += nt) {
        int ly, lx;
        const int p = db_entry<GL>(geo, A.order[k], ly, lx);
        if (A.obj[p] == 0) {
            bool near = false;
            db_for_neighbours<GL>(geo, p, ly, lx, [&](int q, int, int) {
                if (db_member<GL>(geo, A, q) && A.obj[q] != 0) near = true;
            });
            qr[p] = near ? 1 : 0;
            if (near) F[0][atomicAdd(&C->n_f[0], 1)] = p;
        } else if (A.frz[p]) {
            // the key pixel of an object: its record
            if (!pool_ok) {
                if ((long long)C->pool_base + A.st[p] < a.cap_out) pool[A.st[p]].omin = INT_MAX;   // emit skips it
            } else {
                int ly, lx;
                geo.coords(p, ly, lx);
                ORec *o = pool + A.st[p];
                o->f = 0.0; o->sx = 0.0; o->sy = 0.0; o->sxx = 0.0; o->syy = 0.0; o->sxy = 0.0;
                o->peak = 0ull;
                o->key = geo.fidx(ly, lx);
                o->frame = s.frame;
                o->npix = 0;
                o->xmin = INT_MAX; o->xmax = INT_MIN; o->ymin = INT_MAX; o->ymax = INT_MIN;
                o->omin = INT_MAX;
                o->pad[0] = 0; o->pad[1] = 0;
            }
        }
    }
    g.sync();
    for (int round = 1;; ++round) {
        const int cur = (round - 1) & 1, nf = C->n_f[cur];
        if (nf == 0) break;
        const int32_t *Fc = F[cur];
        int32_t *Fn = F[cur ^ 1];
        for (int k = tid; k < nf; k += nt) {   // the brightest assigned neighbour, as of the previous round
            const int p = Fc[k];
            int ly, lx;
            geo.coords(p, ly, lx);
            float best = 0.f;
            int bo = 0;
            db_for_neighbours<GL>(geo, p, ly, lx, [&](int q, int dy, int dx) {
                if (!db_member<GL>(geo, A, q)) return;
                const int oq = A.obj[q];
                if (oq == 0) return;
                const float vq = __ldg(geo.sub + geo.fidx(ly + dy, lx + dx));
                if (bo == 0 || vq > best || (vq == best && oq < bo)) { best = vq; bo = oq; }
            });
            pend[p] = bo;
        }
        if (tid == 0) C->n_f[cur ^ 1] = 0;
        g.sync();
        for (int k = tid; k < nf; k += nt) { const int p = Fc[k]; A.obj[p] = pend[p]; }
        g.sync();
        for (int k = tid; k < nf; k += nt) {   // next frontier: the unassigned neighbours of the pixels just assigned
            const int p = Fc[k];
            int ly, lx;
            geo.coords(p, ly, lx);
            db_for_neighbours<GL>(geo, p, ly, lx, [&](int q, int, int) {
                if (!db_member<GL>(geo, A, q) || A.obj[q] != 0) return;
                if (atomicExch(&qr[q], round + 1) != round + 1) Fn[atomicAdd(&C->n_f[cur ^ 1], 1)] = q;
            });
        }
        g.sync();
    }

    // ---- D8 + the records of the objects: one raster pass over the box, 32 consecutive pixels per warp step ---------
    int32_t *omin = A.T;   // (qr is done with)
    for (int k = tid; k < npix; k += nt) {
        int ly, lx;
        const int p = db_entry<GL>(geo, A.order[k], ly, lx);
        if (A.frz[p]) omin[p] = INT_MAX;
    }
    g.sync();
    {
        const int lane = tid & 31, nchunks = (nbox + 31) >> 5;
        for (int ch = g.warp(); ch < nchunks; ch += g.nwarps()) {
            const int k = ch * 32 + lane;
            int r = -1, f = 0, ly = 0, lx = 0;
            if (k < nbox) {
                ly = k / geo.bw; lx = k - ly * geo.bw;
                f = geo.fidx(ly, lx);
                const int p = geo.aidx(ly, lx);
                const bool mem = GL ? labels[f] == geo.L : A.lvl[p] >= 0;
                if (mem) r = A.obj[p] - 1;
            }
            uint32_t todo = __ballot_sync(0xffffffffu, r >= 0);
            while (todo) {
                const int l0 = __ffs(todo) - 1;
                const int r0 = __shfl_sync(0xffffffffu, r, l0);
                const bool mine = r == r0;
                todo &= ~__ballot_sync(0xffffffffu, mine);
                int ky, kx;
                geo.coords(r0, ky, kx);
                PixAcc v;
                v.f = 0.0; v.sx = 0.0; v.sy = 0.0; v.sxx = 0.0; v.syy = 0.0; v.sxy = 0.0; v.peak = 0ull;
                v.npix = 0; v.xmin = INT_MAX; v.xmax = INT_MIN; v.ymin = INT_MAX; v.ymax = INT_MIN; v.omin = INT_MAX;
                if (mine) {
                    const float fv = __ldg(geo.sub + f);
                    const double I = (double)fv, dx = (double)(lx - kx), dy = (double)(ly - ky);
                    v.f = I; v.sx = I * dx; v.sy = I * dy; v.sxx = I * dx * dx; v.syy = I * dy * dy; v.sxy = I * dx * dy;
                    v.peak = ((u64)f32_to_key(fv) << 32) | (u64)(0xFFFFFFFFu - (uint32_t)f);
                    v.npix = 1; v.xmin = v.xmax = geo.x0 + lx; v.ymin = v.ymax = geo.y0 + ly; v.omin = f;
                }
                pix_reduce(v);
                if (lane == l0) {
                    atomicMin(&omin[r0], v.omin);
                    if (pool_ok) {
                        ORec *o = pool + A.st[r0];
                        atomicAdd(&o->f, v.f); atomicAdd(&o->sx, v.sx); atomicAdd(&o->sy, v.sy);
                        atomicAdd(&o->sxx, v.sxx); atomicAdd(&o->syy, v.syy); atomicAdd(&o->sxy, v.sxy);
                        atomicMax(&o->peak, v.peak);
                        atomicAdd(&o->npix, v.npix);
                        atomicMin(&o->xmin, v.xmin); atomicMax(&o->xmax, v.xmax);
                        atomicMin(&o->ymin, v.ymin); atomicMax(&o->ymax, v.ymax);
                    }
                }
            }
        }
    }
    g.sync();
    for (int k = tid; k < npix; k += nt) {
        int ly, lx;
        const int p = db_entry<GL>(geo, A.order[k], ly, lx);
        const int r = A.obj[p] - 1;
        const int m = ldv<GL>(omin + r);
        labels[geo.fidx(ly, lx)] = m + 1;
        if (A.frz[p]) {
            const int mo = ldv<GL>(omin + p);
            mark_kept(a.w, fo + (size_t)mo);
            if (pool_ok) pool[A.st[p]].omin = mo;
        }
    }
    if (tid == 0) a.w.state[ci] = 1;
    g.sync();
}

// carve a group's shared-memory arrays for `cap` pixels
__device__ __forceinline__ DbArr db_smem_arrays(char *base, int cap) {
    DbArr A;
    A.accf = (double *)base; base += (size_t)cap * 8;
    A.par = (int32_t *)base; base += (size_t)cap * 4;
    A.accn = (int32_t *)base; base += (size_t)cap * 4;
    A.st = (int32_t *)base; base += (size_t)cap * 4;
    A.T = (int32_t *)base; base += (size_t)cap * 4;
    A.obj = (int32_t *)base; base += (size_t)cap * 4;
    A.order = (int32_t *)base; base += (size_t)cap * 4;
    A.lost = (int32_t *)base; base += (size_t)cap * 4;
    A.touched = (int32_t *)base; base += (size_t)cap * 4;
    A.lvl = (int8_t *)base; base += (size_t)cap;
    A.frz = (uint8_t *)base;
    return A;
}
constexpr size_t db_smem_bytes(int cap) { return (size_t)cap * 42; }
constexpr size_t DB_CTL_BYTES = (sizeof(DbCtl) + 15) / 16 * 16;

// tiers 0, 1: one warp per candidate (tier 0: boxes of at most CAP_TINY cells -- half of all candidates -- with half the
// shared memory per warp, so twice as many warps per SM hide the latency of this short, dependent code)
template <int TIER, int CAP, int NWARPS>
__global__ void __launch_bounds__(NWARPS * 32) k9_deblend_warp(DbArgs a) {
    extern __shared__ __align__(16) char smem[];
    const int warp = threadIdx.x >> 5;
    WarpGroup g;
    g.lane = threadIdx.x & 31;
    char *mine = smem + (size_t)warp * (DB_CTL_BYTES + db_smem_bytes(CAP));
    DbCtl *C = (DbCtl *)mine;
    const DbArr A = db_smem_arrays(mine + DB_CTL_BYTES, CAP);
    const uint32_t n = a.w.counters[C_TIER0 + TIER];
    while (true) {
        uint32_t it = 0;
        if (g.lane == 0) it = atomicAdd(&a.w.counters[C_CUR0 + TIER], 1u);
        it = __shfl_sync(0xffffffffu, it, 0);
        if (it >= n) break;
        db_candidate<false>(g, a, A, C, a.w.lists[(size_t)TIER * a.cap_in + it]);
    }
}

// tiers 2, 3: one thread block per candidate, arrays in shared memory
template <int TIER, int CAP, int NT>
__global__ void __launch_bounds__(NT) k9_deblend_block(DbArgs a) {
    extern __shared__ __align__(16) char smem[];
    BlockGroup g;
    DbCtl *C = (DbCtl *)smem;
    const DbArr A = db_smem_arrays(smem + DB_CTL_BYTES, CAP);
    const uint32_t n = a.w.counters[C_TIER0 + TIER];
    while (true) {
        if (threadIdx.x == 0) C->item = (int)atomicAdd(&a.w.counters[C_CUR0 + TIER], 1u);
        __syncthreads();
        const uint32_t it = (uint32_t)C->item;
        __syncthreads();
        if (it >= n) break;
        db_candidate<false>(g, a, A, C, a.w.lists[(size_t)TIER * a.cap_in + it]);
    }
}

// tier 4: one thread block per candidate, arrays in the workspace (frame coordinates)
__global__ void __launch_bounds__(512) k9_deblend_global(DbArgs a) {
    __shared__ DbCtl ctl;
    BlockGroup g;
    DbArr A;
    A.par = a.w.par; A.accn = a.w.accn; A.st = a.w.st; A.T = a.w.T; A.obj = a.w.obj; A.order = a.w.order; A.lost = a.w.lost;
    A.touched = a.w.touched; A.accf = a.w.accf; A.lvl = a.w.lvl; A.frz = a.w.frz;
    const uint32_t n = a.w.counters[C_TIER0 + 4];
    while (true) {
        if (threadIdx.x == 0) ctl.item = (int)atomicAdd(&a.w.counters[C_CUR0 + 4], 1u);
        __syncthreads();
        const uint32_t it = (uint32_t)ctl.item;
        __syncthreads();
        if (it >= n) break;
        db_candidate<true>(g, a, A, &ctl, a.w.lists[(size_t)4 * a.cap_in + it]);
    }
}

// ------------------------------------------------------------------------------------------------ output catalogue
__global__ void __launch_bounds__(256) k9_emit(DbArgs a, bd_source *out, int64_t *n_out) {
    const long long total = db_total(a);
    const size_t HW = (size_t)a.H * a.W;
    const long long t0 = (long long)blockIdx.x * blockDim.x + threadIdx.x, stride = (long long)gridDim.x * blockDim.x;
    if (t0 < a.B)
        n_out[t0] = (int64_t)kept_rank(a.w.keptbits, a.w.blkprefix, (size_t)(t0 + 1) * HW) - (int64_t)kept_rank(a.w.keptbits, a.w.blkprefix, (size_t)t0 * HW);
    if (!out || a.cap_out <= 0) return;
    for (long long i = t0; i < total; i += stride) {
        if (a.w.state[i]) continue;
        const bd_source s = a.cat[i];
        const uint32_t rank = kept_rank(a.w.keptbits, a.w.blkprefix, (size_t)s.frame * HW + (size_t)(s.label - 1));
        if ((int64_t)rank < a.cap_out) out[rank] = s;
    }
    const long long np = min((long long)a.w.counters[C_POOL], (long long)a.cap_out);
    const int W = a.W;
    for (long long j = t0; j < np; j += stride) {
        const ORec o = a.w.pool[j];
        if (o.omin == INT_MAX) continue;   // a slot of a candidate that could not reserve its records
        const uint32_t rank = kept_rank(a.w.keptbits, a.w.blkprefix, (size_t)o.frame * HW + (size_t)o.omin);
        if ((int64_t)rank >= a.cap_out) continue;
        const int yk = o.key / W, xk = o.key - yk * W;
        bd_source s;
        s.frame = o.frame;
        s.label = o.omin + 1;
        s.npix = o.npix;
        s.xmin = o.xmin; s.xmax = o.xmax; s.ymin = o.ymin; s.ymax = o.ymax;
        const uint32_t pidx = 0xFFFFFFFFu - (uint32_t)(o.peak & 0xFFFFFFFFull);
        s.ypeak = (int)(pidx / (uint32_t)W);
        s.xpeak = (int)(pidx - (uint32_t)s.ypeak * (uint32_t)W);
        s.peak = key_to_f32((uint32_t)(o.peak >> 32));
        s.flux = o.f;
        const double mx = o.sx / o.f, my = o.sy / o.f;
        s.x = (double)xk + mx;
        s.y = (double)yk + my;
        s.x2 = o.sxx / o.f - mx * mx;
        s.y2 = o.syy / o.f - my * my;
        s.xy = o.sxy / o.f - mx * my;
        out[rank] = s;
    }
}

}  // namespace

size_t k9_workspace_bytes(int B, int H, int W, int64_t cap_in, int64_t cap_out) {
    DbWs w;
    return carve(w, nullptr, B, H, W, cap_in, cap_out) + 256;
}

int k9_launch(bd_ctx *ctx, const float *d_sub, const float *d_rms, int B, int H, int W, double detect_k, int min_area,
              const bd_deblend_params *p, int32_t *d_labels, const bd_source *d_cat_in, const int64_t *d_n_in, int64_t cap_in,
              bd_source *d_cat_out, int64_t cap_out, int64_t *d_n_out, void *d_ws, size_t ws_bytes, cudaStream_t st) {
    DbArgs a;
    memset(&a, 0, sizeof(a));
    char *base = (char *)bd_align_up((size_t)d_ws, 256);
    const size_t need = carve(a.w, base, B, H, W, cap_in, cap_out);
    if ((size_t)(base - (char *)d_ws) + need > ws_bytes)
        return bd_set_error(ctx, BD_EWORKSPACE, "deblend workspace: need %zu bytes, got %zu", need + 256, ws_bytes);
    int log2n = 0;
    while ((1 << log2n) < p->n_thresh) ++log2n;
    a.sub = d_sub; a.rms = d_rms; a.labels = d_labels; a.cat = d_cat_in; a.n_in = d_n_in; a.cap_in = cap_in; a.cap_out = cap_out;
    a.B = B; a.H = H; a.W = W; a.kf = (float)detect_k; a.min_area = min_area; a.nthr = p->n_thresh; a.log2n = log2n;
    a.min_cont = p->min_cont;
    BD_CUDA_CHECK(ctx, cudaMemsetAsync(a.w.counters, 0, a.w.zero_bytes, st));
    const int nsm = ctx->num_sms;
    k9_classify<<<nsm * 8, 256, 0, st>>>(a);
    constexpr int TINY_WARPS = 16;
    const size_t sm_tiny = TINY_WARPS * (DB_CTL_BYTES + db_smem_bytes(CAP_TINY));
    const size_t sm_warp = WARPS_PER_CTA * (DB_CTL_BYTES + db_smem_bytes(CAP_WARP));
    const size_t sm_mid = DB_CTL_BYTES + db_smem_bytes(CAP_MID), sm_big = DB_CTL_BYTES + db_smem_bytes(CAP_BIG);
    BD_CUDA_CHECK(ctx, cudaFuncSetAttribute(k9_deblend_warp<0, CAP_TINY, TINY_WARPS>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm_tiny));
    BD_CUDA_CHECK(ctx, cudaFuncSetAttribute(k9_deblend_warp<1, CAP_WARP, WARPS_PER_CTA>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm_warp));
    BD_CUDA_CHECK(ctx, cudaFuncSetAttribute(k9_deblend_block<2, CAP_MID, 128>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm_mid));
    BD_CUDA_CHECK(ctx, cudaFuncSetAttribute(k9_deblend_block<3, CAP_BIG, 512>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm_big));
    k9_deblend_warp<0, CAP_TINY, TINY_WARPS><<<nsm * 2, TINY_WARPS * 32, sm_tiny, st>>>(a);
    k9_deblend_warp<1, CAP_WARP, WARPS_PER_CTA><<<nsm * 2, WARPS_PER_CTA * 32, sm_warp, st>>>(a);
    k9_deblend_block<2, CAP_MID, 128><<<nsm * 3, 128, sm_mid, st>>>(a);
    k9_deblend_block<3, CAP_BIG, 512><<<nsm, 512, sm_big, st>>>(a);
    k9_deblend_global<<<nsm * 2, 512, 0, st>>>(a);
    k5s_scan_blocks<<<1, 1024, 0, st>>>(a.w.blkcnt, a.w.NB, a.w.blkprefix, a.w.counters + 32);
    const int nb = nsm * 8 * 256 >= B ? nsm * 8 : (B + 255) / 256;
    k9_emit<<<nb, 256, 0, st>>>(a, d_cat_out, d_n_out);
    BD_CUDA_CHECK(ctx, cudaGetLastError());
    return BD_OK;
}
