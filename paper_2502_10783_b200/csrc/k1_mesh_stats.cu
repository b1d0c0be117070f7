// K1: per-mesh iterative sigma-clipped statistics (step a1).  PAPER.md:67 (rectangular sub-regions),
// :69-76 (eqs. 1-4), :78 ("determine the upper and lower limits based on the calculated central value and
// the specified sigma range, exclude data outside these limits, and recalculate the central value and
// standard deviation ... Once the maximum number of iterations is reached or the data stabilizes ...").
//
// The paper gives one GPU *thread* per sub-region.  Here a mesh is owned by a team of C CTAs (a
// thread-block cluster; C = 1 when the mesh fits one CTA's shared memory): each CTA stages a slab of the
// mesh's rows in shared memory with one TMA bulk-tensor load, and every later sweep reads shared memory
// only, so HBM sees each pixel once (4 B/px).
//
// Structure of the clipping loop.  The survivors of every round are the pixels in a value interval
// [LO, HI] (LO = max of the lower bounds so far, HI = min of the upper bounds).  A round therefore needs
//   (1) one sweep for n, sum(x-p), sum((x-p)^2) over [LO, HI] and the count below LO -- float64 sums
//       against float64 bounds, so the survivor set is the float64 definition's; and
//   (2) the order statistics n_below + (n-1)/2 and n_below + n/2 of the WHOLE mesh.
// (2) is a radix select on order-preserving uint32 keys that avoids per-pixel shared-memory atomics
// (measured: ~1 atomic/clk/SM, which made the first version of this kernel 2.1 ms on a 9216x9232 frame):
//   * the median of a set lies within one (population) standard deviation of its mean, so the search
//     starts from the key range of [mean - sd, mean + sd];
//   * each refinement level histograms that range into <= 64 bins with PER-THREAD byte counters in shared
//     memory (plain load/add/store, bank-conflict free), reduced with dp4a; it descends into the bin that
//     holds the wanted rank until that bin has <= 512 pixels (or is a single key);
//   * the pixels of a window of bins around it (<= 1024 pixels) are gathered, shared by the team, and
//     counting-sorted once; every later round's median is then a table lookup, because later medians move
//     by a fraction of sigma.  A rank that falls outside the window rebuilds the window.
// Team-wide values go through distributed shared memory; with C = 1 everything is CTA-local.
#include <cooperative_groups.h>

#include "common.cuh"

namespace cg = cooperative_groups;

namespace {

constexpr int K1_NBIN = 64;        // bins per refinement level
constexpr int K1_T1 = 512;         // stop refining when the target bin holds <= this many pixels
constexpr int K1_LISTCAP = 1024;   // candidate window capacity (team total)
constexpr int K1_FB = 1024;        // fine bins of the candidate counting sort
constexpr int K1_MAXWARPS = 16;
constexpr int K1_MAXC = 8;

struct K1Args {
    const float *img;
    int B, H, W, mh, mw, ny, nx;
    int slab_rows, use_tma;
    double k_c;
    int iters, skew_guard;
    double median_factor, mean_factor;
    double *bkg_raw, *rms_raw, *median, *mean;
    int32_t *n_kept;
};

struct Xch {   // one CTA's contribution to a team-wide reduction
    double s1, s2;
    int n_in, n_below;
    uint32_t below, m, nextkey, pad;
    uint32_t cnt[K1_NBIN];
};

struct Smem {   // fixed-size part of shared memory; follows the slab
    alignas(16) unsigned long long mbar;
    Xch xch[2];
    Xch tot;
    double red_d[2][K1_MAXWARPS];
    int red_i[2][K1_MAXWARPS];
    uint32_t red_u[K1_MAXWARPS];
    uint32_t win_b0, win_b1;
    uint32_t cand_local[K1_LISTCAP];   // this CTA's candidates (peers read it through DSMEM)
    uint32_t list[K1_LISTCAP];         // the team's candidates
    // the union area (per-thread byte histograms during refinement; sort arrays afterwards) follows
};

struct SortArea {
    uint32_t sorted[K1_LISTCAP];
    uint32_t fcur[K1_FB];
    uint32_t fstart[K1_FB + 1];
};

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

// ---- block-wide reductions (result valid in every thread) -------------------------------------------------
__device__ void block_reduce_stats(Smem &s, double &s1, double &s2, int &n_in, int &n_below) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = blockDim.x >> 5;
#pragma unroll
    for (int o = 16; o; o >>= 1) {
        s1 += __shfl_xor_sync(0xffffffffu, s1, o);
        s2 += __shfl_xor_sync(0xffffffffu, s2, o);
        n_in += __shfl_xor_sync(0xffffffffu, n_in, o);
        n_below += __shfl_xor_sync(0xffffffffu, n_below, o);
    }
    if (lane == 0) { s.red_d[0][warp] = s1; s.red_d[1][warp] = s2; s.red_i[0][warp] = n_in; s.red_i[1][warp] = n_below; }
    __syncthreads();
    s1 = 0; s2 = 0; n_in = 0; n_below = 0;
    for (int w = 0; w < nw; ++w) { s1 += s.red_d[0][w]; s2 += s.red_d[1][w]; n_in += s.red_i[0][w]; n_below += s.red_i[1][w]; }
    __syncthreads();
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

// Team-wide combine.  `mine` holds this CTA's block-reduced scalars (same value in all threads); cnt[] is
// taken from s.xch[slot].cnt, which the caller filled before (when with_cnt).  Sums everything over the team
// in rank order (every CTA computes the same bits), min for nextkey.  Result in s.tot (valid after return).
// phase alternates the exchange slot so a fast CTA's next write cannot overtake a slow CTA's read.
template <int C>
__device__ void team_combine(Smem &s, const Xch &mine, int &phase, bool with_cnt) {
    Xch *slot = &s.xch[phase & 1];
    if constexpr (C == 1) {
        __syncthreads();   // every thread is done with the previous s.tot
        if (threadIdx.x == 0) {
            s.tot.s1 = mine.s1; s.tot.s2 = mine.s2; s.tot.n_in = mine.n_in; s.tot.n_below = mine.n_below;
            s.tot.below = mine.below; s.tot.m = mine.m; s.tot.nextkey = mine.nextkey;
        }
        if (with_cnt && threadIdx.x < K1_NBIN) s.tot.cnt[threadIdx.x] = slot->cnt[threadIdx.x];
        __syncthreads();
        ++phase;
        return;
    }
    if (threadIdx.x == 0) {
        slot->s1 = mine.s1; slot->s2 = mine.s2; slot->n_in = mine.n_in; slot->n_below = mine.n_below;
        slot->below = mine.below; slot->m = mine.m; slot->nextkey = mine.nextkey;
    }
    Team<C>::sync();
    if (threadIdx.x == 0) {
        double s1 = 0, s2 = 0;
        int n_in = 0, n_below = 0;
        uint32_t below = 0, m = 0, nk = 0xFFFFFFFFu;
        for (unsigned r = 0; r < (unsigned)C; ++r) {
            const Xch *o = Team<C>::remote(slot, r);
            s1 += o->s1; s2 += o->s2; n_in += o->n_in; n_below += o->n_below;
            below += o->below; m += o->m; nk = min(nk, o->nextkey);
        }
        s.tot.s1 = s1; s.tot.s2 = s2; s.tot.n_in = n_in; s.tot.n_below = n_below;
        s.tot.below = below; s.tot.m = m; s.tot.nextkey = nk;
    }
    if (with_cnt && threadIdx.x >= 32 && threadIdx.x < 32 + K1_NBIN) {
        const int b = threadIdx.x - 32;
        uint32_t t = 0;
        for (unsigned r = 0; r < (unsigned)C; ++r) t += Team<C>::remote(slot, r)->cnt[b];
        s.tot.cnt[b] = t;
    }
    __syncthreads();
    ++phase;
}

template <int C>
__global__ void k1_mesh_stats(const __grid_constant__ CUtensorMap tmap, K1Args a) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    float *slab = reinterpret_cast<float *>(smem_raw);   // [slab_rows * mw], 128-B aligned for TMA
    const size_t slab_bytes = ((size_t)a.slab_rows * a.mw * sizeof(float) + 127) & ~(size_t)127;
    Smem &s = *reinterpret_cast<Smem *>(smem_raw + slab_bytes);
    unsigned char *area = smem_raw + slab_bytes + ((sizeof(Smem) + 127) & ~(size_t)127);
    uint8_t *hist8 = area;                                   // [K1_NBIN][nt] byte counters
    SortArea &srt = *reinterpret_cast<SortArea *>(area);     // aliases hist8 (used after the gather)

    const unsigned rank = Team<C>::rank();
    const int mesh = blockIdx.x / C;
    const int frame = mesh / (a.ny * a.nx);
    const int mj = (mesh / a.nx) % a.ny, mi = mesh % a.nx;
    const int y0 = mj * a.mh, x0 = mi * a.mw;
    const int vh = min(a.mh, a.H - y0), vw = min(a.mw, a.W - x0);       // valid part of the mesh
    const int row0 = (int)rank * a.slab_rows;                           // first mesh row of this CTA's slab
    const int my_rows = max(0, min(a.slab_rows, vh - row0));
    const int n_c = my_rows * vw;                                       // valid pixels in this slab, a prefix
    const int n_tot = vh * vw;
    const float *frame_ptr = a.img + (size_t)frame * a.H * a.W;
    const int tid = threadIdx.x, nt = blockDim.x;
    const int lane = tid & 31;

    // ---- stage the slab ---------------------------------------------------------------------------------
    const bool tma = a.use_tma && vw == a.mw;
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
    // pivot of the round-0 sums: median of five pixels of the mesh (uniform over the team; a robust centre
    // keeps the one-pass variance accurate even when some of the five are outliers)
    double pivot;
    {
        const int ys[5] = {0, 0, vh - 1, vh - 1, vh / 2}, xs[5] = {0, vw - 1, 0, vw - 1, vw / 2};
        float v[5];
#pragma unroll
        for (int k = 0; k < 5; ++k) v[k] = __ldg(frame_ptr + (size_t)(y0 + ys[k]) * a.W + x0 + xs[k]);
#define K1_CE(i, j) { float lo_ = fminf(v[i], v[j]), hi_ = fmaxf(v[i], v[j]); v[i] = lo_; v[j] = hi_; }
        K1_CE(0, 1) K1_CE(3, 4) K1_CE(2, 4) K1_CE(2, 3) K1_CE(0, 3) K1_CE(0, 2) K1_CE(1, 4) K1_CE(1, 3) K1_CE(1, 2)
#undef K1_CE
        pivot = (double)v[2];
    }
    if (tma) {
        __syncthreads();
        uint32_t bar = smem_u32(&s.mbar), done = 0;
        while (!done) {
            asm volatile(
                "{ .reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], 0; selp.u32 %0, 1, 0, p; }"
                : "=r"(done)
                : "r"(bar)
                : "memory");
        }
    } else {   // plain loader: valid pixels packed row-major
        for (int i = tid; i < n_c; i += nt) {
            int r = i / vw, c = i - r * vw;
            slab[i] = frame_ptr[(size_t)(y0 + row0 + r) * a.W + x0 + c];
        }
        __syncthreads();
    }

    const float4 *slab4 = reinterpret_cast<const float4 *>(slab);
    const int n4 = n_c >> 2, n_tail = n_c & 3;
    int phase = 0;

    // every sweep: whole float4s without per-element bounds checks, then the <= 3 tail pixels
#define K1_SWEEP(BODY)                                                   \
    {                                                                    \
        for (int i_ = tid; i_ < n4; i_ += nt) {                          \
            const float4 v_ = slab4[i_];                                 \
            { const float e = v_.x; BODY }                               \
            { const float e = v_.y; BODY }                               \
            { const float e = v_.z; BODY }                               \
            { const float e = v_.w; BODY }                               \
        }                                                                \
        if (tid < n_tail) { const float e = slab[(n4 << 2) + tid]; BODY }\
    }

    // ---- sweep A: round-0 sums about the pivot -------------------------------------------------------------
    double s1, s2;
    {
        double t1 = 0, t2 = 0;
        K1_SWEEP({ const double d = (double)e - pivot; t1 += d; t2 = fma(d, d, t2); })
        int z0 = 0, z1 = 0;
        block_reduce_stats(s, t1, t2, z0, z1);
        Xch mine; mine.s1 = t1; mine.s2 = t2; mine.n_in = 0; mine.n_below = 0; mine.below = 0; mine.m = 0; mine.nextkey = 0;
        team_combine<C>(s, mine, phase, false);
        s1 = s.tot.s1; s2 = s.tot.s2;
        __syncthreads();
    }

    // ---- candidate window state (uniform over the team) ---------------------------------------------------
    int mode = 0;                 // 0 none, 1 sorted list, 2 single key
    uint32_t list_off = 0, list_m = 0;             // mode 1: ranks [list_off, list_off + list_m) are srt.sorted[]
    uint32_t sel_key = 0, sel_lo = 0, sel_hi = 0;  // mode 2: ranks [sel_lo, sel_hi) all have key sel_key

    // Build the window for 0-based rank `want` of the whole mesh, searching keys [ka, kb] (must contain it).
    auto build = [&](uint32_t want, uint32_t ka, uint32_t kb) {
        uint32_t off = 0;
        bool top = true;
        for (;;) {
            const uint32_t span = kb - ka;
            int shift = 0;
            while ((span >> shift) >= (uint32_t)K1_NBIN) ++shift;
            // -- per-thread byte histogram of the keys in [ka, kb]
            for (int i = tid; i < (K1_NBIN * nt) / 16; i += nt) reinterpret_cast<uint4 *>(hist8)[i] = make_uint4(0, 0, 0, 0);
            __syncthreads();
            uint32_t below = 0;
            uint8_t *col = hist8 + tid;
            K1_SWEEP({
                const uint32_t k = f32_to_key(e);
                const uint32_t t = k - ka;
                if (t <= span) col[(t >> shift) * nt] += 1;
                else if (top && k < ka) ++below;
            })
            __syncthreads();
            // -- reduce the byte columns: G = nt/64 threads per bin, 16 words each, dp4a
            {
                const int G = nt / K1_NBIN, b = tid / G, g = tid - b * G;
                const uint32_t *row = reinterpret_cast<const uint32_t *>(hist8) + (size_t)b * (nt / 4);
                uint32_t acc = 0;
#pragma unroll
                for (int j = 0; j < 16; ++j) acc = __dp4a(row[j * G + g], 0x01010101u, acc);
                for (int o = G >> 1; o; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
                if (g == 0) s.xch[phase & 1].cnt[b] = acc;
            }
            if (top) below = block_reduce_u32<false>(s, below);
            else __syncthreads();
            Xch mine; mine.s1 = 0; mine.s2 = 0; mine.n_in = 0; mine.n_below = 0; mine.below = below; mine.m = 0; mine.nextkey = 0;
            team_combine<C>(s, mine, phase, true);
            if (top) off = s.tot.below;
            top = false;
            // -- locate the bin of `want` (every warp redundantly: lane l owns bins 2l, 2l+1)
            const uint32_t c0 = s.tot.cnt[2 * lane], c1 = s.tot.cnt[2 * lane + 1];
            uint32_t incl = c0 + c1;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                uint32_t t = __shfl_up_sync(0xffffffffu, incl, o);
                if (lane >= o) incl += t;
            }
            const uint32_t excl = incl - c0 - c1;
            const uint32_t r = want - off;
            const bool mine0 = r >= excl && r < excl + c0, mine1 = r >= excl + c0 && r < incl;
            const uint32_t bal = __ballot_sync(0xffffffffu, mine0 || mine1);
            if (bal == 0) {   // cannot happen for a range that brackets the rank; be safe: search all keys
                ka = 0; kb = 0xFFFFFFFFu; off = 0; top = true;
                __syncthreads();
                continue;
            }
            const int src = __ffs(bal) - 1;
            const uint32_t b = __shfl_sync(0xffffffffu, 2 * lane + (mine1 ? 1 : 0), src);
            const uint32_t pre = __shfl_sync(0xffffffffu, mine1 ? excl + c0 : excl, src);
            const uint32_t cntb = __shfl_sync(0xffffffffu, mine1 ? c1 : c0, src);
            if (shift == 0) {   // the bin is a single key
                mode = 2; sel_key = ka + b; sel_lo = off + pre; sel_hi = sel_lo + cntb;
                __syncthreads();
                return;
            }
            if (cntb > (uint32_t)K1_T1) {   // descend
                off += pre;
                ka = ka + (b << shift);
                kb = min(kb, ka + ((1u << shift) - 1u));
                __syncthreads();   // everyone has read s.tot.cnt before the next level rewrites it
                continue;
            }
            // -- window of bins around b with <= K1_LISTCAP pixels (thread 0 decides; same inputs on every CTA)
            if (tid == 0) {
                const int nb = (int)(span >> shift) + 1;
                int b0 = (int)b, b1 = (int)b;
                uint32_t tot = cntb;
                for (int g = 0; g < 8; ++g) {
                    bool grew = false;
                    if (b1 + 1 < nb && tot + s.tot.cnt[b1 + 1] <= (uint32_t)K1_LISTCAP) { ++b1; tot += s.tot.cnt[b1]; grew = true; }
                    if (b0 - 1 >= 0 && tot + s.tot.cnt[b0 - 1] <= (uint32_t)K1_LISTCAP) { --b0; tot += s.tot.cnt[b0]; grew = true; }
                    if (!grew) break;
                }
                s.win_b0 = b0; s.win_b1 = b1;
            }
            __syncthreads();
            const uint32_t b0 = s.win_b0, b1 = s.win_b1;
            // exclusive prefix of bin b0 (lane b0/2 knows it)
            const uint32_t pre0 = __shfl_sync(0xffffffffu, (b0 & 1) ? excl + c0 : excl, (int)(b0 >> 1));
            const uint32_t kga = ka + (b0 << shift);
            const uint32_t kgb = min(kb, ka + (((b1 + 1) << shift) - 1u));
            // -- gather: this thread's count is in its byte column; block scan -> private offset; write pass
            uint32_t mycnt = 0;
            for (uint32_t bb = b0; bb <= b1; ++bb) mycnt += col[bb * nt];
            uint32_t incl2 = mycnt;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                uint32_t t = __shfl_up_sync(0xffffffffu, incl2, o);
                if (lane >= o) incl2 += t;
            }
            if (lane == 31) s.red_u[tid >> 5] = incl2;
            __syncthreads();
            uint32_t wbase = 0, m_c = 0;
            for (int w = 0; w < (nt >> 5); ++w) { if (w < (tid >> 5)) wbase += s.red_u[w]; m_c += s.red_u[w]; }
            uint32_t pos = wbase + incl2 - mycnt;
            const uint32_t gspan = kgb - kga;
            K1_SWEEP({
                const uint32_t k = f32_to_key(e);
                if (k - kga <= gspan) s.cand_local[pos++] = k;
            })
            // -- share the candidates over the team
            Xch mine2; mine2.s1 = 0; mine2.s2 = 0; mine2.n_in = 0; mine2.n_below = 0; mine2.below = 0; mine2.m = m_c; mine2.nextkey = 0;
            const int slot = phase & 1;
            team_combine<C>(s, mine2, phase, false);   // includes the barrier that publishes cand_local
            const uint32_t m = s.tot.m;
            if constexpr (C == 1) {
                for (uint32_t i = tid; i < m; i += nt) s.list[i] = s.cand_local[i];
            } else {
                uint32_t base = 0;
                for (unsigned r = 0; r < (unsigned)C; ++r) {
                    const uint32_t mr = Team<C>::remote(&s.xch[slot], r)->m;
                    const uint32_t *src2 = Team<C>::remote(s.cand_local, r);
                    for (uint32_t i = tid; i < mr; i += nt) s.list[base + i] = src2[i];
                    base += mr;
                }
                Team<C>::sync();   // peers are done reading my cand_local and exchange slot
            }
            // -- counting sort of the list on fine bins (hist8 is dead now; the sort arrays alias it)
            int fshift = 0;
            while ((gspan >> fshift) >= (uint32_t)K1_FB) ++fshift;
            const int nfb = (int)(gspan >> fshift) + 1;
            __syncthreads();
            for (int i = tid; i < nfb; i += nt) srt.fcur[i] = 0;
            __syncthreads();
            for (uint32_t i = tid; i < m; i += nt) atomicAdd(&srt.fcur[(s.list[i] - kga) >> fshift], 1u);
            __syncthreads();
            {   // exclusive scan of fcur[0..nfb) -> fstart, fcur
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
                    srt.fstart[f0 + k] = run;
                    srt.fcur[f0 + k] = run;
                    run += c;
                }
            }
            __syncthreads();
            for (uint32_t i = tid; i < m; i += nt) {
                const uint32_t k = s.list[i];
                srt.sorted[atomicAdd(&srt.fcur[(k - kga) >> fshift], 1u)] = k;
            }
            __syncthreads();
            if (fshift > 0) {   // a fine bin may hold several keys: order it (bins are tiny)
                for (int f = tid; f < nfb; f += nt) {
                    const uint32_t lo = srt.fstart[f], hi = srt.fcur[f];
                    for (uint32_t i = lo + 1; i < hi; ++i) {
                        const uint32_t k = srt.sorted[i];
                        uint32_t j = i;
                        while (j > lo && srt.sorted[j - 1] > k) { srt.sorted[j] = srt.sorted[j - 1]; --j; }
                        srt.sorted[j] = k;
                    }
                }
                __syncthreads();
            }
            mode = 1; list_off = off + pre0; list_m = m;
            return;
        }
    };

    // smallest key strictly greater than `key` in the mesh (only asked when one exists)
    auto next_key = [&](uint32_t key) -> uint32_t {
        uint32_t best = 0xFFFFFFFFu;
        K1_SWEEP({ const uint32_t k = f32_to_key(e); if (k > key) best = min(best, k); })
        best = block_reduce_u32<true>(s, best);
        Xch mine; mine.s1 = 0; mine.s2 = 0; mine.n_in = 0; mine.n_below = 0; mine.below = 0; mine.m = 0; mine.nextkey = best;
        team_combine<C>(s, mine, phase, false);
        const uint32_t r = s.tot.nextkey;
        __syncthreads();
        return r;
    };

    // ---- clipping rounds -----------------------------------------------------------------------------------
    double LO = -INFINITY, HI = INFINITY;
    int n = n_tot, n_below = 0;
    double med = 0, mu = 0, sd = 0;
    for (int round = 0;; ++round) {
        const double inv_n = 1.0 / (double)n;
        const double m1 = s1 * inv_n;
        mu = pivot + m1;
        double var = s2 * inv_n - m1 * m1;
        sd = var > 0.0 ? sqrt(var) : 0.0;
        // median: ranks k0 = n_below + (n-1)/2 and (n even) k0 + 1 of the whole mesh
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
        if (round >= a.iters) break;
        const double lo = fmax(LO, med - a.k_c * sd), hi = fmin(HI, med + a.k_c * sd);
        // sweep: survivors of [lo, hi], sums about the new pivot (= current median: a robust centre that lies
        // inside the surviving interval, so the one-pass variance loses no digits -- and is exactly 0 when all
        // survivors are equal)
        double t1 = 0, t2 = 0;
        int c_in = 0, c_below = 0;
        K1_SWEEP({
            const double x = (double)e;
            if (x < lo) ++c_below;
            else if (x <= hi) {
                const double d = x - med;
                ++c_in;
                t1 += d;
                t2 = fma(d, d, t2);
            }
        })
        block_reduce_stats(s, t1, t2, c_in, c_below);
        Xch mine; mine.s1 = t1; mine.s2 = t2; mine.n_in = c_in; mine.n_below = c_below; mine.below = 0; mine.m = 0; mine.nextkey = 0;
        team_combine<C>(s, mine, phase, false);
        const int n_new = s.tot.n_in;
        const int nb_new = s.tot.n_below;
        const double s1_new = s.tot.s1, s2_new = s.tot.s2;
        __syncthreads();   // s.tot is rewritten by the next combine
        if (n_new == n || n_new == 0) break;   // stable (A7) or would empty the set: keep the current statistics
        LO = lo; HI = hi;
        n = n_new; n_below = nb_new; s1 = s1_new; s2 = s2_new;
        pivot = med;
    }
#undef K1_SWEEP

    if (rank == 0 && tid == 0) {
        double bkg = a.median_factor * med - a.mean_factor * mu;
        if (a.skew_guard) {
            if (sd == 0.0) bkg = mu;
            else if (fabs(mu - med) / sd >= 0.3) bkg = med;
        }
        if (a.bkg_raw) a.bkg_raw[mesh] = bkg;
        if (a.rms_raw) a.rms_raw[mesh] = sd;
        if (a.median) a.median[mesh] = med;
        if (a.mean) a.mean[mesh] = mu;
        if (a.n_kept) a.n_kept[mesh] = n;
    }
    if constexpr (C > 1) Team<C>::sync();   // nobody leaves while a peer may still read its shared memory
}

}  // namespace

// ---- host side ------------------------------------------------------------------------------------------
static size_t k1_smem_bytes(int slab_rows, int mw, int threads) {
    size_t area = (size_t)K1_NBIN * threads;
    if (area < sizeof(SortArea)) area = sizeof(SortArea);
    return bd_align_up((size_t)slab_rows * mw * sizeof(float), 128) + bd_align_up(sizeof(Smem), 128) + area + 128;
}

int k1_plan(const bd_ctx *ctx, int mesh_h, int mesh_w, K1Plan *plan) {
    // Smallest team whose slab stays <= 64 KiB (several CTAs per SM overlap one team's load with another's
    // sweeps); if even 8 CTAs cannot do that, allow slabs up to the opt-in shared-memory limit.
    const size_t soft = 64 * 1024;
    for (int pass = 0; pass < 2; ++pass) {
        for (int c = 1; c <= K1_MAXC; c *= 2) {
            int rows = (mesh_h + c - 1) / c;
            size_t px = (size_t)rows * mesh_w;
            size_t slab = px * sizeof(float);
            int threads = px >= 16384 ? 512 : 256;
            size_t smem = k1_smem_bytes(rows, mesh_w, threads);
            bool ok = pass == 0 ? slab <= soft : true;
            // byte counters: a thread sees at most ceil(px/threads) + 4 pixels of the slab
            if (ok && smem <= ctx->smem_optin && px / threads + 5 <= 255) {
                plan->cluster = c;
                plan->slab_rows = rows;
                plan->smem_bytes = smem;
                plan->threads = threads;
                plan->use_tma = (mesh_w % 4 == 0 && mesh_w <= 256 && rows <= 256) ? 1 : 0;
                return BD_OK;
            }
        }
    }
    return BD_EUNSUPPORTED;
}

template <int C>
static cudaError_t k1_launch_c(const CUtensorMap &tmap, const K1Args &a, const K1Plan &plan, int n_mesh, cudaStream_t st) {
    cudaError_t e = cudaFuncSetAttribute(k1_mesh_stats<C>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)plan.smem_bytes);
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
    return cudaLaunchKernelEx(&cfg, k1_mesh_stats<C>, tmap, a);
}

int k1_launch(bd_ctx *ctx, const float *d_img, int B, int H, int W, const bd_bkg_params *p, double *d_bkg_raw,
              double *d_rms_raw, double *d_median, double *d_mean, int32_t *d_n_kept, cudaStream_t st) {
    K1Plan plan;
    int rc = k1_plan(ctx, p->mesh_h, p->mesh_w, &plan);
    if (rc != BD_OK) return bd_set_error(ctx, rc, "mesh %dx%d does not fit a thread-block cluster's shared memory", p->mesh_h, p->mesh_w);
    K1Args a;
    a.img = d_img; a.B = B; a.H = H; a.W = W; a.mh = p->mesh_h; a.mw = p->mesh_w;
    a.ny = (H + a.mh - 1) / a.mh; a.nx = (W + a.mw - 1) / a.mw;
    a.slab_rows = plan.slab_rows; a.use_tma = plan.use_tma;
    a.k_c = p->clip_sigma; a.iters = p->clip_iters; a.skew_guard = p->skew_guard;
    a.median_factor = p->median_factor; a.mean_factor = p->mean_factor;
    a.bkg_raw = d_bkg_raw; a.rms_raw = d_rms_raw; a.median = d_median; a.mean = d_mean; a.n_kept = d_n_kept;

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
    const int n_mesh = B * a.ny * a.nx;
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
