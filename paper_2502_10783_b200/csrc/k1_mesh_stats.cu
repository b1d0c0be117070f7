// K1: per-mesh iterative sigma-clipped statistics (step a1).  PAPER.md:67 (rectangular sub-regions),
// :69-76 (eqs. 1-4), :78 ("determine the upper and lower limits based on the calculated central value and
// the specified sigma range, exclude data outside these limits, and recalculate the central value and
// standard deviation ... Once the maximum number of iterations is reached or the data stabilizes ...").
//
// The paper gives one GPU *thread* per sub-region.  Here a mesh is owned by a team of C CTAs (a
// thread-block cluster; C = 1 for meshes that fit one CTA's shared memory): each CTA stages a slab of the
// mesh's rows in shared memory with one TMA bulk-tensor load, and every later sweep reads shared memory
// only, so HBM sees each pixel once (4 B/px).
//
// What makes the clipping loop cheap: the survivors of every round are the pixels in a value interval
// [LO, HI] (LO = max of the lower bounds so far, HI = min of the upper bounds), so a round needs
//   (1) one sweep for n, sum(x-p), sum((x-p)^2) over [LO, HI] and the count below LO  -- float64
//       accumulation against float64 bounds, so the survivor set is the float64 definition's; and
//   (2) the order statistics n_below + (n-1)/2 and n_below + n/2 of the WHOLE mesh, found by radix
//       select on order-preserving uint32 keys: a level-0 histogram (2048 bins, bin width = the smallest
//       power of two of key units that covers [kmin, kmax]) is built once per mesh and reused by every
//       round; each lower level refines one bin by 11 more key bits until the key is exact.
// Team-wide values go through distributed shared memory; with C = 1 everything is CTA-local.
#include <cooperative_groups.h>

#include "common.cuh"

namespace cg = cooperative_groups;

namespace {

constexpr int K1_LB = 11;               // key bits resolved per histogram level
constexpr int K1_NB = 1 << K1_LB;       // bins per level
constexpr int K1_MAXWARPS = 32;

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
    uint32_t kmin, kmax;
};

struct Smem {   // fixed-size part of shared memory; the slab follows
    alignas(8) unsigned long long mbar;
    Xch xch[2];
    Xch tot;
    double red_d[2][K1_MAXWARPS];
    int red_i[2][K1_MAXWARPS];
    uint32_t red_u[2][K1_MAXWARPS];
    uint32_t sel_bin, sel_prefix, sel_count;
    uint32_t histp[K1_NB];       // this CTA's partial histogram of the current level
    uint32_t hists[K1_NB];       // team-total histogram of a refinement level
    uint32_t cum0[K1_NB + 1];    // exclusive prefix of the team-total level-0 histogram
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

__device__ void block_reduce_minmax(Smem &s, uint32_t &kmin, uint32_t &kmax) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = blockDim.x >> 5;
#pragma unroll
    for (int o = 16; o; o >>= 1) {
        kmin = min(kmin, __shfl_xor_sync(0xffffffffu, kmin, o));
        kmax = max(kmax, __shfl_xor_sync(0xffffffffu, kmax, o));
    }
    if (lane == 0) { s.red_u[0][warp] = kmin; s.red_u[1][warp] = kmax; }
    __syncthreads();
    for (int w = 0; w < nw; ++w) { kmin = min(kmin, s.red_u[0][w]); kmax = max(kmax, s.red_u[1][w]); }
    __syncthreads();
}

// Team-wide combine of a per-CTA Xch (already block-reduced, same value in all threads of the CTA).
// phase alternates the exchange slot so a fast CTA's next write cannot overtake a slow CTA's read.
template <int C>
__device__ Xch team_combine(Smem &s, const Xch &mine, int &phase) {
    if constexpr (C == 1) return mine;
    Xch *slot = &s.xch[phase & 1];
    if (threadIdx.x == 0) *slot = mine;
    Team<C>::sync();
    if (threadIdx.x == 0) {
        Xch t; t.s1 = 0; t.s2 = 0; t.n_in = 0; t.n_below = 0; t.kmin = 0xFFFFFFFFu; t.kmax = 0;
        for (unsigned r = 0; r < (unsigned)C; ++r) {   // rank order: every CTA computes the same bits
            const Xch *o = Team<C>::remote(slot, r);
            t.s1 += o->s1; t.s2 += o->s2; t.n_in += o->n_in; t.n_below += o->n_below;
            t.kmin = min(t.kmin, o->kmin); t.kmax = max(t.kmax, o->kmax);
        }
        s.tot = t;
    }
    __syncthreads();
    Xch t = s.tot;
    __syncthreads();
    ++phase;
    return t;
}

// Exclusive scan of src[0..nb) (nb <= K1_NB) over the CTA; writes dst[0..nb] if dst != nullptr, and locates
// the bin holding 0-based rank `want` (returns bin, exclusive prefix and count through shared memory).
__device__ void block_scan_locate(Smem &s, const uint32_t *src, uint32_t *dst, int nb, uint32_t want,
                                  uint32_t &bin, uint32_t &prefix, uint32_t &count) {
    const int nt = blockDim.x, per = (nb + nt - 1) / nt;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = nt >> 5;
    const int b0 = threadIdx.x * per;
    uint32_t local = 0;
    for (int k = 0; k < per; ++k) if (b0 + k < nb) local += src[b0 + k];
    uint32_t incl = local;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        uint32_t v = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += v;
    }
    if (lane == 31) s.red_u[0][warp] = incl;
    __syncthreads();
    uint32_t base = 0;
    for (int w = 0; w < warp; ++w) base += s.red_u[0][w];
    uint32_t total = 0;
    for (int w = 0; w < nw; ++w) total += s.red_u[0][w];
    uint32_t run = base + incl - local;
    for (int k = 0; k < per; ++k) {
        if (b0 + k >= nb) break;
        uint32_t c = src[b0 + k];
        if (dst) dst[b0 + k] = run;
        if (want >= run && want < run + c) { s.sel_bin = b0 + k; s.sel_prefix = run; s.sel_count = c; }
        run += c;
    }
    if (dst && threadIdx.x == 0) dst[nb] = total;
    __syncthreads();
    bin = s.sel_bin; prefix = s.sel_prefix; count = s.sel_count;
    __syncthreads();
}

// Sum the C partial histograms (histp of every CTA) into this CTA's hists.  Two team syncs.
template <int C>
__device__ const uint32_t *team_merge_hist(Smem &s, int nb) {
    if constexpr (C == 1) {
        __syncthreads();
        return s.histp;
    }
    Team<C>::sync();
    for (int b = threadIdx.x; b < nb; b += blockDim.x) {
        uint32_t t = 0;
        for (unsigned r = 0; r < (unsigned)C; ++r) t += Team<C>::remote(s.histp, r)[b];
        s.hists[b] = t;
    }
    Team<C>::sync();
    return s.hists;
}

template <int C>
__global__ void k1_mesh_stats(const __grid_constant__ CUtensorMap tmap, K1Args a) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    float *slab = reinterpret_cast<float *>(smem_raw);   // [slab_rows * mw], 128-B aligned for TMA
    Smem &s = *reinterpret_cast<Smem *>(smem_raw + (((size_t)a.slab_rows * a.mw * sizeof(float) + 127) & ~(size_t)127));

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

    // ---- stage the slab ---------------------------------------------------------------------------------
    if (a.use_tma && vw == a.mw) {
        if (tid == 0) {
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
        __syncthreads();
        {
            uint32_t bar = smem_u32(&s.mbar), done = 0;
            while (!done) {
                asm volatile(
                    "{ .reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], 0; selp.u32 %0, 1, 0, p; }"
                    : "=r"(done)
                    : "r"(bar)
                    : "memory");
            }
        }
    } else {   // plain loader: valid pixels packed row-major
        for (int i = tid; i < n_c; i += nt) {
            int r = i / vw, c = i - r * vw;
            slab[i] = frame_ptr[(size_t)(y0 + row0 + r) * a.W + x0 + c];
        }
        __syncthreads();
    }

    const float4 *slab4 = reinterpret_cast<const float4 *>(slab);
    const int n4 = (n_c + 3) >> 2;
    int phase = 0;

    // ---- sweep A: key range and round-0 sums about the pivot (first pixel of the mesh) -------------------
    double pivot = (double)__ldg(frame_ptr + (size_t)y0 * a.W + x0);
    Xch cur;
    {
        double s1 = 0, s2 = 0;
        uint32_t kmin = 0xFFFFFFFFu, kmax = 0;
        for (int i = tid; i < n4; i += nt) {
            float4 v = slab4[i];
            const float e[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
            for (int q = 0; q < 4; ++q)
                if (4 * i + q < n_c) {
                    double d = (double)e[q] - pivot;
                    s1 += d;
                    s2 = fma(d, d, s2);
                    uint32_t k = f32_to_key(e[q]);
                    kmin = min(kmin, k);
                    kmax = max(kmax, k);
                }
        }
        int n_in = 0, n_below = 0;
        block_reduce_stats(s, s1, s2, n_in, n_below);
        block_reduce_minmax(s, kmin, kmax);
        Xch mine; mine.s1 = s1; mine.s2 = s2; mine.n_in = n_c; mine.n_below = 0; mine.kmin = kmin; mine.kmax = kmax;
        cur = team_combine<C>(s, mine, phase);
    }
    const uint32_t kmin = cur.kmin, kmax = cur.kmax;
    int shift0 = 0;
    while (((kmax >> shift0) - (kmin >> shift0)) >= (uint32_t)K1_NB) ++shift0;
    const uint32_t base0 = kmin >> shift0;

    // ---- level-0 histogram of the whole mesh (reused by every round) -------------------------------------
    for (int b = tid; b < K1_NB; b += nt) s.histp[b] = 0;
    __syncthreads();
    for (int i = tid; i < n4; i += nt) {
        float4 v = slab4[i];
        const float e[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
        for (int q = 0; q < 4; ++q)
            if (4 * i + q < n_c) atomicAdd(&s.histp[(f32_to_key(e[q]) >> shift0) - base0], 1u);
    }
    {
        const uint32_t *h = team_merge_hist<C>(s, K1_NB);
        uint32_t b, p, c;
        block_scan_locate(s, h, s.cum0, K1_NB, 0xFFFFFFFFu, b, p, c);
    }

    // exact key of 0-based rank `want` among ALL pixels of the mesh; dup = how many further pixels share it
    auto select_key = [&](uint32_t want, uint32_t &dup_after) -> uint32_t {
        int lo = 0, hi = K1_NB;   // last b with cum0[b] <= want
        while (hi - lo > 1) {
            int mid = (lo + hi) >> 1;
            if (s.cum0[mid] <= want) lo = mid; else hi = mid;
        }
        uint32_t key_hi = base0 + (uint32_t)lo;    // key >> shift
        uint32_t r = want - s.cum0[lo];
        uint32_t cnt = s.cum0[lo + 1] - s.cum0[lo];
        int shift = shift0;
        while (shift > 0) {
            const int nshift = shift > K1_LB ? shift - K1_LB : 0;
            const int nb = 1 << (shift - nshift);
            for (int b = tid; b < nb; b += nt) s.histp[b] = 0;
            __syncthreads();
            for (int i = tid; i < n4; i += nt) {
                float4 v = slab4[i];
                const float e[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    uint32_t k = f32_to_key(e[q]);
                    if (4 * i + q < n_c && (k >> shift) == key_hi) atomicAdd(&s.histp[(k >> nshift) & (uint32_t)(nb - 1)], 1u);
                }
            }
            const uint32_t *h = team_merge_hist<C>(s, nb);
            uint32_t b, p, c;
            block_scan_locate(s, h, nullptr, nb, r, b, p, c);
            key_hi = (key_hi << (shift - nshift)) | b;
            r -= p;
            cnt = c;
            shift = nshift;
        }
        dup_after = cnt - 1 - r;
        return key_hi;
    };

    // smallest key strictly greater than `key` in the mesh (exists whenever it is asked for)
    auto next_key = [&](uint32_t key) -> uint32_t {
        uint32_t best = 0xFFFFFFFFu, dummy = 0;
        for (int i = tid; i < n4; i += nt) {
            float4 v = slab4[i];
            const float e[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                uint32_t k = f32_to_key(e[q]);
                if (4 * i + q < n_c && k > key) best = min(best, k);
            }
        }
        block_reduce_minmax(s, best, dummy);
        Xch mine; mine.s1 = 0; mine.s2 = 0; mine.n_in = 0; mine.n_below = 0; mine.kmin = best; mine.kmax = 0;
        return team_combine<C>(s, mine, phase).kmin;
    };

    // ---- clipping rounds -----------------------------------------------------------------------------------
    double LO = -INFINITY, HI = INFINITY;
    int n = n_tot, n_below = 0;
    double s1 = cur.s1, s2 = cur.s2;
    double med = 0, mu = 0, sd = 0;
    for (int round = 0;; ++round) {
        const double inv_n = 1.0 / (double)n;
        const double m1 = s1 * inv_n;
        mu = pivot + m1;
        double var = s2 * inv_n - m1 * m1;
        sd = var > 0.0 ? sqrt(var) : 0.0;
        uint32_t dup;
        const uint32_t ka = select_key((uint32_t)(n_below + (n - 1) / 2), dup);
        uint32_t kb = ka;
        if ((n & 1) == 0 && dup == 0) kb = next_key(ka);
        med = 0.5 * ((double)key_to_f32(ka) + (double)key_to_f32(kb));
        if (round >= a.iters) break;
        const double lo = fmax(LO, med - a.k_c * sd), hi = fmin(HI, med + a.k_c * sd);
        // sweep: survivors of [lo, hi], sums about the new pivot (= current median: a robust centre that
        // lies inside the surviving interval, so the one-pass variance below loses no digits -- and is
        // exactly 0 when all survivors are equal)
        double t1 = 0, t2 = 0;
        int c_in = 0, c_below = 0;
        for (int i = tid; i < n4; i += nt) {
            float4 v = slab4[i];
            const float e[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
            for (int q = 0; q < 4; ++q)
                if (4 * i + q < n_c) {
                    double x = (double)e[q];
                    if (x < lo) ++c_below;
                    else if (x <= hi) {
                        double d = x - med;
                        ++c_in;
                        t1 += d;
                        t2 = fma(d, d, t2);
                    }
                }
        }
        block_reduce_stats(s, t1, t2, c_in, c_below);
        Xch mine; mine.s1 = t1; mine.s2 = t2; mine.n_in = c_in; mine.n_below = c_below; mine.kmin = 0; mine.kmax = 0;
        Xch t = team_combine<C>(s, mine, phase);
        if (t.n_in == n || t.n_in == 0) break;   // stable (A7) or would empty the set: keep the current statistics
        LO = lo; HI = hi;
        n = t.n_in; n_below = t.n_below; s1 = t.s1; s2 = t.s2;
        pivot = med;
    }

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
static size_t k1_smem_bytes(int slab_rows, int mw) {
    return bd_align_up((size_t)slab_rows * mw * sizeof(float), 128) + sizeof(Smem) + 128;
}

int k1_plan(const bd_ctx *ctx, int mesh_h, int mesh_w, K1Plan *plan) {
    // Smallest team whose slab stays <= 64 KiB (several CTAs per SM overlap one team's load with another's
    // sweeps); if even 8 CTAs cannot do that, allow slabs up to the opt-in shared-memory limit.
    const size_t soft = 64 * 1024;
    for (int pass = 0; pass < 2; ++pass) {
        for (int c = 1; c <= 8; c *= 2) {
            int rows = (mesh_h + c - 1) / c;
            size_t slab = (size_t)rows * mesh_w * sizeof(float);
            size_t smem = k1_smem_bytes(rows, mesh_w);
            bool ok = pass == 0 ? slab <= soft : smem <= ctx->smem_optin;
            if (ok && smem <= ctx->smem_optin) {
                plan->cluster = c;
                plan->slab_rows = rows;
                plan->smem_bytes = smem;
                size_t px = (size_t)rows * mesh_w;
                plan->threads = px >= 16384 ? 512 : 256;
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
