// K4 + K5: 8-connected component labelling and per-component reduction (steps a4, a5).
// PAPER.md:153 ("identify pixels whose flux exceeds a specified main threshold. These pixels are then
// connected to form source candidates ... calculate peak values and total flux for each candidate"),
// :159 (isophotal photometry).  Readings A16 (8-connectivity), A18-A20 (moments, min_area, label map).
//
// The paper scans with one thread per pixel and reduces with Thrust.  Here the frame is cut into 128x64-pixel
// tiles and labelling and reduction are ONE pass over the tile (the first version labelled, flattened and then
// re-read labels and sub twice more: 1.38 ms on 9216x9232; ncu showed the tile kernel instruction-bound on
// divergent per-pixel loops and the re-read passes latency-bound):
//   K4a  per tile (256 threads, one per 32-pixel bit word): mask bytes -> bit rows (+1-pixel halo) in shared memory --
//        or, in FUSED mode (bkg_subtract_detect), the spline evaluation of step a3 itself: the image tile arrives by one
//        TMA load into the label buffer, sub / bkg / rms are written out and the threshold bits go straight into the bit
//        rows; pixels without any foreground neighbour are complete components (labelled on the spot, dropped when
//        min_area > 1); a COMPACT list of the other foreground pixels, so every later phase runs dense; union-find on
//        the list (parent = start of the horizontal run, vertical/diagonal links with the usual pruning, union by
//        minimum index); per-component pixel counts; components that can matter (count >= min_area, or touching a
//        foreground pixel of another tile) get a 96-byte record in a contiguous range the tile reserves with one atomic;
//        partial sums (npix, flux, first/second moments about the tile-local root, peak, bbox) are reduced over the
//        list entries of one (component, row) with a segmented shuffle reduction and added to the record with RED
//        atomics; the label tile (1 + raster index of the tile-local root, 0 = background) is assembled in shared memory
//        and leaves with one TMA bulk-tensor store; the tile's border bit rows/columns are exported (48 B per tile).
//   K4b  seam merge from the exported border bits alone: only real cross-tile links touch the label array
//        (union by atomicMin on the root's label word).
//   K5m  for every record whose tile-local root is no longer a root: add it to the final root's record
//        (float64 atomics, moments shifted to the new origin) and relabel the pixels of its bounding box.
//   K5k  records that are final roots with npix >= min_area set their bit in a per-pixel bitmap and count into
//        4096-pixel blocks;  K5s scans the block counts;  K5f ranks every kept root (= catalogue slot in
//        ascending (frame, label) order) and writes its record.
// Records are a compact array (capacity: one per 2x2-pixel block, the worst case, so nothing can overflow; only the
// records in use are touched); a direct-mapped index by the 2x2 block of the root (two roots can never share one: they
// would be 8-adjacent) finds the record of a root when two records merge.
// Labels are bit-exact by construction; float sums depend on atomic order (not bit-reproducible).
#include "common.cuh"
#include "spline_eval.cuh"

namespace {

typedef unsigned long long u64;

#include "kept_rank.cuh"

constexpr int TW = 128, TH = 64, K4_NT = 256;   // one thread per 32-pixel bit word of the tile
constexpr int TPX = TW * TH;             // 8192 pixels per tile
constexpr int BROWS = TH + 2;            // bit rows incl. halo rows y0-1 and y0+TH
constexpr int BWORDS = 6;                // [0] bit 31 = column x0-1, [1..4] the tile, [5] bit 0 = column x0+TW
constexpr int EDGE_WORDS = 12;           // per tile: top[4], bottom[4], left[2], right[2]

// lab[] word of a foreground pixel p (local index, 13 bits):
//   non-root: index of its parent / (after the flatten) of its root;
//   root:     p | count << 13 (14 bits) | F_RING, and once the record slot is known p | slot << 13 | F_REC | F_RING
constexpr uint32_t IDX_MASK = 0x1FFFu;
constexpr int CNT_SHIFT = 13;
constexpr uint32_t CNT_MASK = 0x3FFFu;   // count <= 8192
constexpr uint32_t F_REC = 0x80000000u;
constexpr uint32_t F_RING = 0x40000000u;

struct Rec {   // 96 bytes; sums are about the record's own root pixel
    double f, sx, sy, sxx, syy, sxy;
    u64 peak;          // (ordered key of sub << 32) | (0xFFFFFFFF - raster index in frame): max -> max value, ties -> min index
    int32_t root;      // raster index of the root within its frame
    int32_t frame;
    int32_t npix;
    int32_t xmin, xmax, ymin, ymax;
    int32_t merged;    // set by K5m: this record was added to another root's record
    int32_t pad[2];
};
static_assert(sizeof(Rec) == 96, "Rec must be 96 bytes");

struct Ws {
    uint32_t *counters;     // [0] n_rec, [1] n_kept
    uint8_t *maskbuf;       // [P] (only used when the caller gave no mask)
    uint32_t *edges;        // [ntiles * EDGE_WORDS]
    uint32_t *recidx;       // [nblk2] direct-mapped by the 2x2 block of a root: index of its record
    uint32_t *keptbits;     // [NWk] one bit per pixel  |
    uint32_t *blkcnt;       // [NB + 1] per 4096 px     |  zeroed together every call
    uint32_t *blkprefix;    // [NB + 2]
    float *wx_tab;          // [W][4] float32 x-weights of every image column  | fused mode: filled by k_spline_tabs
    double *wy_tab;         // [H][4] float64 y-weights of every image row     |
    int32_t *i0_tab, *j0_tab;   // [W], [H] grid cells                          |
    Rec *rec;               // [nblk2] records, compact: 0 .. n_rec-1 (capacity = one per 2x2 block, the worst case)
    size_t P, nblk2, NWk, NB, ntiles;
    size_t zero_bytes;      // bytes from keptbits to the end of blkcnt
    size_t total;
};

size_t carve(Ws &w, void *base, int B, int H, int W) {
    const size_t P = (size_t)B * H * W;
    w.P = P;
    w.nblk2 = (size_t)B * ((H + 1) / 2) * (W / 2);
    w.NWk = (P + 31) / 32 + 32;
    w.NB = (P + 4095) / 4096;            // ranking blocks of 4096 pixels (RB_SHIFT)
    w.ntiles = (size_t)B * ((H + TH - 1) / TH) * ((W + TW - 1) / TW);
    size_t off = 0;
    auto take = [&](size_t bytes) { size_t o = off; off = bd_align_up(off + bytes, 256); return (char *)base + o; };
    w.counters = (uint32_t *)take(64 * sizeof(uint32_t));
    w.maskbuf = (uint8_t *)take(P);
    w.edges = (uint32_t *)take(w.ntiles * EDGE_WORDS * sizeof(uint32_t));
    w.recidx = (uint32_t *)take(w.nblk2 * sizeof(uint32_t));
    w.keptbits = (uint32_t *)take(w.NWk * sizeof(uint32_t));
    w.blkcnt = (uint32_t *)take((w.NB + 8) * sizeof(uint32_t));
    w.zero_bytes = (size_t)((char *)w.blkcnt - (char *)w.keptbits) + (w.NB + 1) * sizeof(uint32_t);
    w.blkprefix = (uint32_t *)take((w.NB + 8) * sizeof(uint32_t));
    w.wx_tab = (float *)take((size_t)W * 4 * sizeof(float));
    w.wy_tab = (double *)take((size_t)H * 4 * sizeof(double));
    w.i0_tab = (int32_t *)take((size_t)W * sizeof(int32_t));
    w.j0_tab = (int32_t *)take((size_t)H * sizeof(int32_t));
    w.rec = (Rec *)take(w.nblk2 * sizeof(Rec));
    w.total = off;
    return off;
}

// ------------------------------------------------------------------------------------------------ mask
// (the same float32 rule as K3 / the fused kernel: spl_above)
__global__ void k_make_mask(const float *sub, const float *rms, size_t n4, float k_d, uint8_t *mask) {
    size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n4) return;
    float4 s = reinterpret_cast<const float4 *>(sub)[i], r = reinterpret_cast<const float4 *>(rms)[i];
    uint32_t m = 0;
    m |= spl_above(s.x, r.x, k_d) ? 1u : 0u;
    m |= spl_above(s.y, r.y, k_d) ? 1u << 8 : 0u;
    m |= spl_above(s.z, r.z, k_d) ? 1u << 16 : 0u;
    m |= spl_above(s.w, r.w, k_d) ? 1u << 24 : 0u;
    reinterpret_cast<uint32_t *>(mask)[i] = m;
}

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

// 4 mask bytes (non-zero = foreground) -> 4 bits
__device__ __forceinline__ uint32_t bytes_to_nibble(uint32_t v) {
    const uint32_t nz = ((((v & 0x7F7F7F7Fu) + 0x7F7F7F7Fu) | v) & 0x80808080u) >> 7;   // bits 0, 8, 16, 24
    return (nz * 0x00204081u >> 21) & 0xFu;
}

// ------------------------------------------------------------------------------------------------ spline weights
// The x-weights of a column and the y-weights of a row are the same for every tile that contains them: computed once
// per call (fused mode) with the functions K3 uses, instead of 5 float64 polynomial evaluations per thread per tile.
__global__ void k_spline_tabs(int H, int W, int mh, int mw, float *wx_tab, double *wy_tab, int32_t *i0_tab, int32_t *j0_tab) {
    // launched programmatically dependent: the weights are computed while the predecessor on the stream drains, the stores wait
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    int i0 = 0, j0 = 0;
    float wx[4] = {0.f, 0.f, 0.f, 0.f};
    double wy[4] = {0.0, 0.0, 0.0, 0.0};
    if (t < W) { i0 = spl_cell_of(t, mw); spl_x_weights(t, mw, i0, wx); }
    if (t < H) { j0 = spl_cell_of(t, mh); spl_y_weights(t, mh, j0, wy); }
    bd_pdl_wait();
    if (t < W) {
        reinterpret_cast<float4 *>(wx_tab)[t] = make_float4(wx[0], wx[1], wx[2], wx[3]);
        i0_tab[t] = i0;
    }
    if (t < H) {
        wy_tab[4 * t + 0] = wy[0]; wy_tab[4 * t + 1] = wy[1]; wy_tab[4 * t + 2] = wy[2]; wy_tab[4 * t + 3] = wy[3];
        j0_tab[t] = j0;
    }
}

// ------------------------------------------------------------------------------------------------ K4a
// shared-memory union-find on lab[]: a root's low 13 bits point to itself, union by minimum index
__device__ __forceinline__ uint32_t sm_find(volatile uint32_t *par, uint32_t x) {
    uint32_t p = par[x] & IDX_MASK;
    while (p != x) { x = p; p = par[x] & IDX_MASK; }
    return x;
}
// bits of columns x-1, x, x+1 of a bit row (bit 0 = x-1); x in [0, TW)
__device__ __forceinline__ uint32_t get3(const uint32_t *row, int x) {
    const int q = x + 31, j = q >> 5;
    return __funnelshift_r(row[j], row[j + 1], q & 31) & 7u;
}

#ifdef K4_TIMING
__device__ unsigned long long g_k4_t[16];
#define K4_T(i) do { if (tid == 0) { const long long t_ = clock64(); atomicAdd(&g_k4_t[i], (unsigned long long)(t_ - t_prev)); t_prev = t_; } } while (0)
#else
#define K4_T(i) do { } while (0)
#endif

struct K4Args {
    const uint8_t *mask;
    const float *sub;
    int H, W, min_area, vec16, use_tma;
    int32_t *labels;
    uint32_t *edges;
    Rec *rec;
    uint32_t *recidx;
    uint32_t *counters;
    int skip_isolated;   // min_area > 1: pixels without any foreground neighbour never enter the list
    // fused mode (FUSED = true): phase A evaluates the background / RMS splines itself (step a3) instead of reading a mask
    const float *img;
    const double *bcoef, *rcoef;
    float *sub_out, *bkg, *rms;
    uint8_t *mask_out;
    int mh, mw, ny, nx, uniform;
    float k_d;
    const float *wx_tab;
    const double *wy_tab;
    const int32_t *i0_tab, *j0_tab;
};

constexpr int SM_LAB = 0;
constexpr int SM_LIST = SM_LAB + TPX * 4;
constexpr int SM_BITS = SM_LIST + TPX * 2;
constexpr int SM_ROOTS = SM_BITS + 1600;              // BROWS * BWORDS * 4 = 1584, padded
constexpr int SM_MISC = SM_ROOTS + (TPX / 4) * 2;     // at most one root per 2x2 block
constexpr int K4_SMEM = SM_MISC + 16 * 4;

// one 32-pixel word of a mask row: the 32 raw bytes (0 outside the frame), loaded first and converted later so
// that a thread's main and halo loads are in flight together
struct Raw8 { uint32_t v[8]; };
__device__ __forceinline__ Raw8 load_mask_raw(const K4Args &a, size_t fbase, int y, int x) {
    Raw8 r;
#pragma unroll
    for (int k = 0; k < 8; ++k) r.v[k] = 0;
    if (y >= 0 && y < a.H && x < a.W) {
        const uint8_t *src = a.mask + fbase + (size_t)y * a.W + x;
        if (a.vec16) {
            if (x + 16 <= a.W) {
                const uint4 v = __ldg(reinterpret_cast<const uint4 *>(src));
                r.v[0] = v.x; r.v[1] = v.y; r.v[2] = v.z; r.v[3] = v.w;
            }
            if (x + 32 <= a.W) {
                const uint4 v = __ldg(reinterpret_cast<const uint4 *>(src + 16));
                r.v[4] = v.x; r.v[5] = v.y; r.v[6] = v.z; r.v[7] = v.w;
            }
        } else {
#pragma unroll
            for (int k = 0; k < 8; ++k)
                if (x + 4 * k < a.W) r.v[k] = __ldg(reinterpret_cast<const uint32_t *>(src + 4 * k));
        }
    }
    return r;
}
__device__ __forceinline__ uint32_t raw_to_word(const Raw8 &r) {
    uint32_t word = 0;
#pragma unroll
    for (int k = 0; k < 8; ++k) word |= bytes_to_nibble(r.v[k]) << (4 * k);
    return word;
}

template <bool FUSED>
__global__ void __launch_bounds__(K4_NT, 4) k4a_tile_label(const __grid_constant__ CUtensorMap tmap_lab,
                                                               const __grid_constant__ CUtensorMap tmap_img, K4Args a) {
    extern __shared__ __align__(128) unsigned char sm[];
    uint32_t *lab = reinterpret_cast<uint32_t *>(sm + SM_LAB);
    uint16_t *list = reinterpret_cast<uint16_t *>(sm + SM_LIST);
    uint32_t(*bits)[BWORDS] = reinterpret_cast<uint32_t(*)[BWORDS]>(sm + SM_BITS);
    uint16_t *roots = reinterpret_cast<uint16_t *>(sm + SM_ROOTS);   // the tile-local roots (filled in D)
    uint32_t *wsum = reinterpret_cast<uint32_t *>(sm + SM_MISC);   // [0..7] warp totals, [8] n_rec, [9] g_base, [10] n_roots

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int frame = blockIdx.z;
    const int x0 = blockIdx.x * TW, y0 = blockIdx.y * TH;
    const int H = a.H, W = a.W;
    const size_t fbase = (size_t)frame * H * W;
    const size_t tile = ((size_t)frame * gridDim.y + blockIdx.y) * gridDim.x + blockIdx.x;
    const int row_w = tid >> 2, w_w = tid & 3;   // this thread's bit word of the tile
#ifdef K4_TIMING
    long long t_prev = clock64();
#endif

    // ---- A: zero the label tile, mask bytes -> bit rows with a 1-pixel halo -------------------------------
    if (tid == 0) { wsum[8] = 0; wsum[10] = 0; }
    if constexpr (FUSED) {
        // the tile's image pixels: one TMA bulk-tensor load into the label buffer (unused until phase B), in flight
        // while the spline table is built; rows / columns past the frame edge are zero-filled and never used
        if (tid == 0) {
            const uint32_t bar = smem_u32(&wsum[12]);
            asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(bar));
            asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
            asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"((uint32_t)(TPX * 4)) : "memory");
            asm volatile(
                "cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];"
                ::"r"(smem_u32(lab)), "l"(&tmap_img), "r"(x0), "r"(y0), "r"(frame), "r"(bar)
                : "memory");
        }
    } else {
#pragma unroll
        for (int k = 0; k < TPX / 4 / K4_NT; ++k) reinterpret_cast<uint4 *>(lab)[k * K4_NT + tid] = make_uint4(0, 0, 0, 0);
    }
    uint32_t M;
    if constexpr (FUSED) {
        // ---- A (fused): step a3 for the tile and its 1-pixel halo: spline table -> sub, bkg, rms (written out),
        //      threshold bits.  Arithmetic shared with K3 (spline_eval.cuh): bit-identical maps and mask.
        float *table = reinterpret_cast<float *>(sm + SM_LIST);   // aliases the list (built in B)
        const double *bc = a.bcoef + (size_t)frame * a.ny * a.nx, *rc = a.rcoef + (size_t)frame * a.ny * a.nx;
        const int ry0 = max(y0 - 1, 0), ry1 = min(y0 + TH, H - 1), cx0 = max(x0 - 1, 0), cx1 = min(x0 + TW, W - 1);
        const int i0_first = spl_cell_of(cx0, a.mw), n_i0 = spl_cell_of(cx1, a.mw) - i0_first + 1;
        const int row_stride = n_i0 * SPL_ENT;
        const int xt = x0 + 4 * lane;                // this thread's four columns
        const bool col_ok = xt < W;
        const float *img = a.img + fbase;
        // halo loads first (the tile itself arrives by TMA): the halo row of warps 0 / 1, one halo-column pixel
        const int yh = warp == 0 ? y0 - 1 : y0 + TH;   // halo row of warp 0 / warp 1
        const bool hrow_ok = warp < 2 && col_ok && yh >= 0 && yh < H;
        float4 pixh = make_float4(0.f, 0.f, 0.f, 0.f);
        if (hrow_ok) pixh = __ldg(reinterpret_cast<const float4 *>(img + (size_t)yh * W + xt));
        const int hcy = y0 - 1 + (tid >> 1), hcx = (tid & 1) ? x0 + TW : x0 - 1;   // halo-column pixel of threads < 2 * BROWS
        const bool hcol_ok = tid < 2 * BROWS && hcy >= 0 && hcy < H && hcx >= 0 && hcx < W;
        float pixc = 0.f;
        if (hcol_ok) pixc = __ldg(img + (size_t)hcy * W + hcx);
        // table: one entry per (row, grid cell) of the halo region
        const int n_ent = (ry1 - ry0 + 1) * n_i0;
        for (int e = tid; e < n_ent; e += K4_NT) {
            const int r = e / n_i0, ii = e - r * n_i0, y = ry0 + r;
            double wy[4];
            wy[0] = __ldg(a.wy_tab + 4 * y); wy[1] = __ldg(a.wy_tab + 4 * y + 1); wy[2] = __ldg(a.wy_tab + 4 * y + 2); wy[3] = __ldg(a.wy_tab + 4 * y + 3);
            spl_table_entry_w(bc, rc, a.ny, a.nx, __ldg(a.j0_tab + y), wy, i0_first + ii, table + (size_t)e * SPL_ENT);
        }
        float wx[4][4];
        int ent_off[4];
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            const int xq = min(xt + q, W - 1);
            const float4 wv = __ldg(reinterpret_cast<const float4 *>(a.wx_tab) + xq);
            wx[q][0] = wv.x; wx[q][1] = wv.y; wx[q][2] = wv.z; wx[q][3] = wv.w;
            ent_off[q] = (__ldg(a.i0_tab + xq) - i0_first) * SPL_ENT;
        }
        K4_T(11);
        __syncthreads();
        K4_T(12);
        auto eval4 = [&](const float4 &px, int y, float o_sub[4], float o_bkg[4], float o_rms[4]) -> uint32_t {
            const float *trow = table + (size_t)(y - ry0) * row_stride;
            const float in[4] = {px.x, px.y, px.z, px.w};
            uint32_t nib = 0;
            float4 t0, t1;
            float t8;
            if (a.uniform) {
                const float *t = trow + ent_off[0];
                t0 = *reinterpret_cast<const float4 *>(t); t1 = *reinterpret_cast<const float4 *>(t + 4); t8 = t[8];
            }
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                if (!a.uniform) {
                    const float *t = trow + ent_off[q];
                    t0 = *reinterpret_cast<const float4 *>(t); t1 = *reinterpret_cast<const float4 *>(t + 4); t8 = t[8];
                }
                nib |= (spl_pixel(t0, t1, t8, wx[q], in[q], a.k_d, o_sub[q], o_bkg[q], o_rms[q]) ? 1u : 0u) << q;
            }
            return nib;
        };
        auto put_bits = [&](uint32_t nib, int hr) {   // 8 lanes x 4 bits -> one word of bit row hr
            uint32_t word = nib << (4 * (lane & 7));
            word |= __shfl_xor_sync(0xffffffffu, word, 1);
            word |= __shfl_xor_sync(0xffffffffu, word, 2);
            word |= __shfl_xor_sync(0xffffffffu, word, 4);
            if ((lane & 7) == 0) bits[hr][1 + (lane >> 3)] = word;
        };
        {   // wait for the tile
            const uint32_t bar = smem_u32(&wsum[12]);
            uint32_t done = 0;
            while (!done)
                asm volatile("{ .reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], 0; selp.u32 %0, 1, 0, p; }"
                             : "=r"(done) : "r"(bar) : "memory");
        }
        K4_T(13);
        const float4 *tile4 = reinterpret_cast<const float4 *>(lab);
#pragma unroll 2
        for (int k = 0; k < TH / 8; ++k) {
            const int row = warp + 8 * k, y = y0 + row;
            uint32_t nib = 0;
            if (col_ok && y < H) {
                float o_sub[4], o_bkg[4], o_rms[4];
                nib = eval4(tile4[row * (TW / 4) + lane], y, o_sub, o_bkg, o_rms);
                const size_t off = fbase + (size_t)y * W + xt;
                *reinterpret_cast<float4 *>(a.sub_out + off) = make_float4(o_sub[0], o_sub[1], o_sub[2], o_sub[3]);
                if (a.bkg) __stcs(reinterpret_cast<float4 *>(a.bkg + off), make_float4(o_bkg[0], o_bkg[1], o_bkg[2], o_bkg[3]));
                if (a.rms) __stcs(reinterpret_cast<float4 *>(a.rms + off), make_float4(o_rms[0], o_rms[1], o_rms[2], o_rms[3]));
                if (a.mask_out)
                    __stcs(reinterpret_cast<uint32_t *>(a.mask_out + off),
                           (nib & 1u) | (nib & 2u) << 7 | (nib & 4u) << 14 | (nib & 8u) << 21);
            }
            put_bits(nib, row + 1);
        }
        K4_T(14);
        if (warp < 2) {   // halo rows: bits only
            uint32_t nib = 0;
            if (hrow_ok) {
                float o_sub[4], o_bkg[4], o_rms[4];
                nib = eval4(pixh, yh, o_sub, o_bkg, o_rms);
            }
            put_bits(nib, warp == 0 ? 0 : BROWS - 1);
        }
        if (tid < 2 * BROWS) {   // halo columns: one pixel each
            uint32_t bit = 0;
            if (hcol_ok) {
                const int i0 = __ldg(a.i0_tab + hcx);
                const float4 wv = __ldg(reinterpret_cast<const float4 *>(a.wx_tab) + hcx);
                const float wxc[4] = {wv.x, wv.y, wv.z, wv.w};
                float o_s, o_b, o_r;
                const float *t = table + (size_t)(hcy - ry0) * row_stride + (i0 - i0_first) * SPL_ENT;
                bit = spl_pixel(*reinterpret_cast<const float4 *>(t), *reinterpret_cast<const float4 *>(t + 4), t[8], wxc, pixc, a.k_d,
                                o_s, o_b, o_r) ? 1u : 0u;
            }
            bits[tid >> 1][(tid & 1) ? 5 : 0] = (tid & 1) ? bit : bit << 31;
        }
        __syncthreads();   // every pixel of the tile buffer has been consumed: it becomes the label array
#pragma unroll
        for (int k = 0; k < TPX / 4 / K4_NT; ++k) reinterpret_cast<uint4 *>(lab)[k * K4_NT + tid] = make_uint4(0, 0, 0, 0);
        M = bits[row_w + 1][1 + w_w];
    } else {
        const Raw8 raw_m = load_mask_raw(a, fbase, y0 + row_w, x0 + 32 * w_w);
        Raw8 raw_h;
        uint32_t hbit = 0;
        const int hcol = tid - 8;   // halo column element (if 0 <= hcol < 2 * BROWS)
        if (tid < 8) {              // halo rows y0-1 and y0+TH
            raw_h = load_mask_raw(a, fbase, y0 - 1 + (tid < 4 ? 0 : BROWS - 1), x0 + 32 * (tid & 3));
        } else if (hcol < BROWS * 2) {   // halo columns x0-1 and x0+TW
            const int y = y0 - 1 + (hcol >> 1), x = (hcol & 1) ? x0 + TW : x0 - 1;
            if (y >= 0 && y < H && x >= 0 && x < W) hbit = __ldg(a.mask + fbase + (size_t)y * W + x) ? 1u : 0u;
        }
        M = raw_to_word(raw_m);
        bits[row_w + 1][1 + w_w] = M;
        if (tid < 8) bits[tid < 4 ? 0 : BROWS - 1][1 + (tid & 3)] = raw_to_word(raw_h);
        else if (hcol < BROWS * 2) bits[hcol >> 1][(hcol & 1) ? 5 : 0] = (hcol & 1) ? hbit : hbit << 31;

    }
    __syncthreads();
    K4_T(0);

    // ---- B: compact list of the foreground pixels that have a foreground neighbour (raster order); parent =
    //      start of the horizontal run.  A pixel whose 3x3 neighbourhood (halo included) is empty is a complete
    //      component of one pixel: it gets its label here and, when min_area > 1, takes no further part.
    uint32_t Mc = M;
    if (a.skip_isolated && M) {
        const uint32_t *ru = bits[row_w], *rm = bits[row_w + 1], *rd = bits[row_w + 2];
        const int j = 1 + w_w;
        const uint32_t U = ru[j], D = rd[j];
        const uint32_t nb = U | (U << 1) | (ru[j - 1] >> 31) | (U >> 1) | (ru[j + 1] << 31) |
                            D | (D << 1) | (rd[j - 1] >> 31) | (D >> 1) | (rd[j + 1] << 31) |
                            (M << 1) | (rm[j - 1] >> 31) | (M >> 1) | (rm[j + 1] << 31);
        Mc = M & nb;
        uint32_t iso = M & ~nb;
        const int gbase_px = (y0 + row_w) * W + x0 + w_w * 32 + 1;
        while (iso) {
            const int i = __ffs(iso) - 1;
            iso &= iso - 1;
            lab[row_w * TW + w_w * 32 + i] = (uint32_t)(gbase_px + i);
        }
    }
    uint32_t incl = __popc(Mc);
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const uint32_t t = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += t;
    }
    if (lane == 31) wsum[warp] = incl;
    __syncthreads();
    K4_T(1);

    // border bit rows / columns for the seam merge
    {
        uint32_t *e = a.edges + tile * EDGE_WORDS;
        if (tid < 4) e[tid] = bits[1][1 + tid];
        else if (tid < 8) e[tid] = bits[TH][1 + tid - 4];
        if (warp == 1 || warp == 2) {
            const int row = tid - 32;
            const uint32_t bl = __ballot_sync(0xffffffffu, bits[row + 1][1] & 1u);
            const uint32_t br = __ballot_sync(0xffffffffu, bits[row + 1][4] >> 31);
            if (lane == 0) { e[8 + warp - 1] = bl; e[10 + warp - 1] = br; }
        }
    }
    uint32_t pos = incl - __popc(Mc);
    int n = 0;
#pragma unroll
    for (int k = 0; k < K4_NT / 32; ++k) {
        const uint32_t t = wsum[k];
        if (k < warp) pos += t;
        n += (int)t;
    }
    if (Mc) {
        const uint32_t prevbit = w_w ? bits[row_w + 1][w_w] >> 31 : 0u;   // left neighbour word of the same tile row
        const uint32_t pbase = (uint32_t)(row_w * TW + w_w * 32);
        uint32_t m = Mc, cur = 0;
        while (m) {
            const int i = __ffs(m) - 1;
            m &= m - 1;
            const uint32_t p = pbase + i;
            const bool cont = i ? ((M >> (i - 1)) & 1u) : prevbit;
            if (!cont) cur = p;
            else if (i == 0) cur = p - 1;
            lab[p] = cur;
            list[pos++] = (uint16_t)p;
        }
    }
    __syncthreads();
    K4_T(2);

    if (n > 0) {
        // sub of this thread's first list entry: requested now, used in F (hides the DRAM latency behind C..E)
        float I_pre = 0.f;
        if (tid < n) {
            const uint32_t p = list[tid];
            const float *ps = a.sub + fbase + (size_t)(y0 + (int)(p >> 7)) * W + x0 + (int)(p & 127);
            I_pre = FUSED ? __ldcg(ps) : __ldg(ps);   // fused: sub was written by this CTA in phase A (L2-coherent load)
        }
        // ---- C: vertical / diagonal links inside the tile.  Rules (w, a, b, c = W, NW, N, NE neighbours):
        //      b && !w -> N;  !b && a && !w -> NW;  !b && c -> NE.  In-tile bits only (a halo pixel never prunes an
        //      in-tile link): the tile-local components are then exactly the components of the tile's own mask, so
        //      two tile-local roots never share a 2x2 block.
        constexpr uint32_t NONE = 0xFFFFFFFFu;
        for (int e = tid; e < n; e += K4_NT) {
            const uint32_t p = list[e];
            const int r = (int)(p >> 7), x = (int)(p & 127);
            if (r == 0) continue;
            const uint32_t u3 = get3(bits[r], x), m3 = get3(bits[r + 1], x);
            const bool w = (m3 & 1u) && x > 0, na = u3 & 1u, nb = u3 & 2u, nc = u3 & 4u;
            uint32_t t0 = NONE, t1 = NONE;
            if (nb) { if (!w) t0 = p - TW; }
            else {
                if (na && !w && x > 0) t0 = p - TW - 1;
                if (nc && x < TW - 1) t1 = p - TW + 1;
            }
#pragma unroll 1
            for (int k = 0; k < 2; ++k) {
                uint32_t ub = k ? t1 : t0;
                if (ub == NONE) continue;
                uint32_t ua = p;
                for (;;) {
                    ua = sm_find(lab, ua);
                    ub = sm_find(lab, ub);
                    if (ua == ub) break;
                    if (ua < ub) { const uint32_t t = ua; ua = ub; ub = t; }
                    const uint32_t old = atomicMin(&lab[ua], ub);
                    if (old == ua) break;
                    ua = old;
                }
            }
        }
        __syncthreads();
        K4_T(3);
        // ---- D: flatten; pixel counts (one atomic per run of equal roots in the list); ring flags -------------
        for (int e0 = 0; e0 < n; e0 += K4_NT) {
            const int e = e0 + tid;
            uint32_t r = 0xFFFF0000u | lane;
            bool ring = false, isroot = false;
            uint32_t p = 0;
            if (e < n) {
                p = list[e];
                r = sm_find(lab, p);
                if (r != p) lab[p] = r;
                isroot = r == p;
                const int row = (int)(p >> 7), x = (int)(p & 127);
                if (row == 0 || row == TH - 1 || x == 0 || x == TW - 1) {
                    const uint32_t u3 = get3(bits[row], x), m3 = get3(bits[row + 1], x), d3 = get3(bits[row + 2], x);
                    uint32_t out = 0;
                    if (row == 0) out |= u3;
                    if (row == TH - 1) out |= d3;
                    if (x == 0) out |= (u3 | m3 | d3) & 1u;
                    if (x == TW - 1) out |= (u3 | m3 | d3) & 4u;
                    ring = out != 0;
                }
            }
            const uint32_t prev = __shfl_up_sync(0xffffffffu, r, 1);
            const bool head = lane == 0 || prev != r;
            const uint32_t hm = __ballot_sync(0xffffffffu, head);
            const uint32_t rest = lane == 31 ? 0u : hm & ~((2u << lane) - 1u);
            const int tail = rest ? __ffs(rest) - 2 : 31;
            if (e < n && head) atomicAdd(&lab[r], (uint32_t)(tail - lane + 1) << CNT_SHIFT);
            if (ring) atomicOr(&lab[r], F_RING);
            const uint32_t rb = __ballot_sync(0xffffffffu, isroot);
            if (rb) {   // the warp's roots go to the root list with one shared atomic
                uint32_t base = 0;
                if (lane == __ffs(rb) - 1) base = atomicAdd(&wsum[10], (uint32_t)__popc(rb));
                base = __shfl_sync(0xffffffffu, base, __ffs(rb) - 1);
                if (isroot) roots[base + __popc(rb & ((1u << lane) - 1u))] = (uint16_t)p;
            }
        }
        __syncthreads();
        K4_T(4);
        const int nroots = (int)wsum[10];
        // ---- E: components that can matter get a record slot; the tile reserves a contiguous range of records -
        for (int e = tid; e < nroots; e += K4_NT) {
            const uint32_t p = roots[e];
            const uint32_t wd = lab[p];
            const int cnt = (int)((wd >> CNT_SHIFT) & CNT_MASK);
            if (cnt >= a.min_area || (wd & F_RING)) {
                const uint32_t slot = atomicAdd(&wsum[8], 1u);
                lab[p] = p | (slot << CNT_SHIFT) | F_REC | (wd & F_RING);
            }
        }
        __syncthreads();
        K4_T(5);
        const int nrec = (int)wsum[8];
        if (nrec > 0) {
            if (tid == 0) wsum[9] = atomicAdd(a.counters + 0, (uint32_t)nrec);
            __syncthreads();
            K4_T(6);
            const uint32_t gbase = wsum[9];
            for (int e = tid; e < nroots; e += K4_NT) {   // zeroed records + the root -> record index
                const uint32_t p = roots[e];
                const uint32_t wd = lab[p];
                if (!(wd & F_REC)) continue;
                const uint32_t slot = (wd >> CNT_SHIFT) & 0x7FFu;
                const int gy = y0 + (int)(p >> 7), gx = x0 + (int)(p & 127);
                a.recidx[((size_t)frame * ((H + 1) / 2) + (gy >> 1)) * (W / 2) + (gx >> 1)] = gbase + slot;
                uint4 *dst = reinterpret_cast<uint4 *>(a.rec + gbase + slot);
                dst[0] = make_uint4(0, 0, 0, 0); dst[1] = make_uint4(0, 0, 0, 0); dst[2] = make_uint4(0, 0, 0, 0);
                dst[3] = make_uint4(0, 0, (uint32_t)(gy * W + gx), (uint32_t)frame);                            // peak, root, frame
                dst[4] = make_uint4(0, 0x7FFFFFFFu, 0xFFFFFFFFu, 0x7FFFFFFFu);    // npix (summed in F), xmin, xmax, ymin
                dst[5] = make_uint4(0xFFFFFFFFu, 0, 0, 0);                                                      // ymax, merged
            }
            __syncthreads();
            K4_T(7);
            // ---- F: partial sums of the recorded components.  One segment = the consecutive list entries of one
            //      (component, row); segmented shuffle reduction, then the head lane adds the run to the record.
            for (int e0 = 0; e0 < n; e0 += K4_NT) {
                const int e = e0 + tid;
                uint32_t key = 0xFFFF0000u | lane, r = 0, rslot = 0;
                int x = 0, row = 0;
                double S0 = 0.0, S1 = 0.0, S2 = 0.0;
                u64 pk = 0;
                bool in = false;
                if (e < n) {
                    const uint32_t p = list[e];
                    const uint32_t own = lab[p];
                    const bool isroot = (own & IDX_MASK) == p;
                    r = isroot ? p : own;
                    const uint32_t rw = isroot ? own : lab[r];
                    in = rw & F_REC;
                    rslot = (rw >> CNT_SHIFT) & 0x7FFu;
                    if (in) {
                        row = (int)(p >> 7); x = (int)(p & 127);
                        key = (r << 6) | (uint32_t)row;
                        const int gidx = (y0 + row) * W + x0 + x;
                        const float I = e0 == 0 ? I_pre : (FUSED ? __ldcg(a.sub + fbase + (size_t)gidx) : __ldg(a.sub + fbase + (size_t)gidx));
                        const double dx = (double)(x - (int)(r & 127));
                        S0 = (double)I; S1 = S0 * dx; S2 = S1 * dx;
                        pk = ((u64)f32_to_key(I) << 32) | (u64)(0xFFFFFFFFu - (uint32_t)gidx);
                    }
                }
                if (!__any_sync(0xffffffffu, in)) continue;
                const uint32_t prev = __shfl_up_sync(0xffffffffu, key, 1);
                const bool head = lane == 0 || prev != key;
                const uint32_t hm = __ballot_sync(0xffffffffu, head);
                const uint32_t rest = lane == 31 ? 0u : hm & ~((2u << lane) - 1u);
                const int tail = rest ? __ffs(rest) - 2 : 31;
                const int maxlen = __reduce_max_sync(0xffffffffu, in ? tail - lane : 0);
                for (int d = 1; d <= maxlen; d <<= 1) {
                    const double o0 = __shfl_down_sync(0xffffffffu, S0, d), o1 = __shfl_down_sync(0xffffffffu, S1, d);
                    const double o2 = __shfl_down_sync(0xffffffffu, S2, d);
                    const u64 opk = __shfl_down_sync(0xffffffffu, pk, d);
                    if (lane + d <= tail) { S0 += o0; S1 += o1; S2 += o2; pk = opk > pk ? opk : pk; }
                }
                const int xlast = __shfl_sync(0xffffffffu, x, tail);
                if (in && head) {
                    const int ry = (int)(r >> 7);
                    Rec *T = a.rec + gbase + rslot;
                    const double dy = (double)(row - ry);
                    atomicAdd(&T->f, S0);
                    atomicAdd(&T->sx, S1);
                    atomicAdd(&T->sy, dy * S0);
                    atomicAdd(&T->sxx, S2);
                    atomicAdd(&T->syy, dy * dy * S0);
                    atomicAdd(&T->sxy, dy * S1);
                    atomicMax(&T->peak, pk);
                    atomicAdd(&T->npix, tail - lane + 1);
                    atomicMin(&T->xmin, x0 + x); atomicMax(&T->xmax, x0 + xlast);
                    atomicMin(&T->ymin, y0 + row); atomicMax(&T->ymax, y0 + row);
                }
            }
        }
        __syncthreads();
        K4_T(8);
        // ---- G: parents -> labels (1 + raster index of the tile-local root) ------------------------------------
        for (int e = tid; e < n; e += K4_NT) {
            const uint32_t p = list[e];
            const uint32_t own = lab[p];
            const uint32_t r = (own & IDX_MASK) == p ? p : own;
            lab[p] = (uint32_t)((y0 + (int)(r >> 7)) * W + x0 + (int)(r & 127) + 1);
        }
    }

    // ---- H: the label tile leaves shared memory ----------------------------------------------------------------
    if (a.use_tma) {
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        __syncthreads();
        K4_T(9);
        if (tid == 0) {
            asm volatile("cp.async.bulk.tensor.3d.global.shared::cta.tile.bulk_group [%0, {%1, %2, %3}], [%4];" ::"l"(&tmap_lab),
                         "r"(x0), "r"(y0), "r"(frame), "r"(smem_u32(lab))
                         : "memory");
            asm volatile("cp.async.bulk.commit_group;" ::: "memory");
            asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
            K4_T(10);
        }
    } else {
        __syncthreads();
        for (int i = tid; i < TPX / 4; i += K4_NT) {
            const int r = i >> 5, c = (i & 31) * 4;
            if (y0 + r < H && x0 + c < W)
                __stcg(reinterpret_cast<uint4 *>(a.labels + fbase + (size_t)(y0 + r) * W + x0 + c), reinterpret_cast<const uint4 *>(lab)[i]);
        }
    }
}

// ------------------------------------------------------------------------------------------------ K4b
// global union-find on the label array of one frame: L[a] = 1 + parent of a; a root has L[a] = a + 1
__device__ __forceinline__ int g_find(const int32_t *L, int a) {
    for (;;) {
        int p = __ldcg(L + a) - 1;
        if (p == a) return a;
        a = p;
    }
}
__device__ __forceinline__ void g_union(int32_t *L, int a, int b) {
    {   // first hop of both walks together (two independent misses instead of two in a row)
        const int pa = __ldcg(L + a) - 1, pb = __ldcg(L + b) - 1;
        a = pa; b = pb;
    }
    for (;;) {
        a = g_find(L, a);
        b = g_find(L, b);
        if (a == b) return;
        if (a < b) { int t = a; a = b; b = t; }
        int old = atomicMin(L + a, b + 1);
        if (old == a + 1) return;   // a was a root and now hangs under b
        a = old - 1;
    }
}

// One WARP per (tile, unit): units 0..3 = the four 32-pixel words of the tile's top row against the bottom
// row of the tile above (links N, NW, NE of row-0 pixels); units 4, 5 = the two 32-row words of the tile's left
// column against the right column of the tile to the left (link W of column-0 pixels, NW of column-0 pixels and
// NE of the left tile's last column, rows >= 1 of the tile; row 0 belongs to units 0..3).  The conditions are
// the pruned rules of K4a evaluated on the true neighbour bits; every lane computes the three task words, lane l
// executes bit l of each (the unions are chains of dependent L2 accesses: one per lane, in parallel).
__global__ void __launch_bounds__(256) k4b_seams(const uint32_t *edges, int32_t *labels, int H, int W, int TX, int TY,
                                                 size_t n_units) {
    bd_pdl_wait();
    bd_pdl_trigger();
    const size_t u = ((size_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (u >= n_units) return;
    const int unit = (int)(u % 6);
    const size_t tile = u / 6;
    const int tx = (int)(tile % TX), ty = (int)((tile / TX) % TY);
    const size_t frame = tile / ((size_t)TX * TY);
    int32_t *L = labels + frame * (size_t)H * W;
    const uint32_t *E = edges + tile * EDGE_WORDS;
    const int x0 = tx * TW, y0 = ty * TH;
    if (unit < 4) {
        if (ty == 0) return;
        const int k = unit;
        const uint32_t M = E[k];
        if (!M) return;
        const uint32_t *EU = E - (size_t)TX * EDGE_WORDS;   // tile above
        const uint32_t Uc = EU[4 + k];
        uint32_t lc, rc, ml;
        if (k > 0) { lc = EU[4 + k - 1] >> 31; ml = E[k - 1] >> 31; }
        else if (tx > 0) { lc = (EU - EDGE_WORDS)[4 + 3] >> 31; ml = (E - EDGE_WORDS)[3] >> 31; }
        else { lc = 0; ml = 0; }
        if (k < 3) rc = EU[4 + k + 1] & 1u;
        else if (tx + 1 < TX) rc = (EU + EDGE_WORDS)[4] & 1u;
        else rc = 0;
        const uint32_t na = (Uc << 1) | lc, nb = Uc, nc = (Uc >> 1) | (rc << 31), wb = (M << 1) | ml;
        const uint32_t tN = M & ~wb & nb, tNW = M & ~wb & ~nb & na, tNE = M & ~nb & nc;
        const int pbase = y0 * W + x0 + 32 * k;
        const int p = pbase + lane;   // lane l owns bit l
        if ((tN >> lane) & 1u) g_union(L, p, p - W);
        if ((tNW >> lane) & 1u) g_union(L, p, p - W - 1);
        if ((tNE >> lane) & 1u) g_union(L, p, p - W + 1);
    } else {
        if (tx == 0) return;
        const int h = unit - 4;
        const uint32_t *EA = E - EDGE_WORDS;   // tile to the left
        const uint32_t R = E[8 + h], Lc = EA[10 + h];
        if (!(R | Lc)) return;
        const uint32_t cl = h ? EA[10] >> 31 : 0u, cr = h ? E[8] >> 31 : 0u;
        const uint32_t Lup = (Lc << 1) | cl, Rup = (R << 1) | cr;
        const uint32_t rows = h ? 0xFFFFFFFFu : 0xFFFFFFFEu;   // row 0 of the tile: units 0..3
        const uint32_t tW = R & Lc, tNW = R & ~Lc & ~Rup & Lup & rows, tNE = Lc & ~Lup & Rup & rows;
        const int ybase = y0 + 32 * h;
        const int p = (ybase + lane) * W + x0;   // lane l owns row l of the word
        if ((tW >> lane) & 1u) g_union(L, p, p - 1);
        if ((tNW >> lane) & 1u) g_union(L, p, p - W - 1);
        if ((tNE >> lane) & 1u) g_union(L, p - 1, p - 1 - W + 1);
    }
}

// ------------------------------------------------------------------------------------------------ K5
__device__ __forceinline__ size_t blk2_of(int frame, int r, int H, int W) {
    const int y = r / W, x = r - y * W;
    return ((size_t)frame * ((H + 1) / 2) + (y >> 1)) * (W / 2) + (x >> 1);
}

// K5m: records whose tile-local root was linked under another root are added to the final root's record and
// their pixels relabelled.  One thread per record (records are contiguous: coalesced reads).  A changed record
// with a small bounding box is served by its own thread; larger boxes are served by the whole warp.
constexpr int K5M_SOLO_AREA = 48;

__device__ __forceinline__ void k5m_merge_into(const Rec *c, Rec *T, int cr, int cR, int W) {
    const int yc = cr / W, xc = cr - yc * W, yR = cR / W, xR = cR - yR * W;
    const double ox = (double)(xc - xR), oy = (double)(yc - yR);
    const double f = c->f, sx = c->sx, sy = c->sy;
    atomicAdd(&T->f, f);
    atomicAdd(&T->sx, sx + f * ox);
    atomicAdd(&T->sy, sy + f * oy);
    atomicAdd(&T->sxx, c->sxx + 2.0 * ox * sx + ox * ox * f);
    atomicAdd(&T->syy, c->syy + 2.0 * oy * sy + oy * oy * f);
    atomicAdd(&T->sxy, c->sxy + ox * sy + oy * sx + ox * oy * f);
    atomicMax(&T->peak, c->peak);
    atomicAdd(&T->npix, c->npix);
    atomicMin(&T->xmin, c->xmin); atomicMax(&T->xmax, c->xmax);
    atomicMin(&T->ymin, c->ymin); atomicMax(&T->ymax, c->ymax);
}

__global__ void __launch_bounds__(256) k5m_merge_relabel(const uint32_t *counters, Rec *rec, const uint32_t *recidx,
                                                         int32_t *labels, int H, int W) {
    bd_pdl_wait();
    bd_pdl_trigger();
    const uint32_t n = counters[0];
    const int lane = threadIdx.x & 31;
    const size_t HW = (size_t)H * W;
    for (size_t base = ((size_t)blockIdx.x * blockDim.x + threadIdx.x) & ~(size_t)31; base < n; base += (size_t)gridDim.x * blockDim.x) {
        const size_t i = base + lane;
        int r = 0, R = 0, frame = 0, bx = 0, by = 0, bw = 0, bh = 0;
        if (i < n) {
            const int4 v = *reinterpret_cast<const int4 *>(&rec[i].peak);       // peak (2 words), root, frame
            const int4 bb = *reinterpret_cast<const int4 *>(&rec[i].npix);      // npix, xmin, xmax, ymin
            r = v.z; frame = v.w;
            bx = bb.y; bw = bb.z - bb.y + 1; by = bb.w; bh = rec[i].ymax - bb.w + 1;
            R = g_find(labels + (size_t)frame * HW, r);
        }
        const bool changed = R != r;
        const bool solo = changed && bw * bh <= K5M_SOLO_AREA;
        if (changed) {
            int32_t *L = labels + (size_t)frame * HW;
            rec[i].merged = 1;
            k5m_merge_into(rec + i, rec + recidx[blk2_of(frame, R, H, W)], r, R, W);
            L[r] = R + 1;
            if (solo) {   // 8 loads in flight, then the stores (a load-compare-store loop waits for every load)
                const int old = r + 1, neu = R + 1, area = bw * bh;
                for (int k0 = 0; k0 < area; k0 += 8) {
                    int32_t *q[8];
                    int v[8];
#pragma unroll
                    for (int k = 0; k < 8; ++k) {
                        const int kk = min(k0 + k, area - 1), yy = kk / bw;
                        q[k] = L + (size_t)(by + yy) * W + bx + (kk - yy * bw);
                        v[k] = __ldcg(q[k]);
                    }
#pragma unroll
                    for (int k = 0; k < 8; ++k)
                        if (v[k] == old) *q[k] = neu;
                }
            }
        }
        uint32_t todo = __ballot_sync(0xffffffffu, changed && !solo);
        while (todo) {   // large boxes: the warp relabels them together
            const int j = __ffs(todo) - 1;
            todo &= todo - 1;
            const int cr = __shfl_sync(0xffffffffu, r, j), cR = __shfl_sync(0xffffffffu, R, j), cf = __shfl_sync(0xffffffffu, frame, j);
            const int cbx = __shfl_sync(0xffffffffu, bx, j), cby = __shfl_sync(0xffffffffu, by, j);
            const int cbw = __shfl_sync(0xffffffffu, bw, j), cbh = __shfl_sync(0xffffffffu, bh, j);
            int32_t *L = labels + (size_t)cf * HW;
            const int old = cr + 1, neu = cR + 1;
            for (int k = lane; k < cbw * cbh; k += 32) {
                const int yy = k / cbw, xx = k - yy * cbw;
                int32_t *q = L + (size_t)(cby + yy) * W + cbx + xx;
                if (*q == old) *q = neu;
            }
        }
    }
}

// K5k: final roots with npix >= min_area -> bit in the per-pixel bitmap, count in the 4096-pixel block
__global__ void __launch_bounds__(256) k5k_mark_kept(const uint32_t *counters, const Rec *rec, int H, int W, int min_area,
                                                     uint32_t *keptbits, uint32_t *blkcnt) {
    bd_pdl_wait();
    bd_pdl_trigger();
    const uint32_t n = counters[0];
    const size_t HW = (size_t)H * W;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        const Rec *c = rec + i;
        if (c->merged || c->npix < min_area) continue;
        const size_t g = (size_t)c->frame * HW + c->root;
        atomicOr(&keptbits[g >> 5], 1u << (g & 31));
        atomicAdd(&blkcnt[g >> RB_SHIFT], 1u);
    }
}

// K5f: catalogue records in ascending (frame, label) order; per-frame counts
__global__ void __launch_bounds__(256) k5f_finalize(const uint32_t *counters, const Rec *rec, int B, int H, int W,
                                                    int min_area, const uint32_t *keptbits, const uint32_t *blkprefix,
                                                    bd_source *cat, int64_t cap, int64_t *n_sources) {
    bd_pdl_wait();
    const uint32_t n = counters[0];
    const size_t HW = (size_t)H * W;
    const size_t t0 = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t0 < (size_t)B)
        n_sources[t0] = (int64_t)kept_rank(keptbits, blkprefix, (t0 + 1) * HW) - (int64_t)kept_rank(keptbits, blkprefix, t0 * HW);
    if (!cat || cap <= 0) return;
    for (size_t i = t0; i < n; i += (size_t)gridDim.x * blockDim.x) {
        const Rec *c = rec + i;
        if (c->merged || c->npix < min_area) continue;
        const Rec a = *c;
        const int r = a.root, frame = a.frame;
        const uint32_t rank = kept_rank(keptbits, blkprefix, (size_t)frame * HW + r);
        if ((int64_t)rank >= cap) continue;
        const int yr = r / W, xr = r - yr * W;
        bd_source s;
        s.frame = frame;
        s.label = r + 1;
        s.npix = a.npix;
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
        cat[rank] = s;
    }
}

}  // namespace

size_t k45_workspace_bytes(int B, int H, int W, int64_t cat_capacity) {
    (void)cat_capacity;   // the record table is sized by the frame, not by the catalogue
    Ws w;
    return carve(w, nullptr, B, H, W) + 256;
}

// the fused tile kernel keeps its spline table (66 rows x cells x 48 B) in the 16 KiB the list occupies later
// and stages the image tile with a TMA box of TW x TH pixels
bool k45_can_fuse(const bd_ctx *ctx, int H, int W, int mesh_w) {
    return ctx->encode_tiled && W >= TW && H >= TH && BROWS * ((TW + 2) / mesh_w + 2) * SPL_ENT * (int)sizeof(float) <= TPX * 2;
}
// the P bytes of the detect workspace that hold a mask when the caller passes none
uint8_t *k45_ws_maskbuf(void *d_ws, int B, int H, int W) {
    Ws w;
    carve(w, (char *)bd_align_up((size_t)d_ws, 256), B, H, W);
    return w.maskbuf;
}

int k45_launch(bd_ctx *ctx, const float *d_sub, const float *d_rms, const uint8_t *d_mask, int B, int H, int W,
               double detect_k, int min_area, int32_t *d_labels, bd_source *d_cat, int64_t cat_capacity,
               int64_t *d_n_sources, void *d_ws, size_t ws_bytes, cudaStream_t st, const K45Fused *fz) {
    Ws w;
    char *base = (char *)bd_align_up((size_t)d_ws, 256);
    size_t need = carve(w, base, B, H, W);
    if ((size_t)(base - (char *)d_ws) + need > ws_bytes)
        return bd_set_error(ctx, BD_EWORKSPACE, "detect workspace: need %zu bytes, got %zu", need + 256, ws_bytes);
    const size_t P = w.P;

    const uint8_t *mask = d_mask;
    if (!mask && !fz) {
        size_t n4 = P / 4;
        k_make_mask<<<(unsigned)((n4 + 255) / 256), 256, 0, st>>>(d_sub, d_rms, n4, (float)detect_k, w.maskbuf);
        mask = w.maskbuf;
    }

    const int TX = (W + TW - 1) / TW, TY = (H + TH - 1) / TH;
    K4Args a;
    memset(&a, 0, sizeof(a));
    a.mask = mask; a.sub = d_sub; a.H = H; a.W = W; a.min_area = min_area;
    a.vec16 = (W % 16 == 0 && ((uintptr_t)mask & 15) == 0) ? 1 : 0;
    a.labels = d_labels; a.edges = w.edges; a.rec = w.rec; a.recidx = w.recidx; a.counters = w.counters;
    a.skip_isolated = min_area > 1 ? 1 : 0;
    if (fz) {
        a.img = fz->img; a.bcoef = fz->bcoef; a.rcoef = fz->rcoef;
        a.sub_out = fz->sub; a.bkg = fz->bkg; a.rms = fz->rms; a.mask_out = fz->mask;
        a.mh = fz->mh; a.mw = fz->mw; a.ny = (H + fz->mh - 1) / fz->mh; a.nx = (W + fz->mw - 1) / fz->mw;
        a.uniform = fz->mw % 8 == 0 ? 1 : 0;
        a.k_d = (float)detect_k;
        a.sub = fz->sub;
        a.wx_tab = w.wx_tab; a.wy_tab = w.wy_tab; a.i0_tab = w.i0_tab; a.j0_tab = w.j0_tab;
        const int nt_tabs = W > H ? W : H;
        BD_CUDA_CHECK(ctx, bd_launch_pdl(k_spline_tabs, dim3((nt_tabs + 255) / 256), dim3(256), 0, st, H, W, fz->mh, fz->mw, w.wx_tab, w.wy_tab,
                                         w.i0_tab, w.j0_tab));
    }
    BD_CUDA_CHECK(ctx, cudaMemsetAsync(w.counters, 0, 64 * sizeof(uint32_t), st));
    BD_CUDA_CHECK(ctx, cudaMemsetAsync(w.keptbits, 0, w.zero_bytes, st));
    a.use_tma = (W >= TW && H >= TH && ctx->encode_tiled) ? 1 : 0;
    CUtensorMap tmap;
    memset(&tmap, 0, sizeof(tmap));
    if (a.use_tma) {
        cuuint64_t dims[3] = {(cuuint64_t)W, (cuuint64_t)H, (cuuint64_t)B};
        cuuint64_t strides[2] = {(cuuint64_t)W * sizeof(int32_t), (cuuint64_t)W * H * sizeof(int32_t)};
        cuuint32_t box[3] = {TW, TH, 1};
        cuuint32_t estr[3] = {1, 1, 1};
        CUresult r = ctx->encode_tiled(&tmap, CU_TENSOR_MAP_DATA_TYPE_INT32, 3, (void *)d_labels, dims, strides, box, estr,
                                       CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                                       CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (r != CUDA_SUCCESS) return bd_set_error(ctx, BD_ECUDA, "cuTensorMapEncodeTiled(labels) failed (%d)", (int)r);
    }
    if (ctx->dbg_ev0) cudaEventRecord(ctx->dbg_ev0, st);
    CUtensorMap tmap_img;
    memset(&tmap_img, 0, sizeof(tmap_img));
    if (fz) {
        cuuint64_t dims[3] = {(cuuint64_t)W, (cuuint64_t)H, (cuuint64_t)B};
        cuuint64_t strides[2] = {(cuuint64_t)W * sizeof(float), (cuuint64_t)W * H * sizeof(float)};
        cuuint32_t box[3] = {TW, TH, 1};
        cuuint32_t estr[3] = {1, 1, 1};
        CUresult r = ctx->encode_tiled(&tmap_img, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, (void *)fz->img, dims, strides, box, estr,
                                       CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                                       CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (r != CUDA_SUCCESS) return bd_set_error(ctx, BD_ECUDA, "cuTensorMapEncodeTiled(img) failed (%d)", (int)r);
    }
    if (fz) {
        BD_CUDA_CHECK(ctx, cudaFuncSetAttribute(k4a_tile_label<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, K4_SMEM));
        k4a_tile_label<true><<<dim3(TX, TY, B), K4_NT, K4_SMEM, st>>>(tmap, tmap_img, a);
    } else {
        BD_CUDA_CHECK(ctx, cudaFuncSetAttribute(k4a_tile_label<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, K4_SMEM));
        k4a_tile_label<false><<<dim3(TX, TY, B), K4_NT, K4_SMEM, st>>>(tmap, tmap_img, a);
    }
    if (ctx->dbg_ev1) cudaEventRecord(ctx->dbg_ev1, st);
    if (TX > 1 || TY > 1) {
        const size_t n_units = w.ntiles * 6;
        BD_CUDA_CHECK(ctx, bd_launch_pdl(k4b_seams, dim3((unsigned)((n_units + 7) / 8)), dim3(256), 0, st, w.edges, d_labels, H, W, TX, TY, n_units));
    }
    const int nb = ctx->num_sms * 32;
    // the five small kernels of the tail are launched programmatically dependent: each becomes resident while its predecessor
    // drains and waits (griddepcontrol.wait) for it to complete
    BD_CUDA_CHECK(ctx, bd_launch_pdl(k5m_merge_relabel, dim3(nb), dim3(256), 0, st, w.counters, w.rec, w.recidx, d_labels, H, W));
    BD_CUDA_CHECK(ctx, bd_launch_pdl(k5k_mark_kept, dim3(nb), dim3(256), 0, st, w.counters, w.rec, H, W, min_area, w.keptbits, w.blkcnt));
    BD_CUDA_CHECK(ctx, bd_launch_pdl(k5s_scan_blocks, dim3(1), dim3(1024), 0, st, w.blkcnt, w.NB, w.blkprefix, w.counters + 1));
    const int nbf = nb * 256 >= B ? nb : (B + 255) / 256;
    BD_CUDA_CHECK(ctx, bd_launch_pdl(k5f_finalize, dim3(nbf), dim3(256), 0, st, w.counters, w.rec, B, H, W, min_area, w.keptbits, w.blkprefix,
                                     d_cat, cat_capacity, d_n_sources));
    BD_CUDA_CHECK(ctx, cudaGetLastError());
    return BD_OK;
}

#ifdef K4_TIMING
extern "C" int bd_debug_k4_timing(unsigned long long *out16, int reset) {
    unsigned long long z[16] = {0};
    if (cudaMemcpyFromSymbol(out16, g_k4_t, sizeof(z)) != cudaSuccess) return BD_ECUDA;
    if (reset && cudaMemcpyToSymbol(g_k4_t, z, sizeof(z)) != cudaSuccess) return BD_ECUDA;
    return BD_OK;
}
#endif

// diagnostics (not part of include/bkgdet.h): CUDA events (cudaEvent_t as void*, 0 = off) that the next calls record
// on their stream immediately before and after the tile kernel, so a caller can time that kernel alone
extern "C" int bd_debug_tile_kernel_events(bd_ctx *ctx, void *ev_before, void *ev_after) {
    if (!ctx) return BD_EINVAL;
    ctx->dbg_ev0 = (cudaEvent_t)ev_before;
    ctx->dbg_ev1 = (cudaEvent_t)ev_after;
    return BD_OK;
}
