// K8: stamp-wise spatially varying convolution of the template and image subtraction.
// PAPER.md:126-147, eqs. 8-10: K(u,v) = sum_n a_n(x,y) K_n(u,v), K_n = exp(-(u^2+v^2)/(2 sigma_k^2)) u^i v^j, R (x) K = I + B;
// "We then allocate a thread block for each stamp of the convolution kernel size; by default, the size of the stamp is 21 x 21
// pixels.  The convolution computation is performed within shared memory, with each thread processing a single pixel in the
// stamp, utilizing the preloaded convolution kernel."  Readings C1-C7; the kernel fit itself is out of scope.
//
// Why this is a CUDA-core stencil and not a tcgen05 contraction.  The kernel of a stamp is fixed inside the stamp (C3), so a
// pixel costs S^2 = 441 multiply-adds: 37.5 G FMA on a 9216 x 9232 frame.  Tensor cores need an operand shared by many output
// rows; the only shared operand is the BASIS (im2col(R) [pixels x 441] times K_n [441 x N]), which multiplies the work by
// the N = 49 basis kernels: 1.84 T FMA = 3.7 TFLOP, i.e. 4.4 ms in one tf32 pass at half the measured bf16 peak (and tf32's
// 10-bit mantissa on ~1000-ADU pixels needs a 3-way split for float32-grade products: ~13 ms), against ~1 ms of plain FFMA at
// 128 FMA/clk/SM.  Per stamp the product is a matrix-VECTOR product (441 outputs x 441 taps, N = 1): nothing for an MMA to
// reuse.  So: float32 FFMA with register blocking, bound by the FMA pipe (bench.py reports it as "alu").
//
// k8_moment_kernels (tiny): the a_n are polynomials in the normalised stamp-centre coordinates (C2), so
//   K(u,v; xc,yc) = sum_t xh^p yh^q M_t(u,v),   M_t = sum_n c[n,t] K_n   -- n_sp (6) "moment kernels" per frame, built once
// in float64 (exp, powers) and rounded to float32, stored flipped (the convolution becomes a correlation with MF).
// k8_stamp_conv<HW> (HW = 10, the paper's 21 x 21): a CTA owns NSX x NSY stamps; the template patch (tile + halo, zero
// outside the frame, C4) sits in shared memory with a pitch = 1 mod 32, the stamps' kernels (6 FMAs per tap from the M_t)
// beside it.  One THREAD per (stamp, stamp row): 21 accumulators, and per kernel row one 41-pixel segment of the patch and
// the 21 taps in registers -> 441 FFMA for 41 + 6 shared-memory loads (9:1; the paper's thread-per-pixel mapping is 1:2 and
// would be bound by shared-memory bandwidth at ~8 ms).  Lanes are consecutive rows, so the segment loads are conflict-free.
// The results leave through shared memory so that diff = I + B - conv is read and written in coalesced rows.
// k8_stamp_conv_generic: any other half-width (<= 15), one thread per pixel, same arithmetic order per pixel is NOT promised
// (float32 sums differ in the last bits between the two kernels).
#include "common.cuh"

namespace {

constexpr int K8_MAX_SP = 15;   // spatial terms (order <= 4)
constexpr int K8_MAX_N = 160;   // basis kernels

struct K8Basis {   // by value: the basis definition (C1)
    int hw, n_gauss, degree[4], spatial_order, bg_order, n_basis, n_sp, n_bg;
    double sigma[4];
};

__host__ __device__ inline int k8_npoly(int o) { return (o + 1) * (o + 2) / 2; }

// M[b][t][w][m] = sum_n c[b][n][t] K_n(u = hw - m, v = hw - w), float64 -> float32.  One thread per (frame, tap).
__global__ void __launch_bounds__(256) k8_moment_kernels(K8Basis bs, const double *kcoef, int B, float *M) {
    const int S = 2 * bs.hw + 1, taps = S * S;
    const int idx = blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= B * taps) return;
    const int b = idx / taps, tap = idx - b * taps, w = tap / S, m = tap - w * S;
    const double u = (double)(bs.hw - m), v = (double)(bs.hw - w);
    double acc[K8_MAX_SP];
    for (int t = 0; t < bs.n_sp; ++t) acc[t] = 0.0;
    const double *c = kcoef + (size_t)b * bs.n_basis * bs.n_sp;
    int n = 0;
    for (int g = 0; g < bs.n_gauss; ++g) {
        const double e = exp(-(u * u + v * v) / (2.0 * bs.sigma[g] * bs.sigma[g]));
        double ui = 1.0;
        for (int i = 0; i <= bs.degree[g]; ++i) {
            double vj = 1.0;
            for (int j = 0; j <= bs.degree[g] - i; ++j) {
                const double val = e * ui * vj;
                for (int t = 0; t < bs.n_sp; ++t) acc[t] = fma(c[(size_t)n * bs.n_sp + t], val, acc[t]);
                ++n;
                vj *= v;
            }
            ui *= u;
        }
    }
    for (int t = 0; t < bs.n_sp; ++t) M[((size_t)b * bs.n_sp + t) * taps + tap] = (float)acc[t];
}

// xh^p yh^q for the terms t = (p, q), p = 0..o, q = 0..o - p (C2), in float64
__device__ __forceinline__ void k8_poly_terms(int order, double xh, double yh, double *out) {
    int t = 0;
    double xp = 1.0;
    for (int p = 0; p <= order; ++p) {
        double yq = 1.0;
        for (int q = 0; q <= order - p; ++q) { out[t++] = xp * yq; yq *= yh; }
        xp *= xh;
    }
}

// B(x, y) = sum_t bc[t] xh^p yh^q (C2), float64, no local array; the coordinates use reciprocals computed once per thread
__device__ __forceinline__ double k8_bg(const double *bc, int order, double xh, double yh) {
    double bg = 0.0, xp = 1.0;
    int t = 0;
    for (int p = 0; p <= order; ++p) {
        double yq = 1.0;
        for (int q = 0; q <= order - p; ++q) { bg = fma(__ldg(bc + t), xp * yq, bg); ++t; yq *= yh; }
        xp *= xh;
    }
    return bg;
}

struct K8Args {
    const float *ref, *img, *M;
    const double *bgcoef;     // [B][n_bg]
    float *diff, *conv;       // conv may be null
    int H, W, hw, spatial_order, bg_order, n_sp, n_bg;
};

template <int HW, int NSX, int NSY>
struct K8Cfg {
    static constexpr int S = 2 * HW + 1;
    static constexpr int NT = ((S * NSX * NSY + 31) / 32) * 32;
    static constexpr int PW = NSX * S + 2 * HW, PH = NSY * S + 2 * HW;          // patch incl. halo
    static constexpr int PITCH = ((PW + 30) / 32) * 32 + 1;                      // = 1 mod 32: lanes = rows -> distinct banks
    static constexpr int KP = (S + 3) / 4 * 4;                                   // padded kernel row (128-bit loads)
    static constexpr int PATCH_FLOATS = (PH * PITCH + 3) / 4 * 4;                // the kernels behind it are read as float4
    static constexpr int KERN_FLOATS = NSX * NSY * S * KP;
    static constexpr int SMEM = (PATCH_FLOATS + KERN_FLOATS + NSX * NSY * 16) * 4;   // + the stamps' spatial terms
};

template <int HW, int NSX, int NSY>
__global__ void __launch_bounds__(K8Cfg<HW, NSX, NSY>::NT, 2) k8_stamp_conv(K8Args a) {
    using C = K8Cfg<HW, NSX, NSY>;
    constexpr int S = C::S, PITCH = C::PITCH, KP = C::KP;
    extern __shared__ __align__(16) float sm8[];
    float *patch = sm8;                           // [PH][PITCH]; after the main loop: the conv tile [NSY*S][PITCH]
    float *kern = sm8 + C::PATCH_FLOATS;          // [stamp][S][KP], flipped
    const int tid = threadIdx.x, frame = blockIdx.z;
    const int H = a.H, W = a.W;
    const size_t fbase = (size_t)frame * H * W;
    const int tx0 = blockIdx.x * NSX * S, ty0 = blockIdx.y * NSY * S;   // first output pixel of the tile

    // ---- template patch (tile + halo), zero outside the frame (C4) ---------------------------------------------------------
    for (int i = tid; i < C::PH * C::PW; i += C::NT) {
        const int r = i / C::PW, c = i - r * C::PW;
        const int y = ty0 - HW + r, x = tx0 - HW + c;
        patch[r * PITCH + c] = (y >= 0 && y < H && x >= 0 && x < W) ? __ldg(a.ref + fbase + (size_t)y * W + x) : 0.0f;
    }
    // ---- the stamps' kernels: K = sum_t xh^p yh^q M_t at the stamp centre (C2, C3), already flipped ------------------------
    float *sterm = kern + C::KERN_FLOATS;         // [stamp][16]: xh^p yh^q of the stamp centres (float64 -> float32)
    if (tid < NSX * NSY) {
        const int sx = blockIdx.x * NSX + tid % NSX, sy = blockIdx.y * NSY + tid / NSX;
        const double xh = (2.0 * (double)(sx * S + HW) - (double)(W - 1)) / (double)W;
        const double yh = (2.0 * (double)(sy * S + HW) - (double)(H - 1)) / (double)H;
        double term[K8_MAX_SP];
        k8_poly_terms(a.spatial_order, xh, yh, term);
        for (int t = 0; t < a.n_sp; ++t) sterm[tid * 16 + t] = (float)term[t];
    }
    __syncthreads();
    {
        const float *M = a.M + (size_t)frame * a.n_sp * S * S;
        for (int i = tid; i < NSX * NSY * S * S; i += C::NT) {
            const int s = i / (S * S), tap = i - s * S * S;
            float k = 0.0f;
            for (int t = 0; t < a.n_sp; ++t) k = fmaf(sterm[s * 16 + t], __ldg(M + (size_t)t * S * S + tap), k);
            kern[(s * S + tap / S) * KP + tap % S] = k;
        }
    }
    __syncthreads();

    // ---- one thread per (stamp, stamp row): acc[x] += KF[w][m] * patch[row + w][x0 + x + m] --------------------------------
    const int s = tid / S, ry = tid - s * S;
    const bool active = s < NSX * NSY;
    float acc[S];
#pragma unroll
    for (int x = 0; x < S; ++x) acc[x] = 0.0f;
    if (active) {
        const int lx0 = (s % NSX) * S, ly = (s / NSX) * S + ry;   // patch coordinates of this row's first needed pixel
        const float *prow = patch + ly * PITCH + lx0;
        const float *krow = kern + s * S * KP;
#pragma unroll 1
        for (int w = 0; w < S; ++w) {
            float seg[S + 2 * HW], kf[KP];
#pragma unroll
            for (int j = 0; j < S + 2 * HW; ++j) seg[j] = prow[w * PITCH + j];
#pragma unroll
            for (int j = 0; j < KP / 4; ++j) {
                const float4 q = *reinterpret_cast<const float4 *>(krow + w * KP + 4 * j);
                kf[4 * j] = q.x; kf[4 * j + 1] = q.y; kf[4 * j + 2] = q.z; kf[4 * j + 3] = q.w;
            }
#pragma unroll
            for (int m = 0; m < S; ++m)
#pragma unroll
                for (int x = 0; x < S; ++x) acc[x] = fmaf(kf[m], seg[x + m], acc[x]);
        }
    }
    __syncthreads();   // the patch is dead: it becomes the conv tile
    if (active) {
        float *orow = patch + ((s / NSX) * S + ry) * PITCH + (s % NSX) * S;
#pragma unroll
        for (int x = 0; x < S; ++x) orow[x] = acc[x];
    }
    __syncthreads();
    // ---- diff = I + B - conv (C5), coalesced rows -------------------------------------------------------------------------
    const double *bc = a.bgcoef + (size_t)frame * a.n_bg;
    const double inv_w = 1.0 / (double)W, inv_h = 1.0 / (double)H;
    for (int i = tid; i < NSY * S * NSX * S; i += C::NT) {
        const int r = i / (NSX * S), c = i - r * (NSX * S);
        const int y = ty0 + r, x = tx0 + c;
        if (y >= H || x >= W) continue;
        const float cv = patch[r * PITCH + c];
        const double bg = k8_bg(bc, a.bg_order, (double)(2 * x - (W - 1)) * inv_w, (double)(2 * y - (H - 1)) * inv_h);
        const size_t off = fbase + (size_t)y * W + x;
        a.diff[off] = (float)(((double)__ldg(a.img + off) + bg) - (double)cv);
        if (a.conv) a.conv[off] = cv;
    }
}

// any half-width <= 15: one CTA per stamp, one thread per pixel (the paper's mapping), patch and kernel in shared memory
__global__ void __launch_bounds__(1024) k8_stamp_conv_generic(K8Args a) {
    extern __shared__ __align__(16) float sm8[];
    const int hw = a.hw, S = 2 * hw + 1, PW = S + 2 * hw;
    float *patch = sm8, *kern = sm8 + PW * PW;
    const int tid = threadIdx.x, nt = blockDim.x, frame = blockIdx.z;
    const int H = a.H, W = a.W;
    const size_t fbase = (size_t)frame * H * W;
    const int sx = blockIdx.x, sy = blockIdx.y, tx0 = sx * S, ty0 = sy * S;
    for (int i = tid; i < PW * PW; i += nt) {
        const int r = i / PW, c = i - r * PW, y = ty0 - hw + r, x = tx0 - hw + c;
        patch[i] = (y >= 0 && y < H && x >= 0 && x < W) ? __ldg(a.ref + fbase + (size_t)y * W + x) : 0.0f;
    }
    {
        const float *M = a.M + (size_t)frame * a.n_sp * S * S;
        const double xh = (2.0 * (double)(sx * S + hw) - (double)(W - 1)) / (double)W;
        const double yh = (2.0 * (double)(sy * S + hw) - (double)(H - 1)) / (double)H;
        double term[K8_MAX_SP];
        k8_poly_terms(a.spatial_order, xh, yh, term);
        for (int tap = tid; tap < S * S; tap += nt) {
            float k = 0.0f;
            for (int t = 0; t < a.n_sp; ++t) k = fmaf((float)term[t], __ldg(M + (size_t)t * S * S + tap), k);
            kern[tap] = k;
        }
    }
    __syncthreads();
    const double *bc = a.bgcoef + (size_t)frame * a.n_bg;
    const double inv_w = 1.0 / (double)W, inv_h = 1.0 / (double)H;
    for (int i = tid; i < S * S; i += nt) {
        const int r = i / S, c = i - r * S, y = ty0 + r, x = tx0 + c;
        if (y >= H || x >= W) continue;
        float acc = 0.0f;
        for (int w = 0; w < S; ++w)
            for (int m = 0; m < S; ++m) acc = fmaf(kern[w * S + m], patch[(r + w) * PW + c + m], acc);
        const double bg = k8_bg(bc, a.bg_order, (double)(2 * x - (W - 1)) * inv_w, (double)(2 * y - (H - 1)) * inv_h);
        const size_t off = fbase + (size_t)y * W + x;
        a.diff[off] = (float)(((double)__ldg(a.img + off) + bg) - (double)acc);
        if (a.conv) a.conv[off] = acc;
    }
}

}  // namespace

static int k8_basis(const bd_conv_params *p, K8Basis *bs) {
    if (!p || p->half_width < 1 || p->half_width > 15 || p->n_gauss < 1 || p->n_gauss > 4 || p->spatial_order < 0 ||
        p->spatial_order > 4 || p->bg_order < 0 || p->bg_order > 4)
        return BD_EINVAL;
    bs->hw = p->half_width; bs->n_gauss = p->n_gauss; bs->spatial_order = p->spatial_order; bs->bg_order = p->bg_order;
    bs->n_basis = 0;
    for (int g = 0; g < 4; ++g) {
        bs->degree[g] = g < p->n_gauss ? p->degree[g] : 0;
        bs->sigma[g] = g < p->n_gauss ? p->sigma[g] : 1.0;
        if (g < p->n_gauss) {
            if (p->degree[g] < 0 || p->degree[g] > 8 || !(p->sigma[g] > 0.0)) return BD_EINVAL;
            bs->n_basis += k8_npoly(p->degree[g]);
        }
    }
    bs->n_sp = k8_npoly(p->spatial_order); bs->n_bg = k8_npoly(p->bg_order);
    return bs->n_basis <= K8_MAX_N ? BD_OK : BD_EINVAL;
}

int k8_num_basis(const bd_conv_params *p) {
    K8Basis bs;
    return k8_basis(p, &bs) == BD_OK ? bs.n_basis : -1;
}

size_t k8_workspace_bytes(int B, const bd_conv_params *p) {
    K8Basis bs;
    if (k8_basis(p, &bs) != BD_OK) return 0;
    const int S = 2 * bs.hw + 1;
    return 256 + (size_t)B * bs.n_sp * S * S * sizeof(float);
}

int k8_launch(bd_ctx *ctx, const float *d_ref, const float *d_img, int B, int H, int W, const bd_conv_params *p,
              const double *d_kcoef, const double *d_bgcoef, float *d_diff, float *d_conv, void *d_ws, cudaStream_t st) {
    K8Basis bs;
    if (k8_basis(p, &bs) != BD_OK) return bd_set_error(ctx, BD_EINVAL, "bad convolution parameters");
    const int S = 2 * bs.hw + 1;
    float *M = (float *)bd_align_up((size_t)d_ws, 256);
    k8_moment_kernels<<<(B * S * S + 255) / 256, 256, 0, st>>>(bs, d_kcoef, B, M);
    K8Args a;
    a.ref = d_ref; a.img = d_img; a.M = M; a.bgcoef = d_bgcoef; a.diff = d_diff; a.conv = d_conv;
    a.H = H; a.W = W; a.hw = bs.hw; a.spatial_order = bs.spatial_order; a.bg_order = bs.bg_order; a.n_sp = bs.n_sp; a.n_bg = bs.n_bg;
    if (bs.hw == 10) {
        using C = K8Cfg<10, 6, 2>;
        BD_CUDA_CHECK(ctx, cudaFuncSetAttribute(k8_stamp_conv<10, 6, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, C::SMEM));
        dim3 grid((W + 6 * S - 1) / (6 * S), (H + 2 * S - 1) / (2 * S), B);
        k8_stamp_conv<10, 6, 2><<<grid, C::NT, C::SMEM, st>>>(a);
    } else {
        const int PW = S + 2 * bs.hw;
        const size_t smem = (size_t)(PW * PW + S * S) * sizeof(float);
        int nt = (S * S + 31) / 32 * 32;
        if (nt > 1024) nt = 1024;
        dim3 grid((W + S - 1) / S, (H + S - 1) / S, B);
        if (grid.y > 65535) return bd_set_error(ctx, BD_EUNSUPPORTED, "frame too tall for this stamp size");
        k8_stamp_conv_generic<<<grid, nt, smem, st>>>(a);
    }
    BD_CUDA_CHECK(ctx, cudaGetLastError());
    return BD_OK;
}
