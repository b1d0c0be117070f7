// Internal declarations shared by the .cu files of libbkgdet (sm_100a only).
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>
#include <string.h>

#include "../../include/bkgdet.h"

struct bd_ctx {
    int device;
    int num_sms;
    size_t smem_optin;
    char err[512];
    int k1_force_slow;   // diagnostics: K1 skips its fast path
    cudaEvent_t dbg_ev0, dbg_ev1;   // diagnostics: recorded around the tile kernel of detect_sources / bkg_subtract_detect
    // cuTensorMapEncodeTiled, fetched through the runtime (no -lcuda link dependency)
    CUresult (*encode_tiled)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                             const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                             CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
    // bd_run_host cache
    void *host_dev;
    size_t host_dev_bytes;
    cudaStream_t host_stream, copy_stream;
    cudaEvent_t host_ev[8];   // BD_HOST_CHUNKS: one per chunk of the frame that bd_run_host copies
};
#define BD_HOST_CHUNKS 8

int bd_set_error(bd_ctx *ctx, int code, const char *fmt, ...);

// Every entry point that touches the device runs with ctx->device current and puts the caller's device back.
struct BdDeviceGuard {
    int prev = -1;
    bool changed = false;
    cudaError_t err;
    explicit BdDeviceGuard(const bd_ctx *ctx) {
        err = cudaGetDevice(&prev);
        if (err == cudaSuccess && prev != ctx->device) {
            err = cudaSetDevice(ctx->device);
            changed = err == cudaSuccess;
        }
    }
    ~BdDeviceGuard() { if (changed) cudaSetDevice(prev); }
};
#define BD_BIND_DEVICE(ctx)                                                                             \
    BdDeviceGuard _bd_guard(ctx);                                                                       \
    if (_bd_guard.err != cudaSuccess)                                                                   \
        return bd_set_error((ctx), BD_ECUDA, "cannot bind CUDA device %d: %s", (ctx)->device, cudaGetErrorString(_bd_guard.err))

#define BD_CUDA_CHECK(ctx, expr)                                                                       \
    do {                                                                                               \
        cudaError_t _e = (expr);                                                                       \
        if (_e != cudaSuccess)                                                                         \
            return bd_set_error((ctx), BD_ECUDA, "%s:%d %s: %s", __FILE__, __LINE__, #expr,            \
                                cudaGetErrorString(_e));                                               \
    } while (0)

static inline size_t bd_align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

// ---- launchers implemented in the kernel files ---------------------------------------------------------
struct K1Plan {
    int cluster;        // CTAs per mesh (1, 2, 4, 8)
    int slab_rows;      // mesh rows held by one CTA
    int threads;        // threads per CTA
    size_t smem_bytes;  // dynamic shared memory per CTA
    int use_tma;
    int tailcap;        // capacity of the tail-pixel list (team total)
    int stream;         // 1: no slab, one CTA per mesh sweeps global memory (meshes larger than one CTA's slab)
    size_t slab_bytes;  // shared memory in front of the fixed part: the slab, or room for the sort arrays
};
int k1_plan(const bd_ctx *ctx, int mesh_h, int mesh_w, K1Plan *plan);
// d_ws: k1_workspace_bytes() of device memory (the worklist of meshes the warp-per-mesh kernel hands to the general path)
size_t k1_workspace_bytes(int B, int ny, int nx);
// d_bad / px / d_n_valid: the background variants (bad-pixel mask, validity rules, valid-pixel counts); all may be null
int k1_launch(bd_ctx *ctx, const float *d_img, int B, int H, int W, const bd_bkg_params *p, double *d_bkg_raw,
              double *d_rms_raw, double *d_median, double *d_mean, int32_t *d_n_kept, void *d_ws, cudaStream_t st,
              const uint8_t *d_bad = nullptr, const bd_bkgx_params *px = nullptr, int32_t *d_n_valid = nullptr);

// doubles of scratch K2 needs per (frame, grid): the Thomas factors of both directions
static inline __host__ __device__ size_t k2_scratch_per_grid(int ny, int nx) { return 2 * ((size_t)ny + (size_t)nx); }
int k2_launch(bd_ctx *ctx, const double *d_bkg_raw, const double *d_rms_raw, int B, int ny, int nx, int fh, int fw,
              float *d_bkg_mesh, float *d_rms_mesh, double *d_bkg_coef, double *d_rms_coef, double *d_scratch,
              cudaStream_t st);

// B3: invalid (NaN) cells filled from their valid neighbours; d_valid may be null
int k2f_launch(bd_ctx *ctx, const double *d_bkg_raw, const double *d_rms_raw, int B, int ny, int nx, double *d_bkg_filled,
               double *d_rms_filled, uint8_t *d_valid, cudaStream_t st);

// B5: out = (bad0 != 0) | dilate(det, grow); det and bad0 may be null (zeros)
int k7_dilate_or(bd_ctx *ctx, const uint8_t *d_det, const uint8_t *d_bad0, int B, int H, int W, int grow, uint8_t *d_out,
                 cudaStream_t st);

// d_sub may be null here (bkg_iterate wants the mask only)
int k3_launch(bd_ctx *ctx, const float *d_img, int B, int H, int W, int mh, int mw, const double *d_bkg_coef,
              const double *d_rms_coef, double detect_k, float *d_sub, float *d_bkg, float *d_rms, uint8_t *d_mask,
              cudaStream_t st);

size_t k45_workspace_bytes(int B, int H, int W, int64_t cat_capacity);
// fused step a3 + a4 + a5: the tile kernel evaluates the splines itself (no mask / sub input)
struct K45Fused {
    const float *img;
    const double *bcoef, *rcoef;
    float *sub, *bkg, *rms;   // sub required; bkg, rms may be null
    uint8_t *mask;            // may be null
    int mh, mw;
};
bool k45_can_fuse(const bd_ctx *ctx, int H, int W, int mesh_w);
uint8_t *k45_ws_maskbuf(void *d_ws, int B, int H, int W);
int k45_launch(bd_ctx *ctx, const float *d_sub, const float *d_rms, const uint8_t *d_mask, int B, int H, int W,
               double detect_k, int min_area, int32_t *d_labels, bd_source *d_cat, int64_t cat_capacity,
               int64_t *d_n_sources, void *d_ws, size_t ws_bytes, cudaStream_t st, const K45Fused *fz);

int k6_launch(bd_ctx *ctx, const float *d_sub, const float *d_rms, int B, int H, int W, const bd_source *d_cat,
              const int64_t *d_n_sources, int64_t cat_capacity, const bd_phot_params *p, bd_phot *d_phot, void *d_ws,
              size_t ws_bytes, cudaStream_t st);
size_t k6_workspace_bytes(int64_t cat_capacity);

size_t k9_workspace_bytes(int B, int H, int W, int64_t cap_in, int64_t cap_out);
int k9_launch(bd_ctx *ctx, const float *d_sub, const float *d_rms, int B, int H, int W, double detect_k, int min_area,
              const bd_deblend_params *p, int32_t *d_labels, const bd_source *d_cat_in, const int64_t *d_n_in, int64_t cap_in,
              bd_source *d_cat_out, int64_t cap_out, int64_t *d_n_out, void *d_ws, size_t ws_bytes, cudaStream_t st);
size_t k10_workspace_bytes(int B, int H, int W, int64_t cap_in);
int k10_launch(bd_ctx *ctx, const float *d_rms, int B, int H, int W, double detect_k, const bd_deblend_params *p, int32_t *d_labels,
               const bd_source *d_cat_in, const int64_t *d_n_in, int64_t cap_in, bd_source *d_cat_out, int64_t cap_out,
               int64_t *d_n_out, uint8_t *d_flags, void *d_ws, size_t ws_bytes, cudaStream_t st);

int k8_num_basis(const bd_conv_params *p);
size_t k8_workspace_bytes(int B, const bd_conv_params *p);
int k8_launch(bd_ctx *ctx, const float *d_ref, const float *d_img, int B, int H, int W, const bd_conv_params *p,
              const double *d_kcoef, const double *d_bgcoef, float *d_diff, float *d_conv, void *d_ws, cudaStream_t st);

// K11: bilinear reprojection through a per-frame affine matrix (d_affine: float64 [B][6], source -> result)
int k11_launch(bd_ctx *ctx, const float *d_src, int B, int Hs, int Ws, const double *d_affine, float fill, float *d_out, int Hd,
               int Wd, cudaStream_t st);

// ---- programmatic dependent launch (the small kernels that follow a large one on the same stream) ------------------
// A kernel launched with bd_launch_pdl may become resident while its predecessor is still draining; it must call
// bd_pdl_wait() before it touches anything the predecessor wrote (the wait returns when the whole predecessor grid has
// completed and its memory is visible).  bd_pdl_trigger() in a kernel lets ITS successor start launching early.  Both are
// no-ops for kernels launched the plain way.
#ifdef __CUDACC__
__device__ __forceinline__ void bd_pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void bd_pdl_trigger() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
template <typename... KArgs, typename... Args>
static inline cudaError_t bd_launch_pdl(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, Args &&...args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kernel, static_cast<KArgs>(args)...);
}
#endif

// ---- small device helpers ------------------------------------------------------------------------------
#ifdef __CUDACC__
__device__ __forceinline__ uint32_t f32_to_key(float f) {   // order-preserving map float32 -> uint32
    uint32_t b = __float_as_uint(f);
    return b ^ ((b >> 31) ? 0xFFFFFFFFu : 0x80000000u);
}
__device__ __forceinline__ float key_to_f32(uint32_t k) {
    uint32_t b = (k >> 31) ? (k ^ 0x80000000u) : ~k;
    return __uint_as_float(b);
}
#endif
