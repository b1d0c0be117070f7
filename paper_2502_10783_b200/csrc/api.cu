// C-ABI entry points of libbkgdet (include/bkgdet.h): argument checks, workspace carving, launch order.
// No computation happens here; every step of the path runs in the kernels of k1..k45.
#include <stdarg.h>
#include <stdlib.h>

#include "common.cuh"

int bd_set_error(bd_ctx *ctx, int code, const char *fmt, ...) {
    if (ctx) {
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(ctx->err, sizeof(ctx->err), fmt, ap);
        va_end(ap);
    }
    return code;
}

static bool aligned16(const void *p) { return ((uintptr_t)p & 15) == 0; }

extern "C" {

int bd_create(bd_ctx **out, int device) {
    if (!out) return BD_EINVAL;
    *out = nullptr;
    int n = 0;
    if (cudaGetDeviceCount(&n) != cudaSuccess || n <= 0 || device < 0 || device >= n) return BD_ECUDA;
    bd_ctx *c = (bd_ctx *)calloc(1, sizeof(bd_ctx));
    if (!c) return BD_ECUDA;
    c->device = device;
    {
        BdDeviceGuard guard(c);   // the caller's current device is put back on return
        if (guard.err != cudaSuccess) { free(c); return BD_ECUDA; }
        cudaDeviceProp prop;
        if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) { free(c); return BD_ECUDA; }
        c->num_sms = prop.multiProcessorCount;
        c->smem_optin = prop.sharedMemPerBlockOptin;
        void *fn = nullptr;
        cudaDriverEntryPointQueryResult qres;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) == cudaSuccess &&
            qres == cudaDriverEntryPointSuccess)
            c->encode_tiled = (decltype(c->encode_tiled))fn;
        cudaGetLastError();
    }
    *out = c;
    return BD_OK;
}

void bd_destroy(bd_ctx *ctx) {
    if (!ctx) return;
    {
        BdDeviceGuard guard(ctx);
        if (ctx->host_dev) cudaFree(ctx->host_dev);
        if (ctx->host_stream) cudaStreamDestroy(ctx->host_stream);
        if (ctx->copy_stream) cudaStreamDestroy(ctx->copy_stream);
        for (int c = 0; c < BD_HOST_CHUNKS; ++c)
            if (ctx->host_ev[c]) cudaEventDestroy(ctx->host_ev[c]);
    }
    free(ctx);
}

const char *bd_last_error(const bd_ctx *ctx) { return ctx ? ctx->err : "null context"; }

void bd_default_bkg_params(bd_bkg_params *p) {
    if (!p) return;
    p->mesh_h = 64; p->mesh_w = 64;
    p->filt_h = 3; p->filt_w = 3;
    p->clip_sigma = 3.0; p->clip_iters = 5;
    p->skew_guard = 0;
    p->median_factor = 3.0; p->mean_factor = 2.0;
}

int bd_grid_shape(int H, int W, int mesh_h, int mesh_w, int *ny, int *nx) {
    if (H <= 0 || W <= 0 || mesh_h <= 0 || mesh_w <= 0 || !ny || !nx) return BD_EINVAL;
    *ny = (H + mesh_h - 1) / mesh_h;
    *nx = (W + mesh_w - 1) / mesh_w;
    return BD_OK;
}

static int check_frame(bd_ctx *ctx, int B, int H, int W) {
    if (!ctx) return BD_EINVAL;
    if (B <= 0 || H <= 0 || W <= 0) return bd_set_error(ctx, BD_EINVAL, "B, H, W must be positive");
    if (B > 65535) return bd_set_error(ctx, BD_EINVAL, "B must be <= 65535");
    if (W % 4) return bd_set_error(ctx, BD_EINVAL, "W must be a multiple of 4");
    if ((long long)H * W >= (1ll << 31)) return bd_set_error(ctx, BD_EINVAL, "H*W must be < 2^31");
    return BD_OK;
}

static int check_params(bd_ctx *ctx, const bd_bkg_params *p) {
    if (!p) return bd_set_error(ctx, BD_EINVAL, "null params");
    if (p->mesh_h <= 0 || p->mesh_w <= 0) return bd_set_error(ctx, BD_EINVAL, "mesh size must be positive");
    if (p->filt_h < 1 || p->filt_w < 1 || !(p->filt_h & 1) || !(p->filt_w & 1) || p->filt_h > 11 || p->filt_w > 11)
        return bd_set_error(ctx, BD_EINVAL, "filter size must be odd and in 1..11");
    if (p->clip_iters < 0 || !(p->clip_sigma > 0.0)) return bd_set_error(ctx, BD_EINVAL, "clip_iters >= 0 and clip_sigma > 0 required");
    return BD_OK;
}

int bd_bkg_workspace_bytes(const bd_ctx *ctx, int B, int H, int W, const bd_bkg_params *p, size_t *bytes) {
    if (!ctx || !p || !bytes || B <= 0 || H <= 0 || W <= 0 || p->mesh_h <= 0 || p->mesh_w <= 0) return BD_EINVAL;
    const int ny = (H + p->mesh_h - 1) / p->mesh_h, nx = (W + p->mesh_w - 1) / p->mesh_w;
    size_t cells = (size_t)B * ny * nx;
    // raw bkg, raw rms, the two filled grids of the variants, K2's scratch, K1's worklist
    *bytes = 4 * bd_align_up(cells * sizeof(double), 256) + bd_align_up(2 * (size_t)B * k2_scratch_per_grid(ny, nx) * sizeof(double), 256) +
             k1_workspace_bytes(B, ny, nx) + 512;
    return BD_OK;
}

int bd_detect_workspace_bytes(const bd_ctx *ctx, int B, int H, int W, int64_t cat_capacity, size_t *bytes) {
    if (!ctx || !bytes || B <= 0 || H <= 0 || W <= 0 || cat_capacity < 0) return BD_EINVAL;
    *bytes = k45_workspace_bytes(B, H, W, cat_capacity);
    return BD_OK;
}

int bd_mesh_stats(bd_ctx *ctx, const float *d_img, int B, int H, int W, const bd_bkg_params *p, double *d_bkg_raw,
                  double *d_rms_raw, double *d_median, double *d_mean, int32_t *d_n_kept, void *d_ws, size_t ws_bytes,
                  void *cuda_stream) {
    int rc = check_frame(ctx, B, H, W);
    if (rc) return rc;
    BD_BIND_DEVICE(ctx);
    if ((rc = check_params(ctx, p))) return rc;
    if (!d_img || !aligned16(d_img)) return bd_set_error(ctx, BD_EINVAL, "d_img null or misaligned");
    const int ny = (H + p->mesh_h - 1) / p->mesh_h, nx = (W + p->mesh_w - 1) / p->mesh_w;
    const size_t need = k1_workspace_bytes(B, ny, nx) + 256;
    if (!d_ws || ws_bytes < need) return bd_set_error(ctx, BD_EWORKSPACE, "mesh statistics workspace: need %zu bytes, got %zu", need, ws_bytes);
    return k1_launch(ctx, d_img, B, H, W, p, d_bkg_raw, d_rms_raw, d_median, d_mean, d_n_kept, (void *)bd_align_up((size_t)d_ws, 256),
                     (cudaStream_t)cuda_stream);
}

int bd_grid_filter_spline(bd_ctx *ctx, const double *d_bkg_raw, const double *d_rms_raw, int B, int ny, int nx,
                          int filt_h, int filt_w, float *d_bkg_mesh, float *d_rms_mesh, double *d_bkg_coef,
                          double *d_rms_coef, void *d_ws, size_t ws_bytes, void *cuda_stream) {
    if (!ctx) return BD_EINVAL;
    if (!d_bkg_raw || !d_rms_raw || !d_bkg_coef || !d_rms_coef || !d_ws) return bd_set_error(ctx, BD_EINVAL, "null pointer");
    if (B <= 0 || ny <= 0 || nx <= 0 || B > 65535) return bd_set_error(ctx, BD_EINVAL, "bad grid shape");
    BD_BIND_DEVICE(ctx);
    if (filt_h < 1 || filt_w < 1 || !(filt_h & 1) || !(filt_w & 1) || filt_h > 11 || filt_w > 11)
        return bd_set_error(ctx, BD_EINVAL, "filter size must be odd and in 1..11");
    size_t need = 2 * (size_t)B * k2_scratch_per_grid(ny, nx) * sizeof(double);
    if (ws_bytes < need) return bd_set_error(ctx, BD_EWORKSPACE, "grid workspace: need %zu bytes, got %zu", need, ws_bytes);
    return k2_launch(ctx, d_bkg_raw, d_rms_raw, B, ny, nx, filt_h, filt_w, d_bkg_mesh, d_rms_mesh, d_bkg_coef, d_rms_coef,
                     (double *)d_ws, (cudaStream_t)cuda_stream);
}

// a1 (+ fill of invalid cells when the variants are on) + a2, shared by bkg_estimate, bkg_estimate_masked, bkg_iterate
static int estimate_impl(bd_ctx *ctx, const float *d_img, const uint8_t *d_bad, int B, int H, int W, const bd_bkg_params *p,
                         const bd_bkgx_params *px, float *d_bkg_mesh, float *d_rms_mesh, double *d_bkg_coef, double *d_rms_coef,
                         uint8_t *d_valid_mesh, void *d_ws, size_t ws_bytes, cudaStream_t st) {
    size_t need = 0;
    bd_bkg_workspace_bytes(ctx, B, H, W, p, &need);
    if (ws_bytes < need) return bd_set_error(ctx, BD_EWORKSPACE, "bkg workspace: need %zu bytes, got %zu", need, ws_bytes);
    const int ny = (H + p->mesh_h - 1) / p->mesh_h, nx = (W + p->mesh_w - 1) / p->mesh_w;
    const size_t cells = (size_t)B * ny * nx, stride = bd_align_up(cells * sizeof(double), 256);
    char *base = (char *)bd_align_up((size_t)d_ws, 256);
    double *raw_b = (double *)base, *raw_r = (double *)(base + stride);
    double *fill_b = (double *)(base + 2 * stride), *fill_r = (double *)(base + 3 * stride), *scratch = (double *)(base + 4 * stride);
    void *k1_ws = base + 4 * stride + bd_align_up(2 * (size_t)B * k2_scratch_per_grid(ny, nx) * sizeof(double), 256);
    int rc = k1_launch(ctx, d_img, B, H, W, p, raw_b, raw_r, nullptr, nullptr, nullptr, k1_ws, st, d_bad, px, nullptr);
    if (rc) return rc;
    if (d_bad || px) {
        if ((rc = k2f_launch(ctx, raw_b, raw_r, B, ny, nx, fill_b, fill_r, d_valid_mesh, st))) return rc;
        raw_b = fill_b; raw_r = fill_r;
    }
    return k2_launch(ctx, raw_b, raw_r, B, ny, nx, p->filt_h, p->filt_w, d_bkg_mesh, d_rms_mesh, d_bkg_coef, d_rms_coef,
                     scratch, st);
}

int bkg_estimate(bd_ctx *ctx, const float *d_img, int B, int H, int W, const bd_bkg_params *p, float *d_bkg_mesh,
                 float *d_rms_mesh, double *d_bkg_coef, double *d_rms_coef, void *d_ws, size_t ws_bytes,
                 void *cuda_stream) {
    int rc = check_frame(ctx, B, H, W);
    if (rc) return rc;
    BD_BIND_DEVICE(ctx);
    if ((rc = check_params(ctx, p))) return rc;
    if (!d_img || !aligned16(d_img)) return bd_set_error(ctx, BD_EINVAL, "d_img null or misaligned");
    if (!d_bkg_coef || !d_rms_coef || !d_ws) return bd_set_error(ctx, BD_EINVAL, "null coefficient or workspace pointer");
    return estimate_impl(ctx, d_img, nullptr, B, H, W, p, nullptr, d_bkg_mesh, d_rms_mesh, d_bkg_coef, d_rms_coef, nullptr, d_ws,
                         ws_bytes, (cudaStream_t)cuda_stream);
}

// ---- background variants (NEXT-3) ------------------------------------------------------------------------------------------
void bd_default_bkgx_params(bd_bkgx_params *px) {
    if (!px) return;
    px->min_valid_px = 100; px->grow = 1; px->max_masked_frac = 1.0; px->max_reject_frac = 1.0;
}

static int check_bkgx(bd_ctx *ctx, const bd_bkgx_params *px) {
    if (!px) return bd_set_error(ctx, BD_EINVAL, "null variant params");
    if (px->min_valid_px < 0 || px->grow < 0 || px->grow > 3 || !(px->max_masked_frac >= 0.0) || !(px->max_reject_frac >= 0.0))
        return bd_set_error(ctx, BD_EINVAL, "variant params: min_valid_px >= 0, grow in 0..3, fractions >= 0 required");
    return BD_OK;
}

int bd_mesh_stats_masked(bd_ctx *ctx, const float *d_img, const uint8_t *d_bad, int B, int H, int W, const bd_bkg_params *p,
                         const bd_bkgx_params *px, double *d_bkg_raw, double *d_rms_raw, double *d_median, double *d_mean,
                         int32_t *d_n_kept, int32_t *d_n_valid, void *d_ws, size_t ws_bytes, void *cuda_stream) {
    int rc = check_frame(ctx, B, H, W);
    if (rc) return rc;
    BD_BIND_DEVICE(ctx);
    if ((rc = check_params(ctx, p))) return rc;
    if ((rc = check_bkgx(ctx, px))) return rc;
    if (!d_img || !aligned16(d_img) || !aligned16(d_bad)) return bd_set_error(ctx, BD_EINVAL, "d_img null, or d_img / d_bad misaligned");
    const int ny = (H + p->mesh_h - 1) / p->mesh_h, nx = (W + p->mesh_w - 1) / p->mesh_w;
    const size_t need = k1_workspace_bytes(B, ny, nx) + 256;
    if (!d_ws || ws_bytes < need) return bd_set_error(ctx, BD_EWORKSPACE, "mesh statistics workspace: need %zu bytes, got %zu", need, ws_bytes);
    return k1_launch(ctx, d_img, B, H, W, p, d_bkg_raw, d_rms_raw, d_median, d_mean, d_n_kept, (void *)bd_align_up((size_t)d_ws, 256),
                     (cudaStream_t)cuda_stream, d_bad, px, d_n_valid);
}

int bkg_estimate_masked(bd_ctx *ctx, const float *d_img, const uint8_t *d_bad, int B, int H, int W, const bd_bkg_params *p,
                        const bd_bkgx_params *px, float *d_bkg_mesh, float *d_rms_mesh, double *d_bkg_coef, double *d_rms_coef,
                        uint8_t *d_valid_mesh, void *d_ws, size_t ws_bytes, void *cuda_stream) {
    int rc = check_frame(ctx, B, H, W);
    if (rc) return rc;
    BD_BIND_DEVICE(ctx);
    if ((rc = check_params(ctx, p))) return rc;
    if ((rc = check_bkgx(ctx, px))) return rc;
    if (!d_img || !aligned16(d_img) || !aligned16(d_bad)) return bd_set_error(ctx, BD_EINVAL, "d_img null, or d_img / d_bad misaligned");
    if (!d_bkg_coef || !d_rms_coef || !d_ws) return bd_set_error(ctx, BD_EINVAL, "null coefficient or workspace pointer");
    return estimate_impl(ctx, d_img, d_bad, B, H, W, p, px, d_bkg_mesh, d_rms_mesh, d_bkg_coef, d_rms_coef, d_valid_mesh, d_ws,
                         ws_bytes, (cudaStream_t)cuda_stream);
}

int bd_bkg_iterate_workspace_bytes(const bd_ctx *ctx, int B, int H, int W, const bd_bkg_params *p, size_t *bytes) {
    if (!bytes) return BD_EINVAL;
    size_t b = 0;
    int rc = bd_bkg_workspace_bytes(ctx, B, H, W, p, &b);
    if (rc) return rc;
    *bytes = bd_align_up(b, 256) + (size_t)B * H * W + 512;   // + the detection mask of one iteration
    return BD_OK;
}

int bkg_iterate(bd_ctx *ctx, const float *d_img, const uint8_t *d_bad0, int B, int H, int W, const bd_bkg_params *p,
                const bd_bkgx_params *px, double detect_k, int n_iter, float *d_bkg_mesh, float *d_rms_mesh, double *d_bkg_coef,
                double *d_rms_coef, uint8_t *d_valid_mesh, uint8_t *d_bad_out, void *d_ws, size_t ws_bytes, void *cuda_stream) {
    int rc = check_frame(ctx, B, H, W);
    if (rc) return rc;
    BD_BIND_DEVICE(ctx);
    if ((rc = check_params(ctx, p))) return rc;
    if ((rc = check_bkgx(ctx, px))) return rc;
    if (!d_img || !aligned16(d_img) || !aligned16(d_bad0) || !d_bad_out || !aligned16(d_bad_out))
        return bd_set_error(ctx, BD_EINVAL, "d_img / d_bad_out null, or a pointer misaligned");
    if (!d_bkg_coef || !d_rms_coef || !d_ws) return bd_set_error(ctx, BD_EINVAL, "null coefficient or workspace pointer");
    if (n_iter < 0 || (n_iter > 0 && !(detect_k > 0.0))) return bd_set_error(ctx, BD_EINVAL, "n_iter >= 0 and detect_k > 0 required");
    size_t need = 0, ws_b = 0;
    bd_bkg_iterate_workspace_bytes(ctx, B, H, W, p, &need);
    bd_bkg_workspace_bytes(ctx, B, H, W, p, &ws_b);
    if (ws_bytes < need) return bd_set_error(ctx, BD_EWORKSPACE, "iterate workspace: need %zu bytes, got %zu", need, ws_bytes);
    char *base = (char *)bd_align_up((size_t)d_ws, 256);
    uint8_t *det = (uint8_t *)(base + bd_align_up(ws_b, 256));
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if ((rc = k7_dilate_or(ctx, nullptr, d_bad0, B, H, W, 0, d_bad_out, st))) return rc;   // bad_out = (bad0 != 0)
    rc = estimate_impl(ctx, d_img, d_bad0 ? d_bad_out : nullptr, B, H, W, p, px, d_bkg_mesh, d_rms_mesh, d_bkg_coef, d_rms_coef,
                       d_valid_mesh, base, ws_b, st);
    for (int it = 0; it < n_iter && !rc; ++it) {
        rc = k3_launch(ctx, d_img, B, H, W, p->mesh_h, p->mesh_w, d_bkg_coef, d_rms_coef, detect_k, nullptr, nullptr, nullptr, det, st);
        if (!rc) rc = k7_dilate_or(ctx, det, d_bad0, B, H, W, px->grow, d_bad_out, st);
        if (!rc) rc = estimate_impl(ctx, d_img, d_bad_out, B, H, W, p, px, d_bkg_mesh, d_rms_mesh, d_bkg_coef, d_rms_coef,
                                    d_valid_mesh, base, ws_b, st);
    }
    return rc;
}

int bkg_subtract(bd_ctx *ctx, const float *d_img, int B, int H, int W, int mesh_h, int mesh_w, const double *d_bkg_coef,
                 const double *d_rms_coef, double detect_k, float *d_sub, float *d_bkg, float *d_rms, uint8_t *d_mask,
                 void *cuda_stream) {
    int rc = check_frame(ctx, B, H, W);
    if (rc) return rc;
    BD_BIND_DEVICE(ctx);
    if (mesh_h <= 0 || mesh_w <= 0) return bd_set_error(ctx, BD_EINVAL, "mesh size must be positive");
    if (!d_img || !d_bkg_coef || !d_rms_coef || !d_sub) return bd_set_error(ctx, BD_EINVAL, "null pointer");
    if (!aligned16(d_img) || !aligned16(d_sub) || !aligned16(d_bkg) || !aligned16(d_rms) || !aligned16(d_mask))
        return bd_set_error(ctx, BD_EINVAL, "misaligned pointer (16 bytes required)");
    if (d_mask && !(detect_k > 0.0)) return bd_set_error(ctx, BD_EINVAL, "detect_k must be > 0 when a mask is requested");
    return k3_launch(ctx, d_img, B, H, W, mesh_h, mesh_w, d_bkg_coef, d_rms_coef, detect_k, d_sub, d_bkg, d_rms, d_mask,
                     (cudaStream_t)cuda_stream);
}

int detect_sources(bd_ctx *ctx, const float *d_sub, const float *d_rms, const uint8_t *d_mask, int B, int H, int W,
                   double detect_k, int32_t min_area, int32_t *d_labels, bd_source *d_cat, int64_t cat_capacity,
                   int64_t *d_n_sources, void *d_ws, size_t ws_bytes, void *cuda_stream) {
    int rc = check_frame(ctx, B, H, W);
    if (rc) return rc;
    BD_BIND_DEVICE(ctx);
    if (!d_sub || !d_labels || !d_n_sources || !d_ws) return bd_set_error(ctx, BD_EINVAL, "null pointer");
    if (!d_mask && (!d_rms || !(detect_k > 0.0))) return bd_set_error(ctx, BD_EINVAL, "no mask: d_rms and detect_k > 0 required");
    if (cat_capacity < 0 || (cat_capacity > 0 && !d_cat)) return bd_set_error(ctx, BD_EINVAL, "bad catalogue buffer");
    if (!aligned16(d_sub) || !aligned16(d_labels) || !aligned16(d_mask) || !aligned16(d_rms))
        return bd_set_error(ctx, BD_EINVAL, "misaligned pointer (16 bytes required)");
    return k45_launch(ctx, d_sub, d_rms, d_mask, B, H, W, detect_k, min_area, d_labels, d_cat, cat_capacity, d_n_sources,
                      d_ws, ws_bytes, (cudaStream_t)cuda_stream, nullptr);
}

int bkg_subtract_detect(bd_ctx *ctx, const float *d_img, int B, int H, int W, int mesh_h, int mesh_w, const double *d_bkg_coef,
                        const double *d_rms_coef, double detect_k, int32_t min_area, float *d_sub, float *d_bkg, float *d_rms,
                        uint8_t *d_mask, int32_t *d_labels, bd_source *d_cat, int64_t cat_capacity, int64_t *d_n_sources,
                        void *d_ws, size_t ws_bytes, void *cuda_stream) {
    int rc = check_frame(ctx, B, H, W);
    if (rc) return rc;
    BD_BIND_DEVICE(ctx);
    if (mesh_h <= 0 || mesh_w <= 0) return bd_set_error(ctx, BD_EINVAL, "mesh size must be positive");
    if (!d_img || !d_bkg_coef || !d_rms_coef || !d_sub || !d_labels || !d_n_sources || !d_ws)
        return bd_set_error(ctx, BD_EINVAL, "null pointer");
    if (!(detect_k > 0.0)) return bd_set_error(ctx, BD_EINVAL, "detect_k must be > 0");
    if (cat_capacity < 0 || (cat_capacity > 0 && !d_cat)) return bd_set_error(ctx, BD_EINVAL, "bad catalogue buffer");
    if (!aligned16(d_img) || !aligned16(d_sub) || !aligned16(d_bkg) || !aligned16(d_rms) || !aligned16(d_mask) || !aligned16(d_labels))
        return bd_set_error(ctx, BD_EINVAL, "misaligned pointer (16 bytes required)");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (!k45_can_fuse(ctx, H, W, mesh_w)) {   // frame smaller than a tile, or mesh too narrow for the tile kernel's spline table:
        size_t need = 0;                      // the two passes one after the other (the mask goes through the workspace if need be)
        bd_detect_workspace_bytes(ctx, B, H, W, cat_capacity, &need);
        if (ws_bytes < need) return bd_set_error(ctx, BD_EWORKSPACE, "detect workspace: need %zu bytes, got %zu", need, ws_bytes);
        uint8_t *mask = d_mask ? d_mask : k45_ws_maskbuf(d_ws, B, H, W);
        rc = k3_launch(ctx, d_img, B, H, W, mesh_h, mesh_w, d_bkg_coef, d_rms_coef, detect_k, d_sub, d_bkg, d_rms, mask, st);
        if (rc) return rc;
        return k45_launch(ctx, d_sub, d_rms, mask, B, H, W, detect_k, min_area, d_labels, d_cat, cat_capacity, d_n_sources, d_ws,
                          ws_bytes, st, nullptr);
    }
    K45Fused fz;
    fz.img = d_img; fz.bcoef = d_bkg_coef; fz.rcoef = d_rms_coef;
    fz.sub = d_sub; fz.bkg = d_bkg; fz.rms = d_rms; fz.mask = d_mask; fz.mh = mesh_h; fz.mw = mesh_w;
    return k45_launch(ctx, d_sub, d_rms, nullptr, B, H, W, detect_k, min_area, d_labels, d_cat, cat_capacity, d_n_sources, d_ws,
                      ws_bytes, st, &fz);
}

// ---- NEXT-1: deblending and cleaning -------------------------------------------------------------------------
void bd_default_deblend_params(bd_deblend_params *p) {
    if (!p) return;
    p->n_thresh = 32; p->pad = 0; p->min_cont = 0.005; p->clean_param = 1.0; p->clean_zone = 4.0;
}

static int check_deblend_params(bd_ctx *ctx, const bd_deblend_params *p) {
    if (!p) return bd_set_error(ctx, BD_EINVAL, "null pointer");
    if (p->n_thresh < 2 || p->n_thresh > 64 || (p->n_thresh & (p->n_thresh - 1)))
        return bd_set_error(ctx, BD_EINVAL, "n_thresh must be a power of two in 2..64");
    if (!(p->min_cont >= 0.0) || !(p->min_cont <= 1.0)) return bd_set_error(ctx, BD_EINVAL, "min_cont must be in [0, 1]");
    if (!(p->clean_param > 0.0) || !(p->clean_param <= 64.0) || !(p->clean_zone > 0.0) || !(p->clean_zone <= 1024.0))
        return bd_set_error(ctx, BD_EINVAL, "clean_param must be in (0, 64], clean_zone in (0, 1024]");
    return BD_OK;
}

int bd_deblend_workspace_bytes(const bd_ctx *ctx, int B, int H, int W, int64_t cap_in, int64_t cap_out, size_t *bytes) {
    if (!ctx || !bytes || B <= 0 || H <= 0 || W <= 0 || cap_in < 0 || cap_out < 0) return BD_EINVAL;
    *bytes = k9_workspace_bytes(B, H, W, cap_in, cap_out);
    return BD_OK;
}

int deblend_sources(bd_ctx *ctx, const float *d_sub, const float *d_rms, int B, int H, int W, double detect_k,
                    int32_t min_area, const bd_deblend_params *p, int32_t *d_labels, const bd_source *d_cat_in,
                    const int64_t *d_n_in, int64_t cap_in, bd_source *d_cat_out, int64_t cap_out, int64_t *d_n_out,
                    void *d_ws, size_t ws_bytes, void *cuda_stream) {
    int rc = check_frame(ctx, B, H, W);
    if (rc) return rc;
    BD_BIND_DEVICE(ctx);
    if (!d_sub || !d_rms || !d_labels || !d_cat_in || !d_n_in || !d_n_out || !d_ws) return bd_set_error(ctx, BD_EINVAL, "null pointer");
    if ((rc = check_deblend_params(ctx, p))) return rc;
    if (cap_in < 0 || cap_out < 0 || (cap_out > 0 && !d_cat_out)) return bd_set_error(ctx, BD_EINVAL, "bad catalogue capacity");
    if (!(detect_k > 0.0) || min_area < 1) return bd_set_error(ctx, BD_EINVAL, "detect_k must be positive, min_area >= 1");
    if (d_cat_out == d_cat_in) return bd_set_error(ctx, BD_EINVAL, "d_cat_out must not alias d_cat_in");
    return k9_launch(ctx, d_sub, d_rms, B, H, W, detect_k, min_area, p, d_labels, d_cat_in, d_n_in, cap_in, d_cat_out, cap_out,
                     d_n_out, d_ws, ws_bytes, (cudaStream_t)cuda_stream);
}

int bd_clean_workspace_bytes(const bd_ctx *ctx, int B, int H, int W, int64_t cap_in, size_t *bytes) {
    if (!ctx || !bytes || B <= 0 || H <= 0 || W <= 0 || cap_in < 0) return BD_EINVAL;
    *bytes = k10_workspace_bytes(B, H, W, cap_in);
    return BD_OK;
}

int clean_sources(bd_ctx *ctx, const float *d_rms, int B, int H, int W, double detect_k, const bd_deblend_params *p,
                  int32_t *d_labels, const bd_source *d_cat_in, const int64_t *d_n_in, int64_t cap_in,
                  bd_source *d_cat_out, int64_t cap_out, int64_t *d_n_out, uint8_t *d_flags, void *d_ws,
                  size_t ws_bytes, void *cuda_stream) {
    int rc = check_frame(ctx, B, H, W);
    if (rc) return rc;
    BD_BIND_DEVICE(ctx);
    if (!d_rms || !d_labels || !d_cat_in || !d_n_in || !d_n_out || !d_ws) return bd_set_error(ctx, BD_EINVAL, "null pointer");
    if ((rc = check_deblend_params(ctx, p))) return rc;
    if (cap_in < 0 || cap_out < 0 || (cap_out > 0 && !d_cat_out)) return bd_set_error(ctx, BD_EINVAL, "bad catalogue capacity");
    if (!(detect_k > 0.0)) return bd_set_error(ctx, BD_EINVAL, "detect_k must be positive");
    if (d_cat_out == d_cat_in) return bd_set_error(ctx, BD_EINVAL, "d_cat_out must not alias d_cat_in");
    return k10_launch(ctx, d_rms, B, H, W, detect_k, p, d_labels, d_cat_in, d_n_in, cap_in, d_cat_out, cap_out, d_n_out, d_flags,
                      d_ws, ws_bytes, (cudaStream_t)cuda_stream);
}

int bd_phot_workspace_bytes(const bd_ctx *ctx, int64_t cat_capacity, size_t *bytes) {
    if (!ctx || !bytes || cat_capacity < 0) return BD_EINVAL;
    *bytes = k6_workspace_bytes(cat_capacity);
    return BD_OK;
}

void bd_default_phot_params(bd_phot_params *p) {
    if (!p) return;
    p->r_aper = 5.0; p->kron_factor = 2.5; p->kron_min_radius = 3.5; p->kron_search = 6.0; p->subpix = 5; p->pad = 0;
}

int photometry(bd_ctx *ctx, const float *d_sub, const float *d_rms, int B, int H, int W, const bd_source *d_cat,
               const int64_t *d_n_sources, int64_t cat_capacity, const bd_phot_params *p, bd_phot *d_phot, void *d_ws,
               size_t ws_bytes, void *cuda_stream) {
    int rc = check_frame(ctx, B, H, W);
    if (rc) return rc;
    BD_BIND_DEVICE(ctx);
    if (!d_sub || !d_rms || !d_cat || !d_n_sources || !d_phot || !p || !d_ws) return bd_set_error(ctx, BD_EINVAL, "null pointer");
    if (cat_capacity < 0) return bd_set_error(ctx, BD_EINVAL, "bad catalogue capacity");
    if (!(p->r_aper > 0.0) || !(p->kron_factor > 0.0) || !(p->kron_min_radius > 0.0) || !(p->kron_search > 0.0) || p->subpix < 1 ||
        p->subpix > 16)
        return bd_set_error(ctx, BD_EINVAL, "photometry parameters must be positive, subpix in 1..16");
    if (!(p->r_aper <= 1024.0) || !(p->kron_factor <= 1024.0) || !(p->kron_min_radius <= 1024.0) || !(p->kron_search <= 1024.0))
        return bd_set_error(ctx, BD_EINVAL, "photometry radii / factors must be <= 1024");
    if (cat_capacity == 0) return BD_OK;
    return k6_launch(ctx, d_sub, d_rms, B, H, W, d_cat, d_n_sources, cat_capacity, p, d_phot, d_ws, ws_bytes, (cudaStream_t)cuda_stream);
}

// ---- stamp convolution + subtraction (NEXT-4) -----------------------------------------------------------------------------
void bd_default_conv_params(bd_conv_params *p) {
    if (!p) return;
    memset(p, 0, sizeof(*p));
    p->half_width = 10; p->n_gauss = 3;
    p->sigma[0] = 0.7; p->sigma[1] = 1.5; p->sigma[2] = 3.0; p->sigma[3] = 1.0;
    p->degree[0] = 6; p->degree[1] = 4; p->degree[2] = 2; p->degree[3] = 0;
    p->spatial_order = 2; p->bg_order = 1;
}

int bd_conv_num_basis(const bd_conv_params *p) {
    const int n = k8_num_basis(p);
    return n < 0 ? BD_EINVAL : n;
}

int bd_subtract_workspace_bytes(const bd_ctx *ctx, int B, const bd_conv_params *p, size_t *bytes) {
    if (!ctx || !bytes || B <= 0 || k8_num_basis(p) < 0) return BD_EINVAL;
    *bytes = k8_workspace_bytes(B, p) + 256;
    return BD_OK;
}

int image_subtract(bd_ctx *ctx, const float *d_ref, const float *d_img, int B, int H, int W, const bd_conv_params *p,
                   const double *d_kcoef, const double *d_bgcoef, float *d_diff, float *d_conv, void *d_ws, size_t ws_bytes,
                   void *cuda_stream) {
    int rc = check_frame(ctx, B, H, W);
    if (rc) return rc;
    BD_BIND_DEVICE(ctx);
    if (!d_ref || !d_img || !d_kcoef || !d_bgcoef || !d_diff || !d_ws) return bd_set_error(ctx, BD_EINVAL, "null pointer");
    if (k8_num_basis(p) < 0) return bd_set_error(ctx, BD_EINVAL, "bad convolution parameters");
    const size_t need = k8_workspace_bytes(B, p) + 256;
    if (ws_bytes < need) return bd_set_error(ctx, BD_EWORKSPACE, "subtract workspace: need %zu bytes, got %zu", need, ws_bytes);
    return k8_launch(ctx, d_ref, d_img, B, H, W, p, d_kcoef, d_bgcoef, d_diff, d_conv, d_ws, (cudaStream_t)cuda_stream);
}

int image_reproject(bd_ctx *ctx, const float *d_src, int B, int Hs, int Ws, const double *d_affine, double fill, float *d_out,
                    int Hd, int Wd, void *cuda_stream) {
    int rc = check_frame(ctx, B, Hs, Ws);
    if (rc) return rc;
    if ((rc = check_frame(ctx, B, Hd, Wd))) return rc;
    BD_BIND_DEVICE(ctx);
    if (!d_src || !d_affine || !d_out) return bd_set_error(ctx, BD_EINVAL, "null pointer");
    if (!aligned16(d_out) || !aligned16(d_src) || ((uintptr_t)d_affine & 7)) return bd_set_error(ctx, BD_EINVAL, "d_src, d_out must be 16-byte, d_affine 8-byte aligned");
    if (d_src == d_out) return bd_set_error(ctx, BD_EINVAL, "d_out must not alias d_src");
    return k11_launch(ctx, d_src, B, Hs, Ws, d_affine, (float)fill, d_out, Hd, Wd, (cudaStream_t)cuda_stream);
}

// bd_run_host returns early on any error; by then copies on the copy stream may still be reading the caller's h_img and
// writing h_n_sources / h_cat.  The guard waits for both streams on every such path (the caller may free its buffers as
// soon as the call returns); the successful path has already synchronised and disarms it.
struct BdHostDrain {
    bd_ctx *ctx;
    bool armed = true;
    explicit BdHostDrain(bd_ctx *c) : ctx(c) {}
    ~BdHostDrain() {
        if (!armed) return;
        if (ctx->copy_stream) cudaStreamSynchronize(ctx->copy_stream);
        if (ctx->host_stream) cudaStreamSynchronize(ctx->host_stream);
        cudaGetLastError();   // the error that brought us here is already recorded in ctx->err
    }
};

int bd_run_host(bd_ctx *ctx, const float *h_img, int B, int H, int W, const bd_bkg_params *p, double detect_k,
                int32_t min_area, bd_source *h_cat, int64_t cat_capacity, int64_t *h_n_sources) {
    int rc = check_frame(ctx, B, H, W);
    if (rc) return rc;
    BD_BIND_DEVICE(ctx);
    if ((rc = check_params(ctx, p))) return rc;
    if (!h_img || !h_n_sources || cat_capacity < 0 || (cat_capacity > 0 && !h_cat))
        return bd_set_error(ctx, BD_EINVAL, "null host pointer");
    if (!ctx->host_stream) BD_CUDA_CHECK(ctx, cudaStreamCreateWithFlags(&ctx->host_stream, cudaStreamNonBlocking));
    cudaStream_t st = ctx->host_stream;
    const size_t P = (size_t)B * H * W;
    const int ny = (H + p->mesh_h - 1) / p->mesh_h, nx = (W + p->mesh_w - 1) / p->mesh_w;
    const size_t cells = (size_t)B * ny * nx;
    size_t ws_b = 0, ws_d = 0;
    bd_bkg_workspace_bytes(ctx, B, H, W, p, &ws_b);
    bd_detect_workspace_bytes(ctx, B, H, W, cat_capacity, &ws_d);
    size_t off = 0;
    auto take = [&](size_t bytes) { size_t o = off; off = bd_align_up(off + bytes, 256); return o; };
    const size_t o_img = take(P * 4), o_sub = take(P * 4), o_rms = take(P * 4), o_mask = take(P), o_lab = take(P * 4);
    const size_t o_cb = take(cells * 8), o_cr = take(cells * 8), o_wsb = take(ws_b), o_wsd = take(ws_d);
    const size_t o_cat = take((size_t)cat_capacity * sizeof(bd_source)), o_n = take((size_t)B * 8);
    if (off > ctx->host_dev_bytes) {
        if (ctx->host_dev) cudaFree(ctx->host_dev);
        ctx->host_dev = nullptr; ctx->host_dev_bytes = 0;
        BD_CUDA_CHECK(ctx, cudaMalloc(&ctx->host_dev, off));
        ctx->host_dev_bytes = off;
    }
    char *d = (char *)ctx->host_dev;
    // The frame arrives in chunks on a copy stream (whole frames of a batch, or strips of mesh rows of a single frame) and
    // K1 runs on every chunk as soon as it is there: the statistics pass hides behind the PCIe transfer.  K2 and the fused
    // pass need the whole mesh grid and follow the last chunk.
    if (!ctx->copy_stream) BD_CUDA_CHECK(ctx, cudaStreamCreateWithFlags(&ctx->copy_stream, cudaStreamNonBlocking));
    for (int c = 0; c < BD_HOST_CHUNKS; ++c)
        if (!ctx->host_ev[c]) BD_CUDA_CHECK(ctx, cudaEventCreateWithFlags(&ctx->host_ev[c], cudaEventDisableTiming));
    BdHostDrain drain(ctx);
    drain.armed = false;
    {
        const size_t stride = bd_align_up(cells * sizeof(double), 256);
        char *base = (char *)bd_align_up((size_t)(d + o_wsb), 256);
        double *raw_b = (double *)base, *raw_r = (double *)(base + stride), *scratch = (double *)(base + 4 * stride);
        void *k1_ws = base + 4 * stride + bd_align_up(2 * (size_t)B * k2_scratch_per_grid(ny, nx) * sizeof(double), 256);
        // units: frames of a batch, mesh rows of a single frame
        const int units = B > 1 ? B : ny;
        const int nch = units < BD_HOST_CHUNKS ? units : BD_HOST_CHUNKS;
        // (the copy stream must not overwrite the frame while work of the previous call still reads it)
        drain.armed = true;   // from the first enqueue on, an early return waits for the streams
        BD_CUDA_CHECK(ctx, cudaEventRecord(ctx->host_ev[BD_HOST_CHUNKS - 1], st));
        BD_CUDA_CHECK(ctx, cudaStreamWaitEvent(ctx->copy_stream, ctx->host_ev[BD_HOST_CHUNKS - 1], 0));
        for (int c = 0; c < nch; ++c) {
            const int u0 = (int)((long long)units * c / nch), u1 = (int)((long long)units * (c + 1) / nch);
            size_t px0, px1, cell0;
            int Bc, Hc;
            if (B > 1) { px0 = (size_t)u0 * H * W; px1 = (size_t)u1 * H * W; cell0 = (size_t)u0 * ny * nx; Bc = u1 - u0; Hc = H; }
            else {
                const int r0 = u0 * p->mesh_h, r1 = u1 == ny ? H : u1 * p->mesh_h;
                px0 = (size_t)r0 * W; px1 = (size_t)r1 * W; cell0 = (size_t)u0 * nx; Bc = 1; Hc = r1 - r0;
            }
            BD_CUDA_CHECK(ctx, cudaMemcpyAsync(d + o_img + px0 * 4, h_img + px0, (px1 - px0) * 4, cudaMemcpyHostToDevice, ctx->copy_stream));
            BD_CUDA_CHECK(ctx, cudaEventRecord(ctx->host_ev[c], ctx->copy_stream));
            BD_CUDA_CHECK(ctx, cudaStreamWaitEvent(st, ctx->host_ev[c], 0));
            rc = k1_launch(ctx, (const float *)(d + o_img) + px0, Bc, Hc, W, p, raw_b + cell0, raw_r + cell0, nullptr, nullptr, nullptr, k1_ws, st);
            if (rc) return rc;
        }
        rc = k2_launch(ctx, raw_b, raw_r, B, ny, nx, p->filt_h, p->filt_w, nullptr, nullptr, (double *)(d + o_cb), (double *)(d + o_cr), scratch, st);
        if (rc) return rc;
    }
    rc = bkg_subtract_detect(ctx, (const float *)(d + o_img), B, H, W, p->mesh_h, p->mesh_w, (const double *)(d + o_cb),
                             (const double *)(d + o_cr), detect_k, min_area, (float *)(d + o_sub), nullptr, (float *)(d + o_rms),
                             (uint8_t *)(d + o_mask), (int32_t *)(d + o_lab), (bd_source *)(d + o_cat), cat_capacity,
                             (int64_t *)(d + o_n), d + o_wsd, ws_d, st);
    if (rc) return rc;
    BD_CUDA_CHECK(ctx, cudaMemcpyAsync(h_n_sources, d + o_n, (size_t)B * 8, cudaMemcpyDeviceToHost, st));
    BD_CUDA_CHECK(ctx, cudaStreamSynchronize(st));
    int64_t total = 0;
    for (int f = 0; f < B; ++f) total += h_n_sources[f];
    if (total > cat_capacity) total = cat_capacity;
    if (total > 0) {
        BD_CUDA_CHECK(ctx, cudaMemcpyAsync(h_cat, d + o_cat, (size_t)total * sizeof(bd_source), cudaMemcpyDeviceToHost, st));
        BD_CUDA_CHECK(ctx, cudaStreamSynchronize(st));
    }
    drain.armed = false;   // both streams are idle here: st was synchronised after the last copy it waited for
    return BD_OK;
}

}  // extern "C"
