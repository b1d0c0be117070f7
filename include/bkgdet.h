/*
 * bkgdet.h -- C ABI of the B200-native background + detection hot path of arxiv 2502.10783
 * ("Image Pre-Processing Framework for Time-Domain Astronomy in the Artificial Intelligence Era").
 *
 * The three calls BASELINE.json names -- bkg_estimate, bkg_subtract, detect_sources -- plus context,
 * workspace queries, two single-step entry points used by the parity tests, and one host-buffer
 * convenience call.  Citations are PAPER.md line numbers with the section
 * they fall in; A<n> are the readings of silent/garbled passages listed in DESIGN.md.
 *
 * Conventions (all calls)
 *   - Frames are float32, row-major, contiguous [B, H, W]; W must be a multiple of 4; H*W < 2^31.
 *   - Every d_* argument is a DEVICE pointer owned by the caller, 16-byte aligned, valid until the
 *     stream work completes.  h_* arguments are HOST pointers.  The library allocates nothing per call
 *     except inside bd_run_host (buffers cached in the context).
 *   - cuda_stream is a cudaStream_t passed as void* (0 = legacy default stream).  Calls enqueue work
 *     and return; they never synchronise (bd_run_host does).
 *   - Return value: BD_OK (0) or a negative BD_E* code; bd_last_error() gives text.
 *   - Non-finite pixels: undefined results.
 *   - Mesh grid: ny = ceil(H/mesh_h), nx = ceil(W/mesh_w); partial edge meshes are their own mesh (A9).
 */
#ifndef BKGDET_H
#define BKGDET_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define BD_OK 0
#define BD_EINVAL (-1)      /* null pointer, non-positive size, even filter, W % 4 != 0, misaligned pointer ... */
#define BD_EWORKSPACE (-2)  /* workspace too small */
#define BD_ECUDA (-3)       /* CUDA runtime/driver error (text in bd_last_error) */
#define BD_EUNSUPPORTED (-4) /* mesh too large for the kernels (see bd_mesh_stats) */

typedef struct bd_ctx bd_ctx; /* opaque: device properties, TMA encode entry point, cached buffers, last error */

/* Parameters of background estimation.  PAPER.md:67 (sub-regions, default 64x64), :78 (sigma range,
 * maximum iterations), :80 (median filter), :69-76 eqs. 1-4 (estimators). */
typedef struct {
    int32_t mesh_h, mesh_w;   /* sub-region size in pixels; default 64, 64 */
    int32_t filt_h, filt_w;   /* median-filter window on the mesh grid, odd, 1..11; default 3, 3   :80 */
    double clip_sigma;        /* k_c of median +- k_c*std; default 3.0                              :78 */
    int32_t clip_iters;       /* maximum rejection rounds (0 = no clipping); default 5             :78 */
    int32_t skew_guard;       /* 0 (default) = estimator formula as printed; 1 = A12 rule: std==0 -> mean,
                                 |mean-median|/std >= 0.3 -> median */
    double median_factor;     /* background = median_factor*median - mean_factor*mean (eq. 4, A2):       */
    double mean_factor;       /* (3,2) mode [default]; (2.5,1.5) eq. 3; (1,0) eq. 1 median; (0,-1) eq. 2 mean */
} bd_bkg_params;

/* One catalogue record (detect_sources).  PAPER.md:153 (peak value, total flux per candidate), :159
 * (isophotal photometry); readings A18-A20.  Coordinates are 0-based, pixel centre at integer
 * coordinates, x = column, y = row.  Moments are intensity-weighted by sub. */
typedef struct {
    int32_t frame;                      /* frame index in the batch */
    int32_t label;                      /* 1 + minimum raster index (y*W + x) of the component, per frame */
    int32_t npix;                       /* pixels in the component */
    int32_t xmin, xmax, ymin, ymax;     /* bounding box, inclusive */
    int32_t xpeak, ypeak;               /* position of the maximum of sub (ties: smallest raster index) */
    float peak;                         /* max of sub over the component */
    double flux;                        /* sum of sub */
    double x, y;                        /* centroid  sum(I*x)/sum(I) */
    double x2, y2, xy;                  /* central second moments  sum(I*(x-xc)^2)/sum(I) ... */
} bd_source;

/* Parameters of aperture / auto photometry (readings A23-A27; the paper, names the methods only). */
typedef struct {
    double r_aper;            /* radius of the circular aperture in pixels; default 5.0                        A23 */
    double kron_factor;       /* auto aperture = kron_factor * first-moment radius; default 2.5               A25 */
    double kron_min_radius;   /* lower limit of the auto radius, in units of the object's 1-sigma ellipse; 3.5    */
    double kron_search;       /* the first-moment radius is measured inside this many sigma; default 6.0          */
    int32_t subpix;           /* sub-pixel samples per axis for the pixels on the aperture's rim; default 5    A23 */
    int32_t pad;
} bd_phot_params;

/* One photometry record per catalogue record (same index).  56 bytes. */
typedef struct {
    double flux_aper, fluxerr_aper, area_aper;   /* sum w*sub, sqrt(sum w*rms^2), sum w over the circular aperture */
    double kron_radius;                          /* in units of the 1-sigma ellipse of the second moments          */
    double flux_auto, fluxerr_auto;              /* sum sub, sqrt(sum rms^2) over the ellipse of kron_radius       */
    int32_t npix_auto;                           /* pixels in that ellipse                                          */
    int32_t flags;                               /* bit 0: the circular aperture is cut by the frame edge; bit 1: the
                                                    bounding box of the search or Kron ellipse leaves the frame; bit 2:
                                                    degenerate record (non-finite centroid / moments or flux <= 0): all
                                                    sums are 0 and nothing was measured                                */
} bd_phot;

/* ---- context ------------------------------------------------------------------------------------ */
int bd_create(bd_ctx **ctx, int device);   /* binds to CUDA device `device`; returns BD_ECUDA if none */
void bd_destroy(bd_ctx *ctx);
const char *bd_last_error(const bd_ctx *ctx);
void bd_default_bkg_params(bd_bkg_params *p);
int bd_grid_shape(int H, int W, int mesh_h, int mesh_w, int *ny, int *nx);

/* ---- workspace sizes (bytes of device memory the caller must pass as d_ws) ------------------------ */
int bd_bkg_workspace_bytes(const bd_ctx *ctx, int B, int H, int W, const bd_bkg_params *p, size_t *bytes);
int bd_detect_workspace_bytes(const bd_ctx *ctx, int B, int H, int W, int64_t cat_capacity, size_t *bytes);

/* ---- a1: per-mesh sigma-clipped statistics (kernel K1).  PAPER.md:67-78, eqs. 1-4. --------------------
 * For every mesh: up to clip_iters rounds of {median, mean, population std of the survivors; reject
 * outside median +- clip_sigma*std (inclusive bounds, A6)}, stop when a round rejects nothing (A7), then
 * the final statistics of the survivors.  Sums are accumulated in float64 against float64 bounds, so
 * the survivor sets equal the float64 definition's.
 * Outputs, each [B, ny, nx], any may be NULL:  d_bkg_raw = median_factor*median - mean_factor*mean
 * (float64), d_rms_raw = std (float64), d_median, d_mean (float64), d_n_kept (int32 survivors).
 * d_ws / ws_bytes: at least bd_bkg_workspace_bytes() (4 bytes per mesh are used: the list of meshes the warp-per-mesh
 * kernel hands to the general path).
 * Limits: a mesh may hold at most 255 * 512 = 130 560 pixels (the sweeps count into per-thread 8-bit histogram
 * columns, 512 threads per mesh), i.e. up to 361 x 361; larger meshes return BD_EUNSUPPORTED.  Meshes of at
 * most 4096 pixels with mesh_w % 4 == 0 are held in the registers of one warp; larger ones are staged in shared
 * memory by TMA (<= 48 KiB) or streamed from global memory / L2 (mesh_w % 4 == 0), other widths use a plain loader. */
int bd_mesh_stats(bd_ctx *ctx, const float *d_img, int B, int H, int W, const bd_bkg_params *p,
                  double *d_bkg_raw, double *d_rms_raw, double *d_median, double *d_mean,
                  int32_t *d_n_kept, void *d_ws, size_t ws_bytes, void *cuda_stream);

/* ---- a2: median filter of both mesh grids + cubic B-spline prefilter (kernel K2).  PAPER.md:80. --------
 * In: raw grids float64 [B, ny, nx].  Out: filtered grids (float32, for the caller; may be NULL) and the
 * spline coefficients (float64) bkg_subtract consumes.  Window truncated at the grid border (A13);
 * both grids filtered (A11); half-sample-symmetric spline boundary (A14).  d_ws: >= 4*B*(ny+nx) doubles. */
int bd_grid_filter_spline(bd_ctx *ctx, const double *d_bkg_raw, const double *d_rms_raw, int B, int ny, int nx,
                          int filt_h, int filt_w, float *d_bkg_mesh, float *d_rms_mesh,
                          double *d_bkg_coef, double *d_rms_coef, void *d_ws, size_t ws_bytes,
                          void *cuda_stream);

/* ---- a2 for callers that cannot allocate device memory.  PAPER.md:80, same operation and same kernels as
 * bd_grid_filter_spline, but without the d_ws / ws_bytes pair.
 * Who needs it: code that gets its device buffers handed to it and has no allocator of its own -- a plug-in inside
 * an application that owns all of the GPU's memory, a real-time loop that may not enter cudaMalloc (it can block and
 * synchronises the device), a process whose memory is fully committed by the time this step runs.  Such a caller can
 * still pass the inputs and outputs it was given, but has nowhere to get the scratch from.
 * Here the scratch (the Thomas factors of the spline prefilter, 4*B*(ny+nx) doubles) is an array compiled into the
 * library: BD_GRID_STATIC_MAX_DOUBLES doubles (256 KiB) of device memory that every GPU which loads libbkgdet holds
 * from module load until the process exits, whether or not this call is ever made.  The call makes no cudaMalloc,
 * cudaFree or other allocating call.
 * Limit: 4*B*(ny+nx) <= BD_GRID_STATIC_MAX_DOUBLES, else BD_EWORKSPACE with the numbers in bd_last_error() and
 * nothing is launched (e.g. B = 64 frames of 32 x 32 meshes, or one frame with ny + nx <= 8192).
 * First call on a device: looks up the array's device address (cudaGetSymbolAddress with ctx's device current) and
 * keeps it for later calls; make that first call outside any stream capture.
 * Sharing: there is ONE array per GPU, used by every call, context and stream.  Nothing in it has to be zero at
 * entry (the kernel writes each factor before reading it) and the last call's contents stay behind.  Two calls
 * whose kernels overlap on the same GPU (different streams, or different host threads) race on the array and
 * produce garbage: keep calls on one stream, or order them with events.  Grids that fit the kernel's shared memory
 * (ny, nx <= 160 and ny*(nx|1) <= 20880) do not touch the array at all.
 * Outputs are bit-identical to bd_grid_filter_spline's. */
#define BD_GRID_STATIC_MAX_DOUBLES 32768
int bd_grid_filter_spline_static(bd_ctx *ctx, const double *d_bkg_raw, const double *d_rms_raw, int B, int ny, int nx,
                                 int filt_h, int filt_w, float *d_bkg_mesh, float *d_rms_mesh,
                                 double *d_bkg_coef, double *d_rms_coef, void *cuda_stream);

/* ---- bkg_estimate = a1 + a2.  PAPER.md:67-80. -------------------------------------------------------
 * d_bkg_mesh, d_rms_mesh: filtered mesh grids, float32 [B, ny, nx] (may be NULL).
 * d_bkg_coef, d_rms_coef: spline coefficients, float64 [B, ny, nx] (required).
 * d_ws / ws_bytes: at least bd_bkg_workspace_bytes(). */
int bkg_estimate(bd_ctx *ctx, const float *d_img, int B, int H, int W, const bd_bkg_params *p,
                 float *d_bkg_mesh, float *d_rms_mesh, double *d_bkg_coef, double *d_rms_coef,
                 void *d_ws, size_t ws_bytes, void *cuda_stream);

/* ---- bkg_subtract = a3 (kernel K3, fused).  PAPER.md:80 (spline interpolation back to full
 * resolution), :61-65 (removal), :153 (threshold scan). -------------------------------------------------
 * Per pixel: bkg, rms = cubic B-spline value of the coefficient grids at u=(x+1/2)/mesh_w-1/2,
 * v=(y+1/2)/mesh_h-1/2 (A14);  sub = img - bkg;  mask = rms > 0 && sub > detect_k*rms (strict, A15).
 * Arithmetic: the y-collapsed spline coefficients of every (row, grid cell) are formed in float64 and split into a
 * float32 hi/lo pair; a pixel is then float32 FMAs with sub = (img - hi) - (lo + sum), which agrees with the float64
 * definition to ~1e-6 ADU.  The comparison is float32 on the float32 outputs: sub > (float)detect_k * rms, one
 * rounded product (the same rule in bkg_subtract, bkg_subtract_detect and detect_sources without a mask).
 * d_sub (required), d_bkg, d_rms: float32 [B,H,W]; d_mask: uint8 [B,H,W] (0/1).  d_bkg, d_rms, d_mask may be
 * NULL (not emitted); detect_k <= 0 with d_mask != NULL is BD_EINVAL. */
int bkg_subtract(bd_ctx *ctx, const float *d_img, int B, int H, int W, int mesh_h, int mesh_w,
                 const double *d_bkg_coef, const double *d_rms_coef, double detect_k,
                 float *d_sub, float *d_bkg, float *d_rms, uint8_t *d_mask, void *cuda_stream);

/* ---- detect_sources = a4 + a5 (kernels K4, K5).  PAPER.md:153 (connect pixels above the main
 * threshold into candidates; peak and total flux per candidate), :159 (isophotal flux). ------------------
 * d_mask: uint8 [B,H,W], non-zero = foreground.  If NULL the mask is computed from (d_sub, d_rms, detect_k) with
 * the bkg_subtract rule (float32: rms > 0 && sub > (float)detect_k * rms), so it equals bkg_subtract's mask bit for bit.
 * d_labels: int32 [B,H,W] out; 8-connected components (A16), label = 1 + minimum raster index of the
 * component within its frame, 0 = background; all components are labelled (A20).
 * d_cat: records of components with npix >= min_area (A19), ascending (frame, label); the first
 * min(n_total, cat_capacity) are written.  d_n_sources: int64 [B] true per-frame counts (device).
 * Catalogue overflow is not an error: records beyond cat_capacity are dropped.
 * Sums use float64 atomics: flux/centroid/moments are not bit-reproducible run to run (labels are).
 * d_ws / ws_bytes: at least bd_detect_workspace_bytes() (about 26 bytes per pixel: the record table is sized for the
 * worst case of one component per 2x2 pixels, so it cannot overflow; only the records in use are touched). */
int detect_sources(bd_ctx *ctx, const float *d_sub, const float *d_rms, const uint8_t *d_mask,
                   int B, int H, int W, double detect_k, int32_t min_area,
                   int32_t *d_labels, bd_source *d_cat, int64_t cat_capacity, int64_t *d_n_sources,
                   void *d_ws, size_t ws_bytes, void *cuda_stream);

/* ---- bkg_subtract_detect = a3 + a4 + a5 in one pass (fused tile kernel).  PAPER.md:80, :61-65, :153, :159. -------
 * Same results as bkg_subtract followed by detect_sources on its mask (the two share their arithmetic: maps, mask
 * and labels are bit-identical; catalogue sums differ only by atomic order), but the 128x64-pixel tile kernel of
 * detect_sources evaluates the splines itself, so the streaming of the maps overlaps the labelling and neither the
 * mask nor sub is read back from HBM.  Arguments as in the two calls: d_sub required; d_bkg, d_rms, d_mask may be
 * NULL (not emitted).  For mesh_w < 33 (spline table too large for the tile kernel) or frames smaller than one tile the
 * call runs the two passes one after the other (same results).
 * d_ws / ws_bytes: at least bd_detect_workspace_bytes(). */
int bkg_subtract_detect(bd_ctx *ctx, const float *d_img, int B, int H, int W, int mesh_h, int mesh_w,
                        const double *d_bkg_coef, const double *d_rms_coef, double detect_k, int32_t min_area,
                        float *d_sub, float *d_bkg, float *d_rms, uint8_t *d_mask, int32_t *d_labels,
                        bd_source *d_cat, int64_t cat_capacity, int64_t *d_n_sources, void *d_ws, size_t ws_bytes,
                        void *cuda_stream);

/* ---- photometry = SURVEY 8(f) NEXT-2: aperture and auto (Kron-like) photometry of every catalogue record (kernel K6).
 * PAPER.md:159 (aperture, isophotal and auto photometry, one object per thread; isophotal = bd_source.flux).
 * d_sub, d_rms: float32 [B,H,W] maps of bkg_subtract; d_cat / d_n_sources: the outputs of detect_sources (records in
 * catalogue order, per-frame counts on the device); the first min(sum n_sources, cat_capacity) records are measured and
 * d_phot[i] belongs to d_cat[i].  Aperture: circle of r_aper about the centroid, rim pixels weighted by the fraction of
 * their subpix^2 sub-pixel centres inside (A23).  Auto: ellipse of the second moments (A24; 1/12 added to x2, y2 of
 * degenerate objects), first-moment radius r1 = sum r*sub / sum sub inside kron_search sigma, kron_radius =
 * max(kron_factor*r1, kron_min_radius) (A25), flux inside that ellipse with a hard edge (A26).  No neighbour masking
 * (A27).  Deterministic (fixed summation order).  Pixels outside the frame contribute nothing (flags).
 * One warp per object; objects whose search ellipse covers more than 4096 pixels are queued in the workspace and
 * measured by one thread block each.  d_ws / ws_bytes: at least bd_phot_workspace_bytes(cat_capacity). */
void bd_default_phot_params(bd_phot_params *p);
int bd_phot_workspace_bytes(const bd_ctx *ctx, int64_t cat_capacity, size_t *bytes);
int photometry(bd_ctx *ctx, const float *d_sub, const float *d_rms, int B, int H, int W, const bd_source *d_cat,
               const int64_t *d_n_sources, int64_t cat_capacity, const bd_phot_params *p, bd_phot *d_phot,
               void *d_ws, size_t ws_bytes, void *cuda_stream);

/* ---- multi-threshold deblending (kernel K9) and cleaning (kernel K10).
 * PAPER.md:155 ("calculate multi-level deblending thresholds.  At each threshold level, the algorithm re-evaluates objects
 * and splits them as necessary, constructing a binary tree structure rooted in the original source candidate ... traversed
 * from bottom to top ... pruning"), :157 ("determine if the current object can be merged with any adjacent objects ...
 * flagged as a false detection ... a parallel operation to remove the marked pixels").  The paper gives no constants and no
 * formulas; readings D1-D12 restate the method it adapts:
 *   D1  candidates = the records of detect_sources;  D2  levels t_i = t_0 q^i, t_0 = (float)detect_k * rms[peak pixel],
 *       q = (peak / t_0)^(1/n_thresh) by repeated float64 square roots (n_thresh a power of two, 2..64);
 *   D3  node of level i = an 8-connected component of {sub > t_i} inside the candidate with >= min_area pixels;
 *   D4  significant = flux > min_cont * candidate flux;  D5  bottom-to-top pruning: a node splits when at least two of its
 *       children are split or significant;  D6  one object: candidate unchanged;
 *   D7  the other pixels join the object of their brightest assigned 8-neighbour, in synchronous rounds;
 *   D8  label of an object = 1 + minimum raster index of its pixels; records as in detect_sources;
 *   D9-D11  cleaning: object i is a false detection when a brighter object j (Moffat-like profile of index clean_param
 *       fitted to j's flux, second moments, area and threshold) within clean_zone isophotal radii of j leaves
 *       flux_i / npix_i - I_j(i) <= t_i;  D12  its pixels become 0 in the label map, its record leaves the catalogue.
 * deblend_sources: d_labels (in/out) int32 [B,H,W] and d_cat_in / d_n_in from detect_sources (the first
 * min(sum n_in, cap_in) records are the candidates; records cut off by cap_in are dropped).  d_cat_out: ascending
 * (frame, label), the first min(n, cap_out) records; d_n_out int64 [B] true counts.  cap_out also bounds the number of NEW
 * objects whose records can be formed: a candidate that cannot reserve its records still gets its new labels and is counted
 * in d_n_out, so sum(d_n_out) > cap_out or missing records tell the caller to retry with more room.  d_cat_out must not
 * alias d_cat_in.  A candidate whose bounding box is 65 535 or more pixels wide or 32 767 or more tall is left whole.
 * Label maps are bit-reproducible; flux sums are float64 atomics (tree decisions within 1e-9 relative of
 * the contrast limit may differ from the float64 definition).
 * clean_sources: d_cat_in / d_n_in are a catalogue of d_labels (normally deblend_sources' output); d_flags (uint8
 * [cap_in], may be NULL) receives 1 for every false detection.  Decisions use float64 pow(): pairs within 1e-9 relative of
 * the limit may differ from the definition.
 * d_ws / ws_bytes: at least bd_deblend_workspace_bytes() (about 42 bytes per pixel: the frame-sized arrays of the
 * candidates too large for shared memory) / bd_clean_workspace_bytes(). */
typedef struct {
    int32_t n_thresh;         /* number of levels, a power of two in 2..64; default 32                      D2 */
    int32_t pad;
    double min_cont;          /* minimum contrast; default 0.005                                            D4 */
    double clean_param;       /* index beta of the neighbour profile; default 1.0                          D10 */
    double clean_zone;        /* reach of a neighbour in isophotal radii; default 4.0                      D11 */
} bd_deblend_params;
void bd_default_deblend_params(bd_deblend_params *p);
int bd_deblend_workspace_bytes(const bd_ctx *ctx, int B, int H, int W, int64_t cap_in, int64_t cap_out, size_t *bytes);
int deblend_sources(bd_ctx *ctx, const float *d_sub, const float *d_rms, int B, int H, int W, double detect_k,
                    int32_t min_area, const bd_deblend_params *p, int32_t *d_labels, const bd_source *d_cat_in,
                    const int64_t *d_n_in, int64_t cap_in, bd_source *d_cat_out, int64_t cap_out, int64_t *d_n_out,
                    void *d_ws, size_t ws_bytes, void *cuda_stream);
int bd_clean_workspace_bytes(const bd_ctx *ctx, int B, int H, int W, int64_t cap_in, size_t *bytes);
int clean_sources(bd_ctx *ctx, const float *d_rms, int B, int H, int W, double detect_k, const bd_deblend_params *p,
                  int32_t *d_labels, const bd_source *d_cat_in, const int64_t *d_n_in, int64_t cap_in,
                  bd_source *d_cat_out, int64_t cap_out, int64_t *d_n_out, uint8_t *d_flags, void *d_ws,
                  size_t ws_bytes, void *cuda_stream);

/* ---- background variants.  PAPER.md:67 ("This division can be based on either predefined masks
 * generated by the Image Quality Assessment function or rectangular regions ... each sub-region containing at least 100
 * pixels"), :181 ("We will iterate to remove background noises with the background estimation and removal function").
 * Readings B1-B6:
 *   B1  d_bad: uint8 [B,H,W], non-zero = excluded; masked pixels leave a mesh's multiset before the first clipping round;
 *   B2  a mesh that keeps fewer than min_valid_px pixels, or of which more than max_masked_frac is masked, is INVALID;
 *   B6  so is a mesh whose clipping rejected more than max_reject_frac of its valid pixels (a crowded mesh);
 *   B3  an invalid cell of the mesh grids takes the median of the valid cells inside the smallest square window
 *       (2r+1)^2, r = 1, 2, ..., truncated at the grid border, that holds one (both grids; 0 if no cell is valid);
 *       then the median filter and the spline prefilter as in bkg_estimate;
 *   B4  bkg_iterate: estimate with the caller's mask, threshold the subtracted frame at detect_k (the bkg_subtract
 *       rule), grow the detections (B5: dilation by the (2 grow + 1)^2 square), OR them with the caller's mask,
 *       estimate again -- n_iter re-estimations.
 * With a mask every mesh takes the general path of kernel K1 (a sweep per clipping round). */
typedef struct {
    int32_t min_valid_px;     /* default 100 */
    int32_t grow;             /* Chebyshev radius of the dilation of the detections, 0..3; default 1           B5 */
    double max_masked_frac;   /* default 1.0 (never)                                                           B2 */
    double max_reject_frac;   /* default 1.0 (never)                                                           B6 */
} bd_bkgx_params;
void bd_default_bkgx_params(bd_bkgx_params *px);

/* a1 with the variants.  Outputs as bd_mesh_stats (invalid meshes: NaN, n_kept 0) plus d_n_valid (int32 [B,ny,nx], pixels
 * left after masking; may be NULL).  d_bad may be NULL (validity rules only).  d_ws: bd_bkg_workspace_bytes(). */
int bd_mesh_stats_masked(bd_ctx *ctx, const float *d_img, const uint8_t *d_bad, int B, int H, int W,
                         const bd_bkg_params *p, const bd_bkgx_params *px, double *d_bkg_raw, double *d_rms_raw,
                         double *d_median, double *d_mean, int32_t *d_n_kept, int32_t *d_n_valid, void *d_ws,
                         size_t ws_bytes, void *cuda_stream);

/* a1 + fill (B3) + a2.  Outputs as bkg_estimate plus d_valid_mesh (uint8 [B,ny,nx], 1 = the mesh was valid; may be NULL).
 * d_ws / ws_bytes: at least bd_bkg_workspace_bytes(). */
int bkg_estimate_masked(bd_ctx *ctx, const float *d_img, const uint8_t *d_bad, int B, int H, int W,
                        const bd_bkg_params *p, const bd_bkgx_params *px, float *d_bkg_mesh, float *d_rms_mesh,
                        double *d_bkg_coef, double *d_rms_coef, uint8_t *d_valid_mesh, void *d_ws, size_t ws_bytes,
                        void *cuda_stream);

/* B4.  d_bad0 may be NULL.  d_bad_out: uint8 [B,H,W], required: the exclusion mask the last estimate used (0/1).
 * n_iter >= 0 (0 = bkg_estimate_masked with d_bad0; d_bad_out is then d_bad0 != 0, or zeros).
 * d_ws / ws_bytes: at least bd_bkg_iterate_workspace_bytes(). */
int bd_bkg_iterate_workspace_bytes(const bd_ctx *ctx, int B, int H, int W, const bd_bkg_params *p, size_t *bytes);
int bkg_iterate(bd_ctx *ctx, const float *d_img, const uint8_t *d_bad0, int B, int H, int W, const bd_bkg_params *p,
                const bd_bkgx_params *px, double detect_k, int n_iter, float *d_bkg_mesh, float *d_rms_mesh,
                double *d_bkg_coef, double *d_rms_coef, uint8_t *d_valid_mesh, uint8_t *d_bad_out, void *d_ws,
                size_t ws_bytes, void *cuda_stream);

/* ---- stamp-wise spatially varying convolution of the template + image subtraction (kernel K8).
 * eq. 8 K(u,v) = sum_n a_n(x,y) K_n(u,v); eq. 9 K_n = exp(-(u^2+v^2)/(2 sigma_k^2)) u^i v^j, i + j <= degree;
 * eq. 10 R (x) K = I + B; one stamp of the kernel size (21 x 21 by default) per thread block with a preloaded kernel.
 * The kernel FIT is out of scope: the coefficients are inputs.  Readings C1-C7:
 *   C1  basis order: Gaussian g = 0.., inside it (i, j) with i = 0..degree[g], j = 0..degree[g] - i;
 *   C2  a_n(x,y) = sum_t kcoef[n][t] xh^p yh^q, t over p = 0..spatial_order, q = 0..spatial_order - p,
 *       xh = (2x - (W-1))/W, yh = (2y - (H-1))/H;  B(x,y) likewise from bgcoef with bg_order;
 *   C3  stamps of S x S pixels (S = 2 half_width + 1) from the top-left corner; a stamp's kernel is K at its nominal
 *       centre (sx S + half_width, sy S + half_width), the same for all its pixels;
 *   C4  conv(x,y) = sum_{u,v} K(u,v) R(x-u, y-v), R = 0 outside the frame;   C5  diff = I + B - conv, B at the pixel.
 * d_ref, d_img: float32 [B,H,W]; d_kcoef: float64 [B][n_basis][n_sp]; d_bgcoef: float64 [B][n_bg]
 * (n_sp = (so+1)(so+2)/2, n_bg likewise); d_diff: float32 [B,H,W]; d_conv: float32 [B,H,W] or NULL.
 * Arithmetic: the kernels are built in float64 and rounded to float32; the 441-term sums are float32 FMAs.
 * d_ws / ws_bytes: at least bd_subtract_workspace_bytes(). */
typedef struct {
    int32_t half_width;       /* 1..15; default 10 (21 x 21; the register-blocked kernel; others use a generic one) */
    int32_t n_gauss;          /* 1..4; default 3 */
    double sigma[4];          /* default 0.7, 1.5, 3.0 */
    int32_t degree[4];        /* 0..8 each; default 6, 4, 2  -> 49 basis kernels */
    int32_t spatial_order;    /* 0..4; default 2 */
    int32_t bg_order;         /* 0..4; default 1 */
} bd_conv_params;
void bd_default_conv_params(bd_conv_params *p);
int bd_conv_num_basis(const bd_conv_params *p);      /* n_basis, or a negative code */
int bd_subtract_workspace_bytes(const bd_ctx *ctx, int B, const bd_conv_params *p, size_t *bytes);
int image_subtract(bd_ctx *ctx, const float *d_ref, const float *d_img, int B, int H, int W, const bd_conv_params *p,
                   const double *d_kcoef, const double *d_bgcoef, float *d_diff, float *d_conv, void *d_ws,
                   size_t ws_bytes, void *cuda_stream);

/* ---- SURVEY 8(f) NEXT-4, second half: bilinear reprojection through an affine matrix (kernel K11).
 * PAPER.md:114 ("we use the affine matrix to obtain the coordinate mapping between the source image and the resulting image.
 * For each pixel in the source image, the pixel value in the resulting image is calculated through bilinear interpolation
 * based on the four neighboring pixels").  The FIT of the matrix is out of scope: the matrix is an input.  Readings R1-R6:
 *   R1  d_affine: float64 [B][6] on the device, one row-major 2 x 3 matrix per frame, the FORWARD map source pixel (x, y) ->
 *       result pixel (x', y') = (a0 x + a1 y + a2, a3 x + a4 y + a5).  The result pulls: result(x', y') is the source
 *       sampled at A^-1 (x', y');   R2  pixel centres at integers, x = column, y = row, 0-based;
 *   R3  neighbours (x0, y0) .. (x0+1, y0+1), x0 = floor(xs), y0 = floor(ys), weights (1-fx)(1-fy), fx(1-fy), (1-fx)fy, fx fy;
 *   R4  a neighbour outside the source frame has the value `fill` and is interpolated like any other;
 *   R5  a matrix without an inverse (det = 0, or non-finite entries) gives a result frame of `fill`;
 *   R6  A^-1 and the source coordinates are float64, fx, fy and the blend float32 (within 1e-6 max|src| of the float64
 *       definition).
 * d_src: float32 [B,Hs,Ws]; d_out: float32 [B,Hd,Wd] (its own shape; Ws and Wd multiples of 4), must not alias d_src.
 * No workspace.  Deterministic. */
int image_reproject(bd_ctx *ctx, const float *d_src, int B, int Hs, int Ws, const double *d_affine, double fill,
                    float *d_out, int Hd, int Wd, void *cuda_stream);

/* ---- whole chain from HOST buffers (pinned or pageable), synchronous. ----------------------------------
 * Copies h_img to the device in up to 8 chunks (whole frames of a batch, strips of mesh rows of a single frame) on a
 * copy stream of its own and runs the statistics kernel of step a1 on every chunk as it arrives, then a2 and
 * bkg_subtract_detect on the whole frame, copies the catalogue and the per-frame counts back, and waits.  Same results as
 * the device calls.  Device buffers, the two streams and the events are cached in ctx between calls.
 * h_cat: [cat_capacity] records; h_n_sources: [B].  Returns BD_OK or an error code. */
int bd_run_host(bd_ctx *ctx, const float *h_img, int B, int H, int W, const bd_bkg_params *p,
                double detect_k, int32_t min_area, bd_source *h_cat, int64_t cat_capacity,
                int64_t *h_n_sources);

#ifdef __cplusplus
}
#endif
#endif /* BKGDET_H */
