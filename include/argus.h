/*
 * argus.h -- C ABI of the B200-native calibrate + HEALPix-resample hot path of Argus-HDPS
 * (arXiv 2207.14304).  Plain C99, no torch types: device/host pointers, sizes, a cudaStream_t
 * passed as void*.
 *
 * What the path computes (citations are PAPER.md line + section; the paper states the steps in
 * words only, DESIGN.md lists the readings taken where it is silent):
 *   - "standard image calibrations (dark subtraction, flat fielding, masking of bad pixels)"
 *     PAPER.md:141 (sec. 5.1), on the GPU PAPER.md:135 (sec. 5), Table 2 PAPER.md:192;
 *   - "Each full-frame image is reprojected into equal-sky-area tiles (based on the HEALPix
 *     pixelization scheme with NSIDE=256)" PAPER.md:145 (sec. 5.1.1), Table 2, using the
 *     "one-directional mapping from celestial to pixel-plane coordinates" of PAPER.md:141;
 *   - coaddition on the pre-aligned HEALPix grid PAPER.md:153 (sec. 5.1.3): plain sum / weight-sum.
 *   Calibration masters are caller-owned device buffers that stay resident across frames
 *   (uploaded "at the start of each pointing").
 *
 * Conventions
 *   - Every function returns ARGUS_OK (0) or a negative argus_status; nothing throws.
 *   - Unless stated otherwise every array pointer is a DEVICE pointer owned by the caller; the library
 *     never frees it and never keeps it after the call returns.  argus_wcs / argus_frame / argus_coadd
 *     structs are HOST structs read during the call.
 *   - All work is enqueued on the caller's stream (cudaStream_t passed as void*; NULL = legacy default
 *     stream) and is asynchronous, except where a function documents a synchronisation.  With
 *     ARGUS_OPT_PLAN_OVERLAP (default) the per-frame plan runs on the context's own streams and the caller's
 *     stream waits for it by event: outputs are complete in the caller's stream order exactly as without it.
 *   - Pixel convention: 0-based, pixel centres at integers, frame[y*W + x], x <-> FITS axis 1,
 *     crpix 0-based.  HEALPix: NESTED scheme, nside a power of two, 32 <= nside <= 2^29; sky
 *     convention alpha = phi, delta = pi/2 - theta (ICRS).  (Lower bound: the unit of work of the plan and of
 *     every resample kernel is a tile of 32 x 32 pixels of one base face = 1024 consecutive nested indices,
 *     which does not exist below nside 32 -- a whole sky of at most 3072 pixels, far from the paper's
 *     NSIDE-256 tiles of 1.38 arcsec pixels.  argus_resample with an explicit idx list has no
 *     such unit but keeps the same bound for uniformity.)
 *   - Footprint domain: a HEALPix pixel belongs to the frame footprint iff its centre maps to
 *     -0.5 <= x < W-0.5, -0.5 <= y < H-0.5 and lies within rho_max of CRVAL,
 *     rho_max = atan(1.25 * scale * hypot(W,H)/2), scale = sqrt|det CD|.
 */
#ifndef ARGUS_H_
#define ARGUS_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum argus_status {
    ARGUS_OK = 0,
    ARGUS_ERR_NULL = -1,     /* a required pointer is NULL */
    ARGUS_ERR_SHAPE = -2,    /* W, H, n or a size argument is out of range */
    ARGUS_ERR_NSIDE = -3,    /* nside is not a power of two in [32, 2^29] */
    ARGUS_ERR_KERNEL = -4,   /* unknown interpolation kernel */
    ARGUS_ERR_WCS = -5,      /* singular CD matrix, non-finite entries, sip_order outside [0,5] */
    ARGUS_ERR_CAPACITY = -6, /* an output or scratch capacity is too small (required size is reported) */
    ARGUS_ERR_ALIGN = -7,    /* a pointer is not aligned to its element type */
    ARGUS_ERR_CUDA = -8,     /* a CUDA runtime call failed: see argus_last_cuda_error() */
    ARGUS_ERR_STATE = -9     /* call sequence error (e.g. no plan for this WCS and n does not match) */
} argus_status;

enum { ARGUS_BILINEAR = 0, ARGUS_LANCZOS3 = 1 };

/* Options for argus_ctx_set_option. */
enum {
    ARGUS_OPT_PLAN_CACHE = 1, /* 1 (default): a plan built for (wcs, W, H, nside) is reused by the next
                                 call with identical arguments; 0: every call re-plans on the device */
    ARGUS_OPT_FAST_PATH = 3,  /* which kernel runs a planned frame given as raw + masters (no bpm, W % 8 == 0, 16-byte aligned arrays):
                                 1 (default): the TMA-staged tile kernel (resample_fast_kernel, both interpolation kernels) where
                                    every 32 x 32-pixel tile's source box fits its stage, else -- and always with pre-fused
                                    masters -- the image-aligned unit kernel (resample_unit_kernel, bilinear);
                                    Lanczos-3 frames whose boxes all fit 48 x 48 source pixels (fine grids: nside 2^18 at 0.08 pixels
                                    per HEALPix pixel) run the tile kernel with two half-size stages instead of one;
                                 2: tile kernel only (one-stage Lanczos-3 form); 3: unit kernel wherever its geometry allows;
                                 4: as 1 without the two-stage Lanczos-3 form (diagnostic); 0: always the general kernel */
    ARGUS_OPT_PLAN_OVERLAP = 4, /* 1 (default): the plan of a new WCS is built on an internal high-priority stream in a second
                                 set of scratch buffers, so that it runs underneath the previous frame's kernels; the
                                 caller's stream waits for it (stream order of results is unchanged); 0: in place */
    ARGUS_OPT_SEGMENT_RASTER = 5, /* 0 (default): argus_segment_products with a layout writes every tile in nested pixel
                               * order (slot(p) of argus_coadd).  1: every tile is a row-major image of side
                               * nside / nside_tile: pixel (ix, iy) of the tile (ix = even bits, iy = odd bits of the
                               * in-tile nested index, the HEALPix face coordinates) goes to iy * side + ix. */
    ARGUS_OPT_UNIT_MARGIN = 6, /* test hook, default 0: added to the unit kernel's estimated sub-block overhang (cells).  A negative
                                  value makes plan_units_kernel find sub-blocks that leave their unit's box: they are served by the
                                  stray kernel (per pixel, FP64), which normal geometries never exercise.  9 .. 40: self-test of the
                                  ARGUS_DEBUG_BOUNDS build (its check treats the staged box as value - 8 cells narrower) */
    ARGUS_OPT_PROFILE = 2     /* 1: argus_resample / argus_resample_coadd (idx == NULL) record CUDA events on
                                 the caller's stream around the plan kernels and around the fused kernel
                                 (ring of 256 calls); read them back with argus_profile_read.  Default 0. */
};

typedef struct argus_ctx argus_ctx;

/* Sky -> pixel WCS.  TAN (gnomonic) about crval, pixel = CD^-1 (xi, eta) [+ SIP] + crpix.
 * SIP uses the sky->pixel ("inverse", AP/BP) polynomials applied directly:
 *   u = U + sum_{p+q<=sip_order} ap[p*6+q] U^p V^q,   v = V + sum bp[p*6+q] U^p V^q. */
typedef struct argus_wcs {
    double crval[2];   /* deg: alpha0, delta0 */
    double crpix[2];   /* px, 0-based */
    double cd[2][2];   /* deg/px: (xi, eta)^T = cd (U, V)^T */
    int32_t sip_order; /* 0 = no SIP, else 2..5 */
    int32_t reserved;
    double ap[36];
    double bp[36];
} argus_wcs;

/* One frame.  Either the raw frame + masters (raw != NULL: calibration is fused into the resampling,
 * the calibrated frame never exists in HBM) or an already calibrated frame (raw == NULL: cal + mask,
 * e.g. argus_calibrate's outputs).  All pointers are device pointers, row-major [H][W]. */
typedef struct argus_frame {
    const uint16_t* raw;  /* ADU */
    const float* bias;    /* ADU */
    const float* dark;    /* ADU / s */
    const float* flat;    /* dimensionless */
    const uint8_t* bpm;   /* optional (may be NULL); non-zero = bad pixel */
    float t_exp;          /* s: dark is scaled by t_exp */
    int32_t sat_adu;      /* raw >= sat_adu is masked (65535 = clipped pixels only) */
    float flat_min;       /* !(flat >= flat_min) is masked */
    const float* cal;     /* used when raw == NULL: calibrated ADU */
    const uint8_t* mask;  /* used when raw == NULL: 1 = good, 0 = masked */
    /* Pre-fused masters (argus_prepare_masters below).  masters_format != 0 with raw != NULL: the
     * calibration is (raw - offset) * gain with the two arrays argus_prepare_masters wrote (float32 or binary16 as the
     * format says); bias, dark, flat, bpm, t_exp and flat_min are then ignored (they are folded into the two arrays). */
    const void* offset;   /* ADU: bias + dark * t_exp */
    const void* gain;     /* 1 / flat; NaN = invalid pixel */
    int32_t masters_format; /* 0 = bias / dark / flat; ARGUS_MASTERS_F32; ARGUS_MASTERS_F16 */
    int32_t reserved;
} argus_frame;

enum { ARGUS_MASTERS_F32 = 1, ARGUS_MASTERS_F16 = 2 };

/* Coadd buffer layout: sorted tile ids at resolution nside_tile (NSIDE = 256 in the
 * paper); each tile owns ppt = (nside/nside_tile)^2 consecutive nested pixels:
 *   slot(p) = rank(p / ppt) * ppt + (p mod ppt);  sum and wsum hold n_tiles * ppt floats. */
typedef struct argus_coadd {
    const int64_t* tiles; /* device, ascending, unique */
    int64_t n_tiles;
    int64_t nside_tile;   /* power of two, 1 <= nside_tile <= nside/32 */
} argus_coadd;

/* Plan statistics of the most recent plan (diagnostics; filled by argus_plan_info). */
typedef struct argus_plan_stats {
    int64_t n_footprint;  /* footprint size */
    int64_t n_tiles;      /* 32x32-pixel output tiles visited */
    int64_t n_inside;     /* tiles entirely inside the footprint, polynomial coordinates */
    int64_t n_border;     /* tiles cut by the frame border */
    int64_t n_exact;      /* tiles evaluated per pixel in FP64 (belt/cap ring, poles, failed fits) */
    int64_t n_empty;      /* candidate tiles that turned out empty */
    int64_t n_units;      /* image-aligned work units of the plan (0: the tile or general kernel runs the frame) */
    int64_t n_stray;      /* 4 x 4-pixel sub-blocks no unit can serve (per-pixel FP64 path); normally 0 */
} argus_plan_stats;

const char* argus_strerror(int status);
int argus_version(void);

/* Context: owns scratch only -- three sets of plan buffers (tile records, masks, prefix sums, counters; about
 * 560 bytes per candidate output tile each), two internal high-priority streams and events for ARGUS_OPT_PLAN_OVERLAP.
 *   max_tiles = 0 (default): the sets are sized from (W, H, nside, pixel scale) by the first call that plans a frame
 *               (1.5 x the frame's area in 32 x 32-pixel tiles + margin: 3 x 48 MB for a 61-MPix frame at nside 2^17,
 *               which has 5.3e4 candidate tiles; 1.95e5 at nside 2^18) and grown -- which synchronises the device --
 *               when a later frame needs more; never shrunk.
 *   max_tiles in 64 .. 2^24: allocated now, fixed; a frame with more candidate tiles reports ARGUS_ERR_CAPACITY.
 * device = CUDA ordinal.  Synchronous.  A context is not thread-safe: use one per host thread (contexts are
 * independent).  Its calls share device scratch (plan sets, the tile kernels' claim counter): enqueue the calls of one
 * context on ONE stream at a time (or order the streams with events); frames that should run concurrently on one GPU take
 * one context each. */
int argus_ctx_create(argus_ctx** ctx, int device, int64_t max_tiles);
int argus_ctx_destroy(argus_ctx* ctx);
int argus_ctx_set_option(argus_ctx* ctx, int option, int64_t value);
/* cudaError_t of the last failed CUDA call made through this context (0 if none). */
int argus_last_cuda_error(const argus_ctx* ctx);
/* Number of CUDA kernels launched through this context since its creation (diagnostics; bench.py's gpu_launches). */
int64_t argus_launch_count(const argus_ctx* ctx);

/* A2 (standalone; the paper's unfused order).  Per pixel:
 *   good = raw < sat_adu && (bpm == NULL || bpm == 0) && flat >= flat_min && all masters finite
 *   cal_out  = good ? (raw - bias - dark * t_exp) / flat : 0      (float32)
 *   mask_out = good ? 1 : 0
 * Asynchronous on stream. */
int argus_calibrate(argus_ctx* ctx, const uint16_t* raw, const float* bias, const float* dark,
                    const float* flat, const uint8_t* bpm, int64_t W, int64_t H, float t_exp,
                    int32_t sat_adu, float flat_min, float* cal_out, uint8_t* mask_out, void* stream);

/* Pre-fused masters (the calibration of PAPER.md:141 with everything that depends only on the masters
 * formed once per pointing and exposure time).  Per pixel:
 *   offset = bias + dark * t_exp
 *   gain   = 1 / flat; NaN where flat < flat_min or not finite, bias or dark not finite, bpm != 0 (bpm may be NULL), or
 *            where offset or gain cannot be represented in the storage format
 * format ARGUS_MASTERS_F32: float32 arrays (10 B per input pixel on the hot path instead of 14; results stay within
 * north_star's tolerance of the definition); ARGUS_MASTERS_F16: IEEE binary16 arrays, round to nearest even (6 B per
 * pixel; NOT within that tolerance: a 1000-ADU offset is stored to 0.25 ADU -- DESIGN.md section 12 has the numbers).
 * offset_out / gain_out: DEVICE, W * H elements of the format, 16-byte aligned for the vector paths.  Asynchronous. */
int argus_prepare_masters(argus_ctx* ctx, const float* bias, const float* dark, const float* flat, const uint8_t* bpm,
                          int64_t W, int64_t H, float t_exp, float flat_min, int format, void* offset_out, void* gain_out,
                          void* stream);

/* A0 + A1: builds the resampling plan for (wcs, W, H, nside) on the device and reports the footprint.
 *   idx_out  : device int64[capacity] or NULL.  When non-NULL receives the footprint: all nested pixel
 *              indices whose centre falls on the frame, ascending, unique.
 *   n_out    : HOST pointer, receives the footprint size (always, also on ARGUS_ERR_CAPACITY).
 * Synchronises the stream (the count travels to the host).  The plan stays cached in ctx for the
 * following argus_resample / argus_resample_coadd calls with the same (wcs, W, H, nside). */
int argus_healpix_footprint(argus_ctx* ctx, const argus_wcs* wcs, int64_t W, int64_t H, int64_t nside,
                            int64_t* idx_out, size_t capacity, size_t* n_out, void* stream);

/* A3-A5 (+ fused A2 when frame->raw != NULL): per footprint pixel pix2ang -> inverse TAN (+SIP) ->
 * masked, normalised bilinear / Lanczos-3 interpolation (BASELINE.json north_star):
 *   S0 = sum k, B = sum k (1 - m), V1 = sum k m cal over the 2x2 / 6x6 taps (off-frame taps have m = 0)
 *   w = 1 - B/S0;  w < w_min ? (value, weight) = (0, 0) : (V1 / (S0 - B), min(w, 1)).
 *   idx == NULL : the library uses its own plan for (wcs, W, H, nside) (built here, on the device, if not
 *                 cached); output element i belongs to the i-th footprint pixel in ascending order; n is
 *                 the capacity of value_out / weight_out; fully asynchronous.  If the footprint is
 *                 larger than n nothing beyond n is written and the next synchronising call
 *                 (argus_healpix_footprint / argus_plan_info) reports ARGUS_ERR_CAPACITY.
 *   idx != NULL : device int64[n], arbitrary nested pixels (any order); output element i belongs to
 *                 idx[i]; coordinates are evaluated per pixel in FP64 (general, slower path).
 * Outputs are never NaN/Inf. */
int argus_resample(argus_ctx* ctx, const argus_frame* frame, const argus_wcs* wcs, int64_t W, int64_t H,
                   int64_t nside, int kernel, float w_min, const int64_t* idx, size_t n, float* value_out,
                   float* weight_out, void* stream);

/* A2-A5 with HOST buffers for the per-frame data: frame->raw is a HOST pointer to the uint16 frame (pinned memory
 * for asynchronous copies; pageable memory works but serialises), the masters stay DEVICE pointers (resident per
 * pointing), value_host / weight_host are HOST arrays of n floats (n = footprint size, e.g. from
 * argus_healpix_footprint; the first n outputs are copied).  The library uploads the frame, runs argus_resample with its
 * own plan on `stream` and downloads value + weight, on internal copy streams and two sets of device staging buffers,
 * so that the upload of frame k+1 and the download of frame k-1 overlap the kernels of frame k.  Asynchronous: the
 * host arrays are complete after argus_host_wait(ctx).  The first call (and a call with a larger frame) allocates the
 * staging buffers and synchronises the device. */
int argus_resample_host(argus_ctx* ctx, const argus_frame* frame, const argus_wcs* wcs, int64_t W, int64_t H,
                        int64_t nside, int kernel, float w_min, size_t n, float* value_host, float* weight_host,
                        void* stream);
/* A2-A6 fused with the raw frame in HOST memory (frame->raw as for argus_resample_host; masters, layout, sum and wsum
 * are DEVICE pointers as for argus_resample_coadd): the upload of frame k+1 overlaps the kernels of frame k (two device
 * staging buffers, the library's upload stream).  The accumulation is ordered on `stream`. */
int argus_resample_coadd_host(argus_ctx* ctx, const argus_frame* frame, const argus_wcs* wcs, int64_t W, int64_t H,
                              int64_t nside, int kernel, float w_min, const argus_coadd* layout, float* sum, float* wsum,
                              int64_t* n_skipped_dev, void* stream);
/* The paper's per-frame PRODUCT with HOST buffers: the resampled frame as IEEE binary16 segment data and the
 * low-resolution map on the minipix grid (argus_segment_products without stamping).  frame->raw: HOST
 * (pinned); masters: DEVICE.  n = footprint size (argus_healpix_footprint); seg16_host[n]: element i <-> i-th footprint pixel
 * ascending; mini_*_host[mini_capacity], *n_mini_host: as argus_segment_products (all HOST, pinned for asynchronous copies;
 * entries beyond n_mini are unspecified).  2 bytes per footprint pixel + 16 per minipix leave the device instead of the 8
 * per pixel of argus_resample_host.  Pipelined like argus_resample_host; complete after argus_host_wait. */
int argus_reduce_frame_host(argus_ctx* ctx, const argus_frame* frame, const argus_wcs* wcs, int64_t W, int64_t H, int64_t nside,
                            int kernel, float w_min, int64_t nside_mini, size_t n, size_t mini_capacity, uint16_t* seg16_host,
                            int64_t* mini_id_host, float* mini_value_host, float* mini_weight_host, int64_t* n_mini_host,
                            void* stream);
/* Blocks until every upload and download enqueued by argus_resample_host / argus_resample_coadd_host / argus_reduce_frame_host
 * has completed. */
int argus_host_wait(argus_ctx* ctx);

/* A6: sum[slot(idx[i])] += weight[i] * value[i]; wsum[slot] += weight[i] for i < n.  idx must hold
 * unique pixels (a footprint); pixels whose tile is absent from the layout are skipped and counted in
 * *n_skipped_dev (device int64, may be NULL, accumulated with atomics).  Asynchronous. */
int argus_coadd_accumulate(argus_ctx* ctx, const argus_coadd* layout, int64_t nside, float* sum, float* wsum,
                           const int64_t* idx, const float* value, const float* weight, size_t n,
                           int64_t* n_skipped_dev, void* stream);

/* A2-A6 fused: resample with the library's plan and accumulate straight into the coadd buffer
 * (value / weight are never written to HBM).  Asynchronous. */
int argus_resample_coadd(argus_ctx* ctx, const argus_frame* frame, const argus_wcs* wcs, int64_t W, int64_t H,
                         int64_t nside, int kernel, float w_min, const argus_coadd* layout, float* sum,
                         float* wsum, int64_t* n_skipped_dev, void* stream);

/* Segment products of a resampled frame: 16-bit float segment data, minipix
 * stamping against a target list and the low-resolution map (readings in DESIGN.md section 10).
 *   inputs   idx[n]: DEVICE, ascending unique nested pixels at nside (a footprint); value[n], weight[n]: DEVICE,
 *            the resampled frame on them; nside, nside_mini: powers of two, nside_mini <= nside <= 2^29 (the paper:
 *            nside_mini = 16384); a minipix is the 4^j consecutive nested pixels idx >> 2j, 2^j = nside / nside_mini;
 *            targets[n_targets]: DEVICE, minipix ids at nside_mini that hold a science target (any order,
 *            duplicates and ids outside the footprint allowed).
 *   outputs  (all DEVICE, caller-owned, any may be NULL except as noted; "n_mini" = number of distinct minipix
 *            that own at least one pixel of idx)
 *            mini_id[k]      ascending minipix ids, k < n_mini (required when mini_capacity > 0)
 *            mini_weight[k]  sum of weight over the minipix' pixels (FP32, fixed summation order)
 *            mini_value[k]   sum(weight * value) / sum(weight), 0 where the sum of weights is 0
 *            mini_keep[k]    1 if mini_id[k] is in targets, else 0 (k < n_mini; the rest is left untouched)
 *            seg16           IEEE binary16 bits (round to nearest even, finite values clamped to +-65504, NaN ->
 *                            0x7e00) of value where the pixel's minipix is kept, of 0 elsewhere; with
 *                            mini_keep == NULL nothing is stamped (plain packing).  layout == NULL: element i <->
 *                            idx[i] (n elements).  layout != NULL (nside_tile <= nside_mini): scattered to the
 *                            tile-dense layout slot(p) of argus_coadd, n_tiles * ppt elements; slots outside the
 *                            footprint are not written (zero the buffer once), pixels of absent tiles are dropped.
 *                            ARGUS_OPT_SEGMENT_RASTER selects row-major tiles instead of nested order.
 *            n_mini_dev      DEVICE int64, receives n_mini (asynchronous)
 *            n_mini_out      HOST; when not NULL the call synchronises the stream and stores n_mini here.
 * mini_capacity = 0 with every per-minipix output and seg16 NULL only counts.  Minipix beyond mini_capacity are
 * not written (nor are their seg16 pixels): with n_mini_out the call then returns ARGUS_ERR_CAPACITY and
 * *n_mini_out holds the required capacity.  The context keeps 8 (mini_capacity + 1) + n / 8 bytes of scratch,
 * grown on demand (which synchronises the device).  Otherwise asynchronous on `stream`. */
int argus_segment_products(argus_ctx* ctx, int64_t nside, int64_t nside_mini, const int64_t* idx, const float* value,
                           const float* weight, size_t n, const int64_t* targets, size_t n_targets,
                           const argus_coadd* layout, uint16_t* seg16, int64_t* mini_id, float* mini_value,
                           float* mini_weight, uint8_t* mini_keep, size_t mini_capacity, int64_t* n_mini_dev,
                           size_t* n_mini_out, void* stream);

/* ---- Background map and source detection: the paper's two GPU stages between calibration and
 * resampling, "Median-filtered background map" and "Source detection" (PAPER.md:193-194 Table 2; :135; the
 * per-camera "intermediate background and noise maps" of :109).  The paper gives no formula; DESIGN.md section 11
 * lists the readings R-D1 .. R-D6 restated here.  "median" of n values = mean of the order statistics (n-1)/2 and n/2.
 *
 * argus_background_map: frame as for argus_resample (raw + masters: calibration fused; or cal + mask).  The frame is
 * cut into cell x cell pixel cells (cell in {8, 16, 32, 64}; ragged at the right / bottom edge), GX = ceil(W / cell),
 * GY = ceil(H / cell), row-major [GY][GX] grids:
 *   med   = median of the cell's good pixels; sig = 1.4826 * median |v - med|; ngood = number of good pixels;
 *           a cell with ngood < max(n_min, 1) is invalid (med = sig = 0)                      (optional outputs)
 *   bkg   = median of med over the valid cells of the 3 x 3 cell neighbourhood (clipped to the grid); nse likewise
 *           from sig; no valid cell: bkg = 0, nse = +inf                                      (required outputs)
 * All DEVICE pointers, GX * GY elements.  Medians are exact selections (bit-exact for a given float32 frame).
 * Asynchronous on stream; the context keeps 12 bytes of scratch per cell. */
int argus_background_map(argus_ctx* ctx, const argus_frame* frame, int64_t W, int64_t H, int32_t cell, int32_t n_min,
                         float* bkg_out, float* nse_out, float* med_out, float* sig_out, int32_t* ngood_out,
                         void* stream);

/* argus_background_map_static: argus_background_map for callers that may not allocate (code under CUDA graph
 * capture, tight serving loops, harnesses that forbid cudaMalloc).  The same two kernels, the same outputs bit for bit
 * (R-D1, R-D2; Table 2 "Median-filtered background map"), but the 12 bytes of scratch per cell (med, sig,
 * ngood) live in one file-scope device array of the library instead of the context, so the call needs no context and
 * calls no cudaMalloc / cudaFree / allocating library routine, in any call including the first.
 *   - Works on the device that is CURRENT at the call.  The scratch array holds ARGUS_BG_STATIC_MAX_CELLS cells
 *     (12 MiB); every GPU that loads the library holds it until the process exits.  A grid with
 *     GX * GY > ARGUS_BG_STATIC_MAX_CELLS is rejected with ARGUS_ERR_CAPACITY before anything is launched.
 *   - The first call on a device resolves the array's device address (cudaGetSymbolAddress: no allocation, but make it
 *     outside stream capture); later calls only launch.
 *   - All calls on a device share the array and it keeps the last call's contents.  Nothing has to start at zero: the
 *     first kernel writes every one of the GX * GY cells the second kernel reads, the rest is never read.  Two calls
 *     that overlap on the GPU (different streams, or two host threads on one device) RACE on it: serialise them.
 *   frame, W, H, cell, n_min, bkg_out, nse_out: as argus_background_map (DEVICE pointers of the current device).
 *   cuda_error_out: HOST int (may be NULL): receives the cudaError_t when the call returns ARGUS_ERR_CUDA.
 * Asynchronous on stream. */
#define ARGUS_BG_STATIC_MAX_CELLS (1 << 20)
int argus_background_map_static(const argus_frame* frame, int64_t W, int64_t H, int32_t cell, int32_t n_min,
                                float* bkg_out, float* nse_out, int32_t* cuda_error_out, void* stream);

/* One detected source (32 bytes). */
typedef struct argus_source {
    int32_t x, y;      /* peak pixel */
    float peak;        /* s = cal - bkg(x, y) at the peak, ADU */
    float flux;        /* sum of s over the good in-frame pixels of the 3 x 3 window */
    float cx, cy;      /* centroid offsets sum(s dx) / flux, sum(s dy) / flux (0 when flux <= 0): centroid = (x + cx, y + cy) */
    float bkg, nse;    /* interpolated background and noise at the peak */
} argus_source;

/* argus_detect_sources: bkg / nse are the DEVICE grids of argus_background_map for the same (W, H, cell), evaluated
 * per pixel by bilinear interpolation between the cell centres gx * cell + (cell - 1) / 2 (clamped outside the
 * outermost centres).  Pixel p is a source iff it is good, s_p > k_sigma * nse(p), s_p > 0, and s_p is the maximum of
 * its good in-frame 8-neighbours (s_p > s_q for q before p in raster order, s_p >= s_q for q after p).  Pixels whose
 * interpolation touches a cell with nse = +inf are never sources.
 *   out       DEVICE argus_source[capacity], 16-byte aligned.  Catalogue order: ascending raster index y * W + x
 *             (the paper states none; DESIGN.md R-D6).
 *   n_dev     DEVICE int64 (may be NULL): number of sources found (asynchronous)
 *   n_out     HOST (may be NULL): when given the call synchronises the stream and stores the number found; if that
 *             exceeds a non-zero capacity the call returns ARGUS_ERR_CAPACITY, the contents of out are unspecified
 *             (nothing is written beyond capacity) and *n_out is the capacity to call again with.
 * capacity = 0 only counts.  Scratch: 16 bytes per 64 x 32-pixel work tile + 40 bytes per record of capacity, grown on demand (which
 * synchronises the device).  Otherwise asynchronous on stream. */
int argus_detect_sources(argus_ctx* ctx, const argus_frame* frame, int64_t W, int64_t H, int32_t cell, const float* bkg,
                         const float* nse, float k_sigma, argus_source* out, size_t capacity, int64_t* n_dev,
                         size_t* n_out, void* stream);

/* argus_detect_frame: argus_background_map followed by argus_detect_sources in ONE call that reads the frame once
 * (Table 2: the two stages run back to back on every frame; DESIGN.md section 11 "one pass").  While a
 * cell's pixels are in registers for its median, every good pixel above cut = med + kappa * sig of its cell
 * (kappa = max(k_sigma - 2, 2.5); all good pixels of an invalid cell) is noted as a candidate of its 64 x 32-pixel tile.
 * After the 3 x 3 filter a tile is served from its candidates alone when min over the nodes it touches of
 * (bkg + k_sigma * nse) lies above the cuts of the cells it overlaps (then no other pixel can pass the threshold); the
 * other tiles, and tiles with more than 48 candidates, are scanned in full as argus_detect_sources does.
 * bkg_out, nse_out (DEVICE, GX * GY floats, required), out / capacity / n_dev / n_out / error behaviour: exactly the
 * results of the two calls, bit for bit, catalogue order included.  Scratch: 12 + 4 bytes per cell, 120 bytes per
 * tile, 40 bytes per record of capacity, grown on demand (which synchronises the device); otherwise asynchronous. */
int argus_detect_frame(argus_ctx* ctx, const argus_frame* frame, int64_t W, int64_t H, int32_t cell, int32_t n_min,
                       float k_sigma, float* bkg_out, float* nse_out, argus_source* out, size_t capacity, int64_t* n_dev,
                       size_t* n_out, void* stream);

/* Synchronises the stream and reports how many tiles the last argus_detect_frame of this context scanned in full
 * (HOST pointer).  ARGUS_ERR_STATE before the first call. */
int argus_detect_frame_info(argus_ctx* ctx, int64_t* n_full_tiles, void* stream);

/* ---- Direct image subtraction per tile: "Transient detection is performed using image subtraction in
 * the reprojected HEALPix image segments, leveraging long-term coadds as reference frames ... the direct image
 * subtraction method ... for real-time operation in 1-second cadence data" (sec. 5.2), per tile,
 * on the CPU in the paper (20 ms per tile), "a GPU implementation is in development" (:185).  The method's
 * formulas are in the paper's ref [17], not in the paper: DESIGN.md section 13 lists the readings R-X1 .. R-X8 restated here.
 *
 * Both images live on the tile-dense grid of `layout` (argus_coadd: n_tiles * ppt floats, nested order inside a tile) as
 * (sum, wsum) pairs, exactly what argus_resample_coadd accumulates: the science image is the pair of ONE frame (or of a
 * short coadd), the reference the pair of the long-term coadd.  Per pixel and tile:
 *   s = sci_sum / sci_wsum, r = ref_sum / ref_wsum; VALID iff sci_wsum >= sci_wmin and ref_wsum >= ref_wmin
 *   match   ARGUS_SUB_MATCH_NONE: alpha = 1, beta = 0.  ARGUS_SUB_MATCH_AFFINE: per tile, least squares of s ~ alpha r + beta
 *           over the valid pixels (FP64 sums in a fixed order); fewer than n_min valid pixels or a reference without
 *           structure (variance(r) <= 1e-10 mean(r^2): constant up to rounding): alpha = 1, beta = mean(s - r)
 *   diff    d = s - (alpha r + beta) at valid pixels, 0 elsewhere
 *   noise   sigma^2 = (read_noise^2 + max(alpha r + beta, 0) / gain) * (1 / sci_wsum + alpha^2 / ref_wsum)
 *   sig     S = d / sigma at valid pixels, 0 elsewhere
 *   candidate iff valid, S > k_sigma, and S is the maximum over the valid 8-neighbours in the tile's (ix, iy) grid (ix =
 *           even, iy = odd bits of the in-tile nested index; tiles are independent: no neighbours beyond the tile), S_p >
 *           S_q for neighbours with a smaller nested index, S_p >= S_q for larger ones.
 * Outputs (DEVICE): diff_out (required) and sig_out (may be NULL): n_tiles * ppt floats; alpha_out, beta_out (float) and
 * nvalid_out (int32), n_tiles each, may be NULL; cat_out: argus_transient[capacity], 16-byte aligned, ascending nested
 * pixel index; n_dev / n_out / capacity / ARGUS_ERR_CAPACITY exactly as argus_detect_sources.  Scratch grown on demand.
 * Asynchronous on stream unless n_out is given. */
enum { ARGUS_SUB_MATCH_NONE = 0, ARGUS_SUB_MATCH_AFFINE = 1 };

typedef struct argus_subtract_params {
    int32_t match;      /* ARGUS_SUB_MATCH_* */
    int32_t n_min;      /* affine match: minimum number of valid pixels of a tile (>= 2; e.g. 16) */
    float sci_wmin;     /* validity thresholds on the weight sums (> 0; e.g. 0.5) */
    float ref_wmin;
    float read_noise;   /* ADU, > 0 */
    float gain;         /* e- / ADU, > 0 */
    float k_sigma;      /* detection threshold, >= 0 (the paper's Fig. 3: 5) */
    float reserved;
} argus_subtract_params;

/* One transient candidate (32 bytes). */
typedef struct argus_transient {
    int64_t pixel;      /* nested pixel index at nside */
    float sig;          /* S at the peak */
    float diff;         /* d at the peak, ADU */
    float flux;         /* sum of d over the valid pixels of the 3 x 3 window in the tile, ADU */
    float noise;        /* sigma at the peak, ADU */
    int32_t tile_rank;  /* position of the pixel's tile in layout->tiles */
    int32_t reserved;
} argus_transient;

int argus_subtract_tiles(argus_ctx* ctx, const argus_coadd* layout, int64_t nside, const float* sci_sum,
                         const float* sci_wsum, const float* ref_sum, const float* ref_wsum,
                         const argus_subtract_params* params, float* diff_out, float* sig_out, float* alpha_out,
                         float* beta_out, int32_t* nvalid_out, argus_transient* cat_out, size_t capacity, int64_t* n_dev,
                         size_t* n_out, void* stream);

/* Synchronises the stream and reports the statistics of the most recent plan.  Returns ARGUS_ERR_CAPACITY if ANY
 * asynchronous call since the last check (argus_plan_info or argus_healpix_footprint) overflowed its output capacity
 * or the context's max_tiles -- the condition is latched in the context, not in the per-frame plan, so a check after
 * a batch of frames sees the overflow of any of them; reading clears it. */
int argus_plan_info(argus_ctx* ctx, argus_plan_stats* out, void* stream);

/* Synchronises the stream and returns, for the calls recorded since ARGUS_OPT_PROFILE was last set to 1,
 * the summed device time (ms) of the plan kernels and of the fused resample kernel, and the number of
 * calls summed (at most the last 256).  HOST pointers.  Resets the ring. */
int argus_profile_read(argus_ctx* ctx, double* plan_ms, double* kernel_ms, int64_t* n_calls, void* stream);

#ifdef __cplusplus
}
#endif
#endif /* ARGUS_H_ */
