/*
 * lacosmic.h -- C ABI of the B200-native L.A.Cosmic hot path (liblacosmic_b200.so).
 *
 * The operation is the cosmic-ray detection-and-cleaning iteration that PAPER.md:53-62
 * (section Methods/Algorithm, items 1-7) lists and BASELINE.json north_star (1)-(7) defines:
 *   (1) L+  : 2x block-replicate, 3x3 Laplacian, clip negatives, 2x2 block-average
 *   (2) N   = sqrt(gain*med5(img) + readnoise^2)/gain
 *   (3) S   = L+/(2N),  S' = S - med5(S)
 *   (4) F   = max(med3(img) - med7(med3(img)), 0.01)
 *   (5) candidates: S' > sigclip and L+/F > objlim
 *   (6) two 3x3 binary dilations gated by S' > sigclip, then S' > sigfrac*sigclip
 *   (7) every flagged pixel <- median of its unflagged 5x5 neighbours
 * repeated niter times on the cleaned image (parameters: PAPER.md:66-74).  The exact arithmetic
 * (operation order, boundary rule, tie rules) is DESIGN.md section 3, readings R1-R20.
 * Every step runs in hand-written sm_100a CUDA kernels; there is no CPU fallback.
 *
 * Conventions for EVERY entry point unless stated otherwise
 *   - Pointers named *_dev / img / mask_out / clean_out / workspace are DEVICE pointers on the
 *     current CUDA device, owned and allocated by the caller; the library keeps no reference to
 *     them once the work enqueued on `stream` has completed and never frees caller memory.
 *   - Images are row-major contiguous [h][w] (h rows, w columns, pitch = w elements).
 *   - `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).  Calls only
 *     ENQUEUE work and return; they never synchronise the host.  Outputs are valid once the
 *     caller has synchronised `stream`.
 *   - Return value: LACOSMIC_OK (0) or a negative LACOSMIC_ERR_* code.  Nothing is printed, no
 *     exception crosses the boundary, the process is never aborted.  On an argument error no
 *     work is enqueued and no output is touched.
 *   - Input pixels must be finite.  NaN/Inf input is a caller error with unspecified output (a
 *     validation pass would cost a full extra read of the frame).
 */
#ifndef LACOSMIC_H_
#define LACOSMIC_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define LACOSMIC_OK 0
#define LACOSMIC_ERR_NULL (-1)      /* a required pointer is NULL */
#define LACOSMIC_ERR_SHAPE (-2)     /* h < 1, w < 1, or h*w >= 2^31 (or n < 0 for a batch) */
#define LACOSMIC_ERR_PARAM (-3)     /* non-finite parameter; gain < 0; readnoise < 0; sigclip <= 0;
                                       sigfrac <= 0 or > 1; objlim < 0; niter < 0 or > LACOSMIC_MAX_NITER;
                                       satlevel NaN; unknown mode; k not in {3,5,7} */
#define LACOSMIC_ERR_ALIGN (-4)     /* fp32 image pointer not 16-byte aligned, workspace not 256-byte aligned */
#define LACOSMIC_ERR_ALIAS (-5)     /* img, mask_out, clean_out (or workspace) overlap */
#define LACOSMIC_ERR_WORKSPACE (-6) /* workspace_bytes smaller than lacosmic_workspace_bytes(h, w) */
#define LACOSMIC_ERR_CUDA (-7)      /* a CUDA call failed; see lacosmic_last_cuda_error() */
#define LACOSMIC_ERR_TOO_LARGE (-8) /* frame larger than the built-in scratch of lacosmic_masked_median_noalloc */

#define LACOSMIC_MAX_NITER 64

/* Parameters of one frame (PAPER.md:66-74 plus niter/satlevel of the north_star signature).
 * gain [e-/ADU] > 0, or 0 = "not supplied": it is then estimated at each iteration from that iteration's
 * input image (reading R21: residual over sqrt(med5), three rounds of rank-based
 * sigma clipping, gain = the positive root of the noise model's variance equation; every iteration then
 * recomputes all planes); readnoise [e-] >= 0;
 * sigclip > 0: detection limit in sigma; sigfrac in (0,1]: fractional limit for neighbours;
 * objlim >= 0: contrast limit L+/F; satlevel: pixels >= satlevel are never flagged (+INF disables);
 * niter in [0, LACOSMIC_MAX_NITER]: number of iterations (0: clean_out = img, mask_out = 0). */
typedef struct lacosmic_params {
    float gain, readnoise, sigclip, sigfrac, objlim, satlevel;
    int32_t niter;
    int32_t mode; /* LACOSMIC_MODE_LAZY (0, default) or LACOSMIC_MODE_DENSE */
} lacosmic_params;

/* Evaluation mode.  Both modes execute the same fp32 operations on the pixels that decide the result
 * and return bit-identical masks, cleaned frames and counts.
 *   LACOSMIC_MODE_DENSE: med5(S), med3 and med7(med3) are selected at every pixel by the fused
 *     k_fine_gates kernel (the reference path; every debug plane is available).
 *   LACOSMIC_MODE_LAZY: after the dense noise/significance pass, the threshold tests S' > sigclip,
 *     S' > sigfrac*sigclip and L+/F > objlim are evaluated only on the pixels with S above the
 *     threshold (S' <= S because med5(S) >= 0), by counting the window elements that satisfy the same
 *     monotone fp32 test (no selection is needed to compare a median with a threshold); from the
 *     second iteration on, S and the tests are only recomputed near the pixels the previous replacement
 *     rewrote (within 2 px for S, within 4 px for the tests). */
#define LACOSMIC_MODE_LAZY 0
#define LACOSMIC_MODE_DENSE 1

/* Optional per-step dump of ONE iteration (used by the parity tests).  Every pointer is a
 * nullable device pointer to a [h][w] plane (fp32 planes 16-byte aligned): fp32 for Lp (step 1), N (2), S, Sp (3), m3, F (4);
 * uint8 0/1 for G1 = (S' > sigclip), G2 = (S' > sigfrac*sigclip) (both AND img < satlevel),
 * M1 (step 5), M2, M3 (step 6) and C (cumulative mask after the iteration).  LACOSMIC_MODE_LAZY never
 * forms Sp, m3, F and evaluates G2 only where step (6) reads it: those four planes are left untouched
 * there; every other plane is filled and identical in both modes.  An iteration that is skipped because an
 * earlier one flagged nothing new (fixed point, R17) leaves the planes untouched. */
typedef struct lacosmic_debug {
    int32_t iter;   /* iteration whose planes are dumped; -1: none (only `gains` is filled) */
    float *Lp, *N, *S, *Sp, *m3, *F;
    uint8_t *G1, *G2, *M1, *M2, *M3, *C;
    float *gains;   /* nullable device array of p->niter floats: the gain each iteration's noise model used
                       (the supplied gain, or the estimates of R21 when p->gain == 0) */
} lacosmic_debug;

/* ---- the whole path ------------------------------------------------------------------------- */

/* North-star signature (BASELINE.json north_star).  Cleans one frame: mask_out[h][w] uint8 is 1
 * where a pixel was flagged (and replaced) in any iteration, else 0; clean_out[h][w] fp32 is the
 * cleaned frame (equal to img wherever mask_out is 0).  img (const), mask_out and clean_out must
 * not overlap; img and clean_out 16-byte aligned.  Scratch comes from the stream-ordered pool
 * (cudaMallocAsync/cudaFreeAsync on `stream`). */
int lacosmic_run(const float *img, int h, int w, float gain, float readnoise, float sigclip,
                 float sigfrac, float objlim, int niter, float satlevel, uint8_t *mask_out,
                 float *clean_out, void *stream);

/* Scratch size in bytes that lacosmic_run_ws / lacosmic_run_batch / lacosmic_masked_median need for
 * an h x w frame (0 if the shape is invalid). */
size_t lacosmic_workspace_bytes(int h, int w);

/* Same as lacosmic_run with caller-supplied scratch (256-byte aligned device memory of at least
 * lacosmic_workspace_bytes(h,w) bytes, contents undefined before and after).  This is the timed
 * entry point.  iter_counts: nullable DEVICE array of p->niter int32; element t receives the number
 * of pixels newly flagged in iteration t (0 for iterations skipped after a fixed point, which
 * leaves the result unchanged -- DESIGN.md R17).  dbg: nullable HOST struct (read during the call)
 * of device planes to fill for iteration dbg->iter. */
int lacosmic_run_ws(const float *img, int h, int w, const lacosmic_params *p, uint8_t *mask_out,
                    float *clean_out, void *workspace, size_t workspace_bytes, int32_t *iter_counts,
                    const lacosmic_debug *dbg, void *stream);

/* ---- fidelity variants (readings R22-R25) ------------------------------ */

#define LACOSMIC_FS_ADU 0          /* R7, the north-star test: L+/F > objlim, F = max(med3 - med7(med3), 0.01) in ADU */
#define LACOSMIC_FS_NORMALISED 1   /* R22: Fn = max((med3 - med7(med3))/N, 0.01), test S'/Fn > objlim */
#define LACOSMIC_MAX_SATGROW 16

/* Optional variants of one frame; a NULL pointer or {LACOSMIC_FS_ADU, -1, NULL, NULL} is the north-star path.
 *   fsmode : which quantity the object test of step (5) compares (above).
 *   satgrow: -1 = off; k in [0, LACOSMIC_MAX_SATGROW] = extended saturated-star mask (R25): the pixels of
 *            dil3^k(med5(img) >= satlevel), computed once from the input frame, are never flagged (they stay donors).
 *   bpm    : nullable DEVICE uint8 [h][w], != 0 = bad pixel (R23): never flagged, never rewritten, never a donor of
 *            the replacement; its value still enters the filters.
 *   var    : nullable DEVICE fp32 [h][w] (16-byte aligned), variance in ADU^2 (R24): N = sqrt(max(var, 1e-8)) replaces
 *            the noise model of step (2); gain and readnoise are then unused (gain = 0 does not trigger the estimate).
 * bpm / var are read during the call's stream work and must overlap neither the outputs nor the workspace
 * (LACOSMIC_ERR_ALIAS). */
typedef struct lacosmic_variant {
    int32_t fsmode;
    int32_t satgrow;
    const uint8_t *bpm;
    const float *var;
} lacosmic_variant;

/* lacosmic_run_ws with variants (v: nullable HOST struct, read during the call).  Same outputs, same modes: both
 * LACOSMIC_MODE_LAZY and LACOSMIC_MODE_DENSE implement every variant and agree bit for bit.  With fsmode =
 * LACOSMIC_FS_NORMALISED the debug plane F holds Fn. */
int lacosmic_run_ex(const float *img, int h, int w, const lacosmic_params *p, const lacosmic_variant *v,
                    uint8_t *mask_out, float *clean_out, void *workspace, size_t workspace_bytes,
                    int32_t *iter_counts, const lacosmic_debug *dbg, void *stream);

/* ---- separable-median COMPARISON path (R26) ---------------------------- */

/* PAPER.md:29,37 argue that the separable median (row pass, then column pass) "can result in the incorrect removal of
 * cosmic rays by incorrectly classifying the center of near-saturated or saturated stars as cosmic rays".  This entry
 * point exists to show that difference: it runs O0-O7 with med5(img), med5(S), med3 and med7 all replaced by the
 * separable median and is otherwise lacosmic_run_ws (p->mode is ignored; p->gain must be > 0).  It is NOT a product
 * path: nothing else in the library calls it.  workspace: lacosmic_sepmed_workspace_bytes(h, w) bytes. */
size_t lacosmic_sepmed_workspace_bytes(int h, int w);
int lacosmic_run_sepmed_compare(const float *img, int h, int w, const lacosmic_params *p, uint8_t *mask_out,
                                float *clean_out, void *workspace, size_t workspace_bytes, int32_t *iter_counts,
                                const lacosmic_debug *dbg, void *stream);
/* out = separable k x k median of in (k in {3,5,7}); tmp: a third fp32 [h][w] plane (receives the row pass). */
int lacosmic_sepmedfilt(const float *in, float *out, float *tmp, int h, int w, int k, void *stream);

/* n independent frames ("batch processing"; BASELINE.json configs[3]).
 * imgs/masks_out/cleans_out are [n][h][w]; params is a HOST array of n structs (per-frame
 * parameters, read during the call); iter_counts: nullable device array [n][LACOSMIC_MAX_NITER].
 * workspace: k = min(n, LACOSMIC_MAX_BATCH_STREAMS, workspace_bytes / lacosmic_workspace_bytes(h,w))
 * frames are in flight at a time, each with its own slice of the workspace, on k internal streams
 * that fork from and join back into `stream` with events (no host synchronisation; outputs are valid
 * once `stream` reaches the end of the call's work).  One frame's worth of workspace (k = 1) runs the
 * frames back to back on `stream` itself.  Most launches of a frame are latency bound, so frames in
 * flight together overlap well: lacosmic_batch_workspace_bytes(h, w, k) gives the size for k. */
size_t lacosmic_batch_workspace_bytes(int h, int w, int concurrency);
#define LACOSMIC_MAX_BATCH_STREAMS 8
int lacosmic_run_batch(const float *imgs, int n, int h, int w, const lacosmic_params *params,
                       uint8_t *masks_out, float *cleans_out, void *workspace,
                       size_t workspace_bytes, int32_t *iter_counts, void *stream);

/* End-to-end variant with HOST buffers: img_host, mask_out_host, clean_out_host are host pointers
 * (pinned memory makes the copies asynchronous); the call enqueues H2D copy, the whole path and
 * the D2H copies on `stream`.  dev_workspace: device scratch of at least
 * lacosmic_host_workspace_bytes(h,w) bytes (frame staging + lacosmic_workspace_bytes), 256-byte
 * aligned.  Results are valid after the caller synchronises `stream`.  For frames of at least 1024 rows (lazy mode,
 * gain supplied, w % 4 == 0) the H2D copy is issued in eight bands on a copy stream the library keeps per calling thread
 * and device (ordered after the work already on `stream`), and the first pass of the path follows it band by band on
 * `stream`; the img_host buffer must stay unchanged until `stream` has been synchronised, as for any asynchronous copy. */
size_t lacosmic_host_workspace_bytes(int h, int w);
/* Diagnostic: the plan of that banded copy for an h x w frame, a function of the shape alone (no GPU needed).  Returns
 * the number of bands n <= LACOSMIC_HOST_BANDS (0: the frame is copied in one piece; negative: error code) and fills the
 * HOST arrays row_end[b] = first row NOT in bands 0..b and tile_rows[b] = how many rows of tiles of the first pass
 * (LACOSMIC_HOST_TILE_ROWS input rows each, reading LACOSMIC_HOST_TILE_MARGIN more rows above and below) are released once
 * band b has arrived.  tests/test_abi_cpu.py checks for every height that no row of tiles is released before the last
 * row it reads is on the device.  (Bands are also conditional on lazy mode, a supplied gain and fp32 input.) */
#define LACOSMIC_HOST_BANDS 8
#define LACOSMIC_HOST_TILE_ROWS 32
#define LACOSMIC_HOST_TILE_MARGIN 2
int lacosmic_host_band_plan(int h, int w, int32_t *row_end, int32_t *tile_rows);
int lacosmic_run_host(const float *img_host, int h, int w, const lacosmic_params *p,
                      uint8_t *mask_out_host, float *clean_out_host, void *dev_workspace,
                      size_t dev_workspace_bytes, void *stream);

/* Raw-frame ingest: as lacosmic_run_host, but the input is the detector's uint16 frame
 * (ADU counts, row-major [h][w], 2-byte aligned); it is copied as 2 bytes per pixel and widened to fp32 on
 * the device (exact: every uint16 is an fp32 value), which halves the host-to-device traffic.  The result
 * equals lacosmic_run_host on the widened frame.  dev_workspace as for lacosmic_run_host. */
int lacosmic_run_host_u16(const uint16_t *img_host, int h, int w, const lacosmic_params *p,
                          uint8_t *mask_out_host, float *clean_out_host, void *dev_workspace,
                          size_t dev_workspace_bytes, void *stream);

/* Sparse results for a pipeline that keeps the input frame on the host: the cleaned
 * frame equals the input outside the mask, so instead of the two full planes (5 bytes per pixel over PCIe)
 * the call returns the final mask as a bit-plane (maskbits_host: [h][lacosmic_bitplane_pitch_words(w)] words,
 * bit k of word j of a row = pixel 32 j + k) and the flagged pixels as a list in ascending flat-index order:
 * idx_host[i] = y*w + x, val_host[i] = the replacement value, for i < min(*count_host, capacity);
 * *count_host is the number of flagged pixels (a value above `capacity` means the list was truncated).
 * `capacity` entries of idx/val are copied whatever the count (no host synchronisation inside the call), so
 * size it to the expected mask fraction.  All four outputs are HOST pointers; dev_workspace as for
 * lacosmic_run_host.  clean[idx[i]] = val[i] applied to a copy of the input reproduces lacosmic_run_host. */
int lacosmic_run_host_sparse(const float *img_host, int h, int w, const lacosmic_params *p,
                             uint32_t *maskbits_host, int32_t *idx_host, float *val_host,
                             int32_t *count_host, int capacity, void *dev_workspace,
                             size_t dev_workspace_bytes, void *stream);

/* The production configuration of a nightly pipeline: a stream of n raw
 * frames in, sparse results out.  imgs_host: [n][h][w] fp32 (input_is_u16 = 0) or uint16 (= 1) host frames;
 * per frame f the call returns maskbits_host[f] ([h][pitch] words), idx_host[f*capacity ...], val_host[f*capacity
 * ...] and counts_host[f] exactly as lacosmic_run_host_sparse does for one frame.  Frames go through staging
 * slots on internal streams like lacosmic_run_host_batch (same dev_workspace sizing), so the H2D copy of one
 * frame overlaps the kernels of another; per frame only 2 or 4 bytes per pixel cross PCIe on the way in and
 * about 0.4 bytes per pixel on the way out. */
int lacosmic_run_host_stream_sparse(const void *imgs_host, int input_is_u16, int n, int h, int w,
                                    const lacosmic_params *params, uint32_t *maskbits_host,
                                    int32_t *idx_host, float *val_host, int32_t *counts_host, int capacity,
                                    void *dev_workspace, size_t dev_workspace_bytes, void *stream);

/* Stream of n independent frames in HOST buffers (a nightly pipeline
 * of >1000 frames per 15 minutes).  imgs_host/masks_host/cleans_host are [n][h][w] host arrays (pinned
 * memory makes the copies asynchronous and lets them overlap), params a host array of n structs.  Frame f
 * uses staging slot f % k on an internal stream (H2D copy, the whole path, D2H copies, in that order),
 * k = min(n, LACOSMIC_MAX_BATCH_STREAMS, dev_workspace_bytes / lacosmic_host_workspace_bytes(h,w)), so with
 * k >= 3 the H2D copy of one frame, the kernels of another and the D2H copy of a third run at the same
 * time; the streams fork from and join back into `stream` with events (no host synchronisation).
 * lacosmic_host_batch_workspace_bytes(h, w, k) gives the device scratch size for k slots. */
size_t lacosmic_host_batch_workspace_bytes(int h, int w, int concurrency);
int lacosmic_run_host_batch(const float *imgs_host, int n, int h, int w, const lacosmic_params *params,
                            uint8_t *masks_host, float *cleans_host, void *dev_workspace,
                            size_t dev_workspace_bytes, void *stream);

/* ---- single steps (each is the kernel the whole path uses; exported for parity tests) -------- */

/* R21 alone: the gain estimate of one image (what the whole path computes at the start of an iteration when
 * p->gain == 0), for the given read noise [e-].  gain_out: DEVICE pointer to one float; stats_out: nullable
 * DEVICE pointer to 6 floats {c, s, lo, hi, kept, mt}: centre, 1.4826 MAD, the interval the last clipping
 * round started from, the number of pixels inside it, the typical signal (rank-(kept-1)/2 element of
 * max(med5, 1e-4) over those pixels).  workspace as for lacosmic_run_ws.  (Version 0.3 of the library wrote a seventh
 * float behind the six; from 0.4 on this symbol writes six again and the seventh has its own pointer below.) */
int lacosmic_estimate_gain(const float *img, int h, int w, float readnoise, float *gain_out,
                           float *stats_out, void *workspace, size_t workspace_bytes, void *stream);
/* The same with path_out: nullable DEVICE pointer to one float that receives 1 if the three clipping rounds were
 * resolved on the zone lists (two reads of the residual plane, csrc/selectz.cuh), 0 if by radix passes over the plane
 * (csrc/select.cuh; taken when the fast path is switched off, on frames of a few pixels or of few distinct values, or
 * when a check of the fast path fails) -- gain and statistics are the same bits either way. */
int lacosmic_estimate_gain_ex(const float *img, int h, int w, float readnoise, float *gain_out, float *stats_out,
                              float *path_out, void *workspace, size_t workspace_bytes, void *stream);

/* Diagnostic: the plan of the last gain estimate that ran in `workspace` (csrc/selectz.cuh, struct SelZone), copied to
 * the HOST array info_host[LACOSMIC_GAIN_ZONE_WORDS] as 32-bit words after synchronising `stream`:
 *   0-1 base, scale of the bucket grid (float bits); 2-7 bucket ranges of Z0, Z-, Z+ (lo, hi each); 8-9 last bucket of
 *   OUT-, first of OUT+; 10 values below Z0; 11-13 values in Z0, Z-, Z+; 14 values between Z- and Z+; 15-16 values in
 *   OUT-, OUT+; 17 pixels; 18-22 list cursors; 23 plan made; 24 rounds resolved on the lists; 25 where the fast path
 *   stopped (0 it did not; 1 off / no grid; 2-4 plan; 10 j + 1..4: round j, bounds / centre / MAD rank / MAD); 26 the
 *   residuals that are exactly +0; 27 the negative residuals in the bucket of 0; the typical signal: 28-29 base, scale of
 *   its bucket grid (float bits); 30-31 bucket range of its zone; 32 values below the zone; 33 values in it; 34 list
 *   cursor; 35 zone made; 36 selected on the list (0: by radix passes over the med5 plane). */
#define LACOSMIC_GAIN_ZONE_WORDS 40
int lacosmic_gain_zone_info(const void *workspace, int h, int w, int32_t *info_host, void *stream);

/* Switches the fast path of the gain estimate on (default; environment LACOSMIC_GAIN_FAST=0 starts with it off)
 * or off, for the whole process.  Results do not depend on it. */
int lacosmic_gain_fast_path_enable(int enable);

/* Step (1): out = L+(in).  in/out fp32 [h][w], distinct. */
int lacosmic_lplus(const float *in, float *out, int h, int w, void *stream);

/* True (non-separable) k x k median with edge-replicate borders, k in {3,5,7}.
 * in/out fp32 [h][w], distinct. */
int lacosmic_medfilt(const float *in, float *out, int h, int w, int k, void *stream);

/* Bit-plane layout used by the mask steps: row pitch lacosmic_bitplane_pitch_words(w) =
 * ceil(w/32) uint32 words, pixel x of a row in word x/32, bit x%32 (LSB = lowest x); pad bits 0. */
int lacosmic_bitplane_pitch_words(int w);
int lacosmic_pack_bits(const uint8_t *mask_u8, uint32_t *bits, int h, int w, void *stream);
int lacosmic_unpack_bits(const uint32_t *bits, uint8_t *mask_u8, int h, int w, void *stream);

/* Step (6) primitive: 3x3 binary dilation (8-connected, outside the frame = 0) on bit-planes.
 * bits_in/bits_out distinct, [h][pitch] uint32. */
int lacosmic_dilate3(const uint32_t *bits_in, uint32_t *bits_out, int h, int w, void *stream);

/* Step (7): out = img where mask_u8 == 0, else the median of the unmasked 5x5 edge-replicated
 * neighbours (even count: mean of the two middle values; none: plain 5x5 median).  workspace as
 * for lacosmic_run_ws. */
int lacosmic_masked_median(const float *img, const uint8_t *mask_u8, float *out, int h, int w,
                           void *workspace, size_t workspace_bytes, void *stream);

/* Step (7) with bad pixels removed from the donors (R23); bpm_u8 nullable (then lacosmic_masked_median). */
int lacosmic_masked_median_bpm(const float *img, const uint8_t *mask_u8, const uint8_t *bpm_u8, float *out, int h,
                               int w, void *workspace, size_t workspace_bytes, void *stream);

/* ---- step (7) for callers that cannot allocate device memory ----------------------------------- */

/* Some code that wants step (7) has no way to obtain scratch memory for it: a plug-in running inside a host
 * application that owns the GPU's memory pool and hands out only the input and output buffers; a real-time loop
 * that may not enter the allocator (cudaMalloc can block, and synchronises the device) once it has started; a
 * process whose memory budget was fixed at start-up and is used up.  Every other entry point of this library
 * that needs scratch takes a `workspace` the caller must have allocated, or (lacosmic_run) draws from the
 * stream-ordered pool.  This one needs neither: its scratch -- five bit-planes and a counter -- is a fixed array
 * inside the library's own device image.
 *
 * Same operation and same kernels as lacosmic_masked_median_bpm (bpm_u8 nullable), same results bit for bit:
 * out = img where mask_u8 == 0, else the median of the unmasked (and not bad) 5x5 edge-replicated neighbours.
 * img, mask_u8, bpm_u8, out are the caller's DEVICE buffers ([h][w]; img and out must not overlap).
 *
 * Limit: h * lacosmic_bitplane_pitch_words(w) <= LACOSMIC_NOALLOC_MAX_WORDS (131072 words: any frame up to 2048 x 2048
 * pixels, or e.g. 1024 x 4096).  A larger frame returns LACOSMIC_ERR_TOO_LARGE and enqueues nothing.  The array
 * occupies LACOSMIC_NOALLOC_SCRATCH_BYTES (2.5 MiB + 256 bytes) of every GPU on which the process loads this library, from the
 * moment the library's device code is loaded there until the process exits, whether or not this call is ever made.
 *
 * The call itself makes no cudaMalloc / cudaFree / cudaMallocAsync and calls no routine that allocates: it enqueues
 * two or three small kernels, one device-to-device copy and two memsets on `stream`.  The FIRST call on each device
 * also looks up the array's address on that device (cudaGetSymbolAddress, with that device current; the result is
 * kept per device under a lock).  That look-up may make the CUDA runtime load the library's device code, so make
 * the first call on a device during set-up, before any stream capture and before the phase that must not allocate.
 *
 * There is ONE array per GPU and every call on that GPU uses it, from whichever thread or stream.  Calls that are
 * ordered on the GPU (same stream, or streams ordered by events) are safe: each call re-initialises the parts it
 * relies on and never reads what an earlier call left behind.  Two calls that can run on the GPU at the same time
 * (different streams with no ordering between them) race on the array and give undefined results: serialise them
 * yourself, or use lacosmic_masked_median_bpm with one workspace per stream. */
#define LACOSMIC_NOALLOC_MAX_WORDS 131072
#define LACOSMIC_NOALLOC_SCRATCH_BYTES (5 * LACOSMIC_NOALLOC_MAX_WORDS * 4 + 256)
int lacosmic_masked_median_noalloc(const float *img, const uint8_t *mask_u8, const uint8_t *bpm_u8, float *out,
                                   int h, int w, void *stream);

/* R25 alone: out_u8[h][w] = 1 on dil3^grow(med5(img) >= satlevel), else 0.  workspace as for lacosmic_run_ws. */
int lacosmic_satstar_mask(const float *img, int h, int w, float satlevel, int grow, uint8_t *out_u8, void *workspace,
                          size_t workspace_bytes, void *stream);

/* ---- diagnostics ---------------------------------------------------------------------------- */
const char *lacosmic_strerror(int code);
/* cudaError_t (as int) of the last failing CUDA call made by this library on the calling thread. */
int lacosmic_last_cuda_error(void);
/* Number of kernel launches the last lacosmic_run* call on this thread enqueued (bench.py reports
 * it as gpu_launches). */
int lacosmic_last_launch_count(void);
const char *lacosmic_version(void);

/* Work counters of the last frame that ran in `workspace` (the lazy path's data-dependent work; bench.py turns them into
 * the per-kernel terms of the whole-step roofline).  stats_host: HOST array
 * [LACOSMIC_NUM_FRAME_STATS][LACOSMIC_MAX_NITER] of int32, row r, iteration t:
 *   0 newly flagged pixels; 1 candidates evaluated (pixels with S > sigclip listed for the tests); 2 quads (aligned groups
 *   of 4 pixels) whose S the incremental pass recomputed; and, only for frames run after lacosmic_stats_enable(1) on the
 *   calling thread (two extra atomics per warp, so off by default): 3 pixels whose replacement value was computed;
 *   4 candidates that passed S' > sigclip and took the fine-structure test.
 * Copies 5 * 64 * 4 bytes device-to-host and SYNCHRONISES `stream`. */
#define LACOSMIC_NUM_FRAME_STATS 5
int lacosmic_stats_enable(int enable);
int lacosmic_frame_stats(const void *workspace, int h, int w, int32_t *stats_host, void *stream);

/* Replay of repeated calls from a CUDA graph (process-wide switch; on by default, also off with the environment
 * variable LACOSMIC_GRAPHS=0).  The launch sequence of lacosmic_run_ws is a function of its arguments alone (pointers,
 * shape, parameters; everything data-dependent is decided on the device), so from the second call with identical
 * arguments on the library captures the sequence once into a CUDA graph and later calls enqueue that graph: the same
 * kernels run on every call, the host-side launch work is reused (about 2 us per dependent kernel; CUDA graphs are the
 * launch mechanism the Blackwell guide recommends for launch-bound loops).  The 16 most recently used argument sets are
 * kept.  Not used when `dbg` is given, while kernel timing or statistics are enabled, on the legacy default stream, or
 * on a stream the caller is capturing (the call then enqueues its kernels directly, as always).  enable = 0 also drops
 * the cached graphs.  Results and ordering on `stream` are identical either way.  Threads: the table of cached graphs is
 * locked only for the look-up; capture, instantiation and launch hold a lock of the one entry, so calls with different
 * arguments (other GPUs, streams, frames) do not serialise on each other.  The switch of the gain estimate's fast path is
 * part of the key, so flipping it never replays a sequence captured under the other setting. */
int lacosmic_graph_replay_enable(int enable);

/* Measured peak of the "alu" roofline (the medians of PAPER.md:23,64 are fp32 min/max selection
 * networks, bound by the rate at which the SMs issue FMNMX).  Runs a register-only kernel of independent min/max chains
 * (kind 0: two-input FMNMX; kind 1: three-input FMNMX3) on every SM of the current device and writes the achieved
 * thread-level instructions per second to *instr_per_s_host (HOST pointer).  Unlike every other entry point this
 * diagnostic allocates 256 bytes of device memory, SYNCHRONISES `stream` and takes about 10 ms. */
int lacosmic_probe_minmax_rate(int kind, double *instr_per_s_host, void *stream);

/* Optional CUDA-event timing per kernel class, per calling thread.  After
 * lacosmic_kernel_timing_enable(1) every launch of the whole-path entry points is bracketed by an
 * event pair on the caller's stream (up to 8192 spans between reads).  Once the caller has
 * synchronised the stream, lacosmic_kernel_timing_read() writes, for each class c <
 * LACOSMIC_NUM_KERNEL_CLASSES, the summed device time ms_sum[c] and the number of spans[c] (HOST
 * arrays), and clears the record.  Class names: lacosmic_kernel_class_name(c); the last class is the
 * whole frame (copies included). */
#define LACOSMIC_NUM_KERNEL_CLASSES 9
int lacosmic_kernel_timing_enable(int enable);
int lacosmic_kernel_timing_read(float *ms_sum, int32_t *spans);
const char *lacosmic_kernel_class_name(int cls);

#ifdef __cplusplus
}
#endif
#endif /* LACOSMIC_H_ */
