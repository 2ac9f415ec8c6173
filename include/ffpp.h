/* ffpp.h — C ABI of libffpp: B200 (sm_100a) post-processing of a single-class anchor-free detector head.
 *
 * The operation (BASELINE.json north_star; the paper states the
 * problem only as "generating bounding boxes with confidence scores" from model output, §2.3, with
 * post-processing the dominant per-frame cost, §3.2, and "mapping chicken positions onto a
 * spatial grid to generate density heatmaps", §2.3 / Algorithm 1 PAPER.md:L193-234 / §3.6):
 *
 *   for every frame f of a (possibly mixed-resolution) batch, independently
 *     1. decode candidate j -> (level, ix, iy); grid point p = ((ix+.5)s, (iy+.5)s);
 *        box = (px - l s, py - t s, px + r s, py + b s) in fp32; survivor iff logit > ln(conf/(1-conf))   [O1-O3]
 *     2. order survivors by (logit descending, candidate index ascending); keep the first min(n, top_k)    [O4]
 *     3. greedy NMS in that order: i is kept iff no earlier kept j has IoU(j,i) > iou_thresh,
 *        IoU = inter / ((areaA + areaB) - inter), every operation a separately rounded fp32 op              [O5]
 *     4. density grid: kept boxes' centroids binned into cell_px cells (in-frame only), convolved with a
 *        separable truncated Gaussian (normalised taps, radius floor(truncate*sigma), reflect border)      [O7]
 *
 * All entry points are plain C, no C++ types, no exceptions across the boundary.  Every pointer is marked
 * HOST or DEVICE.  Return value: FFPP_OK (0) or a negative ffpp_status.
 */
#ifndef FFPP_H_
#define FFPP_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum ffpp_status {
  FFPP_OK = 0,
  FFPP_EINVAL = -1,    /* null pointer, B < 0, bad dtype/stride/dims, N_f != sum_l W*H/s_l^2, misaligned raw, ... */
  FFPP_ECAPACITY = -2, /* batch exceeds the capacities given to ffpp_create                                    */
  FFPP_ECUDA = -3,     /* CUDA runtime / launch error; text via ffpp_last_error                                  */
  FFPP_ENOMEM = -4     /* workspace allocation failed in ffpp_create                                             */
} ffpp_status;

typedef struct ffpp_handle ffpp_handle; /* opaque; owned by the library */

/* Method + capacity parameters.  Zero-initialise, then fill. */
typedef struct ffpp_params {
  int32_t dtype;           /* 0 = fp32, 1 = fp16 (IEEE binary16) rows of the raw head output                       */
  float conf_thresh;       /* threshold on sigmoid(logit), strict >, applied as logit > ln(c/(1-c))  (A7)          */
  float iou_thresh;        /* strict >; must be >= 0                                                   (A11)        */
  int32_t top_k;           /* >= 1; at most 24576 (fp16 rows with N_f <= 65536) or 12288 (otherwise): the top-K set of
                              a frame (keys, spatial bins) is held in one SM's 227 KB of shared memory by a2/a4      */
  int32_t num_levels;      /* 1..4                                                                                  */
  int32_t strides[4];      /* ascending powers of two, e.g. {8,16,32}                                  (A5)         */
  int32_t cell_px;         /* density cell edge in pixels, e.g. 8                                                   */
  float sigma_cells;       /* Gaussian sigma in cells, > 0                                                          */
  float truncate_sigmas;   /* radius R = floor(truncate_sigmas * sigma_cells), 1 <= R <= 32            (A15)        */
  int32_t max_frames;      /* capacity: B <= max_frames                                                             */
  int64_t max_total_candidates; /* capacity: sum_f N_f                                                              */
  int32_t max_frame_w;     /* capacity: W_f <= max_frame_w                                                          */
  int32_t max_frame_h;     /* capacity: H_f <= max_frame_h                                                          */
  int64_t max_total_cells; /* capacity: sum_f (W_f/cell)(H_f/cell); 0 = max_frames * (max_w/cell)(max_h/cell)       */
  int64_t nms_workspace_bytes; /* capacity of the NMS suppression-edge pool in bytes (4 per edge, shared out to the
                                  frames in proportion to min(N_f, top_k)); 0 = nms_edges_per_box edges per box       */
  int32_t nms_edges_per_box; /* 0 = 16.  An edge is one unordered pair {a, b} with IoU > iou_thresh; the flock
                                workloads have 4-9 per box.  The pool is a speed knob, never a correctness limit: a
                                frame that needs more than its share is resolved by the pool-free overflow path of a4
                                (same result, bounded workspace, slower for that frame)                               */
  int32_t reserved_;
} ffpp_params;

/* One kept detection (24 bytes).  score = sigmoid(logit) in fp32; cand_index = candidate index within its frame. */
typedef struct ffpp_box {
  float x1, y1, x2, y2;
  float score;
  int32_t cand_index;
} ffpp_box;

/* Create a handle on the CURRENT CUDA device: validates p, allocates every byte of device workspace and pinned
 * staging the handle will ever use, precomputes the logit threshold and the Gaussian taps ("initialize grid once",
 * PAPER.md:L219).  *out is set only on success.  Errors: EINVAL (bad params), ENOMEM, ECUDA. */
int ffpp_create(const ffpp_params* p /*HOST*/, ffpp_handle** out /*HOST*/);

/* Run the whole path on one batch; everything is enqueued on `stream`, nothing is allocated, the host is never
 * synchronised.  The frame descriptor table of a batch geometry (B, N_per_frame, frame_dims) is built on first
 * sight, uploaded with one stream-ordered copy and cached in one of 32 device slots (least recently used slot is
 * replaced), so alternating geometries cost nothing after their first call.  CUDA-graph capturable when the
 * geometry is cached (run it once before capturing; an uncached geometry under capture returns FFPP_EINVAL).
 * Results are complete when `stream` reaches the point after the call; the caller synchronises.
 *
 *   raw          DEVICE  [sum_f N_f][5] values (l, t, r, b in stride units, score logit) in params.dtype, frames
 *                        tightly concatenated in order (A22); 16-byte aligned base.  Read only.
 *   B            number of frames, 0 <= B <= max_frames.  B == 0: success, touches nothing.
 *   N_per_frame  HOST    [B] candidates per frame; must equal sum_l W*H/s_l^2 (O1, A21).  Read before return.
 *   frame_dims   HOST    [B][2] = (W, H) pixels; W a multiple of the largest stride and of cell_px, H a multiple
 *                        of cell_px, W*H a multiple of s_l^2 for every level.  Read before return.
 *   stream       cudaStream_t (as void*); NULL = legacy default stream.
 *   out_boxes    DEVICE  [B][top_k] ffpp_box, 8-byte aligned base; rows [0, out_counts[f]) of frame f are valid, in keep order
 *                        (= score order); the rest is left untouched.
 *   out_counts   DEVICE  [B] int32: boxes kept by NMS (in-frame or not, A19).
 *   out_density  DEVICE  float32, per-frame row-major [H/cell][W/cell] grids concatenated in frame order; every
 *                        cell is written.
 * The caller owns all five arrays.  Errors: EINVAL, ECAPACITY, ECUDA; no partial-write promise on error. */
int ffpp_run(ffpp_handle* h, const void* raw /*DEVICE*/, int32_t B, const int32_t* N_per_frame /*HOST*/,
             const int32_t* frame_dims /*HOST*/, void* stream, ffpp_box* out_boxes /*DEVICE*/,
             int32_t* out_counts /*DEVICE*/, float* out_density /*DEVICE*/);

/* The same path with HOST buffers (the call a user without device buffers makes): copies raw host->device,
 * runs, copies the three outputs device->host through the handle's own staging, and synchronises `stream`
 * before returning.  raw / out_* are HOST pointers (pinned memory makes the copies asynchronous DMA; a pinned
 * out_boxes is written by one kernel through its device alias).  Batches of >= 16 MB and >= 12 frames are cut by
 * bytes into up to 6 runs of whole frames (frames are independent; consecutive runs alternate between two compute
 * streams and two workspaces, the second one created on the first such call) so that the upload of the next run and the
 * download of the previous one, on two internal copy streams, overlap the kernels of the current run on
 * `stream` (the D2H copy + CPU post-processing the paper blames; L308-310: streams as the remedy). */
int ffpp_run_host(ffpp_handle* h, const void* raw /*HOST*/, int32_t B, const int32_t* N_per_frame /*HOST*/,
                  const int32_t* frame_dims /*HOST*/, void* stream, ffpp_box* out_boxes /*HOST*/,
                  int32_t* out_counts /*HOST*/, float* out_density /*HOST*/);

/* Release all device and pinned memory.  NULL is a no-op. */
int ffpp_destroy(ffpp_handle* h);

/* Static or handle-owned NUL-terminated text of the last error on h (h == NULL: last create error). */
const char* ffpp_last_error(const ffpp_handle* h);

/* Constants the handle derived from its parameters, for cross-checking against an independent computation. */
typedef struct ffpp_info {
  float logit_threshold;   /* T = (float) ln(conf/(1-conf))                                                        */
  int32_t radius;          /* R                                                                                     */
  float taps[65];          /* w[-R..R] at taps[0..2R], fp32-rounded, normalised by their discrete sum in double     */
  int32_t key_bits;        /* 32 or 64: width of the (score, index) sort key                                        */
  int64_t workspace_bytes; /* device bytes owned by the handle                                                      */
  int32_t sm_count;
} ffpp_info;
int ffpp_get_info(const ffpp_handle* h, ffpp_info* out /*HOST*/);

/* Stage timing.  When enabled, ffpp_run records CUDA events on `stream` around each stage of the NEXT runs;
 * ffpp_get_stage_ms (after the caller synchronised the stream) returns the last run's durations in ms:
 *   [0] scheduler upload + counter reset   (a0)      [1] decode/threshold/compaction        (a1)
 *   [2] top-K select + decode + spatial bin (a2)     [3] NMS suppression edges              (a3)
 *   [4] NMS resolve + order + output gather (a4)      [5] density histogram + convolution    (a5-a6)
 * Event recording makes the run non-capturable; leave it off for graph capture. */
#define FFPP_NUM_STAGES 6
int ffpp_set_stage_timing(ffpp_handle* h, int32_t enable);
int ffpp_get_stage_ms(ffpp_handle* h, float* ms_out /*HOST [FFPP_NUM_STAGES]*/);

#ifdef __cplusplus
}
#endif
#endif /* FFPP_H_ */
