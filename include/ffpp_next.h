/* ffpp_next.h — C ABI of the steps around the hot path that SURVEY.md §8(f) ranks next (f1-f4).  Same conventions as
 * ffpp.h: plain C, every pointer marked HOST or DEVICE, return FFPP_OK (0) or a negative ffpp_status, everything is
 * enqueued on `stream`, the host is never synchronised.  The paper names these steps and prints no formula for any
 * of them; the definitions are the readings B1-B6 of DESIGN.md §3 (restated in oracle/ffpp_next_oracle.cpp).
 */
#ifndef FFPP_NEXT_H_
#define FFPP_NEXT_H_

#include "ffpp.h"

#ifdef __cplusplus
extern "C" {
#endif

/* One connected region of a thresholded grid (f1) or mask (f3): 32 bytes. */
typedef struct ffpp_region {
  int32_t label;          /* smallest row-major cell / pixel index of the component (its label in out_labels)       */
  int32_t area;           /* cells / pixels                                                                          */
  int32_t x0, y0, x1, y1; /* inclusive bounding box, cells / pixels                                                  */
  float mass;             /* f1: sum of the density over the region; f3: mean probability over the component (score) */
  int32_t reserved_;
} ffpp_region;

/* f1 — heatmap analytics on density grids (§2.3 Clustering: "Clusters are identified by thresholding
 * these heatmaps and applying connected component analysis to detect areas of local aggregation"; Algorithm 1
 * "Compute heatmap, entropy, clustering degree"; §3.6).  Per frame f of the batch:
 *   out_entropy[f] = -sum p ln p over the cells, p = D / sum(D), cells with D <= 0 skipped; 0 if sum(D) <= 0    (B1)
 *   out_degree[f]  = 1 - entropy / ln(n_cells); 0 if n_cells <= 1 or sum(D) <= 0                                 (B2)
 *   regions        = connected components (connectivity 4 or 8) of {D > threshold}, strict                        (B3)
 *   out_labels     = per cell, the smallest row-major cell index of its region, -1 for background
 *   out_regions[f][k], k < min(count, max_regions): the regions in ascending label order with cell count,
 *                    inclusive bounding box and mass; out_region_counts[f] = number of regions (may exceed max_regions).
 *
 *   density        DEVICE  float32, per-frame row-major [H/cell][W/cell] grids concatenated (ffpp_run's out_density
 *                          layout; any buffer of that layout will do).  Read only.
 *   frame_dims     HOST    [B][2] = (W, H) pixels, multiples of params.cell_px.  Read before return; the per-frame
 *                          grid table is uploaded on first sight of a geometry and cached (8 slots), like ffpp_run's.
 *   out_entropy, out_degree  DEVICE [B] float64.   out_labels  DEVICE int32, same layout as density.
 *   out_regions    DEVICE  [B][max_regions].       out_region_counts  DEVICE [B] int32.
 * Scratch (one int32 per cell, one 64-bit sum per table row, the entropy partials) is allocated by the handle on the
 * first call that needs more than it has; that call is not graph-capturable.  Errors: EINVAL, ECAPACITY, ECUDA. */
int ffpp_heatmap_stats(ffpp_handle* h, const float* density /*DEVICE*/, int32_t B, const int32_t* frame_dims /*HOST*/,
                       float threshold, int32_t connectivity, int32_t max_regions, void* stream,
                       double* out_entropy /*DEVICE*/, double* out_degree /*DEVICE*/, int32_t* out_labels /*DEVICE*/,
                       ffpp_region* out_regions /*DEVICE*/, int32_t* out_region_counts /*DEVICE*/);

/* f2 — exact-position density, the paper's own formulation (Algorithm 1 DefaultClustering: "for all
 * grid cells / for all chickens / Compute distance and update density"; L225 "Vectorized density map (cdist)"; §3.6
 * L242).  Every kept box of frame f whose fp32 centroid (cx, cy) = ((x1+x2)/2, (y1+y2)/2) lies in [0,W) x [0,H) adds
 *     exp(-(dx^2 + dy^2) / (2 sigma^2)) / Z^2,   dx = (ix + 0.5) - cx/cell,  dy = (iy + 0.5) - cy/cell  (fp32)
 * to every cell (ix, iy) with |dx| <= R and |dy| <= R; sigma, R and Z (the discrete tap sum) are the handle's (A15), so a
 * centroid on a cell centre reproduces ffpp_run's binned grid.  No border fold: mass outside the grid is lost   (B4).
 *   boxes / counts DEVICE  ffpp_run's out_boxes [B][top_k] and out_counts [B] (rows [0, counts[f]) are read).
 *   frame_dims     HOST    [B][2]; cached like f1's.     out_density  DEVICE float32, ffpp_run's out_density layout. */
int ffpp_density_exact(ffpp_handle* h, const ffpp_box* boxes /*DEVICE*/, const int32_t* counts /*DEVICE*/, int32_t B,
                       const int32_t* frame_dims /*HOST*/, void* stream, float* out_density /*DEVICE*/);

/* f3 — segmentation-mask post-processing, the step the paper accelerated on the CPU (§2.3: "applying a
 * threshold to the model's output, extracting connected components, and generating bounding boxes from the resulting
 * masks"; §3.2: 40.2 -> 11.4 ms per frame; L310: "remained CPU-bound").  Per frame: foreground = prob >
 * threshold (strict); components under connectivity 4 or 8; label = smallest row-major pixel index; per component the
 * pixel count, inclusive bounding box and score = mean probability; components with area < min_area are left out of
 * the table (not of the label image); the table is in ascending label order                                     (B5).
 *   mask           DEVICE  [B][H][W] probabilities, dtype 0 = fp32, 1 = fp16.  Read only.
 *   out_labels     DEVICE  [B][H][W] int32.   out_components  DEVICE [B][max_components].   out_counts  DEVICE [B].
 * Needs one int32 of scratch per pixel of the batch: allocated by the handle on the first call that needs more than it
 * has (that call is not graph-capturable); W*H < 2^31. */
int ffpp_mask_components(ffpp_handle* h, const void* mask /*DEVICE*/, int32_t dtype, int32_t B, int32_t W, int32_t H,
                         float threshold, int32_t connectivity, int32_t min_area, int32_t max_components, void* stream,
                         int32_t* out_labels /*DEVICE*/, ffpp_region* out_components /*DEVICE*/, int32_t* out_counts /*DEVICE*/);

/* f4 — pre-processing (§2.3: "image resizing, normalization, and conversion to tensor format"; 8.8 ms
 * per frame, L151): bilinear resize with half-pixel centres (src = (dst + 0.5) * scale - 0.5, clamped at 0, the right /
 * lower neighbour clamped at the last pixel), then (v / 255 - mean[c]) / std[c], HWC uint8 -> CHW                (B6).
 *   src   DEVICE  [B][Hs][Ws][3] uint8.     dst   DEVICE  [B][3][Hd][Wd], out_dtype 0 = fp32, 1 = fp16.
 *   mean, std  HOST [3] (passed by value to the kernel).  No handle: the call owns no state. */
int ffpp_preprocess(const uint8_t* src /*DEVICE*/, int32_t B, int32_t Hs, int32_t Ws, int32_t Hd, int32_t Wd,
                    const float* mean /*HOST*/, const float* stdv /*HOST*/, int32_t out_dtype, void* stream, void* dst /*DEVICE*/);

#ifdef __cplusplus
}
#endif
#endif /* FFPP_NEXT_H_ */
