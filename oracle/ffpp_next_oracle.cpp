// ffpp_next_oracle — TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// Plain, slow, single-threaded CPU statements of the four steps around the hot path that SURVEY.md §8(f) ranks
// next (f1-f4).  Same rules as ffpp_oracle.cpp: only tests/, __graft_entry__.smoke() and bench.py's CPU legs may
// build, load or call this file; it shares no code, header, table or helper with the CUDA path and neither includes
// the other.  Every function is the definition written out (double accumulation, no blocking, no fusion).
//
//  f1  heatmap analytics on a density grid: "Clusters are identified by thresholding these heatmaps and applying
//      connected component analysis to detect areas of local aggregation" (§2.3 Clustering);
//      "Compute heatmap, entropy, clustering degree" (Algorithm 1; §3.6).
//  f2  exact-position density: "for all grid cells / for all chickens / Compute distance and update density"
//      (Algorithm 1 DefaultClustering; "Vectorized density map (cdist)" L225, §3.6).
//  f3  segmentation-mask post-processing: "applying a threshold to the model's output, extracting connected
//      components, and generating bounding boxes from the resulting masks" (§2.3 Detection;
//      §3.2: skimage.regionprops -> cv2.connectedComponentsWithStats, 40.2 -> 11.4 ms/frame).
//  f4  pre-processing: "image resizing, normalization, and conversion to tensor format" (8.8 ms per
//      frame, L151).
//
// READINGS (the paper prints no formula for any of these; DESIGN.md §3 lists them; all are PARITY UNPINNED against the
// paper and pinned against the mathematics / library routines in tests/test_oracle_next_pins.py):
//  B1  entropy = Shannon entropy, natural log, of p = D / sum(D) over the cells of one frame; cells with D <= 0
//      contribute 0; sum(D) <= 0 gives 0.
//  B2  clustering degree = 1 - H / ln(n_cells) (0 for a uniform grid, 1 for all mass in one cell); n_cells <= 1 or
//      sum(D) <= 0 gives 0.  The paper names the quantity and never defines it.
//  B3  regions = connected components (4- or 8-connectivity, caller's choice) of {D > threshold}, strict; the label of
//      a component is the smallest row-major cell index in it; per region: cell count, inclusive bounding box, mass
//      = sum of D over its cells; regions are listed in ascending label order.
//  B4  exact-position density: a kept, in-frame centroid (O7's fp32 centroid and in-frame test) at u = cx / cell,
//      v = cy / cell (fp32) adds  exp(-(dx^2 + dy^2) / (2 sigma^2)) / Z^2  to every cell whose centre offset
//      dx = (ix + 0.5) - u, dy = (iy + 0.5) - v (each ONE fp32 subtraction) has |dx| <= R and |dy| <= R; Z and R are the
//      discrete tap sum and radius of O7 (A15), so a centroid exactly on a cell centre reproduces the binned result
//      (G1).  No border handling: mass that falls outside the grid is lost (the paper's loop has no fold).
//  B5  mask components: foreground = prob > threshold (strict), fp16 converted exactly; connectivity 8 by default
//      (cv2.connectedComponentsWithStats' default); label = smallest row-major pixel index; per component: area,
//      inclusive pixel bounding box, score = mean probability over its pixels; components with area < min_area are
//      left out of the table (their labels stay in the label image).
//  B6  pre-processing: bilinear resize with half-pixel centres (src = (dst + 0.5) * scale - 0.5, clamped at 0, the
//      right neighbour clamped at the last pixel: cv2.INTER_LINEAR / torch interpolate(align_corners=False)), then
//      (v / 255 - mean_c) / std_c, HWC uint8 -> CHW float.
#include <cmath>
#include <cstdint>
#include <cstring>
#include <vector>

extern "C" {

typedef struct oracle_region {
  int32_t label;            // smallest row-major index of the component
  int32_t area;             // cells / pixels
  int32_t x0, y0, x1, y1;   // inclusive bounding box
  float mass;               // f1: sum of D over the region; f3: mean probability (score)
  int32_t reserved_;
} oracle_region;

}  // extern "C"

namespace {

float half_bits_to_float(uint16_t h) {
  const int sign = (h >> 15) & 1, e = (h >> 10) & 31, m = h & 1023;
  double v;
  if (e == 0) v = std::ldexp((double)m, -24);
  else if (e == 31) v = m ? NAN : INFINITY;
  else v = std::ldexp((double)(1024 + m), e - 25);
  return (float)(sign ? -v : v);
}

// B3 / B5: flood fill in row-major order; the first cell of a component that the scan meets is its smallest index.
template <typename Fg, typename Val>
int32_t components(int w, int h, int conn, Fg fg, Val val, bool mean, int min_area, int32_t* labels, oracle_region* out, int32_t max_out) {
  const int64_t n = (int64_t)w * h;
  for (int64_t i = 0; i < n; ++i) labels[i] = -1;
  std::vector<int32_t> stack;
  int32_t count = 0;
  static const int dx8[8] = {1, -1, 0, 0, 1, 1, -1, -1}, dy8[8] = {0, 0, 1, -1, 1, -1, 1, -1};
  const int nn = conn == 8 ? 8 : 4;
  for (int64_t i = 0; i < n; ++i) {
    if (!fg(i) || labels[i] >= 0) continue;
    oracle_region r;
    std::memset(&r, 0, sizeof(r));
    r.label = (int32_t)i;
    r.x0 = r.x1 = (int32_t)(i % w);
    r.y0 = r.y1 = (int32_t)(i / w);
    double sum = 0.0;
    labels[i] = (int32_t)i;
    stack.assign(1, (int32_t)i);
    while (!stack.empty()) {
      const int32_t c = stack.back();
      stack.pop_back();
      const int x = c % w, y = c / w;
      ++r.area;
      sum += (double)val(c);
      if (x < r.x0) r.x0 = x;
      if (x > r.x1) r.x1 = x;
      if (y < r.y0) r.y0 = y;
      if (y > r.y1) r.y1 = y;
      for (int k = 0; k < nn; ++k) {
        const int xx = x + dx8[k], yy = y + dy8[k];
        if (xx < 0 || yy < 0 || xx >= w || yy >= h) continue;
        const int64_t j = (int64_t)yy * w + xx;
        if (fg(j) && labels[j] < 0) { labels[j] = (int32_t)i; stack.push_back((int32_t)j); }
      }
    }
    r.mass = (float)(mean ? sum / (double)r.area : sum);
    if (r.area >= min_area) {
      if (count < max_out && out) out[count] = r;
      ++count;
    }
  }
  return count;
}

}  // namespace

extern "C" {

// ---- f1 (B1): Shannon entropy of p = D / sum(D), natural log ----
double oracle_entropy(const float* D, int64_t n) {
  double s = 0.0;
  for (int64_t i = 0; i < n; ++i) if (D[i] > 0.0f) s += (double)D[i];
  if (!(s > 0.0)) return 0.0;
  double h = 0.0;
  for (int64_t i = 0; i < n; ++i) {
    if (!(D[i] > 0.0f)) continue;
    const double p = (double)D[i] / s;
    h -= p * std::log(p);
  }
  return h;
}

// ---- f1 (B2): clustering degree = 1 - H / ln(n) ----
double oracle_clustering_degree(const float* D, int64_t n) {
  double s = 0.0;
  for (int64_t i = 0; i < n; ++i) if (D[i] > 0.0f) s += (double)D[i];
  if (n <= 1 || !(s > 0.0)) return 0.0;
  return 1.0 - oracle_entropy(D, n) / std::log((double)n);
}

// ---- f1 (B3): regions of {D > thr}; returns the number of regions (may exceed max_out; the table holds the first max_out) ----
int32_t oracle_regions(const float* D, int32_t gw, int32_t gh, float thr, int32_t conn, int32_t* labels, oracle_region* out, int32_t max_out) {
  return components(gw, gh, conn, [&](int64_t i) { return D[i] > thr; }, [&](int64_t i) { return D[i]; }, false, 1, labels, out, max_out);
}

// ---- f2 (B4): the literal cell x bird double loop of Algorithm 1 ----
// boxes: [n][4] kept boxes (x1, y1, x2, y2); returns the number of in-frame centroids.
int32_t oracle_density_exact(const float* boxes, int32_t n, int32_t W, int32_t H, int32_t cell, float sigma, float truncate, float* out) {
  const int gw = W / cell, gh = H / cell;
  const int R = (int)std::floor((double)truncate * (double)sigma);
  const double s2 = 2.0 * (double)sigma * (double)sigma;
  double Z = 0.0;
  for (int k = -R; k <= R; ++k) Z += std::exp(-(double)(k * k) / s2);
  std::vector<float> u, v;
  for (int i = 0; i < n; ++i) {
    const float* b = boxes + 4 * (int64_t)i;
    const float cx = (b[0] + b[2]) * 0.5f, cy = (b[1] + b[3]) * 0.5f;
    if (!(cx >= 0.0f && cx < (float)W && cy >= 0.0f && cy < (float)H)) continue;
    u.push_back(cx / (float)cell);
    v.push_back(cy / (float)cell);
  }
  for (int iy = 0; iy < gh; ++iy)
    for (int ix = 0; ix < gw; ++ix) {                       // for all grid cells
      double acc = 0.0;
      for (size_t k = 0; k < u.size(); ++k) {               // for all chickens
        const float dx = ((float)ix + 0.5f) - u[k];         // compute distance ...
        const float dy = ((float)iy + 0.5f) - v[k];
        if (!(std::fabs(dx) <= (float)R && std::fabs(dy) <= (float)R)) continue;
        acc += std::exp(-((double)dx * (double)dx + (double)dy * (double)dy) / s2) / (Z * Z);   // ... and update density
      }
      out[(int64_t)iy * gw + ix] = (float)acc;
    }
  return (int32_t)u.size();
}

// ---- f3 (B5): threshold -> connected components -> per-component box, area, score ----
// mask: [H][W] probabilities, dtype 0 = fp32, 1 = fp16.
int32_t oracle_mask_components(const void* mask, int32_t dtype, int32_t W, int32_t H, float thr, int32_t conn, int32_t min_area,
                               int32_t* labels, oracle_region* out, int32_t max_out) {
  auto val = [&](int64_t i) { return dtype == 1 ? half_bits_to_float(((const uint16_t*)mask)[i]) : ((const float*)mask)[i]; };
  return components(W, H, conn, [&](int64_t i) { return val(i) > thr; }, val, true, min_area < 1 ? 1 : min_area, labels, out, max_out);
}

// ---- f4 (B6): bilinear resize (half-pixel centres) + normalise + HWC uint8 -> CHW ----
void oracle_preprocess(const uint8_t* src, int32_t Hs, int32_t Ws, int32_t Hd, int32_t Wd, const float* mean, const float* stdv, double* dst) {
  const double sy = (double)Hs / (double)Hd, sx = (double)Ws / (double)Wd;
  for (int c = 0; c < 3; ++c)
    for (int y = 0; y < Hd; ++y) {
      double fy = ((double)y + 0.5) * sy - 0.5;
      if (fy < 0.0) fy = 0.0;
      int y0 = (int)std::floor(fy);
      if (y0 > Hs - 1) y0 = Hs - 1;
      const int y1 = y0 + 1 < Hs ? y0 + 1 : Hs - 1;
      const double wy = fy - (double)y0;
      for (int x = 0; x < Wd; ++x) {
        double fx = ((double)x + 0.5) * sx - 0.5;
        if (fx < 0.0) fx = 0.0;
        int x0 = (int)std::floor(fx);
        if (x0 > Ws - 1) x0 = Ws - 1;
        const int x1 = x0 + 1 < Ws ? x0 + 1 : Ws - 1;
        const double wx = fx - (double)x0;
        auto px = [&](int yy, int xx) { return (double)src[((int64_t)yy * Ws + xx) * 3 + c]; };
        const double top = (1.0 - wx) * px(y0, x0) + wx * px(y0, x1);
        const double bot = (1.0 - wx) * px(y1, x0) + wx * px(y1, x1);
        const double val = (1.0 - wy) * top + wy * bot;
        dst[((int64_t)c * Hd + y) * Wd + x] = (val / 255.0 - (double)mean[c]) / (double)stdv[c];
      }
    }
}

}  // extern "C"
