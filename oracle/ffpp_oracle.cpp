// ffpp_oracle — TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// Plain, slow, single-threaded CPU statement of what the hot path computes: batched per-frame
// post-processing of a single-class anchor-free detector head (decode + score threshold ->
// sort + top-K -> greedy IoU NMS -> binned truncated-Gaussian density grid).  Only tests/,
// __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may build, load
// or call this file.  It shares no code, header, table or helper with the CUDA path
// (paper_2512_07009_b200/csrc) and neither includes the other.
//
// Authority: the paper describes the pipeline step this replaces only
// in prose — "generating bounding boxes with confidence scores" from model output (PAPER.md:L70,
// §2.3 Detection), post-processing being the dominant cost (§3.2), and
// "mapping chicken positions onto a spatial grid to generate density heatmaps" (PAPER.md:L86,
// §2.3 Clustering; Algorithm 1: "for all grid cells / for all chickens /
// compute distance and update density").  It prints no formula for decode, IoU, NMS or the
// density kernel, so every definition below is BASELINE.json's north_star as read in SURVEY.md
// §8(c) steps O1-O7 and readings A1-A26 (listed again in DESIGN.md).  Each function cites its step.
//
// Every stage has a plain definition and the oracle is that definition written out: no blocking,
// no fusion, no reordering.  fp32 where the definition fixes fp32 (decode, IoU: every operation a
// separately rounded fp32 op; build with -ffp-contract=off, never -ffast-math), double for the
// density accumulation.
//
// Pins (tests/test_oracle_pins.py): D1 decode hand cases, logit(conf) closed forms, N1 IoU
// just-above/just-below hand case, brute-force O(n^2) NMS on 50 random boxes, torchvision.ops.nms,
// G1 single-centroid closed form + printed constants, grid-sum invariant, scipy correlate1d
// (mode='reflect'), python sorted() for the order.  Parity unpinned against the paper (it is silent):
// A2 cell-centre grid point, A15 radius rule floor(3*sigma), A16 reflect border, A21 720p half row —
// these are readings, pinned only against BASELINE.json's own worked cases.
#include <cmath>
#include <cstdint>
#include <cstring>
#include <vector>

extern "C" {

typedef struct oracle_params {
  int32_t dtype;            // 0 = fp32, 1 = fp16 rows
  float conf_thresh;        // on sigmoid(logit), strict >
  float iou_thresh;         // strict >
  int32_t top_k;
  int32_t num_levels;
  int32_t strides[4];       // ascending, e.g. {8,16,32}
  int32_t cell_px;          // density cell edge, px
  float sigma_cells;
  float truncate_sigmas;
} oracle_params;

typedef struct oracle_box { float x1, y1, x2, y2, score; int32_t cand_index; } oracle_box;

}  // extern "C"

namespace {

// IEEE binary16 -> binary32 (exact).  O2: "if fp16 convert each to fp32 (exact)".
float half_bits_to_float(uint16_t h) {
  const int sign = (h >> 15) & 1, e = (h >> 10) & 31, m = h & 1023;
  double v;
  if (e == 0) v = std::ldexp((double)m, -24);                 // zero / subnormal: m * 2^-24
  else if (e == 31) v = m ? NAN : INFINITY;
  else v = std::ldexp((double)(1024 + m), e - 25);            // (1 + m/1024) * 2^(e-15)
  return (float)(sign ? -v : v);
}

float read_value(const void* raw, int dtype, int64_t row, int col) {
  if (dtype == 1) return half_bits_to_float(((const uint16_t*)raw)[row * 5 + col]);
  return ((const float*)raw)[row * 5 + col];
}

// O3 / A7: T = (float) ln(conf / (1 - conf)) evaluated in double. conf<=0 -> -inf, conf>=1 -> +inf.
float logit_threshold(float conf) {
  if (!(conf > 0.0f)) return -INFINITY;
  if (!(conf < 1.0f)) return INFINITY;
  const double c = (double)conf;
  return (float)std::log(c / (1.0 - c));
}

// O1: candidate j of a W x H frame -> (level, ix, iy).  Level-major, ascending stride; level l has
// n_l = W*H/s_l^2 rows and grid width gw_l = W/s_l; row k of the level: ix = k mod gw, iy = k div gw.
void locate(const oracle_params& p, int W, int H, int64_t j, int& stride, int& ix, int& iy) {
  int64_t start = 0;
  for (int l = 0; l < p.num_levels; ++l) {
    const int s = p.strides[l];
    const int64_t n = (int64_t)W * H / ((int64_t)s * s);
    if (j < start + n || l == p.num_levels - 1) {
      const int64_t k = j - start;
      const int gw = W / s;
      stride = s; ix = (int)(k % gw); iy = (int)(k / gw);
      return;
    }
    start += n;
  }
}

// O2 / A2-A5: grid point = cell centre; distances in stride units; no clipping; all fp32.
void decode(int stride, int ix, int iy, float l, float t, float r, float b, float out[4]) {
  const float s = (float)stride;
  const float px = ((float)ix + 0.5f) * s;
  const float py = ((float)iy + 0.5f) * s;
  out[0] = px - l * s;
  out[1] = py - t * s;
  out[2] = px + r * s;
  out[3] = py + b * s;
}

// O5 / A11-A12: IoU = inter / ((areaA + areaB) - inter), continuous boxes, every op fp32.
float iou(const float a[4], const float b[4]) {
  float iw = std::fmin(a[2], b[2]) - std::fmax(a[0], b[0]);
  float ih = std::fmin(a[3], b[3]) - std::fmax(a[1], b[1]);
  iw = std::fmax(0.0f, iw);
  ih = std::fmax(0.0f, ih);
  const float inter = iw * ih;
  const float area_a = (a[2] - a[0]) * (a[3] - a[1]);
  const float area_b = (b[2] - b[0]) * (b[3] - b[1]);
  const float uni = (area_a + area_b) - inter;
  return inter / uni;   // 0/0 -> NaN -> never "> thr"
}

// O7 / A15: normalised taps w[k], k = -R..R (stored at index k+R), R = floor(truncate * sigma).
int taps(float sigma, float truncate, std::vector<double>& w) {
  const int R = (int)std::floor((double)truncate * (double)sigma);
  w.assign((size_t)(2 * R + 1), 0.0);
  double Z = 0.0;
  for (int k = -R; k <= R; ++k) Z += std::exp(-(double)(k * k) / (2.0 * (double)sigma * (double)sigma));
  for (int k = -R; k <= R; ++k) w[(size_t)(k + R)] = std::exp(-(double)(k * k) / (2.0 * (double)sigma * (double)sigma)) / Z;
  return R;
}

// O7 / A16: half-sample symmetric reflection  d c b a | a b c d | d c b a
int fold(int i, int n) {
  if (i < 0) return -i - 1;
  if (i >= n) return 2 * n - 1 - i;
  return i;
}

struct Cand { float z; int32_t idx; float box[4]; };

// O4 / A9-A10: total order (z descending as float comparison, then candidate index ascending).
bool before(const Cand& a, const Cand& b) {
  if (a.z > b.z) return true;
  if (a.z < b.z) return false;
  return a.idx < b.idx;
}

// Plain insertion-free merge sort on the total order (own code: std::sort's order of equal
// elements does not matter here because `before` is a strict total order, but keep it explicit).
void sort_cands(std::vector<Cand>& v) {
  std::vector<Cand> tmp(v.size());
  for (size_t width = 1; width < v.size(); width *= 2) {
    for (size_t lo = 0; lo < v.size(); lo += 2 * width) {
      size_t mid = lo + width < v.size() ? lo + width : v.size();
      size_t hi = lo + 2 * width < v.size() ? lo + 2 * width : v.size();
      size_t a = lo, b = mid, o = lo;
      while (a < mid && b < hi) tmp[o++] = before(v[b], v[a]) ? v[b++] : v[a++];
      while (a < mid) tmp[o++] = v[a++];
      while (b < hi) tmp[o++] = v[b++];
    }
    v.swap(tmp);
  }
}

}  // namespace

extern "C" {

float oracle_half_to_float(uint16_t h) { return half_bits_to_float(h); }
float oracle_logit_threshold(float conf) { return logit_threshold(conf); }
float oracle_iou(const float* a, const float* b) { return iou(a, b); }
int32_t oracle_fold(int32_t i, int32_t n) { return fold(i, n); }

// w_out must hold 2R+1 doubles (query R first with w_out == NULL).
int32_t oracle_taps(float sigma, float truncate, double* w_out) {
  std::vector<double> w;
  const int R = taps(sigma, truncate, w);
  if (w_out) std::memcpy(w_out, w.data(), w.size() * sizeof(double));
  return R;
}

// Decode candidate j of a W x H frame from its five values.  out = x1,y1,x2,y2.
void oracle_decode_candidate(const oracle_params* p, int32_t W, int32_t H, int64_t j, const float* ltrb, float* out,
                             int32_t* stride_ix_iy) {
  int s, ix, iy;
  locate(*p, W, H, j, s, ix, iy);
  decode(s, ix, iy, ltrb[0], ltrb[1], ltrb[2], ltrb[3], out);
  if (stride_ix_iy) { stride_ix_iy[0] = s; stride_ix_iy[1] = ix; stride_ix_iy[2] = iy; }
}

// O5: greedy NMS over boxes already in score order.  keep_out receives kept positions (ascending).
int32_t oracle_nms_sorted(const float* boxes /*[n][4]*/, int32_t n, float thr, int32_t* keep_out) {
  int32_t nk = 0;
  for (int32_t i = 0; i < n; ++i) {
    bool keep = true;
    for (int32_t k = 0; k < nk && keep; ++k)
      if (iou(boxes + 4 * (int64_t)keep_out[k], boxes + 4 * (int64_t)i) > thr) keep = false;
    if (keep) keep_out[nk++] = i;
  }
  return nk;
}

// O7: density grid of one frame from kept boxes (scatter form, the paper's bird loop inside the
// cell update), accumulated in double, stored as float, row-major [gh][gw].
// Returns the number of in-frame centroids (A18).
int32_t oracle_density(const float* boxes /*[n][4]*/, int32_t n, int32_t W, int32_t H, int32_t cell, float sigma,
                       float truncate, float* out) {
  const int gw = W / cell, gh = H / cell;
  std::vector<double> w;
  const int R = taps(sigma, truncate, w);
  std::vector<double> D((size_t)gw * gh, 0.0);
  int32_t inframe = 0;
  for (int32_t i = 0; i < n; ++i) {
    const float* b = boxes + 4 * (int64_t)i;
    const float cx = (b[0] + b[2]) * 0.5f;
    const float cy = (b[1] + b[3]) * 0.5f;
    if (!(cx >= 0.0f && cx < (float)W && cy >= 0.0f && cy < (float)H)) continue;
    ++inframe;
    const int cxi = (int)std::floor(cx / (float)cell);
    const int cyi = (int)std::floor(cy / (float)cell);
    for (int dy = -R; dy <= R; ++dy)
      for (int dx = -R; dx <= R; ++dx)
        D[(size_t)fold(cyi + dy, gh) * gw + fold(cxi + dx, gw)] += w[(size_t)(dy + R)] * w[(size_t)(dx + R)];
  }
  for (size_t i = 0; i < D.size(); ++i) out[i] = (float)D[i];
  return inframe;
}

// Whole path, O1-O7, frames in a for loop.
//   raw          [sum N_f][5] in p->dtype, frames tightly concatenated (A22)
//   out_boxes    [B][top_k]   rows [0,count) valid, keep order (= score order)
//   out_counts   [B]
//   out_density  concat of per-frame [H/cell][W/cell] row-major
//   sorted_idx   optional [B][top_k]: candidate indices after O4 (debug / stage parity), -1 padded
//   sorted_counts optional [B]: min(n_survivors, top_k);  survivor_counts optional [B]: n_survivors
// Returns 0, or -1 on invalid arguments.
int32_t oracle_run(const oracle_params* p, const void* raw, int32_t B, const int32_t* N_per_frame,
                   const int32_t* frame_dims, oracle_box* out_boxes, int32_t* out_counts, float* out_density,
                   int32_t* sorted_idx, int32_t* sorted_counts, int32_t* survivor_counts) {
  if (!p || B < 0 || (B > 0 && (!raw || !N_per_frame || !frame_dims || !out_boxes || !out_counts || !out_density))) return -1;
  const float T = logit_threshold(p->conf_thresh);
  int64_t off = 0, doff = 0;
  for (int32_t f = 0; f < B; ++f) {
    const int W = frame_dims[2 * f], H = frame_dims[2 * f + 1];
    const int64_t N = N_per_frame[f];
    // O1-O3: decode every candidate, keep those with z > T (NaN fails, A6)
    std::vector<Cand> sv;
    for (int64_t j = 0; j < N; ++j) {
      const float z = read_value(raw, p->dtype, off + j, 4);
      if (!(z > T)) continue;
      Cand c;
      c.z = z; c.idx = (int32_t)j;
      int s, ix, iy;
      locate(*p, W, H, j, s, ix, iy);
      decode(s, ix, iy, read_value(raw, p->dtype, off + j, 0), read_value(raw, p->dtype, off + j, 1),
             read_value(raw, p->dtype, off + j, 2), read_value(raw, p->dtype, off + j, 3), c.box);
      sv.push_back(c);
    }
    if (survivor_counts) survivor_counts[f] = (int32_t)sv.size();
    // O4: sort, cut to top-K
    sort_cands(sv);
    if ((int64_t)sv.size() > p->top_k) sv.resize((size_t)p->top_k);
    if (sorted_counts) sorted_counts[f] = (int32_t)sv.size();
    if (sorted_idx)
      for (int32_t k = 0; k < p->top_k; ++k) sorted_idx[(int64_t)f * p->top_k + k] = k < (int32_t)sv.size() ? sv[(size_t)k].idx : -1;
    // O5: greedy NMS against earlier kept boxes — the same routine the 50-box brute-force pin exercises
    std::vector<float> sb(sv.size() * 4);
    for (size_t i = 0; i < sv.size(); ++i) std::memcpy(&sb[i * 4], sv[i].box, 16);
    std::vector<int32_t> kept(sv.size() + 1);
    kept.resize((size_t)oracle_nms_sorted(sb.data(), (int32_t)sv.size(), p->iou_thresh, kept.data()));
    // O6: outputs; reported score = sigmoid(z) in fp32 (A8)
    std::vector<float> kb(kept.size() * 4);
    for (size_t k = 0; k < kept.size(); ++k) {
      const Cand& c = sv[(size_t)kept[k]];
      oracle_box& o = out_boxes[(int64_t)f * p->top_k + (int64_t)k];
      o.x1 = c.box[0]; o.y1 = c.box[1]; o.x2 = c.box[2]; o.y2 = c.box[3];
      o.score = 1.0f / (1.0f + std::exp(-c.z));
      o.cand_index = c.idx;
      std::memcpy(&kb[k * 4], c.box, 16);
    }
    out_counts[f] = (int32_t)kept.size();
    // O7: density
    oracle_density(kb.data(), (int32_t)kept.size(), W, H, p->cell_px, p->sigma_cells, p->truncate_sigmas, out_density + doff);
    off += N;
    doff += (int64_t)(W / p->cell_px) * (H / p->cell_px);
  }
  return 0;
}

}  // extern "C"
