// flockgen — seeded synthetic "flock" detector-head outputs (INPUT generator only).
//
// This module produces the raw [sum N_f, 5] (l,t,r,b,logit) head output that stands in for
// the paper's private farm videos + trained detector (§4; BASELINE.json
// configs[0..4]).  It serves both the CPU oracle and the CUDA path as *input*; it contains
// none of the post-processing method (no sort/top-K of outputs, no NMS, no density) and
// shares no code with either.  The only method-adjacent logic here is input conditioning
// demanded by BASELINE.json ("generation rejecting any pair within 1e-5 of the IoU
// threshold"): to find such pairs the generator has to know which boxes an implementation
// will compare, so it carries its own double-precision restatement of the layout (SURVEY
// §8(c) O1/O2) and of IoU.  That restatement is private to this file.
//
// Recipe: SURVEY.md §8(d) "Synthetic inputs"; DESIGN.md "Input recipe".
// PRNG: splitmix64-seeded xoshiro256** (hand-written; no std::*_distribution, which are
// implementation-defined).  Frame f of a batch draws from its own stream
// splitmix64(seed + f), so frames can be generated in parallel and in any order.
#include <algorithm>
#include <atomic>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <thread>
#include <vector>

extern "C" {

typedef struct flockgen_frame_spec {
  int32_t W, H;            // frame size in pixels
  double lambda_lo;        // Poisson mean of the bird count; if lambda_hi > lambda_lo the mean
  double lambda_hi;        //   is drawn log-uniform in [lo, hi] first
  double lambda_cap;       //   and then capped at lambda_cap (<= 0: no cap)
  double box_median;       // lognormal median of box w and h, px
  double box_sigma;        // lognormal sigma (0.25)
  int32_t layout;          // 0: Gaussian mixture + uniform; 1: uniform + clustered neighbours
  int32_t n_components;    // layout 0: number of mixture components
  double comp_sigma;       // layout 0: component sigma, px
  double frac;             // layout 0: fraction drawn uniform; layout 1: fraction clustered
  int32_t bg_beta_a;       // background score ~ Beta(a, b), integer a,b (order statistics)
  int32_t bg_beta_b;
} flockgen_frame_spec;

typedef struct flockgen_params {
  int32_t dtype;           // 0 = fp32 rows, 1 = fp16 rows (IEEE binary16, RNE)
  int32_t num_levels;
  int32_t strides[4];
  double conf_thresh;      // needed only for the IoU-margin conditioning
  double iou_thresh;
  int32_t top_k;
  double jitter_px;        // 1.5
  double iou_margin;       // 1e-5
  int32_t threads;         // <= 0: hardware_concurrency
} flockgen_params;

typedef struct flockgen_stats {
  int64_t birds;           // total birds drawn
  int64_t redraws;         // candidates whose distances were re-drawn by the margin rule
  int64_t evicted;         // candidates whose logit was forced to -10 after 16 failed re-draws
} flockgen_stats;

}  // extern "C"

namespace {

struct Rng {
  uint64_t s[4];
  static uint64_t splitmix64(uint64_t& x) {
    uint64_t z = (x += 0x9E3779B97F4A7C15ull);
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
    return z ^ (z >> 31);
  }
  explicit Rng(uint64_t seed) {
    uint64_t x = seed;
    for (int i = 0; i < 4; ++i) s[i] = splitmix64(x);
  }
  static uint64_t rotl(uint64_t x, int k) { return (x << k) | (x >> (64 - k)); }
  uint64_t next() {
    const uint64_t result = rotl(s[1] * 5, 7) * 9;
    const uint64_t t = s[1] << 17;
    s[2] ^= s[0]; s[3] ^= s[1]; s[1] ^= s[2]; s[0] ^= s[3];
    s[2] ^= t; s[3] = rotl(s[3], 45);
    return result;
  }
  double u01() { return (double)(next() >> 11) * (1.0 / 9007199254740992.0); }          // [0,1)
  double u01_open() { return ((double)(next() >> 11) + 0.5) * (1.0 / 9007199254740992.0); }  // (0,1)
  double uniform(double a, double b) { return a + (b - a) * u01(); }
  double normal() {  // Marsaglia polar, no cached second value (keeps the stream position simple)
    for (;;) {
      double u = 2.0 * u01() - 1.0, v = 2.0 * u01() - 1.0;
      double q = u * u + v * v;
      if (q > 0.0 && q < 1.0) return u * std::sqrt(-2.0 * std::log(q) / q);
    }
  }
  int64_t poisson(double lambda) {  // exact: count unit-rate exponential arrivals before lambda
    int64_t k = 0;
    double acc = -std::log(u01_open());
    while (acc < lambda) { ++k; acc += -std::log(u01_open()); }
    return k;
  }
  // Beta(a,b) with integer a,b = a-th smallest of a+b-1 uniforms.
  double beta_int(int a, int b) {
    double buf[64];
    int n = a + b - 1;
    if (n > 64) n = 64;
    for (int i = 0; i < n; ++i) buf[i] = u01_open();
    std::nth_element(buf, buf + (a - 1), buf + n);
    return buf[a - 1];
  }
};

// ---- IEEE binary16 round-to-nearest-even, via float bits (portable, no _Float16) ----
uint16_t f32_to_f16_rne(float f) {
  uint32_t x; std::memcpy(&x, &f, 4);
  uint32_t sign = (x >> 16) & 0x8000u;
  uint32_t em = x & 0x7FFFFFFFu;
  if (em >= 0x7F800000u) return (uint16_t)(sign | (em > 0x7F800000u ? 0x7E00u : 0x7C00u));
  if (em >= 0x477FF000u) return (uint16_t)(sign | 0x7C00u);           // rounds to >= 65520 -> inf
  if (em < 0x33000001u) return (uint16_t)sign;                        // < 2^-25 (or == 2^-25 tie) -> 0
  int32_t e = (int32_t)(em >> 23) - 127;
  uint32_t m = (em & 0x7FFFFFu) | 0x800000u;
  int shift;
  uint32_t base;
  if (e >= -14) { shift = 13; base = (uint32_t)(e + 15) << 10; m &= 0x7FFFFFu; }
  else { shift = 13 + (-14 - e); base = 0; }
  uint32_t q = m >> shift;
  uint32_t rem = m & ((1u << shift) - 1u);
  uint32_t half = 1u << (shift - 1);
  if (rem > half || (rem == half && (q & 1u))) ++q;
  return (uint16_t)(sign | (base + q));                                // carry into exponent is correct
}
float f16_to_f32(uint16_t h) {
  uint32_t sign = (uint32_t)(h & 0x8000u) << 16;
  uint32_t e = (h >> 10) & 0x1Fu, m = h & 0x3FFu, x;
  if (e == 0) {
    if (m == 0) x = sign;
    else { int k = 0; while (!(m & 0x400u)) { m <<= 1; ++k; } x = sign | ((uint32_t)(113 - k) << 23) | ((m & 0x3FFu) << 13); }
  } else if (e == 31) x = sign | 0x7F800000u | (m << 13);
  else x = sign | ((e + 112) << 23) | (m << 13);
  float f; std::memcpy(&f, &x, 4); return f;
}

struct Bird { double cx, cy, w, h; };

struct Level { int stride, gw, rows; int64_t n, start; };

struct FrameGen {
  const flockgen_frame_spec& sp;
  const flockgen_params& pa;
  Rng rng;
  int64_t N = 0;
  std::vector<Level> lv;
  std::vector<Bird> birds;
  std::vector<int32_t> owner;      // per candidate: bird index or -1
  std::vector<float> vals;         // [N][5], already rounded to the storage dtype's value set
  std::vector<uint8_t> tries;
  flockgen_stats st{0, 0, 0};

  FrameGen(const flockgen_frame_spec& s, const flockgen_params& p, uint64_t seed) : sp(s), pa(p), rng(seed) {
    int64_t start = 0;
    for (int l = 0; l < pa.num_levels; ++l) {
      Level L;
      L.stride = pa.strides[l];
      L.gw = sp.W / L.stride;
      L.n = (int64_t)sp.W * sp.H / ((int64_t)L.stride * L.stride);
      L.rows = (int)((L.n + L.gw - 1) / L.gw);
      L.start = start;
      start += L.n;
      lv.push_back(L);
    }
    N = start;
  }

  float q(double v) const {  // round a real to the storage dtype, return as float
    float f = (float)v;
    return pa.dtype == 1 ? f16_to_f32(f32_to_f16_rne(f)) : f;
  }

  void locate(int64_t j, int& l, int& ix, int& iy) const {
    l = 0;
    while (l + 1 < (int)lv.size() && j >= lv[l + 1].start) ++l;
    int64_t k = j - lv[l].start;
    ix = (int)(k % lv[l].gw);
    iy = (int)(k / lv[l].gw);
  }

  void draw_birds() {
    double lambda = sp.lambda_lo;
    if (sp.lambda_hi > sp.lambda_lo) lambda = std::exp(rng.uniform(std::log(sp.lambda_lo), std::log(sp.lambda_hi)));
    if (sp.lambda_cap > 0 && lambda > sp.lambda_cap) lambda = sp.lambda_cap;
    int64_t nb = rng.poisson(lambda);
    std::vector<double> mx, my;
    if (sp.layout == 0)
      for (int c = 0; c < sp.n_components; ++c) {  // component means: central 70 % of the frame
        mx.push_back(rng.uniform(0.15 * sp.W, 0.85 * sp.W));
        my.push_back(rng.uniform(0.15 * sp.H, 0.85 * sp.H));
      }
    birds.reserve((size_t)nb);
    for (int64_t i = 0; i < nb; ++i) {
      Bird b;
      double u = rng.u01();
      if (sp.layout == 0) {
        if (u < sp.frac || sp.n_components == 0) { b.cx = rng.uniform(0, sp.W); b.cy = rng.uniform(0, sp.H); }
        else {
          int c = (int)(rng.u01() * sp.n_components);
          b.cx = mx[c] + sp.comp_sigma * rng.normal();
          b.cy = my[c] + sp.comp_sigma * rng.normal();
        }
      } else {
        if (i > 0 && u < sp.frac) {  // clustered: offset U(0.25,0.55)*m from an existing bird
          const Bird& o = birds[(size_t)(rng.u01() * (double)i)];
          double th = rng.uniform(0, 6.283185307179586), d = rng.uniform(0.25, 0.55) * sp.box_median;
          b.cx = o.cx + d * std::cos(th); b.cy = o.cy + d * std::sin(th);
        } else { b.cx = rng.uniform(0, sp.W); b.cy = rng.uniform(0, sp.H); }
      }
      b.cx = std::min(std::max(b.cx, 1.0), sp.W - 1.0);
      b.cy = std::min(std::max(b.cy, 1.0), sp.H - 1.0);
      b.w = sp.box_median * std::exp(sp.box_sigma * rng.normal());
      b.h = sp.box_median * std::exp(sp.box_sigma * rng.normal());
      birds.push_back(b);
    }
    st.birds = nb;
  }

  void assign_owners() {  // smallest-area bird whose box strictly contains the grid point
    owner.assign((size_t)N, -1);
    std::vector<double> best((size_t)N, 1e300);
    for (size_t bi = 0; bi < birds.size(); ++bi) {
      const Bird& b = birds[bi];
      double x1 = b.cx - 0.5 * b.w, x2 = b.cx + 0.5 * b.w, y1 = b.cy - 0.5 * b.h, y2 = b.cy + 0.5 * b.h, area = b.w * b.h;
      for (const Level& L : lv) {
        double s = L.stride;
        int ix0 = std::max(0, (int)std::floor(x1 / s - 0.5) + 1), ix1 = std::min(L.gw - 1, (int)std::ceil(x2 / s - 0.5) - 1);
        int iy0 = std::max(0, (int)std::floor(y1 / s - 0.5) + 1), iy1 = std::min(L.rows - 1, (int)std::ceil(y2 / s - 0.5) - 1);
        for (int iy = iy0; iy <= iy1; ++iy)
          for (int ix = ix0; ix <= ix1; ++ix) {
            int64_t k = (int64_t)iy * L.gw + ix;
            if (k >= L.n) continue;  // partial last row (1280x720, stride 32)
            size_t j = (size_t)(L.start + k);
            if (area < best[j]) { best[j] = area; owner[j] = (int32_t)bi; }
          }
      }
    }
  }

  void draw_distances(int64_t j) {
    int l, ix, iy; locate(j, l, ix, iy);
    double s = lv[l].stride, px = (ix + 0.5) * s, py = (iy + 0.5) * s;
    float* v = &vals[(size_t)j * 5];
    for (int attempt = 0;; ++attempt) {
      double d[4];
      if (owner[(size_t)j] >= 0) {
        const Bird& b = birds[(size_t)owner[(size_t)j]];
        d[0] = px - (b.cx - 0.5 * b.w) + pa.jitter_px * rng.normal();
        d[1] = py - (b.cy - 0.5 * b.h) + pa.jitter_px * rng.normal();
        d[2] = (b.cx + 0.5 * b.w) - px + pa.jitter_px * rng.normal();
        d[3] = (b.cy + 0.5 * b.h) - py + pa.jitter_px * rng.normal();
      } else {
        for (int k = 0; k < 4; ++k) d[k] = rng.uniform(2.0, 40.0);
      }
      for (int k = 0; k < 4; ++k) v[k] = q(d[k] / s);
      // positive width and height after rounding; practically always true
      if ((double)v[0] + (double)v[2] > 1.0 / s && (double)v[1] + (double)v[3] > 1.0 / s) break;
      if (attempt > 64) { v[0] = v[1] = v[2] = v[3] = q(4.0 / s); break; }
    }
  }

  void draw_logit(int64_t j) {
    double u = owner[(size_t)j] >= 0 ? rng.beta_int(8, 2) : rng.beta_int(sp.bg_beta_a, sp.bg_beta_b);
    u = std::min(std::max(u, 1e-6), 1.0 - 1e-6);
    float z = q(std::log(u / (1.0 - u)));
    if (z == 0.0f) z = 6.103515625e-05f;  // 2^-14: never emit +-0 logits
    vals[(size_t)j * 5 + 4] = z;
  }

  struct DBox { double x1, y1, x2, y2; float z; int32_t idx; };

  DBox decode(int64_t j) const {
    int l, ix, iy; locate(j, l, ix, iy);
    double s = lv[l].stride, px = (ix + 0.5) * s, py = (iy + 0.5) * s;
    const float* v = &vals[(size_t)j * 5];
    DBox b;
    // each coordinate is one fp32 rounding of an exactly representable product/sum
    b.x1 = (double)(float)(px - (double)v[0] * s); b.y1 = (double)(float)(py - (double)v[1] * s);
    b.x2 = (double)(float)(px + (double)v[2] * s); b.y2 = (double)(float)(py + (double)v[3] * s);
    b.z = v[4]; b.idx = (int32_t)j;
    return b;
  }

  // Re-draw until no pair among the frame's top-K survivors has |IoU - thr| < margin.
  void condition_iou_margin() {
    const float T = (float)std::log(pa.conf_thresh / (1.0 - pa.conf_thresh));
    tries.assign((size_t)N, 0);
    const double cell = std::max(32.0, 2.0 * sp.box_median);
    const int cw = (int)(sp.W / cell) + 3, ch = (int)(sp.H / cell) + 3;
    for (int round = 0; round < 1000; ++round) {
      std::vector<DBox> sv;
      for (int64_t j = 0; j < N; ++j)
        if (vals[(size_t)j * 5 + 4] > T) sv.push_back(decode(j));
      std::sort(sv.begin(), sv.end(), [](const DBox& a, const DBox& b) { return a.z > b.z || (a.z == b.z && a.idx < b.idx); });
      if ((int64_t)sv.size() > pa.top_k) sv.resize((size_t)pa.top_k);
      // uniform spatial hash over box extents (clamped into a padded cell grid)
      auto cx = [&](double x) { return std::min(cw - 1, std::max(0, (int)std::floor(x / cell) + 1)); };
      auto cy = [&](double y) { return std::min(ch - 1, std::max(0, (int)std::floor(y / cell) + 1)); };
      std::vector<std::vector<int32_t>> cells((size_t)cw * ch);
      for (size_t r = 0; r < sv.size(); ++r)
        for (int gy = cy(sv[r].y1); gy <= cy(sv[r].y2); ++gy)
          for (int gx = cx(sv[r].x1); gx <= cx(sv[r].x2); ++gx) cells[(size_t)gy * cw + gx].push_back((int32_t)r);
      std::vector<int32_t> bad;
      for (int gy = 0; gy < ch; ++gy)
        for (int gx = 0; gx < cw; ++gx) {
          const auto& c = cells[(size_t)gy * cw + gx];
          for (size_t a = 0; a < c.size(); ++a)
            for (size_t b = a + 1; b < c.size(); ++b) {
              const DBox &A = sv[(size_t)c[a]], &B = sv[(size_t)c[b]];
              double ix1 = std::max(A.x1, B.x1), iy1 = std::max(A.y1, B.y1);
              double iw = std::min(A.x2, B.x2) - ix1, ih = std::min(A.y2, B.y2) - iy1;
              if (iw <= 0 || ih <= 0) continue;
              if (cx(ix1) != gx || cy(iy1) != gy) continue;  // count each pair once
              double inter = iw * ih;
              double uni = (A.x2 - A.x1) * (A.y2 - A.y1) + (B.x2 - B.x1) * (B.y2 - B.y1) - inter;
              double iou = inter / uni;
              if (std::fabs(iou - pa.iou_thresh) < pa.iou_margin) bad.push_back(std::max(c[a], c[b]));  // lower-scored member
            }
        }
      if (bad.empty()) return;
      std::sort(bad.begin(), bad.end());
      bad.erase(std::unique(bad.begin(), bad.end()), bad.end());
      for (int32_t r : bad) {
        int64_t j = sv[(size_t)r].idx;
        if (++tries[(size_t)j] > 16) { vals[(size_t)j * 5 + 4] = q(-10.0); ++st.evicted; }
        else { draw_distances(j); ++st.redraws; }
      }
    }
  }

  void run(void* dst_rows) {
    draw_birds();
    assign_owners();
    vals.assign((size_t)N * 5, 0.f);
    for (int64_t j = 0; j < N; ++j) { draw_distances(j); draw_logit(j); }
    condition_iou_margin();
    if (pa.dtype == 1) {
      uint16_t* o = (uint16_t*)dst_rows;
      for (size_t i = 0; i < vals.size(); ++i) o[i] = f32_to_f16_rne(vals[i]);
    } else {
      std::memcpy(dst_rows, vals.data(), vals.size() * sizeof(float));
    }
  }
};

}  // namespace

extern "C" {

// Candidates per frame for a (W,H) under the level layout n_l = W*H/s_l^2.
int64_t flockgen_frame_candidates(const flockgen_params* pa, int32_t W, int32_t H) {
  int64_t n = 0;
  for (int l = 0; l < pa->num_levels; ++l) n += (int64_t)W * H / ((int64_t)pa->strides[l] * pa->strides[l]);
  return n;
}

// raw_out: HOST buffer of sum_f N_f rows of 5 values in pa->dtype, frames tightly concatenated.
// Returns 0 on success.
int flockgen_generate(const flockgen_params* pa, int32_t B, const flockgen_frame_spec* specs, uint64_t seed,
                      void* raw_out, flockgen_stats* stats_out) {
  if (!pa || !specs || !raw_out || B < 0) return -1;
  std::vector<int64_t> off((size_t)B + 1, 0);
  for (int f = 0; f < B; ++f) off[(size_t)f + 1] = off[(size_t)f] + flockgen_frame_candidates(pa, specs[f].W, specs[f].H);
  const size_t esz = pa->dtype == 1 ? 2 : 4;
  std::vector<flockgen_stats> st((size_t)B);
  int nt = pa->threads > 0 ? pa->threads : (int)std::thread::hardware_concurrency();
  nt = std::max(1, std::min(nt, B));
  std::atomic<int> next{0};
  auto work = [&]() {
    for (;;) {
      int f = next.fetch_add(1);
      if (f >= B) return;
      uint64_t x = seed + (uint64_t)f;
      FrameGen g(specs[f], *pa, Rng::splitmix64(x));
      g.run((char*)raw_out + (size_t)off[(size_t)f] * 5 * esz);
      st[(size_t)f] = g.st;
    }
  };
  std::vector<std::thread> th;
  for (int t = 1; t < nt; ++t) th.emplace_back(work);
  work();
  for (auto& t : th) t.join();
  if (stats_out) {
    stats_out->birds = stats_out->redraws = stats_out->evicted = 0;
    for (auto& s : st) { stats_out->birds += s.birds; stats_out->redraws += s.redraws; stats_out->evicted += s.evicted; }
  }
  return 0;
}

}  // extern "C"
