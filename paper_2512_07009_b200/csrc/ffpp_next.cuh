// the steps around the hot path (include/ffpp_next.h).  Kernels first, then the host entry points.
// This file is included at the end of ffpp.cu (it needs the handle).  Nothing here is shared with oracle/.
#pragma once
#include <climits>

#include "../../include/ffpp_next.h"
#include "ffpp_kernels.cuh"

namespace ffpp {

// one image of a batch: a density grid (f1, f2: ragged, table uploaded by the host) or a mask (f3: uniform, computed)
struct ImgDesc {
  int64_t off;                      // first element of the image in the flat arrays
  int32_t w, h;
};
__device__ __forceinline__ ImgDesc img_desc(const ImgDesc* __restrict__ tab, const int img, const int w, const int h) {
  if (tab) return tab[img];
  ImgDesc d;
  d.off = (int64_t)img * w * h; d.w = w; d.h = h;
  return d;
}
__device__ __forceinline__ float load_prob(const float* p, const int64_t i) { return p[i]; }
__device__ __forceinline__ float load_prob(const __half* p, const int64_t i) { return __half2float(p[i]); }

// =====================================================================================================
// Connected-component labelling shared by f1 (regions of a thresholded density grid) and f3
// (components of a thresholded segmentation mask).  Label equivalence by union-find in the
// label image itself: every foreground pixel starts as its own root (label = its row-major index); a pixel unites
// itself with its already-scanned foreground neighbours (left, up; up-left and up-right under 8-connectivity), a
// union always hanging the LARGER root under the smaller one with atomicMin, so the root of a component is its
// smallest index whatever the interleaving — the result is unique, hence deterministic and equal to the oracle's.
//   kc_init    label = first pixel of the row run inside the warp / -1, area counter of every self-labelled pixel = 0
//   kc_merge   unions
//   kc_flatten label = root; area[root] += 1
//   kr_*       ordered compaction of the roots with area >= min_area into the table (ascending label); the table
//              index of every root goes to the counter array
//   kc_stats   bounding box (atomicMin / atomicMax) and sum (64-bit fixed point, 2^-40: order-independent, so
//              bit-reproducible) of every listed component; a warp whose pixels all belong to one component
//              reduces first and issues one set of atomics
//   kc_final   mass = sum (f1) or sum / area (f3: mean probability)
// =====================================================================================================
constexpr int KC_THREADS = 256;
constexpr int KC_PER = 1;                         // 256-pixel steps per CTA of the per-pixel kernels (a step = 32 consecutive pixels per warp)
constexpr int KC_RANK_THREADS = 1024;
constexpr int KC_RANK_PER = 4;                    // consecutive pixels per thread per step of kc_rank
constexpr double KC_FIX = 1099511627776.0;        // 2^40

template <typename T>
__global__ void __launch_bounds__(KC_THREADS) kc_init(const T* __restrict__ src, const ImgDesc* __restrict__ tab, int w0, int h0,
                                                      float thr, int32_t* __restrict__ labels, int32_t* __restrict__ aux) {
  const ImgDesc d = img_desc(tab, blockIdx.y, w0, h0);
  const int n = d.w * d.h;
  const int lane = threadIdx.x & 31;
  for (int e = 0; e < KC_PER; ++e) {
  const int base = (blockIdx.x * KC_PER + e) * KC_THREADS;
  if (base >= n) break;
  const int i = base + threadIdx.x;
  const bool valid = i < n;
  const bool fg = valid && load_prob(src, d.off + i) > thr;
  // horizontal runs inside the warp's 32 consecutive pixels start labelled with the run's first pixel: the unions
  // along a row are done before the first atomic (a run that continues from the previous warp is united in kc_merge)
  const int x = valid ? i % d.w : 0;
  const uint32_t bits = __ballot_sync(0xffffffffu, fg), rowstart = __ballot_sync(0xffffffffu, valid && x == 0);
  const uint32_t starts = bits & (~(bits << 1) | rowstart);
  const int first = 31 - __clz((int)(starts & (0xFFFFFFFFu >> (31 - lane))));
  if (valid) {
    labels[d.off + i] = fg ? i - (lane - first) : -1;
    if (fg && first == lane) aux[d.off + i] = 0;             // only a pixel that labels itself can end up a root: its area counter
  }
  }
}

__device__ __forceinline__ int cc_find(const int32_t* L, int i) {
  for (;;) {
    const int p = *reinterpret_cast<const volatile int32_t*>(L + i);
    if (p == i) return i;
    i = p;
  }
}
__device__ __forceinline__ void cc_unite(int32_t* L, int a, int b) {
  for (;;) {
    a = cc_find(L, a);
    b = cc_find(L, b);
    if (a == b) return;
    if (a > b) { const int t = a; a = b; b = t; }            // a < b: b's tree goes under a
    const int old = atomicMin(&L[b], a);
    if (old == b) return;                                    // b was still a root: linked
    b = old;                                                 // somebody re-parented b first: unite a with that parent
  }
}

// Unions between rows, one per START of a vertical contact instead of one per pixel: with the left neighbour and the
// upper-left neighbour both foreground, the left neighbour (or a pixel further left in the same run) has already
// joined the two rows.  Under 8-connectivity a diagonal contact counts only where the pixel straight above is
// background (otherwise the upper run already holds both), and only from the end of the run that touches it.
__global__ void __launch_bounds__(KC_THREADS) kc_merge(const ImgDesc* __restrict__ tab, int w0, int h0, int conn, int32_t* __restrict__ labels) {
  const ImgDesc d = img_desc(tab, blockIdx.y, w0, h0);
  const int w = d.w, n = d.w * d.h;
  const int lane = threadIdx.x & 31;
  int32_t* L = labels + d.off;
  for (int e = 0; e < KC_PER; ++e) {
  const int base = (blockIdx.x * KC_PER + e) * KC_THREADS;
  if (base >= n) break;
  const int i = base + threadIdx.x;
  const bool valid = i < n;
  const bool fg = valid && L[i] >= 0;                        // foreground never changes: label >= 0
  const uint32_t bits = __ballot_sync(0xffffffffu, fg);
  if (!fg) continue;
  const int y = i / w, x = i - y * w;
  const bool left = x > 0 && (lane > 0 ? ((bits >> (lane - 1)) & 1u) != 0 : L[i - 1] >= 0);
  if (lane == 0 && left) cc_unite(L, i, i - 1);              // the run continues from the previous warp
  if (y == 0) continue;
  const bool up = L[i - w] >= 0;
  const bool ul = x > 0 && L[i - w - 1] >= 0;
  if (up) {
    if (!(left && ul)) cc_unite(L, i, i - w);
  } else if (conn == 8) {
    if (ul && !left) cc_unite(L, i, i - w - 1);
    if (x + 1 < w && L[i - w + 1] >= 0) {
      const bool right = lane < 31 ? ((bits >> (lane + 1)) & 1u) != 0 : (i + 1 < n && L[i + 1] >= 0);
      if (!right) cc_unite(L, i, i - w + 1);
    }
  }
  }
}

__global__ void __launch_bounds__(KC_THREADS) kc_flatten(const ImgDesc* __restrict__ tab, int w0, int h0, int32_t* __restrict__ labels,
                                                         int32_t* __restrict__ aux) {
  const ImgDesc d = img_desc(tab, blockIdx.y, w0, h0);
  const int n = d.w * d.h;
  int32_t* L = labels + d.off;
  for (int e = 0; e < KC_PER; ++e) {
    const int i = (blockIdx.x * KC_PER + e) * KC_THREADS + threadIdx.x;
    if (i >= n || L[i] < 0) continue;
    const int r = cc_find(L, i);
    if (r != i) L[i] = r;                                    // a chain through i that another thread is walking still ends at r
    // area: lanes of the warp that found the same root count together (runs of one component are the common case)
    const uint32_t peers = __match_any_sync(__activemask(), r);
    if ((int)(__ffs(peers) - 1) == (int)(threadIdx.x & 31)) atomicAdd(&aux[d.off + r], __popc(peers));
  }
}

// Ordered compaction of the roots with area >= min_area into the table (ascending label), in three launches so that a
// 2 M-pixel mask is scanned by hundreds of CTAs: per block of 4096 pixels the number of listed roots (kr_count), per
// image the exclusive scan of the block counts (kr_scan), per block the table rows (kr_place).  The table index of every
// root replaces its area in the counter array (-1: not listed).
constexpr int KR_BLOCK = KC_RANK_THREADS * KC_RANK_PER;

__device__ __forceinline__ int kr_block_scan(const int c, int* s_wsum, const int tid, int* total) {   // exclusive prefix of c over the CTA
  const int lane = tid & 31, warp = tid >> 5;
  int inc = c;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) { const int t = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= o) inc += t; }
  if (lane == 31) s_wsum[warp] = inc;
  __syncthreads();
  const int wv = s_wsum[lane];
  int winc = wv;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) { const int t = __shfl_up_sync(0xffffffffu, winc, o); if (lane >= o) winc += t; }
  *total = __shfl_sync(0xffffffffu, winc, 31);
  return __shfl_sync(0xffffffffu, winc - wv, warp) + inc - c;
}

template <bool kPlace>
__global__ void __launch_bounds__(KC_RANK_THREADS) kr_count_place(const ImgDesc* __restrict__ tab, int w0, int h0, const int32_t* __restrict__ labels,
                                                                  int32_t* __restrict__ aux, int min_area, int max_out, int nblk_max,
                                                                  int32_t* __restrict__ blk, ffpp_region* __restrict__ out,
                                                                  unsigned long long* __restrict__ sums) {
  __shared__ int s_wsum[KC_RANK_THREADS / 32];
  const int img = blockIdx.y;
  const ImgDesc d = img_desc(tab, img, w0, h0);
  const int n = d.w * d.h;
  const int base = blockIdx.x * KR_BLOCK;
  if (base >= n) return;
  const int32_t* L = labels + d.off;
  int32_t* A = aux + d.off;
  const int tid = threadIdx.x;
  const int i0 = base + tid * KC_RANK_PER;
  int area[KC_RANK_PER];
  uint32_t rootm = 0, selm = 0;
#pragma unroll
  for (int e = 0; e < KC_RANK_PER; ++e) {
    const int i = i0 + e;
    area[e] = 0;
    if (i < n && L[i] == i) {
      rootm |= 1u << e;
      area[e] = A[i];
      if (area[e] >= min_area) selm |= 1u << e;
    }
  }
  int total;
  const int excl = kr_block_scan(__popc(selm), s_wsum, tid, &total);
  if (!kPlace) {
    if (tid == 0) blk[(int64_t)img * nblk_max + blockIdx.x] = total;
    return;
  }
  ffpp_region* table = out + (int64_t)img * max_out;
  unsigned long long* sm = sums + (int64_t)img * max_out;
  int pos = blk[(int64_t)img * nblk_max + blockIdx.x] + excl;
#pragma unroll
  for (int e = 0; e < KC_RANK_PER; ++e) {
    if (!((rootm >> e) & 1u)) continue;
    const int i = i0 + e;
    int k = -1;
    if ((selm >> e) & 1u) {
      if (pos < max_out) {
        k = pos;
        ffpp_region r;
        r.label = i; r.area = area[e]; r.x0 = INT_MAX; r.y0 = INT_MAX; r.x1 = -1; r.y1 = -1; r.mass = 0.0f; r.reserved_ = 0;
        table[k] = r;
        sm[k] = 0ull;
      }
      ++pos;
    }
    A[i] = k;                                                // table index of this root, -1 if not listed
  }
}

__global__ void __launch_bounds__(KC_THREADS) kr_scan(const ImgDesc* __restrict__ tab, int w0, int h0, int nblk_max, int32_t* __restrict__ blk,
                                                      int32_t* __restrict__ out_counts) {
  __shared__ int s_wsum[32];
  const int img = blockIdx.x;
  const ImgDesc d = img_desc(tab, img, w0, h0);
  const int nblk = (d.w * d.h + KR_BLOCK - 1) / KR_BLOCK;
  int32_t* b = blk + (int64_t)img * nblk_max;
  const int tid = threadIdx.x;
  if (tid < 32) s_wsum[tid] = 0;                             // kr_block_scan reads 32 warp sums; this CTA has 8 warps
  __syncthreads();
  int running = 0;
  for (int base = 0; base < nblk; base += KC_THREADS) {
    const int k = base + tid;
    const int c = k < nblk ? b[k] : 0;
    int total;
    const int excl = kr_block_scan(c, s_wsum, tid, &total);
    if (k < nblk) b[k] = running + excl;
    running += total;
    __syncthreads();
  }
  if (tid == 0) out_counts[img] = running;
}

template <typename T>
__global__ void __launch_bounds__(KC_THREADS) kc_stats(const T* __restrict__ src, const ImgDesc* __restrict__ tab, int w0, int h0,
                                                       const int32_t* __restrict__ labels, const int32_t* __restrict__ aux, int max_out,
                                                       ffpp_region* __restrict__ out, unsigned long long* __restrict__ sums) {
  const int img = blockIdx.y;
  const ImgDesc d = img_desc(tab, img, w0, h0);
  const int w = d.w, n = d.w * d.h;
  ffpp_region* table = out + (int64_t)img * max_out;
  unsigned long long* sm = sums + (int64_t)img * max_out;
  for (int e = 0; e < KC_PER; ++e) {
  const int base = (blockIdx.x * KC_PER + e) * KC_THREADS;
  if (base >= n) break;
  const int i = base + threadIdx.x;
  int k = -1;
  int x = 0, y = 0;
  unsigned long long fx = 0ull;
  if (i < n) {
    const int l = labels[d.off + i];
    if (l >= 0) k = aux[d.off + l];
    if (k >= 0) {
      y = i / w; x = i - y * w;
      fx = (unsigned long long)__double2ll_rn((double)load_prob(src, d.off + i) * KC_FIX);   // |value| < 2^22
    }
  }
  const uint32_t act = __ballot_sync(0xffffffffu, k >= 0);
  if (act == 0) continue;
  const int k0 = __shfl_sync(0xffffffffu, k, __ffs(act) - 1);
  if (__all_sync(0xffffffffu, k < 0 || k == k0)) {           // one component in this warp: reduce, then one set of atomics
    int x0 = k >= 0 ? x : INT_MAX, x1 = k >= 0 ? x : -1, y0 = k >= 0 ? y : INT_MAX, y1 = k >= 0 ? y : -1;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      x0 = min(x0, __shfl_xor_sync(0xffffffffu, x0, o)); x1 = max(x1, __shfl_xor_sync(0xffffffffu, x1, o));
      y0 = min(y0, __shfl_xor_sync(0xffffffffu, y0, o)); y1 = max(y1, __shfl_xor_sync(0xffffffffu, y1, o));
      fx += __shfl_xor_sync(0xffffffffu, fx, o);
    }
    if ((threadIdx.x & 31) == 0) {
      atomicMin(&table[k0].x0, x0); atomicMax(&table[k0].x1, x1);
      atomicMin(&table[k0].y0, y0); atomicMax(&table[k0].y1, y1);
      atomicAdd(&sm[k0], fx);
    }
  } else if (k >= 0) {
    atomicMin(&table[k].x0, x); atomicMax(&table[k].x1, x);
    atomicMin(&table[k].y0, y); atomicMax(&table[k].y1, y);
    atomicAdd(&sm[k], fx);
  }
  }
}

__global__ void __launch_bounds__(KC_THREADS) kc_final(int max_out, int mean, const int32_t* __restrict__ counts,
                                                       ffpp_region* __restrict__ out, const unsigned long long* __restrict__ sums) {
  const int img = blockIdx.y;
  const int k = blockIdx.x * KC_THREADS + threadIdx.x;
  const int n = min(counts[img], max_out);
  if (k >= n) return;
  ffpp_region* r = out + (int64_t)img * max_out + k;
  const double s = (double)(long long)sums[(int64_t)img * max_out + k] / KC_FIX;   // two's complement: negative terms are fine
  r->mass = (float)(mean ? s / (double)r->area : s);
}

// =====================================================================================================
// f1 — entropy and clustering degree of a density grid (readings B1, B2):  H = -sum p ln p with p = D / A, A = sum D,
// evaluated as  H = ln A - (sum D ln D) / A  so that one pass over the grid suffices.  Double precision, fixed
// summation order (thread-strided partials, shuffle tree, then the block partials in index order): bit-reproducible.
// =====================================================================================================
constexpr int KE_THREADS = 256;
constexpr int KE_PER = 8;                          // cells per thread

__global__ void __launch_bounds__(KE_THREADS) ke_partial(const float* __restrict__ D, const ImgDesc* __restrict__ tab, int nblk_max,
                                                         double2* __restrict__ part) {
  __shared__ double2 s_w[KE_THREADS / 32];
  const int img = blockIdx.y;
  const ImgDesc d = tab[img];
  const int n = d.w * d.h;
  const int base = blockIdx.x * KE_THREADS * KE_PER;
  if (base >= n) return;
  double a = 0.0, b = 0.0;
#pragma unroll
  for (int e = 0; e < KE_PER; ++e) {
    const int i = base + e * KE_THREADS + threadIdx.x;
    if (i < n) {
      const float v = D[d.off + i];
      if (v > 0.0f) { const double dv = (double)v; a += dv; b += dv * log(dv); }
    }
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) { a += __shfl_xor_sync(0xffffffffu, a, o); b += __shfl_xor_sync(0xffffffffu, b, o); }
  if ((threadIdx.x & 31) == 0) s_w[threadIdx.x >> 5] = make_double2(a, b);
  __syncthreads();
  if (threadIdx.x == 0) {
    double2 t = make_double2(0.0, 0.0);
    for (int wv = 0; wv < KE_THREADS / 32; ++wv) { t.x += s_w[wv].x; t.y += s_w[wv].y; }
    part[(int64_t)img * nblk_max + blockIdx.x] = t;
  }
}

__global__ void ke_final(const ImgDesc* __restrict__ tab, int B, int nblk_max, const double2* __restrict__ part,
                         double* __restrict__ out_entropy, double* __restrict__ out_degree) {
  const int img = blockIdx.x * blockDim.x + threadIdx.x;
  if (img >= B) return;
  const ImgDesc d = tab[img];
  const int n = d.w * d.h;
  const int nblk = (n + KE_THREADS * KE_PER - 1) / (KE_THREADS * KE_PER);
  double a = 0.0, b = 0.0;
  for (int k = 0; k < nblk; ++k) { const double2 t = part[(int64_t)img * nblk_max + k]; a += t.x; b += t.y; }
  double H = 0.0, deg = 0.0;
  if (a > 0.0) {
    H = log(a) - b / a;
    if (H < 0.0) H = 0.0;                                    // rounding of the two terms when all mass sits in one cell
    if (n > 1) deg = 1.0 - H / log((double)n);
  }
  out_entropy[img] = H;
  out_degree[img] = deg;
}

// =====================================================================================================
// f2 — exact-position density (reading B4).  Gather form: a CTA owns a tile of 16 x 32 cells and walks
// the frame's kept boxes 256 at a time; every thread turns one box into its centroid in cell units (fp32, the in-frame
// test of O7), the ones whose truncation square reaches the tile are compacted IN KEEP ORDER into shared memory
// (ballot + prefix sums), and every thread then adds the boxes of the list to its two cells.  The summation order of
// a cell is the keep order, whatever the launch: bit-reproducible.  dx, dy and the |d| <= R decisions are single fp32
// operations, the same ones the definition prescribes.
// =====================================================================================================
constexpr int KD_THREADS = 256;
constexpr int KD_TW = 32, KD_TH = 16;

__global__ void __launch_bounds__(KD_THREADS) kd_exact(const ffpp_box* __restrict__ boxes, const int32_t* __restrict__ counts,
                                                       const ImgDesc* __restrict__ tab, Consts cst, float neg_inv_2s2, float inv_z2,
                                                       float* __restrict__ out) {
  __shared__ float2 s_uv[KD_THREADS];
  __shared__ int s_wsum[KD_THREADS / 32];
  const int img = blockIdx.y;
  const ImgDesc d = tab[img];
  const int tiles_x = (d.w + KD_TW - 1) / KD_TW, tiles_y = (d.h + KD_TH - 1) / KD_TH;
  if ((int)blockIdx.x >= tiles_x * tiles_y) return;
  const int ty = (int)blockIdx.x / tiles_x, tx = (int)blockIdx.x - ty * tiles_x;
  const int X0 = tx * KD_TW, Y0 = ty * KD_TH;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int ix = X0 + lane, iy0 = Y0 + warp, iy1 = Y0 + warp + 8;
  const float xc = (float)ix + 0.5f, yc0 = (float)iy0 + 0.5f, yc1 = (float)iy1 + 0.5f;
  const float Rf = (float)cst.radius;
  const float W = (float)(d.w * cst.cell_px), H = (float)(d.h * cst.cell_px);
  // a box can touch the tile only if its centroid (cell units) lies within R of the tile's cell centres
  const float ulo = (float)X0 + 0.5f - Rf, uhi = (float)(X0 + KD_TW - 1) + 0.5f + Rf;
  const float vlo = (float)Y0 + 0.5f - Rf, vhi = (float)(Y0 + KD_TH - 1) + 0.5f + Rf;
  const int n = counts[img];
  const ffpp_box* fb = boxes + (int64_t)img * cst.top_k;
  float acc0 = 0.0f, acc1 = 0.0f;
  for (int base = 0; base < n; base += KD_THREADS) {
    const int b = base + tid;
    bool take = false;
    float u = 0.0f, v = 0.0f;
    if (b < n) {
      const float2* p = reinterpret_cast<const float2*>(fb + b);   // 24-byte records, 8-byte aligned
      const float2 p0 = p[0], p1 = p[1];
      const float cx = __fmul_rn(__fadd_rn(p0.x, p1.x), 0.5f), cy = __fmul_rn(__fadd_rn(p0.y, p1.y), 0.5f);
      if (cx >= 0.0f && cx < W && cy >= 0.0f && cy < H) {
        u = cst.cell_inv != 0.0f ? __fmul_rn(cx, cst.cell_inv) : __fdiv_rn(cx, (float)cst.cell_px);
        v = cst.cell_inv != 0.0f ? __fmul_rn(cy, cst.cell_inv) : __fdiv_rn(cy, (float)cst.cell_px);
        take = u >= ulo - 1e-3f && u <= uhi + 1e-3f && v >= vlo - 1e-3f && v <= vhi + 1e-3f;   // conservative: the exact test is per cell
      }
    }
    const uint32_t bal = __ballot_sync(0xffffffffu, take);
    if (lane == 0) s_wsum[warp] = __popc(bal);
    __syncthreads();
    int before = 0, total = 0;
#pragma unroll
    for (int wv = 0; wv < KD_THREADS / 32; ++wv) { const int c = s_wsum[wv]; if (wv < warp) before += c; total += c; }
    if (take) s_uv[before + __popc(bal & ((1u << lane) - 1u))] = make_float2(u, v);
    __syncthreads();
    for (int k = 0; k < total; ++k) {
      const float2 q = s_uv[k];
      const float dy0 = __fsub_rn(yc0, q.y), dy1 = __fsub_rn(yc1, q.y);
      const bool in0 = fabsf(dy0) <= Rf, in1 = fabsf(dy1) <= Rf;
      if (!(in0 | in1)) continue;                            // warp-uniform: a warp is one row of the tile (and the row 8 below)
      const float dx = __fsub_rn(xc, q.x);
      if (!(fabsf(dx) <= Rf)) continue;
      const float dx2 = dx * dx;
      if (in0) acc0 += expf((dx2 + dy0 * dy0) * neg_inv_2s2) * inv_z2;
      if (in1) acc1 += expf((dx2 + dy1 * dy1) * neg_inv_2s2) * inv_z2;
    }
    __syncthreads();
  }
  if (ix < d.w) {
    if (iy0 < d.h) out[d.off + (int64_t)iy0 * d.w + ix] = acc0;
    if (iy1 < d.h) out[d.off + (int64_t)iy1 * d.w + ix] = acc1;
  }
}

// =====================================================================================================
// f4 — pre-processing (reading B6): bilinear resize + normalise + HWC uint8 -> CHW, one pass.
// Source coordinates are exact rationals: fx = ((2x + 1) Ws - Wd) / (2 Wd), so the left neighbour is an integer division
// and the weight one correctly rounded fp32 division — no drift across a 4 k-pixel row.  A thread produces 4
// consecutive outputs of all three channels (8- or 16-byte stores per channel plane); HBM-bound: 3 bytes read per
// source pixel (each touched once through L1/L2), 3 x 2 or 3 x 4 bytes written per destination pixel.
// =====================================================================================================
constexpr int KP_THREADS = 256;
struct PreNorm { float scale[3], bias[3]; };       // out = v * scale + bias  with scale = 1 / (255 std), bias = -mean / std

__device__ __forceinline__ void kp_axis(const int o, const int S, const int D, int& i0, int& i1, float& w) {
  const int num = (2 * o + 1) * S - D, den = 2 * D;
  if (num <= 0) { i0 = 0; w = 0.0f; }
  else { i0 = num / den; w = __fdiv_rn((float)(num - i0 * den), (float)den); }
  if (i0 > S - 1) i0 = S - 1;
  i1 = i0 + 1 < S ? i0 + 1 : S - 1;
}
__device__ __forceinline__ void kp_store4(float* p, const float4 v) { *reinterpret_cast<float4*>(p) = v; }
__device__ __forceinline__ void kp_store4(__half* p, const float4 v) {
  const __half2 a = __floats2half2_rn(v.x, v.y), b = __floats2half2_rn(v.z, v.w);
  uint2 u;
  u.x = *reinterpret_cast<const uint32_t*>(&a); u.y = *reinterpret_cast<const uint32_t*>(&b);
  *reinterpret_cast<uint2*>(p) = u;
}
__device__ __forceinline__ void kp_store1(float* p, const float v) { *p = v; }
__device__ __forceinline__ void kp_store1(__half* p, const float v) { *p = __float2half_rn(v); }

template <typename OutT>
__global__ void __launch_bounds__(KP_THREADS) kp_preprocess(const uint8_t* __restrict__ src, int Hs, int Ws, int Hd, int Wd, PreNorm nrm,
                                                            OutT* __restrict__ dst) {
  const int img = blockIdx.z, y = blockIdx.y;
  const int x4 = (blockIdx.x * KP_THREADS + threadIdx.x) * 4;
  if (x4 >= Wd) return;
  int y0, y1;
  float wy;
  kp_axis(y, Hs, Hd, y0, y1, wy);
  const uint8_t* r0 = src + ((int64_t)img * Hs + y0) * Ws * 3;
  const uint8_t* r1 = src + ((int64_t)img * Hs + y1) * Ws * 3;
  float o[3][4];
#pragma unroll
  for (int e = 0; e < 4; ++e) {
    int xa, xb;
    float wx;
    kp_axis(min(x4 + e, Wd - 1), Ws, Wd, xa, xb, wx);
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      const float p00 = (float)r0[xa * 3 + c], p01 = (float)r0[xb * 3 + c], p10 = (float)r1[xa * 3 + c], p11 = (float)r1[xb * 3 + c];
      const float top = p00 + wx * (p01 - p00), bot = p10 + wx * (p11 - p10);
      o[c][e] = (top + wy * (bot - top)) * nrm.scale[c] + nrm.bias[c];
    }
  }
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    OutT* p = dst + (((int64_t)img * 3 + c) * Hd + y) * Wd + x4;
    if (x4 + 4 <= Wd && (((uintptr_t)p) & (4 * sizeof(OutT) - 1)) == 0) {
      kp_store4(p, make_float4(o[c][0], o[c][1], o[c][2], o[c][3]));
    } else {
      for (int e = 0; e < 4 && x4 + e < Wd; ++e) kp_store1(p + e, o[c][e]);
    }
  }
}

}  // namespace ffpp

// =====================================================================================================
// host side
// =====================================================================================================
namespace {

// grid table of a batch geometry (f1, f2): found among the handle's cached slots, else built and uploaded
int next_geometry(ffpp_handle* h, int B, const int32_t* dims, cudaStream_t st, const ffpp::ImgDesc** out_tab, int64_t* cells_out,
                  int* max_cells_out, int* max_w_out, int* max_h_out) {
  uint64_t hash = 0x51ED270B9ull ^ (uint64_t)B;
  for (int f = 0; f < 2 * B; ++f) { hash ^= (uint32_t)dims[f] + 0x9E3779B97F4A7C15ull + (hash << 6) + (hash >> 2); hash *= 0xD6E8FEB86659FD93ull; hash ^= hash >> 32; }
  int lru = 0;
  for (int s = 0; s < ffpp_handle::kNextSlots; ++s) {
    ffpp_handle::NextGeo& g = h->ngeo[s];
    if (g.B == B && g.hash == hash && std::memcmp(dims, g.dims.data(), sizeof(int32_t) * 2 * B) == 0) {
      g.last_use = ++h->use_clock;
      *out_tab = static_cast<const ffpp::ImgDesc*>(g.d_tab); *cells_out = g.cells; *max_cells_out = g.max_cells; *max_w_out = g.max_w; *max_h_out = g.max_h;
      return FFPP_OK;
    }
    if (g.last_use < h->ngeo[lru].last_use) lru = s;
  }
  {
    cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
    if (cudaStreamIsCapturing(st, &cap) == cudaSuccess && cap != cudaStreamCaptureStatusNone)
      return fail(h, FFPP_EINVAL, "batch geometry not cached: run it once outside stream capture first");
    cudaGetLastError();
  }
  std::vector<ffpp::ImgDesc> tab((size_t)B);
  int64_t cells = 0;
  int max_cells = 0, max_w = 0, max_h = 0;
  for (int f = 0; f < B; ++f) {
    const int W = dims[2 * f], H = dims[2 * f + 1];
    if (W <= 0 || H <= 0 || W % h->p.cell_px || H % h->p.cell_px) return fail(h, FFPP_EINVAL, "frame_dims: W and H must be positive multiples of cell_px");
    if (W > h->p.max_frame_w || H > h->p.max_frame_h) return fail(h, FFPP_ECAPACITY, "frame exceeds max_frame_w/max_frame_h");
    tab[(size_t)f].off = cells; tab[(size_t)f].w = W / h->p.cell_px; tab[(size_t)f].h = H / h->p.cell_px;
    const int c = tab[(size_t)f].w * tab[(size_t)f].h;
    cells += c;
    max_cells = std::max(max_cells, c); max_w = std::max(max_w, (int)tab[(size_t)f].w); max_h = std::max(max_h, (int)tab[(size_t)f].h);
  }
  if (cells > h->max_total_cells) return fail(h, FFPP_ECAPACITY, "density cells exceed max_total_cells");
  ffpp_handle::NextGeo& g = h->ngeo[lru];
  g.B = -1;
  if (!g.d_tab) FFPP_CUDA(h, cudaMalloc(&g.d_tab, sizeof(ffpp::ImgDesc) * (size_t)h->p.max_frames));
  FFPP_CUDA(h, cudaMemcpyAsync(g.d_tab, tab.data(), sizeof(ffpp::ImgDesc) * (size_t)B, cudaMemcpyHostToDevice, st));   // pageable: staged before return
  g.B = B; g.hash = hash; g.dims.assign(dims, dims + 2 * B);
  g.cells = cells; g.max_cells = max_cells; g.max_w = max_w; g.max_h = max_h;
  g.last_use = ++h->use_clock;
  *out_tab = static_cast<const ffpp::ImgDesc*>(g.d_tab); *cells_out = cells; *max_cells_out = max_cells; *max_w_out = max_w; *max_h_out = max_h;
  return FFPP_OK;
}

// scratch of the component labelling: one int32 per pixel, one 64-bit sum per table row; grown on demand
int next_scratch(ffpp_handle* h, int64_t pixels, int64_t rows, int64_t blocks, cudaStream_t st) {
  if (pixels > h->ccl_aux_cap || rows > h->ccl_sum_cap || blocks > h->ccl_blk_cap) {
    cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
    if (cudaStreamIsCapturing(st, &cap) == cudaSuccess && cap != cudaStreamCaptureStatusNone)
      return fail(h, FFPP_EINVAL, "labelling scratch not allocated yet: run this call once outside stream capture first");
    cudaGetLastError();
  }
  if (pixels > h->ccl_aux_cap) {
    FFPP_CUDA(h, cudaStreamSynchronize(st));                 // earlier work on this stream may still use the old buffer
    cudaFree(h->d_ccl_aux); h->d_ccl_aux = nullptr; h->ccl_aux_cap = 0;
    FFPP_CUDA(h, cudaMalloc((void**)&h->d_ccl_aux, sizeof(int32_t) * (size_t)pixels));
    h->ccl_aux_cap = pixels;
  }
  if (rows > h->ccl_sum_cap) {
    FFPP_CUDA(h, cudaStreamSynchronize(st));
    cudaFree(h->d_ccl_sums); h->d_ccl_sums = nullptr; h->ccl_sum_cap = 0;
    FFPP_CUDA(h, cudaMalloc((void**)&h->d_ccl_sums, sizeof(unsigned long long) * (size_t)rows));
    h->ccl_sum_cap = rows;
  }
  if (blocks > h->ccl_blk_cap) {
    FFPP_CUDA(h, cudaStreamSynchronize(st));
    cudaFree(h->d_ccl_blk); h->d_ccl_blk = nullptr; h->ccl_blk_cap = 0;
    FFPP_CUDA(h, cudaMalloc((void**)&h->d_ccl_blk, sizeof(int32_t) * (size_t)blocks));
    h->ccl_blk_cap = blocks;
  }
  return FFPP_OK;
}

template <typename T>
int run_ccl(ffpp_handle* h, const T* src, const ffpp::ImgDesc* tab, int B, int w0, int h0, int max_px, float thr, int conn, int min_area,
            int max_out, int mean, cudaStream_t st, int32_t* labels, ffpp_region* out, int32_t* counts) {
  using namespace ffpp;
  const dim3 g((unsigned)((max_px + KC_THREADS * KC_PER - 1) / (KC_THREADS * KC_PER)), (unsigned)B);
  kc_init<T><<<g, KC_THREADS, 0, st>>>(src, tab, w0, h0, thr, labels, h->d_ccl_aux);
  kc_merge<<<g, KC_THREADS, 0, st>>>(tab, w0, h0, conn, labels);
  kc_flatten<<<g, KC_THREADS, 0, st>>>(tab, w0, h0, labels, h->d_ccl_aux);
  const int nblk = (max_px + KR_BLOCK - 1) / KR_BLOCK;
  const dim3 gr((unsigned)nblk, (unsigned)B);
  kr_count_place<false><<<gr, KC_RANK_THREADS, 0, st>>>(tab, w0, h0, labels, h->d_ccl_aux, min_area, max_out, nblk, h->d_ccl_blk, out, h->d_ccl_sums);
  kr_scan<<<B, KC_THREADS, 0, st>>>(tab, w0, h0, nblk, h->d_ccl_blk, counts);
  kr_count_place<true><<<gr, KC_RANK_THREADS, 0, st>>>(tab, w0, h0, labels, h->d_ccl_aux, min_area, max_out, nblk, h->d_ccl_blk, out, h->d_ccl_sums);
  kc_stats<T><<<g, KC_THREADS, 0, st>>>(src, tab, w0, h0, labels, h->d_ccl_aux, max_out, out, h->d_ccl_sums);
  const dim3 gf((unsigned)((max_out + KC_THREADS - 1) / KC_THREADS), (unsigned)B);
  kc_final<<<gf, KC_THREADS, 0, st>>>(max_out, mean, counts, out, h->d_ccl_sums);
  FFPP_CUDA(h, cudaGetLastError());
  return FFPP_OK;
}

}  // namespace

extern "C" {

int ffpp_heatmap_stats(ffpp_handle* h, const float* density, int32_t B, const int32_t* frame_dims, float threshold, int32_t connectivity,
                       int32_t max_regions, void* stream, double* out_entropy, double* out_degree, int32_t* out_labels,
                       ffpp_region* out_regions, int32_t* out_region_counts) {
  using namespace ffpp;
  if (!h) return FFPP_EINVAL;
  if (B < 0) return fail(h, FFPP_EINVAL, "B < 0");
  if (B == 0) return FFPP_OK;
  if (!density || !frame_dims || !out_entropy || !out_degree || !out_labels || !out_regions || !out_region_counts) return fail(h, FFPP_EINVAL, "null pointer");
  if (B > h->p.max_frames) return fail(h, FFPP_ECAPACITY, "B exceeds max_frames");
  if (connectivity != 4 && connectivity != 8) return fail(h, FFPP_EINVAL, "connectivity must be 4 or 8");
  if (max_regions < 1) return fail(h, FFPP_EINVAL, "max_regions must be >= 1");
  if (std::isnan(threshold)) return fail(h, FFPP_EINVAL, "threshold is NaN");
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  const ImgDesc* tab = nullptr;
  int64_t cells = 0;
  int max_cells = 0, mw = 0, mh = 0;
  int rc = next_geometry(h, B, frame_dims, st, &tab, &cells, &max_cells, &mw, &mh);
  if (rc != FFPP_OK) return rc;
  const int nblk = (max_cells + KE_THREADS * KE_PER - 1) / (KE_THREADS * KE_PER);
  if ((int64_t)B * nblk > h->ent_part_cap) {
    cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
    if (cudaStreamIsCapturing(st, &cap) == cudaSuccess && cap != cudaStreamCaptureStatusNone)
      return fail(h, FFPP_EINVAL, "entropy scratch not allocated yet: run this call once outside stream capture first");
    cudaGetLastError();
    FFPP_CUDA(h, cudaStreamSynchronize(st));
    cudaFree(h->d_ent_part); h->d_ent_part = nullptr; h->ent_part_cap = 0;
    FFPP_CUDA(h, cudaMalloc((void**)&h->d_ent_part, sizeof(double2) * (size_t)B * nblk));
    h->ent_part_cap = (int64_t)B * nblk;
  }
  if ((rc = next_scratch(h, cells, (int64_t)B * max_regions, (int64_t)B * ((max_cells + KR_BLOCK - 1) / KR_BLOCK), st)) != FFPP_OK) return rc;
  ke_partial<<<dim3((unsigned)nblk, (unsigned)B), KE_THREADS, 0, st>>>(density, tab, nblk, static_cast<double2*>(h->d_ent_part));
  ke_final<<<(B + 127) / 128, 128, 0, st>>>(tab, B, nblk, static_cast<const double2*>(h->d_ent_part), out_entropy, out_degree);
  return run_ccl<float>(h, density, tab, B, 0, 0, max_cells, threshold, connectivity, 1, max_regions, 0, st, out_labels, out_regions, out_region_counts);
}

int ffpp_density_exact(ffpp_handle* h, const ffpp_box* boxes, const int32_t* counts, int32_t B, const int32_t* frame_dims, void* stream,
                       float* out_density) {
  using namespace ffpp;
  if (!h) return FFPP_EINVAL;
  if (B < 0) return fail(h, FFPP_EINVAL, "B < 0");
  if (B == 0) return FFPP_OK;
  if (!boxes || !counts || !frame_dims || !out_density) return fail(h, FFPP_EINVAL, "null pointer");
  if (B > h->p.max_frames) return fail(h, FFPP_ECAPACITY, "B exceeds max_frames");
  if (reinterpret_cast<uintptr_t>(boxes) & 7) return fail(h, FFPP_EINVAL, "boxes must be 8-byte aligned");
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  const ImgDesc* tab = nullptr;
  int64_t cells = 0;
  int max_cells = 0, mw = 0, mh = 0;
  const int rc = next_geometry(h, B, frame_dims, st, &tab, &cells, &max_cells, &mw, &mh);
  if (rc != FFPP_OK) return rc;
  const double s2 = 2.0 * (double)h->p.sigma_cells * (double)h->p.sigma_cells;
  double Z = 0.0;
  for (int k = -h->cst.radius; k <= h->cst.radius; ++k) Z += std::exp(-(double)(k * k) / s2);
  const int tiles = ((mw + KD_TW - 1) / KD_TW) * ((mh + KD_TH - 1) / KD_TH);
  kd_exact<<<dim3((unsigned)tiles, (unsigned)B), KD_THREADS, 0, st>>>(boxes, counts, tab, h->cst, (float)(-1.0 / s2), (float)(1.0 / (Z * Z)), out_density);
  FFPP_CUDA(h, cudaGetLastError());
  return FFPP_OK;
}

int ffpp_mask_components(ffpp_handle* h, const void* mask, int32_t dtype, int32_t B, int32_t W, int32_t H, float threshold, int32_t connectivity,
                         int32_t min_area, int32_t max_components, void* stream, int32_t* out_labels, ffpp_region* out_components,
                         int32_t* out_counts) {
  using namespace ffpp;
  if (!h) return FFPP_EINVAL;
  if (B < 0) return fail(h, FFPP_EINVAL, "B < 0");
  if (B == 0) return FFPP_OK;
  if (!mask || !out_labels || !out_components || !out_counts) return fail(h, FFPP_EINVAL, "null pointer");
  if (dtype != 0 && dtype != 1) return fail(h, FFPP_EINVAL, "dtype must be 0 (fp32) or 1 (fp16)");
  if (W < 1 || H < 1 || (int64_t)W * H >= ((int64_t)1 << 31)) return fail(h, FFPP_EINVAL, "mask dimensions out of range");
  if (B > 65535) return fail(h, FFPP_ECAPACITY, "more than 65535 masks in one call");
  if (connectivity != 4 && connectivity != 8) return fail(h, FFPP_EINVAL, "connectivity must be 4 or 8");
  if (max_components < 1) return fail(h, FFPP_EINVAL, "max_components must be >= 1");
  if (std::isnan(threshold)) return fail(h, FFPP_EINVAL, "threshold is NaN");
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  const int rc = next_scratch(h, (int64_t)B * W * H, (int64_t)B * max_components, (int64_t)B * ((W * H + KR_BLOCK - 1) / KR_BLOCK), st);
  if (rc != FFPP_OK) return rc;
  const int ma = min_area < 1 ? 1 : min_area;
  if (dtype == 1)
    return run_ccl<__half>(h, static_cast<const __half*>(mask), nullptr, B, W, H, W * H, threshold, connectivity, ma, max_components, 1, st,
                           out_labels, out_components, out_counts);
  return run_ccl<float>(h, static_cast<const float*>(mask), nullptr, B, W, H, W * H, threshold, connectivity, ma, max_components, 1, st, out_labels,
                        out_components, out_counts);
}

int ffpp_preprocess(const uint8_t* src, int32_t B, int32_t Hs, int32_t Ws, int32_t Hd, int32_t Wd, const float* mean, const float* stdv,
                    int32_t out_dtype, void* stream, void* dst) {
  using namespace ffpp;
  if (B < 0 || !mean || !stdv) return FFPP_EINVAL;
  if (B == 0) return FFPP_OK;
  if (!src || !dst || Hs < 1 || Ws < 1 || Hd < 1 || Wd < 1 || (out_dtype != 0 && out_dtype != 1)) return FFPP_EINVAL;
  if (Hs > 16384 || Ws > 16384 || Hd > 16384 || Wd > 16384 || Hd > 65535 || B > 65535) return FFPP_ECAPACITY;   // (2x+1)*S stays in int32
  PreNorm n;
  for (int c = 0; c < 3; ++c) {
    if (!(stdv[c] != 0.0f)) return FFPP_EINVAL;
    n.scale[c] = (float)(1.0 / (255.0 * (double)stdv[c]));
    n.bias[c] = (float)(-(double)mean[c] / (double)stdv[c]);
  }
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  const dim3 g((unsigned)((Wd + 4 * KP_THREADS - 1) / (4 * KP_THREADS)), (unsigned)Hd, (unsigned)B);
  if (out_dtype == 1) kp_preprocess<__half><<<g, KP_THREADS, 0, st>>>(src, Hs, Ws, Hd, Wd, n, static_cast<__half*>(dst));
  else kp_preprocess<float><<<g, KP_THREADS, 0, st>>>(src, Hs, Ws, Hd, Wd, n, static_cast<float*>(dst));
  return cudaGetLastError() == cudaSuccess ? FFPP_OK : FFPP_ECUDA;
}

}  // extern "C"
