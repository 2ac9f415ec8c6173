// Dense rank-order bitmask NMS (ffpp_params.nms_mode = 1): the design BASELINE.json north_star (c) sketches, kept as
// the reference point the spatially tiled default (ffpp_kernels.cuh k3/k4) is measured against.
//   a3  k3d_nms_mask  : every 64x64 tile of the upper triangle of the rank-ordered IoU matrix -> suppression words
//   a4  k4d_nms_sweep : one CTA per frame walks the 64-rank chunks in order; one warp resolves a chunk with shuffles
// Work is n(n-1)/2 IoU tests and n^2/16 bytes of mask per frame whatever the geometry.
#pragma once
#include "ffpp_common.cuh"

namespace ffpp {

constexpr int K3D_THREADS = 64;
constexpr int K3D_TILES_PER_UNIT = 16;

__host__ __device__ inline int k3d_units_per_pair(int nb) { return (nb + 1 + K3D_TILES_PER_UNIT - 1) / K3D_TILES_PER_UNIT; }
__host__ __device__ inline int k3d_units(int nb) { return ((nb + 1) / 2) * k3d_units_per_pair(nb); }

// bit (i, j), i < j in rank order, = IoU(box_i, box_j) > thr.  64 threads own the 64 rows of a row block, the 64
// column boxes sit in shared memory (broadcast reads).  Work units pair row block p with row block nb-1-p so every
// unit has the same tile count.
__global__ void __launch_bounds__(K3D_THREADS) k3d_nms_mask(const FrameDesc* __restrict__ frames,
                                                            const int* __restrict__ unit_prefix, int B,
                                                            const float4* __restrict__ sorted_box,
                                                            const int* __restrict__ n_sorted, Consts cst,
                                                            unsigned long long* __restrict__ mask) {
  __shared__ float4 cols[2][kNmsTile];
  const int t = threadIdx.x;
  int lo = 0, hi = B;
  const int u_global = blockIdx.x;
  while (hi - lo > 1) { const int mid = (lo + hi) >> 1; if (unit_prefix[mid] <= u_global) lo = mid; else hi = mid; }
  const int f = lo;
  const int n = n_sorted[f];
  const int nb_act = (n + kNmsTile - 1) / kNmsTile;
  const int nb = frames[f].nbmax;
  const int u = u_global - unit_prefix[f];
  const int upp = k3d_units_per_pair(nb);
  const int p = u / upp, c = u - p * upp;
  if (p >= nb_act && nb - 1 - p >= nb_act) return;
  const int64_t moff = frames[f].mask_off;
  const float4* boxes = sorted_box + (int64_t)f * cst.top_k;

  const int s_begin = c * K3D_TILES_PER_UNIT;
  const int s_end = (s_begin + K3D_TILES_PER_UNIT < nb + 1) ? s_begin + K3D_TILES_PER_UNIT : nb + 1;
  int cur_rb = -1;
  float4 a = make_float4(0.f, 0.f, 0.f, 0.f);
  int buf = 0;
  for (int s = s_begin; s < s_end; ++s) {
    int rb, cb;
    if (s < nb - p) { rb = p; cb = p + s; }
    else { rb = nb - 1 - p; cb = rb + (s - (nb - p)); if (rb == p) break; }
    if (rb >= nb_act || cb >= nb_act) continue;       // block-uniform
    const int row = rb * kNmsTile + t;
    if (rb != cur_rb) { cur_rb = rb; if (row < n) a = boxes[row]; }
    const int col0 = cb * kNmsTile;
    cols[buf][t] = (col0 + t < n) ? boxes[col0 + t] : make_float4(0.f, 0.f, 0.f, 0.f);
    __syncthreads();
    if (row < n) {
      unsigned long long word = 0;
#pragma unroll 8
      for (int j = 0; j < kNmsTile; ++j) {
        const float4 b = cols[buf][j];
        if (boxes_overlap(a, b)) {
          if (iou_exceeds(a, b, cst)) word |= 1ull << j;
        }
      }
      const int ncol = n - col0;                       // valid columns in this tile
      if (ncol < kNmsTile) word &= (1ull << ncol) - 1ull;
      if (cb == rb) word &= (t == 63) ? 0ull : ~((2ull << t) - 1ull);   // strictly later ranks only
      mask[moff + mask_rb_off(rb, nb) + (int64_t)t * (nb - rb) + (cb - rb)] = word;
    }
    buf ^= 1;                                          // double buffer: one barrier per tile
  }
}

constexpr int K4D_THREADS = 256;

// One CTA per frame.  For chunk q of 64 ranks: warp 0 resolves the chunk against `removed[q]` and the diagonal words
// with ffs-driven iterations (one per kept box, register shuffles), emits the chunk's kept boxes in keep order (and
// bins their centroids, a5); then all threads OR the row tails of the kept rows into `removed`.
__global__ void __launch_bounds__(K4D_THREADS) k4d_nms_sweep(const FrameDesc* __restrict__ frames,
                                                             const float4* __restrict__ sorted_box,
                                                             const float* __restrict__ sorted_logit,
                                                             const int* __restrict__ sorted_idx,
                                                             const int* __restrict__ n_sorted, Consts cst,
                                                             const unsigned long long* __restrict__ mask,
                                                             ffpp_box* __restrict__ out_boxes,
                                                             int* __restrict__ out_counts,
                                                             uint32_t* __restrict__ hist32) {
  extern __shared__ unsigned long long removed[];      // nbmax words
  __shared__ unsigned long long s_kept;
  __shared__ FrameDesc fd;
  const int f = blockIdx.x, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  if (tid == 0) fd = frames[f];
  const int n = n_sorted[f];
  const int nb_act = (n + kNmsTile - 1) / kNmsTile;
  __syncthreads();
  const int nb = fd.nbmax;
  const unsigned long long* fm = mask + fd.mask_off;
  const int64_t ibase = (int64_t)f * cst.top_k;
  for (int i = tid; i < nb_act; i += K4D_THREADS) removed[i] = 0ull;
  __syncthreads();
  int kept_total = 0;                                   // meaningful in warp 0
  for (int q = 0; q < nb_act; ++q) {
    const int64_t rbo = mask_rb_off(q, nb);
    const int rl = nb - q;
    if (warp == 0) {
      const int r0 = q * kNmsTile + lane, r1 = r0 + 32;
      const unsigned long long d0 = r0 < n ? fm[rbo + (int64_t)lane * rl] : 0ull;
      const unsigned long long d1 = r1 < n ? fm[rbo + (int64_t)(lane + 32) * rl] : 0ull;
      unsigned long long cur = removed[q];
      const int nrow = n - q * kNmsTile;
      const unsigned long long valid = nrow >= kNmsTile ? ~0ull : ((1ull << nrow) - 1ull);
      unsigned long long alive = ~cur & valid, kept = 0ull;
      while (alive) {
        const int b = __ffsll((long long)alive) - 1;
        kept |= 1ull << b;
        const unsigned long long mine = (b & 32) ? d1 : d0;
        const unsigned long long w = __shfl_sync(0xffffffffu, mine, b & 31);
        cur |= w;
        alive &= ~cur;
        alive &= ~(1ull << b);
      }
      if (lane == 0) s_kept = kept;
#pragma unroll
      for (int h = 0; h < 2; ++h) {
        const int b = lane + 32 * h;
        if ((kept >> b) & 1ull) {
          const int pos = kept_total + __popcll(kept & ((1ull << b) - 1ull));
          const int r = q * kNmsTile + b;
          emit_kept(fd, cst, out_boxes + ibase + pos, sorted_box[ibase + r], sorted_logit[ibase + r], sorted_idx[ibase + r],
                    hist32);
        }
      }
      kept_total += __popcll(kept);
    }
    __syncthreads();
    const unsigned long long km = s_kept;
    if (km) {
      for (int cb = q + 1 + tid; cb < nb_act; cb += K4D_THREADS) {
        unsigned long long acc = 0ull, m = km;
        while (m) {
          const int b = __ffsll((long long)m) - 1;
          m &= m - 1ull;
          acc |= fm[rbo + (int64_t)b * rl + (cb - q)];
        }
        removed[cb] |= acc;
      }
    }
    __syncthreads();
  }
  if (tid == 0) out_counts[f] = kept_total;
}

}  // namespace ffpp
