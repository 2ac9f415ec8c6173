// The five stage kernels of the CUDA path (sm_100a).  See DESIGN.md §"Kernels" for the roofline of each.
// Stage numbering follows SURVEY.md §8(a): a1 threshold+compaction, a2 sort+top-K(+decode), a3 NMS bitmask,
// a4 NMS sweep + output gather, a5-a6 density.
#pragma once
#include "ffpp_common.cuh"

namespace ffpp {

// =====================================================================================================
// a1 — threshold + compaction (BASELINE.json north_star (a); SURVEY §8(a) a1, §8(c) O1+O3).
// HBM-bound stream over the flat [sum N_f, 5] head output.  The TMA engine (1-D cp.async.bulk, UBLKCP)
// moves 20 KB chunks into a 3-stage shared-memory ring so bytes in flight do not depend on thread count;
// threads only look at the score logit of each row (the 16-byte loads of the north_star sketch become
// bulk copies: same coalescing, no register staging).  Survivors get a sort key
//   (descending-monotone score bits) ‖ (candidate index in frame)
// which makes every key of a frame unique, so the slot order inside the per-frame survivor list is
// irrelevant and slots come from warp-aggregated shared-memory counters + one global atomic per
// (chunk, frame).  Boxes are NOT decoded here: only the <= top_k rows that survive the sort are decoded,
// in the a2 epilogue ("re-decoded after the sort").
// =====================================================================================================
constexpr int K1_THREADS = 256;
constexpr int K1_CHUNK_BYTES = 20480;   // multiple of lcm(16, 10, 20) = 80
constexpr int K1_STAGES = 3;
constexpr int K1_MAXF = 16;             // frames a chunk may span on the fast path

template <bool kHalf, typename KeyT>
__device__ __forceinline__ bool k1_eval(const uint8_t* buf, int gl, float T, int idx, KeyT& key) {
  if (kHalf) {
    const uint16_t h = *reinterpret_cast<const uint16_t*>(buf + (size_t)gl * 10 + 8);
    const float z = __half2float(__ushort_as_half(h));
    if (sizeof(KeyT) == 4) key = (KeyT)((desc_key16(h) << 16) | (uint32_t)idx);
    else key = (KeyT)(((uint64_t)desc_key32(z) << 32) | (uint32_t)idx);
    return z > T;
  } else {
    const float z = *reinterpret_cast<const float*>(buf + (size_t)gl * 20 + 16);
    key = (KeyT)(((uint64_t)desc_key32(z) << 32) | (uint32_t)idx);
    return z > T;
  }
}

template <bool kHalf, typename KeyT>
__global__ void __launch_bounds__(K1_THREADS) k1_threshold_compact(const uint8_t* __restrict__ raw, int64_t total_cand,
                                                                   int B, const int64_t* __restrict__ cand_off, float T,
                                                                   KeyT* __restrict__ surv_keys,
                                                                   int* __restrict__ surv_cnt) {
  constexpr int ROW = kHalf ? 10 : 20;
  constexpr int CPC = K1_CHUNK_BYTES / ROW;      // candidates per chunk: 2048 / 1024
  constexpr int CPT = CPC / K1_THREADS;          // per thread: 8 / 4
  extern __shared__ __align__(128) uint8_t ring[];
  __shared__ __align__(8) uint64_t bars[K1_STAGES];
  __shared__ int64_t s_off[K1_MAXF + 1];
  __shared__ int s_cnt[K1_MAXF], s_gbase[K1_MAXF], s_flo, s_nf;

  const int tid = threadIdx.x, lane = tid & 31;
  const int64_t total_bytes = total_cand * ROW;
  const int64_t nchunks = (total_bytes + K1_CHUNK_BYTES - 1) / K1_CHUNK_BYTES;

  auto issue = [&](int stage, int64_t c) {       // thread 0 only
    const int64_t b0 = c * K1_CHUNK_BYTES;
    int64_t len = total_bytes - b0;
    if (len > K1_CHUNK_BYTES) len = K1_CHUNK_BYTES;
    const uint32_t bulk = (uint32_t)(len & ~(int64_t)15);
    mbar_expect_tx(&bars[stage], bulk);
    if (bulk) bulk_g2s(ring + (size_t)stage * K1_CHUNK_BYTES, raw + b0, bulk, &bars[stage]);
  };

  if (tid == 0) {
    for (int s = 0; s < K1_STAGES; ++s) mbar_init(&bars[s], 1);
    mbar_fence_init();
  }
  __syncthreads();
  if (tid == 0)
    for (int s = 0; s < K1_STAGES; ++s) {
      const int64_t c = (int64_t)blockIdx.x + (int64_t)s * gridDim.x;
      if (c < nchunks) issue(s, c);
    }

  int it = 0;
  for (int64_t c = blockIdx.x; c < nchunks; c += gridDim.x, ++it) {
    const int stage = it % K1_STAGES;
    const uint32_t parity = (uint32_t)(it / K1_STAGES) & 1u;
    const int64_t g0 = c * CPC;
    const int64_t g1 = (g0 + CPC < total_cand) ? g0 + CPC : total_cand;
    uint8_t* buf = ring + (size_t)stage * K1_CHUNK_BYTES;

    // ---- chunk metadata (overlaps the copy): frames [flo, flo+nf) intersect [g0, g1) ----
    if (tid == 0) {
      int lo = 0, hi = B;                        // largest f with cand_off[f] <= g0
      while (hi - lo > 1) { const int mid = (lo + hi) >> 1; if (cand_off[mid] <= g0) lo = mid; else hi = mid; }
      int f2 = lo;
      while (f2 + 1 < B && cand_off[f2 + 1] < g1) ++f2;
      s_flo = lo; s_nf = f2 - lo + 1;
    }
    if (tid < K1_MAXF) s_cnt[tid] = 0;
    __syncthreads();
    const int flo = s_flo, nf = s_nf;
    const bool fast = nf <= K1_MAXF;
    if (fast && tid <= nf) s_off[tid] = cand_off[flo + tid];
    __syncthreads();

    mbar_wait(&bars[stage], parity);
    if (c == nchunks - 1) {                      // < 16 trailing bytes the bulk copy cannot carry
      const int64_t b0 = c * K1_CHUNK_BYTES;
      const int len = (int)(total_bytes - b0);
      const int bulk = len & ~15;
      if (tid < len - bulk) buf[bulk + tid] = raw[b0 + bulk + tid];
      __syncthreads();
    }

    if (fast) {
      // phase 1: evaluate, reserve chunk-local slots per frame
      KeyT keys[CPT];
      uint32_t slot[CPT];                        // (local frame << 16) | slot, 0xFFFFFFFF = not a survivor
      int fl = 0;
#pragma unroll
      for (int i = 0; i < CPT; ++i) {
        const int gl = i * K1_THREADS + tid;
        const int64_t g = g0 + gl;
        const bool valid = g < g1;
        if (valid) while (fl + 1 < nf && g >= s_off[fl + 1]) ++fl;
        bool pass = false;
        if (valid) pass = k1_eval<kHalf, KeyT>(buf, gl, T, (int)(g - s_off[fl]), keys[i]);
        const uint32_t tag = pass ? (uint32_t)fl : 0xFFFFu;
        const uint32_t peers = __match_any_sync(0xffffffffu, tag);
        const int leader = __ffs(peers) - 1;
        int base = 0;
        if (pass && lane == leader) base = atomicAdd(&s_cnt[fl], __popc(peers));
        base = __shfl_sync(0xffffffffu, base, leader);
        slot[i] = pass ? (((uint32_t)fl << 16) | (uint32_t)(base + __popc(peers & ((1u << lane) - 1u)))) : 0xFFFFFFFFu;
      }
      __syncthreads();
      // phase 2: one global atomic per (chunk, frame)
      if (tid < nf) s_gbase[tid] = s_cnt[tid] ? atomicAdd(&surv_cnt[flo + tid], s_cnt[tid]) : 0;
      __syncthreads();
      // phase 3: write keys
#pragma unroll
      for (int i = 0; i < CPT; ++i)
        if (slot[i] != 0xFFFFFFFFu) {
          const int f = (int)(slot[i] >> 16);
          surv_keys[s_off[f] + s_gbase[f] + (int)(slot[i] & 0xFFFFu)] = keys[i];
        }
    } else {
      // generic path (chunk spans > K1_MAXF tiny frames): per-candidate global atomics
      for (int i = 0; i < CPT; ++i) {
        const int gl = i * K1_THREADS + tid;
        const int64_t g = g0 + gl;
        if (g >= g1) continue;
        int lo = flo, hi = B;
        while (hi - lo > 1) { const int mid = (lo + hi) >> 1; if (cand_off[mid] <= g) lo = mid; else hi = mid; }
        KeyT key;
        if (k1_eval<kHalf, KeyT>(buf, gl, T, (int)(g - cand_off[lo]), key))
          surv_keys[cand_off[lo] + atomicAdd(&surv_cnt[lo], 1)] = key;
      }
    }
    __syncthreads();                             // every read of this stage is done
    if (tid == 0) {
      const int64_t cn = c + (int64_t)K1_STAGES * gridDim.x;
      if (cn < nchunks) issue(stage, cn);
    }
  }
}

// =====================================================================================================
// a2 — segmented per-frame sort + top-K + decode (north_star (b)).
// One 1024-thread CTA per frame.  (1) If n > K, an MSD radix select over the frame's keys (read from
// L2/HBM, <= keybits/8 histogram passes) finds the K-th smallest key; because keys are unique exactly K keys
// are <= it.  (2) Those keys are staged in shared memory and sorted by a stable LSD block radix sort (8-bit
// digits, per-warp contiguous segments ranked with match_any, passes whose digit is constant are skipped).
// (3) Epilogue: decode the sorted rows from the raw head output (fp32, cell-centre grid point, no clipping)
// and write boxes / logits / candidate indices in rank order.
// =====================================================================================================
constexpr int K2_THREADS = 1024;
constexpr int K2_WARPS = K2_THREADS / 32;

template <typename KeyT> struct KeyBits { static constexpr int value = sizeof(KeyT) * 8; };

// shared layout: KeyT buf0[cap] | KeyT buf1[cap] | uint16 hist[32][256] | uint32 tot[256] | misc
struct K2Misc {
  int wsum[K2_WARPS];
  int sel_digit, sel_kk, sel_tot, skip, count;
};

__device__ __forceinline__ void k2_zero_hist(uint16_t* hist, int tid) {
  uint32_t* h32 = reinterpret_cast<uint32_t*>(hist);
  for (int i = tid; i < K2_WARPS * 256 / 2; i += K2_THREADS) h32[i] = 0;
}

// exclusive scan of hist in (digit major, warp minor) order, in place.  All 1024 threads.
__device__ __forceinline__ void k2_scan_hist(uint16_t* hist, K2Misc* misc, int tid) {
  const int lane = tid & 31, warp = tid >> 5;
  const int d = tid >> 2, w0 = (tid & 3) * 8;
  int v[8], sum = 0;
#pragma unroll
  for (int j = 0; j < 8; ++j) { v[j] = hist[(w0 + j) * 256 + d]; sum += v[j]; }
  int inc = sum;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) { const int t = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= o) inc += t; }
  if (lane == 31) misc->wsum[warp] = inc;
  __syncthreads();
  if (warp == 0) {
    int x = misc->wsum[lane], xi = x;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { const int t = __shfl_up_sync(0xffffffffu, xi, o); if (lane >= o) xi += t; }
    misc->wsum[lane] = xi - x;
  }
  __syncthreads();
  int run = misc->wsum[warp] + inc - sum;
#pragma unroll
  for (int j = 0; j < 8; ++j) { hist[(w0 + j) * 256 + d] = (uint16_t)run; run += v[j]; }
}

template <bool kHalf, typename KeyT>
__global__ void __launch_bounds__(K2_THREADS, 1) k2_sort_topk_decode(const uint8_t* __restrict__ raw,
                                                                      const FrameDesc* __restrict__ frames,
                                                                      const KeyT* __restrict__ surv_keys,
                                                                      const int* __restrict__ surv_cnt, Consts cst,
                                                                      int cap, float4* __restrict__ sorted_box,
                                                                      float* __restrict__ sorted_logit,
                                                                      int* __restrict__ sorted_idx,
                                                                      int* __restrict__ n_sorted) {
  constexpr int KB = KeyBits<KeyT>::value;
  extern __shared__ __align__(16) uint8_t smem[];
  KeyT* buf0 = reinterpret_cast<KeyT*>(smem);
  KeyT* buf1 = buf0 + cap;
  uint16_t* hist = reinterpret_cast<uint16_t*>(buf1 + cap);
  uint32_t* tot = reinterpret_cast<uint32_t*>(hist + K2_WARPS * 256);
  K2Misc* misc = reinterpret_cast<K2Misc*>(tot + 256);
  __shared__ FrameDesc fd;

  const int f = blockIdx.x, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  if (tid == 0) fd = frames[f];
  __syncthreads();
  const int n = surv_cnt[f];
  const int K = cst.top_k;
  const int nsel = n < K ? n : K;
  const KeyT* gk = surv_keys + fd.cand_off;

  if (n > K) {
    // ---- MSD radix select: threshold key = K-th smallest ----
    KeyT prefix = 0, maskbits = 0, thr = 0;
    int kk = K;
    bool done = false;
    for (int shift = KB - 8; shift >= 0 && !done; shift -= 8) {
      k2_zero_hist(hist, tid);
      __syncthreads();
      for (int base = warp * 32; base < n; base += K2_THREADS) {
        const int i = base + lane;
        KeyT key = 0;
        bool m = false;
        if (i < n) { key = gk[i]; m = (key & maskbits) == prefix; }
        const uint32_t dg = m ? (uint32_t)((key >> shift) & 255) : 256u;
        const uint32_t peers = __match_any_sync(0xffffffffu, dg);
        if (m && lane == __ffs(peers) - 1) hist[warp * 256 + dg] += (uint16_t)__popc(peers);
        __syncwarp();
      }
      __syncthreads();
      if (tid < 256) {
        uint32_t s = 0;
#pragma unroll 8
        for (int w = 0; w < K2_WARPS; ++w) s += hist[w * 256 + tid];
        tot[tid] = s;
      }
      __syncthreads();
      if (warp == 0) {
        uint32_t v[8], s = 0;
#pragma unroll
        for (int j = 0; j < 8; ++j) { v[j] = tot[lane * 8 + j]; s += v[j]; }
        uint32_t inc = s;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { const uint32_t t = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= o) inc += t; }
        uint32_t run = inc - s;                          // keys in digits below this lane's first digit
        if (run < (uint32_t)kk && (uint32_t)kk <= inc) {
#pragma unroll
          for (int j = 0; j < 8; ++j) {
            if (run < (uint32_t)kk && (uint32_t)kk <= run + v[j]) {
              misc->sel_digit = lane * 8 + j; misc->sel_kk = kk - (int)run; misc->sel_tot = (int)v[j];
            }
            run += v[j];
          }
        }
      }
      __syncthreads();
      prefix |= (KeyT)misc->sel_digit << shift;
      maskbits |= (KeyT)255 << shift;
      kk = misc->sel_kk;
      if (misc->sel_tot == kk) {                          // the whole bucket is selected
        thr = prefix | (shift ? (((KeyT)1 << shift) - 1) : (KeyT)0);
        done = true;
      }
      __syncthreads();
    }
    if (!done) thr = prefix;
    if (tid == 0) misc->count = 0;
    __syncthreads();
    for (int base = warp * 32; base < n; base += K2_THREADS) {
      const int i = base + lane;
      KeyT key = 0;
      bool m = false;
      if (i < n) { key = gk[i]; m = key <= thr; }
      const uint32_t bal = __ballot_sync(0xffffffffu, m);
      int b = 0;
      if (lane == 0 && bal) b = atomicAdd(&misc->count, __popc(bal));
      b = __shfl_sync(0xffffffffu, b, 0);
      if (m) buf0[b + __popc(bal & ((1u << lane) - 1u))] = key;
    }
  } else {
    for (int i = tid; i < n; i += K2_THREADS) buf0[i] = gk[i];
  }
  __syncthreads();

  // ---- stable LSD radix sort of nsel keys in shared memory ----
  KeyT* src = buf0;
  KeyT* dst = buf1;
  const int seg = ((nsel + K2_WARPS - 1) / K2_WARPS + 31) & ~31;    // per-warp contiguous segment
  const int w_begin = warp * seg < nsel ? warp * seg : nsel;
  const int w_end = (warp + 1) * seg < nsel ? (warp + 1) * seg : nsel;
  if (nsel > 1) {
    for (int shift = 0; shift < KB; shift += 8) {
      k2_zero_hist(hist, tid);
      if (tid == 0) misc->skip = 0;
      __syncthreads();
      for (int base = w_begin; base < w_end; base += 32) {
        const int i = base + lane;
        const bool v = i < w_end;
        const uint32_t dg = v ? (uint32_t)((src[i] >> shift) & 255) : 256u;
        const uint32_t peers = __match_any_sync(0xffffffffu, dg);
        if (v && lane == __ffs(peers) - 1) hist[warp * 256 + dg] += (uint16_t)__popc(peers);
        __syncwarp();
      }
      __syncthreads();
      if (tid < 256) {
        int s = 0;
#pragma unroll 8
        for (int w = 0; w < K2_WARPS; ++w) s += hist[w * 256 + tid];
        if (s == nsel) misc->skip = 1;                    // constant digit: nothing to reorder
      }
      __syncthreads();
      if (misc->skip) { __syncthreads(); continue; }
      k2_scan_hist(hist, misc, tid);
      __syncthreads();
      for (int base = w_begin; base < w_end; base += 32) {
        const int i = base + lane;
        const bool v = i < w_end;
        KeyT key = 0;
        if (v) key = src[i];
        const uint32_t dg = v ? (uint32_t)((key >> shift) & 255) : 256u;
        const uint32_t peers = __match_any_sync(0xffffffffu, dg);
        int b = 0;
        if (v) b = hist[warp * 256 + dg];
        __syncwarp();
        if (v && lane == __ffs(peers) - 1) hist[warp * 256 + dg] = (uint16_t)(b + __popc(peers));
        __syncwarp();
        if (v) dst[b + __popc(peers & ((1u << lane) - 1u))] = key;
      }
      __syncthreads();
      KeyT* t = src; src = dst; dst = t;
    }
  }

  // ---- epilogue: decode sorted rows (O1, O2), write rank-ordered arrays ----
  const int64_t obase = (int64_t)f * K;
  for (int r = tid; r < nsel; r += K2_THREADS) {
    const KeyT key = src[r];
    const int idx = (sizeof(KeyT) == 4) ? (int)((uint32_t)key & 0xFFFFu) : (int)(uint32_t)(key & 0xFFFFFFFFu);
    int l = 0;
    while (l + 1 < cst.num_levels && idx >= fd.lvl_start[l + 1]) ++l;
    const int k = idx - fd.lvl_start[l];
    const int gw = fd.lvl_gw[l];
    const int iy = k / gw, ix = k - iy * gw;
    const float s = (float)(1 << cst.stride_log2[l]);
    float v[5];
    const int64_t row = fd.cand_off + idx;
    if (kHalf) {
      const __half* p = reinterpret_cast<const __half*>(raw) + row * 5;
#pragma unroll
      for (int e = 0; e < 5; ++e) v[e] = __half2float(p[e]);
    } else {
      const float* p = reinterpret_cast<const float*>(raw) + row * 5;
#pragma unroll
      for (int e = 0; e < 5; ++e) v[e] = p[e];
    }
    const float px = __fmul_rn((float)ix + 0.5f, s), py = __fmul_rn((float)iy + 0.5f, s);
    float4 box;
    box.x = __fsub_rn(px, __fmul_rn(v[0], s));
    box.y = __fsub_rn(py, __fmul_rn(v[1], s));
    box.z = __fadd_rn(px, __fmul_rn(v[2], s));
    box.w = __fadd_rn(py, __fmul_rn(v[3], s));
    sorted_box[obase + r] = box;
    sorted_logit[obase + r] = v[4];
    sorted_idx[obase + r] = idx;
  }
  if (tid == 0) n_sorted[f] = nsel;
}

// =====================================================================================================
// a3 — NMS suppression bitmask (north_star (c)).
// bit (i, j), i < j in rank order, = IoU(box_i, box_j) > thr.  64x64 tiles: 64 threads own the 64 rows of a row
// block, the 64 column boxes sit in shared memory (broadcast reads).  A pair is first tested for strict overlap
// with four compares (no overlap => inter = 0 => IoU > thr is false for thr >= 0, so the bit is exactly 0);
// only overlapping pairs (~0.3 % on the flock workloads) evaluate the fp32 IoU of the definition, op by op
// (__f*_rn, no contraction).  Its comparison against thr uses a guard-banded multiply (inter vs thr*union with a
// 2^-20 relative band) that provably agrees with the correctly rounded division, which is evaluated only
// inside the band.  Work units pair row block p with row block nb-1-p so every unit has the same tile count.
// =====================================================================================================
constexpr int K3_THREADS = 64;
constexpr int K3_TILES_PER_UNIT = 16;

__device__ __forceinline__ float box_area(const float4 b) {
  return __fmul_rn(__fsub_rn(b.z, b.x), __fsub_rn(b.w, b.y));
}

__device__ __forceinline__ bool iou_exceeds(const float4 a, const float4 b, const Consts& c) {
  float iw = __fsub_rn(fminf(a.z, b.z), fmaxf(a.x, b.x));
  float ih = __fsub_rn(fminf(a.w, b.w), fmaxf(a.y, b.y));
  iw = fmaxf(0.0f, iw);
  ih = fmaxf(0.0f, ih);
  const float inter = __fmul_rn(iw, ih);
  const float uni = __fsub_rn(__fadd_rn(box_area(a), box_area(b)), inter);
  if (c.iou_fast && uni > 1e-30f && uni < 1e30f && inter < 1e30f) {
    if (inter > __fmul_rn(uni, c.iou_thr_hi)) return true;     // inter/uni > thr(1+2^-21): quotient rounds above thr
    if (inter < __fmul_rn(uni, c.iou_thr_lo)) return false;    // inter/uni < thr: quotient rounds to <= thr
  }
  return __fdiv_rn(inter, uni) > c.iou_thr;
}

__host__ __device__ inline int k3_units_per_pair(int nb) { return (nb + 1 + K3_TILES_PER_UNIT - 1) / K3_TILES_PER_UNIT; }
__host__ __device__ inline int k3_units(int nb) { return ((nb + 1) / 2) * k3_units_per_pair(nb); }

__global__ void __launch_bounds__(K3_THREADS) k3_nms_mask(const FrameDesc* __restrict__ frames,
                                                          const int* __restrict__ unit_prefix, int B,
                                                          const float4* __restrict__ sorted_box,
                                                          const int* __restrict__ n_sorted, Consts cst,
                                                          unsigned long long* __restrict__ mask) {
  __shared__ float4 cols[2][kNmsTile];
  const int t = threadIdx.x;
  // block -> (frame, unit)
  int lo = 0, hi = B;
  const int u_global = blockIdx.x;
  while (hi - lo > 1) { const int mid = (lo + hi) >> 1; if (unit_prefix[mid] <= u_global) lo = mid; else hi = mid; }
  const int f = lo;
  const int n = n_sorted[f];
  const int nb_act = (n + kNmsTile - 1) / kNmsTile;
  const int nb = frames[f].nbmax;
  const int u = u_global - unit_prefix[f];
  const int upp = k3_units_per_pair(nb);
  const int p = u / upp, c = u - p * upp;
  if (p >= nb_act && nb - 1 - p >= nb_act) return;
  const int64_t moff = frames[f].mask_off;
  const float4* boxes = sorted_box + (int64_t)f * cst.top_k;

  const int s_begin = c * K3_TILES_PER_UNIT;
  const int s_end = (s_begin + K3_TILES_PER_UNIT < nb + 1) ? s_begin + K3_TILES_PER_UNIT : nb + 1;
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
        if ((a.z > b.x) & (b.z > a.x) & (a.w > b.y) & (b.w > a.y)) {
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

// =====================================================================================================
// a4 — greedy sweep + output gather (north_star (c) second half).
// One CTA per frame.  For chunk q of 64 ranks: warp 0 resolves the chunk against `removed[q]` and the
// diagonal words with ffs-driven iterations (one per kept box, register shuffles), writes the kept boxes of
// the chunk to out_boxes in keep order; then all threads OR the row tails of the kept rows into `removed`.
// =====================================================================================================
constexpr int K4_THREADS = 256;

__global__ void __launch_bounds__(K4_THREADS) k4_nms_sweep(const FrameDesc* __restrict__ frames,
                                                           const float4* __restrict__ sorted_box,
                                                           const float* __restrict__ sorted_logit,
                                                           const int* __restrict__ sorted_idx,
                                                           const int* __restrict__ n_sorted, Consts cst,
                                                           const unsigned long long* __restrict__ mask,
                                                           ffpp_box* __restrict__ out_boxes,
                                                           int* __restrict__ out_counts) {
  extern __shared__ unsigned long long removed[];      // nbmax words
  __shared__ unsigned long long s_kept;
  const int f = blockIdx.x, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int n = n_sorted[f];
  const int nb_act = (n + kNmsTile - 1) / kNmsTile;
  const int nb = frames[f].nbmax;
  const unsigned long long* fm = mask + frames[f].mask_off;
  const int64_t ibase = (int64_t)f * cst.top_k;
  for (int i = tid; i < nb_act; i += K4_THREADS) removed[i] = 0ull;
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
      // gather the chunk's kept boxes to the output, in keep order
#pragma unroll
      for (int h = 0; h < 2; ++h) {
        const int b = lane + 32 * h;
        if ((kept >> b) & 1ull) {
          const int pos = kept_total + __popcll(kept & ((1ull << b) - 1ull));
          const int r = q * kNmsTile + b;
          const float4 bx = sorted_box[ibase + r];
          ffpp_box o;
          o.x1 = bx.x; o.y1 = bx.y; o.x2 = bx.z; o.y2 = bx.w;
          o.score = __fdiv_rn(1.0f, __fadd_rn(1.0f, expf(-sorted_logit[ibase + r])));
          o.cand_index = sorted_idx[ibase + r];
          out_boxes[ibase + pos] = o;
        }
      }
      kept_total += __popcll(kept);
    }
    __syncthreads();
    const unsigned long long km = s_kept;
    if (km) {
      for (int cb = q + 1 + tid; cb < nb_act; cb += K4_THREADS) {
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

// =====================================================================================================
// a5-a6 — density (north_star (d); the paper's grid-cell x bird loop,
// PAPER.md:L203-208, restated as histogram + separable convolution).
// One CTA per 64x16-cell output tile.  The tile's halo'd histogram is built in shared memory from the frame's
// kept boxes (integer atomics; the reflect border is realised by also binning each centroid's mirror images
// -c-1 and 2n-1-c, i.e. the half-sample symmetric extension), then convolved with the normalised taps along x
// into a second shared buffer and along y into the output.  HBM traffic: out_boxes of the frame (L2-resident)
// + one coalesced 4-byte store per cell.
// =====================================================================================================
constexpr int K5_THREADS = 256;
constexpr int K5_TW = 64, K5_TH = 16;

__global__ void __launch_bounds__(K5_THREADS) k5_density(const FrameDesc* __restrict__ frames,
                                                         const int* __restrict__ tile_prefix, int B,
                                                         const ffpp_box* __restrict__ out_boxes,
                                                         const int* __restrict__ out_counts, Consts cst,
                                                         float* __restrict__ out_density) {
  extern __shared__ __align__(16) uint8_t smem5[];
  const int R = cst.radius;
  const int HW = K5_TW + 2 * R, HH = K5_TH + 2 * R;
  int* hist = reinterpret_cast<int*>(smem5);                       // [HH][HW]
  float* rowc = reinterpret_cast<float*>(hist + HH * HW);          // [HH][K5_TW]
  const int tid = threadIdx.x;
  int lo = 0, hi = B;
  const int tg = blockIdx.x;
  while (hi - lo > 1) { const int mid = (lo + hi) >> 1; if (tile_prefix[mid] <= tg) lo = mid; else hi = mid; }
  const int f = lo;
  const FrameDesc* fd = &frames[f];
  const int gw = fd->gw, gh = fd->gh, W = fd->W, H = fd->H;
  const int tl = tg - tile_prefix[f];
  const int ty = tl / fd->tiles_x, tx = tl - ty * fd->tiles_x;
  const int ex0 = tx * K5_TW - R, ey0 = ty * K5_TH - R;             // extended-grid origin of the halo'd tile

  for (int i = tid; i < HH * HW; i += K5_THREADS) hist[i] = 0;
  __syncthreads();
  const int nk = out_counts[f];
  const ffpp_box* kb = out_boxes + (int64_t)f * cst.top_k;
  const float cell = (float)cst.cell_px, fW = (float)W, fH = (float)H;
  for (int i = tid; i < nk; i += K5_THREADS) {
    const ffpp_box b = kb[i];
    const float cx = __fmul_rn(__fadd_rn(b.x1, b.x2), 0.5f);
    const float cy = __fmul_rn(__fadd_rn(b.y1, b.y2), 0.5f);
    if (!(cx >= 0.0f && cx < fW && cy >= 0.0f && cy < fH)) continue;
    const int cxi = (int)floorf(__fdiv_rn(cx, cell));
    const int cyi = (int)floorf(__fdiv_rn(cy, cell));
    const int xs[3] = {cxi, -cxi - 1, 2 * gw - 1 - cxi};
    const int ys[3] = {cyi, -cyi - 1, 2 * gh - 1 - cyi};
#pragma unroll
    for (int yy = 0; yy < 3; ++yy) {
      const int ly = ys[yy] - ey0;
      if (ly < 0 || ly >= HH) continue;
#pragma unroll
      for (int xx = 0; xx < 3; ++xx) {
        const int lx = xs[xx] - ex0;
        if (lx < 0 || lx >= HW) continue;
        atomicAdd(&hist[ly * HW + lx], 1);
      }
    }
  }
  __syncthreads();
  // x pass: rowc[y][x] = sum_k w[k] * hist[y][x + k]
  for (int i = tid; i < HH * K5_TW; i += K5_THREADS) {
    const int y = i / K5_TW, x = i - y * K5_TW;
    const int* hrow = hist + y * HW + x;
    float acc = 0.0f;
    for (int k = 0; k <= 2 * R; ++k) acc = fmaf(cst.taps[k], (float)hrow[k], acc);
    rowc[i] = acc;
  }
  __syncthreads();
  // y pass + store
  float* out = out_density + fd->dens_off;
  for (int i = tid; i < K5_TH * K5_TW; i += K5_THREADS) {
    const int y = i / K5_TW, x = i - y * K5_TW;
    const int gx = tx * K5_TW + x, gy = ty * K5_TH + y;
    if (gx >= gw || gy >= gh) continue;
    float acc = 0.0f;
    for (int k = 0; k <= 2 * R; ++k) acc = fmaf(cst.taps[k], rowc[(y + k) * K5_TW + x], acc);
    out[(int64_t)gy * gw + gx] = acc;
  }
}

}  // namespace ffpp
