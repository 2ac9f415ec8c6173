// The five stage kernels of the CUDA path (sm_100a).  See DESIGN.md §"Kernels" for the roofline of each.
// Stage numbering follows SURVEY.md §8(a): a1 threshold+compaction, a2 sort+top-K(+decode, +spatial order),
// a3 NMS suppression words, a4 NMS resolve + output gather (+ a5 centroid histogram), a6 density convolution.
#pragma once
#include "ffpp_common.cuh"

namespace ffpp {

// =====================================================================================================
// a1 — threshold + compaction (BASELINE.json north_star (a); SURVEY §8(a) a1, §8(c) O1+O3).
// HBM-bound stream over the flat [sum N_f, 5] head output.  Warp-specialised: one producer warp drives the TMA
// engine (1-D cp.async.bulk, UBLKCP in SASS) through a 3-stage ring of 20 KB chunks guarded by full/empty
// mbarriers; eight consumer warps each own 1/8 of a chunk, look only at the score logit of each row, and compact
// with warp ballots: one global atomicAdd per (warp slice, frame) reserves the slice's slots in the frame's
// survivor list.  Survivors get a sort key
//   (descending-monotone score bits) ‖ (candidate index in frame)
// which makes every key of a frame unique, so slot order inside the list is irrelevant.  Boxes are NOT decoded
// here: only the <= top_k rows that survive the sort are decoded, in the a2 epilogue.
// There is no __syncthreads in the steady state; the frame offset table sits in shared memory.
// =====================================================================================================
constexpr int K1_CONSUMERS = 8;
constexpr int K1_THREADS = 32 * (K1_CONSUMERS + 1);
constexpr int K1_CHUNK_BYTES = 20480;   // multiple of lcm(16, 10, 20) = 80 and of 8 warps x 32 lanes rows
constexpr int K1_STAGES = 3;
constexpr int K1_CTAS_PER_SM = 3;        // 60 KB ring + 8 KB offsets per CTA
constexpr int K1_SMEM_FRAMES = 1024;    // frame offsets cached in shared memory (larger batches read them from L2)

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
  constexpr int CPW = CPC / K1_CONSUMERS;        // per consumer warp: 256 / 128
  constexpr int CPL = CPW / 32;                  // per lane: 8 / 4
  extern __shared__ __align__(128) uint8_t ring[];
  __shared__ __align__(8) uint64_t full[K1_STAGES], empty[K1_STAGES];
  __shared__ int64_t s_coff[K1_SMEM_FRAMES + 1];

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int64_t total_bytes = total_cand * ROW;
  const int64_t nchunks = (total_bytes + K1_CHUNK_BYTES - 1) / K1_CHUNK_BYTES;

  if (tid == 0) {
    for (int s = 0; s < K1_STAGES; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], K1_CONSUMERS); }
    mbar_fence_init();
  }
  const bool coff_in_smem = B <= K1_SMEM_FRAMES;
  if (coff_in_smem)
    for (int i = tid; i <= B; i += K1_THREADS) s_coff[i] = cand_off[i];
  __syncthreads();
  const int64_t* coff = coff_in_smem ? s_coff : cand_off;

  if (warp == K1_CONSUMERS) {
    // ---------------- producer warp ----------------
    int it = 0;
    for (int64_t c = blockIdx.x; c < nchunks; c += gridDim.x, ++it) {
      const int stage = it % K1_STAGES;
      if (it >= K1_STAGES) mbar_wait(&empty[stage], (uint32_t)(it / K1_STAGES - 1) & 1u);
      const int64_t b0 = c * K1_CHUNK_BYTES;
      int64_t len = total_bytes - b0;
      if (len > K1_CHUNK_BYTES) len = K1_CHUNK_BYTES;
      const uint32_t bulk = (uint32_t)(len & ~(int64_t)15);
      uint8_t* dst = ring + (size_t)stage * K1_CHUNK_BYTES;
      if ((uint32_t)len != bulk) {               // < 16 trailing bytes of the stream the bulk copy cannot carry
        if (lane < (int)len - (int)bulk) dst[bulk + lane] = raw[b0 + bulk + lane];
        __syncwarp();
      }
      if (lane == 0) {
        mbar_expect_tx(&full[stage], bulk);
        if (bulk) bulk_g2s(dst, raw + b0, bulk, &full[stage]);
      }
    }
    return;
  }

  // ---------------- consumer warps ----------------
  int it = 0;
  for (int64_t c = blockIdx.x; c < nchunks; c += gridDim.x, ++it) {
    const int stage = it % K1_STAGES;
    const uint8_t* buf = ring + (size_t)stage * K1_CHUNK_BYTES;
    const int64_t gw0 = c * CPC + (int64_t)warp * CPW;          // first candidate of this warp's slice
    int f0 = 0;
    if (gw0 < total_cand) {                                     // frame of gw0 (overlaps the copy)
      int lo = 0, hi = B;
      while (hi - lo > 1) { const int mid = (lo + hi) >> 1; if (coff[mid] <= gw0) lo = mid; else hi = mid; }
      f0 = lo;
    }
    mbar_wait(&full[stage], (uint32_t)(it / K1_STAGES) & 1u);
    if (gw0 < total_cand) {
      KeyT keys[CPL];
      int fr[CPL];
      uint32_t pass = 0;
      int fcur = f0;
      int64_t fend = coff[fcur + 1];
#pragma unroll
      for (int i = 0; i < CPL; ++i) {
        const int gl = warp * CPW + i * 32 + lane;
        const int64_t g = c * CPC + gl;
        fr[i] = -1;
        if (g < total_cand) {
          while (g >= fend) { ++fcur; fend = coff[fcur + 1]; }
          fr[i] = fcur;
          if (k1_eval<kHalf, KeyT>(buf, gl, T, (int)(g - coff[fcur]), keys[i])) pass |= 1u << i;
        }
      }
      const int flast = __reduce_max_sync(0xffffffffu, fcur);
      const uint32_t lt = (1u << lane) - 1u;
      for (int f = f0; f <= flast; ++f) {
        int off[CPL];
        int cnt = 0;
#pragma unroll
        for (int i = 0; i < CPL; ++i) {
          const uint32_t b = __ballot_sync(0xffffffffu, ((pass >> i) & 1u) && fr[i] == f);
          off[i] = cnt + __popc(b & lt);
          cnt += __popc(b);
        }
        if (cnt == 0) continue;
        int base = 0;
        if (lane == 0) base = atomicAdd(&surv_cnt[f], cnt);
        base = __shfl_sync(0xffffffffu, base, 0);
        KeyT* dst = surv_keys + coff[f] + base;
#pragma unroll
        for (int i = 0; i < CPL; ++i)
          if (((pass >> i) & 1u) && fr[i] == f) dst[off[i]] = keys[i];
      }
    }
    __syncwarp();
    if (lane == 0) mbar_arrive(&empty[stage]);
  }
}

// =====================================================================================================
// a2 — segmented per-frame sort + top-K + decode + spatial order (north_star (b)).
// One 1024-thread CTA per frame, everything after the first load in shared memory.
//  (1) the frame's survivor keys are staged in shared memory (read once, coalesced);
//  (2) if n > K, an MSD radix select (8-bit digits) finds the K-th smallest key — keys are unique, so exactly K
//      keys are <= it — and an ordered in-place compaction keeps them;
//  (3) a stable LSD block radix sort (8-bit digits, per-warp contiguous segments ranked with match_any, constant
//      digits skipped) puts them in (score desc, index asc) order;
//  (4) epilogue: decode the sorted rows from the raw head output (fp32, cell-centre grid point, no clipping) and
//      write boxes / logits / candidate indices in rank order;
//  (5) spatial order for the tiled NMS: each box gets the Hilbert index of its centre on a 256 x 256 grid, two more
//      LSD passes sort (hilbert ‖ rank), and the boxes, their ranks and one bounding box per 32 consecutive boxes
//      are written in that order.  The CTA also clears its frame's centroid histogram (a5).
// =====================================================================================================
constexpr int K2_THREADS = 1024;
constexpr int K2_WARPS = K2_THREADS / 32;

template <typename KeyT> struct KeyBits { static constexpr int value = sizeof(KeyT) * 8; };

// shared layout: KeyT keys[cap] | uint16 hist[32][256] | uint32 tot[256] | K2Misc
struct K2Misc {
  int wsum[2][K2_WARPS];
  int sel_digit, sel_kk, sel_tot, skip;
};

__host__ __device__ inline size_t k2_smem_bytes(size_t key_slots, size_t key_bytes) {
  return key_slots * key_bytes + K2_WARPS * 256 * sizeof(uint16_t) + 256 * sizeof(uint32_t) + sizeof(K2Misc) + 16;
}

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
  if (lane == 31) misc->wsum[0][warp] = inc;
  __syncthreads();
  if (warp == 0) {
    int x = misc->wsum[0][lane], xi = x;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { const int t = __shfl_up_sync(0xffffffffu, xi, o); if (lane >= o) xi += t; }
    misc->wsum[0][lane] = xi - x;
  }
  __syncthreads();
  int run = misc->wsum[0][warp] + inc - sum;
#pragma unroll
  for (int j = 0; j < 8; ++j) { hist[(w0 + j) * 256 + d] = (uint16_t)run; run += v[j]; }
}

// One stable LSD pass on the 8-bit digit at `shift`.  Returns true if the keys moved to dst (false: digit constant).
template <typename T>
__device__ __forceinline__ bool k2_lsd_pass(const T* src, T* dst, int n, int shift, uint16_t* hist, K2Misc* misc, int tid) {
  const int lane = tid & 31, warp = tid >> 5;
  const int seg = ((n + K2_WARPS - 1) / K2_WARPS + 31) & ~31;    // per-warp contiguous segment
  const int w_begin = warp * seg < n ? warp * seg : n;
  const int w_end = (warp + 1) * seg < n ? (warp + 1) * seg : n;
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
    if (s == n) misc->skip = 1;                    // constant digit: nothing to reorder
  }
  __syncthreads();
  if (misc->skip) { __syncthreads(); return false; }
  k2_scan_hist(hist, misc, tid);
  __syncthreads();
  for (int base = w_begin; base < w_end; base += 32) {
    const int i = base + lane;
    const bool v = i < w_end;
    T key = 0;
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
  return true;
}

// Hilbert index of cell (x, y) on a 256 x 256 grid (16 bits).  Any bijection would be correct; Hilbert order keeps 32
// consecutive boxes in a compact connected region, which is what makes the a3 tile culling effective.
__device__ __forceinline__ uint32_t hilbert16(uint32_t x, uint32_t y) {
  uint32_t d = 0;
#pragma unroll
  for (uint32_t s = 128; s > 0; s >>= 1) {
    const uint32_t rx = (x & s) ? 1u : 0u, ry = (y & s) ? 1u : 0u;
    d += s * s * ((3u * rx) ^ ry);
    if (ry == 0) {
      if (rx) { x = 255u - x; y = 255u - y; }
      const uint32_t t = x; x = y; y = t;
    }
  }
  return d;
}

template <bool kHalf, typename KeyT>
__global__ void __launch_bounds__(K2_THREADS, 1) k2_sort_topk_decode(
    const uint8_t* __restrict__ raw, const FrameDesc* __restrict__ frames, const KeyT* __restrict__ surv_keys,
    const int* __restrict__ surv_cnt, Consts cst, int key_slots, int nb32cap, float4* __restrict__ sorted_box,
    float* __restrict__ sorted_logit, int* __restrict__ sorted_idx, int* __restrict__ n_sorted,
    float4* __restrict__ sp_box, uint16_t* __restrict__ sp_rank, float4* __restrict__ bbox32,
    uint32_t* __restrict__ hist32, int spatial) {
  constexpr int KB = KeyBits<KeyT>::value;
  extern __shared__ __align__(16) uint8_t smem[];
  KeyT* keys = reinterpret_cast<KeyT*>(smem);
  uint16_t* hist = reinterpret_cast<uint16_t*>(keys + key_slots);
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

  // clear this frame's centroid histogram (uint16 per cell, two per word; boundary words are shared with the
  // neighbouring frames, which clear them too — every a2 CTA finishes before a4 counts)
  {
    const int64_t w0 = fd.dens_off >> 1, w1 = (fd.dens_off + (int64_t)fd.gw * fd.gh + 1) >> 1;
    for (int64_t i = w0 + tid; i < w1; i += K2_THREADS) hist32[i] = 0u;
  }

  // ---- (1) stage ----
  const bool staged = n <= key_slots;
  const KeyT* all = gk;
  if (staged) {
    for (int i = tid; i < n; i += K2_THREADS) keys[i] = gk[i];
    all = keys;
    __syncthreads();
  }

  if (n > K) {
    // ---- (2) MSD radix select: threshold key = K-th smallest ----
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
        if (i < n) { key = all[i]; m = (key & maskbits) == prefix; }
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
    // ordered compaction of the keys <= thr into keys[0, K).  When staged it is in place: element i lands at a
    // position <= i and every read of a 1024-chunk happens before the barrier that precedes its writes.
    int count = 0;
    int par = 0;
    for (int base = 0; base < n; base += K2_THREADS, par ^= 1) {
      const int i = base + tid;
      KeyT key = 0;
      bool m = false;
      if (i < n) { key = all[i]; m = key <= thr; }
      const uint32_t bal = __ballot_sync(0xffffffffu, m);
      if (lane == 0) misc->wsum[par][warp] = __popc(bal);
      __syncthreads();
      const int wv = misc->wsum[par][lane];
      int inc = wv;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) { const int t = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= o) inc += t; }
      const int before = __shfl_sync(0xffffffffu, inc - wv, warp);
      const int total = __shfl_sync(0xffffffffu, inc, 31);
      if (m) keys[count + before + __popc(bal & ((1u << lane) - 1u))] = key;
      count += total;
    }
    __syncthreads();
  } else if (!staged) {
    for (int i = tid; i < n; i += K2_THREADS) keys[i] = gk[i];
    __syncthreads();
  }

  // ---- (3) stable LSD radix sort of nsel keys in shared memory ----
  KeyT* src = keys;
  KeyT* dst = keys + K;
  if (nsel > 1) {
    for (int shift = 0; shift < KB; shift += 8)
      if (k2_lsd_pass<KeyT>(src, dst, nsel, shift, hist, misc, tid)) { KeyT* t = src; src = dst; dst = t; }
  }

  // ---- (4) epilogue: decode sorted rows (O1, O2), write rank-ordered arrays, build (hilbert ‖ rank) keys ----
  const int64_t obase = (int64_t)f * K;
  uint32_t* mk0 = reinterpret_cast<uint32_t*>(dst);
  uint32_t* mk1 = reinterpret_cast<uint32_t*>(src);
  const float cmax = (float)((256 << fd.hshift) - 1);
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
    const float cx = fminf(fmaxf(0.5f * (box.x + box.z), 0.0f), cmax);
    const float cy = fminf(fmaxf(0.5f * (box.y + box.w), 0.0f), cmax);
    const uint32_t hx = (uint32_t)((int)cx >> fd.hshift), hy = (uint32_t)((int)cy >> fd.hshift);
    mk0[r] = (hilbert16(hx, hy) << 16) | (uint32_t)r;
  }
  if (tid == 0) n_sorted[f] = nsel;
  __syncthreads();

  // ---- (5) spatial order ----
  if (!spatial) return;
  uint32_t* ms = mk0;
  uint32_t* md = mk1;
  if (nsel > 1) {
    for (int shift = 16; shift < 32; shift += 8)
      if (k2_lsd_pass<uint32_t>(ms, md, nsel, shift, hist, misc, tid)) { uint32_t* t = ms; ms = md; md = t; }
  }
  const float inf = __int_as_float(0x7f800000);
  for (int s0 = warp * 32; s0 < nsel; s0 += K2_THREADS) {
    const int s = s0 + lane;
    float4 bb = make_float4(inf, inf, -inf, -inf);
    if (s < nsel) {
      const int r = (int)(ms[s] & 0xFFFFu);
      const float4 box = sorted_box[obase + r];
      sp_box[obase + s] = box;
      sp_rank[obase + s] = (uint16_t)r;
      bb = box;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      bb.x = fminf(bb.x, __shfl_xor_sync(0xffffffffu, bb.x, o));
      bb.y = fminf(bb.y, __shfl_xor_sync(0xffffffffu, bb.y, o));
      bb.z = fmaxf(bb.z, __shfl_xor_sync(0xffffffffu, bb.z, o));
      bb.w = fmaxf(bb.w, __shfl_xor_sync(0xffffffffu, bb.w, o));
    }
    if (lane == 0) bbox32[(int64_t)f * nb32cap + (s0 >> 5)] = bb;
  }
}

// =====================================================================================================
// a3 — NMS suppression words, spatially tiled (north_star (c)).
// The bit "box b suppresses box a" = IoU(a, b) > thr and rank(b) < rank(a) is the same bit the rank-ordered matrix
// of the north_star sketch holds; what changes is which bits are looked at.  Boxes are in Hilbert order, 32 per block
// (= one warp of rows, one 32-bit word of columns).  A 32 x 32 tile (row block P, column block Q) is evaluated only
// if the blocks' bounding boxes overlap — otherwise every IoU in it is 0 and every bit is 0, exactly — and inside a
// tile a row is skipped unless its own box overlaps Q's bounding box.  Surviving pairs take the strict-overlap
// pre-test and then the fp32 IoU of the definition (iou_exceeds).  Each row appends its non-zero words to the row
// block's slot range (reserved from the frame's pool with one atomicAdd per CTA): word j of a row lives at
// W32[(slot_base[P] + j) * 32 + lane] with its column block in WQ, and nzc[row] counts them.
// One CTA = 8 warps = 8 row blocks of one frame; the frame's block bounding boxes are staged once per CTA.
// =====================================================================================================
constexpr int K3_WARPS = 8;
constexpr int K3_THREADS = 32 * K3_WARPS;
constexpr int K3_MAX_BLOCKS = 768;              // ceil(24576 / 32)

__global__ void __launch_bounds__(K3_THREADS) k3_nms_tiles(const FrameDesc* __restrict__ frames,
                                                           const int* __restrict__ n_sorted,
                                                           const float4* __restrict__ sp_box,
                                                           const uint16_t* __restrict__ sp_rank,
                                                           const float4* __restrict__ bbox32, Consts cst, int nb32cap,
                                                           int* __restrict__ slot_ctr, int* __restrict__ slot_base,
                                                           uint16_t* __restrict__ nzc, uint32_t* __restrict__ W32,
                                                           uint16_t* __restrict__ WQ, int* __restrict__ frame_err) {
  __shared__ float4 s_bb[K3_MAX_BLOCKS];
  __shared__ float4 s_col[K3_WARPS][kBlk];
  __shared__ uint16_t s_cr[K3_WARPS][kBlk];
  __shared__ int s_cnt[K3_WARPS];
  __shared__ int s_base;

  const int f = blockIdx.y;
  const int n = n_sorted[f];
  if ((int)blockIdx.x * K3_THREADS >= n) return;
  const int nb = (n + kBlk - 1) / kBlk;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int64_t obase = (int64_t)f * cst.top_k;
  const float4* fbb = bbox32 + (int64_t)f * nb32cap;
  for (int i = tid; i < nb; i += K3_THREADS) s_bb[i] = fbb[i];
  __syncthreads();

  const int P = blockIdx.x * K3_WARPS + warp;
  const bool active = P < nb;
  const int row = P * kBlk + lane;
  const bool valid = active && row < n;
  const float nanv = __int_as_float(0x7fc00000);
  float4 a = make_float4(nanv, nanv, nanv, nanv);
  uint32_t ra = 0;
  if (valid) { a = sp_box[obase + row]; ra = sp_rank[obase + row]; }
  const float4 bbP = active ? s_bb[P] : make_float4(nanv, nanv, nanv, nanv);

  // neighbour blocks: word i of the bitmap lives in lane i (nb <= 768 -> <= 24 words)
  uint32_t mybits = 0;
  int total = 0;
  const int nwords = (nb + 31) >> 5;
  for (int i = 0; i < nwords; ++i) {
    const int Q = i * 32 + lane;
    const bool ov = Q < nb && boxes_overlap(bbP, s_bb[Q]);
    const uint32_t b = __ballot_sync(0xffffffffu, ov);
    if (lane == i) mybits = b;
    total += __popc(b);
  }
  if (lane == 0) s_cnt[warp] = total;
  __syncthreads();
  if (tid == 0) {
    int sum = 0;
#pragma unroll
    for (int w = 0; w < K3_WARPS; ++w) sum += s_cnt[w];
    const int base = atomicAdd(&slot_ctr[f], sum);
    s_base = base;
    if (base + sum > frames[f].slot_cap) { frame_err[f] = 1; s_base = -1; }
  }
  __syncthreads();
  if (s_base < 0 || !active) return;       // pool exhausted (only when nms_workspace_bytes was set below worst case)
  int my_base = s_base;
  for (int w = 0; w < warp; ++w) my_base += s_cnt[w];
  const int64_t sb = frames[f].slot_off + my_base;
  if (lane == 0) slot_base[(int64_t)f * nb32cap + P] = (int)sb;

  int nz = 0;
  for (int i = 0; i < nwords; ++i) {
    uint32_t bits = __shfl_sync(0xffffffffu, mybits, i);
    while (bits) {
      const int Q = i * 32 + __ffs(bits) - 1;
      bits &= bits - 1;
      const int col = Q * kBlk + lane;
      float4 cb = make_float4(nanv, nanv, nanv, nanv);
      uint16_t cr = 0xFFFFu;
      if (col < n) { cb = sp_box[obase + col]; cr = sp_rank[obase + col]; }
      __syncwarp();
      s_col[warp][lane] = cb;
      s_cr[warp][lane] = cr;
      __syncwarp();
      uint32_t word = 0;
      if (boxes_overlap(a, s_bb[Q])) {
#pragma unroll 8
        for (int j = 0; j < kBlk; ++j) {
          const float4 b = s_col[warp][j];
          if (boxes_overlap(a, b)) {
            if ((uint32_t)s_cr[warp][j] < ra && iou_exceeds(a, b, cst)) word |= 1u << j;
          }
        }
      }
      if (word) {
        const int64_t at = (sb + nz) * kBlk + lane;
        W32[at] = word;
        WQ[at] = (uint16_t)Q;
        ++nz;
      }
    }
  }
  if (valid) nzc[obase + row] = (uint16_t)nz;
}

// =====================================================================================================
// a4 — greedy resolve + output gather + centroid histogram (north_star (c) second half; SURVEY §8(a) a4-a5,
// §8(c) O5-O7).  One CTA per frame.  Greedy NMS in rank order is the unique solution of
//     kept(a) <=> no b with rank(b) < rank(a), IoU(a,b) > thr is kept,
// so instead of walking the ranks one at a time the CTA iterates to the fixed point: a pending box whose every
// suppressor is known-removed becomes kept, one with a known-kept suppressor becomes removed.  The lowest-ranked
// pending box always resolves, so the loop ends, and the typical depth is a handful of rounds (the longest chain of
// overlapping boxes with decreasing score).  State is two bitmaps in shared memory (monotone, updated with atomicOr).
// Then the kept set is mapped back to rank order, prefix-summed, and written in keep order (= score order) with the
// sigmoid score and candidate index; each kept centroid is binned into the frame's histogram (a5).
// =====================================================================================================
constexpr int K4_THREADS = 1024;

__global__ void __launch_bounds__(K4_THREADS) k4_resolve_emit(
    const FrameDesc* __restrict__ frames, const int* __restrict__ n_sorted, const float4* __restrict__ sorted_box,
    const float* __restrict__ sorted_logit, const int* __restrict__ sorted_idx, const uint16_t* __restrict__ sp_rank,
    const uint16_t* __restrict__ nzc, const int* __restrict__ slot_base, const uint32_t* __restrict__ W32,
    const uint16_t* __restrict__ WQ, const int* __restrict__ frame_err, Consts cst, int nb32cap,
    ffpp_box* __restrict__ out_boxes, int* __restrict__ out_counts, uint32_t* __restrict__ hist32) {
  __shared__ uint32_t kept[K3_MAX_BLOCKS], removed[K3_MAX_BLOCKS], keptR[K3_MAX_BLOCKS], pref[K3_MAX_BLOCKS];
  __shared__ int s_slot[K3_MAX_BLOCKS];
  __shared__ int wsum[32];
  __shared__ FrameDesc fd;
  const int f = blockIdx.x, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  if (frame_err[f]) { if (tid == 0) out_counts[f] = -1; return; }
  if (tid == 0) fd = frames[f];
  const int n = n_sorted[f];
  const int nb = (n + kBlk - 1) / kBlk;
  const int64_t obase = (int64_t)f * cst.top_k;
  for (int i = tid; i < nb; i += K4_THREADS) {
    kept[i] = 0u; removed[i] = 0u; keptR[i] = 0u;
    s_slot[i] = slot_base[(int64_t)f * nb32cap + i];
  }
  __syncthreads();

  const uint32_t bit = 1u << lane;
  uint32_t pending = 0;
  for (int i = 0, a = tid; a < n; ++i, a += K4_THREADS) {
    if (nzc[obase + a] == 0) atomicOr(&kept[a >> 5], bit);
    else pending |= 1u << i;
  }
  __syncthreads();
  while (true) {
    uint32_t m = pending;
    while (m) {
      const int i = __ffs(m) - 1;
      m &= m - 1;
      const int a = tid + i * K4_THREADS;
      const int P = a >> 5;
      const int c = nzc[obase + a];
      const int64_t at = (int64_t)s_slot[P] * kBlk + lane;
      int state = 0;                                   // 0 keep, 1 still pending, 2 remove
      for (int j = 0; j < c; ++j) {
        const uint32_t w = W32[at + (int64_t)j * kBlk];
        const int Q = WQ[at + (int64_t)j * kBlk];
        const uint32_t kq = *(volatile uint32_t*)&kept[Q];
        const uint32_t rq = *(volatile uint32_t*)&removed[Q];
        if (w & kq) { state = 2; break; }
        if (w & ~rq) state = 1;
      }
      if (state == 2) { atomicOr(&removed[P], bit); pending &= ~(1u << i); }
      else if (state == 0) { atomicOr(&kept[P], bit); pending &= ~(1u << i); }
    }
    if (!__syncthreads_or(pending != 0)) break;
  }

  // kept set -> rank order
  for (int a = tid; a < n; a += K4_THREADS)
    if (kept[a >> 5] & bit) {
      const uint32_t r = sp_rank[obase + a];
      atomicOr(&keptR[r >> 5], 1u << (r & 31));
    }
  __syncthreads();
  {
    const int c = tid < nb ? __popc(keptR[tid]) : 0;
    int inc = c;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { const int t = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= o) inc += t; }
    if (lane == 31) wsum[warp] = inc;
    __syncthreads();
    if (warp == 0) {
      const int x = wsum[lane];
      int xi = x;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) { const int t = __shfl_up_sync(0xffffffffu, xi, o); if (lane >= o) xi += t; }
      wsum[lane] = xi - x;
      if (lane == 31) out_counts[f] = xi;
    }
    __syncthreads();
    if (tid < nb) pref[tid] = (uint32_t)(wsum[warp] + inc - c);
  }
  __syncthreads();
  for (int r = tid; r < n; r += K4_THREADS) {
    const uint32_t wd = keptR[r >> 5];
    if (wd & bit) {
      const int pos = (int)pref[r >> 5] + __popc(wd & (bit - 1u));
      emit_kept(fd, cst, out_boxes + obase + pos, sorted_box[obase + r], sorted_logit[obase + r], sorted_idx[obase + r], hist32);
    }
  }
}

// =====================================================================================================
// a6 — density convolution (north_star (d); the paper's grid-cell x bird loop,
// PAPER.md:L203-208, restated as histogram + separable convolution).
// One CTA per 64 x 32-cell output tile.  The tile's halo'd histogram is read through the reflect fold
// (fold(i,n) = -i-1 | 2n-1-i, the half-sample symmetric extension) into shared memory as floats, convolved with the
// normalised taps along x into a second shared buffer and along y into the output, both passes register-blocked
// (8 outputs per thread slide over an 8-wide window, one shared load per tap).  HBM traffic: 2 bytes per cell of
// histogram (L2-resident: written by a2/a4 microseconds earlier) + one coalesced 4-byte store per cell.
// =====================================================================================================
constexpr int K5_THREADS = 256;
constexpr int K5_TW = 64, K5_TH = 32;

__host__ __device__ inline int k5_hs_stride(int R) { return (K5_TW + 2 * R) | 1; }          // odd: conflict-free column walks
__host__ __device__ inline size_t k5_smem_bytes(int R) {
  return sizeof(float) * ((size_t)(K5_TH + 2 * R) * k5_hs_stride(R) + 8 + (size_t)(K5_TH + 2 * R) * (K5_TW + 1));
}

__global__ void __launch_bounds__(K5_THREADS) k5_density(const FrameDesc* __restrict__ frames, Consts cst,
                                                         const uint16_t* __restrict__ hist16,
                                                         float* __restrict__ out_density) {
  extern __shared__ __align__(16) float smem5[];
  const int f = blockIdx.y;
  const FrameDesc* fd = &frames[f];
  const int gw = fd->gw, gh = fd->gh;
  const int tiles_x = (gw + K5_TW - 1) / K5_TW, tiles_y = (gh + K5_TH - 1) / K5_TH;
  if ((int)blockIdx.x >= tiles_x * tiles_y) return;
  const int ty = blockIdx.x / tiles_x, tx = blockIdx.x - ty * tiles_x;
  const int R = cst.radius;
  const int HW = K5_TW + 2 * R, HH = K5_TH + 2 * R, HS = k5_hs_stride(R), RS = K5_TW + 1;
  float* hs = smem5;                       // [HH][HS] (+8 floats of slack for the sliding window's last loads)
  float* rowc = smem5 + (size_t)HH * HS + 8;   // [HH][RS]
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const uint16_t* hsrc = hist16 + fd->dens_off;
  const int ex0 = tx * K5_TW - R, ey0 = ty * K5_TH - R;

  for (int i = tid; i < HH * HW; i += K5_THREADS) {
    const int ly = i / HW, lx = i - ly * HW;
    int gy = ey0 + ly, gx = ex0 + lx;
    gy = gy < 0 ? -gy - 1 : (gy >= gh ? 2 * gh - 1 - gy : gy);
    gx = gx < 0 ? -gx - 1 : (gx >= gw ? 2 * gw - 1 - gx : gx);
    float v = 0.0f;
    if (gy >= 0 && gx >= 0) v = (float)hsrc[(int64_t)gy * gw + gx];   // < 0: overhang beyond the folded range, unused
    hs[ly * HS + lx] = v;
  }
  if (tid < 8) hs[(size_t)HH * HS + tid] = 0.0f;
  __syncthreads();

  // x pass: rowc[y][x] = sum_k w[k] * hs[y][x + k].  lane -> row, 8 consecutive x per thread.
  for (int y0 = 0; y0 < HH; y0 += 32) {
    const int y = y0 + lane;
    if (y < HH) {
      const float* hrow = hs + y * HS + warp * 8;
      float win[8], acc[8];
#pragma unroll
      for (int m = 0; m < 8; ++m) { win[m] = hrow[m]; acc[m] = 0.0f; }
#pragma unroll 8
      for (int k = 0; k <= 2 * R; ++k) {
        const float t = cst.taps[k];
#pragma unroll
        for (int m = 0; m < 8; ++m) acc[m] = fmaf(t, win[m], acc[m]);
#pragma unroll
        for (int m = 0; m < 7; ++m) win[m] = win[m + 1];
        win[7] = hrow[k + 8];
      }
#pragma unroll
      for (int m = 0; m < 8; ++m) rowc[y * RS + warp * 8 + m] = acc[m];
    }
  }
  __syncthreads();

  // y pass + store: thread -> column x, 8 consecutive rows.
  {
    const int x = tid & 63, yg = tid >> 6;                 // 4 groups x 8 rows = 32
    const float* col = rowc + (yg * 8) * RS + x;
    float win[8], acc[8];
#pragma unroll
    for (int m = 0; m < 8; ++m) { win[m] = col[m * RS]; acc[m] = 0.0f; }
#pragma unroll 8
    for (int k = 0; k <= 2 * R; ++k) {
      const float t = cst.taps[k];
#pragma unroll
      for (int m = 0; m < 8; ++m) acc[m] = fmaf(t, win[m], acc[m]);
#pragma unroll
      for (int m = 0; m < 7; ++m) win[m] = win[m + 1];
      const int yy = yg * 8 + k + 8;
      win[7] = yy < HH ? col[(k + 8) * RS] : 0.0f;
    }
    const int gx = tx * K5_TW + x;
    float* out = out_density + fd->dens_off;
    if (gx < gw) {
#pragma unroll
      for (int m = 0; m < 8; ++m) {
        const int gy = ty * K5_TH + yg * 8 + m;
        if (gy < gh) out[(int64_t)gy * gw + gx] = acc[m];
      }
    }
  }
}

}  // namespace ffpp
