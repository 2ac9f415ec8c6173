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
// Block-wide (1024-thread) helpers shared by a2 and a4: exclusive scans and a stable 8-bit LSD radix pass.
// =====================================================================================================
constexpr int BLK_THREADS = 1024;
constexpr int BLK_WARPS = BLK_THREADS / 32;

struct BlkMisc {
  int wsum[2][BLK_WARPS];
  int sel_digit, sel_kk, sel_tot, skip;
  int counter;
};

// inclusive scan of one int per thread over the CTA; returns the inclusive value, *total = sum over the CTA.
// Two barriers; wsum row `par` is scratch (alternate rows between back-to-back calls).
__device__ __forceinline__ int blk_scan_inclusive(int v, BlkMisc* misc, int par, int tid, int* total) {
  const int lane = tid & 31, warp = tid >> 5;
  int inc = v;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) { const int t = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= o) inc += t; }
  if (lane == 31) misc->wsum[par][warp] = inc;
  __syncthreads();
  const int wv = misc->wsum[par][lane];
  int winc = wv;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) { const int t = __shfl_up_sync(0xffffffffu, winc, o); if (lane >= o) winc += t; }
  const int before = __shfl_sync(0xffffffffu, winc - wv, warp);
  *total = __shfl_sync(0xffffffffu, winc, 31);
  __syncthreads();
  return before + inc;
}

__device__ __forceinline__ void blk_zero_hist(uint16_t* hist, int tid) {
  uint32_t* h32 = reinterpret_cast<uint32_t*>(hist);
  for (int i = tid; i < BLK_WARPS * 256 / 2; i += BLK_THREADS) h32[i] = 0;
}

// exclusive scan of the per-warp digit histogram hist[warp][digit] in (digit major, warp minor) order, in place.
__device__ __forceinline__ void blk_scan_hist(uint16_t* hist, BlkMisc* misc, int tid) {
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

// One stable LSD pass on the 8-bit digit at `shift` (per-warp contiguous segments ranked with match_any).
// Returns true if the keys moved to dst (false: the digit is constant, nothing to reorder).
template <typename T>
__device__ __forceinline__ bool blk_lsd_pass(const T* src, T* dst, int n, int shift, uint16_t* hist, BlkMisc* misc, int tid) {
  const int lane = tid & 31, warp = tid >> 5;
  const int seg = ((n + BLK_WARPS - 1) / BLK_WARPS + 31) & ~31;    // per-warp contiguous segment
  const int w_begin = warp * seg < n ? warp * seg : n;
  const int w_end = (warp + 1) * seg < n ? (warp + 1) * seg : n;
  uint32_t* hist32 = reinterpret_cast<uint32_t*>(hist);
  blk_zero_hist(hist, tid);
  if (tid == 0) misc->skip = 0;
  __syncthreads();
  for (int base = w_begin; base < w_end; base += 32) {
    const int i = base + lane;
    const bool v = i < w_end;
    const uint32_t dg = v ? (uint32_t)((src[i] >> shift) & 255) : 256u;
    const uint32_t peers = __match_any_sync(0xffffffffu, dg);
    // two uint16 counters per word; fire-and-forget shared atomics, no carry (a warp segment has < 65536 keys)
    if (v && lane == __ffs(peers) - 1) atomicAdd(&hist32[(warp * 256 + dg) >> 1], (uint32_t)__popc(peers) << (16 * (dg & 1)));
  }
  __syncthreads();
  if (tid < 256) {
    int s = 0;
#pragma unroll 8
    for (int w = 0; w < BLK_WARPS; ++w) s += hist[w * 256 + tid];
    if (s == n) misc->skip = 1;
  }
  __syncthreads();
  if (misc->skip) { __syncthreads(); return false; }
  blk_scan_hist(hist, misc, tid);
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

// Hilbert index of cell (x, y) on a 128 x 128 grid (14 bits).  Any bijection would be correct; Hilbert order keeps
// consecutive boxes in a compact connected region, which is what makes the a3 block culling effective.
__device__ __forceinline__ uint32_t hilbert14(uint32_t x, uint32_t y) {
  uint32_t d = 0;
#pragma unroll
  for (uint32_t s = 64; s > 0; s >>= 1) {
    const uint32_t rx = (x & s) ? 1u : 0u, ry = (y & s) ? 1u : 0u;
    d += s * s * ((3u * rx) ^ ry);
    if (ry == 0) {
      if (rx) { x = 127u - x; y = 127u - y; }
      const uint32_t t = x; x = y; y = t;
    }
  }
  return d;
}

// =====================================================================================================
// a2 — per-frame top-K selection + decode + spatial binning (north_star (b)).
// The total order of O4 is carried by the survivor keys (descending-monotone score bits ‖ candidate index), which are
// unique, so "the first min(n, K) of the order" is exactly the set of keys <= the K-th smallest key.  One 1024-thread
// CTA per frame:
//  (1) MSD radix select on 12-bit digits (3 count sweeps for 32-bit keys, early exit when a whole bucket is taken):
//      CTA-wide counters in shared memory, warp-aggregated (match_any) fire-and-forget shared atomics, keys read
//      straight from the L2-resident survivor list;
//  (2) one sweep appends the keys <= threshold to shared memory (order is irrelevant from here on);
//  (3) decode the selected rows from the raw head output (fp32, cell-centre grid point, no clipping; O1, O2) and bin
//      each box by the Hilbert index of its centre on a 128 x 128 grid with one shared atomic (counting sort);
//  (4) scan the 16384 bins, scatter box / culling box / key to the frame's spatial arrays, and write the bounding
//      box of the culling boxes of every 8 and every 32 consecutive entries.
// The (score desc, index asc) ORDER itself is applied where it is consumed: as key comparisons in a3/a4 (greedy NMS
// only ever asks "which of two boxes comes first") and as a radix sort of the kept keys in a4, which is ~8x fewer
// keys than sorting all top-K entries here.  The CTA also clears its frame's centroid histogram (a5).
// =====================================================================================================
constexpr int K2_THREADS = BLK_THREADS;
constexpr int K2_SEL_BITS = 12;
constexpr int K2_HBINS = 128 * 128;
constexpr int K2_CNT_WORDS = K2_HBINS / 2;     // 32 KB: 4096 select counters (uint32) or 16384 Hilbert counters (uint16)

__host__ __device__ inline size_t k2_smem_bytes(size_t top_k, size_t key_bytes) {
  return top_k * key_bytes + top_k * sizeof(uint32_t) + K2_CNT_WORDS * sizeof(uint32_t) + sizeof(BlkMisc) + 16;
}

template <bool kHalf, typename KeyT>
__global__ void __launch_bounds__(K2_THREADS, 1) k2_select_bin(
    const uint8_t* __restrict__ raw, const FrameDesc* __restrict__ frames, const KeyT* __restrict__ surv_keys,
    const int* __restrict__ surv_cnt, Consts cst, int nb8cap, int nb32cap, float4* __restrict__ sel_box,
    float4* __restrict__ sp_box, float4* __restrict__ sp_sbox, KeyT* __restrict__ sp_key, float4* __restrict__ bbox8,
    float4* __restrict__ bbox32, int* __restrict__ n_sorted, uint32_t* __restrict__ hist32) {
  constexpr int KB = sizeof(KeyT) * 8;
  extern __shared__ __align__(16) uint8_t smem[];
  const int K = cst.top_k;
  KeyT* sel = reinterpret_cast<KeyT*>(smem);
  uint32_t* aux = reinterpret_cast<uint32_t*>(sel + K);
  uint32_t* cnt = aux + K;
  BlkMisc* misc = reinterpret_cast<BlkMisc*>(cnt + K2_CNT_WORDS);
  __shared__ FrameDesc fd;

  const int f = blockIdx.x, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  if (tid == 0) { fd = frames[f]; misc->counter = 0; }
  __syncthreads();
  const int n = surv_cnt[f];
  const int nsel = n < K ? n : K;
  const KeyT* gk = surv_keys + fd.cand_off;

  // clear this frame's centroid histogram (uint16 per cell, two per word; boundary words are shared with the
  // neighbouring frames, which clear them too — every a2 CTA finishes before a4 counts)
  {
    const int64_t w0 = fd.dens_off >> 1, w1 = (fd.dens_off + (int64_t)fd.gw * fd.gh + 1) >> 1;
    for (int64_t i = w0 + tid; i < w1; i += K2_THREADS) hist32[i] = 0u;
  }

  // ---- (1) threshold key = K-th smallest ----
  KeyT thr = ~(KeyT)0;
  if (n > K) {
    KeyT prefix = 0, maskbits = 0;
    int kk = K;
    bool done = false;
    for (int hi = KB; hi > 0 && !done;) {
      const int shift = hi > K2_SEL_BITS ? hi - K2_SEL_BITS : 0;
      const uint32_t dmask = (1u << (hi - shift)) - 1u;
      for (int i = tid; i < (1 << K2_SEL_BITS); i += K2_THREADS) cnt[i] = 0u;
      __syncthreads();
      for (int base = warp * 32; base < n; base += 4 * K2_THREADS) {
        KeyT key[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) { const int i = base + u * K2_THREADS + lane; key[u] = i < n ? gk[i] : ~(KeyT)0; }
#pragma unroll
        for (int u = 0; u < 4; ++u) {
          if (base + u * K2_THREADS < n) {                      // warp-uniform
            const int i = base + u * K2_THREADS + lane;
            const bool m = i < n && (key[u] & maskbits) == prefix;
            const uint32_t dg = m ? (uint32_t)((key[u] >> shift) & dmask) : 0xFFFFFFFFu;
            const uint32_t peers = __match_any_sync(0xffffffffu, dg);
            if (m && lane == __ffs(peers) - 1) atomicAdd(&cnt[dg], (uint32_t)__popc(peers));
          }
        }
      }
      __syncthreads();
      {
        uint32_t v[4];
        int s = 0;
#pragma unroll
        for (int j = 0; j < 4; ++j) { v[j] = cnt[tid * 4 + j]; s += (int)v[j]; }
        int total;
        const int inc = blk_scan_inclusive(s, misc, 0, tid, &total);
        int run = inc - s;                                       // keys in bins below this thread's first bin
        if (run < kk && kk <= inc) {
#pragma unroll
          for (int j = 0; j < 4; ++j) {
            if (run < kk && kk <= run + (int)v[j]) { misc->sel_digit = tid * 4 + j; misc->sel_kk = kk - run; misc->sel_tot = (int)v[j]; }
            run += (int)v[j];
          }
        }
      }
      __syncthreads();
      prefix |= (KeyT)misc->sel_digit << shift;
      maskbits |= (KeyT)dmask << shift;
      kk = misc->sel_kk;
      if (misc->sel_tot == kk) {                                 // the whole bucket is selected
        thr = prefix | (shift ? (((KeyT)1 << shift) - 1) : (KeyT)0);
        done = true;
      }
      hi = shift;
      __syncthreads();
    }
    if (!done) thr = prefix;
  }

  // ---- (2) gather the selected keys into shared memory ----
  for (int base = warp * 32; base < n; base += K2_THREADS) {
    const int i = base + lane;
    KeyT key = 0;
    bool m = false;
    if (i < n) { key = gk[i]; m = key <= thr; }
    const uint32_t bal = __ballot_sync(0xffffffffu, m);
    int at = 0;
    if (lane == 0 && bal) at = atomicAdd(&misc->counter, __popc(bal));
    at = __shfl_sync(0xffffffffu, at, 0);
    if (m) sel[at + __popc(bal & ((1u << lane) - 1u))] = key;
  }
  for (int i = tid; i < K2_CNT_WORDS; i += K2_THREADS) cnt[i] = 0u;
  __syncthreads();

  // ---- (3) decode (O1, O2) + Hilbert bin ----
  const int64_t obase = (int64_t)f * cst.kpad;
  const float cmax = (float)((128 << fd.hshift) - 1);
  for (int i = tid; i < nsel; i += K2_THREADS) {
    const KeyT key = sel[i];
    const int idx = idx_of_key<KeyT>(key);
    int l = 0;
    while (l + 1 < cst.num_levels && idx >= fd.lvl_start[l + 1]) ++l;
    const int k = idx - fd.lvl_start[l];
    const int gw = fd.lvl_gw[l];
    const int iy = k / gw, ix = k - iy * gw;
    const float s = (float)(1 << cst.stride_log2[l]);
    float v[4];
    const int64_t row = fd.cand_off + idx;
    if (kHalf) {
      const __half* p = reinterpret_cast<const __half*>(raw) + row * 5;
#pragma unroll
      for (int e = 0; e < 4; ++e) v[e] = __half2float(p[e]);
    } else {
      const float* p = reinterpret_cast<const float*>(raw) + row * 5;
#pragma unroll
      for (int e = 0; e < 4; ++e) v[e] = p[e];
    }
    const float px = __fmul_rn((float)ix + 0.5f, s), py = __fmul_rn((float)iy + 0.5f, s);
    float4 box;
    box.x = __fsub_rn(px, __fmul_rn(v[0], s));
    box.y = __fsub_rn(py, __fmul_rn(v[1], s));
    box.z = __fadd_rn(px, __fmul_rn(v[2], s));
    box.w = __fadd_rn(py, __fmul_rn(v[3], s));
    sel_box[obase + i] = box;
    const float cx = fminf(fmaxf(0.5f * (box.x + box.z), 0.0f), cmax);   // NaN -> 0
    const float cy = fminf(fmaxf(0.5f * (box.y + box.w), 0.0f), cmax);
    const uint32_t h = hilbert14((uint32_t)((int)cx >> fd.hshift), (uint32_t)((int)cy >> fd.hshift));
    const uint32_t sh = 16u * (h & 1u);
    const uint32_t old = atomicAdd(&cnt[h >> 1], 1u << sh);
    aux[i] = (h << 16) | ((old >> sh) & 0xFFFFu);
  }
  __syncthreads();

  // ---- (4) exclusive scan of the bins (16 per thread), scatter to spatial order ----
  {
    uint32_t w[8];
    int s = 0;
#pragma unroll
    for (int j = 0; j < 8; ++j) { w[j] = cnt[tid * 8 + j]; s += (int)(w[j] & 0xFFFFu) + (int)(w[j] >> 16); }
    int total;
    const int inc = blk_scan_inclusive(s, misc, 1, tid, &total);
    int run = inc - s;
#pragma unroll
    for (int j = 0; j < 8; ++j) {
      const int c0 = (int)(w[j] & 0xFFFFu), c1 = (int)(w[j] >> 16);
      cnt[tid * 8 + j] = (uint32_t)run | ((uint32_t)(run + c0) << 16);
      run += c0 + c1;
    }
  }
  __syncthreads();
  const uint16_t* base16 = reinterpret_cast<const uint16_t*>(cnt);
  for (int i = tid; i < nsel; i += K2_THREADS) {
    const uint32_t a = aux[i];
    const int pos = (int)base16[a >> 16] + (int)(a & 0xFFFFu);
    const float4 box = sel_box[obase + i];
    sp_box[obase + pos] = box;
    sp_sbox[obase + pos] = shrink_box(box, cst.shrink);
    sp_key[obase + pos] = sel[i];
  }
  const float inf = __int_as_float(0x7f800000);
  const int npad = (nsel + kBlk - 1) & ~(kBlk - 1);
  for (int i = nsel + tid; i < npad; i += K2_THREADS) {           // padding of the last block: never overlaps, never first
    sp_sbox[obase + i] = make_float4(inf, inf, -inf, -inf);
    sp_key[obase + i] = ~(KeyT)0;
  }
  if (tid == 0) n_sorted[f] = nsel;
  __syncthreads();

  // ---- bounding boxes of the culling boxes per 8 and per 32 entries ----
  for (int s0 = warp * 32; s0 < nsel; s0 += K2_THREADS) {
    float4 bb = sp_sbox[obase + s0 + lane];                        // padding entries are empty boxes
#pragma unroll
    for (int o = 1; o < 8; o <<= 1) {
      bb.x = fminf(bb.x, __shfl_xor_sync(0xffffffffu, bb.x, o));
      bb.y = fminf(bb.y, __shfl_xor_sync(0xffffffffu, bb.y, o));
      bb.z = fmaxf(bb.z, __shfl_xor_sync(0xffffffffu, bb.z, o));
      bb.w = fmaxf(bb.w, __shfl_xor_sync(0xffffffffu, bb.w, o));
    }
    if ((lane & 7) == 0) bbox8[(int64_t)f * nb8cap + (s0 >> 3) + (lane >> 3)] = bb;
#pragma unroll
    for (int o = 8; o < 32; o <<= 1) {
      bb.x = fminf(bb.x, __shfl_xor_sync(0xffffffffu, bb.x, o));
      bb.y = fminf(bb.y, __shfl_xor_sync(0xffffffffu, bb.y, o));
      bb.z = fmaxf(bb.z, __shfl_xor_sync(0xffffffffu, bb.z, o));
      bb.w = fmaxf(bb.w, __shfl_xor_sync(0xffffffffu, bb.w, o));
    }
    if (lane == 0) bbox32[(int64_t)f * nb32cap + (s0 >> 5)] = bb;
  }
}

// =====================================================================================================
// a3 — NMS suppression edges, spatially tiled (north_star (c)).
// The bit "box b suppresses box a" = IoU(a, b) > thr and b before a in the order of O4 is the same bit the
// rank-ordered matrix of the north_star sketch holds; what changes is which bits are ever looked at.  Boxes are in
// Hilbert order.  One warp owns a block of 32 consecutive rows (lane = row); columns are visited in sub-blocks of 8.
//  (1) block culling: the 32-row block's culling bounding box against every 32-block of the frame (ballots over the
//      bounding boxes staged in shared memory), then each of its four 8-row groups against the four 8-column
//      sub-blocks of every hit; all on culling boxes (boxes shrunk by ~thr/2 per side, see shrink_box), so a pair
//      that is skipped provably has IoU <= thr.  Each group collects its own list of 8-column tiles.
//  (2) pretest: the four groups walk their tile lists in lock step; a row tests its culling box against the tile's
//      8 culling boxes and the order (key(b) < key(a)); 5 + 1 instructions per pair, no divergence.
//  (3) the surviving (row, column) candidates are compacted into a per-warp queue and evaluated 32 at a time, one
//      pair per lane, with the fp32 IoU of the definition (iou_exceeds) — full lanes on the expensive part.
//  (4) hits are appended to the frame's edge pool as (row << 16 | column), spatial positions, via one atomicAdd per
//      flush of the warp's staging buffer.
// One CTA = 8 warps = 8 row blocks of one frame.
// =====================================================================================================
constexpr int K3_WARPS = 8;
constexpr int K3_THREADS = 32 * K3_WARPS;
constexpr int K3_MAX_B32 = kMaxTopK / kBlk;     // 768
constexpr int K3_TCAP = 32;                     // tile-list entries per 8-row group
constexpr int K3_QCAP = 320;                    // candidate queue: <= 31 left over + <= 256 pushed per step
constexpr int K3_SCAP = 96;                     // edge staging per warp

struct K3Warp {
  float4 rowbox[kBlk];
  uint32_t q[K3_QCAP];
  uint32_t sb[K3_SCAP];
  uint16_t tl[4][K3_TCAP];
};

struct K3State {                                 // warp-uniform bookkeeping
  int qcnt, scnt;
};

__device__ __forceinline__ void k3_flush(K3Warp& W, K3State& st, const FrameDesc& fd, int f, int lane,
                                         int* __restrict__ edge_ctr, uint32_t* __restrict__ edges,
                                         int* __restrict__ frame_err) {
  if (st.scnt == 0) return;
  int base = 0;
  if (lane == 0) base = atomicAdd(&edge_ctr[f], st.scnt);
  base = __shfl_sync(0xffffffffu, base, 0);
  if (base + st.scnt <= fd.edge_cap) {
    for (int k = lane; k < st.scnt; k += 32) edges[fd.edge_off + base + k] = W.sb[k];
  } else if (lane == 0) {
    frame_err[f] = 1;                            // pool exhausted (only when nms_workspace_bytes was set too low)
  }
  st.scnt = 0;
  __syncwarp();
}

// evaluate `nb` (<= 32) queued candidates, one per lane, from the top of the queue
__device__ __forceinline__ void k3_exact_batch(K3Warp& W, K3State& st, int nb, const float4* __restrict__ fbox, int row0,
                                               const Consts& cst, const FrameDesc& fd, int f, int lane,
                                               int* __restrict__ edge_ctr, uint32_t* __restrict__ edges,
                                               int* __restrict__ frame_err) {
  bool hit = false;
  uint32_t e = 0;
  if (lane < nb) {
    e = W.q[st.qcnt - nb + lane];
    const float4 a = W.rowbox[e >> 16];
    const float4 b = fbox[e & 0xFFFFu];
    hit = iou_exceeds(a, b, cst);
  }
  const uint32_t bal = __ballot_sync(0xffffffffu, hit);
  if (hit) W.sb[st.scnt + __popc(bal & ((1u << lane) - 1u))] = ((uint32_t)(row0 + (int)(e >> 16)) << 16) | (e & 0xFFFFu);
  st.scnt += __popc(bal);
  st.qcnt -= nb;
  __syncwarp();
  if (st.scnt > K3_SCAP - 32) k3_flush(W, st, fd, f, lane, edge_ctr, edges, frame_err);
}

template <typename KeyT>
__global__ void __launch_bounds__(K3_THREADS) k3_nms_edges(const FrameDesc* __restrict__ frames,
                                                           const int* __restrict__ n_sorted,
                                                           const float4* __restrict__ sp_box,
                                                           const float4* __restrict__ sp_sbox,
                                                           const KeyT* __restrict__ sp_key,
                                                           const float4* __restrict__ bbox8,
                                                           const float4* __restrict__ bbox32, Consts cst, int nb8cap,
                                                           int nb32cap, int* __restrict__ edge_ctr,
                                                           uint32_t* __restrict__ edges, int* __restrict__ frame_err) {
  __shared__ float4 s_bb[K3_MAX_B32];
  __shared__ K3Warp s_w[K3_WARPS];
  __shared__ FrameDesc fd;

  const int f = blockIdx.y;
  const int n = n_sorted[f];
  if ((int)blockIdx.x * K3_THREADS >= n) return;
  const int nb32 = (n + kBlk - 1) / kBlk;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int64_t obase = (int64_t)f * cst.kpad;
  const float4* fbb32 = bbox32 + (int64_t)f * nb32cap;
  const float4* fbb8 = bbox8 + (int64_t)f * nb8cap;
  if (tid == 0) fd = frames[f];
  for (int i = tid; i < nb32; i += K3_THREADS) s_bb[i] = fbb32[i];
  __syncthreads();

  const int P = blockIdx.x * K3_WARPS + warp;
  if (P >= nb32) return;
  K3Warp& W = s_w[warp];
  K3State st;
  st.qcnt = 0; st.scnt = 0;
  const float4* fbox = sp_box + obase;
  const float4* fsbox = sp_sbox + obase;
  const KeyT* fkey = sp_key + obase;
  const int row0 = P * kBlk, row = row0 + lane;
  const float nanv = __int_as_float(0x7fc00000);
  const float inf = __int_as_float(0x7f800000);
  // rows past n are padding: culling box empty, key maximal (a2 wrote both), box NaN
  const float4 sa = fsbox[row];
  const KeyT keyA = fkey[row];
  W.rowbox[lane] = row < n ? fbox[row] : make_float4(nanv, nanv, nanv, nanv);
  const int g = lane >> 3;
  const float4 bbP8 = fbb8[P * 4 + g];
  const float4 bbP = s_bb[P];
  int cnt_g = 0;                                   // entries in this lane's group's tile list (uniform within the group)
  __syncwarp();

  // walk the group tile lists in lock step: pretest, queue, exact batches
  auto drain = [&]() {
    const int T = __reduce_max_sync(0xffffffffu, cnt_g);
    __syncwarp();
    for (int t = 0; t < T; ++t) {
      uint32_t mask = 0;
      int col0 = 0;
      if (t < cnt_g) {
        col0 = (int)W.tl[g][t] * kSub;
#pragma unroll
        for (int j = 0; j < kSub; ++j) {
          const float4 sb = fsbox[col0 + j];
          const KeyT kb = fkey[col0 + j];
          if (boxes_overlap(sa, sb) && kb < keyA) mask |= 1u << j;
        }
      }
      const int c = __popc(mask);
      int inc = c;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) { const int v = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= o) inc += v; }
      const int total = __shfl_sync(0xffffffffu, inc, 31);
      if (total == 0) continue;
      int at = st.qcnt + inc - c;
      while (mask) {
        const int j = __ffs(mask) - 1;
        mask &= mask - 1;
        W.q[at++] = ((uint32_t)lane << 16) | (uint32_t)(col0 + j);
      }
      st.qcnt += total;
      __syncwarp();
      while (st.qcnt >= 32) k3_exact_batch(W, st, 32, fbox, row0, cst, fd, f, lane, edge_ctr, edges, frame_err);
    }
    cnt_g = 0;
  };

  const int nwords = (nb32 + 31) >> 5;
  for (int i = 0; i < nwords; ++i) {
    const int Q = i * 32 + lane;
    uint32_t bits = __ballot_sync(0xffffffffu, Q < nb32 && boxes_overlap(bbP, s_bb[Q]));
    while (bits) {
      const int Q32 = i * 32 + __ffs(bits) - 1;
      bits &= bits - 1;
      // group g's 8-row box against the hit's four 8-column sub-blocks (lanes 0-3 of each group do the tests)
      float4 bq = make_float4(inf, inf, -inf, -inf);
      if ((lane & 4) == 0) bq = fbb8[Q32 * 4 + (lane & 3)];
      const uint32_t b = __ballot_sync(0xffffffffu, boxes_overlap(bbP8, bq));
      const uint32_t mine = (b >> (g * 8)) & 0xFu;
      const int c = __popc(mine);
      const int k = lane & 7;
      if (k < c) {
        uint32_t t = mine;
        for (int z = 0; z < k; ++z) t &= t - 1;
        W.tl[g][cnt_g + k] = (uint16_t)(Q32 * 4 + __ffs(t) - 1);
      }
      cnt_g += c;
      if (__any_sync(0xffffffffu, cnt_g > K3_TCAP - 4)) drain();
    }
  }
  drain();
  if (st.qcnt > 0) k3_exact_batch(W, st, st.qcnt, fbox, row0, cst, fd, f, lane, edge_ctr, edges, frame_err);
  k3_flush(W, st, fd, f, lane, edge_ctr, edges, frame_err);
}

// =====================================================================================================
// a4 — greedy resolve + order + output gather + centroid histogram (north_star (c) second half; SURVEY §8(a) a4-a5,
// §8(c) O5-O7).  One 1024-thread CTA per frame.  Greedy NMS in the order of O4 is the unique solution of
//     kept(a)  <=>  no b before a with IoU(a,b) > thr is kept,
// so instead of walking the order one box at a time the CTA iterates the frame's edge list (a <- b: "b, which comes
// first, overlaps a") to the fixed point:  an edge whose b is kept removes a;  an edge whose b is removed is dropped
// and decrements a's count of undecided suppressors;  a box whose count reaches 0 is kept.  The first undecided box
// in the order always resolves, so the loop ends; the depth is the longest chain of overlapping boxes with
// decreasing score (a handful of rounds).  Each thread owns a strided slice of the edge list and compacts it in
// place, so a round only re-reads the edges that are still undecided.  State (two bitmaps, 16-bit counters) lives
// in shared memory and is monotone.
// Then the kept keys are radix-sorted in shared memory (this is where the (score desc, index asc) order of O4 is
// materialised — on the kept set only), every kept box finds its output row by binary search, and is written with
// its sigmoid score and candidate index; its centroid is binned into the frame's histogram (a5).
// =====================================================================================================
constexpr int K4_THREADS = BLK_THREADS;

__host__ __device__ inline size_t k4_smem_bytes(size_t top_k, size_t kpad, size_t key_bytes) {
  const size_t sort_b = 2 * top_k * key_bytes, pend_b = 2 * kpad;
  return (sort_b > pend_b ? sort_b : pend_b) + BLK_WARPS * 256 * sizeof(uint16_t) + sizeof(BlkMisc) + 16;
}

template <typename KeyT>
__global__ void __launch_bounds__(K4_THREADS, 1) k4_resolve_emit(
    const FrameDesc* __restrict__ frames, const int* __restrict__ n_sorted, const float4* __restrict__ sp_box,
    const KeyT* __restrict__ sp_key, const int* __restrict__ edge_ctr, uint32_t* __restrict__ edges,
    const int* __restrict__ frame_err, Consts cst, ffpp_box* __restrict__ out_boxes, int* __restrict__ out_counts,
    uint32_t* __restrict__ hist32) {
  constexpr int KB = sizeof(KeyT) * 8;
  extern __shared__ __align__(16) uint8_t smem[];
  __shared__ uint32_t kept[K3_MAX_B32], removed[K3_MAX_B32];
  __shared__ FrameDesc fd;
  const int K = cst.top_k;
  const size_t sort_b = 2 * (size_t)K * sizeof(KeyT), pend_b = 2 * (size_t)cst.kpad;
  uint32_t* pend = reinterpret_cast<uint32_t*>(smem);                  // two uint16 counters per word (resolve phase)
  KeyT* list0 = reinterpret_cast<KeyT*>(smem);                         // aliases pend (sort phase)
  KeyT* list1 = list0 + K;
  uint16_t* hist = reinterpret_cast<uint16_t*>(smem + (sort_b > pend_b ? sort_b : pend_b));
  BlkMisc* misc = reinterpret_cast<BlkMisc*>(hist + BLK_WARPS * 256);

  const int f = blockIdx.x, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  if (frame_err[f]) { if (tid == 0) out_counts[f] = -1; return; }
  if (tid == 0) { fd = frames[f]; misc->counter = 0; }
  const int n = n_sorted[f];
  const int nb = (n + kBlk - 1) / kBlk;
  const int E = edge_ctr[f];
  const int64_t obase = (int64_t)f * cst.kpad;
  for (int i = tid; i < nb; i += K4_THREADS) { kept[i] = 0u; removed[i] = 0u; }
  for (int i = tid; i < (n + 1) / 2; i += K4_THREADS) pend[i] = 0u;
  __syncthreads();
  uint32_t* fe = edges + fd.edge_off;

  // in-degrees
  for (int e = tid; e < E; e += K4_THREADS) {
    const uint32_t a = fe[e] >> 16;
    atomicAdd(&pend[a >> 1], 1u << (16 * (a & 1u)));
  }
  __syncthreads();
  for (int a = tid; a < n; a += K4_THREADS)
    if (((pend[a >> 1] >> (16 * (a & 1))) & 0xFFFFu) == 0u) atomicOr(&kept[a >> 5], 1u << (a & 31));
  __syncthreads();

  // fixed point over this thread's strided slice of the edge list, compacted in place
  int mine = E > tid ? (E - tid + K4_THREADS - 1) / K4_THREADS : 0;
  const volatile uint32_t* vk = kept;
  const volatile uint32_t* vr = removed;
  while (true) {
    int w = 0;
    for (int k = 0; k < mine; ++k) {
      const uint32_t e = fe[tid + k * K4_THREADS];
      const uint32_t a = e >> 16, b = e & 0xFFFFu;
      if ((vr[a >> 5] >> (a & 31)) & 1u) continue;                                  // a already removed
      if ((vk[b >> 5] >> (b & 31)) & 1u) { atomicOr(&removed[a >> 5], 1u << (a & 31)); continue; }
      if ((vr[b >> 5] >> (b & 31)) & 1u) {
        const uint32_t sh = 16u * (a & 1u);
        const uint32_t old = atomicSub(&pend[a >> 1], 1u << sh);
        if (((old >> sh) & 0xFFFFu) == 1u) atomicOr(&kept[a >> 5], 1u << (a & 31)); // every suppressor is removed
        continue;
      }
      if (w != k) fe[tid + w * K4_THREADS] = e;
      ++w;
    }
    mine = w;
    if (!__syncthreads_or(mine != 0)) break;
  }

  // kept keys -> shared list (unordered), sorted by key = keep order
  for (int base = warp * 32; base < n; base += K4_THREADS) {
    const int a = base + lane;
    const bool m = a < n && ((kept[a >> 5] >> (a & 31)) & 1u);
    const uint32_t bal = __ballot_sync(0xffffffffu, m);
    int at = 0;
    if (lane == 0 && bal) at = atomicAdd(&misc->counter, __popc(bal));
    at = __shfl_sync(0xffffffffu, at, 0);
    if (m) list0[at + __popc(bal & ((1u << lane) - 1u))] = sp_key[obase + a];
  }
  __syncthreads();
  const int m = misc->counter;
  if (tid == 0) out_counts[f] = m;
  KeyT* src = list0;
  KeyT* dst = list1;
  if (m > 1) {
    for (int shift = 0; shift < KB; shift += 8)
      if (blk_lsd_pass<KeyT>(src, dst, m, shift, hist, misc, tid)) { KeyT* t = src; src = dst; dst = t; }
  }
  __syncthreads();

  // emit: output row = rank of the box's key among the kept keys
  for (int a = tid; a < n; a += K4_THREADS) {
    if ((kept[a >> 5] >> (a & 31)) & 1u) {
      const KeyT key = sp_key[obase + a];
      int lo = 0, hi = m;
      while (hi - lo > 1) { const int mid = (lo + hi) >> 1; if (src[mid] <= key) lo = mid; else hi = mid; }
      emit_kept(fd, cst, out_boxes + (int64_t)f * K + lo, sp_box[obase + a], logit_of_key<KeyT>(key), idx_of_key<KeyT>(key), hist32);
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
