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
// a0 on the device: the per-frame counters of a run (top-K counts, edge counts, overflow flags, one line per frame of
// survivor counts) are cleared by a kernel, not by cudaMemsetAsync: a memset node was seen to queue behind the DMA
// traffic of the chunked host path for tens of microseconds (profiles/r2_e2e_timeline.md), a kernel is not, and a1 can
// be its programmatic dependent.
__global__ void __launch_bounds__(256) k0_clear(int* __restrict__ counters, int max_frames, int B, unsigned long long* __restrict__ work) {
  const int i = blockIdx.x * 256 + threadIdx.x;
  if (i < 3 * B) counters[(i / B) * max_frames + (i % B)] = 0;                 // n_sorted | edge_ctr | frame_err
  else if (i < (3 + kCntStride) * B) counters[3 * max_frames + (i - 3 * B)] = 0;   // survivor counters, kCntStride ints per frame
  if (work && i < 4) work[i] = 0ull;
}

constexpr int K1_CONSUMERS = 8;
constexpr int K1_THREADS = 32 * (K1_CONSUMERS + 1);
constexpr int K1_CHUNK_BYTES = 20480;   // multiple of lcm(16, 10, 20) = 80 and of 8 warps x 32 lanes rows
constexpr int K1_STAGES = 3;
constexpr int K1_CTAS_PER_SM = 3;        // 60 KB ring + 8 KB offsets per CTA
constexpr int K1_BLOCK = 2048;          // rows per entry of the host-built block -> first frame table
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
                                                                   int B, const int64_t* __restrict__ cand_off,
                                                                   const int32_t* __restrict__ block_frame, float T,
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
  pdl_wait();                                                  // the counters are being cleared by k0_clear
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
  // A slice's survivors are stored one chunk LATER: the atomicAdd that reserves their slots in the frame's list is
  // issued, the warp releases the ring stage and evaluates the next chunk, and only then reads the returned base,
  // so the L2 round trip of the (contended, one address per frame) counter is off the critical path.
  KeyT p_keys[kHalf ? 8 : 4];
  uint32_t p_pass = 0;
  int p_total = 0, p_excl = 0, p_base = 0;
  int64_t p_coff = 0;
  auto flush_pending = [&]() {
    if (p_total) {                                              // warp-uniform
      const int base = __shfl_sync(0xffffffffu, p_base, 31);
      KeyT* dst = surv_keys + p_coff + base + p_excl;
#pragma unroll
      for (int i = 0; i < (kHalf ? 8 : 4); ++i)
        if ((p_pass >> i) & 1u) *dst++ = p_keys[i];
      p_total = 0;
    }
  };
  // table entries of this warp's first 32 slices, one per lane, fetched before the loop (a dependent global load per
  // slice would sit on the critical path of every iteration); later slices, if any, look the table up in the loop
  int bf_lane = 0;
  {
    const int64_t g = ((int64_t)blockIdx.x + (int64_t)lane * gridDim.x) * CPC + (int64_t)warp * CPW;
    if (g < total_cand) bf_lane = block_frame[g / K1_BLOCK];
  }
  int it = 0;
  for (int64_t c = blockIdx.x; c < nchunks; c += gridDim.x, ++it) {
    const int stage = it % K1_STAGES;
    const uint8_t* buf = ring + (size_t)stage * K1_CHUNK_BYTES;
    const int64_t gw0 = c * CPC + (int64_t)warp * CPW;          // first candidate of this warp's slice
    int f0 = 0;
    if (gw0 < total_cand) {                                     // frame of gw0: table + short walk in shared memory
      f0 = it < 32 ? __shfl_sync(0xffffffffu, bf_lane, it) : block_frame[gw0 / K1_BLOCK];
      while (coff[f0 + 1] <= gw0) ++f0;
    }
    mbar_wait(&full[stage], (uint32_t)(it / K1_STAGES) & 1u);
    if (gw0 + CPW <= total_cand && gw0 + CPW <= coff[f0 + 1]) {
      // ---- fast path: the warp's whole slice lies in one frame.  A lane owns CPL CONSECUTIVE rows = 80 bytes =
      // five conflict-free 16-byte shared loads, picks the score word of each row out of registers, and the slice is
      // compacted in lane order with one shuffle scan and one global atomicAdd ----
      const uint4* src = reinterpret_cast<const uint4*>(buf + ((size_t)warp * CPW + (size_t)lane * CPL) * ROW);
      uint32_t w[20];
#pragma unroll
      for (int q = 0; q < 5; ++q) { const uint4 t = src[q]; w[4 * q] = t.x; w[4 * q + 1] = t.y; w[4 * q + 2] = t.z; w[4 * q + 3] = t.w; }
      const int idx0 = (int)(gw0 - coff[f0]) + lane * CPL;
      KeyT keys[CPL];
      uint32_t pass = 0;
#pragma unroll
      for (int i = 0; i < CPL; ++i) {
        float z;
        if (kHalf) {
          const int hw = 5 * i + 4;
          const uint16_t h = (uint16_t)(w[hw >> 1] >> (16 * (hw & 1)));
          z = __half2float(__ushort_as_half(h));
          if (sizeof(KeyT) == 4) keys[i] = (KeyT)((desc_key16(h) << 16) | (uint32_t)(idx0 + i));
          else keys[i] = (KeyT)(((uint64_t)desc_key32(z) << 32) | (uint32_t)(idx0 + i));
        } else {
          z = __uint_as_float(w[5 * i + 4]);
          keys[i] = (KeyT)(((uint64_t)desc_key32(z) << 32) | (uint32_t)(idx0 + i));
        }
        if (z > T) pass |= 1u << i;
      }
      const int c = __popc(pass);
      int inc = c;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) { const int t = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= o) inc += t; }
      const int total = __shfl_sync(0xffffffffu, inc, 31);
      flush_pending();                                          // the previous slice: its atomic has had a whole chunk to return
      if (total) {
        if (lane == 31) p_base = atomicAdd(&surv_cnt[f0 * kCntStride], total);   // not consumed until the next flush
        p_total = total; p_pass = pass; p_excl = inc - c; p_coff = coff[f0];
#pragma unroll
        for (int i = 0; i < CPL; ++i) p_keys[i] = keys[i];
      }
    } else if (gw0 < total_cand) {
      flush_pending();
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
        if (lane == 0) base = atomicAdd(&surv_cnt[f * kCntStride], cnt);
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
  flush_pending();
}

// =====================================================================================================
// Block-wide (1024-thread) helper of a2: inclusive scan of one int per thread.
// =====================================================================================================
constexpr int BLK_THREADS = 1024;
constexpr int BLK_WARPS = BLK_THREADS / 32;

struct BlkMisc {
  int wsum[2][BLK_WARPS];
  int sel_digit, sel_kk, sel_tot;
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
//      each box by the spatial cell of its centre (row-major cells of 2^hshift pixels, <= 16384 per frame) with one
//      shared atomic (counting sort);
//  (4) scan the bins, scatter box / key to the frame's spatial arrays, and write the cell-start table
//      (uint16 start position of every cell, row-major) that a3 uses to enumerate the boxes of a window of cells.
// The (score desc, index asc) ORDER itself is applied where it is consumed: as key comparisons in a3/a4 (greedy NMS
// only ever asks "which of two boxes comes first") and as a radix sort of the kept keys in a4, which is ~8x fewer
// keys than sorting all top-K entries here.  The CTA also clears its frame's centroid histogram (a5).
// =====================================================================================================
constexpr int K2_THREADS = BLK_THREADS;
constexpr int K2_SEL_BITS = 12;
constexpr int K2_MAXPERM = 4096;               // batches up to this many frames get the size-ordered CTA -> frame map
constexpr int K2_HBINS = kMaxCells;
constexpr int K2_CNT_WORDS = K2_HBINS / 2;     // 32 KB: 4096 select counters (uint32) or 16384 Hilbert counters (uint16)

__host__ __device__ inline size_t k2_smem_bytes(size_t top_k, size_t key_bytes) {
  return top_k * key_bytes + top_k * sizeof(uint32_t) + K2_CNT_WORDS * sizeof(uint32_t) + sizeof(BlkMisc) + 16;
}

template <bool kHalf, typename KeyT>
__global__ void __launch_bounds__(K2_THREADS, 1) k2_select_bin(
    const uint8_t* __restrict__ raw, const FrameDesc* __restrict__ frames, const KeyT* __restrict__ surv_keys,
    const int* __restrict__ surv_cnt, Consts cst, float4* __restrict__ sel_box, float4* __restrict__ sp_box,
    KeyT* __restrict__ sp_key, uint16_t* __restrict__ cellstart,
    int* __restrict__ n_sorted, uint32_t* __restrict__ hist32, uint32_t* __restrict__ hasin, int sm_count) {
  constexpr int KB = sizeof(KeyT) * 8;
  extern __shared__ __align__(16) uint8_t smem[];
  pdl_wait();
  const int K = cst.top_k;
  KeyT* sel = reinterpret_cast<KeyT*>(smem);
  uint32_t* aux = reinterpret_cast<uint32_t*>(sel + K);
  uint32_t* cnt = aux + K;
  BlkMisc* misc = reinterpret_cast<BlkMisc*>(cnt + K2_CNT_WORDS);
  __shared__ FrameDesc fd;

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  // Which frame this CTA takes: CTAs are handed out in index order, one per SM, so CTA i takes the frame with the
  // i-th largest survivor count — the long frames start in the first wave and the tail is made of short ones.
  __shared__ int s_frame;
  {
    const int B = (int)gridDim.x, i = (int)blockIdx.x;
    if (B <= sm_count || B > K2_MAXPERM) {
      if (tid == 0) s_frame = i;
    } else {
      int* wts = reinterpret_cast<int*>(cnt);                      // the counter array is free until the select
      for (int g = tid; g < B; g += K2_THREADS) wts[g] = surv_cnt[g * kCntStride];
      __syncthreads();
      for (int g = tid; g < B; g += K2_THREADS) {
        const int wg = wts[g];
        int rank = 0;
        for (int h = 0; h < B; ++h) { const int wh = wts[h]; rank += (wh > wg) | ((wh == wg) & (h < g)); }
        if (rank == i) s_frame = g;
      }
    }
    __syncthreads();
  }
  const int f = s_frame;
  if (tid == 0) fd = frames[f];
  __syncthreads();
  const int n = surv_cnt[f * kCntStride];
  const int nsel = n < K ? n : K;
  const KeyT* gk = surv_keys + fd.cand_off;
  FFPP_PHASE2(f, 0);

  // clear this frame's centroid histogram (uint16 per cell, two per word; boundary words are shared with the
  // neighbouring frames, which clear them too — every a2 CTA finishes before a4 counts)
  {
    const int64_t w0 = fd.dens_off >> 1, w1 = (fd.dens_off + (int64_t)fd.gw * fd.gh + 1) >> 1;
    for (int64_t i = w0 + tid; i < w1; i += K2_THREADS) hist32[i] = 0u;
    uint32_t* hz = hasin + (int64_t)f * cst.kpad / 4;                   // a3's victim flags of this frame
    for (int i = tid; i < cst.kpad / 4; i += K2_THREADS) hz[i] = 0u;
  }

  // ---- (1) threshold key = K-th smallest ----
  FFPP_PHASE2(f, 1);
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
          const int i = base + u * K2_THREADS + lane;
          if (i < n && (key[u] & maskbits) == prefix) atomicAdd(&cnt[(uint32_t)((key[u] >> shift) & dmask)], 1u);
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

  // ---- (2) gather the selected keys into shared memory: count per warp, scan the warps, then place (two sweeps
  FFPP_PHASE2(f, 2);
  // over the L2-resident keys instead of one shared atomic per warp step on a single hot counter) ----
  {
    int mine = 0;
    for (int base = warp * 32; base < n; base += 4 * K2_THREADS) {
      KeyT key[4];
#pragma unroll
      for (int u = 0; u < 4; ++u) { const int i = base + u * K2_THREADS + lane; key[u] = i < n ? gk[i] : ~(KeyT)0; }
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        const int i = base + u * K2_THREADS + lane;
        mine += __popc(__ballot_sync(0xffffffffu, i < n && key[u] <= thr));
      }
    }
    int total;
    const int inc = blk_scan_inclusive(lane == 0 ? mine : 0, misc, 0, tid, &total);
    int at = __shfl_sync(0xffffffffu, inc, 0) - mine;            // first slot of this warp
    for (int base = warp * 32; base < n; base += 4 * K2_THREADS) {
      KeyT key[4];
#pragma unroll
      for (int u = 0; u < 4; ++u) { const int i = base + u * K2_THREADS + lane; key[u] = i < n ? gk[i] : ~(KeyT)0; }
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        const int i = base + u * K2_THREADS + lane;
        const bool m = i < n && key[u] <= thr;
        const uint32_t bal = __ballot_sync(0xffffffffu, m);
        if (m) sel[at + __popc(bal & ((1u << lane) - 1u))] = key[u];
        at += __popc(bal);
      }
    }
  }
  for (int i = tid; i < K2_CNT_WORDS; i += K2_THREADS) cnt[i] = 0u;
  __syncthreads();
  FFPP_PHASE2(f, 3);

  // ---- (3) decode (O1, O2) + spatial bin ----
  const int64_t obase = (int64_t)f * cst.kpad;
  const float cmx = (float)((fd.cgw << fd.hshift) - 1), cmy = (float)((fd.cgh << fd.hshift_y) - 1);
  for (int i0 = tid; i0 < nsel; i0 += 4 * K2_THREADS) {
    float v[4][4];
    float ps[4][3];                                                // px, py, stride
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      const int i = i0 + u * K2_THREADS;
      if (i < nsel) {
        const int idx = idx_of_key<KeyT>(sel[i]);
        int l = 0;
        while (l + 1 < cst.num_levels && idx >= fd.lvl_start[l + 1]) ++l;
        const int k = idx - fd.lvl_start[l];
        const int gw = fd.lvl_gw[l];
        int iy = (int)(((float)k + 0.5f) * __frcp_rn((float)gw));        // k < 2^20: off by at most one, fixed below
        int ix = k - iy * gw;
        if (ix < 0) { --iy; ix += gw; } else if (ix >= gw) { ++iy; ix -= gw; }
        const float s = (float)(1 << cst.stride_log2[l]);
        ps[u][0] = __fmul_rn((float)ix + 0.5f, s); ps[u][1] = __fmul_rn((float)iy + 0.5f, s); ps[u][2] = s;
        const int64_t row = fd.cand_off + idx;
        if (kHalf) {
          const __half* p = reinterpret_cast<const __half*>(raw) + row * 5;
#pragma unroll
          for (int e = 0; e < 4; ++e) v[u][e] = __half2float(p[e]);
        } else {
          const float* p = reinterpret_cast<const float*>(raw) + row * 5;
#pragma unroll
          for (int e = 0; e < 4; ++e) v[u][e] = p[e];
        }
      }
    }
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      const int i = i0 + u * K2_THREADS;
      if (i < nsel) {
        const float s = ps[u][2];
        float4 box;
        box.x = __fsub_rn(ps[u][0], __fmul_rn(v[u][0], s));
        box.y = __fsub_rn(ps[u][1], __fmul_rn(v[u][1], s));
        box.z = __fadd_rn(ps[u][0], __fmul_rn(v[u][2], s));
        box.w = __fadd_rn(ps[u][1], __fmul_rn(v[u][3], s));
        sel_box[obase + i] = box;
        const uint32_t h = (uint32_t)(cell_coord(box_centre(box.y, box.w), cmy, fd.hshift_y) * fd.cgw +
                                      cell_coord(box_centre(box.x, box.z), cmx, fd.hshift));
        const uint32_t sh = 16u * (h & 1u);
        const uint32_t old = atomicAdd(&cnt[h >> 1], 1u << sh);
        aux[i] = (h << 16) | ((old >> sh) & 0xFFFFu);
      }
    }
  }
  __syncthreads();
  FFPP_PHASE2(f, 4);

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
  FFPP_PHASE2(f, 5);
  const uint16_t* base16 = reinterpret_cast<const uint16_t*>(cnt);
  for (int i0 = tid; i0 < nsel; i0 += 4 * K2_THREADS) {
    float4 box[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) { const int i = i0 + u * K2_THREADS; if (i < nsel) box[u] = sel_box[obase + i]; }
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      const int i = i0 + u * K2_THREADS;
      if (i < nsel) {
        const uint32_t a = aux[i];
        const int pos = (int)base16[a >> 16] + (int)(a & 0xFFFFu);
        sp_box[obase + pos] = box[u];
        sp_key[obase + pos] = sel[i];
      }
    }
  }
  // cell-start table: after the scan the counter words ARE the uint16 start positions in cell order
  {
    const int ncells = fd.cgw * fd.cgh;
    uint32_t* cs32 = reinterpret_cast<uint32_t*>(cellstart + (int64_t)f * kCellStride);
    for (int i = tid; i < (ncells + 1) / 2; i += K2_THREADS) cs32[i] = cnt[i];
    if (tid == 0) {
      n_sorted[f] = nsel;
      cellstart[(int64_t)f * kCellStride + ncells] = (uint16_t)nsel;      // ncells even or odd: the terminal entry
    }
  }
#ifdef FFPP_PROFILE_PHASES
  __syncthreads();
  FFPP_PHASE2(f, 6);
  if (tid == 0) g_phase2[f][7] = ((unsigned long long)n << 32) | (unsigned long long)nsel;
#endif
}

// =====================================================================================================
// a3 — NMS suppression pairs, cell-windowed (north_star (c)).
// The bit "IoU(a, b) > thr" is the same bit the rank-ordered matrix of the north_star sketch holds; what changes is
// which bits are ever looked at.  Boxes are sorted by the row-major spatial cell of their centre (a2).  A pair with
// IoU > thr has, on each axis, |centre_a - centre_b| < rho * min(w_a, w_b)  (from iw > thr * max(w_a, w_b) and
// |dc| <= (w_a + w_b)/2 - iw;  rho = max(1 - thr, 1/(2 thr) - 1/2), DESIGN.md §6 a3), so the partner of box a lies
// in a window of cells around a's own cell that a computes from its own size.  Every unordered pair is examined once,
// by the member that comes first in the spatial order: its candidates are the rest of its own cell row and the
// window's rows below, each row one contiguous range of the sorted arrays, found through the cell-start table.
// A warp owns 32 consecutive boxes and works in two alternating phases, so that the expensive part runs on full lanes
// whatever the shape of the individual windows:
//  (1) fill: every lane appends its (owner lane, candidate position) pairs of one window row to the warp's work list
//      in shared memory (warp prefix sum of the range lengths; a short divergent loop of 3 instructions per entry);
//  (2) drain: the list is consumed 32 entries at a time, one pair per lane: the owner's box comes from shared memory,
//      the candidate's from the sorted array, and the fp32 IoU of the definition (iou_exceeds) decides.  A hit becomes
//      the edge (victim << 16 | suppressor), spatial positions, the suppressor being the member that comes first in
//      the order of O4 (smaller key); edges are staged per warp and appended to the frame's edge pool with one
//      atomicAdd per flush, and the victim's "has a suppressor" byte is set (a plain store).
// The list is drained only when it is full or the warp has no rows left, so all but the last step of a warp are full.
// =====================================================================================================
constexpr uint32_t ST_U = 0, ST_K = 1, ST_R = 2;   // box state of the greedy fixed point (overflow path, a4)
constexpr int K3_WARPS = 4;
constexpr int K3_THREADS = 32 * K3_WARPS;
constexpr int K3_CHUNK = 16;                    // entries one lane appends per fill step
constexpr int K3_LCAP = 32 * K3_CHUNK + 32;     // work list: one full fill step on top of a < 32 entry remainder
constexpr int K3_SCAP = 256;                    // hit staging per warp (a warp of the flock workloads has ~200)

template <typename KeyT>
struct K3Warp {
  float4 rowbox[32];
  KeyT rowkey[32];
  uint32_t list[K3_LCAP];
  uint32_t sb[K3_SCAP];
};

template <typename KeyT, bool kCount>
__global__ void __launch_bounds__(K3_THREADS, 12) k3_nms_edges(const FrameDesc* __restrict__ frames,
                                                           const int* __restrict__ n_sorted,
                                                           const float4* __restrict__ sp_box,
                                                           const KeyT* __restrict__ sp_key,
                                                           const uint16_t* __restrict__ cellstart, Consts cst,
                                                           int* __restrict__ edge_ctr, uint32_t* __restrict__ edges,
                                                           uint8_t* __restrict__ hasin, int* __restrict__ frame_err,
                                                           unsigned long long* __restrict__ work_ctr) {
  __shared__ K3Warp<KeyT> s_w[K3_WARPS];
  unsigned long long n_exact = 0, n_edge = 0;                 // kCount only: this lane's exact IoUs / edges

  pdl_wait();
  const int f = blockIdx.y;
  const int n = n_sorted[f];
  const int p0 = blockIdx.x * K3_THREADS;
  if (p0 >= n) return;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  if (p0 + warp * 32 >= n) return;
  if (!kCount && *reinterpret_cast<volatile int*>(&frame_err[f])) return;   // the frame already goes to the overflow path
  const FrameDesc* fd = &frames[f];
  const int cgw = fd->cgw, cgh = fd->cgh, hs = fd->hshift, hsy = fd->hshift_y;
  const int64_t obase = (int64_t)f * cst.kpad;
  const float4* fbox = sp_box + obase;
  const KeyT* fkey = sp_key + obase;
  const uint16_t* cs = cellstart + (int64_t)f * kCellStride;
  K3Warp<KeyT>& W = s_w[warp];
  const uint32_t lt = (1u << lane) - 1u;

  const int row0 = p0 + warp * 32;
  const int p = row0 + lane;
  const bool valid = p < n;
  const int pc = valid ? p : n - 1;
  const float4 a = fbox[pc];
  W.rowbox[lane] = a;
  W.rowkey[lane] = fkey[pc];

  // window of cells that can hold a partner's centre
  const float cmx = (float)((cgw << hs) - 1), cmy = (float)((cgh << hsy) - 1);
  const float cxa = box_centre(a.x, a.z), cya = box_centre(a.y, a.w);
  const float ex = fmaxf(cst.rho * (a.z - a.x), 0.0f) * 1.001f + 1e-5f * (fabsf(a.x) + fabsf(a.z));
  const float ey = fmaxf(cst.rho * (a.w - a.y), 0.0f) * 1.001f + 1e-5f * (fabsf(a.y) + fabsf(a.w));
  const int Xlo = cell_coord(cxa - ex, cmx, hs), Xhi = cell_coord(cxa + ex, cmx, hs);
  const int Ya = cell_coord(cya, cmy, hsy);
  const int Yhi = cell_coord(cya + ey, cmy, hsy);
  int lcnt = 0, scnt = 0;                          // warp-uniform
  __syncwarp();

  // staged hits are (owner lane << 16 | candidate position); the flush turns them into edges on full lanes: the
  // suppressor is the member that comes first in the order of O4 (smaller key), the victim's flag byte is set
  const int edge_cap = fd->edge_cap;
  uint32_t* const fedges = edges + fd->edge_off;
  uint8_t* const fhas = hasin + obase;
  auto flush = [&]() {
    if (scnt == 0) return;
    __syncwarp();
    int base = 0;
    if (lane == 0) base = atomicAdd(&edge_ctr[f], scnt);
    base = __shfl_sync(0xffffffffu, base, 0);
    if (base + scnt <= edge_cap) {
      for (int k = lane; k < scnt; k += 32) {
        const uint32_t q = W.sb[k];
        const uint32_t al = q >> 16, b = q & 0xFFFFu, pa = (uint32_t)row0 + al;
        const uint32_t ed = fkey[b] < W.rowkey[al] ? ((pa << 16) | b) : ((b << 16) | pa);
        fhas[ed >> 16] = 1;                        // a4 starts every box that is nobody's victim as kept
        fedges[base + k] = ed;
      }
    } else if (lane == 0) {
      frame_err[f] = 1;                            // the frame's pool share is exhausted: the overflow path resolves the frame
    }
    scnt = 0;
    __syncwarp();
  };
  // record the hits of one step (one pair per lane) in the staging area
  auto stage_hits = [&](const bool hit, const uint32_t q) {
    const uint32_t bal = __ballot_sync(0xffffffffu, hit);
    if (hit) W.sb[scnt + __popc(bal & lt)] = q;
    scnt += __popc(bal);
    if (scnt > K3_SCAP - 32) flush();
  };
  // consume the full 32-entry steps of the list, one pair per lane per step, the next step's entry and candidate box
  // already in flight while this step's IoU is evaluated; the remainder (< 32 entries) moves to the front, or is
  // evaluated too (`all`)
  auto drain = [&](const bool all) {
    int i = 0;
    if (lcnt >= 32) {
      uint32_t q = W.list[lane];
      float4 bb = fbox[q & 0xFFFFu];
      for (; i + 32 <= lcnt; i += 32) {
        uint32_t qn = 0;
        float4 bn = bb;
        if (i + 64 <= lcnt) { qn = W.list[i + 32 + lane]; bn = fbox[qn & 0xFFFFu]; }
        if (kCount) ++n_exact;
        const bool hit = iou_exceeds(W.rowbox[q >> 16], bb, cst);
        if (kCount && hit) ++n_edge;
        stage_hits(hit, q);
        q = qn; bb = bn;
      }
    }
    const int rem = lcnt - i;
    if (rem > 0 && all) {
      bool hit = false;
      uint32_t q = 0;
      if (lane < rem) {
        q = W.list[i + lane];
        if (kCount) ++n_exact;
        hit = iou_exceeds(W.rowbox[q >> 16], fbox[q & 0xFFFFu], cst);
        if (kCount && hit) ++n_edge;
      }
      stage_hits(hit, q);
      lcnt = 0;
      return;
    }
    if (rem > 0 && i > 0) {
      const uint32_t v = lane < rem ? W.list[i + lane] : 0u;
      __syncwarp();
      if (lane < rem) W.list[lane] = v;
      __syncwarp();
    }
    lcnt = rem;
  };

  for (int rr = 0;; ++rr) {
    const int Y = Ya + rr;
    const bool act = valid && Y <= Yhi;
    if (!__any_sync(0xffffffffu, act)) break;
    int j = 0, rem = 0;
    if (act) {
      const uint16_t* r = cs + Y * cgw;
      j = rr == 0 ? p + 1 : (int)r[Xlo];
      rem = max((int)r[Xhi + 1] - j, 0);
    }
    while (__any_sync(0xffffffffu, rem > 0)) {
      const int c = min(rem, K3_CHUNK);
      int inc = c;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) { const int t = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= o) inc += t; }
      const int total = __shfl_sync(0xffffffffu, inc, 31);
      if (lcnt + total > K3_LCAP) drain(false);    // leaves < 32 entries: a whole fill step fits
      uint32_t* dst = W.list + lcnt + inc - c;
      const uint32_t e0 = ((uint32_t)lane << 16) | (uint32_t)j;
      for (int i = 0; i < c; ++i) dst[i] = e0 + (uint32_t)i;
      j += c; rem -= c; lcnt += total;
      __syncwarp();
    }
  }
  drain(true);
  flush();
  if (kCount) {
    n_exact = warp_sum_u64(n_exact); n_edge = warp_sum_u64(n_edge);
    if (lane == 0) { atomicAdd(&work_ctr[1], n_exact); atomicAdd(&work_ctr[2], n_edge); }
  }
}

// =====================================================================================================
// a3/a4 overflow path — a frame whose suppression pairs do not fit its share of the edge pool (k3 raised frame_err[f]).
// Greedy NMS is the unique fixed point of  kept(a) <=> no kept b before a with IoU(a,b) > thr;  the frame's a4 CTA
// iterates to it WITHOUT stored pairs: one state byte per box in shared memory (the same bytes the edge-list fixed
// point uses), and per round every undecided box re-examines its partner window (the same cell window as k3, both
// directions this time):
//     some kept partner before it has IoU > thr          -> removed
//     no undecided-or-kept partner before it has IoU > thr -> kept
//     otherwise                                             -> stays undecided.
// K and R are final, so a decision taken from states another thread is updating in the same round is still right
// (chaotic iteration); the first undecided box of the order always decides, so the loop ends after at most
// (longest chain of overlapping boxes with decreasing score) rounds.  Workspace: the state bytes, whatever the input.
// =====================================================================================================
template <typename KeyT, int kThreads>
__device__ __forceinline__ void overflow_fixed_point(uint8_t* state, const int n, const FrameDesc& fd, const float4* __restrict__ fbox,
                                                     const KeyT* __restrict__ fkey, const uint16_t* __restrict__ cs, const Consts& cst,
                                                     const int tid) {
  const int cgw = fd.cgw, cgh = fd.cgh, hs = fd.hshift, hsy = fd.hshift_y;
  volatile uint8_t* st = state;
  const float cmx = (float)((cgw << hs) - 1), cmy = (float)((cgh << hsy) - 1);
  for (;;) {
    bool undecided = false;
    for (int p = tid; p < n; p += kThreads) {
      if (st[p] != ST_U) continue;
      const float4 a = fbox[p];
      const KeyT ka = fkey[p];
      const float cxa = box_centre(a.x, a.z), cya = box_centre(a.y, a.w);
      const float ex = fmaxf(cst.rho * (a.z - a.x), 0.0f) * 1.001f + 1e-5f * (fabsf(a.x) + fabsf(a.z));
      const float ey = fmaxf(cst.rho * (a.w - a.y), 0.0f) * 1.001f + 1e-5f * (fabsf(a.y) + fabsf(a.w));
      const int Xlo = cell_coord(cxa - ex, cmx, hs), Xhi = cell_coord(cxa + ex, cmx, hs);
      const int Ylo = cell_coord(cya - ey, cmy, hsy), Yhi = cell_coord(cya + ey, cmy, hsy);
      bool removed = false, blocked = false;
      for (int Y = Ylo; Y <= Yhi && !removed; ++Y) {
        const uint16_t* r = cs + Y * cgw;
        const int e = r[Xhi + 1];
        for (int j = r[Xlo]; j < e; ++j) {
          const uint32_t sj = st[j];
          if (sj == ST_R || j == p) continue;
          if (!(fkey[j] < ka)) continue;                       // only a box BEFORE a in the order of O4 can suppress it
          const float4 b = fbox[j];
          if (!boxes_overlap(a, b)) continue;                  // inter == 0: IoU > thr is false for every thr >= 0
          if (!iou_exceeds(a, b, cst)) continue;
          if (sj == ST_K) { removed = true; break; }
          blocked = true;
        }
      }
      if (removed) st[p] = (uint8_t)ST_R;
      else if (!blocked) st[p] = (uint8_t)ST_K;
      else undecided = true;
    }
    if (!__syncthreads_or(undecided)) break;
  }
}

// =====================================================================================================
// a4 — greedy resolve + order (+ k4e_emit: output gather + centroid histogram) (north_star (c) second half; SURVEY §8(a) a4-a5,
// §8(c) O5-O7).  One 512-thread CTA per frame, two CTAs per SM (296 slots: a 256-frame batch is resident at once and
// the barriers of one frame are hidden behind the work of another).
// Greedy NMS in the order of O4 is the unique solution of
//     kept(a)  <=>  no b before a with IoU(a,b) > thr is kept,
// so instead of walking the order one box at a time the CTA iterates the frame's edge list (victim <- suppressor) to
// that fixed point, with one state byte per box in shared memory (U undecided, K kept, R removed) and two flag bytes
// (rem, blk) — plain loads and stores, no atomics.  Boxes that are nobody's victim (a3 flagged every victim) start
// as K; then, per round,
//   phase 1, per edge (v <- s):  v decided -> drop;  s kept -> rem[v] = 1, drop;  s removed -> drop;
//                                s undecided -> blk[v] = 1, keep the edge;
//   phase 2, per box, four state bytes per 32-bit word:  U & rem -> R;  U & !rem & !blk -> K;  flags cleared.
// The first undecided box in the order always resolves, so the loop ends; the depth is the longest chain of
// overlapping boxes with decreasing score (a handful of rounds).  Each thread owns a strided slice of the edge list,
// reads it eight edges at a time (the list lives in L2: memory-level parallelism, not latency, must pace the loop)
// and compacts it in place, so a round only re-reads the edges that are still undecided.
// Then the kept boxes are ordered: their keys and spatial positions are gathered through a prefix sum of the kept
// bitmap and sorted by key (bitonic network up to 1024, LSD radix beyond; this is where the (score desc, index asc)
// order of O4 is materialised — on the kept set only) and the ordered (key, position) list goes to global memory for
// the flat emit kernel k4e_emit.  The sort arrays live in shared memory when they fit, else in a global scratch area.
// =====================================================================================================
constexpr int K4_THREADS = 512;
constexpr int K4_WARPS = K4_THREADS / 32;
constexpr int K4_SMEM_BUDGET = 108 * 1024;       // dynamic shared memory per CTA (two CTAs per SM)
constexpr int K4_MAXPERM = 1024;                 // batches up to this many frames get the weight-ordered CTA -> frame map
constexpr int K4_UNROLL = 8;
constexpr int K4_BITONIC_MAX = 256;              // kept sets up to this size take the bitonic network, larger ones LSD radix

struct K4Misc {
  int wsum[K4_WARPS];
};

__host__ __device__ inline size_t k4_pow2ceil(size_t v) { size_t p = 1; while (p < v) p <<= 1; return p; }
// bytes of the resolve/sort union region and of the fixed tail (kept bitmap, its word prefix, misc)
__host__ __device__ inline size_t k4_tail_bytes(size_t kpad) {
  return kpad / 8 + ((kpad / 32 * 2 + 15) & ~(size_t)15) + K4_WARPS * 256 * sizeof(uint16_t) + sizeof(K4Misc) + 16;
}
// sort arrays for m kept boxes: two (key, position) buffers, m rounded up to a power of two for the bitonic path
__host__ __device__ inline size_t k4_sort_bytes(size_t m, size_t key_bytes) {
  const size_t lsd = 2 * (((m * key_bytes + 15) & ~(size_t)15) + ((m * 2 + 15) & ~(size_t)15));
  const size_t np = k4_pow2ceil(m);                            // bitonic path: two buffers of pow2ceil(m) pairs
  const size_t bit = m <= (size_t)K4_BITONIC_MAX ? 2 * (((np * key_bytes + 15) & ~(size_t)15) + ((np * 2 + 15) & ~(size_t)15)) : 0;
  return lsd > bit ? lsd : bit;
}
__host__ __device__ inline size_t k4_union_bytes(size_t top_k, size_t kpad, size_t key_bytes) {
  const size_t flag_b = 3 * kpad;
  size_t sort_b = k4_sort_bytes(top_k, key_bytes);
  const size_t room = (size_t)K4_SMEM_BUDGET - k4_tail_bytes(kpad);
  if (sort_b > room) sort_b = room;
  return ((sort_b > flag_b ? sort_b : flag_b) + 15) & ~(size_t)15;
}
__host__ __device__ inline size_t k4_smem_bytes(size_t top_k, size_t kpad, size_t key_bytes) {
  return k4_union_bytes(top_k, kpad, key_bytes) + k4_tail_bytes(kpad);
}
__host__ __device__ inline size_t k4_scratch_bytes(size_t top_k, size_t key_bytes) {   // per frame
  return (k4_sort_bytes(top_k, key_bytes) + 15) & ~(size_t)15;
}

// lanes of the warp that hold the same 8-bit digit (ballot per digit bit: a fixed 8 steps whatever the digit mix)
__device__ __forceinline__ uint32_t k4_peers8(const uint32_t dg, const bool v) {
  uint32_t p = __ballot_sync(0xffffffffu, v);
#pragma unroll
  for (int b = 0; b < 8; ++b) {
    const bool bit = (dg >> b) & 1u;
    const uint32_t bal = __ballot_sync(0xffffffffu, bit);
    p &= bit ? bal : ~bal;
  }
  return p;
}

// One stable LSD pass (8-bit digit at `shift`) over m (key, position) pairs, 512 threads.  Returns false (nothing
// moved) when the digit is the same for every key.  hist = 16 warps x 256 digits.
template <typename KeyT>
__device__ __forceinline__ bool k4_lsd_pass(const KeyT* ksrc, const uint16_t* psrc, KeyT* kdst, uint16_t* pdst, int m,
                                            int shift, uint16_t* hist, K4Misc* misc, int tid) {
  const int lane = tid & 31, warp = tid >> 5;
  const int seg = ((m + K4_WARPS - 1) / K4_WARPS + 31) & ~31;      // per-warp contiguous segment
  const int w_begin = warp * seg < m ? warp * seg : m;
  const int w_end = (warp + 1) * seg < m ? (warp + 1) * seg : m;
  uint32_t* hist32 = reinterpret_cast<uint32_t*>(hist);
  for (int i = tid; i < K4_WARPS * 256 / 2; i += K4_THREADS) hist32[i] = 0u;
  __syncthreads();
  for (int base = w_begin; base < w_end; base += 32) {
    const int i = base + lane;
    const bool v = i < w_end;
    // two uint16 counters per word, one row per warp; no carry (a warp segment has < 65536 entries).  Counting needs
    // no peer mask: same-digit lanes simply serialise on the shared atomic.
    if (v) {
      const uint32_t dg = (uint32_t)((ksrc[i] >> shift) & 255);
      atomicAdd(&hist32[(warp * 256 + dg) >> 1], 1u << (16 * (dg & 1)));
    }
  }
  __syncthreads();
  // thread d < 256 owns digit d: counts of the 16 warps, exclusive offsets in (digit major, warp minor) order
  int c[K4_WARPS], s = 0;
  if (tid < 256) {
#pragma unroll
    for (int w = 0; w < K4_WARPS; ++w) { c[w] = hist[w * 256 + tid]; s += c[w]; }
  }
  if (__syncthreads_or(s == m)) return false;
  int inc = s;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) { const int t = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= o) inc += t; }
  if (lane == 31) misc->wsum[warp] = inc;
  __syncthreads();
  if (tid < 256) {
    int run = inc - s;
#pragma unroll
    for (int w = 0; w < 8; ++w) if (w < warp) run += misc->wsum[w];
#pragma unroll
    for (int w = 0; w < K4_WARPS; ++w) { hist[w * 256 + tid] = (uint16_t)run; run += c[w]; }
  }
  __syncthreads();
  for (int base = w_begin; base < w_end; base += 32) {
    const int i = base + lane;
    const bool v = i < w_end;
    KeyT key = 0;
    uint16_t pe = 0;
    if (v) { key = ksrc[i]; pe = psrc[i]; }
    const uint32_t dg = v ? (uint32_t)((key >> shift) & 255) : 0u;
    const uint32_t peers = k4_peers8(dg, v);
    int b = 0;
    if (v) b = hist[warp * 256 + dg];
    __syncwarp();
    if (v && lane == __ffs(peers) - 1) hist[warp * 256 + dg] = (uint16_t)(b + __popc(peers));
    __syncwarp();
    if (v) { const int o = b + __popc(peers & ((1u << lane) - 1u)); kdst[o] = key; pdst[o] = pe; }
  }
  __syncthreads();
  return true;
}

// Bitonic sort of m <= K4_BITONIC_MAX (key, position) pairs held in kA/pA (capacity Np = pow2ceil(m)); kB/pB is a second
// buffer of the same size.  A thread keeps two elements in registers (e0 = 64 warp + lane, e1 = e0 + 32): partner
// distances below 32 are shuffles, 32 is the thread's own pair, and only distances >= 64 go through shared memory —
// 10 block barriers for 1024 keys instead of 55 (a barrier-bound sort crawls when another frame shares the SM).
template <typename KeyT>
__device__ __forceinline__ void k4_bitonic(KeyT* kA, uint16_t* pA, KeyT* kB, uint16_t* pB, const int m, const int Np, const int tid) {
  const int lane = tid & 31, warp = tid >> 5;
  const int e0 = warp * 64 + lane, e1 = e0 + 32;
  const int NE = Np < 64 ? 64 : Np;
  const bool part = e0 < NE;                                   // warp-uniform
  KeyT k0 = ~(KeyT)0, k1 = ~(KeyT)0;                           // padding: maximal keys, sorted to the end, never stored
  uint16_t q0 = 0, q1 = 0;
  if (part) {
    if (e0 < m) { k0 = kA[e0]; q0 = pA[e0]; }
    if (e1 < m) { k1 = kA[e1]; q1 = pA[e1]; }
  }
  KeyT* xk[2] = {kB, kA};
  uint16_t* xq[2] = {pB, pA};
  int cur = 0;
  __syncthreads();                                              // kA is free to be an exchange buffer from here on
  for (int k = 2; k <= NE; k <<= 1) {
    for (int j = k >> 1; j > 0; j >>= 1) {
      if (j >= 64) {
        KeyT* bk = cur ? xk[1] : xk[0];
        uint16_t* bq = cur ? xq[1] : xq[0];
        if (part) { bk[e0] = k0; bq[e0] = q0; bk[e1] = k1; bq[e1] = q1; }
        __syncthreads();
        if (part) {
          {
            const KeyT ok = bk[e0 ^ j]; const uint16_t oq = bq[e0 ^ j];
            const bool take_min = ((e0 & j) == 0) == ((e0 & k) == 0);
            if (take_min ? ok < k0 : ok > k0) { k0 = ok; q0 = oq; }
          }
          {
            const KeyT ok = bk[e1 ^ j]; const uint16_t oq = bq[e1 ^ j];
            const bool take_min = ((e1 & j) == 0) == ((e1 & k) == 0);
            if (take_min ? ok < k1 : ok > k1) { k1 = ok; q1 = oq; }
          }
        }
        cur ^= 1;
      } else if (part) {
        if (j == 32) {
          if ((k0 > k1) == ((e0 & k) == 0)) { const KeyT tk = k0; k0 = k1; k1 = tk; const uint16_t tq = q0; q0 = q1; q1 = tq; }
        } else {
          const bool lower = (lane & j) == 0;
          {
            const KeyT ok = __shfl_xor_sync(0xffffffffu, k0, j); const uint16_t oq = (uint16_t)__shfl_xor_sync(0xffffffffu, (int)q0, j);
            const bool take_min = lower == ((e0 & k) == 0);
            if (take_min ? ok < k0 : ok > k0) { k0 = ok; q0 = oq; }
          }
          {
            const KeyT ok = __shfl_xor_sync(0xffffffffu, k1, j); const uint16_t oq = (uint16_t)__shfl_xor_sync(0xffffffffu, (int)q1, j);
            const bool take_min = lower == ((e1 & k) == 0);
            if (take_min ? ok < k1 : ok > k1) { k1 = ok; q1 = oq; }
          }
        }
      }
    }
  }
  __syncthreads();                                              // every exchange read is done
  if (part) {
    if (e0 < m) { kA[e0] = k0; pA[e0] = q0; }
    if (e1 < m) { kA[e1] = k1; pA[e1] = q1; }
  }
  __syncthreads();
}

template <typename KeyT>
__global__ void __launch_bounds__(K4_THREADS, 2) k4_resolve_order(
    const FrameDesc* __restrict__ frames, const int* __restrict__ n_sorted, const float4* __restrict__ sp_box,
    const KeyT* __restrict__ sp_key, const int* __restrict__ edge_ctr, uint32_t* edges,
    const uint32_t* __restrict__ hasin, const uint16_t* __restrict__ cellstart, const int* __restrict__ frame_err, Consts cst,
    int sm_count, uint8_t* __restrict__ scratch, KeyT* __restrict__ kept_key, uint16_t* __restrict__ kept_pos,
    int* __restrict__ out_counts) {
  extern __shared__ __align__(16) uint8_t smem[];
  __shared__ FrameDesc fd;
  pdl_wait();
  const int K = cst.top_k, kpad = cst.kpad;
  const size_t uni_b = k4_union_bytes((size_t)K, (size_t)kpad, sizeof(KeyT));
  uint32_t* st32 = reinterpret_cast<uint32_t*>(smem);                  // resolve phase: state, rem, blk bytes
  uint32_t* rem32 = reinterpret_cast<uint32_t*>(smem + kpad);
  uint32_t* blk32 = reinterpret_cast<uint32_t*>(smem + 2 * kpad);
  uint8_t* st = smem;
  uint8_t* rem = smem + kpad;
  uint8_t* blk = smem + 2 * kpad;
  uint32_t* keptw = reinterpret_cast<uint32_t*>(smem + uni_b);         // kept bitmap, kpad / 32 words
  uint16_t* wpre = reinterpret_cast<uint16_t*>(smem + uni_b + kpad / 8);   // kept boxes before each bitmap word
  uint16_t* hist = reinterpret_cast<uint16_t*>(smem + uni_b + kpad / 8 + ((kpad / 32 * 2 + 15) & ~15));
  K4Misc* misc = reinterpret_cast<K4Misc*>(hist + K4_WARPS * 256);

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  // Which frame this CTA takes.  All CTAs start at once; the hardware hands out CTAs 0..S-1 one per SM and doubles up
  // after that (measured with %smid: the second CTA of an SM comes in a fixed order that only roughly follows the
  // first, so which SMs stay single is approximate).  The frames are ranked by an estimate of their a4 time (edges,
  // boxes, and the kept count the edge count implies): the 2S-B longest go to the CTAs expected to stay alone, the next
  // longest are paired with the shortest.  What matters most is that long frames never pair with long ones.
  __shared__ __align__(16) int s_w[K4_MAXPERM];
  __shared__ int s_frame;
  {
    const int B = (int)gridDim.x, S = sm_count, i = (int)blockIdx.x;
    if (B <= S || B > K4_MAXPERM) {
      if (tid == 0) s_frame = i;
    } else {
      for (int g = tid; g < B; g += K4_THREADS) {
        const int ng = n_sorted[g], eg = edge_ctr[g];
        const int kept_est = ng - eg / 5 > ng / 10 ? ng - eg / 5 : ng / 10;
        s_w[g] = eg / 2 + 9 * kept_est + 3 * ng;
      }
      __syncthreads();
      const int alone = 2 * S - B > 0 ? 2 * S - B : 0;             // SMs that get a single CTA
      int want;                                                    // rank in descending weight
      if (i >= S) want = i < 2 * S ? B - 1 - (i - S) : alone + (i - S);   // second CTA of an SM: shortest first
      else if (i >= S - alone) want = i - (S - alone);             // alone on its SM: the longest frames
      else want = alone + i;                                       // first CTA of a shared SM
      if (B >= 2 * S) want = i < S ? i : (i < 2 * S ? B - 1 - (i - S) : S + (i - 2 * S));
      // rank of frame g = frames that weigh more (ties: lower index first); the comparisons of one frame are split over
      // K4_THREADS / Bp threads, four weights per shared load
      const int Bp = (B + 3) & ~3;
      for (int g = tid; g < Bp; g += K4_THREADS) if (g >= B) s_w[g] = INT_MIN;   // padding never outranks a frame
      int* s_rank = reinterpret_cast<int*>(smem);                                // the dynamic area is free until the frame is known
      for (int g = tid; g < B; g += K4_THREADS) s_rank[g] = 0;
      __syncthreads();
      const int parts = B <= K4_THREADS / 2 ? K4_THREADS / B : 1;               // threads per frame
      const int g0 = tid / parts, part = tid - g0 * parts;
      for (int g = g0; g < B; g += K4_THREADS / parts) {
        const int wg = s_w[g];
        const int q4 = Bp / 4, qa = q4 * part / parts, qb = q4 * (part + 1) / parts;
        int rank = 0;
        for (int q = qa; q < qb; ++q) {
          const int4 v = reinterpret_cast<const int4*>(s_w)[q];
          const int h = 4 * q;
          rank += (v.x > wg) | ((v.x == wg) & (h < g));
          rank += (v.y > wg) | ((v.y == wg) & (h + 1 < g));
          rank += (v.z > wg) | ((v.z == wg) & (h + 2 < g));
          rank += (v.w > wg) | ((v.w == wg) & (h + 3 < g));
        }
        if (parts > 1) atomicAdd(&s_rank[g], rank); else s_rank[g] = rank;
      }
      __syncthreads();
      for (int g = tid; g < B; g += K4_THREADS) if (s_rank[g] == want) s_frame = g;
    }
    __syncthreads();
  }
  const int f = s_frame;
  FFPP_PHASE(f, 0);
  if (tid == 0) fd = frames[f];
  const int n = n_sorted[f];
  const int64_t obase = (int64_t)f * kpad;
  const bool overflow = frame_err[f] != 0;                             // k3 ran out of this frame's share of the edge pool
  {
    const uint32_t* hin = hasin + obase / 4;
    for (int i = tid; i < kpad / 4; i += K4_THREADS) {
      st32[i] = overflow ? 0u : hin[i] ^ 0x01010101u;                  // victim of some edge (1) -> U, nobody's victim (0) -> K;
                                                                       // overflow path: everybody starts U
      rem32[i] = 0u;
      blk32[i] = 0u;
    }
  }
  __syncthreads();
  FFPP_PHASE(f, 1);
  if (overflow) overflow_fixed_point<KeyT, K4_THREADS>(st, n, fd, sp_box + obase, sp_key + obase, cellstart + (int64_t)f * kCellStride, cst, tid);
  const int E = overflow ? 0 : edge_ctr[f];
  uint32_t* fe = edges + fd.edge_off;

  // ---- fixed point over this thread's strided slice of the edge list, compacted in place ----
  int mine = E > tid ? (E - tid + K4_THREADS - 1) / K4_THREADS : 0;
  const int nw = (n + 3) >> 2;
#ifdef FFPP_PROFILE_PHASES
  int round_ = 0;
#endif
  uint32_t* const fmine = fe + tid;            // this thread's k-th edge sits at fmine[k * K4_THREADS]
  bool first = true;
  for (;;) {
    if (first) {
      // round 1: every victim is still undecided and no box is removed yet, so an edge only needs its suppressor's
      // state (kept -> the victim is removed, undecided -> the victim is blocked); nothing is dropped, nothing written back
      const uint32_t* p = fmine;
      int k0 = 0;
      for (; k0 + K4_UNROLL <= mine; k0 += K4_UNROLL, p += K4_UNROLL * K4_THREADS) {
        uint32_t ed[K4_UNROLL], ss[K4_UNROLL];
#pragma unroll
        for (int u = 0; u < K4_UNROLL; ++u) ed[u] = p[u * K4_THREADS];
#pragma unroll
        for (int u = 0; u < K4_UNROLL; ++u) ss[u] = st[ed[u] & 0xFFFFu];
#pragma unroll
        for (int u = 0; u < K4_UNROLL; ++u) (ss[u] == ST_K ? rem : blk)[ed[u] >> 16] = 1;
      }
      for (; k0 < mine; ++k0, p += K4_THREADS) {
        const uint32_t ed = *p;
        (st[ed & 0xFFFFu] == ST_K ? rem : blk)[ed >> 16] = 1;
      }
    } else {
      int w = 0;
      const uint32_t* p = fmine;
      uint32_t* q = fmine;
      int k0 = 0;
      for (; k0 + K4_UNROLL <= mine; k0 += K4_UNROLL, p += K4_UNROLL * K4_THREADS) {
        uint32_t ed[K4_UNROLL], sv[K4_UNROLL], ss[K4_UNROLL];
#pragma unroll
        for (int u = 0; u < K4_UNROLL; ++u) ed[u] = p[u * K4_THREADS];      // all loads of the batch before its first store
#pragma unroll
        for (int u = 0; u < K4_UNROLL; ++u) { sv[u] = st[ed[u] >> 16]; ss[u] = st[ed[u] & 0xFFFFu]; }
#pragma unroll
        for (int u = 0; u < K4_UNROLL; ++u) {
          if (sv[u] == ST_U) {
            const uint32_t v = ed[u] >> 16;
            if (ss[u] == ST_K) {
              rem[v] = 1;
            } else if (ss[u] == ST_U) {
              blk[v] = 1;
              *q = ed[u]; q += K4_THREADS; ++w;                           // slots at or before the ones this batch read
            }
          }
        }
      }
      for (; k0 < mine; ++k0, p += K4_THREADS) {
        const uint32_t ed = *p;
        if (st[ed >> 16] == ST_U) {
          const uint32_t v = ed >> 16, sst = st[ed & 0xFFFFu];
          if (sst == ST_K) rem[v] = 1;
          else if (sst == ST_U) { blk[v] = 1; *q = ed; q += K4_THREADS; ++w; }
        }
      }
      mine = w;
    }
    first = false;
    __syncthreads();
    for (int i = tid; i < nw; i += K4_THREADS) {
      const uint32_t s4 = st32[i], r4 = rem32[i], b4 = blk32[i];
      const uint32_t isu = ((s4 | (s4 >> 1)) & 0x01010101u) ^ 0x01010101u;          // 1 in every byte that is U
      const uint32_t val = (r4 << 1) | ((r4 | b4) ^ 0x01010101u);                   // R if rem, K if neither, U if blk only
      st32[i] = s4 | (val & (isu | (isu << 1)));
      rem32[i] = 0u;
      blk32[i] = 0u;
    }
#ifdef FFPP_PROFILE_PHASES
    if (round_ < 8) FFPP_PHASE(f, 8 + round_);
    ++round_;
#endif
    if (!__syncthreads_or(mine != 0)) break;
  }
  FFPP_PHASE(f, 2);

  // ---- kept bitmap + its word prefix (the state bytes are about to be overwritten by the sort arrays) ----
  const int nwords = kpad / 32;
  for (int base = warp * 32; base < kpad; base += K4_THREADS) {
    const int a = base + lane;
    const uint32_t bal = __ballot_sync(0xffffffffu, a < n && st[a] == ST_K);
    if (lane == 0) keptw[base >> 5] = bal;
  }
  __syncthreads();
  int m = 0;
  {
    // each thread owns a contiguous run of words; block-wide exclusive scan of the runs' popcounts
    const int per = (nwords + K4_THREADS - 1) / K4_THREADS;
    const int w0 = tid * per, w1 = w0 + per < nwords ? w0 + per : nwords;
    int s = 0;
    for (int i = w0; i < w1; ++i) s += __popc(keptw[i]);
    int inc = s;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { const int t = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= o) inc += t; }
    if (lane == 31) misc->wsum[warp] = inc;
    __syncthreads();
    int run = inc - s;
#pragma unroll
    for (int w = 0; w < K4_WARPS; ++w) { const int ws = misc->wsum[w]; if (w < warp) run += ws; m += ws; }
    for (int i = w0; i < w1; ++i) { wpre[i] = (uint16_t)run; run += __popc(keptw[i]); }
  }
  if (tid == 0) out_counts[f] = m;
  __syncthreads();
  FFPP_PHASE(f, 3);

  // ---- sort arrays: (key, position) pairs; bitonic network for small sets, LSD radix beyond ----
  constexpr int KB = sizeof(KeyT) * 8;
  const bool bitonic = m <= K4_BITONIC_MAX;
  const int Np = bitonic ? (int)k4_pow2ceil((size_t)(m > 1 ? m : 1)) : m;
  uint8_t* lbase = k4_sort_bytes((size_t)m, sizeof(KeyT)) <= uni_b ? smem : scratch + (size_t)f * k4_scratch_bytes((size_t)K, sizeof(KeyT));
  const size_t kbytes = ((size_t)Np * sizeof(KeyT) + 15) & ~(size_t)15, pbytes = ((size_t)Np * 2 + 15) & ~(size_t)15;
  KeyT* kk = reinterpret_cast<KeyT*>(lbase);
  uint16_t* pp = reinterpret_cast<uint16_t*>(lbase + kbytes);
  KeyT* kk1 = reinterpret_cast<KeyT*>(lbase + kbytes + pbytes);          // second buffer (LSD path only)
  uint16_t* pp1 = reinterpret_cast<uint16_t*>(lbase + 2 * kbytes + pbytes);
  for (int base0 = warp * 32; base0 < n; base0 += 4 * K4_THREADS) {
    KeyT key[4];
    uint32_t bal[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      const int base = base0 + u * K4_THREADS;
      bal[u] = base < n ? keptw[base >> 5] : 0u;
      if ((bal[u] >> lane) & 1u) key[u] = sp_key[obase + base + lane];
    }
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      const int base = base0 + u * K4_THREADS;
      if ((bal[u] >> lane) & 1u) {
        const int i = (int)wpre[base >> 5] + __popc(bal[u] & ((1u << lane) - 1u));
        kk[i] = key[u];
        pp[i] = (uint16_t)(base + lane);
      }
    }
  }
  __syncthreads();
  FFPP_PHASE(f, 4);
  if (bitonic) {
    k4_bitonic<KeyT>(kk, pp, kk1, pp1, m, Np, tid);
  }
  // LSD radix: a pass costs ~4 us per 3600 keys (shared-memory atomics and ballots), so only the SCORE half of the key is
  // sorted; boxes of equal score are then put in candidate-index order by ranking inside their (short) tie group while the
  // list is written out.  A tie group longer than 64 (thousands of equal logits: a degenerate input) takes the full-width
  // sort instead.
  constexpr int IB = KB / 2;                                   // index bits of the key: 16 / 32
  bool tie_fix = false;
  if (!bitonic) {
    for (int shift = IB; shift < KB; shift += 8)
      if (k4_lsd_pass<KeyT>(kk, pp, kk1, pp1, m, shift, hist, misc, tid)) {
        KeyT* tk = kk; kk = kk1; kk1 = tk;
        uint16_t* tp = pp; pp = pp1; pp1 = tp;
      }
    bool big = false;
    for (int r = tid; r + 64 < m; r += K4_THREADS) big |= (kk[r] >> IB) == (kk[r + 64] >> IB);
    tie_fix = !__syncthreads_or(big);
    if (!tie_fix)
      for (int shift = 0; shift < KB; shift += 8)
        if (k4_lsd_pass<KeyT>(kk, pp, kk1, pp1, m, shift, hist, misc, tid)) {
          KeyT* tk = kk; kk = kk1; kk1 = tk;
          uint16_t* tp = pp; pp = pp1; pp1 = tp;
        }
  }
  FFPP_PHASE(f, 5);

  // ---- hand the ordered kept list (key, spatial position) to the flat emit kernel: writing 369 k detections is
  // per-box work with no per-frame structure, and on one SM it was a third of a long frame's a4 time ----
  {
    KeyT* ok = kept_key + (int64_t)f * K;
    uint16_t* op = kept_pos + (int64_t)f * K;
    if (!tie_fix) {
      for (int r = tid; r < m; r += K4_THREADS) { ok[r] = kk[r]; op[r] = pp[r]; }
    } else {
      for (int r = tid; r < m; r += K4_THREADS) {
        const KeyT key = kk[r], sc = key >> IB;
        int g0 = r;
        while (g0 > 0 && (kk[g0 - 1] >> IB) == sc) --g0;           // first element of the tie group (<= 64 long)
        int rank = 0;
        for (int j = g0; j < m; ++j) {
          const KeyT kj = kk[j];
          if ((kj >> IB) != sc) break;
          rank += kj < key;                                        // equal score: the smaller candidate index comes first
        }
        ok[g0 + rank] = key; op[g0 + rank] = pp[r];
      }
    }
  }
#ifdef FFPP_PROFILE_PHASES
  __syncthreads();
  FFPP_PHASE(f, 6);
  if (tid == 0) g_phase[f][7] = ((unsigned long long)n << 40) | ((unsigned long long)E << 16) | (unsigned long long)m;
#endif
}

// a4, second launch — FLAT emit over (frame, output row): row r of frame f is the r-th entry of the ordered kept list;
// the detection is written with its sigmoid score and candidate index (O6) and its centroid is binned into the
// frame's histogram (a5, O7 first half).
constexpr int K4E_THREADS = 256;
template <typename KeyT>
__global__ void __launch_bounds__(K4E_THREADS) k4e_emit(const FrameDesc* __restrict__ frames, const float4* __restrict__ sp_box,
                                                        const KeyT* __restrict__ kept_key, const uint16_t* __restrict__ kept_pos,
                                                        const int* __restrict__ out_counts, Consts cst,
                                                        ffpp_box* __restrict__ out_boxes, uint32_t* __restrict__ hist32) {
  pdl_wait();
  const int f = blockIdx.y;
  const int r = blockIdx.x * K4E_THREADS + threadIdx.x;
  if (r >= out_counts[f]) return;
  const int64_t o = (int64_t)f * cst.top_k + r;
  const KeyT key = kept_key[o];
  const float4 bx = sp_box[(int64_t)f * cst.kpad + kept_pos[o]];
  emit_kept(frames[f], cst, out_boxes + o, bx, logit_of_key<KeyT>(key), idx_of_key<KeyT>(key), hist32);
}

// =====================================================================================================
// a6 — density convolution (north_star (d); the paper's grid-cell x bird loop,
// PAPER.md:L203-208, restated as histogram + separable convolution).
// One CTA per tile of th output rows x up to K5_TW output columns of one frame; th (a multiple of 16, chosen per grid
// width by the host scheduler, FrameDesc::k5_th) gives every thread exactly one y-pass unit.  Everything after one
// coalesced read of the uint16 histogram happens in shared memory and registers, in 64 registers per thread so that
// four CTAs share an SM and one tile's staging latency hides behind another tile's arithmetic:
//  (1) stage: rows y0-RT .. y0+th+RT-1 of the histogram (reflect-folded at the top / bottom of the grid) are copied
//      as they are, 16 bytes per cp.async (LDGSTS: asynchronous, no register staging); a thread owns one 8-column
//      group and walks down the rows;
//  (2) y pass: a thread owns TWO adjacent columns and 16 consecutive output rows: one 32-bit shared load brings a
//      pair of counts, two byte-permutes + one packed subtraction turn them into floats (the 2^23 trick: no I2F), and
//      the 16 pairs of sums are updated with packed fma.rn.f32x2 (FFMA2: two fp32 FMAs per issue slot).  The kernel
//      is symmetric, so only RT + 1 (w_k, w_k) tap pairs live in registers.  The sums stay in registers across a
//      barrier and are then written OVER the staged histogram (the two arrays share their shared memory) as
//      s_t[row pair][column] = (t[2p][x], t[2p+1][x]);
//  (3) mirror: window columns outside the grid are reflections of computed ones (reflect border, O7);
//  (4) x pass: a thread owns one ROW PAIR and eight consecutive columns: the packed lanes are now the two rows, so the
//      same (w_k, w_k) tap pairs serve and an output costs exactly 2 RT + 1 FFMA2 per two cells; 16-byte shared loads
//      (row-pair pitch = 2 mod 4 float2: a quarter warp of eight row pairs is conflict-free), two 32-byte sectors
//      written per thread.
// Radii above K5_PACKED_MAX_RT (the tap pairs would not fit the register file) take scalar FMAs with constant-bank taps.
// The tap loops are fully unrolled for the compile-time radius bucket RT >= R (taps zero-padded to RT).
// HBM traffic: 2 bytes per cell of histogram (L2 hits: a4 wrote it microseconds earlier) + one 4-byte store per cell.
// =====================================================================================================
constexpr int K5_THREADS = 256;
constexpr int K5_TW = 256;                      // output columns per CTA at most (wider grids are tiled in x)
constexpr int K5_PACKED_MAX_RT = 12;
constexpr int K5_RB = 16;                       // output rows of one y-pass unit

__host__ __device__ inline int k5_tile_w(int gw) { return gw < K5_TW ? ((gw + 7) & ~7) : K5_TW; }      // multiple of 8
// column pairs the y pass of one tile computes at most (an x-tiled grid adds the RT halo columns on both sides)
__host__ __device__ inline int k5_npair_max(int gw, int RT) { return gw <= K5_TW ? (gw + 1) / 2 : (K5_TW + 2 * RT) / 2 + 1; }
__host__ __device__ inline int k5_tile_h(int gw, int gh, int RT) {        // multiple of 16; units of the y pass <= K5_THREADS
  int nb = K5_THREADS / k5_npair_max(gw, RT);
  if (nb < 1) nb = 1;
  const int cap = (gh + 15) & ~15;
  return K5_RB * nb < cap ? K5_RB * nb : cap;
}
__host__ __device__ inline int k5_pitch_t(int tw, int RT) {               // float2 per row pair: >= tw + 2 RT + 2, = 2 mod 4
  const int need = tw + 2 * RT + 2;
  return ((need - 2 + 3) / 4) * 4 + 2;
}
__host__ __device__ inline int k5_pitch_h(int tw, int RT) { return (tw + 2 * RT + 7 + 8 + 7) & ~7; }  // staged uint16 columns, multiple of 8
__host__ __device__ inline size_t k5_tile_smem(int tw, int th, int RT) {  // the two arrays alias
  const size_t hb = sizeof(uint16_t) * (size_t)(th + 2 * RT) * k5_pitch_h(tw, RT);
  const size_t tb = sizeof(float2) * (size_t)(th / 2) * k5_pitch_t(tw, RT);
  return ((hb > tb ? hb : tb) + 15) & ~(size_t)15;
}
__host__ __device__ inline size_t k5_smem_bytes(int gw_max, int gh_max, int RT) {   // largest tile any grid up to gw_max x gh_max needs
  size_t m = 0;
  for (int gw = 8; gw <= ((gw_max + 7) & ~7); gw += 8) {
    const size_t b = k5_tile_smem(k5_tile_w(gw), k5_tile_h(gw, gh_max, RT), RT);
    if (b > m) m = b;
  }
  return m;
}
__host__ __device__ inline int k5_tiles_x(int gw) { const int tw = k5_tile_w(gw); return (gw + tw - 1) / tw; }
__host__ __device__ inline int k5_tiles(int gw, int gh, int RT) {
  const int th = k5_tile_h(gw, gh, RT);
  return k5_tiles_x(gw) * ((gh + th - 1) / th);
}

__device__ __forceinline__ int k5_fold(int i, const int n) {
  i = i < 0 ? -i - 1 : (i >= n ? 2 * n - 1 - i : i);
  return min(max(i, 0), n - 1);                  // beyond one fold only zero-padded taps look: any in-range cell will do
}
__device__ __forceinline__ void cp_async16(void* dst_smem, const void* src_gmem) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem_u32(dst_smem)), "l"(src_gmem) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }
// u / d for 0 <= u < 2^20 with inv = the correctly rounded 1 / d: (u + 0.5) / d is at least 0.5 / d away from every integer, far more than
// the rounding error of the product
__device__ __forceinline__ int fast_div(const int u, const float inv) { return (int)(((float)u + 0.5f) * inv); }
// packed fp32 pairs (FFMA2 / FADD2)
__device__ __forceinline__ unsigned long long pk2(const float lo, const float hi) {
  unsigned long long r; asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi)); return r;
}
__device__ __forceinline__ void unpk2(const unsigned long long v, float& lo, float& hi) { asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v)); }
__device__ __forceinline__ unsigned long long fma2(const unsigned long long a, const unsigned long long b, const unsigned long long c) {
  unsigned long long d; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c)); return d;
}
__device__ __forceinline__ unsigned long long add2(const unsigned long long a, const unsigned long long b) {
  unsigned long long d; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d;
}

template <int RT>
__global__ void __launch_bounds__(K5_THREADS, (RT <= K5_PACKED_MAX_RT ? 4 : 2)) k5_density(const FrameDesc* __restrict__ frames, Consts cst,
                                                                                         const uint16_t* __restrict__ hist16,
                                                                                         float* __restrict__ out_density) {
  extern __shared__ __align__(16) uint8_t s_k5[];
  constexpr bool kPacked = RT <= K5_PACKED_MAX_RT;
  constexpr int RB = K5_RB, NW = RB + 2 * RT;
  const int f = blockIdx.y;
  const FrameDesc* fd = &frames[f];
  if ((int)blockIdx.x >= fd->k5_tiles) return;                // the descriptor table is older than the whole run
  pdl_wait();
  const int gw = fd->gw, gh = fd->gh;
  const int tw = k5_tile_w(gw), th = fd->k5_th;
  int ty = (int)blockIdx.x, tx = 0;
  if (gw > tw) { const int tiles_x = (gw + tw - 1) / tw; ty = (int)blockIdx.x / tiles_x; tx = (int)blockIdx.x - ty * tiles_x; }
  const int x0 = tx * tw, y0 = ty * th;
  const int x1 = min(gw, x0 + tw);
  const int cx0 = tx > 0 ? x0 - RT : 0, cx1 = min(gw, x1 + (x1 < gw ? RT : 0));   // columns the y pass must compute
  const int sx0 = cx0 & ~7;                                  // first staged column (16-byte copies)
  const int Ph = k5_pitch_h(tw, RT), Pt = k5_pitch_t(tw, RT);
  uint16_t* s_h = reinterpret_cast<uint16_t*>(s_k5);         // [th + 2 RT][Ph]: staged histogram rows, column gx - sx0
  unsigned long long* s_t = reinterpret_cast<unsigned long long*>(s_k5);   // [th / 2][Pt] (t[2p][x], t[2p+1][x]); ALIASES s_h
  constexpr int OD = RT & 1;                                 // s_t column of grid column gx: gx - (x0 - RT) + OD (even gx <-> even column)
  const int tid = threadIdx.x;
  const uint16_t* hsrc = hist16 + fd->dens_off;

  // ---- (1) stage: 8 cells (16 bytes) per copy; a thread keeps its column group and walks down the rows ----
  {
    const int ng = (cx1 - sx0 + 7) >> 3;                    // 8-column groups per row (<= 37)
    const int nrows = th + 2 * RT;
    const float inv_ng = __frcp_rn((float)ng);
    const int rstep = fast_div(K5_THREADS, inv_ng);
    const int r0 = fast_div(tid, inv_ng), g = tid - r0 * ng;
    const bool vec = (((uintptr_t)hsrc & 15) == 0) && ((gw & 7) == 0);
    if (r0 < rstep) {
      const int gx = sx0 + 8 * g;
      uint16_t* dst = s_h + r0 * Ph + 8 * g;
      if (vec && y0 - RT >= 0 && y0 + th + RT <= gh) {        // interior tile: no fold, one pointer bump per copy
        const uint16_t* src = hsrc + (y0 - RT + r0) * gw + gx;
        uint32_t d32 = smem_u32(dst);
        for (int r = r0; r < nrows; r += rstep, d32 += (uint32_t)(rstep * Ph * 2), src += rstep * gw)
          asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(d32), "l"(src) : "memory");
      } else {
        for (int r = r0; r < nrows; r += rstep, dst += rstep * Ph) {
          const uint16_t* src = hsrc + k5_fold(y0 - RT + r, gh) * gw + gx;
          if (vec) {                                          // gw % 8 == 0: a group never straddles the row end
            cp_async16(dst, src);
          } else {
#pragma unroll
            for (int e = 0; e < 8; ++e) dst[e] = gx + e < gw ? src[e] : (uint16_t)0;
          }
        }
      }
    }
    cp_async_wait_all();
  }
  __syncthreads();

  // ---- (2) y pass: one unit (column pair, 16 rows) per thread, sums in registers ----
  const int px0 = cx0 & ~1;                                 // pairs start on an even column (>= sx0)
  const int npair = (cx1 - px0 + 1) >> 1;
  const int q = fast_div(tid, __frcp_rn((float)npair)), c = tid - q * npair;
  const bool yact = q < th / RB && y0 + RB * q < gh;       // else: no such unit, or a block of rows below the grid
  unsigned long long wp[kPacked ? RT + 1 : 1];              // (w_k, w_k) for k = 0 .. RT; w_(2RT - k) = w_k
  if constexpr (kPacked) {
#pragma unroll
    for (int k = 0; k <= RT; ++k) wp[k] = pk2(cst.taps_pad[k], cst.taps_pad[k]);
  }
  unsigned long long acc[RB];
#pragma unroll
  for (int m = 0; m < RB; ++m) acc[m] = 0ull;
  if (yact) {
    const uint32_t* col = reinterpret_cast<const uint32_t*>(s_h + (RB * q) * Ph + (px0 - sx0) + 2 * c);
    const unsigned long long magic = pk2(-8388608.0f, -8388608.0f);
#pragma unroll
    for (int r = 0; r < NW; ++r) {
      const uint32_t v = col[r * (Ph / 2)];
      // count -> float without I2F: 0x4B000000 | c is the float 2^23 + c
      unsigned long long vv = pk2(__uint_as_float(__byte_perm(v, 0x4B000000u, 0x7610)), __uint_as_float(__byte_perm(v, 0x4B000000u, 0x7632)));
      if constexpr (kPacked) {
        vv = add2(vv, magic);
#pragma unroll
        for (int m = 0; m < RB; ++m) {
          const int k = r - m;                              // compile-time after unrolling
          if (k >= 0 && k <= 2 * RT) acc[m] = fma2(wp[k <= RT ? k : 2 * RT - k], vv, acc[m]);
        }
      } else {
        float v0, v1;
        unpk2(vv, v0, v1);
        v0 -= 8388608.0f; v1 -= 8388608.0f;
#pragma unroll
        for (int m = 0; m < RB; ++m) {
          const int k = r - m;
          if (k >= 0 && k <= 2 * RT) {
            float a0, a1;
            unpk2(acc[m], a0, a1);
            acc[m] = pk2(fmaf(cst.taps_pad[k], v0, a0), fmaf(cst.taps_pad[k], v1, a1));
          }
        }
      }
    }
  }
  __syncthreads();                                          // every read of the staged histogram is done: s_t may overwrite it
  if (yact) {
    // acc[m] = (t[m][2c], t[m][2c+1]) -> rows paired: (t[m][2c], t[m+1][2c]), (t[m][2c+1], t[m+1][2c+1]): one 16-byte store
    ulonglong2* dst = reinterpret_cast<ulonglong2*>(s_t + (RB / 2 * q) * Pt + (px0 - (x0 - RT) + OD) + 2 * c);
#pragma unroll
    for (int m = 0; m < RB; m += 2) {
      float a0, a1, b0, b1;
      unpk2(acc[m], a0, a1); unpk2(acc[m + 1], b0, b1);
      dst[(m / 2) * (Pt / 2)] = make_ulonglong2(pk2(a0, b0), pk2(a1, b1));
    }
  }
  __syncthreads();
  // ---- (3) mirror pass: the columns of the window that lie outside the grid are reflections of computed ones ----
  {
    const int nct = (x1 - x0) + 2 * RT;
    const int lo = cx0 - (x0 - RT), hi = cx1 - (x0 - RT);   // computed range, in window columns
    const int nfill = lo + (nct - hi);
    if (nfill) {                                            // block-uniform
      const float inv = __frcp_rn((float)nfill);
      for (int u = tid; u < nfill * (th / 2); u += K5_THREADS) {
        const int y = fast_div(u, inv), e = u - y * nfill;
        const int wc = e < lo ? e : hi + (e - lo);
        const int gx = min(max(k5_fold(x0 - RT + wc, gw), cx0), cx1 - 1);
        s_t[y * Pt + wc + OD] = s_t[y * Pt + (gx - (x0 - RT)) + OD];
      }
      __syncthreads();
    }
  }

  // ---- (4) x pass: unit = (row pair p, 8-column group g); consecutive lanes take consecutive groups of one row pair,
  // so a warp's stores cover whole 128-byte lines (the 4-way bank conflict of its 16-byte shared loads costs a few
  // hundred cycles per tile; stores that scatter over 32 rows cost thousands) ----
  float* out = out_density + fd->dens_off;
  constexpr int NWX = 8 + 2 * RT;                           // window of one 8-output block
  constexpr int NL = (NWX + OD + 1) / 2;                    // 16-byte loads (two columns each)
  const int ngrp = tw / 8;
  const float inv_ngrp = __frcp_rn((float)ngrp);
  for (int u = tid; u < (th / 2) * ngrp; u += K5_THREADS) {
    const int yp = fast_div(u, inv_ngrp), g = u - yp * ngrp;
    const int gy = y0 + 2 * yp, gx = x0 + 8 * g;
    if (gy >= gh || gx >= gw) continue;
    const ulonglong2* row2 = reinterpret_cast<const ulonglong2*>(s_t + yp * Pt + 8 * g);
    unsigned long long xa[8];
#pragma unroll
    for (int m = 0; m < 8; ++m) xa[m] = 0ull;
#pragma unroll
    for (int i = 0; i < NL; ++i) {
      const ulonglong2 t2 = row2[i];
#pragma unroll
      for (int h = 0; h < 2; ++h) {
        const int r = 2 * i + h - OD;                       // window index (compile-time)
        const unsigned long long vv = h ? t2.y : t2.x;
        if (r >= 0 && r < NWX) {
#pragma unroll
          for (int m = 0; m < 8; ++m) {
            const int k = r - m;
            if (k >= 0 && k <= 2 * RT) {
              if constexpr (kPacked) {
                xa[m] = fma2(wp[k <= RT ? k : 2 * RT - k], vv, xa[m]);
              } else {
                float v0, v1, a0, a1;
                unpk2(vv, v0, v1); unpk2(xa[m], a0, a1);
                xa[m] = pk2(fmaf(cst.taps_pad[k], v0, a0), fmaf(cst.taps_pad[k], v1, a1));
              }
            }
          }
        }
      }
    }
    float r0v[8], r1v[8];
#pragma unroll
    for (int m = 0; m < 8; ++m) unpk2(xa[m], r0v[m], r1v[m]);
#pragma unroll
    for (int rr = 0; rr < 2; ++rr) {
      if (gy + rr >= gh) break;
      const float* v = rr ? r1v : r0v;
      float* dst = out + (gy + rr) * gw + gx;
      if ((((uintptr_t)dst & 15) == 0) && gx + 8 <= gw) {
        reinterpret_cast<float4*>(dst)[0] = make_float4(v[0], v[1], v[2], v[3]);
        reinterpret_cast<float4*>(dst)[1] = make_float4(v[4], v[5], v[6], v[7]);
      } else {
#pragma unroll
        for (int m = 0; m < 8; ++m)
          if (gx + m < gw) dst[m] = v[m];
      }
    }
  }
}

// =====================================================================================================
// Host-buffer path only (ffpp_run_host): copy rows [0, count) of every frame's kept list from the device staging
// buffer straight into the caller's PINNED host array through its device alias (zero-copy stores over PCIe): one
// launch instead of one cudaMemcpyAsync per frame.
// =====================================================================================================
constexpr int KH_THREADS = 256;
__global__ void __launch_bounds__(KH_THREADS) kh_copy_kept_rows(const ffpp_box* __restrict__ src, const int* __restrict__ counts,
                                                                int K, ffpp_box* __restrict__ dst_host_alias) {
  const int f = blockIdx.y;
  const int n = counts[f];
  const int64_t base = (int64_t)f * K * 3;                     // in 8-byte words: a record is three of them
  const uint2* s = reinterpret_cast<const uint2*>(src) + base;
  uint2* d = reinterpret_cast<uint2*>(dst_host_alias) + base;
  for (int i = blockIdx.x * KH_THREADS + threadIdx.x; i < n * 3; i += gridDim.x * KH_THREADS) d[i] = s[i];
}

// =====================================================================================================
// Calibration only (ffpp_debug_stream_read): a plain coalesced read of a device buffer, 16 bytes per thread per
// step.  bench.py times it over the raw head output under the same cold-L2 regime as a1 to show what a pure read
// of THIS many bytes achieves on this GPU (tens of MB are far from the asymptote the 2 GB copy peak is measured at).
// =====================================================================================================
__global__ void __launch_bounds__(256) k0_stream_read(const uint4* __restrict__ p, int64_t n16, uint32_t* __restrict__ sink) {
  uint32_t acc = 0;
  for (int64_t i = (int64_t)blockIdx.x * 256 + threadIdx.x; i < n16; i += (int64_t)gridDim.x * 256) {
    const uint4 v = __ldg(p + i);
    acc ^= v.x ^ v.y ^ v.z ^ v.w;
  }
  if (acc == 0x9E3779B9u) sink[0] = acc;             // keeps the loads alive; practically never taken
}

}  // namespace ffpp
