// Shared declarations of the CUDA path (sm_100a only).  Nothing here is shared with oracle/.
#pragma once
#include <cuda_fp16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/ffpp.h"

namespace ffpp {

constexpr int kMaxLevels = 4;
constexpr int kMaxRadius = 32;
constexpr int kNmsTile = 64;        // IoU tile edge = bits per suppression word

// ---- a0: frame descriptor table (device copy built by the host scheduler, one per frame) ----
struct FrameDesc {
  int64_t cand_off;                 // first row of the frame in the flat candidate stream
  int64_t mask_off;                 // first uint64 word of the frame's suppression mask
  int64_t dens_off;                 // first float of the frame's density grid
  int32_t N;                        // candidates
  int32_t W, H;                     // pixels
  int32_t nmax;                     // min(N, top_k): host-known bound on boxes entering NMS
  int32_t nbmax;                    // ceil(nmax / 64): mask layout stride
  int32_t gw, gh;                   // density grid
  int32_t tiles_x, tiles_y;         // density tiles
  int32_t lvl_start[kMaxLevels];    // first candidate of level l within the frame
  int32_t lvl_gw[kMaxLevels];       // W / s_l
  int32_t pad_;
};

// Method constants shared by all kernels (passed by value).
struct Consts {
  float logit_thr;                  // T
  float iou_thr, iou_thr_hi, iou_thr_lo;
  int32_t iou_fast;                 // 1: the guard-banded multiply test is valid for this threshold
  int32_t top_k;
  int32_t num_levels;
  int32_t stride_log2[kMaxLevels];
  int32_t cell_px;
  int32_t radius;
  float taps[2 * kMaxRadius + 1];
};

// ---- suppression-mask layout: row-block major, upper-triangular, row-major inside a row block ----
// word (row r, column block cb >= r/64) of a frame lives at
//   mask_off + rb_off(rb) + (r % 64) * (nbmax - rb) + (cb - rb),  rb = r / 64
__host__ __device__ inline int64_t mask_rb_off(int rb, int nbmax) {
  return (int64_t)kNmsTile * ((int64_t)rb * nbmax - (int64_t)rb * (rb - 1) / 2);
}
__host__ __device__ inline int64_t mask_words(int nbmax) { return (int64_t)kNmsTile * nbmax * (nbmax + 1) / 2; }

// ---- monotone float -> unsigned maps (descending: larger score -> smaller key) ----
__device__ __forceinline__ uint32_t desc_key16(uint16_t h) {
  if (h == 0x8000u) h = 0;                                   // -0 -> +0
  uint32_t asc = (h & 0x8000u) ? (uint32_t)(~h & 0xFFFFu) : (uint32_t)(h | 0x8000u);
  return (~asc) & 0xFFFFu;
}
__device__ __forceinline__ uint32_t desc_key32(float z) {
  uint32_t u = __float_as_uint(z);
  if (u == 0x80000000u) u = 0;
  uint32_t asc = (u & 0x80000000u) ? ~u : (u | 0x80000000u);
  return ~asc;
}

// ---- PTX helpers: mbarrier + 1-D bulk async copy (TMA engine, UBLKCP in SASS) ----
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_fence_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void* dst_smem, const void* src_gmem, uint32_t bytes, uint64_t* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                   smem_u32(dst_smem)),
               "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar))
               : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  asm volatile(
      "{\n\t"
      ".reg .pred p;\n\t"
      "MBAR_WAIT:\n\t"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
      "@p bra MBAR_DONE;\n\t"
      "bra MBAR_WAIT;\n\t"
      "MBAR_DONE:\n\t"
      "}" ::"r"(smem_u32(bar)),
      "r"(parity)
      : "memory");
}

}  // namespace ffpp
