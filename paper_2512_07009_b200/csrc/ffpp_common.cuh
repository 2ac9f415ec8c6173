// Shared declarations of the CUDA path (sm_100a only).  Nothing here is shared with oracle/.
#pragma once
#include <cuda_fp16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/ffpp.h"

namespace ffpp {

constexpr int kMaxLevels = 4;
constexpr int kMaxRadius = 32;
constexpr int kNmsTile = 64;        // dense mode: IoU tile edge = bits per suppression word
constexpr int kBlk = 32;            // tiled mode: boxes per spatial block = bits per suppression word = one warp

// ---- a0: frame descriptor table (device copy built by the host scheduler, one per frame) ----
struct FrameDesc {
  int64_t cand_off;                 // first row of the frame in the flat candidate stream
  int64_t mask_off;                 // dense mode: first uint64 word of the frame's suppression mask
  int64_t dens_off;                 // first float of the frame's density grid (= first uint16 of its histogram)
  int64_t slot_off;                 // tiled mode: first suppression-word slot of the frame's pool
  int32_t slot_cap;                 // tiled mode: slots in the frame's pool
  int32_t N;                        // candidates
  int32_t W, H;                     // pixels
  int32_t nmax;                     // min(N, top_k): host-known bound on boxes entering NMS
  int32_t nbmax;                    // dense mode: ceil(nmax / 64): mask layout stride
  int32_t gw, gh;                   // density grid
  int32_t hshift;                   // Hilbert cell = 2^hshift pixels (256 x 256 cells cover the frame)
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

// ---- dense-mode suppression-mask layout: row-block major, upper-triangular, row-major inside a row block ----
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

// ---- IoU of the definition: every operation a separately rounded fp32 op ----
__device__ __forceinline__ float box_area(const float4 b) {
  return __fmul_rn(__fsub_rn(b.z, b.x), __fsub_rn(b.w, b.y));
}
// strict overlap in both axes; false => inter == 0 => IoU > thr is false for every thr >= 0
__device__ __forceinline__ bool boxes_overlap(const float4 a, const float4 b) {
  return (a.z > b.x) & (b.z > a.x) & (a.w > b.y) & (b.w > a.y);
}
// IoU(a, b) > thr.  The comparison uses a guard-banded multiply (inter vs thr*union with a 2^-20 relative band)
// that provably agrees with the correctly rounded division, which is evaluated only inside the band.
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

// ---- a4 epilogue + a5: write one kept detection and bin its centroid (SURVEY §8(c) O6, O7 first half) ----
// The histogram is uint16 per cell (a count never exceeds top_k <= 24576), two cells per 32-bit word, indexed by the
// global cell number dens_off + cy*gw + cx; the 32-bit atomicAdd on the containing word cannot carry between halves.
__device__ __forceinline__ void emit_kept(const FrameDesc& fd, const Consts& cst, ffpp_box* __restrict__ dst, const float4 bx,
                                          const float logit, const int idx, uint32_t* __restrict__ hist32) {
  ffpp_box o;
  o.x1 = bx.x; o.y1 = bx.y; o.x2 = bx.z; o.y2 = bx.w;
  o.score = __fdiv_rn(1.0f, __fadd_rn(1.0f, expf(-logit)));
  o.cand_index = idx;
  *dst = o;
  const float cx = __fmul_rn(__fadd_rn(bx.x, bx.z), 0.5f);
  const float cy = __fmul_rn(__fadd_rn(bx.y, bx.w), 0.5f);
  if (cx >= 0.0f && cx < (float)fd.W && cy >= 0.0f && cy < (float)fd.H) {
    const float cell = (float)cst.cell_px;
    const int cxi = (int)floorf(__fdiv_rn(cx, cell));
    const int cyi = (int)floorf(__fdiv_rn(cy, cell));
    const int64_t h = fd.dens_off + (int64_t)cyi * fd.gw + cxi;
    atomicAdd(&hist32[h >> 1], 1u << (16 * (int)(h & 1)));
  }
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
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
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
