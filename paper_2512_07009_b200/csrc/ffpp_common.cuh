// Shared declarations of the CUDA path (sm_100a only).  Nothing here is shared with oracle/.
#pragma once
#include <cuda_fp16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/ffpp.h"

namespace ffpp {

constexpr int kMaxLevels = 4;
constexpr int kMaxRadius = 32;
constexpr int kBlk = 32;            // kpad granularity
constexpr int kMaxTopK = 24576;     // positions fit 15 bits (adjacency entries carry one more bit)
constexpr int kCntStride = 32;      // ints between two frames' survivor counters: one 128-byte line each, so the a1 atomics
                                    // of different frames go to different L2 lines
constexpr int kMaxCells = 16384;    // spatial cells per frame (<= 128 x 128)
constexpr int kCellStride = kMaxCells + 8;   // uint16 entries per frame in the cell-start table

// ---- a0: frame descriptor table (device copy built by the host scheduler, one per frame) ----
struct FrameDesc {
  int64_t cand_off;                 // first row of the frame in the flat candidate stream
  int64_t dens_off;                 // first float of the frame's density grid (= first uint16 of its histogram)
  int64_t edge_off;                 // first entry of the frame's suppression-edge pool
  int32_t edge_cap;                 // entries in the frame's pool
  int32_t N;                        // candidates
  int32_t W, H;                     // pixels
  int32_t nmax;                     // min(N, top_k): host-known bound on boxes entering NMS
  int32_t gw, gh;                   // density grid
  int32_t hshift;                   // spatial cell = 2^hshift pixels wide ...
  int32_t hshift_y;                 // ... and 2^hshift_y pixels tall (8 x 16 when that fits kMaxCells: a window row is a
                                    // contiguous range whatever its width in cells, so narrow cells trim it for free)
  int32_t cgw, cgh;                 // spatial cell grid (cgw * cgh <= kMaxCells), covers [0,W) x [0,H)
  int32_t lvl_start[kMaxLevels];    // first candidate of level l within the frame
  int32_t lvl_gw[kMaxLevels];       // W / s_l
  int32_t k5_th, k5_tiles;          // a6: output rows per tile (multiple of 16) and tiles of this frame
};

// Method constants shared by all kernels (passed by value).
struct Consts {
  float logit_thr;                  // T
  float iou_thr, iou_thr_hi, iou_thr_lo;
  int32_t iou_fast;                 // 1: the guard-banded multiply test is valid for this threshold
  float rho;                        // partner-centre window half-extent in units of the box's own width/height (a3)
  int32_t top_k;
  int32_t kpad;                     // top_k rounded up to a multiple of 32: per-frame stride of the spatial arrays
  int32_t num_levels;
  int32_t stride_log2[kMaxLevels];
  int32_t cell_px;
  float cell_inv;                   // 1 / cell_px if cell_px is a power of two (the product is then exact), else 0
  int32_t radius;
  float taps[2 * kMaxRadius + 1];
  int32_t radius_t;                 // compile-time radius bucket RT >= radius that a6 runs with
  float taps_pad[2 * kMaxRadius + 1];   // taps centred in a 2 RT + 1 window, zero outside the real radius
};

// ---- development aid: per-phase %globaltimer stamps (compiled only with -DFFPP_PROFILE_PHASES) ----
#ifdef FFPP_PROFILE_PHASES
__device__ unsigned long long g_phase[4096][16];
__device__ __forceinline__ unsigned long long gtimer() { unsigned long long t; asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t)); return t; }
__device__ unsigned long long g_phase2[4096][16];
#define FFPP_PHASE(f, i) do { if (threadIdx.x == 0) g_phase[(f)][(i)] = gtimer(); } while (0)
#define FFPP_PHASE2(f, i) do { if (threadIdx.x == 0) g_phase2[(f)][(i)] = gtimer(); } while (0)
#else
#define FFPP_PHASE(f, i) do { } while (0)
#define FFPP_PHASE2(f, i) do { } while (0)
#endif

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

// inverse maps: the key carries the score logit exactly (with -0 canonicalised to +0, which has the same sigmoid)
__device__ __forceinline__ float logit_of_key16(uint32_t k16) {
  const uint32_t asc = (~k16) & 0xFFFFu;
  const uint16_t h = (asc & 0x8000u) ? (uint16_t)(asc & 0x7FFFu) : (uint16_t)(~asc & 0xFFFFu);
  return __half2float(__ushort_as_half(h));
}
__device__ __forceinline__ float logit_of_key32(uint32_t k32) {
  const uint32_t asc = ~k32;
  return __uint_as_float((asc & 0x80000000u) ? (asc & 0x7FFFFFFFu) : ~asc);
}
template <typename KeyT> __device__ __forceinline__ int idx_of_key(KeyT key) {
  return sizeof(KeyT) == 4 ? (int)((uint32_t)key & 0xFFFFu) : (int)(uint32_t)((uint64_t)key & 0xFFFFFFFFu);
}
template <typename KeyT> __device__ __forceinline__ float logit_of_key(KeyT key) {
  return sizeof(KeyT) == 4 ? logit_of_key16((uint32_t)key >> 16) : logit_of_key32((uint32_t)((uint64_t)key >> 32));
}

// ---- spatial cells (a2 bins with these, a3 builds its windows with these: the same two functions on both sides) ----
__device__ __forceinline__ float box_centre(const float lo, const float hi) { return __fmul_rn(0.5f, __fadd_rn(lo, hi)); }
__device__ __forceinline__ int cell_coord(const float v, const float cmax, const int hshift) {
  return (int)fminf(fmaxf(v, 0.0f), cmax) >> hshift;          // NaN -> 0; monotone non-decreasing in v
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
  const float score = __fdiv_rn(1.0f, __fadd_rn(1.0f, expf(-logit)));
  float2* d2 = reinterpret_cast<float2*>(dst);                 // a record is 24 bytes, rows start 8-byte aligned
  d2[0] = make_float2(bx.x, bx.y);
  d2[1] = make_float2(bx.z, bx.w);
  d2[2] = make_float2(score, __int_as_float(idx));
  const float cx = __fmul_rn(__fadd_rn(bx.x, bx.z), 0.5f);
  const float cy = __fmul_rn(__fadd_rn(bx.y, bx.w), 0.5f);
  if (cx >= 0.0f && cx < (float)fd.W && cy >= 0.0f && cy < (float)fd.H) {
    const float cell = (float)cst.cell_px;
    // cell_inv != 0: cell_px is a power of two, x * (1/cell) IS the correctly rounded x / cell
    const int cxi = (int)floorf(cst.cell_inv != 0.0f ? __fmul_rn(cx, cst.cell_inv) : __fdiv_rn(cx, cell));
    const int cyi = (int)floorf(cst.cell_inv != 0.0f ? __fmul_rn(cy, cst.cell_inv) : __fdiv_rn(cy, cell));
    const int64_t h = fd.dens_off + (int64_t)cyi * fd.gw + cxi;
    atomicAdd(&hist32[h >> 1], 1u << (16 * (int)(h & 1)));
  }
}

__device__ __forceinline__ unsigned long long warp_sum_u64(unsigned long long v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// ---- programmatic dependent launch: a kernel launched with the stream-serialisation attribute may start before its
// predecessor in the stream has finished (its launch latency overlaps the predecessor's tail); this waits until the
// predecessor has completed and its writes are visible.  A no-op for a kernel launched the ordinary way.
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

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
