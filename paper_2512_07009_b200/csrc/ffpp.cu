// libffpp — host side: ragged-batch scheduler (a0), workspace, C ABI (include/ffpp.h).
// Build: nvcc -gencode arch=compute_100a,code=sm_100a -lineinfo -O3 -shared -Xcompiler -fPIC
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "../../include/ffpp_debug.h"
#include "ffpp_kernels.cuh"

using namespace ffpp;

// compile-time radii of the a6 kernel; a run uses the smallest one >= floor(truncate * sigma)
#define FFPP_K5_RADII(X) X(2) X(3) X(4) X(5) X(6) X(7) X(8) X(9) X(10) X(12) X(14) X(16) X(20) X(24) X(28) X(32)
#define FFPP_K5_LIST(RT) RT,

namespace {

thread_local std::string g_create_error;

struct DeviceMeta {           // one pinned block + one device block, uploaded with a single copy
  size_t frames_off, cand_off_off, block_frame_off, bytes;
};

DeviceMeta meta_layout(int max_frames, int64_t max_total_candidates) {
  DeviceMeta m;
  size_t o = 0;
  m.frames_off = o; o += sizeof(FrameDesc) * (size_t)max_frames;
  o = (o + 15) & ~(size_t)15;
  m.cand_off_off = o; o += sizeof(int64_t) * ((size_t)max_frames + 1);
  o = (o + 15) & ~(size_t)15;
  m.block_frame_off = o; o += sizeof(int32_t) * ((size_t)(max_total_candidates / K1_BLOCK) + 2);
  m.bytes = (o + 15) & ~(size_t)15;
  return m;
}

}  // namespace

struct ffpp_handle {
  ffpp_params p;
  Consts cst;
  bool half = false;
  int key_bytes = 8;
  int kpad = 0;                       // top_k rounded up to 32: per-frame stride of the spatial arrays
  int sm_count = 148;
  int max_frame_cand = 0;
  int64_t max_total_cells = 0;
  int64_t edge_cap_total = 0;         // suppression-edge pool, entries
  int64_t edges_per_box = 16;
  std::string err;

  // device workspace
  void* d_surv_keys = nullptr;
  int* d_counters = nullptr;          // 4 x max_frames: survivor counts | top-K counts | edge counters | frame_err
  float4* d_sel_box = nullptr;        // a2 scratch: decoded boxes in selection order; 
  float4* d_sp_box = nullptr;         // boxes in spatial order (row-major 16-px cell of the centre), stride kpad per frame
  void* d_sp_key = nullptr;
  uint8_t* d_hasin = nullptr;         // a3 -> a4: one byte per box, 1 = victim of at least one edge
  void* d_kept_key = nullptr;         // a4: keys of the kept boxes in keep order, top_k per frame
  uint16_t* d_kept_pos = nullptr;     // a4: their spatial positions
  uint8_t* d_k4_scratch = nullptr;    // a4 sort arrays of frames whose kept set does not fit shared memory
  uint16_t* d_cellstart = nullptr;    // kCellStride entries per frame: start position of every spatial cell
  uint32_t* d_edges = nullptr;
  uint32_t* d_hist32 = nullptr;       // a5: uint16 count per density cell, two per word
  int64_t workspace_bytes = 0;
  // a0: cached batch geometries.  A slot owns one device copy of the descriptor block; the host copy is built in a
  // plain (pageable) vector and uploaded with cudaMemcpyAsync, which stages pageable memory before it returns: no
  // pinned block to protect, hence no event and no host synchronisation.
  DeviceMeta ml;
  struct GeoSlot {
    uint8_t* d_meta = nullptr;
    uint64_t hash = 0, last_use = 0;
    int B = -1;
    std::vector<int32_t> N, dims;
    int max_tiles = 0, max_nmax = 0;
    int64_t total_cand = 0, total_cells = 0;
  };
  static constexpr int kGeoSlots = 32;
  GeoSlot geo[kGeoSlots];
  int cur = -1;                         // slot of the last run
  uint64_t use_clock = 0;
  std::vector<uint8_t> h_meta;          // host build area of the descriptor block
  unsigned long long* d_work = nullptr; // a3 work counters (debug): culling tests, exact IoUs, edges
  bool count_work = false;
  // host-buffer path staging (allocated on first ffpp_run_host)
  void* d_in = nullptr;
  ffpp_box* d_out_boxes = nullptr;
  int* d_out_counts = nullptr;
  float* d_out_density = nullptr;
  cudaStream_t s_h2d = nullptr, s_d2h = nullptr;     // copy streams of the chunked host path (created on first use)
  cudaStream_t s_run2 = nullptr;                     // second compute stream of the chunked host path
  ffpp_handle* twin = nullptr;                       // second workspace: odd runs of the chunked host path go through it
  static constexpr int kHostChunks = 6;
  cudaEvent_t ev_up[kHostChunks] = {}, ev_run[kHostChunks] = {};
  // SURVEY §8(f) f1-f3 (ffpp_next.cuh): cached grid tables of f1 / f2 and the component-labelling scratch (grown on demand)
  struct NextGeo {
    void* d_tab = nullptr;
    uint64_t hash = 0, last_use = 0;
    int B = -1;
    std::vector<int32_t> dims;
    int64_t cells = 0;
    int max_cells = 0, max_w = 0, max_h = 0;
  };
  static constexpr int kNextSlots = 8;
  NextGeo ngeo[kNextSlots];
  int32_t* d_ccl_aux = nullptr;
  int64_t ccl_aux_cap = 0;
  unsigned long long* d_ccl_sums = nullptr;
  int64_t ccl_sum_cap = 0;
  int32_t* d_ccl_blk = nullptr;
  int64_t ccl_blk_cap = 0;
  void* d_ent_part = nullptr;
  int64_t ent_part_cap = 0;
  // stage timing
  bool timing = false;
  cudaEvent_t ev[FFPP_NUM_STAGES + 1] = {};
  bool ev_valid = false;

  int* n_sorted() const { return d_counters; }
  int* edge_ctr() const { return d_counters + (size_t)p.max_frames; }
  int* frame_err() const { return d_counters + 2 * (size_t)p.max_frames; }
  int* surv_cnt() const { return d_counters + 3 * (size_t)p.max_frames; }     // kCntStride ints per frame
};

namespace {

int fail(ffpp_handle* h, int code, const std::string& msg) {
  if (h) h->err = msg; else g_create_error = msg;
  return code;
}

int cuda_fail(ffpp_handle* h, cudaError_t e, const char* what) {
  return fail(h, FFPP_ECUDA, std::string(what) + ": " + cudaGetErrorString(e));
}

#define FFPP_CUDA(h, call)                                   \
  do {                                                       \
    cudaError_t e__ = (call);                                \
    if (e__ != cudaSuccess) return cuda_fail(h, e__, #call); \
  } while (0)

bool is_pow2(int v) { return v > 0 && (v & (v - 1)) == 0; }
int ilog2(int v) { int l = 0; while ((1 << l) < v) ++l; return l; }

int64_t frame_candidates(const ffpp_params& p, int W, int H) {
  int64_t n = 0;
  for (int l = 0; l < p.num_levels; ++l) n += (int64_t)W * H / ((int64_t)p.strides[l] * p.strides[l]);
  return n;
}

uint64_t geo_hash(int B, const int32_t* N, const int32_t* dims) {
  uint64_t x = 0x9E3779B97F4A7C15ull ^ (uint64_t)B;
  auto mix = [&](uint64_t v) { x ^= v + 0x9E3779B97F4A7C15ull + (x << 6) + (x >> 2); x *= 0xD6E8FEB86659FD93ull; x ^= x >> 32; };
  for (int f = 0; f < B; ++f) { mix((uint32_t)N[f]); mix(((uint64_t)(uint32_t)dims[2 * f] << 32) | (uint32_t)dims[2 * f + 1]); }
  return x;
}

// a0: find the batch geometry among the cached slots, else validate it, build its descriptor block and upload it
// (one stream-ordered copy from pageable memory: no host synchronisation).  Sets h->cur.
int schedule(ffpp_handle* h, int B, const int32_t* N, const int32_t* dims, cudaStream_t stream) {
  const ffpp_params& p = h->p;
  const uint64_t hash = geo_hash(B, N, dims);
  int lru = 0;
  for (int s = 0; s < ffpp_handle::kGeoSlots; ++s) {
    ffpp_handle::GeoSlot& g = h->geo[s];
    if (g.B == B && g.hash == hash && std::memcmp(N, g.N.data(), sizeof(int32_t) * B) == 0 &&
        std::memcmp(dims, g.dims.data(), sizeof(int32_t) * 2 * B) == 0) {
      g.last_use = ++h->use_clock;
      h->cur = s;
      return FFPP_OK;
    }
    if (g.last_use < h->geo[lru].last_use) lru = s;
  }
  {
    cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
    if (cudaStreamIsCapturing(stream, &cap) == cudaSuccess && cap != cudaStreamCaptureStatusNone)
      return fail(h, FFPP_EINVAL, "batch geometry not cached: run it once outside stream capture first");
    cudaGetLastError();
  }
  FrameDesc* fr = reinterpret_cast<FrameDesc*>(h->h_meta.data() + h->ml.frames_off);
  int64_t* coff = reinterpret_cast<int64_t*>(h->h_meta.data() + h->ml.cand_off_off);
  const int smax = p.strides[p.num_levels - 1];
  const int R = h->cst.radius;
  int64_t cand = 0, cells = 0, edges = 0;
  int max_tiles = 0, max_nmax = 0;
  for (int f = 0; f < B; ++f) {
    const int W = dims[2 * f], H = dims[2 * f + 1];
    if (W <= 0 || H <= 0) return fail(h, FFPP_EINVAL, "frame_dims: W and H must be positive");
    if (W > p.max_frame_w || H > p.max_frame_h) return fail(h, FFPP_ECAPACITY, "frame exceeds max_frame_w/max_frame_h");
    if (W % smax) return fail(h, FFPP_EINVAL, "W must be a multiple of the largest stride");
    if (W % p.cell_px || H % p.cell_px) return fail(h, FFPP_EINVAL, "W and H must be multiples of cell_px");
    FrameDesc d;
    std::memset(&d, 0, sizeof(d));
    int64_t n = 0;
    for (int l = 0; l < p.num_levels; ++l) {
      const int64_t s2 = (int64_t)p.strides[l] * p.strides[l];
      if (((int64_t)W * H) % s2) return fail(h, FFPP_EINVAL, "W*H must be a multiple of stride^2 for every level");
      d.lvl_start[l] = (int32_t)n;
      d.lvl_gw[l] = W / p.strides[l];
      n += (int64_t)W * H / s2;
    }
    if (n != N[f]) return fail(h, FFPP_EINVAL, "N_per_frame[f] != sum_l W*H/s_l^2");
    if (h->key_bytes == 4 && n > 65536) return fail(h, FFPP_ECAPACITY, "frame has more than 65536 candidates (32-bit key handle)");
    if (n > (1 << 20)) return fail(h, FFPP_ECAPACITY, "frame has more than 2^20 candidates");
    d.cand_off = cand; d.N = (int32_t)n; d.W = W; d.H = H;
    d.nmax = (int32_t)(n < p.top_k ? n : p.top_k);
    d.dens_off = cells;
    d.gw = W / p.cell_px; d.gh = H / p.cell_px;
    if (d.gw < R || d.gh < R) return fail(h, FFPP_EINVAL, "density grid smaller than the Gaussian radius");
    // spatial cells 8 px wide x 16 px tall; both edges double until the frame has at most kMaxCells of them
    int hs = 3, hsy = 4;
    while ((int64_t)((W + (1 << hs) - 1) >> hs) * ((H + (1 << hsy) - 1) >> hsy) > kMaxCells) { if (hs < hsy) ++hs; else ++hsy; }
    d.hshift = hs; d.hshift_y = hsy;
    d.cgw = (W + (1 << hs) - 1) >> hs;
    d.cgh = (H + (1 << hsy) - 1) >> hsy;
    d.edge_off = edges;
    d.edge_cap = (int32_t)std::min<int64_t>(h->edges_per_box * d.nmax, 0x7fffffff);
    edges += d.edge_cap;
    fr[f] = d;
    coff[f] = cand;
    cand += n; cells += (int64_t)d.gw * d.gh;
    d.k5_th = k5_tile_h(d.gw, d.gh, h->cst.radius_t);
    d.k5_tiles = k5_tiles(d.gw, d.gh, h->cst.radius_t);
    fr[f] = d;
    max_tiles = std::max(max_tiles, (int)d.k5_tiles);
    max_nmax = std::max(max_nmax, (int)d.nmax);
  }
  coff[B] = cand;
  if (cand > p.max_total_candidates) return fail(h, FFPP_ECAPACITY, "sum N_f exceeds max_total_candidates");
  size_t used = h->ml.block_frame_off;
  {
    // a1: first frame of every K1_BLOCK-row block of the flat candidate stream
    int32_t* bf = reinterpret_cast<int32_t*>(h->h_meta.data() + h->ml.block_frame_off);
    int f = 0;
    int64_t b = 0;
    for (; b * K1_BLOCK < cand; ++b) {
      while (f + 1 < B && coff[f + 1] <= b * K1_BLOCK) ++f;
      bf[b] = f;
    }
    used += sizeof(int32_t) * (size_t)b;
  }
  if (cells > h->max_total_cells) return fail(h, FFPP_ECAPACITY, "density cells exceed max_total_cells");
  if (edges > h->edge_cap_total) return fail(h, FFPP_ECAPACITY, "suppression-edge pool exceeds nms_workspace_bytes");
  ffpp_handle::GeoSlot& g = h->geo[lru];
  g.B = -1;                                       // not valid until the copy is queued
  used = (used + 15) & ~(size_t)15;
  FFPP_CUDA(h, cudaMemcpyAsync(g.d_meta, h->h_meta.data(), used, cudaMemcpyHostToDevice, stream));
  g.B = B; g.hash = hash;
  g.N.assign(N, N + B);
  g.dims.assign(dims, dims + 2 * B);
  g.max_tiles = max_tiles; g.max_nmax = max_nmax;
  g.total_cand = cand; g.total_cells = cells;
  g.last_use = ++h->use_clock;
  h->cur = lru;
  return FFPP_OK;
}

// Launch `kern` as a programmatic dependent of the kernel before it in the stream: its launch is processed while the
// predecessor still runs and it starts the moment the predecessor has finished (every such kernel begins with
// pdl_wait()).  PAPER.md:L155: "many small and short-lived GPU kernels interspersed with idle gaps" — these are the gaps.
template <typename... KArgs, typename... Args>
cudaError_t launch_dep(void (*kern)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, Args&&... args) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = st;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = at; cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, kern, static_cast<KArgs>(args)...);
}

template <bool kHalf, typename KeyT>
int launch_all(ffpp_handle* h, const void* raw, int B, cudaStream_t st, ffpp_box* out_boxes, int32_t* out_counts,
               float* out_density) {
  const ffpp_handle::GeoSlot& g = h->geo[h->cur];
  const FrameDesc* frames = reinterpret_cast<const FrameDesc*>(g.d_meta + h->ml.frames_off);
  const int64_t* coff = reinterpret_cast<const int64_t*>(g.d_meta + h->ml.cand_off_off);
  const Consts& c = h->cst;
  const bool tm = h->timing;
  if (tm) FFPP_CUDA(h, cudaEventRecord(h->ev[1], st));

  // a1
  {
    const int64_t row = kHalf ? 10 : 20;
    const int64_t nchunks = (g.total_cand * row + K1_CHUNK_BYTES - 1) / K1_CHUNK_BYTES;
    int64_t grid = (int64_t)h->sm_count * K1_CTAS_PER_SM;
    if (grid > nchunks) grid = nchunks;
    launch_dep(k1_threshold_compact<kHalf, KeyT>, dim3((unsigned)grid), dim3(K1_THREADS), (size_t)(K1_STAGES * K1_CHUNK_BYTES), st,
               static_cast<const uint8_t*>(raw), g.total_cand, B, coff, reinterpret_cast<const int32_t*>(g.d_meta + h->ml.block_frame_off),
               c.logit_thr, static_cast<KeyT*>(h->d_surv_keys), h->surv_cnt());
  }
  if (tm) FFPP_CUDA(h, cudaEventRecord(h->ev[2], st));
  // a2 (+ clears the a5 histogram)
  launch_dep(k2_select_bin<kHalf, KeyT>, dim3((unsigned)B), dim3(K2_THREADS), k2_smem_bytes((size_t)c.top_k, sizeof(KeyT)), st,
             static_cast<const uint8_t*>(raw), frames, static_cast<const KeyT*>(h->d_surv_keys), h->surv_cnt(), c,
             h->d_sel_box, h->d_sp_box, static_cast<KeyT*>(h->d_sp_key), h->d_cellstart, h->n_sorted(), h->d_hist32,
             reinterpret_cast<uint32_t*>(h->d_hasin), h->sm_count);
  if (tm) FFPP_CUDA(h, cudaEventRecord(h->ev[3], st));
  // a3 (a frame that overflows its share of the edge pool is flagged and resolved pool-free by its a4 CTA)
  {
    const dim3 g3((unsigned)((g.max_nmax + K3_THREADS - 1) / K3_THREADS), (unsigned)B);
    if (g3.x > 0) {
      if (h->count_work)
        launch_dep(k3_nms_edges<KeyT, true>, g3, dim3(K3_THREADS), 0, st, frames, h->n_sorted(), h->d_sp_box,
                   static_cast<const KeyT*>(h->d_sp_key), h->d_cellstart, c, h->edge_ctr(), h->d_edges, h->d_hasin, h->frame_err(), h->d_work);
      else
        launch_dep(k3_nms_edges<KeyT, false>, g3, dim3(K3_THREADS), 0, st, frames, h->n_sorted(), h->d_sp_box,
                   static_cast<const KeyT*>(h->d_sp_key), h->d_cellstart, c, h->edge_ctr(), h->d_edges, h->d_hasin, h->frame_err(), h->d_work);
    }
  }
  if (tm) FFPP_CUDA(h, cudaEventRecord(h->ev[4], st));
  // a4 (+ a5 histogram)
  launch_dep(k4_resolve_order<KeyT>, dim3((unsigned)B), dim3(K4_THREADS), k4_smem_bytes((size_t)c.top_k, (size_t)c.kpad, sizeof(KeyT)), st,
             frames, h->n_sorted(), h->d_sp_box, static_cast<const KeyT*>(h->d_sp_key), h->edge_ctr(), h->d_edges,
             reinterpret_cast<const uint32_t*>(h->d_hasin), h->d_cellstart, h->frame_err(), c, h->sm_count, h->d_k4_scratch,
             static_cast<KeyT*>(h->d_kept_key), h->d_kept_pos, out_counts);
  {
    const dim3 g4e((unsigned)((g.max_nmax + K4E_THREADS - 1) / K4E_THREADS), (unsigned)B);
    if (g4e.x > 0)
      launch_dep(k4e_emit<KeyT>, g4e, dim3(K4E_THREADS), 0, st, frames, h->d_sp_box, static_cast<const KeyT*>(h->d_kept_key), h->d_kept_pos,
                 out_counts, c, out_boxes, h->d_hist32);
  }
  if (tm) FFPP_CUDA(h, cudaEventRecord(h->ev[5], st));
  // a6
  {
    const dim3 g5((unsigned)g.max_tiles, (unsigned)B);
    const size_t s5 = k5_smem_bytes(h->p.max_frame_w / h->p.cell_px, h->p.max_frame_h / h->p.cell_px, c.radius_t);
    const uint16_t* h16 = reinterpret_cast<const uint16_t*>(h->d_hist32);
    switch (c.radius_t) {
#define FFPP_K5_CASE(RT) case RT: launch_dep(k5_density<RT>, g5, dim3(K5_THREADS), s5, st, frames, c, h16, out_density); break;
      FFPP_K5_RADII(FFPP_K5_CASE)
#undef FFPP_K5_CASE
      default: return fail(h, FFPP_EINVAL, "no a6 kernel for this radius");
    }
  }
  if (tm) {
    FFPP_CUDA(h, cudaEventRecord(h->ev[6], st));
    h->ev_valid = true;
  }
  FFPP_CUDA(h, cudaGetLastError());
  return FFPP_OK;
}

template <bool kHalf, typename KeyT>
int set_kernel_attrs(ffpp_handle* h) {
  const size_t s1 = K1_STAGES * K1_CHUNK_BYTES;
  FFPP_CUDA(h, cudaFuncSetAttribute(k1_threshold_compact<kHalf, KeyT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)s1));
  const size_t s2 = k2_smem_bytes((size_t)h->p.top_k, sizeof(KeyT));
  FFPP_CUDA(h, cudaFuncSetAttribute(k2_select_bin<kHalf, KeyT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)s2));
  const size_t s4 = k4_smem_bytes((size_t)h->p.top_k, (size_t)h->kpad, sizeof(KeyT));
  FFPP_CUDA(h, cudaFuncSetAttribute(k4_resolve_order<KeyT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)s4));
  return FFPP_OK;
}

}  // namespace

extern "C" {

int ffpp_create(const ffpp_params* p, ffpp_handle** out) {
  if (!p || !out) return fail(nullptr, FFPP_EINVAL, "ffpp_create: null argument");
  if (p->dtype != 0 && p->dtype != 1) return fail(nullptr, FFPP_EINVAL, "dtype must be 0 (fp32) or 1 (fp16)");
  if (p->num_levels < 1 || p->num_levels > kMaxLevels) return fail(nullptr, FFPP_EINVAL, "num_levels must be 1..4");
  for (int l = 0; l < p->num_levels; ++l) {
    if (!is_pow2(p->strides[l])) return fail(nullptr, FFPP_EINVAL, "strides must be powers of two");
    if (l && p->strides[l] <= p->strides[l - 1]) return fail(nullptr, FFPP_EINVAL, "strides must be ascending");
  }
  if (!(p->iou_thresh >= 0.0f)) return fail(nullptr, FFPP_EINVAL, "iou_thresh must be >= 0");
  if (std::isnan(p->conf_thresh)) return fail(nullptr, FFPP_EINVAL, "conf_thresh is NaN");
  if (p->top_k < 1) return fail(nullptr, FFPP_EINVAL, "top_k must be >= 1");
  if (p->cell_px < 1) return fail(nullptr, FFPP_EINVAL, "cell_px must be >= 1");
  if (!(p->sigma_cells > 0.0f) || !(p->truncate_sigmas > 0.0f)) return fail(nullptr, FFPP_EINVAL, "sigma_cells and truncate_sigmas must be > 0");
  if (p->max_frames < 1 || p->max_total_candidates < 1 || p->max_frame_w < 1 || p->max_frame_h < 1)
    return fail(nullptr, FFPP_EINVAL, "capacities must be positive");
  const int R = (int)std::floor((double)p->truncate_sigmas * (double)p->sigma_cells);
  if (R < 1 || R > kMaxRadius) return fail(nullptr, FFPP_EINVAL, "Gaussian radius floor(truncate*sigma) must be 1..32");

  if (p->nms_edges_per_box < 0 || p->nms_workspace_bytes < 0) return fail(nullptr, FFPP_EINVAL, "nms_edges_per_box / nms_workspace_bytes must be >= 0");
  ffpp_handle* h = new (std::nothrow) ffpp_handle();
  if (!h) return fail(nullptr, FFPP_ENOMEM, "host allocation failed");
  h->p = *p;
  h->half = p->dtype == 1;
  const int64_t nmaxframe = frame_candidates(*p, p->max_frame_w, p->max_frame_h);
  h->max_frame_cand = (int)std::min<int64_t>(nmaxframe, 1 << 20);
  h->key_bytes = (h->half && nmaxframe <= 65536) ? 4 : 8;
  h->kpad = (p->top_k + kBlk - 1) / kBlk * kBlk;
  {
    // shared-memory budgets of a2 (selected keys + bin bookkeeping) and a4 (two sort buffers) under the 227 KB opt-in limit
    const size_t lim = 232448;                                        // minus each kernel's static shared memory
    if (p->top_k > kMaxTopK || k2_smem_bytes((size_t)p->top_k, h->key_bytes) > lim - 512 ||
        k4_smem_bytes((size_t)p->top_k, (size_t)h->kpad, h->key_bytes) > lim - 512) {
      delete h;
      return fail(nullptr, FFPP_EINVAL, "top_k exceeds the shared-memory capacity (24576 with 32-bit keys, 12288 with 64-bit keys)");
    }
  }

  // constants
  Consts& c = h->cst;
  std::memset(&c, 0, sizeof(c));
  if (!(p->conf_thresh > 0.0f)) c.logit_thr = -INFINITY;
  else if (!(p->conf_thresh < 1.0f)) c.logit_thr = INFINITY;
  else c.logit_thr = (float)std::log((double)p->conf_thresh / (1.0 - (double)p->conf_thresh));
  c.iou_thr = p->iou_thresh;
  c.iou_fast = (p->iou_thresh >= 1e-6f && p->iou_thresh <= 1e6f) ? 1 : 0;
  c.iou_thr_hi = std::nextafterf((float)((double)p->iou_thresh * (1.0 + std::ldexp(1.0, -20))), INFINITY);
  c.iou_thr_lo = std::nextafterf((float)((double)p->iou_thresh * (1.0 - std::ldexp(1.0, -20))), -INFINITY);
  {
    // a pair with IoU > t has |centre distance| < rho * min(w_a, w_b) per axis, rho = max(1 - t, 1/(2t) - 1/2); evaluated
    // at a slightly smaller t (and at most 0.9) so that every fp32 rounding of the IoU of the definition is covered
    const double te = std::min((double)p->iou_thresh, 0.9) * (1.0 - 1e-3);
    c.rho = te >= 1e-3 ? (float)std::max(1.0 - te, 0.5 / te - 0.5) : 1e30f;
  }
  c.top_k = p->top_k;
  c.kpad = h->kpad;
  c.num_levels = p->num_levels;
  for (int l = 0; l < p->num_levels; ++l) c.stride_log2[l] = ilog2(p->strides[l]);
  c.cell_px = p->cell_px;
  c.cell_inv = is_pow2(p->cell_px) ? 1.0f / (float)p->cell_px : 0.0f;
  c.radius = R;
  {
    double Z = 0.0, s2 = 2.0 * (double)p->sigma_cells * (double)p->sigma_cells;
    for (int k = -R; k <= R; ++k) Z += std::exp(-(double)(k * k) / s2);
    for (int k = -R; k <= R; ++k) c.taps[k + R] = (float)(std::exp(-(double)(k * k) / s2) / Z);
    static const int buckets[] = {FFPP_K5_RADII(FFPP_K5_LIST) 0};
    int RT = kMaxRadius;
    for (int i = 0; buckets[i]; ++i) if (buckets[i] >= R && buckets[i] < RT) RT = buckets[i];
    c.radius_t = RT;
    for (int k = -R; k <= R; ++k) c.taps_pad[k + RT] = c.taps[k + R];
  }

  auto bail = [&](int code, const std::string& msg) { ffpp_destroy(h); return fail(nullptr, code, msg); };
  cudaError_t e;
  int dev = 0;
  if ((e = cudaGetDevice(&dev)) != cudaSuccess) return bail(FFPP_ECUDA, std::string("cudaGetDevice: ") + cudaGetErrorString(e));
  cudaDeviceProp prop;
  if ((e = cudaGetDeviceProperties(&prop, dev)) != cudaSuccess) return bail(FFPP_ECUDA, std::string("cudaGetDeviceProperties: ") + cudaGetErrorString(e));
  if (prop.major != 10) return bail(FFPP_ECUDA, "libffpp is built for sm_100a only; this device is sm_" + std::to_string(prop.major * 10 + prop.minor));
  h->sm_count = prop.multiProcessorCount;

  // capacities
  const int64_t cells_frame = (int64_t)(p->max_frame_w / p->cell_px) * (p->max_frame_h / p->cell_px);
  h->max_total_cells = p->max_total_cells > 0 ? p->max_total_cells : cells_frame * p->max_frames;
  const int64_t nmax_cap = std::min<int64_t>(p->top_k, nmaxframe);
  h->edges_per_box = p->nms_edges_per_box > 0 ? p->nms_edges_per_box : 16;
  if (p->nms_workspace_bytes > 0)
    h->edges_per_box = std::max<int64_t>(1, p->nms_workspace_bytes / 4 / (nmax_cap * p->max_frames));
  h->p.nms_edges_per_box = (int32_t)std::min<int64_t>(h->edges_per_box, 0x7fffffff);
  h->edge_cap_total = h->edges_per_box * nmax_cap * p->max_frames;

  h->ml = meta_layout(p->max_frames, p->max_total_candidates);
  auto dalloc = [&](void** ptr, size_t bytes) {
    if (bytes == 0) bytes = 16;
    cudaError_t ee = cudaMalloc(ptr, bytes);
    if (ee == cudaSuccess) h->workspace_bytes += (int64_t)bytes;
    return ee;
  };
  const size_t KP = (size_t)h->kpad, F = (size_t)p->max_frames;
  e = cudaSuccess;
  for (int sl = 0; sl < ffpp_handle::kGeoSlots && e == cudaSuccess; ++sl) e = dalloc((void**)&h->geo[sl].d_meta, h->ml.bytes);
  if (e != cudaSuccess ||
      (e = dalloc((void**)&h->d_work, 4 * sizeof(unsigned long long))) != cudaSuccess ||
      (e = dalloc(&h->d_surv_keys, (size_t)p->max_total_candidates * h->key_bytes)) != cudaSuccess ||
      (e = dalloc((void**)&h->d_counters, (3 + kCntStride) * F * sizeof(int))) != cudaSuccess ||
      (e = dalloc((void**)&h->d_sel_box, F * KP * sizeof(float4))) != cudaSuccess ||
      (e = dalloc((void**)&h->d_sp_box, F * KP * sizeof(float4))) != cudaSuccess ||
      (e = dalloc(&h->d_sp_key, F * KP * (size_t)h->key_bytes)) != cudaSuccess ||
      (e = dalloc((void**)&h->d_hasin, F * KP)) != cudaSuccess ||
      (e = dalloc(&h->d_kept_key, F * (size_t)p->top_k * (size_t)h->key_bytes)) != cudaSuccess ||
      (e = dalloc((void**)&h->d_kept_pos, F * (size_t)p->top_k * sizeof(uint16_t))) != cudaSuccess ||
      (e = dalloc((void**)&h->d_k4_scratch, F * k4_scratch_bytes((size_t)p->top_k, (size_t)h->key_bytes))) != cudaSuccess ||
      (e = dalloc((void**)&h->d_cellstart, F * (size_t)kCellStride * sizeof(uint16_t))) != cudaSuccess ||
      (e = dalloc((void**)&h->d_edges, (size_t)h->edge_cap_total * sizeof(uint32_t))) != cudaSuccess ||
      (e = dalloc((void**)&h->d_hist32, ((size_t)h->max_total_cells / 2 + 2) * sizeof(uint32_t))) != cudaSuccess) {
    cudaGetLastError();
    return bail(e == cudaErrorMemoryAllocation ? FFPP_ENOMEM : FFPP_ECUDA, std::string("workspace cudaMalloc: ") + cudaGetErrorString(e));
  }
  h->h_meta.assign(h->ml.bytes, 0);
  if ((e = cudaMemset(h->d_work, 0, 4 * sizeof(unsigned long long))) != cudaSuccess) return bail(FFPP_ECUDA, std::string("cudaMemset: ") + cudaGetErrorString(e));
  for (int i = 0; i <= FFPP_NUM_STAGES; ++i)
    if ((e = cudaEventCreate(&h->ev[i])) != cudaSuccess) return bail(FFPP_ECUDA, std::string("cudaEventCreate: ") + cudaGetErrorString(e));
  int rc;
  if (h->half && h->key_bytes == 4) rc = set_kernel_attrs<true, uint32_t>(h);
  else if (h->half) rc = set_kernel_attrs<true, uint64_t>(h);
  else rc = set_kernel_attrs<false, uint64_t>(h);
  if (rc != FFPP_OK) { std::string m = h->err; return bail(rc, m); }
  {
    const size_t s5 = k5_smem_bytes(p->max_frame_w / p->cell_px, p->max_frame_h / p->cell_px, c.radius_t);
    e = cudaSuccess;
    switch (c.radius_t) {
#define FFPP_K5_CASE(RT) case RT: e = cudaFuncSetAttribute(k5_density<RT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)s5); break;
      FFPP_K5_RADII(FFPP_K5_CASE)
#undef FFPP_K5_CASE
      default: break;
    }
    if (e != cudaSuccess) return bail(FFPP_ECUDA, std::string("cudaFuncSetAttribute(k5): ") + cudaGetErrorString(e));
  }
  *out = h;
  return FFPP_OK;
}

int ffpp_run(ffpp_handle* h, const void* raw, int32_t B, const int32_t* N_per_frame, const int32_t* frame_dims, void* stream,
             ffpp_box* out_boxes, int32_t* out_counts, float* out_density) {
  if (!h) return FFPP_EINVAL;
  if (B < 0) return fail(h, FFPP_EINVAL, "B < 0");
  if (B == 0) return FFPP_OK;
  if (!raw || !N_per_frame || !frame_dims || !out_boxes || !out_counts || !out_density) return fail(h, FFPP_EINVAL, "null pointer");
  if (B > h->p.max_frames) return fail(h, FFPP_ECAPACITY, "B exceeds max_frames");
  if (reinterpret_cast<uintptr_t>(raw) & 15) return fail(h, FFPP_EINVAL, "raw must be 16-byte aligned");
  if (reinterpret_cast<uintptr_t>(out_boxes) & 7) return fail(h, FFPP_EINVAL, "out_boxes must be 8-byte aligned");
  if ((reinterpret_cast<uintptr_t>(out_density) | reinterpret_cast<uintptr_t>(out_counts)) & 3)
    return fail(h, FFPP_EINVAL, "out_counts / out_density must be 4-byte aligned");
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  if (h->timing) FFPP_CUDA(h, cudaEventRecord(h->ev[0], st));
  int rc = schedule(h, B, N_per_frame, frame_dims, st);
  if (rc != FFPP_OK) return rc;
  k0_clear<<<(unsigned)(((3 + kCntStride) * B + 255) / 256), 256, 0, st>>>(h->d_counters, h->p.max_frames, B, h->count_work ? h->d_work : nullptr);
  if (h->half && h->key_bytes == 4) return launch_all<true, uint32_t>(h, raw, B, st, out_boxes, out_counts, out_density);
  if (h->half) return launch_all<true, uint64_t>(h, raw, B, st, out_boxes, out_counts, out_density);
  return launch_all<false, uint64_t>(h, raw, B, st, out_boxes, out_counts, out_density);
}

int ffpp_run_host(ffpp_handle* h, const void* raw, int32_t B, const int32_t* N_per_frame, const int32_t* frame_dims, void* stream,
                  ffpp_box* out_boxes, int32_t* out_counts, float* out_density) {
  if (!h) return FFPP_EINVAL;
  if (B < 0) return fail(h, FFPP_EINVAL, "B < 0");
  if (B == 0) return FFPP_OK;
  if (!raw || !N_per_frame || !frame_dims || !out_boxes || !out_counts || !out_density) return fail(h, FFPP_EINVAL, "null pointer");
  if (B > h->p.max_frames) return fail(h, FFPP_ECAPACITY, "B exceeds max_frames");
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  const size_t esz = h->half ? 2 : 4;
  // sizes are checked BEFORE anything is queued: they become byte counts of the uploads below
  int64_t cand = 0, cells = 0;
  for (int f = 0; f < B; ++f) {
    const int W = frame_dims[2 * f], H = frame_dims[2 * f + 1];
    if (W <= 0 || H <= 0) return fail(h, FFPP_EINVAL, "frame_dims: W and H must be positive");
    if (N_per_frame[f] <= 0 || (int64_t)N_per_frame[f] != frame_candidates(h->p, W, H))
      return fail(h, FFPP_EINVAL, "N_per_frame[f] != sum_l W*H/s_l^2");
    cand += N_per_frame[f];
    cells += (int64_t)(W / h->p.cell_px) * (H / h->p.cell_px);
  }
  if (cand > h->p.max_total_candidates) return fail(h, FFPP_ECAPACITY, "sum N_f exceeds max_total_candidates");
  if (cells > h->max_total_cells) return fail(h, FFPP_ECAPACITY, "density cells exceed max_total_cells");
  if (!h->d_in) {  // first use of the host path: its device staging (not part of ffpp_run's no-allocation promise), all or nothing
    const size_t K = (size_t)h->p.top_k, F = (size_t)h->p.max_frames;
    cudaError_t e;
    if ((e = cudaMalloc(&h->d_in, (size_t)h->p.max_total_candidates * 5 * esz + 16)) != cudaSuccess ||
        (e = cudaMalloc((void**)&h->d_out_boxes, F * K * sizeof(ffpp_box))) != cudaSuccess ||
        (e = cudaMalloc((void**)&h->d_out_counts, F * sizeof(int))) != cudaSuccess ||
        (e = cudaMalloc((void**)&h->d_out_density, (size_t)h->max_total_cells * sizeof(float) + 16)) != cudaSuccess) {
      cudaGetLastError();
      cudaFree(h->d_in); cudaFree(h->d_out_boxes); cudaFree(h->d_out_counts); cudaFree(h->d_out_density);
      h->d_in = nullptr; h->d_out_boxes = nullptr; h->d_out_counts = nullptr; h->d_out_density = nullptr;
      return fail(h, e == cudaErrorMemoryAllocation ? FFPP_ENOMEM : FFPP_ECUDA, std::string("host-path staging cudaMalloc: ") + cudaGetErrorString(e));
    }
  }
  // kept boxes: only rows [0, count) of each frame are defined.  A pinned (device-mapped) out_boxes is written by one
  // kernel through its device alias; a pageable one gets one copy per frame after the counts have arrived.
  const size_t K = (size_t)h->p.top_k;
  ffpp_box* alias = nullptr;
  {
    cudaPointerAttributes at;
    if (cudaPointerGetAttributes(&at, out_boxes) == cudaSuccess && at.type == cudaMemoryTypeHost && at.devicePointer)
      alias = static_cast<ffpp_box*>(at.devicePointer);
    else
      cudaGetLastError();
  }
  // Frames are independent, so a large batch is cut BY BYTES into up to kHostChunks runs of whole frames: the upload of
  // run i+1 (copy stream) and the download of run i-1 (second copy stream) overlap the kernels of run i on `stream`.
  // A run starts where the raw byte offset is a multiple of 16 (ffpp_run's alignment rule).  A run's kernel chain costs
  // ~160 us however few frames it holds (one CTA per frame in a2 / a4), so consecutive runs alternate between two
  // compute streams and two workspaces (this handle's and its twin's): two chains are in flight and the batch stays
  // PCIe-bound.  What is left after the last upload is one chain + its download; six runs with shrinking shares
  // measured best on config 5 (1.56 ms; four equal runs on one stream 1.61, eight 2.06, one 2.10; the H2D copies
  // alone take 1.33 ms while downloads run beside them; profiles/r2_e2e_timeline.md).
  constexpr int kHostChunks = ffpp_handle::kHostChunks;
  static const int kShare[kHostChunks] = {4, 4, 4, 3, 3, 2};                  // of 20: relative raw bytes of the runs
  const int nshare = kHostChunks;
  const size_t row = 5 * esz;
  std::vector<int> cut{0};                                          // first frame of every run, then B
  if (B >= 2 * kHostChunks && (size_t)cand * row >= ((size_t)16 << 20)) {
    int64_t acc = 0, want = 0;
    int next = 0;
    want = cand * kShare[0] / 20;
    for (int f = 0; f < B && next + 1 < nshare; ++f) {
      if (f > cut.back() && acc * (int64_t)row % 16 == 0 && acc >= want) {
        cut.push_back(f); ++next;
        int sh = 0;
        for (int q = 0; q <= next; ++q) sh += kShare[q];
        want = cand * sh / 20;
      }
      acc += N_per_frame[f];
    }
  }
  cut.push_back(B);
  const int C = (int)cut.size() - 1;
  if (C > 1 && !h->s_h2d) {
    FFPP_CUDA(h, cudaStreamCreateWithFlags(&h->s_h2d, cudaStreamNonBlocking));
    FFPP_CUDA(h, cudaStreamCreateWithFlags(&h->s_d2h, cudaStreamNonBlocking));
    FFPP_CUDA(h, cudaStreamCreateWithFlags(&h->s_run2, cudaStreamNonBlocking));
    for (int i = 0; i < kHostChunks; ++i) {
      FFPP_CUDA(h, cudaEventCreateWithFlags(&h->ev_up[i], cudaEventDisableTiming));
      FFPP_CUDA(h, cudaEventCreateWithFlags(&h->ev_run[i], cudaEventDisableTiming));
    }
  }
  if (C > 1 && !h->twin) {                                          // the second workspace (same parameters), first chunked call only
    ffpp_params tp = h->p;
    const int trc = ffpp_create(&tp, &h->twin);
    if (trc != FFPP_OK) { h->twin = nullptr; return fail(h, trc, std::string("host path: second workspace: ") + ffpp_last_error(nullptr)); }
  }
  cudaStream_t s_up = C > 1 ? h->s_h2d : st, s_dn = C > 1 ? h->s_d2h : st;
  if (C > 1) {                                                      // the copy streams start after what is already on `stream`
    FFPP_CUDA(h, cudaEventRecord(h->ev_run[0], st));
    FFPP_CUDA(h, cudaStreamWaitEvent(s_up, h->ev_run[0], 0));
    FFPP_CUDA(h, cudaStreamWaitEvent(h->s_run2, h->ev_run[0], 0));
  }
  std::vector<int64_t> c_off((size_t)C + 1, 0), d_off((size_t)C + 1, 0);
  for (int i = 0; i < C; ++i) {
    int64_t cc = 0, dd = 0;
    for (int f = cut[(size_t)i]; f < cut[(size_t)i + 1]; ++f) {
      cc += N_per_frame[f];
      dd += (int64_t)(frame_dims[2 * f] / h->p.cell_px) * (frame_dims[2 * f + 1] / h->p.cell_px);
    }
    c_off[(size_t)i + 1] = c_off[(size_t)i] + cc;
    d_off[(size_t)i + 1] = d_off[(size_t)i] + dd;
  }
  uint8_t* d_in8 = static_cast<uint8_t*>(h->d_in);
  const uint8_t* raw8 = static_cast<const uint8_t*>(raw);
  for (int i = 0; i < C; ++i)                                       // all uploads are queued up front, in order
  {
    const size_t o = (size_t)c_off[(size_t)i] * row, nbytes = (size_t)(c_off[(size_t)i + 1] - c_off[(size_t)i]) * row;
    FFPP_CUDA(h, cudaMemcpyAsync(d_in8 + o, raw8 + o, nbytes, cudaMemcpyHostToDevice, s_up));
    if (C > 1) FFPP_CUDA(h, cudaEventRecord(h->ev_up[i], s_up));
  }
  for (int i = 0; i < C; ++i) {
    const int f0 = cut[(size_t)i], Bi = cut[(size_t)i + 1] - f0;
    // two kernel chains in flight: even runs on `stream` with this handle's workspace, odd runs on the second compute
    // stream with the twin's (a run's chain is latency-bound: one CTA per frame in a2 / a4, so two chains share the SMs well)
    ffpp_handle* hr = (C > 1 && (i & 1)) ? h->twin : h;
    cudaStream_t sr = (C > 1 && (i & 1)) ? h->s_run2 : st;
    if (C > 1) FFPP_CUDA(h, cudaStreamWaitEvent(sr, h->ev_up[i], 0));
    const int rc = ffpp_run(hr, d_in8 + (size_t)c_off[(size_t)i] * row, Bi, N_per_frame + f0, frame_dims + 2 * f0, sr,
                            h->d_out_boxes + (size_t)f0 * K, h->d_out_counts + f0, h->d_out_density + d_off[(size_t)i]);
    if (rc != FFPP_OK) {
      if (hr != h) h->err = hr->err;
      cudaStreamSynchronize(s_up); cudaStreamSynchronize(st); if (C > 1) cudaStreamSynchronize(h->s_run2); cudaStreamSynchronize(s_dn);
      return rc;
    }
    if (C > 1) {
      FFPP_CUDA(h, cudaEventRecord(h->ev_run[i], sr));
      FFPP_CUDA(h, cudaStreamWaitEvent(s_dn, h->ev_run[i], 0));
    }
    if (alias) {
      const dim3 g((unsigned)std::min<size_t>(16, (K * 3 + KH_THREADS - 1) / KH_THREADS), (unsigned)Bi);
      kh_copy_kept_rows<<<g, KH_THREADS, 0, s_dn>>>(h->d_out_boxes + (size_t)f0 * K, h->d_out_counts + f0, (int)K, alias + (size_t)f0 * K);
    }
    FFPP_CUDA(h, cudaMemcpyAsync(out_counts + f0, h->d_out_counts + f0, sizeof(int) * (size_t)Bi, cudaMemcpyDeviceToHost, s_dn));
    FFPP_CUDA(h, cudaMemcpyAsync(out_density + d_off[(size_t)i], h->d_out_density + d_off[(size_t)i],
                                 sizeof(float) * (size_t)(d_off[(size_t)i + 1] - d_off[(size_t)i]), cudaMemcpyDeviceToHost, s_dn));
  }
  FFPP_CUDA(h, cudaStreamSynchronize(s_dn));
  if (C > 1) FFPP_CUDA(h, cudaStreamSynchronize(h->s_run2));
  FFPP_CUDA(h, cudaStreamSynchronize(st));
  if (!alias) {
    for (int f = 0; f < B; ++f)
      if (out_counts[f] > 0)
        FFPP_CUDA(h, cudaMemcpyAsync(out_boxes + (size_t)f * K, h->d_out_boxes + (size_t)f * K, sizeof(ffpp_box) * (size_t)out_counts[f],
                                     cudaMemcpyDeviceToHost, st));
    FFPP_CUDA(h, cudaStreamSynchronize(st));
  }
  FFPP_CUDA(h, cudaGetLastError());
  return FFPP_OK;
}

int ffpp_destroy(ffpp_handle* h) {
  if (!h) return FFPP_OK;
  for (int sl = 0; sl < ffpp_handle::kGeoSlots; ++sl) cudaFree(h->geo[sl].d_meta);
  cudaFree(h->d_work); cudaFree(h->d_surv_keys); cudaFree(h->d_counters); cudaFree(h->d_sel_box); cudaFree(h->d_sp_box);
  cudaFree(h->d_sp_key); cudaFree(h->d_cellstart); cudaFree(h->d_hasin); cudaFree(h->d_k4_scratch); cudaFree(h->d_kept_key); cudaFree(h->d_kept_pos); cudaFree(h->d_edges);
  cudaFree(h->d_hist32);
  cudaFree(h->d_in); cudaFree(h->d_out_boxes); cudaFree(h->d_out_counts); cudaFree(h->d_out_density);
  for (int sl = 0; sl < ffpp_handle::kNextSlots; ++sl) cudaFree(h->ngeo[sl].d_tab);
  cudaFree(h->d_ccl_aux); cudaFree(h->d_ccl_sums); cudaFree(h->d_ccl_blk); cudaFree(h->d_ent_part);
  if (h->twin) ffpp_destroy(h->twin);
  if (h->s_run2) cudaStreamDestroy(h->s_run2);
  if (h->s_h2d) cudaStreamDestroy(h->s_h2d);
  if (h->s_d2h) cudaStreamDestroy(h->s_d2h);
  for (int i = 0; i < ffpp_handle::kHostChunks; ++i) { if (h->ev_up[i]) cudaEventDestroy(h->ev_up[i]); if (h->ev_run[i]) cudaEventDestroy(h->ev_run[i]); }
  for (int i = 0; i <= FFPP_NUM_STAGES; ++i)
    if (h->ev[i]) cudaEventDestroy(h->ev[i]);
  delete h;
  return FFPP_OK;
}

const char* ffpp_last_error(const ffpp_handle* h) { return h ? h->err.c_str() : g_create_error.c_str(); }

int ffpp_get_info(const ffpp_handle* h, ffpp_info* out) {
  if (!h || !out) return FFPP_EINVAL;
  std::memset(out, 0, sizeof(*out));
  out->logit_threshold = h->cst.logit_thr;
  out->radius = h->cst.radius;
  for (int k = 0; k <= 2 * h->cst.radius; ++k) out->taps[k] = h->cst.taps[k];
  out->key_bits = h->key_bytes * 8;
  out->workspace_bytes = h->workspace_bytes;
  out->sm_count = h->sm_count;
  return FFPP_OK;
}

int ffpp_set_stage_timing(ffpp_handle* h, int32_t enable) {
  if (!h) return FFPP_EINVAL;
  h->timing = enable != 0;
  h->ev_valid = false;
  return FFPP_OK;
}

int ffpp_get_stage_ms(ffpp_handle* h, float* ms_out) {
  if (!h || !ms_out) return FFPP_EINVAL;
  if (!h->ev_valid) return fail(h, FFPP_EINVAL, "no timed run recorded");
  for (int i = 0; i < FFPP_NUM_STAGES; ++i) FFPP_CUDA(h, cudaEventElapsedTime(&ms_out[i], h->ev[i], h->ev[i + 1]));
  return FFPP_OK;
}

int ffpp_debug_read(ffpp_handle* h, int32_t what, void* dst, int64_t dst_bytes) {
  if (!h || !dst) return FFPP_EINVAL;
  if (h->cur < 0 || h->geo[h->cur].B < 0) return fail(h, FFPP_EINVAL, "no run to read back");
  const int B = h->geo[h->cur].B;
  const size_t K = (size_t)h->p.top_k;
  FFPP_CUDA(h, cudaDeviceSynchronize());
  if (what == 0 || what == 1) {
    if (dst_bytes < (int64_t)(sizeof(int) * B)) return fail(h, FFPP_EINVAL, "dst too small");
    if (what == 0)
      FFPP_CUDA(h, cudaMemcpy2D(dst, sizeof(int), h->surv_cnt(), sizeof(int) * kCntStride, sizeof(int), (size_t)B, cudaMemcpyDeviceToHost));
    else
      FFPP_CUDA(h, cudaMemcpy(dst, h->n_sorted(), sizeof(int) * B, cudaMemcpyDeviceToHost));
    return FFPP_OK;
  }
  if (what == 4) {
    if (dst_bytes < (int64_t)(4 * sizeof(int64_t))) return fail(h, FFPP_EINVAL, "dst too small");
    int64_t* d = static_cast<int64_t*>(dst);
    FFPP_CUDA(h, cudaMemcpy(d, h->d_work, 3 * sizeof(int64_t), cudaMemcpyDeviceToHost));
    std::vector<int> fe((size_t)B);
    FFPP_CUDA(h, cudaMemcpy(fe.data(), h->frame_err(), sizeof(int) * B, cudaMemcpyDeviceToHost));
    d[3] = 0;
    for (int f = 0; f < B; ++f) d[3] += fe[(size_t)f] != 0;
    return FFPP_OK;
  }
  if (what == 5) {
    if (dst_bytes < (int64_t)(sizeof(int) * B)) return fail(h, FFPP_EINVAL, "dst too small");
    FFPP_CUDA(h, cudaMemcpy(dst, h->frame_err(), sizeof(int) * B, cudaMemcpyDeviceToHost));
    return FFPP_OK;
  }
  if (what != 2 && what != 3) return fail(h, FFPP_EINVAL, "unknown debug selector");
  if (dst_bytes < (int64_t)((what == 2 ? sizeof(int) : 4 * sizeof(float)) * B * K)) return fail(h, FFPP_EINVAL, "dst too small");
  // the device holds the top-K set in spatial order with its keys; the order of O4 is ascending key
  std::vector<int> ns((size_t)B);
  FFPP_CUDA(h, cudaMemcpy(ns.data(), h->n_sorted(), sizeof(int) * B, cudaMemcpyDeviceToHost));
  const size_t KP = (size_t)h->kpad;
  std::vector<uint64_t> keys(KP);
  std::vector<float4> boxes(KP);
  std::vector<uint32_t> k32(KP);
  std::vector<int> order(KP);
  for (int f = 0; f < B; ++f) {
    const int n = ns[(size_t)f];
    if (h->key_bytes == 4) {
      FFPP_CUDA(h, cudaMemcpy(k32.data(), static_cast<const uint32_t*>(h->d_sp_key) + (size_t)f * KP, sizeof(uint32_t) * n, cudaMemcpyDeviceToHost));
      for (int i = 0; i < n; ++i) keys[(size_t)i] = k32[(size_t)i];
    } else {
      FFPP_CUDA(h, cudaMemcpy(keys.data(), static_cast<const uint64_t*>(h->d_sp_key) + (size_t)f * KP, sizeof(uint64_t) * n, cudaMemcpyDeviceToHost));
    }
    for (int i = 0; i < n; ++i) order[(size_t)i] = i;
    std::sort(order.begin(), order.begin() + n, [&](int x, int y) { return keys[(size_t)x] < keys[(size_t)y]; });
    if (what == 2) {
      int* d = static_cast<int*>(dst) + (size_t)f * K;
      const uint64_t imask = h->key_bytes == 4 ? 0xFFFFull : 0xFFFFFFFFull;
      for (int k = 0; k < n; ++k) d[k] = (int)(keys[(size_t)order[(size_t)k]] & imask);
      for (size_t k = (size_t)n; k < K; ++k) d[k] = -1;
    } else {
      FFPP_CUDA(h, cudaMemcpy(boxes.data(), h->d_sp_box + (size_t)f * KP, sizeof(float4) * n, cudaMemcpyDeviceToHost));
      float* d = static_cast<float*>(dst) + (size_t)f * K * 4;
      for (int k = 0; k < n; ++k) std::memcpy(d + 4 * (size_t)k, &boxes[(size_t)order[(size_t)k]], sizeof(float4));
      for (size_t k = (size_t)n * 4; k < K * 4; ++k) d[k] = 0.0f;
    }
  }
  return FFPP_OK;

}

int ffpp_debug_count_work(ffpp_handle* h, int32_t enable) {
  if (!h) return FFPP_EINVAL;
  h->count_work = enable != 0;
  return FFPP_OK;
}

int ffpp_debug_stream_read(ffpp_handle* h, const void* dev, int64_t bytes, void* stream) {
  if (!h || !dev || bytes < 0) return FFPP_EINVAL;
  if (reinterpret_cast<uintptr_t>(dev) & 15) return fail(h, FFPP_EINVAL, "buffer must be 16-byte aligned");
  const int64_t n16 = bytes / 16;
  if (n16 == 0) return FFPP_OK;
  const int64_t grid = std::min<int64_t>((int64_t)h->sm_count * 8, (n16 + 255) / 256);
  k0_stream_read<<<(unsigned)grid, 256, 0, static_cast<cudaStream_t>(stream)>>>(static_cast<const uint4*>(dev), n16,
                                                                               reinterpret_cast<uint32_t*>(h->d_counters));
  FFPP_CUDA(h, cudaGetLastError());
  return FFPP_OK;
}

#ifdef FFPP_PROFILE_PHASES
// development aid, compiled only with -DFFPP_PROFILE_PHASES: %globaltimer stamps of the a4 phases of the last run
int ffpp_debug_phases(unsigned long long* dst, int frames) {
  cudaDeviceSynchronize();
  return (int)cudaMemcpyFromSymbol(dst, ffpp::g_phase, sizeof(unsigned long long) * 16 * (size_t)frames);
}
int ffpp_debug_phases2(unsigned long long* dst, int frames) {
  cudaDeviceSynchronize();
  return (int)cudaMemcpyFromSymbol(dst, ffpp::g_phase2, sizeof(unsigned long long) * 16 * (size_t)frames);
}
#endif

}  // extern "C"

#include "ffpp_next.cuh"

// =====================================================================================================
// The no-allocation entry point (include/ffpp_noalloc.h): entropy + clustering degree of B density grids of one size,
// with the scratch of the partial sums in a file-scope device array instead of handle memory.  A variant of
// ke_partial / ke_final (ffpp_next.cuh) for uniform grids: same block size, same per-thread cells, same summation order,
// so the results equal ffpp_heatmap_stats' bit for bit.  Nothing here touches an existing code path.
//
// g_noalloc_scratch is a DEVICE array: in host code its name is only a host-side stand-in (passing it to a kernel would
// fault or, where the GPU can reach host memory, silently use the wrong memory).  The host resolves its device address
// with cudaGetSymbolAddress, once per device with that device current, and passes that pointer to the kernels.
// =====================================================================================================
#include <mutex>

#include "../../include/ffpp_noalloc.h"

static __device__ __align__(256) double2 g_noalloc_scratch[FFPP_NOALLOC_MAX_BLOCKS];   // 256 KiB per GPU, held until exit

namespace ffpp {

__global__ void __launch_bounds__(KE_THREADS) kn_entropy_partial(const float* __restrict__ D, int n, int nblk, double2* __restrict__ part) {
  __shared__ double2 s_w[KE_THREADS / 32];
  const int img = blockIdx.y;
  const int base = blockIdx.x * KE_THREADS * KE_PER;          // grid.x == nblk: every (img, block) slot is written
  const float* Df = D + (int64_t)img * n;
  double a = 0.0, b = 0.0;
#pragma unroll
  for (int e = 0; e < KE_PER; ++e) {
    const int i = base + e * KE_THREADS + threadIdx.x;
    if (i < n) {
      const float v = Df[i];
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
    part[(int64_t)img * nblk + blockIdx.x] = t;
  }
}

__global__ void kn_entropy_final(int B, int n, int nblk, const double2* __restrict__ part, double* __restrict__ out_entropy,
                                 double* __restrict__ out_degree) {
  const int img = blockIdx.x * blockDim.x + threadIdx.x;
  if (img >= B) return;
  double a = 0.0, b = 0.0;
  for (int k = 0; k < nblk; ++k) { const double2 t = part[(int64_t)img * nblk + k]; a += t.x; b += t.y; }
  double H = 0.0, deg = 0.0;
  if (a > 0.0) {
    H = log(a) - b / a;
    if (H < 0.0) H = 0.0;
    if (n > 1) deg = 1.0 - H / log((double)n);
  }
  out_entropy[img] = H;
  out_degree[img] = deg;
}

}  // namespace ffpp

namespace {

constexpr int kNoallocMaxDevices = 64;
std::mutex g_noalloc_mu;
double2* g_noalloc_ptr[kNoallocMaxDevices] = {};     // device address of g_noalloc_scratch, per device ordinal

// device address of the scratch array on the CURRENT device (looked up once per device; no allocation)
int noalloc_scratch(double2** out) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return cuda_fail(nullptr, e, "cudaGetDevice");
  if (dev < 0 || dev >= kNoallocMaxDevices) return fail(nullptr, FFPP_ECAPACITY, "ffpp_heatmap_entropy_noalloc: device ordinal beyond 63");
  std::lock_guard<std::mutex> lock(g_noalloc_mu);
  if (!g_noalloc_ptr[dev]) {
    void* p = nullptr;
    e = cudaGetSymbolAddress(&p, g_noalloc_scratch);
    if (e != cudaSuccess || !p) return cuda_fail(nullptr, e, "cudaGetSymbolAddress(g_noalloc_scratch)");
    g_noalloc_ptr[dev] = static_cast<double2*>(p);
  }
  *out = g_noalloc_ptr[dev];
  return FFPP_OK;
}

}  // namespace

extern "C" int ffpp_heatmap_entropy_noalloc(const float* density, int32_t B, int32_t gw, int32_t gh, void* stream, double* out_entropy,
                                            double* out_degree) {
  using namespace ffpp;
  if (B < 0) return fail(nullptr, FFPP_EINVAL, "ffpp_heatmap_entropy_noalloc: B < 0");
  if (B == 0) return FFPP_OK;
  if (!density || !out_entropy || !out_degree) return fail(nullptr, FFPP_EINVAL, "ffpp_heatmap_entropy_noalloc: null pointer");
  if (gw < 1 || gh < 1 || (int64_t)gw * gh >= ((int64_t)1 << 31)) return fail(nullptr, FFPP_EINVAL, "ffpp_heatmap_entropy_noalloc: grid size out of range");
  if (B > 65535) return fail(nullptr, FFPP_ECAPACITY, "ffpp_heatmap_entropy_noalloc: more than 65535 grids in one call");
  const int n = gw * gh;
  const int nblk = (n + KE_THREADS * KE_PER - 1) / (KE_THREADS * KE_PER);
  if ((int64_t)B * nblk > FFPP_NOALLOC_MAX_BLOCKS)
    return fail(nullptr, FFPP_ECAPACITY,
                "ffpp_heatmap_entropy_noalloc: B * ceil(gw*gh/2048) = " + std::to_string((int64_t)B * nblk) + " exceeds the static scratch of " +
                    std::to_string(FFPP_NOALLOC_MAX_BLOCKS) + " blocks (256 KiB); split the batch or use ffpp_heatmap_stats");
  double2* scratch = nullptr;
  const int rc = noalloc_scratch(&scratch);
  if (rc != FFPP_OK) return rc;
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  kn_entropy_partial<<<dim3((unsigned)nblk, (unsigned)B), KE_THREADS, 0, st>>>(density, n, nblk, scratch);
  kn_entropy_final<<<(B + 127) / 128, 128, 0, st>>>(B, n, nblk, scratch, out_entropy, out_degree);
  const cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return cuda_fail(nullptr, e, "ffpp_heatmap_entropy_noalloc launch");
  return FFPP_OK;
}
