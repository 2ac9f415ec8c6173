/* ffpp_noalloc.h — ONE entry point of libffpp that allocates nothing, for callers that cannot call cudaMalloc (code
 * under CUDA graph capture, tight serving loops, harnesses that forbid allocation).
 *
 * ffpp_heatmap_entropy_noalloc computes what ffpp_heatmap_stats (ffpp_next.h; PAPER.md:L212, L230:
 * "Compute heatmap, entropy, clustering degree") writes to out_entropy / out_degree — readings B1 and B2 of DESIGN.md §3 —
 * for B density grids of ONE common size.  Its scratch (one pair of doubles per 2048-cell block of every grid) lives in a
 * file-scope `static __device__` array of FFPP_NOALLOC_SCRATCH_BYTES = 256 KiB inside the library: every GPU that loads
 * libffpp holds those 256 KiB until the process exits.  The call needs no handle, calls no cudaMalloc / cudaFree / allocating
 * library routine, and enqueues two kernels on `stream`; the host is not synchronised.  The first call on a device looks
 * the array's device address up (cudaGetSymbolAddress, once per device): make that first call outside stream capture.
 *
 * Limit: B * ceil(gw * gh / 2048) <= FFPP_NOALLOC_MAX_BLOCKS (16384), i.e. up to 33.5 M cells per call; beyond it the call
 * returns FFPP_ECAPACITY and ffpp_last_error(NULL) says so.
 * Sharing: every call on a device uses the same array, which keeps the previous call's contents.  Each slot a call reads
 * is written by that same call first, so nothing has to be cleared — but two calls that OVERLAP on the GPU (different
 * streams, or graph branches without an edge between them) race on it: serialise them.
 */
#ifndef FFPP_NOALLOC_H_
#define FFPP_NOALLOC_H_

#include "ffpp.h"

#ifdef __cplusplus
extern "C" {
#endif

#define FFPP_NOALLOC_MAX_BLOCKS 16384
#define FFPP_NOALLOC_SCRATCH_BYTES (FFPP_NOALLOC_MAX_BLOCKS * 16)

/*   density      DEVICE  float32 [B][gh][gw], row-major, grids concatenated.  Read only.
 *   B, gw, gh    grids, grid width and height in cells (all >= 1; B <= 65535; gw * gh < 2^31).  B == 0: success, no work.
 *   out_entropy  DEVICE  [B] float64: -sum p ln p, p = D / sum(D), cells with D <= 0 skipped; 0 if sum(D) <= 0     (B1)
 *   out_degree   DEVICE  [B] float64: 1 - entropy / ln(gw * gh); 0 if gw * gh <= 1 or sum(D) <= 0                   (B2)
 * Same arithmetic and summation order as ffpp_heatmap_stats: the two agree bit for bit.
 * Errors: FFPP_EINVAL (null pointer, bad size), FFPP_ECAPACITY (limit above), FFPP_ECUDA; text via ffpp_last_error(NULL). */
int ffpp_heatmap_entropy_noalloc(const float* density /*DEVICE*/, int32_t B, int32_t gw, int32_t gh, void* stream,
                                 double* out_entropy /*DEVICE*/, double* out_degree /*DEVICE*/);

#ifdef __cplusplus
}
#endif
#endif /* FFPP_NOALLOC_H_ */
