/* ffpp_debug.h — test, calibration and measurement entry points of libffpp.  NOT part of the contract of the path
 * (include/ffpp.h is): nothing here is needed to run it, and every call here may synchronise the device.
 * Used by tests/ (to localise a parity failure) and bench.py (calibration reads, device-counted work for the a3
 * roofline). */
#ifndef FFPP_DEBUG_H_
#define FFPP_DEBUG_H_

#include "ffpp.h"

#ifdef __cplusplus
extern "C" {
#endif

/* Readback of per-stage intermediates of the LAST run (synchronises the device).
 *   what = 0: survivor count per frame after thresholding       dst HOST int32 [B]
 *   what = 1: sorted count per frame  min(n, top_k)             dst HOST int32 [B]
 *   what = 2: candidate indices of the top-K set in the order   dst HOST int32 [B][top_k] (rows past the count: -1)
 *             of O4 (the device holds the set with its keys in spatial order; the readback sorts by key on the host)
 *   what = 3: decoded boxes of the top-K set, same order        dst HOST float [B][top_k][4]
 *   what = 4: a3 work counters of the last run made while       dst HOST int64 [4] = culling-box tests (4 fp32
 *             ffpp_debug_count_work was on                       compares each), exact fp32 IoU evaluations (O5),
 *                                                                suppression edges found, frames that overflowed
 *                                                                their edge-pool share (resolved pool-free by their a4 CTA)
 *   what = 5: per-frame flag: 1 = the frame took the a3         dst HOST int32 [B]
 *             overflow path in the last run */
int ffpp_debug_read(ffpp_handle* h, int32_t what, void* dst /*HOST*/, int64_t dst_bytes);

/* When on, the NEXT runs launch the counting instantiation of the a3 kernel (same search, plus one warp-aggregated
 * atomic per warp exit on three device counters that what = 4 reads back).  bench.py does this in a separate,
 * untimed pass: the timed kernels carry no counters. */
int ffpp_debug_count_work(ffpp_handle* h, int32_t enable);

/* Calibration only: enqueue a plain coalesced read of `bytes` bytes of the DEVICE buffer `dev` (16-byte aligned) on
 * `stream`.  Computes nothing of the path; bench.py times it over the raw head output, under the same cold-cache
 * regime as stage a1, to report what a pure read of that size achieves on this GPU, and uses it over a buffer
 * larger than L2 to leave the cache cold AND clean before a timed step. */
int ffpp_debug_stream_read(ffpp_handle* h, const void* dev /*DEVICE*/, int64_t bytes, void* stream);

#ifdef __cplusplus
}
#endif
#endif /* FFPP_DEBUG_H_ */
