/*
 * bkgdet_debug.h -- diagnostic entry points of libbkgdet.  Not part of the hot path: the parity tests use them to
 * force both paths of kernel K1 and to read its path counters, bench.py uses the event hook to time one kernel of a
 * call on the launching stream.  They change no result.  Same conventions as bkgdet.h (int status codes).
 */
#ifndef BKGDET_DEBUG_H
#define BKGDET_DEBUG_H

#include "bkgdet.h"

#ifdef __cplusplus
extern "C" {
#endif

/* Number of meshes that took K1's general path (a sweep per clipping round + radix select) since the last reset.
 * Reads a device counter: synchronise the stream first.  *out may be NULL. */
int bd_debug_k1_slow_meshes(unsigned long long *out, int reset);

/* Why meshes left K1's fast path, 8 counters: [1] degenerate sample, [2] tail list full, [3] median rank outside the
 * bracket, [4] median bin larger than the candidate window, [5] a round's median rank left the window, [6] a clipping
 * bound entered the core interval, [7] mask-aware statistics requested (bd_mesh_stats_masked).  out8: HOST array. */
int bd_debug_k1_reasons(unsigned long long *out8, int reset);

/* on != 0: K1 skips its fast path for this context (the tests exercise both paths; results are identical). */
int bd_debug_k1_force_slow(bd_ctx *ctx, int on);

/* CUDA events (cudaEvent_t passed as void*, NULL = off) that the following detect_sources / bkg_subtract_detect calls
 * record on their stream immediately before and after the tile kernel, so a caller can time that kernel alone. */
int bd_debug_tile_kernel_events(bd_ctx *ctx, void *ev_before, void *ev_after);

#ifdef __cplusplus
}
#endif
#endif /* BKGDET_DEBUG_H */
