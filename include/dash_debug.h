/*
 * dash_debug.h — tuning overrides of libdash_hash4d.so for sweeps and A/B measurements.  NOT part of the method and not
 * included by the product headers: a program that only uses the encoder never needs this file.  bench.py (--set-debug,
 * --sweep-groups) and a few tests use it to force a schedule the library would not pick on its own.
 */
#ifndef DASH_DEBUG_H_
#define DASH_DEBUG_H_

#include <stdint.h>

#include "dash_hash4d.h"

#ifdef __cplusplus
extern "C" {
#endif

/* Tuning overrides for sweeps and A/B measurements (bench.py --sweep, tests).  Process-wide; value 0 restores the
 * library's own choice; the library reads NO environment variable.  Not part of the method: every setting computes
 * the same result.  Returns INVALID_ARG for an unknown key or a negative value. */
enum dash_debug_key {
    DASH_DEBUG_FWD_GROUP = 0,    /* levels per level group G of fwd / bwd_input / slice_fwd (1..16, power of two) */
    DASH_DEBUG_BWD_GROUP = 1,    /* ... of bwd */
    DASH_DEBUG_SMOOTH_GROUP = 2, /* ... of smooth */
    DASH_DEBUG_DEFORM_PATH = 3,  /* dash_deform_fwd: 1 = fused kernel, 2 = two-pass (encoder -> workspace -> MLP) */
    DASH_DEBUG_BWD_VARIANT = 4,  /* bwd with ZERO_GRAD: 1 = no L2 eviction hints on the zero stores / reductions */
    DASH_DEBUG_BWD_COARSE_LEVELS = 5, /* SORT_COARSE: number of leading levels the run-merged scatter takes */
    DASH_DEBUG_BWD_RUN_CHUNK = 6,     /* SORT_COARSE: consecutive sorted queries per lane pair */
    DASH_DEBUG_FWD_ORDERED_LEVELS = 7, /* SORT_COARSE: number of leading levels the forward walks in the sorted order */
    DASH_DEBUG_SORT_KEY_BITS = 8,      /* SORT_COARSE: cap on the bits of the sort key, 8..22 (bins = 2^bits) */
    DASH_DEBUG_KEY_COUNT = 9
};
DASH_API int dash_hash4d_set_debug(int key, int64_t value);

#ifdef __cplusplus
}
#endif
#endif /* DASH_DEBUG_H_ */
