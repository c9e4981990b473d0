/*
 * dash_ceilings.h — C ABI of the microbenchmarks that establish the chip ceilings of the encoder's access
 * patterns (SURVEY.md §7 step 5, §8d "the L2/atomic ceilings must be measured"): random 8/16/32-byte gathers,
 * random fp32 vector reductions, same-address contention, shared-memory fp32 atomics, TMA bulk gathers, and a
 * stream copy.  `bench.py --ceilings` drives them and prints one JSON line; DESIGN.md §11 and the
 * `roofline.ceilings` object of the normal bench line quote its numbers.  Measurement infrastructure: nothing
 * of the method (Eq. 7-9) is computed here.
 *
 * One call = one kernel launch on `cuda_stream`; the caller times it with CUDA events.  All pointers are DEVICE
 * pointers, caller-owned.  Return codes as dash_hash4d_status (include/dash_hash4d.h).
 */
#ifndef DASH_CEILINGS_H_
#define DASH_CEILINGS_H_

#include <stddef.h>
#include <stdint.h>

#include "dash_hash4d.h"

#ifdef __cplusplus
extern "C" {
#endif

enum dash_ceiling_kind {
    DASH_CEIL_COPY = 0,        /* buf[i] -> sink[i], 16 bytes per thread per iteration (HBM stream)            */
    DASH_CEIL_GATHER = 1,      /* ld.global.nc of `width` bytes (8, 16 or 32 = two 16-byte loads) per lane      */
    DASH_CEIL_RED = 2,         /* red.global.add.f32 / .v2.f32 / .v4.f32 (width 4, 8, 16) per lane, no return   */
    DASH_CEIL_SMEM_ATOMIC = 3, /* atomicAdd(float) on a 32 KB shared array (a CAS loop on sm_100a), width 4     */
    DASH_CEIL_TMA_GATHER = 4,  /* cp.async.bulk global -> shared of 16 bytes per lane, mbarrier completion        */
    DASH_CEIL_SMEM_ATOMIC_U64 = 5 /* atomicAdd(unsigned long long) on the shared array (native ATOMS), width 8  */
};

enum dash_ceiling_pattern {
    DASH_CEIL_INDEPENDENT = 0, /* every lane its own random slot                                               */
    DASH_CEIL_PAIR_ALIGNED = 1,/* lanes 2j, 2j+1 take slots 2r, 2r+1: always one 32-byte sector (width <= 16)   */
    DASH_CEIL_PAIR_XCORNER = 2 /* lanes 2j, 2j+1 take slots r, r+1 (any r): the x-corner pair of the kernels    */
};

typedef struct dash_ceiling_params {
    uint32_t struct_size;     /* = sizeof(dash_ceiling_params)                                                 */
    uint32_t kind;            /* dash_ceiling_kind                                                             */
    uint32_t width;           /* bytes per lane access (see kind)                                              */
    uint32_t pattern;         /* dash_ceiling_pattern                                                          */
    uint64_t footprint_bytes; /* slots are drawn from [0, footprint_bytes): 16 MiB = L2-resident, 1 GiB = HBM;
                                 a tiny footprint gives the same-address contention case                       */
    uint32_t grid;            /* CTAs; 0 = 8 x SM count                                                        */
    uint32_t block;           /* threads per CTA, multiple of 32, <= 1024; 0 = 256                             */
    uint32_t dyn_smem;        /* extra dynamic shared memory per CTA (bytes) to limit CTAs per SM              */
    uint32_t iters;           /* loop trips per thread; each trip issues 8 independent accesses                */
    uint32_t seed;
    uint32_t reserved;
} dash_ceiling_params;

/* Launches the microbenchmark.  buf: footprint_bytes bytes (COPY: also the source), 16-byte aligned; sink:
 * COPY: footprint_bytes bytes, otherwise >= 16 bytes (keeps the loads alive).  *lane_ops (host, nullable)
 * receives the number of lane accesses the launch performs = grid * block * iters * 8 (COPY: 16-byte units). */
DASH_API int dash_ceiling_launch(const dash_ceiling_params* p, void* buf, void* sink, uint64_t* lane_ops,
                                 void* cuda_stream);

#ifdef __cplusplus
}
#endif
#endif /* DASH_CEILINGS_H_ */
