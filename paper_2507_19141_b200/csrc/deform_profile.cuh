// deform_profile.cuh — optional clock64() phase timers of deform_fused_kernel, kept out of the kernel body.
// Compiled to nothing unless the library is built with -DDASH_DEFORM_PROFILE (a development build: CTA 0 then prints
// the time stamps of its producer tiles, MMA issues and epilogues at kernel end).  The product build never defines it.
#pragma once

#ifdef DASH_DEFORM_PROFILE
#include <cstdio>
#define DASH_PROF_ENTRY() const long long prof_entry_ = clock64()
// after the setup barrier: one shared time base for all warp roles
#define DASH_PROF_BEGIN(tid)                                                          \
    __shared__ long long prof_[3][64];                                                \
    __shared__ long long prof_t0_;                                                    \
    if ((tid) == 0) { prof_t0_ = clock64(); prof_[0][40] = prof_[0][41] = prof_[0][42] = 0; } \
    __syncthreads();                                                                  \
    const long long prof_setup_ = prof_t0_
#define DASH_PROF(role, idx) \
    do { if (blockIdx.x == 0 && (idx) < 64) prof_[role][idx] = clock64() - prof_setup_; } while (0)
#define DASH_PROF_CLOCK(name) const long long name = clock64()
#define DASH_PROF_ACCUM(cond, issue, wait)                                            \
    do { if (blockIdx.x == 0 && (cond)) { prof_[0][40] += (issue); prof_[0][41] += (wait); prof_[0][42] += 1; } } while (0)
#define DASH_PROF_REPORT(tid, tiles, layers)                                          \
    do {                                                                              \
        if (blockIdx.x == 0 && (tid) == 0) {                                          \
            printf("tiles=%u setup=%lld end=%lld\n", (tiles), prof_setup_ - prof_entry_, clock64() - prof_setup_); \
            printf("warp0 rounds=%lld issue_cycles=%lld wait_cycles=%lld\n", prof_[0][42], prof_[0][40], prof_[0][41]); \
            for (int k_ = 0; k_ < 2 * (int)(tiles) && k_ < 64; ++k_) printf("prod[%d]=%lld\n", k_, prof_[0][k_]); \
            for (int k_ = 0; k_ < (int)((tiles) + 1) / 2 * 2 * (int)(layers) && k_ < 64; ++k_) \
                printf("mma0[%d]=%lld epi0[%d]=%lld\n", k_, prof_[1][k_], k_, prof_[2][k_]); \
        }                                                                             \
    } while (0)
#else
#define DASH_PROF_ENTRY() do { } while (0)
#define DASH_PROF_BEGIN(tid) do { } while (0)
#define DASH_PROF(role, idx) do { } while (0)
#define DASH_PROF_CLOCK(name) do { } while (0)
#define DASH_PROF_ACCUM(cond, issue, wait) do { } while (0)
#define DASH_PROF_REPORT(tid, tiles, layers) do { } while (0)
#endif
