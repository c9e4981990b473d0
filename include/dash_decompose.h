/*
 * dash_decompose.h — C ABI of DASH's self-supervised decomposition step (arxiv 2507.19141 §4.1):
 * "We compute motion magnitudes ||dp|| for all Gaussians and set a threshold tau at the top k% percentile of these
 * values.  Gaussians with ||dp|| > tau are classified as dynamic Gaussians, while the rest are classified as static.
 * Static Gaussians are constrained by  L_s = (1/N_s) sum_{p in G_s} ||dp||  (Eq. 5)."
 * dp = phi_l(phi_p(G_3D(p))) (Eq. 3) is produced by dash_hash3d_fwd + dash_mlp_fwd; the index list this call writes is
 * the `index` argument of the G_4D calls (the dynamic subset the 4D encoder is queried for).  Readings: DESIGN.md Q31.
 * All data pointers are DEVICE pointers, caller-owned; the call enqueues on `cuda_stream` and does not synchronise.
 * Return codes as dash_hash4d_status.
 */
#ifndef DASH_DECOMPOSE_H_
#define DASH_DECOMPOSE_H_

#include <stddef.h>
#include <stdint.h>

#include "dash_hash4d.h"

#ifdef __cplusplus
extern "C" {
#endif

/* Written by dash_decompose (device memory, 16 bytes). */
typedef struct dash_decompose_result {
    uint32_t n_dynamic; /* entries written to dyn_index                                              */
    uint32_t n_static;  /* N - n_dynamic = N_s of Eq. 5                                              */
    float tau;          /* the threshold: the largest magnitude not among the m = ceil(N k / 100 - 1e-9) largest;
                           +inf when m = 0, -1 when m = N                                            */
    float loss;         /* L_s of Eq. 5 (0 when N_s = 0)                                             */
} dash_decompose_result;

/* Bytes of device workspace for N Gaussians (16-byte aligned). */
DASH_API size_t dash_decompose_workspace_bytes(uint64_t N);

/*   dp          [N][3] fp32: the linear-motion estimate of every Gaussian (Eq. 4).
 *   k_percent   in [0, 100]: the "top k %".
 *   mag         [N] fp32, written: ||dp[n]|| formed in binary32 as sqrt((x*x + y*y) + z*z), no contraction; NaN -> 0.
 *   dyn_index   [N] int32 capacity; the first result->n_dynamic entries are written: the dynamic Gaussians
 *               (mag > tau, strictly) in ascending order.  At most m entries; fewer when magnitudes tie at tau.
 *   result      one dash_decompose_result (device), written.
 *   ddp         nullable, [N][3] fp32, written: grad_scale * dL_s/d dp = grad_scale * dp[n] / (mag[n] * N_s) for static
 *               n with mag[n] > 0, else 0 (the classification is held fixed).
 * Exact k-th order statistic by a hand-written 4-pass radix select on the magnitudes' bit patterns; ascending
 * compaction by block scan.  The index list, counts and tau are unique results (compared bit-exactly with the oracle);
 * the loss is a double-precision sum in a fixed order (deterministic run to run). */
DASH_API int dash_decompose(uint64_t N, const float* dp, double k_percent, float grad_scale, float* mag,
                            int32_t* dyn_index, dash_decompose_result* result, float* ddp,
                            void* workspace, size_t workspace_bytes, void* cuda_stream);

#ifdef __cplusplus
}
#endif
#endif /* DASH_DECOMPOSE_H_ */
