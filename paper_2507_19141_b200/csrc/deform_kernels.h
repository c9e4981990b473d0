// deform_kernels.h — launch plan and host-callable launchers of the fused deformation kernel (deform_kernels.cu).
#pragma once
#include <cuda_runtime.h>

#include <cstddef>
#include <cstdint>

#include "hash4d_plan.h"

namespace dash {

constexpr uint32_t kDeformTileM = 128;      // queries per tile = rows of one tcgen05.mma (M = 128, cta_group::1)
constexpr uint32_t kDeformEncWarps = 24;    // producer warps (multiple of 4 so that the epilogue warps that follow
                                            // have warp % 4 = 0..3, the TMEM lane quarter each may read)
constexpr uint32_t kDeformPipes = 2;        // independent consumer pipelines (even / odd tiles): each has 4 warps
                                            // (MMA issue + epilogue), its own TMEM accumulator, activation buffer
                                            // and barriers, so one tile's epilogue overlaps the other's MMAs
constexpr uint32_t kDeformThreads = (kDeformEncWarps + 4 * kDeformPipes) * 32;   // 1024
constexpr uint32_t kMlpMaxLayers = 4;
constexpr uint32_t kMlpMaxWidth = 256;      // one tcgen05.mma covers N <= 256
constexpr uint32_t kDeformSmemLimit = 227u * 1024u;

// Dense-layer chain: widths, padded operand shapes and the shared-memory map of one CTA.
struct MlpPlan {
    uint64_t N;                  // rows (queries)
    uint32_t num_tiles;          // ceil(N / 128)
    uint32_t grid;               // CTAs: min(SM count, num_tiles)
    uint64_t rows_per_cta;       // ceil(N / grid): CTA b owns rows [b * rows_per_cta, ...)
    uint32_t n_layers;
    uint32_t width[kMlpMaxLayers + 1];  // width[0] inputs, width[l] outputs of layer l (as given)
    uint32_t kbias[kMlpMaxLayers];      // input width of layer l rounded up to 16: column of the bias (hi, lo) pair
    uint32_t kpad[kMlpMaxLayers];       // K of layer l = kbias[l] + 16
    uint32_t npad[kMlpMaxLayers];       // N of layer l: its output width rounded up to 16
    uint32_t p_off[kMlpMaxLayers];      // float offset of W_l in the packed parameter buffer (b_l follows W_l)
    uint32_t w_off[kMlpMaxLayers];      // byte offset of the bf16 operand copy of W_l in shared memory
    uint32_t a0_off;             // two A buffers of the first layer, 128 x kpad[0] bf16 each
    uint32_t out_stage_off;      // 2 KB per consumer warp to transpose a narrow (<= 16 wide) output tile; 0 = unused
    uint32_t smem_bytes;
    uint32_t tmem_cols;          // allocated TMEM columns: power of two >= npipes * tmem_pipe_cols, >= 32
    uint32_t tmem_pipe_cols;     // per pipeline: accumulator (max npad) + bf16 A operand of layers 2..n (max kpad/2)
    uint32_t tmem_a_off;         // column offset of the A operand inside a pipeline's region (= max npad)
    uint32_t npipes;             // consumer pipelines in use: 2 when both fit the 512 TMEM columns, else 1
    uint32_t n_out;              // width[n_layers]
};

// Backward through the chain (mlp_bwd_kernels.cu): shared-memory / tensor-memory map of one CTA.  The forward is
// recomputed per 128-row tile; every operand tile is bf16 in the same no-swizzle core-matrix layout (chunk (row, c) at
// c * (rows*16+16) + row*16), read K-major by the forward / dgrad MMAs and MN-major by the wgrad MMAs.
constexpr uint32_t kMlpBwdThreads = 256;    // warps 0-3: MMA issue + epilogues (TMEM lane quarters); warps 4-7: loaders
struct MlpBwdPlan {
    MlpPlan fwd;                        // widths, paddings, p_off; w_off / a0_off / smem_bytes are re-laid-out below
    uint32_t w_off[kMlpMaxLayers];      // bf16 weights of layer l, [npad][kpad] (as in the forward)
    uint32_t a_off[kMlpMaxLayers];      // activation tile a_l, l = 0..n-1: 128 x kpad[l]; a_0 is double buffered
    uint32_t a0_bytes;                  // bytes of one a_0 buffer
    uint32_t d_off[2];                  // delta tiles (ping-pong), 128 x 128
    uint32_t dn_off;                    // delta_n tile (from dout), 128 x npad[n-1]
    uint32_t bar_off;                   // mbarriers + TMEM slot
    uint32_t smem_bytes;
    uint32_t acc_col;                   // working accumulator (forward z_l / dgrad g): columns [acc_col, acc_col + acc_cols)
    uint32_t acc_cols;
    uint32_t dw_col[kMlpMaxLayers];     // persistent wgrad accumulators: kpad[l] columns each, lane = output row j
    uint32_t tmem_cols;                 // power of two >= total, <= 512
};

cudaError_t launch_mlp_bwd(const MlpBwdPlan& B, const float* feat, const float* params, const float* dout,
                           float* dfeat, float* dparams, cudaStream_t s);

cudaError_t launch_deform_fused(const Plan& P, const MlpPlan& M, const float* xyz, const float* t,
                                const int32_t* index, const void* table, bool table_half,
                                const float* params, const float* base, float* out, int sms,
                                cudaStream_t s);
cudaError_t launch_mlp(const MlpPlan& M, const float* feat, const float* params, const float* base,
                       float* out, int sms, cudaStream_t s);

void count_launch();   // bumps the per-thread launch counter kept in hash4d_kernels.cu
int device_sm_count();      // of the current device, cached per device ordinal
size_t device_l2_bytes();

}  // namespace dash
