// hash4d_kernels.h — host-callable launchers of the sm_100a kernels (hash4d_kernels.cu).
#pragma once
#include <cuda_runtime.h>

#include <cstddef>
#include <cstdint>

#include "hash4d_plan.h"

namespace dash {

// Header of the caller's workspace when a flag needs one (DETERMINISTIC_BWD / VALIDATE_INPUTS).
// What a SORT_COARSE sort was computed for: written behind the order by the sort's last kernel, compared by a later
// ORDER_READY call when VALIDATE_INPUTS lets it synchronise (hash4d_api.cu).  Plain words so that memcmp decides.
struct OrderStamp {
    uint32_t w[12];
};

struct WorkspaceHeader {
    uint32_t absmax_bits;   // max |dout| as binary32 bits (deterministic bwd)
    float scale;            // fixed-point scale 2^s
    double inv_scale;       // 2^-s
    uint32_t bad_inputs;    // VALIDATE_INPUTS: coordinates that are NaN or outside [0,1)
    uint32_t pad0[11];      // the first 64 bytes are per-call scratch (zeroed by VALIDATE_INPUTS)
    OrderStamp order_stamp; // bytes 64..111: survives from the call that sorted to the calls that reuse the order
    uint32_t pad1[4];
};
static_assert(sizeof(WorkspaceHeader) == 128, "workspace header is 128 bytes");
constexpr size_t kHeaderScratchBytes = 64;

// order / sorted_q (both or neither; G_4D only): walk the queries in the cell-sorted order of launch_coarse_sort
cudaError_t launch_fwd(const Plan& P, const float* xyz, const float* t, const int32_t* index,
                       const void* table, bool table_half, float* out, cudaStream_t s,
                       const int32_t* order = nullptr, const float4* sorted_q = nullptr);
cudaError_t launch_bwd_input(const Plan& P, const float* xyz, const float* t, const int32_t* index,
                             const void* table, bool table_half, const float* dout, float* dq,
                             cudaStream_t s, const int32_t* order = nullptr, const float4* sorted_q = nullptr);
cudaError_t launch_smooth(const Plan& P, const float* xyz, const float* t, const int32_t* index,
                          const float* eps, uint32_t eps_stride, const void* table, bool table_half,
                          float two_scale, float* loss, float* dtable, cudaStream_t s);
cudaError_t launch_bwd(const Plan& P, const float* xyz, const float* t, const int32_t* index,
                       const float* dout, float* dtable, cudaStream_t s, bool l2_hint = false);
cudaError_t launch_bwd_fixed(const Plan& P, const float* xyz, const float* t, const int32_t* index,
                             const float* dout, long long* acc, const WorkspaceHeader* hdr,
                             cudaStream_t s);
cudaError_t launch_indices(const Plan& P, const float* xyz, const float* t, const int32_t* index,
                           uint32_t* idx_out, float* w_out, cudaStream_t s);
cudaError_t launch_zero(void* ptr, size_t bytes, cudaStream_t s, bool l2_hint = false);
cudaError_t launch_absmax(const float* v, size_t count, WorkspaceHeader* hdr, uint64_t N,
                          cudaStream_t s);
cudaError_t launch_fixed_finalize(const long long* acc, float* dtable, size_t count,
                                  const WorkspaceHeader* hdr, bool overwrite, cudaStream_t s);
cudaError_t launch_sort_queries(uint64_t N, const float* xyz, uint32_t xyz_stride, const int32_t* index,
                                uint32_t bits, int32_t* order, uint32_t* keys, uint32_t* bins, uint32_t* totals,
                                cudaStream_t s);
constexpr uint32_t kScanTile = 4096;   // bins one CTA of the exclusive scan covers
cudaError_t launch_exclusive_scan_u32(uint32_t* bins, uint32_t n_bins, uint32_t* totals, cudaStream_t s,
                                      bool add_offsets = true);
// Run-merged scatter of the coarse levels (bwd_runs_kernels.cu; DASH_HASH4D_FLAG_SORT_COARSE): sort the queries by the
// 4D cell of level `key_level`, then reduce runs of queries that share a cell in registers before they reach L2.
struct CoarseSort {
    uint32_t levels;      // leading levels [0, levels) taken by the run-merged scatter (0: path not used)
    uint32_t levels_fwd;  // leading levels the FORWARD walks in the sorted order (>= levels)
    uint32_t key_level;   // the cell of this level is the sort key (the finest of them)
    uint32_t bits_s, bits_t, shift_s, shift_t;  // Morton key: (cell >> shift) per axis, bits per spatial axis / for t
    uint32_t chunk;       // consecutive sorted queries walked by one lane pair
    uint32_t n_bins;      // 1 << (3 bits_s + bits_t)
};
// order[i] = number of the i-th query in key order, sorted_q[i] = its (x, y, z, t); keys / bins / totals: scratch
cudaError_t launch_coarse_sort(const Plan& P, const CoarseSort& cs, const float* xyz, const float* t,
                               const int32_t* index, int32_t* order, float4* sorted_q, uint32_t* keys, uint32_t* bins,
                               uint32_t* totals, cudaStream_t s, WorkspaceHeader* hdr, const OrderStamp& stamp);
cudaError_t launch_bwd_runs(const Plan& P, const CoarseSort& cs, const float* dout, float* dtable, const int32_t* order,
                            const float4* sorted_q, cudaStream_t s, bool l2_hint);
cudaError_t launch_slice_t(const Plan& P, const float* t, const void* table, bool table_half, float* slice,
                           cudaStream_t s);
cudaError_t launch_adam(size_t count, double lr, double beta1, double beta2, double eps, uint32_t step,
                        bool zero_grad, float* theta, void* theta16, float* grad, float* m, float* v,
                        cudaStream_t s);
cudaError_t launch_validate(const Plan& P, const float* xyz, const float* t, const int32_t* index,
                            WorkspaceHeader* hdr, cudaStream_t s);

uint64_t launch_counter(bool reset);

}  // namespace dash
