// decompose_kernels.cu — self-supervised decomposition (include/dash_decompose.h; Eq. 5; DESIGN.md
// Q31): motion magnitudes, the exact top-k % threshold by a 4-pass radix select on the fp32 bit patterns (non-negative
// floats order like their bits), the ascending index list of the dynamic Gaussians by block scan, L_s and its gradient.
#include <cuda_runtime.h>

#include <cmath>
#include <cstdint>

#include "../../include/dash_decompose.h"
#include "api_errors.h"       // api_fail, api_cuda_fail, api_ok
#include "deform_kernels.h"   // count_launch, device_sm_count

namespace dash {
namespace {

constexpr int kThreads = 1024;   // one block = 1024 Gaussians in the classify / compact passes

struct SelectState {     // in the workspace
    uint32_t prefix;     // bits of tau decided so far (from the most significant byte down)
    uint32_t mask;       // which bits of `prefix` are decided
    uint32_t rank;       // rank still to descend, counted from the largest (0-based)
    uint32_t tau_bits;   // final threshold
    uint32_t hist[4][256];
};

__global__ void __launch_bounds__(256)
magnitude_kernel(uint64_t N, const float* __restrict__ dp, float* __restrict__ mag) {
    const uint64_t n = static_cast<uint64_t>(blockIdx.x) * 256 + threadIdx.x;
    if (n >= N) return;
    const float x = __ldg(dp + n * 3), y = __ldg(dp + n * 3 + 1), z = __ldg(dp + n * 3 + 2);
    const float v = __fsqrt_rn(__fadd_rn(__fadd_rn(__fmul_rn(x, x), __fmul_rn(y, y)), __fmul_rn(z, z)));
    mag[n] = (v != v) ? 0.0f : v;
}

// pass p (3 = most significant byte): histogram of byte p over the magnitudes whose decided bits match the prefix
__global__ void __launch_bounds__(256)
select_hist_kernel(uint64_t N, const float* __restrict__ mag, SelectState* __restrict__ st, int pass) {
    __shared__ uint32_t h[256];
    h[threadIdx.x] = 0;
    __syncthreads();
    const uint32_t prefix = st->prefix, mask = st->mask;
    const size_t stride = static_cast<size_t>(gridDim.x) * 256;
    for (uint64_t n = static_cast<uint64_t>(blockIdx.x) * 256 + threadIdx.x; n < N; n += stride) {
        const uint32_t key = __float_as_uint(__ldg(mag + n));
        if (((key ^ prefix) & mask) == 0u) atomicAdd(&h[(key >> (8 * pass)) & 0xffu], 1u);
    }
    __syncthreads();
    if (h[threadIdx.x]) atomicAdd(&st->hist[pass][threadIdx.x], h[threadIdx.x]);
}

// descend: the bin (from the top) that holds the element of the remaining rank
__global__ void select_pick_kernel(SelectState* st, int pass) {
    if (threadIdx.x != 0) return;
    uint32_t rank = st->rank, above = 0;
    int b = 255;
    for (; b > 0; --b) {
        const uint32_t c = st->hist[pass][b];
        if (rank < above + c) break;
        above += c;
    }
    st->rank = rank - above;
    st->prefix |= static_cast<uint32_t>(b) << (8 * pass);
    st->mask |= 0xffu << (8 * pass);
    if (pass == 0) st->tau_bits = st->prefix;
}

__global__ void set_tau_kernel(SelectState* st, uint32_t bits) { st->tau_bits = bits; }

// per block of 1024: how many are dynamic, and the double-precision sum of the static magnitudes
__global__ void __launch_bounds__(kThreads)
classify_count_kernel(uint64_t N, const float* __restrict__ mag, const SelectState* __restrict__ st,
                      uint32_t* __restrict__ block_dyn, double* __restrict__ block_sum) {
    __shared__ uint32_t cnt[32];
    __shared__ double sum[32];
    const float tau = __uint_as_float(st->tau_bits);
    const uint64_t n = static_cast<uint64_t>(blockIdx.x) * kThreads + threadIdx.x;
    const float m = n < N ? mag[n] : 0.0f;
    const bool dyn = n < N && m > tau;
    const uint32_t lane = threadIdx.x & 31u, w = threadIdx.x >> 5;
    const uint32_t c = __popc(__ballot_sync(0xffffffffu, dyn));
    double s = (n < N && !dyn) ? static_cast<double>(m) : 0.0;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if (lane == 0) { cnt[w] = c; sum[w] = s; }
    __syncthreads();
    if (threadIdx.x == 0) {
        uint32_t ct = 0;
        double st2 = 0.0;
        for (int i = 0; i < 32; ++i) { ct += cnt[i]; st2 += sum[i]; }   // fixed order: deterministic
        block_dyn[blockIdx.x] = ct;
        block_sum[blockIdx.x] = st2;
    }
}

// one CTA: exclusive scan of the block counts in place, total + loss -> result
__global__ void __launch_bounds__(1024)
scan_finalize_kernel(uint64_t N, uint32_t blocks, uint32_t* __restrict__ block_dyn, const double* __restrict__ block_sum,
                     const SelectState* __restrict__ st, dash_decompose_result* __restrict__ result) {
    __shared__ uint32_t warp_sum[32];
    __shared__ uint32_t carry;
    __shared__ double partial[1024];
    if (threadIdx.x == 0) carry = 0;
    __syncthreads();
    const uint32_t lane = threadIdx.x & 31u, w = threadIdx.x >> 5;
    for (uint32_t base = 0; base < blocks; base += 1024u) {
        const uint32_t i = base + threadIdx.x;
        const uint32_t v = i < blocks ? block_dyn[i] : 0u;
        uint32_t x = v;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t y = __shfl_up_sync(0xffffffffu, x, o);
            if (lane >= static_cast<uint32_t>(o)) x += y;
        }
        if (lane == 31) warp_sum[w] = x;
        __syncthreads();
        if (w == 0) {
            uint32_t s = warp_sum[lane];
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const uint32_t y = __shfl_up_sync(0xffffffffu, s, o);
                if (lane >= static_cast<uint32_t>(o)) s += y;
            }
            warp_sum[lane] = s;
        }
        __syncthreads();
        const uint32_t before = carry + (w ? warp_sum[w - 1] : 0u);
        if (i < blocks) block_dyn[i] = before + x - v;
        __syncthreads();
        if (threadIdx.x == 1023) carry = before + x;
        __syncthreads();
    }
    // loss: strided partial sums, then a fixed-order tree
    double s = 0.0;
    for (uint32_t i = threadIdx.x; i < blocks; i += 1024u) s += block_sum[i];
    partial[threadIdx.x] = s;
    __syncthreads();
    for (uint32_t o = 512; o > 0; o >>= 1) {
        if (threadIdx.x < o) partial[threadIdx.x] += partial[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        const uint32_t nd = carry, ns = static_cast<uint32_t>(N) - nd;
        result->n_dynamic = nd;
        result->n_static = ns;
        result->tau = __uint_as_float(st->tau_bits);
        result->loss = ns ? static_cast<float>(partial[0] / static_cast<double>(ns)) : 0.0f;
    }
}

// ascending compaction + gradient of Eq. 5
__global__ void __launch_bounds__(kThreads)
compact_grad_kernel(uint64_t N, const float* __restrict__ dp, const float* __restrict__ mag,
                    const SelectState* __restrict__ st, const uint32_t* __restrict__ block_off,
                    const dash_decompose_result* __restrict__ result, float grad_scale,
                    int32_t* __restrict__ dyn_index, float* __restrict__ ddp) {
    __shared__ uint32_t warp_cnt[32];
    const float tau = __uint_as_float(st->tau_bits);
    const uint64_t n = static_cast<uint64_t>(blockIdx.x) * kThreads + threadIdx.x;
    const float m = n < N ? mag[n] : 0.0f;
    const bool dyn = n < N && m > tau;
    const uint32_t lane = threadIdx.x & 31u, w = threadIdx.x >> 5;
    const uint32_t ballot = __ballot_sync(0xffffffffu, dyn);
    if (lane == 0) warp_cnt[w] = __popc(ballot);
    __syncthreads();
    if (w == 0) {
        uint32_t s = warp_cnt[lane];
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t y = __shfl_up_sync(0xffffffffu, s, o);
            if (lane >= static_cast<uint32_t>(o)) s += y;
        }
        warp_cnt[lane] = s;   // inclusive over warps
    }
    __syncthreads();
    if (dyn) {
        const uint32_t pos = block_off[blockIdx.x] + (w ? warp_cnt[w - 1] : 0u) + __popc(ballot & ((1u << lane) - 1u));
        dyn_index[pos] = static_cast<int32_t>(n);
    }
    if (ddp && n < N) {
        const float ns = static_cast<float>(result->n_static);
        const float g = (!dyn && m > 0.0f) ? __fdiv_rn(grad_scale, __fmul_rn(m, ns)) : 0.0f;
#pragma unroll
        for (int d = 0; d < 3; ++d) ddp[n * 3 + d] = g == 0.0f ? 0.0f : __fmul_rn(g, __ldg(dp + n * 3 + d));
    }
}

__global__ void zero_state_kernel(SelectState* st, uint32_t rank) {
    uint32_t* p = reinterpret_cast<uint32_t*>(st);
    for (uint32_t i = threadIdx.x; i < sizeof(SelectState) / 4; i += blockDim.x) p[i] = 0;
    __syncthreads();
    if (threadIdx.x == 0) st->rank = rank;
}

size_t round16(size_t v) { return (v + 15u) & ~static_cast<size_t>(15u); }

}  // namespace
}  // namespace dash

extern "C" {

DASH_API size_t dash_decompose_workspace_bytes(uint64_t N) {
    const size_t blocks = (N + dash::kThreads - 1) / dash::kThreads;
    return dash::round16(sizeof(dash::SelectState)) + dash::round16(blocks * 4) + dash::round16(blocks * 8);
}

DASH_API int dash_decompose(uint64_t N, const float* dp, double k_percent, float grad_scale, float* mag,
                            int32_t* dyn_index, dash_decompose_result* result, float* ddp, void* workspace,
                            size_t workspace_bytes, void* cuda_stream) {
    using namespace dash;
    if (!(k_percent >= 0.0 && k_percent <= 100.0))
        return api_fail(DASH_HASH4D_INVALID_ARG, "decompose: k_percent = %g outside [0, 100]", k_percent);
    if (!result) return api_fail(DASH_HASH4D_INVALID_ARG, "decompose: result is NULL");
    if (N > 0x7fffffffull) return api_fail(DASH_HASH4D_UNSUPPORTED, "decompose: N too large for an int32 index list");
    if (N && (!dp || !mag || !dyn_index))
        return api_fail(DASH_HASH4D_INVALID_ARG, "decompose: dp, mag or dyn_index is NULL");
    const size_t need = dash_decompose_workspace_bytes(N);
    if (!workspace || workspace_bytes < need)
        return api_fail(DASH_HASH4D_WORKSPACE_TOO_SMALL, "decompose needs %zu workspace bytes, got %zu", need,
                        workspace ? workspace_bytes : static_cast<size_t>(0));
    if (reinterpret_cast<uintptr_t>(workspace) & 15u)
        return api_fail(DASH_HASH4D_INVALID_ARG, "decompose: workspace not 16-byte aligned");
    if (reinterpret_cast<uintptr_t>(result) & 3u)
        return api_fail(DASH_HASH4D_INVALID_ARG, "decompose: result not 4-byte aligned");
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    const uint32_t blocks = static_cast<uint32_t>((N + kThreads - 1) / kThreads);
    char* w = static_cast<char*>(workspace);
    SelectState* st = reinterpret_cast<SelectState*>(w);
    uint32_t* block_dyn = reinterpret_cast<uint32_t*>(w + round16(sizeof(SelectState)));
    double* block_sum = reinterpret_cast<double*>(w + round16(sizeof(SelectState)) + round16(static_cast<size_t>(blocks) * 4));
    const double md = std::ceil(static_cast<double>(N) * k_percent / 100.0 - 1e-9);
    const uint64_t m = md <= 0.0 ? 0 : (md >= static_cast<double>(N) ? N : static_cast<uint64_t>(md));
    // every launch is counted and checked on its own, so a failure names the kernel that caused it
#define DASH_DECOMPOSE_LAUNCHED(what)                                                   \
    do {                                                                                \
        count_launch();                                                                 \
        const cudaError_t le_ = cudaGetLastError();                                     \
        if (le_ != cudaSuccess) return api_cuda_fail(le_, "decompose: " what " launch"); \
    } while (0)
    zero_state_kernel<<<1, 256, 0, s>>>(st, static_cast<uint32_t>(m));
    DASH_DECOMPOSE_LAUNCHED("zero_state");
    if (N) {
        magnitude_kernel<<<static_cast<unsigned>((N + 255) / 256), 256, 0, s>>>(N, dp, mag);
        DASH_DECOMPOSE_LAUNCHED("magnitude");
    }
    if (m == 0 || m >= N) {
        set_tau_kernel<<<1, 1, 0, s>>>(st, m == 0 ? 0x7f800000u : 0xbf800000u);   // +inf / -1
        DASH_DECOMPOSE_LAUNCHED("set_tau");
    } else {
        const size_t want = (N + 255) / 256, cap = static_cast<size_t>(device_sm_count()) * 8;
        const unsigned grid = static_cast<unsigned>(want > cap ? cap : want);
        for (int pass = 3; pass >= 0; --pass) {
            select_hist_kernel<<<grid, 256, 0, s>>>(N, mag, st, pass);
            DASH_DECOMPOSE_LAUNCHED("select_hist");
            select_pick_kernel<<<1, 32, 0, s>>>(st, pass);
            DASH_DECOMPOSE_LAUNCHED("select_pick");
        }
    }
    if (N) {
        classify_count_kernel<<<blocks, kThreads, 0, s>>>(N, mag, st, block_dyn, block_sum);
        DASH_DECOMPOSE_LAUNCHED("classify_count");
    }
    scan_finalize_kernel<<<1, 1024, 0, s>>>(N, blocks, block_dyn, block_sum, st, result);
    DASH_DECOMPOSE_LAUNCHED("scan_finalize");
    if (N) {
        compact_grad_kernel<<<blocks, kThreads, 0, s>>>(N, dp, mag, st, block_dyn, result, grad_scale, dyn_index, ddp);
        DASH_DECOMPOSE_LAUNCHED("compact_grad");
    }
#undef DASH_DECOMPOSE_LAUNCHED
    return api_ok();
}

}  // extern "C"
