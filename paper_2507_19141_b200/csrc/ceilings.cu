// ceilings.cu — microbenchmarks behind include/dash_ceilings.h: the chip ceilings of the encoder's access patterns
// (random gathers, vector reductions, contention, shared-memory atomics, TMA bulk gathers, stream copy).
// Measurement infrastructure, driven by `bench.py --ceilings`; nothing of the method is computed here.
#include <cuda_runtime.h>

#include <cstdint>

#include "../../include/dash_ceilings.h"

namespace dash {
namespace {

constexpr int kUnroll = 8;  // independent accesses per loop trip (the kernels keep 8 gathers / REDs in flight)

struct CeilArgs {
    unsigned char* buf;
    unsigned char* sink;
    uint64_t slot_mask;  // slots - 1 (power of two)
    uint32_t width, pattern, iters, seed;
    uint64_t n16;        // COPY: 16-byte units in buf
};

__device__ __forceinline__ uint32_t mix(uint32_t x) {
    x ^= x >> 16; x *= 0x7feb352du; x ^= x >> 15; x *= 0x846ca68bu; x ^= x >> 16;
    return x;
}

// slot of access j of trip i for this lane under the pattern
__device__ __forceinline__ uint64_t pick_slot(const CeilArgs& a, uint32_t gid, uint32_t i, int j) {
    const uint32_t who = a.pattern == DASH_CEIL_INDEPENDENT ? gid : (gid >> 1);
    const uint32_t r = mix(a.seed + who * 0x9E3779B1u + (i * kUnroll + j) * 0x85EBCA6Bu);
    uint64_t r64 = (static_cast<uint64_t>(mix(r ^ 0x68bc21ebu)) << 32 | r) & a.slot_mask;
    if (a.pattern == DASH_CEIL_PAIR_ALIGNED) r64 = (r64 & ~1ull) | (gid & 1u);
    if (a.pattern == DASH_CEIL_PAIR_XCORNER) r64 = (r64 + (gid & 1u)) & a.slot_mask;
    return r64;
}

__global__ void copy_kernel(const CeilArgs a) {
    const uint64_t threads = static_cast<uint64_t>(gridDim.x) * blockDim.x;
    const uint64_t gid = static_cast<uint64_t>(blockIdx.x) * blockDim.x + threadIdx.x;
    const uint4* src = reinterpret_cast<const uint4*>(a.buf);
    uint4* dst = reinterpret_cast<uint4*>(a.sink);
    for (uint32_t i = 0; i < a.iters; ++i) {
        uint4 v[kUnroll];
#pragma unroll
        for (int j = 0; j < kUnroll; ++j) {
            const uint64_t e = (static_cast<uint64_t>(i) * kUnroll + j) * threads + gid;
            v[j] = e < a.n16 ? __ldcs(src + e) : make_uint4(0, 0, 0, 0);
        }
#pragma unroll
        for (int j = 0; j < kUnroll; ++j) {
            const uint64_t e = (static_cast<uint64_t>(i) * kUnroll + j) * threads + gid;
            if (e < a.n16) __stcs(dst + e, v[j]);
        }
    }
}

template <int WIDTH>
__global__ void gather_kernel(const CeilArgs a) {
    const uint32_t gid = blockIdx.x * blockDim.x + threadIdx.x;
    uint32_t acc = 0;
    for (uint32_t i = 0; i < a.iters; ++i) {
        uint32_t got[kUnroll];
#pragma unroll
        for (int j = 0; j < kUnroll; ++j) {
            const unsigned char* p = a.buf + pick_slot(a, gid, i, j) * WIDTH;
            if constexpr (WIDTH == 4) {
                got[j] = __ldg(reinterpret_cast<const uint32_t*>(p));
            } else if constexpr (WIDTH == 8) {
                const uint2 v = __ldg(reinterpret_cast<const uint2*>(p));
                got[j] = v.x ^ v.y;
            } else if constexpr (WIDTH == 16) {
                const uint4 v = __ldg(reinterpret_cast<const uint4*>(p));
                got[j] = v.x ^ v.y ^ v.z ^ v.w;
            } else {
                const uint4 v = __ldg(reinterpret_cast<const uint4*>(p));
                const uint4 w = __ldg(reinterpret_cast<const uint4*>(p) + 1);
                got[j] = v.x ^ v.y ^ v.z ^ v.w ^ w.x ^ w.y ^ w.z ^ w.w;
            }
        }
#pragma unroll
        for (int j = 0; j < kUnroll; ++j) acc ^= got[j];
    }
    if (acc == 0x9e3779b9u) reinterpret_cast<uint32_t*>(a.sink)[0] = acc;  // keeps the loads alive
}

template <int WIDTH>
__global__ void red_kernel(const CeilArgs a) {
    const uint32_t gid = blockIdx.x * blockDim.x + threadIdx.x;
    for (uint32_t i = 0; i < a.iters; ++i) {
#pragma unroll
        for (int j = 0; j < kUnroll; ++j) {
            float* p = reinterpret_cast<float*>(a.buf + pick_slot(a, gid, i, j) * WIDTH);
            if constexpr (WIDTH == 4)
                asm volatile("red.global.add.f32 [%0], %1;" ::"l"(p), "f"(1.0f) : "memory");
            else if constexpr (WIDTH == 8)
                asm volatile("red.global.add.v2.f32 [%0], {%1, %2};" ::"l"(p), "f"(1.0f), "f"(2.0f) : "memory");
            else
                asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(p), "f"(1.0f), "f"(2.0f),
                             "f"(3.0f), "f"(4.0f)
                             : "memory");
        }
    }
}

constexpr int kSmemAtomicBytes = 32 * 1024;

template <typename T>
__global__ void smem_atomic_kernel(const CeilArgs a) {
    __shared__ T acc[kSmemAtomicBytes / sizeof(T)];
    constexpr uint32_t kSlots = kSmemAtomicBytes / sizeof(T);
    for (uint32_t e = threadIdx.x; e < kSlots; e += blockDim.x) acc[e] = T(0);
    __syncthreads();
    const uint32_t gid = blockIdx.x * blockDim.x + threadIdx.x;
    for (uint32_t i = 0; i < a.iters; ++i) {
#pragma unroll
        for (int j = 0; j < kUnroll; ++j) {
            const uint32_t s = static_cast<uint32_t>(pick_slot(a, gid, i, j)) & (kSlots - 1u);
            atomicAdd(&acc[s], T(1));
        }
    }
    __syncthreads();
    if (acc[threadIdx.x & (kSlots - 1u)] == T(123456789)) reinterpret_cast<uint32_t*>(a.sink)[0] = 1u;
}

__global__ void tma_gather_kernel(const CeilArgs a) {
    extern __shared__ __align__(128) unsigned char dyn[];
    __shared__ __align__(8) uint64_t bar;
    const uint32_t bar_s = static_cast<uint32_t>(__cvta_generic_to_shared(&bar));
    const uint32_t dst0 = static_cast<uint32_t>(__cvta_generic_to_shared(dyn)) + threadIdx.x * (kUnroll * 16);
    if (threadIdx.x == 0) {
        asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(bar_s) : "memory");
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    const uint32_t gid = blockIdx.x * blockDim.x + threadIdx.x;
    const uint32_t bytes = blockDim.x * kUnroll * 16;
    for (uint32_t i = 0; i < a.iters; ++i) {
        if (threadIdx.x == 0)
            asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar_s), "r"(bytes) : "memory");
#pragma unroll
        for (int j = 0; j < kUnroll; ++j) {
            const unsigned char* src = a.buf + pick_slot(a, gid, i, j) * 16;
            asm volatile(
                "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], 16, [%2];" ::"r"(
                    dst0 + j * 16),
                "l"(src), "r"(bar_s)
                : "memory");
        }
        uint32_t done = 0;
        while (!done) {
            asm volatile(
                "{\n.reg .pred p;\nmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\nselp.u32 %0, 1, 0, p;\n}"
                : "=r"(done)
                : "r"(bar_s), "r"(i & 1u)
                : "memory");
        }
    }
}

}  // namespace
}  // namespace dash

namespace {
// Built as its own library (libdash_ceilings.so): nothing here is shared with the product library.
uint32_t sm_count_of_current_device() {
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess ||
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms <= 0)
        return 148u;
    return static_cast<uint32_t>(sms);
}
#ifndef DASH_CEIL_BUILD_ID_STRING
#define DASH_CEIL_BUILD_ID_STRING "unknown"
#endif
__attribute__((used)) const char kCeilBuildId[] = "DASH_CEIL_BUILD_ID=" DASH_CEIL_BUILD_ID_STRING;
}  // namespace

extern "C" DASH_API int dash_ceiling_launch(const dash_ceiling_params* p, void* buf, void* sink,
                                            uint64_t* lane_ops, void* cuda_stream) {
    using namespace dash;
    if (!p || p->struct_size != sizeof(dash_ceiling_params) || !buf || !sink) return DASH_HASH4D_INVALID_ARG;
    if ((reinterpret_cast<uintptr_t>(buf) | reinterpret_cast<uintptr_t>(sink)) & 15u) return DASH_HASH4D_INVALID_ARG;
    const uint32_t block = p->block ? p->block : 256u;
    const uint32_t grid = p->grid ? p->grid : 8u * sm_count_of_current_device();
    if (block % 32u || block > 1024u || p->iters == 0 || p->pattern > DASH_CEIL_PAIR_XCORNER)
        return DASH_HASH4D_INVALID_ARG;
    const uint32_t w = p->width;
    uint32_t unit = w;
    if (p->kind == DASH_CEIL_COPY || p->kind == DASH_CEIL_TMA_GATHER) unit = 16;
    if (unit == 0 || p->footprint_bytes < unit) return DASH_HASH4D_INVALID_ARG;
    uint64_t slots = 1;
    while (slots * 2 * unit <= p->footprint_bytes) slots *= 2;
    CeilArgs a;
    a.buf = static_cast<unsigned char*>(buf);
    a.sink = static_cast<unsigned char*>(sink);
    a.slot_mask = slots - 1;
    a.width = w;
    a.pattern = p->pattern;
    a.iters = p->iters;
    a.seed = p->seed;
    a.n16 = p->footprint_bytes / 16;
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    size_t dyn = p->dyn_smem;
    cudaError_t e = cudaSuccess;
#define DASH_CEIL_LAUNCH(KERNEL)                                                                            \
    do {                                                                                                    \
        if (dyn > 48 * 1024)                                                                                \
            e = cudaFuncSetAttribute(KERNEL, cudaFuncAttributeMaxDynamicSharedMemorySize, static_cast<int>(dyn)); \
        if (e == cudaSuccess) KERNEL<<<grid, block, dyn, s>>>(a);                                           \
    } while (0)
    switch (p->kind) {
        case DASH_CEIL_COPY: DASH_CEIL_LAUNCH(copy_kernel); break;
        case DASH_CEIL_GATHER:
            if (w == 4) DASH_CEIL_LAUNCH(gather_kernel<4>);
            else if (w == 8) DASH_CEIL_LAUNCH(gather_kernel<8>);
            else if (w == 16) DASH_CEIL_LAUNCH(gather_kernel<16>);
            else if (w == 32) DASH_CEIL_LAUNCH(gather_kernel<32>);
            else return DASH_HASH4D_INVALID_ARG;
            break;
        case DASH_CEIL_RED:
            if (w == 4) DASH_CEIL_LAUNCH(red_kernel<4>);
            else if (w == 8) DASH_CEIL_LAUNCH(red_kernel<8>);
            else if (w == 16) DASH_CEIL_LAUNCH(red_kernel<16>);
            else return DASH_HASH4D_INVALID_ARG;
            break;
        case DASH_CEIL_SMEM_ATOMIC: DASH_CEIL_LAUNCH(smem_atomic_kernel<float>); break;
        case DASH_CEIL_SMEM_ATOMIC_U64: DASH_CEIL_LAUNCH(smem_atomic_kernel<unsigned long long>); break;
        case DASH_CEIL_TMA_GATHER:
            dyn += static_cast<size_t>(block) * kUnroll * 16;
            DASH_CEIL_LAUNCH(tma_gather_kernel);
            break;
        default: return DASH_HASH4D_INVALID_ARG;
    }
#undef DASH_CEIL_LAUNCH
    if (e == cudaSuccess) e = cudaGetLastError();
    if (e != cudaSuccess) return DASH_HASH4D_CUDA_ERROR;
    if (lane_ops) *lane_ops = static_cast<uint64_t>(grid) * block * p->iters * kUnroll;
    return DASH_HASH4D_OK;
}
