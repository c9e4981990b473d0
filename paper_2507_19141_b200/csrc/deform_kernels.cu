// deform_kernels.cu — render path of the 4D hash deformation field, fused:
//     f_h = G_4D(x)  ->  f_4D = phi_d(f_h)  ->  (dx, dr, ds) = heads(f_4D)  ->  out = base + delta
// (Eq. 9-10; Q27).  ONE persistent, warp-specialised kernel per SM:
//
//   warps 0..23   ENCODER   the lane-pair gather / quadrilinear interpolation of hash4d_kernels.cu for a tile
//                           of 128 queries x all L levels; the L*F features never go to HBM: they are written
//                           as bf16 straight into the shared-memory A operand of the first dense layer
//                           (UMMA K-major, no-swizzle core-matrix layout), double buffered.
//   warp  28      MMA       one elected thread issues tcgen05.mma (kind::f16, bf16 x bf16 -> fp32, M = 128,
//                           N = layer width, K = 16 per instruction); accumulators live in TMEM.
//   warps 24..27  EPILOGUE  tcgen05.ld the accumulator rows (warp e owns TMEM lanes 32e..32e+31), + bias, relu,
//                           -> bf16 -> the next layer's A operand in shared memory; last layer: + base, store.
//
// The weights of every layer are converted to bf16 once per CTA and stay resident in shared memory.  Hand-offs
// are mbarriers (full/empty per A buffer, accumulator-done via tcgen05.commit, activations-ready); no
// __syncthreads in the steady state.  The gathers are the bound (L1 wavefronts, as in the forward kernel); the
// tensor pipe and the epilogue run underneath them.  With FUSED = false the producer warps read a feature
// matrix from global memory instead (two-pass path for tables that do not fit L2 in one level group).
#include <cuda_bf16.h>
#include <cuda_fp16.h>
#include <cuda_runtime.h>

#include "deform_kernels.h"
#include "hash4d_device.cuh"

namespace dash {

namespace {

constexpr uint32_t kProducerThreads = kDeformEncWarps * 32;
constexpr uint32_t kEpilogueThreads = kDeformEpiWarps * 32;

// ---------------------------------------------------------------------------------------------- PTX wrappers
__device__ __forceinline__ uint32_t smem_u32(const void* p) {
    return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred P1;\n"
        "LAB_WAIT:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n"
        "@P1 bra DONE;\n"
        "bra LAB_WAIT;\n"
        "DONE:\n"
        "}" ::"r"(bar),
        "r"(parity)
        : "memory");
}
// generic-proxy shared-memory writes -> visible to the async proxy (tcgen05.mma operand reads)
__device__ __forceinline__ void fence_async_smem() {
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}
__device__ __forceinline__ void tc_fence_before() {
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
}
__device__ __forceinline__ void tc_fence_after() {
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
}
__device__ __forceinline__ void tc_commit(uint32_t bar) {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar)
                 : "memory");
}
// D[tmem] (+)= A[smem] * B[smem]^T ; A: 128 x 16 bf16 K-major, B: N x 16 bf16 K-major
__device__ __forceinline__ void tc_mma_bf16(uint32_t tmem_d, uint64_t adesc, uint64_t bdesc, uint32_t idesc,
                                            uint32_t accumulate) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "setp.ne.b32 p, %4, 0;\n"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n"
        "}" ::"r"(tmem_d),
        "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate)
        : "memory");
}
// 16 consecutive fp32 accumulator columns of this thread's TMEM lane
__device__ __forceinline__ void tc_ld16(uint32_t taddr, float v[16]) {
    uint32_t r[16];
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, "
        "%14, %15}, [%16];"
        : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]),
          "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
        : "r"(taddr)
        : "memory");
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
    for (int i = 0; i < 16; ++i) v[i] = __uint_as_float(r[i]);
}

// UMMA shared-memory matrix descriptor, K-major, SWIZZLE_NONE ("interleave"): core matrices of 8 rows x 16 bytes
// stored as 128 contiguous bytes; SBO = distance between 8-row groups, LBO = distance between the two 16-byte
// K-chunks one K = 16 instruction reads.  Bits: [0,14) address >> 4, [16,30) LBO >> 4, [32,46) SBO >> 4,
// [46,48) version = 1 (sm_100), [61,64) layout type = 0.
__device__ __forceinline__ uint64_t umma_desc(uint32_t saddr, uint32_t lbo_bytes, uint32_t sbo_bytes) {
    return static_cast<uint64_t>((saddr >> 4) & 0x3fffu) |
           (static_cast<uint64_t>((lbo_bytes >> 4) & 0x3fffu) << 16) |
           (static_cast<uint64_t>((sbo_bytes >> 4) & 0x3fffu) << 32) | (1ull << 46);
}
// kind::f16 instruction descriptor: D fp32 (bits [4,6) = 1), A and B bf16 ([7,10) = [10,13) = 1), both K-major,
// N >> 3 at [17,23), M >> 4 at [24,29).
__device__ __forceinline__ uint32_t umma_idesc(uint32_t n) {
    return (1u << 4) | (1u << 7) | (1u << 10) | ((n >> 3) << 17) | ((kDeformTileM >> 4) << 24);
}

// byte offset of element (row, col) of a K-major operand with `rows` rows in the layout umma_desc() describes:
// 16-byte chunk (col / 8) of row `row` sits at chunk * rows*16 + row*16.
__device__ __forceinline__ uint32_t operand_offset(uint32_t rows, uint32_t row, uint32_t col) {
    return (col >> 3) * (rows * 16u) + row * 16u + (col & 7u) * 2u;
}

__device__ __forceinline__ uint32_t pack_bf16(float lo, float hi) {
    const __nv_bfloat162 h = __floats2bfloat162_rn(lo, hi);  // .x = lo (low 16 bits)
    return *reinterpret_cast<const uint32_t*>(&h);
}

}  // namespace

// ------------------------------------------------------------------------------------------------------------
template <int F, bool HALF, bool FUSED>
__global__ void __launch_bounds__(kDeformThreads, 1)
deform_fused_kernel(const __grid_constant__ Plan P, const __grid_constant__ MlpPlan M,
                    const float* __restrict__ xyz, const float* __restrict__ t,
                    const int32_t* __restrict__ index, const void* __restrict__ table,
                    const float* __restrict__ feat, const float* __restrict__ params,
                    const float* __restrict__ base, float* __restrict__ out) {
    extern __shared__ __align__(128) unsigned char smem[];
    const uint32_t sbase = smem_u32(smem);
    const uint32_t tid = threadIdx.x, warp = tid >> 5, lane = tid & 31u;
    // barriers: [0] full0 [1] full1 [2] empty0 [3] empty1 [4] mma_done [5] act_ready ; [8] (u32) TMEM base
    const uint32_t bar_full = sbase + 0, bar_empty = sbase + 16, bar_mma = sbase + 32, bar_act = sbase + 40;
    volatile uint32_t* tmem_slot = reinterpret_cast<volatile uint32_t*>(smem + 64);

    // ---- one-time setup: barriers, TMEM, weights -> bf16 operand layout, zero padding of the A buffers
    if (tid == 0) {
        mbar_init(bar_full + 0, kProducerThreads);
        mbar_init(bar_full + 8, kProducerThreads);
        mbar_init(bar_empty + 0, 1);
        mbar_init(bar_empty + 8, 1);
        mbar_init(bar_mma, 1);
        mbar_init(bar_act, kEpilogueThreads);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == kDeformMmaWarp) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(sbase + 64),
                     "r"(M.tmem_cols)
                     : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    for (uint32_t l = 0; l < M.n_layers; ++l) {
        const uint32_t K = M.width[l], J = M.width[l + 1], kp = M.kpad[l], np = M.npad[l];
        const float* W = params + M.p_off[l];
        const float* b = W + static_cast<size_t>(J) * K;
        for (uint32_t i = tid; i < np * kp; i += kDeformThreads) {
            const uint32_t j = i / kp, k = i - j * kp;
            const float w = (j < J && k < K) ? __ldg(W + static_cast<size_t>(j) * K + k) : 0.0f;
            *reinterpret_cast<__nv_bfloat16*>(smem + M.w_off[l] + operand_offset(np, j, k)) =
                __float2bfloat16_rn(w);
        }
        float* bs = reinterpret_cast<float*>(smem + M.b_off[l]);
        for (uint32_t j = tid; j < np; j += kDeformThreads) bs[j] = j < J ? __ldg(b + j) : 0.0f;
    }
    for (uint32_t i = tid; i < (2u * kDeformTileM * M.kpad[0] * 2u) / 16u; i += kDeformThreads)
        reinterpret_cast<uint4*>(smem + M.a0_off)[i] = make_uint4(0u, 0u, 0u, 0u);
    fence_async_smem();
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot;

    const uint32_t a0_bytes = kDeformTileM * M.kpad[0] * 2u;
    const uint32_t my_tiles =
        blockIdx.x < M.num_tiles ? (M.num_tiles - blockIdx.x + gridDim.x - 1) / gridDim.x : 0u;

    if (warp < kDeformEncWarps) {
        // ================================================================================== PRODUCER
        for (uint32_t i = 0; i < my_tiles; ++i) {
            const uint32_t s = i & 1u;
            const uint64_t row0 = (static_cast<uint64_t>(blockIdx.x) + static_cast<uint64_t>(i) * gridDim.x) *
                                  kDeformTileM;
            mbar_wait(bar_empty + 8 * s, ((i >> 1) & 1u) ^ 1u);  // first use of each buffer passes at once
            unsigned char* a0 = smem + M.a0_off + s * a0_bytes;
            if constexpr (FUSED) {
                const uint32_t pair = lane >> 1, xc = lane & 1u;
                const uint32_t items = kDeformTileM * P.L;  // multiple of 16: whole warps stay together
                for (uint32_t it = warp * 16u + pair; it < items; it += kDeformEncWarps * 16u) {
                    const uint32_t q = it / P.L, l = it - q * P.L;
                    uint64_t n = row0 + q;
                    if (n >= P.N) n = P.N - 1;  // tail tile: duplicate work, rows never stored
                    const LevelParams lp = P.lv[l];
                    const Query qq = load_query<4>(P, lp, n, xyz, t, index);
                    uint32_t slot[8];
                    float W[8];
                    half_cell<4>(P, lp, qq, xc, slot, W);
                    constexpr size_t kElem = HALF ? 2 : 4;
                    const char* level_base =
                        static_cast<const char*>(table) + static_cast<size_t>(l) * P.T * (F * kElem);
                    float v[8][F];
#pragma unroll
                    for (int j = 0; j < 8; ++j) load_slot<F, HALF>(level_base, slot[j], v[j]);
                    float acc[F];
#pragma unroll
                    for (int f = 0; f < F; ++f) acc[f] = 0.0f;
#pragma unroll
                    for (int j = 0; j < 8; ++j)
#pragma unroll
                        for (int f = 0; f < F; ++f) acc[f] = fmaf(W[j], v[j][f], acc[f]);
#pragma unroll
                    for (int f = 0; f < F; ++f) acc[f] += __shfl_xor_sync(0xffffffffu, acc[f], 1);
                    if (xc == 0) {  // fp32 feature -> bf16 operand element (row q, column l*F + f)
                        unsigned char* dst = a0 + operand_offset(kDeformTileM, q, l * F);
                        if constexpr (F == 1) {
                            *reinterpret_cast<__nv_bfloat16*>(dst) = __float2bfloat16_rn(acc[0]);
                        } else if constexpr (F == 2) {
                            *reinterpret_cast<uint32_t*>(dst) = pack_bf16(acc[0], acc[1]);
                        } else if constexpr (F == 4) {
                            *reinterpret_cast<uint2*>(dst) =
                                make_uint2(pack_bf16(acc[0], acc[1]), pack_bf16(acc[2], acc[3]));
                        } else {
                            *reinterpret_cast<uint4*>(dst) =
                                make_uint4(pack_bf16(acc[0], acc[1]), pack_bf16(acc[2], acc[3]),
                                           pack_bf16(acc[4], acc[5]), pack_bf16(acc[6], acc[7]));
                        }
                    }
                }
            } else {
                // feature rows from global memory: one 8-column chunk (32 bytes in, 16 bytes out) per step
                const uint32_t K = M.width[0], chunks = M.kpad[0] >> 3;
                for (uint32_t i2 = tid; i2 < kDeformTileM * chunks; i2 += kProducerThreads) {
                    const uint32_t q = i2 / chunks, c = i2 - q * chunks;
                    const uint64_t n = row0 + q;
                    float x[8];
#pragma unroll
                    for (int e = 0; e < 8; ++e) {
                        const uint32_t k = c * 8u + e;
                        x[e] = (n < M.N && k < K) ? __ldcs(feat + n * K + k) : 0.0f;
                    }
                    *reinterpret_cast<uint4*>(a0 + operand_offset(kDeformTileM, q, c * 8u)) =
                        make_uint4(pack_bf16(x[0], x[1]), pack_bf16(x[2], x[3]), pack_bf16(x[4], x[5]),
                                   pack_bf16(x[6], x[7]));
                }
            }
            fence_async_smem();
            mbar_arrive(bar_full + 8 * s);
        }
    } else if (warp == kDeformMmaWarp) {
        // ================================================================================== MMA ISSUER
        if (lane == 0) {
            uint32_t act_phase = 0, batch = 0;
            for (uint32_t i = 0; i < my_tiles; ++i) {
                const uint32_t s = i & 1u;
                for (uint32_t l = 0; l < M.n_layers; ++l, ++batch) {
                    if (l == 0) mbar_wait(bar_full + 8 * s, (i >> 1) & 1u);
                    if (batch > 0) {  // TMEM drained (and, for l > 0, the activations written) by the epilogue
                        mbar_wait(bar_act, act_phase);
                        act_phase ^= 1u;
                    }
                    tc_fence_after();
                    const uint32_t a_addr = sbase + (l == 0 ? M.a0_off + s * a0_bytes : M.act_off);
                    const uint32_t w_addr = sbase + M.w_off[l];
                    const uint32_t np = M.npad[l], ksteps = M.kpad[l] >> 4;
                    const uint32_t a_lbo = kDeformTileM * 16u, w_lbo = np * 16u;
                    const uint32_t idesc = umma_idesc(np);
                    for (uint32_t kk = 0; kk < ksteps; ++kk) {
                        const uint64_t ad = umma_desc(a_addr + kk * 2u * a_lbo, a_lbo, 128u);
                        const uint64_t bd = umma_desc(w_addr + kk * 2u * w_lbo, w_lbo, 128u);
                        tc_mma_bf16(tmem_base, ad, bd, idesc, kk > 0 ? 1u : 0u);
                    }
                    if (l == 0) tc_commit(bar_empty + 8 * s);  // A buffer free once these MMAs have read it
                    tc_commit(bar_mma);
                }
            }
        }
    } else {
        // ================================================================================== EPILOGUE
        const uint32_t e = warp - kDeformEncWarps;          // == warp % 4: owns TMEM lanes 32e .. 32e+31
        const uint32_t r = e * 32u + lane;                  // accumulator row = query within the tile
        const uint32_t taddr_row = tmem_base + ((e * 32u) << 16);
        uint32_t mma_phase = 0;
        for (uint32_t i = 0; i < my_tiles; ++i) {
            const uint64_t n = (static_cast<uint64_t>(blockIdx.x) + static_cast<uint64_t>(i) * gridDim.x) *
                                   kDeformTileM + r;
            for (uint32_t l = 0; l < M.n_layers; ++l) {
                mbar_wait(bar_mma, mma_phase);
                mma_phase ^= 1u;
                tc_fence_after();
                const float* bs = reinterpret_cast<const float*>(smem + M.b_off[l]);
                const uint32_t np = M.npad[l];
                const bool last = l + 1 == M.n_layers;
                for (uint32_t c = 0; c < np; c += 16u) {
                    float v[16];
                    tc_ld16(taddr_row + c, v);
#pragma unroll
                    for (int j = 0; j < 16; ++j) v[j] += bs[c + j];
                    if (!last) {
#pragma unroll
                        for (int j = 0; j < 16; ++j) v[j] = fmaxf(v[j], 0.0f);
                        unsigned char* dst = smem + M.act_off + operand_offset(kDeformTileM, r, c);
                        *reinterpret_cast<uint4*>(dst) = make_uint4(pack_bf16(v[0], v[1]), pack_bf16(v[2], v[3]),
                                                                    pack_bf16(v[4], v[5]), pack_bf16(v[6], v[7]));
                        *reinterpret_cast<uint4*>(dst + kDeformTileM * 16u) =
                            make_uint4(pack_bf16(v[8], v[9]), pack_bf16(v[10], v[11]),
                                       pack_bf16(v[12], v[13]), pack_bf16(v[14], v[15]));
                    } else if (n < M.N) {
                        float* o = out + n * M.n_out;
                        const float* bb = base ? base + n * M.n_out : nullptr;
#pragma unroll
                        for (int j = 0; j < 16; ++j)
                            if (c + j < M.n_out) __stcs(o + c + j, v[j] + (bb ? __ldcs(bb + c + j) : 0.0f));
                    }
                }
                if (!last) fence_async_smem();
                tc_fence_before();
                mbar_arrive(bar_act);
            }
        }
    }

    // ---- teardown: every TMEM read has completed (each epilogue thread waited on its loads)
    tc_fence_before();
    __syncthreads();
    if (warp == kDeformMmaWarp) {
        tc_fence_after();
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(M.tmem_cols)
                     : "memory");
    }
}

// ------------------------------------------------------------------------------------------------------------
template <int F, bool HALF, bool FUSED>
static cudaError_t launch_t(const Plan& P, const MlpPlan& M, const float* xyz, const float* t,
                            const int32_t* index, const void* table, const float* feat, const float* params,
                            const float* base, float* out, int sms, cudaStream_t s) {
    auto* k = deform_fused_kernel<F, HALF, FUSED>;
    cudaError_t e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         static_cast<int>(M.smem_bytes));
    if (e != cudaSuccess) return e;
    const unsigned grid = M.num_tiles < static_cast<uint32_t>(sms) ? M.num_tiles : static_cast<unsigned>(sms);
    k<<<grid, kDeformThreads, M.smem_bytes, s>>>(P, M, xyz, t, index, table, feat, params, base, out);
    count_launch();
    return cudaGetLastError();
}

cudaError_t launch_deform_fused(const Plan& P, const MlpPlan& M, const float* xyz, const float* t,
                                const int32_t* index, const void* table, bool table_half,
                                const float* params, const float* base, float* out, int sms,
                                cudaStream_t s) {
#define DASH_DF(FV, HV) \
    return launch_t<FV, HV, true>(P, M, xyz, t, index, table, nullptr, params, base, out, sms, s)
    switch (P.F * 2 + (table_half ? 1 : 0)) {
        case 2: DASH_DF(1, false);
        case 3: DASH_DF(1, true);
        case 4: DASH_DF(2, false);
        case 5: DASH_DF(2, true);
        case 8: DASH_DF(4, false);
        case 9: DASH_DF(4, true);
        case 16: DASH_DF(8, false);
        case 17: DASH_DF(8, true);
        default: return cudaErrorInvalidValue;
    }
#undef DASH_DF
}

cudaError_t launch_mlp(const MlpPlan& M, const float* feat, const float* params, const float* base,
                       float* out, int sms, cudaStream_t s) {
    Plan P{};  // unused by the non-fused instantiation
    return launch_t<1, false, false>(P, M, nullptr, nullptr, nullptr, nullptr, feat, params, base, out, sms,
                                     s);
}

}  // namespace dash
