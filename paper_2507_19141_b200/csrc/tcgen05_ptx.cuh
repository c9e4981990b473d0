// tcgen05_ptx.cuh — thin inline-PTX wrappers for the sm_100a tensor-core path (tcgen05.mma / ld / st / commit, TMEM,
// mbarriers) and the shared-memory operand layout helpers used by deform_kernels.cu and mlp_bwd_kernels.cu.
// Product code: shares nothing with oracle/.
#pragma once
#include <cuda_bf16.h>
#include <cuda_runtime.h>

#include <cstdint>

#include "deform_kernels.h"

namespace dash {
namespace {

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
// D[tmem] (+)= A[tmem] * B[smem]^T ; A: 128 lanes x 8 columns, each 32-bit column two bf16 along K (even k low)
__device__ __forceinline__ void tc_mma_bf16_ts(uint32_t tmem_d, uint32_t tmem_a, uint64_t bdesc, uint32_t idesc,
                                               uint32_t accumulate) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "setp.ne.b32 p, %4, 0;\n"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], [%1], %2, %3, p;\n"
        "}" ::"r"(tmem_d),
        "r"(tmem_a), "l"(bdesc), "r"(idesc), "r"(accumulate)
        : "memory");
}
// registers -> 16 / 8 consecutive 32-bit columns of this thread's TMEM lane
__device__ __forceinline__ void tc_st16(uint32_t taddr, const uint32_t r[16]) {
    asm volatile(
        "tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, "
        "%14, %15, %16};" ::"r"(taddr),
        "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]), "r"(r[8]),
        "r"(r[9]), "r"(r[10]), "r"(r[11]), "r"(r[12]), "r"(r[13]), "r"(r[14]), "r"(r[15])
        : "memory");
}
__device__ __forceinline__ void tc_st8(uint32_t taddr, const uint32_t r[8]) {
    asm volatile(
        "tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8};" ::"r"(taddr),
        "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7])
        : "memory");
}
__device__ __forceinline__ void tc_st_wait() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }

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

// 32 consecutive columns, no wait: several loads are issued back to back, then tc_ld_wait() once
__device__ __forceinline__ void tc_ld32_nowait(uint32_t taddr, uint32_t r[32]) {
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x32.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, "
        "%14, %15, %16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
        : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]),
          "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]),
          "=r"(r[16]), "=r"(r[17]), "=r"(r[18]), "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]),
          "=r"(r[23]), "=r"(r[24]), "=r"(r[25]), "=r"(r[26]), "=r"(r[27]), "=r"(r[28]), "=r"(r[29]),
          "=r"(r[30]), "=r"(r[31])
        : "r"(taddr)
        : "memory");
}
__device__ __forceinline__ void tc_ld_wait() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }

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

// byte offset of element (row, col) of a K-major operand in the layout umma_desc() describes: the 16-byte chunk
// (col / 8) of row `row` sits at chunk * LBO + row * 16.  LBO = rows*16 + 16: the 16 spare bytes skew successive
// K-chunks across the shared-memory banks (stores that walk along K would otherwise all hit one bank group).
__device__ __forceinline__ uint32_t operand_lbo(uint32_t rows) { return rows * 16u + 16u; }
__device__ __forceinline__ uint32_t operand_offset(uint32_t lbo, uint32_t row, uint32_t col) {
    return (col >> 3) * lbo + row * 16u + (col & 7u) * 2u;
}

// Explicit shared-space stores on 32-bit shared addresses.  Stores through generic pointers into `extern
// __shared__` made the compiler rebuild the shared window base (S2UR SR_CgaCtaId + ULEA) in the hot loop: 25 % of
// the producers' stall samples were short-scoreboard waits on that chain (round-1 ncu source page; the
// current kernel's stall mix is in profiles/ncu_render_r02.md).
__device__ __forceinline__ void sts16(uint32_t a, uint16_t v) {
    asm volatile("st.shared.b16 [%0], %1;" ::"r"(a), "h"(v) : "memory");
}
__device__ __forceinline__ void sts32(uint32_t a, uint32_t v) {
    asm volatile("st.shared.b32 [%0], %1;" ::"r"(a), "r"(v) : "memory");
}
__device__ __forceinline__ void sts64(uint32_t a, uint32_t x, uint32_t y) {
    asm volatile("st.shared.v2.b32 [%0], {%1, %2};" ::"r"(a), "r"(x), "r"(y) : "memory");
}
__device__ __forceinline__ void sts128(uint32_t a, uint32_t x, uint32_t y, uint32_t z, uint32_t w) {
    asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(a), "r"(x), "r"(y), "r"(z), "r"(w) : "memory");
}

// One lane of a converged warp.  The MMA issue runs as "whole warp enters, elected lane issues" with every operand
// derived from warp-uniform values: behind a per-thread `if (lane == 0)` the compiler cannot prove the descriptors
// uniform and wraps EVERY tcgen05.mma in an ELECT / R2UR.BROADCAST / BRA.U.ANY loop (~120 cycles per instruction,
// 3.2K cycles of issue per tile in the round-1 kernel: clock64 phase timers, profiles/experiments_r02.md §3).
__device__ __forceinline__ bool elect_one() {
    uint32_t pred;
    asm volatile(
        "{\n"
        ".reg .pred P;\n"
        "elect.sync _|P, 0xffffffff;\n"
        "selp.u32 %0, 1, 0, P;\n"
        "}"
        : "=r"(pred));
    return pred != 0;
}
__device__ __forceinline__ uint32_t uniform(uint32_t v) { return __shfl_sync(0xffffffffu, v, 0); }

// max(x, 0) and round to bf16, two values per instruction (cvt.rn.relu.bf16x2.f32: NaN -> canonical NaN)
__device__ __forceinline__ uint32_t pack_bf16_relu(float lo, float hi) {
    uint32_t r;
    asm("cvt.rn.relu.bf16x2.f32 %0, %1, %2;" : "=r"(r) : "f"(hi), "f"(lo));   // first source -> upper half
    return r;
}

__device__ __forceinline__ uint32_t pack_bf16(float lo, float hi) {
    const __nv_bfloat162 h = __floats2bfloat162_rn(lo, hi);  // .x = lo (low 16 bits)
    return *reinterpret_cast<const uint32_t*>(&h);
}


// W_l (fp32, row-major [J][K], bias behind it) -> the bf16 B operand [npad][kpad] of layer l in shared memory: one
// 16-byte chunk (8 consecutive k of one output row j) per step at chunk * LBO + j * 16, LBO = npad*16 + 16; columns
// kb, kb+1 carry the bias as bf16 hi + lo (the A operand has 1.0 there).  Each thread takes up to four chunks per batch
// and issues ALL their global loads before converting any: one L2 round trip per batch instead of one per chunk (the
// one-chunk-at-a-time loop cost 5-6K cycles per CTA, 10 % of dash_mlp_fwd at N = 300k).
__device__ __forceinline__ void stage_weights_bf16(const float* __restrict__ W, uint32_t K, uint32_t J, uint32_t kp,
                                                   uint32_t np, uint32_t kb, unsigned char* ws, uint32_t first,
                                                   uint32_t nthreads) {
    const float* b = W + static_cast<size_t>(J) * K;
    const uint32_t cpr = kp >> 3, w_lbo = operand_lbo(np), total = np * cpr;
    const bool vec = (K & 7u) == 0 && (reinterpret_cast<uintptr_t>(W) & 15u) == 0;  // float4 row chunks
    for (uint32_t i0 = first; i0 < total; i0 += 4u * nthreads) {
        float w[4][8];
        uint32_t dst[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const uint32_t i = i0 + u * nthreads;
            const uint32_t ii = i < total ? i : i0;
            const uint32_t j = ii / cpr, c = ii - j * cpr, k0 = c * 8u;
            dst[u] = c * w_lbo + j * 16u;
#pragma unroll
            for (int e = 0; e < 8; ++e) w[u][e] = 0.0f;
            if (j < J) {
                const float* src = W + static_cast<size_t>(j) * K + k0;
                if (k0 < kb) {
                    if (vec && k0 + 8u <= K) {
                        const float4 lo = __ldg(reinterpret_cast<const float4*>(src));
                        const float4 hi = __ldg(reinterpret_cast<const float4*>(src) + 1);
                        w[u][0] = lo.x; w[u][1] = lo.y; w[u][2] = lo.z; w[u][3] = lo.w;
                        w[u][4] = hi.x; w[u][5] = hi.y; w[u][6] = hi.z; w[u][7] = hi.w;
                    } else {
#pragma unroll
                        for (int e = 0; e < 8; ++e)
                            if (k0 + e < K) w[u][e] = __ldg(src + e);
                    }
                } else if (k0 == kb) {
                    w[u][0] = __ldg(b + j);   // split into hi + lo below
                }
            }
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const uint32_t i = i0 + u * nthreads;
            if (i >= total) continue;
            const uint32_t j = i / cpr, c = i - j * cpr;
            if (c * 8u == kb && j < J) {
                const float bj = w[u][0];
                w[u][0] = __bfloat162float(__float2bfloat16_rn(bj));
                w[u][1] = bj - w[u][0];
            }
            *reinterpret_cast<uint4*>(ws + dst[u]) = make_uint4(pack_bf16(w[u][0], w[u][1]), pack_bf16(w[u][2], w[u][3]),
                                                                pack_bf16(w[u][4], w[u][5]), pack_bf16(w[u][6], w[u][7]));
        }
    }
}

}  // namespace
}  // namespace dash
