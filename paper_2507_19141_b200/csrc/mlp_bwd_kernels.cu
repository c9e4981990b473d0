// mlp_bwd_kernels.cu — backward through phi_d and the heads (include/dash_deform.h dash_mlp_bwd; Q30):
//     delta_n = dout;   for l = n .. 1:   dW_l += delta_l^T a_{l-1},  db_l += sum_rows delta_l,
//     g_{l-1} = delta_l W_l,   delta_{l-1} = g_{l-1} * [a_{l-1} > 0],   dfeat = g_0
// on the tensor cores (tcgen05, kind::f16: bf16 operands, fp32 accumulation in tensor memory).  One persistent CTA
// per SM walks its rows in tiles of 128 and, per tile, RECOMPUTES the forward activations (nothing is saved by
// dash_mlp_fwd: 128 x width bf16 per layer would be written and read back through HBM), then runs the chain backwards.
//
//   operand tiles   every operand is a bf16 tile [128 rows x C columns] in ONE shared-memory layout (no swizzle: the
//                   16-byte chunk c of row r at c * LBO + r * 16, LBO = 128*16 + 16).  The SAME bytes serve as
//                     K-major  operands (contraction over the columns):  forward a_{l-1} W_l^T,  dgrad delta_l W_l
//                     MN-major operands (contraction over the 128 ROWS):  wgrad delta_l^T a_{l-1}
//                   — only the descriptor changes (a_major / b_major bits, LBO <-> SBO roles).  The bf16 weight copy
//                   W_l [npad x kpad] of the forward is the K-major B operand there and, unchanged, the MN-major B
//                   operand of the dgrad (contraction over its rows j).
//   wgrad           D[M = j (128 lanes, rows >= J_l unused)][N = kpad_l] accumulates in tensor memory
//                   across ALL tiles of the CTA (lane j, column k <-> dW_l[j][k]; the "ones" column of a_{l-1} makes
//                   column kbias_l the bias gradient); one flush of fp32 reductions per CTA at the end.
//   roles           warps 0-3: the epilogues (TMEM lane quarter = warp).  warp 4: one elected lane issues every MMA, so
//                   that no epilogue warp spends its time in the issue loop (the wgrad MMAs are issued while the
//                   epilogue of the dgrad before them already runs).  warps 5-7: load the next tile's features
//                   (-> a_0, double buffered) and dout (-> delta_n) as bf16 while the current tile computes.
// The dgrad of a layer is issued before its wgrad and committed alone, so the epilogue that forms delta_{l-1} runs
// while the wgrad MMAs of layer l execute (they read delta_l, the epilogue writes the other ping-pong buffer).
#include <cuda_bf16.h>
#include <cuda_runtime.h>

#include "deform_kernels.h"
#include "tcgen05_ptx.cuh"

namespace dash {

namespace {

constexpr uint32_t kBwdComputeThreads = 128, kBwdLoaderThreads = 96;   // warps 0-3 | warp 4 issues | warps 5-7 load
constexpr uint32_t kTileLbo = kDeformTileM * 16u + 16u;   // operand_lbo(128)

// kind::f16 instruction descriptor with selectable major-ness: bit 15 = A is MN-major, bit 16 = B is MN-major
__device__ __forceinline__ uint32_t umma_idesc_mn(uint32_t n, bool a_mn, bool b_mn) {
    return umma_idesc(n) | (a_mn ? (1u << 15) : 0u) | (b_mn ? (1u << 16) : 0u);
}
// MN-major view of a tile in the layout above: 8 consecutive K' (rows) 16 bytes apart, 8-row groups 128 bytes apart
// (LBO field), 8-column chunks `chunk_stride` bytes apart (SBO field); one K' = 16 step advances the start by 256 B.
__device__ __forceinline__ uint64_t umma_desc_mn(uint32_t saddr, uint32_t chunk_stride) {
    return umma_desc(saddr, 128u, chunk_stride);
}

__device__ __forceinline__ uint4 lds128(uint32_t a) {
    uint4 v;
    asm volatile("ld.shared.v4.b32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(a) : "memory");
    return v;
}
// relu mask of a PAIR of activations, as a bit mask over a packed bf16 pair: 0xffff in each half whose activation is
// > 0.  The activations are relu outputs (cvt.rn.relu: never negative, never -0), so "> 0" is "bits != 0": adding
// 0x7fff to a 15-bit magnitude sets bit 15 exactly when it is non-zero (no carry between the halves), and
// (t >> 15) * 0xffff spreads the two flag bits over their halves.  Four integer operations per pair; the first version
// built two 0/1 floats per pair with compares and selects and spent 2.4K cycles per hidden layer in this epilogue.
__device__ __forceinline__ uint32_t relu_mask2(uint32_t packed) {
    const uint32_t t = ((packed & 0x7fff7fffu) + 0x7fff7fffu) & 0x80008000u;
    return (t >> 15) * 0xffffu;
}

}  // namespace

__global__ void __launch_bounds__(kMlpBwdThreads, 1)
mlp_bwd_kernel(const __grid_constant__ MlpBwdPlan B, const float* __restrict__ feat,
               const float* __restrict__ params, const float* __restrict__ dout, float* __restrict__ dfeat,
               float* __restrict__ dparams) {
    extern __shared__ __align__(128) unsigned char smem[];
    const MlpPlan& M = B.fwd;
    const uint32_t tid = threadIdx.x, lane = tid & 31u;
    const uint32_t warp = uniform(tid >> 5);
    const uint32_t sb = uniform(smem_u32(smem));
    const uint32_t nl = M.n_layers;
    // barriers (8 bytes each) at bar_off: full_a0[2] +0, empty_a0[2] +16, full_dn +32, empty_dn +40, mma_done +48;
    // TMEM base slot +64
    const uint32_t bar = sb + B.bar_off;
    const uint32_t bar_full_a0 = bar, bar_empty_a0 = bar + 16, bar_full_dn = bar + 32, bar_empty_dn = bar + 40,
                   bar_mma = bar + 48;
    volatile uint32_t* tmem_slot = reinterpret_cast<volatile uint32_t*>(smem + B.bar_off + 64);
    const uint4 ones_chunk = make_uint4(0x3f803f80u, 0u, 0u, 0u);

    if (tid == 0) {
        mbar_init(bar_full_a0 + 0, kBwdLoaderThreads);
        mbar_init(bar_full_a0 + 8, kBwdLoaderThreads);
        mbar_init(bar_empty_a0 + 0, 1);
        mbar_init(bar_empty_a0 + 8, 1);
        mbar_init(bar_full_dn, kBwdLoaderThreads);
        mbar_init(bar_empty_dn, 1);
        mbar_init(bar_mma, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(bar + 64),
                     "r"(B.tmem_cols)
                     : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    // weights -> bf16 operand copies, exactly as the forward stages them (bias as bf16 hi + lo in columns kb, kb+1)
    for (uint32_t l = 0; l < nl; ++l)
        stage_weights_bf16(params + M.p_off[l], M.width[l], M.width[l + 1], M.kpad[l], M.npad[l], M.kbias[l],
                           smem + B.w_off[l], tid, kMlpBwdThreads);
    // activation tiles: zeros, (1, 1) in the chunk behind the data columns (bias column of the forward, bias
    // gradient of the wgrad); a_0 has two buffers.  delta tiles: zeros (columns an epilogue never writes stay 0).
    for (uint32_t l = 0; l < nl; ++l) {
        const uint32_t chunks = M.kpad[l] >> 3, copies = l == 0 ? 2u : 1u;
        for (uint32_t i = tid; i < copies * chunks * (kTileLbo / 16u); i += kMlpBwdThreads) {
            const uint32_t within = (i * 16u) % (chunks * kTileLbo);
            reinterpret_cast<uint4*>(smem + B.a_off[l])[i] =
                (within / kTileLbo == (M.kbias[l] >> 3)) ? ones_chunk : make_uint4(0u, 0u, 0u, 0u);
        }
    }
    for (uint32_t i = tid; i < (2u * 16u * kTileLbo) / 16u; i += kMlpBwdThreads)
        reinterpret_cast<uint4*>(smem + B.d_off[0])[i] = make_uint4(0u, 0u, 0u, 0u);   // d_off[1] follows d_off[0]
    for (uint32_t i = tid; i < ((M.npad[nl - 1] >> 3) * kTileLbo) / 16u; i += kMlpBwdThreads)
        reinterpret_cast<uint4*>(smem + B.dn_off)[i] = make_uint4(0u, 0u, 0u, 0u);
    fence_async_smem();
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = uniform(*tmem_slot);

    const uint64_t r_begin = static_cast<uint64_t>(blockIdx.x) * M.rows_per_cta;
    const uint64_t r_end = r_begin + M.rows_per_cta < M.N ? r_begin + M.rows_per_cta : M.N;
    const uint32_t my_tiles =
        r_begin < r_end ? static_cast<uint32_t>((r_end - r_begin + kDeformTileM - 1) / kDeformTileM) : 0u;
    const uint32_t n_out = M.n_out;

    if (warp >= 5) {
        // ============================================================================================ LOADERS
        const uint32_t lt = tid - kBwdComputeThreads - 32u;
        const uint32_t K0 = M.width[0], chunks0 = M.kbias[0] >> 3, chunksn = M.npad[nl - 1] >> 3;
        for (uint32_t i = 0; i < my_tiles; ++i) {
            const uint32_t s = i & 1u;
            const uint64_t row0 = r_begin + static_cast<uint64_t>(i) * kDeformTileM;
            const uint32_t rows_here = r_end - row0 < kDeformTileM ? static_cast<uint32_t>(r_end - row0) : kDeformTileM;
            mbar_wait(bar_empty_a0 + 8 * s, ((i >> 1) & 1u) ^ 1u);
            const uint32_t a0 = sb + B.a_off[0] + s * B.a0_bytes;
            for (uint32_t i2 = lt; i2 < kDeformTileM * chunks0; i2 += kBwdLoaderThreads) {
                const uint32_t q = i2 / chunks0, c = i2 - q * chunks0;
                float x[8];
#pragma unroll
                for (int e = 0; e < 8; ++e) {
                    const uint32_t k = c * 8u + e;
                    x[e] = (q < rows_here && k < K0) ? __ldcs(feat + (row0 + q) * K0 + k) : 0.0f;   // rows past the
                }                                                                                    // range: zeros
                sts128(a0 + c * kTileLbo + q * 16u, pack_bf16(x[0], x[1]), pack_bf16(x[2], x[3]),
                       pack_bf16(x[4], x[5]), pack_bf16(x[6], x[7]));
            }
            fence_async_smem();
            mbar_arrive(bar_full_a0 + 8 * s);
            mbar_wait(bar_empty_dn, (i & 1u) ^ 1u);
            const uint32_t dn = sb + B.dn_off;
            for (uint32_t i2 = lt; i2 < kDeformTileM * chunksn; i2 += kBwdLoaderThreads) {
                const uint32_t q = i2 / chunksn, c = i2 - q * chunksn;
                float x[8];
#pragma unroll
                for (int e = 0; e < 8; ++e) {
                    const uint32_t k = c * 8u + e;
                    x[e] = (q < rows_here && k < n_out) ? __ldcs(dout + (row0 + q) * n_out + k) : 0.0f;
                }
                sts128(dn + c * kTileLbo + q * 16u, pack_bf16(x[0], x[1]), pack_bf16(x[2], x[3]),
                       pack_bf16(x[4], x[5]), pack_bf16(x[6], x[7]));
            }
            fence_async_smem();
            mbar_arrive(bar_full_dn);
        }
    } else if (warp == 4) {
        // ============================================================================================ MMA ISSUE
        // Mirrors the epilogue warps' step sequence; after issuing the MMAs of a step it waits (named barrier 1, 160
        // threads) until their epilogue has consumed the accumulator and written its tile.
        const uint32_t acc = tmem_base + B.acc_col;
        for (uint32_t i = 0; i < my_tiles; ++i) {
            const uint32_t s = i & 1u;
            const uint32_t a0 = sb + B.a_off[0] + s * B.a0_bytes;
            for (uint32_t l = 0; l + 1 < nl; ++l) {   // forward recompute
                if (l == 0) mbar_wait(bar_full_a0 + 8 * s, (i >> 1) & 1u);
                tc_fence_after();
                if (elect_one()) {
                    const uint32_t a_addr = l == 0 ? a0 : sb + B.a_off[l];
                    const uint32_t w_addr = sb + B.w_off[l], np = M.npad[l], w_lbo = operand_lbo(np);
                    const uint32_t idesc = umma_idesc(np);
                    for (uint32_t kk = 0; kk < (M.kpad[l] >> 4); ++kk)
                        tc_mma_bf16(acc, umma_desc(a_addr + kk * 2u * kTileLbo, kTileLbo, 128u),
                                    umma_desc(w_addr + kk * 2u * w_lbo, w_lbo, 128u), idesc, kk > 0 ? 1u : 0u);
                    tc_commit(bar_mma);
                }
                __syncwarp();
                asm volatile("bar.sync 1, 160;" ::: "memory");
            }
            for (int l = static_cast<int>(nl) - 1; l >= 0; --l) {   // backward
                const bool last = l == static_cast<int>(nl) - 1;
                const uint32_t dsrc = last ? sb + B.dn_off : sb + B.d_off[(l + 1) & 1];   // delta of this layer's output
                const bool need_dgrad = l > 0 || dfeat != nullptr;
                if (last) mbar_wait(bar_full_dn, i & 1u);
                tc_fence_after();
                if (elect_one()) {
                    const uint32_t w_lbo = operand_lbo(M.npad[l]);
                    if (need_dgrad) {   // g = delta W_l: contraction over the layer's outputs j (K-major A, MN-major B)
                        const uint32_t idesc = umma_idesc_mn(M.kbias[l], false, true);
                        for (uint32_t kk = 0; kk < (M.npad[l] >> 4); ++kk)
                            tc_mma_bf16(acc, umma_desc(dsrc + kk * 2u * kTileLbo, kTileLbo, 128u),
                                        umma_desc_mn(sb + B.w_off[l] + kk * 256u, w_lbo), idesc, kk > 0 ? 1u : 0u);
                    }
                    tc_commit(bar_mma);   // the dgrad alone (and everything before it): its epilogue may start
                    // dW_l (+)= delta^T a_l: contraction over the 128 rows (both operands MN-major); accumulates over
                    // all tiles of this CTA
                    const uint32_t a_l = l == 0 ? a0 : sb + B.a_off[l];
                    const uint32_t idesc_w = umma_idesc_mn(M.kpad[l], true, true);
                    for (uint32_t kk = 0; kk < kDeformTileM / 16u; ++kk)
                        tc_mma_bf16(tmem_base + B.dw_col[l], umma_desc_mn(dsrc + kk * 256u, kTileLbo),
                                    umma_desc_mn(a_l + kk * 256u, kTileLbo), idesc_w, (i > 0 || kk > 0) ? 1u : 0u);
                    if (last) tc_commit(bar_empty_dn);            // delta_n consumed (dgrad + wgrad of layer n)
                    if (l == 0) tc_commit(bar_empty_a0 + 8 * s);  // a_0 consumed (forward + wgrad of layer 1)
                }
                __syncwarp();
                asm volatile("bar.sync 1, 160;" ::: "memory");
            }
        }
        if (my_tiles > 0) {
            tc_fence_after();
            if (elect_one()) tc_commit(bar_mma);   // covers the last wgrad MMAs: the flush may read the accumulators
            __syncwarp();
        }
    } else {
        // ============================================================================================ EPILOGUES
        const uint32_t r = warp * 32u + lane;              // row of the tile = TMEM lane this thread reads
        const uint32_t lane_off = (warp * 32u) << 16;
        const uint32_t acc = tmem_base + B.acc_col;
        uint32_t mma_phase = 0;
        for (uint32_t i = 0; i < my_tiles; ++i) {
            const uint64_t n = r_begin + static_cast<uint64_t>(i) * kDeformTileM + r;
            // ---------------------------------------------------------------- forward recompute: a_1 .. a_{n-1}
            for (uint32_t l = 0; l + 1 < nl; ++l) {
                mbar_wait(bar_mma, mma_phase);
                mma_phase ^= 1u;
                __syncwarp();
                tc_fence_after();
                const uint32_t np = M.npad[l], dst = sb + B.a_off[l + 1] + r * 16u;
                for (uint32_t c = 0; c < np; c += 32u) {
                    uint32_t rr[32];
                    tc_ld32_nowait(acc + lane_off + c, rr);
                    tc_ld_wait();
#pragma unroll
                    for (uint32_t q = 0; q < 4; ++q)
                        if (c + 8u * q < np)
                            sts128(dst + ((c >> 3) + q) * kTileLbo,
                                   pack_bf16_relu(__uint_as_float(rr[8 * q + 0]), __uint_as_float(rr[8 * q + 1])),
                                   pack_bf16_relu(__uint_as_float(rr[8 * q + 2]), __uint_as_float(rr[8 * q + 3])),
                                   pack_bf16_relu(__uint_as_float(rr[8 * q + 4]), __uint_as_float(rr[8 * q + 5])),
                                   pack_bf16_relu(__uint_as_float(rr[8 * q + 6]), __uint_as_float(rr[8 * q + 7])));
                }
                fence_async_smem();
                tc_fence_before();
                asm volatile("bar.sync 1, 160;" ::: "memory");
            }
            // ---------------------------------------------------------------- backward: layers n .. 1 (l = n-1 .. 0)
            for (int l = static_cast<int>(nl) - 1; l >= 0; --l) {
                mbar_wait(bar_mma, mma_phase);
                mma_phase ^= 1u;
                __syncwarp();
                tc_fence_after();
                if (l > 0) {
                    // delta_l = g * [a_l > 0] -> bf16 -> the delta buffer the running wgrad does NOT read
                    const uint32_t kc = M.kbias[l], dst = sb + B.d_off[l & 1] + r * 16u, src = sb + B.a_off[l] + r * 16u;
                    for (uint32_t c = 0; c < kc; c += 32u) {
                        uint32_t rr[32];
                        tc_ld32_nowait(acc + lane_off + c, rr);
                        uint4 av[4];   // the activations' chunks are fetched under the tensor-memory load
#pragma unroll
                        for (uint32_t q = 0; q < 4; ++q)
                            av[q] = c + 8u * q < kc ? lds128(src + ((c >> 3) + q) * kTileLbo) : make_uint4(0u, 0u, 0u, 0u);
                        tc_ld_wait();
#pragma unroll
                        for (uint32_t q = 0; q < 4; ++q) {
                            if (c + 8u * q < kc)
                                sts128(dst + ((c >> 3) + q) * kTileLbo,
                                       pack_bf16(__uint_as_float(rr[8 * q + 0]), __uint_as_float(rr[8 * q + 1])) & relu_mask2(av[q].x),
                                       pack_bf16(__uint_as_float(rr[8 * q + 2]), __uint_as_float(rr[8 * q + 3])) & relu_mask2(av[q].y),
                                       pack_bf16(__uint_as_float(rr[8 * q + 4]), __uint_as_float(rr[8 * q + 5])) & relu_mask2(av[q].z),
                                       pack_bf16(__uint_as_float(rr[8 * q + 6]), __uint_as_float(rr[8 * q + 7])) & relu_mask2(av[q].w));
                        }
                    }
                    fence_async_smem();
                } else if (dfeat != nullptr) {
                    const uint32_t K0 = M.width[0];
                    for (uint32_t c = 0; c < M.kbias[0]; c += 16u) {
                        float v[16];
                        tc_ld16(acc + lane_off + c, v);
                        if (n < r_end) {
                            float* o = dfeat + n * K0 + c;
                            if ((K0 & 3u) == 0u && c + 16u <= K0) {
#pragma unroll
                                for (int q = 0; q < 4; ++q)
                                    __stcs(reinterpret_cast<float4*>(o) + q,
                                           make_float4(v[4 * q], v[4 * q + 1], v[4 * q + 2], v[4 * q + 3]));
                            } else {
#pragma unroll
                                for (int j = 0; j < 16; ++j)
                                    if (c + j < K0) __stcs(o + j, v[j]);
                            }
                        }
                    }
                }
                tc_fence_before();
                asm volatile("bar.sync 1, 160;" ::: "memory");
            }
        }
        // ---------------------------------------------------------------- flush the wgrad accumulators
        if (my_tiles > 0) {
            mbar_wait(bar_mma, mma_phase);
            __syncwarp();
            tc_fence_after();
            // every CTA adds into the same dparams: start at a different layer / column block per CTA so that the
            // 148 flushes do not walk the same addresses in lock step; 16-byte vector reductions where aligned
            for (uint32_t ll = 0; ll < nl; ++ll) {
                const uint32_t l = (ll + blockIdx.x) % nl;
                const uint32_t K = M.width[l], J = M.width[l + 1], kb = M.kbias[l], blocks = M.kpad[l] >> 4;
                float* dW = dparams + M.p_off[l];
                float* db = dW + static_cast<size_t>(J) * K;
                for (uint32_t cc = 0; cc < blocks; ++cc) {
                    const uint32_t c = ((cc + blockIdx.x) % blocks) << 4;
                    float v[16];
                    tc_ld16(tmem_base + B.dw_col[l] + lane_off + c, v);   // lane r = output row j, columns = inputs k
                    if (r < J) {
                        float* row = dW + static_cast<size_t>(r) * K + c;
                        if (c + 16u <= K && (reinterpret_cast<uintptr_t>(row) & 15u) == 0) {
#pragma unroll
                            for (int q = 0; q < 4; ++q)
                                asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(row + 4 * q),
                                             "f"(v[4 * q]), "f"(v[4 * q + 1]), "f"(v[4 * q + 2]), "f"(v[4 * q + 3])
                                             : "memory");
                        } else {
#pragma unroll
                            for (int jj = 0; jj < 16; ++jj) {
                                const uint32_t k = c + jj;
                                if (k < K) atomicAdd(row + jj, v[jj]);
                                else if (k == kb) atomicAdd(db + r, v[jj]);
                            }
                        }
                    }
                }
            }
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 0) {
        tc_fence_after();
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(B.tmem_cols)
                     : "memory");
    }
}

cudaError_t launch_mlp_bwd(const MlpBwdPlan& B, const float* feat, const float* params, const float* dout,
                           float* dfeat, float* dparams, cudaStream_t s) {
    cudaError_t e = cudaFuncSetAttribute(mlp_bwd_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         static_cast<int>(B.smem_bytes));
    if (e != cudaSuccess) return e;
    mlp_bwd_kernel<<<B.fwd.grid, kMlpBwdThreads, B.smem_bytes, s>>>(B, feat, params, dout, dfeat, dparams);
    count_launch();
    return cudaGetLastError();
}

}  // namespace dash
