// deform_kernels.cu — render path of the 4D hash deformation field, fused:
//     f_h = G_4D(x)  ->  f_4D = phi_d(f_h)  ->  (dx, dr, ds) = heads(f_4D)  ->  out = base + delta
// (Eq. 9-10; Q27).  ONE persistent, warp-specialised kernel per SM:
//
//   warps 0..23   ENCODER   the lane-pair gather / quadrilinear interpolation of hash4d_kernels.cu for a tile
//                           of 128 queries x all L levels; the L*F features never go to HBM: they are written
//                           as bf16 straight into the shared-memory A operand of the first dense layer
//                           (UMMA K-major, no-swizzle core-matrix layout), double buffered.
//   warps 24..31  two independent CONSUMER pipelines p = 0, 1 (even / odd tiles) of 4 warps each:
//                 MMA       the pipeline's first thread issues tcgen05.mma (kind::f16, bf16 x bf16 -> fp32,
//                           M = 128, N = layer width, K = 16 per instruction); accumulators live in TMEM.  The
//                           bias rides in the MMA: two extra K columns hold b as bf16 hi + lo against 1.0 in A.
//                 EPILOGUE  all 4 warps tcgen05.ld the accumulator rows (warp e owns TMEM lanes 32e..32e+31),
//                           relu, -> bf16 -> tcgen05.st into the TMEM A operand of the next layer (TS-form MMA);
//                           last layer: + base, store.  No shared-memory traffic at all between layers: the
//                           SM's LSU queue belongs to the producers' gathers.
//   The layers of one tile are a dependent chain (MMA -> epilogue -> MMA ...); two pipelines keep the tensor
//   pipe and the epilogue of one tile busy while the other tile waits on a hand-off.
//
// The weights of every layer are converted to bf16 once per CTA and stay resident in shared memory.  Hand-offs:
// mbarriers full/empty per A buffer, accumulator-done via tcgen05.commit, a 128-thread named barrier inside a
// pipeline; no __syncthreads in the steady state.  The gathers are the bound (issue + latency of 24 warps; L1 at
// ~70 % of its wavefront rate); the tensor pipe (~4 % busy) and the epilogue run underneath them.  D = 3: 8-corner
// gathers in a per-frame time slice of the tables (Q29).  FUSED = false: the producer warps read a
// feature matrix from global memory instead (two-pass path for tables that do not fit L2 in one level group).
// Phase timers for development builds live in deform_profile.cuh (DASH_PROF_* macros; empty in the product build).
#include <cuda_bf16.h>
#include <cuda_fp16.h>
#include <cuda_runtime.h>

#include "deform_kernels.h"
#include "deform_profile.cuh"
#include "hash4d_device.cuh"
#include "tcgen05_ptx.cuh"

namespace dash {

namespace {

constexpr uint32_t kEpilogueThreads = 4 * 32;   // per pipeline

}  // namespace

// ------------------------------------------------------------------------------------------------------------
template <int F, bool HALF, bool FUSED, int D>
__global__ void __launch_bounds__(kDeformThreads, 1)
deform_fused_kernel(const __grid_constant__ Plan P, const __grid_constant__ MlpPlan M,
                    const float* __restrict__ xyz, const float* __restrict__ t,
                    const int32_t* __restrict__ index, const void* __restrict__ table,
                    const float* __restrict__ feat, const float* __restrict__ params,
                    const float* __restrict__ base, float* __restrict__ out) {
    extern __shared__ __align__(128) unsigned char smem[];
    constexpr uint32_t kThreads = kDeformThreads, kProducerThreads = kDeformEncWarps * 32;
    DASH_PROF_ENTRY();
    uint32_t sbase = smem_u32(smem);
    asm volatile("" : "+r"(sbase));   // opaque: keep it in a register instead of re-deriving the shared window base
    const uint32_t tid = threadIdx.x, warp = tid >> 5, lane = tid & 31u;
    // barriers (8 bytes each): full[2] @0, empty[2] @16, mma_done[2] @32; TMEM base (u32) @64.
    // A buffer s, pipeline p and tile parity coincide: tile i of this CTA uses s = p = i & 1.
    const uint32_t bar_full = sbase + 0, bar_empty = sbase + 16, bar_mma0 = sbase + 32;
    volatile uint32_t* tmem_slot = reinterpret_cast<volatile uint32_t*>(smem + 64);
    const uint32_t a_lbo = operand_lbo(kDeformTileM);           // A operands: 128 rows
    const uint32_t a0_bytes = (M.kpad[0] >> 3) * a_lbo;
    // one 16-byte chunk holding (1, 1, 0, ...) in bf16: the two "ones" columns that multiply the bias columns of W
    const uint4 ones_chunk = make_uint4(0x3f803f80u, 0u, 0u, 0u);

    // ---- one-time setup: barriers, TMEM, weights (+ bias columns) -> bf16 operand layout, A buffers
    if (tid == 0) {
        mbar_init(bar_full + 0, kProducerThreads);
        mbar_init(bar_full + 8, kProducerThreads);
        mbar_init(bar_empty + 0, 1);
        mbar_init(bar_empty + 8, 1);
        mbar_init(bar_mma0 + 0, 1);
        mbar_init(bar_mma0 + 8, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == kDeformEncWarps) {  // first consumer warp owns the TMEM allocation
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(sbase + 64),
                     "r"(M.tmem_cols)
                     : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    fence_async_smem();
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = uniform(*tmem_slot);
    DASH_PROF_BEGIN(tid);

    // FUSED: the weights are staged by the CONSUMER warps only, while the producers already gather their first tile
    // (the producers never read them): the 5-6K cycles of setup of the round-1 kernel leave the critical path.
    // MLP-only mode has nothing to overlap them with: all threads stage, then one CTA barrier.
    auto stage_weights = [&](const uint32_t first, const uint32_t stagers) {
        for (uint32_t l = 0; l < M.n_layers; ++l) {
            // W_l as the B operand [npad][kpad], one 16-byte chunk (8 consecutive k of one output row j) per step;
            // consecutive threads take consecutive chunks of a row: coalesced (float4 when aligned) global reads; the
            // skewed LBO keeps the shared stores of neighbouring chunks on different banks.
            // Columns kb, kb+1 carry the bias as bf16 hi + bf16 lo (the A operand has 1.0 there): the tensor core
            // adds b_j = hi + lo (>= 16 significant bits) and the epilogue needs no bias loads.
            const uint32_t K = M.width[l], J = M.width[l + 1], kp = M.kpad[l], np = M.npad[l], kb = M.kbias[l];
            const float* W = params + M.p_off[l];
            const float* b = W + static_cast<size_t>(J) * K;
            unsigned char* ws = smem + M.w_off[l];
            const uint32_t cpr = kp >> 3, w_lbo = operand_lbo(np);
            const bool vec = (K & 7u) == 0 && (reinterpret_cast<uintptr_t>(W) & 15u) == 0;  // float4 row chunks
            for (uint32_t i = tid - first; i < np * cpr; i += stagers) {
                const uint32_t j = i / cpr, c = i - j * cpr, k0 = c * 8u;   // consecutive threads: consecutive chunks
                float w[8];
#pragma unroll
                for (int e = 0; e < 8; ++e) w[e] = 0.0f;
                if (j < J) {
                    const float* src = W + static_cast<size_t>(j) * K + k0;
                    if (k0 < kb) {
                        if (vec && k0 + 8u <= K) {
                            const float4 lo = __ldg(reinterpret_cast<const float4*>(src));
                            const float4 hi = __ldg(reinterpret_cast<const float4*>(src) + 1);
                            w[0] = lo.x; w[1] = lo.y; w[2] = lo.z; w[3] = lo.w;
                            w[4] = hi.x; w[5] = hi.y; w[6] = hi.z; w[7] = hi.w;
                        } else {
#pragma unroll
                            for (int e = 0; e < 8; ++e)
                                if (k0 + e < K) w[e] = __ldg(src + e);
                        }
                    } else if (k0 == kb) {
                        const float bj = __ldg(b + j);
                        w[0] = __bfloat162float(__float2bfloat16_rn(bj));
                        w[1] = bj - w[0];
                    }
                }
                *reinterpret_cast<uint4*>(ws + c * w_lbo + j * 16u) =
                    make_uint4(pack_bf16(w[0], w[1]), pack_bf16(w[2], w[3]), pack_bf16(w[4], w[5]),
                               pack_bf16(w[6], w[7]));
            }
        }
    };
    if constexpr (!FUSED) {
        stage_weights(0u, kThreads);
        fence_async_smem();
        __syncthreads();
    }

    // Each CTA owns a contiguous range of rows [r_begin, r_end) — an equal share of N, not a whole number of
    // tiles — and walks it in tiles of 128; in its last, partial tile the producers skip the missing rows, so the
    // gather work (the bound) is balanced to a row, whatever N is.
    const uint64_t r_begin = static_cast<uint64_t>(blockIdx.x) * M.rows_per_cta;
    const uint64_t r_end = r_begin + M.rows_per_cta < M.N ? r_begin + M.rows_per_cta : M.N;
    const uint32_t my_tiles =
        r_begin < r_end ? static_cast<uint32_t>((r_end - r_begin + kDeformTileM - 1) / kDeformTileM) : 0u;

    // From here on the two roles never share a code path again (until the teardown).  (Measured: with the set-up of
    // each role inside its own branch the fused modes run 3-4 % faster than with a shared prologue.)
    if (warp < kDeformEncWarps) {
        // ================================================================================== PRODUCER
        // the A buffers are the producers': zeros, and (1, 1) in the chunk that multiplies the bias columns; their
        // tile writes follow behind a producers-only barrier, and every producer fences before it signals "full"
        for (uint32_t i = tid; i < (2u * a0_bytes) / 16u; i += kProducerThreads) {
            const uint32_t within = (i * 16u) % a0_bytes;                 // byte offset inside one A buffer
            reinterpret_cast<uint4*>(smem + M.a0_off)[i] =
                (within / a_lbo == (M.kbias[0] >> 3)) ? ones_chunk : make_uint4(0u, 0u, 0u, 0u);
        }
        asm volatile("bar.sync %0, %1;" ::"r"(4u), "r"(kProducerThreads) : "memory");
        for (uint32_t i = 0; i < my_tiles; ++i) {
            const uint32_t s = i & 1u;
            const uint64_t row0 = r_begin + static_cast<uint64_t>(i) * kDeformTileM;
            const uint32_t rows_here = r_end - row0 < kDeformTileM ? static_cast<uint32_t>(r_end - row0) : kDeformTileM;
            mbar_wait(bar_empty + 8 * s, ((i >> 1) & 1u) ^ 1u);  // first use of each buffer passes at once
            if (tid == 0) DASH_PROF(0, 2 * i);
            const uint32_t a0 = sbase + M.a0_off + s * a0_bytes;   // shared-space address of this tile's A buffer
            if constexpr (FUSED) {
                // One ROUND = 16 (query, level) items = one warp instruction's worth of lane pairs; a full tile has
                // 8*L rounds, taken by the warps round-robin.  The coordinates of a warp's NEXT round are loaded under
                // the gathers of the current one (one global round trip on the critical path instead of two).  The
                // warp -> round assignment rotates from tile to tile: 8*L is rarely a multiple of the warp count, and
                // the producers may run up to two tiles ahead, so the rotation evens the work out.  (Two rounds per
                // iteration, 16 gathers per lane in flight, was measured SLOWER: 34K instead of 21K cycles per tile.)
                const uint32_t pair = lane >> 1, xc = lane & 1u;
                const uint32_t rounds = (rows_here * P.L + 15u) >> 4;   // rounds that hold at least one real row
                const uint32_t w0 = (warp + 8u * i) % kDeformEncWarps;
                constexpr size_t kElem = HALF ? 2 : 4;
                auto item_row = [&](uint32_t rr) -> uint64_t {
                    const uint32_t it = rr * 16u + pair;
                    const uint64_t n = row0 + ((P.L & (P.L - 1u)) == 0u ? it >> (31u - __clz(P.L)) : it / P.L);
                    return n < r_end ? n : r_end - 1;  // ragged last round: duplicate work, rows never stored
                };
                constexpr int NC = 1 << (D - 1);   // D = 3: lookups in a time slice (8 corners), D = 4: Eq. 9 as is
                // Gathers in flight set the rate: the SM's load queue is served at ~1 wavefront per cycle behind a
                // fixed ~1.2K-cycle L2 round trip, so throughput ~ W / (W + 1.2K) with W the queued wavefronts
                // (24 warps x 8 loads x 17 lines = 3.3K -> 0.73, measured).  R rounds per warp iteration: R = 2 was
                // measured slower for both D = 4 (34K vs 21K cycles per tile) and D = 3 (87 vs 75 us at C2), so R = 1.
                constexpr int R = 1;
                constexpr uint32_t kStep = R * kDeformEncWarps;
                // When L divides 16 a lane pair serves the SAME level in every round (l = pair mod L): its level
                // constants and table base are then fetched once, not per round — the indexed constant loads and
                // the integer divisions were 2K of the ~3.2K cycles a round took (clock64 phase timers).
                const bool fixed_level = (16u % P.L) == 0u;
                const uint32_t l_shift = 31u - __clz(P.L);           // valid when L is a power of two
                LevelParams lp_fix = P.lv[pair % P.L];
                const char* base_fix =
                    static_cast<const char*>(table) + static_cast<size_t>(pair % P.L) * P.T * (F * kElem);
                float cq[R][4];
#pragma unroll
                for (int k = 0; k < R; ++k) {
                    const uint32_t rk = w0 + k * kDeformEncWarps;
                    if (w0 < rounds) load_coords<D>(P, item_row(rk < rounds ? rk : w0), xyz, t, index, cq[k]);
                }
                for (uint32_t ra = w0; ra < rounds; ra += kStep) {
                    DASH_PROF_CLOCK(q0);
                    uint32_t rk[R];
                    uint32_t slot[R][NC];
                    float W[R][NC];
                    float v[R][NC][F];
#pragma unroll
                    for (int k = 0; k < R; ++k) {
                        rk[k] = ra + k * kDeformEncWarps < rounds ? ra + k * kDeformEncWarps : ra;  // past the end:
                        LevelParams lp = lp_fix;                                         // redo round ra, no store
                        const char* level_base = base_fix;
                        if (!fixed_level) {
                            const uint32_t l = (rk[k] * 16u + pair) % P.L;
                            lp = P.lv[l];
                            level_base = static_cast<const char*>(table) + static_cast<size_t>(l) * P.T * (F * kElem);
                        }
                        const Query qq = make_query<D>(lp, cq[k][0], cq[k][1], cq[k][2], cq[k][3]);
                        half_cell<D>(P, lp, qq, xc, slot[k], W[k]);
#pragma unroll
                        for (int j = 0; j < NC; ++j) load_slot<F, HALF>(level_base, slot[k][j], v[k][j]);
                    }
                    DASH_PROF_CLOCK(q1);
                    if (ra + kStep < rounds) {   // next iteration's coordinates, under the gathers
#pragma unroll
                        for (int k = 0; k < R; ++k) {
                            const uint32_t rn = ra + kStep + k * kDeformEncWarps;
                            load_coords<D>(P, item_row(rn < rounds ? rn : ra + kStep), xyz, t, index, cq[k]);
                        }
                    }
#pragma unroll
                    for (int k = 0; k < R; ++k) {
                        float acc[F];
#pragma unroll
                        for (int f = 0; f < F; ++f) acc[f] = 0.0f;
#pragma unroll
                        for (int j = 0; j < NC; ++j)
#pragma unroll
                            for (int f = 0; f < F; ++f) acc[f] = fmaf(W[k][j], v[k][j][f], acc[f]);
#pragma unroll
                        for (int f = 0; f < F; ++f) acc[f] += __shfl_xor_sync(0xffffffffu, acc[f], 1);
                        DASH_PROF_ACCUM(tid == 0, q1 - q0, clock64() - q1);
                        if (xc == 0 && (k == 0 || rk[k] != ra)) {
                            // fp32 feature -> bf16 operand element (row q, column l*F + f)
                            const uint32_t it = rk[k] * 16u + pair;
                            const uint32_t q = (P.L & (P.L - 1u)) == 0u ? it >> l_shift : it / P.L, l = it - q * P.L;
                            const uint32_t dst = a0 + operand_offset(a_lbo, q, l * F);
                            if constexpr (F == 1) {
                                sts16(dst, __bfloat16_as_ushort(__float2bfloat16_rn(acc[0])));
                            } else if constexpr (F == 2) {
                                sts32(dst, pack_bf16(acc[0], acc[1]));
                            } else if constexpr (F == 4) {
                                sts64(dst, pack_bf16(acc[0], acc[1]), pack_bf16(acc[2], acc[3]));
                            } else {
                                sts128(dst, pack_bf16(acc[0], acc[1]), pack_bf16(acc[2], acc[3]),
                                       pack_bf16(acc[4], acc[5]), pack_bf16(acc[6], acc[7]));
                            }
                        }
                    }
                }
            } else {
                // feature rows from global memory: one 8-column chunk (32 bytes in, 16 bytes out) per step;
                // only the data chunks — the bias ("ones") chunk behind them was written once at setup
                const uint32_t K = M.width[0], chunks = M.kbias[0] >> 3;
                for (uint32_t i2 = tid; i2 < rows_here * chunks; i2 += kProducerThreads) {
                    const uint32_t q = i2 / chunks, c = i2 - q * chunks;
                    const uint64_t n = row0 + q;
                    float x[8];
#pragma unroll
                    for (int e = 0; e < 8; ++e) {
                        const uint32_t k = c * 8u + e;
                        x[e] = k < K ? __ldcs(feat + n * K + k) : 0.0f;
                    }
                    sts128(a0 + operand_offset(a_lbo, q, c * 8u), pack_bf16(x[0], x[1]), pack_bf16(x[2], x[3]),
                           pack_bf16(x[4], x[5]), pack_bf16(x[6], x[7]));
                }
            }
            fence_async_smem();
            mbar_arrive(bar_full + 8 * s);
            if (tid == 0) DASH_PROF(0, 2 * i + 1);
        }
    } else {
        // ================================================================================== CONSUMER PIPELINE p
        if constexpr (FUSED) {
            stage_weights(kProducerThreads, kThreads - kProducerThreads);
            fence_async_smem();   // the staged weights are read by the async proxy (tcgen05.mma)
            asm volatile("bar.sync %0, %1;" ::"r"(3u), "r"(kThreads - kProducerThreads) : "memory");
        }
        // Tile i of this CTA: A buffer s = i & 1, pipeline p = i % npipes.  Layer 1 reads its A operand from shared
        // memory (written by the producers); the hidden activations go accumulator -> registers -> TENSOR MEMORY
        // (tcgen05.st) and the next layer's MMA reads its A operand from there (TS form).  A consumer thread touches
        // shared memory only to wait on an mbarrier: everything that goes through the SM's LSU queue waits behind
        // the producers' gathers (measured: 6-14K cycles per layer with shared-memory activations, profiles/).
        const uint32_t cw = uniform(warp) - kDeformEncWarps;   // warp-uniform by construction (see elect_one)
        const uint32_t p = cw >> 2, e = cw & 3u;            // e == warp % 4: owns TMEM lanes 32e .. 32e+31
        const bool issue_warp = e == 0;                     // this pipeline's MMA-issuing warp (one elected lane)
        const uint32_t sb = uniform(sbase);
        const uint32_t r = e * 32u + lane;                  // accumulator row = query within the tile
        const uint32_t tmem_d = tmem_base + p * M.tmem_pipe_cols;        // accumulator columns of this pipeline
        const uint32_t tmem_a = tmem_d + M.tmem_a_off;                   // bf16 A operand of layers 2..n
        const uint32_t lane_off = (e * 32u) << 16;
        const uint32_t bar_mma = bar_mma0 + 8 * p;
        uint32_t mma_phase = 0, batch = 0;
        for (uint32_t i = p; i < my_tiles && p < M.npipes; i += M.npipes) {
            const uint32_t s = i & 1u;
            const uint64_t n = r_begin + static_cast<uint64_t>(i) * kDeformTileM + r;
#pragma unroll
            for (uint32_t l = 0; l < kMlpMaxLayers; ++l, ++batch) {   // unrolled: M.*[l] become direct constant reads
                if (l >= M.n_layers) break;
                if (issue_warp) {
                    if (l == 0) mbar_wait(sb + 8 * s, (i >> 1) & 1u);   // bar_full[s]
                    tc_fence_after();
                    if (p == 0 && lane == 0) DASH_PROF(1, 2 * batch);
                    if (elect_one()) {
                        const uint32_t w_addr = sb + M.w_off[l];
                        const uint32_t np = M.npad[l], ksteps = M.kpad[l] >> 4;
                        const uint32_t w_lbo = operand_lbo(np);
                        const uint32_t idesc = umma_idesc(np);
                        if (l == 0) {
                            const uint32_t a_addr = sb + M.a0_off + s * a0_bytes;
                            for (uint32_t kk = 0; kk < ksteps; ++kk) {
                                const uint64_t ad = umma_desc(a_addr + kk * 2u * a_lbo, a_lbo, 128u);
                                const uint64_t bd = umma_desc(w_addr + kk * 2u * w_lbo, w_lbo, 128u);
                                tc_mma_bf16(tmem_d, ad, bd, idesc, kk > 0 ? 1u : 0u);
                            }
                            tc_commit(sb + 16 + 8 * s);  // bar_empty[s]: A buffer free once these MMAs have read it
                        } else {
                            for (uint32_t kk = 0; kk < ksteps; ++kk) {   // K = 16 per instruction = 8 TMEM columns of A
                                const uint64_t bd = umma_desc(w_addr + kk * 2u * w_lbo, w_lbo, 128u);
                                tc_mma_bf16_ts(tmem_d, tmem_a + kk * 8u, bd, idesc, kk > 0 ? 1u : 0u);
                            }
                        }
                        tc_commit(sb + 32 + 8 * p);      // bar_mma[p]
                    }
                    __syncwarp();
                    if (p == 0 && lane == 0) DASH_PROF(1, 2 * batch + 1);
                }
                mbar_wait(bar_mma, mma_phase);
                mma_phase ^= 1u;
                __syncwarp();
                tc_fence_after();
                if (cw == 0 && lane == 0) DASH_PROF(2, 2 * batch);
                const uint32_t np = M.npad[l];
                if (l + 1 < M.n_layers) {
                    // hidden layer: relu, -> bf16 pairs, -> tensor memory (the bias came out of the MMA).  (A version
                    // with 16-column steps and one load kept in flight under the conversion was measured slower:
                    // 1.2K instead of 1.0K cycles per layer, profiles/experiments_r02.md §3.)
                    for (uint32_t c = 0; c < np; c += 32u) {   // np is a multiple of 16: the last round may be half
                        uint32_t rr[32];
                        tc_ld32_nowait(tmem_d + lane_off + c, rr);
                        tc_ld_wait();
                        uint32_t w[16];
#pragma unroll
                        for (int j = 0; j < 16; ++j)
                            w[j] = pack_bf16_relu(__uint_as_float(rr[2 * j]), __uint_as_float(rr[2 * j + 1]));
                        if (c + 16u < np) {
                            tc_st16(tmem_a + lane_off + (c >> 1), w);
                        } else {
                            tc_st8(tmem_a + lane_off + (c >> 1), w);
                        }
                    }
                    // the "ones" pair that multiplies the next layer's bias columns, zeros behind it
                    const uint32_t tail[8] = {0x3f803f80u, 0u, 0u, 0u, 0u, 0u, 0u, 0u};
                    tc_st8(tmem_a + lane_off + (np >> 1), tail);
                    tc_st_wait();
                } else if (M.out_stage_off != 0u) {
                    // narrow last layer (n_out <= 16, the deformation heads): a thread owns a row, i.e. n_out floats
                    // at a 4*n_out-byte stride from its neighbours' — stored directly, every store instruction touches
                    // 32 sectors (measured: 1.5K of the 2.1K cycles of this epilogue, profiles/experiments_r02.md §3).
                    // The warp's 32 rows are ONE contiguous block of `out`: transpose through 2 KB of shared memory
                    // and store it with lane-contiguous (fully coalesced) instructions; `base` is read the same way.
                    float v[16];
                    tc_ld16(tmem_d + lane_off, v);
                    const uint32_t stage = sb + M.out_stage_off + cw * 2048u;
                    const uint32_t n_out = M.n_out;
#pragma unroll
                    for (int j = 0; j < 16; ++j)
                        if (static_cast<uint32_t>(j) < n_out) sts32(stage + (lane * n_out + j) * 4u, __float_as_uint(v[j]));
                    __syncwarp();
                    const uint64_t n0 = n - lane;                                   // first row of this warp
                    const uint32_t rows_valid = n0 < r_end ? (r_end - n0 < 32u ? static_cast<uint32_t>(r_end - n0) : 32u) : 0u;
                    const uint32_t count = rows_valid * n_out;
                    float* o = out + n0 * n_out;
                    const float* bb = base ? base + n0 * n_out : nullptr;
#pragma unroll 4
                    for (uint32_t k = lane; k < count; k += 32u) {
                        float val;
                        asm volatile("ld.shared.f32 %0, [%1];" : "=f"(val) : "r"(stage + k * 4u) : "memory");
                        __stcs(o + k, val + (bb ? __ldcs(bb + k) : 0.0f));
                    }
                    __syncwarp();   // the staging block is rewritten by this warp's next tile
                } else {
                    for (uint32_t c = 0; c < np; c += 16u) {
                        float v[16];
                        tc_ld16(tmem_d + lane_off + c, v);
                        if (n < r_end) {   // rows past the range hold stale operands: never stored
                            float* o = out + n * M.n_out;
                            const float* bb = base ? base + n * M.n_out : nullptr;
#pragma unroll
                            for (int j = 0; j < 16; ++j)
                                if (c + j < M.n_out) __stcs(o + c + j, v[j] + (bb ? __ldcs(bb + c + j) : 0.0f));
                        }
                    }
                }
                tc_fence_before();
                // the 4 warps of this pipeline: activations written and TMEM drained before the next MMAs
                asm volatile("bar.sync %0, %1;" ::"r"(1u + p), "r"(kEpilogueThreads) : "memory");
                if (cw == 0 && lane == 0) DASH_PROF(2, 2 * batch + 1);
            }
        }
    }

    // ---- teardown: every TMEM read has completed (each consumer thread waited on its loads)
    tc_fence_before();
    __syncthreads();
    DASH_PROF_REPORT(tid, my_tiles, M.n_layers);
    if (warp == kDeformEncWarps) {
        tc_fence_after();
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(M.tmem_cols)
                     : "memory");
    }
}

// ------------------------------------------------------------------------------------------------------------
template <int F, bool HALF, bool FUSED, int D>
static cudaError_t launch_t(const Plan& P, const MlpPlan& M, const float* xyz, const float* t,
                            const int32_t* index, const void* table, const float* feat, const float* params,
                            const float* base, float* out, int sms, cudaStream_t s) {
    auto* k = deform_fused_kernel<F, HALF, FUSED, D>;
    cudaError_t e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         static_cast<int>(M.smem_bytes));
    if (e != cudaSuccess) return e;
    (void)sms;
    k<<<M.grid, kDeformThreads, M.smem_bytes, s>>>(P, M, xyz, t, index, table, feat, params, base, out);
    count_launch();
    return cudaGetLastError();
}

cudaError_t launch_deform_fused(const Plan& P, const MlpPlan& M, const float* xyz, const float* t,
                                const int32_t* index, const void* table, bool table_half,
                                const float* params, const float* base, float* out, int sms,
                                cudaStream_t s) {
#define DASH_DF(FV, HV) \
    return launch_t<FV, HV, true, 4>(P, M, xyz, t, index, table, nullptr, params, base, out, sms, s)
#define DASH_DF3(FV) \
    return launch_t<FV, false, true, 3>(P, M, xyz, t, index, table, nullptr, params, base, out, sms, s)
    if (P.dims == 3) {  // lookups in a time slice (fp32, Q29) or a G_3D table
        if (table_half) return cudaErrorInvalidValue;
        switch (P.F) {
            case 1: DASH_DF3(1);
            case 2: DASH_DF3(2);
            case 4: DASH_DF3(4);
            case 8: DASH_DF3(8);
            default: return cudaErrorInvalidValue;
        }
    }
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
#undef DASH_DF3
}

cudaError_t launch_mlp(const MlpPlan& M, const float* feat, const float* params, const float* base,
                       float* out, int sms, cudaStream_t s) {
    Plan P{};  // unused by the non-fused instantiation
    return launch_t<1, false, false, 4>(P, M, nullptr, nullptr, nullptr, nullptr, feat, params, base, out, sms,
                                     s);
}

}  // namespace dash
