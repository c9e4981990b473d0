// hash4d_kernels.cu — hand-written sm_100a kernels of the DASH 4D hash encoder.
//
// Work decomposition: one LANE PAIR per (query n, level l) item.  The two lanes of
// a pair take the two x-corners of the 4D cell (pi_x = 1 keeps them in adjacent table slots, so a
// pair's two 8/16-byte accesses fall in one 32-byte sector 50-75 % of the time and almost always
// in one 128-byte line: half the L1 wavefronts of a lane-per-item mapping), each lane walks the 8
// (y,z,t) corners, and one shuffle folds the two halves.  A warp holds 16 items = (16/G) queries x
// G consecutive levels, so the warp's store of `out` (and load of `dout`) covers G*F*4 contiguous
// bytes per query.  Blocks are ordered level-group-major (blockIdx.y = group) so that the tables
// (fwd) / gradient slices (bwd) of one group stay L2-resident while all queries stream past.
//
// This is a gather/scatter path: no tensor cores (no dense contraction), no TMA (8-byte random
// accesses cannot be expressed as tiles).
#include <cuda_fp16.h>
#include <cuda_runtime.h>

#include <cmath>

#include "hash4d_device.cuh"
#include "deform_kernels.h"
#include "hash4d_kernels.h"

namespace dash {

namespace {

thread_local uint64_t g_launches = 0;

// Item coordinates of this lane pair.  Inactive pairs (tail tile, L not a multiple of G) are clamped
// onto a valid item so that every lane reaches the shuffles; they skip their stores / reductions.
struct Item {
    uint64_t n;
    uint32_t l;
    uint32_t xc;
    bool active;
};

__device__ __forceinline__ Item this_item(const Plan& P, uint32_t tile, uint32_t grp) {
    const uint32_t pair = threadIdx.x >> 1;
    Item it;
    it.xc = threadIdx.x & 1u;
    it.n = static_cast<uint64_t>(tile) * P.q_per_block + (pair >> P.group_log2);
    it.l = P.level_begin + grp * P.group + (pair & (P.group - 1u));
    it.active = (it.n < P.N) && (it.l < P.level_end);
    if (it.n >= P.N) it.n = P.N - 1;
    if (it.l >= P.level_end) it.l = P.level_end - 1;
    return it;
}

__device__ __forceinline__ Item this_item(const Plan& P) { return this_item(P, blockIdx.x, blockIdx.y); }

// ------------------------------------------------------------------------------------------------
// Forward: gather + quadrilinear interpolation (Eq. 9)
// ------------------------------------------------------------------------------------------------
template <int F, bool HALF, int D, bool ORDERED>
__global__ void __launch_bounds__(kBlockThreads)
hash4d_fwd_kernel(const __grid_constant__ Plan P, const float* __restrict__ xyz,
                  const float* __restrict__ t, const int32_t* __restrict__ index,
                  const void* __restrict__ table, float* __restrict__ out,
                  const int32_t* __restrict__ order, const float4* __restrict__ sorted_q) {
    constexpr int NC = 1 << (D - 1);
    Item it = this_item(P);
    const LevelParams lp = P.lv[it.l];
    Query q;
    if constexpr (ORDERED) {   // SORT_COARSE: position it.n of the cell-sorted order (bwd_runs_kernels.cu): neighbouring
                               // lanes then gather from the same cells; the row of `out` is the query's own
        const float4 c = __ldg(sorted_q + it.n);
        q = make_query<D>(lp, c.x, c.y, c.z, c.w);
        const uint64_t n = static_cast<uint64_t>(static_cast<uint32_t>(__ldg(order + it.n)));
        it.n = n < P.N ? n : P.N - 1;   // memory-safe even if the caller's ORDER_READY claim is false
    } else {
        q = load_query<D>(P, lp, it.n, xyz, t, index);
    }
    uint32_t slot[NC];
    float W[NC];
    half_cell<D>(P, lp, q, it.xc, slot, W);

    constexpr size_t kElem = HALF ? 2 : 4;
    const char* level_base =
        static_cast<const char*>(table) + static_cast<size_t>(it.l) * P.T * (F * kElem);
    float v[NC][F];
#pragma unroll
    for (int j = 0; j < NC; ++j) load_slot<F, HALF>(level_base, slot[j], v[j]);  // NC loads in flight
    float acc[F];
#pragma unroll
    for (int f = 0; f < F; ++f) acc[f] = 0.0f;
#pragma unroll
    for (int j = 0; j < NC; ++j)
#pragma unroll
        for (int f = 0; f < F; ++f) acc[f] = fmaf(W[j], v[j][f], acc[f]);
#pragma unroll
    for (int f = 0; f < F; ++f) acc[f] += __shfl_xor_sync(0xffffffffu, acc[f], 1);  // fold x-corners

    if (!it.active) return;
    float* o = out + it.n * (static_cast<size_t>(P.L) * F) + static_cast<size_t>(it.l) * F;
    if constexpr (F == 1) {
        if (it.xc == 0) __stcs(o, acc[0]);
    } else if constexpr (F == 2) {
        __stcs(o + it.xc, it.xc ? acc[1] : acc[0]);
    } else if constexpr (F == 4) {
        const float2 s = it.xc ? make_float2(acc[2], acc[3]) : make_float2(acc[0], acc[1]);
        __stcs(reinterpret_cast<float2*>(o) + it.xc, s);
    } else {
        const float4 s = it.xc ? make_float4(acc[4], acc[5], acc[6], acc[7])
                               : make_float4(acc[0], acc[1], acc[2], acc[3]);
        __stcs(reinterpret_cast<float4*>(o) + it.xc, s);
    }
}

// Each lane of a pair loads half of the item's F upstream gradients; one shuffle gives both all F.
template <int F>
__device__ __forceinline__ void load_dout(const float* __restrict__ d, uint32_t xc, float g[F]) {
    if constexpr (F == 1) {
        g[0] = __ldcs(d);
    } else if constexpr (F == 2) {
        const float mine = __ldcs(d + xc);
        const float other = __shfl_xor_sync(0xffffffffu, mine, 1);
        g[0] = xc ? other : mine;
        g[1] = xc ? mine : other;
    } else if constexpr (F == 4) {
        const float2 mine = __ldcs(reinterpret_cast<const float2*>(d) + xc);
        float2 other;
        other.x = __shfl_xor_sync(0xffffffffu, mine.x, 1);
        other.y = __shfl_xor_sync(0xffffffffu, mine.y, 1);
        const float2 lo = xc ? other : mine, hi = xc ? mine : other;
        g[0] = lo.x; g[1] = lo.y; g[2] = hi.x; g[3] = hi.y;
    } else {
        const float4 mine = __ldcs(reinterpret_cast<const float4*>(d) + xc);
        float4 other;
        other.x = __shfl_xor_sync(0xffffffffu, mine.x, 1);
        other.y = __shfl_xor_sync(0xffffffffu, mine.y, 1);
        other.z = __shfl_xor_sync(0xffffffffu, mine.z, 1);
        other.w = __shfl_xor_sync(0xffffffffu, mine.w, 1);
        const float4 lo = xc ? other : mine, hi = xc ? mine : other;
        g[0] = lo.x; g[1] = lo.y; g[2] = lo.z; g[3] = lo.w;
        g[4] = hi.x; g[5] = hi.y; g[6] = hi.z; g[7] = hi.w;
    }
}

// ------------------------------------------------------------------------------------------------
// Backward: scatter-add of W_k * dY into the table gradient (transpose of Eq. 9)
// ------------------------------------------------------------------------------------------------
template <int F, int D, bool HINT = false>
__global__ void __launch_bounds__(kBlockThreads)
hash4d_bwd_kernel(const __grid_constant__ Plan P, const float* __restrict__ xyz,
                  const float* __restrict__ t, const int32_t* __restrict__ index,
                  const float* __restrict__ dout, float* __restrict__ dtable) {
    constexpr int NC = 1 << (D - 1);
    const Item it = this_item(P);
    const LevelParams lp = P.lv[it.l];
    float g[F];
    load_dout<F>(dout + it.n * (static_cast<size_t>(P.L) * F) + static_cast<size_t>(it.l) * F,
                 it.xc, g);
    const Query q = load_query<D>(P, lp, it.n, xyz, t, index);
    uint32_t slot[NC];
    float W[NC];
    half_cell<D>(P, lp, q, it.xc, slot, W);  // recomputed, never cached from fwd (128 B per item)
    if (!it.active) return;
    float* level_base = dtable + static_cast<size_t>(it.l) * P.T * F;
    uint64_t pol = 0;
    if constexpr (HINT) pol = l2_policy_evict_last();
#pragma unroll
    for (int j = 0; j < NC; ++j) {
        float c[F];
#pragma unroll
        for (int f = 0; f < F; ++f) c[f] = W[j] * g[f];
        if constexpr (HINT) red_add_hint<F>(level_base + static_cast<size_t>(slot[j]) * F, c, pol);
        else red_add<F>(level_base + static_cast<size_t>(slot[j]) * F, c);
    }
}

// Deterministic variant: 64-bit fixed-point accumulation.  Integer addition is associative, so the
// sums do not depend on the order in which the L2 applies the reductions.
template <int F, int D>
__global__ void __launch_bounds__(kBlockThreads)
hash4d_bwd_fixed_kernel(const __grid_constant__ Plan P, const float* __restrict__ xyz,
                        const float* __restrict__ t, const int32_t* __restrict__ index,
                        const float* __restrict__ dout, long long* __restrict__ acc,
                        const WorkspaceHeader* __restrict__ hdr) {
    constexpr int NC = 1 << (D - 1);
    const Item it = this_item(P);
    const LevelParams lp = P.lv[it.l];
    float g[F];
    load_dout<F>(dout + it.n * (static_cast<size_t>(P.L) * F) + static_cast<size_t>(it.l) * F,
                 it.xc, g);
    const Query q = load_query<D>(P, lp, it.n, xyz, t, index);
    uint32_t slot[NC];
    float W[NC];
    half_cell<D>(P, lp, q, it.xc, slot, W);
    if (!it.active) return;
    const float scale = hdr->scale;  // power of two: the products below are exact rescalings
    unsigned long long* level_base =
        reinterpret_cast<unsigned long long*>(acc) + static_cast<size_t>(it.l) * P.T * F;
#pragma unroll
    for (int j = 0; j < NC; ++j) {
#pragma unroll
        for (int f = 0; f < F; ++f) {
            const long long fx = __float2ll_rn(__fmul_rn(__fmul_rn(W[j], g[f]), scale));
            atomicAdd(level_base + static_cast<size_t>(slot[j]) * F + f,
                      static_cast<unsigned long long>(fx));
        }
    }
}

// ------------------------------------------------------------------------------------------------
// Coordinate gradient (Q24): dq[n][d] = d<dout[n], G_4D(x_n)>/dx_d.
// Same gathers as the forward.  Per corner the F features collapse to one scalar S_j = <dout, v_j>;
// the multilinear form is then folded axis by axis (y, z, t), keeping at every fold both the
// interpolated value and the difference along the folded axis, so each axis derivative costs one
// extra subtraction per fold instead of a second pass over the 16 corners.
// ------------------------------------------------------------------------------------------------
template <int F, bool HALF, int D, bool ORDERED>
__global__ void __launch_bounds__(kBlockThreads)
hash4d_bwd_input_kernel(const __grid_constant__ Plan P, const float* __restrict__ xyz,
                        const float* __restrict__ t, const int32_t* __restrict__ index,
                        const void* __restrict__ table, const float* __restrict__ dout,
                        float* __restrict__ dq, const int32_t* __restrict__ order,
                        const float4* __restrict__ sorted_q) {
    constexpr int NC = 1 << (D - 1);   // D = 3: G_3D, 4 (y,z) corners per lane, dq is [N][3]
    Item it = this_item(P);
    const LevelParams lp = P.lv[it.l];
    Query q;
    float g[F];
    if constexpr (ORDERED) {   // SORT_COARSE: the it.n-th query of the cell-sorted order; rows of dout / dq are its own
        const float4 c = __ldg(sorted_q + it.n);
        q = make_query<D>(lp, c.x, c.y, c.z, c.w);
        const uint64_t n = static_cast<uint64_t>(static_cast<uint32_t>(__ldg(order + it.n)));
        it.n = n < P.N ? n : P.N - 1;
        load_dout<F>(dout + it.n * (static_cast<size_t>(P.L) * F) + static_cast<size_t>(it.l) * F, it.xc, g);
    } else {                   // a separate instantiation: the plain kernel is the one that was tuned (32 registers)
        load_dout<F>(dout + it.n * (static_cast<size_t>(P.L) * F) + static_cast<size_t>(it.l) * F, it.xc, g);
        q = load_query<D>(P, lp, it.n, xyz, t, index);
    }
    uint32_t slot[NC];
    float W[NC];
    half_cell<D>(P, lp, q, it.xc, slot, W);  // W unused here; slots shared with fwd
    constexpr size_t kElem = HALF ? 2 : 4;
    const char* level_base =
        static_cast<const char*>(table) + static_cast<size_t>(it.l) * P.T * (F * kElem);
    float v[NC][F];
#pragma unroll
    for (int j = 0; j < NC; ++j) load_slot<F, HALF>(level_base, slot[j], v[j]);
    float S[NC];
#pragma unroll
    for (int j = 0; j < NC; ++j) {
        S[j] = 0.0f;
#pragma unroll
        for (int f = 0; f < F; ++f) S[j] = fmaf(g[f], v[j][f], S[j]);
    }
    const float wy = q.w[1], wz = q.w[2], wt = q.w[3];
    // fold y (corner bit 0): value and d/dy for the NC/2 (z[,t]) combinations
    float a[NC / 2], ay[NC / 2];
#pragma unroll
    for (int m = 0; m < NC / 2; ++m) {
        ay[m] = S[2 * m + 1] - S[2 * m];
        a[m] = fmaf(wy, ay[m], S[2 * m]);
    }
    // fold z (corner bit 1)
    float b[NC / 4], by[NC / 4], bz[NC / 4];
#pragma unroll
    for (int m = 0; m < NC / 4; ++m) {
        bz[m] = a[2 * m + 1] - a[2 * m];
        b[m] = fmaf(wz, bz[m], a[2 * m]);
        by[m] = fmaf(wz, ay[2 * m + 1] - ay[2 * m], ay[2 * m]);
    }
    float val, dy, dz, dt;
    if constexpr (D == 4) {   // fold t (corner bit 2)
        val = fmaf(wt, b[1] - b[0], b[0]);
        dy = fmaf(wt, by[1] - by[0], by[0]);
        dz = fmaf(wt, bz[1] - bz[0], bz[0]);
        dt = b[1] - b[0];
    } else {
        val = b[0]; dy = by[0]; dz = bz[0]; dt = 0.0f;
    }
    // this lane is x-corner xc: d/dx takes the sign, the other axes the x weight
    const float wx = it.xc ? q.w[0] : 1.0f - q.w[0];
    float d4[4] = {it.xc ? val : -val, wx * dy, wx * dz, wx * dt};
    const float scale[4] = {lp.ns_f, lp.ns_f, lp.ns_f, lp.nt_f};  // dw_d/dx_d = N_{l,d}
#pragma unroll
    for (int d = 0; d < 4; ++d) {
        d4[d] *= scale[d];
        if (!it.active || ((q.moved >> d) & 1u) || d >= D) d4[d] = 0.0f;
    }
    // sum the lane pair, then the G levels of this query that sit in this warp (2G adjacent lanes)
    const uint32_t span = 2u * P.group;
#pragma unroll
    for (uint32_t o = 1; o < 32; o <<= 1) {
        if (o < span) {
#pragma unroll
            for (int d = 0; d < D; ++d) d4[d] += __shfl_xor_sync(0xffffffffu, d4[d], o);
        }
    }
    if (it.active && (threadIdx.x & (span - 1u)) == 0) {
        if constexpr (D == 4) {
            float* o = dq + it.n * 4;
            asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(o), "f"(d4[0]),
                         "f"(d4[1]), "f"(d4[2]), "f"(d4[3])
                         : "memory");
        } else {
            float* o = dq + it.n * 3;   // rows of 12 bytes: scalar reductions
#pragma unroll
            for (int d = 0; d < 3; ++d) asm volatile("red.global.add.f32 [%0], %1;" ::"l"(o + d), "f"(d4[d]) : "memory");
        }
    }
}

// ------------------------------------------------------------------------------------------------
// Smoothness regulariser, Eq. 11 (Q25):
//     loss[n] = || G(x_n) - G(x'_n) ||^2 ,  x' = fl32(x + eps),   dtable += 2*scale*(J(x)^T d - J(x')^T d).
// One pass per (query, level): gather the cell of x; if x' falls in the SAME cell (the common case on
// coarse levels for a small eps) its 16 corners are the same slots, so the difference is formed directly
// as sum (W - W') v — no second gather, no cancellation between two large sums — and the scatter is ONE
// reduction per corner with weight (W - W') instead of two.  Only items whose cell differs pay the second
// gather and the second set of reductions.
// ------------------------------------------------------------------------------------------------
template <int F, bool HALF, bool GRAD>
__global__ void __launch_bounds__(kBlockThreads)
hash4d_smooth_kernel(const __grid_constant__ Plan P, const float* __restrict__ xyz,
                     const float* __restrict__ t, const int32_t* __restrict__ index,
                     const float* __restrict__ eps, uint32_t eps_stride,
                     const void* __restrict__ table, float two_scale, float* __restrict__ loss,
                     float* __restrict__ dtable) {
    const Item it = this_item(P);
    const LevelParams lp = P.lv[it.l];
    float c[4];
    load_coords(P, it.n, xyz, t, index, c);
    const float* e = eps + it.n * eps_stride;
    const Query q1 = make_query(lp, c[0], c[1], c[2], c[3]);
    const Query q2 = make_query(lp, __fadd_rn(c[0], __ldg(e + 0)), __fadd_rn(c[1], __ldg(e + 1)),
                                __fadd_rn(c[2], __ldg(e + 2)), __fadd_rn(c[3], __ldg(e + 3)));
    uint32_t s1[8], s2[8];
    float W1[8], W2[8];
    half_cell(P, lp, q1, it.xc, s1, W1);
    half_cell(P, lp, q2, it.xc, s2, W2);
    const bool same = q1.c[0] == q2.c[0] && q1.c[1] == q2.c[1] && q1.c[2] == q2.c[2] &&
                      q1.c[3] == q2.c[3];  // identical for both lanes of the pair

    constexpr size_t kElem = HALF ? 2 : 4;
    const char* level_base =
        static_cast<const char*>(table) + static_cast<size_t>(it.l) * P.T * (F * kElem);
    float d[F];
    {
        float v[8][F];
#pragma unroll
        for (int j = 0; j < 8; ++j) load_slot<F, HALF>(level_base, s1[j], v[j]);
        float y[F], ds[F];
#pragma unroll
        for (int f = 0; f < F; ++f) y[f] = ds[f] = 0.0f;
#pragma unroll
        for (int j = 0; j < 8; ++j) {
            const float dw = W1[j] - W2[j];
#pragma unroll
            for (int f = 0; f < F; ++f) {
                y[f] = fmaf(W1[j], v[j][f], y[f]);
                ds[f] = fmaf(dw, v[j][f], ds[f]);
            }
        }
        if (same) {
#pragma unroll
            for (int f = 0; f < F; ++f) d[f] = ds[f];
        } else {
#pragma unroll
            for (int j = 0; j < 8; ++j) load_slot<F, HALF>(level_base, s2[j], v[j]);
#pragma unroll
            for (int j = 0; j < 8; ++j)
#pragma unroll
                for (int f = 0; f < F; ++f) y[f] = fmaf(-W2[j], v[j][f], y[f]);
#pragma unroll
            for (int f = 0; f < F; ++f) d[f] = y[f];
        }
    }
#pragma unroll
    for (int f = 0; f < F; ++f) d[f] += __shfl_xor_sync(0xffffffffu, d[f], 1);  // both x-corners

    // loss: sum_f d^2, once per item (lane xc = 0), summed over the G levels of the query in this warp
    float lsum = 0.0f;
    if (it.active && it.xc == 0) {
#pragma unroll
        for (int f = 0; f < F; ++f) lsum = fmaf(d[f], d[f], lsum);
    }
    const uint32_t span = 2u * P.group;
#pragma unroll
    for (uint32_t o = 1; o < 32; o <<= 1)
        if (o < span) lsum += __shfl_xor_sync(0xffffffffu, lsum, o);
    if (it.active && (threadIdx.x & (span - 1u)) == 0)
        asm volatile("red.global.add.f32 [%0], %1;" ::"l"(loss + it.n), "f"(lsum) : "memory");

    if constexpr (GRAD) {
        if (!it.active) return;
        float* gbase = dtable + static_cast<size_t>(it.l) * P.T * F;
        float g[F];
#pragma unroll
        for (int f = 0; f < F; ++f) g[f] = two_scale * d[f];
        if (same) {
#pragma unroll
            for (int j = 0; j < 8; ++j) {
                const float dw = W1[j] - W2[j];
                float cc[F];
#pragma unroll
                for (int f = 0; f < F; ++f) cc[f] = dw * g[f];
                red_add<F>(gbase + static_cast<size_t>(s1[j]) * F, cc);
            }
        } else {
#pragma unroll
            for (int j = 0; j < 8; ++j) {
                float cc[F];
#pragma unroll
                for (int f = 0; f < F; ++f) cc[f] = W1[j] * g[f];
                red_add<F>(gbase + static_cast<size_t>(s1[j]) * F, cc);
#pragma unroll
                for (int f = 0; f < F; ++f) cc[f] = -W2[j] * g[f];
                red_add<F>(gbase + static_cast<size_t>(s2[j]) * F, cc);
            }
        }
    }
}

// ------------------------------------------------------------------------------------------------
// Debug: all 16 slots + weights per (query, level)
// ------------------------------------------------------------------------------------------------
template <int D>
__global__ void __launch_bounds__(kBlockThreads)
hash4d_indices_kernel(const __grid_constant__ Plan P, const float* __restrict__ xyz,
                      const float* __restrict__ t, const int32_t* __restrict__ index,
                      uint32_t* __restrict__ idx_out, float* __restrict__ w_out) {
    constexpr int NC = 1 << (D - 1);
    const uint64_t i = static_cast<uint64_t>(blockIdx.x) * kBlockThreads + threadIdx.x;
    if (i >= P.N * P.L) return;
    const uint64_t n = i / P.L;
    const uint32_t l = static_cast<uint32_t>(i - n * P.L);
    const LevelParams lp = P.lv[l];
    const Query q = load_query<D>(P, lp, n, xyz, t, index);
#pragma unroll
    for (uint32_t xc = 0; xc < 2; ++xc) {
        uint32_t slot[NC];
        float W[NC];
        half_cell<D>(P, lp, q, xc, slot, W);
#pragma unroll
        for (int j = 0; j < NC; ++j) {
            idx_out[i * (2 * NC) + (xc | (j << 1))] = slot[j];
            if (w_out) w_out[i * (2 * NC) + (xc | (j << 1))] = W[j];
        }
    }
}

// ------------------------------------------------------------------------------------------------
// Small helpers: fill, |dout| max, fixed-point finalize, input validation
// ------------------------------------------------------------------------------------------------
template <bool HINT>
__global__ void __launch_bounds__(kBlockThreads)
zero_kernel(unsigned char* __restrict__ base, size_t head, size_t n32, size_t tail) {
    // [base, base+head) bytes up to 32-byte alignment, then n32 aligned 32-byte stores (STG.256), then tail bytes
    unsigned char* body = base + head;
    const size_t stride = static_cast<size_t>(gridDim.x) * kBlockThreads;
    uint64_t pol = 0;
    if constexpr (HINT) pol = l2_policy_evict_last();
    for (size_t i = static_cast<size_t>(blockIdx.x) * kBlockThreads + threadIdx.x; i < n32; i += stride) {
        if constexpr (HINT)
            asm volatile("st.global.L2::cache_hint.v8.b32 [%0], {%1, %1, %1, %1, %1, %1, %1, %1}, %2;" ::"l"(body + i * 32),
                         "r"(0u), "l"(pol)
                         : "memory");
        else
            asm volatile("st.global.v8.b32 [%0], {%1, %1, %1, %1, %1, %1, %1, %1};" ::"l"(body + i * 32), "r"(0u)
                         : "memory");
    }
    if (blockIdx.x == 0) {
        if (threadIdx.x < head) base[threadIdx.x] = 0;
        if (threadIdx.x < tail) base[head + n32 * 32 + threadIdx.x] = 0;
    }
}

__global__ void __launch_bounds__(kBlockThreads)
absmax_kernel(const float* __restrict__ v, size_t count, WorkspaceHeader* __restrict__ hdr) {
    const size_t stride = static_cast<size_t>(gridDim.x) * kBlockThreads;
    uint32_t m = 0;
    for (size_t i = static_cast<size_t>(blockIdx.x) * kBlockThreads + threadIdx.x; i < count;
         i += stride)
        m = max(m, __float_as_uint(fabsf(__ldg(v + i))));  // non-negative floats order as uints
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) m = max(m, __shfl_xor_sync(0xffffffffu, m, o));
    if ((threadIdx.x & 31) == 0 && m) atomicMax(&hdr->absmax_bits, m);
}

// scale = 2^s with N * max|dY| * 2^s <= 2^61: no slot can overflow int64 (weights of one query sum to 1).
__global__ void fixed_scale_kernel(WorkspaceHeader* hdr, uint64_t N) {
    const float amax = __uint_as_float(hdr->absmax_bits);
    int e = 0;
    if (amax > 0.0f && amax < __int_as_float(0x7f800000)) frexpf(amax, &e);  // amax < 2^e
    int k = 0;
    while ((1ull << k) < N && k < 62) ++k;  // N <= 2^k
    int s = 61 - e - k;
    s = max(-100, min(100, s));
    hdr->scale = ldexpf(1.0f, s);
    hdr->inv_scale = ldexp(1.0, -s);
}

__global__ void __launch_bounds__(kBlockThreads)
fixed_finalize_kernel(const long long* __restrict__ acc, float* __restrict__ dtable, size_t count,
                      const WorkspaceHeader* __restrict__ hdr, int overwrite) {
    const size_t stride = static_cast<size_t>(gridDim.x) * kBlockThreads;
    const double inv = hdr->inv_scale;
    for (size_t i = static_cast<size_t>(blockIdx.x) * kBlockThreads + threadIdx.x; i < count;
         i += stride) {
        const double sum = __ll2double_rn(acc[i]) * inv;
        dtable[i] = static_cast<float>(overwrite ? sum : static_cast<double>(dtable[i]) + sum);
    }
}

__global__ void __launch_bounds__(kBlockThreads)
validate_kernel(const __grid_constant__ Plan P, const float* __restrict__ xyz,
                const float* __restrict__ t, const int32_t* __restrict__ index,
                WorkspaceHeader* __restrict__ hdr) {
    const size_t stride = static_cast<size_t>(gridDim.x) * kBlockThreads;
    uint32_t bad = 0;
    for (uint64_t n = static_cast<uint64_t>(blockIdx.x) * kBlockThreads + threadIdx.x; n < P.N;
         n += stride) {
        const uint64_t row = index ? static_cast<uint64_t>(index[n]) : n;
        const float* p = xyz + row * P.xyz_stride;
        const float c[4] = {p[0], p[1], p[2], P.dims == 3 ? 0.0f : t[n * P.t_stride]};
#pragma unroll
        for (int d = 0; d < 4; ++d) bad += !(c[d] >= 0.0f && c[d] < 1.0f);  // NaN fails both
    }
    if (bad) atomicAdd(&hdr->bad_inputs, bad);
}


// ------------------------------------------------------------------------------------------------
// Sparse Adam over the touched table entries (Q28): entries whose gradient is
// exactly zero are skipped — theta, m, v untouched, and (four at a time) not even read.  Streaming, HBM-bound:
// 4 B per untouched entry, 34-36 B per touched one (g, m, v, theta in; m, v, theta, [half copy], g = 0 out).
// ------------------------------------------------------------------------------------------------
struct AdamParams {
    float lr, beta1, beta2, eps;
    float omb1, omb2;      // 1 - beta1, 1 - beta2
    float inv_c1, inv_c2;  // 1 / (1 - beta1^t), 1 / (1 - beta2^t), evaluated in double on the host
    int zero_grad;
};

__device__ __forceinline__ void adam_one(const AdamParams& A, float g, float& th, float& m, float& v) {
    if (g != 0.0f) {
        m = fmaf(A.beta1, m, A.omb1 * g);
        v = fmaf(A.beta2, v, A.omb2 * g * g);
        th -= __fdiv_rn(A.lr * (m * A.inv_c1), sqrtf(v * A.inv_c2) + A.eps);
    }
}

__global__ void __launch_bounds__(kBlockThreads)
adam_step_kernel(const AdamParams A, size_t n4, size_t count, float* __restrict__ theta,
                 __half* __restrict__ theta16, float* __restrict__ grad, float* __restrict__ m,
                 float* __restrict__ v) {
    const size_t stride = static_cast<size_t>(gridDim.x) * kBlockThreads;
    for (size_t i = static_cast<size_t>(blockIdx.x) * kBlockThreads + threadIdx.x; i < n4; i += stride) {
        const float4 g = reinterpret_cast<const float4*>(grad)[i];
        if (g.x == 0.0f && g.y == 0.0f && g.z == 0.0f && g.w == 0.0f) continue;  // untouched: 16 bytes read
        float4 th = reinterpret_cast<float4*>(theta)[i];
        float4 mm = reinterpret_cast<float4*>(m)[i];
        float4 vv = reinterpret_cast<float4*>(v)[i];
        adam_one(A, g.x, th.x, mm.x, vv.x);
        adam_one(A, g.y, th.y, mm.y, vv.y);
        adam_one(A, g.z, th.z, mm.z, vv.z);
        adam_one(A, g.w, th.w, mm.w, vv.w);
        reinterpret_cast<float4*>(theta)[i] = th;
        reinterpret_cast<float4*>(m)[i] = mm;
        reinterpret_cast<float4*>(v)[i] = vv;
        if (theta16) {
            const __half2 lo = __floats2half2_rn(th.x, th.y), hi = __floats2half2_rn(th.z, th.w);
            uint2 packed;
            packed.x = *reinterpret_cast<const uint32_t*>(&lo);
            packed.y = *reinterpret_cast<const uint32_t*>(&hi);
            reinterpret_cast<uint2*>(theta16)[i] = packed;
        }
        if (A.zero_grad) reinterpret_cast<float4*>(grad)[i] = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
    }
    // the last count % 4 entries
    if (blockIdx.x == 0 && threadIdx.x < count - n4 * 4) {
        const size_t e = n4 * 4 + threadIdx.x;
        const float g = grad[e];
        if (g != 0.0f) {
            float th = theta[e], mm = m[e], vv = v[e];
            adam_one(A, g, th, mm, vv);
            theta[e] = th; m[e] = mm; v[e] = vv;
            if (theta16) theta16[e] = __float2half_rn(th);
            if (A.zero_grad) grad[e] = 0.0f;
        }
    }
}

// ------------------------------------------------------------------------------------------------
// Time slice of the tables at ONE timestamp (render path, "one timestamp per rendered frame";
// DESIGN.md Q29).  For a fixed t the 16-corner interpolation of Eq. 9 factors into a blend of the two
// t-layers, done here once per frame over the whole level, and an 8-corner lookup per query (the D = 3
// kernels on the slice):  hashed level, power-of-two T:  slice[u] = (1-w) tab[u ^ a] + w tab[u ^ b],
// a = (c_t pi_4) mod T, b = ((c_t+1) pi_4) mod T ("mod 2^k" commutes with XOR);  dense level:
// slice[s3] = (1-w) tab[s3 + S^3 c_t] + w tab[s3 + S^3 (c_t+1)], s3 < S^3.  Streaming: 2 reads, 1 write.
// ------------------------------------------------------------------------------------------------
template <int F, bool HALF>
__global__ void __launch_bounds__(kBlockThreads)
slice_t_kernel(const __grid_constant__ Plan P, const float* __restrict__ t,
               const void* __restrict__ table, float* __restrict__ slice) {
    const uint32_t l = blockIdx.y;
    const LevelParams lp = P.lv[l];
    uint32_t ct;
    float wt;
    locate(__ldg(t), lp.nt_f, ct, wt);
    const uint32_t count = lp.dense ? lp.m[3] : P.T;           // dense: m[3] = S^3 vertices per t-layer
    const uint32_t a = lp.dense ? lp.m[3] * ct : (ct * lp.m[3]) & P.t_mask;
    const uint32_t b = lp.dense ? a + lp.m[3] : ((ct + 1u) * lp.m[3]) & P.t_mask;
    constexpr size_t kElem = HALF ? 2 : 4;
    const char* level_base = static_cast<const char*>(table) + static_cast<size_t>(l) * P.T * (F * kElem);
    float* dst = slice + static_cast<size_t>(l) * P.T * F;
    const float w0 = 1.0f - wt;
    for (uint32_t u = blockIdx.x * kBlockThreads + threadIdx.x; u < count; u += gridDim.x * kBlockThreads) {
        float v0[F], v1[F], r[F];
        load_slot<F, HALF>(level_base, lp.dense ? u + a : u ^ a, v0);
        load_slot<F, HALF>(level_base, lp.dense ? u + b : u ^ b, v1);
#pragma unroll
        for (int f = 0; f < F; ++f) r[f] = fmaf(wt, v1[f], w0 * v0[f]);
        float* o = dst + static_cast<size_t>(u) * F;
        if constexpr (F == 1) {
            o[0] = r[0];
        } else if constexpr (F == 2) {
            *reinterpret_cast<float2*>(o) = make_float2(r[0], r[1]);
        } else if constexpr (F == 4) {
            *reinterpret_cast<float4*>(o) = make_float4(r[0], r[1], r[2], r[3]);
        } else {
            *reinterpret_cast<float4*>(o) = make_float4(r[0], r[1], r[2], r[3]);
            *(reinterpret_cast<float4*>(o) + 1) = make_float4(r[4], r[5], r[6], r[7]);
        }
    }
}

// ------------------------------------------------------------------------------------------------
// Spatial counting sort of the queries (dash_hash4d_sort_queries): key = Morton code of the coarse cell.
// keys + histogram -> 3-launch exclusive scan over the bins (1024 bins per CTA) -> scatter through per-bin cursors.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t spread3(uint32_t v) {   // 7 bits -> every third bit
    v &= 0x7fu;
    v = (v | (v << 8)) & 0x0000700fu;
    v = (v | (v << 4)) & 0x000430c3u;
    v = (v | (v << 2)) & 0x00049249u;
    return v;
}

__global__ void __launch_bounds__(kBlockThreads)
sort_keys_kernel(uint64_t N, const float* __restrict__ xyz, uint32_t xyz_stride,
                 const int32_t* __restrict__ index, float scale, uint32_t cell_max,
                 uint32_t* __restrict__ keys, uint32_t* __restrict__ hist) {
    const size_t stride = static_cast<size_t>(gridDim.x) * kBlockThreads;
    for (uint64_t n = static_cast<uint64_t>(blockIdx.x) * kBlockThreads + threadIdx.x; n < N; n += stride) {
        const uint64_t row = index ? static_cast<uint64_t>(__ldg(index + n)) : n;
        const float* p = xyz + row * xyz_stride;
        uint32_t key = 0;
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            const uint32_t c = min(static_cast<uint32_t>(clamp_unit(__ldg(p + d)) * scale), cell_max);
            key |= spread3(c) << d;
        }
        keys[n] = key;
        atomicAdd(hist + key, 1u);
    }
}

// exclusive scan, phase 1: each CTA of 256 threads scans kScanTile = 4096 bins in place (16 per thread, four 16-byte
// loads) and writes its total.  The bins array is allocated in multiples of 16 bytes; elements >= n_bins count as 0.
__global__ void __launch_bounds__(kBlockThreads) sort_scan_local_kernel(uint32_t* __restrict__ bins, uint32_t n_bins,
                                                                        uint32_t* __restrict__ totals) {
    __shared__ uint32_t warp_sum[kBlockThreads / 32];
    const uint32_t lane = threadIdx.x & 31u, w = threadIdx.x >> 5;
    const uint32_t first = blockIdx.x * kScanTile + threadIdx.x * 16u;
    uint4* p = reinterpret_cast<uint4*>(bins + first);
    uint32_t v[16];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        uint4 a = make_uint4(0u, 0u, 0u, 0u);
        if (first + 4u * k < n_bins) a = p[k];
        v[4 * k] = a.x; v[4 * k + 1] = a.y; v[4 * k + 2] = a.z; v[4 * k + 3] = a.w;
    }
    uint32_t sum = 0;
#pragma unroll
    for (int k = 0; k < 16; ++k) {
        const uint32_t x = (first + k < n_bins) ? v[k] : 0u;
        v[k] = sum;            // exclusive within the thread
        sum += x;
    }
    uint32_t x = sum;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const uint32_t y = __shfl_up_sync(0xffffffffu, x, o);
        if (lane >= static_cast<uint32_t>(o)) x += y;
    }
    if (lane == 31) warp_sum[w] = x;
    __syncthreads();
    uint32_t before = x - sum;   // exclusive within the warp
#pragma unroll
    for (uint32_t k = 0; k < kBlockThreads / 32; ++k)
        if (k < w) before += warp_sum[k];
#pragma unroll
    for (int k = 0; k < 4; ++k)
        if (first + 4u * k < n_bins)
            p[k] = make_uint4(before + v[4 * k], before + v[4 * k + 1], before + v[4 * k + 2], before + v[4 * k + 3]);
    if (threadIdx.x == kBlockThreads - 1) totals[blockIdx.x] = before + sum;
}

// phase 2: one CTA turns the CTA totals into exclusive offsets
__global__ void __launch_bounds__(1024) sort_scan_totals_kernel(uint32_t* __restrict__ totals, uint32_t n) {
    __shared__ uint32_t warp_sum[32];
    __shared__ uint32_t carry;
    if (threadIdx.x == 0) carry = 0;
    __syncthreads();
    for (uint32_t base = 0; base < n; base += 1024u) {
        const uint32_t i = base + threadIdx.x, lane = threadIdx.x & 31u, w = threadIdx.x >> 5;
        const uint32_t v = i < n ? totals[i] : 0u;
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
        if (i < n) totals[i] = before + x - v;
        __syncthreads();
        if (threadIdx.x == 1023) carry = before + x;
        __syncthreads();
    }
}

// phase 3: add the CTA offsets (callers that index bins through their own kernel add totals[i / kScanTile] there)
__global__ void __launch_bounds__(kBlockThreads) sort_scan_add_kernel(uint32_t* __restrict__ bins, uint32_t n_bins,
                                                                      const uint32_t* __restrict__ totals) {
    const uint32_t first = blockIdx.x * kScanTile + threadIdx.x * 16u;
    const uint32_t off = totals[blockIdx.x];
    uint4* p = reinterpret_cast<uint4*>(bins + first);
#pragma unroll
    for (int k = 0; k < 4; ++k)
        if (first + 4u * k < n_bins) {
            uint4 a = p[k];
            a.x += off; a.y += off; a.z += off; a.w += off;
            p[k] = a;
        }
}

__global__ void __launch_bounds__(kBlockThreads)
sort_scatter_kernel(uint64_t N, const uint32_t* __restrict__ keys, uint32_t* __restrict__ cursor,
                    int32_t* __restrict__ order) {
    const size_t stride = static_cast<size_t>(gridDim.x) * kBlockThreads;
    for (uint64_t n = static_cast<uint64_t>(blockIdx.x) * kBlockThreads + threadIdx.x; n < N; n += stride)
        order[atomicAdd(cursor + keys[n], 1u)] = static_cast<int32_t>(n);
}

// SM count / L2 bytes of the CURRENT device, cached per device ordinal (a process may drive several GPUs).
struct DeviceInfo {
    int sms;
    size_t l2;
};

const DeviceInfo& device_info() {
    constexpr int kMaxDevices = 64;
    static DeviceInfo cache[kMaxDevices] = {};  // sms == 0: not queried yet; races write identical values
    static thread_local DeviceInfo scratch;
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) dev = -1;
    DeviceInfo* slot = (dev >= 0 && dev < kMaxDevices) ? &cache[dev] : &scratch;
    if (slot == &scratch || slot->sms == 0) {
        int sms = 0, l2 = 0;
        if (dev < 0 || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms <= 0)
            sms = 148;
        if (dev < 0 || cudaDeviceGetAttribute(&l2, cudaDevAttrL2CacheSize, dev) != cudaSuccess || l2 <= 0)
            l2 = 64 << 20;
        slot->l2 = static_cast<size_t>(l2);
        slot->sms = sms;
    }
    return *slot;
}

int sm_count() { return device_info().sms; }

inline cudaError_t after_launch() {
    ++g_launches;
    return cudaGetLastError();
}

inline dim3 item_grid(const Plan& P) {
    const uint64_t tiles = (P.N + P.q_per_block - 1) / P.q_per_block;
    return dim3(static_cast<unsigned>(tiles), P.num_groups, 1);
}

}  // namespace

void count_launch() { ++g_launches; }

int device_sm_count() { return sm_count(); }

size_t device_l2_bytes() { return device_info().l2; }

uint64_t launch_counter(bool reset) {
    const uint64_t v = g_launches;
    if (reset) g_launches = 0;
    return v;
}

cudaError_t launch_fwd(const Plan& P, const float* xyz, const float* t, const int32_t* index,
                       const void* table, bool table_half, float* out, cudaStream_t s, const int32_t* order,
                       const float4* sorted_q) {
    const dim3 grid = item_grid(P), block(kBlockThreads);
#define DASH_FWD_D(FV, HV, DV)                                                                               \
    do {                                                                                                     \
        if (order)                                                                                           \
            hash4d_fwd_kernel<FV, HV, DV, true><<<grid, block, 0, s>>>(P, xyz, t, index, table, out, order,   \
                                                                       sorted_q);                            \
        else                                                                                                 \
            hash4d_fwd_kernel<FV, HV, DV, false><<<grid, block, 0, s>>>(P, xyz, t, index, table, out, nullptr, \
                                                                        nullptr);                            \
    } while (0)
#define DASH_FWD(FV, HV)                        \
    do {                                        \
        if (P.dims == 3) DASH_FWD_D(FV, HV, 3); \
        else DASH_FWD_D(FV, HV, 4);             \
    } while (0)
    switch (P.F * 2 + (table_half ? 1 : 0)) {
        case 2: DASH_FWD(1, false); break;
        case 3: DASH_FWD(1, true); break;
        case 4: DASH_FWD(2, false); break;
        case 5: DASH_FWD(2, true); break;
        case 8: DASH_FWD(4, false); break;
        case 9: DASH_FWD(4, true); break;
        case 16: DASH_FWD(8, false); break;
        case 17: DASH_FWD(8, true); break;
        default: return cudaErrorInvalidValue;
    }
#undef DASH_FWD
#undef DASH_FWD_D
    return after_launch();
}

cudaError_t launch_bwd_input(const Plan& P, const float* xyz, const float* t, const int32_t* index,
                             const void* table, bool table_half, const float* dout, float* dq,
                             cudaStream_t s, const int32_t* order, const float4* sorted_q) {
    const dim3 grid = item_grid(P), block(kBlockThreads);
#define DASH_BWI_D(FV, HV, DV)                                                                                 \
    do {                                                                                                       \
        if (order)                                                                                             \
            hash4d_bwd_input_kernel<FV, HV, DV, true><<<grid, block, 0, s>>>(P, xyz, t, index, table, dout, dq, \
                                                                             order, sorted_q);                 \
        else                                                                                                   \
            hash4d_bwd_input_kernel<FV, HV, DV, false><<<grid, block, 0, s>>>(P, xyz, t, index, table, dout, dq, \
                                                                              nullptr, nullptr);               \
    } while (0)
#define DASH_BWI(FV, HV)                        \
    do {                                        \
        if (P.dims == 3) DASH_BWI_D(FV, HV, 3); \
        else DASH_BWI_D(FV, HV, 4);             \
    } while (0)
    switch (P.F * 2 + (table_half ? 1 : 0)) {
        case 2: DASH_BWI(1, false); break;
        case 3: DASH_BWI(1, true); break;
        case 4: DASH_BWI(2, false); break;
        case 5: DASH_BWI(2, true); break;
        case 8: DASH_BWI(4, false); break;
        case 9: DASH_BWI(4, true); break;
        case 16: DASH_BWI(8, false); break;
        case 17: DASH_BWI(8, true); break;
        default: return cudaErrorInvalidValue;
    }
#undef DASH_BWI
#undef DASH_BWI_D
    return after_launch();
}

template <int F, bool HALF>
static cudaError_t launch_smooth_t(const Plan& P, const float* xyz, const float* t,
                                   const int32_t* index, const float* eps, uint32_t eps_stride,
                                   const void* table, float two_scale, float* loss, float* dtable,
                                   cudaStream_t s) {
    const dim3 grid = item_grid(P), block(kBlockThreads);
    if (dtable)
        hash4d_smooth_kernel<F, HALF, true><<<grid, block, 0, s>>>(P, xyz, t, index, eps, eps_stride,
                                                                   table, two_scale, loss, dtable);
    else
        hash4d_smooth_kernel<F, HALF, false><<<grid, block, 0, s>>>(P, xyz, t, index, eps, eps_stride,
                                                                    table, two_scale, loss, dtable);
    return after_launch();
}

cudaError_t launch_smooth(const Plan& P, const float* xyz, const float* t, const int32_t* index,
                          const float* eps, uint32_t eps_stride, const void* table, bool table_half,
                          float two_scale, float* loss, float* dtable, cudaStream_t s) {
#define DASH_SM(FV, HV) \
    return launch_smooth_t<FV, HV>(P, xyz, t, index, eps, eps_stride, table, two_scale, loss, dtable, s)
    switch (P.F * 2 + (table_half ? 1 : 0)) {
        case 2: DASH_SM(1, false);
        case 3: DASH_SM(1, true);
        case 4: DASH_SM(2, false);
        case 5: DASH_SM(2, true);
        case 8: DASH_SM(4, false);
        case 9: DASH_SM(4, true);
        case 16: DASH_SM(8, false);
        case 17: DASH_SM(8, true);
        default: return cudaErrorInvalidValue;
    }
#undef DASH_SM
}

cudaError_t launch_bwd(const Plan& P, const float* xyz, const float* t, const int32_t* index,
                       const float* dout, float* dtable, cudaStream_t s, bool l2_hint) {
    const dim3 grid = item_grid(P), block(kBlockThreads);
#define DASH_BWD(FV)                                                                                 \
    do {                                                                                             \
        if (P.dims == 3 && l2_hint)                                                                  \
            hash4d_bwd_kernel<FV, 3, true><<<grid, block, 0, s>>>(P, xyz, t, index, dout, dtable);   \
        else if (P.dims == 3)                                                                        \
            hash4d_bwd_kernel<FV, 3><<<grid, block, 0, s>>>(P, xyz, t, index, dout, dtable);         \
        else if (l2_hint)                                                                            \
            hash4d_bwd_kernel<FV, 4, true><<<grid, block, 0, s>>>(P, xyz, t, index, dout, dtable);   \
        else                                                                                         \
            hash4d_bwd_kernel<FV, 4><<<grid, block, 0, s>>>(P, xyz, t, index, dout, dtable);         \
    } while (0)
    switch (P.F) {
        case 1: DASH_BWD(1); break;
        case 2: DASH_BWD(2); break;
        case 4: DASH_BWD(4); break;
        case 8: DASH_BWD(8); break;
        default: return cudaErrorInvalidValue;
    }
#undef DASH_BWD
    return after_launch();
}

cudaError_t launch_bwd_fixed(const Plan& P, const float* xyz, const float* t, const int32_t* index,
                             const float* dout, long long* acc, const WorkspaceHeader* hdr,
                             cudaStream_t s) {
    const dim3 grid = item_grid(P), block(kBlockThreads);
#define DASH_BWDF(FV)                                                                               \
    do {                                                                                            \
        if (P.dims == 3)                                                                            \
            hash4d_bwd_fixed_kernel<FV, 3><<<grid, block, 0, s>>>(P, xyz, t, index, dout, acc, hdr); \
        else                                                                                        \
            hash4d_bwd_fixed_kernel<FV, 4><<<grid, block, 0, s>>>(P, xyz, t, index, dout, acc, hdr); \
    } while (0)
    switch (P.F) {
        case 1: DASH_BWDF(1); break;
        case 2: DASH_BWDF(2); break;
        case 4: DASH_BWDF(4); break;
        case 8: DASH_BWDF(8); break;
        default: return cudaErrorInvalidValue;
    }
#undef DASH_BWDF
    return after_launch();
}

cudaError_t launch_indices(const Plan& P, const float* xyz, const float* t, const int32_t* index,
                           uint32_t* idx_out, float* w_out, cudaStream_t s) {
    const uint64_t items = P.N * P.L;
    const uint64_t blocks = (items + kBlockThreads - 1) / kBlockThreads;
    if (P.dims == 3)
        hash4d_indices_kernel<3><<<static_cast<unsigned>(blocks), kBlockThreads, 0, s>>>(
            P, xyz, t, index, idx_out, w_out);
    else
        hash4d_indices_kernel<4><<<static_cast<unsigned>(blocks), kBlockThreads, 0, s>>>(
            P, xyz, t, index, idx_out, w_out);
    return after_launch();
}

cudaError_t launch_zero(void* ptr, size_t bytes, cudaStream_t s, bool l2_hint) {
    if (bytes == 0) return cudaSuccess;
    size_t head = (32 - (reinterpret_cast<uintptr_t>(ptr) & 31u)) & 31u;
    if (head > bytes) head = bytes;
    const size_t n32 = (bytes - head) / 32, tail = (bytes - head) % 32;
    const size_t want = (n32 + kBlockThreads - 1) / kBlockThreads;
    const size_t cap = static_cast<size_t>(sm_count()) * 16;
    const unsigned blocks = static_cast<unsigned>(want < 1 ? 1 : (want > cap ? cap : want));
    if (l2_hint)
        zero_kernel<true><<<blocks, kBlockThreads, 0, s>>>(static_cast<unsigned char*>(ptr), head, n32, tail);
    else
        zero_kernel<false><<<blocks, kBlockThreads, 0, s>>>(static_cast<unsigned char*>(ptr), head, n32, tail);
    return after_launch();
}

cudaError_t launch_absmax(const float* v, size_t count, WorkspaceHeader* hdr, uint64_t N,
                          cudaStream_t s) {
    const size_t want = (count + kBlockThreads - 1) / kBlockThreads;
    const size_t cap = static_cast<size_t>(sm_count()) * 8;
    const unsigned blocks = static_cast<unsigned>(want < 1 ? 1 : (want > cap ? cap : want));
    absmax_kernel<<<blocks, kBlockThreads, 0, s>>>(v, count, hdr);
    cudaError_t e = after_launch();
    if (e != cudaSuccess) return e;
    fixed_scale_kernel<<<1, 1, 0, s>>>(hdr, N);
    return after_launch();
}

cudaError_t launch_fixed_finalize(const long long* acc, float* dtable, size_t count,
                                  const WorkspaceHeader* hdr, bool overwrite, cudaStream_t s) {
    const size_t want = (count + kBlockThreads - 1) / kBlockThreads;
    const size_t cap = static_cast<size_t>(sm_count()) * 16;
    const unsigned blocks = static_cast<unsigned>(want < 1 ? 1 : (want > cap ? cap : want));
    fixed_finalize_kernel<<<blocks, kBlockThreads, 0, s>>>(acc, dtable, count, hdr, overwrite ? 1 : 0);
    return after_launch();
}

// bins[i] <- sum of bins[0..i) in place; totals: scratch of ceil(n_bins / kScanTile) uint32.  add_offsets = false
// leaves the scan per tile of kScanTile bins: the full value is bins[i] + totals[i / kScanTile] (one launch less).
cudaError_t launch_exclusive_scan_u32(uint32_t* bins, uint32_t n_bins, uint32_t* totals, cudaStream_t s,
                                      bool add_offsets) {
    const uint32_t scan_ctas = (n_bins + kScanTile - 1u) / kScanTile;
    cudaError_t e;
    sort_scan_local_kernel<<<scan_ctas, kBlockThreads, 0, s>>>(bins, n_bins, totals);
    if ((e = after_launch()) != cudaSuccess) return e;
    sort_scan_totals_kernel<<<1, 1024, 0, s>>>(totals, scan_ctas);
    if ((e = after_launch()) != cudaSuccess || !add_offsets) return e;
    sort_scan_add_kernel<<<scan_ctas, kBlockThreads, 0, s>>>(bins, n_bins, totals);
    return after_launch();
}

cudaError_t launch_sort_queries(uint64_t N, const float* xyz, uint32_t xyz_stride, const int32_t* index,
                                uint32_t bits, int32_t* order, uint32_t* keys, uint32_t* bins, uint32_t* totals,
                                cudaStream_t s) {
    const uint32_t n_bins = 1u << (3u * bits);
    const size_t want = (N + kBlockThreads - 1) / kBlockThreads;
    const size_t cap = static_cast<size_t>(sm_count()) * 16;
    const unsigned blocks = static_cast<unsigned>(want < 1 ? 1 : (want > cap ? cap : want));
    cudaError_t e = launch_zero(bins, static_cast<size_t>(n_bins) * sizeof(uint32_t), s);
    if (e != cudaSuccess) return e;
    sort_keys_kernel<<<blocks, kBlockThreads, 0, s>>>(N, xyz, xyz_stride, index, static_cast<float>(1u << bits),
                                                      (1u << bits) - 1u, keys, bins);
    if ((e = after_launch()) != cudaSuccess) return e;
    if ((e = launch_exclusive_scan_u32(bins, n_bins, totals, s)) != cudaSuccess) return e;
    sort_scatter_kernel<<<blocks, kBlockThreads, 0, s>>>(N, keys, bins, order);
    return after_launch();
}

cudaError_t launch_slice_t(const Plan& P, const float* t, const void* table, bool table_half, float* slice,
                           cudaStream_t s) {
    const unsigned per_level = (P.T + kBlockThreads - 1) / kBlockThreads;
    const unsigned cap = static_cast<unsigned>(sm_count()) * 8u / (P.L < 8 ? 1u : P.L / 8u);
    const dim3 grid(per_level < cap ? per_level : (cap ? cap : 1u), P.L, 1), block(kBlockThreads);
#define DASH_SL(FV, HV) slice_t_kernel<FV, HV><<<grid, block, 0, s>>>(P, t, table, slice)
    switch (P.F * 2 + (table_half ? 1 : 0)) {
        case 2: DASH_SL(1, false); break;
        case 3: DASH_SL(1, true); break;
        case 4: DASH_SL(2, false); break;
        case 5: DASH_SL(2, true); break;
        case 8: DASH_SL(4, false); break;
        case 9: DASH_SL(4, true); break;
        case 16: DASH_SL(8, false); break;
        case 17: DASH_SL(8, true); break;
        default: return cudaErrorInvalidValue;
    }
#undef DASH_SL
    return after_launch();
}

cudaError_t launch_adam(size_t count, double lr, double beta1, double beta2, double eps, uint32_t step,
                        bool zero_grad, float* theta, void* theta16, float* grad, float* m, float* v,
                        cudaStream_t s) {
    AdamParams A;
    A.lr = static_cast<float>(lr);
    A.beta1 = static_cast<float>(beta1);
    A.beta2 = static_cast<float>(beta2);
    A.eps = static_cast<float>(eps);
    A.omb1 = static_cast<float>(1.0 - beta1);
    A.omb2 = static_cast<float>(1.0 - beta2);
    A.inv_c1 = static_cast<float>(1.0 / (1.0 - std::pow(beta1, static_cast<double>(step))));
    A.inv_c2 = static_cast<float>(1.0 / (1.0 - std::pow(beta2, static_cast<double>(step))));
    A.zero_grad = zero_grad ? 1 : 0;
    const size_t n4 = count / 4;
    const size_t want = (n4 + kBlockThreads - 1) / kBlockThreads;
    const size_t cap = static_cast<size_t>(sm_count()) * 8;
    const unsigned blocks = static_cast<unsigned>(want < 1 ? 1 : (want > cap ? cap : want));
    adam_step_kernel<<<blocks, kBlockThreads, 0, s>>>(A, n4, count, theta, static_cast<__half*>(theta16), grad,
                                                      m, v);
    return after_launch();
}

cudaError_t launch_validate(const Plan& P, const float* xyz, const float* t, const int32_t* index,
                            WorkspaceHeader* hdr, cudaStream_t s) {
    const size_t want = (P.N + kBlockThreads - 1) / kBlockThreads;
    const size_t cap = static_cast<size_t>(sm_count()) * 8;
    const unsigned blocks = static_cast<unsigned>(want < 1 ? 1 : (want > cap ? cap : want));
    validate_kernel<<<blocks, kBlockThreads, 0, s>>>(P, xyz, t, index, hdr);
    return after_launch();
}

}  // namespace dash
