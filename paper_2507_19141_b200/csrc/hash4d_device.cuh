// hash4d_device.cuh — device-side building blocks of the hash encoder shared by the sm_100a kernels
// (hash4d_kernels.cu, deform_kernels.cu): cell location, vertex -> slot (Eq. 8 / dense index), multilinear
// weights, table slot loads, vector reductions.  Product code: shares nothing with oracle/.
#pragma once
#include <cuda_fp16.h>
#include <cuda_runtime.h>

#include <cstddef>
#include <cstdint>

#include "hash4d_plan.h"

namespace dash {
namespace {

// ------------------------------------------------------------------------------------------------
// Cell location and vertex -> slot (Eq. 8 / dense index)
// ------------------------------------------------------------------------------------------------

// Reading Q12: clamp to [0, 1-2^-24]; fmaxf(NaN, 0) = 0.
__device__ __forceinline__ float clamp_unit(float v) { return fminf(fmaxf(v, 0.0f), 0x1.fffffep-1f); }

// floor(x * N_l) with ONE binary32 multiply (reading Q4): __fmul_rn is never contracted into an FMA.
__device__ __forceinline__ void locate(float x, float res, uint32_t& cell, float& frac) {
    const float pos = __fmul_rn(clamp_unit(x), res);
    const float fl = floorf(pos);
    cell = static_cast<uint32_t>(fl);
    frac = pos - fl;  // exact
}

struct Query {
    uint32_t c[4];   // cell (floor) per axis x,y,z,t
    float w[4];      // fractional offset per axis
    uint32_t moved;  // bit d: the Q12 clamp changed coordinate d (NaN, < 0, > 1-2^-24)
};

__device__ __forceinline__ uint32_t moved_bit(float v, int d) {
    return (v >= 0.0f && v <= 0x1.fffffep-1f) ? 0u : (1u << d);  // NaN fails both comparisons
}

template <int D = 4>
__device__ __forceinline__ Query make_query(const LevelParams& lp, float x, float y, float z, float tt) {
    Query q;
    locate(x, lp.ns_f, q.c[0], q.w[0]);
    locate(y, lp.ns_f, q.c[1], q.w[1]);
    locate(z, lp.ns_f, q.c[2], q.w[2]);
    q.moved = moved_bit(x, 0) | moved_bit(y, 1) | moved_bit(z, 2);
    if constexpr (D == 4) {
        locate(tt, lp.nt_f, q.c[3], q.w[3]);
        q.moved |= moved_bit(tt, 3);
    } else {  // G_3D: no temporal axis
        q.c[3] = 0u;
        q.w[3] = 0.0f;
    }
    return q;
}

template <int D = 4>
__device__ __forceinline__ void load_coords(const Plan& P, uint64_t n, const float* __restrict__ xyz,
                                            const float* __restrict__ t,
                                            const int32_t* __restrict__ index, float c[4]) {
    const uint64_t row = index ? static_cast<uint64_t>(__ldg(index + n)) : n;
    const float* p = xyz + row * P.xyz_stride;
    c[0] = __ldg(p + 0);
    c[1] = __ldg(p + 1);
    c[2] = __ldg(p + 2);
    if constexpr (D == 4) c[3] = __ldg(t + n * P.t_stride);
    else c[3] = 0.0f;
}

template <int D = 4>
__device__ __forceinline__ Query load_query(const Plan& P, const LevelParams& lp, uint64_t n,
                                            const float* __restrict__ xyz,
                                            const float* __restrict__ t,
                                            const int32_t* __restrict__ index) {
    float c[4];
    load_coords<D>(P, n, xyz, t, index, c);
    return make_query<D>(lp, c[0], c[1], c[2], c[3]);
}

// The 2^(D-1) corners that share x-corner `xc` (0: floor, 1: floor+1).  Corner j: bit0 = y, bit1 = z,
// bit2 = t (D = 4 only), i.e. full corner number k = xc | (j << 1) (reading Q6).  Hashed level: slot =
// (XOR of g_d*pi_d) mod T (Eq. 8, uint32 wraparound, Q8/Q9); dense level: slot = sum of g_d*stride_d (Q10).
// D = 3 is G_3D of the decomposition stage (Eq. 3; Q26): 4 (y,z) corners.
template <int D = 4>
__device__ __forceinline__ void half_cell_slots(const Plan& P, const LevelParams& lp, const Query& q,
                                                uint32_t xc, uint32_t* __restrict__ slot) {
    constexpr int NC = 1 << (D - 1);
    const uint32_t ax = (q.c[0] + xc) * lp.m[0];
    const uint32_t ay0 = q.c[1] * lp.m[1], ay1 = ay0 + lp.m[1];
    const uint32_t az0 = q.c[2] * lp.m[2], az1 = az0 + lp.m[2];
    if (lp.dense) {
        const uint32_t p0 = ax + ay0, p1 = ax + ay1;
        if constexpr (D == 4) {
            const uint32_t at0 = q.c[3] * lp.m[3], at1 = at0 + lp.m[3];
            const uint32_t q0 = az0 + at0, q1 = az1 + at0, q2 = az0 + at1, q3 = az1 + at1;
            slot[0] = p0 + q0; slot[1] = p1 + q0; slot[2] = p0 + q1; slot[3] = p1 + q1;
            slot[4] = p0 + q2; slot[5] = p1 + q2; slot[6] = p0 + q3; slot[7] = p1 + q3;
        } else {
            slot[0] = p0 + az0; slot[1] = p1 + az0; slot[2] = p0 + az1; slot[3] = p1 + az1;
        }
    } else {
        const uint32_t p0 = ax ^ ay0, p1 = ax ^ ay1;
        if constexpr (D == 4) {
            const uint32_t at0 = q.c[3] * lp.m[3], at1 = at0 + lp.m[3];
            const uint32_t q0 = az0 ^ at0, q1 = az1 ^ at0, q2 = az0 ^ at1, q3 = az1 ^ at1;
            slot[0] = p0 ^ q0; slot[1] = p1 ^ q0; slot[2] = p0 ^ q1; slot[3] = p1 ^ q1;
            slot[4] = p0 ^ q2; slot[5] = p1 ^ q2; slot[6] = p0 ^ q3; slot[7] = p1 ^ q3;
        } else {
            slot[0] = p0 ^ az0; slot[1] = p1 ^ az0; slot[2] = p0 ^ az1; slot[3] = p1 ^ az1;
        }
        if (P.t_pow2) {
#pragma unroll
            for (int j = 0; j < NC; ++j) slot[j] &= P.t_mask;
        } else {
#pragma unroll
            for (int j = 0; j < NC; ++j) slot[j] %= P.T;
        }
    }
}

// multilinear weights: W = prod_d (corner bit ? w_d : 1 - w_d), fp32
template <int D = 4>
__device__ __forceinline__ void half_cell_weights(const Query& q, uint32_t xc, float* __restrict__ W) {
    const float wx = xc ? q.w[0] : 1.0f - q.w[0];
    const float py0 = wx * (1.0f - q.w[1]), py1 = wx * q.w[1];
    const float z0 = 1.0f - q.w[2], z1 = q.w[2];
    if constexpr (D == 4) {
        const float t0 = 1.0f - q.w[3], t1 = q.w[3];
        const float r0 = z0 * t0, r1 = z1 * t0, r2 = z0 * t1, r3 = z1 * t1;
        W[0] = py0 * r0; W[1] = py1 * r0; W[2] = py0 * r1; W[3] = py1 * r1;
        W[4] = py0 * r2; W[5] = py1 * r2; W[6] = py0 * r3; W[7] = py1 * r3;
    } else {
        W[0] = py0 * z0; W[1] = py1 * z0; W[2] = py0 * z1; W[3] = py1 * z1;
    }
}

template <int D = 4>
__device__ __forceinline__ void half_cell(const Plan& P, const LevelParams& lp, const Query& q,
                                          uint32_t xc, uint32_t* __restrict__ slot,
                                          float* __restrict__ W) {
    half_cell_slots<D>(P, lp, q, xc, slot);
    half_cell_weights<D>(q, xc, W);
}

// ------------------------------------------------------------------------------------------------
// Table slot access
// ------------------------------------------------------------------------------------------------

// 8-byte table gather: ld.global.nc with default L1 allocation.  Measured alternatives on C4/C3/C5
// (profiles/experiments_r02.md §9b, a round-1 record): L1::no_allocate +41 %/+12 %/+28 % time, ld.global.cg
// +3 %/+1 %/+5 %, L1::evict_last +-1 %.
__device__ __forceinline__ uint2 gather8(const void* p) { return __ldg(static_cast<const uint2*>(p)); }

template <int F, bool HALF>
__device__ __forceinline__ void load_slot(const void* __restrict__ level_base, uint32_t slot,
                                          float v[F]) {
    if constexpr (!HALF) {
        const float* p = static_cast<const float*>(level_base) + static_cast<size_t>(slot) * F;
        if constexpr (F == 1) {
            v[0] = __ldg(p);
        } else if constexpr (F == 2) {
            const uint2 raw = gather8(p);
            v[0] = __uint_as_float(raw.x); v[1] = __uint_as_float(raw.y);
        } else if constexpr (F == 4) {
            const float4 a = __ldg(reinterpret_cast<const float4*>(p));
            v[0] = a.x; v[1] = a.y; v[2] = a.z; v[3] = a.w;
        } else {
            const float4 a = __ldg(reinterpret_cast<const float4*>(p));
            const float4 b = __ldg(reinterpret_cast<const float4*>(p) + 1);
            v[0] = a.x; v[1] = a.y; v[2] = a.z; v[3] = a.w;
            v[4] = b.x; v[5] = b.y; v[6] = b.z; v[7] = b.w;
        }
    } else {  // IEEE half table, converted exactly to fp32 (reading Q13)
        const __half* p = static_cast<const __half*>(level_base) + static_cast<size_t>(slot) * F;
        if constexpr (F == 1) {
            const unsigned short raw = __ldg(reinterpret_cast<const unsigned short*>(p));
            v[0] = __half2float(__ushort_as_half(raw));
        } else if constexpr (F == 2) {
            const uint32_t raw = __ldg(reinterpret_cast<const uint32_t*>(p));
            const float2 a = __half22float2(*reinterpret_cast<const __half2*>(&raw));
            v[0] = a.x; v[1] = a.y;
        } else if constexpr (F == 4) {
            const uint2 raw = gather8(p);
            const float2 a = __half22float2(*reinterpret_cast<const __half2*>(&raw.x));
            const float2 b = __half22float2(*reinterpret_cast<const __half2*>(&raw.y));
            v[0] = a.x; v[1] = a.y; v[2] = b.x; v[3] = b.y;
        } else {
            const uint4 raw = __ldg(reinterpret_cast<const uint4*>(p));
            const float2 a = __half22float2(*reinterpret_cast<const __half2*>(&raw.x));
            const float2 b = __half22float2(*reinterpret_cast<const __half2*>(&raw.y));
            const float2 c = __half22float2(*reinterpret_cast<const __half2*>(&raw.z));
            const float2 d = __half22float2(*reinterpret_cast<const __half2*>(&raw.w));
            v[0] = a.x; v[1] = a.y; v[2] = b.x; v[3] = b.y;
            v[4] = c.x; v[5] = c.y; v[6] = d.x; v[7] = d.y;
        }
    }
}

// fp32 vector reduction at L2, no return value (REDG.E.ADD.F32x2 / .F32x4 on sm_100a).
template <int F>
__device__ __forceinline__ void red_add(float* p, const float v[F]) {
    if constexpr (F == 1) {
        asm volatile("red.global.add.f32 [%0], %1;" ::"l"(p), "f"(v[0]) : "memory");
    } else if constexpr (F == 2) {
        asm volatile("red.global.add.v2.f32 [%0], {%1, %2};" ::"l"(p), "f"(v[0]), "f"(v[1])
                     : "memory");
    } else if constexpr (F == 4) {
        asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(p), "f"(v[0]),
                     "f"(v[1]), "f"(v[2]), "f"(v[3])
                     : "memory");
    } else {
        asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(p), "f"(v[0]),
                     "f"(v[1]), "f"(v[2]), "f"(v[3])
                     : "memory");
        asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(p + 4), "f"(v[4]),
                     "f"(v[5]), "f"(v[6]), "f"(v[7])
                     : "memory");
    }
}

// The same reductions carrying an L2 eviction-priority hint (createpolicy): experiment of round 2 on keeping a level
// group's gradient slice resident against the streamed dout / coordinates.
__device__ __forceinline__ uint64_t l2_policy_evict_last() {
    uint64_t pol;
    asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(pol));
    return pol;
}

template <int F>
__device__ __forceinline__ void red_add_hint(float* p, const float v[F], uint64_t pol) {
    if constexpr (F == 1) {
        asm volatile("red.global.add.L2::cache_hint.f32 [%0], %1, %2;" ::"l"(p), "f"(v[0]), "l"(pol) : "memory");
    } else if constexpr (F == 2) {
        asm volatile("red.global.add.L2::cache_hint.v2.f32 [%0], {%1, %2}, %3;" ::"l"(p), "f"(v[0]), "f"(v[1]),
                     "l"(pol)
                     : "memory");
    } else {
#pragma unroll
        for (int h = 0; h < F / 4; ++h)
            asm volatile("red.global.add.L2::cache_hint.v4.f32 [%0], {%1, %2, %3, %4}, %5;" ::"l"(p + 4 * h),
                         "f"(v[4 * h]), "f"(v[4 * h + 1]), "f"(v[4 * h + 2]), "f"(v[4 * h + 3]), "l"(pol)
                         : "memory");
    }
}

}  // namespace
}  // namespace dash
