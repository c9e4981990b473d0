// bwd_runs_kernels.cu — the collision-aware scatter of the coarse levels (DASH_HASH4D_FLAG_SORT_COARSE):
// north_star's "sort-by-slot segmented reduction for the high-collision case" (BASELINE.json config 5; the gradient
// scatter is the transpose of Eq. 9).
//
// On the coarse levels many queries fall into the same 4D cell (C5 level 0: 853 contributions per slot on average),
// so most of their reductions can be merged before they leave the SM — but only when queries of one cell are
// processed one after the other.  Two steps:
//   1. a counting sort of the queries by the Morton code of their cell on the finest coarse level (keys + histogram,
//      3-launch scan, scatter of the query numbers AND of the packed coordinates, so that step 2 streams them);
//   2. hash4d_bwd_runs_kernel: a lane pair (the two x-corners, as everywhere in this library) walks a chunk of
//      consecutive SORTED queries on one level and keeps the 8 x F partial sums of the current cell in REGISTERS:
//      W_k * dY is added with an FMA as long as the cell stays the same, and the 8 vector reductions are issued once
//      per run of equal cells instead of once per query.  No shared-memory atomics (sm_100a has no native fp32 one),
//      no shuffles: a segmented reduction whose segments are the runs.
// The fine levels keep the one-reduction-per-corner kernel in the caller's query order (sorted order makes THAT
// kernel slower: profiles/experiments_r02.md §5).  Product code: shares nothing with oracle/.
#include <cuda_runtime.h>

#include "deform_kernels.h"   // count_launch, device_sm_count
#include "hash4d_device.cuh"
#include "hash4d_kernels.h"

namespace dash {

namespace {

// Morton code of (cx, cy, cz, ct): bit b of every axis that still has a bit b, b ascending, axis order x,y,z,t.
__device__ __forceinline__ uint32_t morton4(const uint32_t c[4], uint32_t bits_s, uint32_t bits_t) {
    uint32_t key = 0, pos = 0;
#pragma unroll
    for (uint32_t b = 0; b < 8; ++b) {
        if (b < bits_s) {
            key |= ((c[0] >> b) & 1u) << pos;
            key |= ((c[1] >> b) & 1u) << (pos + 1);
            key |= ((c[2] >> b) & 1u) << (pos + 2);
            pos += 3;
        }
        if (b < bits_t) {
            key |= ((c[3] >> b) & 1u) << pos;
            pos += 1;
        }
    }
    return key;
}

template <int D>
__device__ __forceinline__ uint32_t coarse_key(const Plan& P, const CoarseSort& cs, uint64_t n,
                                               const float* __restrict__ xyz, const float* __restrict__ t,
                                               const int32_t* __restrict__ index, float4& coords) {
    float c[4];
    load_coords<D>(P, n, xyz, t, index, c);   // D = 3 (G_3D): no timestamp, c[3] = 0, bits_t = 0
    coords = make_float4(c[0], c[1], c[2], c[3]);
    const LevelParams& lp = P.lv[cs.key_level];
    uint32_t cell[4];
    float frac;
    locate(c[0], lp.ns_f, cell[0], frac);
    locate(c[1], lp.ns_f, cell[1], frac);
    locate(c[2], lp.ns_f, cell[2], frac);
    locate(c[3], lp.nt_f, cell[3], frac);
    cell[0] >>= cs.shift_s; cell[1] >>= cs.shift_s; cell[2] >>= cs.shift_s; cell[3] >>= cs.shift_t;
    return morton4(cell, cs.bits_s, cs.bits_t);
}

template <int D>
__global__ void __launch_bounds__(kBlockThreads)
sort4d_keys_kernel(const __grid_constant__ Plan P, const CoarseSort cs, const float* __restrict__ xyz,
                   const float* __restrict__ t, const int32_t* __restrict__ index, uint32_t* __restrict__ keys,
                   uint32_t* __restrict__ hist) {
    const size_t stride = static_cast<size_t>(gridDim.x) * kBlockThreads;
    for (uint64_t n = static_cast<uint64_t>(blockIdx.x) * kBlockThreads + threadIdx.x; n < P.N; n += stride) {
        float4 q;
        const uint32_t key = coarse_key<D>(P, cs, n, xyz, t, index, q);
        keys[n] = key;
        atomicAdd(hist + key, 1u);
    }
}

// order[pos] = n and sorted_q[pos] = (x, y, z, t) of query n: the run kernel streams both
template <int D>
__global__ void __launch_bounds__(kBlockThreads)
sort4d_scatter_kernel(const __grid_constant__ Plan P, const float* __restrict__ xyz, const float* __restrict__ t,
                      const int32_t* __restrict__ index, const uint32_t* __restrict__ keys,
                      uint32_t* __restrict__ cursor, const uint32_t* __restrict__ tile_offset,
                      int32_t* __restrict__ order, float4* __restrict__ sorted_q, WorkspaceHeader* __restrict__ hdr,
                      const OrderStamp stamp) {
    if (blockIdx.x == 0 && threadIdx.x < 12) hdr->order_stamp.w[threadIdx.x] = stamp.w[threadIdx.x];
    const size_t stride = static_cast<size_t>(gridDim.x) * kBlockThreads;
    for (uint64_t n = static_cast<uint64_t>(blockIdx.x) * kBlockThreads + threadIdx.x; n < P.N; n += stride) {
        float c[4];
        load_coords<D>(P, n, xyz, t, index, c);
        const uint32_t key = keys[n];   // the scan is per tile of kScanTile bins: add the tile's offset here
        const uint32_t pos = atomicAdd(cursor + key, 1u) + __ldg(tile_offset + key / kScanTile);
        order[pos] = static_cast<int32_t>(n);
        sorted_q[pos] = make_float4(c[0], c[1], c[2], c[3]);
    }
}

template <int F>
__device__ __forceinline__ void load_row(const float* __restrict__ d, float g[F]) {
    if constexpr (F == 1) {
        g[0] = __ldg(d);
    } else if constexpr (F == 2) {
        const float2 a = __ldg(reinterpret_cast<const float2*>(d));
        g[0] = a.x; g[1] = a.y;
    } else {
#pragma unroll
        for (int h = 0; h < F / 4; ++h) {
            const float4 a = __ldg(reinterpret_cast<const float4*>(d) + h);
            g[4 * h] = a.x; g[4 * h + 1] = a.y; g[4 * h + 2] = a.z; g[4 * h + 3] = a.w;
        }
    }
}

// One run of equal cells is closed: one vector reduction per corner slot.
template <int F, bool HINT, int NC>
__device__ __forceinline__ void flush_run(const uint32_t slot[NC], float* __restrict__ level_base,
                                          const float acc[NC][F], uint64_t pol) {
#pragma unroll
    for (int j = 0; j < NC; ++j) {
        if constexpr (HINT) red_add_hint<F>(level_base + static_cast<size_t>(slot[j]) * F, acc[j], pol);
        else red_add<F>(level_base + static_cast<size_t>(slot[j]) * F, acc[j]);
    }
}

// One lane pair = (chunk of `chunk` consecutive sorted queries, one coarse level); adjacent pairs take the coarse
// levels of the SAME chunk, so their coordinate loads coincide and their dY loads are neighbours in one row.
// N < 2^31 here (the order is an int32 list): positions are 32-bit.
// D = 3: G_3D (dash_hash3d_bwd), 4 (y,z) corners per lane.
template <int F, bool HINT, int D>
__global__ void __launch_bounds__(kBlockThreads, F >= 8 ? 1 : (F == 4 ? 3 : 4))   // F = 4: 80 registers, three CTAs per SM; F <= 2: 64, four
hash4d_bwd_runs_kernel(const __grid_constant__ Plan P, const uint32_t levels, const uint32_t chunk,
                       const float4* __restrict__ sorted_q, const int32_t* __restrict__ order,
                       const float* __restrict__ dout, float* __restrict__ dtable) {
    const uint32_t xc = threadIdx.x & 1u;
    const uint64_t pair = (static_cast<uint64_t>(blockIdx.x) * kBlockThreads + threadIdx.x) >> 1;
    const uint64_t ch = pair / levels;
    const uint32_t l = static_cast<uint32_t>(pair - ch * levels);
    const uint32_t n_total = static_cast<uint32_t>(P.N);
    if (ch * chunk >= n_total) return;
    const uint32_t begin = static_cast<uint32_t>(ch * chunk);
    const uint32_t end = (n_total - begin > chunk) ? begin + chunk : n_total;
    const LevelParams lp = P.lv[l];
    const uint32_t row = P.L * F;
    const float* dcol = dout + static_cast<size_t>(l) * F;
    float* level_base = dtable + static_cast<size_t>(l) * P.T * F;
    uint64_t pol = 0;
    if constexpr (HINT) pol = l2_policy_evict_last();

    constexpr int NC = 1 << (D - 1);
    float acc[NC][F];
    uint32_t slot[NC];
#pragma unroll
    for (int j = 0; j < NC; ++j) slot[j] = 0u;
    uint32_t pc[4] = {0xffffffffu, 0xffffffffu, 0xffffffffu, 0xffffffffu};  // no cell: the first query opens a run
#pragma unroll
    for (int j = 0; j < NC; ++j)
#pragma unroll
        for (int f = 0; f < F; ++f) acc[j][f] = 0.0f;
    // two-deep software pipeline: coordinates and dY of query s+1 and the query number of s+2 are in flight
    // while query s is accumulated
    const uint32_t n_max = n_total - 1u;   // clamped: memory-safe even if ORDER_READY was a false claim
    float4 q_next = __ldg(sorted_q + begin);
    float g_next[F];
    load_row<F>(dcol + static_cast<size_t>(min(static_cast<uint32_t>(__ldg(order + begin)), n_max)) * row, g_next);
    uint32_t n_ahead = (begin + 1 < end) ? min(static_cast<uint32_t>(__ldg(order + begin + 1)), n_max) : 0u;
#pragma unroll 1
    for (uint32_t s = begin; s < end; ++s) {
        const float4 qc = q_next;
        float g[F];
#pragma unroll
        for (int f = 0; f < F; ++f) g[f] = g_next[f];
        if (s + 1 < end) {
            q_next = __ldg(sorted_q + s + 1);
            load_row<F>(dcol + static_cast<size_t>(n_ahead) * row, g_next);
            if (s + 2 < end) n_ahead = min(static_cast<uint32_t>(__ldg(order + s + 2)), n_max);
        }
        const Query q = make_query<D>(lp, qc.x, qc.y, qc.z, qc.w);
        if ((q.c[0] != pc[0]) | (q.c[1] != pc[1]) | (q.c[2] != pc[2]) | (q.c[3] != pc[3])) {
            if (pc[0] != 0xffffffffu) flush_run<F, HINT, NC>(slot, level_base, acc, pol);
            half_cell_slots<D>(P, lp, q, xc, slot);
#pragma unroll
            for (int d = 0; d < 4; ++d) pc[d] = q.c[d];
#pragma unroll
            for (int j = 0; j < NC; ++j)
#pragma unroll
                for (int f = 0; f < F; ++f) acc[j][f] = 0.0f;
        }
        float W[NC];
        half_cell_weights<D>(q, xc, W);
#pragma unroll
        for (int j = 0; j < NC; ++j)
#pragma unroll
            for (int f = 0; f < F; ++f) acc[j][f] = fmaf(W[j], g[f], acc[j][f]);
    }
    flush_run<F, HINT, NC>(slot, level_base, acc, pol);
}

inline cudaError_t launched() {
    count_launch();
    return cudaGetLastError();
}

}  // namespace

cudaError_t launch_coarse_sort(const Plan& P, const CoarseSort& cs, const float* xyz, const float* t,
                               const int32_t* index, int32_t* order, float4* sorted_q, uint32_t* keys, uint32_t* bins,
                               uint32_t* totals, cudaStream_t s, WorkspaceHeader* hdr, const OrderStamp& stamp) {
    const size_t want = (P.N + kBlockThreads - 1) / kBlockThreads;
    const size_t cap = static_cast<size_t>(device_sm_count()) * 16;
    const unsigned blocks = static_cast<unsigned>(want < 1 ? 1 : (want > cap ? cap : want));
    cudaError_t e = launch_zero(bins, static_cast<size_t>(cs.n_bins) * sizeof(uint32_t), s);
    if (e != cudaSuccess) return e;
    if (P.dims == 3) sort4d_keys_kernel<3><<<blocks, kBlockThreads, 0, s>>>(P, cs, xyz, t, index, keys, bins);
    else sort4d_keys_kernel<4><<<blocks, kBlockThreads, 0, s>>>(P, cs, xyz, t, index, keys, bins);
    if ((e = launched()) != cudaSuccess) return e;
    if ((e = launch_exclusive_scan_u32(bins, cs.n_bins, totals, s, false)) != cudaSuccess) return e;
    if (P.dims == 3)
        sort4d_scatter_kernel<3><<<blocks, kBlockThreads, 0, s>>>(P, xyz, t, index, keys, bins, totals, order, sorted_q, hdr,
                                                                  stamp);
    else
        sort4d_scatter_kernel<4><<<blocks, kBlockThreads, 0, s>>>(P, xyz, t, index, keys, bins, totals, order, sorted_q, hdr,
                                                                  stamp);
    return launched();
}

cudaError_t launch_bwd_runs(const Plan& P, const CoarseSort& cs, const float* dout, float* dtable, const int32_t* order,
                            const float4* sorted_q, cudaStream_t s, bool l2_hint) {
    const uint64_t chunks = (P.N + cs.chunk - 1) / cs.chunk;
    const uint64_t threads = chunks * cs.levels * 2;
    const uint64_t grid = (threads + kBlockThreads - 1) / kBlockThreads;
    if (grid > 0x7fffffffull) return cudaErrorInvalidValue;
#define DASH_RUNS_D(FV, HV, DV)                                                                         \
    hash4d_bwd_runs_kernel<FV, HV, DV><<<static_cast<unsigned>(grid), kBlockThreads, 0, s>>>(           \
        P, cs.levels, cs.chunk, sorted_q, order, dout, dtable)
#define DASH_RUNS(FV)                                        \
    do {                                                     \
        if (P.dims == 3) {                                   \
            if (l2_hint) DASH_RUNS_D(FV, true, 3);           \
            else DASH_RUNS_D(FV, false, 3);                  \
        } else {                                             \
            if (l2_hint) DASH_RUNS_D(FV, true, 4);           \
            else DASH_RUNS_D(FV, false, 4);                  \
        }                                                    \
    } while (0)
    switch (P.F) {
        case 1: DASH_RUNS(1); break;
        case 2: DASH_RUNS(2); break;
        case 4: DASH_RUNS(4); break;
        case 8: DASH_RUNS(8); break;
        default: return cudaErrorInvalidValue;
    }
#undef DASH_RUNS
#undef DASH_RUNS_D
    return launched();
}

}  // namespace dash
