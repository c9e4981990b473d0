// hash4d_api.cu — C ABI (include/dash_hash4d.h) and host-side scheduler of the 4D hash encoder.
//
// Host work per call: validate, evaluate Eq. 7 once, decide dense vs hashed per
// level (reading Q10), pick the level-group size G from the L2 capacity, launch.  No allocation,
// no synchronisation (except VALIDATE_INPUTS), no state kept between calls.
#include <cuda_runtime.h>

#include <atomic>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>

#include "../../include/dash_debug.h"
#include "../../include/dash_deform.h"
#include "../../include/dash_hash4d.h"
#include "api_errors.h"
#include "deform_kernels.h"
#include "hash4d_kernels.h"
#include "hash4d_plan.h"

namespace {

using dash::Plan;
using dash::WorkspaceHeader;

thread_local char g_error[512] = "";

int fail(int code, const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_error, sizeof(g_error), fmt, ap);
    va_end(ap);
    return code;
}

int ok() {
    g_error[0] = '\0';
    return DASH_HASH4D_OK;
}

const uint32_t kDefaultPrimes[4] = {1u, 2654435761u, 805459861u, 3674653429u};  // reading Q7
constexpr uint32_t kMaxResolution = 1u << 22;
constexpr size_t kHeaderBytes = sizeof(WorkspaceHeader);

int check_config(const dash_hash4d_config* c, int dims = 4) {
    if (!c) return fail(DASH_HASH4D_INVALID_ARG, "config is NULL");
    if (c->struct_size != sizeof(dash_hash4d_config))
        return fail(DASH_HASH4D_INVALID_ARG, "struct_size %u != %zu", c->struct_size,
                    sizeof(dash_hash4d_config));
    if (c->L < 1 || c->L > dash::kMaxLevels)
        return fail(DASH_HASH4D_INVALID_ARG, "L = %u outside 1..%d", c->L, dash::kMaxLevels);
    if (c->F == 0 || c->F > 8) return fail(DASH_HASH4D_INVALID_ARG, "F = %u outside 1..8", c->F);
    if (!(c->F == 1 || c->F == 2 || c->F == 4 || c->F == 8))
        return fail(DASH_HASH4D_UNSUPPORTED, "F = %u not in {1,2,4,8}", c->F);
    if (c->T < 1) return fail(DASH_HASH4D_INVALID_ARG, "T = 0");
    if (c->res_s_min < 1 || c->res_s_min > c->res_s_max || c->res_s_max > kMaxResolution)
        return fail(DASH_HASH4D_INVALID_ARG, "spatial resolution range [%u, %u] invalid",
                    c->res_s_min, c->res_s_max);
    if (dims == 4 && (c->res_t_min < 1 || c->res_t_min > c->res_t_max || c->res_t_max > kMaxResolution))
        return fail(DASH_HASH4D_INVALID_ARG, "temporal resolution range [%u, %u] invalid",
                    c->res_t_min, c->res_t_max);
    if (c->table_dtype != DASH_HASH4D_FP32 && c->table_dtype != DASH_HASH4D_FP16)
        return fail(DASH_HASH4D_INVALID_ARG, "table_dtype = %u", c->table_dtype);
    if (c->flags & ~63u) return fail(DASH_HASH4D_INVALID_ARG, "unknown flag bits 0x%x", c->flags);
    return DASH_HASH4D_OK;
}

// Eq. 7 with the exponent restored (reading Q1): N_l = floor(N_min * (N_max/N_min)^(l/(L-1))).
// Reading Q2: IEEE double, +1e-6 before the floor so mathematically-integer levels are not lost.
uint32_t geometric_level(uint32_t lo, uint32_t hi, uint32_t l, uint32_t L) {
    if (L == 1) return lo;
    const double ratio = static_cast<double>(hi) / static_cast<double>(lo);
    const double expo = static_cast<double>(l) / static_cast<double>(L - 1);
    return static_cast<uint32_t>(std::floor(static_cast<double>(lo) * std::pow(ratio, expo) + 1e-6));
}

bool fits_dense(uint32_t ns, uint32_t nt, uint32_t T) {  // (Ns+1)^3 (Nt+1) <= T, in 128-bit-safe steps
    const unsigned long long S = static_cast<unsigned long long>(ns) + 1ull;
    unsigned long long v = S * S;               // <= 2^46
    if (v > T) return false;
    v *= S;                                      // v <= T * S < 2^55
    if (v > T) return false;
    v *= static_cast<unsigned long long>(nt) + 1ull;
    return v <= T;
}

bool fits_dense3(uint32_t ns, uint32_t T) {  // (Ns+1)^3 <= T: the d = 3 form of reading Q10 (Q26)
    const unsigned long long S = static_cast<unsigned long long>(ns) + 1ull;
    const unsigned long long v = S * S;
    return v <= T && v * S <= T;
}

struct Schedule {
    uint32_t res_s[dash::kMaxLevels], res_t[dash::kMaxLevels];
    uint8_t dense[dash::kMaxLevels];
};

void make_schedule(const dash_hash4d_config* c, Schedule* s, int dims = 4) {
    for (uint32_t l = 0; l < c->L; ++l) {
        s->res_s[l] = geometric_level(c->res_s_min, c->res_s_max, l, c->L);
        s->res_t[l] = dims == 4 ? geometric_level(c->res_t_min, c->res_t_max, l, c->L) : 1u;
        s->dense[l] = (c->flags & DASH_HASH4D_FLAG_DENSE_COARSE) &&
                      (dims == 4 ? fits_dense(s->res_s[l], s->res_t[l], c->T)
                                 : fits_dense3(s->res_s[l], c->T));
    }
}

size_t l2_bytes() { return dash::device_l2_bytes(); }  // current device, cached per ordinal

// Tuning overrides for sweeps (dash_hash4d_set_debug): process-wide, 0 = the library decides.  No environment
// variable is ever read.
std::atomic<int64_t> g_debug[DASH_DEBUG_KEY_COUNT];

uint32_t debug_u32(int key) { return static_cast<uint32_t>(g_debug[key].load(std::memory_order_relaxed)); }

// Level-group size G (power of two <= 8): as many levels as keep the group's randomly accessed
// bytes (tables in fwd, fp32 gradient slices in bwd) within 0.3 x L2 — measured (profiles/
// group_sweep_r02.md): B200's 126 MB L2 is two 63 MB halves and read-only lines are replicated in
// both, so ~40 MB is what stays resident next to the streamed inputs/outputs — but at least enough
// that a query's slice of `out`/`dout` is one full 32-byte sector (G*F*4 >= 32), and without idling
// more than a quarter of the lanes when L is not a multiple of G.  G = 16 (one query per warp) is
// never picked: every warp would then run both the dense and the hashed index path (measured 7-12 %
// slower than G = 8 at F = 2).  dash_hash4d_set_debug(DASH_DEBUG_{FWD,BWD,SMOOTH}_GROUP, G) overrides G (1..16).
uint32_t pick_group(const dash_hash4d_config* c, size_t bytes_per_level, int debug_key,
                    bool row_sector_rule = true) {
    uint32_t forced = debug_u32(debug_key);
    if (forced) {
        uint32_t g = 1;
        while (g * 2 <= forced && g * 2 <= dash::kMaxGroup) g *= 2;
        return g;
    }
    const size_t budget = l2_bytes() * 3 / 10;
    uint32_t g_min = 1;
    while (row_sector_rule && g_min * c->F * 4 < 32 && g_min < dash::kMaxGroup) g_min *= 2;
    uint32_t best = 0;
    for (uint32_t g = dash::kMaxGroup / 2; g >= 1; g /= 2) {
        const uint32_t groups = (c->L + g - 1) / g;
        const bool efficient = 4 * c->L >= 3 * groups * g;
        const bool resident = g * bytes_per_level <= budget;
        if (efficient && (resident || g <= g_min)) {
            best = g;
            break;
        }
    }
    return best ? best : 1;
}

int fill_plan(const dash_hash4d_config* c, uint64_t N, uint32_t xyz_stride, uint32_t t_stride,
              uint32_t group, Plan* P, int dims = 4) {
    Schedule s;
    make_schedule(c, &s, dims);
    std::memset(P, 0, sizeof(*P));
    P->dims = static_cast<uint32_t>(dims);
    P->N = N;
    P->L = c->L;
    P->F = c->F;
    P->T = c->T;
    P->t_pow2 = (c->T & (c->T - 1)) == 0;
    P->t_mask = c->T - 1;
    P->xyz_stride = xyz_stride;
    P->t_stride = t_stride;
    P->group = group;
    uint32_t lg = 0;
    while ((1u << lg) < group) ++lg;
    P->group_log2 = lg;
    P->level_begin = 0;
    P->level_end = c->L;
    P->num_groups = (c->L + group - 1) / group;
    P->q_per_block = dash::kItemsPerBlock >> lg;
    const bool defaults = !(c->primes[0] | c->primes[1] | c->primes[2] | c->primes[3]);
    for (uint32_t l = 0; l < c->L; ++l) {
        dash::LevelParams& lp = P->lv[l];
        lp.ns_f = static_cast<float>(s.res_s[l]);
        lp.nt_f = static_cast<float>(s.res_t[l]);
        lp.dense = s.dense[l];
        if (s.dense[l]) {
            const uint32_t S = s.res_s[l] + 1;
            lp.m[0] = 1;
            lp.m[1] = S;
            lp.m[2] = S * S;
            lp.m[3] = dims == 4 ? S * S * S : 0u;
        } else {
            for (int d = 0; d < 4; ++d) lp.m[d] = defaults ? kDefaultPrimes[d] : c->primes[d];
        }
    }
    if (N) {
        const uint64_t tiles = (N + P->q_per_block - 1) / P->q_per_block;
        if (tiles > 0x7fffffffull)
            return fail(DASH_HASH4D_UNSUPPORTED, "N = %llu too large for one launch",
                        static_cast<unsigned long long>(N));
    }
    return DASH_HASH4D_OK;
}

int check_queries(const float* xyz, uint32_t xyz_stride, const float* t, uint32_t t_stride,
                  const int32_t* index, int dims = 4) {
    if (!xyz || (dims == 4 && !t)) return fail(DASH_HASH4D_INVALID_ARG, "xyz or t is NULL");
    if (!(xyz_stride == 3 || xyz_stride == 4))
        return fail(DASH_HASH4D_INVALID_ARG, "xyz_stride = %u (want 3 or 4)", xyz_stride);
    if (!(t_stride == 0 || t_stride == 1 || t_stride == 4))
        return fail(DASH_HASH4D_INVALID_ARG, "t_stride = %u (want 0, 1 or 4)", t_stride);
    if ((reinterpret_cast<uintptr_t>(xyz) | reinterpret_cast<uintptr_t>(t) |
         reinterpret_cast<uintptr_t>(index)) & 3u)
        return fail(DASH_HASH4D_INVALID_ARG, "xyz / t / index not 4-byte aligned");
    return DASH_HASH4D_OK;
}

bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

int cuda_fail(cudaError_t e, const char* what) {
    return fail(DASH_HASH4D_CUDA_ERROR, "%s: %s", what, cudaGetErrorString(e));
}

size_t table_elems(const dash_hash4d_config* c) {
    return static_cast<size_t>(c->L) * c->T * c->F;
}

int run_validation(const dash_hash4d_config* c, const Plan& P, const float* xyz, const float* t,
                   const int32_t* index, void* workspace, size_t workspace_bytes, cudaStream_t s) {
    if (!(c->flags & DASH_HASH4D_FLAG_VALIDATE_INPUTS)) return DASH_HASH4D_OK;
    if (!workspace || workspace_bytes < kHeaderBytes)
        return fail(DASH_HASH4D_WORKSPACE_TOO_SMALL, "VALIDATE_INPUTS needs %zu workspace bytes",
                    kHeaderBytes);
    WorkspaceHeader* hdr = static_cast<WorkspaceHeader*>(workspace);
    cudaError_t e = dash::launch_zero(hdr, dash::kHeaderScratchBytes, s);   // not the order stamp behind it
    if (e == cudaSuccess) e = dash::launch_validate(P, xyz, t, index, hdr, s);
    if (e != cudaSuccess) return cuda_fail(e, "validate launch");
    uint32_t bad = 0;
    e = cudaMemcpyAsync(&bad, &hdr->bad_inputs, sizeof(bad), cudaMemcpyDeviceToHost, s);
    if (e == cudaSuccess) e = cudaStreamSynchronize(s);
    if (e != cudaSuccess) return cuda_fail(e, "validate readback");
    if (bad)
        return fail(DASH_HASH4D_INVALID_ARG, "%u coordinates are NaN or outside [0,1)", bad);
    return DASH_HASH4D_OK;
}

}  // namespace

namespace dash {  // api_errors.h: the same channel for the other translation units

int api_fail(int code, const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_error, sizeof(g_error), fmt, ap);
    va_end(ap);
    return code;
}
int api_cuda_fail(cudaError_t e, const char* what) { return cuda_fail(e, what); }
int api_ok() { return ok(); }

}  // namespace dash

extern "C" {

DASH_API const char* dash_hash4d_last_error(void) { return g_error; }

#ifndef DASH_BUILD_ID_STRING
#define DASH_BUILD_ID_STRING "unknown"
#endif
// hash of the sources this library was built from (paper_2507_19141_b200/build.py); the binding refuses a
// library whose id differs from the sources beside it
DASH_API const char* dash_hash4d_build_id(void) {
    static const char id[] = "DASH_BUILD_ID=" DASH_BUILD_ID_STRING;
    return id + 14;
}

DASH_API uint64_t dash_hash4d_launch_count(int reset) { return dash::launch_counter(reset != 0); }

DASH_API int dash_hash4d_set_debug(int key, int64_t value) {
    if (key < 0 || key >= DASH_DEBUG_KEY_COUNT) return fail(DASH_HASH4D_INVALID_ARG, "debug key %d unknown", key);
    if (value < 0) return fail(DASH_HASH4D_INVALID_ARG, "debug value must be >= 0");
    g_debug[key].store(value, std::memory_order_relaxed);
    return ok();
}

DASH_API int dash_hash4d_resolutions(const dash_hash4d_config* cfg, uint32_t* res_s,
                                     uint32_t* res_t, uint8_t* is_dense) {
    if (int rc = check_config(cfg)) return rc;
    if (!res_s || !res_t) return fail(DASH_HASH4D_INVALID_ARG, "res_s or res_t is NULL");
    Schedule s;
    make_schedule(cfg, &s);
    for (uint32_t l = 0; l < cfg->L; ++l) {
        res_s[l] = s.res_s[l];
        res_t[l] = s.res_t[l];
        if (is_dense) is_dense[l] = s.dense[l];
    }
    return ok();
}

static size_t round16(size_t v) { return (v + 15u) & ~static_cast<size_t>(15u); }

// DASH_HASH4D_FLAG_SORT_COARSE: which leading levels the run-merged scatter takes and how the queries are keyed.
// Levels whose cell count Ns^3 Nt is at most 2N (on average >= 1/2 query per cell; clustered inputs fill far fewer
// cells) — measured rule, profiles/experiments_r02.md §8.  The key is the Morton code of the cell on the finest of
// them, coarsened until it has at most 22 bits.  DASH_DEBUG_BWD_COARSE_LEVELS / _RUN_CHUNK override for sweeps.
static bool plan_coarse(const dash_hash4d_config* c, uint64_t N, dash::CoarseSort* cs, int dims = 4) {
    std::memset(cs, 0, sizeof(*cs));
    if (!(c->flags & DASH_HASH4D_FLAG_SORT_COARSE) || (c->flags & DASH_HASH4D_FLAG_DETERMINISTIC_BWD) || N == 0 ||
        N > 0x7fffffffull)   // the order is an int32 list
        return false;
    Schedule s;
    make_schedule(c, &s, dims);   // dims = 3 (G_3D): res_t = 1 on every level, the key has no t bits
    uint32_t nl = 0;
    const uint32_t forced = debug_u32(DASH_DEBUG_BWD_COARSE_LEVELS);
    if (forced) {
        nl = forced < c->L ? forced : c->L;
    } else if (N * c->F >= (1ull << 21)) {
        // below that the sort costs more than it saves: measured crossover ~350k queries at F = 4 (C4's encoder), ~750k at
        // F = 2 (C3's encoder; C3 itself, 300k: +8 %) — profiles/experiments_r02.md §8
        while (nl < c->L && nl < 8) {
            const double cells = static_cast<double>(s.res_s[nl]) * s.res_s[nl] * s.res_s[nl] * s.res_t[nl];
            if (cells > 2.0 * static_cast<double>(N)) break;
            ++nl;
        }
    }
    if (nl == 0) return false;
    cs->levels = nl;
    cs->key_level = nl - 1;
    auto ceil_log2 = [](uint32_t v) { uint32_t b = 0; while ((1ull << b) < v) ++b; return b; };
    uint32_t bs = ceil_log2(s.res_s[nl - 1]), bt = ceil_log2(s.res_t[nl - 1]);
    uint32_t max_bits = debug_u32(DASH_DEBUG_SORT_KEY_BITS);
    max_bits = max_bits ? (max_bits < 8 ? 8u : (max_bits > 22 ? 22u : max_bits)) : 22u;
    while (3 * (bs - cs->shift_s) + (bt - cs->shift_t) > max_bits || bs - cs->shift_s > 7 || bt - cs->shift_t > 7) {
        if (bt - cs->shift_t > bs - cs->shift_s) ++cs->shift_t; else ++cs->shift_s;
    }
    cs->bits_s = bs - cs->shift_s;
    cs->bits_t = bt - cs->shift_t;
    cs->n_bins = 1u << (3 * cs->bits_s + cs->bits_t);
    // The forward walks EVERY level in the sorted order: neighbouring lanes share cells and lines well past the levels
    // whose reductions merge (C4, key 48 per axis: levels of 16-48 per axis -40 %, 70-101 -38 %, 147-212 -21 %, finer
    // ones -3 %), and one launch over all levels beats any split (profiles/experiments_r02.md §8).
    const uint32_t forced_fwd = debug_u32(DASH_DEBUG_FWD_ORDERED_LEVELS);
    cs->levels_fwd = forced_fwd ? (forced_fwd < c->L ? forced_fwd : c->L) : c->L;
    const uint32_t chunk = debug_u32(DASH_DEBUG_BWD_RUN_CHUNK);
    cs->chunk = chunk ? chunk : 32u;   // 24-48 measure alike (C4, C5); 8 and 128 lose 1-3 %
    return true;
}

static size_t coarse_workspace(const dash::CoarseSort& cs, uint64_t N) {
    return round16(N * 4) * 2 + round16(N * 16) + round16(static_cast<size_t>(cs.n_bins) * 4) +
           round16((static_cast<size_t>(cs.n_bins) + 1023) / 1024 * 4);
}

struct CoarseBuffers {
    int32_t* order;
    uint32_t* keys;
    float4* sorted_q;
    uint32_t* bins;
    uint32_t* totals;
};

static CoarseBuffers carve_coarse(void* workspace, const dash::CoarseSort& cs, uint64_t N) {
    char* w = static_cast<char*>(workspace) + kHeaderBytes;
    CoarseBuffers b;
    b.order = reinterpret_cast<int32_t*>(w);
    b.keys = reinterpret_cast<uint32_t*>(w + round16(N * 4));
    b.sorted_q = reinterpret_cast<float4*>(w + 2 * round16(N * 4));
    b.bins = reinterpret_cast<uint32_t*>(w + 2 * round16(N * 4) + round16(N * 16));
    b.totals = b.bins + round16(static_cast<size_t>(cs.n_bins) * 4) / 4;
    return b;
}

// What identifies the queries and the key an order was computed for.  The sort writes it behind the order; a later
// ORDER_READY call can compare it (verify_order).
static dash::OrderStamp order_stamp(const Plan& P, const dash::CoarseSort& cs, const float* xyz, const float* t,
                                    const int32_t* index) {
    dash::OrderStamp st;
    const uint64_t px = reinterpret_cast<uintptr_t>(xyz), pt = reinterpret_cast<uintptr_t>(t),
                   pi = reinterpret_cast<uintptr_t>(index);
    st.w[0] = 0x44415348u;   // "DASH": a workspace that no sort has written never matches
    st.w[1] = static_cast<uint32_t>(P.N);
    st.w[2] = static_cast<uint32_t>(P.N >> 32);
    st.w[3] = P.dims | (P.xyz_stride << 8) | (P.t_stride << 16);
    st.w[4] = cs.key_level | (cs.bits_s << 8) | (cs.bits_t << 16);
    st.w[5] = cs.shift_s | (cs.shift_t << 8);
    st.w[6] = static_cast<uint32_t>(px); st.w[7] = static_cast<uint32_t>(px >> 32);
    st.w[8] = static_cast<uint32_t>(pt); st.w[9] = static_cast<uint32_t>(pt >> 32);
    st.w[10] = static_cast<uint32_t>(pi); st.w[11] = static_cast<uint32_t>(pi >> 32);
    return st;
}

// ORDER_READY is a promise the library cannot check without reading the workspace back.  Under VALIDATE_INPUTS, which
// synchronises the stream anyway, it does: the stamp the sort left must be the one this call would write.
static int verify_order(const dash_hash4d_config* cfg, const Plan& P, const dash::CoarseSort& cs, const float* xyz,
                        const float* t, const int32_t* index, void* workspace, cudaStream_t s) {
    constexpr uint32_t kBoth = DASH_HASH4D_FLAG_ORDER_READY | DASH_HASH4D_FLAG_VALIDATE_INPUTS;
    if ((cfg->flags & kBoth) != kBoth) return DASH_HASH4D_OK;
    dash::OrderStamp got;
    cudaError_t e = cudaMemcpyAsync(&got, &static_cast<WorkspaceHeader*>(workspace)->order_stamp, sizeof(got),
                                    cudaMemcpyDeviceToHost, s);
    if (e == cudaSuccess) e = cudaStreamSynchronize(s);
    if (e != cudaSuccess) return cuda_fail(e, "ORDER_READY stamp readback");
    const dash::OrderStamp want = order_stamp(P, cs, xyz, t, index);
    if (std::memcmp(&got, &want, sizeof(want)) != 0)
        return fail(DASH_HASH4D_INVALID_ARG, "ORDER_READY: the workspace does not hold an order for these queries (%s)",
                    got.w[0] != want.w[0] ? "no SORT_COARSE call has sorted into it" :
                    (got.w[1] != want.w[1] || got.w[2] != want.w[2]) ? "it was computed for a different N" :
                    std::memcmp(&got.w[6], &want.w[6], 24) != 0 ? "xyz, t or index pointer differs" :
                    "strides or sort key differ");
    return DASH_HASH4D_OK;
}

static size_t workspace_need(const dash_hash4d_config* cfg, int op, uint64_t N, int dims = 4) {
    size_t bytes = 0;
    if ((cfg->flags & DASH_HASH4D_FLAG_VALIDATE_INPUTS) && op != DASH_HASH4D_OP_INDICES)
        bytes = kHeaderBytes;
    if (op == DASH_HASH4D_OP_BWD && (cfg->flags & DASH_HASH4D_FLAG_DETERMINISTIC_BWD))
        bytes = kHeaderBytes + table_elems(cfg) * sizeof(long long);
    dash::CoarseSort cs;
    if ((op == DASH_HASH4D_OP_BWD || op == DASH_HASH4D_OP_FWD || op == DASH_HASH4D_OP_BWD_INPUT) &&
        plan_coarse(cfg, N, &cs, dims))
        bytes = kHeaderBytes + coarse_workspace(cs, N);
    return bytes;
}

DASH_API size_t dash_hash4d_workspace_bytes(const dash_hash4d_config* cfg, uint64_t N, int op) {
    if (check_config(cfg, 4)) return 0;
    g_error[0] = '\0';
    return workspace_need(cfg, op, N, 4);
}

DASH_API size_t dash_hash3d_workspace_bytes(const dash_hash4d_config* cfg, uint64_t N, int op) {
    if (check_config(cfg, 3)) return 0;  // the temporal fields are ignored
    g_error[0] = '\0';
    return workspace_need(cfg, op, N, 3);
}

static int fwd_impl(int dims, const dash_hash4d_config* cfg, uint64_t N, const float* xyz,
                    uint32_t xyz_stride, const float* t, uint32_t t_stride, const int32_t* index,
                    const void* table, float* out, void* workspace, size_t workspace_bytes,
                    void* cuda_stream) {
    if (int rc = check_config(cfg, dims)) return rc;
    if (N == 0) return ok();
    if (int rc = check_queries(xyz, xyz_stride, t, t_stride, index, dims)) return rc;
    if (!table || !out) return fail(DASH_HASH4D_INVALID_ARG, "table or out is NULL");
    if (!aligned16(table) || !aligned16(out))
        return fail(DASH_HASH4D_INVALID_ARG, "table / out not 16-byte aligned");
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    const bool half = cfg->table_dtype == DASH_HASH4D_FP16;
    const size_t level_bytes = static_cast<size_t>(cfg->T) * cfg->F * (half ? 2 : 4);
    Plan P;
    uint32_t group = pick_group(cfg, level_bytes, DASH_DEBUG_FWD_GROUP);
    // 8-corner gathers: 4 levels per group measured best (G_3D workload: 0.423 ms at G = 4, 0.476 at G = 8,
    // 0.454 at G = 2) as long as a query's row slice stays a full 32-byte sector
    if (dims == 3 && group > 4 && 4 * cfg->F * sizeof(float) >= 32 && !debug_u32(DASH_DEBUG_FWD_GROUP))
        group = 4;
    if (int rc = fill_plan(cfg, N, xyz_stride, t_stride, group, &P, dims)) return rc;
    dash::CoarseSort cs;
    const bool coarse = plan_coarse(cfg, N, &cs, dims);
    const size_t need = workspace_need(cfg, DASH_HASH4D_OP_FWD, N, dims);
    if (coarse && (!workspace || workspace_bytes < need))
        return fail(DASH_HASH4D_WORKSPACE_TOO_SMALL, "fwd needs %zu workspace bytes, got %zu", need, workspace_bytes);
    if (coarse && !aligned16(workspace)) return fail(DASH_HASH4D_INVALID_ARG, "workspace not 16-byte aligned");
    if (int rc = run_validation(cfg, P, xyz, t, index, workspace, workspace_bytes, s)) return rc;
    if (coarse)
        if (int rc = verify_order(cfg, P, cs, xyz, t, index, workspace, s)) return rc;
    cudaError_t e = cudaSuccess;
    if (coarse) {
        // SORT_COARSE: the coarse levels in cell-sorted order (a warp's lanes then share cells and lines: C4 levels 0-3
        // 120 -> 72 us, profiles/experiments_r02.md §8), the others in the caller's order
        const CoarseBuffers b = carve_coarse(workspace, cs, N);
        if (!(cfg->flags & DASH_HASH4D_FLAG_ORDER_READY))
            e = dash::launch_coarse_sort(P, cs, xyz, t, index, b.order, b.sorted_q, b.keys, b.bins, b.totals, s,
                                         static_cast<WorkspaceHeader*>(workspace), order_stamp(P, cs, xyz, t, index));
        if (e != cudaSuccess) return cuda_fail(e, "coarse sort launch");
        Plan Pc = P;
        const uint32_t lf = cs.levels_fwd;
        uint32_t g = P.group;
        // in the sorted order 4 levels per group beat 8 (C5: 0.850 -> 0.822 ms) as long as a query's row slice stays a
        // full 32-byte sector: neighbouring lanes then hold 4 queries of one neighbourhood instead of 2
        if (g > 4 && 4 * cfg->F * sizeof(float) >= 32 && !debug_u32(DASH_DEBUG_FWD_GROUP)) g = 4;
        while (g > lf) g /= 2;
        uint32_t lg = 0;
        while ((1u << lg) < g) ++lg;
        Pc.group = g;
        Pc.group_log2 = lg;
        Pc.q_per_block = dash::kItemsPerBlock >> lg;
        Pc.level_end = lf;
        Pc.num_groups = (lf + g - 1) / g;
        e = dash::launch_fwd(Pc, xyz, t, index, table, half, out, s, b.order, b.sorted_q);
        if (e != cudaSuccess) return cuda_fail(e, "coarse fwd launch");
        // the other levels: whole groups of P.group in one launch, a ragged rest as smaller power-of-two groups
        for (uint32_t l0 = lf; l0 < cfg->L;) {
            uint32_t gr = P.group;
            while (gr > cfg->L - l0) gr /= 2;
            Plan Pr = P;
            lg = 0;
            while ((1u << lg) < gr) ++lg;
            Pr.group = gr;
            Pr.group_log2 = lg;
            Pr.q_per_block = dash::kItemsPerBlock >> lg;
            Pr.level_begin = l0;
            Pr.num_groups = (cfg->L - l0) / gr;
            e = dash::launch_fwd(Pr, xyz, t, index, table, half, out, s);
            if (e != cudaSuccess) return cuda_fail(e, "fwd launch");
            l0 += Pr.num_groups * gr;
        }
        return ok();
    }
    e = dash::launch_fwd(P, xyz, t, index, table, half, out, s);
    if (e != cudaSuccess) return cuda_fail(e, "fwd launch");
    return ok();
}

DASH_API int dash_hash4d_fwd(const dash_hash4d_config* cfg, uint64_t N, const float* xyz,
                             uint32_t xyz_stride, const float* t, uint32_t t_stride,
                             const int32_t* index, const void* table, float* out, void* workspace,
                             size_t workspace_bytes, void* cuda_stream) {
    return fwd_impl(4, cfg, N, xyz, xyz_stride, t, t_stride, index, table, out, workspace,
                    workspace_bytes, cuda_stream);
}

DASH_API int dash_hash3d_fwd(const dash_hash4d_config* cfg, uint64_t N, const float* xyz,
                             uint32_t xyz_stride, const int32_t* index, const void* table,
                             float* out, void* workspace, size_t workspace_bytes,
                             void* cuda_stream) {
    return fwd_impl(3, cfg, N, xyz, xyz_stride, nullptr, 0, index, table, out, workspace,
                    workspace_bytes, cuda_stream);
}

static int bwd_input_impl(int dims, const dash_hash4d_config* cfg, uint64_t N, const float* xyz,
                          uint32_t xyz_stride, const float* t, uint32_t t_stride, const int32_t* index,
                          const void* table, const float* dout, float* dq, void* workspace,
                          size_t workspace_bytes, void* cuda_stream) {
    if (int rc = check_config(cfg, dims)) return rc;
    if (N == 0) return ok();
    if (int rc = check_queries(xyz, xyz_stride, t, t_stride, index, dims)) return rc;
    if (!table || !dout || !dq) return fail(DASH_HASH4D_INVALID_ARG, "table, dout or dq is NULL");
    if (!aligned16(table) || !aligned16(dout) || (dims == 4 ? !aligned16(dq) : (reinterpret_cast<uintptr_t>(dq) & 3u)))
        return fail(DASH_HASH4D_INVALID_ARG, "table / dout / dq not aligned (16 bytes; dq of the 3D call 4 bytes)");
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    const bool half = cfg->table_dtype == DASH_HASH4D_FP16;
    const size_t level_bytes = static_cast<size_t>(cfg->T) * cfg->F * (half ? 2 : 4);
    Plan P;
    uint32_t group = pick_group(cfg, level_bytes, DASH_DEBUG_FWD_GROUP);
    if (dims == 3 && group > 4 && 4 * cfg->F * sizeof(float) >= 32 && !debug_u32(DASH_DEBUG_FWD_GROUP)) group = 4;
    if (int rc = fill_plan(cfg, N, xyz_stride, t_stride, group, &P, dims)) return rc;
    dash::CoarseSort cs;
    const bool coarse = plan_coarse(cfg, N, &cs, dims);   // SORT_COARSE: the same gathers as the forward, same order
    const size_t need = workspace_need(cfg, DASH_HASH4D_OP_BWD_INPUT, N, dims);
    if (coarse && (!workspace || workspace_bytes < need))
        return fail(DASH_HASH4D_WORKSPACE_TOO_SMALL, "bwd_input needs %zu workspace bytes, got %zu", need,
                    workspace_bytes);
    if (coarse && !aligned16(workspace)) return fail(DASH_HASH4D_INVALID_ARG, "workspace not 16-byte aligned");
    if (int rc = run_validation(cfg, P, xyz, t, index, workspace, workspace_bytes, s)) return rc;
    if (coarse)
        if (int rc = verify_order(cfg, P, cs, xyz, t, index, workspace, s)) return rc;
    cudaError_t e = dash::launch_zero(dq, static_cast<size_t>(N) * dims * sizeof(float), s);
    if (e == cudaSuccess && coarse) {
        const CoarseBuffers b = carve_coarse(workspace, cs, N);
        if (!(cfg->flags & DASH_HASH4D_FLAG_ORDER_READY))
            e = dash::launch_coarse_sort(P, cs, xyz, t, index, b.order, b.sorted_q, b.keys, b.bins, b.totals, s,
                                         static_cast<WorkspaceHeader*>(workspace), order_stamp(P, cs, xyz, t, index));
        if (e == cudaSuccess)
            e = dash::launch_bwd_input(P, xyz, t, index, table, half, dout, dq, s, b.order, b.sorted_q);
    } else if (e == cudaSuccess) {
        e = dash::launch_bwd_input(P, xyz, t, index, table, half, dout, dq, s);
    }
    if (e != cudaSuccess) return cuda_fail(e, "bwd_input launch");
    return ok();
}

DASH_API int dash_hash4d_bwd_input(const dash_hash4d_config* cfg, uint64_t N, const float* xyz,
                                   uint32_t xyz_stride, const float* t, uint32_t t_stride,
                                   const int32_t* index, const void* table, const float* dout,
                                   float* dq, void* workspace, size_t workspace_bytes,
                                   void* cuda_stream) {
    return bwd_input_impl(4, cfg, N, xyz, xyz_stride, t, t_stride, index, table, dout, dq, workspace,
                          workspace_bytes, cuda_stream);
}

DASH_API int dash_hash3d_bwd_input(const dash_hash4d_config* cfg, uint64_t N, const float* xyz,
                                   uint32_t xyz_stride, const int32_t* index, const void* table,
                                   const float* dout, float* dq, void* workspace, size_t workspace_bytes,
                                   void* cuda_stream) {
    return bwd_input_impl(3, cfg, N, xyz, xyz_stride, nullptr, 0, index, table, dout, dq, workspace,
                          workspace_bytes, cuda_stream);
}

DASH_API int dash_hash4d_smooth(const dash_hash4d_config* cfg, uint64_t N, const float* xyz,
                                uint32_t xyz_stride, const float* t, uint32_t t_stride,
                                const int32_t* index, const float* eps, uint32_t eps_stride,
                                const void* table, float grad_scale, float* loss, float* dtable,
                                void* workspace, size_t workspace_bytes, void* cuda_stream) {
    if (int rc = check_config(cfg)) return rc;
    if (dtable && (cfg->flags & DASH_HASH4D_FLAG_DETERMINISTIC_BWD))
        return fail(DASH_HASH4D_UNSUPPORTED, "smooth: DETERMINISTIC_BWD is not supported");
    if (N == 0) return ok();
    if (int rc = check_queries(xyz, xyz_stride, t, t_stride, index)) return rc;
    if (!eps || !table || !loss) return fail(DASH_HASH4D_INVALID_ARG, "eps, table or loss is NULL");
    if (!(eps_stride == 0 || eps_stride == 4))
        return fail(DASH_HASH4D_INVALID_ARG, "eps_stride = %u (want 0 or 4)", eps_stride);
    if ((reinterpret_cast<uintptr_t>(eps) | reinterpret_cast<uintptr_t>(loss)) & 3u)
        return fail(DASH_HASH4D_INVALID_ARG, "eps / loss not 4-byte aligned");
    if (!aligned16(table) || (dtable && !aligned16(dtable)))
        return fail(DASH_HASH4D_INVALID_ARG, "table / dtable not 16-byte aligned");
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    const bool half = cfg->table_dtype == DASH_HASH4D_FP16;
    // a level group keeps its table slice AND (with dtable) its gradient slice in L2; there is no
    // [N][L*F] row to keep sector-complete, so G may go down to 1
    const size_t level_bytes =
        static_cast<size_t>(cfg->T) * cfg->F * ((half ? 2 : 4) + (dtable ? 4 : 0));
    Plan P;
    if (int rc = fill_plan(cfg, N, xyz_stride, t_stride,
                           pick_group(cfg, level_bytes, DASH_DEBUG_SMOOTH_GROUP, false), &P))
        return rc;
    if (int rc = run_validation(cfg, P, xyz, t, index, workspace, workspace_bytes, s)) return rc;
    cudaError_t e = dash::launch_zero(loss, static_cast<size_t>(N) * sizeof(float), s);
    if (e == cudaSuccess)
        e = dash::launch_smooth(P, xyz, t, index, eps, eps_stride, table, half, 2.0f * grad_scale,
                                loss, dtable, s);
    if (e != cudaSuccess) return cuda_fail(e, "smooth launch");
    return ok();
}

static int bwd_impl(int dims, const dash_hash4d_config* cfg, uint64_t N, const float* xyz,
                    uint32_t xyz_stride, const float* t, uint32_t t_stride, const int32_t* index,
                    const float* dout, float* dtable, void* workspace, size_t workspace_bytes,
                    void* cuda_stream) {
    if (int rc = check_config(cfg, dims)) return rc;
    if (!dtable && (N || (cfg->flags & DASH_HASH4D_FLAG_ZERO_GRAD)))
        return fail(DASH_HASH4D_INVALID_ARG, "dtable is NULL");
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    const bool zero_first = (cfg->flags & DASH_HASH4D_FLAG_ZERO_GRAD) != 0;
    const size_t level_bytes = static_cast<size_t>(cfg->T) * cfg->F * sizeof(float);
    if (N == 0) {
        if (zero_first) {
            if (!aligned16(dtable))
                return fail(DASH_HASH4D_INVALID_ARG, "dtable not 16-byte aligned");
            cudaError_t e = dash::launch_zero(dtable, level_bytes * cfg->L, s);
            if (e != cudaSuccess) return cuda_fail(e, "zero launch");
        }
        return ok();
    }
    if (int rc = check_queries(xyz, xyz_stride, t, t_stride, index, dims)) return rc;
    if (!dout) return fail(DASH_HASH4D_INVALID_ARG, "dout is NULL");
    if (!aligned16(dout) || !aligned16(dtable))
        return fail(DASH_HASH4D_INVALID_ARG, "dout / dtable not 16-byte aligned");
    const bool fixed = (cfg->flags & DASH_HASH4D_FLAG_DETERMINISTIC_BWD) != 0;
    const size_t need = workspace_need(cfg, DASH_HASH4D_OP_BWD, N, dims);
    if (need && (!workspace || workspace_bytes < need))
        return fail(DASH_HASH4D_WORKSPACE_TOO_SMALL, "bwd needs %zu workspace bytes, got %zu", need,
                    workspace_bytes);
    if (need && !aligned16(workspace))
        return fail(DASH_HASH4D_INVALID_ARG, "workspace not 16-byte aligned");
    Plan P;
    const size_t scatter_bytes = fixed ? 2 * level_bytes : level_bytes;
    if (int rc = fill_plan(cfg, N, xyz_stride, t_stride,
                           pick_group(cfg, scatter_bytes, DASH_DEBUG_BWD_GROUP), &P, dims))
        return rc;
    if (int rc = run_validation(cfg, P, xyz, t, index, workspace, workspace_bytes, s)) return rc;

    cudaError_t e = cudaSuccess;
    if (fixed) {
        WorkspaceHeader* hdr = static_cast<WorkspaceHeader*>(workspace);
        long long* acc = reinterpret_cast<long long*>(static_cast<char*>(workspace) + kHeaderBytes);
        const size_t elems = table_elems(cfg);
        e = dash::launch_zero(workspace, kHeaderBytes + elems * sizeof(long long), s);
        if (e == cudaSuccess)
            e = dash::launch_absmax(dout, static_cast<size_t>(N) * cfg->L * cfg->F, hdr, N, s);
        if (e == cudaSuccess) e = dash::launch_bwd_fixed(P, xyz, t, index, dout, acc, hdr, s);
        if (e == cudaSuccess) e = dash::launch_fixed_finalize(acc, dtable, elems, hdr, zero_first, s);
        if (e != cudaSuccess) return cuda_fail(e, "deterministic bwd launch");
        return ok();
    }
    // SORT_COARSE: the leading `cs.levels` levels go through the sort + run-merged scatter (bwd_runs_kernels.cu),
    // the others through the one-reduction-per-corner kernel in the caller's order.
    dash::CoarseSort cs;
    const bool coarse = plan_coarse(cfg, N, &cs, dims);
    if (coarse)
        if (int rc = verify_order(cfg, P, cs, xyz, t, index, workspace, s)) return rc;
    const uint32_t l_first = coarse ? cs.levels : 0u;
    auto scatter_coarse = [&](bool hint) -> cudaError_t {
        const CoarseBuffers b = carve_coarse(workspace, cs, N);
        cudaError_t ce = cudaSuccess;
        if (!(cfg->flags & DASH_HASH4D_FLAG_ORDER_READY))
            ce = dash::launch_coarse_sort(P, cs, xyz, t, index, b.order, b.sorted_q, b.keys, b.bins, b.totals, s,
                                         static_cast<WorkspaceHeader*>(workspace), order_stamp(P, cs, xyz, t, index));
        if (ce == cudaSuccess) ce = dash::launch_bwd_runs(P, cs, dout, dtable, b.order, b.sorted_q, s, hint);
        return ce;
    };
    // the levels [l0, L) in groups of P.group (a ragged last group shrinks to the largest power of two that fits)
    auto scatter_rest = [&](uint32_t l0, bool hint) -> cudaError_t {
        if (l0 >= cfg->L) return cudaSuccess;
        Plan Pr = P;
        Pr.level_begin = l0;
        Pr.num_groups = (cfg->L - l0 + P.group - 1) / P.group;
        return dash::launch_bwd(Pr, xyz, t, index, dout, dtable, s, hint);
    };
    if (!zero_first) {
        if (coarse) e = scatter_coarse(false);
        if (e == cudaSuccess) e = scatter_rest(l_first, false);
        if (e != cudaSuccess) return cuda_fail(e, "bwd launch");
        return ok();
    }
    const bool hint = debug_u32(DASH_DEBUG_BWD_VARIANT) != 1;
    // ZERO_GRAD, small tables: when the WHOLE gradient buffer fits the L2 budget there is nothing to keep resident group
    // by group — one zero launch and one scatter launch over all groups (C2: 2 launches instead of 4).
    if (level_bytes * cfg->L <= l2_bytes() * 3 / 10) {
        e = dash::launch_zero(dtable, level_bytes * cfg->L, s, hint);
        if (e == cudaSuccess && coarse) e = scatter_coarse(hint);
        if (e == cudaSuccess) e = scatter_rest(l_first, hint);
        if (e != cudaSuccess) return cuda_fail(e, "bwd launch");
        return ok();
    }
    // ZERO_GRAD: zero one level group, scatter into it while the zeros are still in L2, next group.
    // (A one-launch variant whose tail CTAs zero the next group's slice was built and measured in round 2: slower,
    // profiles/experiments_r02.md §1.)  L2 evict_last hints on the zero stores and the reductions keep the group's
    // slice resident against the streamed dout / coordinates: C4 bwd 1.190 -> 1.168 ms, DRAM bytes per call 2.76 ->
    // 1.54 GB (ncu, profiles/experiments_r02.md §2).  DASH_DEBUG_BWD_VARIANT = 1 turns the hints off for A/B runs.
    if (coarse) {   // the coarse levels' slices first: only their dense / touched part is ever fetched again
        e = dash::launch_zero(dtable, static_cast<size_t>(l_first) * level_bytes, s, hint);
        if (e == cudaSuccess) e = scatter_coarse(hint);
        if (e != cudaSuccess) return cuda_fail(e, "coarse bwd launch");
    }
    for (uint32_t l0 = l_first; l0 < cfg->L;) {
        uint32_t g = P.group;
        while (g > cfg->L - l0) g /= 2;   // ragged tail: a smaller power of two instead of idle lanes
        char* base = reinterpret_cast<char*>(dtable) + static_cast<size_t>(l0) * level_bytes;
        e = dash::launch_zero(base, static_cast<size_t>(g) * level_bytes, s, hint);  // handles 4-byte aligned slices
        if (e != cudaSuccess) return cuda_fail(e, "zero launch");
        Plan Pg = P;
        uint32_t lg = 0;
        while ((1u << lg) < g) ++lg;
        Pg.group = g;
        Pg.group_log2 = lg;
        Pg.q_per_block = dash::kItemsPerBlock >> lg;
        Pg.level_begin = l0;
        Pg.num_groups = 1;
        e = dash::launch_bwd(Pg, xyz, t, index, dout, dtable, s, hint);
        if (e != cudaSuccess) return cuda_fail(e, "bwd launch");
        l0 += g;
    }
    return ok();
}

DASH_API int dash_hash4d_bwd(const dash_hash4d_config* cfg, uint64_t N, const float* xyz,
                             uint32_t xyz_stride, const float* t, uint32_t t_stride,
                             const int32_t* index, const float* dout, float* dtable,
                             void* workspace, size_t workspace_bytes, void* cuda_stream) {
    return bwd_impl(4, cfg, N, xyz, xyz_stride, t, t_stride, index, dout, dtable, workspace,
                    workspace_bytes, cuda_stream);
}

DASH_API int dash_hash3d_bwd(const dash_hash4d_config* cfg, uint64_t N, const float* xyz,
                             uint32_t xyz_stride, const int32_t* index, const float* dout,
                             float* dtable, void* workspace, size_t workspace_bytes,
                             void* cuda_stream) {
    return bwd_impl(3, cfg, N, xyz, xyz_stride, nullptr, 0, index, dout, dtable, workspace,
                    workspace_bytes, cuda_stream);
}

static int indices_impl(int dims, const dash_hash4d_config* cfg, uint64_t N, const float* xyz,
                        uint32_t xyz_stride, const float* t, uint32_t t_stride,
                        const int32_t* index, uint32_t* idx_out, float* w_out, void* cuda_stream) {
    if (int rc = check_config(cfg, dims)) return rc;
    if (N == 0) return ok();
    if (int rc = check_queries(xyz, xyz_stride, t, t_stride, index, dims)) return rc;
    if (!idx_out) return fail(DASH_HASH4D_INVALID_ARG, "idx_out is NULL");
    if (N * cfg->L > 0x7fffffffull * dash::kBlockThreads)
        return fail(DASH_HASH4D_UNSUPPORTED, "N*L too large for one launch");
    Plan P;
    if (int rc = fill_plan(cfg, N, xyz_stride, t_stride, 1, &P, dims)) return rc;
    cudaError_t e = dash::launch_indices(P, xyz, t, index, idx_out, w_out,
                                         static_cast<cudaStream_t>(cuda_stream));
    if (e != cudaSuccess) return cuda_fail(e, "indices launch");
    return ok();
}

DASH_API int dash_hash4d_indices(const dash_hash4d_config* cfg, uint64_t N, const float* xyz,
                                 uint32_t xyz_stride, const float* t, uint32_t t_stride,
                                 const int32_t* index, uint32_t* idx_out, float* w_out,
                                 void* cuda_stream) {
    return indices_impl(4, cfg, N, xyz, xyz_stride, t, t_stride, index, idx_out, w_out, cuda_stream);
}

DASH_API int dash_hash3d_indices(const dash_hash4d_config* cfg, uint64_t N, const float* xyz,
                                 uint32_t xyz_stride, const int32_t* index, uint32_t* idx_out,
                                 float* w_out, void* cuda_stream) {
    return indices_impl(3, cfg, N, xyz, xyz_stride, nullptr, 0, index, idx_out, w_out, cuda_stream);
}

DASH_API int dash_hash3d_resolutions(const dash_hash4d_config* cfg, uint32_t* res_s,
                                     uint8_t* is_dense) {
    if (int rc = check_config(cfg, 3)) return rc;
    if (!res_s) return fail(DASH_HASH4D_INVALID_ARG, "res_s is NULL");
    Schedule s;
    make_schedule(cfg, &s, 3);
    for (uint32_t l = 0; l < cfg->L; ++l) {
        res_s[l] = s.res_s[l];
        if (is_dense) is_dense[l] = s.dense[l];
    }
    return ok();
}

DASH_API int dash_hash4d_adam_step(const dash_hash4d_config* cfg, const dash_adam_config* opt,
                                   float* theta, void* table16, float* dtable, float* m, float* v,
                                   void* cuda_stream) {
    if (int rc = check_config(cfg, 3)) return rc;
    if (!opt || opt->struct_size != sizeof(dash_adam_config))
        return fail(DASH_HASH4D_INVALID_ARG, "adam config NULL or wrong struct_size");
    if (opt->step < 1) return fail(DASH_HASH4D_INVALID_ARG, "adam step must be >= 1");
    if (!(opt->beta1 >= 0.0f && opt->beta1 < 1.0f && opt->beta2 >= 0.0f && opt->beta2 < 1.0f) ||
        !(opt->eps >= 0.0f) || !(opt->lr == opt->lr))
        return fail(DASH_HASH4D_INVALID_ARG, "adam hyper-parameters out of range");
    if (opt->flags & ~static_cast<uint32_t>(DASH_ADAM_ZERO_GRAD))
        return fail(DASH_HASH4D_INVALID_ARG, "unknown adam flag bits 0x%x", opt->flags);
    if (!theta || !dtable || !m || !v) return fail(DASH_HASH4D_INVALID_ARG, "theta, dtable, m or v is NULL");
    if (!aligned16(theta) || !aligned16(dtable) || !aligned16(m) || !aligned16(v) ||
        (table16 && !aligned16(table16)))
        return fail(DASH_HASH4D_INVALID_ARG, "adam buffers not 16-byte aligned");
    cudaError_t e = dash::launch_adam(table_elems(cfg), opt->lr, opt->beta1, opt->beta2, opt->eps, opt->step,
                                      (opt->flags & DASH_ADAM_ZERO_GRAD) != 0, theta, table16, dtable, m, v,
                                      static_cast<cudaStream_t>(cuda_stream));
    if (e != cudaSuccess) return cuda_fail(e, "adam launch");
    return ok();
}

DASH_API size_t dash_hash4d_sort_workspace_bytes(uint64_t N, uint32_t bits) {
    if (bits < 1 || bits > 7) return 0;
    const size_t n_bins = static_cast<size_t>(1) << (3 * bits);
    return round16(N * 4) + round16(n_bins * 4) + round16((n_bins + 1023) / 1024 * 4);
}

DASH_API int dash_hash4d_sort_queries(uint64_t N, const float* xyz, uint32_t xyz_stride, const int32_t* index,
                                      uint32_t bits, int32_t* order, void* workspace, size_t workspace_bytes,
                                      void* cuda_stream) {
    if (bits < 1 || bits > 7) return fail(DASH_HASH4D_INVALID_ARG, "bits = %u outside 1..7", bits);
    if (N == 0) return ok();
    if (N > 0x7fffffffull) return fail(DASH_HASH4D_UNSUPPORTED, "N too large for an int32 order list");
    if (!xyz || !order) return fail(DASH_HASH4D_INVALID_ARG, "xyz or order is NULL");
    if (!(xyz_stride == 3 || xyz_stride == 4))
        return fail(DASH_HASH4D_INVALID_ARG, "xyz_stride = %u (want 3 or 4)", xyz_stride);
    const size_t need = dash_hash4d_sort_workspace_bytes(N, bits);
    if (!workspace || workspace_bytes < need)
        return fail(DASH_HASH4D_WORKSPACE_TOO_SMALL, "sort needs %zu workspace bytes, got %zu", need, workspace_bytes);
    if (!aligned16(workspace)) return fail(DASH_HASH4D_INVALID_ARG, "workspace not 16-byte aligned");
    const size_t n_bins = static_cast<size_t>(1) << (3 * bits);
    char* w = static_cast<char*>(workspace);
    uint32_t* keys = reinterpret_cast<uint32_t*>(w);
    uint32_t* bins = reinterpret_cast<uint32_t*>(w + round16(N * 4));
    uint32_t* totals = reinterpret_cast<uint32_t*>(w + round16(N * 4) + round16(n_bins * 4));
    cudaError_t e = dash::launch_sort_queries(N, xyz, xyz_stride, index, bits, order, keys, bins, totals,
                                              static_cast<cudaStream_t>(cuda_stream));
    if (e != cudaSuccess) return cuda_fail(e, "sort launch");
    return ok();
}

DASH_API int dash_hash4d_zero(const dash_hash4d_config* cfg, float* dtable, void* cuda_stream) {
    if (int rc = check_config(cfg, 3)) return rc;  // only L, T, F matter here (serves G_3D tables too)
    if (!dtable) return fail(DASH_HASH4D_INVALID_ARG, "dtable is NULL");
    if (!aligned16(dtable)) return fail(DASH_HASH4D_INVALID_ARG, "dtable not 16-byte aligned");
    cudaError_t e = dash::launch_zero(dtable, table_elems(cfg) * sizeof(float),
                                      static_cast<cudaStream_t>(cuda_stream));
    if (e != cudaSuccess) return cuda_fail(e, "zero launch");
    return ok();
}

}  // extern "C"

// ------------------------------------------------------------------------------------------------------------
// dash_hash4d_sort_queries_static: the query sort for callers that must not allocate device memory.
//
// The counting sort needs scratch besides its input and output: one key per query, the histogram bins and the
// scan's per-CTA totals.  dash_hash4d_sort_queries takes that scratch from the caller; this variant takes it from
// the array below, which lives in the library's own device data segment.  The CUDA runtime places the array on
// every GPU whose context loads the library and keeps it there until the process exits, so no call ever
// allocates, and the price is kSortStaticBytes (about 5 MB) of HBM per GPU whether or not the call is used.
//
// `g_sort_static` is only a device address inside device code.  In host code the same name is a host-side handle:
// handing it to a kernel as if it were a pointer makes the kernel fault, or (on systems where the GPU can
// dereference host addresses) scribble over host memory.  The host therefore asks the runtime where the array
// lives on the CURRENT device (cudaGetSymbolAddress), once per device, and passes that address on.
// ------------------------------------------------------------------------------------------------------------
namespace {

constexpr size_t kSortStaticKeysBytes = static_cast<size_t>(DASH_HASH4D_SORT_STATIC_MAX_N) * 4;
constexpr size_t kSortStaticBinsBytes = (static_cast<size_t>(1) << (3 * DASH_HASH4D_SORT_STATIC_MAX_BITS)) * 4;
constexpr size_t kSortStaticTotalsBytes = 1024;  // >= one uint32 per 1024 bins at the maximum bin count
constexpr size_t kSortStaticBytes = kSortStaticKeysBytes + kSortStaticBinsBytes + kSortStaticTotalsBytes;
static_assert(kSortStaticTotalsBytes >= (kSortStaticBinsBytes / 4 + 1023) / 1024 * 4, "totals region too small");
static_assert(kSortStaticKeysBytes % 256 == 0 && kSortStaticBinsBytes % 256 == 0, "regions keep the alignment");

static __device__ __align__(256) unsigned char g_sort_static[kSortStaticBytes];

constexpr int kSortStaticMaxDevices = 64;
std::mutex g_sort_static_mutex;
unsigned char* g_sort_static_addr[kSortStaticMaxDevices] = {};  // per device ordinal; NULL = not looked up yet

// Device address of g_sort_static on the current device.  The first call on a device performs the look-up (which
// also makes the runtime load the module there); later calls return the cached address.
int sort_static_address(unsigned char** out) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return cuda_fail(e, "cudaGetDevice");
    if (dev < 0 || dev >= kSortStaticMaxDevices)
        return fail(DASH_HASH4D_UNSUPPORTED, "device ordinal %d outside 0..%d", dev, kSortStaticMaxDevices - 1);
    std::lock_guard<std::mutex> lock(g_sort_static_mutex);
    if (!g_sort_static_addr[dev]) {
        void* p = nullptr;
        e = cudaGetSymbolAddress(&p, g_sort_static);
        if (e != cudaSuccess) return cuda_fail(e, "cudaGetSymbolAddress(static sort scratch)");
        if (!p) return fail(DASH_HASH4D_CUDA_ERROR, "cudaGetSymbolAddress returned NULL for the static sort scratch");
        g_sort_static_addr[dev] = static_cast<unsigned char*>(p);
    }
    *out = g_sort_static_addr[dev];
    return DASH_HASH4D_OK;
}

}  // namespace

extern "C" DASH_API int dash_hash4d_sort_queries_static(uint64_t N, const float* xyz, uint32_t xyz_stride,
                                                        const int32_t* index, uint32_t bits, int32_t* order,
                                                        void* cuda_stream) {
    if (bits < 1 || bits > DASH_HASH4D_SORT_STATIC_MAX_BITS)
        return fail(DASH_HASH4D_UNSUPPORTED, "bits = %u outside 1..%d: the built-in scratch holds at most 2^%d bins; "
                    "use dash_hash4d_sort_queries with a caller-supplied workspace", bits,
                    DASH_HASH4D_SORT_STATIC_MAX_BITS, 3 * DASH_HASH4D_SORT_STATIC_MAX_BITS);
    if (N > DASH_HASH4D_SORT_STATIC_MAX_N)
        return fail(DASH_HASH4D_UNSUPPORTED, "N = %llu exceeds the %llu queries the built-in scratch holds; "
                    "use dash_hash4d_sort_queries with a caller-supplied workspace",
                    static_cast<unsigned long long>(N), static_cast<unsigned long long>(DASH_HASH4D_SORT_STATIC_MAX_N));
    if (N == 0) return ok();
    if (!xyz || !order) return fail(DASH_HASH4D_INVALID_ARG, "xyz or order is NULL");
    if (!(xyz_stride == 3 || xyz_stride == 4))
        return fail(DASH_HASH4D_INVALID_ARG, "xyz_stride = %u (want 3 or 4)", xyz_stride);
    unsigned char* base = nullptr;
    if (int rc = sort_static_address(&base)) return rc;
    uint32_t* keys = reinterpret_cast<uint32_t*>(base);
    uint32_t* bins = reinterpret_cast<uint32_t*>(base + kSortStaticKeysBytes);
    uint32_t* totals = reinterpret_cast<uint32_t*>(base + kSortStaticKeysBytes + kSortStaticBinsBytes);
    // Same five launches as dash_hash4d_sort_queries.  The array still holds whatever the previous call left: the
    // first launch zeroes the bins this call counts into; keys[0..N) and the totals are fully rewritten before read.
    cudaError_t e = dash::launch_sort_queries(N, xyz, xyz_stride, index, bits, order, keys, bins, totals,
                                              static_cast<cudaStream_t>(cuda_stream));
    if (e != cudaSuccess) return cuda_fail(e, "static sort launch");
    return ok();
}

// ------------------------------------------------------------------------------------------------------------
// Render path: G_4D -> phi_d -> heads (include/dash_deform.h; Eq. 9-10; Q27)
// ------------------------------------------------------------------------------------------------------------
namespace {

int check_mlp(const dash_mlp_config* m) {
    if (!m) return fail(DASH_HASH4D_INVALID_ARG, "mlp config is NULL");
    if (m->struct_size != sizeof(dash_mlp_config))
        return fail(DASH_HASH4D_INVALID_ARG, "mlp struct_size %u != %zu", m->struct_size,
                    sizeof(dash_mlp_config));
    if (m->n_layers < 1 || m->n_layers > dash::kMlpMaxLayers)
        return fail(DASH_HASH4D_INVALID_ARG, "n_layers = %u outside 1..%u", m->n_layers,
                    dash::kMlpMaxLayers);
    for (uint32_t l = 0; l <= m->n_layers; ++l)
        if (m->width[l] < 1 || m->width[l] > dash::kMlpMaxWidth)
            return fail(DASH_HASH4D_INVALID_ARG, "width[%u] = %u outside 1..%u", l, m->width[l],
                        dash::kMlpMaxWidth);
    if (m->flags) return fail(DASH_HASH4D_INVALID_ARG, "unknown mlp flag bits 0x%x", m->flags);
    return DASH_HASH4D_OK;
}

uint32_t round_up(uint32_t v, uint32_t m) { return (v + m - 1) / m * m; }

// Shared-memory map of one CTA: [barriers + TMEM slot: 128 B][biases][weights][A0 x 2][activations]
int fill_mlp_plan(const dash_mlp_config* m, uint64_t N, dash::MlpPlan* M) {
    std::memset(M, 0, sizeof(*M));
    M->N = N;
    const uint64_t tiles = (N + dash::kDeformTileM - 1) / dash::kDeformTileM;
    if (tiles > 0x7fffffffull) return fail(DASH_HASH4D_UNSUPPORTED, "N too large for one launch");
    M->num_tiles = static_cast<uint32_t>(tiles);
    const uint64_t sms = static_cast<uint64_t>(dash::device_sm_count());
    M->grid = static_cast<uint32_t>(tiles < sms ? tiles : sms);
    M->rows_per_cta = M->grid ? (N + M->grid - 1) / M->grid : 0;
    M->n_layers = m->n_layers;
    for (uint32_t l = 0; l <= m->n_layers; ++l) M->width[l] = m->width[l];
    M->n_out = m->width[m->n_layers];
    uint32_t off = 128, p = 0, nmax = 0, kmax = 0;
    for (uint32_t l = 0; l < m->n_layers; ++l) {
        M->kbias[l] = round_up(m->width[l], 16);
        M->kpad[l] = M->kbias[l] + 16;   // two bias columns (bf16 hi + lo), padded to one K = 16 step
        M->npad[l] = round_up(m->width[l + 1], 16);
        M->p_off[l] = p;
        p += m->width[l + 1] * m->width[l] + m->width[l + 1];
        if (M->npad[l] > nmax) nmax = M->npad[l];
        if (l > 0 && M->kpad[l] > kmax) kmax = M->kpad[l];
    }
    // operands are stored chunk-major with LBO = rows*16 + 16 bytes (deform_kernels.cu operand_lbo)
    for (uint32_t l = 0; l < m->n_layers; ++l) {
        M->w_off[l] = off;
        off += (M->kpad[l] / 8) * (M->npad[l] * 16 + 16);
    }
    off = round_up(off, 128);
    const uint32_t a_lbo = dash::kDeformTileM * 16 + 16;
    M->a0_off = off;
    off += 2 * (M->kpad[0] / 8) * a_lbo;
    // narrow last layer: the consumer warps transpose their 32 x n_out output block through shared memory
    M->out_stage_off = 0;
    if (M->npad[m->n_layers - 1] == 16 && off + 4 * dash::kDeformPipes * 2048u <= dash::kDeformSmemLimit) {
        off = round_up(off, 16);
        M->out_stage_off = off;
        off += 4 * dash::kDeformPipes * 2048u;
    }
    M->smem_bytes = off;
    // tensor memory per pipeline: fp32 accumulator (nmax columns) + the bf16 A operand of layers 2..n (two
    // elements per 32-bit column: kmax / 2 columns).  Two pipelines when both fit the SM's 512 columns.
    M->tmem_a_off = nmax;
    M->tmem_pipe_cols = nmax + kmax / 2;
    M->npipes = (2 * M->tmem_pipe_cols <= 512) ? dash::kDeformPipes : 1;
    uint32_t cols = 32;
    while (cols < M->npipes * M->tmem_pipe_cols) cols *= 2;
    M->tmem_cols = cols;
    if (M->smem_bytes > dash::kDeformSmemLimit)
        return fail(DASH_HASH4D_UNSUPPORTED,
                    "this layer chain needs %u bytes of shared memory per CTA (limit %u)", M->smem_bytes,
                    dash::kDeformSmemLimit);
    return DASH_HASH4D_OK;
}

size_t mlp_params(const dash_mlp_config* m) {
    size_t p = 0;
    for (uint32_t l = 0; l < m->n_layers; ++l)
        p += static_cast<size_t>(m->width[l + 1]) * m->width[l] + m->width[l + 1];
    return p;
}

// the fused kernel walks all L levels per tile: the whole table (or fp32 time slice) must stay L2-resident
bool deform_fused_applies(const dash_hash4d_config* enc, bool slice = false) {
    if (const uint32_t forced = debug_u32(DASH_DEBUG_DEFORM_PATH)) return forced == 1;  // 1 fused, 2 two-pass
    const size_t elem = (!slice && enc->table_dtype == DASH_HASH4D_FP16) ? 2 : 4;
    const size_t table_bytes = static_cast<size_t>(enc->L) * enc->T * enc->F * elem;
    return table_bytes <= l2_bytes() / 100 * 55;
}

}  // namespace

extern "C" {

DASH_API size_t dash_mlp_param_count(const dash_mlp_config* mlp) {
    if (check_mlp(mlp)) return 0;
    g_error[0] = '\0';
    return mlp_params(mlp);
}

DASH_API int dash_mlp_fwd(const dash_mlp_config* mlp, uint64_t N, const float* feat,
                          const float* params, const float* base, float* out, void* cuda_stream) {
    if (int rc = check_mlp(mlp)) return rc;
    dash::MlpPlan M;
    if (int rc = fill_mlp_plan(mlp, N, &M)) return rc;
    if (N == 0) return ok();
    if (!feat || !params || !out) return fail(DASH_HASH4D_INVALID_ARG, "feat, params or out is NULL");
    if ((reinterpret_cast<uintptr_t>(feat) | reinterpret_cast<uintptr_t>(params) |
         reinterpret_cast<uintptr_t>(base) | reinterpret_cast<uintptr_t>(out)) & 3u)
        return fail(DASH_HASH4D_INVALID_ARG, "feat / params / base / out not 4-byte aligned");
    cudaError_t e = dash::launch_mlp(M, feat, params, base, out, dash::device_sm_count(), static_cast<cudaStream_t>(cuda_stream));
    if (e != cudaSuccess) return cuda_fail(e, "mlp launch");
    return ok();
}

}  // extern "C"

namespace {

// Shared-memory / tensor-memory map of mlp_bwd_kernel (deform_kernels.h MlpBwdPlan).
int fill_mlp_bwd_plan(const dash_mlp_config* m, uint64_t N, dash::MlpBwdPlan* B) {
    std::memset(B, 0, sizeof(*B));
    if (int rc = fill_mlp_plan(m, N, &B->fwd)) return rc;
    const dash::MlpPlan& M = B->fwd;
    const uint32_t nl = M.n_layers, tile_lbo = dash::kDeformTileM * 16 + 16;
    uint32_t off = 0;
    for (uint32_t l = 0; l < nl; ++l) {
        if (M.kpad[l] > 256)
            return fail(DASH_HASH4D_UNSUPPORTED, "mlp_bwd: width[%u] = %u exceeds 240 (one wgrad MMA covers N <= 256)",
                        l, M.width[l]);
        // One M = 128 wgrad issue and 16-chunk delta buffers per layer: a wider OUTPUT would lose rows >= 128 of dW / db
        // and write its delta tile past the shared-memory allocation.
        if (M.width[l + 1] > 128)
            return fail(DASH_HASH4D_UNSUPPORTED, "mlp_bwd: width[%u] = %u exceeds 128 (a layer's output is one M = 128 "
                        "weight-gradient tile)", l + 1, M.width[l + 1]);
        B->w_off[l] = off;
        off += (M.kpad[l] / 8) * (M.npad[l] * 16 + 16);
    }
    off = round_up(off, 128);
    B->a_off[0] = off;
    B->a0_bytes = (M.kpad[0] / 8) * tile_lbo;
    off += 2 * B->a0_bytes;
    for (uint32_t l = 1; l < nl; ++l) {
        B->a_off[l] = off;
        off += (M.kpad[l] / 8) * tile_lbo;
    }
    B->dn_off = off;                       // delta_n first: the wgrad reads 16 chunks from it, the overrun lands in
    off += (M.npad[nl - 1] / 8) * tile_lbo;   // the delta buffers behind it (garbage rows of the accumulator, never read)
    B->d_off[0] = off;
    B->d_off[1] = off + 16 * tile_lbo;
    off += 32 * tile_lbo;
    B->bar_off = round_up(off, 128);
    B->smem_bytes = B->bar_off + 128;
    if (B->smem_bytes > dash::kDeformSmemLimit)
        return fail(DASH_HASH4D_UNSUPPORTED, "mlp_bwd: this layer chain needs %u bytes of shared memory per CTA (limit %u)",
                    B->smem_bytes, dash::kDeformSmemLimit);
    uint32_t acc = 32;
    for (uint32_t l = 0; l + 1 < nl; ++l) acc = M.npad[l] > acc ? M.npad[l] : acc;
    for (uint32_t l = 0; l < nl; ++l) acc = M.kbias[l] > acc ? M.kbias[l] : acc;
    B->acc_col = 0;
    B->acc_cols = round_up(acc, 32);
    uint32_t col = B->acc_cols;
    for (uint32_t l = 0; l < nl; ++l) {
        B->dw_col[l] = col;
        col += M.kpad[l];
    }
    if (col > 512)
        return fail(DASH_HASH4D_UNSUPPORTED, "mlp_bwd: %u tensor-memory columns needed (accumulator %u + weight "
                    "gradients), 512 available", col, B->acc_cols);
    uint32_t cols = 32;
    while (cols < col) cols *= 2;
    B->tmem_cols = cols;
    return DASH_HASH4D_OK;
}

}  // namespace

extern "C" {

DASH_API int dash_mlp_bwd(const dash_mlp_config* mlp, uint64_t N, const float* feat, const float* params,
                          const float* dout, float* dfeat, float* dparams, void* cuda_stream) {
    if (int rc = check_mlp(mlp)) return rc;
    dash::MlpBwdPlan B;
    if (int rc = fill_mlp_bwd_plan(mlp, N, &B)) return rc;
    if (N == 0) return ok();
    if (!feat || !params || !dout || !dparams)
        return fail(DASH_HASH4D_INVALID_ARG, "feat, params, dout or dparams is NULL");
    if ((reinterpret_cast<uintptr_t>(feat) | reinterpret_cast<uintptr_t>(params) | reinterpret_cast<uintptr_t>(dout) |
         reinterpret_cast<uintptr_t>(dparams)) & 3u)
        return fail(DASH_HASH4D_INVALID_ARG, "feat / params / dout / dparams not 4-byte aligned");
    if (dfeat && !aligned16(dfeat)) return fail(DASH_HASH4D_INVALID_ARG, "dfeat not 16-byte aligned");
    cudaError_t e = dash::launch_mlp_bwd(B, feat, params, dout, dfeat, dparams, static_cast<cudaStream_t>(cuda_stream));
    if (e != cudaSuccess) return cuda_fail(e, "mlp_bwd launch");
    return ok();
}

DASH_API size_t dash_deform_bwd_workspace_bytes(const dash_hash4d_config* enc, const dash_mlp_config* mlp,
                                                uint64_t N) {
    if (check_config(enc) || check_mlp(mlp)) return 0;
    g_error[0] = '\0';
    // feature matrix + its gradient, then (SORT_COARSE) the encoder's sort workspace
    return 2 * round16(static_cast<size_t>(N) * enc->L * enc->F * sizeof(float)) +
           round16(workspace_need(enc, DASH_HASH4D_OP_FWD, N, 4));
}

DASH_API int dash_deform_bwd(const dash_hash4d_config* enc, const dash_mlp_config* mlp, uint64_t N,
                             const float* xyz, uint32_t xyz_stride, const float* t, uint32_t t_stride,
                             const int32_t* index, const void* table, const float* params, const float* dout,
                             float* dtable, float* dparams, float* dq, void* workspace, size_t workspace_bytes,
                             void* cuda_stream) {
    if (int rc = check_config(enc)) return rc;
    if (int rc = check_mlp(mlp)) return rc;
    constexpr uint32_t kAllowed = DASH_HASH4D_FLAG_DENSE_COARSE | DASH_HASH4D_FLAG_ZERO_GRAD | DASH_HASH4D_FLAG_SORT_COARSE;
    if (enc->flags & ~kAllowed)
        return fail(DASH_HASH4D_INVALID_ARG,
                    "deform_bwd: only DENSE_COARSE | ZERO_GRAD | SORT_COARSE may be set in enc->flags");
    if (mlp->width[0] != enc->L * enc->F)
        return fail(DASH_HASH4D_INVALID_ARG, "mlp width[0] = %u != L*F = %u", mlp->width[0], enc->L * enc->F);
    const size_t half = round16(static_cast<size_t>(N) * enc->L * enc->F * sizeof(float));
    const size_t sort_bytes = round16(workspace_need(enc, DASH_HASH4D_OP_FWD, N, 4));
    if (N && (!workspace || workspace_bytes < 2 * half + sort_bytes))
        return fail(DASH_HASH4D_WORKSPACE_TOO_SMALL, "deform_bwd needs %zu workspace bytes, got %zu",
                    2 * half + sort_bytes, workspace_bytes);
    if (N && !aligned16(workspace)) return fail(DASH_HASH4D_INVALID_ARG, "workspace not 16-byte aligned");
    float* feat = static_cast<float*>(workspace);
    float* dfeat = reinterpret_cast<float*>(static_cast<char*>(workspace) + half);
    void* sort_ws = sort_bytes ? static_cast<char*>(workspace) + 2 * half : nullptr;
    // SORT_COARSE: ONE sort (inside the forward) serves the forward, the table gradient and the coordinate gradient
    const uint32_t sorted = enc->flags & DASH_HASH4D_FLAG_SORT_COARSE;
    const uint32_t ready = sorted ? (sorted | DASH_HASH4D_FLAG_ORDER_READY) : 0u;
    dash_hash4d_config fcfg = *enc, bcfg = *enc, icfg = *enc;
    fcfg.flags = (enc->flags & DASH_HASH4D_FLAG_DENSE_COARSE) | sorted;
    bcfg.flags = (enc->flags & (DASH_HASH4D_FLAG_DENSE_COARSE | DASH_HASH4D_FLAG_ZERO_GRAD)) | ready;
    icfg.flags = (enc->flags & DASH_HASH4D_FLAG_DENSE_COARSE) | ready;
    if (int rc = fwd_impl(4, &fcfg, N, xyz, xyz_stride, t, t_stride, index, table, feat, sort_ws, sort_bytes, cuda_stream))
        return rc;
    if (int rc = dash_mlp_bwd(mlp, N, feat, params, dout, dfeat, dparams, cuda_stream)) return rc;
    if (int rc = bwd_impl(4, &bcfg, N, xyz, xyz_stride, t, t_stride, index, dfeat, dtable, sort_ws, sort_bytes,
                          cuda_stream))
        return rc;
    if (dq)
        if (int rc = dash_hash4d_bwd_input(&icfg, N, xyz, xyz_stride, t, t_stride, index, table, dfeat, dq, sort_ws,
                                           sort_bytes, cuda_stream))
            return rc;
    return ok();
}

DASH_API size_t dash_deform_workspace_bytes(const dash_hash4d_config* enc, const dash_mlp_config* mlp,
                                            uint64_t N) {
    if (check_config(enc) || check_mlp(mlp)) return 0;
    g_error[0] = '\0';
    if (deform_fused_applies(enc)) return 0;
    return static_cast<size_t>(N) * enc->L * enc->F * sizeof(float);
}

DASH_API int dash_deform_fwd(const dash_hash4d_config* enc, const dash_mlp_config* mlp, uint64_t N,
                             const float* xyz, uint32_t xyz_stride, const float* t, uint32_t t_stride,
                             const int32_t* index, const void* table, const float* params,
                             const float* base, float* out, void* workspace, size_t workspace_bytes,
                             void* cuda_stream) {
    if (int rc = check_config(enc)) return rc;
    if (int rc = check_mlp(mlp)) return rc;
    if (enc->flags & ~static_cast<uint32_t>(DASH_HASH4D_FLAG_DENSE_COARSE))
        return fail(DASH_HASH4D_INVALID_ARG, "deform_fwd: only DENSE_COARSE may be set in enc->flags");
    if (mlp->width[0] != enc->L * enc->F)
        return fail(DASH_HASH4D_INVALID_ARG, "mlp width[0] = %u != L*F = %u", mlp->width[0],
                    enc->L * enc->F);
    dash::MlpPlan M;
    if (int rc = fill_mlp_plan(mlp, N, &M)) return rc;
    if (N == 0) return ok();
    if (int rc = check_queries(xyz, xyz_stride, t, t_stride, index)) return rc;
    if (!table || !params || !out) return fail(DASH_HASH4D_INVALID_ARG, "table, params or out is NULL");
    if (!aligned16(table)) return fail(DASH_HASH4D_INVALID_ARG, "table not 16-byte aligned");
    if ((reinterpret_cast<uintptr_t>(params) | reinterpret_cast<uintptr_t>(base) |
         reinterpret_cast<uintptr_t>(out)) & 3u)
        return fail(DASH_HASH4D_INVALID_ARG, "params / base / out not 4-byte aligned");
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    const bool half = enc->table_dtype == DASH_HASH4D_FP16;
    if (deform_fused_applies(enc)) {
        Plan P;
        if (int rc = fill_plan(enc, N, xyz_stride, t_stride, 1, &P)) return rc;
        cudaError_t e = dash::launch_deform_fused(P, M, xyz, t, index, table, half, params, base, out,
                                                  dash::device_sm_count(), s);
        if (e != cudaSuccess) return cuda_fail(e, "deform launch");
        return ok();
    }
    const size_t need = static_cast<size_t>(N) * enc->L * enc->F * sizeof(float);
    if (!workspace || workspace_bytes < need)
        return fail(DASH_HASH4D_WORKSPACE_TOO_SMALL, "deform_fwd (two-pass) needs %zu workspace bytes, got %zu",
                    need, workspace_bytes);
    if (!aligned16(workspace)) return fail(DASH_HASH4D_INVALID_ARG, "workspace not 16-byte aligned");
    float* feat = static_cast<float*>(workspace);
    if (int rc = fwd_impl(4, enc, N, xyz, xyz_stride, t, t_stride, index, table, feat, nullptr, 0, cuda_stream))
        return rc;
    cudaError_t e = dash::launch_mlp(M, feat, params, base, out, dash::device_sm_count(), s);
    if (e != cudaSuccess) return cuda_fail(e, "mlp launch");
    return ok();
}

}  // extern "C"

// ------------------------------------------------------------------------------------------------------------
// Time slice (render path; Q29): collapse the tables at one timestamp, then 8-corner lookups
// ------------------------------------------------------------------------------------------------------------
namespace {

// the plan of the D = 3 kernels on a slice: the 4D schedule's dense/hashed decision per level, three axes
int fill_slice_plan(const dash_hash4d_config* cfg, uint64_t N, uint32_t xyz_stride, uint32_t group, Plan* P) {
    if (int rc = fill_plan(cfg, N, xyz_stride, 0, group, P, 4)) return rc;
    P->dims = 3;
    for (uint32_t l = 0; l < cfg->L; ++l) P->lv[l].m[3] = 0;
    return DASH_HASH4D_OK;
}

int check_sliceable(const dash_hash4d_config* cfg) {
    if (int rc = check_config(cfg)) return rc;
    if (cfg->flags & ~static_cast<uint32_t>(DASH_HASH4D_FLAG_DENSE_COARSE))
        return fail(DASH_HASH4D_INVALID_ARG, "slice calls: only DENSE_COARSE may be set in cfg->flags");
    if ((cfg->T & (cfg->T - 1)) != 0) {
        Schedule s;
        make_schedule(cfg, &s);
        for (uint32_t l = 0; l < cfg->L; ++l)
            if (!s.dense[l])
                return fail(DASH_HASH4D_UNSUPPORTED,
                            "time slice needs a power-of-two T on hashed levels (level %u, T = %u)", l, cfg->T);
    }
    return DASH_HASH4D_OK;
}

}  // namespace

extern "C" {

DASH_API int dash_hash4d_slice_t(const dash_hash4d_config* cfg, const float* t, const void* table,
                                 float* slice, void* cuda_stream) {
    if (int rc = check_sliceable(cfg)) return rc;
    if (!t || !table || !slice) return fail(DASH_HASH4D_INVALID_ARG, "t, table or slice is NULL");
    if (!aligned16(table) || !aligned16(slice))
        return fail(DASH_HASH4D_INVALID_ARG, "table / slice not 16-byte aligned");
    Plan P;
    if (int rc = fill_plan(cfg, 1, 3, 0, 1, &P, 4)) return rc;
    cudaError_t e = dash::launch_slice_t(P, t, table, cfg->table_dtype == DASH_HASH4D_FP16, slice,
                                         static_cast<cudaStream_t>(cuda_stream));
    if (e != cudaSuccess) return cuda_fail(e, "slice launch");
    return ok();
}

DASH_API int dash_hash4d_slice_fwd(const dash_hash4d_config* cfg, uint64_t N, const float* xyz,
                                   uint32_t xyz_stride, const int32_t* index, const float* slice,
                                   float* out, void* cuda_stream) {
    if (int rc = check_sliceable(cfg)) return rc;
    if (N == 0) return ok();
    if (int rc = check_queries(xyz, xyz_stride, nullptr, 0, index, 3)) return rc;
    if (!slice || !out) return fail(DASH_HASH4D_INVALID_ARG, "slice or out is NULL");
    if (!aligned16(slice) || !aligned16(out))
        return fail(DASH_HASH4D_INVALID_ARG, "slice / out not 16-byte aligned");
    const size_t level_bytes = static_cast<size_t>(cfg->T) * cfg->F * sizeof(float);
    Plan P;
    uint32_t group = pick_group(cfg, level_bytes, DASH_DEBUG_FWD_GROUP);
    if (group > 4 && 4 * cfg->F * sizeof(float) >= 32 && !debug_u32(DASH_DEBUG_FWD_GROUP)) group = 4;
    if (int rc = fill_slice_plan(cfg, N, xyz_stride, group, &P)) return rc;
    cudaError_t e = dash::launch_fwd(P, xyz, nullptr, index, slice, false, out,
                                     static_cast<cudaStream_t>(cuda_stream));
    if (e != cudaSuccess) return cuda_fail(e, "slice fwd launch");
    return ok();
}

DASH_API size_t dash_deform_slice_workspace_bytes(const dash_hash4d_config* enc, const dash_mlp_config* mlp,
                                                  uint64_t N) {
    if (check_sliceable(enc) || check_mlp(mlp)) return 0;
    g_error[0] = '\0';
    if (deform_fused_applies(enc, true)) return 0;
    return static_cast<size_t>(N) * enc->L * enc->F * sizeof(float);
}

DASH_API int dash_deform_slice_fwd(const dash_hash4d_config* enc, const dash_mlp_config* mlp, uint64_t N,
                                   const float* xyz, uint32_t xyz_stride, const int32_t* index,
                                   const float* slice, const float* params, const float* base, float* out,
                                   void* workspace, size_t workspace_bytes, void* cuda_stream) {
    if (int rc = check_sliceable(enc)) return rc;
    if (int rc = check_mlp(mlp)) return rc;
    if (mlp->width[0] != enc->L * enc->F)
        return fail(DASH_HASH4D_INVALID_ARG, "mlp width[0] = %u != L*F = %u", mlp->width[0], enc->L * enc->F);
    dash::MlpPlan M;
    if (int rc = fill_mlp_plan(mlp, N, &M)) return rc;
    if (N == 0) return ok();
    if (int rc = check_queries(xyz, xyz_stride, nullptr, 0, index, 3)) return rc;
    if (!slice || !params || !out) return fail(DASH_HASH4D_INVALID_ARG, "slice, params or out is NULL");
    if (!aligned16(slice)) return fail(DASH_HASH4D_INVALID_ARG, "slice not 16-byte aligned");
    if ((reinterpret_cast<uintptr_t>(params) | reinterpret_cast<uintptr_t>(base) |
         reinterpret_cast<uintptr_t>(out)) & 3u)
        return fail(DASH_HASH4D_INVALID_ARG, "params / base / out not 4-byte aligned");
    if (!deform_fused_applies(enc, true)) {   // slice beyond L2: level-grouped 8-corner lookups, then the MLP kernel
        const size_t need = static_cast<size_t>(N) * enc->L * enc->F * sizeof(float);
        if (!workspace || workspace_bytes < need)
            return fail(DASH_HASH4D_WORKSPACE_TOO_SMALL,
                        "deform_slice_fwd (two-pass) needs %zu workspace bytes, got %zu", need, workspace_bytes);
        if (!aligned16(workspace)) return fail(DASH_HASH4D_INVALID_ARG, "workspace not 16-byte aligned");
        float* feat = static_cast<float*>(workspace);
        if (int rc = dash_hash4d_slice_fwd(enc, N, xyz, xyz_stride, index, slice, feat, cuda_stream)) return rc;
        cudaError_t e2 = dash::launch_mlp(M, feat, params, base, out, dash::device_sm_count(), static_cast<cudaStream_t>(cuda_stream));
        if (e2 != cudaSuccess) return cuda_fail(e2, "mlp launch");
        return ok();
    }
    Plan P;
    if (int rc = fill_slice_plan(enc, N, xyz_stride, 1, &P)) return rc;
    cudaError_t e = dash::launch_deform_fused(P, M, xyz, nullptr, index, slice, false, params, base, out,
                                              dash::device_sm_count(), static_cast<cudaStream_t>(cuda_stream));
    if (e != cudaSuccess) return cuda_fail(e, "deform slice launch");
    return ok();
}

}  // extern "C"
