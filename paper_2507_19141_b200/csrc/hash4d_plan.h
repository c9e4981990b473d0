// hash4d_plan.h — launch plan shared by the host scheduler (hash4d_api.cu) and the sm_100a kernels
// (hash4d_kernels.cu).  Plain data only.  Product code: shares nothing with oracle/.
#pragma once
#include <cstdint>

namespace dash {

constexpr int kMaxLevels = 32;
constexpr int kBlockThreads = 256;              // 8 warps
constexpr int kItemsPerBlock = kBlockThreads / 2;  // one lane PAIR per (query, level) item
constexpr int kMaxGroup = 16;                   // levels per level group (<= items per warp)

// Per-level constants (Eq. 7 resolutions; Eq. 8 multipliers or dense strides).  32 bytes.
struct LevelParams {
    float ns_f, nt_f;     // N_l of the spatial / temporal axis as binary32 (exact: N_l <= 2^22)
    uint32_t m[4];        // vertex term multipliers: hashed level -> pi_x..pi_t (Eq. 8);
                          // dense level -> 1, S, S^2, S^3 with S = Ns+1 (reading Q10)
    uint32_t dense;       // 1: slot = sum of terms; 0: slot = (XOR of terms) mod T
    uint32_t pad;
};

struct Plan {
    uint64_t N;           // queries
    uint32_t L, F, T;
    uint32_t t_mask;      // T-1 when T is a power of two
    uint32_t t_pow2;      // 1 when T is a power of two
    uint32_t xyz_stride, t_stride;
    uint32_t group;       // levels per level group G (power of two <= 16)
    uint32_t group_log2;
    uint32_t level_begin; // first level this launch covers (per-group launches), else 0
    uint32_t level_end;   // one past the last level this launch covers (L unless a launch takes a leading part)
    uint32_t num_groups;  // level groups this launch covers (gridDim.y)
    uint32_t q_per_block; // kItemsPerBlock >> group_log2
    uint32_t dims;        // 4: G_4D (x,y,z,t); 3: G_3D of the decomposition stage (x,y,z), t unused
    LevelParams lv[kMaxLevels];
};

}  // namespace dash
