/*
 * dash_hash4d.h — C ABI of the B200-native multiresolution 4D hash encoder G_4D of DASH
 * (arxiv 2507.19141, §4.2 "4D Hash Encoding", lines 123-138).
 *
 * The encoder maps a query x = (P, t) = (x, y, z, t) in [0,1)^4 to f_h = G_4D(x) in R^{L*F}
 * (Eq. 9): for each of L levels with per-axis resolutions N_l in geometric progression
 * (Eq. 7) it locates the enclosing 4D cell floor(x*N_l), maps each of
 * the cell's 16 vertices to a table slot with the spatial-temporal hash h_l = (XOR_i x_i*pi_i) mod T
 * (Eq. 8), and quadrilinearly interpolates the F-dimensional "learnable feature
 * vectors" stored there.  The backward call is the transpose of that linear map: it
 * scatter-adds upstream gradients into a table-shaped gradient buffer.  Every reading of a point the
 * paper leaves open (Q1..Q21) is listed in DESIGN.md §3.
 *
 * General conventions
 *   - All data pointers are DEVICE pointers unless marked "host".  Every buffer is caller-owned; the
 *     library allocates nothing persistent, keeps no state between calls and never frees.
 *   - Calls enqueue work on `cuda_stream` (a cudaStream_t passed as void*; NULL = default stream) and
 *     return without synchronising, except under DASH_HASH4D_FLAG_VALIDATE_INPUTS.
 *   - `table`, `out`, `dout`, `dtable`, `workspace` must be 16-byte aligned; `xyz`, `t`, `index`,
 *     `idx_out`, `w_out` 4-byte aligned.
 *   - Return codes: see dash_hash4d_status.  No exceptions, no abort.  N == 0 is DASH_HASH4D_OK and
 *     a no-op.  dash_hash4d_last_error() gives a thread-local message for the last non-OK return.
 *   - There is no CPU fallback: without a CUDA device every compute call returns
 *     DASH_HASH4D_CUDA_ERROR.
 */
#ifndef DASH_HASH4D_H_
#define DASH_HASH4D_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#if defined(_WIN32)
#define DASH_API __declspec(dllexport)
#else
#define DASH_API __attribute__((visibility("default")))
#endif

enum dash_hash4d_status {
    DASH_HASH4D_OK = 0,
    DASH_HASH4D_INVALID_ARG = 1,         /* null pointer, bad L/F/T/resolutions/stride/alignment/struct_size,
                                            or (VALIDATE_INPUTS) a NaN / out-of-[0,1) coordinate          */
    DASH_HASH4D_UNSUPPORTED = 2,         /* e.g. F not in {1,2,4,8}, N too large for one launch          */
    DASH_HASH4D_WORKSPACE_TOO_SMALL = 3, /* workspace_bytes < dash_hash4d_workspace_bytes(...)            */
    DASH_HASH4D_CUDA_ERROR = 4           /* launch / runtime error; text via dash_hash4d_last_error()    */
};

enum dash_hash4d_dtype { DASH_HASH4D_FP32 = 0, DASH_HASH4D_FP16 = 1 };

enum dash_hash4d_flags {
    DASH_HASH4D_FLAG_DENSE_COARSE = 1u,     /* levels with (Ns+1)^3 (Nt+1) <= T use the injective dense index
                                               x + S(y + S(z + S t)), S = Ns+1, instead of Eq. 8 (reading Q10).
                                               Clear => Eq. 8 literally on every level.                      */
    DASH_HASH4D_FLAG_DETERMINISTIC_BWD = 2u,/* bwd accumulates in 64-bit fixed point (order-independent):
                                               bitwise identical results run to run; needs workspace.       */
    DASH_HASH4D_FLAG_VALIDATE_INPUTS = 4u,  /* debug: scan coordinates for NaN / values outside [0,1) before
                                               the op; synchronises the stream; needs workspace.            */
    DASH_HASH4D_FLAG_ZERO_GRAD = 8u,        /* bwd OVERWRITES: the library zeroes each level group of dtable
                                               immediately before scattering into it (keeps it L2-resident)
                                               instead of accumulating into the caller's contents.          */
    DASH_HASH4D_FLAG_SORT_COARSE = 16u,     /* the high-collision case (BASELINE.json config 5; the gradient scatter is
                                               the transpose of Eq. 9).  The queries are counting-
                                               sorted by the Morton code of their 4D cell on the finest COARSE level
                                               (the last level with Ns^3 Nt <= 2N) and walked in that order:
                                                 fwd / bwd_input  every level: neighbouring lanes gather from the
                                                                  same cells and lines; values unchanged (bitwise);
                                                 bwd              the coarse levels: a segmented reduction — runs of
                                                                  queries in one cell are summed in registers, one
                                                                  vector reduction per run and corner (same sums in
                                                                  another order: same tolerance); the finer levels
                                                                  keep the caller's order.
                                               Taken only when N*F >= 2^21 and a coarse level exists, else the flag
                                               does nothing.  Needs workspace (dash_hash4d_workspace_bytes).  Honoured
                                               by dash_hash4d_fwd / _bwd / _bwd_input, their dash_hash3d_* forms (3D
                                               cells, no t in the key) and dash_deform_bwd; ignored under
                                               DETERMINISTIC_BWD and by the other calls.                          */
    DASH_HASH4D_FLAG_ORDER_READY = 32u      /* with SORT_COARSE: `workspace` still holds the order that an earlier
                                               fwd / bwd / bwd_input call with SORT_COARSE wrote for the SAME queries
                                               (N, xyz, t, index unchanged, e.g. the forward of this training step):
                                               the sort (five launches) is skipped.  A false claim gives wrong
                                               values but no out-of-bounds access.  The sort leaves a stamp (N, strides,
                                               sort key, the xyz / t / index pointers) in the workspace; together with
                                               VALIDATE_INPUTS, which synchronises anyway, the claim is checked against it
                                               and a mismatch is INVALID_ARG.  Changed CONTENTS behind unchanged pointers
                                               are not detected.                                                */
};

enum dash_hash4d_op { DASH_HASH4D_OP_FWD = 0, DASH_HASH4D_OP_BWD = 1, DASH_HASH4D_OP_INDICES = 2,
                      DASH_HASH4D_OP_BWD_INPUT = 3, DASH_HASH4D_OP_SMOOTH = 4 };

/* Encoder hyper-parameters.  POD, passed by pointer (host memory). */
typedef struct dash_hash4d_config {
    uint32_t struct_size;          /* = sizeof(dash_hash4d_config): ABI versioning                          */
    uint32_t L;                    /* number of levels, 1..32                                               */
    uint32_t F;                    /* features per table entry: 1, 2, 4 or 8                                */
    uint32_t T;                    /* entries per level (T_l of Eq. 8; uniform over levels), >= 1.
                                      Power of two uses `& (T-1)`, anything else an unsigned remainder.     */
    uint32_t res_s_min, res_s_max; /* N_min, N_max of Eq. 7 for the three spatial axes                      */
    uint32_t res_t_min, res_t_max; /* N_min, N_max of Eq. 7 for the temporal axis; all resolutions <= 2^22 */
    uint32_t primes[4];            /* pi_x, pi_y, pi_z, pi_t of Eq. 8; all zero => defaults
                                      (1, 2654435761, 805459861, 3674653429), reading Q7                    */
    uint32_t table_dtype;          /* dash_hash4d_dtype of `table`; out/dout/dtable are always fp32         */
    uint32_t flags;                /* OR of dash_hash4d_flags                                               */
} dash_hash4d_config;

/* Eq. 7: the per-level resolutions N_l = floor(N_min * b^l), b = (N_max/N_min)^(1/(L-1)),
 * for the spatial and the temporal range, and which levels use the dense index (reading Q10).
 * res_s, res_t: host arrays of L uint32 (written).  is_dense: host array of L bytes, nullable.
 * Returns INVALID_ARG on a bad config or null output pointer.  Needs no GPU. */
DASH_API int dash_hash4d_resolutions(const dash_hash4d_config* cfg, uint32_t* res_s, uint32_t* res_t,
                                     uint8_t* is_dense);

/* Bytes of device workspace `op` needs for N queries under cfg->flags (0 for the default paths; SORT_COARSE:
 * 24 bytes per query + the sort's bins, the same for OP_FWD and OP_BWD so that one buffer serves a step).
 * Returns 0 on a bad config as well.  Needs no GPU. */
DASH_API size_t dash_hash4d_workspace_bytes(const dash_hash4d_config* cfg, uint64_t N, int op);
/* The same for the dash_hash3d_* calls (op: DASH_HASH4D_OP_FWD / _BWD / _BWD_INPUT / _INDICES); the temporal fields of cfg
 * are ignored, as in those calls. */
DASH_API size_t dash_hash3d_workspace_bytes(const dash_hash4d_config* cfg, uint64_t N, int op);

/* Forward, Eq. 9:  out[n][l*F + f] = sum_{k<16} W_k * table[l][slot_k][f].
 *   N          number of queries.
 *   xyz        query n reads the three floats at xyz + row*xyz_stride, row = index ? index[n] : n;
 *              xyz_stride (in floats) is 3 or 4.
 *   t          query n reads t[n * t_stride]; t_stride is 0 (one timestamp for the whole call), 1 or 4.
 *              A packed [N][4] array is the view xyz = base, xyz_stride = 4, t = base + 3, t_stride = 4.
 *   index      nullable int32 [N] row list (the dynamic subset of PAPER.md:111); rows must be valid.
 *   table      [L][T][F] row-major, element type cfg->table_dtype (read only).
 *   out        [N][L*F] fp32, level-major columns (written, every element).
 *   workspace  only read when dash_hash4d_workspace_bytes(cfg, N, OP_FWD) > 0.
 * Coordinates are clamped to [0, 1-2^-24], NaN -> 0 (reading Q12).  fp16 tables are converted to fp32
 * exactly; weights, products and sums are fp32 (reading Q13). */
DASH_API int dash_hash4d_fwd(const dash_hash4d_config* cfg, uint64_t N,
                             const float* xyz, uint32_t xyz_stride,
                             const float* t, uint32_t t_stride,
                             const int32_t* index,
                             const void* table,
                             float* out,
                             void* workspace, size_t workspace_bytes, void* cuda_stream);

/* Backward (table gradient), the transpose of Eq. 9:
 *     dtable[l][slot_k][f] += W_k * dout[n][l*F + f]      for every query n, level l, corner k.
 *   dout       [N][L*F] fp32 upstream gradient (read only).
 *   dtable     [L][T][F] fp32, ACCUMULATED into (+=) — the caller zeroes it (dash_hash4d_zero) unless
 *              DASH_HASH4D_FLAG_ZERO_GRAD is set, in which case it is overwritten.
 * Default path: fp32 vector reductions at L2 (`red.global.add.v2/.v4.f32`): summation order, hence the
 * last bits, vary run to run; subnormal partial sums flush to zero.  DETERMINISTIC_BWD: 64-bit
 * fixed-point accumulation in `workspace`, bitwise reproducible.  SORT_COARSE: see the flag; the sort (five launches)
 * and the run-merged scatter run inside this call, on `cuda_stream`, in `workspace`.  Other arguments as in fwd. */
DASH_API int dash_hash4d_bwd(const dash_hash4d_config* cfg, uint64_t N,
                             const float* xyz, uint32_t xyz_stride,
                             const float* t, uint32_t t_stride,
                             const int32_t* index,
                             const float* dout,
                             float* dtable,
                             void* workspace, size_t workspace_bytes, void* cuda_stream);

/* Coordinate gradient (not in the paper, which is silent on whether gradients reach the Gaussian
 * positions through G_4D — PAPER.md:140-144 makes x both encoder input and learnable; Q24):
 *     dq[n][d] = sum_{l,f} dout[n][l*F+f] * d out[n][l*F+f] / d x_d ,   d = 0:x 1:y 2:z 3:t,
 * with d out / d x_d = N_{l,d} * sum_k s_d(k) prod_{e != d} omega_e(k) table[l][slot_k][f] on the open cell
 * (the one-sided derivative from the right at a grid vertex).  A coordinate changed by the clamp
 * (NaN, < 0, > 1-2^-24) gets 0.
 *   dq         [N][4] fp32, OVERWRITTEN (the library zeroes it, then adds one partial sum per level group).
 *              Per QUERY, not per xyz row: with an index list the caller reduces rows itself.
 * Other arguments as in fwd. */
DASH_API int dash_hash4d_bwd_input(const dash_hash4d_config* cfg, uint64_t N,
                                   const float* xyz, uint32_t xyz_stride,
                                   const float* t, uint32_t t_stride,
                                   const int32_t* index,
                                   const void* table,
                                   const float* dout,
                                   float* dq,
                                   void* workspace, size_t workspace_bytes, void* cuda_stream);

/* Smoothness regulariser, Eq. 11:  L_r = || G_4D(x) - G_4D(x + eps_x) ||_2^2.
 *   eps        the "small random perturbation" eps_x = (eps_P, eps_t), DRAWN BY THE CALLER: query n reads
 *              eps[n*eps_stride + d], d = 0..3; eps_stride (in floats) is 4, or 0 for one perturbation shared
 *              by all queries.  The perturbed query is x'_d = fl32(x_d + eps_d), then clamped like any query.
 *   loss       [N] fp32, OVERWRITTEN: loss[n] = sum over the L*F features of (G(x_n) - G(x'_n))^2 — the plain
 *              squared norm, nothing averaged or scaled (reading Q25).
 *   dtable     nullable; [L][T][F] fp32, ACCUMULATED: += grad_scale * d(sum_n loss[n]) / d table
 *              = grad_scale * 2 * sum_n (J(x_n)^T d_n - J(x'_n)^T d_n),  d_n = G(x_n) - G(x'_n)
 *              (pass lambda_r of Eq. 12 as grad_scale; call after dash_hash4d_bwd to add into the same buffer).
 * One fused pass: where x and x' share a cell (coarse levels, small eps) the 16 corners are gathered once
 * and scattered once with weight (W - W').  DETERMINISTIC_BWD is not supported here (UNSUPPORTED when
 * dtable != NULL); ZERO_GRAD is ignored.  Other arguments as in fwd. */
DASH_API int dash_hash4d_smooth(const dash_hash4d_config* cfg, uint64_t N,
                                const float* xyz, uint32_t xyz_stride,
                                const float* t, uint32_t t_stride,
                                const int32_t* index,
                                const float* eps, uint32_t eps_stride,
                                const void* table,
                                float grad_scale,
                                float* loss,
                                float* dtable,
                                void* workspace, size_t workspace_bytes, void* cuda_stream);

/* Debug: the 16 table slots and interpolation weights of every (query, level)
 * (Eq. 8).  Corner k: bit d of k set => vertex floor(x_d*N_l)+1 along axis d,
 * d = 0:x 1:y 2:z 3:t (readings Q5, Q6).
 *   idx_out    [N][L][16] uint32 (written).     w_out  [N][L][16] fp32, nullable. */
DASH_API int dash_hash4d_indices(const dash_hash4d_config* cfg, uint64_t N,
                                 const float* xyz, uint32_t xyz_stride,
                                 const float* t, uint32_t t_stride,
                                 const int32_t* index,
                                 uint32_t* idx_out, float* w_out, void* cuda_stream);

/* ---- G_3D: the 3D hash encoder of the decomposition stage (Eq. 3: "a 3D hash encoder
 * G_3D from Instant-NGP"; Q26) -------------------------------------------------------------------
 * Eq. 7-9 with d = 3: per level the cell floor(p * Ns_l) of a point p = (x,y,z), its 8 vertices hashed with
 * pi_x, pi_y, pi_z (Eq. 8) or, where (Ns_l+1)^3 <= T and DENSE_COARSE is set, indexed gx + S(gy + S gz),
 * S = Ns_l+1; trilinear weights; levels concatenated to R^{L*F}.  The same config struct is used; its temporal
 * fields (res_t_min, res_t_max, primes[3]) are ignored.  Same kernels as the 4D path with 4 instead of 8
 * corners per lane, same level-group-major schedule, flags (ZERO_GRAD, DETERMINISTIC_BWD, VALIDATE_INPUTS),
 * alignment, ownership, error and N == 0 behaviour as dash_hash4d_fwd / _bwd / _indices.
 *   idx_out / w_out of dash_hash3d_indices: [N][L][8], corner k bit d => +1 along axis d (0:x 1:y 2:z).
 *   dash_hash3d_resolutions: res_s [L] host (written), is_dense [L] host, nullable.  Needs no GPU. */
DASH_API int dash_hash3d_resolutions(const dash_hash4d_config* cfg, uint32_t* res_s, uint8_t* is_dense);
DASH_API int dash_hash3d_fwd(const dash_hash4d_config* cfg, uint64_t N,
                             const float* xyz, uint32_t xyz_stride,
                             const int32_t* index,
                             const void* table,
                             float* out,
                             void* workspace, size_t workspace_bytes, void* cuda_stream);
DASH_API int dash_hash3d_bwd(const dash_hash4d_config* cfg, uint64_t N,
                             const float* xyz, uint32_t xyz_stride,
                             const int32_t* index,
                             const float* dout,
                             float* dtable,
                             void* workspace, size_t workspace_bytes, void* cuda_stream);
/* Coordinate gradient of G_3D: dq[n][d] = d<dout[n], G_3D(p_n)>/dp_d, d = x,y,z; dq [N][3] fp32 (overwritten, 4-byte
 * aligned).  The D = 3 form of dash_hash4d_bwd_input (reading Q24: one-sided at vertices, 0 for a clamped coordinate). */
DASH_API int dash_hash3d_bwd_input(const dash_hash4d_config* cfg, uint64_t N,
                                   const float* xyz, uint32_t xyz_stride, const int32_t* index,
                                   const void* table, const float* dout, float* dq,
                                   void* workspace, size_t workspace_bytes, void* cuda_stream);
DASH_API int dash_hash3d_indices(const dash_hash4d_config* cfg, uint64_t N,
                                 const float* xyz, uint32_t xyz_stride,
                                 const int32_t* index,
                                 uint32_t* idx_out, float* w_out, void* cuda_stream);

/* ---- Sparse optimiser step over the touched table entries (Q28) -------------------
 * The paper does not name its optimiser; 3DGS [14] and Instant-NGP [25], which it builds on, train with Adam.
 * Adam (bias-corrected) applied only to entries whose gradient is not exactly zero; an entry no query touched
 * keeps theta, m and v unchanged (the rule of torch.optim.SparseAdam), and is not even read beyond its gradient:
 *     m <- beta1 m + (1-beta1) g;  v <- beta2 v + (1-beta2) g^2;
 *     theta <- theta - lr * (m / (1-beta1^t)) / (sqrt(v / (1-beta2^t)) + eps)          (fp32 arithmetic). */
typedef struct dash_adam_config {
    uint32_t struct_size; /* = sizeof(dash_adam_config)                                                     */
    uint32_t step;        /* t >= 1, the global step count of the bias correction                           */
    float lr, beta1, beta2, eps;
    uint32_t flags;       /* bit0 DASH_ADAM_ZERO_GRAD: set every touched gradient entry to 0 afterwards, so
                             the buffer is all-zero again and the next backward can accumulate into it      */
} dash_adam_config;
enum dash_adam_flags { DASH_ADAM_ZERO_GRAD = 1u };

/*   theta    [L][T][F] fp32 master parameters (read/written).  For a fp32 table this IS the table.
 *   table16  nullable; [L][T][F] IEEE half: receives the rounding of every updated theta (the fp16 table the
 *            encoder reads).  Untouched entries are not rewritten.
 *   dtable   [L][T][F] fp32 gradient (read; zeroed where touched under DASH_ADAM_ZERO_GRAD).
 *   m, v     [L][T][F] fp32 first / second moments (read/written where touched).
 * All five 16-byte aligned.  Only cfg->L, T, F are used. */
DASH_API int dash_hash4d_adam_step(const dash_hash4d_config* cfg, const dash_adam_config* opt,
                                   float* theta, void* table16, float* dtable, float* m, float* v,
                                   void* cuda_stream);

/* Optional helper: a spatial ordering of the queries (the counting sort SURVEY.md §7 step 7 asks to be decided on a
 * kernel; measured in profiles/experiments_r02.md §5).  Key of query n = Morton code of floor(clamp(x_d) * 2^bits) over
 * the three spatial axes of its row (row = index ? index[n] : n); `order` ([N] int32, written) receives the query
 * numbers n sorted by non-decreasing key (ties in no particular order).  Nothing else changes: a caller that wants its
 * queries processed in this order passes `order` (composed with its own index list) as `index` and permutes t / dout
 * alike.  bits: 1..7.  workspace: dash_hash4d_sort_workspace_bytes(N, bits) bytes, 16-byte aligned.  Hand-written
 * histogram + scan + scatter, five launches on `cuda_stream`; PAPER.md:111 (the dynamic subset is an index list). */
DASH_API size_t dash_hash4d_sort_workspace_bytes(uint64_t N, uint32_t bits);
DASH_API int dash_hash4d_sort_queries(uint64_t N, const float* xyz, uint32_t xyz_stride, const int32_t* index,
                                      uint32_t bits, int32_t* order, void* workspace, size_t workspace_bytes,
                                      void* cuda_stream);

/* dash_hash4d_sort_queries for callers that are not able to allocate device memory.
 *
 * Who that is: code that runs inside somebody else's GPU budget.  A plug-in of a renderer or trainer is handed its input
 * and output buffers by the host application, which owns every other byte of HBM through its own pool; a per-frame loop
 * (the paper renders at 264 FPS) must not call cudaMalloc / cudaFree because they serialise the whole device
 * and stall every other stream; and on a GPU whose memory is already committed to tables and Gaussians a late cudaMalloc
 * can simply fail.  Such a caller has nowhere to get the `workspace` that dash_hash4d_sort_queries asks for.
 *
 * This call needs none: the sort's scratch (a key per query, the histogram bins, the scan totals) is a fixed array inside
 * the library's own device data segment.  The call itself runs no cudaMalloc, cudaFree or any allocating library routine.
 *   - The array is DASH_HASH4D_SORT_STATIC_MAX_N * 4 + 8^DASH_HASH4D_SORT_STATIC_MAX_BITS * 4 + 1024 bytes (5 243 904 B,
 *     about 5 MB).  Every GPU on which this process uses the library carries it from the moment the library's device code
 *     is loaded there until the process exits, whether or not this call is ever made.
 *   - Limits: N <= DASH_HASH4D_SORT_STATIC_MAX_N and bits <= DASH_HASH4D_SORT_STATIC_MAX_BITS.  Anything larger returns
 *     DASH_HASH4D_UNSUPPORTED with a message naming the limit (nothing is launched); use dash_hash4d_sort_queries then.
 *   - The first call on each device looks up where the array lives on that device (cudaGetSymbolAddress, with that device
 *     current) and remembers it; make that first call before starting any stream capture on that device.
 *   - All calls on a device share the one array, and it keeps the previous call's contents; each call re-zeroes the part
 *     it counts into, so back-to-back calls on one stream are fine.  Two calls that may execute on the GPU at the same
 *     time (different streams, or different host threads on different streams) race on it and give a wrong `order`:
 *     serialise them yourself.
 * Arguments, key, result (`order` = query numbers by non-decreasing Morton key, ties in any order), launches (five, on
 * `cuda_stream`, no synchronisation) and N == 0 behaviour are those of dash_hash4d_sort_queries. */
#define DASH_HASH4D_SORT_STATIC_MAX_N 1048576ull /* 2^20 queries */
#define DASH_HASH4D_SORT_STATIC_MAX_BITS 6       /* 2^18 bins    */
DASH_API int dash_hash4d_sort_queries_static(uint64_t N, const float* xyz, uint32_t xyz_stride, const int32_t* index,
                                             uint32_t bits, int32_t* order, void* cuda_stream);

/* dtable <- 0 for the whole [L][T][F] fp32 gradient buffer (the accumulation's initial state), with the
 * library's own fill kernel on `cuda_stream`. */
DASH_API int dash_hash4d_zero(const dash_hash4d_config* cfg, float* dtable, void* cuda_stream);

/* Thread-local, never NULL; empty string when the last call on this thread succeeded. */
DASH_API const char* dash_hash4d_last_error(void);

/* Number of kernels the library launched on this thread since the last call with reset != 0
 * (used by bench.py for "gpu_launches"). */
DASH_API uint64_t dash_hash4d_launch_count(int reset);

/* Hash of the sources the library was built from (never NULL).  The Python binding compares it with the sources
 * beside it and refuses (rebuilds, else raises) a library that is out of date. */
DASH_API const char* dash_hash4d_build_id(void);

#ifdef __cplusplus
}
#endif
#endif /* DASH_HASH4D_H_ */
