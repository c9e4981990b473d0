/*
 * dash_deform.h — C ABI of the render path of DASH's 4D hash deformation field (arxiv 2507.19141, §4.2,
 * lines 133-142):
 *
 *     f_h = G_4D(x)                          Eq. 9, the hash encoder of dash_hash4d.h
 *     f_4D = phi_d(f_h)                      "followed by a tiny MLP phi_d"
 *     dx = phi_x(f_4D), dr = phi_r(f_4D), ds = phi_s(f_4D)      multi-head deformation decoder
 *     (x', r', s') = (x + dx, r + dr, s + ds)                   Eq. 10
 *
 * The paper gives neither layer sizes nor the activation.  Reading (Q27): phi_d and the heads form ONE
 * chain of n <= 4 dense layers with relu between them and none after the last,
 *     a_0 = f_h;  a_l = relu(W_l a_{l-1} + b_l) for l < n;  delta = W_n a_{n-1} + b_n;  out = base + delta,
 * the three heads being row blocks of the last layer (a block-diagonal W expresses per-head hidden layers).
 *
 * Arithmetic: the products run on the tensor cores (tcgen05.mma kind::f16): weights and each layer's input
 * vector are rounded to bfloat16 (round-to-nearest-even), products and sums are fp32, biases / base / out fp32.
 * The features f_h are formed in fp32 exactly as dash_hash4d_fwd forms them, then rounded to bf16 as the first
 * layer's input.
 *
 * Conventions as in dash_hash4d.h: device pointers, caller-owned buffers, nothing allocated or kept, work is
 * enqueued on `cuda_stream`, return codes of dash_hash4d_status, N == 0 is a no-op, no CPU fallback.
 */
#ifndef DASH_DEFORM_H_
#define DASH_DEFORM_H_

#include "dash_hash4d.h"

#ifdef __cplusplus
extern "C" {
#endif

/* The dense-layer chain.  POD, passed by pointer (host memory). */
typedef struct dash_mlp_config {
    uint32_t struct_size; /* = sizeof(dash_mlp_config)                                                       */
    uint32_t n_layers;    /* 1..4                                                                            */
    uint32_t width[5];    /* width[0]: inputs (must equal L*F in dash_deform_fwd); width[l]: outputs of layer
                             l, l = 1..n_layers; each 1..256 (internally padded to multiples of 16)          */
    uint32_t flags;       /* reserved, 0                                                                     */
} dash_mlp_config;

/* Number of floats in the packed parameter buffer [W_1 | b_1 | W_2 | b_2 | ...], W_l row-major
 * [width[l]][width[l-1]] (the layout of a torch.nn.Linear weight), b_l [width[l]].  0 on a bad config. */
DASH_API size_t dash_mlp_param_count(const dash_mlp_config* mlp);

/* out[n][j] = (base ? base[n][j] : 0) + MLP(feat[n])[j].
 *   feat    [N][width[0]] fp32.     params  packed fp32 parameters (see dash_mlp_param_count).
 *   base    nullable, [N][width[n_layers]] fp32 (the Gaussian attributes x, r, s of Eq. 10, concatenated).
 *   out     [N][width[n_layers]] fp32, written.
 * UNSUPPORTED when the bf16 weights and tile buffers of the chain exceed one SM's 227 KB of shared memory. */
DASH_API int dash_mlp_fwd(const dash_mlp_config* mlp, uint64_t N,
                          const float* feat, const float* params, const float* base,
                          float* out, void* cuda_stream);

/* Backward of dash_mlp_fwd by the chain rule (the paper trains phi_d and the heads by gradient descent on the losses
 * of PAPER.md:146-156 and gives no formulas; Q30).  With delta_n = dout, for l = n .. 1:
 *     dW_l += delta_l^T a_{l-1},   db_l += sum over rows of delta_l,
 *     g_{l-1} = delta_l W_l,   delta_{l-1} = g_{l-1} * [a_{l-1} > 0]  (relu'(0) = 0),   dfeat = g_0.
 * The forward activations are recomputed from `feat` (dash_mlp_fwd saves nothing).  Like the forward, the products run
 * on the tensor cores with bf16 operands (W, a_{l-1}, delta_l rounded to nearest even) and fp32 accumulation.
 *   feat     [N][width[0]] fp32.     params   packed fp32 parameters.     dout   [N][width[n_layers]] fp32 = dL/d out
 *            (dL/d base is dout itself).
 *   dfeat    nullable, [N][width[0]] fp32, 16-byte aligned, written: dL/d feat — the `dout` of dash_hash4d_bwd /
 *            dash_hash4d_bwd_input when feat = G_4D(x).
 *   dparams  [dash_mlp_param_count] fp32, packed like params, ACCUMULATED into (+=): the caller zeroes it.
 * UNSUPPORTED when width[0] exceeds 240 or any later width exceeds 128, or the tiles / accumulators of the chain exceed 227 KB of shared memory or
 * the 512 tensor-memory columns of an SM (accumulator + one kpad-wide weight-gradient block per layer). */
DASH_API int dash_mlp_bwd(const dash_mlp_config* mlp, uint64_t N, const float* feat, const float* params,
                          const float* dout, float* dfeat, float* dparams, void* cuda_stream);

/* Training backward of dash_deform_fwd (out = base + MLP(G_4D(x)), Eq. 9-10), composed of the calls above and of
 * include/dash_hash4d.h on `cuda_stream`; given dout = dL/d out [N][width[n_layers]]:
 *     feat   = G_4D(x)                         dash_hash4d_fwd, recomputed into the workspace
 *     dfeat, dparams += backward of the chain  dash_mlp_bwd
 *     dtable += J(x)^T dfeat                   dash_hash4d_bwd (enc->flags: DENSE_COARSE, ZERO_GRAD honoured)
 *     dq = d<dfeat, G_4D(x)>/d(x,y,z,t)        dash_hash4d_bwd_input, when dq ([N][4] fp32, overwritten) is not NULL
 * dL/d base is dout itself.  workspace: dash_deform_bwd_workspace_bytes = 2 * N * L*F * 4 bytes (+ the encoder's sort
 * workspace under SORT_COARSE), 16-byte aligned.  SORT_COARSE in enc->flags: ONE sort of the queries by coarse cell
 * (inside the forward) serves all three encoder calls (dash_hash4d_bwd and _bwd_input run with ORDER_READY).
 * enc->flags other than DENSE_COARSE | ZERO_GRAD | SORT_COARSE: INVALID_ARG.  Errors of the composed calls are passed
 * through. */
DASH_API size_t dash_deform_bwd_workspace_bytes(const dash_hash4d_config* enc, const dash_mlp_config* mlp, uint64_t N);
DASH_API int dash_deform_bwd(const dash_hash4d_config* enc, const dash_mlp_config* mlp, uint64_t N,
                             const float* xyz, uint32_t xyz_stride, const float* t, uint32_t t_stride,
                             const int32_t* index, const void* table, const float* params, const float* dout,
                             float* dtable, float* dparams, float* dq,
                             void* workspace, size_t workspace_bytes, void* cuda_stream);

/* Device workspace dash_deform_fwd needs: 0 when the fused kernel applies (the table fits L2 as one level
 * group), else N * L*F * 4 bytes for the feature matrix of the two-pass path. */
DASH_API size_t dash_deform_workspace_bytes(const dash_hash4d_config* enc, const dash_mlp_config* mlp,
                                            uint64_t N);

/* out[n] = base[n] + MLP(G_4D(x_n)): Eq. 9-10 in one call.
 * Query arguments (xyz, xyz_stride, t, t_stride, index) and `table` as in dash_hash4d_fwd; t_stride = 0 is the
 * render path's one timestamp per frame.  mlp->width[0] must equal enc->L * enc->F.
 * Fused kernel (default when L*T*F*sizeof(table element) <= 0.55 x L2): per 128-query tile the gathers write the
 * features as bf16 into shared memory, tcgen05.mma runs the layers out of shared / tensor memory, only `out`
 * goes to HBM.  Otherwise: dash_hash4d_fwd into `workspace`, then the same kernel in feature-matrix mode.
 * enc->flags: DENSE_COARSE honoured; the other flags must be clear (INVALID_ARG). */
DASH_API int dash_deform_fwd(const dash_hash4d_config* enc, const dash_mlp_config* mlp, uint64_t N,
                             const float* xyz, uint32_t xyz_stride,
                             const float* t, uint32_t t_stride,
                             const int32_t* index,
                             const void* table,
                             const float* params, const float* base,
                             float* out,
                             void* workspace, size_t workspace_bytes, void* cuda_stream);

/* ---- Time slice: the render path at ONE timestamp (the rendered frame has one t; Q29) -----
 * For a fixed t, Eq. 9 factors: the two t-layers of every level are blended ONCE per frame,
 *     hashed level (power-of-two T):  slice[l][u]  = (1-w_t) table[l][u ^ a] + w_t table[l][u ^ b],
 *                                     a = (c_t pi_t) mod T, b = ((c_t+1) pi_t) mod T      (mod 2^k commutes with XOR)
 *     dense level:                    slice[l][s3] = (1-w_t) table[l][s3 + S^3 c_t] + w_t table[l][s3 + S^3 (c_t+1)]
 * and every query then interpolates 8 instead of 16 vertices, at slot (g_x pi_x ^ g_y pi_y ^ g_z pi_z) mod T resp.
 * g_x + S(g_y + S g_z).  Same value as dash_hash4d_fwd with t_stride = 0 up to fp32 rounding; half the gathers.
 * Pays when N is not small against T (the blend streams 3 * L*T*F entries).
 *   t       DEVICE pointer to the one timestamp.       slice   [L][T][F] fp32 (written; 16-byte aligned).
 * UNSUPPORTED when a hashed level exists and T is not a power of two.  cfg->flags: DENSE_COARSE only. */
DASH_API int dash_hash4d_slice_t(const dash_hash4d_config* cfg, const float* t, const void* table,
                                 float* slice, void* cuda_stream);

/* out[n][l*F+f] = G_4D(xyz_n, t)[l*F+f] from a slice made by dash_hash4d_slice_t with the same cfg ([N][L*F] fp32). */
DASH_API int dash_hash4d_slice_fwd(const dash_hash4d_config* cfg, uint64_t N,
                                   const float* xyz, uint32_t xyz_stride, const int32_t* index,
                                   const float* slice, float* out, void* cuda_stream);

/* dash_deform_fwd on a slice: out[n] = base[n] + MLP(G_4D(xyz_n, t)).  The fused kernel with 8-corner gathers when
 * the fp32 slice (L*T*F*4 bytes) stays L2-resident; otherwise, like dash_deform_fwd, two passes (level-grouped
 * dash_hash4d_slice_fwd into the workspace, then the MLP kernel).  dash_deform_slice_workspace_bytes gives the bytes
 * that second case needs (0 when the fused kernel applies); workspace 16-byte aligned, nullable when 0. */
DASH_API size_t dash_deform_slice_workspace_bytes(const dash_hash4d_config* enc, const dash_mlp_config* mlp,
                                                  uint64_t N);
DASH_API int dash_deform_slice_fwd(const dash_hash4d_config* enc, const dash_mlp_config* mlp, uint64_t N,
                                   const float* xyz, uint32_t xyz_stride, const int32_t* index,
                                   const float* slice, const float* params, const float* base,
                                   float* out, void* workspace, size_t workspace_bytes, void* cuda_stream);

#ifdef __cplusplus
}
#endif
#endif /* DASH_DEFORM_H_ */
