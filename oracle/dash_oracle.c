/*
 * dash_oracle.c — CPU ORACLE for the DASH multiresolution 4D hash encoder G_4D.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may load it.  It shares no code, header,
 * table or constant generator with the CUDA path (paper_2507_19141_b200/csrc, include/).
 *
 * What it computes: the plain definition of, written out in the paper's order
 *   Eq. 7  resolution schedule N_l            -> dash_oracle_resolutions
 *   PAPER.md:129           cell location  floor(x * N_l)      -> locate()
 *   Eq. 8  spatial-temporal hash of a vertex  -> vertex_slot()
 *   PAPER.md:133 / Eq. 9   quadrilinear interpolation, levels concatenated to f_h in R^{LF}
 *                                                              -> dash_oracle_fwd
 *   PAPER.md:133 ("learnable feature vectors"): the transpose of that linear map, i.e. the
 *   table gradient dtable[l][h] += W * dY                      -> dash_oracle_bwd
 * Where the paper is silent or garbled the reading taken is the numbered one in DESIGN.md §3
 * (Q1..Q21); each is marked "Q<n>" below.
 *
 * Precision: cell location is ONE binary32 multiply (Q4) so that indices are a bit-exact
 * contract; interpolation weights, feature sums and gradient sums are formed in double and
 * rounded to fp32 once (Q11, Q14).  No blocking, no SIMD, no reordering.  OpenMP only splits
 * independent work: queries in fwd/indices, levels (disjoint tables) in bwd.
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): printed resolution lists, hand-derived hash
 * values, dense-index bijection by brute force, weights sum to 1, exact table value at grid
 * vertices, multi-affine reproduction, scipy RegularGridInterpolator on dense levels,
 * linearity, adjoint identity, finite differences, pure-Python brute force on tiny inputs.
 * Parity with the paper's OWN (unavailable) CUDA code on hashed levels: "parity unpinned"
 * (its primes / scale convention are not in the paper) — see DESIGN.md §3.
 *
 * Build: gcc -O2 -std=c11 -fopenmp -ffp-contract=off -shared -fPIC (oracle/build.py).
 */
#include <math.h>
#include <stddef.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct dash_oracle_config {
    uint32_t struct_size;
    uint32_t L, F, T;
    uint32_t res_s_min, res_s_max;
    uint32_t res_t_min, res_t_max;
    uint32_t primes[4];
    uint32_t table_dtype; /* 0 fp32, 1 fp16 */
    uint32_t flags;       /* bit0: dense indexing on coarse levels (Q10) */
} dash_oracle_config;

enum { ORACLE_OK = 0, ORACLE_INVALID = 1, ORACLE_NOMEM = 5 };
#define ORACLE_MAX_L 32

/* Q7: default multipliers (pi_1 = 1 keeps x-neighbours adjacent; the other three are large primes) */
static const uint32_t k_default_primes[4] = {1u, 2654435761u, 805459861u, 3674653429u};

static int config_ok(const dash_oracle_config *c) {
    if (!c || c->struct_size != sizeof(dash_oracle_config)) return 0;
    if (c->L < 1 || c->L > ORACLE_MAX_L) return 0;
    if (!(c->F == 1 || c->F == 2 || c->F == 4 || c->F == 8)) return 0;
    if (c->T < 1) return 0;
    if (c->res_s_min < 1 || c->res_s_min > c->res_s_max) return 0;
    if (c->res_t_min < 1 || c->res_t_min > c->res_t_max) return 0;
    if (c->table_dtype > 1) return 0;
    return 1;
}

static void get_primes(const dash_oracle_config *c, uint32_t pi[4]) {
    int all_zero = !(c->primes[0] | c->primes[1] | c->primes[2] | c->primes[3]);
    for (int d = 0; d < 4; ++d) pi[d] = all_zero ? k_default_primes[d] : c->primes[d];
}

/* Eq. 7 read as N_l = floor(N_min * b^l), b = exp((ln N_max - ln N_min)/(L-1))
 * (Q1: the exponent l is lost in the extracted text; "geometric progression").
 * Q2: evaluated in IEEE double as N_min * pow(N_max/N_min, l/(L-1)), floor(r + 1e-6) so that
 * levels that are mathematically integers (64, 128, 300, 4096 ...) do not fall one short. */
static uint32_t level_resolution(uint32_t n_min, uint32_t n_max, uint32_t l, uint32_t L) {
    if (L == 1) return n_min;
    double r = (double)n_min * pow((double)n_max / (double)n_min, (double)l / (double)(L - 1));
    return (uint32_t)floor(r + 1e-6);
}

/* Q10: a level is dense iff its vertex count (Ns+1)^3 (Nt+1) fits in T. */
static int level_is_dense(const dash_oracle_config *c, uint32_t ns, uint32_t nt) {
    if (!(c->flags & 1u)) return 0;
    long double v = (long double)(ns + 1.0L) * (ns + 1.0L) * (ns + 1.0L) * (nt + 1.0L);
    return v <= (long double)c->T;
}

int dash_oracle_resolutions(const dash_oracle_config *c, uint32_t *res_s, uint32_t *res_t,
                            uint8_t *is_dense) {
    if (!config_ok(c) || !res_s || !res_t) return ORACLE_INVALID;
    for (uint32_t l = 0; l < c->L; ++l) {
        res_s[l] = level_resolution(c->res_s_min, c->res_s_max, l, c->L); /* Q3: spatial range */
        res_t[l] = level_resolution(c->res_t_min, c->res_t_max, l, c->L); /* Q3: temporal range */
        if (is_dense) is_dense[l] = (uint8_t)level_is_dense(c, res_s[l], res_t[l]);
    }
    return ORACLE_OK;
}

/* Q12: inputs live in [0,1); clamp to [0, 1-2^-24], NaN -> 0. */
static float clamp_unit(float v) {
    if (isnan(v)) return 0.0f;
    if (v < 0.0f) return 0.0f;
    if (v > 0x1.fffffep-1f) return 0x1.fffffep-1f;
    return v;
}

/* floor(x_l) = floor(x * N_l).  Q4: one binary32 multiply, no offset.
 * (volatile + -ffp-contract=off keep the compiler from widening or fusing it.) */
static void locate(float x, uint32_t n, uint32_t *cell, float *frac) {
    volatile float pos = x * (float)n;
    float fl = floorf(pos);
    *cell = (uint32_t)fl;
    *frac = pos - fl; /* exact in fp32 */
}

/* Eq. 8: h = (XOR_i g_i * pi_i) mod T, products in uint32 wraparound (Q8),
 * uniform T (Q9); or the dense injective index on coarse levels (Q10), x fastest. */
static uint32_t vertex_slot(const uint32_t g[4], const uint32_t pi[4], uint32_t T, int dense,
                            uint32_t ns) {
    if (dense) {
        uint32_t S = ns + 1u;
        return g[0] + S * (g[1] + S * (g[2] + S * g[3]));
    }
    uint32_t h = 0;
    for (int d = 0; d < 4; ++d) h ^= g[d] * pi[d];
    return h % T;
}

/* Q13: IEEE half -> double, exact, by the format's definition. */
static double half_to_double(uint16_t h) {
    int sign = (h >> 15) & 1, e = (h >> 10) & 0x1f, m = h & 0x3ff;
    double v;
    if (e == 0) v = ldexp((double)m, -24);
    else if (e == 31) v = m ? NAN : INFINITY;
    else v = ldexp((double)(m + 1024), e - 25);
    return sign ? -v : v;
}

typedef struct {
    uint32_t res_s[ORACLE_MAX_L], res_t[ORACLE_MAX_L];
    uint8_t dense[ORACLE_MAX_L];
    uint32_t pi[4];
} level_plan;

static int make_plan(const dash_oracle_config *c, level_plan *p) {
    int rc = dash_oracle_resolutions(c, p->res_s, p->res_t, p->dense);
    if (rc) return rc;
    get_primes(c, p->pi);
    return ORACLE_OK;
}

/* Steps 1-5 of DESIGN.md §2 for one (query, level): the 16 slots and 16 weights.
 * Corner k: bit d of k set => +1 along dimension d, d = 0:x 1:y 2:z 3:t (Q5, Q6). */
static void corners(const dash_oracle_config *c, const level_plan *p, uint32_t l,
                    const float q[4], uint32_t slot[16], double W[16]) {
    uint32_t cell[4];
    float frac[4];
    for (int d = 0; d < 4; ++d) {
        uint32_t n = (d < 3) ? p->res_s[l] : p->res_t[l];
        locate(clamp_unit(q[d]), n, &cell[d], &frac[d]);
    }
    for (int k = 0; k < 16; ++k) {
        uint32_t g[4];
        double w = 1.0;
        for (int d = 0; d < 4; ++d) {
            int up = (k >> d) & 1;
            g[d] = cell[d] + (uint32_t)up; /* Q5: upper corner is floor+1 always */
            w *= up ? (double)frac[d] : 1.0 - (double)frac[d];
        }
        slot[k] = vertex_slot(g, p->pi, c->T, p->dense[l], p->res_s[l]);
        W[k] = w;
    }
}

static void fetch_query(uint64_t n, const float *xyz, uint32_t xyz_stride, const float *t,
                        uint32_t t_stride, const int32_t *index, float q[4]) {
    uint64_t row = index ? (uint64_t)index[n] : n;
    q[0] = xyz[row * xyz_stride + 0];
    q[1] = xyz[row * xyz_stride + 1];
    q[2] = xyz[row * xyz_stride + 2];
    q[3] = t[n * (uint64_t)t_stride]; /* Q21: t_stride 0 = one timestamp for all */
}

static int args_ok(const float *xyz, uint32_t xyz_stride, const float *t, uint32_t t_stride) {
    if (!xyz || !t) return 0;
    if (!(xyz_stride == 3 || xyz_stride == 4)) return 0;
    if (!(t_stride == 0 || t_stride == 1 || t_stride == 4)) return 0;
    return 1;
}

/* idx_out [N][L][16] u32; w_out [N][L][16] double (nullable). */
int dash_oracle_indices(const dash_oracle_config *c, uint64_t N, const float *xyz,
                        uint32_t xyz_stride, const float *t, uint32_t t_stride,
                        const int32_t *index, uint32_t *idx_out, double *w_out) {
    level_plan p;
    if (!config_ok(c) || make_plan(c, &p)) return ORACLE_INVALID;
    if (N == 0) return ORACLE_OK;
    if (!args_ok(xyz, xyz_stride, t, t_stride) || !idx_out) return ORACLE_INVALID;
#pragma omp parallel for schedule(static)
    for (int64_t n = 0; n < (int64_t)N; ++n) {
        float q[4];
        fetch_query((uint64_t)n, xyz, xyz_stride, t, t_stride, index, q);
        for (uint32_t l = 0; l < c->L; ++l) {
            uint32_t slot[16];
            double W[16];
            corners(c, &p, l, q, slot, W);
            size_t base = ((size_t)n * c->L + l) * 16;
            for (int k = 0; k < 16; ++k) {
                idx_out[base + k] = slot[k];
                if (w_out) w_out[base + k] = W[k];
            }
        }
    }
    return ORACLE_OK;
}

static double table_value(const dash_oracle_config *c, const void *table, uint32_t l,
                          uint32_t slot, uint32_t f) {
    size_t e = ((size_t)l * c->T + slot) * c->F + f; /* D1: [L][T][F] */
    if (c->table_dtype == 1) return half_to_double(((const uint16_t *)table)[e]);
    return (double)((const float *)table)[e];
}

/* Eq. 9: out[n][l*F+f] = sum_k W_k * table[l][slot_k][f]  (Q11: level-major).
 * out_abs (nullable, [N][L*F] double) receives sum_k |W_k * v_k| — the conditioning term A of
 * the elementwise tolerance (DESIGN.md §3 Q17). */
int dash_oracle_fwd(const dash_oracle_config *c, uint64_t N, const float *xyz, uint32_t xyz_stride,
                    const float *t, uint32_t t_stride, const int32_t *index, const void *table,
                    float *out, double *out_abs) {
    level_plan p;
    if (!config_ok(c) || make_plan(c, &p)) return ORACLE_INVALID;
    if (N == 0) return ORACLE_OK;
    if (!args_ok(xyz, xyz_stride, t, t_stride) || !table || !out) return ORACLE_INVALID;
    const uint32_t L = c->L, F = c->F;
#pragma omp parallel for schedule(static)
    for (int64_t n = 0; n < (int64_t)N; ++n) {
        float q[4];
        fetch_query((uint64_t)n, xyz, xyz_stride, t, t_stride, index, q);
        for (uint32_t l = 0; l < L; ++l) {
            uint32_t slot[16];
            double W[16];
            corners(c, &p, l, q, slot, W);
            for (uint32_t f = 0; f < F; ++f) {
                double acc = 0.0, mag = 0.0;
                for (int k = 0; k < 16; ++k) {
                    double term = W[k] * table_value(c, table, l, slot[k], f);
                    acc += term;
                    mag += fabs(term);
                }
                size_t o = (size_t)n * L * F + (size_t)l * F + f;
                out[o] = (float)acc; /* rounded to fp32 once */
                if (out_abs) out_abs[o] = mag;
            }
        }
    }
    return ORACLE_OK;
}

/* Transpose of Eq. 9: dtable[l][slot_k][f] += W_k * dout[n][l*F+f]   (Q15: accumulate).
 * Per level: a double accumulator over the whole level, queries in order n = 0..N-1, rounded to
 * fp32 once and added to the caller's dtable.  grad_abs (nullable, [L][T][F] double) receives
 * sum |W * dY| per entry; hits (nullable, [L][T] u32) the number of contributions per slot. */
int dash_oracle_bwd(const dash_oracle_config *c, uint64_t N, const float *xyz, uint32_t xyz_stride,
                    const float *t, uint32_t t_stride, const int32_t *index, const float *dout,
                    float *dtable, double *grad_abs, uint32_t *hits) {
    level_plan p;
    if (!config_ok(c) || make_plan(c, &p)) return ORACLE_INVALID;
    if (N == 0) return ORACLE_OK;
    if (!args_ok(xyz, xyz_stride, t, t_stride) || !dout || !dtable) return ORACLE_INVALID;
    const uint32_t L = c->L, F = c->F;
    const size_t TF = (size_t)c->T * F;
    int failed = 0;
#pragma omp parallel for schedule(dynamic, 1)
    for (int32_t l = 0; l < (int32_t)L; ++l) {
        double *acc = (double *)calloc(TF, sizeof(double));
        double *mag = grad_abs ? grad_abs + (size_t)l * TF : NULL;
        uint32_t *cnt = hits ? hits + (size_t)l * c->T : NULL;
        if (!acc) {
            failed = 1;
            continue;
        }
        if (mag) memset(mag, 0, TF * sizeof(double));
        if (cnt) memset(cnt, 0, (size_t)c->T * sizeof(uint32_t));
        for (uint64_t n = 0; n < N; ++n) {
            float q[4];
            uint32_t slot[16];
            double W[16];
            fetch_query(n, xyz, xyz_stride, t, t_stride, index, q);
            corners(c, &p, (uint32_t)l, q, slot, W);
            for (int k = 0; k < 16; ++k) {
                for (uint32_t f = 0; f < F; ++f) {
                    double term = W[k] * (double)dout[(size_t)n * L * F + (size_t)l * F + f];
                    acc[(size_t)slot[k] * F + f] += term;
                    if (mag) mag[(size_t)slot[k] * F + f] += fabs(term);
                }
                if (cnt) cnt[slot[k]] += 1u;
            }
        }
        float *dst = dtable + (size_t)l * TF;
        for (size_t e = 0; e < TF; ++e) dst[e] = (float)((double)dst[e] + acc[e]);
        free(acc);
    }
    return failed ? ORACLE_NOMEM : ORACLE_OK;
}

int dash_oracle_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void dash_oracle_set_threads(int n) {
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

/* ---- debug exports used only by the pin tests ---- */

/* Slot of grid vertex g = (gx,gy,gz,gt) at level l (Eq. 8 or the dense index). */
int dash_oracle_vertex_slot(const dash_oracle_config *c, uint32_t l, const uint32_t g[4],
                            uint32_t *slot) {
    level_plan p;
    if (!config_ok(c) || make_plan(c, &p) || l >= c->L || !g || !slot) return ORACLE_INVALID;
    *slot = vertex_slot(g, p.pi, c->T, p.dense[l], p.res_s[l]);
    return ORACLE_OK;
}

/* Cell and fractional offset of coordinate x at resolution n (after the Q12 clamp). */
void dash_oracle_locate(float x, uint32_t n, uint32_t *cell, float *frac) {
    locate(clamp_unit(x), n, cell, frac);
}

double dash_oracle_half_to_double(uint16_t h) { return half_to_double(h); }

/* ---- NEXT #1: gradient with respect to the query coordinates -------------------
 * The paper is silent on whether gradients flow through G_4D into the Gaussian positions
 * (DESIGN.md §3 Q14); PAPER.md:140-144 makes x both the encoder input and a learnable quantity.
 * Inside a cell Eq. 9 is multilinear in the fractional offsets w_d = x_d*N_{l,d} - c_d, so
 *   d out[n][l*F+f] / d x_d = N_{l,d} * sum_k s_d(k) * prod_{d' != d} omega_{d'}(k) * table[l][slot_k][f]
 * with omega_d(k) = (bit_d(k) ? w_d : 1-w_d), s_d(k) = (bit_d(k) ? +1 : -1), and
 *   dq[n][d] = sum_{l,f} dout[n][l*F+f] * d out[n][l*F+f] / d x_d.
 * The derivative is taken on the open cell (one-sided from the right at a vertex, because c = floor);
 * a coordinate that the Q12 clamp moved (NaN, < 0, > 1-2^-24) has derivative 0.
 * dq: [N][4] fp32 (x,y,z,t), overwritten.  dq_abs (nullable, [N][4] double): sum of |terms|. */
int dash_oracle_bwd_input(const dash_oracle_config *c, uint64_t N, const float *xyz,
                          uint32_t xyz_stride, const float *t, uint32_t t_stride,
                          const int32_t *index, const void *table, const float *dout, float *dq,
                          double *dq_abs) {
    level_plan p;
    if (!config_ok(c) || make_plan(c, &p)) return ORACLE_INVALID;
    if (N == 0) return ORACLE_OK;
    if (!args_ok(xyz, xyz_stride, t, t_stride) || !table || !dout || !dq) return ORACLE_INVALID;
    const uint32_t L = c->L, F = c->F;
#pragma omp parallel for schedule(static)
    for (int64_t n = 0; n < (int64_t)N; ++n) {
        float q[4];
        fetch_query((uint64_t)n, xyz, xyz_stride, t, t_stride, index, q);
        double acc[4] = {0, 0, 0, 0}, mag[4] = {0, 0, 0, 0};
        for (uint32_t l = 0; l < L; ++l) {
            uint32_t cell[4];
            float frac[4];
            double res[4];
            for (int d = 0; d < 4; ++d) {
                uint32_t nres = (d < 3) ? p.res_s[l] : p.res_t[l];
                locate(clamp_unit(q[d]), nres, &cell[d], &frac[d]);
                res[d] = (double)nres;
            }
            for (int k = 0; k < 16; ++k) {
                uint32_t g[4];
                for (int d = 0; d < 4; ++d) g[d] = cell[d] + (uint32_t)((k >> d) & 1);
                uint32_t slot = vertex_slot(g, p.pi, c->T, p.dense[l], p.res_s[l]);
                for (int d = 0; d < 4; ++d) {
                    double wd = ((k >> d) & 1) ? 1.0 : -1.0; /* d omega_d / d w_d */
                    for (int e = 0; e < 4; ++e)
                        if (e != d) wd *= ((k >> e) & 1) ? (double)frac[e] : 1.0 - (double)frac[e];
                    for (uint32_t f = 0; f < F; ++f) {
                        double term = (double)dout[(size_t)n * L * F + (size_t)l * F + f] * res[d] *
                                      wd * table_value(c, table, l, slot, f);
                        acc[d] += term;
                        mag[d] += fabs(term);
                    }
                }
            }
        }
        for (int d = 0; d < 4; ++d) {
            int moved = isnan(q[d]) || q[d] < 0.0f || q[d] > 0x1.fffffep-1f;
            dq[(size_t)n * 4 + d] = moved ? 0.0f : (float)acc[d];
            if (dq_abs) dq_abs[(size_t)n * 4 + d] = moved ? 0.0 : mag[d];
        }
    }
    return ORACLE_OK;
}

/* ---- NEXT #2: smoothness regulariser, Eq. 11 -------------------
 *     L_r(x) = || G_4D(x) - G_4D(x + eps_x) ||_2^2 ,   eps_x = (eps_P, eps_t) a small random perturbation.
 * The random numbers are an INPUT (eps, drawn by the caller): eps_stride = 4 -> eps[n*4 + d], 0 -> one
 * perturbation for all queries.  Readings (Q25): the perturbed query is x'_d = fl32(x_d + eps_d),
 * then clamped like any query (Q12); the norm is over the L*F features; nothing is averaged: loss[n] is the
 * plain squared norm of query n, and the table gradient is that of  grad_scale * sum_n loss[n]:
 *     dtable += grad_scale * 2 * sum_n ( J(x_n)^T d_n - J(x'_n)^T d_n ),   d_n = G(x_n) - G(x'_n).
 * Everything in double from the fp32 cell offsets; loss rounded to fp32 once, dtable as in dash_oracle_bwd.
 * loss_abs [N] (nullable): sum_{l,f} 2|d| (A + A'), A = sum_k |W_k v_k| — conditioning of loss[n];
 * feat_abs [N] (nullable): max over (l,f) of (A + A')  (second-order term of the tolerance);
 * grad_abs [L][T][F] (nullable): sum over contributions of |2 grad_scale W| (A + A'). */
int dash_oracle_smooth(const dash_oracle_config *c, uint64_t N, const float *xyz, uint32_t xyz_stride,
                       const float *t, uint32_t t_stride, const int32_t *index, const float *eps,
                       uint32_t eps_stride, const void *table, double grad_scale, float *loss,
                       float *dtable, double *loss_abs, double *feat_abs, double *grad_abs) {
    level_plan p;
    if (!config_ok(c) || make_plan(c, &p)) return ORACLE_INVALID;
    if (N == 0) return ORACLE_OK;
    if (!args_ok(xyz, xyz_stride, t, t_stride) || !eps || !table || !loss) return ORACLE_INVALID;
    if (!(eps_stride == 0 || eps_stride == 4)) return ORACLE_INVALID;
    const uint32_t L = c->L, F = c->F;
    const size_t TF = (size_t)c->T * F;
    for (uint64_t n = 0; n < N; ++n) {
        loss[n] = 0.0f;
        if (loss_abs) loss_abs[n] = 0.0;
        if (feat_abs) feat_abs[n] = 0.0;
    }
    int failed = 0;
    /* level by level (disjoint tables); per-query loss terms are summed over levels in double below */
    double *loss_acc = (double *)calloc(N, sizeof(double));
    if (!loss_acc) return ORACLE_NOMEM;
#pragma omp parallel for schedule(dynamic, 1)
    for (int32_t l = 0; l < (int32_t)L; ++l) {
        double *acc = dtable ? (double *)calloc(TF, sizeof(double)) : NULL;
        double *mag = grad_abs ? grad_abs + (size_t)l * TF : NULL;
        if (dtable && !acc) {
            failed = 1;
            continue;
        }
        if (mag) memset(mag, 0, TF * sizeof(double));
        for (uint64_t n = 0; n < N; ++n) {
            float q[4], q2[4];
            fetch_query(n, xyz, xyz_stride, t, t_stride, index, q);
            for (int d = 0; d < 4; ++d) {
                volatile float moved = q[d] + eps[n * (uint64_t)eps_stride + d]; /* one fp32 add */
                q2[d] = moved;
            }
            uint32_t s1[16], s2[16];
            double W1[16], W2[16];
            corners(c, &p, (uint32_t)l, q, s1, W1);
            corners(c, &p, (uint32_t)l, q2, s2, W2);
            double lsum = 0.0, labs = 0.0, fabs_max = 0.0;
            for (uint32_t f = 0; f < F; ++f) {
                double y1 = 0, y2 = 0, a1 = 0, a2 = 0;
                for (int k = 0; k < 16; ++k) {
                    double t1 = W1[k] * table_value(c, table, (uint32_t)l, s1[k], f);
                    double t2 = W2[k] * table_value(c, table, (uint32_t)l, s2[k], f);
                    y1 += t1; y2 += t2; a1 += fabs(t1); a2 += fabs(t2);
                }
                double dd = y1 - y2;
                lsum += dd * dd;
                labs += 2.0 * fabs(dd) * (a1 + a2);
                if (a1 + a2 > fabs_max) fabs_max = a1 + a2;
                if (acc) {
                    for (int k = 0; k < 16; ++k) {
                        double g1 = 2.0 * grad_scale * W1[k], g2 = 2.0 * grad_scale * W2[k];
                        acc[(size_t)s1[k] * F + f] += g1 * dd;
                        acc[(size_t)s2[k] * F + f] -= g2 * dd;
                        if (mag) {
                            mag[(size_t)s1[k] * F + f] += fabs(g1) * (a1 + a2);
                            mag[(size_t)s2[k] * F + f] += fabs(g2) * (a1 + a2);
                        }
                    }
                }
            }
#pragma omp atomic
            loss_acc[n] += lsum;
            if (loss_abs) {
#pragma omp atomic
                loss_abs[n] += labs;
            }
            if (feat_abs) {
#pragma omp critical
                { if (fabs_max > feat_abs[n]) feat_abs[n] = fabs_max; }
            }
        }
        if (acc) {
            float *dst = dtable + (size_t)l * TF;
            for (size_t e = 0; e < TF; ++e) dst[e] = (float)((double)dst[e] + acc[e]);
            free(acc);
        }
    }
    for (uint64_t n = 0; n < N; ++n) loss[n] = (float)loss_acc[n];
    free(loss_acc);
    return failed ? ORACLE_NOMEM : ORACLE_OK;
}

/* ---- NEXT #4: the 3D hash encoder G_3D of the decomposition stage -------------------
 * PAPER.md:97-101, Eq. 3: "we extract spatial features f_3D using a 3D hash encoder G_3D from Instant-NGP
 * [25]".  The paper gives no separate definition, so G_3D is Eq. 7-9 with d = 3 (Q26): the
 * spatial resolution schedule Ns_l of Eq. 7, cell floor(p * Ns_l) per axis (one binary32 multiply, Q4),
 * the 8 vertices of the cell (corner k: bit d set => +1 along d, d = 0:x 1:y 2:z), Eq. 8 over three
 * coordinates with pi_1..pi_3, trilinear weights, levels concatenated to R^{LF}.  A level is dense iff
 * (Ns+1)^3 <= T (the d = 3 form of Q10), dense index gx + S(gy + S gz), S = Ns+1.  The temporal fields of
 * the config are ignored.  Precision as in the 4D functions: weights and sums in double, rounded once. */

static int config3_ok(const dash_oracle_config *c) {
    if (!c || c->struct_size != sizeof(dash_oracle_config)) return 0;
    if (c->L < 1 || c->L > ORACLE_MAX_L) return 0;
    if (!(c->F == 1 || c->F == 2 || c->F == 4 || c->F == 8)) return 0;
    if (c->T < 1) return 0;
    if (c->res_s_min < 1 || c->res_s_min > c->res_s_max) return 0;
    if (c->table_dtype > 1) return 0;
    return 1;
}

static int level3_is_dense(const dash_oracle_config *c, uint32_t ns) {
    if (!(c->flags & 1u)) return 0;
    long double v = (long double)(ns + 1.0L) * (ns + 1.0L) * (ns + 1.0L);
    return v <= (long double)c->T;
}

int dash_oracle3d_resolutions(const dash_oracle_config *c, uint32_t *res_s, uint8_t *is_dense) {
    if (!config3_ok(c) || !res_s) return ORACLE_INVALID;
    for (uint32_t l = 0; l < c->L; ++l) {
        res_s[l] = level_resolution(c->res_s_min, c->res_s_max, l, c->L);
        if (is_dense) is_dense[l] = (uint8_t)level3_is_dense(c, res_s[l]);
    }
    return ORACLE_OK;
}

/* the 8 slots and 8 trilinear weights of point p at a level of resolution ns */
static void corners3(const dash_oracle_config *c, const uint32_t pi[4], uint32_t ns, int dense,
                     const float p[3], uint32_t slot[8], double W[8]) {
    uint32_t cell[3];
    float frac[3];
    for (int d = 0; d < 3; ++d) locate(clamp_unit(p[d]), ns, &cell[d], &frac[d]);
    for (int k = 0; k < 8; ++k) {
        uint32_t g[3];
        double w = 1.0;
        for (int d = 0; d < 3; ++d) {
            int up = (k >> d) & 1;
            g[d] = cell[d] + (uint32_t)up;
            w *= up ? (double)frac[d] : 1.0 - (double)frac[d];
        }
        if (dense) {
            uint32_t S = ns + 1u;
            slot[k] = g[0] + S * (g[1] + S * g[2]);
        } else {
            uint32_t h = 0;
            for (int d = 0; d < 3; ++d) h ^= g[d] * pi[d]; /* Eq. 8 with d = 3, uint32 wraparound */
            slot[k] = h % c->T;
        }
        W[k] = w;
    }
}

static void fetch_point(uint64_t n, const float *xyz, uint32_t xyz_stride, const int32_t *index,
                        float p[3]) {
    uint64_t row = index ? (uint64_t)index[n] : n;
    for (int d = 0; d < 3; ++d) p[d] = xyz[row * xyz_stride + d];
}

/* idx_out [N][L][8] u32; w_out [N][L][8] double (nullable). */
int dash_oracle3d_indices(const dash_oracle_config *c, uint64_t N, const float *xyz,
                          uint32_t xyz_stride, const int32_t *index, uint32_t *idx_out,
                          double *w_out) {
    uint32_t res[ORACLE_MAX_L], pi[4];
    uint8_t dn[ORACLE_MAX_L];
    if (dash_oracle3d_resolutions(c, res, dn)) return ORACLE_INVALID;
    if (N == 0) return ORACLE_OK;
    if (!xyz || !(xyz_stride == 3 || xyz_stride == 4) || !idx_out) return ORACLE_INVALID;
    get_primes(c, pi);
#pragma omp parallel for schedule(static)
    for (int64_t n = 0; n < (int64_t)N; ++n) {
        float p[3];
        fetch_point((uint64_t)n, xyz, xyz_stride, index, p);
        for (uint32_t l = 0; l < c->L; ++l) {
            uint32_t slot[8];
            double W[8];
            corners3(c, pi, res[l], dn[l], p, slot, W);
            size_t base = ((size_t)n * c->L + l) * 8;
            for (int k = 0; k < 8; ++k) {
                idx_out[base + k] = slot[k];
                if (w_out) w_out[base + k] = W[k];
            }
        }
    }
    return ORACLE_OK;
}

/* out[n][l*F+f] = sum_{k<8} W_k * table[l][slot_k][f]; out_abs (nullable): sum |terms|. */
int dash_oracle3d_fwd(const dash_oracle_config *c, uint64_t N, const float *xyz, uint32_t xyz_stride,
                      const int32_t *index, const void *table, float *out, double *out_abs) {
    uint32_t res[ORACLE_MAX_L], pi[4];
    uint8_t dn[ORACLE_MAX_L];
    if (dash_oracle3d_resolutions(c, res, dn)) return ORACLE_INVALID;
    if (N == 0) return ORACLE_OK;
    if (!xyz || !(xyz_stride == 3 || xyz_stride == 4) || !table || !out) return ORACLE_INVALID;
    get_primes(c, pi);
    const uint32_t L = c->L, F = c->F;
#pragma omp parallel for schedule(static)
    for (int64_t n = 0; n < (int64_t)N; ++n) {
        float p[3];
        fetch_point((uint64_t)n, xyz, xyz_stride, index, p);
        for (uint32_t l = 0; l < L; ++l) {
            uint32_t slot[8];
            double W[8];
            corners3(c, pi, res[l], dn[l], p, slot, W);
            for (uint32_t f = 0; f < F; ++f) {
                double acc = 0.0, mag = 0.0;
                for (int k = 0; k < 8; ++k) {
                    double term = W[k] * table_value(c, table, l, slot[k], f);
                    acc += term;
                    mag += fabs(term);
                }
                size_t o = (size_t)n * L * F + (size_t)l * F + f;
                out[o] = (float)acc;
                if (out_abs) out_abs[o] = mag;
            }
        }
    }
    return ORACLE_OK;
}

/* dtable[l][slot_k][f] += W_k * dout[n][l*F+f]; accumulators as in dash_oracle_bwd. */
int dash_oracle3d_bwd(const dash_oracle_config *c, uint64_t N, const float *xyz, uint32_t xyz_stride,
                      const int32_t *index, const float *dout, float *dtable, double *grad_abs,
                      uint32_t *hits) {
    uint32_t res[ORACLE_MAX_L], pi[4];
    uint8_t dn[ORACLE_MAX_L];
    if (dash_oracle3d_resolutions(c, res, dn)) return ORACLE_INVALID;
    if (N == 0) return ORACLE_OK;
    if (!xyz || !(xyz_stride == 3 || xyz_stride == 4) || !dout || !dtable) return ORACLE_INVALID;
    get_primes(c, pi);
    const uint32_t L = c->L, F = c->F;
    const size_t TF = (size_t)c->T * F;
    int failed = 0;
#pragma omp parallel for schedule(dynamic, 1)
    for (int32_t l = 0; l < (int32_t)L; ++l) {
        double *acc = (double *)calloc(TF, sizeof(double));
        double *mag = grad_abs ? grad_abs + (size_t)l * TF : NULL;
        uint32_t *cnt = hits ? hits + (size_t)l * c->T : NULL;
        if (!acc) {
            failed = 1;
            continue;
        }
        if (mag) memset(mag, 0, TF * sizeof(double));
        if (cnt) memset(cnt, 0, (size_t)c->T * sizeof(uint32_t));
        for (uint64_t n = 0; n < N; ++n) {
            float p[3];
            uint32_t slot[8];
            double W[8];
            fetch_point(n, xyz, xyz_stride, index, p);
            corners3(c, pi, res[l], dn[l], p, slot, W);
            for (int k = 0; k < 8; ++k) {
                for (uint32_t f = 0; f < F; ++f) {
                    double term = W[k] * (double)dout[(size_t)n * L * F + (size_t)l * F + f];
                    acc[(size_t)slot[k] * F + f] += term;
                    if (mag) mag[(size_t)slot[k] * F + f] += fabs(term);
                }
                if (cnt) cnt[slot[k]] += 1u;
            }
        }
        float *dst = dtable + (size_t)l * TF;
        for (size_t e = 0; e < TF; ++e) dst[e] = (float)((double)dst[e] + acc[e]);
        free(acc);
    }
    return failed ? ORACLE_NOMEM : ORACLE_OK;
}

/* Coordinate gradient of G_3D (DESIGN.md §9 item 2; the d = 3 form of dash_oracle_bwd_input, reading Q24):
 *   dq[n][d] = sum_{l,f} dout[n][l*F+f] * N_l * sum_k s_d(k) * prod_{e != d} omega_e(k) * table[l][slot_k][f],  d = x,y,z
 * on the open cell; a coordinate the Q12 clamp moved has derivative 0.  dq [N][3] fp32; dq_abs (nullable): sum |terms|. */
int dash_oracle3d_bwd_input(const dash_oracle_config *c, uint64_t N, const float *xyz, uint32_t xyz_stride,
                            const int32_t *index, const void *table, const float *dout, float *dq,
                            double *dq_abs) {
    uint32_t res[ORACLE_MAX_L], pi[4];
    uint8_t dn[ORACLE_MAX_L];
    if (dash_oracle3d_resolutions(c, res, dn)) return ORACLE_INVALID;
    if (N == 0) return ORACLE_OK;
    if (!xyz || !(xyz_stride == 3 || xyz_stride == 4) || !table || !dout || !dq) return ORACLE_INVALID;
    get_primes(c, pi);
    const uint32_t L = c->L, F = c->F;
#pragma omp parallel for schedule(static)
    for (int64_t n = 0; n < (int64_t)N; ++n) {
        float p[3];
        fetch_point((uint64_t)n, xyz, xyz_stride, index, p);
        double acc[3] = {0, 0, 0}, mag[3] = {0, 0, 0};
        for (uint32_t l = 0; l < L; ++l) {
            uint32_t cell[3], slot[8];
            float frac[3];
            double W[8];
            for (int d = 0; d < 3; ++d) locate(clamp_unit(p[d]), res[l], &cell[d], &frac[d]);
            corners3(c, pi, res[l], dn[l], p, slot, W); /* the slots; the weights are differentiated below */
            for (int k = 0; k < 8; ++k)
                for (int d = 0; d < 3; ++d) {
                    double wd = ((k >> d) & 1) ? 1.0 : -1.0;
                    for (int e = 0; e < 3; ++e)
                        if (e != d) wd *= ((k >> e) & 1) ? (double)frac[e] : 1.0 - (double)frac[e];
                    for (uint32_t f = 0; f < F; ++f) {
                        double term = (double)dout[(size_t)n * L * F + (size_t)l * F + f] * (double)res[l] * wd *
                                      table_value(c, table, l, slot[k], f);
                        acc[d] += term;
                        mag[d] += fabs(term);
                    }
                }
        }
        for (int d = 0; d < 3; ++d) {
            int moved = isnan(p[d]) || p[d] < 0.0f || p[d] > 0x1.fffffep-1f;
            dq[(size_t)n * 3 + d] = moved ? 0.0f : (float)acc[d];
            if (dq_abs) dq_abs[(size_t)n * 3 + d] = moved ? 0.0 : mag[d];
        }
    }
    return ORACLE_OK;
}

/* ---- NEXT #3: the tiny MLP phi_d and the multi-head deformation decoder ---------------
 * "quadrilinear interpolation ..., followed by a tiny MLP phi_d", f_4D = phi_d(f_h) (Eq. 9);
 * "a multi-head deformation decoder D = {phi_x, phi_r, phi_s}": dx = phi_x(f_4D), dr = phi_r(f_4D),
 * ds = phi_s(f_4D), and (x', r', s') = (x + dx, r + dr, s + ds) (Eq. 10).  Layer sizes and activation are
 * not in the paper (Q27): the decoder is taken as ONE chain of dense layers
 *     a_0 = f_h;   a_l = relu(W_l a_{l-1} + b_l), l < n;   delta = W_n a_{n-1} + b_n;   out = base + delta
 * (the three heads are the row blocks of the last layer(s); a block-diagonal matrix expresses separate
 * hidden layers per head).  params = [W_1 (width1 x width0, row-major) | b_1 | W_2 | b_2 | ...], fp32.
 * Arithmetic: double.  flags bit0 (QUANT_BF16): the operands of every product — the weights and each
 * layer's input vector — are first rounded to bfloat16 (round-to-nearest-even), which is the precision the
 * CUDA path feeds its tensor cores with (Q27); biases, sums and the output stay unrounded.
 * out_abs (nullable, [N][width_n] double): |b_n| + sum_k |W_n[j][k]| * A_k with A the same bound propagated
 * from the input (A_0 = |a_0|, A_l = |b_l| + |W_l| A_{l-1}) — the conditioning term of the tolerance. */

typedef struct dash_oracle_mlp_config {
    uint32_t struct_size;
    uint32_t n_layers; /* 1..4 */
    uint32_t width[5]; /* width[0] inputs, width[l] outputs of layer l */
    uint32_t flags;    /* bit0: round product operands to bf16 */
} dash_oracle_mlp_config;

/* round-to-nearest-even to the 8-bit-significand bfloat16 grid, from double via one fp32 rounding */
static double to_bf16(double v) {
    float f = (float)v;
    uint32_t u;
    memcpy(&u, &f, 4);
    if ((u & 0x7f800000u) == 0x7f800000u) return (double)f; /* inf / nan unchanged */
    uint32_t lsb = (u >> 16) & 1u;
    u += 0x7fffu + lsb;
    u &= 0xffff0000u;
    memcpy(&f, &u, 4);
    return (double)f;
}

double dash_oracle_to_bf16(double v) { return to_bf16(v); }

int dash_oracle_mlp(const dash_oracle_mlp_config *m, uint64_t N, const float *in, const float *params,
                    const float *base, float *out, double *out_abs) {
    if (!m || m->struct_size != sizeof(*m) || m->n_layers < 1 || m->n_layers > 4) return ORACLE_INVALID;
    for (uint32_t l = 0; l <= m->n_layers; ++l)
        if (m->width[l] < 1 || m->width[l] > 4096) return ORACLE_INVALID;
    if (N == 0) return ORACLE_OK;
    if (!in || !params || !out) return ORACLE_INVALID;
    const int quant = (m->flags & 1u) != 0;
    const uint32_t n_out = m->width[m->n_layers];
    uint32_t wmax = 0;
    for (uint32_t l = 0; l <= m->n_layers; ++l)
        if (m->width[l] > wmax) wmax = m->width[l];
    int failed = 0;
#pragma omp parallel
    {
        double *a = (double *)malloc(sizeof(double) * wmax * 4);
        if (!a) {
#pragma omp atomic write
            failed = 1;
        }
        double *A = a ? a + wmax : NULL, *z = a ? a + 2 * wmax : NULL, *Z = a ? a + 3 * wmax : NULL;
#pragma omp for schedule(static)
        for (int64_t n = 0; n < (int64_t)N; ++n) {
            if (!a) continue;
            for (uint32_t k = 0; k < m->width[0]; ++k) {
                a[k] = (double)in[(size_t)n * m->width[0] + k];
                A[k] = fabs(a[k]);
            }
            const float *p = params;
            for (uint32_t l = 1; l <= m->n_layers; ++l) {
                const uint32_t K = m->width[l - 1], J = m->width[l];
                const float *W = p, *b = p + (size_t)J * K;
                for (uint32_t j = 0; j < J; ++j) {
                    double s = (double)b[j], S = fabs((double)b[j]);
                    for (uint32_t k = 0; k < K; ++k) {
                        double w = (double)W[(size_t)j * K + k], x = a[k];
                        if (quant) {
                            w = to_bf16(w);
                            x = to_bf16(x);
                        }
                        s += w * x;
                        S += fabs(w) * A[k];
                    }
                    z[j] = (l < m->n_layers && s < 0.0) ? 0.0 : s; /* relu on hidden layers */
                    Z[j] = S;
                }
                for (uint32_t j = 0; j < J; ++j) {
                    a[j] = z[j];
                    A[j] = Z[j];
                }
                p = b + J;
            }
            for (uint32_t j = 0; j < n_out; ++j) {
                double v = a[j] + (base ? (double)base[(size_t)n * n_out + j] : 0.0);
                out[(size_t)n * n_out + j] = (float)v;
                if (out_abs) out_abs[(size_t)n * n_out + j] = A[j] + (base ? fabs((double)base[(size_t)n * n_out + j]) : 0.0);
            }
        }
        free(a);
    }
    return failed ? ORACLE_NOMEM : ORACLE_OK;
}

/* ---- beyond §8f (DESIGN.md §9 "missing CUDA work" item 1): backward through phi_d and the heads ----------------
 * The chain of dash_oracle_mlp is differentiated by the chain rule (the paper trains phi_d and the heads by gradient
 * descent on the losses of PAPER.md:146-156; it gives no formulas, the ones below are the textbook ones):
 *     delta_n = dout;   for l = n .. 1:   dW_l += delta_l a_{l-1}^T,   db_l += delta_l,
 *     g_{l-1} = W_l^T delta_l,   delta_{l-1} = g_{l-1} * [z_{l-1} > 0]   (relu'(0) = 0),   dfeat = g_0.
 * The forward activations are recomputed here exactly as dash_oracle_mlp computes them (nothing is saved).
 * Arithmetic: double.  flags bit0 (QUANT_BF16): the operands of every product — W, a_{l-1} and delta_l — are first
 * rounded to bfloat16, which is what the CUDA path feeds its tensor cores with (Q30).
 *   dfeat        [N][width_0] fp32 (nullable), rounded once.
 *   dparams      [param_count] double, OVERWRITTEN with the sums over all N rows, packed like params.
 *   dfeat_abs    (nullable, [N][width_0] double): |W_1|^T ( ... |W_n|^T |dout| ) with the same relu masks.
 *   dparams_abs  (nullable, [param_count] double): sum over rows of Delta_l[j] |a_{l-1}[k]| (and of Delta_l[j]), Delta
 *                the bound |W|^T ... |dout| of dfeat_abs one layer up: delta_l carries the rounding of everything
 *                above it, so ITS conditioning, not |delta_l|, scales the error of dW_l.
 *   margin       (nullable, [N] double): min over the hidden units of |z| / (|b| + sum |w x|): how far the row is from
 *                a relu kink, relative to the rounding scale of z.  The mask is a DECISION taken from a floating-point
 *                value; rows closer to a kink than the arithmetic's accuracy have no unique gradient. */
int dash_oracle_mlp_bwd(const dash_oracle_mlp_config *m, uint64_t N, const float *in, const float *params,
                        const float *dout, float *dfeat, double *dparams, double *dfeat_abs,
                        double *dparams_abs, double *margin) {
    if (!m || m->struct_size != sizeof(*m) || m->n_layers < 1 || m->n_layers > 4) return ORACLE_INVALID;
    for (uint32_t l = 0; l <= m->n_layers; ++l)
        if (m->width[l] < 1 || m->width[l] > 4096) return ORACLE_INVALID;
    if (!dparams) return ORACLE_INVALID;
    const uint32_t n_layers = m->n_layers;
    size_t P = 0, p_off[5] = {0, 0, 0, 0, 0};
    uint32_t wmax = 0;
    for (uint32_t l = 1; l <= n_layers; ++l) {
        p_off[l] = P;
        P += (size_t)m->width[l] * m->width[l - 1] + m->width[l];
    }
    for (uint32_t l = 0; l <= n_layers; ++l)
        if (m->width[l] > wmax) wmax = m->width[l];
    for (size_t i = 0; i < P; ++i) {
        dparams[i] = 0.0;
        if (dparams_abs) dparams_abs[i] = 0.0;
    }
    if (N == 0) return ORACLE_OK;
    if (!in || !params || !dout) return ORACLE_INVALID;
    const int quant = (m->flags & 1u) != 0;
    /* one row at a time, in order: obviously correct, deterministic sums */
    double *a = (double *)malloc(sizeof(double) * wmax * (n_layers + 1) * 2 + sizeof(double) * wmax * 4);
    if (!a) return ORACLE_NOMEM;
    double *mask = a + (size_t)wmax * (n_layers + 1);        /* [l][k]: 1 if z_l[k] > 0 (hidden layers) */
    double *delta = mask + (size_t)wmax * (n_layers + 1), *Delta = delta + wmax, *g = Delta + wmax, *G = g + wmax;
    for (uint64_t n = 0; n < N; ++n) {
        double worst = INFINITY;
        for (uint32_t k = 0; k < m->width[0]; ++k) a[k] = (double)in[(size_t)n * m->width[0] + k];
        for (uint32_t l = 1; l <= n_layers; ++l) { /* forward, as dash_oracle_mlp */
            const uint32_t K = m->width[l - 1], J = m->width[l];
            const float *W = params + p_off[l], *b = W + (size_t)J * K;
            const double *x = a + (size_t)(l - 1) * wmax;
            double *y = a + (size_t)l * wmax, *mk = mask + (size_t)l * wmax;
            for (uint32_t j = 0; j < J; ++j) {
                double s = (double)b[j], S = fabs((double)b[j]);
                for (uint32_t k = 0; k < K; ++k) {
                    double w = (double)W[(size_t)j * K + k], xv = x[k];
                    if (quant) {
                        w = to_bf16(w);
                        xv = to_bf16(xv);
                    }
                    s += w * xv;
                    S += fabs(w * xv);
                }
                if (l < n_layers) {
                    mk[j] = s > 0.0 ? 1.0 : 0.0;
                    y[j] = s > 0.0 ? s : 0.0;
                    double rel = S > 0.0 ? fabs(s) / S : INFINITY;
                    if (rel < worst) worst = rel;
                } else {
                    y[j] = s;
                }
            }
        }
        if (margin) margin[n] = worst;
        const uint32_t n_out = m->width[n_layers];
        for (uint32_t j = 0; j < n_out; ++j) {
            delta[j] = (double)dout[(size_t)n * n_out + j];
            Delta[j] = fabs(delta[j]);
        }
        for (uint32_t l = n_layers; l >= 1; --l) { /* backward */
            const uint32_t K = m->width[l - 1], J = m->width[l];
            const float *W = params + p_off[l];
            double *dW = dparams + p_off[l], *db = dW + (size_t)J * K;
            double *dWa = dparams_abs ? dparams_abs + p_off[l] : NULL, *dba = dWa ? dWa + (size_t)J * K : NULL;
            const double *x = a + (size_t)(l - 1) * wmax;
            for (uint32_t k = 0; k < K; ++k) g[k] = G[k] = 0.0;
            for (uint32_t j = 0; j < J; ++j) {
                const double d = quant ? to_bf16(delta[j]) : delta[j];
                db[j] += d;
                if (dba) dba[j] += Delta[j];
                for (uint32_t k = 0; k < K; ++k) {
                    double w = (double)W[(size_t)j * K + k], xv = x[k];
                    if (quant) {
                        w = to_bf16(w);
                        xv = to_bf16(xv);
                    }
                    dW[(size_t)j * K + k] += d * xv;
                    if (dWa) dWa[(size_t)j * K + k] += Delta[j] * fabs(xv);
                    g[k] += w * d;
                    G[k] += fabs(w) * Delta[j];
                }
            }
            if (l > 1) {
                const double *mk = mask + (size_t)(l - 1) * wmax;
                for (uint32_t k = 0; k < K; ++k) {
                    delta[k] = g[k] * mk[k];
                    Delta[k] = G[k] * mk[k];
                }
            } else {
                for (uint32_t k = 0; k < K; ++k) {
                    if (dfeat) dfeat[(size_t)n * K + k] = (float)g[k];
                    if (dfeat_abs) dfeat_abs[(size_t)n * K + k] = G[k];
                }
            }
        }
    }
    free(a);
    return ORACLE_OK;
}

/* ---- beyond §8f (Q31): self-supervised decomposition (Eq. 5) ----------------------
 * "We compute motion magnitudes ||dp|| for all Gaussians and set a threshold tau at the top k% percentile of these
 * values.  Gaussians with ||dp|| > tau are classified as dynamic, the rest as static.  Static Gaussians are constrained
 * by L_s = (1/N_s) sum_{static} ||dp||."  Readings (Q31):
 *   mag[n] = fl32 sqrt of fl32( fl32( fl32(x*x) + fl32(y*y) ) + fl32(z*z) ): binary32 throughout, no contraction (the
 *            classification is a decision on this value, so both sides form it identically); a NaN magnitude counts as 0.
 *   m      = ceil(N * k / 100 - 1e-9), clamped to [0, N]: the size of "the top k %".
 *   tau    = the largest magnitude NOT among the m largest (the (m+1)-th largest); m = 0 -> +inf; m = N -> -1.
 *   dynamic = { n : mag[n] > tau } in ascending n (what nonzero(mask) yields; at most m entries, fewer on ties at tau).
 *   L_s    = sum over static n of mag[n] / N_s (double; 0 when N_s = 0).
 *   ddp[n] = grad_scale * dp[n] / (mag[n] * N_s) for static n with mag[n] > 0, else 0  (d L_s / d dp; the
 *            classification is held fixed, as any top-k selection is when differentiated). */
static int cmp_desc_f32(const void *a, const void *b) {
    float x = *(const float *)a, y = *(const float *)b;
    return (x < y) - (x > y);
}

int dash_oracle_decompose(uint64_t N, const float *dp, double k_percent, double grad_scale, float *mag,
                          float *tau_out, int32_t *dyn_index, uint64_t *n_dyn_out, double *loss_out,
                          float *ddp) {
    if (!mag || !tau_out || !dyn_index || !n_dyn_out || !loss_out) return ORACLE_INVALID;
    if (!(k_percent >= 0.0 && k_percent <= 100.0)) return ORACLE_INVALID;
    *n_dyn_out = 0;
    *loss_out = 0.0;
    *tau_out = INFINITY;
    if (N == 0) return ORACLE_OK;
    if (!dp) return ORACLE_INVALID;
    for (uint64_t n = 0; n < N; ++n) {
        volatile float xx = dp[n * 3 + 0] * dp[n * 3 + 0];
        volatile float yy = dp[n * 3 + 1] * dp[n * 3 + 1];
        volatile float zz = dp[n * 3 + 2] * dp[n * 3 + 2];
        volatile float s = xx + yy;
        s = s + zz;
        float v = sqrtf(s);
        mag[n] = isnan(v) ? 0.0f : v;
    }
    double md = ceil((double)N * k_percent / 100.0 - 1e-9);
    uint64_t m = md <= 0.0 ? 0 : (md >= (double)N ? N : (uint64_t)md);
    float tau;
    if (m == 0) {
        tau = INFINITY;
    } else if (m >= N) {
        tau = -1.0f;
    } else {
        float *sorted = (float *)malloc(sizeof(float) * N);
        if (!sorted) return ORACLE_NOMEM;
        memcpy(sorted, mag, sizeof(float) * N);
        qsort(sorted, N, sizeof(float), cmp_desc_f32);
        tau = sorted[m];
        free(sorted);
    }
    *tau_out = tau;
    uint64_t nd = 0;
    double sum = 0.0;
    for (uint64_t n = 0; n < N; ++n) {
        if (mag[n] > tau) dyn_index[nd++] = (int32_t)n;
        else sum += (double)mag[n];
    }
    const uint64_t ns = N - nd;
    *n_dyn_out = nd;
    *loss_out = ns ? sum / (double)ns : 0.0;
    if (ddp)
        for (uint64_t n = 0; n < N; ++n)
            for (int d = 0; d < 3; ++d)
                ddp[n * 3 + d] = (!(mag[n] > tau) && mag[n] > 0.0f)
                                     ? (float)(grad_scale * (double)dp[n * 3 + d] / ((double)mag[n] * (double)ns))
                                     : 0.0f;
    return ORACLE_OK;
}

/* ---- NEXT #4: sparse optimiser step over the touched table entries -------------------
 * The paper does not name its optimiser ("primarily based on the PyTorch framework"; 3DGS [14]
 * and Instant-NGP [25], which it follows, both train with Adam).  Reading (Q28): Adam (Kingma & Ba),
 * bias-corrected, applied ONLY to entries whose gradient is not exactly zero — an entry no query touched in
 * this step keeps theta, m and v unchanged (no moment decay), which is what makes the step sparse on the
 * coarse dense levels (1-27 % of T touched at C4) and is the rule of torch.optim.SparseAdam.  For g != 0:
 *     m <- beta1 m + (1 - beta1) g ;  v <- beta2 v + (1 - beta2) g^2
 *     theta <- theta - lr * (m / (1 - beta1^t)) / (sqrt(v / (1 - beta2^t)) + eps)
 * theta is the fp32 master copy; theta16 (nullable) receives its IEEE-half rounding (the fp16 table the encoder
 * reads).  With zero_grad != 0 every gradient entry is set to 0 afterwards (the next backward accumulates into
 * it).  Arithmetic in double from the fp32 state, each stored value rounded once. */
static uint16_t double_to_half(double d) {
    /* round-to-nearest-even to IEEE binary16 by search over the format's definition (slow, obviously right) */
    if (isnan(d)) return 0x7e00u;
    uint16_t sign = (uint16_t)(signbit(d) ? 0x8000u : 0u);
    double a = fabs(d);
    if (a >= 65520.0) return (uint16_t)(sign | 0x7c00u); /* rounds to inf */
    /* spacing: subnormal step 2^-24 below 2^-14, else 2^(e-10) */
    int e;
    (void)frexp(a, &e); /* a = f * 2^e, f in [0.5, 1) -> a in [2^(e-1), 2^e) */
    double step = (a < ldexp(1.0, -14)) ? ldexp(1.0, -24) : ldexp(1.0, e - 1 - 10);
    double q = a / step; /* exact: power-of-two scaling */
    double lo = floor(q), frac = q - lo;
    if (frac > 0.5 || (frac == 0.5 && fmod(lo, 2.0) == 1.0)) lo += 1.0;
    double r = lo * step;
    if (r == 0.0) return sign;
    if (r < ldexp(1.0, -14)) return (uint16_t)(sign | (uint16_t)(r / ldexp(1.0, -24)));
    int er;
    double fr = frexp(r, &er); /* r = fr * 2^er, fr in [0.5,1) */
    uint16_t expo = (uint16_t)(er - 1 + 15);
    uint16_t mant = (uint16_t)((fr * 2.0 - 1.0) * 1024.0);
    return (uint16_t)(sign | (uint16_t)(expo << 10) | mant);
}

uint16_t dash_oracle_double_to_half(double d) { return double_to_half(d); }

int dash_oracle_adam_step(uint64_t count, double lr, double beta1, double beta2, double eps, uint32_t t,
                          float *theta, uint16_t *theta16, float *grad, float *m, float *v,
                          int zero_grad, uint64_t *touched) {
    if (!theta || !grad || !m || !v || t < 1) return ORACLE_INVALID;
    const double c1 = 1.0 - pow(beta1, (double)t), c2 = 1.0 - pow(beta2, (double)t);
    uint64_t n_touched = 0;
#pragma omp parallel for schedule(static) reduction(+ : n_touched)
    for (int64_t i = 0; i < (int64_t)count; ++i) {
        const double g = (double)grad[i];
        if (g != 0.0) {
            const double mn = beta1 * (double)m[i] + (1.0 - beta1) * g;
            const double vn = beta2 * (double)v[i] + (1.0 - beta2) * g * g;
            const double th = (double)theta[i] - lr * (mn / c1) / (sqrt(vn / c2) + eps);
            m[i] = (float)mn;
            v[i] = (float)vn;
            theta[i] = (float)th;
            if (theta16) theta16[i] = double_to_half((double)theta[i]);
            ++n_touched;
        }
        if (zero_grad) grad[i] = 0.0f;
    }
    if (touched) *touched = n_touched;
    return ORACLE_OK;
}
