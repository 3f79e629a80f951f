/* ddf_hash_oracle.h - CPU oracle for the paper's own DDF architecture:
 * multiresolution hash grid on the ray origin + sinusoidal direction bands + a small MLP.
 * TEST INFRASTRUCTURE, NOT PRODUCT (same rules as ddf_oracle.h).
 *
 * PAPER.md:64 (Sec. III-A): "a multiresolution hash grid that encodes the point x, following
 * [8], together with a small encoding of the direction d.  A two-layer MLP of width 64 reads
 * this code and outputs t and xi."   PAPER.md:84 (Sec. III-D): "16 levels, two features per
 * level, a table of 2^19 entries per level, base resolution 16, and growth 1.5, over a box that
 * bounds the normalized object ... direction d with four sinusoidal bands ... The hash table
 * holds about 13M parameters and the MLP about 8k, for a stored field of 52 MB."
 *
 * What [8] (the multiresolution hash encoding the paper follows) defines, restated (DESIGN.md
 * readings H1-H6):
 *   H1  level l has resolution N_l = floor(base * growth^l); its grid has (N_l + 1)^3 vertices.
 *   H2  x01 = clamp((x - box_min) / (box_max - box_min), 0, 1), evaluated in fp32.
 *   H3  pos = x01 * N_l (fp32); cell = min(floor(pos), N_l - 1); w = pos - cell  (per axis).
 *   H4  a vertex (ix, iy, iz) is stored at  ix + (N_l+1) * (iy + (N_l+1) * iz)  when the whole
 *       grid fits the table ((N_l+1)^3 <= T), else at
 *       (ix ^ iy * 2654435761 ^ iz * 805459861) mod T   (32-bit wrap-around products).
 *   H5  feature_f = sum over the 8 cell corners of  prod_axis (w or 1-w) * table[l][index][f].
 *   H6  MLP input = [features of level 0, level 1, ... ; gamma_Ld(d)]  (gamma as in
 *       ddf_oracle.h: identity, then per band 3 sines and 3 cosines of 2^k pi d).
 * Everything after the integer decisions of H2-H4 (which the paper's fp32 inputs fix) is fp64.
 *
 * Pins (tests/test_hash_oracle_pins.py): the paper's own counts (13.06M table parameters,
 * 52.2 MB, 8130 MLP parameters); partition of unity; exact reproduction of linear fields on
 * dense levels; table value at a vertex; hand-computed dense and hashed indices; continuity
 * across cell faces; brute-force numpy re-evaluation.  Parity unpinned: the absolute (t, xi) of
 * the seeded random field (no trained field exists in the container).
 */
#ifndef DDF_HASH_ORACLE_H
#define DDF_HASH_ORACLE_H
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct orc_hash_layout {
  int32_t n_levels;        /* 16 */
  int32_t n_features;      /* 2 */
  int32_t log2_table;      /* 19: T = 2^19 entries per level */
  int32_t base_res;        /* 16 */
  double  growth;          /* 1.5 */
  float   box_min[3], box_max[3];
  int32_t n_freq_dir;      /* 4 */
  int32_t n_hidden;        /* 2 */
  int32_t width;           /* 64 */
  int32_t n_out;           /* 2 */
  int32_t table_dtype;     /* 0 = fp32, 2 = fp16 (raw uint16) */
  int32_t mlp_dtype;       /* 0 = fp32, 1 = bf16 (raw uint16) */
} orc_hash_layout;

/* resolution N_l, number of stored entries, entry offset of the level in the table, hashed? */
int  orc_hash_level(const orc_hash_layout* L, int level, int64_t* res, int64_t* entries,
                    int64_t* offset, int* hashed);
int64_t orc_hash_table_entries(const orc_hash_layout* L);       /* all levels */
int  orc_hash_mlp_in(const orc_hash_layout* L);                 /* n_levels*n_features + 3 + 6*L_d */
int64_t orc_hash_mlp_params(const orc_hash_layout* L);          /* weights + biases */
/* storage index of vertex (ix, iy, iz) of `level` within that level (H4) */
int64_t orc_hash_index(const orc_hash_layout* L, int level, uint32_t ix, uint32_t iy, uint32_t iz);
/* feat[n][n_levels*n_features] (fp64) of the points x[n][3] */
int  orc_hash_encode(const orc_hash_layout* L, const void* table, const float* x, int64_t n, double* feat);
/* mode 0 exact fp64; 1 quantised (features, gamma(d) and hidden activations but the last rounded
 * to bf16; fp32 MLP weights rounded to bf16).  mlp blob: layers then head, W[out][in] + b[out]. */
int  orc_hash_forward(const orc_hash_layout* L, const void* table, const void* mlp,
                      const float* o, const float* d, int64_t n, int mode,
                      double* z, double* dist, double* vis, int nthreads);

/* ---------------------------------------------------------------- training
 * PAPER.md:70 (Sec. III-B): "The loss is an L1 term on distance, clamped to a maximum so far-away
 * surfaces do not dominate, plus a cross-entropy term on the hit flag."  PAPER.md:86 (Sec. III-D):
 * "Adam for 30,000 steps, a batch of 16,384 rays, and a learning rate of 3e-3 decayed by cosine to
 * five percent of its value.  The loss is an L1 term on distance, clamped at the box scale, plus a
 * cross-entropy term on the hit weighted at 0.3."  Readings T1-T5:
 *   T1  per ray  l = hit * min(|softplus(z0) - t|, clamp) + ce_weight * CE(sigmoid(z1), hit),
 *       CE = softplus(-z1) if hit else softplus(z1);  loss = mean over the batch.
 *   T2  the distance term exists only for rays that hit (a miss has no distance).
 *   T3  Adam as published (Kingma & Ba): m = b1 m + (1-b1) g; v = b2 v + (1-b2) g^2;
 *       p -= lr * (m / (1-b1^s)) / (sqrt(v / (1-b2^s)) + eps), s = 1, 2, ...
 *   T4  lr(s) = lr0 * (f + (1-f) * (1 + cos(pi * min(s, S) / S)) / 2), f = 0.05, s = 0 .. S.
 *   T5  fp32 master parameters; this oracle evaluates everything in fp64 from them.
 * Pins (tests/test_train_oracle_pins.py): gradients against central finite differences of the
 * loss; Adam's first step = -lr * sign(g); constant gradient; schedule end points. */
typedef struct orc_train_params {
  double lr0, lr_final_frac; int32_t total_steps;
  double beta1, beta2, adam_eps, dist_clamp, ce_weight;
} orc_train_params;
/* loss (returned) and gradients of the mean loss w.r.t. every table value (grad_table
 * [entries * n_features]) and every MLP parameter (grad_mlp, blob order); either may be NULL.
 * table and mlp are fp32 here (table_dtype / mlp_dtype of L are ignored). */
double orc_hash_loss_grads(const orc_hash_layout* L, const float* table, const float* mlp,
                           const float* o, const float* d, const float* t, const uint8_t* hit,
                           int64_t n, const orc_train_params* P, double* grad_table, double* grad_mlp);
/* margin[i] = min over the hidden units of |pre-activation| of ray i (fp32 table and MLP, as in
 * orc_hash_loss_grads): how far the ray is from a ReLU kink, where the loss has no gradient
 * (reading T7). */
int orc_hash_relu_margin(const orc_hash_layout* L, const float* table, const float* mlp,
                         const float* o, const float* d, int64_t n, double* margin);
double orc_lr_at(const orc_train_params* P, int64_t step);
/* one Adam update of n parameters in place; `step` is 1-based (T3) */
void orc_adam_step(float* p, const double* g, double* m, double* v, int64_t n, int64_t step,
                   double lr, const orc_train_params* P);

/* ---- analytic supervision (stands in for the paper's mesh ray cast): distance to
 * the FIRST SURFACE along d of a sphere and an axis-aligned box, from any origin
 * (inside an object the first surface is where the ray leaves it).  Returns t, or -1 for a miss. */
double orc_solid_scene_raycast(const double o[3], const double d[3], const double sphere_c[3],
                               double sphere_r, const double bmin[3], const double bmax[3]);

/* one training batch, reading T6 (ddf.h ddf_gen_train_batch): counters (step n + k) 16 + j.
 * Pinned by tests/test_train_oracle_pins.py::test_train_batch_generator_pins: the draws recomputed
 * with the numpy counter generator say which rays must be anchored / shifted; geometry judged by implicit surface
 * functions and brute-force sampling along the ray. */
void orc_gen_train_batch(const double sphere_c[3], double sphere_r, const double bmin[3], const double bmax[3],
                         uint64_t seed, uint64_t stream, int64_t step, int64_t n, double sample_half,
                         float* o, float* d, float* t, uint8_t* hit);

#ifdef __cplusplus
}
#endif
#endif
