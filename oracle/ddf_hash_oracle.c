/* ddf_hash_oracle.c - CPU oracle of the hash-grid DDF.  TEST INFRASTRUCTURE, NOT PRODUCT.
 * Definitions, citations and pins: ddf_hash_oracle.h.  Built into libddf_oracle.so together
 * with ddf_oracle.c (gcc -O2 -ffp-contract=off, no fast-math). */
#include "ddf_hash_oracle.h"
#include "ddf_oracle.h"
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define HPI 3.14159265358979323846

static int hl_ok(const orc_hash_layout* L) {
  if (L->n_levels < 1 || L->n_levels > 32 || L->n_features < 1 || L->n_features > 8) return 0;
  if (L->log2_table < 4 || L->log2_table > 28 || L->base_res < 1 || !(L->growth >= 1.0)) return 0;
  if (L->n_freq_dir < 0 || L->n_hidden < 1 || L->width < 1 || L->n_out < 1 || L->n_out > 2) return 0;
  if (!(L->table_dtype == 0 || L->table_dtype == 2) || L->mlp_dtype < 0 || L->mlp_dtype > 1) return 0;
  for (int a = 0; a < 3; ++a) if (!(L->box_max[a] > L->box_min[a])) return 0;
  return 1;
}

/* H1: N_l = floor(base * growth^l) */
static int64_t level_res(const orc_hash_layout* L, int level) {
  return (int64_t)floor((double)L->base_res * pow(L->growth, (double)level));
}

int orc_hash_level(const orc_hash_layout* L, int level, int64_t* res, int64_t* entries,
                   int64_t* offset, int* hashed) {
  if (!hl_ok(L) || level < 0 || level >= L->n_levels) return -1;
  const int64_t T = (int64_t)1 << L->log2_table;
  int64_t off = 0;
  for (int l = 0; l <= level; ++l) {
    const int64_t N = level_res(L, l), V = N + 1;
    /* (N+1)^3 <= T without overflow: V is at most a few hundred thousand here */
    const int dense = (V <= 2097151) && (V * V * V <= T);
    const int64_t cnt = dense ? V * V * V : T;
    if (l == level) {
      if (res) *res = N;
      if (entries) *entries = cnt;
      if (offset) *offset = off;
      if (hashed) *hashed = !dense;
    }
    off += cnt;
  }
  return 0;
}

int64_t orc_hash_table_entries(const orc_hash_layout* L) {
  int64_t e = 0, o = 0;
  if (orc_hash_level(L, L->n_levels - 1, NULL, &e, &o, NULL)) return -1;
  return o + e;
}

int orc_hash_mlp_in(const orc_hash_layout* L) { return L->n_levels * L->n_features + 3 + 6 * L->n_freq_dir; }

int64_t orc_hash_mlp_params(const orc_hash_layout* L) {
  int64_t p = 0, in = orc_hash_mlp_in(L);
  for (int l = 0; l < L->n_hidden; ++l) { p += (int64_t)L->width * in + L->width; in = L->width; }
  return p + (int64_t)L->n_out * in + L->n_out;
}

/* H4 */
int64_t orc_hash_index(const orc_hash_layout* L, int level, uint32_t ix, uint32_t iy, uint32_t iz) {
  int64_t N = 0; int hashed = 0;
  if (orc_hash_level(L, level, &N, NULL, NULL, &hashed)) return -1;
  if (!hashed) { const int64_t V = N + 1; return (int64_t)ix + V * ((int64_t)iy + V * (int64_t)iz); }
  const uint32_t h = (ix * 1u) ^ (iy * 2654435761u) ^ (iz * 805459861u);      /* mod 2^32 products */
  return (int64_t)(h & (uint32_t)(((int64_t)1 << L->log2_table) - 1));
}

static double half_bits_to_double(uint16_t h) {
  const int s = h >> 15, e = (h >> 10) & 31, m = h & 1023;
  double v;
  if (e == 0) v = ldexp((double)m, -24);
  else if (e == 31) v = m ? NAN : INFINITY;
  else v = ldexp((double)(1024 + m), e - 25);
  return s ? -v : v;
}

static double table_at(const orc_hash_layout* L, const void* table, int64_t entry, int f) {
  const size_t i = (size_t)entry * L->n_features + f;
  return L->table_dtype == 2 ? half_bits_to_double(((const uint16_t*)table)[i]) : (double)((const float*)table)[i];
}

/* features of one point (H2, H3, H5) */
static void encode_point(const orc_hash_layout* L, const void* table, const float* x, double* feat) {
  float x01[3];
  for (int a = 0; a < 3; ++a) {
    /* H2, in fp32: one subtraction, one subtraction, one division, each correctly rounded */
    const float num = x[a] - L->box_min[a];
    const float den = L->box_max[a] - L->box_min[a];
    float v = num / den;
    v = v < 0.0f ? 0.0f : (v > 1.0f ? 1.0f : v);
    x01[a] = v;
  }
  for (int l = 0; l < L->n_levels; ++l) {
    int64_t N = 0, off = 0;
    orc_hash_level(L, l, &N, NULL, &off, NULL);
    uint32_t c0[3]; double w[3];
    for (int a = 0; a < 3; ++a) {
      const float pos = x01[a] * (float)N;                      /* H3, fp32 product */
      float fl = floorf(pos);
      if (fl > (float)(N - 1)) fl = (float)(N - 1);
      c0[a] = (uint32_t)fl;
      w[a] = (double)(pos - fl);                                /* exact in fp32 */
    }
    for (int f = 0; f < L->n_features; ++f) feat[l * L->n_features + f] = 0.0;
    for (int corner = 0; corner < 8; ++corner) {
      const int bx = corner & 1, by = (corner >> 1) & 1, bz = (corner >> 2) & 1;
      const double wt = (bx ? w[0] : 1.0 - w[0]) * (by ? w[1] : 1.0 - w[1]) * (bz ? w[2] : 1.0 - w[2]);
      const int64_t idx = off + orc_hash_index(L, l, c0[0] + bx, c0[1] + by, c0[2] + bz);
      for (int f = 0; f < L->n_features; ++f) feat[l * L->n_features + f] += wt * table_at(L, table, idx, f);
    }
  }
}

int orc_hash_encode(const orc_hash_layout* L, const void* table, const float* x, int64_t n, double* feat) {
  if (!hl_ok(L)) return -1;
  const int F = L->n_levels * L->n_features;
  #pragma omp parallel for schedule(static)
  for (int64_t i = 0; i < n; ++i) encode_point(L, table, x + 3 * i, feat + (size_t)F * i);
  return 0;
}

static double mlp_at(const orc_hash_layout* L, const void* mlp, size_t i, int quantise) {
  if (L->mlp_dtype == 1) {
    uint32_t b = ((uint32_t)((const uint16_t*)mlp)[i]) << 16; float f; memcpy(&f, &b, 4); return (double)f;
  }
  const float f = ((const float*)mlp)[i];
  return quantise ? orc_round_bf16((double)f) : (double)f;
}

int orc_hash_forward(const orc_hash_layout* L, const void* table, const void* mlp,
                     const float* o, const float* d, int64_t n, int mode,
                     double* z, double* dist, double* vis, int nthreads) {
  if (!hl_ok(L)) return -1;
  const int F = L->n_levels * L->n_features, E = orc_hash_mlp_in(L), W = L->width;
  const int S = (E > W ? E : W);
#ifdef _OPENMP
  if (nthreads > 0) omp_set_num_threads(nthreads);
#endif
  #pragma omp parallel
  {
    double* in = (double*)malloc(sizeof(double) * S);
    double* h  = (double*)malloc(sizeof(double) * S);
    #pragma omp for schedule(dynamic, 64)
    for (int64_t i = 0; i < n; ++i) {
      /* H6: [hash features ; gamma(d)] */
      encode_point(L, table, o + 3 * i, in);
      int m = F;
      for (int c = 0; c < 3; ++c) in[m++] = (double)d[3 * i + c];
      for (int k = 0; k < L->n_freq_dir; ++k) {
        for (int c = 0; c < 3; ++c) in[m++] = sin(HPI * ldexp((double)d[3 * i + c], k));
        for (int c = 0; c < 3; ++c) in[m++] = cos(HPI * ldexp((double)d[3 * i + c], k));
      }
      if (mode) for (int k = 0; k < E; ++k) in[k] = orc_round_bf16(in[k]);
      int nin = E; size_t off = 0;
      for (int l = 0; l < L->n_hidden; ++l) {
        const size_t boff = off + (size_t)W * nin;
        for (int j = 0; j < W; ++j) {
          double acc = mlp_at(L, mlp, boff + j, 0);
          for (int k = 0; k < nin; ++k) acc += mlp_at(L, mlp, off + (size_t)j * nin + k, mode) * in[k];
          acc = acc > 0.0 ? acc : 0.0;
          h[j] = (mode && l != L->n_hidden - 1) ? orc_round_bf16(acc) : acc;
        }
        for (int j = 0; j < W; ++j) in[j] = h[j];
        off = boff + W; nin = W;
      }
      const size_t boff = off + (size_t)L->n_out * nin;
      double zz[2] = {0.0, 0.0};
      for (int j = 0; j < L->n_out; ++j) {
        double acc = mlp_at(L, mlp, boff + j, 0);
        for (int k = 0; k < nin; ++k) acc += mlp_at(L, mlp, off + (size_t)j * nin + k, mode) * in[k];
        zz[j] = acc;
      }
      for (int j = 0; j < L->n_out; ++j) z[(size_t)i * L->n_out + j] = zz[j];
      if (dist) dist[i] = orc_softplus(zz[0]);                     /* (t, xi) */
      if (vis && L->n_out == 2) vis[i] = orc_sigmoid(zz[1]);
    }
    free(in); free(h);
  }
  return 0;
}

/* ------------------------------------------------------------------ training (readings T1-T5) */

/* corners of one level for a point: indices (into the whole table) and trilinear weights */
static void level_corners(const orc_hash_layout* L, int l, const float x01[3], int64_t idx[8], double wt[8]) {
  int64_t N = 0, off = 0;
  orc_hash_level(L, l, &N, NULL, &off, NULL);
  uint32_t c0[3]; double w[3];
  for (int a = 0; a < 3; ++a) {
    const float pos = x01[a] * (float)N;
    float fl = floorf(pos);
    if (fl > (float)(N - 1)) fl = (float)(N - 1);
    c0[a] = (uint32_t)fl; w[a] = (double)(pos - fl);
  }
  for (int c = 0; c < 8; ++c) {
    const int bx = c & 1, by = (c >> 1) & 1, bz = (c >> 2) & 1;
    wt[c] = (bx ? w[0] : 1.0 - w[0]) * (by ? w[1] : 1.0 - w[1]) * (bz ? w[2] : 1.0 - w[2]);
    idx[c] = off + orc_hash_index(L, l, c0[0] + bx, c0[1] + by, c0[2] + bz);
  }
}

double orc_hash_loss_grads(const orc_hash_layout* L, const float* table, const float* mlp,
                           const float* o, const float* d, const float* t, const uint8_t* hit,
                           int64_t n, const orc_train_params* P, double* grad_table, double* grad_mlp) {
  if (!hl_ok(L) || L->n_out != 2) return NAN;
  const int F = L->n_features, NF = L->n_levels * F, E = orc_hash_mlp_in(L), W = L->width, H = L->n_hidden;
  const int64_t n_mlp = orc_hash_mlp_params(L);
  if (grad_table) memset(grad_table, 0, sizeof(double) * (size_t)orc_hash_table_entries(L) * F);
  if (grad_mlp) memset(grad_mlp, 0, sizeof(double) * (size_t)n_mlp);
  /* activations of every layer for one ray: act[0] = input (E), act[l+1] = output of layer l (W) */
  const int S = E > W ? E : W;
  double* act = (double*)malloc(sizeof(double) * (size_t)(H + 1) * S);
  double* del = (double*)malloc(sizeof(double) * S);
  double* dprev = (double*)malloc(sizeof(double) * S);
  double loss = 0.0;
  for (int64_t i = 0; i < n; ++i) {
    float x01[3];
    for (int a = 0; a < 3; ++a) {
      const float num = o[3 * i + a] - L->box_min[a], den = L->box_max[a] - L->box_min[a];
      float v = num / den; v = v < 0.0f ? 0.0f : (v > 1.0f ? 1.0f : v); x01[a] = v;
    }
    double* in = act;
    for (int l = 0; l < L->n_levels; ++l) {
      int64_t idx[8]; double wt[8];
      level_corners(L, l, x01, idx, wt);
      for (int f = 0; f < F; ++f) {
        double s = 0.0;
        for (int c = 0; c < 8; ++c) s += wt[c] * (double)table[(size_t)idx[c] * F + f];
        in[l * F + f] = s;
      }
    }
    int m = NF;
    for (int c = 0; c < 3; ++c) in[m++] = (double)d[3 * i + c];
    for (int k = 0; k < L->n_freq_dir; ++k) {
      for (int c = 0; c < 3; ++c) in[m++] = sin(HPI * ldexp((double)d[3 * i + c], k));
      for (int c = 0; c < 3; ++c) in[m++] = cos(HPI * ldexp((double)d[3 * i + c], k));
    }
    /* forward */
    size_t off = 0; int nin = E;
    for (int l = 0; l < H; ++l) {
      const double* a_in = act + (size_t)l * S; double* a_out = act + (size_t)(l + 1) * S;
      const size_t boff = off + (size_t)W * nin;
      for (int j = 0; j < W; ++j) {
        double acc = (double)mlp[boff + j];
        for (int k = 0; k < nin; ++k) acc += (double)mlp[off + (size_t)j * nin + k] * a_in[k];
        a_out[j] = acc > 0.0 ? acc : 0.0;
      }
      off = boff + W; nin = W;
    }
    const size_t head_off = off, head_b = off + (size_t)2 * nin;
    const double* hl = act + (size_t)H * S;
    double z[2];
    for (int j = 0; j < 2; ++j) {
      double acc = (double)mlp[head_b + j];
      for (int k = 0; k < nin; ++k) acc += (double)mlp[head_off + (size_t)j * nin + k] * hl[k];
      z[j] = acc;
    }
    /* loss (T1, T2) and its derivative w.r.t. the logits */
    const double that = orc_softplus(z[0]), err = that - (double)t[i];
    const int h = hit[i] != 0;
    double dz[2] = {0.0, 0.0};
    if (h) {
      const double ae = fabs(err);
      loss += ae < P->dist_clamp ? ae : P->dist_clamp;
      if (ae < P->dist_clamp) dz[0] = (err > 0.0 ? 1.0 : (err < 0.0 ? -1.0 : 0.0)) * orc_sigmoid(z[0]);   /* d softplus = sigmoid */
    }
    loss += P->ce_weight * (h ? orc_softplus(-z[1]) : orc_softplus(z[1]));
    dz[1] = P->ce_weight * (orc_sigmoid(z[1]) - (double)h);
    dz[0] /= (double)n; dz[1] /= (double)n;
    /* backward: head */
    for (int k = 0; k < nin; ++k) del[k] = 0.0;
    for (int j = 0; j < 2; ++j) {
      if (grad_mlp) { grad_mlp[head_b + j] += dz[j]; for (int k = 0; k < nin; ++k) grad_mlp[head_off + (size_t)j * nin + k] += dz[j] * hl[k]; }
      for (int k = 0; k < nin; ++k) del[k] += (double)mlp[head_off + (size_t)j * nin + k] * dz[j];
    }
    /* hidden layers, last to first; del = dLoss/d(output of layer l) */
    for (int l = H - 1; l >= 0; --l) {
      const int lin = (l == 0) ? E : W;
      size_t woff = 0; { int q = E; for (int r = 0; r < l; ++r) { woff += (size_t)W * q + W; q = W; } }
      const size_t boff = woff + (size_t)W * lin;
      const double* a_in = act + (size_t)l * S; const double* a_out = act + (size_t)(l + 1) * S;
      for (int k = 0; k < lin; ++k) dprev[k] = 0.0;
      for (int j = 0; j < W; ++j) {
        const double g = a_out[j] > 0.0 ? del[j] : 0.0;          /* ReLU */
        if (grad_mlp) { grad_mlp[boff + j] += g; for (int k = 0; k < lin; ++k) grad_mlp[woff + (size_t)j * lin + k] += g * a_in[k]; }
        for (int k = 0; k < lin; ++k) dprev[k] += (double)mlp[woff + (size_t)j * lin + k] * g;
      }
      for (int k = 0; k < lin; ++k) del[k] = dprev[k];
    }
    /* table: d feature / d table value = the trilinear weight */
    if (grad_table)
      for (int l = 0; l < L->n_levels; ++l) {
        int64_t idx[8]; double wt[8];
        level_corners(L, l, x01, idx, wt);
        for (int c = 0; c < 8; ++c) for (int f = 0; f < F; ++f) grad_table[(size_t)idx[c] * F + f] += wt[c] * del[l * F + f];
      }
  }
  free(act); free(del); free(dprev);
  return loss / (double)n;
}

/* Distance of a ray from the nearest ReLU kink: min over all hidden units of |pre-activation|, fp64,
 * the same forward pass as orc_hash_loss_grads.  The loss is not differentiable where a
 * pre-activation is 0, and an implementation whose forward pass is rounded differently picks the
 * other side of the kink for a ray within its rounding error of one (reading T7); the
 * gradient parity tests use this to keep such rays out of large batches. */
int orc_hash_relu_margin(const orc_hash_layout* L, const float* table, const float* mlp,
                         const float* o, const float* d, int64_t n, double* margin) {
  if (!hl_ok(L)) return -1;
  const int E = orc_hash_mlp_in(L), W = L->width, H = L->n_hidden, NF = L->n_levels * L->n_features;
  const int S = E > W ? E : W;
  double* in = (double*)malloc(sizeof(double) * S);
  double* out = (double*)malloc(sizeof(double) * S);
  for (int64_t i = 0; i < n; ++i) {
    encode_point(L, table, o + 3 * i, in);
    int m = NF;
    for (int c = 0; c < 3; ++c) in[m++] = (double)d[3 * i + c];
    for (int k = 0; k < L->n_freq_dir; ++k) {
      for (int c = 0; c < 3; ++c) in[m++] = sin(HPI * ldexp((double)d[3 * i + c], k));
      for (int c = 0; c < 3; ++c) in[m++] = cos(HPI * ldexp((double)d[3 * i + c], k));
    }
    double best = INFINITY;
    size_t off = 0; int nin = E;
    for (int l = 0; l < H; ++l) {
      const size_t boff = off + (size_t)W * nin;
      for (int j = 0; j < W; ++j) {
        double acc = (double)mlp[boff + j];
        for (int k = 0; k < nin; ++k) acc += (double)mlp[off + (size_t)j * nin + k] * in[k];
        if (fabs(acc) < best) best = fabs(acc);
        out[j] = acc > 0.0 ? acc : 0.0;
      }
      for (int j = 0; j < W; ++j) in[j] = out[j];
      off = boff + W; nin = W;
    }
    margin[i] = best;
  }
  free(in); free(out);
  return 0;
}

double orc_lr_at(const orc_train_params* P, int64_t step) {
  const double s = step < P->total_steps ? (double)step : (double)P->total_steps;
  const double f = P->lr_final_frac;
  return P->lr0 * (f + (1.0 - f) * 0.5 * (1.0 + cos(HPI * s / (double)P->total_steps)));
}

void orc_adam_step(float* p, const double* g, double* m, double* v, int64_t n, int64_t step,
                   double lr, const orc_train_params* P) {
  const double c1 = 1.0 - pow(P->beta1, (double)step), c2 = 1.0 - pow(P->beta2, (double)step);
  for (int64_t i = 0; i < n; ++i) {
    m[i] = P->beta1 * m[i] + (1.0 - P->beta1) * g[i];
    v[i] = P->beta2 * v[i] + (1.0 - P->beta2) * g[i] * g[i];
    p[i] = (float)((double)p[i] - lr * (m[i] / c1) / (sqrt(v[i] / c2) + P->adam_eps));
  }
}

double orc_solid_scene_raycast(const double o[3], const double d[3], const double sphere_c[3],
                               double sphere_r, const double bmin[3], const double bmax[3]) {
  double best = -1.0;
  const double ts = orc_ray_sphere(o, d, sphere_c, sphere_r);      /* smallest t > 0, from inside too */
  if (ts > 0.0) best = ts;
  /* slabs: the ray is inside the box for t in [tn, tf] */
  double tn = -INFINITY, tf = INFINITY; int ok = 1;
  for (int a = 0; a < 3; ++a) {
    if (d[a] != 0.0) {
      double t0 = (bmin[a] - o[a]) / d[a], t1 = (bmax[a] - o[a]) / d[a];
      if (t0 > t1) { const double q = t0; t0 = t1; t1 = q; }
      if (t0 > tn) tn = t0;
      if (t1 < tf) tf = t1;
    } else if (o[a] < bmin[a] || o[a] > bmax[a]) ok = 0;
  }
  if (ok && tn <= tf && tf > 0.0) {
    const double tb = tn > 0.0 ? tn : tf;                          /* entering, or leaving from inside */
    if (best < 0.0 || tb < best) best = tb;
  }
  return best;
}

/* reading T6: "Camera rays ... Rays that start on the surface and point in all
 * directions ... a point moved forward by s should report distance t-s"; "We replace
 * 30 percent of each batch with the ray-march shifted points". */
void orc_gen_train_batch(const double sphere_c[3], double sphere_r, const double bmin[3], const double bmax[3],
                         uint64_t seed, uint64_t stream, int64_t step, int64_t n, double sample_half,
                         float* o, float* d, float* t, uint8_t* hit) {
  for (int64_t k = 0; k < n; ++k) {
    const uint64_t base = ((uint64_t)step * (uint64_t)n + (uint64_t)k) * 16ull;
    double u[11];
    for (int j = 0; j < 11; ++j) u[j] = orc_uniform01(seed, stream, base + j);
    double oo[3], dd[3], q[3];
    for (int a = 0; a < 3; ++a) oo[a] = (2.0 * u[a] - 1.0) * sample_half;
    for (int a = 0; a < 3; ++a) q[a] = (2.0 * u[3 + a] - 1.0) - oo[a];
    const double len = sqrt(q[0]*q[0] + q[1]*q[1] + q[2]*q[2]);
    if (len > 1e-6) { for (int a = 0; a < 3; ++a) dd[a] = q[a] / len; } else { dd[0] = 0; dd[1] = 0; dd[2] = 1; }
    double tt = orc_solid_scene_raycast(oo, dd, sphere_c, sphere_r, bmin, bmax);
    if (u[6] >= 0.5 && tt > 0.0) {                        /* surface-anchored, omnidirectional */
      for (int a = 0; a < 3; ++a) oo[a] += (tt - 1e-3) * dd[a];
      orc_dir_from_u(u[7], u[8], dd);
      tt = orc_solid_scene_raycast(oo, dd, sphere_c, sphere_r, bmin, bmax);
    }
    double tf = tt > 0.0 ? tt : 0.0;
    if (tt > 0.0 && u[9] < 0.3) {                         /* ray-march shifted point */
      const double s = u[10] * tf;
      for (int a = 0; a < 3; ++a) oo[a] += s * dd[a];
      tf -= s;
    }
    for (int a = 0; a < 3; ++a) { o[3 * k + a] = (float)oo[a]; d[3 * k + a] = (float)dd[a]; }
    t[k] = (float)tf; hit[k] = tt > 0.0 ? 1 : 0;
  }
}
