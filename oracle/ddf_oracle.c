/* ddf_oracle.c - CPU oracle for the DDF hot path.  TEST INFRASTRUCTURE, NOT PRODUCT.
 * See ddf_oracle.h for scope, pins and the "parity unpinned" statement.
 * Build: gcc -O2 -fopenmp -fPIC -shared -o libddf_oracle.so ddf_oracle.c -lm   (no fast-math)
 */
#include "ddf_oracle.h"
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORC_PI 3.14159265358979323846

/* ------------------------------------------------------------------ scalar pieces */

/* softplus, beta = 1, stable form (reading A1; BASELINE.json configs[0] "distance via softplus") */
double orc_softplus(double z) { return fmax(z, 0.0) + log1p(exp(-fabs(z))); }

/* logistic sigmoid (reading A1; configs[0] "visibility via sigmoid") */
double orc_sigmoid(double z) { return 1.0 / (1.0 + exp(-z)); }

/* bf16 = top 16 bits of fp32, round to nearest even (reading A11) */
static float bf16_rne_f32(float f) {
  uint32_t b; memcpy(&b, &f, 4);
  if ((b & 0x7F800000u) == 0x7F800000u) return f;            /* inf / nan unchanged */
  b = (b + 0x7FFFu + ((b >> 16) & 1u)) & 0xFFFF0000u;
  memcpy(&f, &b, 4);
  return f;
}
double orc_round_bf16(double x) { return (double)bf16_rne_f32((float)x); }

static double bf16_bits_to_double(uint16_t h) {
  uint32_t b = ((uint32_t)h) << 16; float f; memcpy(&f, &b, 4); return (double)f;
}

/* counter-based generator, reading A8 */
uint64_t orc_mix64(uint64_t z) {
  z += 0x9E3779B97F4A7C15ull;
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
  return z ^ (z >> 31);
}
uint64_t orc_u64_at(uint64_t seed, uint64_t stream, uint64_t idx) {
  return orc_mix64(orc_mix64(orc_mix64(seed) ^ stream) ^ idx);
}
double orc_uniform01(uint64_t seed, uint64_t stream, uint64_t idx) {
  return (double)(orc_u64_at(seed, stream, idx) >> 40) * (1.0 / 16777216.0);
}

/* ------------------------------------------------------------------ encoding */

int orc_enc_dim(const orc_layout* L) {
  int e = 3 + 6 * L->n_freq_origin;
  if (L->input_kind == 0) e += 3 + 6 * L->n_freq_dir;
  return e;
}

/* gamma(v) = [v, sin(2^0 pi v), cos(2^0 pi v), ..., sin(2^(L-1) pi v), cos(2^(L-1) pi v)],
 * each sin/cos block holding the 3 components of v (readings A2, A3; "four
 * sinusoidal bands"; configs[0] "identity plus sin/cos(2^k pi x)"). */
static int encode_vec(const float* v, int nfreq, double* out) {
  int m = 0;
  for (int c = 0; c < 3; ++c) out[m++] = (double)v[c];
  for (int k = 0; k < nfreq; ++k) {
    for (int c = 0; c < 3; ++c) out[m++] = sin(ORC_PI * ldexp((double)v[c], k));
    for (int c = 0; c < 3; ++c) out[m++] = cos(ORC_PI * ldexp((double)v[c], k));
  }
  return m;
}

static void encode_ray(const orc_layout* L, const float* o, const float* d, double* g) {
  int m = encode_vec(o, L->n_freq_origin, g);
  if (L->input_kind == 0) encode_vec(d, L->n_freq_dir, g + m);
}

void orc_encode(const orc_layout* L, const float* o, const float* d, int64_t n, double* gamma) {
  int E = orc_enc_dim(L);
  for (int64_t i = 0; i < n; ++i)
    encode_ray(L, o + 3 * i, (L->input_kind == 0) ? d + 3 * i : NULL, gamma + (size_t)E * i);
}

/* ------------------------------------------------------------------ network */

static int layout_ok(const orc_layout* L) {
  if (L->input_kind < 0 || L->input_kind > 1) return 0;
  if (L->n_freq_origin < 0 || L->n_freq_dir < 0 || L->n_hidden < 1 || L->width < 1) return 0;
  if (L->skip_layer != -1 && (L->skip_layer < 1 || L->skip_layer >= L->n_hidden)) return 0;
  if (L->n_out < 1 || L->n_out > 2) return 0;
  if (L->weight_dtype < 0 || L->weight_dtype > 1) return 0;
  return 1;
}

static double blob_at(const orc_layout* L, const void* blob, size_t i, int quantise) {
  if (L->weight_dtype == 1) return bf16_bits_to_double(((const uint16_t*)blob)[i]);
  float f = ((const float*)blob)[i];
  return quantise ? (double)bf16_rne_f32(f) : (double)f;
}

/* one ray: gamma -> hidden layers -> logits.  h, hin are scratch of size width + E. */
static void forward_one(const orc_layout* L, const void* blob, const double* gamma, int mode,
                        double* h, double* hin, double* z) {
  const int E = orc_enc_dim(L), W = L->width;
  int nin = E;
  size_t off = 0;
  for (int k = 0; k < E; ++k) h[k] = mode ? orc_round_bf16(gamma[k]) : gamma[k];
  for (int l = 0; l < L->n_hidden; ++l) {
    /* input of this layer: h, or [h ; gamma] at the skip layer (reading A5) */
    for (int k = 0; k < nin; ++k) hin[k] = h[k];
    if (l == L->skip_layer) {
      for (int k = 0; k < E; ++k) hin[nin + k] = mode ? orc_round_bf16(gamma[k]) : gamma[k];
      nin += E;
    }
    const size_t boff = off + (size_t)W * nin;
    for (int j = 0; j < W; ++j) {
      double acc = blob_at(L, blob, boff + j, 0);              /* bias (never re-rounded) */
      for (int k = 0; k < nin; ++k) acc += blob_at(L, blob, off + (size_t)j * nin + k, mode) * hin[k];
      acc = acc > 0.0 ? acc : 0.0;                             /* ReLU */
      /* reading A11: every post-ReLU activation is stored as bf16, except the last one,
       * which feeds the head from the un-rounded accumulator */
      h[j] = (mode && l != L->n_hidden - 1) ? orc_round_bf16(acc) : acc;
    }
    off = boff + W;
    nin = W;
  }
  /* head (linear) - in quantised mode the head weights are used as stored (fp32 or bf16) */
  const size_t boff = off + (size_t)L->n_out * nin;
  for (int j = 0; j < L->n_out; ++j) {
    double acc = blob_at(L, blob, boff + j, 0);
    for (int k = 0; k < nin; ++k) acc += blob_at(L, blob, off + (size_t)j * nin + k, mode) * h[k];
    z[j] = acc;
  }
}

int orc_forward(const orc_layout* L, const void* blob, const float* o, const float* d,
                int64_t n, int mode, double* z, double* dist, double* vis, int nthreads) {
  if (!layout_ok(L)) return -1;
  const int E = orc_enc_dim(L);
  const int S = L->width + E > 2 * E ? L->width + E : 2 * E;
#ifdef _OPENMP
  if (nthreads > 0) omp_set_num_threads(nthreads);
#endif
  #pragma omp parallel
  {
    double* g   = (double*)malloc(sizeof(double) * E);
    double* h   = (double*)malloc(sizeof(double) * S);
    double* hin = (double*)malloc(sizeof(double) * S);
    #pragma omp for schedule(dynamic, 4)
    for (int64_t i = 0; i < n; ++i) {
      double zz[2] = {0.0, 0.0};
      encode_ray(L, o + 3 * i, (L->input_kind == 0) ? d + 3 * i : NULL, g);
      forward_one(L, blob, g, mode, h, hin, zz);
      for (int j = 0; j < L->n_out; ++j) z[(size_t)i * L->n_out + j] = zz[j];
      /* PAPER.md:58-62 Eq.1: f(x,d) = (t, xi); order (distance, visibility) */
      if (dist) dist[i] = orc_softplus(zz[0]);
      if (vis && L->n_out == 2) vis[i] = orc_sigmoid(zz[1]);
    }
    free(g); free(h); free(hin);
  }
  return 0;
}

/* ------------------------------------------------------------------ analytic intersections */

static double dot3(const double a[3], const double b[3]) { return a[0]*b[0] + a[1]*b[1] + a[2]*b[2]; }
static void cross3(const double a[3], const double b[3], double o[3]) {
  o[0] = a[1]*b[2] - a[2]*b[1]; o[1] = a[2]*b[0] - a[0]*b[2]; o[2] = a[0]*b[1] - a[1]*b[0];
}
static void normalize3(double v[3]) {
  double n = sqrt(dot3(v, v)); v[0] /= n; v[1] /= n; v[2] /= n;
}

/* |o + t d - c|^2 = r^2 with |d| = 1:  t = -b -+ sqrt(b^2 - (|oc|^2 - r^2)), b = oc.d
 * (pin P9).  Returns the smallest t > 0, or -1. */
double orc_ray_sphere(const double o[3], const double d[3], const double c[3], double r) {
  double oc[3] = { o[0]-c[0], o[1]-c[1], o[2]-c[2] };
  double b = dot3(oc, d), cc = dot3(oc, oc) - r * r;
  double disc = b * b - cc;
  if (disc < 0.0) return -1.0;
  double sq = sqrt(disc);
  double t0 = -b - sq, t1 = -b + sq;
  if (t0 > 0.0) return t0;
  if (t1 > 0.0) return t1;
  return -1.0;
}

/* slab method from a point inside the box: the exit distance is the smallest of the
 * per-axis distances to the face the ray is heading to. */
double orc_ray_box_exit(const double o[3], const double d[3], const double bmin[3],
                        const double bmax[3], int* face) {
  double tbest = INFINITY; int fbest = -1;
  for (int a = 0; a < 3; ++a) {
    if (d[a] > 0.0) { double t = (bmax[a] - o[a]) / d[a]; if (t < tbest) { tbest = t; fbest = 2*a + 1; } }
    else if (d[a] < 0.0) { double t = (bmin[a] - o[a]) / d[a]; if (t < tbest) { tbest = t; fbest = 2*a; } }
  }
  if (face) *face = fbest;
  return tbest;
}

/* ------------------------------------------------------------------ generators */

/* reading A9: z = 2 u1 - 1, phi = 2 pi u2 */
void orc_dir_from_u(double u1, double u2, double out[3]) {
  double z = 2.0 * u1 - 1.0, phi = 2.0 * ORC_PI * u2;
  double s = sqrt(fmax(0.0, 1.0 - z * z));
  out[0] = s * cos(phi); out[1] = s * sin(phi); out[2] = z;
}

/* reading A13: camera on a seeded sphere of the given radius, looking at the origin */
void orc_camera_from_seed(uint64_t seed, uint64_t stream, double radius, orc_camera* cam) {
  double v[3];
  orc_dir_from_u(orc_uniform01(seed, stream, 0), orc_uniform01(seed, stream, 1), v);
  for (int a = 0; a < 3; ++a) { cam->pos[a] = radius * v[a]; cam->look_at[a] = 0.0; }
  cam->fov_deg = 50.0;
}

static void camera_frame(const orc_camera* cam, double f[3], double right[3], double up2[3]) {
  for (int a = 0; a < 3; ++a) f[a] = cam->look_at[a] - cam->pos[a];
  normalize3(f);
  double up[3] = { 0.0, 0.0, 1.0 };
  if (fabs(dot3(f, up)) > 0.999) { up[1] = 1.0; up[2] = 0.0; }
  cross3(f, up, right); normalize3(right);
  cross3(right, f, up2);
}

static void camera_dir(const double f[3], const double right[3], const double up2[3],
                       double tanh_fov, int width, int height, int col, int row, double d[3]) {
  double u = (2.0 * (col + 0.5) / width - 1.0) * tanh_fov;
  double v = (1.0 - 2.0 * (row + 0.5) / height) * tanh_fov;
  for (int a = 0; a < 3; ++a) d[a] = f[a] + u * right[a] + v * up2[a];
  normalize3(d);
}

/* PAPER.md:80 "To trace a primary ray we evaluate f at the camera"; pinhole model A13 */
void orc_gen_camera(const orc_camera* cam, int width, int height, float* o, float* d) {
  double f[3], right[3], up2[3], dd[3];
  camera_frame(cam, f, right, up2);
  double th = tan(0.5 * cam->fov_deg * ORC_PI / 180.0);
  for (int row = 0; row < height; ++row)
    for (int col = 0; col < width; ++col) {
      size_t i = (size_t)row * width + col;
      camera_dir(f, right, up2, th, width, height, col, row, dd);
      for (int a = 0; a < 3; ++a) { o[3*i + a] = (float)cam->pos[a]; d[3*i + a] = (float)dd[a]; }
    }
}

/* reading A14: p_i uniform on the sphere of the given radius, n_i = p_i / radius */
void orc_gen_sphere_points(uint64_t seed, uint64_t stream, int64_t n, double radius,
                           float* p, float* nrm) {
  for (int64_t i = 0; i < n; ++i) {
    double v[3];
    orc_dir_from_u(orc_uniform01(seed, stream, 2 * (uint64_t)i),
                   orc_uniform01(seed, stream, 2 * (uint64_t)i + 1), v);
    for (int a = 0; a < 3; ++a) { nrm[3*i + a] = (float)v[a]; p[3*i + a] = (float)(radius * v[a]); }
  }
}

/* PAPER.md:80 "take a surface point, offset it slightly along its normal, and evaluate f
 * toward the light"; tmax = distance to the light (reading A14) */
void orc_gen_shadow(const float* p, const float* nrm, int64_t n, const double light[3],
                    double eps, float* o, float* d, float* tmax) {
  for (int64_t i = 0; i < n; ++i) {
    double oo[3], dd[3];
    for (int a = 0; a < 3; ++a) oo[a] = (double)p[3*i + a] + eps * (double)nrm[3*i + a];
    for (int a = 0; a < 3; ++a) oo[a] = (double)(float)oo[a];   /* the origin the query will see */
    for (int a = 0; a < 3; ++a) dd[a] = light[a] - oo[a];
    double len = sqrt(dot3(dd, dd));
    for (int a = 0; a < 3; ++a) { o[3*i + a] = (float)oo[a]; d[3*i + a] = (float)(dd[a] / len); }
    if (tmax) tmax[i] = (float)len;
  }
}

/* reading A15: primary hits against a sphere inside an axis-aligned room seen from inside;
 * wall normals point inward. */
void orc_gen_gbuffer(const orc_camera* cam, const orc_scene* sc, int width, int height,
                     float* p, float* nrm, float* t_hit) {
  double f[3], right[3], up2[3], dd[3];
  camera_frame(cam, f, right, up2);
  double th = tan(0.5 * cam->fov_deg * ORC_PI / 180.0);
  for (int row = 0; row < height; ++row)
    for (int col = 0; col < width; ++col) {
      size_t i = (size_t)row * width + col;
      camera_dir(f, right, up2, th, width, height, col, row, dd);
      /* the ray the GPU sees has an fp32 direction */
      for (int a = 0; a < 3; ++a) dd[a] = (double)(float)dd[a];
      double oo[3] = { (double)(float)cam->pos[0], (double)(float)cam->pos[1], (double)(float)cam->pos[2] };
      int face = -1;
      double ts = orc_ray_sphere(oo, dd, sc->sphere_c, sc->sphere_r);
      double tb = orc_ray_box_exit(oo, dd, sc->box_min, sc->box_max, &face);
      double t, nn[3] = { 0.0, 0.0, 0.0 };
      if (ts > 0.0 && ts < tb) {
        t = ts;
        for (int a = 0; a < 3; ++a) nn[a] = (oo[a] + t * dd[a] - sc->sphere_c[a]) / sc->sphere_r;
      } else {
        t = tb;
        nn[face / 2] = (face & 1) ? -1.0 : 1.0;                /* inward */
      }
      for (int a = 0; a < 3; ++a) { p[3*i + a] = (float)(oo[a] + t * dd[a]); nrm[3*i + a] = (float)nn[a]; }
      if (t_hit) t_hit[i] = (float)t;
    }
}

/* reading A16: cosine-weighted hemisphere samples around n; rays pixel-major */
void orc_gen_ao(const float* p, const float* nrm, int64_t n_pts, int spp, uint64_t seed,
                uint64_t stream, double eps, float* o, float* d) {
  for (int64_t i = 0; i < n_pts; ++i) {
    double n[3] = { nrm[3*i], nrm[3*i + 1], nrm[3*i + 2] };
    /* tangent frame: cross the normal with the axis of its smallest-magnitude component */
    int ax = 0;
    if (fabs(n[1]) < fabs(n[ax])) ax = 1;
    if (fabs(n[2]) < fabs(n[ax])) ax = 2;
    double e[3] = { 0.0, 0.0, 0.0 }, t1[3], t2[3];
    e[ax] = 1.0;
    cross3(e, n, t1); normalize3(t1);
    cross3(n, t1, t2);
    for (int s = 0; s < spp; ++s) {
      uint64_t k = (uint64_t)i * (uint64_t)spp + (uint64_t)s;
      double u1 = orc_uniform01(seed, stream, 2 * k), u2 = orc_uniform01(seed, stream, 2 * k + 1);
      double r = sqrt(u1), phi = 2.0 * ORC_PI * u2;
      double lx = r * cos(phi), ly = r * sin(phi), lz = sqrt(1.0 - u1);
      double dd[3];
      for (int a = 0; a < 3; ++a) dd[a] = lx * t1[a] + ly * t2[a] + lz * n[a];
      normalize3(dd);
      for (int a = 0; a < 3; ++a) {
        o[3*k + a] = (float)((double)p[3*i + a] + eps * n[a]);
        d[3*k + a] = (float)dd[a];
      }
    }
  }
}

/* PAPER.md:80 "evaluate f along a set of directions over the hemisphere and average the hit
 * flag"; reading A17: ao = 1 - mean(xi > 0.5 and t < ao_radius) */
void orc_ao_reduce(const float* vis, const float* dist, int64_t n_pts, int spp,
                   double ao_radius, float* ao) {
  for (int64_t i = 0; i < n_pts; ++i) {
    int hits = 0;
    for (int s = 0; s < spp; ++s) {
      size_t k = (size_t)i * spp + s;
      if (vis[k] > 0.5f && (double)dist[k] < ao_radius) ++hits;
    }
    ao[i] = (float)(1.0 - (double)hits / (double)spp);
  }
}

/* ------------------------------------------------------------------ sphere tracing */

/* s(p) = (|p| - R) + alpha * MLP(p)   (reading A20); |p| in fp32 with a fixed fma order, the
 * MLP in fp64 (mode), the sum in fp32 - the same places the kernel uses fp32. */
static float sdf_value(const orc_layout* L, const void* blob, const float p[3], float base_radius,
                       float alpha, int mode, double* g, double* h, double* hin) {
  double z[2] = { 0.0, 0.0 };
  if (alpha != 0.0f) {
    encode_ray(L, p, NULL, g);
    forward_one(L, blob, g, mode, h, hin, z);
  }
  float n2 = fmaf(p[2], p[2], fmaf(p[1], p[1], p[0] * p[0]));
  return fmaf(alpha, (float)z[0], sqrtf(n2) - base_radius);
}

int orc_sdf_eval(const orc_layout* L, const void* blob, const float* p, int64_t n,
                 float base_radius, float alpha, int mode, double* s, int nthreads) {
  if (!layout_ok(L) || L->input_kind != 1 || L->n_out != 1) return -1;
  const int E = orc_enc_dim(L), S = L->width + E > 2 * E ? L->width + E : 2 * E;
#ifdef _OPENMP
  if (nthreads > 0) omp_set_num_threads(nthreads);
#endif
  #pragma omp parallel
  {
    double* g = (double*)malloc(sizeof(double) * E);
    double* h = (double*)malloc(sizeof(double) * S);
    double* hin = (double*)malloc(sizeof(double) * S);
    #pragma omp for schedule(dynamic, 4)
    for (int64_t i = 0; i < n; ++i)
      s[i] = (double)sdf_value(L, blob, p + 3 * i, base_radius, alpha, mode, g, h, hin);
    free(g); free(h); free(hin);
  }
  return 0;
}

/* PAPER.md:19 "Sphere tracing takes many small steps along each ray, and each step is a full
 * network evaluation"; "a sequential loop".  Step rule = reading A19:
 *   t = 0; for step in 0..max_steps-1: p = o + t d; s = SDF(p);
 *     if |s| < eps: hit, stop;  t += s;  if t > t_max or t < 0: miss, stop.
 *   not converged after max_steps: miss.   steps = number of SDF evaluations made. */
int orc_sphere_trace(const orc_layout* L, const void* blob, const float* o, const float* d,
                     int64_t n, int max_steps, float eps, float t_max, float base_radius,
                     float alpha, int mode, float* out_t, uint8_t* out_hit, int32_t* out_steps,
                     float* trace_p, float* trace_s, int nthreads) {
  return orc_sphere_trace_relaxed(L, blob, o, d, n, max_steps, eps, t_max, base_radius, alpha, 1.0f, mode,
                                  out_t, out_hit, out_steps, trace_p, trace_s, nthreads);
}

/* Over-relaxed sphere tracing (reading A19'): steps of omega * s with 1 <= omega < 2; when the
 * spheres at the previous and at the current point do not touch (|s| + |s_prev| < t - t_prev) the
 * relaxed step may have jumped a surface: go back to the plain position t_prev + s_prev and never
 * relax this ray again.  omega = 1 is the plain rule of A19, bit for bit. */
int orc_sphere_trace_relaxed(const orc_layout* L, const void* blob, const float* o, const float* d,
                             int64_t n, int max_steps, float eps, float t_max, float base_radius,
                             float alpha, float omega, int mode, float* out_t, uint8_t* out_hit, int32_t* out_steps,
                             float* trace_p, float* trace_s, int nthreads) {
  if (!layout_ok(L) || L->input_kind != 1 || L->n_out != 1) return -1;
  const int E = orc_enc_dim(L), S = L->width + E > 2 * E ? L->width + E : 2 * E;
#ifdef _OPENMP
  if (nthreads > 0) omp_set_num_threads(nthreads);
#endif
  #pragma omp parallel
  {
    double* g = (double*)malloc(sizeof(double) * E);
    double* h = (double*)malloc(sizeof(double) * S);
    double* hin = (double*)malloc(sizeof(double) * S);
    #pragma omp for schedule(dynamic, 1)
    for (int64_t i = 0; i < n; ++i) {
      float t = 0.0f, t_prev = 0.0f, s_prev = 0.0f, om = omega > 1.0f ? omega : 1.0f; int hit = 0, steps = 0, have_prev = 0;
      if (trace_p) for (int k = 0; k < 3 * max_steps; ++k) trace_p[(size_t)i * 3 * max_steps + k] = NAN;
      if (trace_s) for (int k = 0; k < max_steps; ++k) trace_s[(size_t)i * max_steps + k] = NAN;
      for (int step = 0; step < max_steps; ++step) {
        float p[3];
        for (int a = 0; a < 3; ++a) p[a] = fmaf(t, d[3*i + a], o[3*i + a]);
        float s = sdf_value(L, blob, p, base_radius, alpha, mode, g, h, hin);
        steps = step + 1;
        if (trace_p) for (int a = 0; a < 3; ++a) trace_p[((size_t)i * max_steps + step) * 3 + a] = p[a];
        if (trace_s) trace_s[(size_t)i * max_steps + step] = s;
        if (om > 1.0f && have_prev && fabsf(s) + fabsf(s_prev) < t - t_prev) {
          t = t_prev + s_prev; om = 1.0f; have_prev = 0;          /* redo from the plain position */
          if (t > t_max || t < 0.0f) break;
          continue;
        }
        if (fabsf(s) < eps) { hit = 1; break; }
        t_prev = t; s_prev = s; have_prev = 1;
        t = fmaf(om, s, t);
        if (t > t_max || t < 0.0f) break;
      }
      out_t[i] = t; out_hit[i] = (uint8_t)hit; out_steps[i] = steps;
    }
    free(g); free(h); free(hin);
  }
  return 0;
}

/* ------------------------------------------------------------------ wavefront secondary rays */

int64_t orc_gen_shadow_from_hits(const float* o, const float* d, const float* dist, const float* vis,
                                 int64_t n, const double light[3], float eps, float* o2, float* d2,
                                 float* tmax, int32_t* index) {
  int64_t k = 0;
  for (int64_t i = 0; i < n; ++i) {
    if (!(vis[i] > 0.5f)) continue;                       /* "when xi is high" */
    const float t = dist[i] - eps;                        /* stepped back along the ray */
    double p[3], v[3];
    for (int a = 0; a < 3; ++a) p[a] = (double)o[3 * i + a] + (double)t * (double)d[3 * i + a];
    for (int a = 0; a < 3; ++a) v[a] = light[a] - (double)(float)p[a];
    const double len = sqrt(v[0] * v[0] + v[1] * v[1] + v[2] * v[2]);
    for (int a = 0; a < 3; ++a) { o2[3 * k + a] = (float)p[a]; d2[3 * k + a] = (float)(v[a] / len); }
    tmax[k] = (float)len;
    index[k] = (int32_t)i;
    ++k;
  }
  return k;
}

void orc_shadow_lit(const float* vis2, const float* dist2, const float* tmax, const int32_t* index,
                    int64_t count, int64_t n, uint8_t* lit) {
  for (int64_t i = 0; i < n; ++i) lit[i] = 0;
  for (int64_t k = 0; k < count; ++k)                     /* occluded within the distance to the light */
    lit[index[k]] = (vis2[k] > 0.5f && dist2[k] < tmax[k]) ? 0 : 1;
}

/* reading W5: normal from the hit-point image */
static int pick_neighbour(const float* dist, const float* vis, int64_t i, int64_t step, int has_f, int has_b) {
  const int f = has_f && vis[i + step] > 0.5f, b = has_b && vis[i - step] > 0.5f;
  if (f && b) {
    const float df = fabsf(dist[i + step] - dist[i]), db = fabsf(dist[i - step] - dist[i]);   /* fp32 */
    return df <= db ? +1 : -1;
  }
  return f ? +1 : (b ? -1 : 0);
}

int64_t orc_hit_normals(const float* o, const float* d, const float* dist, const float* vis,
                        int width, int height, float* p, float* nrm, int32_t* index) {
  int64_t k = 0;
  for (int y = 0; y < height; ++y)
    for (int x = 0; x < width; ++x) {
      const int64_t i = (int64_t)y * width + x;
      if (!(vis[i] > 0.5f)) continue;
      double P[3], du[3], dv[3], n[3];
      for (int a = 0; a < 3; ++a) P[a] = (double)o[3 * i + a] + (double)dist[i] * (double)d[3 * i + a];
      const int su = pick_neighbour(dist, vis, i, 1, x + 1 < width, x >= 1);
      const int sv = pick_neighbour(dist, vis, i, width, y + 1 < height, y >= 1);
      int ok = su != 0 && sv != 0;
      if (ok) {
        const int64_t ju = i + su, jv = i + (int64_t)sv * width;
        for (int a = 0; a < 3; ++a) {
          const double Pu = (double)o[3 * ju + a] + (double)dist[ju] * (double)d[3 * ju + a];
          const double Pv = (double)o[3 * jv + a] + (double)dist[jv] * (double)d[3 * jv + a];
          du[a] = su * (Pu - P[a]);
          dv[a] = sv * (Pv - P[a]);
        }
        n[0] = du[1] * dv[2] - du[2] * dv[1];
        n[1] = du[2] * dv[0] - du[0] * dv[2];
        n[2] = du[0] * dv[1] - du[1] * dv[0];
        const double len = sqrt(n[0] * n[0] + n[1] * n[1] + n[2] * n[2]);
        if (len > 0.0 && len < INFINITY) {
          double dot = 0.0;
          for (int a = 0; a < 3; ++a) { n[a] /= len; dot += n[a] * (double)d[3 * i + a]; }
          if (dot > 0.0) for (int a = 0; a < 3; ++a) n[a] = -n[a];
        } else ok = 0;
      }
      if (!ok) for (int a = 0; a < 3; ++a) n[a] = -(double)d[3 * i + a];
      for (int a = 0; a < 3; ++a) { p[3 * k + a] = (float)P[a]; nrm[3 * k + a] = (float)n[a]; }
      index[k] = (int32_t)i;
      ++k;
    }
  return k;
}
