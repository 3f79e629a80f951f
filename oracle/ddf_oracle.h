/* ddf_oracle.h - CPU oracle for the DDF hot path.  TEST INFRASTRUCTURE, NOT PRODUCT.
 *
 * A plain, slow, obviously-correct restatement of what the path computes, written from
 * /root/reference/PAPER.md (cited as PAPER.md:<line>) and BASELINE.json's configs; fp64
 * arithmetic throughout (libm sin/cos/exp/log1p).  It shares no code with the CUDA path
 * under paper_2606_00817_b200/ and may only be used by tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs.
 *
 * Pins (tests/test_oracle_pins.py, -m "not gpu"): closed forms P1-P5, P7, brute force P6
 * (independent numpy evaluator), encoding worked example P3, generator analytics P9-P11,
 * sphere-tracer vs analytic ray-sphere P12 - see DESIGN.md "Oracle pins".
 * Parity unpinned: the absolute values of (t, xi) on the seeded random benchmark networks
 * have no external ground truth (no trained weights exist in the container).
 */
#ifndef DDF_ORACLE_H
#define DDF_ORACLE_H
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct orc_layout {
  int32_t input_kind;      /* 0 = ray (origin + direction), 1 = point */
  int32_t n_freq_origin;   /* L_o */
  int32_t n_freq_dir;      /* L_d (ignored for input_kind 1) */
  int32_t n_hidden;        /* Linear+ReLU layers */
  int32_t width;
  int32_t skip_layer;      /* layer whose input is [h ; gamma]; -1 none */
  int32_t n_out;           /* 2 = (distance logit, visibility logit); 1 = linear SDF value */
  int32_t weight_dtype;    /* 0 = fp32 blob, 1 = bf16 blob (uint16) */
} orc_layout;

typedef struct orc_camera { double pos[3]; double look_at[3]; double fov_deg; } orc_camera;
typedef struct orc_scene  { double sphere_c[3]; double sphere_r; double box_min[3]; double box_max[3]; } orc_scene;

/* ---- scalar pieces ---- */
double   orc_softplus(double z);                 /* max(z,0) + log1p(exp(-|z|))            */
double   orc_sigmoid(double z);                  /* 1/(1+exp(-z))                          */
double   orc_round_bf16(double x);               /* RNE to bf16 (of the fp32 rounding of x)*/
uint64_t orc_mix64(uint64_t z);
uint64_t orc_u64_at(uint64_t seed, uint64_t stream, uint64_t idx);
double   orc_uniform01(uint64_t seed, uint64_t stream, uint64_t idx);

/* ---- encoding + network ---- */
int  orc_enc_dim(const orc_layout* L);
/* gamma[n][E] (fp64).  d may be NULL for input_kind 1. */
void orc_encode(const orc_layout* L, const float* o, const float* d, int64_t n, double* gamma);
/* mode 0 = exact fp64; 1 = quantised (gamma and every post-ReLU activation rounded to bf16,
 * and fp32 weight blobs rounded to bf16, exactly where the GPU rounds - reading A11).
 * z[n][n_out] logits; dist[n] = softplus(z0), vis[n] = sigmoid(z1) when n_out == 2
 * (either may be NULL).  Returns 0, or -1 on a bad layout. */
int  orc_forward(const orc_layout* L, const void* blob, const float* o, const float* d,
                 int64_t n, int mode, double* z, double* dist, double* vis, int nthreads);

/* ---- analytic intersections (pins for the generators) ---- */
/* nearest t > 0 with |o + t d - c| = r, or -1 */
double orc_ray_sphere(const double o[3], const double d[3], const double c[3], double r);
/* exit distance of a ray starting inside the box; face = 0..5 (-x,+x,-y,+y,-z,+z) */
double orc_ray_box_exit(const double o[3], const double d[3], const double bmin[3],
                        const double bmax[3], int* face);

/* ---- generators (CPU twins of SURVEY.md rows a9-a11) ---- */
void orc_dir_from_u(double u1, double u2, double out[3]);            /* reading A9 */
void orc_camera_from_seed(uint64_t seed, uint64_t stream, double radius, orc_camera* cam);
void orc_gen_camera(const orc_camera* cam, int width, int height, float* o, float* d);
void orc_gen_sphere_points(uint64_t seed, uint64_t stream, int64_t n, double radius,
                           float* p, float* nrm);
void orc_gen_shadow(const float* p, const float* nrm, int64_t n, const double light[3],
                    double eps, float* o, float* d, float* tmax);
void orc_gen_gbuffer(const orc_camera* cam, const orc_scene* sc, int width, int height,
                     float* p, float* nrm, float* t_hit);
void orc_gen_ao(const float* p, const float* nrm, int64_t n_pts, int spp, uint64_t seed,
                uint64_t stream, double eps, float* o, float* d);
void orc_ao_reduce(const float* vis, const float* dist, int64_t n_pts, int spp,
                   double ao_radius, float* ao);

/* ---- wavefront secondary rays (PAPER.md:62 hit point x + t d; PAPER.md:80 shadow test) ----
 * for every i with vis[i] > 0.5, in increasing i: o2 = o_i + (dist_i - eps) d_i (fp32 subtraction,
 * the rest in fp64, rounded to fp32), d2 = normalise(light - o2), tmax = |light - o2|, index = i.
 * Returns the number of secondary rays. */
int64_t orc_gen_shadow_from_hits(const float* o, const float* d, const float* dist, const float* vis,
                                 int64_t n, const double light[3], float eps, float* o2, float* d2,
                                 float* tmax, int32_t* index);
/* lit[i] = 1 iff ray i hit and its shadow ray is not occluded (vis2 > 0.5 and dist2 < tmax) */
void orc_shadow_lit(const float* vis2, const float* dist2, const float* tmax, const int32_t* index,
                    int64_t count, int64_t n, uint8_t* lit);

/* ---- normals of the field's own hits (reading W5; "offset it slightly
 * along its normal": the field returns no normal, so it is estimated from the hit-point image) ----
 * The primary batch is a width x height image, ray i = y * width + x.  For every i with vis[i] > 0.5,
 * in increasing i: P_i = o_i + dist_i d_i; along x the difference is taken toward the neighbour that
 * also hit (both hit: the one with the smaller |dist_j - dist_i| in fp32, forward on ties): forward
 * P_{i+1} - P_i, backward P_i - P_{i-1}; along y likewise with +-width.  n = normalise(du x dv), turned
 * so that n . d_i <= 0; if an axis has no hit neighbour, or the product vanishes, n = -d_i.
 * Writes the compacted p, nrm [count][3] and index [count]; returns count.  fp64 but for the stated
 * fp32 comparison. */
int64_t orc_hit_normals(const float* o, const float* d, const float* dist, const float* vis,
                        int width, int height, float* p, float* nrm, int32_t* index);

/* ---- sphere tracing of s(p) = (|p| - base_radius) + alpha * MLP(p)  (readings A19, A20) ----
 * Ray state (t, p, s) is carried in fp32 exactly as the kernel carries it; the MLP itself is
 * evaluated by orc_forward in `mode`.  trace_p/trace_s (may be NULL) receive, for every ray,
 * the visited points [n][max_steps][3] and values [n][max_steps] (unvisited = NaN). */
int orc_sphere_trace(const orc_layout* L, const void* blob, const float* o, const float* d,
                     int64_t n, int max_steps, float eps, float t_max, float base_radius,
                     float alpha, int mode, float* out_t, uint8_t* out_hit, int32_t* out_steps,
                     float* trace_p, float* trace_s, int nthreads);
/* the same with over-relaxed steps (rule in ddf_oracle.c); omega <= 1: plain */
int orc_sphere_trace_relaxed(const orc_layout* L, const void* blob, const float* o, const float* d,
                             int64_t n, int max_steps, float eps, float t_max, float base_radius,
                             float alpha, float omega, int mode, float* out_t, uint8_t* out_hit,
                             int32_t* out_steps, float* trace_p, float* trace_s, int nthreads);
/* value of s at given points (teacher forcing, pin P12) */
int orc_sdf_eval(const orc_layout* L, const void* blob, const float* p, int64_t n,
                 float base_radius, float alpha, int mode, double* s, int nthreads);

#ifdef __cplusplus
}
#endif
#endif
