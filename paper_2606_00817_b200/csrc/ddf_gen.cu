// ddf_gen.cu - device-side secondary-ray generators and reducers (Sec. III-C:
// primary ray / shadow test / ambient occlusion recipes; shapes from BASELINE.json configs 1-3).
// Streaming kernels: one thread per ray (or point), coalesced through 3-float rows.
#include "ddf_common.cuh"
#include "ddf_camera.cuh"
#include <math.h>

namespace ddf {

static inline uint64_t host_mix64(uint64_t z) {
  z += 0x9E3779B97F4A7C15ull;
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
  return z ^ (z >> 31);
}
static inline uint64_t host_key(uint64_t seed, uint64_t stream) { return host_mix64(host_mix64(seed) ^ stream); }

__global__ void gen_camera_kernel(CamFrame c, int width, int height, float* __restrict__ o, float* __restrict__ d) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= (int64_t)width * height) return;
  float dd[3];
  pixel_dir(c, width, height, (int)(i % width), (int)(i / width), dd);
  #pragma unroll
  for (int a = 0; a < 3; ++a) { o[3 * i + a] = c.pos[a]; d[3 * i + a] = dd[a]; }
}

__device__ __forceinline__ void dir_from_u(float u1, float u2, float v[3]) {
  float z = 2.0f * u1 - 1.0f, s, c;
  sincospif(2.0f * u2, &s, &c);
  float r = sqrtf(fmaxf(0.0f, 1.0f - z * z));
  v[0] = r * c; v[1] = r * s; v[2] = z;
}

__global__ void gen_sphere_points_kernel(uint64_t key, int64_t n, float radius, float* __restrict__ p, float* __restrict__ nrm) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  float v[3];
  dir_from_u(dev_uniform01(key, 2 * (uint64_t)i), dev_uniform01(key, 2 * (uint64_t)i + 1), v);
  #pragma unroll
  for (int a = 0; a < 3; ++a) { nrm[3 * i + a] = v[a]; p[3 * i + a] = radius * v[a]; }
}

__global__ void gen_shadow_kernel(const float* __restrict__ p, const float* __restrict__ nrm, int64_t n,
                                  float lx, float ly, float lz, float eps,
                                  float* __restrict__ o, float* __restrict__ d, float* __restrict__ tmax) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  float ox = fmaf(eps, nrm[3 * i], p[3 * i]), oy = fmaf(eps, nrm[3 * i + 1], p[3 * i + 1]), oz = fmaf(eps, nrm[3 * i + 2], p[3 * i + 2]);
  float dx = lx - ox, dy = ly - oy, dz = lz - oz;
  float len = sqrtf(fmaf(dz, dz, fmaf(dy, dy, dx * dx)));
  float inv = 1.0f / len;
  o[3 * i] = ox; o[3 * i + 1] = oy; o[3 * i + 2] = oz;
  d[3 * i] = dx * inv; d[3 * i + 1] = dy * inv; d[3 * i + 2] = dz * inv;
  if (tmax) tmax[i] = len;
}

// G-buffer: ray-sphere by the quadratic, ray-box by slabs from inside; the intersection itself is
// done in fp64 so that grazing rays agree with the analytic result.
__global__ void gen_gbuffer_kernel(CamFrame c, ddf_scene sc, int width, int height,
                                   float* __restrict__ p, float* __restrict__ nrm, float* __restrict__ t_hit) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= (int64_t)width * height) return;
  float df[3];
  pixel_dir(c, width, height, (int)(i % width), (int)(i / width), df);
  double o[3] = { c.pos[0], c.pos[1], c.pos[2] }, d[3] = { df[0], df[1], df[2] };
  double oc[3] = { o[0] - sc.sphere_c[0], o[1] - sc.sphere_c[1], o[2] - sc.sphere_c[2] };
  double b = oc[0]*d[0] + oc[1]*d[1] + oc[2]*d[2];
  double cc = oc[0]*oc[0] + oc[1]*oc[1] + oc[2]*oc[2] - (double)sc.sphere_r * (double)sc.sphere_r;
  double disc = b * b - cc, ts = -1.0;
  if (disc >= 0.0) { double sq = sqrt(disc); ts = (-b - sq > 0.0) ? -b - sq : ((-b + sq > 0.0) ? -b + sq : -1.0); }
  double tb = INFINITY; int face = -1;
  #pragma unroll
  for (int a = 0; a < 3; ++a) {
    if (d[a] > 0.0) { double t = ((double)sc.box_max[a] - o[a]) / d[a]; if (t < tb) { tb = t; face = 2 * a + 1; } }
    else if (d[a] < 0.0) { double t = ((double)sc.box_min[a] - o[a]) / d[a]; if (t < tb) { tb = t; face = 2 * a; } }
  }
  double t; double nn[3] = { 0.0, 0.0, 0.0 };
  if (ts > 0.0 && ts < tb) {
    t = ts;
    #pragma unroll
    for (int a = 0; a < 3; ++a) nn[a] = (o[a] + t * d[a] - (double)sc.sphere_c[a]) / (double)sc.sphere_r;
  } else {
    t = tb;
    #pragma unroll
    for (int a = 0; a < 3; ++a) if (face / 2 == a) nn[a] = (face & 1) ? -1.0 : 1.0;
  }
  #pragma unroll
  for (int a = 0; a < 3; ++a) { p[3 * i + a] = (float)(o[a] + t * d[a]); nrm[3 * i + a] = (float)nn[a]; }
  if (t_hit) t_hit[i] = (float)t;
}

// AO rays: one thread per ray (pixel-major, spp consecutive rays per point).
// n_pts_dev (device, optional) overrides n_pts; it can only be smaller.
__global__ void gen_ao_kernel(const float* __restrict__ p, const float* __restrict__ nrm, int64_t n_pts,
                              const int64_t* __restrict__ n_pts_dev, int spp,
                              uint64_t key, float eps, float* __restrict__ o, float* __restrict__ d) {
  int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (n_pts_dev) n_pts = *n_pts_dev;
  if (k >= n_pts * spp) return;
  int64_t i = k / spp;
  const float n[3] = { nrm[3 * i], nrm[3 * i + 1], nrm[3 * i + 2] };
  const float pp[3] = { p[3 * i], p[3 * i + 1], p[3 * i + 2] };
  float oo[3], dd[3];
  ao_ray_from_point(pp, n, key, k, eps, oo, dd);
  #pragma unroll
  for (int a = 0; a < 3; ++a) { o[3 * k + a] = oo[a]; d[3 * k + a] = dd[a]; }
}

__global__ void ao_reduce_kernel(const float* __restrict__ vis, const float* __restrict__ dist, int64_t n_pts, int spp,
                                 float ao_radius, float* __restrict__ ao) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n_pts) return;
  int hits = 0;
  if (spp % 4 == 0 && (((uintptr_t)vis | (uintptr_t)dist) & 15) == 0) {
    const float4* v4 = reinterpret_cast<const float4*>(vis + i * spp);
    const float4* d4 = reinterpret_cast<const float4*>(dist + i * spp);
    for (int s = 0; s < spp / 4; ++s) {
      float4 v = v4[s], t = d4[s];
      hits += (v.x > 0.5f && t.x < ao_radius) + (v.y > 0.5f && t.y < ao_radius) +
              (v.z > 0.5f && t.z < ao_radius) + (v.w > 0.5f && t.w < ao_radius);
    }
  } else {
    for (int s = 0; s < spp; ++s) hits += (vis[i * spp + s] > 0.5f && dist[i * spp + s] < ao_radius);
  }
  ao[i] = 1.0f - (float)hits / (float)spp;
}

__global__ void shadow_test_kernel(const float* __restrict__ vis, const float* __restrict__ dist,
                                   const float* __restrict__ tmax, int64_t n, uint8_t* __restrict__ shadow) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) shadow[i] = (vis[i] > 0.5f && dist[i] < tmax[i]) ? 1 : 0;
}

static inline unsigned blocks_for(int64_t n, int t) { return (unsigned)((n + t - 1) / t); }

uint64_t gen_key(uint64_t seed, uint64_t rng_stream) { return host_key(seed, rng_stream); }

int gen_ao_launch(const float* p, const float* nrm, int64_t n_pts, const int64_t* n_pts_dev, int spp, uint64_t seed,
                  uint64_t rng_stream, float eps, float* o, float* d, cudaStream_t st) {
  gen_ao_kernel<<<blocks_for(n_pts * spp, 256), 256, 0, st>>>(p, nrm, n_pts, n_pts_dev, spp, host_key(seed, rng_stream), eps, o, d);
  DDF_CUDA_TRY(cudaGetLastError());
  return DDF_OK;
}

}  // namespace ddf

using namespace ddf;

extern "C" int ddf_camera_from_seed(uint64_t seed, uint64_t stream, float radius, ddf_camera* out) {
  if (!out) return DDF_E_INVALID_ARG;
  uint64_t key = host_key(seed, stream);
  double u1 = (double)(host_mix64(key ^ 0ull) >> 40) / 16777216.0;
  double u2 = (double)(host_mix64(key ^ 1ull) >> 40) / 16777216.0;
  double z = 2.0 * u1 - 1.0, phi = 2.0 * 3.14159265358979323846 * u2, s = sqrt(fmax(0.0, 1.0 - z * z));
  out->pos[0] = (float)(radius * s * cos(phi)); out->pos[1] = (float)(radius * s * sin(phi)); out->pos[2] = (float)(radius * z);
  out->look_at[0] = out->look_at[1] = out->look_at[2] = 0.0f;
  out->fov_deg = 50.0f;
  return DDF_OK;
}

extern "C" int ddf_gen_camera(const ddf_camera* cam, int width, int height, float* o, float* d, void* stream) {
  if (!cam || width < 0 || height < 0) return DDF_E_INVALID_ARG;
  int64_t n = (int64_t)width * height;
  if (n == 0) return DDF_OK;
  if (!o || !d) return DDF_E_INVALID_ARG;
  gen_camera_kernel<<<blocks_for(n, 256), 256, 0, (cudaStream_t)stream>>>(make_frame(cam), width, height, o, d);
  DDF_CUDA_TRY(cudaGetLastError());
  return DDF_OK;
}

extern "C" int ddf_gen_sphere_points(uint64_t seed, uint64_t rng_stream, int64_t n, float radius,
                                     float* p, float* nrm, void* stream) {
  if (n < 0) return DDF_E_INVALID_ARG;
  if (n == 0) return DDF_OK;
  if (!p || !nrm) return DDF_E_INVALID_ARG;
  gen_sphere_points_kernel<<<blocks_for(n, 256), 256, 0, (cudaStream_t)stream>>>(host_key(seed, rng_stream), n, radius, p, nrm);
  DDF_CUDA_TRY(cudaGetLastError());
  return DDF_OK;
}

extern "C" int ddf_gen_shadow(const float* p, const float* nrm, int64_t n, const float light[3], float eps,
                              float* o, float* d, float* tmax, void* stream) {
  if (n < 0 || !light) return DDF_E_INVALID_ARG;
  if (n == 0) return DDF_OK;
  if (!p || !nrm || !o || !d) return DDF_E_INVALID_ARG;
  gen_shadow_kernel<<<blocks_for(n, 256), 256, 0, (cudaStream_t)stream>>>(p, nrm, n, light[0], light[1], light[2], eps, o, d, tmax);
  DDF_CUDA_TRY(cudaGetLastError());
  return DDF_OK;
}

extern "C" int ddf_gen_gbuffer(const ddf_camera* cam, const ddf_scene* scene, int width, int height,
                               float* p, float* nrm, float* t_hit, void* stream) {
  if (!cam || !scene || width < 0 || height < 0) return DDF_E_INVALID_ARG;
  int64_t n = (int64_t)width * height;
  if (n == 0) return DDF_OK;
  if (!p || !nrm) return DDF_E_INVALID_ARG;
  gen_gbuffer_kernel<<<blocks_for(n, 256), 256, 0, (cudaStream_t)stream>>>(make_frame(cam), *scene, width, height, p, nrm, t_hit);
  DDF_CUDA_TRY(cudaGetLastError());
  return DDF_OK;
}

extern "C" int ddf_gen_ao(const float* p, const float* nrm, int64_t n_pts, int spp, uint64_t seed,
                          uint64_t rng_stream, float eps, float* o, float* d, void* stream) {
  if (n_pts < 0 || spp <= 0) return DDF_E_INVALID_ARG;
  if (n_pts == 0) return DDF_OK;
  if (!p || !nrm || !o || !d) return DDF_E_INVALID_ARG;
  return gen_ao_launch(p, nrm, n_pts, nullptr, spp, seed, rng_stream, eps, o, d, (cudaStream_t)stream);
}

extern "C" int ddf_ao_reduce(const float* vis, const float* dist, int64_t n_pts, int spp, float ao_radius,
                             float* ao, void* stream) {
  if (n_pts < 0 || spp <= 0) return DDF_E_INVALID_ARG;
  if (n_pts == 0) return DDF_OK;
  if (!vis || !dist || !ao) return DDF_E_INVALID_ARG;
  ao_reduce_kernel<<<blocks_for(n_pts, 128), 128, 0, (cudaStream_t)stream>>>(vis, dist, n_pts, spp, ao_radius, ao);
  DDF_CUDA_TRY(cudaGetLastError());
  return DDF_OK;
}

extern "C" int ddf_shadow_test(const float* vis, const float* dist, const float* tmax, int64_t n,
                               uint8_t* shadow, void* stream) {
  if (n < 0) return DDF_E_INVALID_ARG;
  if (n == 0) return DDF_OK;
  if (!vis || !dist || !tmax || !shadow) return DDF_E_INVALID_ARG;
  shadow_test_kernel<<<blocks_for(n, 256), 256, 0, (cudaStream_t)stream>>>(vis, dist, tmax, n, shadow);
  DDF_CUDA_TRY(cudaGetLastError());
  return DDF_OK;
}
