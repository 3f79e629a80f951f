// ddf_camera.cuh - the pinhole camera frame shared by the camera generator (ddf_gen.cu) and the
// kernels that generate primary rays themselves (ddf_query_camera): one definition, so both give
// the same bits (reading A13: up = z with a y fall-back, pixel centres, fov = full angle).
#pragma once
#include "ddf_common.cuh"
#include <math.h>

namespace ddf {

struct CamFrame { float pos[3], f[3], r[3], u[3], tan_half; };

static inline CamFrame make_frame(const ddf_camera* cam) {
  double f[3], up[3] = {0, 0, 1}, r[3], u[3];
  for (int a = 0; a < 3; ++a) f[a] = (double)cam->look_at[a] - (double)cam->pos[a];
  double n = sqrt(f[0]*f[0] + f[1]*f[1] + f[2]*f[2]);
  for (int a = 0; a < 3; ++a) f[a] /= n;
  if (fabs(f[2]) > 0.999) { up[1] = 1; up[2] = 0; }
  r[0] = f[1]*up[2] - f[2]*up[1]; r[1] = f[2]*up[0] - f[0]*up[2]; r[2] = f[0]*up[1] - f[1]*up[0];
  n = sqrt(r[0]*r[0] + r[1]*r[1] + r[2]*r[2]);
  for (int a = 0; a < 3; ++a) r[a] /= n;
  u[0] = r[1]*f[2] - r[2]*f[1]; u[1] = r[2]*f[0] - r[0]*f[2]; u[2] = r[0]*f[1] - r[1]*f[0];
  CamFrame cf;
  for (int a = 0; a < 3; ++a) { cf.pos[a] = cam->pos[a]; cf.f[a] = (float)f[a]; cf.r[a] = (float)r[a]; cf.u[a] = (float)u[a]; }
  cf.tan_half = (float)tan(0.5 * (double)cam->fov_deg * 3.14159265358979323846 / 180.0);
  return cf;
}

__device__ __forceinline__ void pixel_dir(const CamFrame& c, int width, int height, int col, int row, float d[3]) {
  float u = (2.0f * ((float)col + 0.5f) / (float)width - 1.0f) * c.tan_half;
  float v = (1.0f - 2.0f * ((float)row + 0.5f) / (float)height) * c.tan_half;
  float x = fmaf(v, c.u[0], fmaf(u, c.r[0], c.f[0]));
  float y = fmaf(v, c.u[1], fmaf(u, c.r[1], c.f[1]));
  float z = fmaf(v, c.u[2], fmaf(u, c.r[2], c.f[2]));
  float inv = 1.0f / sqrtf(fmaf(z, z, fmaf(y, y, x * x)));
  d[0] = x * inv; d[1] = y * inv; d[2] = z * inv;
}


}  // namespace ddf
