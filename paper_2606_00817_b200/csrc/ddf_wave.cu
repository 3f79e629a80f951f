// ddf_wave.cu - wavefront secondary rays: primary query -> hit points -> compacted shadow rays ->
// second query -> lit flags (include/ddf.h).  The compaction is a stable
// three-kernel scan (per-block counts, one-block scan of the counts, scatter), so the secondary
// batch is in increasing primary-ray order and reproducible; its size stays on the device and is
// read by the query kernels themselves (n_dev), so the loop needs no host round trip.
#include "ddf_common.cuh"
#include <mutex>

namespace ddf {

constexpr int kWaveBlock = 256;

__global__ void wave_count_kernel(const float* __restrict__ vis, int64_t n, int32_t* __restrict__ block_counts) {
  const int64_t i = (int64_t)blockIdx.x * kWaveBlock + threadIdx.x;
  const int hit = (i < n) && (vis[i] > 0.5f);
  const int c = __syncthreads_count(hit);
  if (threadIdx.x == 0) block_counts[blockIdx.x] = c;
}

// exclusive scan of the block counts in place (one block), total -> *count
__global__ void wave_scan_kernel(int32_t* __restrict__ block_counts, int64_t n_blocks, int64_t* __restrict__ count,
                                 int64_t* __restrict__ count_scaled, int scale) {
  __shared__ int32_t warp_sums[32];
  __shared__ int64_t carry;
  if (threadIdx.x == 0) carry = 0;
  __syncthreads();
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  for (int64_t base = 0; base < n_blocks; base += blockDim.x) {
    const int64_t i = base + threadIdx.x;
    const int32_t v = (i < n_blocks) ? block_counts[i] : 0;
    int32_t x = v;
    #pragma unroll
    for (int s = 1; s < 32; s <<= 1) { const int32_t y = __shfl_up_sync(0xffffffffu, x, s); if (lane >= s) x += y; }
    if (lane == 31) warp_sums[warp] = x;
    __syncthreads();
    if (warp == 0) {
      int32_t w = (lane < (int)(blockDim.x >> 5)) ? warp_sums[lane] : 0;
      #pragma unroll
      for (int s = 1; s < 32; s <<= 1) { const int32_t y = __shfl_up_sync(0xffffffffu, w, s); if (lane >= s) w += y; }
      warp_sums[lane] = w;                                   // inclusive over warps
    }
    __syncthreads();
    const int64_t before = carry + (warp ? warp_sums[warp - 1] : 0) + (x - v);
    if (i < n_blocks) block_counts[i] = (int32_t)before;     // n <= 2^31 - 1 rays
    __syncthreads();
    if (threadIdx.x == blockDim.x - 1) carry += warp_sums[(blockDim.x >> 5) - 1];
    __syncthreads();
  }
  if (threadIdx.x == 0) { *count = carry; if (count_scaled) *count_scaled = carry * scale; }
}

__global__ void wave_scatter_kernel(const float* __restrict__ o, const float* __restrict__ d,
                                    const float* __restrict__ dist, const float* __restrict__ vis, int64_t n,
                                    float lx, float ly, float lz, float eps, const int32_t* __restrict__ block_offsets,
                                    float* __restrict__ o2, float* __restrict__ d2, float* __restrict__ tmax,
                                    int32_t* __restrict__ index) {
  __shared__ int32_t warp_base[kWaveBlock / 32];
  const int64_t i = (int64_t)blockIdx.x * kWaveBlock + threadIdx.x;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const bool hit = (i < n) && (vis[i] > 0.5f);
  const uint32_t m = __ballot_sync(0xffffffffu, hit);
  if (lane == 0) warp_base[warp] = __popc(m);
  __syncthreads();
  if (threadIdx.x == 0) {
    int32_t run = 0;
    for (int w = 0; w < kWaveBlock / 32; ++w) { const int32_t c = warp_base[w]; warp_base[w] = run; run += c; }
  }
  __syncthreads();
  if (!hit) return;
  const int64_t k = (int64_t)block_offsets[blockIdx.x] + warp_base[warp] + __popc(m & ((1u << lane) - 1u));
  const float t = dist[i] - eps;
  const float ox = fmaf(t, d[3 * i], o[3 * i]), oy = fmaf(t, d[3 * i + 1], o[3 * i + 1]), oz = fmaf(t, d[3 * i + 2], o[3 * i + 2]);
  const float dx = lx - ox, dy = ly - oy, dz = lz - oz;
  const float len = sqrtf(fmaf(dz, dz, fmaf(dy, dy, dx * dx)));
  const float inv = 1.0f / len;
  o2[3 * k] = ox; o2[3 * k + 1] = oy; o2[3 * k + 2] = oz;
  d2[3 * k] = dx * inv; d2[3 * k + 1] = dy * inv; d2[3 * k + 2] = dz * inv;
  tmax[k] = len;
  index[k] = (int32_t)i;
}

// bit `bit` of lit[index[k]] = light not occluded, for k < *count (lit was zeroed before: primary misses stay 0;
// every k owns its own byte, and the lights run one after the other in the stream); the last light also
// reports the number of shadow rays traced, *count x n_lights
__global__ void wave_lit_kernel(const float* __restrict__ vis2, const float* __restrict__ dist2,
                                const float* __restrict__ tmax, const int32_t* __restrict__ index,
                                const int64_t* __restrict__ count, uint8_t* __restrict__ lit, int bit,
                                int64_t* __restrict__ out_count, int n_lights) {
  const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (k == 0 && out_count) *out_count = *count * n_lights;
  if (k >= *count) return;
  if (!(vis2[k] > 0.5f && dist2[k] < tmax[k])) lit[index[k]] |= (uint8_t)(1u << bit);
}

// ---- ambient occlusion at the field's own hits (readings W5 / W6) ----
// which neighbour the difference along one image axis goes to: +1 forward, -1 backward, 0 none
__device__ __forceinline__ int wave_pick_neighbour(const float* __restrict__ dist, const float* __restrict__ vis,
                                                   int64_t i, int64_t step, bool has_f, bool has_b) {
  const bool f = has_f && vis[i + step] > 0.5f, b = has_b && vis[i - step] > 0.5f;
  if (f && b) {
    const float t = dist[i];
    return fabsf(__fsub_rn(dist[i + step], t)) <= fabsf(__fsub_rn(dist[i - step], t)) ? 1 : -1;
  }
  return f ? 1 : (b ? -1 : 0);
}
__device__ __forceinline__ void wave_hit_point(const float* __restrict__ o, const float* __restrict__ d,
                                               const float* __restrict__ dist, int64_t i, float P[3]) {
  const float t = dist[i];
  #pragma unroll
  for (int a = 0; a < 3; ++a) P[a] = fmaf(t, d[3 * i + a], o[3 * i + a]);
}

// stable compaction of the hits of a width x height primary batch with the hit point and the normal
// estimated from the hit-point image; nrm_img (optional, [n][3]) also receives the normal per pixel (0 = miss)
__global__ void wave_normals_scatter_kernel(const float* __restrict__ o, const float* __restrict__ d,
                                            const float* __restrict__ dist, const float* __restrict__ vis,
                                            int width, int height, const int32_t* __restrict__ block_offsets,
                                            float* __restrict__ p_c, float* __restrict__ n_c, int32_t* __restrict__ index,
                                            float* __restrict__ nrm_img) {
  __shared__ int32_t warp_base[kWaveBlock / 32];
  const int64_t n = (int64_t)width * height;
  const int64_t i = (int64_t)blockIdx.x * kWaveBlock + threadIdx.x;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const bool hit = (i < n) && (vis[i] > 0.5f);
  const uint32_t m = __ballot_sync(0xffffffffu, hit);
  if (lane == 0) warp_base[warp] = __popc(m);
  __syncthreads();
  if (threadIdx.x == 0) {
    int32_t run = 0;
    for (int w = 0; w < kWaveBlock / 32; ++w) { const int32_t c = warp_base[w]; warp_base[w] = run; run += c; }
  }
  __syncthreads();
  if (!hit) {
    if (nrm_img && i < n) { nrm_img[3 * i] = 0.0f; nrm_img[3 * i + 1] = 0.0f; nrm_img[3 * i + 2] = 0.0f; }
    return;
  }
  const int64_t k = (int64_t)block_offsets[blockIdx.x] + warp_base[warp] + __popc(m & ((1u << lane) - 1u));
  const int x = (int)(i % width), y = (int)(i / width);
  float P[3], nn[3] = { -d[3 * i], -d[3 * i + 1], -d[3 * i + 2] };
  wave_hit_point(o, d, dist, i, P);
  const int su = wave_pick_neighbour(dist, vis, i, 1, x + 1 < width, x >= 1);
  const int sv = wave_pick_neighbour(dist, vis, i, width, y + 1 < height, y >= 1);
  if (su != 0 && sv != 0) {
    float Pu[3], Pv[3], du[3], dv[3];
    wave_hit_point(o, d, dist, i + su, Pu);
    wave_hit_point(o, d, dist, i + (int64_t)sv * width, Pv);
    #pragma unroll
    for (int a = 0; a < 3; ++a) { du[a] = (float)su * (Pu[a] - P[a]); dv[a] = (float)sv * (Pv[a] - P[a]); }
    const float cx = du[1] * dv[2] - du[2] * dv[1], cy = du[2] * dv[0] - du[0] * dv[2], cz = du[0] * dv[1] - du[1] * dv[0];
    const float len = sqrtf(fmaf(cz, cz, fmaf(cy, cy, cx * cx)));
    if (len > 0.0f && len < INFINITY) {
      const float inv = 1.0f / len;
      float c[3] = { cx * inv, cy * inv, cz * inv };
      const float dot = fmaf(c[2], d[3 * i + 2], fmaf(c[1], d[3 * i + 1], c[0] * d[3 * i]));
      const float sgn = dot > 0.0f ? -1.0f : 1.0f;
      #pragma unroll
      for (int a = 0; a < 3; ++a) nn[a] = sgn * c[a];
    }
  }
  #pragma unroll
  for (int a = 0; a < 3; ++a) { p_c[3 * k + a] = P[a]; n_c[3 * k + a] = nn[a]; }
  index[k] = (int32_t)i;
  if (nrm_img) { nrm_img[3 * i] = nn[0]; nrm_img[3 * i + 1] = nn[1]; nrm_img[3 * i + 2] = nn[2]; }
}

// out_ao[i] = 1 where the primary ray missed, the AO of its compacted slot where it hit; also reports
// the number of AO rays traced
__global__ void wave_ao_scatter_kernel(const float* __restrict__ vis, int64_t n, const float* __restrict__ ao_c,
                                       const int32_t* __restrict__ index, const int64_t* __restrict__ count,
                                       float* __restrict__ out_ao, int64_t* __restrict__ out_count, int spp) {
  const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (k == 0 && out_count) *out_count = *count * spp;
  if (k < n && !(vis[k] > 0.5f)) out_ao[k] = 1.0f;
  if (k < *count) out_ao[index[k]] = ao_c[k];
}

int scan_block_counts(int32_t* block_counts, int64_t n_blocks, int64_t* count, cudaStream_t st) {
  wave_scan_kernel<<<1, 1024, 0, st>>>(block_counts, n_blocks, count, nullptr, 1);
  DDF_CUDA_TRY(cudaGetLastError());
  return DDF_OK;
}

int wave_reserve_bytes(Model* m, size_t need) {
  if (need <= m->wave_ws_bytes) return DDF_OK;
  cudaFree(m->wave_ws); m->wave_ws = nullptr; m->wave_ws_bytes = 0;
  DDF_CUDA_TRY(cudaMalloc(&m->wave_ws, need));
  m->wave_ws_bytes = need;
  return DDF_OK;
}
// the largest workspace any wavefront call needs for n primary rays (spp AO rays per hit; 0: shadows only)
int wave_reserve(Model* m, int64_t n, int spp) {
  const size_t nb = (size_t)((n + kWaveBlock - 1) / kWaveBlock);
  const size_t a = (size_t)((n + 63) / 64 * 64);
  const size_t head = ((nb * 4 + 255) / 256) * 256 + 256;
  size_t need = head + a * (12 + 12 + 4 + 4 + 4 + 4);
  if (spp > 0) { const size_t ao = head + a * (12 + 12 + 4 + 4) + a * (size_t)spp * 24; if (ao > need) need = ao; }
  return wave_reserve_bytes(m, need);
}

struct WaveWs { int32_t* block_counts; float *o2, *d2, *tmax, *dist2, *vis2; int32_t* index; int64_t* count; };

// workspace: block counts always; the ray buffers only for ddf_query_shadowed (full = true)
static int wave_ws(Model* m, int64_t n, bool full, WaveWs* w) {
  const size_t nb = (size_t)((n + kWaveBlock - 1) / kWaveBlock);
  const size_t a = (size_t)((n + 63) / 64 * 64);
  size_t need = ((nb * 4 + 255) / 256) * 256 + 256;
  if (full) need += a * (12 + 12 + 4 + 4 + 4 + 4);
  { int rc = wave_reserve_bytes(m, need); if (rc != DDF_OK) return rc; }
  uint8_t* b = (uint8_t*)m->wave_ws;
  w->count = (int64_t*)b;                 b += 256;
  w->block_counts = (int32_t*)b;          b += ((nb * 4 + 255) / 256) * 256;
  if (full) {
    w->o2 = (float*)b;    b += a * 12;
    w->d2 = (float*)b;    b += a * 12;
    w->tmax = (float*)b;  b += a * 4;
    w->dist2 = (float*)b; b += a * 4;
    w->vis2 = (float*)b;  b += a * 4;
    w->index = (int32_t*)b;
  }
  return DDF_OK;
}

// count + scan once per primary batch, then one scatter per light
static int wave_count(const WaveWs& w, const float* vis, int64_t n, int64_t* count, cudaStream_t st,
                      int64_t* count_scaled = nullptr, int scale = 1) {
  const unsigned nb = (unsigned)((n + kWaveBlock - 1) / kWaveBlock);
  wave_count_kernel<<<nb, kWaveBlock, 0, st>>>(vis, n, w.block_counts);
  wave_scan_kernel<<<1, 1024, 0, st>>>(w.block_counts, (int64_t)nb, count, count_scaled, scale);
  DDF_CUDA_TRY(cudaGetLastError());
  return DDF_OK;
}
static int wave_scatter(const WaveWs& w, const float* o, const float* d, const float* dist, const float* vis,
                        int64_t n, const float light[3], float eps, float* o2, float* d2, float* tmax, int32_t* index,
                        cudaStream_t st) {
  const unsigned nb = (unsigned)((n + kWaveBlock - 1) / kWaveBlock);
  wave_scatter_kernel<<<nb, kWaveBlock, 0, st>>>(o, d, dist, vis, n, light[0], light[1], light[2], eps,
                                                w.block_counts, o2, d2, tmax, index);
  DDF_CUDA_TRY(cudaGetLastError());
  return DDF_OK;
}

}  // namespace ddf

using namespace ddf;

extern "C" int ddf_gen_shadow_from_hits(ddf_model* model, const float* o, const float* d, const float* dist,
                                        const float* vis, int64_t n, const float light[3], float eps,
                                        float* o2, float* d2, float* tmax, int32_t* index, int64_t* count,
                                        void* stream) {
  if (!model || !light || !count || n < 0 || n > 0x7fffffff) return DDF_E_INVALID_ARG;
  cudaStream_t st = (cudaStream_t)stream;
  if (n == 0) { DDF_CUDA_TRY(cudaMemsetAsync(count, 0, 8, st)); return DDF_OK; }
  if (!o || !d || !dist || !vis || !o2 || !d2 || !tmax || !index) return DDF_E_INVALID_ARG;
  Model* m = reinterpret_cast<Model*>(model);
  { const int rc_dev = check_device(m->device); if (rc_dev != DDF_OK) return rc_dev; }
  WaveWs w;
  int rc = wave_ws(m, n, false, &w);
  if (rc != DDF_OK) return rc;
  if ((rc = wave_count(w, vis, n, count, st)) != DDF_OK) return rc;
  rc = wave_scatter(w, o, d, dist, vis, n, light, eps, o2, d2, tmax, index, st);
  m->last_launches = 3;
  return rc;
}

// do_primary = false: out_dist / out_vis already hold the primary results (ddf_query_shaded)
static int shadowed_lights_impl(ddf_model* model, const float* o, const float* d, int64_t n,
                                const float* lights, int n_lights, float eps, float* out_dist,
                                float* out_vis, uint8_t* out_lit_mask, int64_t* out_count, void* stream, bool do_primary) {
  if (!model || !lights || n < 0 || n > 0x7fffffff || n_lights < 1 || n_lights > 8) return DDF_E_INVALID_ARG;
  Model* m = reinterpret_cast<Model*>(model);
  { const int rc_dev = check_device(m->device); if (rc_dev != DDF_OK) return rc_dev; }
  if (m->lay.input_kind != 0 || m->lay.n_out != 2) return DDF_E_INVALID_ARG;
  cudaStream_t st = (cudaStream_t)stream;
  if (n == 0) { if (out_count) DDF_CUDA_TRY(cudaMemsetAsync(out_count, 0, 8, st)); m->last_launches = 0; return DDF_OK; }
  if (!o || !d || !out_dist || !out_vis || !out_lit_mask) return DDF_E_INVALID_ARG;
  WaveWs w;
  int rc = wave_ws(m, n, true, &w);
  if (rc != DDF_OK) return rc;
  // 1. primary rays
  int launches = 0;
  if (do_primary) {
    if ((rc = ddf_query(model, o, d, n, out_dist, out_vis, stream)) != DDF_OK) return rc;
    launches = m->last_launches;
  }
  // 2. where the hits go in the compacted batch (the same for every light)
  if ((rc = wave_count(w, out_vis, n, w.count, st)) != DDF_OK) return rc;
  launches += 2;
  DDF_CUDA_TRY(cudaMemsetAsync(out_lit_mask, 0, (size_t)n, st));
  int64_t live = -1;
  for (int j = 0; j < n_lights; ++j) {
    // 3. shadow rays toward light j, 4. second query; the fused paths read the batch size on the device
    if ((rc = wave_scatter(w, o, d, out_dist, out_vis, n, lights + 3 * j, eps, w.o2, w.d2, w.tmax, w.index, st)) != DDF_OK) return rc;
    if (has_fused_path(m)) rc = fused_forward(m, w.o2, w.d2, n, w.count, 0, w.dist2, w.vis2, 0, 0.0f, st);
    else {
      if (live < 0) {                                      // the SIMT path sizes its grids on the host
        DDF_CUDA_TRY(cudaMemcpyAsync(&live, w.count, 8, cudaMemcpyDeviceToHost, st));
        DDF_CUDA_TRY(cudaStreamSynchronize(st));
      }
      rc = live > 0 ? simt_forward(m, w.o2, w.d2, live, 0, w.dist2, w.vis2, st) : DDF_OK;
      if (live == 0) m->last_launches = 0;
    }
    if (rc != DDF_OK) return rc;
    launches += 1 + m->last_launches;
    // 5. shadow decision for light j, scattered back to bit j of the primary rays
    wave_lit_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(w.vis2, w.dist2, w.tmax, w.index, w.count, out_lit_mask, j,
                                                                 j == n_lights - 1 ? out_count : nullptr, n_lights);
    DDF_CUDA_TRY(cudaGetLastError());
    launches += 1;
  }
  m->last_launches = launches;
  return DDF_OK;
}

extern "C" int ddf_query_shadowed_lights(ddf_model* model, const float* o, const float* d, int64_t n,
                                         const float* lights, int n_lights, float eps, float* out_dist,
                                         float* out_vis, uint8_t* out_lit_mask, int64_t* out_count, void* stream) {
  return shadowed_lights_impl(model, o, d, n, lights, n_lights, eps, out_dist, out_vis, out_lit_mask, out_count, stream, true);
}

extern "C" int ddf_query_shadowed(ddf_model* model, const float* o, const float* d, int64_t n,
                                  const float light[3], float eps, float* out_dist, float* out_vis,
                                  uint8_t* out_lit, int64_t* out_count, void* stream) {
  if (!light) return DDF_E_INVALID_ARG;
  return ddf_query_shadowed_lights(model, o, d, n, light, 1, eps, out_dist, out_vis, out_lit, out_count, stream);
}

// ---- ambient occlusion at the field's own hits ----------------------------------------------
namespace ddf {

struct WaveAoWs { int64_t *count, *count_rays; int32_t* block_counts; float *p_c, *n_c, *ao_c, *o2, *d2; int32_t* index; };

// workspace of ddf_query_ao_wavefront / ddf_gen_ao_from_hits (full = false: counts only)
static int wave_ao_ws(Model* m, int64_t n, int spp, bool full, WaveAoWs* w) {
  const size_t nb = (size_t)((n + kWaveBlock - 1) / kWaveBlock);
  const size_t a = (size_t)((n + 63) / 64 * 64);
  size_t need = ((nb * 4 + 255) / 256) * 256 + 256;
  if (full) need += a * (12 + 12 + 4 + 4) + a * (size_t)spp * 24;
  { int rc = wave_reserve_bytes(m, need); if (rc != DDF_OK) return rc; }
  uint8_t* b = (uint8_t*)m->wave_ws;
  w->count = (int64_t*)b; w->count_rays = (int64_t*)(b + 8);  b += 256;
  w->block_counts = (int32_t*)b;                              b += ((nb * 4 + 255) / 256) * 256;
  if (full) {
    w->p_c = (float*)b;     b += a * 12;
    w->n_c = (float*)b;     b += a * 12;
    w->ao_c = (float*)b;    b += a * 4;
    w->index = (int32_t*)b; b += a * 4;
    w->o2 = (float*)b;      b += a * (size_t)spp * 12;
    w->d2 = (float*)b;
  }
  return DDF_OK;
}

// count + scan + (hit point, normal, index) scatter + AO rays about the normals; 4 launches (3 without rays)
static int wave_ao_rays(Model* m, const WaveAoWs& w, const float* o, const float* d, const float* dist, const float* vis,
                        int width, int height, int spp, uint64_t seed, uint64_t rng_stream, float eps, float* p_c,
                        float* n_c, int32_t* index, float* nrm_img, float* o2, float* d2, int64_t* count,
                        int64_t* count_rays, cudaStream_t st) {
  const int64_t n = (int64_t)width * height;
  const unsigned nb = (unsigned)((n + kWaveBlock - 1) / kWaveBlock);
  WaveWs cw; cw.block_counts = w.block_counts;
  int rc = wave_count(cw, vis, n, count, st, count_rays, spp);
  if (rc != DDF_OK) return rc;
  wave_normals_scatter_kernel<<<nb, kWaveBlock, 0, st>>>(o, d, dist, vis, width, height, w.block_counts, p_c, n_c, index, nrm_img);
  DDF_CUDA_TRY(cudaGetLastError());
  m->last_launches = 3;
  if (o2) {
    if ((rc = gen_ao_launch(p_c, n_c, n, count, spp, seed, rng_stream, eps, o2, d2, st)) != DDF_OK) return rc;
    m->last_launches = 4;
  }
  return DDF_OK;
}

}  // namespace ddf

extern "C" int ddf_gen_ao_from_hits(ddf_model* model, const float* o, const float* d, const float* dist,
                                    const float* vis, int width, int height, int spp, uint64_t seed,
                                    uint64_t rng_stream, float eps, float* p_c, float* nrm_c, int32_t* index,
                                    float* o2, float* d2, int64_t* count, void* stream) {
  if (!model || !count || width < 0 || height < 0 || spp <= 0 || (int64_t)width * height * spp > 0x7fffffff) return DDF_E_INVALID_ARG;
  if ((o2 == nullptr) != (d2 == nullptr)) return DDF_E_INVALID_ARG;
  cudaStream_t st = (cudaStream_t)stream;
  Model* m = reinterpret_cast<Model*>(model);
  { const int rc_dev = check_device(m->device); if (rc_dev != DDF_OK) return rc_dev; }
  const int64_t n = (int64_t)width * height;
  if (n == 0) { DDF_CUDA_TRY(cudaMemsetAsync(count, 0, 8, st)); m->last_launches = 0; return DDF_OK; }
  if (!o || !d || !dist || !vis || !p_c || !nrm_c || !index) return DDF_E_INVALID_ARG;
  WaveAoWs w;
  int rc = wave_ao_ws(m, n, spp, false, &w);
  if (rc != DDF_OK) return rc;
  return wave_ao_rays(m, w, o, d, dist, vis, width, height, spp, seed, rng_stream, eps, p_c, nrm_c, index, nullptr,
                      o2, d2, count, nullptr, st);
}

static int ao_wavefront_impl(ddf_model* model, const float* o, const float* d, int width, int height,
                             int spp, uint64_t seed, uint64_t rng_stream, float eps, float ao_radius,
                             float* out_dist, float* out_vis, float* out_nrm, float* out_ao,
                             int64_t* out_count, void* stream, bool do_primary) {
  if (!model || width < 0 || height < 0 || spp <= 0 || (int64_t)width * height * spp > 0x7fffffff) return DDF_E_INVALID_ARG;
  Model* m = reinterpret_cast<Model*>(model);
  { const int rc_dev = check_device(m->device); if (rc_dev != DDF_OK) return rc_dev; }
  if (m->lay.input_kind != 0 || m->lay.n_out != 2) return DDF_E_INVALID_ARG;
  cudaStream_t st = (cudaStream_t)stream;
  const int64_t n = (int64_t)width * height;
  if (n == 0) { if (out_count) DDF_CUDA_TRY(cudaMemsetAsync(out_count, 0, 8, st)); m->last_launches = 0; return DDF_OK; }
  if (!o || !d || !out_dist || !out_vis || !out_ao) return DDF_E_INVALID_ARG;
  // a hash-grid field generates the AO rays inside its query kernel (ddf_query_ao_points): no ray buffer, no generator launch
  const bool rays_in_kernel = m->hg && spp <= 32 && 32 % spp == 0;
  WaveAoWs w;
  int rc = wave_ao_ws(m, n, rays_in_kernel ? 0 : spp, true, &w);
  if (rc != DDF_OK) return rc;
  // 1. primary rays
  int launches = 0;
  if (do_primary) {
    if ((rc = ddf_query(model, o, d, n, out_dist, out_vis, stream)) != DDF_OK) return rc;
    launches = m->last_launches;
  }
  // 2. hit points, normals from the hit-point image, spp rays about each normal (compacted, size on the device)
  if ((rc = wave_ao_rays(m, w, o, d, out_dist, out_vis, width, height, spp, seed, rng_stream, eps, w.p_c, w.n_c, w.index,
                         out_nrm, rays_in_kernel ? nullptr : w.o2, rays_in_kernel ? nullptr : w.d2, w.count, w.count_rays,
                         st)) != DDF_OK) return rc;
  launches += m->last_launches;
  // 3. second query with the AO reduce fused when a pixel's rays sit in one warp; else through ddf_query_ao
  if (rays_in_kernel) {
    rc = hash_forward_ao_points(m, w.p_c, w.n_c, n, w.count_rays, spp, gen_key(seed, rng_stream), eps, ao_radius, w.ao_c, st);
  } else if (has_fused_path(m) && spp <= 32 && 32 % spp == 0) {
    rc = fused_forward(m, w.o2, w.d2, n * spp, w.count_rays, 2, w.ao_c, nullptr, spp, ao_radius, st);
  } else {
    int64_t live = 0;
    DDF_CUDA_TRY(cudaMemcpyAsync(&live, w.count, 8, cudaMemcpyDeviceToHost, st));
    DDF_CUDA_TRY(cudaStreamSynchronize(st));
    rc = ddf_query_ao(model, w.o2, w.d2, live, spp, ao_radius, w.ao_c, stream);
    if (live == 0) m->last_launches = 0;
  }
  if (rc != DDF_OK) return rc;
  launches += m->last_launches;
  // 4. back to the pixels
  wave_ao_scatter_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(out_vis, n, w.ao_c, w.index, w.count, out_ao, out_count, spp);
  DDF_CUDA_TRY(cudaGetLastError());
  m->last_launches = launches + 1;
  return DDF_OK;
}

extern "C" int ddf_query_ao_wavefront(ddf_model* model, const float* o, const float* d, int width, int height,
                                      int spp, uint64_t seed, uint64_t rng_stream, float eps, float ao_radius,
                                      float* out_dist, float* out_vis, float* out_nrm, float* out_ao,
                                      int64_t* out_count, void* stream) {
  return ao_wavefront_impl(model, o, d, width, height, spp, seed, rng_stream, eps, ao_radius, out_dist, out_vis, out_nrm,
                           out_ao, out_count, stream, true);
}

// shadows and ambient occlusion of one frame from ONE primary query (the field as the renderer's
// secondary-ray oracle; its Table VI reports exactly these two effects)
extern "C" int ddf_query_shaded(ddf_model* model, const float* o, const float* d, int width, int height,
                                const float* lights, int n_lights, int spp, uint64_t seed, uint64_t rng_stream,
                                float eps, float ao_radius, float* out_dist, float* out_vis, uint8_t* out_lit_mask,
                                float* out_nrm, float* out_ao, int64_t* out_counts, void* stream) {
  if (!model || width < 0 || height < 0 || (int64_t)width * height > 0x7fffffff || n_lights < 0 || n_lights > 8 || spp < 0)
    return DDF_E_INVALID_ARG;
  if ((n_lights > 0 && (!lights || !out_lit_mask)) || (spp > 0 && !out_ao)) return DDF_E_INVALID_ARG;
  Model* m = reinterpret_cast<Model*>(model);
  { const int rc_dev = check_device(m->device); if (rc_dev != DDF_OK) return rc_dev; }
  if (m->lay.input_kind != 0 || m->lay.n_out != 2) return DDF_E_INVALID_ARG;
  cudaStream_t st = (cudaStream_t)stream;
  const int64_t n = (int64_t)width * height;
  if (out_counts) DDF_CUDA_TRY(cudaMemsetAsync(out_counts, 0, 16, st));
  if (n == 0) { m->last_launches = 0; return DDF_OK; }
  if (!o || !d || !out_dist || !out_vis) return DDF_E_INVALID_ARG;
  int rc = ddf_query(model, o, d, n, out_dist, out_vis, stream);
  if (rc != DDF_OK) return rc;
  int launches = m->last_launches;
  if (n_lights > 0) {
    if ((rc = shadowed_lights_impl(model, o, d, n, lights, n_lights, eps, out_dist, out_vis, out_lit_mask, out_counts, stream, false)) != DDF_OK) return rc;
    launches += m->last_launches;
  }
  if (spp > 0) {
    if ((rc = ao_wavefront_impl(model, o, d, width, height, spp, seed, rng_stream, eps, ao_radius, out_dist, out_vis, out_nrm,
                                out_ao, out_counts ? out_counts + 1 : nullptr, stream, false)) != DDF_OK) return rc;
    launches += m->last_launches;
  }
  m->last_launches = launches;
  return DDF_OK;
}

// ---- ddf_gen_shadow_from_hits for hosts that cannot allocate device memory ---------------------
// The compaction above needs one int32 per 256 primary rays between its three launches (how many hits each block
// saw, then where each block's hits start).  Every other entry point keeps those numbers in a workspace that belongs
// to a model and is obtained with cudaMalloc.  Some hosts cannot do that: a renderer or a training framework that
// took the whole device for its own pool at start-up and has nothing left for the driver to hand out, or a frame
// loop that cannot accept the device-wide stall a cudaMalloc / cudaFree brings.  For them the numbers live in the
// array below, which is part of the library image: every GPU that loads libddf.so carries its 256 KB until the
// process ends, whether or not this entry point is ever called.  65,536 entries cover DDF_STATIC_MAX_RAYS = 2^24
// primary rays (configs[3]'s 1024 x 1024 x 16 batch).
namespace ddf {

constexpr int64_t kStaticMaxRays = DDF_STATIC_MAX_RAYS;
constexpr int64_t kStaticBlocks = kStaticMaxRays / kWaveBlock;
static_assert(kStaticBlocks * kWaveBlock == kStaticMaxRays, "the ray limit is a whole number of count blocks");

static __device__ __align__(256) int32_t g_static_block_counts[kStaticBlocks];

// In host code `g_static_block_counts` is only a handle the runtime knows the array by - handing it to a kernel as a
// pointer would make the kernel read host memory or fault.  The address the kernels need is asked from the runtime,
// once per device and with that device current, and remembered here.
constexpr int kStaticMaxDevices = 64;
static std::mutex g_static_mu;
static int32_t* g_static_dev_ptr[kStaticMaxDevices];

static int static_block_counts(int32_t** out) {
  int dev = -1;
  DDF_CUDA_TRY(cudaGetDevice(&dev));
  if (dev < 0 || dev >= kStaticMaxDevices) return DDF_E_UNSUPPORTED;
  std::lock_guard<std::mutex> lock(g_static_mu);
  if (!g_static_dev_ptr[dev]) {
    void* p = nullptr;
    DDF_CUDA_TRY(cudaGetSymbolAddress(&p, g_static_block_counts));
    if (!p) return DDF_E_CUDA;
    g_static_dev_ptr[dev] = static_cast<int32_t*>(p);
  }
  *out = g_static_dev_ptr[dev];
  return DDF_OK;
}

}  // namespace ddf

extern "C" int ddf_gen_shadow_from_hits_static(const float* o, const float* d, const float* dist, const float* vis,
                                               int64_t n, const float light[3], float eps, float* o2, float* d2,
                                               float* tmax, int32_t* index, int64_t* count, void* stream) {
  if (!light || !count || n < 0) return DDF_E_INVALID_ARG;
  if (n > kStaticMaxRays) return DDF_E_TOO_LARGE;
  cudaStream_t st = (cudaStream_t)stream;
  if (n == 0) { DDF_CUDA_TRY(cudaMemsetAsync(count, 0, 8, st)); return DDF_OK; }
  if (!o || !d || !dist || !vis || !o2 || !d2 || !tmax || !index) return DDF_E_INVALID_ARG;
  WaveWs w = {};
  int rc = static_block_counts(&w.block_counts);
  if (rc != DDF_OK) return rc;
  // Nothing in the array has to be cleared between calls: the count launch writes every one of the ceil(n / 256)
  // entries the scan and the scatter go on to read, and no launch reads past them, so whatever an earlier
  // (possibly larger) batch left behind is never seen.
  if ((rc = wave_count(w, vis, n, count, st)) != DDF_OK) return rc;
  return wave_scatter(w, o, d, dist, vis, n, light, eps, o2, d2, tmax, index, st);
}
