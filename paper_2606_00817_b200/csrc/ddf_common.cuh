// ddf_common.cuh - shared declarations of libddf (model object, error plumbing, device helpers).
// Product code: shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <cuda_bf16.h>
#include <stdint.h>
#include "../../include/ddf.h"

namespace ddf {

extern thread_local int g_last_cuda_error;

#define DDF_CUDA_TRY(expr)                                   \
  do {                                                       \
    cudaError_t _e = (expr);                                 \
    if (_e != cudaSuccess) {                                 \
      ddf::g_last_cuda_error = (int)_e;                      \
      (void)cudaGetLastError();                              \
      return DDF_E_CUDA;                                     \
    }                                                        \
  } while (0)

constexpr int kMaxLayers = 32;
constexpr int kKBlock = 64;          // K granularity of the tiled weight copy (bf16 elements)

inline int round_up(int x, int m) { return (x + m - 1) / m * m; }

// One Linear layer of the device weight copy.  W is bf16 [n_out_pad][k_pad] row-major with
// k_pad = k0_pad + k1_pad: segment 0 multiplies h (or gamma for layer 0), segment 1 multiplies
// gamma at the skip layer.  Pad rows / columns are zero.
struct LayerDesc {
  int n_out;            // true output count
  int k0, k0_pad;       // first input segment (true, padded to kKBlock)
  int k1, k1_pad;       // second input segment (skip: gamma), 0 if none
  int k_pad;            // row stride of W in elements
  size_t w_off;         // element offset of W in the bf16 weight arena
  size_t b_off;         // element offset of the bias in the fp32 bias arena
};

struct TcPlan;          // tcgen05 path state (ddf_tc.cu)
struct HashPlan;        // hash-grid field state (ddf_hash.cu)
struct NarrowPlan;      // tcgen05 path for narrow networks (ddf_narrow.cu)

struct Model {
  ddf_layout lay;
  int E, E_pad;                    // encoded width, padded to kKBlock
  int width_pad;                   // width padded to kKBlock
  int n_layers;                    // n_hidden + 1 (head last)
  LayerDesc layers[kMaxLayers];
  __nv_bfloat16* d_w;              // weight arena (hidden layers, padded; head stored too)
  float* d_b;                      // bias arena (fp32)
  float* d_head_w;                 // head weights as fp32 [n_out][width] (bf16-rounded values)
  size_t w_elems, b_elems;
  // workspace for the SIMT path and the sphere tracer (grown on demand, never in the hot loop
  // once sized): two bf16 activation buffers + one fp32 buffer for the last hidden layer
  int64_t ws_rows;
  __nv_bfloat16 *ws_gamma, *ws_act0, *ws_act1;
  float* ws_last;
  float *ws_dist, *ws_vis;         // ddf_query_ao fallback
  int64_t ws_out_rows;
  // staging for ddf_query_host
  float *h2d_o, *h2d_d, *d2h_dist, *d2h_vis;
  int64_t host_rows;
  float *cam_o, *cam_d; int64_t cam_rows;  // ddf_query_camera workspace for the kernels that read rays from memory
  cudaStream_t host_s_in, host_s_out;      // ddf_query_host: copy streams (created on first use)
  cudaEvent_t host_ev[16];                 // [0..7] chunk uploaded, [8..15] chunk computed
  // sphere tracer state
  void* trace_ws; size_t trace_ws_bytes;
  // wavefront secondary rays (ddf_wave.cu)
  void* wave_ws; size_t wave_ws_bytes;
  int path;                        // 0 auto, 1 SIMT, 2 tcgen05
  TcPlan* tc;                      // non-null when the tcgen05 path can serve the layout
  NarrowPlan* nw;                  // non-null when the narrow tcgen05 path (width 64 / 128, weights in smem) serves it
  HashPlan* hg;                    // non-null: this model is a hash-grid field (ddf_create_hashgrid)
  int sm_count;
  int last_launches;
  int device;                      // CUDA device ordinal the model was created on: every call must find it current
};

// A model's (and a trainer's) pointers, tensor maps and per-context function attributes belong to the device it was
// created on; a call made with another device current would launch there on foreign addresses.  Refuse it instead.
inline int check_device(int owner) {
  int cur = -1;
  if (cudaGetDevice(&cur) != cudaSuccess) { (void)cudaGetLastError(); return DDF_E_CUDA; }
  return cur == owner ? DDF_OK : DDF_E_INVALID_ARG;
}

// ---- SIMT path (ddf_simt.cu)
constexpr int64_t kSimtChunkRows = 16384;   // rays per pass of simt_forward: the most rows its activation workspace ever holds
int simt_forward(Model* m, const float* o, const float* d, int64_t n, int mode_out,
                 float* out0, float* out1, cudaStream_t st);
int ensure_workspace(Model* m, int64_t rows);

// ---- tcgen05 path (ddf_tc.cu)
int tc_plan_create(Model* m);                 // sets m->tc or leaves it null (unsupported shape)
void tc_plan_destroy(Model* m);
// mode_out: 0 = heads (dist, vis), 1 = raw logits into out0 [n][n_out], 2 = AO reduce into out0
int tc_forward(Model* m, const float* o, const float* d, int64_t n, const int64_t* n_dev,
               int mode_out, float* out0, float* out1, int spp, float ao_radius, cudaStream_t st);

// ---- workspaces sized ahead of time (ddf_reserve) or on first use
int trace_reserve(Model* m, int64_t n, int max_steps);          // ddf_trace.cu
int wave_reserve_bytes(Model* m, size_t need);                  // ddf_wave.cu
int wave_reserve(Model* m, int64_t n, int spp);
// exclusive scan of n_blocks int32 block counts in place (one block), the total to *count (device): the middle step of
// every stable compaction in the library
int scan_block_counts(int32_t* block_counts, int64_t n_blocks, int64_t* count, cudaStream_t st);

// ---- hash-grid field (ddf_hash.cu)
void hash_plan_destroy(Model* m);
int hash_forward(Model* m, const float* o, const float* d, int64_t n, const int64_t* n_dev, int mode_out,
                 float* out0, float* out1, int spp, float ao_radius, cudaStream_t st);

int hash_forward_camera(Model* m, const ddf_camera* cam, int width, int height, float* out0, float* out1, cudaStream_t st);
// AO of n_pts points (n_pts_dev: device-side count or null), the spp rays of a point generated in the kernel
int hash_forward_ao_points(Model* m, const float* pts, const float* nrm, int64_t n_pts, const int64_t* n_rays_dev, int spp,
                           uint64_t key, float eps, float ao_radius, float* ao, cudaStream_t st);
uint64_t gen_key(uint64_t seed, uint64_t rng_stream);   // ddf_gen.cu: the generators' counter key

// ---- narrow-network tcgen05 path (ddf_narrow.cu)
int narrow_plan_create(Model* m, const uint16_t* hw_host, const float* hb_host);   // sets m->nw or leaves it null
void narrow_plan_destroy(Model* m);
int narrow_forward(Model* m, const float* o, const float* d, int64_t n, const int64_t* n_dev, int mode_out,
                   float* out0, float* out1, int spp, float ao_radius, cudaStream_t st);

// ---- generators (ddf_gen.cu): AO rays about (p, nrm); n_pts_dev (device) overrides n_pts when non-null
int gen_ao_launch(const float* p, const float* nrm, int64_t n_pts, const int64_t* n_pts_dev, int spp, uint64_t seed,
                  uint64_t rng_stream, float eps, float* o, float* d, cudaStream_t st);

// one dispatch for every fused path: tcgen05 wide, tcgen05 narrow, hash grid (n_dev: device-side count or null)
inline bool has_fused_path(const Model* m) { return m->hg || ((m->tc || m->nw) && m->path != 1); }
inline int fused_forward(Model* m, const float* o, const float* d, int64_t n, const int64_t* n_dev, int mode_out,
                         float* out0, float* out1, int spp, float ao_radius, cudaStream_t st) {
  if (m->hg) return hash_forward(m, o, d, n, n_dev, mode_out, out0, out1, spp, ao_radius, st);
  if (m->tc) return tc_forward(m, o, d, n, n_dev, mode_out, out0, out1, spp, ao_radius, st);
  return narrow_forward(m, o, d, n, n_dev, mode_out, out0, out1, spp, ao_radius, st);
}

// ---- device helpers -------------------------------------------------------------------------
#ifdef __CUDACC__
__device__ __forceinline__ uint64_t dev_mix64(uint64_t z) {
  z += 0x9E3779B97F4A7C15ull;
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
  return z ^ (z >> 31);
}
// key = mix64(mix64(seed) ^ stream) is computed once on the host
__device__ __forceinline__ float dev_uniform01(uint64_t key, uint64_t idx) {
  return (float)(uint32_t)(dev_mix64(key ^ idx) >> 40) * (1.0f / 16777216.0f);
}

__device__ __forceinline__ float softplus_f(float z) {
  return fmaxf(z, 0.0f) + log1pf(expf(-fabsf(z)));
}
__device__ __forceinline__ float sigmoid_f(float z) { return 1.0f / (1.0f + expf(-z)); }

// AO ray k (= point k / spp, sample k % spp) about the unit normal n at p: origin p + eps n, cosine-weighted
// direction in the frame (t1, t2, n) (reading A9 / row a11).  Shared by the generator kernel and by the
// kernels that generate the rays themselves, so both produce the same bits.
__device__ __forceinline__ void ao_ray_from_point(const float p[3], const float n[3], uint64_t key, int64_t k, float eps,
                                                  float o[3], float d[3]) {
  int ax = 0;
  if (fabsf(n[1]) < fabsf(n[ax])) ax = 1;
  if (fabsf(n[2]) < fabsf(n[ax])) ax = 2;
  float e[3] = { ax == 0 ? 1.0f : 0.0f, ax == 1 ? 1.0f : 0.0f, ax == 2 ? 1.0f : 0.0f };
  // every product and sum below is an explicit round-to-nearest operation: the kernels that inline this helper must
  // produce the same bits whatever FMA contraction the optimiser would choose in each of them
  #define DDF_CROSS(a, b, c, d) __fsub_rn(__fmul_rn(a, b), __fmul_rn(c, d))
  #define DDF_SUMSQ(v) __fadd_rn(__fadd_rn(__fmul_rn(v[0], v[0]), __fmul_rn(v[1], v[1])), __fmul_rn(v[2], v[2]))
  float t1[3] = { DDF_CROSS(e[1], n[2], e[2], n[1]), DDF_CROSS(e[2], n[0], e[0], n[2]), DDF_CROSS(e[0], n[1], e[1], n[0]) };
  float inv = __frcp_rn(__fsqrt_rn(DDF_SUMSQ(t1)));
  t1[0] = __fmul_rn(t1[0], inv); t1[1] = __fmul_rn(t1[1], inv); t1[2] = __fmul_rn(t1[2], inv);
  float t2[3] = { DDF_CROSS(n[1], t1[2], n[2], t1[1]), DDF_CROSS(n[2], t1[0], n[0], t1[2]), DDF_CROSS(n[0], t1[1], n[1], t1[0]) };
  float u1 = dev_uniform01(key, 2 * (uint64_t)k), u2 = dev_uniform01(key, 2 * (uint64_t)k + 1);
  float r = __fsqrt_rn(u1), s, c;
  sincospif(__fmul_rn(2.0f, u2), &s, &c);
  float lx = __fmul_rn(r, c), ly = __fmul_rn(r, s), lz = __fsqrt_rn(__fsub_rn(1.0f, u1));
  float dd[3];
  #pragma unroll
  for (int a = 0; a < 3; ++a) dd[a] = __fmaf_rn(lz, n[a], __fmaf_rn(ly, t2[a], __fmul_rn(lx, t1[a])));
  inv = __frcp_rn(__fsqrt_rn(DDF_SUMSQ(dd)));
  #pragma unroll
  for (int a = 0; a < 3; ++a) { o[a] = __fmaf_rn(eps, n[a], p[a]); d[a] = __fmul_rn(dd[a], inv); }
  #undef DDF_CROSS
  #undef DDF_SUMSQ
}

// The 3-vectors of 32 consecutive rays (first ray `first`, AoS float[n][3]) into registers, lane j <- ray first + j:
// the warp reads its 384 contiguous bytes as 24 coalesced 16-byte loads and regroups them by shuffles (SURVEY.md row a1
// "flat float4 over the n*3 array, regroup in shuffles").  Falls back to per-ray scalar loads for a 4-byte-aligned
// buffer or a ragged last warp.  All 32 lanes must call it; lanes whose ray is >= n get zeros.
__device__ __forceinline__ void load_ray_vec3(const float* __restrict__ base, int64_t first, int64_t n, int lane, float v[3]) {
  const float* w = base + 3 * first;
  const bool fast = first + 32 <= n && (reinterpret_cast<uintptr_t>(w) & 15) == 0;       // warp-uniform
  if (fast) {
    float4 q = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
    if (lane < 24) q = __ldg(reinterpret_cast<const float4*>(w) + lane);
    #pragma unroll
    for (int i = 0; i < 3; ++i) {
      const int f = 3 * lane + i, src = f >> 2, comp = f & 3;
      const float s0 = __shfl_sync(0xffffffffu, q.x, src), s1 = __shfl_sync(0xffffffffu, q.y, src);
      const float s2 = __shfl_sync(0xffffffffu, q.z, src), s3 = __shfl_sync(0xffffffffu, q.w, src);
      v[i] = comp == 0 ? s0 : (comp == 1 ? s1 : (comp == 2 ? s2 : s3));
    }
  } else {
    const int64_t g = first + lane;
    const bool ok = g < n;
    v[0] = ok ? base[3 * g] : 0.0f; v[1] = ok ? base[3 * g + 1] : 0.0f; v[2] = ok ? base[3 * g + 2] : 0.0f;
  }
}

// gamma of one ray into a bf16 row (E_pad entries, pad = 0).  sin/cos(2^k pi x) via sincospif
// of the exactly scaled argument (ldexp), so high bands keep full fp32 accuracy.
__device__ __forceinline__ void encode_vec_bf16(const float v[3], int nfreq, __nv_bfloat16* row) {
  row[0] = __float2bfloat16_rn(v[0]); row[1] = __float2bfloat16_rn(v[1]); row[2] = __float2bfloat16_rn(v[2]);
  for (int k = 0; k < nfreq; ++k) {
    #pragma unroll
    for (int c = 0; c < 3; ++c) {
      float s, co;
      sincospif(ldexpf(v[c], k), &s, &co);
      row[3 + 6 * k + c] = __float2bfloat16_rn(s);
      row[6 + 6 * k + c] = __float2bfloat16_rn(co);
    }
  }
}
#endif

}  // namespace ddf
