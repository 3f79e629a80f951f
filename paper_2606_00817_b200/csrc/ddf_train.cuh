// ddf_train.cuh - what the two training kernels share (ddf_train.cu: fp32 CUDA cores,
// ddf_train_tc.cu: split-bf16 tensor cores): the parameter block, the trainer object, the corner rule.
#pragma once
#include "ddf_common.cuh"
#include <utility>

namespace ddf {

constexpr int kTrRays = 128;            // rays per CTA
constexpr int kTrThreads = 256;         // two threads per ray
constexpr int kTrPitch = 129;
constexpr int kTrW = 64;
constexpr int kTrMaxLevels = 16;
constexpr int kTrRep = 8;               // copies of the coarse levels' gradient accumulator (tensor-core path)
constexpr int64_t kTrRepLevelMax = 32768;   // levels with at most this many entries are replicated

struct TrLevel { float scale; uint32_t verts; uint32_t offset; uint32_t hashed; };

struct TrParams {
  TrLevel lv[kTrMaxLevels];
  const float* table; const float* mlp;          // fp32 master copies
  float* g_table; float* g_mlp; float* loss;
  const float* o; const float* d; const float* t; const uint8_t* hit;
  int64_t n;
  float bmin[3], den[3];
  float dist_clamp, ce_weight;
  uint32_t tmask;
  int n_levels, Ld, n_hidden, E, NF;
  int w_off[3], b_off[3];                        // blob offsets of layer l (l = n_hidden: head)
  float* feat; float* dfeat; float* slab;        // tensor-core path: level features / their gradients [n][32], per-CTA dW
  float* rep; uint32_t rep_entries; int rep_levels;   // kTrRep private copies of the gradient of the first rep_levels levels (rep_entries entries)
};

struct Trainer {
  ddf_hashgrid_layout lay;
  ddf_train_params prm;
  int64_t entries, n_table, n_mlp, step;
  float *p_table, *p_mlp, *m, *v, *g;            // m, v, g hold table values first, then the MLP
  float* loss_dev;
  TrParams base;
  size_t smem_bytes;
  float *ws_feat, *ws_dfeat, *ws_slab, *ws_rep;  // tensor-core path workspace; ws_feat / ws_dfeat hold ws_rays rays
  int64_t ws_rays;
  int sms;
  int device;                                    // CUDA device ordinal of every pointer below (check_device)
};

// corner indices (into the table, in float2 units) and weights of one level
__device__ __forceinline__ void tr_corners(const TrLevel& lv, uint32_t tmask, const float x01[3], uint32_t idx[8], float wt[8]) {
  uint32_t c0[3]; float w1[3];
  #pragma unroll
  for (int a = 0; a < 3; ++a) {
    const float pos = __fmul_rn(x01[a], lv.scale);
    const float fl = fminf(floorf(pos), lv.scale - 1.0f);
    c0[a] = (uint32_t)fl; w1[a] = pos - fl;
  }
  uint32_t kx[2], ky[2], kz[2];
  if (lv.hashed) {
    kx[0] = c0[0]; kx[1] = c0[0] + 1u;
    ky[0] = c0[1] * 2654435761u; ky[1] = (c0[1] + 1u) * 2654435761u;
    kz[0] = c0[2] * 805459861u;  kz[1] = (c0[2] + 1u) * 805459861u;
  } else {
    kx[0] = c0[0]; kx[1] = c0[0] + 1u;
    ky[0] = c0[1] * lv.verts; ky[1] = ky[0] + lv.verts;
    kz[0] = c0[2] * lv.verts * lv.verts; kz[1] = kz[0] + lv.verts * lv.verts;
  }
  #pragma unroll
  for (int c = 0; c < 8; ++c) {
    const uint32_t a = kx[c & 1], b = ky[(c >> 1) & 1], e = kz[c >> 2];
    idx[c] = lv.offset + (lv.hashed ? ((a ^ b ^ e) & tmask) : (a + b + e));
    wt[c] = ((c & 1) ? w1[0] : 1.0f - w1[0]) * (((c >> 1) & 1) ? w1[1] : 1.0f - w1[1]) * ((c >> 2) ? w1[2] : 1.0f - w1[2]);
  }
}

// Programmatic dependent launch: a kernel launched with launch_pdl may be scheduled while its predecessor in
// the stream is still running (as soon as every CTA of the predecessor has executed pdl_launch_dependents or
// exited); it must execute pdl_wait before it touches anything the predecessor writes.  pdl_wait returns when
// the predecessor grid has completed and its writes are visible.  Used along the chain gather -> MLP ->
// scatter -> Adam, so that launch latencies and the MLP kernel's prologue overlap the kernel before.
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
template <typename... KArgs, typename... Args>
inline cudaError_t launch_pdl(void (*kernel)(KArgs...), unsigned grid, unsigned block, size_t smem, cudaStream_t st, Args&&... args) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(grid); cfg.blockDim = dim3(block); cfg.dynamicSmemBytes = smem; cfg.stream = st;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = at; cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, kernel, std::forward<Args>(args)...);
}
// the same kernel (it may still execute pdl_wait: a no-op then) launched the ordinary way, after its predecessor
template <typename... KArgs, typename... Args>
inline cudaError_t launch_plain(void (*kernel)(KArgs...), unsigned grid, unsigned block, size_t smem, cudaStream_t st, Args&&... args) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(grid); cfg.blockDim = dim3(block); cfg.dynamicSmemBytes = smem; cfg.stream = st;
  return cudaLaunchKernelEx(&cfg, kernel, std::forward<Args>(args)...);
}

// ddf_train_tc.cu
size_t train_tc_slab_floats();
size_t train_tc_feat_pitch();
cudaError_t train_tc_prepare();
cudaError_t train_tc_launch(const TrParams& p, unsigned grid, cudaStream_t st);

}  // namespace ddf
