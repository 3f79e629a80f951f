// ddf_narrow.cu - the tcgen05 path for NARROW frequency-encoded networks (width 64 or 128, e.g.
// BASELINE.json configs[0] (3 x 64) and the paper's "sinusoidal MLP 128 x 4"): the
// whole weight set fits in shared memory, so one CTA = 128 rays runs encode -> layers -> heads
// without touching global memory in between.
//
//   thread t = ray t of the tile = row t of the operand tiles = TMEM lane t
//   G tile : gamma(o, d) as bf16, 128 rows x E_pad (64-column blocks of 16 KB, 128-byte swizzle);
//            kept for the skip layer
//   H tile : the hidden activation, 128 rows x width, overwritten in place once the MMAs that
//            read it have completed
//   layer  : D[128 x width] = sum over 64-column blocks of  A_block[128 x 64] W_block[width x 64]^T,
//            tcgen05.mma M128 N{64,128} K16, fp32 accumulator in TMEM; the skip layer just adds the
//            G blocks to the same accumulator
//   epilogue: tcgen05.ld 64 columns at a time -> +bias, ReLU -> bf16 row into the H tile; the
//            last layer feeds the fused heads from fp32 (same heads / AO reduce as ddf_tc.cu)
// Several CTAs per SM when the weights are small (configs[0]: 56 KB), so one tile's encoding
// overlaps another's MMAs.  Numerics and rounding points as in ddf_tc.cu (reading A11).
#include "ddf_common.cuh"
#include "ddf_tc_ptx.cuh"
#include <stdlib.h>
#include <string.h>
#include <new>
#include <vector>

namespace ddf {

constexpr int kNwThreads = 128;
constexpr int kNwMaxLayers = 16;

struct NwParams {
  const __nv_bfloat16* w;        // per layer, per 64-column K block: [width rows][64] bf16
  const float* bias;             // [n_hidden][width]
  const float* head_w;           // [n_out][width]
  const float* o; const float* d;
  float* out0; float* out1;
  int64_t n; const int64_t* n_dev;
  float head_b[2];
  float ao_radius;
  int n_hidden, width, skip_layer, n_out, input_kind, Lo, Ld, E, gblocks, hblocks;
  int mode_out, spp;
  int w_blk_off[kNwMaxLayers];   // first weight block of layer l (in blocks of width x 64)
  int total_blocks;
};

struct NarrowPlan {
  __nv_bfloat16* d_w; float* d_bias;
  NwParams base;
  size_t smem_bytes;
  int ctas_per_sm;
};

__device__ __forceinline__ uint32_t nw_pack(float a, float b) {
  __nv_bfloat162 t = __floats2bfloat162_rn(a, b);
  return *reinterpret_cast<uint32_t*>(&t);
}

__global__ void __launch_bounds__(kNwThreads) ddf_narrow_kernel(const __grid_constant__ NwParams p) {
  extern __shared__ uint8_t smem_raw[];
  const uint32_t smem_base = (ptx::smem_u32(smem_raw) + 1023u) & ~1023u;
  const int W = p.width;
  const uint32_t wblk_bytes = (uint32_t)W * 128u;
  const uint32_t g_smem = smem_base;                                   // gblocks x 16 KB
  const uint32_t h_smem = g_smem + (uint32_t)p.gblocks * 16384u;       // hblocks x 16 KB
  const uint32_t w_smem = h_smem + (uint32_t)p.hblocks * 16384u;       // total_blocks x (W x 128 B)
  const uint32_t f_smem = w_smem + (uint32_t)p.total_blocks * wblk_bytes;
  const uint32_t bar = f_smem + (uint32_t)((p.n_hidden + 2) * W) * 4u;
  const uint32_t tmem_slot = bar + 8u;
  uint8_t* gen = smem_raw + (smem_base - ptx::smem_u32(smem_raw));
  float* fsm = reinterpret_cast<float*>(gen + (f_smem - smem_base));   // bias [n_hidden][W], head [2][W]

  const int t = threadIdx.x, warp = t >> 5, lane = t & 31;

  // ---- one-time: weights (already in block order) into swizzled shared memory
  {
    const int chunks = p.total_blocks * W * 8;                          // 16-byte chunks
    for (int e = t; e < chunks; e += kNwThreads) {
      const int blk = e / (W * 8), r = (e >> 3) % W, j = e & 7;
      const uint4 v = __ldg(reinterpret_cast<const uint4*>(p.w) + e);
      ptx::st_shared_v4(w_smem + (uint32_t)blk * wblk_bytes + (uint32_t)r * 128u + (uint32_t)((j ^ (r & 7)) << 4), v);
    }
    for (int e = t; e < p.n_hidden * W; e += kNwThreads) fsm[e] = __ldg(p.bias + e);
    for (int e = t; e < 2 * W; e += kNwThreads) fsm[p.n_hidden * W + e] = (e < p.n_out * W) ? __ldg(p.head_w + e) : 0.0f;
  }
  if (t == 0) { ptx::mbar_init(bar, 1); ptx::fence_mbar_init(); }
  if (warp == 0) { ptx::tmem_alloc<1>(tmem_slot, 128); ptx::tmem_relinquish<1>(); }
  ptx::fence_proxy_async_smem();
  ptx::tc_fence_before();
  __syncthreads();
  ptx::tc_fence_after();
  uint32_t tmem_base;
  asm volatile("ld.shared.u32 %0, [%1];" : "=r"(tmem_base) : "r"(tmem_slot));
  const uint32_t taddr = tmem_base + ((uint32_t)(warp * 32) << 16);
  const uint32_t idesc = ptx::idesc_bf16_f32(128, W);
  uint32_t phase = 0;
  const int last_layer = p.n_hidden - 1;

  const int64_t n_rays = p.n_dev ? *p.n_dev : p.n;
  const int64_t num_tiles = (n_rays + kNwThreads - 1) / kNwThreads;
  for (int64_t tile = blockIdx.x; tile < num_tiles; tile += gridDim.x) {
    const int64_t ray = tile * kNwThreads + t;
    const bool valid = ray < n_rays;
    // ---- gamma(o, d) -> bf16 row of the G tile
    {
      __align__(16) __nv_bfloat16 enc[128];
      for (int k = 0; k < p.gblocks * 64; ++k) enc[k] = __float2bfloat16_rn(0.0f);
      if (valid) {
        float v[3] = { p.o[3 * ray], p.o[3 * ray + 1], p.o[3 * ray + 2] };
        encode_vec_bf16(v, p.Lo, enc);
        if (p.input_kind == 0) {
          float w3[3] = { p.d[3 * ray], p.d[3 * ray + 1], p.d[3 * ray + 2] };
          encode_vec_bf16(w3, p.Ld, enc + 3 + 6 * p.Lo);
        }
      }
      const uint4* src = reinterpret_cast<const uint4*>(enc);
      for (int c = 0; c < p.gblocks * 8; ++c)
        ptx::st_shared_v4(g_smem + (uint32_t)(c >> 3) * 16384u + (uint32_t)t * 128u + (uint32_t)(((c & 7) ^ (t & 7)) << 4), src[c]);
    }
    float z0 = 0.0f, z1 = 0.0f;
    for (int l = 0; l < p.n_hidden; ++l) {
      ptx::fence_proxy_async_smem();
      ptx::tc_fence_before();
      __syncthreads();
      if (warp == 0) {
        ptx::tc_fence_after();
        if (ptx::elect_one()) {
          const int nb0 = (l == 0) ? p.gblocks : p.hblocks;             // blocks of the layer's own input
          const int nb1 = (l == p.skip_layer) ? p.gblocks : 0;          // + gamma at the skip layer
          const uint32_t a0 = (l == 0) ? g_smem : h_smem;
          uint32_t acc = 0;
          for (int kb = 0; kb < nb0 + nb1; ++kb) {
            const uint32_t a_addr = (kb < nb0) ? a0 + (uint32_t)kb * 16384u : g_smem + (uint32_t)(kb - nb0) * 16384u;
            const uint64_t adesc = ptx::smem_desc_k_sw128(a_addr);
            const uint64_t bdesc = ptx::smem_desc_k_sw128(w_smem + (uint32_t)(p.w_blk_off[l] + kb) * wblk_bytes);
            #pragma unroll
            for (int k = 0; k < 4; ++k) { ptx::umma_bf16<1>(tmem_base, adesc + 2u * k, bdesc + 2u * k, idesc, acc); acc = 1u; }
          }
          ptx::umma_commit<1>(bar);
        }
        __syncwarp();
      }
      ptx::mbar_wait_bounded(bar, phase);
      phase ^= 1u;
      ptx::tc_fence_after();
      const float* bl = fsm + l * W;
      for (int hb = 0; hb < p.hblocks; ++hb) {                          // 64 output columns at a time
        uint32_t r[64];
        ptx::tmem_ld32(taddr + hb * 64, *reinterpret_cast<uint32_t(*)[32]>(&r[0]));
        ptx::tmem_ld32(taddr + hb * 64 + 32, *reinterpret_cast<uint32_t(*)[32]>(&r[32]));
        ptx::tmem_ld_wait();
        #pragma unroll
        for (int i = 0; i < 16; ++i) {                                  // bias: broadcast 16-byte loads
          const float4 b4 = reinterpret_cast<const float4*>(bl + hb * 64)[i];
          r[4 * i + 0] = __float_as_uint(fmaxf(__uint_as_float(r[4 * i + 0]) + b4.x, 0.0f));
          r[4 * i + 1] = __float_as_uint(fmaxf(__uint_as_float(r[4 * i + 1]) + b4.y, 0.0f));
          r[4 * i + 2] = __float_as_uint(fmaxf(__uint_as_float(r[4 * i + 2]) + b4.z, 0.0f));
          r[4 * i + 3] = __float_as_uint(fmaxf(__uint_as_float(r[4 * i + 3]) + b4.w, 0.0f));
        }
        if (l < last_layer) {
          // every MMA of this layer has completed (commit observed): the H tile may be overwritten
          #pragma unroll
          for (int j = 0; j < 8; ++j) {
            uint4 pk;
            pk.x = nw_pack(__uint_as_float(r[8 * j + 0]), __uint_as_float(r[8 * j + 1]));
            pk.y = nw_pack(__uint_as_float(r[8 * j + 2]), __uint_as_float(r[8 * j + 3]));
            pk.z = nw_pack(__uint_as_float(r[8 * j + 4]), __uint_as_float(r[8 * j + 5]));
            pk.w = nw_pack(__uint_as_float(r[8 * j + 6]), __uint_as_float(r[8 * j + 7]));
            ptx::st_shared_v4(h_smem + (uint32_t)hb * 16384u + (uint32_t)t * 128u + (uint32_t)((j ^ (t & 7)) << 4), pk);
          }
        } else {
          const float* hw = fsm + p.n_hidden * W + hb * 64;
          #pragma unroll
          for (int i = 0; i < 16; ++i) {
            const float4 a4 = reinterpret_cast<const float4*>(hw)[i], c4 = reinterpret_cast<const float4*>(hw + W)[i];
            z0 = fmaf(__uint_as_float(r[4 * i + 0]), a4.x, z0); z1 = fmaf(__uint_as_float(r[4 * i + 0]), c4.x, z1);
            z0 = fmaf(__uint_as_float(r[4 * i + 1]), a4.y, z0); z1 = fmaf(__uint_as_float(r[4 * i + 1]), c4.y, z1);
            z0 = fmaf(__uint_as_float(r[4 * i + 2]), a4.z, z0); z1 = fmaf(__uint_as_float(r[4 * i + 2]), c4.z, z1);
            z0 = fmaf(__uint_as_float(r[4 * i + 3]), a4.w, z0); z1 = fmaf(__uint_as_float(r[4 * i + 3]), c4.w, z1);
          }
        }
      }
    }
    // ---- heads (t = distance, xi = visibility)
    z0 += p.head_b[0]; z1 += p.head_b[1];
    if (p.mode_out == 1) {
      if (valid) { p.out0[ray * p.n_out] = z0; if (p.n_out == 2) p.out0[ray * p.n_out + 1] = z1; }
    } else if (p.mode_out == 0) {
      if (valid) {
        if (p.n_out == 2) { p.out0[ray] = softplus_f(z0); if (p.out1) p.out1[ray] = sigmoid_f(z1); }
        else p.out0[ray] = z0;
      }
    } else {
      const bool hit = valid && (sigmoid_f(z1) > 0.5f) && (softplus_f(z0) < p.ao_radius);
      const uint32_t m = __ballot_sync(0xffffffffu, hit);
      const int g0 = (lane / p.spp) * p.spp;
      const uint32_t bits = (p.spp == 32) ? m : ((m >> g0) & ((1u << p.spp) - 1u));
      if (valid && (lane % p.spp) == 0) p.out0[ray / p.spp] = 1.0f - (float)__popc(bits) / (float)p.spp;
    }
    ptx::tc_fence_before();
  }
  __syncthreads();
  if (warp == 0) ptx::tmem_dealloc<1>(tmem_base, 128);
}

// ------------------------------------------------------------------------------------------ host
void narrow_plan_destroy(Model* m) {
  if (!m->nw) return;
  cudaFree(m->nw->d_w); cudaFree(m->nw->d_bias);
  delete m->nw;
  m->nw = nullptr;
}

// hw: the padded host copy ddf_create built ([round_up(out,128)][k_pad] per layer); hb: biases
int narrow_plan_create(Model* m, const uint16_t* hw, const float* hb) {
  m->nw = nullptr;
  const ddf_layout& L = m->lay;
  const int W = (int)L.width;
  if ((W != 64 && W != 128) || L.n_hidden > (uint32_t)kNwMaxLayers || m->E_pad > 128) return DDF_OK;   // not this path's shape
  const int gblocks = m->E_pad / 64, hblocks = W / 64;
  int total = 0;
  int blk_off[kNwMaxLayers];
  for (int l = 0; l < (int)L.n_hidden; ++l) { blk_off[l] = total; total += m->layers[l].k_pad / 64; }
  const size_t smem = (size_t)(gblocks + hblocks) * 16384 + (size_t)total * W * 128 + (size_t)(L.n_hidden + 2) * W * 4 + 64 + 1024;
  int dev = 0; cudaDeviceProp prop;
  DDF_CUDA_TRY(cudaGetDevice(&dev));
  DDF_CUDA_TRY(cudaGetDeviceProperties(&prop, dev));
  if (smem > prop.sharedMemPerBlockOptin) return DDF_OK;               // weights do not fit: SIMT path serves it
  NarrowPlan* t = new (std::nothrow) NarrowPlan();
  if (!t) return DDF_E_NOMEM;
  memset(t, 0, sizeof(NarrowPlan));
  m->nw = t;
  std::vector<uint16_t> blocks((size_t)total * W * 64, 0);
  std::vector<float> bias((size_t)L.n_hidden * W, 0.0f);
  for (int l = 0; l < (int)L.n_hidden; ++l) {
    const LayerDesc& d = m->layers[l];
    for (int kb = 0; kb < d.k_pad / 64; ++kb)
      for (int j = 0; j < W; ++j)
        memcpy(&blocks[((size_t)(blk_off[l] + kb) * W + j) * 64], hw + d.w_off + (size_t)j * d.k_pad + (size_t)kb * 64, 128);
    for (int j = 0; j < W; ++j) bias[(size_t)l * W + j] = hb[d.b_off + j];
  }
  DDF_CUDA_TRY(cudaMalloc(&t->d_w, blocks.size() * 2));
  DDF_CUDA_TRY(cudaMalloc(&t->d_bias, bias.size() * 4));
  DDF_CUDA_TRY(cudaMemcpy(t->d_w, blocks.data(), blocks.size() * 2, cudaMemcpyHostToDevice));
  DDF_CUDA_TRY(cudaMemcpy(t->d_bias, bias.data(), bias.size() * 4, cudaMemcpyHostToDevice));
  NwParams& p = t->base;
  p.w = t->d_w; p.bias = t->d_bias; p.head_w = m->d_head_w;
  p.head_b[0] = hb[m->layers[L.n_hidden].b_off]; p.head_b[1] = L.n_out == 2 ? hb[m->layers[L.n_hidden].b_off + 1] : 0.0f;
  p.n_hidden = (int)L.n_hidden; p.width = W; p.skip_layer = L.skip_layer; p.n_out = (int)L.n_out; p.input_kind = (int)L.input_kind;
  p.Lo = (int)L.n_freq_origin; p.Ld = (int)L.n_freq_dir; p.E = m->E; p.gblocks = gblocks; p.hblocks = hblocks;
  for (int l = 0; l < (int)L.n_hidden; ++l) p.w_blk_off[l] = blk_off[l];
  p.total_blocks = total;
  t->smem_bytes = smem;
  // function attributes are process-wide: the limit is the device's, the carve-out the largest any live or past model asked
  // for, so creating a smaller network never lowers what an existing larger one launches with
  DDF_CUDA_TRY(cudaFuncSetAttribute(ddf_narrow_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)prop.sharedMemPerBlockOptin));
  cudaFuncAttributes fa;
  DDF_CUDA_TRY(cudaFuncGetAttributes(&fa, ddf_narrow_kernel));
  const int regs_cta = ((fa.numRegs * 32 + 255) / 256 * 256) * (kNwThreads / 32);
  int occ = prop.regsPerMultiprocessor / (regs_cta > 0 ? regs_cta : 1);
  const int by_smem = (int)(prop.sharedMemPerMultiprocessor / (smem + prop.reservedSharedMemPerBlock));
  if (by_smem < occ) occ = by_smem;
  if (occ > 4) occ = 4;                                                 // 4 x 128 TMEM columns
  if (occ < 1) { narrow_plan_destroy(m); return DDF_OK; }
  t->ctas_per_sm = occ;
  int pct = (int)((occ * (smem + prop.reservedSharedMemPerBlock) * 100 + prop.sharedMemPerMultiprocessor - 1) / prop.sharedMemPerMultiprocessor);
  if (pct > 100) pct = 100;
  static int s_carveout = 0;
  if (pct > s_carveout) s_carveout = pct;
  DDF_CUDA_TRY(cudaFuncSetAttribute(ddf_narrow_kernel, cudaFuncAttributePreferredSharedMemoryCarveout, s_carveout));
  return DDF_OK;
}

int narrow_forward(Model* m, const float* o, const float* d, int64_t n, const int64_t* n_dev, int mode_out,
                   float* out0, float* out1, int spp, float ao_radius, cudaStream_t st) {
  NarrowPlan* t = m->nw;
  if (!t) return DDF_E_UNSUPPORTED;
  NwParams p = t->base;
  p.o = o; p.d = d; p.n = n; p.n_dev = n_dev; p.out0 = out0; p.out1 = out1;
  p.mode_out = mode_out; p.spp = spp > 0 ? spp : 1; p.ao_radius = ao_radius;
  const int64_t tiles = (n + kNwThreads - 1) / kNwThreads;
  int64_t grid = (int64_t)m->sm_count * t->ctas_per_sm;
  if (tiles < grid) grid = tiles;
  ddf_narrow_kernel<<<(unsigned)grid, kNwThreads, t->smem_bytes, st>>>(p);
  DDF_CUDA_TRY(cudaGetLastError());
  m->last_launches = 1;
  return DDF_OK;
}

}  // namespace ddf
