// ddf_hash.cu - the paper's own field: multiresolution hash grid on the ray
// origin + sinusoidal direction bands + a small ReLU MLP, one fused kernel per query batch.
//
// One CTA = 128 threads = one tile of 128 rays; thread t owns ray t of the tile, row t of the
// operand tile in shared memory and TMEM lane t of the accumulator.
//   gather    : 16 levels x 8 corners, one 8-byte (fp32) or 4-byte (fp16) load per corner, all 8
//               of a level in flight together; trilinear weights in fp32.  This is what bounds
//               the kernel (L2 sector traffic: 128 sectors per ray), not the arithmetic.
//   operand   : row t = [gamma(d) | 0 pad to 32 | level features | 0 pad to 64] as bf16, written
//               with the 128-byte swizzle the tensor core reads (the MLP weight columns are
//               permuted to this order at create).
//   layers    : D[128 x 64] = X[128 x 64] W_l^T on tcgen05 (4 MMAs of K = 16, fp32 accumulator
//               in 64 TMEM columns); tcgen05.ld -> +bias, ReLU -> bf16 row back into the operand
//               tile for the next layer; the last layer feeds the fused heads from fp32.
// Several CTAs are resident per SM (34 KB of shared memory, 64 TMEM columns each), so the
// gathers of one tile overlap the MMAs / epilogues of the others.
// Operation and readings H1-H7: include/ddf.h, DESIGN.md.
#include "ddf_common.cuh"
#include "ddf_tc_ptx.cuh"
#include "ddf_camera.cuh"
#include <cuda_fp16.h>
#include <math.h>
#include <stdlib.h>
#include <string.h>
#include <new>
#include <vector>

namespace ddf {

constexpr int kHgMaxLevels = 16;
constexpr int kHgMaxHidden = 4;
constexpr int kHgWidth = 64;
constexpr int kHgThreads = 128;
constexpr int kHgFeatCol = 32;            // operand column of the first level feature

struct HgLevel { float scale; uint32_t verts; uint32_t offset; uint32_t hashed; };

struct HgParams {
  HgLevel lv[kHgMaxLevels];
  const void* table;
  const __nv_bfloat16* w;       // [n_hidden][64][64], K-major, operand column order
  const float* bias;            // [n_hidden][64]
  const float* head_w;          // [2][64] (bf16-rounded values)
  const float* o; const float* d;
  float* out0; float* out1;
  int64_t n; const int64_t* n_dev;        // n_dev (device) overrides n when non-null; it can only be smaller
  float bmin[3], den[3];
  float head_b[2];
  float ao_radius;
  uint32_t tmask;
  int n_levels, Ld, n_hidden, n_out, table_f16, mode_out, spp;
  // primary rays generated in the kernel (ddf_query_camera): every ray starts at cam.pos, so the
  // level features are computed once per CTA; o and d are not read
  int cam_mode, cam_w, cam_h;
  CamFrame cam;
  // AO rays generated in the kernel (ddf_query_ao_points): ray k = sample k % spp of point k / spp; o and d are not read
  int ao_mode; float ao_eps; uint64_t ao_key;
  const float* ao_p; const float* ao_n;
};

struct HashPlan {
  void* d_table; __nv_bfloat16* d_w; float* d_bias; float* d_head_w;
  HgParams base;
  int ctas_per_sm;
  size_t smem_bytes;
};

__device__ __forceinline__ uint32_t pack_bf16(float a, float b) {
  __nv_bfloat162 t = __floats2bfloat162_rn(a, b);
  return *reinterpret_cast<uint32_t*>(&t);
}

// features (2 values, packed bf16) of one level at the point x01 (readings H3-H5)
template <bool F16>
__device__ __forceinline__ uint32_t hg_level_feature(const HgLevel lv, uint32_t tmask, const void* table, const float x01[3]) {
  uint32_t c0[3]; float w1[3];
  #pragma unroll
  for (int a = 0; a < 3; ++a) {
    const float pos = __fmul_rn(x01[a], lv.scale);
    const float fl = fminf(floorf(pos), lv.scale - 1.0f);
    c0[a] = (uint32_t)fl; w1[a] = pos - fl;
  }
  uint32_t kx[2], ky[2], kz[2];
  if (lv.hashed) {
    kx[0] = c0[0];                  kx[1] = c0[0] + 1u;
    ky[0] = c0[1] * 2654435761u;    ky[1] = (c0[1] + 1u) * 2654435761u;
    kz[0] = c0[2] * 805459861u;     kz[1] = (c0[2] + 1u) * 805459861u;
  } else {
    kx[0] = c0[0];                          kx[1] = c0[0] + 1u;
    ky[0] = c0[1] * lv.verts;               ky[1] = ky[0] + lv.verts;
    kz[0] = c0[2] * lv.verts * lv.verts;    kz[1] = kz[0] + lv.verts * lv.verts;
  }
  float2 v[8];
  #pragma unroll
  for (int c = 0; c < 8; ++c) {
    const uint32_t a = kx[c & 1], b = ky[(c >> 1) & 1], e = kz[c >> 2];
    const uint32_t idx = lv.offset + (lv.hashed ? ((a ^ b ^ e) & tmask) : (a + b + e));
    if (F16) v[c] = __half22float2(__ldg(reinterpret_cast<const __half2*>(table) + idx));
    else     v[c] = __ldg(reinterpret_cast<const float2*>(table) + idx);
  }
  float f0 = 0.0f, f1 = 0.0f;
  #pragma unroll
  for (int c = 0; c < 8; ++c) {
    const float wt = ((c & 1) ? w1[0] : 1.0f - w1[0]) * (((c >> 1) & 1) ? w1[1] : 1.0f - w1[1])
                   * ((c >> 2) ? w1[2] : 1.0f - w1[2]);
    f0 = fmaf(wt, v[c].x, f0); f1 = fmaf(wt, v[c].y, f1);
  }
  return pack_bf16(f0, f1);
}

// AOP: the rays are generated in the kernel from surface points (ddf_query_ao_points); a template parameter so that
// the kernels that read rays from memory carry none of it
template <bool F16, bool AOP = false>
__global__ void __launch_bounds__(kHgThreads, 5) ddf_hash_kernel(const __grid_constant__ HgParams p) {
  extern __shared__ uint8_t smem_raw[];
  const uint32_t smem_base = (ptx::smem_u32(smem_raw) + 1023u) & ~1023u;
  const uint32_t x_smem = smem_base;                                   // 128 rows x 128 B
  const uint32_t w_smem = smem_base + 16384u;                          // n_hidden x (64 rows x 128 B)
  const uint32_t f_smem = w_smem + (uint32_t)p.n_hidden * 8192u;       // bias [n_hidden][64], head [2][64]
  const uint32_t bar = f_smem + (uint32_t)(p.n_hidden + 2) * 256u;
  const uint32_t tmem_slot = bar + 8u;
  uint8_t* gen = smem_raw + (smem_base - ptx::smem_u32(smem_raw));
  float* fsm = reinterpret_cast<float*>(gen + 16384 + p.n_hidden * 8192);

  const int t = threadIdx.x, warp = t >> 5, lane = t & 31;

  // ---- one-time: weights into shared memory (swizzled K-major rows), barrier, TMEM
  for (int e = t; e < p.n_hidden * 64 * 8; e += kHgThreads) {          // 16-byte chunks
    const int l = e >> 9, r = (e >> 3) & 63, j = e & 7;
    const uint4 v = __ldg(reinterpret_cast<const uint4*>(p.w) + e);
    ptx::st_shared_v4(w_smem + (uint32_t)l * 8192u + (uint32_t)r * 128u + (uint32_t)((j ^ (r & 7)) << 4), v);
  }
  for (int e = t; e < p.n_hidden * 64; e += kHgThreads) fsm[e] = __ldg(p.bias + e);
  for (int e = t; e < 128; e += kHgThreads) fsm[p.n_hidden * 64 + e] = (e < p.n_out * 64) ? __ldg(p.head_w + e) : 0.0f;
  if (t == 0) { ptx::mbar_init(bar, 1); ptx::fence_mbar_init(); }
  if (warp == 0) { ptx::tmem_alloc<1>(tmem_slot, 64); ptx::tmem_relinquish<1>(); }
  ptx::fence_proxy_async_smem();
  ptx::tc_fence_before();
  __syncthreads();
  ptx::tc_fence_after();
  uint32_t tmem_base;
  asm volatile("ld.shared.u32 %0, [%1];" : "=r"(tmem_base) : "r"(tmem_slot));
  const uint32_t taddr = tmem_base + ((uint32_t)(warp * 32) << 16);
  constexpr uint32_t idesc = ptx::idesc_bf16_f32(128, kHgWidth);
  const uint32_t xrow = x_smem + (uint32_t)t * 128u;
  uint32_t phase = 0;

  // shared origin: thread l computes level l once for the whole CTA
  uint32_t* cam_feat = nullptr;
  if (p.cam_mode) {
    cam_feat = reinterpret_cast<uint32_t*>(gen + (bar - smem_base) + 16);
    if (t < p.n_levels) {
      float x01[3];
      #pragma unroll
      for (int a = 0; a < 3; ++a) {
        const float v = __fdiv_rn(__fsub_rn(p.cam.pos[a], p.bmin[a]), p.den[a]);
        x01[a] = fminf(fmaxf(v, 0.0f), 1.0f);
      }
      cam_feat[t] = hg_level_feature<F16>(p.lv[t], p.tmask, p.table, x01);
    }
    __syncthreads();
  }
  const int64_t n_rays = p.n_dev ? *p.n_dev : p.n;
  const int64_t num_tiles = (n_rays + kHgThreads - 1) / kHgThreads;
  for (int64_t tile = blockIdx.x; tile < num_tiles; tile += gridDim.x) {
    const int64_t ray = tile * kHgThreads + t;
    const bool valid = ray < n_rays;
    uint32_t rw[32];                                   // the operand row, 64 bf16
    #pragma unroll
    for (int i = 0; i < 32; ++i) rw[i] = 0u;
    float ov[3] = {0.0f, 0.0f, 0.0f};                  // the origin when the kernel generates the ray itself (ao_mode)
    if (valid) {
      // ---- gamma(d): identity, then per band 3 sines and 3 cosines (ddf.h), columns 0..26
      float g[32];
      #pragma unroll
      for (int i = 0; i < 32; ++i) g[i] = 0.0f;
      float dv[3];
      if (p.cam_mode) pixel_dir(p.cam, p.cam_w, p.cam_h, (int)(ray % p.cam_w), (int)(ray / p.cam_w), dv);
      else if (AOP) {
        const int64_t pt = ray / p.spp;
        const float pp[3] = { p.ao_p[3 * pt], p.ao_p[3 * pt + 1], p.ao_p[3 * pt + 2] };
        const float nn[3] = { p.ao_n[3 * pt], p.ao_n[3 * pt + 1], p.ao_n[3 * pt + 2] };
        ao_ray_from_point(pp, nn, p.ao_key, ray, p.ao_eps, ov, dv);
      }
      else { dv[0] = p.d[3 * ray]; dv[1] = p.d[3 * ray + 1]; dv[2] = p.d[3 * ray + 2]; }
      g[0] = dv[0]; g[1] = dv[1]; g[2] = dv[2];
      #pragma unroll
      for (int k = 0; k < 4; ++k) {
        if (k < p.Ld) {
          #pragma unroll
          for (int c = 0; c < 3; ++c) {
            float s, co;
            sincospif(ldexpf(dv[c], k), &s, &co);
            g[3 + 6 * k + c] = s; g[6 + 6 * k + c] = co;
          }
        }
      }
      #pragma unroll
      for (int i = 0; i < 16; ++i) rw[i] = pack_bf16(g[2 * i], g[2 * i + 1]);
    }
    // ---- hash grid on the origin (readings H1-H5)
    float x01[3] = {0.0f, 0.0f, 0.0f};
    if (valid && !p.cam_mode) {
      #pragma unroll
      for (int a = 0; a < 3; ++a) {
        const float oa = AOP ? ov[a] : p.o[3 * ray + a];
        const float v = __fdiv_rn(__fsub_rn(oa, p.bmin[a]), p.den[a]);
        x01[a] = fminf(fmaxf(v, 0.0f), 1.0f);
      }
    }
    // Rays that share an origin share its level features.  When every aligned group of 16 rays of this warp
    // does (the rays of an AO point, of a camera, of a light sample), lane j of a group computes level j once
    // and the group exchanges the results: 8 gathers per ray instead of 128, the same function of the same
    // point, so the same bits.  The test is warp-uniform; any other warp takes the per-ray path below.
    static_assert(kHgMaxLevels <= 16, "one level per lane of a 16-lane group");
    bool shared16 = false;
    if (!p.cam_mode) {
      const int leader = lane & ~15;
      float xg[3];
      bool same = true;
      #pragma unroll
      for (int a = 0; a < 3; ++a) {
        xg[a] = __shfl_sync(0xffffffffu, x01[a], leader);
        same = same && (__float_as_uint(xg[a]) == __float_as_uint(x01[a]));
      }
      shared16 = __all_sync(0xffffffffu, same || !valid);
      if (shared16) {
        const int lj = lane & 15;
        const uint32_t f = (lj < p.n_levels) ? hg_level_feature<F16>(p.lv[lj], p.tmask, p.table, xg) : 0u;
        #pragma unroll
        for (int l = 0; l < kHgMaxLevels; ++l) {
          const uint32_t v = __shfl_sync(0xffffffffu, f, leader + l);
          if (valid && l < p.n_levels) rw[kHgFeatCol / 2 + l] = v;
        }
      }
    }
    if (valid && !shared16) {
      #pragma unroll
      for (int l = 0; l < kHgMaxLevels; ++l) {
        if (l < p.n_levels) {
          rw[kHgFeatCol / 2 + l] = cam_feat ? cam_feat[l] : hg_level_feature<F16>(p.lv[l], p.tmask, p.table, x01);
        }
      }
    }
    #pragma unroll
    for (int j = 0; j < 8; ++j)
      ptx::st_shared_v4(xrow + (uint32_t)((j ^ (t & 7)) << 4), make_uint4(rw[4 * j], rw[4 * j + 1], rw[4 * j + 2], rw[4 * j + 3]));

    float z0 = 0.0f, z1 = 0.0f;
    for (int l = 0; l < p.n_hidden; ++l) {
      ptx::fence_proxy_async_smem();                   // operand rows -> visible to the tensor core
      ptx::tc_fence_before();
      __syncthreads();
      if (warp == 0) {
        ptx::tc_fence_after();
        if (ptx::elect_one()) {
          const uint64_t adesc = ptx::smem_desc_k_sw128(x_smem);
          const uint64_t bdesc = ptx::smem_desc_k_sw128(w_smem + (uint32_t)l * 8192u);
          #pragma unroll
          for (int k = 0; k < 4; ++k) ptx::umma_bf16<1>(tmem_base, adesc + 2u * k, bdesc + 2u * k, idesc, (uint32_t)(k != 0));
          ptx::umma_commit<1>(bar);
        }
        __syncwarp();
      }
      ptx::mbar_wait_bounded(bar, phase);
      phase ^= 1u;
      ptx::tc_fence_after();
      uint32_t r[64];
      ptx::tmem_ld32(taddr, *reinterpret_cast<uint32_t(*)[32]>(&r[0]));
      ptx::tmem_ld32(taddr + 32, *reinterpret_cast<uint32_t(*)[32]>(&r[32]));
      ptx::tmem_ld_wait();
      const float* bl = fsm + l * 64;
      #pragma unroll
      for (int i = 0; i < 16; ++i) {                                    // bias: broadcast 16-byte loads
        const float4 b4 = reinterpret_cast<const float4*>(bl)[i];
        r[4 * i + 0] = __float_as_uint(fmaxf(__uint_as_float(r[4 * i + 0]) + b4.x, 0.0f));
        r[4 * i + 1] = __float_as_uint(fmaxf(__uint_as_float(r[4 * i + 1]) + b4.y, 0.0f));
        r[4 * i + 2] = __float_as_uint(fmaxf(__uint_as_float(r[4 * i + 2]) + b4.z, 0.0f));
        r[4 * i + 3] = __float_as_uint(fmaxf(__uint_as_float(r[4 * i + 3]) + b4.w, 0.0f));
      }
      if (l < p.n_hidden - 1) {
        // MMA l has completed (the commit arrived), so the operand tile may be overwritten
        #pragma unroll
        for (int j = 0; j < 8; ++j) {
          uint4 pk;
          pk.x = pack_bf16(__uint_as_float(r[8 * j + 0]), __uint_as_float(r[8 * j + 1]));
          pk.y = pack_bf16(__uint_as_float(r[8 * j + 2]), __uint_as_float(r[8 * j + 3]));
          pk.z = pack_bf16(__uint_as_float(r[8 * j + 4]), __uint_as_float(r[8 * j + 5]));
          pk.w = pack_bf16(__uint_as_float(r[8 * j + 6]), __uint_as_float(r[8 * j + 7]));
          ptx::st_shared_v4(xrow + (uint32_t)((j ^ (t & 7)) << 4), pk);
        }
      } else {
        const float* hw = fsm + p.n_hidden * 64;
        #pragma unroll
        for (int i = 0; i < 16; ++i) {
          const float4 a4 = reinterpret_cast<const float4*>(hw)[i], c4 = reinterpret_cast<const float4*>(hw + 64)[i];
          z0 = fmaf(__uint_as_float(r[4 * i + 0]), a4.x, z0); z1 = fmaf(__uint_as_float(r[4 * i + 0]), c4.x, z1);
          z0 = fmaf(__uint_as_float(r[4 * i + 1]), a4.y, z0); z1 = fmaf(__uint_as_float(r[4 * i + 1]), c4.y, z1);
          z0 = fmaf(__uint_as_float(r[4 * i + 2]), a4.z, z0); z1 = fmaf(__uint_as_float(r[4 * i + 2]), c4.z, z1);
          z0 = fmaf(__uint_as_float(r[4 * i + 3]), a4.w, z0); z1 = fmaf(__uint_as_float(r[4 * i + 3]), c4.w, z1);
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
    // the next tile's operand rows are written after this point; every thread's tcgen05.ld of
    // the last layer is complete (wait::ld above) and the next MMA is issued only after the
    // __syncthreads at the top of the layer loop
    ptx::tc_fence_before();
  }
  __syncthreads();
  if (warp == 0) ptx::tmem_dealloc<1>(tmem_base, 64);
}

// ------------------------------------------------------------------------------------------ host
static int hg_check(const ddf_hashgrid_layout* L) {
  if (L->struct_size != sizeof(ddf_hashgrid_layout) || L->version != DDF_LAYOUT_VERSION) return DDF_E_BAD_LAYOUT;
  if (L->n_levels < 1 || L->n_features < 1 || L->log2_table_size < 4 || L->log2_table_size > 28) return DDF_E_BAD_LAYOUT;
  if (L->base_resolution < 1 || !(L->growth >= 1.0f) || L->n_hidden < 1 || L->width < 1) return DDF_E_BAD_LAYOUT;
  if (L->n_out < 1 || L->n_out > 2 || L->mlp_dtype > 1 || L->weights_on_device > 1) return DDF_E_BAD_LAYOUT;
  if (L->table_dtype != 0 && L->table_dtype != 2) return DDF_E_BAD_LAYOUT;
  for (int a = 0; a < 3; ++a) if (!(L->box_max[a] > L->box_min[a])) return DDF_E_BAD_LAYOUT;
  if (L->n_levels > 32 || L->n_features > 8) return DDF_E_UNSUPPORTED;
  return DDF_OK;
}

// reading H1 / H4: resolution, stored entries, offset of every level
static int hg_levels(const ddf_hashgrid_layout* L, std::vector<HgLevel>* out, int64_t* total) {
  const int64_t T = (int64_t)1 << L->log2_table_size;
  int64_t off = 0;
  for (uint32_t l = 0; l < L->n_levels; ++l) {
    const double nd = floor((double)L->base_resolution * pow((double)L->growth, (double)l));
    if (!(nd >= 1.0) || nd > 16777215.0) return DDF_E_UNSUPPORTED;     // N_l must be exact in fp32
    const int64_t N = (int64_t)nd, V = N + 1;
    const bool dense = V <= 1024 && V * V * V <= T;
    HgLevel lv;
    lv.scale = (float)N; lv.verts = (uint32_t)V; lv.hashed = dense ? 0u : 1u;
    if (off > 0xFFFFFFFFll - T) return DDF_E_UNSUPPORTED;
    lv.offset = (uint32_t)off;
    off += dense ? V * V * V : T;
    if (out) out->push_back(lv);
  }
  *total = off;
  return DDF_OK;
}

void hash_plan_destroy(Model* m) {
  if (!m->hg) return;
  cudaFree(m->hg->d_table); cudaFree(m->hg->d_w); cudaFree(m->hg->d_bias); cudaFree(m->hg->d_head_w);
  delete m->hg;
  m->hg = nullptr;
}

int hash_forward_camera(Model* m, const ddf_camera* cam, int width, int height, float* out0, float* out1, cudaStream_t st) {
  HashPlan* h = m->hg;
  HgParams p = h->base;
  const int64_t n = (int64_t)width * height;
  p.o = nullptr; p.d = nullptr; p.n = n; p.n_dev = nullptr; p.out0 = out0; p.out1 = out1;
  p.mode_out = 0; p.spp = 1; p.ao_radius = 0.0f;
  p.cam_mode = 1; p.cam_w = width; p.cam_h = height; p.cam = make_frame(cam);
  const int64_t tiles = (n + kHgThreads - 1) / kHgThreads;
  int64_t grid = (int64_t)m->sm_count * h->ctas_per_sm;
  if (tiles < grid) grid = tiles;
  if (p.table_f16) ddf_hash_kernel<true><<<(unsigned)grid, kHgThreads, h->smem_bytes, st>>>(p);
  else             ddf_hash_kernel<false><<<(unsigned)grid, kHgThreads, h->smem_bytes, st>>>(p);
  DDF_CUDA_TRY(cudaGetLastError());
  m->last_launches = 1;
  return DDF_OK;
}

int hash_forward_ao_points(Model* m, const float* pts, const float* nrm, int64_t n_pts, const int64_t* n_rays_dev, int spp,
                           uint64_t key, float eps, float ao_radius, float* ao, cudaStream_t st) {
  HashPlan* h = m->hg;
  HgParams p = h->base;
  const int64_t n = n_pts * spp;
  p.o = nullptr; p.d = nullptr; p.n = n; p.n_dev = n_rays_dev; p.out0 = ao; p.out1 = nullptr;
  p.mode_out = 2; p.spp = spp; p.ao_radius = ao_radius;
  p.ao_mode = 1; p.ao_eps = eps; p.ao_key = key; p.ao_p = pts; p.ao_n = nrm;
  const int64_t tiles = (n + kHgThreads - 1) / kHgThreads;
  int64_t grid = (int64_t)m->sm_count * h->ctas_per_sm;
  if (tiles < grid) grid = tiles;
  if (p.table_f16) ddf_hash_kernel<true, true><<<(unsigned)grid, kHgThreads, h->smem_bytes, st>>>(p);
  else             ddf_hash_kernel<false, true><<<(unsigned)grid, kHgThreads, h->smem_bytes, st>>>(p);
  DDF_CUDA_TRY(cudaGetLastError());
  m->last_launches = 1;
  return DDF_OK;
}

int hash_forward(Model* m, const float* o, const float* d, int64_t n, const int64_t* n_dev, int mode_out,
                 float* out0, float* out1, int spp, float ao_radius, cudaStream_t st) {
  HashPlan* h = m->hg;
  HgParams p = h->base;
  p.o = o; p.d = d; p.n = n; p.n_dev = n_dev; p.out0 = out0; p.out1 = out1;
  p.mode_out = mode_out; p.spp = spp > 0 ? spp : 1; p.ao_radius = ao_radius;
  const int64_t tiles = (n + kHgThreads - 1) / kHgThreads;
  int64_t grid = (int64_t)m->sm_count * h->ctas_per_sm;
  if (tiles < grid) grid = tiles;
  if (p.table_f16) ddf_hash_kernel<true><<<(unsigned)grid, kHgThreads, h->smem_bytes, st>>>(p);
  else             ddf_hash_kernel<false><<<(unsigned)grid, kHgThreads, h->smem_bytes, st>>>(p);
  DDF_CUDA_TRY(cudaGetLastError());
  m->last_launches = 1;
  return DDF_OK;
}

}  // namespace ddf

using namespace ddf;

extern "C" int64_t ddf_hashgrid_table_entries(const ddf_hashgrid_layout* layout) {
  if (!layout) return DDF_E_INVALID_ARG;
  int rc = hg_check(layout);
  if (rc != DDF_OK) return rc;
  int64_t total = 0;
  rc = hg_levels(layout, nullptr, &total);
  return rc != DDF_OK ? rc : total;
}

static inline uint16_t hg_f32_to_bf16(float f) {
  uint32_t b; memcpy(&b, &f, 4);
  if ((b & 0x7F800000u) == 0x7F800000u) return (uint16_t)(b >> 16);
  return (uint16_t)((b + 0x7FFFu + ((b >> 16) & 1u)) >> 16);
}
static inline float hg_bf16_to_f32(uint16_t h) { uint32_t b = (uint32_t)h << 16; float f; memcpy(&f, &b, 4); return f; }

extern "C" int ddf_create_hashgrid(const void* table, const void* mlp, const ddf_hashgrid_layout* layout,
                                   ddf_model** out) {
  if (out) *out = nullptr;
  if (!table || !mlp || !layout || !out) return DDF_E_INVALID_ARG;
  int rc = hg_check(layout);
  if (rc != DDF_OK) return rc;
  const ddf_hashgrid_layout& L = *layout;
  // shapes this kernel serves
  const int n_dir = 3 + 6 * (int)L.n_freq_dir, n_feat = (int)(L.n_levels * L.n_features);
  if (L.n_features != 2 || L.n_levels > (uint32_t)kHgMaxLevels || L.n_freq_dir > 4 || L.width != (uint32_t)kHgWidth ||
      L.n_hidden > (uint32_t)kHgMaxHidden)
    return DDF_E_UNSUPPORTED;
  std::vector<HgLevel> lv;
  int64_t entries = 0;
  if ((rc = hg_levels(&L, &lv, &entries)) != DDF_OK) return rc;
  int dev = 0; cudaDeviceProp prop;
  DDF_CUDA_TRY(cudaGetDevice(&dev));
  DDF_CUDA_TRY(cudaGetDeviceProperties(&prop, dev));
  if (prop.major != 10) return DDF_E_UNSUPPORTED;

  Model* m = new (std::nothrow) Model();
  if (!m) return DDF_E_NOMEM;
  memset(m, 0, sizeof(Model));
  HashPlan* h = new (std::nothrow) HashPlan();
  if (!h) { delete m; return DDF_E_NOMEM; }
  memset(h, 0, sizeof(HashPlan));
  m->hg = h;
  m->device = dev;
  m->sm_count = prop.multiProcessorCount;
  m->E = n_feat + n_dir;
  m->lay.struct_size = sizeof(ddf_layout); m->lay.version = DDF_LAYOUT_VERSION;
  m->lay.input_kind = 0; m->lay.n_freq_dir = L.n_freq_dir; m->lay.n_hidden = L.n_hidden;
  m->lay.width = L.width; m->lay.skip_layer = -1; m->lay.n_out = L.n_out;

  auto fail = [&](int code, cudaError_t e) { if (code == DDF_E_CUDA) { g_last_cuda_error = (int)e; (void)cudaGetLastError(); }
                                             hash_plan_destroy(m); delete m; return code; };
  // ---- table: copied as is (fp32 pairs or fp16 pairs)
  const size_t tbytes = (size_t)entries * L.n_features * (L.table_dtype == 2 ? 2 : 4);
  cudaError_t e;
  if ((e = cudaMalloc(&h->d_table, tbytes)) != cudaSuccess) return fail(e == cudaErrorMemoryAllocation ? DDF_E_NOMEM : DDF_E_CUDA, e);
  if ((e = cudaMemcpy(h->d_table, table, tbytes, L.weights_on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice)) != cudaSuccess)
    return fail(DDF_E_CUDA, e);
  // ---- MLP: bf16 operands in the kernel's column order [gamma(d) | pad | features | pad]
  size_t mlp_elems = 0;
  { size_t in = (size_t)m->E; for (uint32_t l = 0; l < L.n_hidden; ++l) { mlp_elems += (size_t)L.width * in + L.width; in = L.width; }
    mlp_elems += (size_t)L.n_out * in + L.n_out; }
  const size_t esz = L.mlp_dtype == 1 ? 2 : 4;
  std::vector<uint8_t> hostm(mlp_elems * esz);
  if (L.weights_on_device) { if ((e = cudaMemcpy(hostm.data(), mlp, mlp_elems * esz, cudaMemcpyDeviceToHost)) != cudaSuccess) return fail(DDF_E_CUDA, e); }
  else memcpy(hostm.data(), mlp, mlp_elems * esz);
  auto w_bf16 = [&](size_t i) -> uint16_t { return L.mlp_dtype == 1 ? ((const uint16_t*)hostm.data())[i] : hg_f32_to_bf16(((const float*)hostm.data())[i]); };
  auto w_f32 = [&](size_t i) -> float { return L.mlp_dtype == 1 ? hg_bf16_to_f32(((const uint16_t*)hostm.data())[i]) : ((const float*)hostm.data())[i]; };
  std::vector<uint16_t> hw((size_t)L.n_hidden * 64 * 64, 0);
  std::vector<float> hb((size_t)L.n_hidden * 64, 0.0f), hh(128, 0.0f);
  size_t off = 0; int in = m->E;
  for (uint32_t l = 0; l < L.n_hidden; ++l) {
    for (int j = 0; j < 64; ++j)
      for (int k = 0; k < in; ++k) {
        // blob input order: features first, then gamma(d); operand order: gamma(d) at 0, features at 32
        const int col = (l == 0) ? (k < n_feat ? kHgFeatCol + k : k - n_feat) : k;
        hw[((size_t)l * 64 + j) * 64 + col] = w_bf16(off + (size_t)j * in + k);
      }
    off += (size_t)64 * in;
    for (int j = 0; j < 64; ++j) hb[(size_t)l * 64 + j] = w_f32(off + j);
    off += 64; in = 64;
  }
  for (uint32_t j = 0; j < L.n_out; ++j)
    for (int k = 0; k < 64; ++k) hh[(size_t)j * 64 + k] = hg_bf16_to_f32(w_bf16(off + (size_t)j * 64 + k));
  off += (size_t)L.n_out * 64;
  HgParams& p = h->base;
  p.head_b[0] = w_f32(off); p.head_b[1] = L.n_out == 2 ? w_f32(off + 1) : 0.0f;
  if ((e = cudaMalloc(&h->d_w, hw.size() * 2)) != cudaSuccess || (e = cudaMalloc(&h->d_bias, hb.size() * 4)) != cudaSuccess ||
      (e = cudaMalloc(&h->d_head_w, hh.size() * 4)) != cudaSuccess ||
      (e = cudaMemcpy(h->d_w, hw.data(), hw.size() * 2, cudaMemcpyHostToDevice)) != cudaSuccess ||
      (e = cudaMemcpy(h->d_bias, hb.data(), hb.size() * 4, cudaMemcpyHostToDevice)) != cudaSuccess ||
      (e = cudaMemcpy(h->d_head_w, hh.data(), hh.size() * 4, cudaMemcpyHostToDevice)) != cudaSuccess)
    return fail(e == cudaErrorMemoryAllocation ? DDF_E_NOMEM : DDF_E_CUDA, e);
  for (uint32_t l = 0; l < L.n_levels; ++l) p.lv[l] = lv[l];
  p.table = h->d_table; p.w = h->d_w; p.bias = h->d_bias; p.head_w = h->d_head_w;
  for (int a = 0; a < 3; ++a) { p.bmin[a] = L.box_min[a]; p.den[a] = L.box_max[a] - L.box_min[a]; }
  p.tmask = (1u << L.log2_table_size) - 1u;
  p.n_levels = (int)L.n_levels; p.Ld = (int)L.n_freq_dir; p.n_hidden = (int)L.n_hidden; p.n_out = (int)L.n_out;
  p.table_f16 = L.table_dtype == 2;
  h->smem_bytes = 16384 + (size_t)L.n_hidden * 8192 + (L.n_hidden + 2) * 256 + 128 + 1024;
  // function attributes are process-wide: the limit is the device's, the carve-out (below) the largest any model asked for,
  // so creating a smaller field never lowers what an existing larger one launches with
  const int optin = (int)prop.sharedMemPerBlockOptin;
  if ((size_t)optin < h->smem_bytes) return fail(DDF_E_UNSUPPORTED, cudaSuccess);
  if ((e = cudaFuncSetAttribute(ddf_hash_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, optin)) != cudaSuccess ||
      (e = cudaFuncSetAttribute(ddf_hash_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, optin)) != cudaSuccess ||
      (e = cudaFuncSetAttribute(ddf_hash_kernel<false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, optin)) != cudaSuccess ||
      (e = cudaFuncSetAttribute(ddf_hash_kernel<true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, optin)) != cudaSuccess)
    return fail(DDF_E_CUDA, e);
  // resident CTAs per SM from the kernel's own resource use (the runtime's occupancy query answers
  // for the current carve-out, which another library in the process may have left at "prefer L1")
  cudaFuncAttributes fa;
  if ((e = (L.table_dtype == 2 ? cudaFuncGetAttributes(&fa, ddf_hash_kernel<true>) : cudaFuncGetAttributes(&fa, ddf_hash_kernel<false>))) != cudaSuccess ||
      false)
    return fail(DDF_E_CUDA, e);
  const int regs_cta = ((fa.numRegs * 32 + 255) / 256 * 256) * (kHgThreads / 32);
  int occ = prop.regsPerMultiprocessor / (regs_cta > 0 ? regs_cta : 1);
  const int by_smem = (int)(prop.sharedMemPerMultiprocessor / (h->smem_bytes + prop.reservedSharedMemPerBlock));
  if (by_smem < occ) occ = by_smem;
  if (occ < 1) return fail(DDF_E_UNSUPPORTED, cudaSuccess);
  // measured on B200: 4 resident CTAs is the best trade between latency hiding
  // and the L1 left for the coarse levels (8 x 64 TMEM columns would be the hard limit)
  h->ctas_per_sm = occ > 4 ? 4 : occ;
  // shared-memory carve-out: just what the resident CTAs need; the rest of the 256 KB stays L1,
  // which is what serves the coarse (small) levels of the grid
  {
    int pct = (int)((h->ctas_per_sm * (h->smem_bytes + prop.reservedSharedMemPerBlock) * 100 + prop.sharedMemPerMultiprocessor - 1) / prop.sharedMemPerMultiprocessor);
    if (pct > 100) pct = 100;
    static int s_carveout = 0;
    if (pct > s_carveout) s_carveout = pct;
    pct = s_carveout;
    if ((e = cudaFuncSetAttribute(ddf_hash_kernel<false>, cudaFuncAttributePreferredSharedMemoryCarveout, pct)) != cudaSuccess ||
        (e = cudaFuncSetAttribute(ddf_hash_kernel<true>, cudaFuncAttributePreferredSharedMemoryCarveout, pct)) != cudaSuccess ||
        (e = cudaFuncSetAttribute(ddf_hash_kernel<false, true>, cudaFuncAttributePreferredSharedMemoryCarveout, pct)) != cudaSuccess ||
        (e = cudaFuncSetAttribute(ddf_hash_kernel<true, true>, cudaFuncAttributePreferredSharedMemoryCarveout, pct)) != cudaSuccess)
      return fail(DDF_E_CUDA, e);
  }
  if ((e = cudaDeviceSynchronize()) != cudaSuccess) return fail(DDF_E_CUDA, e);
  *out = reinterpret_cast<ddf_model*>(m);
  return DDF_OK;
}
