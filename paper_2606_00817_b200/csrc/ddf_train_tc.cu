// ddf_train_tc.cu - the training step's forward / backward pass on the tensor cores
// (include/ddf.h "training", arithmetic = DDF_TRAIN_BF16X3).
//
// Three kernels per pass, because they want opposite things from an SM.  The table gather and the
// gradient scatter are random 8-byte accesses: they want many threads and a large L1 (its lines hold
// the misses in flight), so they run one thread per (ray, level) with no shared memory.  The MLP
// wants 200 KB of shared memory for its operand tiles, which leaves an L1 so small that the same
// gather issued from inside it ran at a quarter of the rate.  The level features
// [n][32] and their gradients pass between the kernels through L2 (2 MB each at the paper's batch).
//
// tc_mlp_kernel: one CTA = one tile of 128 rays (= the M of a tcgen05.mma), 256 threads: thread (r, h)
// owns ray r and half h of the columns of whatever it reads back from tensor memory.  Every fp32
// operand x is written to shared memory as two bf16 terms, hi = bf16(x) and lo = bf16(x - hi)
// (16 mantissa bits together), and every matrix product is three kind::f16 MMAs,
// hi hi + hi lo + lo hi, accumulated in fp32 in tensor memory (the lo lo term, 2^-18 of the
// product, is dropped):
//
//   forward    Z_{l+1} = A_l  W_l^T          A_l K-major,        W_l K-major            (K = 64: 4 steps of 16)
//   backward   dA_l    = G_{l+1} W_l        G_{l+1} K-major,    W_l MN-major           (K = 64)
//   weights    dW_l    = G_{l+1}^T A_l      both MN-major, K = the 128 rays            (8 steps)
//
// A tile [128 rays][64 units] of bf16 has 128-byte rows in the 128-byte swizzle; read K-major it
// is an operand whose K runs over the units, read MN-major the SAME bytes are an operand whose K
// runs over the rays, so no transposed copy is ever written.  (tf32 operands would not allow
// this: an MN-major 32-bit operand needs its own 32-byte-based swizzle.)  The weight-gradient
// products of all layers are one M = 128 chain: the G tiles lie one after the other
// (M = [units of layer H-1 | units of layer H-2]) and so do the A tiles (N likewise); the
// diagonal 64 x 64 blocks of the 128 x 128 result are the dW_l, the rest is not read.  That
// accumulator stays in tensor memory over all tiles of a CTA and is written once, to the CTA's own
// slab; tc_scatter_kernel's last blocks add the slabs up (atomics from every CTA onto the same 8k
// addresses were the slowest phase of the first version).
// The head (2 outputs), the loss, the ReLU masks and the bias gradients stay on the CUDA cores.  The fp32 kernel of ddf_train.cu remains as DDF_TRAIN_FP32.
#include "ddf_train.cuh"
#include "ddf_tc_ptx.cuh"
#include <cuda_bf16.h>

namespace ddf {
namespace {

constexpr int kTile = 16384;                      // [128][64] bf16
constexpr int kWTile = 8192;                      // [64][64] bf16
constexpr int kOffAh = 0;                         // slot b: input of layer H-1-b (hi terms)
constexpr int kOffAl = 2 * kTile;                 //                              (lo terms)
constexpr int kOffGh = 4 * kTile;                 // slot b: delta at the output of layer H-1-b
constexpr int kOffGl = 6 * kTile;
constexpr int kOffWh = 8 * kTile;                 // W_l [j][k], k >= fan-in zero
constexpr int kOffWl = kOffWh + 2 * kWTile;
constexpr int kOffTop = kOffWl + 2 * kWTile;      // top activations [unit][ray], pitch 129, fp32
constexpr int kOffSmall = kOffTop + kTrW * kTrPitch * 4;
constexpr int kSmallFloats = 2 * kTrW + 2 * kTrW + 2 * kTrRays + 4 * kTrRays;   // bias, head, dz, partial logits
constexpr int kSmemBytes = kOffSmall + kSmallFloats * 4 + 16 + 1024;           // + barrier, tmem slot, alignment slack
constexpr uint32_t kTmemCols = 256;               // Z 64 | dA 64 | dW 128
constexpr int kFeatPitch = 2 * kTrMaxLevels;      // floats per ray in feat / dfeat
constexpr int kSlabFloats = 2 * kTrW * kTrW;      // per CTA: block b = dW of layer H-1-b, [j][k] pitch 64
constexpr int kReduceBlocks = kSlabFloats / 256;
constexpr int kSlabSplit = 8;

// byte offset of element (row, col) of a tile with 128-byte rows (64 bf16), 128-byte swizzle
__device__ __forceinline__ uint32_t tile_off(int r, int u) {
  return (uint32_t)(((r >> 3) << 10) + ((r & 7) << 7) + (((u >> 3) ^ (r & 7)) << 4) + ((u & 7) << 1));
}
__device__ __forceinline__ void split_bf16(float x, __nv_bfloat16& hi, __nv_bfloat16& lo) {
  hi = __float2bfloat16_rn(x);
  lo = __float2bfloat16_rn(x - __bfloat162float(hi));
}
__device__ __forceinline__ void put(uint8_t* hi_tile, uint8_t* lo_tile, int r, int u, float x) {
  __nv_bfloat16 hi, lo; split_bf16(x, hi, lo);
  const uint32_t off = tile_off(r, u);
  *reinterpret_cast<__nv_bfloat16*>(hi_tile + off) = hi; *reinterpret_cast<__nv_bfloat16*>(lo_tile + off) = lo;
}
__device__ __forceinline__ float get(const uint8_t* hi_tile, const uint8_t* lo_tile, int r, int u) {
  const uint32_t off = tile_off(r, u);
  return __bfloat162float(*reinterpret_cast<const __nv_bfloat16*>(hi_tile + off)) + __bfloat162float(*reinterpret_cast<const __nv_bfloat16*>(lo_tile + off));
}
// the 32 columns [32 half, 32 half + 32) of row r: 4 swizzled 16-byte chunks in each of the two tiles
__device__ __forceinline__ void row_store32(uint8_t* hi_tile, uint8_t* lo_tile, int r, int half, const float (&x)[32]) {
  const uint32_t row = (uint32_t)(((r >> 3) << 10) + ((r & 7) << 7));
  #pragma unroll
  for (int c = 0; c < 4; ++c) {
    uint32_t ph[4], pl[4];
    #pragma unroll
    for (int q = 0; q < 4; ++q) {
      __nv_bfloat16 h0, l0, h1, l1;
      split_bf16(x[8 * c + 2 * q], h0, l0); split_bf16(x[8 * c + 2 * q + 1], h1, l1);
      ph[q] = (uint32_t)__bfloat16_as_ushort(h0) | ((uint32_t)__bfloat16_as_ushort(h1) << 16);
      pl[q] = (uint32_t)__bfloat16_as_ushort(l0) | ((uint32_t)__bfloat16_as_ushort(l1) << 16);
    }
    const uint32_t off = row + (uint32_t)((((4 * half + c) ^ (r & 7))) << 4);
    *reinterpret_cast<uint4*>(hi_tile + off) = make_uint4(ph[0], ph[1], ph[2], ph[3]);
    *reinterpret_cast<uint4*>(lo_tile + off) = make_uint4(pl[0], pl[1], pl[2], pl[3]);
  }
}
// sign information of the same 32 entries is all the ReLU mask needs: the hi terms
__device__ __forceinline__ void row_load32_hi(const uint8_t* hi_tile, int r, int half, float (&x)[32]) {
  const uint32_t row = (uint32_t)(((r >> 3) << 10) + ((r & 7) << 7));
  #pragma unroll
  for (int c = 0; c < 4; ++c) {
    const uint4 v = *reinterpret_cast<const uint4*>(hi_tile + row + (uint32_t)((((4 * half + c) ^ (r & 7))) << 4));
    const uint32_t w[4] = {v.x, v.y, v.z, v.w};
    #pragma unroll
    for (int q = 0; q < 4; ++q) { x[8 * c + 2 * q] = __uint_as_float(w[q] << 16); x[8 * c + 2 * q + 1] = __uint_as_float(w[q] & 0xFFFF0000u); }
  }
}

// D (+)= A B as hi hi + hi lo + lo hi over nk K-steps of 16.  A K-major operand advances 32 bytes
// per step inside its 128-byte rows, an MN-major one 16 rows = 2048 bytes.
template <bool A_MN, bool B_MN>
__device__ __forceinline__ void mma_x3(uint32_t d, uint32_t a_hi, uint32_t a_lo, uint32_t b_hi, uint32_t b_lo, int nk,
                                       uint32_t a_lbo, uint32_t b_lbo, uint32_t idesc, uint32_t acc = 0) {
  for (int ks = 0; ks < nk; ++ks) {
    const uint32_t as = (uint32_t)ks * (A_MN ? 2048u : 32u), bs = (uint32_t)ks * (B_MN ? 2048u : 32u);
    #pragma unroll
    for (int term = 0; term < 3; ++term) {
      const uint32_t aa = (term == 2 ? a_lo : a_hi) + as, bb = (term == 1 ? b_lo : b_hi) + bs;
      const uint64_t ad = A_MN ? ptx::smem_desc_mn_sw128(aa, a_lbo) : ptx::smem_desc_k_sw128(aa);
      const uint64_t bd = B_MN ? ptx::smem_desc_mn_sw128(bb, b_lbo) : ptx::smem_desc_k_sw128(bb);
      ptx::umma_bf16<1>(d, ad, bd, idesc, acc);
      acc = 1;
    }
  }
}

// one thread per (ray, level): feat[ray][2 l .. 2 l + 1] = the interpolated features of that level
__global__ void __launch_bounds__(256) tc_gather_kernel(const __grid_constant__ TrParams p) {
  pdl_wait();                                                  // the table is the previous step's Adam output
  pdl_launch_dependents();
  const int L = p.n_levels;
  const int64_t idx = (int64_t)blockIdx.x * 256 + threadIdx.x;
  if (idx == 0 && p.loss) *p.loss = 0.0f;
  if (idx >= p.n * L) return;
  const int64_t ray = idx / L;
  const int l = (int)(idx - ray * L);
  float x01[3];
  #pragma unroll
  for (int a = 0; a < 3; ++a) {
    const float v = __fdiv_rn(__fsub_rn(p.o[3 * ray + a], p.bmin[a]), p.den[a]);
    x01[a] = fminf(fmaxf(v, 0.0f), 1.0f);
  }
  uint32_t ix[8]; float wt[8];
  tr_corners(p.lv[l], p.tmask, x01, ix, wt);
  // The two x-neighbours of a cell edge are entries i and i ^ 1 half of the time (always when x is even on a
  // hashed level: the hash is an XOR with x): then they are one aligned 16-byte access instead of two 8-byte ones.
  float f0 = 0.0f, f1 = 0.0f;
  #pragma unroll
  for (int c = 0; c < 8; c += 2) {
    if ((ix[c] ^ ix[c + 1]) == 1u) {
      const float4 v = __ldg(reinterpret_cast<const float4*>(p.table) + (ix[c] >> 1));
      const bool sw = ix[c] & 1u;                              // corner c is the odd entry
      const float wa = sw ? wt[c + 1] : wt[c], wb = sw ? wt[c] : wt[c + 1];
      f0 = fmaf(wa, v.x, f0); f1 = fmaf(wa, v.y, f1); f0 = fmaf(wb, v.z, f0); f1 = fmaf(wb, v.w, f1);
    } else {
      const float2 v0 = __ldg(reinterpret_cast<const float2*>(p.table) + ix[c]), v1 = __ldg(reinterpret_cast<const float2*>(p.table) + ix[c + 1]);
      f0 = fmaf(wt[c], v0.x, f0); f1 = fmaf(wt[c], v0.y, f1); f0 = fmaf(wt[c + 1], v1.x, f0); f1 = fmaf(wt[c + 1], v1.y, f1);
    }
  }
  *reinterpret_cast<float2*>(p.feat + ray * kFeatPitch + 2 * l) = make_float2(f0, f1);
}

// the first kReduceBlocks * kSlabSplit blocks: the sum of the CTAs' dW slabs, one thread per MLP weight and
// 1/kSlabSplit of the slabs (they go first: they are the long ones); the rest: one thread per (ray, level),
// the 8 float2 atomics of that level's gradient
__global__ void __launch_bounds__(256) tc_scatter_kernel(const __grid_constant__ TrParams p, int n_slabs) {
  constexpr int kHead = kReduceBlocks * kSlabSplit;
  pdl_wait();
  pdl_launch_dependents();
  if ((int)blockIdx.x < kHead) {
    const int part = (int)blockIdx.x / kReduceBlocks;
    const int e = ((int)blockIdx.x - part * kReduceBlocks) * 256 + threadIdx.x;
    const int b = e / (kTrW * kTrW), j = (e / kTrW) % kTrW, k = e % kTrW;
    if (b >= p.n_hidden) return;
    const int l = p.n_hidden - 1 - b, nin = l == 0 ? p.E : kTrW;
    if (k >= nin) return;
    float s = 0.0f;
    #pragma unroll 8
    for (int c = part; c < n_slabs; c += kSlabSplit) s += p.slab[(size_t)c * kSlabFloats + e];
    atomicAdd(p.g_mlp + p.w_off[l] + j * nin + k, s);
    return;
  }
  const int L = p.n_levels;
  const int64_t idx = (int64_t)(blockIdx.x - kHead) * 256 + threadIdx.x;
  if (idx >= p.n * L) return;
  const int64_t ray = idx / L;
  const int l = (int)(idx - ray * L);
  const float2 g = *reinterpret_cast<const float2*>(p.dfeat + ray * kFeatPitch + 2 * l);
  float x01[3];
  #pragma unroll
  for (int a = 0; a < 3; ++a) {
    const float v = __fdiv_rn(__fsub_rn(p.o[3 * ray + a], p.bmin[a]), p.den[a]);
    x01[a] = fminf(fmaxf(v, 0.0f), 1.0f);
  }
  uint32_t ix[8]; float wt[8];
  tr_corners(p.lv[l], p.tmask, x01, ix, wt);
  // The coarsest levels have few entries (17^3, 25^3 for the paper's grid) and every ray of the batch lands on
  // them: 8-27 atomics per address.  They go to one of kTrRep private copies, chosen by the ray; the Adam pass
  // (or fold_rep_kernel) adds the copies up.
  float2* dst = reinterpret_cast<float2*>(p.g_table);
  if (l < p.rep_levels) dst = reinterpret_cast<float2*>(p.rep) + (size_t)(ray & (kTrRep - 1)) * p.rep_entries;
  #pragma unroll
  for (int c = 0; c < 8; c += 2) {
    if ((ix[c] ^ ix[c + 1]) == 1u) {                           // entries i, i ^ 1: one 16-byte atomic (see the gather)
      const bool sw = ix[c] & 1u;
      const float wa = sw ? wt[c + 1] : wt[c], wb = sw ? wt[c] : wt[c + 1];
      atomicAdd(reinterpret_cast<float4*>(dst) + (ix[c] >> 1), make_float4(wa * g.x, wa * g.y, wb * g.x, wb * g.y));
    } else {
      atomicAdd(dst + ix[c], make_float2(wt[c] * g.x, wt[c] * g.y));
      atomicAdd(dst + ix[c + 1], make_float2(wt[c + 1] * g.x, wt[c + 1] * g.y));
    }
  }
}

__global__ void __launch_bounds__(kTrThreads, 1) tc_mlp_kernel(const __grid_constant__ TrParams p) {
  extern __shared__ uint8_t sm_raw[];
  const uint32_t raw_u32 = ptx::smem_u32(sm_raw);
  uint8_t* sm = sm_raw + (((raw_u32 + 1023u) & ~1023u) - raw_u32);
  const uint32_t sm_u32 = ptx::smem_u32(sm);
  const int t = threadIdx.x, r = t & (kTrRays - 1), h = t >> 7, warp = t >> 5, H = p.n_hidden, E = p.E;
  float* bias = reinterpret_cast<float*>(sm + kOffSmall);      // [2][64]
  float* Wh = bias + 2 * kTrW;                                  // [2][64]
  float* dzs = Wh + 2 * kTrW;                                   // [2][128]
  float* zp = dzs + 2 * kTrRays;                                // [half][2][128]
  uint64_t* bar_p = reinterpret_cast<uint64_t*>(zp + 4 * kTrRays);
  uint32_t* tmem_slot_p = reinterpret_cast<uint32_t*>(bar_p + 1);
  float* top = reinterpret_cast<float*>(sm + kOffTop);
  const uint32_t bar = ptx::smem_u32(bar_p);

  // ---- once per CTA: weights (columns past the fan-in are zero), barrier, tensor memory
  for (int l = 0; l < H; ++l) {
    const int nin = l == 0 ? E : kTrW;
    for (int e = t; e < kTrW * kTrW; e += kTrThreads) {
      const int j = e >> 6, k = e & 63;
      put(sm + kOffWh + l * kWTile, sm + kOffWl + l * kWTile, j, k, k < nin ? p.mlp[p.w_off[l] + j * nin + k] : 0.0f);
    }
    for (int e = t; e < kTrW; e += kTrThreads) bias[l * kTrW + e] = p.mlp[p.b_off[l] + e];
  }
  for (int e = t; e < 2 * kTrW; e += kTrThreads) Wh[e] = p.mlp[p.w_off[H] + e];
  const float hb0 = p.mlp[p.b_off[H]], hb1 = p.mlp[p.b_off[H] + 1];
  if (t == 0) { ptx::mbar_init(bar, 1); ptx::fence_mbar_init(); }
  if (warp == 0) { ptx::tmem_alloc<1>(ptx::smem_u32(tmem_slot_p), kTmemCols); ptx::tmem_relinquish<1>(); }
  ptx::fence_proxy_async_smem();
  ptx::tc_fence_before();
  __syncthreads();
  ptx::tc_fence_after();
  const uint32_t tmem = *tmem_slot_p;
  const uint32_t tmZ = tmem, tmDA = tmem + 64, tmDW = tmem + 128;
  const uint32_t lane_sel = (uint32_t)(32 * (warp & 3)) << 16;
  const uint32_t idF = ptx::idesc_bf16_f32_major(128, 64, 0, 0), idB = ptx::idesc_bf16_f32_major(128, 64, 0, 1),
                 idW = ptx::idesc_bf16_f32_major(128, 64 * H, 1, 1);
  uint32_t phase = 0;
  // everything above read only the MLP parameters (final since the gather kernel started: it waited for the
  // Adam pass before it); what follows reads the gather kernel's features
  pdl_wait();
  pdl_launch_dependents();

  float block_loss = 0.0f;
  bool first_tile = true;
  const int64_t num_tiles = (p.n + kTrRays - 1) / kTrRays;
  for (int64_t tile = blockIdx.x; tile < num_tiles; tile += gridDim.x) {
    const int64_t ray = tile * kTrRays + r;
    const bool valid = ray < p.n;
    // ---- the input row [level features | gamma(d) | 0]: thread h = 0 takes the features, h = 1 the rest
    {
      uint8_t* A0h = sm + kOffAh + (H - 1) * kTile; uint8_t* A0l = sm + kOffAl + (H - 1) * kTile;
      if (p.NF == kFeatPitch) {                                // the paper's 16 levels: whole 32-column halves
        float x[32];
        if (h == 0) {
          #pragma unroll
          for (int c = 0; c < 8; ++c) {
            const float4 v = valid ? *(reinterpret_cast<const float4*>(p.feat + ray * kFeatPitch) + c) : make_float4(0.0f, 0.0f, 0.0f, 0.0f);
            x[4 * c] = v.x; x[4 * c + 1] = v.y; x[4 * c + 2] = v.z; x[4 * c + 3] = v.w;
          }
        } else {
          #pragma unroll
          for (int c = 0; c < 32; ++c) x[c] = 0.0f;
          if (valid) {
            const float dv[3] = { p.d[3 * ray], p.d[3 * ray + 1], p.d[3 * ray + 2] };
            #pragma unroll
            for (int c = 0; c < 3; ++c) x[c] = dv[c];
            #pragma unroll
            for (int k = 0; k < 4; ++k)
              if (k < p.Ld) {
                #pragma unroll
                for (int c = 0; c < 3; ++c) sincospif(ldexpf(dv[c], k), &x[3 + 6 * k + c], &x[6 + 6 * k + c]);
              }
          }
        }
        row_store32(A0h, A0l, r, h, x);
      } else if (h == 0) {
        for (int c = 0; c < p.NF; ++c) put(A0h, A0l, r, c, valid ? p.feat[ray * kFeatPitch + c] : 0.0f);
      } else {
        int m = p.NF;
        if (valid) {
          const float dv[3] = { p.d[3 * ray], p.d[3 * ray + 1], p.d[3 * ray + 2] };
          for (int c = 0; c < 3; ++c) put(A0h, A0l, r, m++, dv[c]);
          for (int k = 0; k < p.Ld; ++k) {
            float sn[3], co[3];
            for (int c = 0; c < 3; ++c) sincospif(ldexpf(dv[c], k), &sn[c], &co[c]);
            for (int c = 0; c < 3; ++c) put(A0h, A0l, r, m++, sn[c]);
            for (int c = 0; c < 3; ++c) put(A0h, A0l, r, m++, co[c]);
          }
        }
        for (; m < kTrW; ++m) put(A0h, A0l, r, m, 0.0f);
      }
    }
    ptx::fence_proxy_async_smem();
    __syncthreads();

    // ---- forward
    float a[32];                                               // own half of the top activations
    for (int l = 0; l < H; ++l) {
      if (t == 0) {
        ptx::tc_fence_after();
        mma_x3<false, false>(tmZ, sm_u32 + kOffAh + (H - 1 - l) * kTile, sm_u32 + kOffAl + (H - 1 - l) * kTile,
                             sm_u32 + kOffWh + l * kWTile, sm_u32 + kOffWl + l * kWTile, 4, 0u, 0u, idF);
        ptx::umma_commit<1>(bar);
      }
      ptx::mbar_wait_bounded(bar, phase);
      phase ^= 1u;
      ptx::tc_fence_after();
      uint32_t v[32];
      ptx::tmem_ld32(tmZ + lane_sel + 32u * h, v);
      ptx::tmem_ld_wait();
      #pragma unroll
      for (int c = 0; c < 32; ++c) a[c] = fmaxf(__uint_as_float(v[c]) + bias[l * kTrW + 32 * h + c], 0.0f);
      ptx::tc_fence_before();
      if (l < H - 1) {
        row_store32(sm + kOffAh + (H - 2 - l) * kTile, sm + kOffAl + (H - 2 - l) * kTile, r, h, a);
        ptx::fence_proxy_async_smem();
        __syncthreads();
      }
    }
    // ---- head, loss, d loss / d logits (readings T1, T2)
    {
      float z0p = 0.0f, z1p = 0.0f;
      #pragma unroll
      for (int c = 0; c < 32; ++c) {
        const int u = 32 * h + c;
        top[u * kTrPitch + r] = a[c];
        z0p = fmaf(Wh[u], a[c], z0p); z1p = fmaf(Wh[kTrW + u], a[c], z1p);
      }
      zp[(2 * h) * kTrRays + r] = z0p; zp[(2 * h + 1) * kTrRays + r] = z1p;
    }
    __syncthreads();
    float dz0 = 0.0f, dz1 = 0.0f;
    {
      const float z0 = (hb0 + zp[r]) + zp[2 * kTrRays + r], z1 = (hb1 + zp[kTrRays + r]) + zp[3 * kTrRays + r];
      if (valid) {
        const int hitf = p.hit[ray] != 0;
        const float sp = softplus_f(z0), err = sp - p.t[ray], ae = fabsf(err);
        float l = p.ce_weight * (hitf ? softplus_f(-z1) : softplus_f(z1));
        if (hitf) { l += fminf(ae, p.dist_clamp); if (ae < p.dist_clamp) dz0 = (err > 0.0f ? 1.0f : (err < 0.0f ? -1.0f : 0.0f)) * sigmoid_f(z0); }
        if (h == 0) block_loss += l;
        dz1 = p.ce_weight * (sigmoid_f(z1) - (float)hitf);
        const float inv_n = 1.0f / (float)p.n;
        dz0 *= inv_n; dz1 *= inv_n;
      }
      float g[32];
      #pragma unroll
      for (int c = 0; c < 32; ++c) { const int u = 32 * h + c; g[c] = a[c] > 0.0f ? fmaf(Wh[u], dz0, Wh[kTrW + u] * dz1) : 0.0f; }
      row_store32(sm + kOffGh, sm + kOffGl, r, h, g);
      if (h == 0) { dzs[r] = dz0; dzs[kTrRays + r] = dz1; }
    }
    ptx::fence_proxy_async_smem();
    __syncthreads();

    // ---- backward, last hidden layer first
    for (int l = H - 1; l >= 0; --l) {
      const int slot = H - 1 - l;
      if (t == 0) {
        ptx::tc_fence_after();
        mma_x3<false, true>(tmDA, sm_u32 + kOffGh + slot * kTile, sm_u32 + kOffGl + slot * kTile,
                            sm_u32 + kOffWh + l * kWTile, sm_u32 + kOffWl + l * kWTile, 4, 0u, (uint32_t)kWTile, idB);
        if (l == 0)
          mma_x3<true, true>(tmDW, sm_u32 + kOffGh, sm_u32 + kOffGl, sm_u32 + kOffAh, sm_u32 + kOffAl, 8,
                             (uint32_t)kTile, (uint32_t)kTile, idW, first_tile ? 0u : 1u);
        ptx::umma_commit<1>(bar);
      }
      // meanwhile, on the CUDA cores: head gradients (once) and the bias gradient of this layer
      if (l == H - 1) {
        if (t < 2 * kTrW) {
          const int k = t & (kTrW - 1), c = t >> 6;
          float s = 0.0f;
          for (int q = 0; q < kTrRays; ++q) s = fmaf(dzs[c * kTrRays + q], top[k * kTrPitch + q], s);
          atomicAdd(p.g_mlp + p.w_off[H] + c * kTrW + k, s);
        } else if (t >= 3 * kTrW && t < 3 * kTrW + 2) {
          float s = 0.0f;
          for (int q = 0; q < kTrRays; ++q) s += dzs[(t - 3 * kTrW) * kTrRays + q];
          atomicAdd(p.g_mlp + p.b_off[H] + (t - 3 * kTrW), s);
        }
      }
      if (t >= 2 * kTrW && t < 3 * kTrW) {
        const int u = t - 2 * kTrW;
        const uint8_t* Gh = sm + kOffGh + slot * kTile; const uint8_t* Gl = sm + kOffGl + slot * kTile;
        float s = 0.0f;
        for (int q = 0; q < kTrRays; ++q) s += get(Gh, Gl, q, u);
        atomicAdd(p.g_mlp + p.b_off[l] + u, s);
      }
      ptx::mbar_wait_bounded(bar, phase);
      phase ^= 1u;
      ptx::tc_fence_after();
      if (l > 0) {                                             // delta of the layer below: ReLU mask of its output
        uint32_t v[32]; float al[32], g[32];
        ptx::tmem_ld32(tmDA + lane_sel + 32u * h, v);
        row_load32_hi(sm + kOffAh + slot * kTile, r, h, al);
        ptx::tmem_ld_wait();
        #pragma unroll
        for (int c = 0; c < 32; ++c) g[c] = al[c] > 0.0f ? __uint_as_float(v[c]) : 0.0f;
        row_store32(sm + kOffGh + (slot + 1) * kTile, sm + kOffGl + (slot + 1) * kTile, r, h, g);
        ptx::tc_fence_before();
        ptx::fence_proxy_async_smem();
        __syncthreads();
      }
    }
    // ---- d loss / d input: its first 32 columns are the level-feature gradients tc_scatter_kernel wants
    if (h == 0) {
      uint32_t v[32];
      ptx::tmem_ld32(tmDA + lane_sel, v);
      ptx::tmem_ld_wait();
      if (valid) {
        #pragma unroll
        for (int c = 0; c < 8; ++c)
          *(reinterpret_cast<float4*>(p.dfeat + ray * kFeatPitch) + c) =
              make_float4(__uint_as_float(v[4 * c]), __uint_as_float(v[4 * c + 1]), __uint_as_float(v[4 * c + 2]), __uint_as_float(v[4 * c + 3]));
      }
    }
    first_tile = false;
    ptx::tc_fence_before();
    __syncthreads();
  }
  // ---- weight gradients of all tiles: lanes [64 b, 64 b + 64) x columns [64 b, 64 b + 64) is dW of layer H-1-b
  {
    ptx::tc_fence_after();
    const int b = r >> 6;
    uint32_t v[32];
    ptx::tmem_ld32(tmDW + lane_sel + 64u * b + 32u * h, v);
    ptx::tmem_ld_wait();
    if (b < H) {
      float4* dst = reinterpret_cast<float4*>(p.slab + (size_t)blockIdx.x * kSlabFloats + (b * kTrW + (r & 63)) * kTrW + 32 * h);
      #pragma unroll
      for (int c = 0; c < 8; ++c)
        dst[c] = make_float4(__uint_as_float(v[4 * c]), __uint_as_float(v[4 * c + 1]), __uint_as_float(v[4 * c + 2]), __uint_as_float(v[4 * c + 3]));
    }
    ptx::tc_fence_before();
  }
  #pragma unroll
  for (int sft = 16; sft > 0; sft >>= 1) block_loss += __shfl_xor_sync(0xffffffffu, block_loss, sft);
  if ((t & 31) == 0 && p.loss) atomicAdd(p.loss, block_loss / (float)p.n);
  __syncthreads();
  ptx::tc_fence_after();
  if (warp == 0) ptx::tmem_dealloc<1>(tmem, kTmemCols);
}

}  // namespace

size_t train_tc_slab_floats() { return (size_t)kSlabFloats; }
size_t train_tc_feat_pitch() { return (size_t)kFeatPitch; }
cudaError_t train_tc_prepare() {
  return cudaFuncSetAttribute(tc_mlp_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemBytes);
}
// p.feat / p.dfeat: n x 32 floats each; p.slab: grid x train_tc_slab_floats()
cudaError_t train_tc_launch(const TrParams& p, unsigned grid, cudaStream_t st) {
  const unsigned pair_blocks = (unsigned)((p.n * p.n_levels + 255) / 256);
  cudaError_t e;
  if ((e = launch_pdl(tc_gather_kernel, pair_blocks, 256, 0, st, p)) != cudaSuccess) return e;
  if ((e = launch_pdl(tc_mlp_kernel, grid, kTrThreads, kSmemBytes, st, p)) != cudaSuccess) return e;
  return launch_pdl(tc_scatter_kernel, pair_blocks + kReduceBlocks * kSlabSplit, 256, 0, st, p, (int)grid);
}

}  // namespace ddf
