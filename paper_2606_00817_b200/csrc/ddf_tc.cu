// ddf_tc.cu - the tcgen05 path: ONE persistent, warp-specialised kernel that runs the whole DDF
// forward pass (encode -> n_hidden x [GEMM + bias + ReLU + bf16] -> heads) for tiles of 128 rays
// per CTA (256 per CTA pair with cta_group::2).
//
//   warp 0      TMA producer  : streams activation (A) and weight (B) K-blocks into a smem ring
//   warp 1      MMA issuer    : tcgen05.mma (bf16 x bf16 -> fp32 in TMEM), 128x256 (or 256x256 per
//                               pair) x K accumulators, double-buffered in the 512 TMEM columns
//   warps 2-3   encoder       : gamma(o, d) of the NEXT tile, in registers, written as bf16
//                               (warp 2 also owns the TMEM allocation)
//   warps 4-11  epilogue      : tcgen05.ld -> +bias, ReLU, bf16 -> swizzled smem box -> TMA store
//                               = next layer's operand; the last layer feeds the fused heads
//                               (softplus / sigmoid / AO reduction)
//
// Layer hand-off: a 128 x width bf16 activation tile does not fit next to a weight pipeline in
// 227 KB of shared memory (320 KB at width 1280), so the epilogue writes it to a per-CTA scratch
// tile that is re-read by TMA as the next layer's A operand.  The scratch (148 CTAs x 2 x 320 KB)
// is written once and re-read at once by the same SM, i.e. it lives in the 126 MB L2; no
// activation makes a round trip through a separate kernel launch.  Producer gating is per
// 256-column output chunk (mbarriers), so layer l+1 starts its K loop while layer l's last
// chunk is still in the epilogue: the tensor pipe never drains between layers or tiles.
//
// Operation: include/ddf.h header comment (Eq.1).
#include "ddf_common.cuh"
#include "ddf_tc_ptx.cuh"
#include <cuda.h>
#include <stdlib.h>
#include <string.h>
#include <new>

namespace ddf {

constexpr int kTileM = 128;          // rays per CTA
constexpr int kChunkN = 256;         // output columns per accumulator
constexpr int kMaxTcLayers = 16;
constexpr int kMaxChunks = 8;
constexpr int kABytes = kTileM * kKBlock * 2;           // 16 KB
constexpr int kThreads = 384;

template <int CG> struct TcCfg {
  static constexpr int kBBytes = (CG == 2 ? 128 : 256) * kKBlock * 2;
  static constexpr int kStageBytes = kABytes + kBBytes;
  static constexpr int kStages = (CG == 2) ? 6 : 4;
  static constexpr int kBarBytes = 2048;
  static constexpr int kSmemBytes = kStages * kStageBytes + 8 * 4096 + kBarBytes + 1024;   // + alignment slack
};

struct TcParams {
  CUtensorMap w[kMaxTcLayers];
  CUtensorMap x0, x1, g;
  CUtensorMap xs0, xs1;              // store maps (32-row boxes) on the same activation buffers
  int hint_act, hint_w, hint_st;     // L2 eviction class of the three TMA streams (0 normal, 1 evict_last, 2 evict_first)
  int res_stages, res_e16;           // activation-resident kernel: weight stages that fit, gamma rows (E rounded up to 16)
  const float* o; const float* d;
  int64_t n; const int64_t* n_dev;
  const float* bias; const float* head_w;
  __nv_bfloat16 *x0p, *x1p, *gp;
  float* out0; float* out1;
  uint32_t* dbg;
  int n_hidden, width, n_chunks, skip_layer, n_out, input_kind, Lo, Ld, E, E_pad;
  int mode_out, spp; float ao_radius;
  int g_last_nk16;
  int b_off[kMaxTcLayers + 1];
  int nkb0[kMaxTcLayers], nkb1[kMaxTcLayers];
};

struct TcPlan {
  int cg;
  int grid;
  bool res_ok;                       // the activation-resident kernel serves this layout
  size_t res_smem;
  __nv_bfloat16 *x0, *x1, *g;
  float2* zpart;                     // column-split path: head partials [rows][n_chunks][2 halves]
  uint32_t* dbg_host; uint32_t* dbg_dev;
  TcParams base;
};

// ------------------------------------------------------------------------------------------
__device__ __forceinline__ uint64_t globaltimer_ns() {
  uint64_t t; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t)); return t;
}

// Bounded wait: a protocol error becomes a trap with a code in mapped host memory, not a hang.
template <bool CLUSTER>
__device__ __forceinline__ void wait_bar(uint32_t bar, uint32_t parity, uint32_t* dbg, uint32_t code) {
  uint32_t spins = 0; uint64_t t0 = 0;
  while (true) {
    bool ok = CLUSTER ? ptx::mbar_try_wait_cluster(bar, parity) : ptx::mbar_try_wait(bar, parity);
    if (ok) return;
    if ((++spins & 1023u) == 0) {
      uint64_t now = globaltimer_ns();
      if (t0 == 0) t0 = now;
      else if (now - t0 > ptx::kWaitTrapNs) {
        if (dbg && atomicCAS(dbg, 0u, code) == 0u) { dbg[1] = blockIdx.x; dbg[2] = parity; dbg[3] = threadIdx.x; __threadfence_system(); }
        __trap();
      }
    }
  }
}

// ---- pieces shared by the persistent and the column-split kernel (one instruction sequence, so both return the same bits)
// the MMAs of one 64-K stage into accumulator d_tmem: 4 steps of K = 16 (fewer for gamma's last block)
__device__ __forceinline__ void tc_issue_stage(uint32_t d_tmem, uint32_t a_addr, uint32_t b_addr, int nk16, int kb, uint32_t idesc) {
  const uint64_t adesc = ptx::smem_desc_k_sw128(a_addr);
  const uint64_t bdesc = ptx::smem_desc_k_sw128(b_addr);
  if (nk16 == 4) {
    ptx::umma_bf16<2>(d_tmem, adesc, bdesc, idesc, (uint32_t)(kb != 0));
    ptx::umma_bf16<2>(d_tmem, adesc + 2u, bdesc + 2u, idesc, 1u);
    ptx::umma_bf16<2>(d_tmem, adesc + 4u, bdesc + 4u, idesc, 1u);
    ptx::umma_bf16<2>(d_tmem, adesc + 6u, bdesc + 6u, idesc, 1u);
  } else {
    for (int k = 0; k < nk16; ++k)
      ptx::umma_bf16<2>(d_tmem, adesc + 2u * k, bdesc + 2u * k, idesc, (uint32_t)((kb | k) != 0));
  }
}

// An epilogue warp's 32 rows x 128 columns of a finished accumulator chunk: tcgen05.ld, + bias, ReLU, then either
// bf16 -> swizzled 32 x 64 staging box -> TMA store at (col0 + 64 box, out_row) (hidden layers), or this chunk's share
// of the head dot products from the un-rounded values (last layer).  The accumulator is handed back to the MMA warp
// (arrival on tempty_addr, the leader CTA's barrier) as soon as its last column has been read.
__device__ __forceinline__ void tc_epilogue_chunk(const TcParams& p, uint32_t taddr, uint32_t tempty_addr, int lane, const float* bias,
                                                  int col0, bool hidden, const CUtensorMap* smap, int out_row, uint32_t stage, int hint_st,
                                                  float& pc0, float& pc1) {
  #pragma unroll 1
  for (int box = 0; box < 2; ++box) {
    uint32_t r[64];
    ptx::tmem_ld32(taddr + box * 64, *reinterpret_cast<uint32_t(*)[32]>(&r[0]));
    ptx::tmem_ld32(taddr + box * 64 + 32, *reinterpret_cast<uint32_t(*)[32]>(&r[32]));
    ptx::tmem_ld_wait();
    if (box == 1) {
      ptx::tc_fence_before();
      __syncwarp();
      if (lane == 0) ptx::mbar_arrive_cluster(tempty_addr);
    }
    const int col = col0 + box * 64;
    const float4* b4 = reinterpret_cast<const float4*>(bias + col);
    #pragma unroll
    for (int i = 0; i < 16; ++i) {
      float4 bb = __ldg(b4 + i);
      r[4 * i + 0] = __float_as_uint(fmaxf(__uint_as_float(r[4 * i + 0]) + bb.x, 0.0f));
      r[4 * i + 1] = __float_as_uint(fmaxf(__uint_as_float(r[4 * i + 1]) + bb.y, 0.0f));
      r[4 * i + 2] = __float_as_uint(fmaxf(__uint_as_float(r[4 * i + 2]) + bb.z, 0.0f));
      r[4 * i + 3] = __float_as_uint(fmaxf(__uint_as_float(r[4 * i + 3]) + bb.w, 0.0f));
    }
    if (hidden) {
      if (lane == 0) ptx::bulk_wait_read<0>();          // staging box free again
      __syncwarp();
      #pragma unroll
      for (int j = 0; j < 8; ++j) {
        uint4 pk;
        __nv_bfloat162 t0 = __floats2bfloat162_rn(__uint_as_float(r[8 * j + 0]), __uint_as_float(r[8 * j + 1]));
        __nv_bfloat162 t1 = __floats2bfloat162_rn(__uint_as_float(r[8 * j + 2]), __uint_as_float(r[8 * j + 3]));
        __nv_bfloat162 t2 = __floats2bfloat162_rn(__uint_as_float(r[8 * j + 4]), __uint_as_float(r[8 * j + 5]));
        __nv_bfloat162 t3 = __floats2bfloat162_rn(__uint_as_float(r[8 * j + 6]), __uint_as_float(r[8 * j + 7]));
        pk.x = *reinterpret_cast<uint32_t*>(&t0); pk.y = *reinterpret_cast<uint32_t*>(&t1);
        pk.z = *reinterpret_cast<uint32_t*>(&t2); pk.w = *reinterpret_cast<uint32_t*>(&t3);
        ptx::st_shared_v4(stage + (uint32_t)lane * 128u + (uint32_t)((j ^ (lane & 7)) << 4), pk);
      }
      ptx::fence_proxy_async_smem();
      __syncwarp();
      if (lane == 0) {
        if (hint_st) ptx::tma_store_2d_hint(smap, stage, col, out_row, ptx::policy_of(hint_st));
        else ptx::tma_store_2d(smap, stage, col, out_row);
        ptx::bulk_commit();
      }
    } else {
      const float4* w0 = reinterpret_cast<const float4*>(p.head_w + col);
      #pragma unroll
      for (int i = 0; i < 16; ++i) {
        float4 ww = __ldg(w0 + i);
        pc0 = fmaf(__uint_as_float(r[4 * i + 0]), ww.x, pc0); pc0 = fmaf(__uint_as_float(r[4 * i + 1]), ww.y, pc0);
        pc0 = fmaf(__uint_as_float(r[4 * i + 2]), ww.z, pc0); pc0 = fmaf(__uint_as_float(r[4 * i + 3]), ww.w, pc0);
      }
      if (p.n_out == 2) {
        const float4* w1 = reinterpret_cast<const float4*>(p.head_w + p.width + col);
        #pragma unroll
        for (int i = 0; i < 16; ++i) {
          float4 ww = __ldg(w1 + i);
          pc1 = fmaf(__uint_as_float(r[4 * i + 0]), ww.x, pc1); pc1 = fmaf(__uint_as_float(r[4 * i + 1]), ww.y, pc1);
          pc1 = fmaf(__uint_as_float(r[4 * i + 2]), ww.z, pc1); pc1 = fmaf(__uint_as_float(r[4 * i + 3]), ww.w, pc1);
        }
      }
    }
  }
}

__global__ void __launch_bounds__(kThreads, 1) ddf_tc_kernel(const __grid_constant__ TcParams p) {
  constexpr int CG = 2;
  using Cfg = TcCfg<CG>;
  constexpr int S = Cfg::kStages;
  extern __shared__ uint8_t smem_raw[];
  const uint32_t smem_base = (ptx::smem_u32(smem_raw) + 1023u) & ~1023u;
  const uint32_t stg_base = smem_base + S * Cfg::kStageBytes;          // 8 x 4 KB epilogue staging boxes
  const uint32_t bar_base = stg_base + 8u * 4096u;
  // barrier map (8 bytes each)
  auto full_bar   = [&](int s) { return bar_base + 8u * s; };
  auto empty_bar  = [&](int s) { return bar_base + 8u * (8 + s); };
  auto tfull_bar  = [&](int b) { return bar_base + 8u * (16 + b); };
  auto tempty_bar = [&](int b) { return bar_base + 8u * (18 + b); };
  auto act_bar    = [&](int j) { return bar_base + 8u * (20 + j); };
  auto gready_bar = [&](int b) { return bar_base + 8u * (28 + b); };
  auto gfree_bar  = [&](int b) { return bar_base + 8u * (30 + b); };
  const uint32_t tmem_slot = bar_base + 8u * 32;
  const uint32_t zbuf = bar_base + 8u * 40;                            // 128 x float2 head partials
  auto a_smem = [&](int s) { return smem_base + s * Cfg::kStageBytes; };
  auto b_smem = [&](int s) { return smem_base + s * Cfg::kStageBytes + kABytes; };

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint32_t rank = (CG == 2) ? ptx::cluster_ctarank() : 0u;
  const bool leader = (rank == 0);
  const int pid = blockIdx.x / CG, num_pairs = gridDim.x / CG;
  const int cta_global = blockIdx.x;
  const int64_t n = p.n_dev ? *p.n_dev : p.n;
  const int64_t tile_rays = (int64_t)kTileM * CG;
  const int64_t num_tiles = (n + tile_rays - 1) / tile_rays;
  const int last_layer = p.n_hidden - 1;
  const int gamma_layer = p.skip_layer >= 0 ? p.skip_layer : 0;      // last layer that reads gamma

  if (threadIdx.x == 0) {
    for (int s = 0; s < S; ++s) { ptx::mbar_init(full_bar(s), 1); ptx::mbar_init(empty_bar(s), 1); }
    for (int b = 0; b < 2; ++b) {
      ptx::mbar_init(tfull_bar(b), 1); ptx::mbar_init(tempty_bar(b), 8 * CG);
      ptx::mbar_init(gready_bar(b), 64); ptx::mbar_init(gfree_bar(b), 1);
    }
    for (int j = 0; j < kMaxChunks; ++j) ptx::mbar_init(act_bar(j), 8);
    ptx::fence_mbar_init();
  }
  if (warp == 0 && lane == 0) {
    for (int l = 0; l < p.n_hidden; ++l) ptx::prefetch_tmap(&p.w[l]);
    ptx::prefetch_tmap(&p.x0); ptx::prefetch_tmap(&p.x1); ptx::prefetch_tmap(&p.g);
    ptx::prefetch_tmap(&p.xs0); ptx::prefetch_tmap(&p.xs1);
  }
  if (warp == 2) { ptx::tmem_alloc<CG>(tmem_slot, 512); ptx::tmem_relinquish<CG>(); }
  ptx::tc_fence_before();
  if (CG == 2) ptx::cluster_sync(); else __syncthreads();
  ptx::tc_fence_after();
  uint32_t tmem_base;
  asm volatile("ld.shared.u32 %0, [%1];" : "=r"(tmem_base) : "r"(tmem_slot));

  if (warp == 0) {
    // ================================================================ TMA producer
    {
      uint32_t it = 0, act_phase = 0;                    // bit j of act_phase: parity for act_bar(j)
      int tile_local = 0;
      const uint64_t pol_a = ptx::policy_of(p.hint_act), pol_w = ptx::policy_of(p.hint_w);
      for (int64_t tile = pid; tile < num_tiles; tile += num_pairs, ++tile_local) {
        const int gb = tile_local & 1;
        const int g_row = (cta_global * 2 + gb) * kTileM;
        for (int l = 0; l < p.n_hidden; ++l) {
          const int nk0 = p.nkb0[l], nk1 = p.nkb1[l];
          const CUtensorMap* amap = (l == 0) ? &p.g : (((l - 1) & 1) ? &p.x1 : &p.x0);
          const int a_row = (l == 0) ? g_row : cta_global * kTileM;
          for (int c = 0; c < p.n_chunks; ++c) {
            for (int kb = 0; kb < nk0 + nk1; ++kb) {
              if (c == 0 && kb < nk0) {
                if (l == 0) {
                  if (kb == 0) wait_bar<false>(gready_bar(gb), (tile_local >> 1) & 1, p.dbg, 0x100 + gb);
                } else if ((kb & 3) == 0) {
                  const int j = kb >> 2;
                  wait_bar<false>(act_bar(j), (act_phase >> j) & 1u, p.dbg, 0x200 + j);
                  act_phase ^= (1u << j);
                }
              }
              const int s = it % S; const uint32_t ph = (it / S) & 1u;
              wait_bar<CG == 2>(empty_bar(s), ph ^ 1u, p.dbg, 0x300 + s);
              const int brow = c * kChunkN + (CG == 2 ? (int)rank * 128 : 0);
              if (ptx::elect_one()) {
                if (leader) ptx::mbar_arrive_expect_tx(full_bar(s), 2u * Cfg::kStageBytes);
                const uint32_t fb = ptx::mapa(full_bar(s), 0);
                if (kb < nk0) ptx::tma_load_2d_cg2_hint(a_smem(s), amap, fb, kb * kKBlock, a_row, pol_a);
                else          ptx::tma_load_2d_cg2_hint(a_smem(s), &p.g, fb, (kb - nk0) * kKBlock, g_row, pol_a);
                ptx::tma_load_2d_cg2_hint(b_smem(s), &p.w[l], fb, kb * kKBlock, brow, pol_w);
              }
              __syncwarp();
              ++it;
            }
          }
        }
      }
    }
  } else if (warp == 1) {
    // ================================================================ MMA issuer
    // the whole warp walks the schedule (warp-uniform control flow and operands); one elected
    // lane issues the tcgen05 instructions
    if (leader) {
      constexpr uint32_t idesc = ptx::idesc_bf16_f32(128 * CG, kChunkN);
      uint32_t it = 0, cc = 0;
      int tile_local = 0;
      for (int64_t tile = pid; tile < num_tiles; tile += num_pairs, ++tile_local) {
        const int gb = tile_local & 1;
        for (int l = 0; l < p.n_hidden; ++l) {
          const int nk0 = p.nkb0[l], nk1 = p.nkb1[l], nk = nk0 + nk1;
          for (int c = 0; c < p.n_chunks; ++c, ++cc) {
            const uint32_t buf = cc & 1u, use = cc >> 1;
            wait_bar<CG == 2>(tempty_bar(buf), (use & 1u) ^ 1u, p.dbg, 0x400 + buf);
            ptx::tc_fence_after();
            const uint32_t d_tmem = tmem_base + buf * kChunkN;
            for (int kb = 0; kb < nk; ++kb, ++it) {
              const int s = it % S; const uint32_t ph = (it / S) & 1u;
              wait_bar<CG == 2>(full_bar(s), ph, p.dbg, 0x500 + s);
              ptx::tc_fence_after();
              const bool g_last = (l == 0) ? (kb == nk0 - 1) : (kb == nk - 1 && nk1 > 0);
              const int nk16 = g_last ? p.g_last_nk16 : 4;
              const bool free_gamma = (l == gamma_layer && c == p.n_chunks - 1 && kb == nk - 1);
              if (ptx::elect_one()) {
                tc_issue_stage(d_tmem, a_smem(s), b_smem(s), nk16, kb, idesc);
                ptx::umma_commit<CG>(empty_bar(s));
                if (free_gamma) ptx::umma_commit<CG>(gfree_bar(gb));
                if (kb == nk - 1) ptx::umma_commit<CG>(tfull_bar(buf));
              }
              __syncwarp();
            }
          }
        }
      }
    }
  } else if (warp >= 4) {
    // ================================================================ epilogue (8 warps)
    // warp w owns TMEM lanes 32*(w%4).. (hardware rule) and columns 128*h.. of each 256-column
    // chunk, h = (w-4)/4.  Output rows go through a 32x64 bf16 staging box (128B swizzle) and a
    // TMA store, so the next layer's TMA loads read what the async proxy itself wrote.
    const int q = warp & 3, h = (warp - 4) >> 2;
    const int row = q * 32 + lane;
    const uint32_t stage = stg_base + (uint32_t)(warp - 4) * 4096u;
    const uint32_t tempty_remote = (CG == 2) ? ptx::mapa(tempty_bar(0), 0) : 0u;
    uint32_t cc = 0;
    for (int64_t tile = pid; tile < num_tiles; tile += num_pairs) {
      const int64_t grow = tile * tile_rays + (int64_t)rank * kTileM + row;
      const bool valid = grow < n;
      float z0 = 0.0f, z1 = 0.0f;
      for (int l = 0; l < p.n_hidden; ++l) {
        const CUtensorMap* smap = (l & 1) ? &p.xs1 : &p.xs0;
        const float* bias = p.bias + p.b_off[l];
        for (int c = 0; c < p.n_chunks; ++c, ++cc) {
          const uint32_t buf = cc & 1u, use = cc >> 1;
          wait_bar<CG == 2>(tfull_bar(buf), use & 1u, p.dbg, 0x600 + buf);
          ptx::tc_fence_after();
          const uint32_t taddr = tmem_base + ((uint32_t)(q * 32) << 16) + buf * kChunkN + h * 128;
          float pc0 = 0.0f, pc1 = 0.0f;           // this chunk's share of the head dot products
          tc_epilogue_chunk(p, taddr, tempty_remote + 8u * buf, lane, bias, c * kChunkN + h * 128, l < last_layer, smap,
                            cta_global * kTileM + q * 32, stage, p.hint_st, pc0, pc1);
          // chunk partials are summed in chunk order: the column-split path (below) adds the same
          // partials in the same order, so both give the same bits
          if (l == last_layer) { z0 += pc0; z1 += pc1; }
          if (l < last_layer && lane == 0) {
            ptx::bulk_wait<0>();                  // this warp's part of chunk c is in global memory
            ptx::mbar_arrive(act_bar(c));
          }
        }
      }
      // ---- fused heads (t = distance, xi = visibility); the two column halves
      // of a row meet through shared memory, always added in the same order
      if (h == 1) { asm volatile("st.shared.v2.f32 [%0], {%1, %2};" :: "r"(zbuf + (uint32_t)row * 8u), "f"(z0), "f"(z1) : "memory"); }
      ptx::named_bar_sync(1, 256);
      if (h == 0) {
        float y0, y1;
        asm volatile("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(y0), "=f"(y1) : "r"(zbuf + (uint32_t)row * 8u) : "memory");
        z0 = (z0 + y0) + p.bias[p.b_off[p.n_hidden]];
        if (p.n_out == 2) z1 = (z1 + y1) + p.bias[p.b_off[p.n_hidden] + 1];
        if (p.mode_out == 1) {
          if (valid) { p.out0[grow * p.n_out] = z0; if (p.n_out == 2) p.out0[grow * p.n_out + 1] = z1; }
        } else if (p.mode_out == 0) {
          if (valid) {
            if (p.n_out == 2) { p.out0[grow] = softplus_f(z0); if (p.out1) p.out1[grow] = sigmoid_f(z1); }
            else p.out0[grow] = z0;
          }
        } else {
          // AO: 1 - mean over the pixel's spp consecutive rays of (xi > 0.5 and t < ao_radius)
          const bool hit = valid && (sigmoid_f(z1) > 0.5f) && (softplus_f(z0) < p.ao_radius);
          const uint32_t m = __ballot_sync(0xffffffffu, hit);
          const int g0 = (lane / p.spp) * p.spp;
          const uint32_t bits = (p.spp == 32) ? m : ((m >> g0) & ((1u << p.spp) - 1u));
          if (valid && (lane % p.spp) == 0) p.out0[grow / p.spp] = 1.0f - (float)__popc(bits) / (float)p.spp;
        }
      }
      ptx::named_bar_sync(1, 256);
    }
  } else {
    // ================================================================ encoder (warps 2, 3)
    // gamma(o, d) of this CTA's 128 rays, two rays per thread, one tile ahead of the MMAs
    const int t64 = (warp - 2) * 32 + lane;
    int tile_local = 0;
    for (int64_t tile = pid; tile < num_tiles; tile += num_pairs, ++tile_local) {
      const int gb = tile_local & 1;
      wait_bar<CG == 2>(gfree_bar(gb), ((tile_local >> 1) & 1) ^ 1, p.dbg, 0x700 + gb);
      #pragma unroll 1
      for (int rr = 0; rr < 2; ++rr) {
        const int row = t64 + rr * 64;
        const int64_t grow = tile * tile_rays + (int64_t)rank * kTileM + row;
        __align__(16) __nv_bfloat16 enc[256];
        #pragma unroll 1
        for (int k = 0; k < p.E_pad; ++k) enc[k] = __float2bfloat16_rn(0.0f);
        float v[3], w[3];
        load_ray_vec3(p.o, grow - lane, n, lane, v);                     // coalesced 16-byte loads, regrouped by shuffles
        if (p.input_kind == 0) load_ray_vec3(p.d, grow - lane, n, lane, w);
        if (grow < n) {
          encode_vec_bf16(v, p.Lo, enc);
          if (p.input_kind == 0) encode_vec_bf16(w, p.Ld, enc + 3 + 6 * p.Lo);
        }
        uint4* dst = reinterpret_cast<uint4*>(p.gp + ((size_t)(cta_global * 2 + gb) * kTileM + row) * p.E_pad);
        const uint4* src = reinterpret_cast<const uint4*>(enc);
        #pragma unroll 1
        for (int k = 0; k < p.E_pad / 8; ++k) dst[k] = src[k];
      }
      ptx::fence_proxy_async();
      __threadfence();
      ptx::mbar_arrive(gready_bar(gb));
    }
  }

  ptx::tc_fence_before();
  if (CG == 2) ptx::cluster_sync(); else __syncthreads();
  if (warp == 2) ptx::tmem_dealloc<CG>(tmem_base, 512);
}

}  // namespace ddf
#include "ddf_tc_res.cuh"
namespace ddf {

// ------------------------------------------------------------------------------------------
// Column-split path for small batches.  With fewer ray tiles than CTA pairs the persistent kernel
// above leaves most of the chip idle (a tile walks all layers on one pair: ~0.35 ms whatever n).
// Here a layer is one launch and the work item is (ray tile, 256-column output chunk), so a batch
// of t tiles keeps min(74, t * n_chunks) pairs busy; activations go through the same scratch
// (rows indexed by ray, not by CTA) and the launch boundary is the layer hand-off.  The chain
//   encode -> layer 0 .. layer n_hidden-1 -> finish
// is linked by programmatic dependent launch, so each prologue (barrier init, TMEM allocation,
// descriptor prefetch) overlaps the launch before.  Every accumulator is produced by the same MMA
// sequence as in the persistent kernel and the head partials are added in the same order:
// both paths return the same bits (tests/test_gpu_contract.py).
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

// gamma(o, d) of every row of the batch's tiles (rows >= n: zero).  One warp per row, one lane per
// slot of the row (the identity triple or one frequency band of o or d): the call is latency-bound and a
// thread per row would walk its 84 sincospif one after the other (13.9 us for one tile; 2 us this way).
// Same functions on the same arguments as encode_vec_bf16, so the same bits.
constexpr int kSplitEncRows = 4;                       // rows per 128-thread block
__global__ void __launch_bounds__(32 * kSplitEncRows) ddf_tc_split_encode_kernel(const __grid_constant__ TcParams p) {
  pdl_launch_dependents();
  const int64_t n = p.n_dev ? *p.n_dev : p.n;
  const int64_t rows = (n + 2 * kTileM - 1) / (2 * kTileM) * (2 * kTileM);
  const int lane = threadIdx.x & 31;
  const int64_t grow = (int64_t)blockIdx.x * kSplitEncRows + (threadIdx.x >> 5);
  if (grow >= rows) return;
  __nv_bfloat16* row = p.gp + (size_t)grow * p.E_pad;
  const __nv_bfloat16 zero = __float2bfloat16_rn(0.0f);
  if (grow >= n) {
    for (int k = lane; k < p.E_pad; k += 32) row[k] = zero;
    return;
  }
  const int Eo = 3 + 6 * p.Lo;
  const int so = 1 + p.Lo, sd = (p.input_kind == 0) ? 1 + p.Ld : 0;
  const int E = Eo + ((p.input_kind == 0) ? 3 + 6 * p.Ld : 0);
  for (int k = E + lane; k < p.E_pad; k += 32) row[k] = zero;
  for (int s = lane; s < so + sd; s += 32) {
    const bool is_d = s >= so;
    const float* src = is_d ? p.d : p.o;
    const int k = (is_d ? s - so : s) - 1;             // -1: the identity triple
    __nv_bfloat16* dst = row + (is_d ? Eo : 0);
    const float v[3] = { src[3 * grow], src[3 * grow + 1], src[3 * grow + 2] };
    if (k < 0) {
      #pragma unroll
      for (int c = 0; c < 3; ++c) dst[c] = __float2bfloat16_rn(v[c]);
    } else {
      #pragma unroll
      for (int c = 0; c < 3; ++c) {
        float sn, cs;
        sincospif(ldexpf(v[c], k), &sn, &cs);
        dst[3 + 6 * k + c] = __float2bfloat16_rn(sn);
        dst[6 + 6 * k + c] = __float2bfloat16_rn(cs);
      }
    }
  }
}

// one hidden layer: item = (tile, chunk), tile = 256 rays of a CTA pair, chunk = 256 output columns
__global__ void __launch_bounds__(kThreads, 1) ddf_tc_split_layer_kernel(const __grid_constant__ TcParams p, const int l,
                                                                          float2* __restrict__ zpart) {
  constexpr int CG = 2;
  using Cfg = TcCfg<CG>;
  constexpr int S = Cfg::kStages;
  extern __shared__ uint8_t smem_raw[];
  const uint32_t smem_base = (ptx::smem_u32(smem_raw) + 1023u) & ~1023u;
  const uint32_t stg_base = smem_base + S * Cfg::kStageBytes;
  const uint32_t bar_base = stg_base + 8u * 4096u;
  auto full_bar   = [&](int s) { return bar_base + 8u * s; };
  auto empty_bar  = [&](int s) { return bar_base + 8u * (8 + s); };
  auto tfull_bar  = [&](int b) { return bar_base + 8u * (16 + b); };
  auto tempty_bar = [&](int b) { return bar_base + 8u * (18 + b); };
  const uint32_t tmem_slot = bar_base + 8u * 32;
  auto a_smem = [&](int s) { return smem_base + s * Cfg::kStageBytes; };
  auto b_smem = [&](int s) { return smem_base + s * Cfg::kStageBytes + kABytes; };

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint32_t rank = ptx::cluster_ctarank();
  const bool leader = (rank == 0);
  const int pid = blockIdx.x / CG, num_pairs = gridDim.x / CG;
  const int last_layer = p.n_hidden - 1;

  if (threadIdx.x == 0) {
    pdl_launch_dependents();
    for (int s = 0; s < S; ++s) { ptx::mbar_init(full_bar(s), 1); ptx::mbar_init(empty_bar(s), 1); }
    for (int b = 0; b < 2; ++b) { ptx::mbar_init(tfull_bar(b), 1); ptx::mbar_init(tempty_bar(b), 8 * CG); }
    ptx::fence_mbar_init();
  }
  if (warp == 0 && lane == 0) {
    ptx::prefetch_tmap(&p.w[l]); ptx::prefetch_tmap(&p.g);
    ptx::prefetch_tmap(((l - 1) & 1) ? &p.x1 : &p.x0); ptx::prefetch_tmap((l & 1) ? &p.xs1 : &p.xs0);
  }
  if (warp == 2) { ptx::tmem_alloc<CG>(tmem_slot, 512); ptx::tmem_relinquish<CG>(); }
  ptx::tc_fence_before();
  ptx::cluster_sync();
  ptx::tc_fence_after();
  uint32_t tmem_base;
  asm volatile("ld.shared.u32 %0, [%1];" : "=r"(tmem_base) : "r"(tmem_slot));
  // n_dev (if any) was written before the chain's first, ordinary launch: safe to read before the wait
  const int64_t n = p.n_dev ? *p.n_dev : p.n;
  const int64_t tile_rays = (int64_t)kTileM * CG;
  const int64_t num_tiles = (n + tile_rays - 1) / tile_rays;
  const int64_t items = num_tiles * p.n_chunks;
  const int nk0 = p.nkb0[l], nk1 = p.nkb1[l], nk = nk0 + nk1;

  if (warp == 0) {
    // ================================================================ TMA producer
    // The weights do not depend on the launch before: the first item's first S weight blocks are
    // requested before the dependency wait, the activations after it.
    const CUtensorMap* amap = (l == 0) ? &p.g : (((l - 1) & 1) ? &p.x1 : &p.x0);
    const int pre = (pid < items) ? (nk < S ? nk : S) : 0;
    if (pre > 0 && ptx::elect_one()) {
      const int brow = (int)(pid % p.n_chunks) * kChunkN + (int)rank * 128;
      for (int kb = 0; kb < pre; ++kb) {
        if (leader) ptx::mbar_arrive_expect_tx(full_bar(kb), 2u * Cfg::kStageBytes);
        ptx::tma_load_2d_cg2(b_smem(kb), &p.w[l], ptx::mapa(full_bar(kb), 0), kb * kKBlock, brow);
      }
    }
    __syncwarp();
    pdl_wait();                        // everything below reads or overwrites what the launch before produced
    ptx::fence_proxy_async();          // ... some of it written through the generic proxy (gamma) and read by TMA
    uint32_t it = 0;
    for (int64_t item = pid; item < items; item += num_pairs) {
      const int tile = (int)(item / p.n_chunks), c = (int)(item - (int64_t)tile * p.n_chunks);
      const int a_row = tile * (int)tile_rays + (int)rank * kTileM;
      const int brow = c * kChunkN + (int)rank * 128;
      for (int kb = 0; kb < nk; ++kb, ++it) {
        const int s = it % S; const uint32_t ph = (it / S) & 1u;
        const bool early = it < (uint32_t)pre;             // stage armed and its weights requested above
        if (!early) wait_bar<true>(empty_bar(s), ph ^ 1u, p.dbg, 0x1300 + s);
        if (ptx::elect_one()) {
          if (leader && !early) ptx::mbar_arrive_expect_tx(full_bar(s), 2u * Cfg::kStageBytes);
          const uint32_t fb = ptx::mapa(full_bar(s), 0);
          if (kb < nk0) ptx::tma_load_2d_cg2(a_smem(s), amap, fb, kb * kKBlock, a_row);
          else          ptx::tma_load_2d_cg2(a_smem(s), &p.g, fb, (kb - nk0) * kKBlock, a_row);
          if (!early) ptx::tma_load_2d_cg2(b_smem(s), &p.w[l], fb, kb * kKBlock, brow);
        }
        __syncwarp();
      }
    }
  } else if (warp == 1) {
    // ================================================================ MMA issuer (same instruction sequence per accumulator as ddf_tc_kernel)
    pdl_wait();
    if (leader) {
      constexpr uint32_t idesc = ptx::idesc_bf16_f32(128 * CG, kChunkN);
      uint32_t it = 0, cc = 0;
      for (int64_t item = pid; item < items; item += num_pairs, ++cc) {
        const uint32_t buf = cc & 1u, use = cc >> 1;
        wait_bar<true>(tempty_bar(buf), (use & 1u) ^ 1u, p.dbg, 0x1400 + buf);
        ptx::tc_fence_after();
        const uint32_t d_tmem = tmem_base + buf * kChunkN;
        for (int kb = 0; kb < nk; ++kb, ++it) {
          const int s = it % S; const uint32_t ph = (it / S) & 1u;
          wait_bar<true>(full_bar(s), ph, p.dbg, 0x1500 + s);
          ptx::tc_fence_after();
          const bool g_last = (l == 0) ? (kb == nk0 - 1) : (kb == nk - 1 && nk1 > 0);
          const int nk16 = g_last ? p.g_last_nk16 : 4;
          if (ptx::elect_one()) {
            tc_issue_stage(d_tmem, a_smem(s), b_smem(s), nk16, kb, idesc);
            ptx::umma_commit<CG>(empty_bar(s));
            if (kb == nk - 1) ptx::umma_commit<CG>(tfull_bar(buf));
          }
          __syncwarp();
        }
      }
    }
  } else if (warp >= 4) {
    // ================================================================ epilogue (8 warps), as in ddf_tc_kernel
    const int q = warp & 3, h = (warp - 4) >> 2;
    const int row = q * 32 + lane;
    const uint32_t stage = stg_base + (uint32_t)(warp - 4) * 4096u;
    const uint32_t tempty_remote = ptx::mapa(tempty_bar(0), 0);
    const CUtensorMap* smap = (l & 1) ? &p.xs1 : &p.xs0;
    const float* bias = p.bias + p.b_off[l];
    uint32_t cc = 0;
    pdl_wait();
    for (int64_t item = pid; item < items; item += num_pairs, ++cc) {
      const int tile = (int)(item / p.n_chunks), c = (int)(item - (int64_t)tile * p.n_chunks);
      const int t_row = tile * (int)tile_rays + (int)rank * kTileM;
      const uint32_t buf = cc & 1u, use = cc >> 1;
      wait_bar<true>(tfull_bar(buf), use & 1u, p.dbg, 0x1600 + buf);
      ptx::tc_fence_after();
      const uint32_t taddr = tmem_base + ((uint32_t)(q * 32) << 16) + buf * kChunkN + h * 128;
      float pc0 = 0.0f, pc1 = 0.0f;
      tc_epilogue_chunk(p, taddr, tempty_remote + 8u * buf, lane, bias, c * kChunkN + h * 128, l < last_layer, smap, t_row + q * 32,
                        stage, 0, pc0, pc1);
      if (l == last_layer) zpart[((size_t)(t_row + row) * p.n_chunks + c) * 2 + h] = make_float2(pc0, pc1);
    }
    if (lane == 0) ptx::bulk_wait_read<0>();     // the staging boxes must outlive the bulk stores that read them
  } else {
    pdl_wait();
  }

  ptx::tc_fence_before();
  ptx::cluster_sync();
  if (warp == 2) ptx::tmem_dealloc<CG>(tmem_base, 512);
}

// heads from the chunk partials, added in the order ddf_tc_kernel adds them; one thread per ray
__global__ void __launch_bounds__(128) ddf_tc_split_finish_kernel(const __grid_constant__ TcParams p, const float2* __restrict__ zpart) {
  pdl_wait();
  const int64_t n = p.n_dev ? *p.n_dev : p.n;
  const int64_t rows = (n + 2 * kTileM - 1) / (2 * kTileM) * (2 * kTileM);
  const int64_t grow = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (grow >= rows) return;                      // whole warps: rows is a multiple of 256
  const int lane = threadIdx.x & 31;
  const bool valid = grow < n;
  float z0 = 0.0f, z1 = 0.0f, y0 = 0.0f, y1 = 0.0f;
  for (int c = 0; c < p.n_chunks; ++c) {
    const float2 a = zpart[((size_t)grow * p.n_chunks + c) * 2 + 0];
    const float2 b = zpart[((size_t)grow * p.n_chunks + c) * 2 + 1];
    z0 += a.x; z1 += a.y; y0 += b.x; y1 += b.y;
  }
  z0 = (z0 + y0) + p.bias[p.b_off[p.n_hidden]];
  if (p.n_out == 2) z1 = (z1 + y1) + p.bias[p.b_off[p.n_hidden] + 1];
  if (p.mode_out == 1) {
    if (valid) { p.out0[grow * p.n_out] = z0; if (p.n_out == 2) p.out0[grow * p.n_out + 1] = z1; }
  } else if (p.mode_out == 0) {
    if (valid) {
      if (p.n_out == 2) { p.out0[grow] = softplus_f(z0); if (p.out1) p.out1[grow] = sigmoid_f(z1); }
      else p.out0[grow] = z0;
    }
  } else {
    const bool hit = valid && (sigmoid_f(z1) > 0.5f) && (softplus_f(z0) < p.ao_radius);
    const uint32_t m = __ballot_sync(0xffffffffu, hit);
    const int g0 = (lane / p.spp) * p.spp;
    const uint32_t bits = (p.spp == 32) ? m : ((m >> g0) & ((1u << p.spp) - 1u));
    if (valid && (lane % p.spp) == 0) p.out0[grow / p.spp] = 1.0f - (float)__popc(bits) / (float)p.spp;
  }
}

// ------------------------------------------------------------------------------------------ host
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static EncodeTiledFn get_encode_fn() {
  static EncodeTiledFn fn = nullptr;
  if (!fn) {
    void* sym = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &sym, cudaEnableDefault, &qres) != cudaSuccess ||
        qres != cudaDriverEntryPointSuccess)
      return nullptr;
    fn = (EncodeTiledFn)sym;
  }
  return fn;
}

// bf16 row-major [rows][cols] with row pitch `pitch_elems`; box = 64 columns x 128 rows, 128B swizzle
static int make_map(CUtensorMap* out, void* base, uint64_t cols, uint64_t rows, uint64_t pitch_elems, uint32_t box_rows = 128u) {
  EncodeTiledFn fn = get_encode_fn();
  if (!fn) return DDF_E_UNSUPPORTED;
  cuuint64_t dims[2] = { cols, rows };
  cuuint64_t strides[1] = { pitch_elems * 2 };
  cuuint32_t box[2] = { (cuuint32_t)kKBlock, box_rows };
  cuuint32_t estr[2] = { 1u, 1u };
  CUresult r = fn(out, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, base, dims, strides, box, estr,
                  CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
                  CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  return r == CUDA_SUCCESS ? DDF_OK : DDF_E_CUDA;
}

void tc_plan_destroy(Model* m) {
  if (!m->tc) return;
  cudaFree(m->tc->x0); cudaFree(m->tc->x1); cudaFree(m->tc->g); cudaFree(m->tc->zpart);
  if (m->tc->dbg_host) cudaFreeHost(m->tc->dbg_host);
  delete m->tc;
  m->tc = nullptr;
}

int tc_plan_create(Model* m) {
  m->tc = nullptr;
  const ddf_layout& L = m->lay;
  // shapes this kernel serves: width a multiple of 256 (whole accumulator chunks), <= 16 layers
  if (L.width % kChunkN != 0 || L.width / kChunkN > (uint32_t)kMaxChunks) return DDF_OK;
  if (L.n_hidden > (uint32_t)kMaxTcLayers || m->E_pad > 256) return DDF_OK;
  TcPlan* t = new (std::nothrow) TcPlan();
  if (!t) return DDF_E_NOMEM;
  memset(t, 0, sizeof(TcPlan));
  m->tc = t;
  t->cg = 2;
  t->grid = (m->sm_count / 2) * 2;
  const size_t rows = (size_t)t->grid * kTileM;
  DDF_CUDA_TRY(cudaMalloc(&t->x0, rows * L.width * 2));
  DDF_CUDA_TRY(cudaMalloc(&t->x1, rows * L.width * 2));
  DDF_CUDA_TRY(cudaMalloc(&t->g, rows * 2 * m->E_pad * 2));
  DDF_CUDA_TRY(cudaMemset(t->x0, 0, rows * L.width * 2));
  DDF_CUDA_TRY(cudaMemset(t->x1, 0, rows * L.width * 2));
  DDF_CUDA_TRY(cudaMemset(t->g, 0, rows * 2 * m->E_pad * 2));
  DDF_CUDA_TRY(cudaMalloc(&t->zpart, rows * (L.width / kChunkN) * 2 * sizeof(float2)));
  DDF_CUDA_TRY(cudaHostAlloc(&t->dbg_host, 64, cudaHostAllocMapped));
  memset(t->dbg_host, 0, 64);
  DDF_CUDA_TRY(cudaHostGetDevicePointer((void**)&t->dbg_dev, t->dbg_host, 0));

  TcParams& p = t->base;
  int rc;
  for (int l = 0; l < (int)L.n_hidden; ++l) {
    const LayerDesc& d = m->layers[l];
    rc = make_map(&p.w[l], m->d_w + d.w_off, (uint64_t)d.k_pad, (uint64_t)round_up(d.n_out, 128), (uint64_t)d.k_pad);
    if (rc != DDF_OK) return rc;
    p.nkb0[l] = d.k0_pad / kKBlock; p.nkb1[l] = d.k1_pad / kKBlock;
    p.b_off[l] = (int)d.b_off;
  }
  p.b_off[L.n_hidden] = (int)m->layers[L.n_hidden].b_off;
  if ((rc = make_map(&p.x0, t->x0, L.width, rows, L.width)) != DDF_OK) return rc;
  if ((rc = make_map(&p.x1, t->x1, L.width, rows, L.width)) != DDF_OK) return rc;
  if ((rc = make_map(&p.xs0, t->x0, L.width, rows, L.width, 32u)) != DDF_OK) return rc;
  if ((rc = make_map(&p.xs1, t->x1, L.width, rows, L.width, 32u)) != DDF_OK) return rc;
  if ((rc = make_map(&p.g, t->g, (uint64_t)m->E_pad, rows * 2, (uint64_t)m->E_pad)) != DDF_OK) return rc;
  // L2 priorities of the persistent kernel's TMA streams: activation and weight loads evict_last, stores default
  p.hint_act = 1; p.hint_w = 1; p.hint_st = 0;
  p.bias = m->d_b; p.head_w = m->d_head_w;
  p.x0p = t->x0; p.x1p = t->x1; p.gp = t->g;
  p.dbg = t->dbg_dev;
  p.n_hidden = (int)L.n_hidden; p.width = (int)L.width; p.n_chunks = (int)L.width / kChunkN;
  p.skip_layer = L.skip_layer; p.n_out = (int)L.n_out; p.input_kind = (int)L.input_kind;
  p.Lo = (int)L.n_freq_origin; p.Ld = (int)L.n_freq_dir; p.E = m->E; p.E_pad = m->E_pad;
  p.g_last_nk16 = (m->E - (m->E_pad - kKBlock) + 15) / 16;
  DDF_CUDA_TRY(cudaFuncSetAttribute(ddf_tc_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, TcCfg<2>::kSmemBytes));
  DDF_CUDA_TRY(cudaFuncSetAttribute(ddf_tc_split_layer_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, TcCfg<2>::kSmemBytes));
  // activation-resident kernel: 64 rays x width bf16 resident per CTA, parked chunks in 256 TMEM columns (<= 5 chunks)
  p.res_e16 = (m->E + 15) / 16 * 16;
  p.res_stages = 0;
  for (int s = kResMaxStages; s >= 2; --s)
    if (res_smem_bytes((int)L.width, p.res_e16, s) <= (size_t)TcCfg<2>::kSmemBytes) { p.res_stages = s; break; }
  // two hidden layers at least: with one, nothing orders a tile's head partials (zbuf) before the next tile's writes
  t->res_ok = p.res_stages >= 2 && L.width / kChunkN <= 5 && m->E_pad <= 128 && L.n_hidden >= 2;
  if (t->res_ok) {
    t->res_smem = res_smem_bytes((int)L.width, p.res_e16, p.res_stages);
    DDF_CUDA_TRY(cudaFuncSetAttribute(ddf_tc_res_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, TcCfg<2>::kSmemBytes));
  }
  return DDF_OK;
}

// Batches of at most this many 256-ray tiles take the column-split path when the choice is automatic
// (measured on one B200: the split path wins below ~2^14 rays).
constexpr int kSplitAutoTiles = 40;

// encode -> one launch per hidden layer -> finish, chained by programmatic dependent launch
static int tc_forward_split(Model* m, const TcParams& p, int64_t tiles, cudaStream_t st) {
  TcPlan* t = m->tc;
  const int n_chunks = p.n_chunks;
  int64_t pairs = tiles * n_chunks;
  if (pairs > t->grid / 2) pairs = t->grid / 2;
  cudaLaunchAttribute attr[2];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  attr[1].id = cudaLaunchAttributeClusterDimension;
  attr[1].val.clusterDim.x = 2; attr[1].val.clusterDim.y = 1; attr[1].val.clusterDim.z = 1;
  cudaLaunchConfig_t cfg;
  memset(&cfg, 0, sizeof(cfg));
  cfg.stream = st;
  // the first launch of the chain is an ordinary one: it waits for everything queued before it
  cfg.gridDim = dim3((unsigned)(tiles * (2 * kTileM / kSplitEncRows))); cfg.blockDim = dim3(32 * kSplitEncRows);
  DDF_CUDA_TRY(cudaLaunchKernelEx(&cfg, ddf_tc_split_encode_kernel, p));
  cfg.gridDim = dim3((unsigned)(pairs * 2)); cfg.blockDim = dim3(kThreads);
  cfg.dynamicSmemBytes = TcCfg<2>::kSmemBytes; cfg.attrs = attr; cfg.numAttrs = 2;
  for (int l = 0; l < p.n_hidden; ++l)
    DDF_CUDA_TRY(cudaLaunchKernelEx(&cfg, ddf_tc_split_layer_kernel, p, l, t->zpart));
  cfg.gridDim = dim3((unsigned)(tiles * 2)); cfg.blockDim = dim3(128);
  cfg.dynamicSmemBytes = 0; cfg.numAttrs = 1;
  DDF_CUDA_TRY(cudaLaunchKernelEx(&cfg, ddf_tc_split_finish_kernel, p, (const float2*)t->zpart));
  m->last_launches = p.n_hidden + 2;
  return DDF_OK;
}

int tc_forward(Model* m, const float* o, const float* d, int64_t n, const int64_t* n_dev, int mode_out,
               float* out0, float* out1, int spp, float ao_radius, cudaStream_t st) {
  TcPlan* t = m->tc;
  if (!t) return DDF_E_UNSUPPORTED;
  if (t->dbg_host[0] != 0) return DDF_E_CUDA;           // an earlier launch tripped a bounded wait
  TcParams p = t->base;
  p.o = o; p.d = d; p.n = n; p.n_dev = n_dev;
  p.out0 = out0; p.out1 = out1; p.mode_out = mode_out; p.spp = spp > 0 ? spp : 1; p.ao_radius = ao_radius;
  const int64_t tile_rays = (int64_t)kTileM * t->cg;
  int64_t tiles = (n + tile_rays - 1) / tile_rays;
  // small batches: split the output columns of a layer over the CTA pairs (ddf_set_path 3 / 4 pin the choice)
  const int64_t split_max = (m->path == 3 || m->path == 5) ? 0 : (m->path == 4 ? t->grid / 2 : kSplitAutoTiles);
  if (tiles <= split_max) return tc_forward_split(m, p, tiles, st);
  if (m->path == 5 && t->res_ok) {
    // activation-resident kernel: tiles of 128 rays per CTA pair, same equal-tiles grid rule
    const int64_t rtiles = (n + 2 * kResRays - 1) / (2 * kResRays);
    const int64_t units = t->grid / 2, waves = (rtiles + units - 1) / units;
    const int rgrid = (int)((rtiles + waves - 1) / waves) * 2;
    cudaLaunchConfig_t cfg;
    memset(&cfg, 0, sizeof(cfg));
    cfg.gridDim = dim3((unsigned)rgrid); cfg.blockDim = dim3(kThreads); cfg.stream = st;
    cfg.dynamicSmemBytes = t->res_smem;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = 2; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr; cfg.numAttrs = 1;
    DDF_CUDA_TRY(cudaLaunchKernelEx(&cfg, ddf_tc_res_kernel, p));
    m->last_launches = 1;
    return DDF_OK;
  }
  // as many CTAs (pairs) as give every one the same number of tiles (+-1): the last wave of a persistent grid is
  // otherwise part empty, and the CTAs that would idle through it only add L2 contention and power in the others
  const int64_t units = t->grid / t->cg;
  const int64_t waves = (tiles + units - 1) / units;
  int grid = (int)((tiles + waves - 1) / waves) * t->cg;  // <= t->grid; n_dev can only shrink n
  cudaLaunchConfig_t cfg;
  memset(&cfg, 0, sizeof(cfg));
  cfg.gridDim = dim3((unsigned)grid); cfg.blockDim = dim3(kThreads); cfg.stream = st;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeClusterDimension;
  attr[0].val.clusterDim.x = (unsigned)t->cg; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
  cfg.attrs = attr; cfg.numAttrs = 1;
  cfg.dynamicSmemBytes = TcCfg<2>::kSmemBytes;
  DDF_CUDA_TRY(cudaLaunchKernelEx(&cfg, ddf_tc_kernel, p));
  m->last_launches = 1;
  return DDF_OK;
}

}  // namespace ddf
