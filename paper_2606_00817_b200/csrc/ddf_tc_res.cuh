// ddf_tc_res.cuh - the activation-resident tcgen05 kernel (included by ddf_tc.cu).
//
// Same forward pass as ddf_tc_kernel (include/ddf.h; Eq. 1, "Every query is one forward
// pass"), with the layer hand-off kept in shared and tensor memory: no activation is written to global memory.
// The GEMM is transposed, D^T[features x rays] = W[features x K] . H^T[K x rays]:
//
//   A operand  = weights, streamed by TMA (this CTA's 128 of the pair's 256 output features x 64 K per stage)
//   B operand  = activations, RESIDENT in shared memory: 64 rays per CTA x all K, MN-major (row = k, the 64 rays of
//                the CTA contiguous in one 128-byte swizzled row), so cta_group::2 gives M = 256 features x N = 128 rays
//   D          = fp32 in TMEM, 128 lanes (features) x 128 columns (rays of the pair), double buffered (256 columns)
//
// An output chunk (256 features of the pair) cannot overwrite the layer's input while later chunks still read it, so
// the epilogue parks chunks 0 .. nc-2 as packed bf16 in the other 256 TMEM columns (tcgen05.st).  Every chunk walks K
// in natural order (gamma blocks, then input chunks 0 .. nc-1); the layer's LAST output chunk commits to a per-chunk
// "dead" barrier as it leaves each 256-row input chunk behind, and the epilogue copies parked chunk j back over input
// chunk j (tcgen05.ld -> st.shared) as soon as that barrier fires - while the last chunk is still running.  The last
// chunk's own accumulator completes only when every MMA of the layer has, and is written straight into its rows.
// Layer 0 reads gamma, not H, so it writes every chunk directly.  Each CTA computes half of the features for ALL 128
// rays but needs, as its next B operand, all features for ITS 64 rays: the other half of every chunk crosses to the
// peer CTA through distributed shared memory.  The next layer's first output chunk waits per 256-row input chunk
// (mbarriers) for both halves to be in place.  Needs at least two hidden layers: the layer-0 hand-over barriers are
// what keeps a tile's head partials from being overwritten by the next tile (tc_plan_create checks).
//
//   warp 0      TMA producer (weights only)        warps 2-3   encoder: gamma of the next tile, registers -> smem
//   warp 1      MMA issuer (leader CTA)            warps 4-11  epilogue: +bias, ReLU, bf16, park / hand over; heads
//
// The heads need sum_f w[f] h8[f] with f on TMEM lanes: a butterfly transpose-reduce over the 32 lanes of a warp,
// then the 8 warp partials of a ray (4 lane quarters x 2 CTAs) meet in the ray owner's shared memory and are added
// in a fixed order - results do not depend on n or on the ray's position (same contract as ddf_tc_kernel).
#pragma once

namespace ddf {

constexpr int kResRays = 64;                 // rays per CTA; a tile = 128 rays per CTA pair
constexpr int kResStageBytes = 128 * kKBlock * 2;      // one weight tile: 128 features x 64 K = 16 KB
constexpr int kResMaxStages = 8;
constexpr int kResZBytes = 8 * kResRays * 8;           // head partials: 8 slots x 64 rays x (z0, z1)
constexpr int kResBarBytes = 1024;

// dynamic shared memory of the kernel for a (width, E16) network with `stages` weight stages
__host__ __device__ inline size_t res_smem_bytes(int width, int e16, int stages) {
  return 1024 + (size_t)stages * kResStageBytes + (size_t)width * 128 + (size_t)e16 * 128 + kResZBytes + kResBarBytes;
}

__device__ __forceinline__ uint32_t pack_bf16x2(float lo, float hi) {
  __nv_bfloat162 t = __floats2bfloat162_rn(lo, hi);
  return *reinterpret_cast<uint32_t*>(&t);
}

// one K row (128 bytes = 64 rays) of the resident operand: 8 x 16 bytes, 128-byte swizzle.  Into this CTA's own rows:
// plain stores (the caller fences and arrives).  Into the peer's: asynchronous stores that count their bytes on the
// peer's barrier `bar_peer` (a shared::cluster address) - nothing to fence, nothing to wait for.
__device__ __forceinline__ void res_store_row(uint32_t h_base, int row, const uint32_t (&w)[32], bool local, uint32_t peer, uint32_t bar_peer) {
  const uint32_t a = h_base + (uint32_t)row * 128u;
  const uint32_t ar = local ? 0u : ptx::mapa(a, peer);
  #pragma unroll
  for (int i = 0; i < 8; ++i) {
    const uint4 v = make_uint4(w[4 * i], w[4 * i + 1], w[4 * i + 2], w[4 * i + 3]);
    const uint32_t off = (uint32_t)((i ^ (row & 7)) << 4);
    if (local) ptx::st_shared_v4(a + off, v);
    else ptx::st_async_v4(ar + off, v, bar_peer);
  }
}

__global__ void __launch_bounds__(kThreads, 1) ddf_tc_res_kernel(const __grid_constant__ TcParams p) {
  extern __shared__ uint8_t smem_raw[];
  const int S = p.res_stages;
  const uint32_t ring = (ptx::smem_u32(smem_raw) + 1023u) & ~1023u;
  const uint32_t Hs = ring + (uint32_t)S * kResStageBytes;             // [width][64 rays] bf16, MN-major, 128B swizzle
  const uint32_t Gs = Hs + (uint32_t)p.width * 128u;                   // [E16][64 rays]: gamma, kept for the skip layer
  const uint32_t zbuf = Gs + (uint32_t)p.res_e16 * 128u;
  const uint32_t bar = zbuf + kResZBytes;
  auto full_bar   = [&](int s) { return bar + 8u * s; };
  auto empty_bar  = [&](int s) { return bar + 8u * (8 + s); };
  auto tfull_bar  = [&](int b) { return bar + 8u * (16 + b); };
  auto tempty_bar = [&](int b) { return bar + 8u * (18 + b); };
  // chunk j of the next layer's input is in place in THIS CTA: 4 arrivals of the local epilogue warps (one of them
  // announcing the 16 KB the peer's warps send asynchronously) + those bytes
  auto hready_bar = [&](int j) { return bar + 8u * (20 + j); };
  auto pready_bar = [&](int j) { return bar + 8u * (33 + j); };        // leader only: chunk j is in place in the peer CTA too
  const uint32_t gready_bar = bar + 8u * 28, gfree_bar = bar + 8u * 29, zready_bar = bar + 8u * 30;
  // rows of input chunk j are dead: the layer's LAST output chunk (every other one finished before it started) has
  // completed its MMAs over them (tcgen05.commit, both CTAs)
  auto hdead_bar = [&](int j) { return bar + 8u * (41 + j); };
  const uint32_t tmem_slot = bar + 8u * 32;

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint32_t rank = ptx::cluster_ctarank();
  const bool leader = (rank == 0);
  const int pid = blockIdx.x >> 1, num_pairs = gridDim.x >> 1;
  const int64_t n = p.n_dev ? *p.n_dev : p.n;
  const int64_t tile_rays = 2 * kResRays;
  const int64_t num_tiles = (n + tile_rays - 1) / tile_rays;
  const int nc = p.n_chunks, last_layer = p.n_hidden - 1;
  const int gamma_layer = p.skip_layer >= 0 ? p.skip_layer : 0;        // last layer that reads gamma

  if (threadIdx.x == 0) {
    for (int s = 0; s < S; ++s) { ptx::mbar_init(full_bar(s), 1); ptx::mbar_init(empty_bar(s), 1); }
    for (int b = 0; b < 2; ++b) { ptx::mbar_init(tfull_bar(b), 1); ptx::mbar_init(tempty_bar(b), 16); }
    for (int j = 0; j < kMaxChunks; ++j) { ptx::mbar_init(hready_bar(j), 4); ptx::mbar_init(pready_bar(j), 1); ptx::mbar_init(hdead_bar(j), 1); }
    ptx::mbar_init(gready_bar, 4); ptx::mbar_init(gfree_bar, 1); ptx::mbar_init(zready_bar, 8);
    ptx::fence_mbar_init();
  }
  if (warp == 0 && lane == 0)
    for (int l = 0; l < p.n_hidden; ++l) ptx::prefetch_tmap(&p.w[l]);
  if (warp == 2) { ptx::tmem_alloc<2>(tmem_slot, 512); ptx::tmem_relinquish<2>(); }
  ptx::tc_fence_before();
  ptx::cluster_sync();
  ptx::tc_fence_after();
  uint32_t tmem_base;
  asm volatile("ld.shared.u32 %0, [%1];" : "=r"(tmem_base) : "r"(tmem_slot));

  // K-block order of a layer: the gamma blocks first (always in place), then the hidden blocks in natural order, chunk 0
  // .. nc-1; the first output chunk of a layer waits for each input chunk's hand-over as it reaches it.  Producer and
  // issuer walk it with counters only (no division: the issuer's loop must stay well under the 256 clocks its four
  // MMAs of a stage take).
  if (warp == 0) {
    // ================================================================ TMA producer: this CTA's 128 feature rows of each weight tile
    const uint64_t pol_w = ptx::policy_evict_last();
    const uint32_t full0 = ptx::mapa(full_bar(0), 0);
    int s = 0; uint32_t ph = 0;
    auto load = [&](const CUtensorMap* wmap, int wcol, int wrow) {
      wait_bar<true>(empty_bar(s), ph ^ 1u, p.dbg, 0x2300 + s);
      if (ptx::elect_one()) {
        if (leader) ptx::mbar_arrive_expect_tx(full_bar(s), 2u * kResStageBytes);
        ptx::tma_load_2d_cg2_hint(ring + (uint32_t)s * kResStageBytes, wmap, full0 + 8u * s, wcol, wrow, pol_w);
      }
      __syncwarp();
      if (++s == S) { s = 0; ph ^= 1u; }
    };
    for (int64_t tile = pid; tile < num_tiles; tile += num_pairs) {
      for (int l = 0; l < p.n_hidden; ++l) {
        const int ng = (l == 0) ? p.nkb0[0] : p.nkb1[l];
        const int gcol0 = (l == 0) ? 0 : p.nkb0[l] * kKBlock;
        for (int c = 0; c < nc; ++c) {
          const int wrow = c * kChunkN + (int)rank * 128;
          for (int g = 0; g < ng; ++g) load(&p.w[l], gcol0 + g * kKBlock, wrow);
          if (l > 0)
            for (int kb = 0; kb < 4 * nc; ++kb) load(&p.w[l], kb * kKBlock, wrow);
        }
      }
    }
  } else if (warp == 1) {
    // ================================================================ MMA issuer
    if (leader) {
      constexpr uint32_t idesc = ptx::idesc_bf16_f32_major(256, 2 * kResRays, 0, 1);
      const uint64_t adesc0 = ptx::smem_desc_k_sw128(ring), gdesc0 = ptx::smem_desc_mn_sw128(Gs, 8192u), hdesc0 = ptx::smem_desc_mn_sw128(Hs, 8192u);
      int s = 0; uint32_t ph = 0, cc = 0, hphase = 0;
      int tile_local = 0;
      // one stage = one 64-K block: 4 (or fewer, for gamma's last block) MMAs of K = 16.  A advances 32 bytes per step
      // inside its 128-byte rows, the MN-major B 16 rows = 2048 bytes; descriptors carry addresses in 16-byte units.
      auto issue = [&](uint32_t d_tmem, uint64_t bdesc, int nk16, bool first, uint32_t extra_commit) {
        wait_bar<true>(full_bar(s), ph, p.dbg, 0x2500 + s);
        ptx::tc_fence_after();
        const uint64_t adesc = adesc0 + (uint64_t)((uint32_t)s * (kResStageBytes >> 4));
        if (ptx::elect_one()) {
          if (nk16 == 4) {
            ptx::umma_bf16<2>(d_tmem, adesc, bdesc, idesc, first ? 0u : 1u);
            ptx::umma_bf16<2>(d_tmem, adesc + 2u, bdesc + 128u, idesc, 1u);
            ptx::umma_bf16<2>(d_tmem, adesc + 4u, bdesc + 256u, idesc, 1u);
            ptx::umma_bf16<2>(d_tmem, adesc + 6u, bdesc + 384u, idesc, 1u);
          } else {
            for (int k = 0; k < nk16; ++k)
              ptx::umma_bf16<2>(d_tmem, adesc + 2u * k, bdesc + 128u * k, idesc, (first && k == 0) ? 0u : 1u);
          }
          ptx::umma_commit<2>(empty_bar(s));
          if (extra_commit) ptx::umma_commit<2>(extra_commit);
        }
        __syncwarp();
        if (++s == S) { s = 0; ph ^= 1u; }
      };
      for (int64_t tile = pid; tile < num_tiles; tile += num_pairs, ++tile_local) {
        for (int l = 0; l < p.n_hidden; ++l) {
          const int ng = (l == 0) ? p.nkb0[0] : p.nkb1[l];
          for (int c = 0; c < nc; ++c, ++cc) {
            const uint32_t buf = cc & 1u, use = cc >> 1;
            wait_bar<true>(tempty_bar(buf), (use & 1u) ^ 1u, p.dbg, 0x2400 + buf);
            ptx::tc_fence_after();
            const uint32_t d_tmem = tmem_base + buf * (2 * kResRays);
            const bool last_c = c == nc - 1;
            if (l == 0 && c == 0) {
              wait_bar<true>(gready_bar, (uint32_t)(tile_local & 1), p.dbg, 0x2100);
              ptx::tc_fence_after();
            }
            for (int g = 0; g < ng; ++g) {
              const bool glast = g == ng - 1;
              // the last reader of gamma frees it for the encoder; a layer without hidden blocks (layer 0) ends its chunk here
              const uint32_t extra = (glast && l == 0) ? tfull_bar(buf) : ((glast && l == gamma_layer && last_c) ? gfree_bar : 0u);
              issue(d_tmem, gdesc0 + (uint64_t)((uint32_t)g * (kKBlock * 128u >> 4)), glast ? p.g_last_nk16 : 4, g == 0, extra);
            }
            if (l == 0) {
              if (gamma_layer == 0 && last_c && ptx::elect_one()) ptx::umma_commit<2>(gfree_bar);
              __syncwarp();
            } else {
              // the layer's last output chunk frees the input rows chunk by chunk as it walks K: the parked output
              // chunks are copied over them while it is still running (no hand-over at the layer's end to wait for)
              const bool frees = last_c && l < last_layer;
              for (int chunk = 0; chunk < nc; ++chunk) {
                if (c == 0) {
                  wait_bar<true>(hready_bar(chunk), (hphase >> chunk) & 1u, p.dbg, 0x2200 + chunk);
                  wait_bar<true>(pready_bar(chunk), (hphase >> chunk) & 1u, p.dbg, 0x2900 + chunk);
                  hphase ^= (1u << chunk);
                  ptx::fence_proxy_async_smem();                 // the peer's asynchronous stores -> the tensor core's reads
                  ptx::tc_fence_after();
                }
                const uint64_t hd = hdesc0 + (uint64_t)((uint32_t)chunk * (4u * kKBlock * 128u >> 4));
                #pragma unroll
                for (int b = 0; b < 4; ++b)
                  issue(d_tmem, hd + (uint64_t)((uint32_t)b * (kKBlock * 128u >> 4)), 4, ng == 0 && chunk == 0 && b == 0,
                        b < 3 ? 0u : (chunk == nc - 1 ? tfull_bar(buf) : (frees ? hdead_bar(chunk) : 0u)));
              }
            }
          }
        }
      }
    } else {
      // the peer CTA's warp 1 relays "chunk in place here" to the leader, whose MMAs read both CTAs' operands
      uint32_t hphase = 0;
      for (int64_t tile = pid; tile < num_tiles; tile += num_pairs) {
        for (int l = 1; l < p.n_hidden; ++l) {
          for (int chunk = 0; chunk < nc; ++chunk) {
            wait_bar<true>(hready_bar(chunk), (hphase >> chunk) & 1u, p.dbg, 0x2a00 + chunk);
            hphase ^= (1u << chunk);
            ptx::fence_proxy_async_smem();
            __syncwarp();
            if (lane == 0) ptx::mbar_arrive_cluster(ptx::mapa(pready_bar(chunk), 0));
          }
        }
      }
    }
  } else if (warp >= 4) {
    // ================================================================ epilogue (8 warps)
    // warp (q, h): TMEM lanes 32q .. 32q+31 (features) and columns 64h .. 64h+63 of an accumulator = the rays CTA h owns
    const int q = warp & 3, h = (warp - 4) >> 2;
    const bool local = ((uint32_t)h == rank);
    const int fl = q * 32 + lane;                                        // feature inside this CTA's 128 of a chunk
    const uint32_t lane_sel = (uint32_t)(q * 32) << 16;
    const uint32_t tempty_remote = ptx::mapa(tempty_bar(0), 0);
    const uint32_t stash = tmem_base + lane_sel + 4u * kResRays + (uint32_t)h * 32u;    // + 64 columns per parked chunk
    const uint32_t hready_peer = ptx::mapa(hready_bar(0), (uint32_t)h);
    // rows of chunk j written: the local warps publish them to the async proxy and arrive on this CTA's barrier (lane
    // quarter 0 also announces the peer's 16 KB); the warps that sent to the peer have nothing left to do
    auto hand_over = [&](int j) {
      if (local) {
        ptx::fence_proxy_async_smem();
        __syncwarp();
        if (lane == 0) { if (q == 0) ptx::mbar_arrive_expect_tx(hready_bar(j), 128u * 128u); else ptx::mbar_arrive(hready_bar(j)); }
      }
    };
    uint32_t cc = 0, dphase = 0;
    int tile_local = 0;
    for (int64_t tile = pid; tile < num_tiles; tile += num_pairs, ++tile_local) {
      float za[4] = { 0.0f, 0.0f, 0.0f, 0.0f };                           // (z0, z1) of rays 2 lane, 2 lane + 1 of half h (last layer)
      for (int l = 0; l < p.n_hidden; ++l) {
        const float* bias = p.bias + p.b_off[l];
        for (int c = 0; c < nc; ++c, ++cc) {
          const uint32_t buf = cc & 1u, use = cc >> 1;
          const int fg = c * kChunkN + (int)rank * 128 + fl;             // this thread's output feature = next layer's K row
          const float bf = __ldg(bias + fg);
          wait_bar<true>(tfull_bar(buf), use & 1u, p.dbg, 0x2600 + buf);
          ptx::tc_fence_after();
          uint32_t r[64];
          const uint32_t taddr = tmem_base + lane_sel + buf * (2 * kResRays) + (uint32_t)h * kResRays;
          ptx::tmem_ld32(taddr, *reinterpret_cast<uint32_t(*)[32]>(&r[0]));
          ptx::tmem_ld32(taddr + 32, *reinterpret_cast<uint32_t(*)[32]>(&r[32]));
          ptx::tmem_ld_wait();
          ptx::tc_fence_before();
          __syncwarp();
          if (lane == 0) ptx::mbar_arrive_cluster(tempty_remote + 8u * buf);       // accumulator read: back to the MMA warp
          if (l < last_layer) {
            uint32_t w[32];
            #pragma unroll
            for (int i = 0; i < 32; ++i)
              w[i] = pack_bf16x2(fmaxf(__uint_as_float(r[2 * i]) + bf, 0.0f), fmaxf(__uint_as_float(r[2 * i + 1]) + bf, 0.0f));
            if (l == 0 || c == nc - 1) {
              // layer 0 reads gamma, not H (whose rows the tile before has finished with); a last chunk's accumulator
              // completes only when every MMA of the layer has: either way the rows are dead in both CTAs
              res_store_row(Hs, fg, w, local, (uint32_t)h, hready_peer + 8u * c);
              hand_over(c);
            } else {
              ptx::tmem_st32(stash + (uint32_t)c * kResRays, w);          // park: the layer's input is still being read
              ptx::tmem_st_wait();
              if (c == nc - 2) {
                // the last chunk is now walking K and frees the input chunk by chunk: copy the parked chunks over it
                for (int j = 0; j < nc - 1; ++j) {
                  wait_bar<true>(hdead_bar(j), (dphase >> j) & 1u, p.dbg, 0x2b00 + j);
                  dphase ^= (1u << j);
                  ptx::tc_fence_after();
                  ptx::tmem_ld32(stash + (uint32_t)j * kResRays, w);
                  ptx::tmem_ld_wait();
                  res_store_row(Hs, j * kChunkN + (int)rank * 128 + fl, w, local, (uint32_t)h, hready_peer + 8u * j);
                  hand_over(j);
                }
                ptx::tc_fence_before();
              }
            }
          } else {
            // heads: this warp's 32 features x 64 rays -> per-ray partial sums, lane L ends with rays 2L, 2L+1
            #pragma unroll
            for (int o = 0; o < 2; ++o) {
              if (o == 1 && p.n_out != 2) break;
              const float hw = __ldg(p.head_w + o * p.width + fg);
              float v[32];
              const bool up16 = (lane & 16) != 0;
              #pragma unroll
              for (int i = 0; i < 32; ++i) {
                const float a = fmaxf(__uint_as_float(r[i]) + bf, 0.0f) * hw, b = fmaxf(__uint_as_float(r[i + 32]) + bf, 0.0f) * hw;
                v[i] = (up16 ? b : a) + __shfl_xor_sync(0xffffffffu, up16 ? a : b, 16);
              }
              #define DDF_RES_FOLD(half, m) { const bool up = (lane & m) != 0; _Pragma("unroll") for (int i = 0; i < half; ++i) \
                  v[i] = (up ? v[i + half] : v[i]) + __shfl_xor_sync(0xffffffffu, up ? v[i] : v[i + half], m); }
              DDF_RES_FOLD(16, 8) DDF_RES_FOLD(8, 4) DDF_RES_FOLD(4, 2) DDF_RES_FOLD(2, 1)
              #undef DDF_RES_FOLD
              // after masks 16, 8, 4, 2, 1 two values remain: rays 2 lane and 2 lane + 1
              za[o] += v[0]; za[2 + o] += v[1];
            }
          }
        }
      }
      // ---- heads: the 8 partials of a ray (slot = 4 rank + q) meet in the shared memory of the CTA that owns the ray
      {
        const uint32_t a = zbuf + (uint32_t)(((int)rank * 4 + q) * kResRays + 2 * lane) * 8u;
        const uint4 v = make_uint4(__float_as_uint(za[0]), __float_as_uint(za[1]), __float_as_uint(za[2]), __float_as_uint(za[3]));
        if (local) ptx::st_shared_v4(a, v); else ptx::st_cluster_v4(ptx::mapa(a, (uint32_t)h), v);
        __syncwarp();
        if (lane == 0) ptx::mbar_arrive_release_cluster(ptx::mapa(zready_bar, (uint32_t)h));
      }
      if (warp < 6) {                                                      // warps 4, 5: one thread per ray of this CTA
        const int j = (warp - 4) * 32 + lane;
        wait_bar<true>(zready_bar, (uint32_t)(tile_local & 1), p.dbg, 0x2700);
        ptx::fence_acq_rel_cluster();
        float z0 = 0.0f, z1 = 0.0f;
        #pragma unroll
        for (int sl = 0; sl < 8; ++sl) {
          float y0, y1;
          asm volatile("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(y0), "=f"(y1) : "r"(zbuf + (uint32_t)(sl * kResRays + j) * 8u) : "memory");
          z0 += y0; z1 += y1;
        }
        z0 += p.bias[p.b_off[p.n_hidden]];
        if (p.n_out == 2) z1 += p.bias[p.b_off[p.n_hidden] + 1];
        const int64_t grow = tile * tile_rays + (int64_t)rank * kResRays + j;
        const bool valid = grow < n;
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
    }
  } else {
    // ================================================================ encoder (warps 2, 3): one ray per thread, registers -> shared memory
    const int j = (warp - 2) * 32 + lane;
    int tile_local = 0;
    for (int64_t tile = pid; tile < num_tiles; tile += num_pairs, ++tile_local) {
      const int64_t grow = tile * tile_rays + (int64_t)rank * kResRays + j;
      __align__(16) __nv_bfloat16 enc[128];
      #pragma unroll 1
      for (int k = 0; k < p.res_e16; ++k) enc[k] = __float2bfloat16_rn(0.0f);
      float v[3], w[3];
      load_ray_vec3(p.o, grow - lane, n, lane, v);                         // coalesced 16-byte loads, regrouped by shuffles
      if (p.input_kind == 0) load_ray_vec3(p.d, grow - lane, n, lane, w);
      if (grow < n) {
        encode_vec_bf16(v, p.Lo, enc);
        if (p.input_kind == 0) encode_vec_bf16(w, p.Ld, enc + 3 + 6 * p.Lo);
      }
      // gamma of the tile before is read until the skip layer's last chunk: one buffer, freed by that MMA's commit
      wait_bar<true>(gfree_bar, (uint32_t)((tile_local & 1) ^ 1), p.dbg, 0x2800);
      const uint32_t col = (uint32_t)(j & 7) * 2u, chunk16 = (uint32_t)(j >> 3);
      #pragma unroll 1
      for (int k = 0; k < p.res_e16; ++k) {
        const uint32_t a = Gs + (uint32_t)k * 128u + ((chunk16 ^ (uint32_t)(k & 7)) << 4) + col;
        asm volatile("st.shared.b16 [%0], %1;" :: "r"(a), "h"(*reinterpret_cast<const uint16_t*>(&enc[k])) : "memory");
      }
      ptx::fence_proxy_async_smem();
      __syncwarp();
      if (lane == 0) ptx::mbar_arrive_release_cluster(ptx::mapa(gready_bar, 0));
    }
  }

  ptx::tc_fence_before();
  ptx::cluster_sync();
  if (warp == 2) ptx::tmem_dealloc<2>(tmem_base, 512);
}

}  // namespace ddf
